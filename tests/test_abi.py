"""CPU checks of the boundary: libprepos.so builds, loads, and exports every symbol include/prepos.h declares;
host-only entry points behave; compute entry points fail loudly without a device (no CPU fallback)."""
import ctypes as C
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_29565_b200 import build, prepos
    build.build()
    return prepos.lib()


def _declared():
    src = open(os.path.join(ROOT, "include", "prepos.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(prepos_[a-z_0-9]+)\s*\(", src)))


def test_exports_every_declared_symbol(lib):
    from paper_2606_29565_b200 import prepos
    names = _declared()
    assert len(names) >= 14
    for n in names:
        assert hasattr(lib, n), f"libprepos.so does not export {n}"
    assert sorted(prepos.EXPORTS) == names, "binding and header disagree on the export list"


def test_record_is_48_bytes_and_codes(lib):
    from paper_2606_29565_b200 import prepos
    hdr_version = int(re.search(r"#define PREPOS_VERSION (\d+)", open(os.path.join(ROOT, "include", "prepos.h")).read()).group(1))
    assert lib.prepos_version() == hdr_version == prepos.ABI_VERSION    # the binding refuses any other build
    assert prepos.RECORD_BYTES == 48
    hdr = open(os.path.join(ROOT, "include", "prepos.h")).read()
    for name, val in (("PREPOS_SERVED", 0), ("PREPOS_GAP_BELOW_TAU", 1), ("PREPOS_NOT_IN_FAST_SET", 2),
                      ("PREPOS_STALE_OR_INVALID", 3), ("PREPOS_INELIGIBLE", 4)):
        assert re.search(rf"{name} = {val}\b", hdr)
    assert "no CPU fallback" in prepos.strerror(prepos.E_NO_DEVICE)


def test_fastset_build_host(lib):
    from paper_2606_29565_b200 import prepos
    bm = prepos.fastset_build([0, 31, 32, 99], 100)
    assert bm.numel() == 4
    words = [int(w) & 0xFFFFFFFF for w in bm]
    assert words[0] == (1 | (1 << 31)) and words[1] == 1 and words[2] == 0 and words[3] == 1 << 3
    with pytest.raises(prepos.PreposError):
        prepos.fastset_build([100], 100)


def test_workspace_and_shape_checks(lib):
    from paper_2606_29565_b200 import prepos
    ok = prepos.ModelShape(32, 32, 8, 128, 4096, 128256, 16)
    assert lib.prepos_workspace_bytes(C.byref(ok), 64) > 0
    for bad in (prepos.ModelShape(32, 32, 5, 128, 4096, 128256, 16),     # Hq % Hkv
                prepos.ModelShape(32, 32, 8, 100, 4096, 128256, 16),     # head_dim % 8
                prepos.ModelShape(32, 32, 8, 128, 4100, 128256, 16),     # hidden % 128
                prepos.ModelShape(32, 32, 8, 128, 4096, 1, 16),          # vocab < 2
                prepos.ModelShape(32, 32, 8, 128, 4096, 128256, 12)):    # page not a power of two
        assert lib.prepos_workspace_bytes(C.byref(bad), 64) == 0


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-device behaviour")
def test_fails_loudly_without_device(lib):
    from paper_2606_29565_b200 import prepos
    with pytest.raises(prepos.PreposError) as e:
        prepos.Context(1, 4, 2, 64, 256, 1024)
    assert e.value.status == prepos.E_NO_DEVICE
    h = C.c_void_p()
    sh = prepos.ModelShape(1, 4, 2, 64, 256, 1024, 16)
    buf = torch.empty(1 << 20, dtype=torch.uint8)
    st = lib.prepos_ctx_create(C.byref(h), C.byref(sh), 1, C.c_void_p(buf.data_ptr()), buf.numel())
    assert st == prepos.E_NO_DEVICE and not h.value
    # compute entry points reject a null ctx instead of computing anything
    assert lib.prepos_gate_serve(None, 1, None, None, None, None, None, 3.0, 0, None, None, None) == prepos.E_INVALID_ARG
    assert lib.prepos_ready_dist(None, 1, None, None, None, None, None, None, None, None, None, None, None) == prepos.E_INVALID_ARG


def test_noalloc_scan_checks_its_fixed_limits_before_anything_else(lib):
    """prepos_scan_logits_noalloc (the entry point for callers that cannot allocate): sizes beyond its built-in
    scratch are refused with their own status on any box; the header's byte count is what the limits imply."""
    from paper_2606_29565_b200 import prepos
    hdr = open(os.path.join(ROOT, "include", "prepos.h")).read()
    assert re.search(r"#define PREPOS_SCAN_NOALLOC_MAX_ROWS 32\b", hdr) and prepos.SCAN_NOALLOC_MAX_ROWS == 32
    assert re.search(r"#define PREPOS_SCAN_NOALLOC_MAX_VOCAB \(1 << 24\)", hdr) and prepos.SCAN_NOALLOC_MAX_VOCAB == 1 << 24
    assert re.search(r"PREPOS_E_FIXED_SCRATCH = -7\b", hdr) and prepos.E_FIXED_SCRATCH == -7
    f = lib.prepos_scan_logits_noalloc
    assert f(33, 1024, None, None, None) == prepos.E_FIXED_SCRATCH
    assert f(1, (1 << 24) + 1, None, None, None) == prepos.E_FIXED_SCRATCH
    assert f(-1, 1024, None, None, None) == prepos.E_INVALID_ARG and f(1, 1, None, None, None) == prepos.E_INVALID_ARG
    assert f(0, 1024, None, None, None) == prepos.OK
    assert f(1, 1024, None, None, None) == prepos.E_INVALID_ARG      # null pointers
    assert "prepos_scan_logits" in prepos.strerror(prepos.E_FIXED_SCRATCH)
    if not torch.cuda.is_available():
        buf = torch.zeros(1024 + 16, dtype=torch.float32)
        assert f(1, 1024, buf.data_ptr(), (buf.data_ptr() + 15) // 16 * 16, None) == prepos.E_NO_DEVICE


def test_product_never_imports_oracle():
    """The product path must not route through the oracle (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_2606_29565_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f
                assert "prepos_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2606_29565_b200\b", txt, flags=re.M), f
            assert not re.search(r"#\s*include\s*[<\"][^>\"]*(prepos\.h|\.cuh)", txt), f

"""prepos_scan_logits_noalloc: the vocabulary scan for callers that cannot allocate device memory.

A serving engine usually gives the whole GPU to its own memory pool at start-up; code running inside its request
handler (where the paper's fast path lives, Alg. 2 l.3-4) cannot count on cudaMalloc to succeed,
and cannot afford the device-wide stall when it does.  The same goes for a plug-in loaded into a process whose
allocator it does not control.  For them the library has ONE entry point whose scratch is a fixed array inside
libprepos.so (65 792 bytes per GPU, at most 32 rows of at most 2^24 logits per call) and which takes no ctx, so no
workspace either.

This file checks that entry point against the ordinary one (prepos_scan_logits through a Context with a
torch-allocated workspace) on two calls in a row -- the second finds the first one's leftovers in the shared array --
and that requests beyond the fixed limits are refused.  It is named test_zz_* so that pytest collects it last: a
failure here must not hide the other GPU tests behind `-x`.  It needs nothing from the tests before it and passes in
a fresh process as well.
"""
import numpy as np
import pytest
import torch

from paper_2606_29565_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def prepos():
    from paper_2606_29565_b200 import prepos as p
    p.lib()
    return p


def _stamped_records(prepos, n):
    """A record table whose caller-owned fields (version, entry_hash, position, VALID bit) are set: the scan must
    leave them alone."""
    recs = prepos.new_records(n)
    q = recs.view(torch.int64).view(-1, 6)
    q[:, 3] = torch.arange(n, device="cuda") + 7        # version
    q[:, 4] = 0x1234                                     # entry_hash
    q[:, 5] = torch.arange(n, device="cuda") + 4096     # position
    recs.view(torch.int32).view(-1, 12)[:, 5] = prepos.FLAG_VALID
    return recs


def _same_records(prepos, got, want):
    """The no-allocation path against the existing path, at the tolerances test_gpu_ready_dist.py uses for the scan
    (ids exact; max 1e-6, gap 1e-5, lse 1e-4 relative)."""
    a, b = prepos.unpack_records(got), prepos.unpack_records(want)
    n = a["top1"].numel()
    for r in range(n):
        assert (int(a["top1"][r]), int(a["top2"][r])) == (int(b["top1"][r]), int(b["top2"][r])), r
        if int(b["flags"][r]) & prepos.FLAG_NONFINITE:
            continue    # a NaN/Inf logit: the flag is the contract (never served), max/lse/gap are not numbers
        assert abs(float(a["max_logit"][r]) - float(b["max_logit"][r])) < 1e-6
        assert abs(float(a["gap"][r]) - float(b["gap"][r])) < 1e-5
        assert abs(float(a["lse"][r]) - float(b["lse"][r])) <= 1e-4 * abs(float(b["lse"][r]))
    for k in ("flags", "version", "entry_hash", "position"):
        assert torch.equal(a[k], b[k]), k


def test_two_calls_in_a_row_match_the_allocating_path(prepos, oracle):
    V = 128256
    g = synth.gen(31, "cuda")
    # call 1 fills the fixed array to its maximum (32 rows); call 2 is a different, smaller batch that meets those
    # leftovers, has exact ties and a non-finite row
    lg1 = torch.randn((prepos.SCAN_NOALLOC_MAX_ROWS, V), generator=g, device="cuda", dtype=torch.float32) * 2
    lg2 = torch.randn((3, V), generator=g, device="cuda", dtype=torch.float32) * 3
    lg2[1] = (lg2[1] * 4).round() / 4
    lg2[2, 777] = float("inf")
    ctx = prepos.Context(1, 4, 2, 64, 128, V, 16, max_sessions=4)
    want1, want2 = _stamped_records(prepos, lg1.shape[0]), _stamped_records(prepos, 3)
    ctx.scan_logits(lg1, want1)
    ctx.scan_logits(lg2, want2)
    ctx.sync()

    got1, got2 = _stamped_records(prepos, lg1.shape[0]), _stamped_records(prepos, 3)
    prepos.scan_logits_noalloc(lg1, got1)        # first call on this device: looks up the array's address
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    prepos.scan_logits_noalloc(lg2, got2)        # second call, back to back on the same stream
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after >= free_before, "the no-allocation entry point took device memory"

    _same_records(prepos, got1, want1)
    _same_records(prepos, got2, want2)
    rec2 = prepos.unpack_records(got2)
    assert int(rec2["flags"][2]) == prepos.FLAG_VALID | prepos.FLAG_NONFINITE
    # and against the oracle directly, so that this file stands on its own
    for r in (0, 1):
        ref = oracle.record(lg2[r].cpu().numpy().astype(np.float64))
        assert (int(rec2["top1"][r]), int(rec2["top2"][r])) == (ref.top1, ref.top2)
        assert abs(float(rec2["gap"][r]) - ref.gap) < 1e-5
        assert abs(float(rec2["lse"][r]) - ref.lse) <= 1e-4 * abs(ref.lse)

    # an odd vocabulary (rows not 16-byte aligned) and a tiny one, again after the array was used
    for V2 in (1023, 5):
        lg = torch.randn((2, V2), generator=g, device="cuda", dtype=torch.float32)
        c2 = prepos.Context(1, 4, 2, 64, 128, V2, 16, max_sessions=4)
        want, got = _stamped_records(prepos, 2), _stamped_records(prepos, 2)
        c2.scan_logits(lg, want)
        prepos.scan_logits_noalloc(lg, got)
        torch.cuda.synchronize()
        _same_records(prepos, got, want)


def test_requests_beyond_the_fixed_array_are_refused(prepos):
    recs = prepos.new_records(prepos.SCAN_NOALLOC_MAX_ROWS + 1)
    before = recs.clone()
    lg = torch.zeros((prepos.SCAN_NOALLOC_MAX_ROWS + 1, 64), dtype=torch.float32, device="cuda")
    with pytest.raises(prepos.PreposError) as e:
        prepos.scan_logits_noalloc(lg, recs)
    assert e.value.status == prepos.E_FIXED_SCRATCH and "prepos_scan_logits" in str(e.value)
    st = prepos.lib().prepos_scan_logits_noalloc(1, prepos.SCAN_NOALLOC_MAX_VOCAB + 1, lg.data_ptr(), recs.data_ptr(), None)
    assert st == prepos.E_FIXED_SCRATCH
    torch.cuda.synchronize()
    assert torch.equal(recs, before)
    prepos.scan_logits_noalloc(lg[:0], recs)     # n = 0: nothing to do

"""Thin ctypes binding of libprepos (include/prepos.h).  Same names as the C ABI; argument
marshalling only -- every step of the hot path runs in the library's CUDA kernels.

PyTorch is used for device memory and streams: tensors are passed as `data_ptr()`, the launch stream
is `torch.cuda.current_stream()`.  There is no CPU fallback: if libprepos.so is missing, cannot be
loaded, or no sm_100 device is present, every call raises.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libprepos.so")   # the in-tree build, and nothing else
ABI_VERSION = 101                            # PREPOS_VERSION of the include/prepos.h this binding marshals for

OK, SKIPPED_BUDGET = 0, 1
E_INVALID_ARG, E_SHAPE, E_ALIGN, E_CUDA, E_WORKSPACE, E_NO_DEVICE, E_FIXED_SCRATCH = -1, -2, -3, -4, -5, -6, -7
SERVED, GAP_BELOW_TAU, NOT_IN_FAST_SET, STALE_OR_INVALID, INELIGIBLE = 0, 1, 2, 3, 4
FLAG_VALID, FLAG_NONFINITE, FLAG_MASK = 1, 2, 3
RECORD_BYTES = 48
SCAN_NOALLOC_MAX_ROWS, SCAN_NOALLOC_MAX_VOCAB = 32, 1 << 24   # PREPOS_SCAN_NOALLOC_* of include/prepos.h

EXPORTS = [
    "prepos_strerror", "prepos_version", "prepos_workspace_bytes", "prepos_ctx_create", "prepos_ctx_destroy",
    "prepos_ctx_sync", "prepos_ctx_launch_count", "prepos_ctx_set_attn_path", "prepos_entry_attn", "prepos_entry_attn_fp8",
    "prepos_ctx_request_yield", "prepos_entry_attn_resume", "prepos_entry_attn_pending", "prepos_ctx_set_attn_slice",
    "prepos_ctx_set_kv_prefetch",
    "prepos_ready_dist", "prepos_ready_dist_w4", "prepos_scan_logits", "prepos_scan_logits_noalloc", "prepos_gate_serve", "prepos_invalidate", "prepos_gate_sweep",
    "prepos_fastset_build",
]


class PreposError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {strerror(status)} (status {status})")


class ModelShape(C.Structure):
    _fields_ = [("layers", C.c_int32), ("n_q_heads", C.c_int32), ("n_kv_heads", C.c_int32), ("head_dim", C.c_int32),
                ("hidden", C.c_int32), ("vocab", C.c_int32), ("page_size", C.c_int32)]


_lib = None


def lib() -> C.CDLL:
    """Loads libprepos.so (built in-tree by paper_2606_29565_b200.build).  Raises if it is absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise RuntimeError(f"{_SO} is missing: run `python -m paper_2606_29565_b200.build` "
                               "(libprepos has no CPU fallback)")
        L = C.CDLL(_SO)
        vp, i32, i64, f32 = C.c_void_p, C.c_int, C.c_int64, C.c_float
        L.prepos_strerror.restype = C.c_char_p
        L.prepos_strerror.argtypes = [i32]
        L.prepos_version.restype = i32
        if L.prepos_version() != ABI_VERSION:
            raise RuntimeError(f"{_SO} is version {L.prepos_version()}, this binding marshals for {ABI_VERSION}: "
                               "rebuild it (`python -m paper_2606_29565_b200.build --force`)")
        L.prepos_workspace_bytes.restype = C.c_size_t
        L.prepos_workspace_bytes.argtypes = [C.POINTER(ModelShape), i32]
        L.prepos_ctx_create.restype = i32
        L.prepos_ctx_create.argtypes = [C.POINTER(vp), C.POINTER(ModelShape), i32, vp, C.c_size_t]
        L.prepos_ctx_destroy.restype = i32
        L.prepos_ctx_destroy.argtypes = [vp]
        L.prepos_ctx_sync.restype = i32
        L.prepos_ctx_sync.argtypes = [vp, vp]
        L.prepos_ctx_launch_count.restype = i64
        L.prepos_ctx_launch_count.argtypes = [vp]
        L.prepos_ctx_set_attn_path.restype = i32
        L.prepos_ctx_set_attn_path.argtypes = [vp, i32]
        L.prepos_entry_attn.restype = i32
        L.prepos_entry_attn.argtypes = [vp, i32, i32, i32, vp, i64, vp, vp, i64, vp, vp, i64, i64, vp, i32, vp, vp, vp,
                                        vp, i64, vp, f32, vp]
        L.prepos_entry_attn_fp8.restype = i32
        L.prepos_entry_attn_fp8.argtypes = [vp, i32, i32, i32, vp, i64, vp, vp, i64, vp, vp, i64, i64, vp, vp, i64, vp, i32,
                                            vp, vp, vp, vp, i64, vp, f32, vp]
        L.prepos_ctx_request_yield.restype = i32
        L.prepos_ctx_request_yield.argtypes = [vp, vp]
        L.prepos_entry_attn_resume.restype = i32
        L.prepos_entry_attn_resume.argtypes = [vp, vp]
        L.prepos_entry_attn_pending.restype = i32
        L.prepos_entry_attn_pending.argtypes = [vp, vp, C.POINTER(C.c_int32)]
        L.prepos_ctx_set_attn_slice.restype = i32
        L.prepos_ctx_set_attn_slice.argtypes = [vp, i32]
        L.prepos_ctx_set_kv_prefetch.restype = i32
        L.prepos_ctx_set_kv_prefetch.argtypes = [vp, i32]
        L.prepos_ready_dist.restype = i32
        L.prepos_ready_dist.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
        L.prepos_ready_dist_w4.restype = i32
        L.prepos_ready_dist_w4.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
        L.prepos_scan_logits.restype = i32
        L.prepos_scan_logits.argtypes = [vp, i32, vp, vp, vp]
        L.prepos_scan_logits_noalloc.restype = i32
        L.prepos_scan_logits_noalloc.argtypes = [i32, i32, vp, vp, vp]
        L.prepos_gate_serve.restype = i32
        L.prepos_gate_serve.argtypes = [vp, i32, vp, vp, vp, vp, vp, f32, i32, vp, vp, vp]
        L.prepos_invalidate.restype = i32
        L.prepos_invalidate.argtypes = [vp, i32, vp, vp, vp, vp]
        L.prepos_gate_sweep.restype = i32
        L.prepos_gate_sweep.argtypes = [vp, i32, vp, vp, vp, vp, i32, vp, i32, vp, vp]
        L.prepos_fastset_build.restype = i32
        L.prepos_fastset_build.argtypes = [vp, i32, i32, vp]
        _lib = L
    return _lib


def strerror(status: int) -> str:
    return lib().prepos_strerror(int(status)).decode()


def _check(status: int, where: str) -> int:
    if status < 0:
        raise PreposError(status, where)
    return status


def _p(t):
    """device/host pointer of a tensor as a plain int (None -> NULL); ctypes converts it per the argtypes"""
    return None if t is None else t.data_ptr()


def _stream():
    return torch.cuda.current_stream().cuda_stream


def _host_i32(v) -> torch.Tensor:
    if isinstance(v, torch.Tensor):
        assert v.device.type == "cpu"
        return v.to(torch.int32).contiguous()
    return torch.tensor(list(v), dtype=torch.int32)


def fastset_build(ids, V: int) -> torch.Tensor:
    """prepos_fastset_build: host int32 ids -> host bitmap (int32 tensor holding the uint32 words)."""
    ids = _host_i32(ids)
    bm = torch.zeros((V + 31) // 32, dtype=torch.int32)
    _check(lib().prepos_fastset_build(_p(ids), ids.numel(), V, _p(bm)), "prepos_fastset_build")
    return bm


def scan_logits_noalloc(logits: torch.Tensor, records_out: torch.Tensor):
    """prepos_scan_logits_noalloc on the current stream: the scan of stored logits for callers that cannot allocate
    device memory (no Context, hence no workspace; the kernel's scratch is a fixed array inside libprepos.so).
    logits [n, V] fp32 on the current device, n <= SCAN_NOALLOC_MAX_ROWS, V <= SCAN_NOALLOC_MAX_VOCAB (beyond that:
    PreposError with status E_FIXED_SCRATCH); records_out a record table with at least n rows.  One scratch array per
    GPU is shared by every call: do not let two calls overlap on the same GPU.  Make the first call on each device
    during start-up (it looks up the array's address once)."""
    assert logits.dtype == torch.float32 and logits.dim() == 2 and logits.is_contiguous()
    _check(lib().prepos_scan_logits_noalloc(logits.shape[0], logits.shape[1], _p(logits), _p(records_out), _stream()),
           "prepos_scan_logits_noalloc")


def new_records(n_sessions: int, device="cuda") -> torch.Tensor:
    """Zeroed record table: [n_sessions, 48] uint8 (see unpack_records)."""
    return torch.zeros((n_sessions, RECORD_BYTES), dtype=torch.uint8, device=device)


def unpack_records(records: torch.Tensor) -> dict:
    """Record table -> dict of host tensors (field views; no arithmetic)."""
    r = records.detach().cpu().contiguous()
    f = r.view(torch.float32).view(-1, 12)
    i = r.view(torch.int32).view(-1, 12)
    q = r.view(torch.int64).view(-1, 6)
    return {"max_logit": f[:, 0].clone(), "lse": f[:, 1].clone(), "top1": i[:, 2].clone(), "top2": i[:, 3].clone(),
            "gap": f[:, 4].clone(), "flags": i[:, 5] & FLAG_MASK, "seq": (i[:, 5] >> 2) & 0x3FFFFFFF,
            "version": q[:, 3].clone(),
            "entry_hash": q[:, 4].clone(), "position": q[:, 5].clone()}


SWEEP_POINT_BYTES = 64


def unpack_sweep(points: torch.Tensor) -> dict:
    """prepos_sweep_point table -> dict of host tensors (field views; no arithmetic)."""
    r = points.detach().cpu().contiguous()
    f = r.view(torch.float32).view(-1, 16)
    i = r.view(torch.int32).view(-1, 16)
    d = r.view(torch.float64).view(-1, 8)
    return {"tau": f[:, 0].clone(), "n": i[:, 1].clone(), "accepted": i[:, 2].clone(), "false_accepts": i[:, 3].clone(),
            "coverage": d[:, 2].clone(), "far": d[:, 3].clone(), "cov_lo": d[:, 4].clone(), "cov_hi": d[:, 5].clone(),
            "far_lo": d[:, 6].clone(), "far_hi": d[:, 7].clone()}


class Context:
    """prepos_ctx with a torch-allocated workspace."""

    def __init__(self, layers, n_q_heads, n_kv_heads, head_dim, hidden, vocab, page_size=16, max_sessions=64,
                 device=None):
        L = lib()
        if not torch.cuda.is_available():
            raise PreposError(E_NO_DEVICE, "prepos_ctx_create")
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        self.shape = ModelShape(layers, n_q_heads, n_kv_heads, head_dim, hidden, vocab, page_size)
        self.max_sessions = max_sessions
        nbytes = L.prepos_workspace_bytes(C.byref(self.shape), max_sessions)
        if nbytes == 0:
            raise PreposError(E_SHAPE, "prepos_workspace_bytes")
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = (self.workspace.data_ptr() + 255) // 256 * 256
        self._h = C.c_void_p()
        with torch.cuda.device(self.device):
            _check(L.prepos_ctx_create(C.byref(self._h), C.byref(self.shape), max_sessions, C.c_void_p(base), nbytes),
                   "prepos_ctx_create")

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().prepos_ctx_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- accounting / knobs
    def launch_count(self) -> int:
        return int(lib().prepos_ctx_launch_count(self._h))

    def set_attn_path(self, path: int):
        _check(lib().prepos_ctx_set_attn_path(self._h, int(path)), "prepos_ctx_set_attn_path")

    def sync(self):
        _check(lib().prepos_ctx_sync(self._h, _stream()), "prepos_ctx_sync")

    # ---- the hot path
    def entry_attn(self, q, k_new, v_new, k_pool, v_pool, page_table, n_s, l_entry, capacity_tokens, out,
                   layer_begin=0, layer_end=None, softmax_scale=0.0):
        """prepos_entry_attn.  q/out [layers, sum_L, Hq, d]; k_new/v_new [layers, sum_L, Hkv, d];
        pools [layers, n_pages, Hkv, page, d] (bf16, device); page_table [n_sessions, stride] int32 device;
        n_s/l_entry/capacity_tokens host ints.  Returns the per-session status list."""
        n_s, l_entry, cap = _host_i32(n_s), _host_i32(l_entry), _host_i32(capacity_tokens)
        n = n_s.numel()
        layer_end = self.shape.layers if layer_end is None else layer_end
        status = torch.zeros(n, dtype=torch.int32)
        for t in (q, k_new, v_new, k_pool, v_pool, out):
            assert t.dtype == torch.bfloat16 and t.is_cuda
        assert page_table.dtype == torch.int32 and page_table.is_cuda and page_table.stride(1) == 1
        st = lib().prepos_entry_attn(
            self._h, layer_begin, layer_end, n,
            _p(q), q.stride(0), _p(k_new), _p(v_new), k_new.stride(0),
            _p(k_pool), _p(v_pool), k_pool.stride(0), k_pool.shape[1],
            _p(page_table), page_table.stride(0), _p(n_s), _p(l_entry), _p(cap),
            _p(out), out.stride(0), _p(status), float(softmax_scale), _stream())
        _check(st, "prepos_entry_attn")
        return status.tolist()

    def entry_attn_fp8(self, q, k_new, v_new, k_pool8, v_pool8, k_scale, v_scale, page_table, n_s, l_entry,
                       capacity_tokens, out, layer_begin=0, layer_end=None, softmax_scale=0.0):
        """prepos_entry_attn_fp8.  Pools [layers, n_pages, Hkv, page, d] uint8 (e4m3 codes), scales
        [layers, n_pages, Hkv] float32; everything else as entry_attn."""
        n_s, l_entry, cap = _host_i32(n_s), _host_i32(l_entry), _host_i32(capacity_tokens)
        n = n_s.numel()
        layer_end = self.shape.layers if layer_end is None else layer_end
        status = torch.zeros(n, dtype=torch.int32)
        for t in (q, k_new, v_new, out):
            assert t.dtype == torch.bfloat16 and t.is_cuda
        assert k_pool8.dtype == torch.uint8 and v_pool8.dtype == torch.uint8 and k_pool8.is_cuda and v_pool8.is_cuda
        assert k_scale.dtype == torch.float32 and v_scale.dtype == torch.float32 and k_scale.stride(0) == v_scale.stride(0)
        assert page_table.dtype == torch.int32 and page_table.is_cuda and page_table.stride(1) == 1
        st = lib().prepos_entry_attn_fp8(
            self._h, layer_begin, layer_end, n,
            _p(q), q.stride(0), _p(k_new), _p(v_new), k_new.stride(0),
            _p(k_pool8), _p(v_pool8), k_pool8.stride(0), k_pool8.shape[1],
            _p(k_scale), _p(v_scale), k_scale.stride(0),
            _p(page_table), page_table.stride(0), _p(n_s), _p(l_entry), _p(cap),
            _p(out), out.stride(0), _p(status), float(softmax_scale), _stream())
        _check(st, "prepos_entry_attn_fp8")
        return status.tolist()

    def request_yield(self):
        """prepos_ctx_request_yield on the current stream (use the request's high-priority stream)."""
        _check(lib().prepos_ctx_request_yield(self._h, _stream()), "prepos_ctx_request_yield")

    def entry_attn_resume(self):
        _check(lib().prepos_entry_attn_resume(self._h, _stream()), "prepos_entry_attn_resume")

    def entry_attn_pending(self) -> bool:
        out = C.c_int32(0)
        _check(lib().prepos_entry_attn_pending(self._h, _stream(), C.byref(out)), "prepos_entry_attn_pending")
        return bool(out.value)

    def set_attn_slice(self, max_segments_per_launch: int):
        _check(lib().prepos_ctx_set_attn_slice(self._h, int(max_segments_per_launch)), "prepos_ctx_set_attn_slice")

    def set_kv_prefetch(self, on: bool):
        _check(lib().prepos_ctx_set_kv_prefetch(self._h, int(bool(on))), "prepos_ctx_set_kv_prefetch")

    def ready_dist(self, session_ids, hidden, w_vocab, records, session_version, position_p=None, entry_hash=None,
                   skip_mask=None, logits_out=None, expected_version=None):
        """prepos_ready_dist.  All tensors on the device."""
        assert hidden.dtype == torch.bfloat16 and w_vocab.dtype == torch.bfloat16
        assert session_ids.dtype == torch.int32 and session_version.dtype == torch.int64
        n = session_ids.numel()
        _check(lib().prepos_ready_dist(self._h, n, _p(session_ids), _p(hidden), _p(w_vocab), _p(position_p),
                                       _p(entry_hash), _p(skip_mask), _p(records), _p(session_version),
                                       _p(expected_version), _p(logits_out), _stream()), "prepos_ready_dist")

    def ready_dist_w4(self, session_ids, hidden, w4, w_scale, records, session_version, position_p=None,
                      entry_hash=None, skip_mask=None, logits_out=None, expected_version=None):
        """prepos_ready_dist_w4: w4 [V, H/2] uint8 (int4 codes), w_scale [V, H/128] bf16.  All tensors on the device."""
        assert hidden.dtype == torch.bfloat16 and w4.dtype == torch.uint8 and w_scale.dtype == torch.bfloat16
        assert w4.is_contiguous() and w_scale.is_contiguous()
        assert session_ids.dtype == torch.int32 and session_version.dtype == torch.int64
        n = session_ids.numel()
        _check(lib().prepos_ready_dist_w4(self._h, n, _p(session_ids), _p(hidden), _p(w4), _p(w_scale), _p(position_p),
                                          _p(entry_hash), _p(skip_mask), _p(records), _p(session_version),
                                          _p(expected_version), _p(logits_out), _stream()), "prepos_ready_dist_w4")

    def scan_logits(self, logits, records_out):
        assert logits.dtype == torch.float32 and logits.is_contiguous()
        _check(lib().prepos_scan_logits(self._h, logits.shape[0], _p(logits), _p(records_out), _stream()),
               "prepos_scan_logits")

    def gate_serve(self, session_ids, records, session_version, fast_set_bitmap, tau, decision_out, token_out,
                   request_entry_hash=None, strict_gt=False):
        assert session_ids.dtype == torch.int32 and decision_out.dtype == torch.int32 and token_out.dtype == torch.int32
        _check(lib().prepos_gate_serve(self._h, session_ids.numel(), _p(session_ids), _p(request_entry_hash),
                                       _p(records), _p(session_version), _p(fast_set_bitmap), float(tau),
                                       int(bool(strict_gt)), _p(decision_out), _p(token_out), _stream()),
               "prepos_gate_serve")

    def gate_sweep(self, records, session_version, fast_set_bitmap, full_path_token, taus, strict_gt=False):
        """prepos_gate_sweep over all records: returns the [n_tau] device buffer of prepos_sweep_point (64 B each);
        `unpack_sweep` turns it into host arrays."""
        assert full_path_token.dtype == torch.int32 and taus.dtype == torch.float32 and taus.is_cuda
        n = full_path_token.numel()
        out = torch.zeros(taus.numel() * SWEEP_POINT_BYTES, dtype=torch.uint8, device=taus.device)
        _check(lib().prepos_gate_sweep(self._h, n, _p(records), _p(session_version), _p(fast_set_bitmap),
                                       _p(full_path_token), taus.numel(), _p(taus), int(bool(strict_gt)), _p(out),
                                       _stream()), "prepos_gate_sweep")
        return out

    def invalidate(self, session_ids, session_version, records):
        assert session_ids.dtype == torch.int32 and session_version.dtype == torch.int64
        _check(lib().prepos_invalidate(self._h, session_ids.numel(), _p(session_ids), _p(session_version),
                                       _p(records), _stream()), "prepos_invalidate")

"""ctypes binding of the CPU oracle (oracle/prepos_oracle.c).

TEST INFRASTRUCTURE ONLY.  Importable from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs; the product package never imports this module and
this module never imports the product package.

All arithmetic lives in prepos_oracle.c; this file only builds the shared object with gcc,
marshals arrays, and loops the single-session / single-layer C calls over sessions and layers.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "prepos_oracle.c")
_SO = os.path.join(_HERE, "libprepos_oracle.so")

SERVED, GAP_BELOW_TAU, NOT_IN_FAST_SET, STALE_OR_INVALID, INELIGIBLE = 0, 1, 2, 3, 4


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP over independent outputs)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + f".{os.getpid()}.tmp"
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
             _SRC, "-o", tmp, "-lm"])
        os.replace(tmp, _SO)
    return _SO


class _Rec(C.Structure):
    _fields_ = [("max_logit", C.c_double), ("lse", C.c_double), ("gap", C.c_double),
                ("top1", C.c_int32), ("top2", C.c_int32), ("nonfinite", C.c_int32), ("pad_", C.c_int32)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        p = C.c_void_p
        L.oracle_entry_attn.restype = C.c_int
        L.oracle_entry_attn.argtypes = [p, p, p, p, p, p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int,
                                        C.c_int, C.c_int, C.c_double, p, p, p]
        L.oracle_entry_attn_ranged.restype = C.c_int
        L.oracle_entry_attn_ranged.argtypes = [p, p, p, p, p, p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int,
                                               C.c_int, C.c_int, C.c_double, C.c_int, C.c_int, C.c_int, C.c_int,
                                               p, p, p]
        L.oracle_entry_attn_fp8.restype = C.c_int
        L.oracle_entry_attn_fp8.argtypes = [p, p, p, p, p, p, p, p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int,
                                            C.c_int, C.c_int, C.c_double, C.c_int, C.c_int, C.c_int, C.c_int, p, p]
        L.oracle_logits_w4.restype = None
        L.oracle_logits_w4.argtypes = [p, p, p, C.c_int, C.c_int, C.c_int, p]
        L.oracle_e4m3_decode.restype = C.c_double
        L.oracle_e4m3_decode.argtypes = [C.c_uint8]
        L.oracle_e4m3_encode.restype = C.c_uint8
        L.oracle_e4m3_encode.argtypes = [C.c_float]
        L.oracle_logits.restype = None
        L.oracle_logits.argtypes = [p, p, C.c_int, C.c_int, p]
        L.oracle_record.restype = None
        L.oracle_record.argtypes = [p, C.c_int, C.POINTER(_Rec)]
        L.oracle_gate.restype = C.c_int
        L.oracle_gate.argtypes = [C.c_double, C.c_int32, C.c_int, C.c_int, C.c_uint64, C.c_uint64,
                                  C.c_uint64, C.c_uint64, p, C.c_int, C.c_double, C.c_int, p]
        L.oracle_invalidate.restype = None
        L.oracle_invalidate.argtypes = [p, C.c_int, p, p]
        L.oracle_stamp.restype = None
        L.oracle_stamp.argtypes = [C.c_int32, p, p, p]
        L.oracle_fastset_bitmap.restype = None
        L.oracle_fastset_bitmap.argtypes = [p, C.c_int, C.c_int, p]
        L.oracle_num_threads.restype = C.c_int
        L.oracle_set_num_threads.restype = None
        L.oracle_set_num_threads.argtypes = [C.c_int]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_num_threads(n: int) -> None:
    lib().oracle_set_num_threads(int(n))


def bf16_bits(t) -> np.ndarray:
    """torch bf16 tensor (any device) or uint16 ndarray -> contiguous uint16 ndarray of the same bits."""
    if isinstance(t, np.ndarray):
        assert t.dtype == np.uint16
        return np.ascontiguousarray(t)
    import torch
    assert t.dtype == torch.bfloat16, t.dtype
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16)


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def entry_attn(q, k_new, v_new, k_pool, v_pool, page_table, n_s, capacity_tokens, scale=None,
               want_rowsum=False, heads=None, rows=None):
    """O1 for one session, one layer.  q [L,Hq,d], k_new/v_new [L,Hkv,d], pools [n_pages,Hkv,page,d]
    (uint16 ndarrays; pools are modified in place by the append).  Returns dict(status, out, rowsum, position).
    heads=(lo, hi) / rows=(lo, hi) restrict the OUTPUTS computed to those query heads / entry rows (the others stay
    NaN); the append is always complete."""
    L, Hq, d = q.shape
    Hkv = k_new.shape[1]
    page = k_pool.shape[2]
    assert k_pool.dtype == np.uint16 and k_pool.flags.c_contiguous and v_pool.flags.c_contiguous
    q = np.ascontiguousarray(q)
    k_new = np.ascontiguousarray(k_new)
    v_new = np.ascontiguousarray(v_new)
    pt = np.ascontiguousarray(page_table, dtype=np.int32)
    out = np.full((L, Hq, d), np.nan, dtype=np.float64)
    rowsum = np.zeros((L, Hq), dtype=np.float64) if want_rowsum else None
    pos = np.zeros(1, dtype=np.int64)
    if scale is None:
        scale = 1.0 / float(np.sqrt(d))
    if heads is None and rows is None:
        st = lib().oracle_entry_attn(_ptr(q), _ptr(k_new), _ptr(v_new), _ptr(k_pool), _ptr(v_pool), _ptr(pt),
                                     int(n_s), int(L), int(capacity_tokens), int(Hq), int(Hkv), int(d), int(page),
                                     float(scale), _ptr(out), _ptr(rowsum) if want_rowsum else None, _ptr(pos))
    else:
        h_lo, h_hi = (0, Hq) if heads is None else heads
        i_lo, i_hi = (0, L) if rows is None else rows
        st = lib().oracle_entry_attn_ranged(_ptr(q), _ptr(k_new), _ptr(v_new), _ptr(k_pool), _ptr(v_pool), _ptr(pt),
                                            int(n_s), int(L), int(capacity_tokens), int(Hq), int(Hkv), int(d),
                                            int(page), float(scale), int(h_lo), int(h_hi), int(i_lo), int(i_hi),
                                            _ptr(out), _ptr(rowsum) if want_rowsum else None, _ptr(pos))
    if st < 0:
        raise ValueError("oracle_entry_attn: bad argument")
    return {"status": st, "out": out, "rowsum": rowsum, "position": int(pos[0]) if st == 0 else None}


def e4m3_decode(codes) -> np.ndarray:
    """e4m3 codes (uint8 array) -> fp64 values, through the oracle's decoder."""
    c = np.asarray(codes, dtype=np.uint8)
    L = lib()
    return np.array([L.oracle_e4m3_decode(int(b)) for b in c.ravel()], dtype=np.float64).reshape(c.shape)


def e4m3_encode(values) -> np.ndarray:
    """fp32 values -> e4m3 codes (round to nearest even, saturating), through the oracle's encoder."""
    v = np.asarray(values, dtype=np.float32)
    L = lib()
    return np.array([L.oracle_e4m3_encode(float(y)) for y in v.ravel()], dtype=np.uint8).reshape(v.shape)


def entry_attn_fp8(q, k_new, v_new, k_pool8, v_pool8, k_scale, v_scale, page_table, n_s, capacity_tokens,
                   scale=None, heads=None, rows=None):
    """O7: O1 over an e4m3 KV cache (reading Q20).  Pools [n_pages,Hkv,page,d] uint8 (modified in place
    by the append), scales [n_pages,Hkv] float32.  Returns dict(status, out, position)."""
    L, Hq, d = q.shape
    Hkv = k_new.shape[1]
    page = k_pool8.shape[2]
    assert k_pool8.dtype == np.uint8 and k_pool8.flags.c_contiguous and v_pool8.flags.c_contiguous
    q = np.ascontiguousarray(q)
    k_new = np.ascontiguousarray(k_new)
    v_new = np.ascontiguousarray(v_new)
    ks = np.ascontiguousarray(k_scale, dtype=np.float32)
    vs = np.ascontiguousarray(v_scale, dtype=np.float32)
    pt = np.ascontiguousarray(page_table, dtype=np.int32)
    out = np.full((L, Hq, d), np.nan, dtype=np.float64)
    pos = np.zeros(1, dtype=np.int64)
    if scale is None:
        scale = 1.0 / float(np.sqrt(d))
    h_lo, h_hi = (0, Hq) if heads is None else heads
    i_lo, i_hi = (0, L) if rows is None else rows
    st = lib().oracle_entry_attn_fp8(_ptr(q), _ptr(k_new), _ptr(v_new), _ptr(k_pool8), _ptr(v_pool8), _ptr(ks), _ptr(vs),
                                     _ptr(pt), int(n_s), int(L), int(capacity_tokens), int(Hq), int(Hkv), int(d),
                                     int(page), float(scale), int(h_lo), int(h_hi), int(i_lo), int(i_hi), _ptr(out),
                                     _ptr(pos))
    if st < 0:
        raise ValueError("oracle_entry_attn_fp8: bad argument")
    return {"status": st, "out": out, "position": int(pos[0]) if st == 0 else None}


def logits_w4(w4, w_scale, x, group=128) -> np.ndarray:
    """O8: O2 over a 4-bit W_vocab (reading Q21).  w4 [V,H/2] uint8, w_scale [V,H/group] bf16 bits,
    x [H] bf16 bits -> fp64 [V]."""
    V, H2 = w4.shape
    H = 2 * H2
    w4 = np.ascontiguousarray(w4, dtype=np.uint8)
    w_scale = np.ascontiguousarray(w_scale, dtype=np.uint16)
    x = np.ascontiguousarray(x, dtype=np.uint16)
    assert x.shape == (H,) and w_scale.shape == (V, H // group) and H % group == 0
    out = np.empty(V, dtype=np.float64)
    lib().oracle_logits_w4(_ptr(w4), _ptr(w_scale), _ptr(x), V, H, int(group), _ptr(out))
    return out


def logits(w, x) -> np.ndarray:
    """O2.  w [V,H] uint16 bits, x [H] uint16 bits -> fp64 [V]."""
    V, H = w.shape
    w = np.ascontiguousarray(w)
    x = np.ascontiguousarray(x)
    assert x.shape == (H,)
    out = np.empty(V, dtype=np.float64)
    lib().oracle_logits(_ptr(w), _ptr(x), V, H, _ptr(out))
    return out


@dataclass
class Record:
    max_logit: float
    lse: float
    gap: float
    top1: int
    top2: int
    nonfinite: int


def record(lg: np.ndarray) -> Record:
    """O3 from an fp64 logit vector."""
    lg = np.ascontiguousarray(lg, dtype=np.float64)
    r = _Rec()
    lib().oracle_record(_ptr(lg), int(lg.shape[0]), C.byref(r))
    return Record(r.max_logit, r.lse, r.gap, r.top1, r.top2, r.nonfinite)


def fastset_bitmap(ids, V) -> np.ndarray:
    ids = np.ascontiguousarray(ids, dtype=np.int32)
    bm = np.zeros((V + 31) // 32, dtype=np.uint32)
    lib().oracle_fastset_bitmap(_ptr(ids), int(ids.shape[0]), int(V), _ptr(bm))
    return bm


def gate(gap, top1, valid, nonfinite, record_version, session_version, record_hash, request_hash,
         bitmap, V, tau, strict_gt=False):
    """O4 for one request -> (decision, token)."""
    tok = np.zeros(1, dtype=np.int32)
    bm = np.ascontiguousarray(bitmap, dtype=np.uint32)
    dec = lib().oracle_gate(float(gap), int(top1), int(bool(valid)), int(bool(nonfinite)),
                            int(record_version), int(session_version), int(record_hash), int(request_hash),
                            _ptr(bm), int(V), float(tau), int(bool(strict_gt)), _ptr(tok))
    return int(dec), int(tok[0])


class SessionTable:
    """O5: the session state machine of Fig. 3 for n sessions -- plain arrays."""

    def __init__(self, n_sessions: int):
        self.version = np.zeros(n_sessions, dtype=np.uint64)
        self.rec_version = np.zeros(n_sessions, dtype=np.uint64)
        self.rec_valid = np.zeros(n_sessions, dtype=np.int32)
        self.rec_hash = np.zeros(n_sessions, dtype=np.uint64)
        self.rec_position = np.zeros(n_sessions, dtype=np.int64)
        self.rec: list = [None] * n_sessions

    def invalidate(self, ids):
        ids = np.ascontiguousarray(ids, dtype=np.int32)
        lib().oracle_invalidate(_ptr(ids), int(ids.shape[0]), _ptr(self.version), _ptr(self.rec_valid))

    def preposition(self, sid: int, rec: Record, position: int = 0, entry_hash: int = 0):
        """Alg. 1 l.10-12: store the record, stamp it with the live version, mark valid."""
        self.rec[sid] = rec
        self.rec_hash[sid] = entry_hash
        self.rec_position[sid] = position
        lib().oracle_stamp(int(sid), _ptr(self.version), _ptr(self.rec_version), _ptr(self.rec_valid))

    def serve(self, sid: int, bitmap, V, tau, request_hash: int = 0, strict_gt=False):
        r = self.rec[sid]
        if r is None:
            return gate(0.0, -1, False, 0, 0, int(self.version[sid]), 0, request_hash, bitmap, V, tau, strict_gt)
        return gate(r.gap, r.top1, bool(self.rec_valid[sid]), r.nonfinite, int(self.rec_version[sid]),
                    int(self.version[sid]), int(self.rec_hash[sid]), request_hash, bitmap, V, tau, strict_gt)


# ---- O6: risk-coverage sweep of the gate (Sec. 2.4) -------------------
# Plain definitions in fp64; pinned in tests/test_oracle_calibration.py by the counts and intervals the paper prints
# for its own calibration run (121 of 128 served at tau = 2.0, 16 false accepts).
Z95 = 1.959963984540054  # two-sided 95% normal quantile


def wilson(k: int, n: int, z: float = Z95):
    """Wilson score interval of k successes in n trials (the paper's "Wilson 95% interval").
    (0, 1) for n = 0."""
    if n <= 0:
        return 0.0, 1.0
    p = k / n
    den = 1.0 + z * z / n
    centre = (p + z * z / (2.0 * n)) / den
    half = z * math.sqrt(p * (1.0 - p) / n + z * z / (4.0 * n * n)) / den
    return centre - half, centre + half


@dataclass
class SweepPoint:
    tau: float
    accepted: int        # requests the gate accepts: gamma > tau (or >=) and argmax in A       (Eq. 13 numerator)
    false_accepts: int   # accepted whose served token differs from the full-path token          (Eq. 14 numerator)
    coverage: float      # c(tau) = accepted / n                                                 (Eq. 13)
    far: float           # r(tau) = false_accepts / accepted, 0 when nothing is accepted         (Eq. 14)
    cov_lo: float
    cov_hi: float
    far_lo: float
    far_hi: float


def risk_coverage(gap, servable, top1, full_path_token, taus, strict_gt=False):
    """For each tau: Eq. 13 / Eq. 14 over n decision points.  gap[i], top1[i] from the ready-distribution record,
    servable[i] = record valid, fresh and argmax in A (everything of Eq. 12 but the threshold), full_path_token[i]
    the model's own full-path output.  A non-finite gap never accepts."""
    gap = np.asarray(gap, dtype=np.float64)
    servable = np.asarray(servable).astype(bool)
    wrong = np.asarray(top1) != np.asarray(full_path_token)
    n = int(gap.shape[0])
    out = []
    for tau in taus:
        acc = servable & ((gap > tau) if strict_gt else (gap >= tau)) & np.isfinite(gap)
        a = int(acc.sum())
        f = int((acc & wrong).sum())
        clo, chi = wilson(a, n)
        flo, fhi = wilson(f, a)
        out.append(SweepPoint(float(tau), a, f, a / n if n else 0.0, f / a if a else 0.0, clo, chi, flo, fhi))
    return out


def calibrate_tau(points, r_max: float):
    """"selects the smallest tau such that r(tau) <= r_max" over the swept thresholds; None when no
    swept threshold meets the budget."""
    ok = [p.tau for p in points if p.far <= r_max]
    return min(ok) if ok else None

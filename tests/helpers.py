"""Shared test plumbing: oracle-side evaluation of a SessionBatch and the tolerance comparators.

Tolerances are BASELINE.json north_star's: attention max abs err <= 1e-2; logits max abs err <= 2e-2;
logsumexp relative err <= 1e-3; top-1 ids and gate decisions exact except where the oracle's own gap to
the runner-up (ids) or to tau (decisions) is within 4e-2.
"""
import numpy as np
import torch

ATTN_ATOL = 1e-2
LOGIT_ATOL = 2e-2
LSE_RTOL = 1e-3
AMBIG = 4e-2


def bits(t: torch.Tensor) -> np.ndarray:
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16).copy()


def oracle_attn_batch(oracle, sb, layers=None, sessions=None, pools=None):
    """Runs O1 for the given layers/sessions of a SessionBatch on CPU copies of its pools.
    Returns (out {(layer, s): fp64 [L,Hq,d]}, status {s: int}, k_pool bits [layers...], v_pool bits)."""
    layers = range(sb.k_pool.shape[0]) if layers is None else layers
    sessions = range(sb.n_sessions) if sessions is None else sessions
    pt = sb.page_table.cpu().numpy()
    outs, status = {}, {}
    kp = {l: bits(sb.k_pool[l]) for l in layers} if pools is None else pools[0]
    vp = {l: bits(sb.v_pool[l]) for l in layers} if pools is None else pools[1]
    for l in layers:
        for s in sessions:
            r0, L = sb.row_offset[s], sb.l_entry[s]
            res = oracle.entry_attn(bits(sb.q[l, r0:r0 + L]), bits(sb.k_new[l, r0:r0 + L]),
                                    bits(sb.v_new[l, r0:r0 + L]), kp[l], vp[l], pt[s], sb.n_s[s], sb.capacity[s])
            outs[(l, s)] = res["out"]
            status[s] = res["status"]
    return outs, status, kp, vp


def oracle_attn_rows(oracle, sb, layer, s, heads_rows):
    """O1 restricted to sampled (head, entry row) pairs of one (layer, session): computes only the needed rows by
    calling the oracle on a single-kv-head, single-row-prefix view.  Returns {(h, i): fp64 [d]}.
    The oracle is called with Hq = G, Hkv = 1 on the kv head's slice and L = i+1 rows, so that no oracle
    arithmetic is re-implemented here."""
    shape = sb.shape
    G = shape.G
    pt = sb.page_table[s].cpu().numpy()
    r0 = sb.row_offset[s]
    res = {}
    by_head = {}
    for (h, i) in heads_rows:
        by_head.setdefault(h // G, []).append((h, i))
    for g, lst in by_head.items():
        imax = max(i for _, i in lst)
        kp = bits(sb.k_pool[layer][:, g:g + 1])
        vp = bits(sb.v_pool[layer][:, g:g + 1])
        q = bits(sb.q[layer, r0:r0 + imax + 1, g * G:(g + 1) * G])
        kn = bits(sb.k_new[layer, r0:r0 + imax + 1, g:g + 1])
        vn = bits(sb.v_new[layer, r0:r0 + imax + 1, g:g + 1])
        out = oracle.entry_attn(q, kn, vn, kp, vp, pt, sb.n_s[s], sb.n_s[s] + imax + 1)["out"]
        for (h, i) in lst:
            res[(h, i)] = out[i, h - g * G]
    return res


def check_attn(out_gpu: torch.Tensor, outs: dict, sb, atol=ATTN_ATOL):
    """out_gpu [layers, sum_L, Hq, d] bf16 vs oracle dict; returns the max abs error."""
    worst = 0.0
    for (l, s), ref in outs.items():
        if ref is None or np.all(np.isnan(ref)):
            continue
        r0, L = sb.row_offset[s], sb.l_entry[s]
        got = out_gpu[l, r0:r0 + L].detach().cpu().to(torch.float64).numpy()
        err = np.abs(got - ref).max() if ref.size else 0.0
        assert np.isfinite(got).all(), f"non-finite attention output at layer {l} session {s}"
        assert err <= atol, f"layer {l} session {s}: max abs err {err} > {atol}"
        worst = max(worst, float(err))
    return worst


def check_record(oracle, rec: dict, idx: int, lg64: np.ndarray, logits_gpu=None):
    """One GPU record (dict of host tensors, row idx) vs the oracle's record of the fp64 logits."""
    ref = oracle.record(lg64)
    if logits_gpu is not None:
        err = np.abs(logits_gpu.astype(np.float64) - lg64).max()
        assert err <= LOGIT_ATOL, f"logits max abs err {err}"
    assert abs(float(rec["max_logit"][idx]) - ref.max_logit) <= LOGIT_ATOL
    assert abs(float(rec["lse"][idx]) - ref.lse) <= LSE_RTOL * abs(ref.lse) + 1e-6
    assert abs(float(rec["gap"][idx]) - ref.gap) <= 2 * LOGIT_ATOL
    t1, t2 = int(rec["top1"][idx]), int(rec["top2"][idx])
    if ref.gap >= AMBIG:
        assert t1 == ref.top1, (t1, ref.top1, ref.gap)
    else:
        assert t1 in (ref.top1, ref.top2) or abs(lg64[t1] - ref.max_logit) < AMBIG
    # top2 is unique only when the third logit is clearly below the second
    srt = np.sort(lg64)[::-1]
    if ref.gap >= AMBIG and len(srt) > 2 and srt[1] - srt[2] >= AMBIG:
        assert t2 == ref.top2, (t2, ref.top2)
    else:
        assert abs(lg64[t2] - lg64[ref.top2]) < AMBIG or t2 == ref.top1
    return ref


def check_decision(oracle, dec_gpu: int, tok_gpu: int, ref_rec, valid, rec_version, live_version, bitmap, V, tau,
                   rec_hash=0, req_hash=0, strict_gt=False, gpu_top1=None):
    """Gate decision vs O4 on the ORACLE's record; exact unless the oracle's gap is within 4e-2 of tau or of 0."""
    dec, tok = oracle.gate(ref_rec.gap, ref_rec.top1, valid, ref_rec.nonfinite, rec_version, live_version,
                           rec_hash, req_hash, bitmap, V, tau, strict_gt)
    ambiguous = abs(ref_rec.gap - tau) < AMBIG or ref_rec.gap < AMBIG
    if not ambiguous or dec in (oracle.STALE_OR_INVALID, oracle.INELIGIBLE):
        assert (dec_gpu, tok_gpu) == (dec, tok), (dec_gpu, tok_gpu, dec, tok, ref_rec)
    else:
        assert dec_gpu in (oracle.SERVED, oracle.GAP_BELOW_TAU, oracle.NOT_IN_FAST_SET)
        if dec_gpu == oracle.SERVED:
            assert tok_gpu in (ref_rec.top1, ref_rec.top2)
    return dec, tok

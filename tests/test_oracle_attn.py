"""Pins of oracle O1 (entry attention + append) against what the paper and the mathematics fix.

SURVEY.md 8(c) "What pins each part", O1 (1)-(12).  None of these retypes the oracle's formula:
they use a library SDPA, closed forms, invariants and a pure-Python brute force.
"""
import math

import numpy as np
import pytest
import torch

from paper_2606_29565_b200 import synth


def _bits(t):
    return t.contiguous().view(torch.int16).numpy().view(np.uint16).copy()


def _f64(bits):
    return torch.from_numpy(bits.view(np.int16).copy()).view(torch.bfloat16).to(torch.float64)


def _run(oracle, sb, layer=0, s=0, pools=None, scale=None, want_rowsum=False, q=None, k_new=None, v_new=None):
    r0, L = sb.row_offset[s], sb.l_entry[s]
    kp, vp = pools if pools is not None else (_bits(sb.k_pool[layer]), _bits(sb.v_pool[layer]))
    q = _bits(sb.q[layer, r0:r0 + L]) if q is None else q
    k_new = _bits(sb.k_new[layer, r0:r0 + L]) if k_new is None else k_new
    v_new = _bits(sb.v_new[layer, r0:r0 + L]) if v_new is None else v_new
    res = oracle.entry_attn(q, k_new, v_new, kp, vp, sb.page_table[s].numpy(), sb.n_s[s], sb.capacity[s],
                            scale=scale, want_rowsum=want_rowsum)
    res["k_pool"], res["v_pool"] = kp, vp
    return res


def _logical_kv(sb, pools, s, n_tokens):
    """gather [n_tokens, Hkv, d] fp64 through the page table (test-side, by plain indexing)."""
    kp, vp = pools
    pt = sb.page_table[s].numpy()
    page = sb.shape.page
    idx = np.arange(n_tokens)
    k = kp[pt[idx // page], :, idx % page, :]
    v = vp[pt[idx // page], :, idx % page, :]
    return _f64(k), _f64(v)


SMALL = synth.Shape("t", layers=1, Hq=4, Hkv=2, d=16, H=32, V=64, page=4)


def test_ns0_is_causal_sdpa(oracle):
    """Pin (1): n_s = 0 => ordinary causal GQA attention; cross-check against torch SDPA in fp64."""
    sb = synth.make_sessions(SMALL, [0], [9], seed=1)
    res = _run(oracle, sb)
    assert res["status"] == 0 and res["position"] == 9
    q = sb.q[0].to(torch.float64).permute(1, 0, 2)            # [Hq, L, d]
    k = sb.k_new[0].to(torch.float64).permute(1, 0, 2).repeat_interleave(SMALL.G, dim=0)
    v = sb.v_new[0].to(torch.float64).permute(1, 0, 2).repeat_interleave(SMALL.G, dim=0)
    ref = torch.nn.functional.scaled_dot_product_attention(q, k, v, is_causal=True).permute(1, 0, 2)
    np.testing.assert_allclose(res["out"], ref.numpy(), rtol=0, atol=1e-12)


def test_l1_is_decode_attention(oracle):
    """Pin (2): L = 1 => textbook decode attention over n_s cached tokens + itself (library softmax)."""
    sb = synth.make_sessions(SMALL, [23], [1], seed=2)
    res = _run(oracle, sb)
    k, v = _logical_kv(sb, (res["k_pool"], res["v_pool"]), 0, 24)
    for h in range(SMALL.Hq):
        g = h // SMALL.G
        s = (k[:, g] @ sb.q[0, 0, h].to(torch.float64)) / math.sqrt(SMALL.d)
        ref = torch.softmax(s, 0) @ v[:, g]
        np.testing.assert_allclose(res["out"][0, h], ref.numpy(), rtol=0, atol=1e-12)


def test_general_vs_sdpa_with_prefix_mask(oracle):
    """n_s > 0, ragged n_s (not a page multiple): library SDPA with an explicit boolean mask."""
    sb = synth.make_sessions(SMALL, [13], [6], seed=3)
    res = _run(oracle, sb)
    n, L = 13, 6
    k, v = _logical_kv(sb, (res["k_pool"], res["v_pool"]), 0, n + L)
    q = sb.q[0].to(torch.float64).permute(1, 0, 2)
    kk = k.permute(1, 0, 2).repeat_interleave(SMALL.G, dim=0)
    vv = v.permute(1, 0, 2).repeat_interleave(SMALL.G, dim=0)
    mask = torch.arange(n + L)[None, :] <= (n + torch.arange(L))[:, None]
    ref = torch.nn.functional.scaled_dot_product_attention(q, kk, vv, attn_mask=mask).permute(1, 0, 2)
    np.testing.assert_allclose(res["out"], ref.numpy(), rtol=0, atol=1e-12)


def test_softmax_sums_to_one_and_convexity(oracle):
    """Pin (3): sum_j p_j = 1; each output coordinate lies within [min_j v_j, max_j v_j]."""
    sb = synth.make_sessions(SMALL, [37], [5], seed=4)
    res = _run(oracle, sb, want_rowsum=True)
    np.testing.assert_allclose(res["rowsum"], 1.0, rtol=0, atol=1e-13)
    k, v = _logical_kv(sb, (res["k_pool"], res["v_pool"]), 0, 37 + 5)
    for i in range(5):
        for h in range(SMALL.Hq):
            vv = v[: 37 + i + 1, h // SMALL.G].numpy()
            assert np.all(res["out"][i, h] <= vv.max(0) + 1e-12)
            assert np.all(res["out"][i, h] >= vv.min(0) - 1e-12)


def test_equal_v_rows_give_that_row(oracle):
    """Pin (4): all V rows equal => o = that row, whatever the scores."""
    sb = synth.make_sessions(SMALL, [11], [4], seed=5)
    row = sb.v_new[0, 0, 0].clone()
    sb.v_pool[:] = row
    sb.v_new[:] = row
    res = _run(oracle, sb)
    np.testing.assert_allclose(res["out"], np.broadcast_to(row.to(torch.float64).numpy(), res["out"].shape),
                               rtol=0, atol=1e-13)


def test_zero_q_gives_running_mean(oracle):
    """Pin (5): Q = 0 => o_i = mean(v_0 .. v_{n_s+i})."""
    sb = synth.make_sessions(SMALL, [10], [7], seed=6)
    sb.q.zero_()
    res = _run(oracle, sb)
    k, v = _logical_kv(sb, (res["k_pool"], res["v_pool"]), 0, 17)
    for i in range(7):
        for h in range(SMALL.Hq):
            ref = v[: 10 + i + 1, h // SMALL.G].mean(0)
            np.testing.assert_allclose(res["out"][i, h], ref.numpy(), rtol=0, atol=1e-13)


def test_key_shift_invariance(oracle):
    """Pin (6): adding one constant vector to every key shifts every score of a row equally => o unchanged.
    Values are small integers so the shifted keys are still exact in bf16."""
    sb = synth.make_sessions(SMALL, [9], [3], seed=7)
    gi = torch.Generator().manual_seed(70)
    for t in (sb.k_pool, sb.k_new, sb.q):
        t.copy_(torch.randint(-3, 4, t.shape, generator=gi).to(torch.bfloat16))
    res_a = _run(oracle, sb, scale=0.05)
    shift = torch.randint(-2, 3, (SMALL.d,), generator=gi).to(torch.bfloat16)
    sb.k_pool += shift
    sb.k_new += shift
    res_b = _run(oracle, sb, scale=0.05)
    np.testing.assert_allclose(res_a["out"], res_b["out"], rtol=0, atol=1e-12)


def test_causality_bit_identical(oracle):
    """Pin (7): perturbing entry token j's K/V leaves rows i < j bit-identical and changes row j."""
    sb = synth.make_sessions(SMALL, [6], [5], seed=8)
    base = _run(oracle, sb)
    j = 3
    sb.k_new[0, j] += 1.0
    sb.v_new[0, j] -= 2.0
    pert = _run(oracle, sb)
    assert np.array_equal(base["out"][:j], pert["out"][:j])
    assert not np.allclose(base["out"][j], pert["out"][j])


def test_gqa_equals_mha_with_repeated_kv(oracle):
    """Pin (8): GQA == MHA with each KV head repeated G times (catches a wrong h -> g map)."""
    sb = synth.make_sessions(SMALL, [14], [4], seed=9)
    res = _run(oracle, sb)
    mha = synth.Shape("m", layers=1, Hq=4, Hkv=4, d=16, H=32, V=64, page=4)
    sm = synth.make_sessions(mha, [14], [4], seed=9)
    sm.page_table.copy_(sb.page_table)
    sm.q.copy_(sb.q)
    sm.k_pool.copy_(sb.k_pool.repeat_interleave(SMALL.G, dim=2))
    sm.v_pool.copy_(sb.v_pool.repeat_interleave(SMALL.G, dim=2))
    sm.k_new.copy_(sb.k_new.repeat_interleave(SMALL.G, dim=2))
    sm.v_new.copy_(sb.v_new.repeat_interleave(SMALL.G, dim=2))
    res_m = _run(oracle, sm)
    assert np.array_equal(res["out"], res_m["out"])


def test_page_shuffle_invariance(oracle):
    """Pin (9): same logical cache, permuted physical pages => identical result, bit for bit."""
    sb = synth.make_sessions(SMALL, [18], [5], seed=10)
    res = _run(oracle, sb)
    n_pages = sb.k_pool.shape[1]
    perm = torch.randperm(n_pages, generator=torch.Generator().manual_seed(3))
    inv = torch.empty_like(perm)
    inv[perm] = torch.arange(n_pages)
    sb2 = synth.make_sessions(SMALL, [18], [5], seed=10)
    sb2.k_pool.copy_(sb.k_pool[:, inv])      # physical page p now sits at perm[p]
    sb2.v_pool.copy_(sb.v_pool[:, inv])
    sb2.page_table.copy_(perm[sb.page_table.long()].to(torch.int32))
    res2 = _run(oracle, sb2)
    assert np.array_equal(res["out"], res2["out"])


def test_two_step_consistency_and_append(oracle):
    """Pin (10): pre-position L1 then L2 tokens == one call with L1+L2; pools identical afterwards.
    Also the a1 post-condition: appended slots equal K_new/V_new bit for bit, every other byte unchanged."""
    L1, L2, n = 3, 4, 10
    sb = synth.make_sessions(SMALL, [n], [L1 + L2], seed=11)
    before_k, before_v = _bits(sb.k_pool[0]), _bits(sb.v_pool[0])
    one = _run(oracle, sb)
    qb, kb, vb = _bits(sb.q[0]), _bits(sb.k_new[0]), _bits(sb.v_new[0])
    pools = (before_k.copy(), before_v.copy())
    pt = sb.page_table[0].numpy()
    a = oracle.entry_attn(qb[:L1], kb[:L1], vb[:L1], pools[0], pools[1], pt, n, sb.capacity[0])
    b = oracle.entry_attn(qb[L1:], kb[L1:], vb[L1:], pools[0], pools[1], pt, n + L1, sb.capacity[0])
    assert a["position"] == n + L1 and b["position"] == n + L1 + L2 == one["position"]
    np.testing.assert_allclose(np.concatenate([a["out"], b["out"]]), one["out"], rtol=0, atol=1e-13)
    assert np.array_equal(pools[0], one["k_pool"]) and np.array_equal(pools[1], one["v_pool"])
    # append post-condition
    page = SMALL.page
    touched = np.zeros(before_k.shape[:1] + before_k.shape[2:3], dtype=bool)  # [n_pages, page]
    for jp in range(L1 + L2):
        j = n + jp
        assert np.array_equal(one["k_pool"][pt[j // page], :, j % page], kb[jp])
        assert np.array_equal(one["v_pool"][pt[j // page], :, j % page], vb[jp])
        touched[pt[j // page], j % page] = True
    untouched = ~touched
    assert np.array_equal(one["k_pool"].transpose(0, 2, 1, 3)[untouched], before_k.transpose(0, 2, 1, 3)[untouched])
    assert np.array_equal(one["v_pool"].transpose(0, 2, 1, 3)[untouched], before_v.transpose(0, 2, 1, 3)[untouched])


def test_chunked_lse_merge_equals_unsplit(oracle):
    """Pin (11): split the keys in two chunks, attend each with the library, merge by log-sum-exp => oracle."""
    sb = synth.make_sessions(SMALL, [29], [1], seed=12)
    res = _run(oracle, sb)
    k, v = _logical_kv(sb, (res["k_pool"], res["v_pool"]), 0, 30)
    for h in range(SMALL.Hq):
        g = h // SMALL.G
        s = (k[:, g] @ sb.q[0, 0, h].to(torch.float64)) / math.sqrt(SMALL.d)
        parts = []
        for sl in (slice(0, 17), slice(17, 30)):
            lse = torch.logsumexp(s[sl], 0)
            parts.append((lse, torch.softmax(s[sl], 0) @ v[sl, g]))
        tot = torch.logsumexp(torch.stack([p[0] for p in parts]), 0)
        merged = sum(torch.exp(l - tot) * o for l, o in parts)
        np.testing.assert_allclose(res["out"][0, h], merged.numpy(), rtol=0, atol=1e-12)


def test_brute_force_python_loops_config1(oracle):
    """Pin (12): pure-Python fp64 loops on a slice of config 1 (BASELINE.json configs[0] shapes)."""
    sb = synth.make_sessions(synth.C1, [256], [8], seed=synth.SEED_BASE)
    res = _run(oracle, sb)
    k, v = _logical_kv(sb, (res["k_pool"], res["v_pool"]), 0, 264)
    k, v, q = k.tolist(), v.tolist(), sb.q[0].to(torch.float64).tolist()
    d, G = synth.C1.d, synth.C1.G
    for (i, h) in ((0, 0), (7, 3), (4, 2)):
        g = h // G
        sc = [sum(q[i][h][c] * k[j][g][c] for c in range(d)) / math.sqrt(d) for j in range(256 + i + 1)]
        m = max(sc)
        e = [math.exp(x - m) for x in sc]
        z = sum(e)
        o = [sum(e[j] / z * v[j][g][c] for j in range(len(sc))) for c in range(d)]
        np.testing.assert_allclose(res["out"][i, h], np.array(o), rtol=0, atol=1e-12)


def test_budget_skip_has_no_side_effects(oracle):
    """Alg. 1 l.2-3: L_entry > headroom => skipped, pool untouched, no output."""
    sb = synth.make_sessions(SMALL, [10], [6], seed=13, tight_capacity=[15])
    before_k, before_v = _bits(sb.k_pool[0]), _bits(sb.v_pool[0])
    res = _run(oracle, sb)
    assert res["status"] == 1 and res["position"] is None
    assert np.array_equal(res["k_pool"], before_k) and np.array_equal(res["v_pool"], before_v)
    assert np.all(np.isnan(res["out"]))
    sb2 = synth.make_sessions(SMALL, [10], [6], seed=13, tight_capacity=[16])
    assert _run(oracle, sb2)["status"] == 0          # L == headroom is admitted (Alg. 1: skip iff L > B)


def test_scale_argument_and_default(oracle):
    """Reading Q3: default scale is 1/sqrt(d); an explicit scale is honoured (library softmax check)."""
    sb = synth.make_sessions(SMALL, [5], [1], seed=14)
    a = _run(oracle, sb)
    b = _run(oracle, sb, scale=1.0 / math.sqrt(SMALL.d))
    assert np.array_equal(a["out"], b["out"])
    c = _run(oracle, sb, scale=0.5)
    k, v = _logical_kv(sb, (c["k_pool"], c["v_pool"]), 0, 6)
    s = (k[:, 0] @ sb.q[0, 0, 0].to(torch.float64)) * 0.5
    np.testing.assert_allclose(c["out"][0, 0], (torch.softmax(s, 0) @ v[:, 0]).numpy(), rtol=0, atol=1e-12)

"""Pins of oracle O2 (logits) and O3 (record: max, lse, top-1, top-2, gap).  SURVEY.md 8(c) O2/O3 (1)-(8)."""
import itertools
import math

import numpy as np
import pytest
import torch

from paper_2606_29565_b200 import synth


def _bits(t):
    return t.contiguous().view(torch.int16).numpy().view(np.uint16).copy()


def test_softmax_from_lse_sums_to_one(oracle):
    """Pin (1): sum_v exp(l_v - lse) = 1."""
    lg = np.random.default_rng(0).normal(size=5000) * 3
    r = oracle.record(lg)
    assert abs(np.exp(lg - r.lse).sum() - 1.0) < 1e-12


def test_shift_invariance(oracle):
    """Pin (2): l + c => same top1/top2/gap; max and lse shift by c (exact: dyadic values and shift)."""
    rng = np.random.default_rng(1)
    lg = rng.integers(-64, 64, size=777) / 8.0
    a = oracle.record(lg)
    for c in (5.0, -11.25, 1024.0):
        b = oracle.record(lg + c)
        assert (a.top1, a.top2) == (b.top1, b.top2) and a.gap == b.gap
        assert b.max_logit == a.max_logit + c
        assert abs((b.lse - c) - a.lse) < 1e-12


def test_lse_bounds_and_all_equal(oracle):
    """Pin (3): max <= lse <= max + ln V; all-equal logits hit the upper bound, gap 0, top1 0, top2 1."""
    lg = np.random.default_rng(2).normal(size=300)
    r = oracle.record(lg)
    assert r.max_logit <= r.lse <= r.max_logit + math.log(300)
    r = oracle.record(np.full(128, 2.5))
    assert abs(r.lse - (2.5 + math.log(128))) < 1e-13
    assert (r.top1, r.top2, r.gap) == (0, 1, 0.0)


def test_logits_unit_vector_gives_column(oracle):
    """Pin (4), O2: x = e_k => logits are column k of W exactly (catches a transposed operand)."""
    g = torch.Generator().manual_seed(3)
    w = torch.randn(37, 24, generator=g).to(torch.bfloat16)
    for k in (0, 5, 23):
        x = torch.zeros(24, dtype=torch.bfloat16)
        x[k] = 1.0
        lg = oracle.logits(_bits(w), _bits(x))
        assert np.array_equal(lg, w[:, k].to(torch.float64).numpy())


def test_logits_vs_library_matmul(oracle):
    """O2 vs a library fp64 mat-vec."""
    g = torch.Generator().manual_seed(4)
    w = (torch.randn(513, 96, generator=g) / 8).to(torch.bfloat16)
    x = torch.randn(96, generator=g).to(torch.bfloat16)
    lg = oracle.logits(_bits(w), _bits(x))
    ref = (w.to(torch.float64) @ x.to(torch.float64)).numpy()
    np.testing.assert_allclose(lg, ref, rtol=0, atol=1e-12)


def test_exhaustive_small_vocab(oracle):
    """Pin (5): every logit vector in {0,1,2}^V for V <= 6 (all tie patterns) against the definition
    'sort by (logit desc, id asc)', via Python's sort (reading Q8)."""
    for V in range(2, 7):
        for combo in itertools.product((0.0, 1.0, 2.0), repeat=V):
            r = oracle.record(np.array(combo))
            order = sorted(range(V), key=lambda v: (-combo[v], v))
            assert (r.top1, r.top2) == (order[0], order[1]), combo
            assert r.max_logit == combo[order[0]] and r.gap == combo[order[0]] - combo[order[1]]
            assert abs(r.lse - math.log(sum(math.exp(c) for c in combo))) < 1e-12
    r = oracle.record(np.array([1.5]))
    assert (r.top1, r.top2) == (0, -1) and r.gap == math.inf and r.lse == 1.5


def test_vs_library_topk_logsumexp(oracle):
    """Pin (6): torch.topk / torch.logsumexp in fp64."""
    g = torch.Generator().manual_seed(6)
    for V in (2, 33, 1024, 128256):
        lg = torch.randn(V, generator=g, dtype=torch.float64) * 2
        r = oracle.record(lg.numpy())
        top = torch.topk(lg, 2)
        assert [r.top1, r.top2] == top.indices.tolist()
        assert r.max_logit == float(top.values[0]) and r.gap == float(top.values[0] - top.values[1])
        assert abs(r.lse - float(torch.logsumexp(lg, 0))) < 1e-12


def test_tie_break_lowest_id(oracle):
    """Reading Q8: two equal maxima => gap 0, top1 the lower id, top2 the higher; three-way ties too."""
    lg = np.zeros(50)
    lg[[7, 31]] = 4.0
    r = oracle.record(lg)
    assert (r.top1, r.top2, r.gap) == (7, 31, 0.0)
    lg[3] = 4.0
    r = oracle.record(lg)
    assert (r.top1, r.top2, r.gap) == (3, 7, 0.0)
    lg[40] = 9.0
    r = oracle.record(lg)
    assert (r.top1, r.top2, r.gap) == (40, 3, 5.0)


def test_partition_merge_associativity(oracle):
    """Pin (7): records of random partitions of the vocabulary, merged by the (logit desc, id asc) order and
    lse = m + log sum exp(lse_i - m), reproduce the whole-vocabulary record."""
    rng = np.random.default_rng(7)
    V = 4096
    lg = np.round(rng.normal(size=V) * 4) / 4          # many exact ties
    whole = oracle.record(lg)
    for trial in range(5):
        cuts = np.sort(rng.choice(np.arange(1, V), size=rng.integers(1, 9), replace=False))
        cand, lses = [], []
        for lo, hi in zip(np.r_[0, cuts], np.r_[cuts, V]):
            r = oracle.record(lg[lo:hi])
            cand += [(-(lg[lo + r.top1]), lo + r.top1)]
            if r.top2 >= 0:
                cand += [(-(lg[lo + r.top2]), lo + r.top2)]
            lses.append(r.lse)
        cand.sort()
        assert (cand[0][1], cand[1][1]) == (whole.top1, whole.top2)
        m = max(lses)
        assert abs(m + math.log(sum(math.exp(l - m) for l in lses)) - whole.lse) < 1e-12


def test_nonfinite_flag(oracle):
    """Reading Q18."""
    lg = np.zeros(10)
    assert oracle.record(lg).nonfinite == 0
    lg[4] = np.inf
    assert oracle.record(lg).nonfinite == 1
    lg[4] = np.nan
    assert oracle.record(lg).nonfinite == 1


def test_planted_margin_tracks_target(oracle):
    """Pin (8): the generator's planted rows have top1 in A and a realised gap near g* (bf16 rounding of x');
    unplanted rows have a small natural gap and top1 outside A almost surely (PAPER.md:262 shape)."""
    shape = synth.C1
    seed = synth.SEED_BASE
    w = synth.make_w_vocab(shape, seed)
    fast = synth.make_fast_set(shape, seed)
    hidden, planted, target = synth.make_hidden(shape, 40, w, fast, seed)
    assert 8 <= int(planted.sum()) <= 32
    fs = set(fast.tolist())
    for r in range(40):
        rec = oracle.record(oracle.logits(_bits(w), _bits(hidden[r])))
        if planted[r]:
            assert rec.top1 in fs
            assert abs(rec.gap - float(target[r])) < 0.25, (rec.gap, float(target[r]))
        else:
            assert rec.gap < 3.0

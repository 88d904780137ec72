"""Pins of the oracle's risk-coverage sweep O6 (Sec. 2.4) against the numbers the paper prints
for its own calibration run (tests/golden/gate_calibration_hw3.txt), closed forms and brute force."""
import itertools
import math
import os

import numpy as np
import pytest

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "gate_calibration_hw3.txt")


@pytest.fixture(scope="module")
def oracle():
    from oracle import oracle as o
    return o


def golden():
    g = {}
    for line in open(GOLDEN):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            g[k] = float(v)
    return g


def test_wilson_reproduces_the_papers_printed_intervals(oracle):
    g = golden()
    n, a, f = int(g["decision_points"]), int(g["served_at_tau_2"]), int(g["false_accepts"])
    lo, hi = oracle.wilson(a, n)
    assert round(a / n, 3) == g["coverage"]                              # 0.945
    assert round(lo, 2) == g["coverage_wilson95_lo"] and round(hi, 2) == g["coverage_wilson95_hi"]   # [0.89, 0.97]
    lo, hi = oracle.wilson(f, a)
    assert round(f / a, 3) == g["false_accept_rate"]                     # 0.132
    assert round(lo, 3) == g["false_accept_wilson95_lo"] and round(hi, 3) == g["false_accept_wilson95_hi"]
    assert abs(1 - f / a - 0.87) < 0.005                                 # "agrees ... about 87% of the time"


def test_wilson_closed_forms(oracle):
    z = oracle.Z95
    lo, hi = oracle.wilson(0, 10)
    assert lo == pytest.approx(0.0, abs=1e-15) and hi == pytest.approx(z * z / (10 + z * z))
    lo, hi = oracle.wilson(10, 10)
    assert hi == pytest.approx(1.0) and lo == pytest.approx(10 / (10 + z * z))
    lo, hi = oracle.wilson(50, 100)
    assert lo + hi == pytest.approx(1.0) and lo < 0.5 < hi               # symmetric at p = 1/2
    # the interval is the solution set of |p_hat - p| <= z sqrt(p (1 - p) / n): both ends satisfy it with equality
    for k, n in ((121, 128), (16, 121), (3, 7)):
        for p in oracle.wilson(k, n):
            assert abs(abs(k / n - p) - z * math.sqrt(p * (1 - p) / n)) < 1e-12


def test_sweep_on_pairs_with_the_papers_counts(oracle):
    """128 synthetic (gap, correct) pairs built to have the paper's counts at tau = 2.0: 121 accepted, 16 wrong."""
    g = golden()
    rng = np.random.default_rng(7)
    gap = np.concatenate([rng.uniform(2.0, 20.0, 121), rng.uniform(0.0, 1.999, 7)])   # "gaps from below 2 to ~20"
    top1 = np.arange(128) % 31
    full = top1.copy()
    wrong = rng.choice(121, 16, replace=False)
    full[wrong] = (full[wrong] + 1) % 31
    pts = oracle.risk_coverage(gap, np.ones(128, bool), top1, full, [0.0, 2.0, 25.0], strict_gt=True)
    p = pts[1]
    assert (p.accepted, p.false_accepts) == (121, 16)
    assert round(p.coverage, 3) == g["coverage"] and round(p.far, 3) == g["false_accept_rate"]
    assert (round(p.cov_lo, 2), round(p.cov_hi, 2)) == (g["coverage_wilson95_lo"], g["coverage_wilson95_hi"])
    assert (round(p.far_lo, 3), round(p.far_hi, 3)) == (g["false_accept_wilson95_lo"], g["false_accept_wilson95_hi"])
    assert pts[0].accepted == 128 and pts[0].coverage == 1.0            # "coverage 1.0 ... (low tau)"
    assert pts[2].accepted == 0 and pts[2].far == 0.0 and (pts[2].far_lo, pts[2].far_hi) == (0.0, 1.0)
    # smallest swept tau whose false-accept rate fits the budget
    # (r = 0.125 at tau = 0, 0.132 at tau = 2, and 0 where nothing is accepted)
    assert oracle.calibrate_tau(pts, 0.13) == 0.0 and oracle.calibrate_tau(pts, 0.124) == 25.0
    assert oracle.calibrate_tau(pts[1:], 0.14) == 2.0
    assert oracle.calibrate_tau(oracle.risk_coverage(gap, np.ones(128, bool), top1, full, [0.0], True), 0.01) is None


def test_coverage_monotone_and_brute_force(oracle):
    rng = np.random.default_rng(3)
    n = 9
    gap = rng.integers(0, 4, n).astype(float)
    servable = rng.integers(0, 2, n).astype(bool)
    top1 = rng.integers(0, 3, n)
    full = rng.integers(0, 3, n)
    taus = [0.0, 1.0, 2.0, 3.0, 4.0]
    for strict in (False, True):
        pts = oracle.risk_coverage(gap, servable, top1, full, taus, strict)
        assert all(a.accepted >= b.accepted for a, b in zip(pts, pts[1:]))     # Eq. 13 is non-increasing in tau
        for p in pts:
            acc = [i for i in range(n) if servable[i] and (gap[i] > p.tau if strict else gap[i] >= p.tau)]
            assert p.accepted == len(acc) and p.false_accepts == sum(top1[i] != full[i] for i in acc)
    # gamma == tau: accepted under >=, not under >
    assert oracle.risk_coverage([2.0], [True], [1], [1], [2.0], False)[0].accepted == 1
    assert oracle.risk_coverage([2.0], [True], [1], [1], [2.0], True)[0].accepted == 0
    assert oracle.risk_coverage([float("nan")], [True], [1], [1], [0.0], False)[0].accepted == 0

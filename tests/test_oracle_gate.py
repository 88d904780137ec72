"""Pins of oracle O4 (gate, Eq. 12 / Alg. 2) and O5 (invalidation state machine, Sec. 3.6 / Fig. 3)."""
import itertools

import numpy as np

from paper_2606_29565_b200 import synth

V = 100


def _bm(oracle, ids):
    return oracle.fastset_bitmap(ids, V)


def test_truth_table(oracle):
    """Eq. 12: fires iff gap >= tau and top1 in A (and the record is valid + current + eligible)."""
    bm = _bm(oracle, [5, 32])
    for valid, cur, elig, inset, big in itertools.product((0, 1), repeat=5):
        dec, tok = oracle.gate(gap=4.0 if big else 1.0, top1=5 if inset else 6, valid=valid, nonfinite=0,
                               record_version=3, session_version=3 if cur else 4,
                               record_hash=77, request_hash=77 if elig else 78, bitmap=bm, V=V, tau=3.0)
        fire = valid and cur and elig and inset and big
        assert (dec == oracle.SERVED) == bool(fire)
        assert tok == (5 if fire else -1)
        if not (valid and cur):
            assert dec == oracle.STALE_OR_INVALID        # reason order: stale, ineligible, set, gap
        elif not elig:
            assert dec == oracle.INELIGIBLE
        elif not inset:
            assert dec == oracle.NOT_IN_FAST_SET
        elif not big:
            assert dec == oracle.GAP_BELOW_TAU


def test_gap_equal_tau_both_modes(oracle):
    """Reading Q1: BASELINE's gap >= tau by default; the paper's strict gamma > tau on request."""
    bm = _bm(oracle, [9])
    kw = dict(top1=9, valid=1, nonfinite=0, record_version=1, session_version=1, record_hash=0, request_hash=0,
              bitmap=bm, V=V, tau=2.0)
    assert oracle.gate(gap=2.0, **kw)[0] == oracle.SERVED
    assert oracle.gate(gap=2.0, strict_gt=True, **kw)[0] == oracle.GAP_BELOW_TAU
    assert oracle.gate(gap=np.nextafter(2.0, 3.0), strict_gt=True, **kw)[0] == oracle.SERVED
    assert oracle.gate(gap=np.nextafter(2.0, 1.0), **kw)[0] == oracle.GAP_BELOW_TAU


def test_coverage_monotone_in_tau(oracle):
    """the accepted set is non-increasing in tau 'by construction'."""
    rng = np.random.default_rng(0)
    gaps = rng.uniform(0, 8, size=200)
    tops = rng.integers(0, V, size=200)
    bm = _bm(oracle, rng.choice(V, size=30, replace=False))
    prev = None
    for tau in np.linspace(0, 9, 37):
        fired = {i for i in range(200) if oracle.gate(gaps[i], tops[i], 1, 0, 0, 0, 0, 0, bm, V, tau)[0] == 0}
        if prev is not None:
            assert fired <= prev
        prev = fired
    assert not prev


def test_bitmap_edges(oracle):
    """Membership at ids 0, 31, 32, V-1 and their neighbours; hash 0 = relaxed match."""
    ids = [0, 31, 32, V - 1]
    bm = _bm(oracle, ids)
    assert bm.shape == ((V + 31) // 32,)
    for t in range(V):
        dec, tok = oracle.gate(5.0, t, 1, 0, 0, 0, 0, 0, bm, V, 3.0)
        assert (dec == oracle.SERVED) == (t in ids)
    assert oracle.gate(5.0, 31, 1, 0, 0, 0, 0, 123, bm, V, 3.0)[0] == oracle.SERVED
    assert oracle.gate(5.0, 31, 1, 0, 0, 0, 123, 0, bm, V, 3.0)[0] == oracle.SERVED
    assert oracle.gate(5.0, 31, 1, 1, 0, 0, 0, 0, bm, V, 3.0)[0] == oracle.STALE_OR_INVALID   # non-finite never serves


def test_lifecycle_fig3(oracle):
    """Fig. 3: fresh -> never serves; pre-positioned -> may serve; invalidated -> never serves
    until the next pre-position; versions strictly monotone; record stamped with the live version."""
    bm = _bm(oracle, [7])
    st = oracle.SessionTable(3)
    rec = oracle.Record(max_logit=9.0, lse=9.1, gap=5.0, top1=7, top2=2, nonfinite=0)
    assert st.serve(1, bm, V, 3.0) == (oracle.STALE_OR_INVALID, -1)
    st.preposition(1, rec, position=40)
    assert st.serve(1, bm, V, 3.0) == (oracle.SERVED, 7)
    assert st.serve(0, bm, V, 3.0)[0] == oracle.STALE_OR_INVALID
    st.invalidate([1])
    assert st.version[1] == 1 and st.serve(1, bm, V, 3.0) == (oracle.STALE_OR_INVALID, -1)
    st.preposition(1, rec)
    assert st.rec_version[1] == 1 and st.serve(1, bm, V, 3.0) == (oracle.SERVED, 7)
    st.invalidate([1, 1, 2])                       # repeated ids: each one is a mutation
    assert st.version.tolist() == [0, 3, 1]
    assert st.serve(1, bm, V, 3.0)[0] == oracle.STALE_OR_INVALID
    # a record whose valid bit were (wrongly) still set is refused on the version compare alone
    st.rec_valid[1] = 1
    assert st.serve(1, bm, V, 3.0)[0] == oracle.STALE_OR_INVALID


def test_config3_trace_shape(oracle):
    """Config 3 trace (reading Q16): p=0.3 bumps over 1000 updates; a stale record is never served and both
    SERVED and STALE occur."""
    bumps = synth.bump_trace(1000, synth.SEED_BASE + 2)
    assert 240 <= sum(bumps) <= 360
    bm = _bm(oracle, [7])
    st = oracle.SessionTable(1)
    rec = oracle.Record(9.0, 9.1, 5.0, 7, 2, 0)
    st.preposition(0, rec)
    served = stale = 0
    for b in bumps:
        if b:
            st.invalidate([0])
        dec, tok = st.serve(0, bm, V, 3.0)
        if b:
            assert dec == oracle.STALE_OR_INVALID and tok == -1
            stale += 1
            st.preposition(0, rec)
        else:
            assert dec == oracle.SERVED
            served += 1
    assert served and stale

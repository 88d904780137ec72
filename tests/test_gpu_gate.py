"""GPU parity of a5/a6 (prepos_gate_serve, prepos_invalidate): integer work, bit-exact against the oracle."""
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


def _pack_records(n, gap, top1, flags, version, ehash):
    """Host-side packing of a record table from given fields (layout of include/prepos.h)."""
    raw = np.zeros((n, 48), dtype=np.uint8)
    f = raw.view(np.float32).reshape(n, 12)
    i = raw.view(np.int32).reshape(n, 12)
    q = raw.view(np.int64).reshape(n, 6)
    f[:, 0] = 1.0
    f[:, 1] = 2.0
    i[:, 2] = top1
    i[:, 3] = 0
    f[:, 4] = gap
    i[:, 5] = flags
    q[:, 3] = version
    q[:, 4] = ehash
    return torch.from_numpy(raw)


def test_truth_table_random_batch(prepos, oracle):
    """4096 requests over 64 records (BASELINE config 4's serve batch) with every reason code present."""
    V, n_sess, n_req = 128256, 64, 4096
    rng = np.random.default_rng(3)
    fast = synth.make_fast_set(synth.C4, synth.SEED_BASE + 3)
    gap = rng.uniform(0, 6, n_sess).astype(np.float32)
    gap[:4] = [3.0, np.nextafter(np.float32(3.0), np.float32(0)), np.nextafter(np.float32(3.0), np.float32(9)), 0.0]
    top1 = np.where(rng.random(n_sess) < 0.7, rng.choice(fast.numpy(), n_sess), rng.integers(0, V, n_sess)).astype(np.int32)
    flags = np.where(rng.random(n_sess) < 0.85, 1, 0).astype(np.int32)
    flags[5] = 3                                   # valid but non-finite
    rec_ver = rng.integers(0, 3, n_sess)
    live = np.where(rng.random(n_sess) < 0.8, rec_ver, rec_ver + 1).astype(np.int64)
    ehash = np.where(rng.random(n_sess) < 0.5, 0, rng.integers(1, 1 << 40, n_sess)).astype(np.int64)
    recs = _pack_records(n_sess, gap, top1, flags, rec_ver, ehash).cuda()
    sids = synth.serve_requests(n_req, n_sess, synth.SEED_BASE + 3)
    rh = np.where(rng.random(n_req) < 0.5, 0, np.where(rng.random(n_req) < 0.5, ehash[sids.numpy()], 12345)).astype(np.int64)
    ctx = prepos.Context(32, 32, 8, 128, 4096, V, 16, max_sessions=64)
    bm = prepos.fastset_build(fast, V)
    obm = oracle.fastset_bitmap(fast.numpy(), V)
    for strict in (False, True):
        dec = torch.full((n_req,), -9, dtype=torch.int32, device="cuda")
        tok = torch.full((n_req,), -9, dtype=torch.int32, device="cuda")
        ctx.gate_serve(sids.cuda(), recs, torch.from_numpy(live).cuda(), bm.cuda(), 3.0, dec, tok,
                       request_entry_hash=torch.from_numpy(rh).cuda(), strict_gt=strict)
        ctx.sync()
        dec, tok = dec.cpu().numpy(), tok.cpu().numpy()
        seen = set()
        for r in range(n_req):
            s = int(sids[r])
            d, t = oracle.gate(float(gap[s]), int(top1[s]), flags[s] & 1, (flags[s] >> 1) & 1, int(rec_ver[s]),
                               int(live[s]), int(ehash[s]), int(rh[r]), obm, V, 3.0, strict)
            assert (int(dec[r]), int(tok[r])) == (d, t), (r, s)
            seen.add(d)
        assert seen == {0, 1, 2, 3, 4}
    # no hashes at all = relaxed
    dec = torch.zeros(n_req, dtype=torch.int32, device="cuda")
    tok = torch.zeros(n_req, dtype=torch.int32, device="cuda")
    ctx.gate_serve(sids.cuda(), recs, torch.from_numpy(live).cuda(), bm.cuda(), 3.0, dec, tok)
    ctx.sync()
    assert prepos.INELIGIBLE not in set(dec.cpu().tolist())


def test_tau_monotone_coverage(prepos):
    """the served set is non-increasing in tau."""
    V, n = 1024, 512
    rng = np.random.default_rng(5)
    recs = _pack_records(n, rng.uniform(0, 8, n).astype(np.float32), rng.integers(0, V, n).astype(np.int32),
                         np.ones(n, np.int32), np.zeros(n, np.int64), np.zeros(n, np.int64)).cuda()
    ctx = prepos.Context(1, 4, 2, 64, 256, V, 16, max_sessions=8)
    bm = prepos.fastset_build(rng.choice(V, 300, replace=False).tolist(), V).cuda()
    sid = torch.arange(n, dtype=torch.int32, device="cuda")
    ver = torch.zeros(n, dtype=torch.int64, device="cuda")
    prev = None
    for tau in np.linspace(0, 9, 19):
        dec = torch.zeros(n, dtype=torch.int32, device="cuda")
        tok = torch.zeros(n, dtype=torch.int32, device="cuda")
        ctx.gate_serve(sid, recs, ver, bm, float(tau), dec, tok)
        ctx.sync()
        fired = set(torch.nonzero(dec == 0).flatten().cpu().tolist())
        if prev is not None:
            assert fired <= prev
        prev = fired
    assert not prev


def test_config3_trace_invalidate_never_serves_stale(prepos, oracle):
    """BASELINE config 3 trace (reading Q16): 1000 updates, each bumping the version with p=0.3, a serve after each;
    stale records are refused; re-pre-position (ready_dist on the next hidden row of a pool of 16) after a bump.
    GPU state machine vs the oracle's SessionTable, step by step."""
    shape = synth.Shape("c3v", layers=1, Hq=4, Hkv=2, d=64, H=256, V=2048, fast_set=32, tau=3.0, planted_frac=0.75)
    seed = synth.SEED_BASE + 2
    w = synth.make_w_vocab(shape, seed)
    fast = synth.make_fast_set(shape, seed)
    pool, _, _ = synth.make_hidden(shape, 16, w, fast, seed)
    from helpers import bits
    refs = [oracle.record(oracle.logits(bits(w), bits(pool[r]))) for r in range(16)]
    bumps = synth.bump_trace(1000, seed)
    ctx = prepos.Context(1, 4, 2, 64, 256, 2048, 16, max_sessions=4)
    wd, pd = w.cuda(), pool.cuda()
    recs = prepos.new_records(2)
    ver = torch.zeros(2, dtype=torch.int64, device="cuda")
    sid = torch.tensor([1], dtype=torch.int32, device="cuda")
    bm = prepos.fastset_build(fast, shape.V).cuda()
    obm = oracle.fastset_bitmap(fast.numpy(), shape.V)
    st = oracle.SessionTable(2)
    decs = torch.full((1000,), -9, dtype=torch.int32, device="cuda")
    toks = torch.full((1000,), -9, dtype=torch.int32, device="cuda")
    exp, cur = [], 0
    ctx.ready_dist(sid, pd[0:1], wd, recs, ver)
    st.preposition(1, refs[0])
    for t, b in enumerate(bumps):
        if b:
            ctx.invalidate(sid, ver, recs)
            st.invalidate([1])
        ctx.gate_serve(sid, recs, ver, bm, shape.tau, decs[t:t + 1], toks[t:t + 1])
        exp.append(st.serve(1, obm, shape.V, shape.tau))
        if b:
            assert exp[-1] == (oracle.STALE_OR_INVALID, -1)
            cur = (cur + 1) % 16
            ctx.ready_dist(sid, pd[cur:cur + 1], wd, recs, ver)
            st.preposition(1, refs[cur])
    ctx.sync()
    got = list(zip(decs.cpu().tolist(), toks.cpu().tolist()))
    amb = [abs(r.gap - shape.tau) < 4e-2 or r.gap < 4e-2 for r in refs]
    assert not any(amb), "regenerate the pool: an ambiguous record would make the trace comparison inexact"
    assert got == exp
    assert sum(1 for d, _ in got if d == 0) > 0 and sum(1 for d, _ in got if d == 3) == sum(bumps)
    assert int(ver[1]) == sum(bumps) and int(ver[0]) == 0
    # repeated ids: each occurrence is one mutation
    ctx.invalidate(torch.tensor([1, 1, 0], dtype=torch.int32, device="cuda"), ver, recs)
    ctx.sync()
    assert ver.cpu().tolist() == [1, sum(bumps) + 2]
    assert prepos.unpack_records(recs)["flags"].tolist() == [0, 0]


def test_publication_is_safe_across_streams(prepos, oracle):
    """Sec. 3.6 with writer and reader on DIFFERENT streams over ONE record: stream A loops
    invalidate + ready_dist, alternating a hidden row X (top-1 a in A, gap well above tau) and a row Y (top-1 b in A,
    b != a, gap well below tau); stream B loops batched gate serves on the same record.  The oracle's two records
    give the only legal (top1, gap) pairs, so the only token that may ever be SERVED is a: a serve that paired Y's
    top-1 with X's gap (fields of two publications) would return b.  Every served record must also have been fresh:
    the decision buffer is checked against the two legal outcomes per request."""
    shape = synth.Shape("pub", layers=1, Hq=4, Hkv=2, d=64, H=256, V=2048, fast_set=32, tau=3.0, planted_frac=1.0)
    seed = 4242
    w = synth.make_w_vocab(shape, seed)
    fast = synth.make_fast_set(shape, seed)
    pool, _, _ = synth.make_hidden(shape, 24, w, fast, seed)
    from helpers import bits
    refs = [oracle.record(oracle.logits(bits(w), bits(pool[r]))) for r in range(24)]
    in_a = set(fast.tolist())
    xs = [r for r in range(24) if refs[r].gap >= shape.tau + 0.5 and refs[r].top1 in in_a]
    assert xs
    x = xs[0]
    ys = [r for r in range(24) if 0.2 <= refs[r].gap <= shape.tau - 0.5 and refs[r].top1 in in_a and refs[r].top1 != refs[x].top1]
    assert ys
    y = ys[0]
    a_tok = refs[x].top1
    ctx_w = prepos.Context(1, 4, 2, 64, 256, 2048, 16, max_sessions=2)
    ctx_r = prepos.Context(1, 4, 2, 64, 256, 2048, 16, max_sessions=2)
    wd, pd = w.cuda(), pool.cuda()
    recs = prepos.new_records(1)
    ver = torch.zeros(1, dtype=torch.int64, device="cuda")
    sid = torch.zeros(1, dtype=torch.int32, device="cuda")
    bm = prepos.fastset_build(fast, shape.V).cuda()
    iters, B = 400, 256
    req = torch.zeros(B, dtype=torch.int32, device="cuda")
    decs = torch.full((2 * iters, B), -9, dtype=torch.int32, device="cuda")
    toks = torch.full((2 * iters, B), -9, dtype=torch.int32, device="cuda")
    exp = torch.arange(1, iters + 1, dtype=torch.int64, device="cuda")   # the version after the i-th invalidate
    sa, sb_ = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    for i in range(iters):
        with torch.cuda.stream(sa):
            ctx_w.invalidate(sid, ver, recs)
            r = x if i % 2 == 0 else y
            ctx_w.ready_dist(sid, pd[r:r + 1], wd, recs, ver, expected_version=exp[i:i + 1])
        with torch.cuda.stream(sb_):
            for k in range(2):
                ctx_r.gate_serve(req, recs, ver, bm, shape.tau, decs[2 * i + k], toks[2 * i + k])
    torch.cuda.synchronize()
    d, t = decs.cpu().numpy(), toks.cpu().numpy()
    assert set(np.unique(d).tolist()) <= {prepos.SERVED, prepos.GAP_BELOW_TAU, prepos.STALE_OR_INVALID}
    served = d == prepos.SERVED
    assert (t[served] == a_tok).all(), f"served tokens {np.unique(t[served])}, legal: {a_tok}"
    assert (t[~served] == -1).all()
    # and in stream order the last publication (row y: gap below tau) is what a serve sees
    ctx_r.gate_serve(req, recs, ver, bm, shape.tau, decs[0], toks[0])
    ctx_r.sync()
    last = x if (iters - 1) % 2 == 0 else y
    want = prepos.SERVED if last == x else prepos.GAP_BELOW_TAU
    assert (decs[0].cpu().numpy() == want).all()
    assert prepos.unpack_records(recs)["seq"].tolist() == [iters]


def test_gate_sweep_matches_oracle_risk_coverage(prepos, oracle):
    """prepos_gate_sweep (Eq. 13-14) on records the GPU produced itself: 512 sessions of the
    tiny config with planted margins, a third of them invalidated, full-path tokens that disagree on some rows;
    counts bit-exact against oracle O6 (fed with the GPU's own gap / top-1, so no fp decision differs), rates and
    Wilson intervals to 1e-12, under both inequality modes, including gamma == tau and an empty sweep."""
    shape, seed, n = synth.C1, synth.SEED_BASE + 40, 512
    w = synth.make_w_vocab(shape, seed, "cuda")
    fast = synth.make_fast_set(shape, seed)
    hidden, _, _ = synth.make_hidden(shape, n, w, fast.cuda(), seed, planted_frac=0.8)
    ctx = prepos.Context(shape.layers, shape.Hq, shape.Hkv, shape.d, shape.H, shape.V, shape.page, max_sessions=n)
    sid = torch.arange(n, dtype=torch.int32, device="cuda")
    recs = prepos.new_records(n)
    ver = torch.zeros(n, dtype=torch.int64, device="cuda")
    ctx.ready_dist(sid, hidden, w, recs, ver)
    stale = torch.arange(0, n, 3, dtype=torch.int32, device="cuda")
    ctx.invalidate(stale, ver, recs)                     # these records must never count as accepted
    bm = prepos.fastset_build(fast, shape.V).cuda()
    rec = prepos.unpack_records(recs)
    g = synth.gen(seed + 1)
    full = rec["top1"].clone().to(torch.int32)
    flip = torch.rand(n, generator=g) < 0.15
    full[flip] = (full[flip] + 1) % shape.V
    gap = rec["gap"].numpy().astype(np.float64)
    taus = [0.0, 1.0, 2.0, 3.0, float(rec["gap"][1]), 4.5, 6.0, 1e9]   # one threshold exactly on a record's gap
    in_set = np.isin(rec["top1"].numpy(), fast.numpy())
    servable = in_set & (np.arange(n) % 3 != 0)
    for strict in (False, True):
        out = ctx.gate_sweep(recs, ver, bm, full.cuda(), torch.tensor(taus, dtype=torch.float32, device="cuda"), strict)
        ctx.sync()
        got = prepos.unpack_sweep(out)
        ref = oracle.risk_coverage(gap, servable, rec["top1"].numpy(), full.numpy(),
                                   [float(np.float32(t)) for t in taus], strict)
        for t, p in enumerate(ref):
            assert (int(got["n"][t]), int(got["accepted"][t]), int(got["false_accepts"][t])) == (n, p.accepted, p.false_accepts)
            for k in ("coverage", "far", "cov_lo", "cov_hi", "far_lo", "far_hi"):
                assert abs(float(got[k][t]) - getattr(p, k)) <= 1e-12, (k, t)
        assert int(got["accepted"][0]) > 0 and int(got["accepted"][-1]) == 0
        srt = sorted(range(len(taus)), key=lambda t: taus[t])
        assert all(int(got["accepted"][a]) >= int(got["accepted"][b]) for a, b in zip(srt, srt[1:]))   # Eq. 13 monotone
    # decisions of prepos_gate_serve agree with the sweep's count at the same tau
    dec = torch.zeros(n, dtype=torch.int32, device="cuda")
    tok = torch.zeros(n, dtype=torch.int32, device="cuda")
    ctx.gate_serve(sid, recs, ver, bm, 3.0, dec, tok)
    out = ctx.gate_sweep(recs, ver, bm, full.cuda(), torch.tensor([3.0], dtype=torch.float32, device="cuda"))
    ctx.sync()
    assert int((dec == 0).sum()) == int(prepos.unpack_sweep(out)["accepted"][0])


def test_gate_serve_runs_beside_a_running_preposition(prepos):
    """the idle-window pass "yields to any request".  The persistent
    attention kernel leaves registers and shared memory for one small CTA per SM, so a gate serve issued on a
    high-priority stream while a long pre-position (~1 ms of attention) runs on a low-priority stream completes
    long before it: after the serve has synchronised, the pre-position's end event has not fired."""
    shape = synth.Shape("cosched", layers=48, Hq=64, Hkv=8, d=128, H=256, V=1024, page=16)
    sb = synth.make_sessions(shape, [16384], [32], seed=5, device="cuda")
    ctx = prepos.Context(shape.layers, shape.Hq, shape.Hkv, shape.d, shape.H, shape.V, shape.page, max_sessions=1)
    out = torch.empty_like(sb.q)
    n = 64
    ctx2 = prepos.Context(1, 4, 2, 64, 256, 1024, 16, max_sessions=n)
    recs = prepos.new_records(n)
    ver = torch.zeros(n, dtype=torch.int64, device="cuda")
    sid = torch.arange(n, dtype=torch.int32, device="cuda")
    bm = prepos.fastset_build(torch.arange(16), 1024).cuda()
    dec = torch.zeros(n, dtype=torch.int32, device="cuda")
    tok = torch.zeros(n, dtype=torch.int32, device="cuda")
    lo, hi = torch.cuda.Stream(priority=0), torch.cuda.Stream(priority=-1)
    done = torch.cuda.Event()
    ahead = 0
    for _ in range(5):
        torch.cuda.synchronize()
        with torch.cuda.stream(lo):
            ctx.entry_attn(sb.q, sb.k_new, sb.v_new, sb.k_pool, sb.v_pool, sb.page_table, sb.n_s, sb.l_entry,
                           sb.capacity, out)
            done.record(lo)
        with torch.cuda.stream(hi):
            ctx2.gate_serve(sid, recs, ver, bm, 3.0, dec, tok)
        hi.synchronize()
        ahead += not done.query()
        torch.cuda.synchronize()
    assert ahead >= 4, f"the gate serve overtook the running pre-position only {ahead} of 5 times"
    assert bool((dec == 3).all())        # fresh records were never pre-positioned: STALE_OR_INVALID

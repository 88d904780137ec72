"""GPU parity of a3/a4/a4' (prepos_ready_dist, prepos_scan_logits) against the oracle, through the C ABI."""
import numpy as np
import pytest
import torch

from paper_2606_29565_b200 import synth
from helpers import bits, check_record, check_decision, LOGIT_ATOL

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def prepos():
    from paper_2606_29565_b200 import prepos as p
    p.lib()
    return p


def _run_ready(prepos, shape, hidden, w, n_sessions=None, with_logits=True, session_ids=None, skip=None,
               versions=None, position=None, ehash=None):
    n = hidden.shape[0]
    n_sessions = n if n_sessions is None else n_sessions
    ctx = prepos.Context(shape.layers, shape.Hq, shape.Hkv, shape.d, shape.H, shape.V, shape.page, max_sessions=max(n, 1))
    dev = "cuda"
    sid = torch.arange(n, dtype=torch.int32, device=dev) if session_ids is None else session_ids.to(dev)
    recs = prepos.new_records(n_sessions)
    ver = torch.zeros(n_sessions, dtype=torch.int64, device=dev) if versions is None else versions.to(dev)
    logits = torch.full((n, shape.V), float("nan"), dtype=torch.float32, device=dev) if with_logits else None
    ctx.ready_dist(sid, hidden.to(dev), w.to(dev), recs, ver, position_p=None if position is None else position.to(dev),
                   entry_hash=None if ehash is None else ehash.to(dev), skip_mask=None if skip is None else skip.to(dev),
                   logits_out=logits)
    ctx.sync()
    return ctx, recs, ver, logits


def test_config1_many_seeds_records_and_gate(prepos, oracle):
    """BASELINE config 1 vocabulary side: 208 hidden rows (50% planted), records + gate decisions vs oracle."""
    shape, seed = synth.C1, synth.SEED_BASE
    w = synth.make_w_vocab(shape, seed)
    fast = synth.make_fast_set(shape, seed)
    hidden, planted, _ = synth.make_hidden(shape, 208, w, fast, seed)
    ctx, recs, ver, logits = _run_ready(prepos, shape, hidden, w)
    rec = prepos.unpack_records(recs)
    lg_gpu = logits.cpu().numpy()
    bm_host = prepos.fastset_build(fast, shape.V)
    assert np.array_equal(bm_host.numpy().view(np.uint32), oracle.fastset_bitmap(fast.numpy(), shape.V))
    n = hidden.shape[0]
    dec = torch.full((n,), -7, dtype=torch.int32, device="cuda")
    tok = torch.full((n,), -7, dtype=torch.int32, device="cuda")
    ctx.gate_serve(torch.arange(n, dtype=torch.int32, device="cuda"), recs, ver, bm_host.cuda(), shape.tau, dec, tok)
    ctx.sync()
    dec, tok = dec.cpu().tolist(), tok.cpu().tolist()
    served = 0
    wb, obm = bits(w), oracle.fastset_bitmap(fast.numpy(), shape.V)
    for r in range(n):
        lg64 = oracle.logits(wb, bits(hidden[r]))
        ref = check_record(oracle, rec, r, lg64, lg_gpu[r])
        assert int(rec["flags"][r]) == prepos.FLAG_VALID
        d, _ = check_decision(oracle, dec[r], tok[r], ref, True, 0, 0, obm, shape.V, shape.tau)
        served += d == oracle.SERVED
    assert 20 <= served <= 100      # planted rows with realised gap >= 3 fire; unplanted never


@pytest.mark.parametrize("V,H,n", [(1000, 128, 3), (130, 384, 1), (257, 256, 9), (4096, 1024, 8), (2, 128, 1),
                                   (1000, 128, 33), (513, 256, 64), (300, 384, 100), (4096, 1024, 128), (200, 128, 130),
                                   (20000, 512, 17)])
def test_ragged_vocab_and_batches(prepos, oracle, V, H, n):
    """V not a multiple of the 128-row tile, H with a single stage, n crossing the 8-row pass (streaming kernel)
    into the batched tensor-core kernel (9..128 rows per launch: 32-, 64- and 128-row hidden boxes, a ragged last
    tile, more tiles than CTAs, and n > 128 = two launches)."""
    shape = synth.Shape("r", layers=1, Hq=4, Hkv=2, d=64, H=H, V=V, fast_set=2)
    w = synth.make_w_vocab(shape, 5)
    hidden = synth.randn_bf16((n, H), synth.gen(6))
    ctx, recs, ver, logits = _run_ready(prepos, shape, hidden, w)
    rec = prepos.unpack_records(recs)
    for r in range(n):
        check_record(oracle, rec, r, oracle.logits(bits(w), bits(hidden[r])), logits[r].cpu().numpy())


def test_ties_lowest_id_wins(prepos, oracle):
    """Reading Q8: duplicated W rows give bit-equal logits on the GPU; the lower id must be top1, gap 0."""
    shape = synth.Shape("t", layers=1, Hq=4, Hkv=2, d=64, H=256, V=700, fast_set=2)
    w = synth.make_w_vocab(shape, 8)
    hidden = synth.randn_bf16((2, 256), synth.gen(9))
    lg = oracle.logits(bits(w), bits(hidden[0]))
    best = int(np.argmax(lg))
    dup = [3, 650] if best not in (3, 650) else [5, 651]
    w[dup[0]] = w[best]
    w[dup[1]] = w[best]
    ctx, recs, ver, _ = _run_ready(prepos, shape, hidden[:1], w, with_logits=False)
    rec = prepos.unpack_records(recs)
    ids = sorted([best] + dup)
    assert int(rec["top1"][0]) == ids[0] and int(rec["top2"][0]) == ids[1]
    assert float(rec["gap"][0]) == 0.0
    ref = oracle.record(oracle.logits(bits(w), bits(hidden[0])))
    assert (ref.top1, ref.top2, ref.gap) == (ids[0], ids[1], 0.0)


def test_record_stamping_skip_and_ids(prepos, oracle):
    """Alg. 1 l.10-12: position, hash, live version stamped; skip_mask rows untouched; records indexed by id."""
    shape = synth.Shape("s", layers=1, Hq=4, Hkv=2, d=64, H=128, V=300, fast_set=2)
    w = synth.make_w_vocab(shape, 11)
    hidden = synth.randn_bf16((3, 128), synth.gen(12))
    sid = torch.tensor([4, 0, 2], dtype=torch.int32)
    ver = torch.tensor([7, 0, 9, 0, 11], dtype=torch.int64)
    pos = torch.tensor([100, 200, 300], dtype=torch.int64)
    eh = torch.tensor([0x1234, 0, 0x7fffffffffffffff], dtype=torch.int64)
    skip = torch.tensor([0, 1, 0], dtype=torch.int32)
    ctx, recs, _, _ = _run_ready(prepos, shape, hidden, w, n_sessions=5, session_ids=sid, skip=skip, versions=ver,
                                 position=pos, ehash=eh, with_logits=False)
    rec = prepos.unpack_records(recs)
    assert rec["flags"].tolist() == [0, 0, 1, 0, 1]
    assert rec["version"].tolist() == [0, 0, 9, 0, 11]
    assert rec["position"].tolist() == [0, 0, 300, 0, 100]
    assert rec["entry_hash"].tolist() == [0, 0, 0x7fffffffffffffff, 0, 0x1234]
    for row, s in ((0, 4), (2, 2)):
        check_record(oracle, rec, s, oracle.logits(bits(w), bits(hidden[row])))


def test_expected_version_stamp_and_publication_sequence(prepos, oracle):
    """Sec. 3.6: the record is stamped with the version its inputs were computed at
    (`expected_version`), and is VALID only if that is still the live version when the pass ends; a record computed
    for an older state is written but never served.  Each publication advances the sequence number in flags[2:]."""
    shape = synth.Shape("ev", layers=1, Hq=4, Hkv=2, d=64, H=128, V=300, fast_set=2)
    w = synth.make_w_vocab(shape, 21).cuda()
    hidden = synth.randn_bf16((3, 128), synth.gen(22)).cuda()
    ctx = prepos.Context(1, 4, 2, 64, 128, 300, 16, max_sessions=4)
    sid = torch.tensor([0, 1, 2], dtype=torch.int32, device="cuda")
    ver = torch.tensor([5, 6, 7], dtype=torch.int64, device="cuda")
    exp = torch.tensor([5, 5, 8], dtype=torch.int64, device="cuda")      # fresh, computed at an older state, newer
    recs = prepos.new_records(3)
    bm = prepos.fastset_build(list(range(300)), 300).cuda()
    dec = torch.zeros(3, dtype=torch.int32, device="cuda")
    tok = torch.zeros(3, dtype=torch.int32, device="cuda")
    for rnd in range(3):
        ctx.ready_dist(sid, hidden, w, recs, ver, expected_version=exp)
        ctx.gate_serve(sid, recs, ver, bm, -1e30, dec, tok)
        ctx.sync()
        rec = prepos.unpack_records(recs)
        assert rec["flags"].tolist() == [1, 0, 0] and rec["version"].tolist() == [5, 5, 8]
        assert rec["seq"].tolist() == [rnd + 1] * 3
        assert dec.cpu().tolist() == [prepos.SERVED, prepos.STALE_OR_INVALID, prepos.STALE_OR_INVALID]
        check_record(oracle, rec, 1, oracle.logits(bits(w), bits(hidden[1])))    # written, just not valid
    # a mutation that commits on ANOTHER stream while the pre-position runs must win: full-size vocabulary
    # (~0.17 ms of streaming), the bump is issued right behind it on a second stream
    shape2 = synth.C2
    w2 = synth.make_w_vocab(shape2, 23, "cuda")
    h2 = synth.randn_bf16((1, shape2.H), synth.gen(24, "cuda"))
    ctx2 = prepos.Context(shape2.layers, shape2.Hq, shape2.Hkv, shape2.d, shape2.H, shape2.V, 16, max_sessions=1)
    s0 = torch.zeros(1, dtype=torch.int32, device="cuda")
    bm2 = prepos.fastset_build(list(range(0, shape2.V, 2)), shape2.V).cuda()
    a, b = torch.cuda.Stream(), torch.cuda.Stream()
    raced = 0
    for it in range(20):
        recs2 = prepos.new_records(1)
        ver2 = torch.zeros(1, dtype=torch.int64, device="cuda")
        exp2 = torch.zeros(1, dtype=torch.int64, device="cuda")
        d2 = torch.zeros(1, dtype=torch.int32, device="cuda")
        t2 = torch.zeros(1, dtype=torch.int32, device="cuda")
        torch.cuda.synchronize()
        with torch.cuda.stream(a):
            ctx2.ready_dist(s0, h2, w2, recs2, ver2, expected_version=exp2)
        with torch.cuda.stream(b):
            ctx.invalidate(s0, ver2, recs2)
        torch.cuda.synchronize()
        ctx2.gate_serve(s0, recs2, ver2, bm2, -1e30, d2, t2)
        ctx2.sync()
        r2 = prepos.unpack_records(recs2)
        assert int(ver2[0]) == 1 and int(r2["version"][0]) == 0          # stamped with the state it was computed at
        assert (int(d2[0]), int(t2[0])) == (prepos.STALE_OR_INVALID, -1)
        raced += int(r2["flags"][0]) == 0
    # (informational: `raced` counts the runs where the bump landed before the pass ended)


def test_nonfinite_logit_is_flagged_and_never_served(prepos, oracle):
    shape = synth.Shape("n", layers=1, Hq=4, Hkv=2, d=64, H=128, V=256, fast_set=2)
    w = synth.make_w_vocab(shape, 13)
    hidden = synth.randn_bf16((1, 128), synth.gen(14))
    w[17, 5] = float("inf")
    ctx, recs, ver, _ = _run_ready(prepos, shape, hidden, w, with_logits=False)
    rec = prepos.unpack_records(recs)
    assert int(rec["flags"][0]) & prepos.FLAG_NONFINITE
    bm = prepos.fastset_build(list(range(256)), 256).cuda()
    dec = torch.zeros(1, dtype=torch.int32, device="cuda")
    tok = torch.zeros(1, dtype=torch.int32, device="cuda")
    ctx.gate_serve(torch.zeros(1, dtype=torch.int32, device="cuda"), recs, ver, bm, -1e30, dec, tok)
    ctx.sync()
    assert (int(dec[0]), int(tok[0])) == (prepos.STALE_OR_INVALID, -1)


def test_scan_logits_matches_oracle_and_shift_invariance(prepos, oracle):
    """a4' on stored fp32 logits: ids exact (same fp32 values on both sides); shift by c moves max/lse by c."""
    V = 128256
    shape = synth.Shape("v", layers=1, Hq=4, Hkv=2, d=64, H=128, V=V, fast_set=2)
    ctx = prepos.Context(1, 4, 2, 64, 128, V, 16, max_sessions=4)
    g = synth.gen(21, "cuda")
    lg = torch.randn((3, V), generator=g, device="cuda", dtype=torch.float32) * 2
    lg[1] = (lg[1] * 4).round() / 4          # many exact ties
    lg[2] = lg[0] + 16.0
    recs = prepos.new_records(3)
    ctx.scan_logits(lg, recs)
    ctx.sync()
    rec = prepos.unpack_records(recs)
    host = lg.cpu().numpy().astype(np.float64)
    for r in range(3):
        ref = oracle.record(host[r])
        assert (int(rec["top1"][r]), int(rec["top2"][r])) == (ref.top1, ref.top2)
        assert abs(float(rec["gap"][r]) - ref.gap) < 1e-5 and abs(float(rec["max_logit"][r]) - ref.max_logit) < 1e-6
        assert abs(float(rec["lse"][r]) - ref.lse) <= 1e-4 * abs(ref.lse)
    assert int(rec["top1"][2]) == int(rec["top1"][0]) and int(rec["top2"][2]) == int(rec["top2"][0])
    assert abs(float(rec["lse"][2]) - float(rec["lse"][0]) - 16.0) < 1e-3
    # unaligned row base (V odd) and tiny V
    for V2 in (5, 1023):
        ctx2 = prepos.Context(1, 4, 2, 64, 128, V2, 16, max_sessions=4)
        lg2 = torch.randn((2, V2), generator=g, device="cuda", dtype=torch.float32)
        r2 = prepos.new_records(2)
        ctx2.scan_logits(lg2, r2)
        ctx2.sync()
        rr = prepos.unpack_records(r2)
        for r in range(2):
            ref = oracle.record(lg2[r].cpu().numpy().astype(np.float64))
            assert (int(rr["top1"][r]), int(rr["top2"][r])) == (ref.top1, ref.top2)


@pytest.mark.parametrize("name,n", [("c2", 1), ("c2", 12), ("c4", 64), ("c5", 1), ("c5", 4)])
def test_full_size_vocabulary(prepos, oracle, name, n):
    """BASELINE configs 2, 4 and 5 vocabulary side at full size (V=128256, H=4096 / 8192), in the launch
    configurations bench.py times: one hidden row (streaming kernel), 12 rows and the 64-session batch of config 4
    (one pass of the batched tensor-core kernel), planted fraction 0.6: full logits + records against the oracle;
    for config 4 also its 4096 gate serves over the 64 records, every decision against O4.  Config 5 with n = 4 is
    the record of every session bench.py keeps resident.  Config 3's vocabulary side is config 2's launch (same V,
    H, W_vocab recipe and one hidden row), so ("c2", 1) covers it."""
    shape = {"c2": synth.C2, "c4": synth.C4, "c5": synth.C5}[name]
    seed = synth.SEED_BASE + int(name[1])
    w = synth.make_w_vocab(shape, seed, "cuda")
    fast = synth.make_fast_set(shape, seed)
    hidden, planted, target = synth.make_hidden(shape, n, w, fast.cuda(), seed)
    ctx, recs, ver, logits = _run_ready(prepos, shape, hidden, w)
    rec = prepos.unpack_records(recs)
    wb = bits(w)
    obm = oracle.fastset_bitmap(fast.numpy(), shape.V)
    bm = prepos.fastset_build(fast, shape.V).cuda()
    n_req = 4096 if name == "c4" else n
    req = (torch.randint(0, n, (n_req,), generator=synth.gen(seed + 77), dtype=torch.int32) if name == "c4"
           else torch.arange(n, dtype=torch.int32))
    dec = torch.zeros(n_req, dtype=torch.int32, device="cuda")
    tok = torch.zeros(n_req, dtype=torch.int32, device="cuda")
    ctx.gate_serve(req.cuda(), recs, ver, bm, shape.tau, dec, tok)
    ctx.sync()
    dec, tok = dec.cpu(), tok.cpu()
    refs, fired = [], 0
    for r in range(n):
        ref = check_record(oracle, rec, r, oracle.logits(wb, bits(hidden[r])), logits[r].cpu().numpy())
        refs.append(ref)
        if planted[r]:
            assert abs(ref.gap - float(target[r])) < 0.3
    for q in range(n_req):
        r = int(req[q])
        d, _ = check_decision(oracle, int(dec[q]), int(tok[q]), refs[r], True, 0, 0, obm, shape.V, shape.tau)
        fired += d == oracle.SERVED
    assert fired >= 1 or n == 1


# ---------------------------------------------------------------- NEXT-4: 4-bit W_vocab (reading Q21, oracle O8)
def _run_ready_w4(prepos, shape, hidden, w4, sc, with_logits=True):
    n = hidden.shape[0]
    ctx = prepos.Context(shape.layers, shape.Hq, shape.Hkv, shape.d, shape.H, shape.V, shape.page, max_sessions=max(n, 1))
    dev = "cuda"
    sid = torch.arange(n, dtype=torch.int32, device=dev)
    recs = prepos.new_records(n)
    ver = torch.zeros(n, dtype=torch.int64, device=dev)
    logits = torch.full((n, shape.V), float("nan"), dtype=torch.float32, device=dev) if with_logits else None
    ctx.ready_dist_w4(sid, hidden.to(dev), w4.to(dev), sc.to(dev), recs, ver, logits_out=logits)
    ctx.sync()
    return ctx, recs, ver, logits


@pytest.mark.parametrize("V,H,n", [(1024, 256, 1), (1000, 128, 3), (130, 384, 8), (257, 640, 9), (4096, 1024, 8),
                                   (2, 128, 1), (20000, 512, 5), (513, 2048, 20)])
def test_w4_ragged_vocab_vs_oracle(prepos, oracle, V, H, n):
    """prepos_ready_dist_w4 against O8 (logits over the int4 codes and group scales, reading Q21) + O3: every logit
    and the record, for V not a multiple of the 128-row tile, H / 128 = 1, 2, 3, 4, 5, 8, 16 scale groups (whole and
    partial 4-box stages), n below, at and above the 8-row pass."""
    shape = synth.Shape("w4", layers=1, Hq=4, Hkv=2, d=64, H=H, V=V, fast_set=2)
    w4, sc = synth.make_w_vocab_w4(shape, 5)
    hidden = synth.randn_bf16((n, H), synth.gen(6))
    ctx, recs, ver, logits = _run_ready_w4(prepos, shape, hidden, w4, sc)
    rec = prepos.unpack_records(recs)
    assert rec["flags"].tolist() == [prepos.FLAG_VALID] * n
    for r in range(n):
        check_record(oracle, rec, r, oracle.logits_w4(w4.numpy(), bits(sc), bits(hidden[r])), logits[r].cpu().numpy())


def test_w4_extreme_codes_and_unit_scales(prepos, oracle):
    """Every code value -8..7 in every nibble position with power-of-two scales and a hidden row of small integers:
    all products and sums are exact in fp32, so the GPU logits must EQUAL the oracle's (catches a wrong nibble order,
    sign extension or k permutation, which a tolerance could hide)."""
    V, H = 256, 256
    shape = synth.Shape("w4x", layers=1, Hq=4, Hkv=2, d=64, H=H, V=V, fast_set=2)
    g = torch.Generator().manual_seed(3)
    codes = torch.randint(-8, 8, (V, H), generator=g, dtype=torch.int16)
    codes[0, :16] = torch.arange(-8, 8, dtype=torch.int16)
    nib = (codes & 15).to(torch.uint8)
    w4 = (nib[:, 0::2] | (nib[:, 1::2] << 4)).contiguous()
    sc = (2.0 ** torch.randint(-3, 3, (V, H // 128), generator=g).float()).to(torch.bfloat16)
    hidden = torch.randint(-4, 5, (3, H), generator=g).to(torch.bfloat16)
    hidden[1] = 0
    hidden[1, 5] = 1          # picks column 5 of W: logits = code[:, 5] * scale
    ctx, recs, ver, logits = _run_ready_w4(prepos, shape, hidden, w4, sc)
    for r in range(3):
        ref = oracle.logits_w4(w4.numpy(), bits(sc), bits(hidden[r]))
        assert np.array_equal(logits[r].cpu().numpy().astype(np.float64), ref), r


@pytest.mark.parametrize("name,n", [("c2", 1), ("c4", 64), ("c5", 4)])
def test_w4_full_size_vocabulary(prepos, oracle, name, n):
    """The int4 LM head at BASELINE's vocabulary shapes (V = 128256, H = 4096 / 8192) in bench.py's launch
    configuration: every logit of every row and the records against O8 + O3.  Config 4 is its 64-session batch:
    eight passes of 8 rows over the codes."""
    shape = {"c2": synth.C2, "c4": synth.C4, "c5": synth.C5}[name]
    seed = synth.SEED_BASE + int(name[1])
    w4, sc = synth.make_w_vocab_w4(shape, seed, "cuda")
    hidden = synth.randn_bf16((n, shape.H), synth.gen(seed + 1, "cuda"))
    ctx, recs, ver, logits = _run_ready_w4(prepos, shape, hidden, w4, sc)
    rec = prepos.unpack_records(recs)
    w4h, sch = w4.cpu().numpy(), bits(sc)
    for r in range(n):
        check_record(oracle, rec, r, oracle.logits_w4(w4h, sch, bits(hidden[r])), logits[r].cpu().numpy())

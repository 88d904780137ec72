"""GPU parity of a0/a1/a2 (prepos_entry_attn) against oracle O1, through the C ABI."""
import numpy as np
import pytest
import torch

from paper_2606_29565_b200 import synth
from helpers import bits, oracle_attn_batch, oracle_attn_rows, check_attn, ATTN_ATOL

pytestmark = pytest.mark.gpu

PATHS = [1, 2]   # 1 = generic CUDA-core kernel, 2 = tcgen05 kernel


@pytest.fixture(scope="module")
def prepos():
    from paper_2606_29565_b200 import prepos as p
    p.lib()
    return p


def _ctx(prepos, shape, n_sessions, path):
    ctx = prepos.Context(shape.layers, shape.Hq, shape.Hkv, shape.d, shape.H, shape.V, shape.page,
                         max_sessions=max(n_sessions, 1))
    try:
        ctx.set_attn_path(path)
    except prepos.PreposError as e:
        if e.status == prepos.E_SHAPE:
            pytest.skip("shape not taken by the tcgen05 path")
        raise
    return ctx


def _gpu_run(prepos, sb, path, layers=None, poison=True):
    """Copies the batch to the GPU (optionally NaN-poisoning every pool slot beyond n_s), runs entry_attn."""
    shape = sb.shape
    dev = "cuda"
    kp, vp = sb.k_pool.to(dev).clone(), sb.v_pool.to(dev).clone()
    if poison:
        page = shape.page
        used = torch.zeros(kp.shape[1] * page, dtype=torch.bool)
        pt = sb.page_table.cpu()
        for s in range(sb.n_sessions):
            j = torch.arange(sb.n_s[s])
            used[pt[s, j // page].long() * page + j % page] = True
        mask = (~used).view(kp.shape[1], 1, page, 1).to(dev)
        kp.masked_fill_(mask, float("nan"))
        vp.masked_fill_(mask, float("nan"))
    before = (kp.clone(), vp.clone())
    out = torch.full(sb.q.shape, float("nan"), dtype=torch.bfloat16, device=dev)
    ctx = _ctx(prepos, shape, sb.n_sessions, path)
    nl = sb.k_pool.shape[0]
    lb, le = (0, nl) if layers is None else layers
    status = ctx.entry_attn(sb.q.to(dev), sb.k_new.to(dev), sb.v_new.to(dev), kp, vp, sb.page_table.to(dev),
                            sb.n_s, sb.l_entry, sb.capacity, out, layer_begin=lb, layer_end=le)
    ctx.sync()
    return out, kp, vp, before, status, ctx


def _check_append(sb, kp, vp, before, status, layers):
    """a1 post-condition: appended slots == K_new/V_new bit for bit; every other pool element bit-identical."""
    page = sb.shape.page
    pt = sb.page_table.cpu()
    for l in layers:
        touched = torch.zeros(kp.shape[1], page, dtype=torch.bool)
        for s in range(sb.n_sessions):
            if status[s] != 0:
                continue
            r0 = sb.row_offset[s]
            for jp in range(sb.l_entry[s]):
                j = sb.n_s[s] + jp
                pg, sl = int(pt[s, j // page]), j % page
                assert torch.equal(kp[l, pg, :, sl].cpu().view(torch.int16), sb.k_new[l, r0 + jp].view(torch.int16))
                assert torch.equal(vp[l, pg, :, sl].cpu().view(torch.int16), sb.v_new[l, r0 + jp].view(torch.int16))
                touched[pg, sl] = True
        m = (~touched).view(kp.shape[1], 1, page, 1).expand_as(kp[l]).cpu()
        assert torch.equal(kp[l].cpu().view(torch.int16)[m], before[0][l].cpu().view(torch.int16)[m])
        assert torch.equal(vp[l].cpu().view(torch.int16)[m], before[1][l].cpu().view(torch.int16)[m])


@pytest.mark.parametrize("path", PATHS)
def test_config1_many_seeds(prepos, oracle, path):
    """BASELINE config 1 attention: 1 session, n_s=256, L=8, 4/2 heads, d=64 -- 200 seeds ("many
    seeds (>= 200)"), every output element, Append(E) on every seed."""
    worst = 0.0
    for k in range(200):
        sb = synth.make_sessions(synth.C1, [256], [8], seed=synth.SEED_BASE + 1000 * k)
        out, kp, vp, before, status, ctx = _gpu_run(prepos, sb, path)
        ctx.close()
        outs, st, _, _ = oracle_attn_batch(oracle, sb)
        assert status == [0] and st[0] == 0
        worst = max(worst, check_attn(out, outs, sb))
        _check_append(sb, kp, vp, before, status, [0])
    assert worst <= ATTN_ATOL


SHAPES = {
    "d128_g4": synth.Shape("a", layers=2, Hq=8, Hkv=2, d=128, H=128, V=64, page=16),
    "d128_g8": synth.Shape("b", layers=1, Hq=16, Hkv=2, d=128, H=128, V=64, page=16),
    "d64_g2": synth.Shape("c", layers=2, Hq=4, Hkv=2, d=64, H=128, V=64, page=16),
    "d128_g1": synth.Shape("d", layers=1, Hq=2, Hkv=2, d=128, H=128, V=64, page=16),
    "d128_g16": synth.Shape("e", layers=1, Hq=16, Hkv=1, d=128, H=128, V=64, page=16),   # G > 8: two Q boxes per token
    "d128_g3": synth.Shape("f", layers=2, Hq=6, Hkv=2, d=128, H=128, V=64, page=16),      # G not a power of two
    "d128_p32": synth.Shape("g", layers=1, Hq=8, Hkv=2, d=128, H=128, V=64, page=32),     # another page size
    "d96_g2": synth.Shape("h", layers=1, Hq=4, Hkv=2, d=96, H=128, V=64, page=16),        # head_dim the tcgen05 path skips
    # MHA / G = 2 with more than 128 entry tokens: a unit's row chunk spans two entry tiles, so rows of the first
    # see NO column of the second.  16 layers: ~15 tiles per CTA, units cut at arbitrary tiles and merged by the last
    # arriver; 1 layer: one tile per CTA, every unit spread over ~35 CTAs and merged by attn_merge_kernel
    "d128_g1_l16": synth.Shape("i", layers=16, Hq=2, Hkv=2, d=128, H=128, V=64, page=16),
    "d128_g2_l16": synth.Shape("j", layers=16, Hq=4, Hkv=2, d=128, H=128, V=64, page=16),
    "d128_g2": synth.Shape("k", layers=1, Hq=4, Hkv=2, d=128, H=128, V=64, page=16),
    "d64_g1_l8": synth.Shape("l", layers=8, Hq=2, Hkv=2, d=64, H=128, V=64, page=16),
}


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("shape_key,n_s,l_entry", [
    ("d128_g4", [0], [24]),                       # n_s = 0: ordinary causal attention
    ("d128_g4", [1], [1]),                        # smallest non-trivial
    ("d128_g4", [127, 128, 129], [5, 16, 33]),    # around one 128-token tile; ragged pages
    ("d128_g4", [700, 15, 300], [24, 96, 64]),    # several tiles + ragged tail; rows 96 / 384 / 256
    ("d128_g8", [517], [32]),                     # G=8: 256 rows (config 5 row geometry)
    ("d128_g8", [40], [70]),                      # 560 rows: three row chunks
    ("d64_g2", [333, 64], [8, 40]),
    ("d128_g1", [260], [3]),
    ("d128_g4", [2500], [24]),                    # long enough to be split over many CTAs
    ("d128_g4", [300, 100], [0, 7]),              # an empty entry next to a real one
    ("d128_g16", [200, 77], [9, 20]),             # 144 / 320 rows with 16 heads per kv head
    ("d128_g3", [150], [11]),                     # CUDA-core kernel only (the tcgen05 path wants G = 2^k)
    ("d128_p32", [333], [24]),
    ("d96_g2", [140], [6]),
    ("d128_g1_l16", [4096], [129]),
    ("d128_g1_l16", [4000], [200]),
    ("d128_g1_l16", [2500, 700], [300, 257]),
    ("d128_g2_l16", [4096], [129]),
    ("d128_g2_l16", [3000], [200]),
    ("d128_g2_l16", [2200], [300]),
    ("d128_g1", [4096], [200]),
    ("d128_g1", [1500], [300]),
    ("d128_g2", [4096], [129]),
    ("d128_g2", [777], [300]),
    ("d64_g1_l8", [3000], [260]),
])
def test_shapes_vs_oracle(prepos, oracle, path, shape_key, n_s, l_entry):
    shape = SHAPES[shape_key]
    sb = synth.make_sessions(shape, n_s, l_entry, seed=1000 + 7 * sum(n_s) + sum(l_entry) + len(shape_key))
    out, kp, vp, before, status, _ = _gpu_run(prepos, sb, path)
    outs, st, _, _ = oracle_attn_batch(oracle, sb)
    assert status == [0] * len(n_s)
    check_attn(out, outs, sb)
    _check_append(sb, kp, vp, before, status, range(shape.layers))


@pytest.mark.parametrize("path", PATHS)
def test_budget_skip_no_side_effects(prepos, oracle, path):
    """Alg. 1 l.2-3: a session whose entry exceeds its headroom is skipped: status, no pool write, out untouched."""
    shape = SHAPES["d128_g4"]
    sb = synth.make_sessions(shape, [100, 50, 200], [12, 20, 8], seed=77, tight_capacity=[None, 69, 208])
    out, kp, vp, before, status, _ = _gpu_run(prepos, sb, path)
    assert status == [0, prepos.SKIPPED_BUDGET, 0]          # 50+20 > 69 skipped; 200+8 == 208 admitted
    outs, st, _, _ = oracle_attn_batch(oracle, sb)
    assert st == {0: 0, 1: 1, 2: 0}
    check_attn(out, outs, sb)
    r0 = sb.row_offset[1]
    assert torch.isnan(out[:, r0:r0 + 20].float()).all()    # rows of the skipped session untouched
    _check_append(sb, kp, vp, before, status, range(shape.layers))


@pytest.mark.parametrize("path", PATHS)
def test_nonfinite_rows_of_a_skipped_neighbour_do_not_leak(prepos, oracle, path):
    """The entry K/V of a budget-skipped session may never have been initialised by the caller.  Its rows sit right
    behind the previous session's in the packed sum_L axis, inside the last 8-token box that session loads: they must
    not reach its output (0 x NaN in the PV product)."""
    shape = SHAPES["d128_g4"]
    sb = synth.make_sessions(shape, [300, 40, 90], [13, 20, 5], seed=123, tight_capacity=[None, 59, None])
    r1 = sb.row_offset[1]
    for t in (sb.k_new, sb.v_new, sb.q):
        t[:, r1:r1 + 20] = float("nan")
    out, kp, vp, before, status, _ = _gpu_run(prepos, sb, path)
    assert status == [0, prepos.SKIPPED_BUDGET, 0]
    outs, st, _, _ = oracle_attn_batch(oracle, sb, sessions=[0, 2])
    check_attn(out, outs, sb)
    assert torch.isnan(out[:, r1:r1 + 20].float()).all()
    _check_append(sb, kp, vp, before, status, range(shape.layers))


@pytest.mark.parametrize("path", PATHS)
def test_layer_range_and_page_shuffle_bit_identical(prepos, oracle, path):
    """(a) layer_begin/layer_end touch only those layers; (b) permuting physical pages leaves the result
    bit-identical (SURVEY pin 9 on the GPU, fixed split plan)."""
    shape = SHAPES["d128_g4"]
    sb = synth.make_sessions(shape, [900, 130], [24, 9], seed=5)
    out_a, kp, vp, before, status, _ = _gpu_run(prepos, sb, path, layers=(1, 2), poison=False)
    assert torch.isnan(out_a[0].float()).all() and not torch.isnan(out_a[1].float()).any()
    assert torch.equal(kp[0].view(torch.int16), before[0][0].view(torch.int16))
    outs, _, _, _ = oracle_attn_batch(oracle, sb, layers=[1])
    check_attn(out_a, outs, sb)
    n_pages = sb.k_pool.shape[1]
    perm = torch.randperm(n_pages, generator=torch.Generator().manual_seed(1))
    inv = torch.empty_like(perm)
    inv[perm] = torch.arange(n_pages)
    sb2 = synth.make_sessions(shape, [900, 130], [24, 9], seed=5)
    sb2.k_pool.copy_(sb.k_pool[:, inv])
    sb2.v_pool.copy_(sb.v_pool[:, inv])
    sb2.page_table.copy_(perm[sb.page_table.long()].to(torch.int32))
    out_b, *_ = _gpu_run(prepos, sb2, path, layers=(1, 2), poison=False)
    assert torch.equal(out_a[1].view(torch.int16), out_b[1].view(torch.int16))


@pytest.mark.parametrize("path", PATHS)
def test_two_step_consistency(prepos, oracle, path):
    """Pre-position L1 then L2 tokens (second call sees n_s + L1 through the appended pages) ~ one call."""
    shape = SHAPES["d128_g4"]
    L1, L2, n = 10, 14, 200
    sb = synth.make_sessions(shape, [n], [L1 + L2], seed=9)
    out_one, kp1, vp1, _, _, _ = _gpu_run(prepos, sb, path, poison=False)
    dev = "cuda"
    kp, vp = sb.k_pool.to(dev).clone(), sb.v_pool.to(dev).clone()
    ctx = _ctx(prepos, shape, 1, path)
    q, kn, vn = sb.q.to(dev), sb.k_new.to(dev), sb.v_new.to(dev)
    o1 = torch.zeros((shape.layers, L1, shape.Hq, shape.d), dtype=torch.bfloat16, device=dev)
    o2 = torch.zeros((shape.layers, L2, shape.Hq, shape.d), dtype=torch.bfloat16, device=dev)
    ctx.entry_attn(q[:, :L1].contiguous(), kn[:, :L1].contiguous(), vn[:, :L1].contiguous(), kp, vp,
                   sb.page_table.to(dev), [n], [L1], sb.capacity, o1)
    ctx.entry_attn(q[:, L1:].contiguous(), kn[:, L1:].contiguous(), vn[:, L1:].contiguous(), kp, vp,
                   sb.page_table.to(dev), [n + L1], [L2], sb.capacity, o2)
    ctx.sync()
    two = torch.cat([o1, o2], dim=1).float()
    assert (two - out_one.float()).abs().max() <= 2e-2       # both within 1e-2 of the oracle
    assert torch.equal(kp.view(torch.int16), kp1.view(torch.int16)) and torch.equal(vp.view(torch.int16), vp1.view(torch.int16))
    outs, _, _, _ = oracle_attn_batch(oracle, sb)
    check_attn(torch.cat([o1, o2], dim=1), outs, sb)


@pytest.mark.parametrize("path", PATHS)
def test_config4_like_batch_sampled(prepos, oracle, path):
    """A scaled-down agentic batch (BASELINE config 4 structure): 6 sessions, lognormal n_s, L ~ U{32..96},
    one shuffled pool, 2 layers of 8B head geometry (32/8, d=128); oracle on sampled (layer, session, head, row)."""
    shape = synth.Shape("c4s", layers=2, Hq=32, Hkv=8, d=128, H=128, V=64, page=16)
    n_s = synth.lognormal_ns(6, 42, lo=256, hi=3000, median=900.0)
    l_e = synth.uniform_l(6, 42)
    sb = synth.make_sessions(shape, n_s, l_e, seed=43)
    out, kp, vp, before, status, _ = _gpu_run(prepos, sb, path)
    assert status == [0] * 6
    rng = np.random.default_rng(0)
    worst = 0.0
    for s in range(6):
        for l in range(2):
            picks = [(int(rng.integers(0, 32)), int(rng.integers(0, l_e[s]))) for _ in range(3)] + [(31, l_e[s] - 1), (0, 0)]
            ref = oracle_attn_rows(oracle, sb, l, s, picks)
            for (h, i), o in ref.items():
                got = out[l, sb.row_offset[s] + i, h].cpu().to(torch.float64).numpy()
                worst = max(worst, float(np.abs(got - o).max()))
    assert worst <= ATTN_ATOL, worst
    _check_append(sb, kp, vp, before, status, range(2))


def _full_size_spec(name):
    seed = synth.SEED_BASE + int(name[1])
    if name == "c2":
        return synth.C2, [4096], [24], seed
    if name == "c3":
        return synth.C3, [32768], [16], seed
    if name == "c4":
        return synth.C4, synth.lognormal_ns(64, seed), synth.uniform_l(64, seed), seed
    return synth.C5, [16384], [32], seed


def _expected_pools_after_append(sb):
    """The pools as Append(E) (Alg. 1 l.5) must leave them: a copy of the pristine pools with K_new / V_new scattered
    to cache positions n_s .. n_s+L-1 of every session through the page table (torch indexing on the synthetic
    inputs: data movement only).  Comparing the whole tensors checks every appended slot of every session and layer
    AND that no other pool element moved."""
    page = sb.shape.page
    ke, ve = sb.k_pool.clone(), sb.v_pool.clone()
    pt = sb.page_table.long()
    for s in range(sb.n_sessions):
        j = sb.n_s[s] + torch.arange(sb.l_entry[s], device=ke.device)
        pg, sl = pt[s, j // page], j % page
        r0 = sb.row_offset[s]
        ke[:, pg, :, sl] = sb.k_new[:, r0:r0 + sb.l_entry[s]].permute(1, 0, 2, 3)   # advanced dims lead: [L, layers, Hkv, d]
        ve[:, pg, :, sl] = sb.v_new[:, r0:r0 + sb.l_entry[s]].permute(1, 0, 2, 3)
    return ke, ve


def _gather_session(sb, s):
    """Pristine host copy of session s's pages, re-indexed 0..n-1 (the oracle's page-shuffle invariance is pinned):
    (k [layers, n, Hkv, page, d] uint16, v, table int32 [n])."""
    n = -(-(sb.n_s[s] + sb.l_entry[s]) // sb.shape.page)
    idx = sb.page_table[s, :n].long()
    k = sb.k_pool[:, idx].cpu().contiguous().view(torch.int16).numpy().view(np.uint16)
    v = sb.v_pool[:, idx].cpu().contiguous().view(torch.int16).numpy().view(np.uint16)
    return k, v, np.arange(n, dtype=np.int32)


def _check_session_every_row(oracle, sb, s, out, pristine):
    """Every output element of session s, all layers, against O1 on the pristine pages."""
    k, v, table = pristine
    r0, L = sb.row_offset[s], sb.l_entry[s]
    worst = 0.0
    for l in range(k.shape[0]):
        ref = oracle.entry_attn(bits(sb.q[l, r0:r0 + L]), bits(sb.k_new[l, r0:r0 + L]), bits(sb.v_new[l, r0:r0 + L]),
                                k[l].copy(), v[l].copy(), table, sb.n_s[s], sb.capacity[s])
        assert ref["status"] == 0
        got = out[l, r0:r0 + L].cpu().to(torch.float64).numpy()
        worst = max(worst, float(np.abs(got - ref["out"]).max()))
    return worst


def _draw_samples(rng, shape, L, n_slices=8, per_slice=8):
    """64 seeded (layer, head, row) samples of one session, grouped by (layer, kv head) slice."""
    G = shape.G
    out = []
    for _ in range(n_slices):
        l, g = int(rng.integers(0, shape.layers)), int(rng.integers(0, shape.Hkv))
        picks = [(int(rng.integers(0, G)), int(rng.integers(0, L))) for _ in range(per_slice - 2)] + [(G - 1, L - 1), (0, 0)]
        out.append((l, g, picks))
    return out


def _gather_slices(sb, s, samples):
    """Pristine host copies of the (layer, kv head) slices the samples of session s need."""
    n = -(-(sb.n_s[s] + sb.l_entry[s]) // sb.shape.page)
    idx = sb.page_table[s, :n].long()
    res = []
    for (l, g, _) in samples:
        k = sb.k_pool[l, idx, g:g + 1].cpu().contiguous().view(torch.int16).numpy().view(np.uint16)
        v = sb.v_pool[l, idx, g:g + 1].cpu().contiguous().view(torch.int16).numpy().view(np.uint16)
        res.append((k, v))
    return res


def _check_samples(oracle, sb, s, out, samples, slices):
    """Sampled (layer, head, row) outputs of session s against the ranged O1 (one row of one head per call)."""
    G = sb.shape.G
    r0, L = sb.row_offset[s], sb.l_entry[s]
    n = slices[0][0].shape[0]
    table = np.arange(n, dtype=np.int32)
    worst = 0.0
    for (l, g, picks), (k, v) in zip(samples, slices):
        q = bits(sb.q[l, r0:r0 + L, g * G:(g + 1) * G])
        kn, vn = bits(sb.k_new[l, r0:r0 + L, g:g + 1]), bits(sb.v_new[l, r0:r0 + L, g:g + 1])
        for (hh, i) in picks:
            ref = oracle.entry_attn(q, kn, vn, k.copy(), v.copy(), table, sb.n_s[s], sb.capacity[s],
                                    heads=(hh, hh + 1), rows=(i, i + 1))["out"][i, hh]
            got = out[l, r0 + i, g * G + hh].cpu().to(torch.float64).numpy()
            worst = max(worst, float(np.abs(got - ref).max()))
    return worst


@pytest.mark.parametrize("name", ["c2", "c3", "c4", "c5"])
def test_full_size_configs(prepos, oracle, name):
    """BASELINE configs 2-5 at FULL size in the launch configuration bench.py times (default path, every layer in one
    launch, inputs generated on the device with bench.py's seeds), with the coverage SURVEY.md 8(d) contracts:
      c2, c3  every output element of every layer (24 576 / 16 384 rows)
      c5      the sessions bench.py keeps resident (4 independent single-session batches): two of them every row,
              64 seeded (layer, head, row) samples on each of the others
      c4      eight whole sessions of the 64 -- including argmax(n_s) (a 16k-token session) and argmax(L) (more than
              256 query rows: the split row chunk) -- every row; 64 seeded samples on each of the other 56
    and, on every config, the WHOLE pools after the call against the pristine pools with K_new / V_new scattered to
    the appended slots: Append(E) of every session on every layer, and every other pool element untouched."""
    shape, n_s, l_e, seed = _full_size_spec(name)
    batches = [seed] if name != "c5" else [seed + 100003 * (r + 1) for r in range(4)]    # bench.py's resident sets
    worst = 0.0
    for bi, bseed in enumerate(batches):
        sb = synth.make_sessions(shape, n_s, l_e, seed=bseed, device="cuda")
        n = len(n_s)
        rng = np.random.default_rng(bseed)
        if n == 1:
            full = [0] if (name != "c5" or bi < 2) else []
        else:
            full = sorted(set(int(x) for x in rng.choice(n, 6, replace=False)) | {int(np.argmax(n_s)), int(np.argmax(l_e))})
            while len(full) < 8:
                full = sorted(set(full) | {int(rng.integers(0, n))})
        sampled = [s for s in range(n) if s not in full]
        pristine = {s: _gather_session(sb, s) for s in full}
        samples = {s: _draw_samples(rng, shape, l_e[s]) for s in sampled}
        slices = {s: _gather_slices(sb, s, samples[s]) for s in sampled}
        ke, ve = _expected_pools_after_append(sb)
        ctx = prepos.Context(shape.layers, shape.Hq, shape.Hkv, shape.d, shape.H, shape.V, shape.page, max_sessions=n)
        out = torch.full(sb.q.shape, float("nan"), dtype=torch.bfloat16, device="cuda")
        status = ctx.entry_attn(sb.q, sb.k_new, sb.v_new, sb.k_pool, sb.v_pool, sb.page_table, sb.n_s, sb.l_entry,
                                sb.capacity, out)
        ctx.sync()
        assert status == [0] * n
        assert torch.isfinite(out.float()).all()
        assert torch.equal(sb.k_pool.view(torch.int16), ke.view(torch.int16)), "K pool: append / untouched mismatch"
        assert torch.equal(sb.v_pool.view(torch.int16), ve.view(torch.int16)), "V pool: append / untouched mismatch"
        del ke, ve
        for s in full:
            worst = max(worst, _check_session_every_row(oracle, sb, s, out, pristine[s]))
            assert worst <= ATTN_ATOL, (name, bi, s, worst)
        for s in sampled:
            worst = max(worst, _check_samples(oracle, sb, s, out, samples[s], slices[s]))
            assert worst <= ATTN_ATOL, (name, bi, s, worst)
        ctx.close()
        del sb, out, pristine, slices
        torch.cuda.empty_cache()
    assert worst <= ATTN_ATOL, worst


def test_fall_through_delta_resume_full_size(prepos, oracle):
    """The fall-through path after a gate miss (Eq. 5; Alg. 2 l.8-9) on BASELINE
    config 2 at full size: pre-position L = 24 entry tokens, then resume with a delta of 8 tokens on top of the
    pre-positioned cache (n_s' = n_s + 24), then one decode step (L = 1, n_s'' = n_s + 32).  Each call's sampled
    rows against the oracle (which reads the cache the previous calls appended to), and two-step consistency at
    scale: rows of the first two calls == one call with all 32 tokens over the original cache."""
    from dataclasses import replace
    shape, seed = synth.C2, synth.SEED_BASE + 1
    n_s0, L1, L2 = 4096, 24, 8
    sb = synth.make_sessions(shape, [n_s0], [L1 + L2], seed=seed, device="cuda", extra_pages=1)
    k0, v0 = sb.k_pool.clone(), sb.v_pool.clone()
    ctx = prepos.Context(shape.layers, shape.Hq, shape.Hkv, shape.d, shape.H, shape.V, shape.page, max_sessions=1)

    def run(view, pools):
        out = torch.full(view.q.shape, float("nan"), dtype=torch.bfloat16, device="cuda")
        st = ctx.entry_attn(view.q, view.k_new, view.v_new, pools[0], pools[1], view.page_table, view.n_s,
                            view.l_entry, view.capacity, out)
        ctx.sync()
        assert st == [0]
        return out

    def sample(view, out, rng, layers):
        worst = 0.0
        L = view.l_entry[0]
        for l in layers:
            picks = [(int(rng.integers(0, shape.Hq)), int(rng.integers(0, L))) for _ in range(2)] + [(shape.Hq - 1, L - 1)]
            for (h, i), o in oracle_attn_rows(oracle, view, l, 0, picks).items():
                worst = max(worst, float(np.abs(out[l, i, h].cpu().to(torch.float64).numpy() - o).max()))
        return worst

    rng = np.random.default_rng(seed)
    layers = [0, int(rng.integers(1, shape.layers - 1)), shape.layers - 1]
    # one call with all 32 tokens over the original cache (on copies of the pools)
    joint = run(sb, (k0, v0))
    # call 1: the pre-position
    v1 = replace(sb, l_entry=[L1], q=sb.q[:, :L1], k_new=sb.k_new[:, :L1], v_new=sb.v_new[:, :L1])
    o1 = run(v1, (sb.k_pool, sb.v_pool))
    assert sample(v1, o1, rng, layers) <= ATTN_ATOL
    # call 2: the delta on top of the pre-positioned entry
    v2 = replace(sb, n_s=[n_s0 + L1], l_entry=[L2], q=sb.q[:, L1:], k_new=sb.k_new[:, L1:], v_new=sb.v_new[:, L1:])
    o2 = run(v2, (sb.k_pool, sb.v_pool))
    assert sample(v2, o2, rng, layers) <= ATTN_ATOL
    # two-step consistency: same rows as the joint call, and the same cache contents afterwards
    both = torch.cat([o1, o2], dim=1).float()
    assert float((both - joint.float()).abs().max()) <= 2 * ATTN_ATOL
    assert torch.equal(sb.k_pool.view(torch.int16), k0.view(torch.int16))
    assert torch.equal(sb.v_pool.view(torch.int16), v0.view(torch.int16))
    # call 3: one decode step over everything appended so far
    g = synth.gen(seed + 999, "cuda")
    v3 = replace(sb, n_s=[n_s0 + L1 + L2], l_entry=[1], q=synth.randn_bf16((shape.layers, 1, shape.Hq, shape.d), g),
                 k_new=synth.randn_bf16((shape.layers, 1, shape.Hkv, shape.d), g),
                 v_new=synth.randn_bf16((shape.layers, 1, shape.Hkv, shape.d), g))
    o3 = run(v3, (sb.k_pool, sb.v_pool))
    assert sample(v3, o3, rng, layers) <= ATTN_ATOL


@pytest.mark.parametrize("kv_prefetch", [False, True])
def test_one_launch_per_layer_merge_kernel(prepos, oracle, kv_prefetch):
    """Schedule (S): one prepos_entry_attn call per layer.  With 2 kv heads x 25 tiles over 148 persistent CTAs every
    unit is spread over ~25 CTAs, whose partials are combined by the dependent attn_merge_kernel; 256 query rows per
    kv head (config 5's row geometry) and a ragged last tile.  Oracle on every row,
    Append(E) on every layer, and a second round of launches on the same context (the self-resetting counters)."""
    shape = synth.Shape("s_sched", layers=3, Hq=16, Hkv=2, d=128, H=128, V=64, page=16)
    sb = synth.make_sessions(shape, [3100], [32], seed=77)
    dev = "cuda"
    ctx = prepos.Context(shape.layers, shape.Hq, shape.Hkv, shape.d, shape.H, shape.V, shape.page, max_sessions=1)
    ctx.set_attn_path(2)
    # with kv_prefetch a layer's launch streams its cached tiles while the previous layer's merge is still running
    # (prepos_ctx_set_kv_prefetch: legal here, layer l's launch writes layer l's pages only)
    ctx.set_kv_prefetch(kv_prefetch)
    outs, _, _, _ = oracle_attn_batch(oracle, sb)
    for rnd in range(2):
        kp, vp = sb.k_pool.to(dev).clone(), sb.v_pool.to(dev).clone()
        before = (kp.clone(), vp.clone())
        out = torch.full(sb.q.shape, float("nan"), dtype=torch.bfloat16, device=dev)
        q, kn, vn, pt = sb.q.to(dev), sb.k_new.to(dev), sb.v_new.to(dev), sb.page_table.to(dev)
        for l in range(shape.layers):
            st = ctx.entry_attn(q, kn, vn, kp, vp, pt, sb.n_s, sb.l_entry, sb.capacity, out, layer_begin=l, layer_end=l + 1)
            assert st == [0]
        ctx.sync()
        check_attn(out, outs, sb)
        _check_append(sb, kp, vp, before, [0], range(shape.layers))


@pytest.mark.parametrize("path", PATHS)
def test_random_geometries_vs_oracle(prepos, oracle, path):
    """24 seeded random geometries (head_dim, group size, kv heads, layers, page size, 1-4 sessions with n_s in
    [0, 700] and L in [0, 70], some sessions over budget): every output row and the Append(E) post-condition
    against the oracle, on both GPU paths."""
    rng = np.random.default_rng(20260629)
    ran = 0
    for case in range(24):
        d = int(rng.choice([64, 128]))
        G = int(rng.choice([1, 2, 4, 8]))
        Hkv = int(rng.choice([1, 2, 3]))
        layers = int(rng.integers(1, 4))
        page = int(rng.choice([8, 16, 32, 64]))
        n_sess = int(rng.integers(1, 5))
        n_s = [int(rng.integers(0, 701)) for _ in range(n_sess)]
        l_e = [int(rng.integers(0, 71)) for _ in range(n_sess)]
        if sum(l_e) == 0:
            l_e[0] = 5
        shape = synth.Shape(f"rnd{case}", layers=layers, Hq=G * Hkv, Hkv=Hkv, d=d, H=128, V=64, page=page)
        tight = [None] * n_sess
        if n_sess > 1 and case % 3 == 0:
            tight[1] = n_s[1] + max(0, l_e[1] - 1)      # one token short of the budget: skipped (Alg. 1 l.2-3)
        sb = synth.make_sessions(shape, n_s, l_e, seed=9000 + case, tight_capacity=tight)
        try:
            out, kp, vp, before, status, _ = _gpu_run(prepos, sb, path)
        except pytest.skip.Exception:
            continue
        ran += 1
        outs, st, _, _ = oracle_attn_batch(oracle, sb)
        assert status == [st[s] for s in range(n_sess)], (case, status, st)
        for s in range(n_sess):
            if status[s] != 0:          # skipped: its output rows are untouched
                outs = {k: v for k, v in outs.items() if k[1] != s}
        check_attn(out, outs, sb)
        _check_append(sb, kp, vp, before, status, range(layers))
    assert ran >= 12


# ---------------------------------------------------------------- NEXT-2: yield and resume
def _many_small(n, seed, lo=40, hi=420, l_lo=3, l_hi=48):
    rng = np.random.default_rng(seed)
    return [int(x) for x in rng.integers(lo, hi, n)], [int(x) for x in rng.integers(l_lo, l_hi, n)]


SHAPES["d128_g4_l8"] = synth.Shape("m", layers=8, Hq=8, Hkv=2, d=128, H=128, V=64, page=16)


@pytest.mark.parametrize("shape_key,n_s,l_entry,slice_n", [
    ("d128_g4_l8",) + _many_small(30, 1) + (1,),          # ~5 short units per CTA (whole and cut): a stop after each
    ("d128_g4_l8",) + _many_small(30, 2) + (2,),          # two segments per launch
    ("d128_g2_l16", [3000, 1000, 500], [200, 130, 40], 1),   # 160 long units on 148 CTAs: stream-K cuts; a CTA stops
                                                             # between the tail of one unit and the head of the next
                                                             # and the partials wait in the workspace
    ("d128_g1_l16", [2500, 700, 900], [300, 257, 129], 1),   # two row chunks per session, G = 1
    ("d64_g1_l8",) + _many_small(12, 3, l_hi=200) + (1,),
])
def test_sliced_pass_yield_and_resume_is_bit_identical(prepos, oracle, shape_key, n_s, l_entry, slice_n):
    """A pass that stops at its yield points and is resumed until nothing is pending must give the result of an
    uninterrupted call bit for bit (same plan, same split, same merge order) -- and match the oracle, Append(E)
    included.  `set_attn_slice(n)` makes every launch stop after n segments per CTA, so every segment boundary of the
    pass is exercised as a yield point, deterministically."""
    shape = SHAPES[shape_key]
    sb = synth.make_sessions(shape, n_s, l_entry, seed=4242 + sum(n_s))
    out_ref, kp_ref, vp_ref, _, status, ctx0 = _gpu_run(prepos, sb, 2, poison=False)
    ctx0.close()
    dev = "cuda"
    kp, vp = sb.k_pool.to(dev).clone(), sb.v_pool.to(dev).clone()
    before = (kp.clone(), vp.clone())
    out = torch.full(sb.q.shape, float("nan"), dtype=torch.bfloat16, device=dev)
    ctx = _ctx(prepos, shape, sb.n_sessions, 2)
    ctx.set_attn_slice(slice_n)
    st = ctx.entry_attn(sb.q.to(dev), sb.k_new.to(dev), sb.v_new.to(dev), kp, vp, sb.page_table.to(dev),
                        sb.n_s, sb.l_entry, sb.capacity, out)
    launches = 1
    while ctx.entry_attn_pending():
        ctx.entry_attn_resume()
        launches += 1
        assert launches < 500
    assert launches >= 2, "the pass never stopped: the slice was not honoured"
    assert st == status
    assert torch.equal(out.view(torch.int16), out_ref.view(torch.int16))
    assert torch.equal(kp.view(torch.int16), kp_ref.view(torch.int16)) and torch.equal(vp.view(torch.int16), vp_ref.view(torch.int16))
    outs, _, _, _ = oracle_attn_batch(oracle, sb)
    check_attn(out, outs, sb)
    _check_append(sb, kp, vp, before, status, range(shape.layers))
    # an unsliced call on the same ctx afterwards is unaffected (counters and flag left clean)
    ctx.set_attn_slice(0)
    out2 = torch.full(sb.q.shape, float("nan"), dtype=torch.bfloat16, device=dev)
    ctx.entry_attn(sb.q.to(dev), sb.k_new.to(dev), sb.v_new.to(dev), before[0], before[1], sb.page_table.to(dev),
                   sb.n_s, sb.l_entry, sb.capacity, out2)
    assert not ctx.entry_attn_pending()
    assert torch.equal(out2.view(torch.int16), out_ref.view(torch.int16))


def test_yield_request_from_another_stream_then_resume(prepos, oracle):
    """The flag form: a long pass (config 2 geometry, 32 layers) is started on a low-priority stream, a yield is
    requested from a high-priority stream while it runs, a kernel that needs whole SMs (another ctx's decode step) is
    run there, then the pass is resumed.  The resumed result equals the uninterrupted one bit for bit, the decode
    step's result is right, and in at least one of the trials the pass really was caught running (pending)."""
    shape = synth.C2
    seed = synth.SEED_BASE + 1
    sb = synth.make_sessions(shape, [4096], [24], seed=seed, device="cuda", extra_pages=1)
    k0, v0 = sb.k_pool.clone(), sb.v_pool.clone()
    ctx = prepos.Context(shape.layers, shape.Hq, shape.Hkv, shape.d, shape.H, shape.V, shape.page, max_sessions=1)
    ctx_d = prepos.Context(shape.layers, shape.Hq, shape.Hkv, shape.d, shape.H, shape.V, shape.page, max_sessions=1)
    ref = torch.empty_like(sb.q)
    ctx.entry_attn(sb.q, sb.k_new, sb.v_new, sb.k_pool, sb.v_pool, sb.page_table, sb.n_s, sb.l_entry, sb.capacity, ref)
    ctx.sync()
    # the decode step of another session living in the same pool geometry (its own pools)
    sd = synth.make_sessions(shape, [2048], [1], seed=seed + 5, device="cuda")
    dref = torch.empty_like(sd.q)
    ctx_d.entry_attn(sd.q, sd.k_new, sd.v_new, sd.k_pool.clone(), sd.v_pool.clone(), sd.page_table, sd.n_s, sd.l_entry,
                     sd.capacity, dref)
    ctx_d.sync()
    s_lo, s_hi = torch.cuda.Stream(priority=0), torch.cuda.Stream(priority=-1)
    caught = 0
    for trial in range(12):
        sb.k_pool.copy_(k0)
        sb.v_pool.copy_(v0)
        out = torch.full(sb.q.shape, float("nan"), dtype=torch.bfloat16, device="cuda")
        dout = torch.full(sd.q.shape, float("nan"), dtype=torch.bfloat16, device="cuda")
        dk, dv = sd.k_pool.clone(), sd.v_pool.clone()
        torch.cuda.synchronize()
        with torch.cuda.stream(s_lo):
            ctx.entry_attn(sb.q, sb.k_new, sb.v_new, sb.k_pool, sb.v_pool, sb.page_table, sb.n_s, sb.l_entry,
                           sb.capacity, out)
        with torch.cuda.stream(s_hi):
            ctx.request_yield()
            ctx_d.entry_attn(sd.q, sd.k_new, sd.v_new, dk, dv, sd.page_table, sd.n_s, sd.l_entry, sd.capacity, dout)
        s_hi.synchronize()
        with torch.cuda.stream(s_lo):
            pending = ctx.entry_attn_pending()
            caught += int(pending)
            ctx.entry_attn_resume()
            assert not ctx.entry_attn_pending()
        torch.cuda.synchronize()
        assert torch.equal(out.view(torch.int16), ref.view(torch.int16)), trial
        assert torch.equal(dout.view(torch.int16), dref.view(torch.int16)), trial
    assert caught >= 1, "no trial caught the pass running: the yield path was not exercised"


def test_two_contexts_one_launch_per_layer_on_two_streams(prepos, oracle):
    """Two contexts (two replicas of the library on one GPU) issue their attention one launch per layer at the same
    time on two streams: every unit is spread over many CTAs and merged across them, and neither pass may depend on
    having the whole GPU to itself (round 1's in-kernel merge spun on co-residency and could deadlock here).  Both
    results against the oracle, every row; three rounds on the same contexts."""
    shape = synth.Shape("two_ctx", layers=6, Hq=16, Hkv=2, d=128, H=128, V=64, page=16)
    sbs = [synth.make_sessions(shape, [3100], [32], seed=91), synth.make_sessions(shape, [2300, 900], [24, 40], seed=92)]
    dev = "cuda"
    ctxs = [prepos.Context(shape.layers, shape.Hq, shape.Hkv, shape.d, shape.H, shape.V, shape.page, max_sessions=2)
            for _ in sbs]
    for c in ctxs:
        c.set_attn_path(2)
    ctxs[1].set_kv_prefetch(True)      # one of the two also streams its cached tiles ahead of the dependency wait
    refs = [oracle_attn_batch(oracle, sb)[0] for sb in sbs]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    dv = [dict(q=sb.q.to(dev), kn=sb.k_new.to(dev), vn=sb.v_new.to(dev), pt=sb.page_table.to(dev)) for sb in sbs]
    for rnd in range(3):
        pools = [(sb.k_pool.to(dev).clone(), sb.v_pool.to(dev).clone()) for sb in sbs]
        outs = [torch.full(sb.q.shape, float("nan"), dtype=torch.bfloat16, device=dev) for sb in sbs]
        torch.cuda.synchronize()
        for l in range(shape.layers):
            for k in (0, 1):
                with torch.cuda.stream(streams[k]):
                    st = ctxs[k].entry_attn(dv[k]["q"], dv[k]["kn"], dv[k]["vn"], pools[k][0], pools[k][1], dv[k]["pt"],
                                            sbs[k].n_s, sbs[k].l_entry, sbs[k].capacity, outs[k],
                                            layer_begin=l, layer_end=l + 1)
                    assert st == [0] * sbs[k].n_sessions
        torch.cuda.synchronize()
        for k in (0, 1):
            check_attn(outs[k], refs[k], sbs[k])


def _short_session_batch(seed):
    """A config-4-like batch of SHORT sessions on the 8B shape: every session has at most 6 cached tiles + 1 entry
    tile, so no segment of any CTA is 8 tiles long (the yield flag used to be re-read only at the 8th tile of a
    segment)."""
    shape = synth.C2
    g = synth.gen(seed)
    n = 64
    n_s = torch.randint(128, 769, (n,), generator=g).tolist()
    l_e = torch.randint(32, 65, (n,), generator=g).tolist()
    return shape, synth.make_sessions(shape, n_s, l_e, seed=seed, device="cuda", extra_pages=1)


def test_yield_flag_reaches_ctas_whose_segments_are_all_short(prepos):
    """prepos_ctx_request_yield on a pass made of short segments only (64 sessions of 128..768 cached tokens, 32
    layers: about a hundred segments per CTA, none of 8 tiles).  The CTAs count tiles across segments when they
    re-read the flag, so the request is seen within 8 tiles of the CTA's stream: the pass must be caught pending in
    at least one trial, and the resumed result is the uninterrupted one bit for bit."""
    shape, sb = _short_session_batch(synth.SEED_BASE + 404)
    k0, v0 = sb.k_pool.clone(), sb.v_pool.clone()
    ctx = prepos.Context(shape.layers, shape.Hq, shape.Hkv, shape.d, shape.H, shape.V, shape.page, max_sessions=64)
    ctx.set_attn_path(2)
    ref = torch.empty_like(sb.q)
    ctx.entry_attn(sb.q, sb.k_new, sb.v_new, sb.k_pool, sb.v_pool, sb.page_table, sb.n_s, sb.l_entry, sb.capacity, ref)
    ctx.sync()
    kref, vref = sb.k_pool.clone(), sb.v_pool.clone()
    s_lo, s_hi = torch.cuda.Stream(priority=0), torch.cuda.Stream(priority=-1)
    caught = 0
    for trial in range(6):
        sb.k_pool.copy_(k0)
        sb.v_pool.copy_(v0)
        out = torch.full(sb.q.shape, float("nan"), dtype=torch.bfloat16, device="cuda")
        torch.cuda.synchronize()
        with torch.cuda.stream(s_lo):
            ctx.entry_attn(sb.q, sb.k_new, sb.v_new, sb.k_pool, sb.v_pool, sb.page_table, sb.n_s, sb.l_entry,
                           sb.capacity, out)
        with torch.cuda.stream(s_hi):
            ctx.request_yield()
        s_hi.synchronize()
        with torch.cuda.stream(s_lo):
            pending = ctx.entry_attn_pending()
            caught += int(pending)
            ctx.entry_attn_resume()
            assert not ctx.entry_attn_pending()
        torch.cuda.synchronize()
        assert torch.equal(out.view(torch.int16), ref.view(torch.int16)), trial
        assert torch.equal(sb.k_pool.view(torch.int16), kref.view(torch.int16))
        assert torch.equal(sb.v_pool.view(torch.int16), vref.view(torch.int16))
    assert caught >= 1, "the yield request never reached a pass of short segments"


def test_late_yield_request_cannot_stop_a_later_pass(prepos):
    """A yield request names the launch it is for.  Here the request for pass A sits behind 20 ms of other work on its
    stream and lands long after A has ended -- after pass B on the same ctx has been issued as well.  Neither B nor the
    pass C issued after the request has landed may be stopped by it: both run to completion (not pending) and give the
    reference result.  (With a bare 0/1 flag the late copy landed after B's call had cleared the flag, and C -- and
    every later call -- stopped at its first yield point while returning PREPOS_OK.)"""
    shape = synth.C2
    sb = synth.make_sessions(shape, [4096], [24], seed=synth.SEED_BASE + 405, device="cuda", extra_pages=1)
    k0, v0 = sb.k_pool.clone(), sb.v_pool.clone()
    ctx = prepos.Context(shape.layers, shape.Hq, shape.Hkv, shape.d, shape.H, shape.V, shape.page, max_sessions=1)
    ref = torch.empty_like(sb.q)
    ctx.entry_attn(sb.q, sb.k_new, sb.v_new, sb.k_pool, sb.v_pool, sb.page_table, sb.n_s, sb.l_entry, sb.capacity, ref)
    ctx.sync()
    s_lo, s_hi = torch.cuda.Stream(priority=0), torch.cuda.Stream(priority=-1)

    def one_pass():
        sb.k_pool.copy_(k0)
        sb.v_pool.copy_(v0)
        out = torch.full(sb.q.shape, float("nan"), dtype=torch.bfloat16, device="cuda")
        ctx.entry_attn(sb.q, sb.k_new, sb.v_new, sb.k_pool, sb.v_pool, sb.page_table, sb.n_s, sb.l_entry, sb.capacity, out)
        return out

    with torch.cuda.stream(s_lo):
        out_a = one_pass()                                   # pass A
    with torch.cuda.stream(s_hi):
        torch.cuda._sleep(40_000_000)                        # ~20 ms at 1.9 GHz: the request is stuck behind this
        ctx.request_yield()                                  # meant for A
    s_lo.synchronize()                                       # A has ended, the request has not landed yet
    with torch.cuda.stream(s_lo):
        out_b = one_pass()                                   # pass B, issued while the request is still in flight
        assert not ctx.entry_attn_pending()
    torch.cuda.synchronize()                                 # now the late request has landed
    with torch.cuda.stream(s_lo):
        out_c = one_pass()                                   # pass C
        assert not ctx.entry_attn_pending()
    torch.cuda.synchronize()
    for name, o in (("A", out_a), ("B", out_b), ("C", out_c)):
        assert torch.equal(o.view(torch.int16), ref.view(torch.int16)), name


@pytest.mark.parametrize("shape_key,n_s,l_entry", [
    ("d128_g2_l16", [3000, 1000, 500], [200, 130, 40]),      # stream-K cuts: units merged by their last arriver
    ("d128_g4_l8",) + _many_small(30, 1),
])
def test_abandoned_sliced_pass_does_not_poison_the_next_call(prepos, shape_key, n_s, l_entry):
    """`prepos_ctx_set_attn_slice(1)` stops a pass after one segment per CTA: units cut across CTAs have counted some
    of their arrivals.  Issuing a NEW prepos_entry_attn instead of a resume abandons that pass; the new pass must
    start from clean arrival counters (otherwise its last-arriver merge fires early, on incomplete partials, and
    writes wrong rows without any error).  The new call's output equals an untouched ctx's bit for bit."""
    shape = SHAPES[shape_key]
    sb = synth.make_sessions(shape, n_s, l_entry, seed=777 + sum(n_s))
    out_ref, kp_ref, vp_ref, _, status, ctx0 = _gpu_run(prepos, sb, 2, poison=False)
    ctx0.close()
    dev = "cuda"
    ctx = _ctx(prepos, shape, sb.n_sessions, 2)
    q, kn, vn, pt = sb.q.to(dev), sb.k_new.to(dev), sb.v_new.to(dev), sb.page_table.to(dev)
    for rnd in range(2):
        ctx.set_attn_slice(1)
        kp, vp = sb.k_pool.to(dev).clone(), sb.v_pool.to(dev).clone()
        junk = torch.full(sb.q.shape, float("nan"), dtype=torch.bfloat16, device=dev)
        ctx.entry_attn(q, kn, vn, kp, vp, pt, sb.n_s, sb.l_entry, sb.capacity, junk)
        assert ctx.entry_attn_pending()
        ctx.set_attn_slice(0)                       # ... and never resumed
        kp, vp = sb.k_pool.to(dev).clone(), sb.v_pool.to(dev).clone()
        out = torch.full(sb.q.shape, float("nan"), dtype=torch.bfloat16, device=dev)
        ctx.entry_attn(q, kn, vn, kp, vp, pt, sb.n_s, sb.l_entry, sb.capacity, out)
        assert not ctx.entry_attn_pending()
        assert torch.equal(out.view(torch.int16), out_ref.view(torch.int16)), rnd
        assert torch.equal(kp.view(torch.int16), kp_ref.view(torch.int16)) and torch.equal(vp.view(torch.int16), vp_ref.view(torch.int16))

"""GPU parity of prepos_entry_attn_fp8 (a1 + a2 over an e4m3 KV cache, DESIGN.md reading
Q20) against oracle O7, through the C ABI: every output row within the attention tolerance, and the pools after the
call -- the codes Append(E) wrote for every entry token, and every other byte untouched -- bit for bit."""
import numpy as np
import pytest
import torch

from paper_2606_29565_b200 import synth
from helpers import bits, ATTN_ATOL

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def prepos():
    from paper_2606_29565_b200 import prepos as p
    p.lib()
    return p


def _oracle_fp8(oracle, fb, layers=None):
    """O7 per (layer, session) on host copies of the code pools (the oracle appends into them in place).
    Returns ({(l, s): out fp64 [L, Hq, d]}, {s: status}, k codes after [layers...], v codes after)."""
    sb = fb.base
    layers = range(fb.k_pool8.shape[0]) if layers is None else layers
    pt = sb.page_table.cpu().numpy()
    k8 = {l: fb.k_pool8[l].cpu().numpy().copy() for l in layers}
    v8 = {l: fb.v_pool8[l].cpu().numpy().copy() for l in layers}
    outs, status = {}, {}
    for l in layers:
        ks, vs = fb.k_scale[l].cpu().numpy(), fb.v_scale[l].cpu().numpy()
        for s in range(sb.n_sessions):
            r0, L = sb.row_offset[s], sb.l_entry[s]
            res = oracle.entry_attn_fp8(bits(sb.q[l, r0:r0 + L]), bits(sb.k_new[l, r0:r0 + L]), bits(sb.v_new[l, r0:r0 + L]),
                                        k8[l], v8[l], ks, vs, pt[s], sb.n_s[s], sb.capacity[s])
            outs[(l, s)] = res["out"]
            status[s] = res["status"]
    return outs, status, k8, v8


PATHS = [1, 2]   # 1 = CUDA-core kernel, 2 = tcgen05 kernel (d = 128, pages of >= 16 tokens)


def _run(prepos, fb, path=0):
    sb, shape, dev = fb.base, fb.base.shape, "cuda"
    ctx = prepos.Context(shape.layers, shape.Hq, shape.Hkv, shape.d, shape.H, shape.V, shape.page,
                         max_sessions=max(sb.n_sessions, 1))
    if path:
        try:
            ctx.set_attn_path(path)
        except prepos.PreposError as e:
            if e.status == prepos.E_SHAPE:
                pytest.skip("shape not taken by the tcgen05 FP8 path")
            raise
    k8, v8 = fb.k_pool8.to(dev).clone(), fb.v_pool8.to(dev).clone()
    out = torch.full(sb.q.shape, float("nan"), dtype=torch.bfloat16, device=dev)
    try:
        st = ctx.entry_attn_fp8(sb.q.to(dev), sb.k_new.to(dev), sb.v_new.to(dev), k8, v8, fb.k_scale.to(dev),
                                fb.v_scale.to(dev), sb.page_table.to(dev), sb.n_s, sb.l_entry, sb.capacity, out)
    except prepos.PreposError as e:
        if e.status == prepos.E_SHAPE:
            pytest.skip("shape not taken by the tcgen05 FP8 path")
        raise
    ctx.sync()
    return out, k8, v8, st, ctx


SHAPES = {
    "d128_g4": synth.Shape("a", layers=2, Hq=8, Hkv=2, d=128, H=128, V=64, page=16),
    "d128_g8": synth.Shape("b", layers=1, Hq=16, Hkv=2, d=128, H=128, V=64, page=16),
    "d64_g2": synth.Shape("c", layers=2, Hq=4, Hkv=2, d=64, H=128, V=64, page=16),
    "d128_g1": synth.Shape("d", layers=1, Hq=2, Hkv=2, d=128, H=128, V=64, page=16),
    "d128_p32": synth.Shape("g", layers=1, Hq=8, Hkv=2, d=128, H=128, V=64, page=32),
    "d128_g1_l16": synth.Shape("i", layers=16, Hq=2, Hkv=2, d=128, H=128, V=64, page=16),
    "d128_g4_l8": synth.Shape("j", layers=8, Hq=8, Hkv=2, d=128, H=128, V=64, page=16),
    "d96_g2": synth.Shape("h", layers=1, Hq=4, Hkv=2, d=96, H=128, V=64, page=8),
}


@pytest.mark.parametrize("shape_key,n_s,l_entry,tight", [
    ("d128_g4", [0], [24], None),                         # n_s = 0: ordinary causal attention over the entry's own codes
    ("d128_g4", [1], [1], None),
    ("d128_g4", [127, 128, 129], [5, 16, 33], None),      # ragged pages: appends land in partly filled pages
    ("d128_g4", [700, 15, 300], [24, 96, 64], None),
    ("d128_g8", [517], [32], None),
    ("d64_g2", [333, 64], [8, 40], None),
    ("d128_g1", [260], [3], None),
    ("d128_g4", [2500], [24], None),
    ("d128_g4", [300, 100], [0, 7], None),                # an empty entry next to a real one
    ("d128_p32", [333], [24], None),
    ("d96_g2", [140], [6], None),
    ("d128_g4", [100, 50, 200], [12, 20, 8], [None, 69, 208]),   # a budget skip (Alg. 1 l.2-3): nothing touched
    ("d128_g1_l16", [2500, 700], [300, 257], None),       # G = 1, > 256 rows: two row chunks; units cut and merged
    ("d128_g4_l8", [3000], [40], None),                   # 8 layers over 148 CTAs: stream-K cuts inside units
])
@pytest.mark.parametrize("path", PATHS)
def test_fp8_shapes_vs_oracle(prepos, oracle, path, shape_key, n_s, l_entry, tight):
    shape = SHAPES[shape_key]
    fb = synth.make_sessions_fp8(shape, n_s, l_entry, seed=3000 + 7 * sum(n_s) + sum(l_entry), tight_capacity=tight)
    sb = fb.base
    out, k8, v8, st, _ = _run(prepos, fb, path)
    outs, ost, ok8, ov8 = _oracle_fp8(oracle, fb)
    assert st == [ost[s] for s in range(sb.n_sessions)]
    worst = 0.0
    for (l, s), ref in outs.items():
        r0, L = sb.row_offset[s], sb.l_entry[s]
        got = out[l, r0:r0 + L].cpu().to(torch.float64).numpy()
        if st[s] != 0:
            assert np.isnan(got).all()          # skipped: rows untouched
            continue
        assert np.isfinite(got).all()
        if ref.size:
            worst = max(worst, float(np.abs(got - ref).max()))
    assert worst <= ATTN_ATOL, worst
    # Append(E): the codes the kernel stored == the oracle's, and every other byte of the pools unchanged
    for l in range(shape.layers):
        assert np.array_equal(k8[l].cpu().numpy(), ok8[l]), f"K codes differ at layer {l}"
        assert np.array_equal(v8[l].cpu().numpy(), ov8[l]), f"V codes differ at layer {l}"


def test_fp8_two_step_equals_one_step(prepos, oracle):
    """Reading Q20: Forward(E) sees the entry tokens through their stored codes, so pre-positioning L1 then L2 tokens
    is the same computation as L1 + L2 in one call: identical pools, rows equal up to the kernel's own rounding."""
    shape = SHAPES["d128_g4"]
    L1, L2, n = 10, 14, 200
    fb = synth.make_sessions_fp8(shape, [n], [L1 + L2], seed=9)
    sb, dev = fb.base, "cuda"
    out_one, k1, v1, _, _ = _run(prepos, fb)
    ctx = prepos.Context(shape.layers, shape.Hq, shape.Hkv, shape.d, shape.H, shape.V, shape.page, max_sessions=1)
    k8, v8 = fb.k_pool8.to(dev).clone(), fb.v_pool8.to(dev).clone()
    ks, vs, pt = fb.k_scale.to(dev), fb.v_scale.to(dev), sb.page_table.to(dev)
    q, kn, vn = sb.q.to(dev), sb.k_new.to(dev), sb.v_new.to(dev)
    o1 = torch.zeros((shape.layers, L1, shape.Hq, shape.d), dtype=torch.bfloat16, device=dev)
    o2 = torch.zeros((shape.layers, L2, shape.Hq, shape.d), dtype=torch.bfloat16, device=dev)
    ctx.entry_attn_fp8(q[:, :L1].contiguous(), kn[:, :L1].contiguous(), vn[:, :L1].contiguous(), k8, v8, ks, vs, pt,
                       [n], [L1], sb.capacity, o1)
    ctx.entry_attn_fp8(q[:, L1:].contiguous(), kn[:, L1:].contiguous(), vn[:, L1:].contiguous(), k8, v8, ks, vs, pt,
                       [n + L1], [L2], sb.capacity, o2)
    ctx.sync()
    assert torch.equal(k8, k1) and torch.equal(v8, v1)
    two = torch.cat([o1, o2], dim=1).float()
    assert float((two - out_one.float()).abs().max()) <= 2 * ATTN_ATOL


def test_fp8_config2_slice_sampled(prepos, oracle):
    """BASELINE config 2 geometry (32/8 heads, d = 128, n_s = 4096, L = 24) on 2 of its layers at full session
    length: every row of one layer and the appended codes of both."""
    shape = synth.Shape("c2f", layers=2, Hq=32, Hkv=8, d=128, H=128, V=64, page=16)
    fb = synth.make_sessions_fp8(shape, [4096], [24], seed=synth.SEED_BASE + 1, device="cuda")
    sb = fb.base
    out, k8, v8, st, _ = _run(prepos, fb)
    assert st == [0]
    outs, ost, ok8, ov8 = _oracle_fp8(oracle, fb, layers=[1])
    got = out[1].cpu().to(torch.float64).numpy()
    assert float(np.abs(got - outs[(1, 0)]).max()) <= ATTN_ATOL
    assert np.array_equal(k8[1].cpu().numpy(), ok8[1]) and np.array_equal(v8[1].cpu().numpy(), ov8[1])


@pytest.mark.parametrize("name", ["c2", "c3", "c5"])
def test_fp8_full_size_configs(prepos, oracle, name):
    """The FP8 pass at BASELINE's full sizes in the launch configuration bench.py times (tcgen05 FP8 kernel, every
    layer in one launch, sessions generated on the device with bench.py's seeds and quantised by the synthetic
    quantiser): configs 2 and 3 (n_s = 32768, L = 16: 64 query rows per unit, 256 tiles per unit, the one shape where
    the FP8 pass is faster than the bf16 one) -- every output row of every layer; config 5 -- 64 seeded (layer, head, row) samples through
    the ranged O7; and on both the WHOLE code pools after the call: the codes Append(E) stored for every entry token
    of every layer equal the oracle's on the sampled layers, and no other byte moved."""
    shape = {"c2": synth.C2, "c3": synth.C3, "c5": synth.C5}[name]
    n_s, l_e = {"c2": ([4096], [24]), "c3": ([32768], [16]), "c5": ([16384], [32])}[name]
    seed = synth.SEED_BASE + int(name[1])
    chunk = max(64, (1 << 28) // (shape.layers * shape.Hkv * shape.page * shape.d))
    sb = synth.make_sessions(shape, n_s, l_e, seed=seed, device="cuda")
    fb = synth.quantise_sessions_fp8(sb, chunk_pages=chunk)
    del sb.k_pool, sb.v_pool
    torch.cuda.empty_cache()
    k0, v0 = fb.k_pool8.clone(), fb.v_pool8.clone()
    ctx = prepos.Context(shape.layers, shape.Hq, shape.Hkv, shape.d, shape.H, shape.V, shape.page, max_sessions=1)
    out = torch.full(sb.q.shape, float("nan"), dtype=torch.bfloat16, device="cuda")
    st = ctx.entry_attn_fp8(sb.q, sb.k_new, sb.v_new, fb.k_pool8, fb.v_pool8, fb.k_scale, fb.v_scale, sb.page_table,
                            sb.n_s, sb.l_entry, sb.capacity, out)
    ctx.sync()
    assert st == [0] and torch.isfinite(out.float()).all()
    L, page = l_e[0], shape.page
    n_pg = -(-(n_s[0] + L) // page)
    idx = sb.page_table[0, :n_pg].long()
    table = np.arange(n_pg, dtype=np.int32)
    # untouched bytes: everything outside the L appended slots of this session
    j = n_s[0] + torch.arange(L, device="cuda")
    pg, sl = sb.page_table[0].long()[j // page], j % page
    ka, va = fb.k_pool8.clone(), fb.v_pool8.clone()
    ka[:, pg, :, sl] = k0[:, pg, :, sl]
    va[:, pg, :, sl] = v0[:, pg, :, sl]
    assert torch.equal(ka, k0) and torch.equal(va, v0), "a byte outside the appended slots changed"
    del ka, va
    rng = np.random.default_rng(seed)
    G = shape.G
    worst = 0.0
    every_row = name in ("c2", "c3")
    if every_row:
        layers = range(shape.layers)
    else:
        layers = sorted(set(int(x) for x in rng.integers(0, shape.layers, 8)))
    for l in layers:
        k8 = k0[l, idx].cpu().numpy().copy()
        v8 = v0[l, idx].cpu().numpy().copy()
        ks, vs = fb.k_scale[l, idx].cpu().numpy(), fb.v_scale[l, idx].cpu().numpy()
        q, kn, vn = bits(sb.q[l]), bits(sb.k_new[l]), bits(sb.v_new[l])
        if every_row:
            ref = oracle.entry_attn_fp8(q, kn, vn, k8, v8, ks, vs, table, n_s[0], sb.capacity[0])
            worst = max(worst, float(np.abs(out[l].cpu().to(torch.float64).numpy() - ref["out"]).max()))
        else:
            for _ in range(8):
                h, i = int(rng.integers(0, shape.Hq)), int(rng.integers(0, L))
                ref = oracle.entry_attn_fp8(q, kn, vn, k8, v8, ks, vs, table, n_s[0], sb.capacity[0],
                                            heads=(h, h + 1), rows=(i, i + 1))["out"][i, h]
                worst = max(worst, float(np.abs(out[l, i, h].cpu().to(torch.float64).numpy() - ref).max()))
        # the oracle appended into its copies: the stored codes of this layer must be the kernel's
        assert np.array_equal(fb.k_pool8[l, idx].cpu().numpy(), k8), f"K codes differ at layer {l}"
        assert np.array_equal(fb.v_pool8[l, idx].cpu().numpy(), v8), f"V codes differ at layer {l}"
    assert worst <= ATTN_ATOL, worst


@pytest.mark.parametrize("shape_key,n_s,l_entry,slice_n", [
    ("d128_g4_l8", [300, 150, 410, 90, 222, 377, 64, 199, 350, 120, 280, 333], [12, 40, 7, 33, 21, 16, 45, 9, 28, 3, 37, 24], 1),
    ("d128_g1_l16", [2500, 700, 900], [300, 257, 129], 1),   # two row chunks per session; stream-K cuts inside units
    ("d128_g4_l8", [60 + 37 * i % 400 for i in range(40)], [1 + 13 * i % 64 for i in range(40)], 2),   # 640 units on
                                                             # 148 CTAs, up to 256 rows (two M-tiles), two segments a launch
])
def test_fp8_sliced_pass_and_resume_is_bit_identical(prepos, oracle, shape_key, n_s, l_entry, slice_n):
    """The yield points of attn_umma_kernel<128, kFp8>: a pass that stops after `slice_n` segments per CTA and is resumed
    until nothing is pending gives the uninterrupted call's outputs and code pools bit for bit (the FP8 path shares the
    admission words, progress counters and merge of the bf16 path, but has its own producer warp and its own polling
    site), and an unsliced call on the same ctx afterwards is unaffected."""
    shape = SHAPES[shape_key]
    fb = synth.make_sessions_fp8(shape, n_s, l_entry, seed=5151 + sum(n_s))
    sb, dev = fb.base, "cuda"
    out_ref, k_ref, v_ref, st_ref, ctx0 = _run(prepos, fb, 2)
    ctx0.close()
    ctx = prepos.Context(shape.layers, shape.Hq, shape.Hkv, shape.d, shape.H, shape.V, shape.page,
                         max_sessions=max(sb.n_sessions, 1))
    ctx.set_attn_path(2)
    args = (sb.q.to(dev), sb.k_new.to(dev), sb.v_new.to(dev))
    tail = (fb.k_scale.to(dev), fb.v_scale.to(dev), sb.page_table.to(dev), sb.n_s, sb.l_entry, sb.capacity)
    k8, v8 = fb.k_pool8.to(dev).clone(), fb.v_pool8.to(dev).clone()
    out = torch.full(sb.q.shape, float("nan"), dtype=torch.bfloat16, device=dev)
    ctx.set_attn_slice(slice_n)
    st = ctx.entry_attn_fp8(*args, k8, v8, *tail, out)
    launches = 1
    while ctx.entry_attn_pending():
        ctx.entry_attn_resume()
        launches += 1
        assert launches < 500
    assert launches >= 2, "the pass never stopped: the slice was not honoured"
    assert st == st_ref
    assert torch.equal(out.view(torch.int16), out_ref.view(torch.int16))
    assert torch.equal(k8, k_ref) and torch.equal(v8, v_ref)
    # a sliced pass that is ABANDONED after its first launch (a new call instead of a resume) must not leak its
    # half-counted arrival counters into the new pass
    k8b, v8b = fb.k_pool8.to(dev).clone(), fb.v_pool8.to(dev).clone()
    junk = torch.full(sb.q.shape, float("nan"), dtype=torch.bfloat16, device=dev)
    ctx.entry_attn_fp8(*args, k8b, v8b, *tail, junk)
    assert ctx.entry_attn_pending()
    ctx.set_attn_slice(0)
    k8c, v8c = fb.k_pool8.to(dev).clone(), fb.v_pool8.to(dev).clone()
    out2 = torch.full(sb.q.shape, float("nan"), dtype=torch.bfloat16, device=dev)
    ctx.entry_attn_fp8(*args, k8c, v8c, *tail, out2)
    assert not ctx.entry_attn_pending()
    assert torch.equal(out2.view(torch.int16), out_ref.view(torch.int16))
    assert torch.equal(k8c, k_ref) and torch.equal(v8c, v_ref)


def test_one_ctx_alternating_bf16_and_fp8_pools_at_the_same_address(prepos):
    """A ctx caches the TMA descriptors of the KV pools it was last given.  The bf16 pools take a 5-D map, the e4m3
    pools a 3-D byte map, and for one geometry the bf16 layer stride in elements EQUALS the FP8 layer stride in bytes:
    when an allocator hands the FP8 pools the address the bf16 pools had, (address, stride, pages) alone cannot tell
    the two apart.  Here both precisions deliberately live at the same base address (views of one buffer) and one ctx
    alternates between them; every call must give what a fresh ctx gives, bit for bit."""
    shape = SHAPES["d128_g4"]
    fb = synth.make_sessions_fp8(shape, [700, 15, 300], [24, 96, 64], seed=77)
    sb, dev = fb.base, "cuda"
    n_el = sb.k_pool.numel()
    bufs = [torch.zeros(2 * n_el, dtype=torch.uint8, device=dev) for _ in range(2)]
    q, kn, vn, pt = sb.q.to(dev), sb.k_new.to(dev), sb.v_new.to(dev), sb.page_table.to(dev)
    ks, vs = fb.k_scale.to(dev), fb.v_scale.to(dev)

    def pools_bf16():
        kp, vp = (b.view(torch.bfloat16).view(sb.k_pool.shape) for b in bufs)
        kp.copy_(sb.k_pool)
        vp.copy_(sb.v_pool)
        return kp, vp

    def pools_fp8():
        k8, v8 = (b[:n_el].view(fb.k_pool8.shape) for b in bufs)
        k8.copy_(fb.k_pool8)
        v8.copy_(fb.v_pool8)
        return k8, v8

    def run_bf16(ctx):
        kp, vp = pools_bf16()
        out = torch.full(sb.q.shape, float("nan"), dtype=torch.bfloat16, device=dev)
        ctx.entry_attn(q, kn, vn, kp, vp, pt, sb.n_s, sb.l_entry, sb.capacity, out)
        ctx.sync()
        return out

    def run_fp8(ctx):
        k8, v8 = pools_fp8()
        assert k8.data_ptr() == bufs[0].data_ptr() and k8.stride(0) == sb.k_pool.stride(0)   # same key as the bf16 pools
        out = torch.full(sb.q.shape, float("nan"), dtype=torch.bfloat16, device=dev)
        ctx.entry_attn_fp8(q, kn, vn, k8, v8, ks, vs, pt, sb.n_s, sb.l_entry, sb.capacity, out)
        ctx.sync()
        return out

    def new_ctx():
        c = prepos.Context(shape.layers, shape.Hq, shape.Hkv, shape.d, shape.H, shape.V, shape.page, max_sessions=3)
        c.set_attn_path(2)
        return c

    ref16, ref8 = run_bf16(new_ctx()), run_fp8(new_ctx())
    ctx = new_ctx()
    for rnd in range(2):
        assert torch.equal(run_bf16(ctx).view(torch.int16), ref16.view(torch.int16)), rnd
        assert torch.equal(run_fp8(ctx).view(torch.int16), ref8.view(torch.int16)), rnd

"""Pins of the quantised oracle variants O7 (FP8 e4m3 KV cache) and O8 (4-bit W_vocab) -- SURVEY.md 8(f) NEXT-4;
the paper's headline model "runs at 4-bit precision" but gives no storage format, so the rules
are DESIGN.md readings Q20 / Q21.  Each variant dequantises exactly and then IS O1 / O2, so the pins are:
the codec against a library's e4m3 (torch.float8_e4m3fn) and the format's closed forms, and equality with the
already-pinned O1 / O2 wherever every code * scale is exactly representable in bf16.  Also pins the ranged form of
O1 that the sampled full-size parity tests call.  CPU only."""
import numpy as np
import pytest
import torch

from paper_2606_29565_b200 import synth
from helpers import bits


def _bf16_bits_of(values64: np.ndarray) -> np.ndarray:
    """fp64 values that are exactly representable in bf16 -> their bf16 bit patterns."""
    t = torch.from_numpy(np.asarray(values64, dtype=np.float64)).to(torch.bfloat16)
    assert np.array_equal(t.to(torch.float64).numpy(), values64), "value not representable in bf16"
    return bits(t)


# ---------------------------------------------------------------- e4m3 codec
def test_e4m3_decode_all_codes_match_library(oracle):
    codes = np.arange(256, dtype=np.uint8)
    lib = torch.from_numpy(codes).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    got = oracle.e4m3_decode(codes)
    assert np.array_equal(np.isnan(got), np.isnan(lib)) and np.isnan(got).sum() == 2      # S.1111.111 only
    ok = ~np.isnan(lib)
    assert np.array_equal(got[ok], lib[ok])
    # closed forms of the format: largest finite 448, smallest subnormal 2^-9, smallest normal 2^-6, 1.0
    assert got[0x7e] == 448.0 and got[0x01] == 2.0 ** -9 and got[0x08] == 2.0 ** -6 and got[0x38] == 1.0
    assert got[0x80] == 0.0 and np.signbit(got[0x80]) and got[0xfe] == -448.0


def test_e4m3_encode_matches_library_and_saturates(oracle):
    rng = np.random.default_rng(1)
    y = np.concatenate([rng.normal(0, 1, 20000), rng.uniform(-448, 448, 20000), rng.normal(0, 0.01, 5000),
                        np.linspace(-448, 448, 7169)]).astype(np.float32)
    lib = torch.from_numpy(y).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    got = oracle.e4m3_encode(y)
    same = (got == lib) | ((got & 0x7f) == 0) & ((lib & 0x7f) == 0)      # +-0 count as equal
    assert same.all(), (y[~same][:5], got[~same][:5], lib[~same][:5])
    # every representable value encodes to itself; exact midpoints go to the even code
    finite = np.array([c for c in range(256) if (c & 0x7f) != 0x7f], dtype=np.uint8)
    assert np.array_equal(oracle.e4m3_encode(oracle.e4m3_decode(finite).astype(np.float32)), finite)
    lo = np.arange(0, 0x7e, dtype=np.uint8)
    mid = ((oracle.e4m3_decode(lo) + oracle.e4m3_decode(lo + 1)) / 2).astype(np.float32)
    assert np.array_equal(oracle.e4m3_encode(mid), np.where(lo % 2 == 0, lo, lo + 1))
    # saturating: anything beyond +-448 (incl. inf) is +-448; NaN is the NaN code
    big = np.array([448.0, 449.0, 464.0, 1e6, np.inf, -1e6, -np.inf], dtype=np.float32)
    assert oracle.e4m3_encode(big).tolist() == [0x7e] * 5 + [0xfe] * 2
    assert oracle.e4m3_encode(np.array([np.nan], dtype=np.float32))[0] == 0x7f


# ---------------------------------------------------------------- O7: FP8 KV attention
def _fp8_case(oracle, rng, n_s, L, Hq=4, Hkv=2, d=16, page=8, scale_exp=(0, 0), extra_pages=1):
    """Random finite e4m3 codes for cache and entry, power-of-two page scales: every code * scale is exactly
    representable in bf16, so the same session exists as a bf16 one."""
    n_pages = (n_s + L + page - 1) // page + extra_pages
    table = rng.permutation(n_pages).astype(np.int32)
    finite = np.array([c for c in range(256) if (c & 0x7f) != 0x7f and 0x08 <= (c & 0x7f) <= 0x5f], dtype=np.uint8)
    kp8 = rng.choice(finite, (n_pages, Hkv, page, d)).astype(np.uint8)
    vp8 = rng.choice(finite, (n_pages, Hkv, page, d)).astype(np.uint8)
    ks = (2.0 ** rng.integers(scale_exp[0], scale_exp[1] + 1, (n_pages, Hkv))).astype(np.float32)
    vs = (2.0 ** rng.integers(scale_exp[0], scale_exp[1] + 1, (n_pages, Hkv))).astype(np.float32)
    q = bits(torch.from_numpy(rng.normal(0, 1, (L, Hq, d))).to(torch.bfloat16))
    # entry K/V = representable code * the scale of the page they will land in
    kn_c = rng.choice(finite, (L, Hkv, d)).astype(np.uint8)
    vn_c = rng.choice(finite, (L, Hkv, d)).astype(np.uint8)
    pg = table[(n_s + np.arange(L)) // page]
    kn = _bf16_bits_of(oracle.e4m3_decode(kn_c) * ks[pg][:, :, None].astype(np.float64))
    vn = _bf16_bits_of(oracle.e4m3_decode(vn_c) * vs[pg][:, :, None].astype(np.float64))
    kp16 = _bf16_bits_of(oracle.e4m3_decode(kp8) * ks[:, :, None, None].astype(np.float64))
    vp16 = _bf16_bits_of(oracle.e4m3_decode(vp8) * vs[:, :, None, None].astype(np.float64))
    return dict(q=q, kn=kn, vn=vn, kp8=kp8, vp8=vp8, ks=ks, vs=vs, kp16=kp16, vp16=vp16, table=table, n_s=n_s,
                cap=n_pages * page, kn_c=kn_c, vn_c=vn_c, page=page)


@pytest.mark.parametrize("n_s,L,scale_exp", [(0, 7, (0, 0)), (37, 5, (0, 0)), (21, 12, (-3, 2)), (64, 1, (-2, 2))])
def test_fp8_attention_equals_o1_on_representable_values(oracle, n_s, L, scale_exp):
    """All scales 1 (and then powers of two) with representable values: O7 == O1 on the widened pool, and the
    appended codes are the entry codes (quantise o dequantise = identity on representable values)."""
    c = _fp8_case(oracle, np.random.default_rng(n_s * 100 + L), n_s, L, scale_exp=scale_exp)
    ref = oracle.entry_attn(c["q"], c["kn"], c["vn"], c["kp16"], c["vp16"], c["table"], n_s, c["cap"])
    got = oracle.entry_attn_fp8(c["q"], c["kn"], c["vn"], c["kp8"], c["vp8"], c["ks"], c["vs"], c["table"], n_s, c["cap"])
    assert ref["status"] == got["status"] == 0 and got["position"] == n_s + L
    assert np.abs(got["out"] - ref["out"]).max() <= 1e-12
    page = c["page"]
    for jp in range(L):
        pg, sl = c["table"][(n_s + jp) // page], (n_s + jp) % page
        assert np.array_equal(c["kp8"][pg, :, sl], c["kn_c"][jp]) and np.array_equal(c["vp8"][pg, :, sl], c["vn_c"][jp])
    # and the dequantised appended cache is O1's appended cache
    assert np.array_equal(oracle.e4m3_decode(c["kp8"]) * c["ks"][:, :, None, None], torch.from_numpy(
        c["kp16"].view(np.int16)).view(torch.bfloat16).to(torch.float64).numpy())


def test_fp8_append_rule_scale_saturation_and_untouched_bytes(oracle):
    """Append(E): code = e4m3(fp32(x) / scale), round to nearest even, saturating; nothing else in the pool moves."""
    rng = np.random.default_rng(5)
    c = _fp8_case(oracle, rng, 19, 6)
    c["ks"][:] = rng.uniform(0.002, 0.005, c["ks"].shape).astype(np.float32)      # |x| / 0.003 > 448 beyond 1.3: saturates
    c["vs"][:] = rng.uniform(0.002, 0.005, c["vs"].shape).astype(np.float32)
    kn = bits(torch.from_numpy(rng.normal(0, 1, (6, 2, 16))).to(torch.bfloat16))
    vn = bits(torch.from_numpy(rng.normal(0, 1, (6, 2, 16))).to(torch.bfloat16))
    k0, v0 = c["kp8"].copy(), c["vp8"].copy()
    oracle.entry_attn_fp8(c["q"], kn, vn, c["kp8"], c["vp8"], c["ks"], c["vs"], c["table"], 19, c["cap"])
    touched = np.zeros(k0.shape[:1] + k0.shape[2:3], dtype=bool)
    saturated = 0
    for jp in range(6):
        pg, sl = c["table"][(19 + jp) // 8], (19 + jp) % 8
        touched[pg, sl] = True
        for g in range(2):
            x = torch.from_numpy(kn[jp, g].view(np.int16)).view(torch.bfloat16).to(torch.float32).numpy()
            y = (x / c["ks"][pg, g]).astype(np.float32)                          # fp32 division, round to nearest
            want = torch.from_numpy(np.clip(y, -448, 448)).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
            got = c["kp8"][pg, g, sl]
            assert np.array_equal(got & 0x7f, want & 0x7f) and np.array_equal((got >> 7)[want & 0x7f != 0], (want >> 7)[want & 0x7f != 0])
            saturated += int((np.abs(y) > 448).sum())
    assert saturated > 0
    m = ~touched[:, None, :, None] & np.ones(k0.shape, dtype=bool)
    assert np.array_equal(c["kp8"][m], k0[m]) and np.array_equal(c["vp8"][m], v0[m])


def test_fp8_two_step_ranged_and_budget(oracle):
    """Forward(E) runs after Append(E) on the stored codes, so L1 then L2 tokens == L1 + L2 tokens bit for bit;
    the ranged call returns the same rows; a budget skip touches nothing."""
    rng = np.random.default_rng(9)
    c = _fp8_case(oracle, rng, 30, 11, scale_exp=(-8, -6))
    kn = bits(torch.from_numpy(rng.normal(0, 1, (11, 2, 16))).to(torch.bfloat16))    # NOT representable: real rounding
    vn = bits(torch.from_numpy(rng.normal(0, 1, (11, 2, 16))).to(torch.bfloat16))
    a = {k: v.copy() for k, v in c.items() if isinstance(v, np.ndarray)}
    one = oracle.entry_attn_fp8(c["q"], kn, vn, a["kp8"], a["vp8"], c["ks"], c["vs"], c["table"], 30, c["cap"])
    b = {k: v.copy() for k, v in c.items() if isinstance(v, np.ndarray)}
    s1 = oracle.entry_attn_fp8(c["q"][:4], kn[:4], vn[:4], b["kp8"], b["vp8"], c["ks"], c["vs"], c["table"], 30, c["cap"])
    s2 = oracle.entry_attn_fp8(c["q"][4:], kn[4:], vn[4:], b["kp8"], b["vp8"], c["ks"], c["vs"], c["table"], 34, c["cap"])
    assert np.array_equal(np.concatenate([s1["out"], s2["out"]]), one["out"])
    assert np.array_equal(a["kp8"], b["kp8"]) and np.array_equal(a["vp8"], b["vp8"])
    d = {k: v.copy() for k, v in c.items() if isinstance(v, np.ndarray)}
    part = oracle.entry_attn_fp8(c["q"], kn, vn, d["kp8"], d["vp8"], c["ks"], c["vs"], c["table"], 30, c["cap"],
                                 heads=(1, 3), rows=(5, 9))
    assert np.array_equal(part["out"][5:9, 1:3], one["out"][5:9, 1:3])
    mask = np.ones(one["out"].shape, dtype=bool)
    mask[5:9, 1:3] = False
    assert np.isnan(part["out"][mask]).all() and np.array_equal(d["kp8"], a["kp8"])
    e = {k: v.copy() for k, v in c.items() if isinstance(v, np.ndarray)}
    skip = oracle.entry_attn_fp8(c["q"], kn, vn, e["kp8"], e["vp8"], c["ks"], c["vs"], c["table"], 30, 40)
    assert skip["status"] == 1 and np.array_equal(e["kp8"], c["kp8"]) and np.isnan(skip["out"]).all()


def test_fp8_scale_is_per_page_and_kv_head(oracle):
    """Doubling one (page, kv head) K scale is the same as doubling that page's K values for that head only."""
    rng = np.random.default_rng(11)
    c = _fp8_case(oracle, rng, 40, 3, scale_exp=(-1, 1))
    base = oracle.entry_attn_fp8(c["q"], c["kn"], c["vn"], c["kp8"].copy(), c["vp8"].copy(), c["ks"], c["vs"], c["table"], 40, c["cap"])
    pg = int(c["table"][2])                                   # logical page 2 = cached tokens 16..23
    ks2 = c["ks"].copy()
    ks2[pg, 1] *= 2
    kp16 = c["kp16"].copy()
    kp16[pg, 1] = _bf16_bits_of(oracle.e4m3_decode(c["kp8"][pg, 1]) * float(ks2[pg, 1]))
    ref = oracle.entry_attn(c["q"], c["kn"], c["vn"], kp16, c["vp16"].copy(), c["table"], 40, c["cap"])
    got = oracle.entry_attn_fp8(c["q"], c["kn"], c["vn"], c["kp8"].copy(), c["vp8"].copy(), ks2, c["vs"], c["table"], 40, c["cap"])
    assert np.abs(got["out"] - ref["out"]).max() <= 1e-12
    assert np.array_equal(got["out"][:, :2], base["out"][:, :2])      # heads of kv head 0 unchanged
    assert np.abs(got["out"][:, 2:] - base["out"][:, 2:]).max() > 1e-6


# ---------------------------------------------------------------- O8: 4-bit W_vocab logits
def _w4_case(rng, V, H, group, scale_exp=(0, 0)):
    codes = rng.integers(-8, 8, (V, H))
    nib = np.where(codes < 0, codes + 16, codes).astype(np.uint8)
    w4 = (nib[:, 0::2] | (nib[:, 1::2] << 4)).astype(np.uint8)                # even k in the low nibble
    sc = 2.0 ** rng.integers(scale_exp[0], scale_exp[1] + 1, (V, H // group)).astype(np.float64)
    w_scale = _bf16_bits_of(sc)
    w16 = _bf16_bits_of(codes * np.repeat(sc, group, axis=1))
    return codes, w4, sc, w_scale, w16


@pytest.mark.parametrize("scale_exp", [(0, 0), (-9, -4)])
def test_w4_logits_equal_o2_on_representable_weights(oracle, scale_exp):
    rng = np.random.default_rng(3)
    V, H, group = 97, 256, 128
    codes, w4, sc, w_scale, w16 = _w4_case(rng, V, H, group, scale_exp)
    x = bits(torch.from_numpy(rng.normal(0, 1, H)).to(torch.bfloat16))
    assert np.abs(oracle.logits_w4(w4, w_scale, x, group) - oracle.logits(w16, x)).max() <= 1e-12
    # the record of those logits is O3's (nothing quantisation-specific after the dequantisation)
    lg = oracle.logits_w4(w4, w_scale, x, group)
    assert oracle.record(lg).top1 == int(np.argmax(lg))


def test_w4_nibble_order_sign_and_group_boundaries(oracle):
    """x = e_k picks column k: low nibble = even k, two's-complement sign, scale index k // group."""
    rng = np.random.default_rng(4)
    V, H, group = 33, 384, 128
    codes, w4, sc, w_scale, _ = _w4_case(rng, V, H, group, (-3, 3))
    assert codes.min() == -8 and codes.max() == 7
    for k in (0, 1, 2, 127, 128, 129, 255, 256, 383):
        x = np.zeros(H)
        x[k] = 1.0
        lg = oracle.logits_w4(w4, w_scale, _bf16_bits_of(x), group)
        assert np.array_equal(lg, codes[:, k] * sc[:, k // group]), k


# ---------------------------------------------------------------- ranged O1 (used by the sampled parity tests)
def test_ranged_attention_is_the_full_one_on_its_range(oracle):
    sb = synth.make_sessions(synth.C1, [100], [9], seed=17)
    args = lambda: (bits(sb.q[0]), bits(sb.k_new[0]), bits(sb.v_new[0]), bits(sb.k_pool[0]), bits(sb.v_pool[0]),
                    sb.page_table[0].numpy(), 100, sb.capacity[0])
    full = oracle.entry_attn(*args(), want_rowsum=True)
    a = args()
    part = oracle.entry_attn(*a, heads=(2, 3), rows=(4, 7), want_rowsum=True)
    assert np.array_equal(part["out"][4:7, 2:3], full["out"][4:7, 2:3])
    mask = np.ones(full["out"].shape, dtype=bool)
    mask[4:7, 2:3] = False
    assert np.isnan(part["out"][mask]).all()
    b = args()
    oracle.entry_attn(*b)
    assert np.array_equal(a[3], b[3]) and np.array_equal(a[4], b[4])          # the append is complete either way
    with pytest.raises(ValueError):
        oracle.entry_attn(*args(), heads=(0, 5))

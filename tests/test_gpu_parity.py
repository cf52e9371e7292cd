"""GPU parity (-m gpu): libfenc's CUDA path, called through the C ABI, against the CPU oracle element by element on
the same seeded inputs.  Bar: bit-exact on every RNS limb (integer work); decoded outputs within 1e-3 of plaintext
fp64 convolution (BASELINE.json north_star).  Parity starts at integer plaintext coefficients (A7)."""
from fractions import Fraction

import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mods():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from oracle import ckks as ck
    from oracle import fragment as fr
    import paper_2606_16359_b200 as fenc
    return ck, fr, fenc


def make(mods, name, **over):
    ck, fr, fenc = mods
    p = dict(wl.PARAMS[name], **over)
    P = ck.Params(*wl.oracle_params_args(p))
    ctx = fenc.Context(**p)
    assert ctx.q == P.q and ctx.p == P.p and ctx.dlen == P.dlen
    return P, ctx


@pytest.mark.parametrize("q_bits,p_bits", [(30, 31), (50, 60), (58, 60)])
def test_long_mac_every_accumulation_mode(mods, q_bits, p_bits):
    """PMult-accumulate of 2100 terms: the MAC kernel's three accumulation modes (20-bit limbs in fp64 below 2^40,
    26-bit limbs below 2^52, 128-bit otherwise) each fold their pending sum back at least once (a7)."""
    ck, fr, fenc = mods
    P, ctx = make(mods, "toy64", q_bits=q_bits, p_bits=p_bits)
    N, L = P.N, P.nq
    rng = np.random.default_rng(5)
    limbs = [wl.random_ct_limbs(100 + i, P.q, L, N) for i in range(5)]
    ws = [ck.encode(P, rng.normal(0, 0.5, P.n), L, 2.0 ** 20) for _ in range(7)]
    octs = [ck.Ciphertext(x, L, 2.0 ** 20) for x in limbs]
    gcts = [ctx.ct_import(x, 2.0 ** 20) for x in limbs]
    gpts = [ctx.pt_from_coeffs(w.coeffs, L, float(w.scale)) for w in ws]
    n_terms = 2100
    acc = np.zeros_like(limbs[0])
    for t in range(n_terms):
        ck.pmult_acc(P, acc, octs[t % 5], ws[t % 7])
    got = ctx.pmult_sum([gcts[t % 5] for t in range(n_terms)], [gpts[t % 7] for t in range(n_terms)])
    assert np.array_equal(ctx.ct_export(got), acc)
    ctx.close()


@pytest.mark.parametrize("name", ["toy64", "mid10", "mid12"])
def test_primitives_bit_exact(mods, name):
    ck, fr, fenc = mods
    P, ctx = make(mods, name)
    N, L = P.N, P.nq
    rng = np.random.default_rng(11)
    limbs = wl.random_ct_limbs(3, P.q, L, N)
    assert np.array_equal(ctx.ct_export(ctx.ct_import(limbs, 2.0 ** 20)), limbs)  # NTT round trip at full N
    steps = [1, 2, 5, P.n - 1, P.n // 2]
    ok = ck.keygen(P, 42, steps, want_relin=True)
    gk = ctx.keygen(42, steps, want_relin=True)
    assert np.array_equal(ctx.secret_export(gk), ok.s)
    for kid in steps + [ck.RELIN_KEY_ID]:
        b, a = ctx.evk_export(gk, kid)
        assert np.array_equal(a, ok.evk[kid][1]) and np.array_equal(b, ok.evk[kid][0]), kid
    z = rng.uniform(-1, 1, P.n)
    opt = ck.encode(P, z, L)
    oct_ = ck.encrypt(P, ok, opt, 7)
    gct = ctx.encrypt(gk, ctx.pt_from_coeffs(opt.coeffs, L, float(opt.scale)), 7)
    assert np.array_equal(ctx.ct_export(gct), oct_.c)
    assert np.abs(ctx.decrypt_slots(gk, gct) - z).max() < 1e-4
    # batched rotation, including step 0 and a repeated step
    st = steps + [0, 1]
    outs = ctx.rotate(gk, [gct] * len(st), st)
    for r, o in zip(st, outs):
        assert np.array_equal(ctx.ct_export(o), ck.rotate(P, ok, oct_, r).c), r
    assert np.abs(ctx.decrypt_slots(gk, outs[1]) - np.roll(z, -2)).max() < 1e-4  # left shift (R2.7)
    # PMult-accumulate of three terms, then rescale
    ws = [ck.encode(P, rng.normal(0, 0.1, P.n), L, P.q[L - 1]) for _ in range(3)]
    acc = np.zeros_like(oct_.c)
    rots = [ck.rotate(P, ok, oct_, r) for r in (0, 1, 2)]
    for x, w in zip(rots, ws):
        ck.pmult_acc(P, acc, x, w)
    gp = ctx.pmult_sum([outs[5], outs[0], outs[1]], [ctx.pt_from_coeffs(w.coeffs, L, float(w.scale)) for w in ws])
    assert np.array_equal(ctx.ct_export(gp), acc)
    ors = ck.rescale(P, ck.Ciphertext(acc, L, oct_.scale * ws[0].scale))
    grs = ctx.rescale([gp])[0]
    assert np.array_equal(ctx.ct_export(grs), ors.c) and grs.L == L - 1
    assert abs(grs.scale - float(ors.scale)) <= 1e-9 * float(ors.scale)
    # add, square + relinearise + rescale
    assert np.array_equal(ctx.ct_export(ctx.add(gct, outs[0])), ck.add(P, oct_, rots[1]).c)
    assert np.array_equal(ctx.ct_export(ctx.square_relin(gk, gct)), ck.square_relin(P, ok, oct_).c)
    # rotation below the top level (short last digit: 5 limbs -> 3 limbs, dlen 2 -> digits 2,1)
    o2 = ck.rescale(P, ors) if ors.L > 2 else ors
    g2 = ctx.rescale([grs])[0] if ors.L > 2 else grs
    assert np.array_equal(ctx.ct_export(ctx.rotate(gk, [g2], [5])[0]), ck.rotate(P, ok, o2, 5).c)
    ctx.close()


@pytest.mark.parametrize("name", ["toy64", "mid12"])
def test_keys_import_host_generated_material(mods, name):
    """fenc_keys_import: the ORACLE's secret and switching keys (generated on the host from the seed, R2.3/R2.4) uploaded
    verbatim; rotations, a hoisted rotation and x^2 with the imported keys equal the oracle's bit for bit, and the imported
    key set re-exports to the same material."""
    ck, fr, fenc = mods
    P, ctx = make(mods, name)
    steps = [1, 7, P.n - 1]
    ok = ck.keygen(P, 99, steps, want_relin=True)
    gk = ctx.keys_import(ok.s, {kid: ok.evk[kid] for kid in steps + [ck.RELIN_KEY_ID]})
    assert np.array_equal(ctx.secret_export(gk), ok.s)
    b, a = ctx.evk_export(gk, 7)
    assert np.array_equal(b, ok.evk[7][0]) and np.array_equal(a, ok.evk[7][1])
    L = P.nq
    pt = ck.encode(P, np.random.default_rng(1).uniform(-1, 1, P.n), L)
    oct_ = ck.encrypt(P, ok, pt, 5)
    gct = ctx.encrypt(gk, ctx.pt_from_coeffs(pt.coeffs, L, float(pt.scale)), 5)
    assert np.array_equal(ctx.ct_export(gct), oct_.c)
    for r, o in zip(steps, ctx.rotate(gk, [gct] * 3, steps)):
        assert np.array_equal(ctx.ct_export(o), ck.rotate(P, ok, oct_, r).c), r
    assert np.array_equal(ctx.ct_export(ctx.rotate_hoisted(gk, [gct], [7])[0][0]), ck.rotate_hoisted(P, ok, oct_, 7).c)
    assert np.array_equal(ctx.ct_export(ctx.square_relin(gk, gct)), ck.square_relin(P, ok, oct_).c)
    with pytest.raises(fenc.FencError):
        ctx.keys_import(np.full(P.N, 2, dtype=np.int64), {})  # not ternary
    ctx.close()


def test_errors_and_edges(mods):
    ck, fr, fenc = mods
    P, ctx = make(mods, "toy64")
    gk = ctx.keygen(1, [1])
    ct = ctx.encrypt(gk, ctx.encode_slots(np.zeros(P.n), 1), 3)
    with pytest.raises(fenc.FencError, match="NO_KEY"):
        ctx.rotate(gk, [ct], [2])
    with pytest.raises(fenc.FencError, match="LEVEL"):
        ctx.rescale([ct])
    with pytest.raises(fenc.FencError, match="NO_KEY"):
        ctx.square_relin(gk, ct)
    assert ctx.rotate(gk, [], []) == []
    with pytest.raises(fenc.FencError):
        fenc.Context(log2N=6, n_q=4, q_bits=30, n_p=1, p_bits=31, dnum=1)  # P < Q_j without allow_noisy_ks
    ctx.close()


def test_library_encoder_close_to_oracle(mods):
    ck, fr, fenc = mods
    P, ctx = make(mods, "mid12")
    rng = np.random.default_rng(5)
    z = rng.uniform(-1, 1, P.n) + 1j * rng.uniform(-1, 1, P.n)
    mine = ctx.pt_coeffs(ctx.encode_slots(z, 2))
    assert np.abs(mine - ck.encode_coeffs(z, P.N, P.scale)).max() <= 1  # A7: rounding may differ by one
    const = ctx.pt_coeffs(ctx.encode_slots(np.full(P.n, 0.25), 2))
    assert const[0] == round(0.25 * 2 ** 40) and not const[1:].any()       # closed form (R2.2)
    ctx.close()


def run_hconv(mods, P, ctx, conv_kw, S, seed, do_rescale=True, kaiming=False, hoist=False):
    """GPU fenc_hconv vs oracle hconv for every batch group; returns (max decoded error, layout)."""
    ck, fr, fenc = mods
    x, w = wl.conv_inputs(seed, conv_kw, kaiming=kaiming)
    od = fr.ConvDesc(S=S, **conv_kw)  # (seg_v / B_cap / bsgs ride along in conv_kw: both descriptors take them)
    graph = fr.ConvGraph(od, P.n)
    conv = ctx.conv_desc(S=S, **conv_kw)
    lay = ctx.layout_plan(conv)
    c = graph.counts()
    assert (lay.n_in_ct, lay.n_out_ct, lay.n_inner_rot, lay.n_outer_rot, lay.n_pmult, lay.n_distinct_pt) == \
        (c["n_in_ct"], c["n_out_ct"], c["n_inner_rot"], c["n_outer_rot"], c["n_pmult"], c["n_distinct_pt"])
    assert lay.steps() == c["rot_steps"]
    L = P.nq
    ok = ck.keygen(P, 100 + seed, c["rot_steps"])
    gk = ctx.keygen(100 + seed, c["rot_steps"])
    oW = fr.encode_weights(ck, P, graph, w, L)
    keys = ctx.wts_keys(conv, lay)
    coeffs = np.stack([oW[tuple(int(v) for v in k)].coeffs for k in keys])
    gW = ctx.conv_weights_from_coeffs(conv, lay, coeffs, L, float(P.q[L - 1]))
    lin = graph.lin
    g_in, o_in = [], {}
    for bg in range(lin.BG):
        for g in range(lin.G):
            for u in range(S):
                for v in range(S):
                    pt = ck.encode(P, lin.gather(x, u, v, g, bg), L)
                    o_in[(bg, u, v, g)] = ck.encrypt(P, ok, pt, 1000 + len(g_in))
                    g_in.append(ctx.encrypt(gk, ctx.pt_from_coeffs(pt.coeffs, L, float(pt.scale)), 1000 + len(g_in)))
    ctx.set_hoisting(hoist)
    g_out = ctx.hconv(gk, conv, lay, gW, g_in, do_rescale=do_rescale)
    So, lout = graph.S_out, graph.lout
    Y = np.zeros((od.BS, od.C_out, od.H_out, od.W_out))
    for bg in range(lin.BG):
        ins = {(u, v, g): o_in[(bg, u, v, g)] for g in range(lin.G) for u in range(S) for v in range(S)}
        o_out = fr.hconv(ck, P, ok, graph, ins, oW, do_rescale=do_rescale, hoist=hoist)
        for go in range(lout.G):
            for uo in range(So):
                for vo in range(So):
                    gct = g_out[((bg * lout.G + go) * So + uo) * So + vo]
                    ref = o_out[(uo, vo, go)]
                    assert np.array_equal(ctx.ct_export(gct), ref.c), (bg, go, uo, vo)
                    assert abs(gct.scale - float(ref.scale)) <= 1e-9 * float(ref.scale)
                    ctx.decrypt_decode(gk, gct, conv, lay, 1, uo, vo, go, bg, Y)
    err = np.abs(Y - fr.direct_conv(od, x, w)).max()
    return err, lay


@pytest.mark.parametrize("conv_kw,S", [
    (dict(BS=2, C_in=4, H=8, W=8, C_out=4, K=3, stride=1, pad=1), 2),      # inner + outer rotations, 2 samples per ct
    (dict(BS=1, C_in=3, H=7, W=6, C_out=5, K=3, stride=1, pad=1), 1),      # ragged channels and frame, row-major (S=1)
    (dict(BS=3, C_in=2, H=8, W=8, C_out=4, K=3, stride=2, pad=1), 2),      # stride by dropping fragments; BS not 2^k
    (dict(BS=1, C_in=4, H=8, W=8, C_out=4, K=3, stride=1, pad=1, depthwise=True), 4),
    (dict(BS=40, C_in=2, H=8, W=8, C_out=3, K=1, stride=1, pad=0), 2),     # several batch groups (B=32, BG=2), 1x1
])
def test_hconv_bit_exact_small(mods, conv_kw, S):
    P, ctx = make(mods, "mid10")
    err, _ = run_hconv(mods, P, ctx, conv_kw, S, seed=3)
    assert err < 1e-3
    ctx.close()


@pytest.mark.parametrize("name", ["mid10", "mid12"])
@pytest.mark.parametrize("conv_kw,S", [
    (dict(BS=2, C_in=4, H=8, W=8, C_out=4, K=3, stride=1, pad=1), 2),      # 3 inner rotations per input ciphertext
    (dict(BS=1, C_in=3, H=7, W=6, C_out=5, K=3, stride=1, pad=1), 1),      # 8 inner rotations of one ciphertext, outer ones plain
    (dict(BS=40, C_in=2, H=8, W=8, C_out=3, K=3, stride=1, pad=1), 2),     # two batch groups: sources of both in one batch
])
def test_hconv_hoisted_inner_rotations_bit_exact(mods, name, conv_kw, S):
    """R2.7b: one decomposition per input ciphertext, automorphism on the extended digits; compared limb by limb with
    the oracle's hoisted variant (ragged digits: 5 limbs, dlen 2), decoded result against the plain convolution."""
    P, ctx = make(mods, name)
    err, _ = run_hconv(mods, P, ctx, conv_kw, S, seed=5, hoist=True)
    assert err < 1e-3
    ctx.close()


def run_hconv_factored(mods, P, ctx, conv_kw, S, seed, hoist=False, w_scale=1.0):
    """GPU fenc_hconv with factored weights (R2.9c) vs the oracle's hconv_factored for every batch group; parity starts at
    the integer multipliers and the masks' integer coefficients (A7).  Returns the max decoded error."""
    ck, fr, fenc = mods
    x, w = wl.conv_inputs(seed, conv_kw)
    w = w * w_scale
    od = fr.ConvDesc(S=S, **conv_kw)
    graph = fr.ConvGraph(od, P.n)
    conv = ctx.conv_desc(S=S, **conv_kw)
    lay = ctx.layout_plan(conv)
    assert lay.ch == 1
    c = graph.counts()
    L = P.nq
    ok, gk = ck.keygen(P, 200 + seed, c["rot_steps"]), ctx.keygen(200 + seed, c["rot_steps"])
    values, masks, E1 = fr.factor_weights(ck, P, graph, w, L)
    E2 = next(iter(masks.values())).scale
    keys = [tuple(int(v) for v in k) for k in ctx.wts_keys(conv, lay)]
    mask_of, n_masks = ctx.wts_factors(conv, lay)
    assert n_masks == len(masks) and len(mask_of) == len(keys)
    by_id = {}
    for wk, mid in zip(keys, mask_of):
        assert by_id.setdefault(int(mid), graph.mask_of[wk]) == graph.mask_of[wk]  # the same partition of the weights
    assert len(set(by_id.values())) == n_masks
    for mid, mk in by_id.items():
        assert np.array_equal(ctx.wts_mask_slots(conv, lay, mid), graph.mask_slots(mk))
    k = np.array([ck.round_half_up(Fraction(values[wk]) * E1) for wk in keys], dtype=np.int64)
    mc = np.stack([masks[by_id[i]].coeffs for i in range(n_masks)])
    gW = ctx.conv_weights_factored_from_ints(conv, lay, k, mc, L, float(E1), float(E2))
    lin = graph.lin
    g_in, o_in = [], {}
    for bg in range(lin.BG):
        for g in range(lin.G):
            for u in range(S):
                for v in range(S):
                    pt = ck.encode(P, lin.gather(x, u, v, g, bg), L)
                    o_in[(bg, u, v, g)] = ck.encrypt(P, ok, pt, 1000 + len(g_in))
                    g_in.append(ctx.encrypt(gk, ctx.pt_from_coeffs(pt.coeffs, L, float(pt.scale)), 1000 + len(g_in)))
    ctx.set_hoisting(hoist)
    g_out = ctx.hconv(gk, conv, lay, gW, g_in)
    So, lout = graph.S_out, graph.lout
    Y = np.zeros((od.BS, od.C_out, od.H_out, od.W_out))
    for bg in range(lin.BG):
        ins = {(u, v, g): o_in[(bg, u, v, g)] for g in range(lin.G) for u in range(S) for v in range(S)}
        o_out = fr.hconv_factored(ck, P, ok, graph, ins, values, masks, E1, hoist=hoist)
        for go in range(lout.G):
            for uo in range(So):
                for vo in range(So):
                    gct = g_out[((bg * lout.G + go) * So + uo) * So + vo]
                    ref = o_out[(uo, vo, go)]
                    assert np.array_equal(ctx.ct_export(gct), ref.c), (bg, go, uo, vo)
                    assert abs(gct.scale - float(ref.scale)) <= 1e-9 * float(ref.scale)
                    ctx.decrypt_decode(gk, gct, conv, lay, 1, uo, vo, go, bg, Y)
    err = np.abs(Y - fr.direct_conv(od, x, w)).max()
    # the library's own factoring (fp64 weights in, multipliers rounded and masks encoded on the library side)
    outs2 = ctx.hconv(gk, conv, lay, ctx.conv_weights_factored(conv, lay, w, L), g_in)
    Y2 = np.zeros_like(Y)
    i = 0
    for bg in range(lin.BG):
        for go in range(lout.G):
            for uo in range(So):
                for vo in range(So):
                    ctx.decrypt_decode(gk, outs2[i], conv, lay, 1, uo, vo, go, bg, Y2)
                    i += 1
    assert np.abs(Y2 - Y).max() < 1e-5 * max(1.0, w_scale)
    return err


@pytest.mark.parametrize("name,over,conv_kw,S,hoist", [
    ("mid10", {}, dict(BS=32, C_in=3, H=4, W=4, C_out=5, K=3, stride=1, pad=1), 1, False),           # 27 terms, border masks
    ("mid10", {}, dict(BS=64, C_in=2, H=7, W=6, C_out=3, K=3, stride=2, pad=1), 2, True),            # stride, frame > data, BG=2, hoisted
    ("mid10", {}, dict(BS=32, C_in=4, H=4, W=4, C_out=4, K=3, stride=1, pad=1, depthwise=True), 1, False),
    ("mid10", {}, dict(BS=40, C_in=9, H=4, W=4, C_out=11, K=1, stride=1, pad=0), 1, False),          # point-wise: groups of 8 + 3 outputs, ragged batch
    ("mid12", dict(q_bits=50, log2_scale=50), dict(BS=32, C_in=3, H=8, W=8, C_out=9, K=3, stride=1, pad=1), 1, True),  # 50-bit: fp64 sums reduced every 7 terms
    ("toy64", dict(q_bits=58, p_bits=60, log2_scale=30), dict(BS=8, C_in=5, H=2, W=2, C_out=3, K=1, stride=1, pad=0), 1, False),  # 58-bit: integer mode
])
def test_hconv_factored_weights_bit_exact(mods, name, over, conv_kw, S, hoist):
    """R2.9c (large-batch layouts, ch = 1): weight plaintexts replaced by integer multipliers and shared mask plaintexts;
    limbs against the oracle's factored variant, decoded result against direct convolution."""
    P, ctx = make(mods, name, **over)
    err = run_hconv_factored(mods, P, ctx, conv_kw, S, seed=6, hoist=hoist)
    assert err < (1e-3 if name != "toy64" else 5e-2)
    ctx.close()


@pytest.mark.parametrize("mode", ["1", "2", "3"])
@pytest.mark.parametrize("name,over", [("mid12", dict(q_bits=50, log2_scale=50)), ("mid10", {})])
def test_smac_modes_give_identical_limbs(mods, monkeypatch, name, over, mode):
    """The scalar MAC's arithmetic modes (fenc_elem.cu: exact fp64 products of residues; the ciphertext word split in
    2 x 25 or 3 x 17 bits times the SIGNED multiplier) forced one by one on the same layer: each equals the oracle's
    factored variant limb by limb.  9 output channels: groups of 8 + 1 outputs (4 + 4 + 1 in the 3-piece mode), hoisted."""
    monkeypatch.setenv("FENC_SMAC_MODE", mode)
    P, ctx = make(mods, name, **over)
    err = run_hconv_factored(mods, P, ctx, dict(BS=32, C_in=3, H=8, W=8, C_out=9, K=3, stride=1, pad=1), 1, seed=7, hoist=True)
    assert err < 1e-3
    ctx.close()


@pytest.mark.parametrize("w_scale,bound", [(12.0, 1e-3), (4000.0, None)])
def test_smac_mode_selection_for_large_multipliers(mods, w_scale, bound):
    """Weights 12 x larger (|k| up to 2^30: the 2-piece products no longer sum exactly, the library picks 3 pieces) and
    4000 x larger (|k| beyond 2^36: back to exact products of residues): limbs against the oracle in both; the decoded
    bar only where the outputs stay of ordinary size."""
    P, ctx = make(mods, "mid12", q_bits=50, log2_scale=50)
    err = run_hconv_factored(mods, P, ctx, dict(BS=32, C_in=3, H=8, W=8, C_out=5, K=3, stride=1, pad=1), 1, seed=9, w_scale=w_scale)
    assert bound is None or err < bound
    ctx.close()


def test_factored_weights_need_one_channel_per_ciphertext(mods):
    ck, fr, fenc = mods
    P, ctx = make(mods, "mid10")
    conv = ctx.conv_desc(S=1, BS=1, C_in=4, H=4, W=4, C_out=4, K=3, stride=1, pad=1)
    lay = ctx.layout_plan(conv)
    assert lay.ch > 1
    with pytest.raises(fenc.FencError, match="LAYOUT"):
        ctx.conv_weights_factored(conv, lay, np.zeros((4, 4, 3, 3)), P.nq)
    ctx.close()


@pytest.mark.parametrize("conv_kw,S,hoist", [
    (dict(BS=4, C_in=2, H=4, W=4, C_out=8, K=3, stride=1, pad=1, seg_v=2, B_cap=4), 1, False),    # n=512: m=4, B=4, chp=8, 4 segments
    (dict(BS=7, C_in=2, H=4, W=4, C_out=5, K=1, stride=1, pad=0, seg_v=2, B_cap=1), 1, False),    # chp=32, 16 segments, ragged
    (dict(BS=16, C_in=3, H=8, W=8, C_out=8, K=3, stride=2, pad=1, seg_v=4, B_cap=2), 2, True),    # S=2, B=2, chp=16, v=4, two output groups, hoisted
])
def test_hconv_segmented_layout_bit_exact(mods, conv_kw, S, hoist):
    """R2.11b: fenc_hconv over the segmented layout AAC's compaction produces (diagonal d as two partial sums rotated by
    d*cs and (d - v)*cs), every limb against the oracle's graph, decoded against direct convolution."""
    P, ctx = make(mods, "mid10")
    err, lay = run_hconv(mods, P, ctx, conv_kw, S, seed=8, hoist=hoist)
    assert lay.seg > 1 and lay.ch == conv_kw["seg_v"] and lay.ch_phys == lay.seg * lay.ch
    assert err < 1e-3
    ctx.close()


def test_bottleneck_compress_then_segmented_conv_bit_exact(mods):
    """Fig. 5 through the C ABI: reduce 8 -> 2 channels (1x1) on plain-layout ciphertexts, fenc_compress
    the 25 %-full outputs of four batch groups into one dense ciphertext, expand 2 -> 8 (3x3) with fenc_hconv on the
    segmented layout.  Every ciphertext of the chain equals the oracle's; the decoded result equals the two convolutions."""
    ck, fr, fenc = mods
    p = dict(wl.PARAMS["mid10"], log2N=8)
    P = ck.Params(*wl.oracle_params_args(p))
    ctx = fenc.Context(**p)
    n, L = P.n, P.nq
    red = dict(BS=4, C_in=8, H=4, W=4, C_out=2, K=1, stride=1, pad=0, B_cap=1)
    exp = dict(BS=4, C_in=2, H=4, W=4, C_out=8, K=3, stride=1, pad=1, B_cap=1, seg_v=2)
    rng = np.random.default_rng(3)
    x = rng.uniform(-1, 1, (4, 8, 4, 4))
    w1, w2 = rng.normal(0, 0.3, (2, 8, 1, 1)), rng.normal(0, 0.3, (8, 2, 3, 3))
    g1, g2 = fr.ConvGraph(fr.ConvDesc(S=1, **red), n), fr.ConvGraph(fr.ConvDesc(S=1, **exp), n)
    c1, c2 = ctx.conv_desc(S=1, **red), ctx.conv_desc(S=1, **exp)
    l1, l2 = ctx.layout_plan(c1), ctx.layout_plan(c2)
    assert (l1.ch, l1.BG, l2.seg, l2.BG, l2.G_out, l2.n_in_ct, l2.n_out_ct) == (8, 4, 4, 1, 4, 1, 4)
    plan = fr.compress_plan(n, 8, g1.lin.cs, 2, 4)
    steps = sorted(set(l1.steps()) | set(l2.steps()) | {r for tl in plan for _, r in tl if r})
    assert set(l2.steps()) == set(g2.counts()["rot_steps"])
    ok, gk = ck.keygen(P, 4, steps), ctx.keygen(4, steps)
    W1, W2 = fr.encode_weights(ck, P, g1, w1, L), fr.encode_weights(ck, P, g2, w2, L - 1)
    gW1 = ctx.conv_weights_from_coeffs(c1, l1, np.stack([W1[tuple(int(v) for v in k)].coeffs for k in ctx.wts_keys(c1, l1)]), L, float(P.q[L - 1]))
    gW2 = ctx.conv_weights_from_coeffs(c2, l2, np.stack([W2[tuple(int(v) for v in k)].coeffs for k in ctx.wts_keys(c2, l2)]), L - 1, float(P.q[L - 2]))
    o_mid, g_in = [], []
    for bg in range(4):
        pt = ck.encode(P, g1.lin.gather(x, 0, 0, 0, bg), L)
        o_mid.append(fr.hconv(ck, P, ok, g1, {(0, 0, 0): ck.encrypt(P, ok, pt, 40 + bg)}, W1)[(0, 0, 0)])
        g_in.append(ctx.encrypt(gk, ctx.pt_from_coeffs(pt.coeffs, L, float(pt.scale)), 40 + bg))
    g_mid = ctx.hconv(gk, c1, l1, gW1, g_in)
    for a, b in zip(g_mid, o_mid):
        assert np.array_equal(ctx.ct_export(a), b.c)
    o_packed = fr.compress(ck, P, ok, plan, o_mid)
    g_packed = ctx.compress(gk, g_mid, [(t, i, r) for t, tl in enumerate(plan) for i, r in tl], len(plan))
    assert len(g_packed) == 1 and np.array_equal(ctx.ct_export(g_packed[0]), o_packed[0].c)
    o_out = fr.hconv(ck, P, ok, g2, {(0, 0, 0): o_packed[0]}, W2)
    g_out = ctx.hconv(gk, c2, l2, gW2, g_packed)
    Y = np.zeros((4, 8, 4, 4))
    for go in range(4):
        assert np.array_equal(ctx.ct_export(g_out[go]), o_out[(0, 0, go)].c), go
        ctx.decrypt_decode(gk, g_out[go], c2, l2, 1, 0, 0, go, 0, Y)
    want = fr.direct_conv(fr.ConvDesc(**exp), fr.direct_conv(fr.ConvDesc(**red), x, w1), w2)
    assert np.abs(Y - want).max() < 1e-3
    ctx.close()


@pytest.mark.parametrize("S_src,S_dst,shape", [(2, 1, (1, 4, 8, 8)), (1, 2, (2, 2, 8, 8)), (2, 4, (1, 8, 7, 6))])
def test_repack_block_size_bit_exact(mods, S_src, S_dst, shape):
    """fenc_repack (R2.11c; PAPER.md:290 block-size re-adaptation) against the oracle's repack on the plan between two
    block sizes: every limb, one level consumed, and the decoded tensor unchanged."""
    ck, fr, fenc = mods
    P, ctx = make(mods, "mid10")
    L = P.nq
    BS, C, H, W = shape
    M = fr.next_pow2(max(H, W))
    src, dst = fr.Layout(P.n, M, S_src, BS, C), fr.Layout(P.n, M, S_dst, BS, C)
    x = np.random.default_rng(15).uniform(-1, 1, shape)
    plan = fr.repack_plan(src, dst, shape)
    steps = sorted({r for terms in plan.values() for _, r, _ in terms if r})
    ok, gk = ck.keygen(P, 6, steps), ctx.keygen(6, steps)
    skeys = src.ct_keys()
    o_in, g_in = {}, []
    for i, k in enumerate(skeys):
        pt = ck.encode(P, src.gather(x, *k), L)
        o_in[k] = ck.encrypt(P, ok, pt, 60 + i)
        g_in.append(ctx.encrypt(gk, ctx.pt_from_coeffs(pt.coeffs, L, float(pt.scale)), 60 + i))
    ref = fr.repack(ck, P, ok, plan, o_in, L)
    dkeys = dst.ct_keys()
    terms = []
    for t, dk in enumerate(dkeys):
        for skey, r, mask in plan[dk]:
            m = ck.encode(P, mask, L, P.q[L - 1])
            terms.append((t, skeys.index(skey), r, ctx.pt_from_coeffs(m.coeffs, L, float(m.scale))))
    got = ctx.repack(gk, g_in, terms, len(dkeys))
    Y = np.zeros(shape)
    for t, dk in enumerate(dkeys):
        assert got[t].L == L - 1 and np.array_equal(ctx.ct_export(got[t]), ref[dk].c), dk
        dst.scatter(Y, ctx.decrypt_slots(gk, got[t]).real, *dk)
    assert np.abs(Y - x).max() < 1e-4
    ctx.close()


@pytest.mark.parametrize("conv_kw,S,hoist", [
    (dict(BS=1, C_in=8, H=8, W=8, C_out=8, K=3, stride=1, pad=1, bsgs=2), 1, False),    # n=512: ch=8, 17 inner + 3 outer
    (dict(BS=1, C_in=5, H=8, W=8, C_out=7, K=3, stride=1, pad=1, bsgs=4), 1, True),     # ragged channels, hoisted composite amounts
    (dict(BS=2, C_in=4, H=8, W=8, C_out=8, K=3, stride=2, pad=1, bsgs=2), 2, True),     # S=2, stride 2, two output groups
    (dict(BS=1, C_in=16, H=4, W=4, C_out=16, K=3, stride=1, pad=1, bsgs=0), 1, True),   # ch=32: the auto rule picks g=2
    (dict(BS=4, C_in=8, H=4, W=4, C_out=16, K=3, stride=1, pad=1, B_cap=1, seg_v=8, bsgs=2), 1, True),  # segmented layout (R2.11b) + BSGS
])
def test_hconv_bsgs_channel_diagonals_bit_exact(mods, conv_kw, S, hoist):
    """R2.9d: baby-step giant-step over the convolution's channel diagonals (baby step folded into the inner rotation,
    weight plaintexts shifted, giant steps as outer rotations): every limb against the oracle's variant, same counts and
    rotation amounts on both sides (asserted in run_hconv), decoded against direct convolution."""
    P, ctx = make(mods, "mid10")
    plain = ctx.layout_plan(ctx.conv_desc(S=S, **dict(conv_kw, bsgs=1)))
    err, lay = run_hconv(mods, P, ctx, conv_kw, S, seed=10, hoist=hoist)
    assert err < 1e-3
    assert lay.n_outer_rot < plain.n_outer_rot and lay.n_pmult == plain.n_pmult and lay.n_distinct_pt == plain.n_distinct_pt
    if conv_kw["bsgs"] == 0:
        assert lay.n_inner_rot + lay.n_outer_rot < plain.n_inner_rot + plain.n_outer_rot
    ctx.close()


def test_hconv_fig4_toy(mods):
    """PAPER.md:160 (Fig. 4): input 1x16x4x4, conv(16,16,3,1), 16-slot ciphertexts, S in {1,2,4}."""
    ck, fr, fenc = mods
    for S, rots in ((1, 128), (2, 96), (4, 240)):
        P = ck.Params(5, 3, 30, 1, 31, 3, 25)
        ctx = fenc.Context(log2N=5, n_q=3, q_bits=30, n_p=1, p_bits=31, dnum=3, log2_scale=25)
        err, lay = run_hconv(mods, P, ctx, wl.CONVS["fig4_toy"], S, seed=4)
        assert lay.n_inner_rot + lay.n_outer_rot == rots
        assert err < 5e-2  # 25-bit scale, 30-bit primes: the toy's own precision
        ctx.close()


def test_hconv_config1_full_size(mods):
    """BASELINE config 1 (LeNet conv1-shaped, N=2^13, primary reading A1) at the size bench.py times."""
    P, ctx = make(mods, "cfg1")
    conv = ctx.conv_desc(**wl.CONVS["lenet_conv1"])
    assert ctx.layout_plan(conv).S == 1  # Conv-aware selection (Eq. 7 bound < 1 -> smallest feasible)
    err, lay = run_hconv(mods, P, ctx, wl.CONVS["lenet_conv1"], 1, seed=1001)
    assert (lay.n_in_ct, lay.n_out_ct, lay.n_inner_rot, lay.n_outer_rot, lay.n_pmult, lay.n_rot_keys) == (1, 2, 24, 4, 150, 27)
    assert err < 1e-3
    ctx.close()


def test_hconv_config1_literal_dnum1_bit_exact_only(mods):
    """Literal dnum=1 (one digit of 3 limbs, P < Q): decoded check waived (A1), limbs must still match."""
    ck, fr, fenc = mods
    P, ctx = make(mods, "cfg1_literal")
    assert ctx.dlen == 3 and ctx.beta_max == 1
    ok = ck.keygen(P, 9, [1, 33])
    gk = ctx.keygen(9, [1, 33])
    limbs = wl.random_ct_limbs(8, P.q, 3, P.N)
    outs = ctx.rotate(gk, [ctx.ct_import(limbs)] * 2, [1, 33])
    for r, o in zip((1, 33), outs):
        assert np.array_equal(ctx.ct_export(o), ck.rotate(P, ok, ck.Ciphertext(limbs, 3, 1), r).c)
    ctx.close()


def test_compress_fig5_shape(mods):
    """PAPER.md:258-262 (Fig. 5): 4 sparse ciphertexts at 25% -> 1 dense; maskless keeps the level, the split-scale
    masked mode consumes exactly one rescale."""
    ck, fr, fenc = mods
    P, ctx = make(mods, "mid10")
    n, L, ch, v = P.n, P.nq, 8, 2
    cs = n // ch
    plan = fr.compress_plan(n, ch, cs, v, 4)
    steps = sorted({r for terms in plan for _, r in terms if r})
    ok, gk = ck.keygen(P, 77, steps), ctx.keygen(77, steps)
    rng = np.random.default_rng(6)
    srcs_o, srcs_g, vecs = [], [], []
    for i in range(4):
        z = np.zeros(n)
        z[: v * cs] = rng.uniform(-1, 1, v * cs)
        pt = ck.encode(P, z, L)
        srcs_o.append(ck.encrypt(P, ok, pt, 50 + i))
        srcs_g.append(ctx.encrypt(gk, ctx.pt_from_coeffs(pt.coeffs, L, float(pt.scale)), 50 + i))
        vecs.append(z)
    terms = [(t, i, r) for t, tl in enumerate(plan) for i, r in tl]
    ref = fr.compress(ck, P, ok, plan, srcs_o)
    got = ctx.compress(gk, srcs_g, terms, len(plan))
    assert len(got) == 1 and got[0].L == L
    assert np.array_equal(ctx.ct_export(got[0]), ref[0].c)
    want = sum(np.roll(vecs[i], -r) for i, r in plan[0])
    assert np.abs(ctx.decrypt_slots(gk, got[0]).real - want).max() < 1e-4
    # masked, split scale: mask at Delta2 = q_{L-1} here, one rescale after
    mask = ck.encode(P, fr.compress_mask(n, cs, v), L, P.q[L - 1])
    ref = fr.compress(ck, P, ok, plan, srcs_o, mask_pt=mask, do_rescale=True)
    got = ctx.compress(gk, srcs_g, terms, len(plan), mask=ctx.pt_from_coeffs(mask.coeffs, L, float(mask.scale)), do_rescale=True)
    assert got[0].L == L - 1 and np.array_equal(ctx.ct_export(got[0]), ref[0].c)
    ctx.close()


def test_rotation_full_size_config3_sampled(mods):
    """N=2^16, 24+4 limbs, dlen 4 (config 3): one batched rotation at the bench's launch configuration; the oracle
    checks two limbs of each polynomial fully (the oracle's key switch costs ~1 min at this size)."""
    ck, fr, fenc = mods
    P, ctx = make(mods, "cfg3")
    steps = [1, 12345]
    gk = ctx.keygen(5, steps)
    ok = ck.keygen(P, 5, steps[:1])
    L = P.nq
    limbs = wl.random_ct_limbs(21, P.q, L, P.N)
    gin = ctx.ct_import(limbs)
    outs = ctx.rotate(gk, [gin, gin], steps)
    ref = ck.rotate(P, ok, ck.Ciphertext(limbs, L, 1), 1)
    assert np.array_equal(ctx.ct_export(outs[0]), ref.c)
    ctx.close()


@pytest.mark.parametrize("n_q,q_bits,n_p,dnum", [(7, 40, 5, 1), (9, 50, 9, 1), (12, 50, 6, 2), (20, 40, 10, 2)])
def test_rotation_wide_digit_groups(mods, n_q, q_bits, n_p, dnum):
    """Digit groups of 6 and more limbs (config 5's dnum = 1, 2 points): the fused column kernel runs 2 or 4 thread
    groups per block over shared source tiles (ragged target counts per group); a second rotation one level down has a
    short last digit.  N = 2^12: four column tiles per limb."""
    ck, fr, fenc = mods
    p = dict(log2N=12, n_q=n_q, q_bits=q_bits, n_p=n_p, p_bits=60, dnum=dnum, log2_scale=q_bits)
    P = ck.Params(*wl.oracle_params_args(p))
    ctx = fenc.Context(**p)
    assert ctx.q == P.q and ctx.p == P.p and ctx.dlen == P.dlen
    steps = [3, P.n - 7]
    ok, gk = ck.keygen(P, 9, steps), ctx.keygen(9, steps)
    for L in (P.nq, P.nq - 1):
        limbs = wl.random_ct_limbs(100 + L, P.q, L, P.N)
        gin = ctx.ct_import(limbs)
        outs = ctx.rotate(gk, [gin, gin, gin], steps + [3])
        for r, o in zip(steps + [3], outs):
            assert np.array_equal(ctx.ct_export(o), ck.rotate(P, ok, ck.Ciphertext(limbs, L, 1), r).c), (L, r)
    ctx.close()


@pytest.mark.parametrize("name", ["toy64", "mid10", "mid12"])
def test_rotate_hoisted_bit_exact(mods, name):
    """fenc_rotate_hoisted (R2.7b) against the oracle's hoisted rotation: several ciphertexts by several amounts
    (including 0 and n-1) at the top level and one level down (short last digit)."""
    ck, fr, fenc = mods
    P, ctx = make(mods, name)
    steps = [1, 5, 0, P.n - 1, P.n // 2]
    ok, gk = ck.keygen(P, 17, steps), ctx.keygen(17, steps)
    for L in (P.nq, P.nq - 1):
        limbs = [wl.random_ct_limbs(40 + 3 * L + i, P.q, L, P.N) for i in range(3)]
        outs = ctx.rotate_hoisted(gk, [ctx.ct_import(a) for a in limbs], steps)
        for a, row in zip(limbs, outs):
            for r, o in zip(steps, row):
                assert np.array_equal(ctx.ct_export(o), ck.rotate_hoisted(P, ok, ck.Ciphertext(a, L, 1), r).c), (L, r)
    z = np.random.default_rng(2).uniform(-1, 1, P.n)
    pt = ck.encode(P, z, P.nq)
    g = ctx.encrypt(gk, ctx.pt_from_coeffs(pt.coeffs, P.nq, float(pt.scale)), 3)
    assert np.abs(ctx.decrypt_slots(gk, ctx.rotate_hoisted(gk, [g], [5])[0][0]).real - np.roll(z, -5)).max() < 1e-3
    ctx.close()


def test_rotate_hoisted_full_size_config3_sampled(mods):
    """N=2^16, 24+4 limbs (config 3), the launch configuration of the hoisted sweep: two ciphertexts by two amounts, the
    oracle checks one of the four fully."""
    ck, fr, fenc = mods
    P, ctx = make(mods, "cfg3")
    steps = [1, 12345]
    gk = ctx.keygen(5, steps)
    ok = ck.keygen(P, 5, steps[1:])
    L = P.nq
    limbs = [wl.random_ct_limbs(21 + i, P.q, L, P.N) for i in range(2)]
    outs = ctx.rotate_hoisted(gk, [ctx.ct_import(a) for a in limbs], steps)
    ref = ck.rotate_hoisted(P, ok, ck.Ciphertext(limbs[1], L, 1), 12345)
    assert np.array_equal(ctx.ct_export(outs[1][1]), ref.c)
    ctx.close()


def test_import_async_matches_import(mods):
    """fenc_ct_import_async (copy stream + staging ring) gives the ciphertexts of fenc_ct_import, also when the ring wraps
    (more uploads in flight than slots would be needed: 70 > 64), when the level changes between uploads, and with work
    queued on the compute stream in between."""
    import torch
    ck, fr, fenc = mods
    P, ctx = make(mods, "mid12")
    gk = ctx.keygen(3, [1])
    hosts = []
    for i in range(70):
        L = P.nq if i % 3 else P.nq - 2
        a = wl.random_ct_limbs(500 + i, P.q, L, P.N)
        hosts.append(torch.from_numpy(a.view(np.int64)).pin_memory())
    views = [t.numpy().view(np.uint64) for t in hosts]
    cts = []
    for i, a in enumerate(views):
        cts.append(ctx.ct_import_async(a))
        if i % 7 == 0:
            cts[-1] = ctx.rotate(gk, [cts[-1]], [0])[0]  # compute-stream work between uploads (step 0: a copy)
    for a, c in zip(views, cts):
        assert c.L == a.shape[1]
        assert np.array_equal(ctx.ct_export(c), a)
    ref = ctx.rotate(gk, [ctx.ct_import(views[1])], [1])[0]
    got = ctx.rotate(gk, [ctx.ct_import_async(views[1])], [1])[0]
    assert np.array_equal(ctx.ct_export(got), ctx.ct_export(ref))
    # asynchronous export: results land in page-locked buffers, complete after export_wait, with later work enqueued behind
    outs = [torch.zeros(v.shape, dtype=torch.int64).pin_memory().numpy().view(np.uint64) for v in views[:5]]
    for c, o in zip(cts[:5], outs):
        ctx.ct_export_async(c, o)
    later = ctx.rotate(gk, [cts[1]], [1])[0]
    ctx.export_wait()
    for a, o in zip(views[:5], outs):
        assert np.array_equal(a, o)
    assert np.array_equal(ctx.ct_export(later), ctx.ct_export(ref))
    ctx.close()


def test_export_async_survives_free_and_reuse_of_the_ciphertext(mods):
    """fenc_ct_export_async reads the ciphertext in stream order and copies on a stream of its own (include/fenc.h): the
    handle may be freed right after the call and its memory reused by later work; the staging queue of the imports grows
    with a cap (FENC_STAGE_MAX_MB, here 1 MiB = two slots: every upload then waits for its slot's previous transform);
    fenc_sync, not only fenc_export_wait, makes the results visible; the device bytes held return to their level once the
    exports have landed."""
    import os
    import torch
    ck, fr, fenc = mods
    os.environ["FENC_STAGE_MAX_MB"] = "1"
    try:
        P, ctx = make(mods, "mid12")
        gk = ctx.keygen(4, [1, 2])
        views = []
        for i in range(24):
            a = wl.random_ct_limbs(700 + i, P.q, P.nq, P.N)
            views.append(torch.from_numpy(a.view(np.int64)).pin_memory().numpy().view(np.uint64))
        want = [ctx.ct_export(ctx.rotate(gk, [ctx.ct_import(a)], [1])[0]) for a in views]
        ctx.sync()
        base, held = ctx.device_bytes(), None
        for rnd in range(2):  # second round: the export buffers and events of the first are reused
            outs = [torch.zeros(v.shape, dtype=torch.int64).pin_memory().numpy().view(np.uint64) for v in views]
            for a, o in zip(views, outs):
                c = ctx.rotate(gk, [ctx.ct_import_async(a)], [1])[0]
                ctx.ct_export_async(c, o)
                del c  # freed while the export is in flight: the next iteration's buffers come from the same pool
            junk = ctx.rotate(gk, [ctx.ct_import(views[0])] * 8, [2] * 8)  # more work behind the exports, reusing freed blocks
            if rnd == 0:
                ctx.export_wait()
            else:
                ctx.sync()
            for w_, o in zip(want, outs):
                assert np.array_equal(w_, o)
            del junk
            ctx.sync()
            if held is None:
                held = ctx.device_bytes()  # what stays after a round: staging slots (capped), the grown workspace
                assert held > base
            assert ctx.device_bytes() == held  # steady state: every export buffer has returned, nothing else grew
        ctx.close()
    finally:
        del os.environ["FENC_STAGE_MAX_MB"]


# ------------------------------------------------------------------------------------------------ fc, pooling, pipeline
@pytest.mark.parametrize("kw", [
    dict(BS=2, n_in=32, n_out=5, in_C=2, in_H=4, in_W=4, in_M=4),
    dict(BS=40, n_in=3 * 3 * 3, n_out=20, in_C=3, in_H=3, in_W=3, in_M=4),   # B=32, BG=2, P=16, two output cts
    dict(BS=64, n_in=20, n_out=11, in_M=4),                                  # flat input
    # baby-step giant-step (R2.12b): explicit g and the library's choice (bsgs=0), several input / output ciphertexts
    dict(BS=2, n_in=32, n_out=5, in_C=2, in_H=4, in_W=4, in_M=4, bsgs=4),
    dict(BS=40, n_in=3 * 3 * 3, n_out=20, in_C=3, in_H=3, in_W=3, in_M=4, bsgs=0),
    dict(BS=64, n_in=20, n_out=11, in_M=4, bsgs=2),
    dict(BS=16, n_in=70, n_out=40, in_M=2, bsgs=0),                          # P = 32: 3 input cts, 2 output cts
    dict(BS=16, n_in=70, n_out=40, in_M=2, bsgs=0, hoist=True),              # baby steps in the hoisted form (R2.7b)
    dict(BS=40, n_in=3 * 3 * 3, n_out=20, in_C=3, in_H=3, in_W=3, in_M=4, bsgs=4, hoist=True),
    # fragment-encoded token embeddings (R2.13): E = S P exactly (the paper's case), ragged, mixed orders, with BSGS
    dict(BS=16, n_in=64, n_out=64, in_M=2, frag_in=2, frag_out=2),           # P = 32 = E / S
    dict(BS=40, n_in=30, n_out=20, in_M=4, frag_in=2, frag_out=4, bsgs=0),   # two batch groups, ragged sub-blocks
    dict(BS=16, n_in=60, n_out=40, in_M=2, frag_in=4, bsgs=0, hoist=True),   # fragment-encoded in, positional out
    dict(BS=16, n_in=40, n_out=64, in_M=2, frag_out=2),                      # positional in, fragment-encoded out
])
def test_fc_bit_exact(mods, kw):
    ck, fr, fenc = mods
    from oracle import network as nw
    kw = dict(kw)
    hoist = kw.pop("hoist", False)
    P, ctx = make(mods, "mid10")
    ctx.set_hoisting(hoist)
    g = nw.FcGraph(P.n, **kw)
    fcd = ctx.fc_desc(**kw)
    info = ctx.fc_plan(fcd)
    c = g.counts()
    assert {k: info[k] for k in c} == c
    if kw.get("bsgs", 1) != 1:
        assert info["bsgs"] > 1 and info["n_rot"] < nw.FcGraph(P.n, **dict(kw, bsgs=1)).counts()["n_rot"]
    L = P.nq
    rng = np.random.default_rng(9)
    X = rng.uniform(-1, 1, (kw["BS"], kw["n_in"]))
    W = rng.normal(0, 0.3, (kw["n_out"], kw["n_in"]))
    ok, gk = ck.keygen(P, 31, c["rot_steps"]), ctx.keygen(31, c["rot_steps"])
    oW = nw.encode_fc_weights(ck, P, g, W, L)
    coeffs = np.stack([oW[tuple(int(v) for v in k)].coeffs for k in ctx.fc_wts_keys(fcd)])
    gW = ctx.fc_weights_from_coeffs(fcd, coeffs, L, float(P.q[L - 1]))
    o_in, g_in = [], []
    for bg in range(g.BG):
        for ci in range(g.n_in_ct):
            pt = ck.encode(P, g.gather_in(X, ci, bg), L)
            o_in.append(ck.encrypt(P, ok, pt, 70 + len(o_in)))
            g_in.append(ctx.encrypt(gk, ctx.pt_from_coeffs(pt.coeffs, L, float(pt.scale)), 70 + len(g_in)))
    g_out = ctx.fc(gk, fcd, gW, g_in)
    Y = np.zeros((kw["BS"], kw["n_out"]))
    for bg in range(g.BG):
        ref = nw.fc(ck, P, ok, g, o_in[bg * g.n_in_ct:(bg + 1) * g.n_in_ct], oW, hoist=hoist)
        for co, r in enumerate(ref):
            got = g_out[bg * g.n_out_ct + co]
            assert np.array_equal(ctx.ct_export(got), r.c), (bg, co)
            g.scatter_out(Y, ctx.decrypt_slots(gk, got).real, co, bg)
    assert np.abs(Y - X @ W.T).max() < 1e-3
    # the library's own weight encoder lands within one unit of the oracle's integers (A7)
    gW2 = ctx.fc_weights(fcd, W, L)
    assert gW2 is not None
    # fenc_fc_encode_input / fenc_fc_decrypt_decode: the library's gather + encoder lands within one unit of the oracle's
    # integers on every input ciphertext, and its scatter places the decrypted slots where the oracle's does
    for bg in range(g.BG):
        for ci in range(g.n_in_ct):
            want = ck.encode(P, g.gather_in(X, ci, bg), L).coeffs
            got = ctx.pt_coeffs(ctx.fc_encode_input(fcd, X, ci, bg, L))
            assert np.abs(got - want).max() <= 1, (bg, ci)
    Y2 = np.zeros_like(Y)
    for bg in range(g.BG):
        for co in range(g.n_out_ct):
            ctx.fc_decrypt_decode(gk, g_out[bg * g.n_out_ct + co], fcd, 1, co, bg, Y2)
    assert np.array_equal(Y2, Y)
    X2 = np.zeros_like(X)
    for bg in range(g.BG):
        for ci in range(g.n_in_ct):
            ctx.fc_decrypt_decode(gk, g_in[bg * g.n_in_ct + ci], fcd, 0, ci, bg, X2)
    assert np.abs(X2 - X).max() < 1e-6
    ctx.close()


def test_square_sum_relin_bit_exact(mods):
    """fenc_square_sum_relin (R2.12c) against the oracle's square_sum_relin: groups of 4, 2 and 1 ciphertexts at two ring
    sizes (merged and unmerged ModDown + rescale), and the decoded sum of squares."""
    ck, fr, fenc = mods
    for name in ("mid10", "mid12"):
        P, ctx = make(mods, name)
        ok, gk = ck.keygen(P, 23, [], want_relin=True), ctx.keygen(23, [], want_relin=True)
        rng = np.random.default_rng(12)
        zs = [rng.uniform(-1, 1, P.n) for _ in range(8)]
        o_in, g_in = [], []
        for i, z in enumerate(zs):
            pt = ck.encode(P, z, P.nq)
            o_in.append(ck.encrypt(P, ok, pt, 300 + i))
            g_in.append(ctx.encrypt(gk, ctx.pt_from_coeffs(pt.coeffs, P.nq, float(pt.scale)), 300 + i))
        for group in (4, 2, 1):
            got = ctx.square_sum_relin(gk, g_in, group)
            assert len(got) == 8 // group
            for o, g in enumerate(got):
                ref = ck.square_sum_relin(P, ok, o_in[o * group:(o + 1) * group])
                assert g.L == ref.L and np.array_equal(ctx.ct_export(g), ref.c), (name, group, o)
                assert abs(g.scale - float(ref.scale)) <= 1e-9 * float(ref.scale)
            want = sum(z * z for z in zs[:group])
            assert np.abs(ctx.decrypt_slots(gk, got[0]).real - want).max() < 1e-4
        ctx.close()


@pytest.mark.parametrize("bsgs,hoist,lazy", [(1, False, False), (0, False, False), (0, True, False), (0, True, True)])
def test_pipeline_toy_network_bit_exact(mods, bsgs, hoist, lazy):
    """conv - square - pool - fc - fc through Pipeline (one batched C-ABI call per layer) vs the oracle's network."""
    ck, fr, fenc = mods
    from oracle import network as nw
    from paper_2606_16359_b200.pipeline import Pipeline
    from test_oracle_network import plain_network, toy_network
    p = dict(log2N=9, n_q=5, q_bits=40, n_p=2, p_bits=60, dnum=3, log2_scale=40)
    P = ck.Params(*wl.oracle_params_args(p))
    ctx = fenc.Context(**p)
    ctx.set_hoisting(hoist)
    layers, x = toy_network(bsgs=bsgs)
    pipe = Pipeline(ctx, layers)
    steps, relin = nw.network_rot_steps(layers, P.n)
    assert sorted(pipe.steps) == steps and pipe.need_relin == relin

    def enc_w(entry):
        L = entry["L"]
        if entry["op"] == "conv":
            g = fr.ConvGraph(fr.ConvDesc(S=int(entry["conv"].S), **{k: int(getattr(entry["conv"], k)) for k in
                             ("BS", "C_in", "H", "W", "C_out", "K", "stride", "pad")}), P.n)
            oW = fr.encode_weights(ck, P, g, entry["w"], L)
            return np.stack([oW[tuple(int(v) for v in k)].coeffs for k in ctx.wts_keys(entry["conv"], entry["lay"])])
        fcd = entry["fc"]
        g = nw.FcGraph(P.n, **{k: int(getattr(fcd, k)) for k in ("BS", "n_in", "n_out", "in_C", "in_H", "in_W", "in_M")},
                       bsgs=0 if fcd.bsgs == 0xFFFFFFFF else int(fcd.bsgs))
        oW = nw.encode_fc_weights(ck, P, g, entry["w"], L)
        return np.stack([oW[tuple(int(v) for v in k)].coeffs for k in ctx.fc_wts_keys(fcd)])

    gk = pipe.setup(key_seed=11, encode_weight=enc_w)
    ok = ck.keygen(P, 11, steps, want_relin=relin)
    lin = fr.Layout(P.n, 8, 2, 2, 1)
    o_in, g_in = [], []
    for i, (u, v, g, bg) in enumerate(lin.ct_keys()):
        pt = ck.encode(P, lin.gather(x, u, v, g, bg), P.nq)
        o_in.append(ck.encrypt(P, ok, pt, 100 + i))
        g_in.append(ctx.encrypt(gk, ctx.pt_from_coeffs(pt.coeffs, P.nq, float(pt.scale)), 100 + i))
    o_out, o_trace = nw.run_network(ck, P, ok, layers, o_in, P.nq, hoist=hoist, lazy_relin=lazy)
    g_trace = []
    g_out = pipe.forward(g_in, trace=g_trace, lazy_relin=lazy)
    for li, (ol, gl) in enumerate(zip(o_trace, g_trace)):
        assert len(ol) == len(gl), li
        for a, b in zip(ol, gl):
            assert np.array_equal(ctx.ct_export(b), a.c), li
    fg = nw.FcGraph(P.n, **layers[-1]["fc"])
    Y = np.zeros((2, 3))
    fg.scatter_out(Y, ctx.decrypt_slots(gk, g_out[0]).real, 0, 0)
    assert np.abs(Y - plain_network(layers, x)).max() < 1e-3
    # the same network with the library's own encoder (Algorithm 1 gather + fp64 encode on the library side)
    pipe2 = Pipeline(ctx, layers)
    pipe2.setup(key_seed=12)
    out2 = pipe2.forward(pipe2.encrypt_input(x, 500))
    fg.scatter_out(Y, ctx.decrypt_slots(pipe2.keys, out2[0]).real, 0, 0)
    assert np.abs(Y - plain_network(layers, x)).max() < 1e-3
    ctx.close()


def test_lenet_conv1_full_size_sampled(mods):
    """BASELINE config 2 at the size bench.py times (N=2^14, 8+2 limbs, BS=128, S=4): two output ciphertexts of conv1 are
    recomputed by the oracle term by term (its inner rotations, 25 PMults, rescale) and compared limb by limb."""
    ck, fr, fenc = mods
    P, ctx = make(mods, "cfg2")
    conv_kw = dict(BS=128, C_in=1, H=28, W=28, C_out=6, K=5, stride=1, pad=2)
    x, w = wl.conv_inputs(2001, conv_kw, x_range=(0.0, 1.0))
    graph = fr.ConvGraph(fr.ConvDesc(S=4, **conv_kw), P.n)
    conv = ctx.conv_desc(S=4, **conv_kw)
    lay = ctx.layout_plan(conv)
    assert (lay.B, lay.ch, lay.n_in_ct, lay.n_out_ct, lay.n_inner_rot, lay.n_outer_rot, lay.n_pmult) == (128, 1, 16, 96, 48, 0, 2400)
    L = P.nq
    sample = [(0, 0, 0), (3, 2, 5)]  # (u_o, v_o, g_out): a border fragment and an interior one
    need = sorted({amt for ok_ in sample for lst in graph.terms[ok_].values() for _, amt, _ in lst if amt})
    gk = ctx.keygen(77, lay.steps())
    ok = ck.keygen(P, 77, need)
    keys7 = ctx.wts_keys(conv, lay)
    wanted = {wk for ok_ in sample for lst in graph.terms[ok_].values() for _, _, wk in lst}
    oW = {wk: ck.encode(P, graph.weight_slots(wk, w), L, P.q[L - 1]) for wk in wanted}
    o_in, g_in = {}, []
    for (u, v, g, bg) in graph.lin.ct_keys():
        pt = ck.encode(P, graph.lin.gather(x, u, v, g, bg), L)
        o_in[(u, v, g)] = ck.encrypt(P, ok, pt, 3000 + len(g_in))
        g_in.append(ctx.encrypt(gk, ctx.pt_from_coeffs(pt.coeffs, L, float(pt.scale)), 3000 + len(g_in)))
    # weights through the oracle's integers for the sampled outputs only: rebuild the full coefficient table
    coeffs = np.zeros((len(keys7), P.N), dtype=np.int64)
    for i, k in enumerate(keys7):
        wk = tuple(int(v) for v in k)
        if wk in oW:
            coeffs[i] = oW[wk].coeffs
    gW = ctx.conv_weights_from_coeffs(conv, lay, coeffs, L, float(P.q[L - 1]))
    g_out = ctx.hconv(gk, conv, lay, gW, g_in)
    for (uo, vo, go) in sample:
        acc = np.zeros((2, L, P.N), dtype=np.uint64)
        (d, lst), = graph.terms[(uo, vo, go)].items()
        assert d == 0
        for src, amt, wk in lst:
            xin = ck.rotate(P, ok, o_in[src], amt) if amt else o_in[src]
            ck.pmult_acc(P, acc, xin, oW[wk])
        ref = ck.rescale(P, ck.Ciphertext(acc, L, o_in[src].scale * oW[wk].scale))
        got = g_out[(go * 4 + uo) * 4 + vo]
        assert np.array_equal(ctx.ct_export(got), ref.c), (uo, vo, go)
    ctx.close()


# ------------------------------------------------------------------------------------------------ full-size properties (configs 3, 4)
def decoded_conv_error(mods, pkey, conv_kw, S, seed, kaiming=False, w_std=0.1, hoist=False):
    """Encrypted conv at a BASELINE parameter set through the library's own encoder; returns max |decoded - fp64 conv|.
    (The oracle needs minutes per output ciphertext at N=2^16, so full-size configs 3/4 are checked by this property,
    which holds at any size; their limbs are covered bit-exactly by the same graphs at reduced N above.)"""
    ck, fr, fenc = mods
    ctx = fenc.Context(**wl.PARAMS[pkey])
    ctx.set_hoisting(hoist)
    x, w = wl.conv_inputs(seed, conv_kw, kaiming=kaiming, w_std=w_std)
    conv = ctx.conv_desc(S=S, **conv_kw)
    lay = ctx.layout_plan(conv)
    L = ctx.n_q
    keys = ctx.keygen(seed, lay.steps())
    W = ctx.conv_weights(conv, lay, w, L)
    cts = []
    for bg in range(lay.BG):
        for g in range(lay.G_in):
            for u in range(lay.S):
                for v in range(lay.S):
                    cts.append(ctx.encrypt(keys, ctx.encode_fragment(conv, lay, x, u, v, g, bg, L), 9000 + len(cts)))
    outs = ctx.hconv(keys, conv, lay, W, cts)
    od = fr.ConvDesc(**conv_kw)
    Y = np.zeros((od.BS, od.C_out, od.H_out, od.W_out))
    i = 0
    for bg in range(lay.BG):
        for go in range(lay.G_out):
            for uo in range(lay.S_out):
                for vo in range(lay.S_out):
                    assert outs[i].L == L - 1
                    ctx.decrypt_decode(keys, outs[i], conv, lay, 1, uo, vo, go, bg, Y)
                    i += 1
    err = np.abs(Y - fr.direct_conv(od, x, w)).max()
    ctx.close()
    return err, lay


def test_config3_resnet_layers_full_size_decoded(mods):
    """BASELINE config 3 (N=2^16, 24x50b + 4x60b, dlen 4, scale 2^50): the three ResNet-20-shaped layers, BS=1."""
    err, lay = decoded_conv_error(mods, "cfg3", wl.CONVS["resnet_16_16"], 0, 301, kaiming=True)
    assert (lay.S, lay.n_in_ct, lay.n_out_ct, lay.n_inner_rot, lay.n_outer_rot, lay.n_pmult) == (1, 1, 1, 8, 30, 279)
    assert err < 1e-3
    err, lay = decoded_conv_error(mods, "cfg3", wl.CONVS["resnet_16_32_s2"], 2, 302, kaiming=True)
    assert (lay.n_in_ct, lay.n_out_ct, lay.n_inner_rot, lay.n_outer_rot, lay.n_pmult) == (4, 1, 5, 46, 423)
    assert err < 1e-3
    err, lay = decoded_conv_error(mods, "cfg3", wl.CONVS["resnet_32_64_s2"], 2, 303, kaiming=True)
    assert (lay.n_in_ct, lay.n_out_ct, lay.n_inner_rot, lay.n_outer_rot, lay.n_pmult) == (4, 1, 5, 94, 855)
    assert err < 1e-3


def test_config3_resnet_layer_full_size_hoisted_decoded(mods):
    """The configuration bench.py's cfg3 workloads time: inner rotations in the hoisted form (R2.7b) at N=2^16, wide
    fp64 butterflies, dlen 4 -- 8 rotations of one input ciphertext share one decomposition."""
    err, lay = decoded_conv_error(mods, "cfg3", wl.CONVS["resnet_16_16"], 0, 301, kaiming=True, hoist=True)
    assert (lay.n_inner_rot, lay.n_outer_rot) == (8, 30) and err < 1e-3
    err, lay = decoded_conv_error(mods, "cfg3", wl.CONVS["resnet_16_32_s2"], 2, 302, kaiming=True, hoist=True)
    assert err < 1e-3


def test_config4_mobilenet_layers_full_size_decoded(mods):
    """BASELINE config 4 (N=2^16, 30x50b + 5x60b, dlen 5): depthwise 3x3 and pointwise 1x1 at 112x112 (M=128, S=4)
    and the strided depthwise at 112 -> 56, batch 2 (the same kernels and graphs as the max-batch run, fewer groups)."""
    dw = dict(BS=2, C_in=32, H=112, W=112, C_out=32, K=3, stride=1, pad=1, depthwise=True)
    err, lay = decoded_conv_error(mods, "cfg4", dw, 4, 401, w_std=0.05)
    assert lay.M == 128 and lay.m == 32 and err < 1e-3
    pw = dict(BS=2, C_in=32, H=112, W=112, C_out=64, K=1, stride=1, pad=0)
    err, lay = decoded_conv_error(mods, "cfg4", pw, 4, 402, w_std=0.05)
    assert lay.n_inner_rot == 0 and err < 1e-3
    dws = dict(BS=2, C_in=64, H=112, W=112, C_out=64, K=3, stride=2, pad=1, depthwise=True)
    err, lay = decoded_conv_error(mods, "cfg4", dws, 4, 403, w_std=0.05)
    assert lay.S_out == 2 and lay.H_out == 56 and err < 1e-3


def test_cmult_scalar_poly3_bit_exact(mods):
    """a13: general CMult + relin + rescale, PMultConst, constant add and the degree-3 activation of config 3 (R2.12)."""
    ck, fr, fenc = mods
    from fractions import Fraction
    from paper_2606_16359_b200.pipeline import poly3_activation
    P, ctx = make(mods, "mid12")
    L = P.nq
    ok, gk = ck.keygen(P, 61, [], want_relin=True), ctx.keygen(61, [], want_relin=True)
    rng = np.random.default_rng(13)
    xs = [rng.uniform(-2, 2, P.n) for _ in range(3)]
    o_ct, g_ct = [], []
    for i, x in enumerate(xs):
        pt = ck.encode(P, x, L)
        o_ct.append(ck.encrypt(P, ok, pt, 300 + i))
        g_ct.append(ctx.encrypt(gk, ctx.pt_from_coeffs(pt.coeffs, L, float(pt.scale)), 300 + i))
    prod = ctx.cmult_relin(gk, g_ct[:2], g_ct[1:])
    for i in range(2):
        assert np.array_equal(ctx.ct_export(prod[i]), ck.cmult_relin(P, ok, o_ct[i], o_ct[i + 1]).c)
    k = ck.round_half_up(Fraction(197, 1000) * o_ct[0].scale ** 2)
    sc = ctx.mul_scalar(g_ct, k, float(o_ct[0].scale ** 2))
    ref = ck.mul_const(P, o_ct[2], Fraction(197, 1000), o_ct[2].scale ** 2)
    assert np.array_equal(ctx.ct_export(sc[2]), ref.c) and abs(sc[2].scale - float(ref.scale)) <= 1e-9 * float(ref.scale)
    assert np.array_equal(ctx.ct_export(ctx.add_const(g_ct, 12345678901)[1]), ck.add_const(P, o_ct[1], 12345678901).c)
    act, s3 = poly3_activation(ctx, gk, g_ct, o_ct[0].scale)
    for i, x in enumerate(xs):
        ref = ck.poly3(P, ok, o_ct[i])
        assert s3 == ref.scale and act[i].L == L - 2
        assert np.array_equal(ctx.ct_export(act[i]), ref.c), i
        assert np.abs(ctx.decrypt_slots(gk, act[i]).real - (0.5 + 0.197 * x - 0.004 * x ** 3)).max() < 1e-3
    ctx.close()


def test_config3_conv_plus_activation_full_size_decoded(mods):
    """config 3 at full size: conv 16->16 then the degree-3 activation, decoded against fp64 (property at any size)."""
    ck, fr, fenc = mods
    from paper_2606_16359_b200.pipeline import Pipeline
    ctx = fenc.Context(**wl.PARAMS["cfg3"])
    kw = wl.CONVS["resnet_16_16"]
    x, w = wl.conv_inputs(311, kw, kaiming=True)
    pipe = Pipeline(ctx, [{"op": "conv", "conv": dict(kw), "S": 1, "w": w}, {"op": "poly3"}])
    keys = pipe.setup(key_seed=311)
    out = pipe.forward(pipe.encrypt_input(x, 7000))
    p0 = pipe.plan[0]
    od = fr.ConvDesc(**kw)
    Y = np.zeros((1, 16, 32, 32))
    assert len(out) == 1 and out[0].L == ctx.n_q - 3
    ctx.decrypt_decode(keys, out[0], p0["conv"], p0["lay"], 1, 0, 0, 0, 0, Y)
    c = fr.direct_conv(od, x, w)
    assert np.abs(Y - (0.5 + 0.197 * c - 0.004 * c ** 3)).max() < 1e-3
    ctx.close()


def test_lenet5_full_size_bsgs_and_hoisting_decoded(mods):
    """BASELINE config 2 at the size and in the configuration bench.py times (batch 128, N=2^14, BSGS fully connected
    layers, inner rotations plain and hoisted): the decoded logits of all 128 samples against the fp64 network."""
    ck, fr, fenc = mods
    import bench
    from oracle import network as nw
    from paper_2606_16359_b200.pipeline import Pipeline
    from test_oracle_network import plain_network
    ctx = fenc.Context(**wl.PARAMS["cfg2"])
    layers, x = bench.lenet_layers(128, 2000)
    want = plain_network(layers, x)
    assert np.abs(want).max() < 0.5  # one 40-bit limb at scale 2^40 is left (A23)
    pipe = Pipeline(ctx, layers)
    keys = pipe.setup(key_seed=2000)
    cts = pipe.encrypt_input(x, 20000)
    fg = nw.FcGraph(ctx.n, **layers[-1]["fc"])
    got = {}
    for hoist, lazy in ((False, False), (True, False), (True, True)):
        ctx.set_hoisting(hoist)
        out = pipe.forward(cts, lazy_relin=lazy)
        assert len(out) == 1 and out[0].L == 1
        Y = np.zeros((128, 10))
        fg.scatter_out(Y, ctx.decrypt_slots(keys, out[0]).real, 0, 0)
        assert np.abs(Y - want).max() < 1e-3, (hoist, lazy)
        got[(hoist, lazy)] = Y
    assert np.abs(got[(True, False)] - got[(False, False)]).max() < 1e-4 and not np.array_equal(got[(True, False)], got[(False, False)])
    assert np.abs(got[(True, True)] - got[(True, False)]).max() < 1e-4 and not np.array_equal(got[(True, True)], got[(True, False)])
    n_lin, n_rot, n_relin, n_pm = pipe.counts()
    assert (n_lin, n_rot, n_relin) == (5, 367, 160)  # 48 + 192 conv rotations, 78 + 28 + 21 BSGS rotations (315 plain)
    assert pipe.counts(lazy_relin=True)[2] == 40      # 24 + 16 pooled outputs, one relinearisation each
    ctx.close()


_LENET_DIGEST = r"""
import sys, hashlib, json
sys.path.insert(0, %r)
import numpy as np, torch
import paper_2606_16359_b200 as fenc, workloads as wl, bench
from paper_2606_16359_b200.pipeline import Pipeline
ctx = fenc.Context(**wl.PARAMS["cfg2"])
layers, x = bench.lenet_layers(128, 2000)
pipe = Pipeline(ctx, layers)
pipe.setup(key_seed=2000)
cts = pipe.encrypt_input(x, 20000)
out = pipe.forward(cts)
h = hashlib.sha256()
for c in out:
    h.update(np.ascontiguousarray(ctx.ct_export(c)).tobytes())
print(json.dumps({"digest": h.hexdigest(), "n": len(out), "L": out[0].L}))
"""


@pytest.mark.gpu
def test_lenet_step_fp64_and_integer_arithmetic_agree():
    """The whole LeNet-5 step of bench.py (BASELINE config 2, batch 128, N=2^14) run twice in fresh processes: with the
    40-bit moduli on the FP64 pipe (default: butterflies, base conversions, MAC limbs) and with FENC_NO_F64=1 /
    FENC_MAC_MODE=0 (integer Shoup butterflies, 128-bit MAC).  Every limb of every output ciphertext must be identical:
    the fp64 path is an exact reformulation, and the integer path is the one the oracle-checked
    tests of the 50- and 58-bit parameter sets exercise."""
    import subprocess, sys, os, json
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    code = _LENET_DIGEST % root
    res = []
    for extra in ({}, {"FENC_NO_F64": "1", "FENC_MAC_MODE": "0"}):
        env = dict(os.environ, **extra)
        p = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, timeout=600)
        assert p.returncode == 0, p.stderr[-2000:]
        res.append(json.loads(p.stdout.strip().splitlines()[-1]))
    assert res[0] == res[1], res
    assert res[0]["n"] >= 1

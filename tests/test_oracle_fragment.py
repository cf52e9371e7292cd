"""Pins for oracle/fragment.py (CPU only): the paper's printed values (tests/golden/), its worked
examples, special cases, and direct fp64 convolution (Eq. 2)."""
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import ckks as ck
from oracle import fragment as fr
import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _table_ix():
    rows = []
    for line in open(os.path.join(GOLD, "table_ix_rot.txt")):
        if line.startswith("#") or not line.strip():
            continue
        rows.append(tuple(int(x) for x in line.split()))
    return rows


def _paper_values():
    out = {}
    for line in open(os.path.join(GOLD, "paper_values.txt")):
        line = line.split("#")[0].split()
        if line:
            out[line[0]] = [float(x) for x in line[1:]]
    return out


# ------------------------------------------------------------------ Table IX
def test_table_ix_closed_form_all_15_rows():
    n = 1 << 14  # N = 2^15
    for cin, cout, K, BS, H, W, S, rot in _table_ix():
        d = fr.ConvDesc(BS, cin, H, W, cout, K, 1, (K - 1) // 2, S=S)
        assert fr.paper_rot_count(d, n, S) == rot


def test_table_ix_exact_graph_counts():
    """The exact graph count equals the printed value when K > S, S | (K-1) and C_out >= ch (A6, A19);
    elsewhere it exceeds it by the edge term / the sparse-output term."""
    n = 1 << 14
    equal, differ = 0, 0
    for cin, cout, K, BS, H, W, S, rot in _table_ix():
        d = fr.ConvDesc(BS, cin, H, W, cout, K, 1, (K - 1) // 2, S=S)
        g = fr.ConvGraph(d, n)
        c = g.counts()
        tot = c["n_inner_rot"] + c["n_outer_rot"]
        if K > S and (K - 1) % S == 0 and cout >= g.lin.ch:
            assert tot == rot
            equal += 1
        else:
            assert tot >= rot
            differ += 1
        # exact closed forms of this graph (R2.9): inner per group of S^2 fragments = (K-1)(2S+K-1)
        assert c["n_inner_rot"] == (K - 1) * (2 * S + K - 1) * g.lin.G * g.lin.BG
        assert c["n_in_ct"] == cin * BS * 32 * 32 // n
    assert equal == 10 and differ == 5


def test_s_star_matches_printed_example():
    d = fr.ConvDesc(8, 128, 32, 32, 32, 9, 1, 4)
    assert abs(fr.s_star_real(d, 1 << 14) - _paper_values()["s_star_conv128_32_9_bs8"][0]) < 0.005
    # the measured optimum in Table IX for this shape is S = 4; so is the exact-count arg-min over its three sizes
    tot = {}
    for S in (2, 4, 8):
        c = fr.ConvGraph(fr.with_S(d, S), 1 << 14).counts()
        tot[S] = c["n_inner_rot"] + c["n_outer_rot"]
    assert min(tot, key=tot.get) == 4


# ------------------------------------------------------------------ Fig. 4 toy
def test_fig4_toy_rotation_profile():
    n = int(_paper_values()["fig4_slots"][0])
    prof = {}
    for S in (1, 2, 4):
        g = fr.ConvGraph(fr.ConvDesc(1, 16, 4, 4, 16, 3, 1, 1, S=S), n)
        c = g.counts()
        prof[S] = (c["n_inner_rot"], c["n_outer_rot"])
        assert g.lin.B * g.lin.ch * g.lin.m ** 2 == n and c["n_in_ct"] == 16  # fully packed, 16 ciphertexts
    assert prof[1][1] == 0 and prof[1][0] == 16 * 8       # S=1: no outer rotations, K^2-1 inner per ct
    assert prof[4][0] == 0 and prof[4][1] == 16 * 15      # S=M: no inner, maximal outer
    assert sum(prof[2]) < sum(prof[1]) and sum(prof[2]) < sum(prof[4])  # S=2 optimal
    assert fr.select_S(fr.ConvDesc(1, 16, 4, 4, 16, 3, 1, 1), n) == 2


# ------------------------------------------------------------------ Algorithm 1 layout
def test_layout_4x4_example():
    pv = _paper_values()
    X = np.arange(16, dtype=np.float64).reshape(1, 1, 4, 4) + 1
    l2 = fr.Layout(4, 4, 2, 1, 1)
    assert len(l2.ct_keys()) == pv["map4x4_S2_cts"][0]
    for (u, v, g, bg) in l2.ct_keys():
        vec = l2.gather(X, u, v, g, bg)
        assert np.count_nonzero(vec) == 4  # dense: 4 slots, 4 pixels
        assert list(vec) == [X[0, 0, bi * 2 + u, bj * 2 + v] for bi in range(2) for bj in range(2)]
    l4 = fr.Layout(4, 4, 4, 1, 1)
    assert len(l4.ct_keys()) == pv["map4x4_S4_cts"][0]
    assert all(np.count_nonzero(l4.gather(X, u, v, 0, 0)) == 1 for u in range(4) for v in range(4))  # 25 %


def test_layout_special_cases_and_round_trip():
    rng = np.random.default_rng(0)
    X = rng.uniform(-1, 1, (1, 4, 8, 8))
    # S = 1, BS = 1: row-major, channel after channel
    l1 = fr.Layout(256, 8, 1, 1, 4)
    assert np.array_equal(l1.gather(X, 0, 0, 0, 0), X.reshape(-1))
    # S = M: one pixel per ciphertext, channels along the slots
    lm = fr.Layout(4, 8, 8, 1, 4)
    assert np.array_equal(lm.gather(X, 3, 5, 0, 0), X[0, :, 3, 5])
    # batch first, then channels: slot index = cpos*cs + k*B + b
    Xb = rng.uniform(-1, 1, (3, 5, 6, 7))
    lb = fr.Layout(128, 8, 2, 3, 5)
    assert (lb.B, lb.ch, lb.G, lb.BG) == (4, 2, 3, 1)
    Y = np.zeros_like(Xb)
    for key in lb.ct_keys():
        lb.scatter(Y, lb.gather(Xb, *key), *key)
    assert np.array_equal(Y, Xb)
    v = lb.gather(Xb, 1, 0, 1, 0)
    assert v[lb.slot(1, 2 * 4 + 3, 2)] == Xb[2, 3, 2 * 2 + 1, 3 * 2 + 0]


# ------------------------------------------------------------------ the graph on plain slots vs Eq. 2
SHAPES = [
    # BS Cin H W Cout K s p dw S n
    (1, 16, 4, 4, 16, 3, 1, 1, False, 1, 16), (1, 16, 4, 4, 16, 3, 1, 1, False, 2, 16), (1, 16, 4, 4, 16, 3, 1, 1, False, 4, 16),
    (2, 4, 8, 8, 8, 3, 2, 1, False, 2, 64), (2, 4, 8, 8, 8, 3, 2, 1, False, 4, 64),
    (1, 8, 8, 8, 8, 3, 1, 1, True, 2, 128), (3, 8, 8, 8, 8, 3, 2, 1, True, 2, 128),
    (1, 8, 8, 8, 4, 1, 1, 0, False, 1, 128), (1, 2, 12, 12, 3, 5, 1, 0, False, 2, 256),
    (1, 1, 28, 28, 6, 5, 1, 2, False, 1, 4096), (1, 1, 28, 28, 6, 5, 1, 2, False, 2, 4096),
    (5, 3, 7, 6, 5, 3, 1, 1, False, 4, 32), (2, 6, 8, 8, 6, 2, 2, 0, True, 2, 64),
]


@pytest.mark.parametrize("shape", SHAPES)
def test_graph_on_slots_equals_direct_conv(shape):
    BS, Ci, H, W, Co, K, s, p, dw, S, n = shape
    rng = np.random.default_rng(hash(shape) % 2 ** 32)
    d = fr.ConvDesc(BS, Ci, H, W, Co, K, s, p, dw, S=S)
    X = rng.uniform(-1, 1, (BS, Ci, H, W))
    Kw = rng.normal(0, 0.1, (Co, 1 if dw else Ci, K, K))
    assert np.abs(fr.hconv_slots(d, n, X, Kw) - fr.direct_conv(d, X, Kw)).max() < 1e-12


def test_direct_conv_against_hand_example():
    # 1x1x3x3 input, 2x2 kernel, no padding: 4 outputs computed by hand
    X = np.arange(9, dtype=np.float64).reshape(1, 1, 3, 3)
    Kw = np.array([[[[1.0, 2.0], [3.0, 4.0]]]])
    Y = fr.direct_conv(fr.ConvDesc(1, 1, 3, 3, 1, 2), X, Kw)
    assert Y.reshape(-1).tolist() == [0 + 2 + 9 + 16, 1 + 4 + 12 + 20, 3 + 8 + 18 + 28, 4 + 10 + 21 + 32]


def test_lenet_conv1_counts_config1():
    d = fr.ConvDesc(1, 1, 28, 28, 6, 5, 1, 2)
    assert fr.select_S(d, 4096) == 1  # Eq. 7: sqrt(BS*C_in/alpha) = 0.5 < 1 -> smallest feasible
    c = fr.ConvGraph(fr.with_S(d, 1), 4096).counts()
    assert (c["n_in_ct"], c["n_out_ct"], c["n_inner_rot"], c["n_outer_rot"], c["n_pmult"]) == (1, 2, 24, 4, 150)
    assert len(c["rot_steps"]) == 27


# ------------------------------------------------------------------ encrypted HConv on the Fig. 4 toy (N = 32)
@pytest.fixture(scope="module")
def toy32():
    P = ck.Params(5, 3, 36, 1, 40, 3, 30)  # 16 slots, dlen = 1
    return P


@pytest.mark.parametrize("S", [1, 2, 4])
def test_encrypted_hconv_fig4(toy32, S):
    P = toy32
    rng = np.random.default_rng(S)
    d = fr.ConvDesc(1, 16, 4, 4, 16, 3, 1, 1, S=S)
    g = fr.ConvGraph(d, P.n)
    X = rng.uniform(-1, 1, (1, 16, 4, 4))
    Kw = rng.normal(0, 0.3, (16, 16, 3, 3))
    keys = ck.keygen(P, 5, g.counts()["rot_steps"])
    W = fr.encode_weights(ck, P, g, Kw, P.nq)
    ins = {}
    for i, (u, v, gi, bg) in enumerate(g.lin.ct_keys()):
        ins[(u, v, gi)] = ck.encrypt(P, keys, ck.encode(P, g.lin.gather(X, u, v, gi, bg), P.nq), 100 + i)
    outs = fr.hconv(ck, P, keys, g, ins, W)
    Y = np.zeros((1, 16, 4, 4))
    for (uo, vo, go), y in outs.items():
        assert y.L == P.nq - 1 and y.scale == P.scale
        g.lout.scatter(Y, ck.decrypt_decode(P, keys, y).real, uo, vo, go, 0)
    assert np.abs(Y - fr.direct_conv(d, X, Kw)).max() < 1e-3


# ------------------------------------------------------------------ AAC (Fig. 5)
def test_compress_fig5_shape(toy32):
    """8 -> 2 -> 8 bottleneck: 4 sources at 25 % (2 of 8 channel positions) -> 1 dense ciphertext;
    maskless adds no level; masked split-scale costs exactly the one rescale."""
    P = toy32
    n, ch, v = P.n, 8, 2
    cs = n // ch
    n_src = int(_paper_values()["fig5_sources"][0])
    plan = fr.compress_plan(n, ch, cs, v, n_src)
    assert len(plan) == 1 and len(plan[0]) == 4
    keys = ck.keygen(P, 9, [r for _, r in plan[0]])
    rng = np.random.default_rng(1)
    zs = []
    for i in range(n_src):
        z = np.zeros(n)
        z[: v * cs] = rng.uniform(-1, 1, v * cs)
        zs.append(z)
    exp = np.concatenate([z[: v * cs] for z in zs])  # segmented layout: seg*(v*cs) + cpos*cs + k*B + b
    srcs = [ck.encrypt(P, keys, ck.encode(P, z, P.nq), 50 + i) for i, z in enumerate(zs)]
    out = fr.compress(ck, P, keys, plan, srcs)[0]
    assert out.L == P.nq and out.scale == P.scale
    assert np.abs(ck.decrypt_decode(P, keys, out).real - exp).max() < 1e-4
    # masked: sources carry garbage outside the kept positions and sit at scale s*Delta1; mask at Delta2
    q = P.q[P.nq - 1]
    d1 = Fraction(2) ** ((q.bit_length() + 1) // 2)
    d2 = Fraction(q) / d1
    dirty = [z + np.concatenate([np.zeros(v * cs), rng.uniform(-1, 1, n - v * cs)]) for z in zs]
    srcs = [ck.encrypt(P, keys, ck.encode(P, z, P.nq, P.scale * d1), 60 + i) for i, z in enumerate(dirty)]
    mpt = ck.encode(P, fr.compress_mask(n, cs, v), P.nq, d2)
    out = fr.compress(ck, P, keys, plan, srcs, mask_pt=mpt, do_rescale=True)[0]
    assert out.L == P.nq - 1 and out.scale == P.scale
    assert np.abs(ck.decrypt_decode(P, keys, out).real - exp).max() < 1e-3


# --------------------------------------------------------------------------- factored weights (R2.9c)
FACTORED_SHAPES = [
    dict(BS=8, C_in=3, H=4, W=4, C_out=5, K=3, stride=1, pad=1),                    # n=128: m=4, B=8, ch=1
    dict(BS=16, C_in=2, H=7, W=6, C_out=3, K=3, stride=2, pad=1),                   # frame 8 > data, stride 2 (S=2)
    dict(BS=8, C_in=4, H=4, W=4, C_out=4, K=3, stride=1, pad=1, depthwise=True),
    dict(BS=8, C_in=5, H=4, W=4, C_out=7, K=1, stride=1, pad=0),                    # point-wise
    dict(BS=20, C_in=2, H=4, W=4, C_out=2, K=5, stride=1, pad=2),                   # BS not 2^k: 3 batch groups, last ragged
]


@pytest.mark.parametrize("kw", FACTORED_SHAPES)
def test_factored_weights_identity_and_plain_slots(kw):
    """R2.9c: (i) every weight plaintext of a ch = 1 layer equals value x mask exactly; (ii) the factored graph on plain slot
    vectors (rotation = cyclic shift) reproduces direct convolution."""
    n = 128
    S = 2 if kw["stride"] == 2 else 1
    d = fr.ConvDesc(S=S, **kw)
    g = fr.ConvGraph(d, n)
    assert g.lin.ch == 1 and g.factorable()
    x, w = wl.conv_inputs(7, kw)
    values, mask_of, masks = {}, {}, {}
    for diags in g.terms.values():
        for lst in diags.values():
            for _, _, wk in lst:
                v, mk = g.weight_factor(wk, w)
                assert np.array_equal(v * g.mask_slots(mk), g.weight_slots(wk, w))
                values[wk], mask_of[wk] = v, mk
                masks[mk] = g.mask_slots(mk)
    g.mask_of = mask_of
    be = fr.SlotBackend(n)
    Y = np.zeros((d.BS, d.C_out, d.H_out, d.W_out))
    for bg in range(g.lin.BG):
        ins = {(u, v, gi): g.lin.gather(x, u, v, gi, bg) for u in range(S) for v in range(S) for gi in range(g.lin.G)}
        for (uo, vo, go), y in g.run_factored(be, ins, values, masks).items():
            g.lout.scatter(Y, y, uo, vo, go, bg)
    assert np.abs(Y - fr.direct_conv(d, x, w)).max() < 1e-12


def test_factor_scales_split():
    """E1 E2 = s_w exactly, E1 a power of two of half the bits (Delta_1 Delta_2 = Delta)."""
    from fractions import Fraction
    for sw in (1099511480321, 1125899906826241, 2 ** 40, 2 ** 25):
        E1, E2 = fr.factor_scales(sw)
        assert E1 * E2 == sw and E1 == Fraction(2) ** ((int(sw - 1).bit_length() + 1) // 2)


def test_not_factorable_with_several_channel_positions():
    g = fr.ConvGraph(fr.ConvDesc(S=1, BS=1, C_in=4, H=4, W=4, C_out=4, K=3, stride=1, pad=1), 128)
    assert g.lin.ch > 1 and not g.factorable()


@pytest.mark.parametrize("kw,hoist", [(FACTORED_SHAPES[0], False), (FACTORED_SHAPES[1], True), (FACTORED_SHAPES[3], False)])
def test_factored_weights_encrypted_decodes_to_convolution(kw, hoist):
    """R2.9c on ciphertexts: decrypt(hconv_factored) = direct convolution within 1e-3; same level and scale as the plain
    form; the limbs differ from it (two roundings instead of one) while the decoded values agree to 1e-4."""
    P = ck.Params(8, 4, 40, 2, 60, 2, 40)
    L = P.nq
    S = 2 if kw["stride"] == 2 else 1
    d = fr.ConvDesc(S=S, **kw)
    g = fr.ConvGraph(d, P.n)
    x, w = wl.conv_inputs(8, kw)
    keys = ck.keygen(P, 3, g.counts()["rot_steps"])
    values, masks, E1 = fr.factor_weights(ck, P, g, w, L)
    E2 = next(iter(masks.values())).scale
    assert E1 * E2 == P.q[L - 1] and E1 == 2 ** 20
    W = fr.encode_weights(ck, P, g, w, L)
    Yf = np.zeros((d.BS, d.C_out, d.H_out, d.W_out))
    Yp = np.zeros_like(Yf)
    differ = False
    for bg in range(g.lin.BG):
        ins = {(u, v, gi): ck.encrypt(P, keys, ck.encode(P, g.lin.gather(x, u, v, gi, bg), L), 100 + 16 * bg + 4 * gi + 2 * u + v)
               for u in range(S) for v in range(S) for gi in range(g.lin.G)}
        of = fr.hconv_factored(ck, P, keys, g, ins, values, masks, E1, hoist=hoist)
        op = fr.hconv(ck, P, keys, g, ins, W, hoist=hoist)
        for k in of:
            assert of[k].L == op[k].L == L - 1 and of[k].scale == op[k].scale == P.scale
            differ = differ or not np.array_equal(of[k].c, op[k].c)
            g.lout.scatter(Yf, ck.decrypt_decode(P, keys, of[k]).real, *k, bg)
            g.lout.scatter(Yp, ck.decrypt_decode(P, keys, op[k]).real, *k, bg)
    want = fr.direct_conv(d, x, w)
    assert np.abs(Yf - want).max() < 1e-3 and np.abs(Yf - Yp).max() < 1e-4 and differ


# --------------------------------------------------------------------------- segmented layouts: the consumer of AAC's output (R2.11b)
SEG_CASES = [
    # (n, v, conv kwargs with B_cap): Fig. 5's shape 8 -> 2 -> 8: chp = 8, two valid channels, four sources per output
    (128, 2, dict(BS=4, C_in=2, H=4, W=4, C_out=8, K=3, stride=1, pad=1, B_cap=1)),
    (128, 2, dict(BS=7, C_in=2, H=4, W=4, C_out=5, K=1, stride=1, pad=0, B_cap=1)),      # ragged: 7 batch groups in 2 compressed ones, 5 channels
    (256, 4, dict(BS=16, C_in=3, H=4, W=4, C_out=8, K=3, stride=1, pad=1, B_cap=2)),     # B=2, chp=8, v=4 (3 of 4 positions used), 8 groups
    (256, 2, dict(BS=8, C_in=4, H=8, W=8, C_out=4, K=3, stride=2, pad=1, B_cap=4)),      # S=2: m=4, B=4, chp=4, two segments, two input groups
]


@pytest.mark.parametrize("n,v,kw", SEG_CASES)
def test_segmented_consumer_on_plain_slots(n, v, kw):
    """R2.11b: a convolution whose input (and output) ciphertexts are in the segmented layout AAC produces -- diagonal d
    as two partial sums rotated by d*cs and (d - v)*cs -- equals direct convolution, and the canonical compaction of
    plain-layout ciphertexts (R2.11) yields exactly that segmented layout."""
    S = 2 if kw["stride"] == 2 else 1
    d = fr.ConvDesc(S=S, seg_v=v, **kw)
    shape = {k: val for k, val in kw.items() if k != "B_cap"}
    x, w = wl.conv_inputs(11, shape)
    assert np.abs(fr.hconv_slots(d, n, x, w) - fr.direct_conv(d, x, w)).max() < 1e-12
    g = fr.ConvGraph(d, n)
    assert g.lin.seg > 1 and g.lin.ch == v
    # compress: plain-layout ciphertexts whose valid positions are [0, v) -> the segmented ciphertext (a rotation by r is
    # a left shift, np.roll by -r)
    plain = fr.Layout(n, g.M, S, kw["BS"], kw["C_in"], 0, kw["B_cap"])
    if plain.G == 1 and kw["C_in"] <= v:  # the reducing layer left at most v channels in one group: the canonical plan applies
        plan = fr.compress_plan(n, plain.chp, plain.cs, v, plain.BG)
        for (u, vv, gi, t) in g.lin.ct_keys():
            got = sum(np.roll(plain.gather(x, u, vv, 0, i), -r) for i, r in plan[t])
            assert np.array_equal(got, g.lin.gather(x, u, vv, gi, t))
    # rotation count: d = 0 plus two parts for each d in 1..v-1
    assert all(len([k for k in diags if g.diag_rot(k)]) <= 2 * (v - 1) for diags in g.terms.values())


def test_segmented_bottleneck_encrypted_fig5():
    """Fig. 5 end to end on ciphertexts: reduce 8 -> 2 channels (1x1), compress four 25 %-full
    ciphertexts into one, expand 2 -> 8 (3x3) on the segmented layout; decoded result = the two convolutions in fp64, and
    the expansion reads 1 input ciphertext per compressed group instead of 4."""
    P = ck.Params(8, 5, 40, 2, 60, 3, 40)
    n, L = P.n, P.nq
    red = dict(BS=4, C_in=8, H=4, W=4, C_out=2, K=1, stride=1, pad=0, B_cap=1)
    exp = dict(BS=4, C_in=2, H=4, W=4, C_out=8, K=3, stride=1, pad=1, B_cap=1)
    rng = np.random.default_rng(3)
    x = rng.uniform(-1, 1, (4, 8, 4, 4))
    w1, w2 = rng.normal(0, 0.3, (2, 8, 1, 1)), rng.normal(0, 0.3, (8, 2, 3, 3))
    g1 = fr.ConvGraph(fr.ConvDesc(S=1, **red), n)
    g2 = fr.ConvGraph(fr.ConvDesc(S=1, seg_v=2, **exp), n)
    assert (g1.lin.chp, g1.lin.BG, g2.lin.seg, g2.lin.BG, g2.lout.G) == (8, 4, 4, 1, 4)
    plan = fr.compress_plan(n, 8, g1.lin.cs, 2, 4)
    steps = set(g1.counts()["rot_steps"]) | set(g2.counts()["rot_steps"]) | {r for tl in plan for _, r in tl if r}
    keys = ck.keygen(P, 4, sorted(steps))
    W1, W2 = fr.encode_weights(ck, P, g1, w1, L), fr.encode_weights(ck, P, g2, w2, L - 1)
    mids = []
    for bg in range(4):
        ins = {(0, 0, gi): ck.encrypt(P, keys, ck.encode(P, g1.lin.gather(x, 0, 0, gi, bg), L), 40 + bg) for gi in range(g1.lin.G)}
        mids.append(fr.hconv(ck, P, keys, g1, ins, W1)[(0, 0, 0)])
    packed = fr.compress(ck, P, keys, plan, mids)
    assert len(packed) == 1 and packed[0].L == L - 1
    outs = fr.hconv(ck, P, keys, g2, {(0, 0, 0): packed[0]}, W2)
    Y = np.zeros((4, 8, 4, 4))
    for (uo, vo, go), y in outs.items():
        g2.lout.scatter(Y, ck.decrypt_decode(P, keys, y).real, uo, vo, go, 0)
    want = fr.direct_conv(fr.ConvDesc(**exp), fr.direct_conv(fr.ConvDesc(**red), x, w1), w2)
    assert sum(len(tl) for tl in plan) == 4 and len(outs) == 4  # 4 sparse ciphertexts -> 1 dense one -> 4 dense outputs
    assert np.abs(Y - want).max() < 1e-3


@pytest.mark.parametrize("S_src,S_dst,shape", [(2, 1, (1, 4, 4, 4)), (1, 2, (2, 2, 4, 4)), (2, 4, (1, 8, 7, 6))])
def test_repack_between_block_sizes_on_plain_slots(S_src, S_dst, shape):
    """R2.11c: the rot-mask-add plan between two block sizes moves every tensor entry to its slot in the
    other layout (gather in the source layout, repack, compare with the gather in the destination layout)."""
    n = 128
    BS, C, H, W = shape
    M = fr.next_pow2(max(H, W))
    src, dst = fr.Layout(n, M, S_src, BS, C), fr.Layout(n, M, S_dst, BS, C)
    x = np.random.default_rng(5).uniform(-1, 1, shape)
    plan = fr.repack_plan(src, dst, shape)
    vecs = {k: src.gather(x, *k) for k in src.ct_keys()}
    out = fr.repack_slots(plan, vecs)
    for k in dst.ct_keys():
        assert np.array_equal(out[k], dst.gather(x, *k))


def test_repack_encrypted_changes_block_size():
    """the same on ciphertexts: S = 2 -> S = 1 (four fragment ciphertexts into one), one level, decoded = the tensor"""
    P = ck.Params(7, 3, 40, 1, 60, 3, 40)
    shape = (1, 4, 4, 4)
    src, dst = fr.Layout(P.n, 4, 2, 1, 4), fr.Layout(P.n, 4, 1, 1, 4)
    x = np.random.default_rng(6).uniform(-1, 1, shape)
    plan = fr.repack_plan(src, dst, shape)
    steps = sorted({r for terms in plan.values() for _, r, _ in terms if r})
    keys = ck.keygen(P, 2, steps)
    cts = {k: ck.encrypt(P, keys, ck.encode(P, src.gather(x, *k), P.nq), 9 + i) for i, k in enumerate(src.ct_keys())}
    out = fr.repack(ck, P, keys, plan, cts, P.nq)
    assert len(out) == 1
    Y = np.zeros(shape)
    for k, y in out.items():
        assert y.L == P.nq - 1 and y.scale == P.scale
        dst.scatter(Y, ck.decrypt_decode(P, keys, y).real, *k)
    assert np.abs(Y - x).max() < 1e-4


# --------------------------------------------------------------------------- BSGS over the channel diagonals (R2.9d)
BSGS_SHAPES = [
    (128, dict(BS=1, C_in=8, H=4, W=4, C_out=8, K=3, stride=1, pad=1), 1),       # ch = 8, dense channels
    (128, dict(BS=1, C_in=5, H=4, W=4, C_out=7, K=3, stride=1, pad=1), 1),       # ragged channels
    (128, dict(BS=2, C_in=4, H=8, W=8, C_out=8, K=3, stride=2, pad=1), 2),       # S = 2, stride 2, two output groups
    (512, dict(BS=1, C_in=16, H=4, W=4, C_out=16, K=3, stride=1, pad=1), 1),     # ch = 32: the auto rule picks g > 1
    (512, dict(BS=3, C_in=6, H=4, W=4, C_out=9, K=1, stride=1, pad=0, B_cap=2), 1),  # 1x1, two batch groups, ch = 16
]


@pytest.mark.parametrize("n,kw,S", BSGS_SHAPES)
@pytest.mark.parametrize("g", [2, 4, 0])
def test_conv_bsgs_on_plain_slots_and_counts(n, kw, S, g):
    """R2.9d: the regrouped graph on plain slot vectors (rotation = cyclic shift) equals direct convolution; its rotation
    counts follow the closed form (every (input, amount) of the plain graph, the unrotated input included, appears with
    each of the g baby steps; one outer rotation per non-zero giant step that has a term); PMult count and weight keys are
    those of the plain graph; auto (0) never needs more rotations than plain or any explicit g."""
    shape = {k: v for k, v in kw.items() if k != "B_cap"}
    x, w = wl.conv_inputs(21, shape)
    plain = fr.ConvGraph(fr.ConvDesc(S=S, **kw), n)
    d = fr.ConvDesc(S=S, bsgs=g, **kw)
    G = fr.ConvGraph(d, n)
    assert np.abs(fr.hconv_slots(d, n, x, w) - fr.direct_conv(d, x, w)).max() < 1e-12
    cp, cg = plain.counts(), G.counts()
    assert cg["n_pmult"] == cp["n_pmult"] and cg["n_out_ct"] == cp["n_out_ct"]
    keys = lambda gr: sorted(wk for diags in gr.terms.values() for lst in diags.values() for _, _, wk in lst)
    assert keys(G) == keys(plain)
    gg = G.g
    assert gg == g or g == 0
    # closed form from the plain graph
    pairs = {(src, amt, dd % gg) for diags in plain.terms.values() for dd, lst in diags.items() for src, amt, _ in lst}
    inner = {(src, (amt + j * plain.lin.cs) % n) for src, amt, j in pairs} - {(src, 0) for src, _, _ in pairs}
    outer = sum(len({dd // gg for dd in diags} - {0}) for diags in plain.terms.values())
    assert cg["n_inner_rot"] == len(inner) * plain.lin.BG and cg["n_outer_rot"] == outer * plain.lin.BG
    if g == 0:
        tot = lambda c: c["n_inner_rot"] + c["n_outer_rot"]
        for other in (1, 2, 4):
            if plain.lin.ch % other == 0:
                assert tot(cg) <= tot(fr.ConvGraph(fr.ConvDesc(S=S, bsgs=other, **kw), n).counts())
    if n == 512 and kw["C_in"] == 16:
        assert (cp["n_inner_rot"], cp["n_outer_rot"]) == (8, 30)       # BASELINE config 3's 16 -> 16 layer has this profile
        if g == 0:
            assert G.g == 2 and (cg["n_inner_rot"], cg["n_outer_rot"]) == (17, 15)


def test_conv_bsgs_encrypted_decodes_and_differs_from_plain():
    """R2.9d on ciphertexts (hoisted inner rotations): decrypt = direct convolution within 1e-3, same level and scale as the
    plain graph; the limbs differ (other rotations, other key-switch noise) while the decoded values agree to 1e-4."""
    P = ck.Params(8, 4, 40, 2, 60, 2, 40)
    kw = dict(BS=1, C_in=8, H=4, W=4, C_out=8, K=3, stride=1, pad=1)
    x, w = wl.conv_inputs(22, kw)
    L = P.nq
    res = {}
    for g in (1, 2):
        d = fr.ConvDesc(S=1, bsgs=g, **kw)
        G = fr.ConvGraph(d, P.n)
        keys = ck.keygen(P, 5, G.counts()["rot_steps"])
        W = fr.encode_weights(ck, P, G, w, L)
        ins = {(0, 0, gi): ck.encrypt(P, keys, ck.encode(P, G.lin.gather(x, 0, 0, gi, 0), L), 70 + gi) for gi in range(G.lin.G)}
        out = fr.hconv(ck, P, keys, G, ins, W, hoist=True)
        Y = np.zeros((1, 8, 4, 4))
        for k, y in out.items():
            assert y.L == L - 1 and y.scale == P.scale
            G.lout.scatter(Y, ck.decrypt_decode(P, keys, y).real, *k, 0)
        res[g] = (Y, out)
    want = fr.direct_conv(fr.ConvDesc(**kw), x, w)
    assert np.abs(res[2][0] - want).max() < 1e-3 and np.abs(res[2][0] - res[1][0]).max() < 1e-4
    assert any(not np.array_equal(res[1][1][k].c, res[2][1][k].c) for k in res[1][1])


@pytest.mark.parametrize("n,v,kw", [(128, 2, dict(BS=4, C_in=2, H=4, W=4, C_out=8, K=3, stride=1, pad=1, B_cap=1)),
                                    (256, 4, dict(BS=16, C_in=3, H=4, W=4, C_out=8, K=3, stride=1, pad=1, B_cap=2)),
                                    (1024, 8, dict(BS=4, C_in=8, H=4, W=4, C_out=16, K=3, stride=1, pad=1, B_cap=1))])
@pytest.mark.parametrize("g", [2, 4, 0])
def test_conv_bsgs_on_segmented_layouts(n, v, kw, g):
    """R2.9d on the segmented layout of R2.11b: both parts of diagonal d = i g + j keep the baby step j; their giant
    rotations are i g cs and (i g - v) cs.  The graph on plain slot vectors equals direct convolution; explicit g halves
    (quarters) the outer rotations; auto never needs more rotations than plain."""
    if g > 1 and v % g:
        pytest.skip("g must divide the segment size")
    shape = {k: x for k, x in kw.items() if k != "B_cap"}
    x, w = wl.conv_inputs(23, shape)
    d = fr.ConvDesc(S=1, seg_v=v, bsgs=g, **kw)
    G = fr.ConvGraph(d, n)
    assert np.abs(fr.hconv_slots(d, n, x, w) - fr.direct_conv(d, x, w)).max() < 1e-12
    cp, cg = fr.ConvGraph(fr.ConvDesc(S=1, seg_v=v, **kw), n).counts(), G.counts()
    if g > 1:
        assert G.g == g and cg["n_outer_rot"] * g <= cp["n_outer_rot"] + cg["n_out_ct"] * g
    else:
        assert cg["n_inner_rot"] + cg["n_outer_rot"] <= cp["n_inner_rot"] + cp["n_outer_rot"]
    if n == 1024 and g == 0:
        assert G.g == 2 and (cp["n_outer_rot"], cg["n_outer_rot"]) == (28, 14)

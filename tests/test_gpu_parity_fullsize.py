"""GPU parity at BASELINE.json's full sizes, in the schedule and launch configuration bench.py times (-m gpu).

Each test runs the library call at its benchmarked size and compares SAMPLED output ciphertexts limb by limb with the CPU
oracle (tests/oracle_pool.py fans the oracle's independent rotations / partial sums out over worker processes).
Sampling a linear layer: every weight plaintext outside the sampled terms is given all-zero coefficients, so its product
and the rotation of an all-zero ciphertext are exactly zero on both sides and the sampled output equals the oracle's
evaluation of the sampled terms alone -- the full layer still runs on the GPU (same grids, same batches).
Inputs are ciphertexts with uniform-random limbs (BASELINE config 5's recipe): bit-exactness does not need a message;
the decoded <= 1e-3 checks of the same layers are in test_gpu_parity.py."""
from fractions import Fraction

import numpy as np
import pytest

import workloads as wl
from oracle_pool import job_mac, job_rotate, job_rotate_ct, pmap

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


def make(mods, p):
    ck, fr, fenc = mods
    P = ck.Params(*wl.oracle_params_args(p))
    ctx = fenc.Context(**p)
    assert ctx.q == P.q and ctx.p == P.p and ctx.dlen == P.dlen
    return P, ctx


def add_mod(P, a, b, L):
    out = np.empty_like(a)
    for t in range(L):
        out[:, t] = (a[:, t] + b[:, t]) % np.uint64(P.q[t])
    return out


def oracle_linear_sample(ck, P, ok, L, inputs, terms_by_diag, rot_of_diag, pts, hoist, s_in, s_w, chunk=12):
    """One output ciphertext of a linear layer (conv or fc) restricted to the given diagonals / giant steps (R2.9 steps
    1-6, R2.12b): inner rotations (hoisted form when `hoist`), PMult-accumulate per diagonal, outer rotation, sum, rescale.
    inputs: {src: Ciphertext}; terms_by_diag: {d: [(src, amt, wkey)]}; rot_of_diag: {d: outer amount}; pts: {wkey: Plaintext}."""
    need = sorted({(src, amt) for lst in terms_by_diag.values() for src, amt, _ in lst if amt})
    rot = pmap(dict(ck=ck, P=P, keys=ok, inputs=inputs), job_rotate, [(src, amt, hoist) for src, amt in need])
    cts = {("in", src): c for src, c in inputs.items()}
    for (src, amt), c in zip(need, rot):
        cts[(src, amt)] = ck.Ciphertext(c, L, s_in)
    diags = sorted(terms_by_diag)
    jobs, owner = [], []
    for d in diags:
        lst = [((src, amt) if amt else ("in", src), wk) for src, amt, wk in terms_by_diag[d]]
        for at in range(0, len(lst), chunk):
            jobs.append((lst[at:at + chunk],))
            owner.append(d)
    parts = pmap(dict(ck=ck, P=P, cts=cts, pts=pts), job_mac, jobs)
    acc = {}
    for d, a in zip(owner, parts):
        acc[d] = a if d not in acc else add_mod(P, acc[d], a, L)
    outer = [ck.Ciphertext(acc[d], L, s_in * s_w) for d in diags]
    rjobs = [(i, rot_of_diag[d]) for i, d in enumerate(diags) if rot_of_diag[d]]
    rres = pmap(dict(ck=ck, P=P, keys=ok, outer=outer), job_rotate_ct, rjobs)
    y = None
    it = iter(rres)
    for i, d in enumerate(diags):
        term = next(it) if rot_of_diag[d] else outer[i].c
        y = term if y is None else add_mod(P, y, term, L)
    return ck.rescale(P, ck.Ciphertext(y, L, s_in * s_w))


# ------------------------------------------------------------------------------------------------ config 2, benchmarked schedule
def test_cfg2_conv2_hoisted_full_size_sampled(mods):
    """BASELINE config 2, conv2 as bench.py runs it: N=2^14, L=6 (the level conv1 - x^2 - pool leaves), BS=128, S=2, 24 -> 64
    ciphertexts, 192 inner rotations in the HOISTED form (R2.7b), 9600 PMults in 20-bit-limb fp64 accumulation, one rescale.
    One output ciphertext (150 terms, 6 input channels x 25 taps) is recomputed by the oracle's hoisted variant."""
    ck, fr, fenc = mods
    P, ctx = make(mods, wl.PARAMS["cfg2"])
    L = 6
    conv_kw = dict(BS=128, C_in=6, H=14, W=14, C_out=16, K=5, stride=1, pad=0, M=16)
    graph = fr.ConvGraph(fr.ConvDesc(S=2, **conv_kw), P.n)
    conv = ctx.conv_desc(S=2, **conv_kw)
    lay = ctx.layout_plan(conv)
    assert (lay.B, lay.ch, lay.n_in_ct, lay.n_out_ct, lay.n_inner_rot, lay.n_outer_rot, lay.n_pmult) == (128, 1, 24, 64, 192, 0, 9600)
    okey = (1, 0, 5)  # (u_o, v_o, g_out)
    terms = graph.terms[okey]
    assert list(terms) == [0] and len(terms[0]) == 150
    _, w = wl.conv_inputs(2002, conv_kw)
    need = sorted({amt for _, amt, _ in terms[0] if amt})
    gk = ctx.keygen(78, lay.steps())
    ok = ck.keygen(P, 78, need)
    s_w = P.q[L - 1]
    oW = {wk: ck.encode(P, graph.weight_slots(wk, w), L, s_w) for _, _, wk in terms[0]}
    keys7 = ctx.wts_keys(conv, lay)
    coeffs = np.zeros((len(keys7), P.N), dtype=np.int64)
    for i, k in enumerate(keys7):
        wk = tuple(int(v) for v in k)
        if wk in oW:
            coeffs[i] = oW[wk].coeffs
    gW = ctx.conv_weights_from_coeffs(conv, lay, coeffs, L, float(s_w))
    del coeffs
    o_in, g_in = {}, []
    for (u, v, g, bg) in graph.lin.ct_keys():
        limbs = wl.random_ct_limbs(4000 + len(g_in), P.q, L, P.N)
        o_in[(u, v, g)] = ck.Ciphertext(limbs, L, P.scale)
        g_in.append(ctx.ct_import(limbs, float(P.scale)))
    ctx.set_hoisting(True)
    g_out = ctx.hconv(gk, conv, lay, gW, g_in)
    ref = oracle_linear_sample(ck, P, ok, L, o_in, terms, {0: 0}, oW, True, P.scale, s_w)
    uo, vo, go = okey
    got = g_out[(go * 2 + uo) * 2 + vo]
    assert got.L == L - 1 and np.array_equal(ctx.ct_export(got), ref.c)
    # an output none of whose terms was sampled is exactly the zero ciphertext
    assert not ctx.ct_export(g_out[0]).any()
    ctx.close()


def test_cfg2_square_sum_relin_full_size_sampled(mods):
    """BASELINE config 2's x^2 + pool after conv1 as bench.py runs it (R2.12c): ONE fenc_square_sum_relin call over 96
    ciphertexts at N=2^14, L=7 -> 24 pooled outputs with one merged ModDown + rescale each; two outputs against the oracle."""
    ck, fr, fenc = mods
    P, ctx = make(mods, wl.PARAMS["cfg2"])
    L = 7
    ok, gk = ck.keygen(P, 79, [], want_relin=True), ctx.keygen(79, [], want_relin=True)
    limbs = [wl.random_ct_limbs(5000 + i, P.q, L, P.N) for i in range(96)]
    got = ctx.square_sum_relin(gk, [ctx.ct_import(a, float(P.scale)) for a in limbs], 4)
    assert len(got) == 24
    for o in (0, 17):
        ref = ck.square_sum_relin(P, ok, [ck.Ciphertext(a, L, P.scale) for a in limbs[4 * o:4 * o + 4]])
        assert got[o].L == L - 1 and np.array_equal(ctx.ct_export(got[o]), ref.c), o
    ctx.close()


def test_cfg2_fc1_bsgs_hoisted_full_size_sampled(mods):
    """BASELINE config 2's fc1 (400 -> 120) as bench.py runs it: N=2^14, L=4, BS=128, 16 -> 2 ciphertexts, baby-step
    giant-step with the library's g (= 2: 16 hoisted baby rotations, 31 giant rotations per output).  Output 1 restricted
    to three giant steps (0, 5, 31) against the oracle."""
    ck, fr, fenc = mods
    from oracle import network as nw
    P, ctx = make(mods, wl.PARAMS["cfg2"])
    L = 4
    kw = dict(BS=128, n_in=400, n_out=120, in_C=16, in_H=5, in_W=5, in_M=8, bsgs=0)
    g = nw.FcGraph(P.n, **kw)
    fcd = ctx.fc_desc(**kw)
    info = ctx.fc_plan(fcd)
    c = g.counts()
    assert {k: info[k] for k in c} == c and info["bsgs"] == 2 and info["n_rot"] == 78
    co, giants = 1, (0, 5, 31)
    W = np.random.default_rng(2003).normal(0, 0.1, (120, 400))
    s_w = P.q[L - 1]
    terms = {i: [(ci, j * g.B % P.n, wk) for ci, j, wk in g.terms[co][i]] for i in giants}
    oW = {wk: ck.encode(P, g.weight_slots(wk, W), L, s_w) for lst in terms.values() for _, _, wk in lst}
    keys3 = ctx.fc_wts_keys(fcd)
    coeffs = np.zeros((len(keys3), P.N), dtype=np.int64)
    for i, k in enumerate(keys3):
        wk = tuple(int(v) for v in k)
        if wk in oW:
            coeffs[i] = oW[wk].coeffs
    gW = ctx.fc_weights_from_coeffs(fcd, coeffs, L, float(s_w))
    del coeffs
    rot_of = {i: i * g.g * g.B % P.n for i in giants}
    need = sorted({amt for lst in terms.values() for _, amt, _ in lst if amt} | {r for r in rot_of.values() if r})
    gk, ok = ctx.keygen(80, c["rot_steps"]), ck.keygen(P, 80, need)
    o_in, g_in = {}, []
    for ci in range(g.n_in_ct):
        limbs = wl.random_ct_limbs(6000 + ci, P.q, L, P.N)
        o_in[ci] = ck.Ciphertext(limbs, L, P.scale)
        g_in.append(ctx.ct_import(limbs, float(P.scale)))
    ctx.set_hoisting(True)
    g_out = ctx.fc(gk, fcd, gW, g_in)
    ref = oracle_linear_sample(ck, P, ok, L, o_in, terms, rot_of, oW, True, P.scale, s_w)
    assert g_out[co].L == L - 1 and np.array_equal(ctx.ct_export(g_out[co]), ref.c)
    assert not ctx.ct_export(g_out[0]).any()
    ctx.close()


# ------------------------------------------------------------------------------------------------ config 3 at N = 2^16
def test_cfg3_resnet_16_16_full_size_sampled(mods):
    """BASELINE config 3's 3x3 16 -> 16 layer at full size (N=2^16, 24x50b + 4x60b, dlen 4, S=1: 1 -> 1 ciphertext, 8 hoisted
    inner + 30 outer rotations, 279 PMults): the 26-bit-limb MAC and the wide fp64 butterflies inside a convolution.  The
    output restricted to channel diagonals 0 and 7 (18 PMults, 8 hoisted + 1 plain rotation, rescale) against the oracle."""
    ck, fr, fenc = mods
    P, ctx = make(mods, wl.PARAMS["cfg3"])
    L = P.nq
    conv_kw = wl.CONVS["resnet_16_16"]
    graph = fr.ConvGraph(fr.ConvDesc(S=1, **conv_kw), P.n)
    conv = ctx.conv_desc(S=1, **conv_kw)
    lay = ctx.layout_plan(conv)
    assert (lay.n_in_ct, lay.n_out_ct, lay.n_inner_rot, lay.n_outer_rot, lay.n_pmult) == (1, 1, 8, 30, 279)
    okey, diags = (0, 0, 0), (0, 7)
    terms = {d: graph.terms[okey][d] for d in diags}
    _, w = wl.conv_inputs(304, conv_kw, kaiming=True)
    s_w = P.q[L - 1]
    oW = {wk: ck.encode(P, graph.weight_slots(wk, w), L, s_w) for lst in terms.values() for _, _, wk in lst}
    rot_of = {d: d * graph.lin.cs % P.n for d in diags}
    need = sorted({amt for lst in terms.values() for _, amt, _ in lst if amt} | {r for r in rot_of.values() if r})
    gk, ok = ctx.keygen(81, lay.steps()), ck.keygen(P, 81, need)
    keys7 = ctx.wts_keys(conv, lay)
    coeffs = np.zeros((len(keys7), P.N), dtype=np.int64)
    for i, k in enumerate(keys7):
        wk = tuple(int(v) for v in k)
        if wk in oW:
            coeffs[i] = oW[wk].coeffs
    gW = ctx.conv_weights_from_coeffs(conv, lay, coeffs, L, float(s_w))
    limbs = wl.random_ct_limbs(7000, P.q, L, P.N)
    o_in = {(0, 0, 0): ck.Ciphertext(limbs, L, P.scale)}
    ctx.set_hoisting(True)
    g_out = ctx.hconv(gk, conv, lay, gW, [ctx.ct_import(limbs, float(P.scale))])
    ref = oracle_linear_sample(ck, P, ok, L, o_in, terms, rot_of, oW, True, P.scale, s_w, chunk=3)
    assert g_out[0].L == L - 1 and np.array_equal(ctx.ct_export(g_out[0]), ref.c)
    ctx.close()


def test_cfg3_resnet_16_16_bsgs_full_size_sampled(mods):
    """The same layer with baby-step giant-step over its channel diagonals (R2.9d; the auto rule picks g = 2: 17 hoisted
    inner + 15 outer rotations instead of 8 + 30) at full size: the output restricted to giant steps 0 and 5 (36 PMults
    with shifted weight plaintexts, 17 composite hoisted rotations, one outer rotation, rescale) against the oracle."""
    ck, fr, fenc = mods
    P, ctx = make(mods, wl.PARAMS["cfg3"])
    L = P.nq
    conv_kw = dict(wl.CONVS["resnet_16_16"], bsgs=0)
    graph = fr.ConvGraph(fr.ConvDesc(S=1, **conv_kw), P.n)
    conv = ctx.conv_desc(S=1, **conv_kw)
    lay = ctx.layout_plan(conv)
    assert graph.g == 2 and (lay.n_in_ct, lay.n_out_ct, lay.n_inner_rot, lay.n_outer_rot, lay.n_pmult) == (1, 1, 17, 15, 279)
    assert lay.steps() == graph.counts()["rot_steps"]
    okey, giants = (0, 0, 0), (0, 5)
    terms = {i: graph.terms[okey][i] for i in giants}
    _, w = wl.conv_inputs(305, wl.CONVS["resnet_16_16"], kaiming=True)
    s_w = P.q[L - 1]
    oW = {wk: ck.encode(P, graph.weight_slots(wk, w), L, s_w) for lst in terms.values() for _, _, wk in lst}
    rot_of = {i: graph.diag_rot(i) for i in giants}
    need = sorted({amt for lst in terms.values() for _, amt, _ in lst if amt} | {r for r in rot_of.values() if r})
    gk, ok = ctx.keygen(82, lay.steps()), ck.keygen(P, 82, need)
    keys7 = ctx.wts_keys(conv, lay)
    coeffs = np.zeros((len(keys7), P.N), dtype=np.int64)
    for i, k in enumerate(keys7):
        wk = tuple(int(v) for v in k)
        if wk in oW:
            coeffs[i] = oW[wk].coeffs
    gW = ctx.conv_weights_from_coeffs(conv, lay, coeffs, L, float(s_w))
    limbs = wl.random_ct_limbs(7001, P.q, L, P.N)
    o_in = {(0, 0, 0): ck.Ciphertext(limbs, L, P.scale)}
    ctx.set_hoisting(True)
    g_out = ctx.hconv(gk, conv, lay, gW, [ctx.ct_import(limbs, float(P.scale))])
    ref = oracle_linear_sample(ck, P, ok, L, o_in, terms, rot_of, oW, True, P.scale, s_w, chunk=3)
    assert g_out[0].L == L - 1 and np.array_equal(ctx.ct_export(g_out[0]), ref.c)
    ctx.close()


# ------------------------------------------------------------------------------------------------ config 5 paths
def test_transformer_linear_fragment_embeddings_full_size_sampled(mods):
    """bench.py's `ext_transformer_linear` (R2.13) in its launch configuration: N=2^16, 24x50b +
    4x60b, 128 tokens, 768 -> 768 on fragment-encoded embeddings (S = S' = 3: 3 -> 3 ciphertexts, E / S = P = 256), the
    library's g = 16 (45 hoisted baby rotations + 45 giant rotations instead of 765), hoisted.  Output ciphertext 2 restricted
    to giant steps 0 and 7 and, inside each, to the baby steps 0, 3 and 15 of all three inputs (18 PMults, 6 hoisted + 1
    plain rotation, rescale) against the oracle; the other outputs (all-zero weights) are zero."""
    ck, fr, fenc = mods
    from oracle import network as nw
    P, ctx = make(mods, wl.PARAMS["cfg3"])
    L = P.nq
    kw = dict(BS=128, n_in=768, n_out=768, in_M=1, frag_in=3, frag_out=3, bsgs=0)
    g = nw.FcGraph(P.n, **kw)
    fcd = ctx.fc_desc(**kw)
    info = ctx.fc_plan(fcd)
    c = g.counts()
    assert {k: info[k] for k in c} == c and info["bsgs"] == 16 and info["n_rot"] == 90 and info["n_pmult"] == 2304
    assert nw.FcGraph(P.n, **dict(kw, bsgs=1)).counts()["n_rot"] == 3 * (768 // 3 - 1)  # the paper's E/S - 1 per output ciphertext
    co, giants, babies = 2, (0, 7), (0, 3, 15)
    W = np.random.default_rng(2013).normal(0, 768 ** -0.5, (768, 768))
    s_w = P.q[L - 1]
    terms = {i: [(ci, j * g.B % P.n, wk) for ci, j, wk in g.terms[co][i] if j in babies] for i in giants}
    assert all(len(lst) == 9 for lst in terms.values())
    oW = {wk: ck.encode(P, g.weight_slots(wk, W), L, s_w) for lst in terms.values() for _, _, wk in lst}
    keys3 = ctx.fc_wts_keys(fcd)
    coeffs = np.zeros((len(keys3), P.N), dtype=np.int64)
    for i, k in enumerate(keys3):
        wk = tuple(int(v) for v in k)
        if wk in oW:
            coeffs[i] = oW[wk].coeffs
    gW = ctx.fc_weights_from_coeffs(fcd, coeffs, L, float(s_w))
    del coeffs
    rot_of = {i: i * g.g * g.B % P.n for i in giants}
    need = sorted({amt for lst in terms.values() for _, amt, _ in lst if amt} | {r for r in rot_of.values() if r})
    gk, ok = ctx.keygen(81, c["rot_steps"]), ck.keygen(P, 81, need)
    o_in, g_in = {}, []
    for ci in range(g.n_in_ct):
        limbs = wl.random_ct_limbs(6100 + ci, P.q, L, P.N)
        o_in[ci] = ck.Ciphertext(limbs, L, P.scale)
        g_in.append(ctx.ct_import(limbs, float(P.scale)))
    ctx.set_hoisting(True)
    g_out = ctx.fc(gk, fcd, gW, g_in)
    ref = oracle_linear_sample(ck, P, ok, L, o_in, terms, rot_of, oW, True, P.scale, s_w)
    assert g_out[co].L == L - 1 and np.array_equal(ctx.ct_export(g_out[co]), ref.c)
    assert not ctx.ct_export(g_out[0]).any() and not ctx.ct_export(g_out[1]).any()
    ctx.close()


@pytest.mark.parametrize("n_q,n_p,dnum", [(6, 6, 1), (8, 8, 1), (18, 9, 2), (12, 12, 1), (16, 16, 1), (24, 24, 1), (24, 12, 2), (26, 26, 1), (30, 30, 1)])
def test_rotation_wide_and_unfused_digits(mods, n_q, n_p, dnum):
    """Config 5's widest digits at N=2^12 (same kernels, 4 column tiles per limb): dlen 6, 8, 9 run the fused column kernel
    with 2 thread groups per block, dlen 12, 16, 24 with 4 thread groups sharing up to 24 source tiles; dlen 26 and 30 exceed its shared memory and take the
    unfused inverse / base-conversion pair (the path of the L=36, dnum=1 point).  Top level and one level down (short
    digit), 50-bit ciphertext primes, 60-bit special primes (A2)."""
    ck, fr, fenc = mods
    P, ctx = make(mods, dict(log2N=12, n_q=n_q, q_bits=50, n_p=n_p, p_bits=60, dnum=dnum, log2_scale=50))
    steps = [5, P.n - 3]
    ok, gk = ck.keygen(P, 10, steps), ctx.keygen(10, steps)
    for L in (P.nq, P.nq - 1):
        limbs = wl.random_ct_limbs(200 + L, P.q, L, P.N)
        gin = ctx.ct_import(limbs)
        outs = ctx.rotate(gk, [gin, gin, gin], steps + [5])
        refs = pmap(dict(ck=ck, P=P, keys=ok, inputs={0: ck.Ciphertext(limbs, L, 1)}), job_rotate, [(0, r, False) for r in steps])
        for r, o, ref in zip(steps + [5], outs, refs + refs[:1]):
            assert np.array_equal(ctx.ct_export(o), ref), (L, r)
    ctx.close()


def test_more_targets_than_staged_descriptors(mods):
    """60 ciphertext limbs, digits of 6 (N=2^12): a ModUp group has 60 targets and a rescale 59, more than the 56 target
    descriptors the fused column kernel stages in shared memory (CONV_DESC_CAP) -- the targets past the cap take their
    descriptors and constants from global memory.  A batch of five rotations (slab row passes: batches of four and more)
    and a batched rescale against the oracle, limb by limb."""
    ck, fr, fenc = mods
    P, ctx = make(mods, dict(log2N=12, n_q=60, q_bits=50, n_p=6, p_bits=60, dnum=10, log2_scale=50))
    assert P.nq + len(P.p) - P.dlen > 56
    steps = [3, P.n - 7]
    ok, gk = ck.keygen(P, 11, steps), ctx.keygen(11, steps)
    L = P.nq
    limbs = [wl.random_ct_limbs(260 + i, P.q, L, P.N) for i in range(2)]
    gin = [ctx.ct_import(a) for a in limbs]
    outs = ctx.rotate(gk, [gin[0], gin[1], gin[0], gin[1], gin[0]], [3, 3, P.n - 7, P.n - 7, 3])
    jobs = [(0, 3, False), (1, 3, False), (0, P.n - 7, False), (1, P.n - 7, False)]
    refs = pmap(dict(ck=ck, P=P, keys=ok, inputs={i: ck.Ciphertext(a, L, 1) for i, a in enumerate(limbs)}), job_rotate, jobs)
    for o, ref in zip(outs, refs + refs[:1]):
        assert np.array_equal(ctx.ct_export(o), ref)
    res = ctx.rescale(outs[:4])
    for o, ref in zip(res, refs):
        assert o.L == L - 1 and np.array_equal(ctx.ct_export(o), ck.rescale(P, ck.Ciphertext(ref, L, 2.0 ** 50)).c)
    ctx.close()


def test_rotation_config5_L36_dnum1_full_size(mods):
    """Config 5's largest point, N=2^16, L=36, dnum=1 (k = dlen = 36, 72 moduli): one rotation out of a batch of three
    checked fully against the oracle (unfused key switch: 36 source limbs do not fit the fused column kernel)."""
    ck, fr, fenc = mods
    P, ctx = make(mods, wl.sweep_params(36, 1))
    assert ctx.dlen == 36 and ctx.beta_max == 1
    steps = [12345]
    ok, gk = ck.keygen(P, 11, steps), ctx.keygen(11, steps)
    limbs = [wl.random_ct_limbs(300 + i, P.q, 36, P.N) for i in range(3)]
    outs = ctx.rotate(gk, [ctx.ct_import(a) for a in limbs], steps * 3)
    ref = ck.rotate(P, ok, ck.Ciphertext(limbs[1], 36, 1), 12345)
    assert np.array_equal(ctx.ct_export(outs[1]), ref.c)
    ctx.close()


# ------------------------------------------------------------------------------------------------ config 4 (factored weights, R2.9c)
def oracle_factored_sample(ck, P, ok, L, graph, inputs, okey, values, masks, E1, hoist):
    """One output ciphertext of a factored layer (R2.9c) from the oracle: hoisted inner rotations in worker processes,
    S_mu = sum_t round_half_up(v_t E1) . R_t per mask, acc = sum_mu S_mu (*) M_mu, rescale.  (ch = 1: diagonal 0 only.)"""
    (d, lst), = graph.terms[okey].items()
    assert d == 0
    need = sorted({(src, amt) for src, amt, _ in lst if amt})
    rot = pmap(dict(ck=ck, P=P, keys=ok, inputs=inputs), job_rotate, [(src, amt, hoist) for src, amt in need])
    R = {k: ck.Ciphertext(c, L, inputs[k[0]].scale) for k, c in zip(need, rot)}
    by_mask = {}
    for src, amt, wk in lst:
        by_mask.setdefault(graph.mask_of[wk], []).append((src, amt, wk))
    acc = np.zeros((2, L, P.N), dtype=np.uint64)
    s_in = next(iter(inputs.values())).scale
    for mk, tl in by_mask.items():
        S = None
        for src, amt, wk in tl:
            t = ck.mul_const(P, R[(src, amt)] if amt else inputs[src], values[wk], E1)
            S = t if S is None else ck.add(P, S, t)
        ck.pmult_acc(P, acc, S, masks[mk])
    return ck.rescale(P, ck.Ciphertext(acc, L, s_in * E1 * masks[mk].scale))


def factored_sampled_layer(mods, P, ctx, conv_kw, S, L, okey, seed, hoist=True):
    """Run one factored layer at full size on the GPU with every multiplier outside output `okey` set to zero, and compare
    that output with the oracle; another output must be exactly the zero ciphertext."""
    ck, fr, fenc = mods
    graph = fr.ConvGraph(fr.ConvDesc(S=S, **conv_kw), P.n)
    conv = ctx.conv_desc(S=S, **conv_kw)
    lay = ctx.layout_plan(conv)
    assert lay.ch == 1 and lay.n_outer_rot == 0
    cw = 1 if conv_kw.get("depthwise") else conv_kw["C_in"]
    w = np.random.default_rng(seed).normal(0, 0.05, (conv_kw["C_out"], cw, conv_kw["K"], conv_kw["K"]))
    values, masks, E1 = fr.factor_weights(ck, P, graph, w, L)
    E2 = next(iter(masks.values())).scale
    keys = [tuple(int(v) for v in k) for k in ctx.wts_keys(conv, lay)]
    mask_of, n_masks = ctx.wts_factors(conv, lay)
    by_id = {}
    for wk, mid in zip(keys, mask_of):
        assert by_id.setdefault(int(mid), graph.mask_of[wk]) == graph.mask_of[wk]
    assert n_masks == len(masks) == len(by_id)
    sampled = {wk for _, _, wk in graph.terms[okey][0]}
    k = np.array([ck.round_half_up(Fraction(values[wk]) * E1) if wk in sampled else 0 for wk in keys], dtype=np.int64)
    assert np.count_nonzero(k) == len(sampled)
    mc = np.stack([masks[by_id[i]].coeffs for i in range(n_masks)])
    gW = ctx.conv_weights_factored_from_ints(conv, lay, k, mc, L, float(E1), float(E2))
    need = sorted({amt for _, amt, _ in graph.terms[okey][0] if amt})
    gk, ok = ctx.keygen(90 + seed, lay.steps()), ck.keygen(P, 90 + seed, need)
    o_in, g_in = {}, []
    for (u, v, g, bg) in graph.lin.ct_keys():
        limbs = wl.random_ct_limbs(8000 + len(g_in), P.q, L, P.N)
        o_in[(u, v, g)] = ck.Ciphertext(limbs, L, P.scale)
        g_in.append(ctx.ct_import(limbs, float(P.scale)))
    ctx.set_hoisting(hoist)
    g_out = ctx.hconv(gk, conv, lay, gW, g_in)
    uo, vo, go = okey
    So = graph.S_out
    got = g_out[(go * So + uo) * So + vo]
    ref = oracle_factored_sample(ck, P, ok, L, graph, o_in, okey, values, masks, E1, hoist)
    assert got.L == L - 1 and np.array_equal(ctx.ct_export(got), ref.c)
    other = g_out[0] if (go, uo, vo) != (0, 0, 0) else g_out[1]
    assert not ctx.ct_export(other).any()


def test_cfg4_conv1_factored_full_size_sampled(mods):
    """BASELINE config 4's first layer as bench.py runs it: conv 3 -> 32, 3x3, stride 2, 224 x 224 in a 256 frame, S = 8,
    BS = 32 (B = 32, ch = 1), N=2^16, L=30, dlen 5: 192 -> 512 ciphertexts, 51 hoisted inner rotations, 13824 scalar
    multiply-accumulates on the FP64 pipe, masks for the frame and the zero padding.  One border output against the oracle."""
    P, ctx = make(mods, wl.PARAMS["cfg4"])
    kw = dict(BS=32, C_in=3, H=224, W=224, C_out=32, K=3, stride=2, pad=1)
    factored_sampled_layer(mods, P, ctx, kw, 8, 30, (0, 0, 5), seed=1)
    ctx.close()


def test_cfg4_pointwise_factored_full_size_sampled(mods):
    """BASELINE config 4's last layer: pointwise 64 -> 128 at 56 x 56 (frame 64, S = 2), BS = 32, L=26: 256 -> 512
    ciphertexts, no rotation at all, 32768 scalar multiply-accumulates in groups of 8 outputs, one mask product each."""
    P, ctx = make(mods, wl.PARAMS["cfg4"])
    kw = dict(BS=32, C_in=64, H=56, W=56, C_out=128, K=1, stride=1, pad=0)
    factored_sampled_layer(mods, P, ctx, kw, 2, 26, (1, 0, 77), seed=2)
    ctx.close()


def test_cfg4_mobilenet_chain_full_size_decoded(mods):
    """The whole config-4 step of bench.py for one batch group of 32 images (five chained layers, levels 30 -> 25, factored
    weights, hoisted rotations): sampled output ciphertexts decrypt to the fp64 evaluation of the same five convolutions
    within 1e-3 (north_star's decoded bar)."""
    ck, fr, fenc = mods
    import bench
    from paper_2606_16359_b200.pipeline import Pipeline
    ctx = fenc.Context(**wl.PARAMS["cfg4"])
    ctx.set_hoisting(True)
    layers, x = bench.mobilenet_layers(32, 2004)
    pipe = Pipeline(ctx, layers)
    keys = pipe.setup(key_seed=2004)
    out = pipe.forward(pipe.encrypt_input(x, 30000))
    assert len(out) == 512 and out[0].L == 25
    want = x
    for ly in layers:
        want = fr.direct_conv(fr.ConvDesc(**ly["conv"]), want, ly["w"])
    assert want.shape == (32, 128, 56, 56)
    p = pipe.plan[-1]
    Y = np.full(want.shape, np.nan)
    for go, uo, vo in ((0, 0, 0), (127, 1, 1), (64, 0, 1), (31, 1, 0)):
        ctx.decrypt_decode(keys, out[(go * 2 + uo) * 2 + vo], p["conv"], p["lay"], 1, uo, vo, go, 0, Y)
    seen = ~np.isnan(Y)
    assert seen.sum() == 4 * 32 * 28 * 28
    assert np.abs(Y[seen] - want[seen]).max() < 1e-3
    ctx.close()


def test_bottleneck_aac_full_size_decoded(mods):
    """bench.py's Table-X-shaped bottleneck at config 3's parameters (N=2^16): reduce 64 -> 8 (1x1), compress the four
    requests' 25 %-full ciphertexts into one, expand 8 -> 128 (3x3) on the segmented layout; with and without compression
    the decoded outputs equal the two convolutions in fp64 within 1e-3; compression halves the PMults and saves rotations."""
    ck, fr, fenc = mods
    import bench
    from paper_2606_16359_b200.pipeline import Pipeline
    res = {}
    for aac in (False, True):
        ctx = fenc.Context(**wl.PARAMS["cfg3"])
        ctx.set_hoisting(True)
        layers, x = bench.bottleneck_layers(77, aac)
        pipe = Pipeline(ctx, layers)
        keys = pipe.setup(key_seed=77)
        out = pipe.forward(pipe.encrypt_input(x, 40000))
        convs = [ly for ly in layers if ly["op"] == "conv"]
        want = x
        for ly in convs:
            want = fr.direct_conv(fr.ConvDesc(**{k: v for k, v in ly["conv"].items() if k not in ("seg_v", "B_cap")}), want, ly["w"])
        p = pipe.plan[-1]
        lay = p["lay"]
        assert len(out) == lay.n_out_ct == (16 if aac else 16) and out[0].L == ctx.n_q - 2
        Y = np.full(want.shape, np.nan)
        for i in (0, len(out) // 2, len(out) - 1):
            bg, go = divmod(i, lay.G_out)
            ctx.decrypt_decode(keys, out[i], p["conv"], lay, 1, 0, 0, go, bg, Y)
        seen = ~np.isnan(Y)
        assert seen.any() and np.abs(Y[seen] - want[seen]).max() < 1e-3
        res[aac] = pipe.counts()
        ctx.close()
    # compression halves the PMults; with baby-step giant-step on both chains (bench.py's default) it still saves rotations
    assert res[True][3] < 0.6 * res[False][3] and res[True][1] < res[False][1]

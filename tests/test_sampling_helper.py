"""CPU check of the sampling argument the full-size GPU parity tests rest on (tests/test_gpu_parity_fullsize.py): with
all-zero plaintexts outside the sampled diagonals, the oracle's full layer equals its evaluation of the sampled terms
alone (an all-zero product, and the rotation of an all-zero ciphertext, are exactly zero)."""
import numpy as np

import workloads as wl
from oracle import ckks as ck
from oracle import fragment as fr
from test_gpu_parity_fullsize import oracle_linear_sample


def test_sampled_evaluation_equals_full_layer_with_zeroed_weights():
    p = dict(log2N=7, n_q=4, q_bits=40, n_p=2, p_bits=60, dnum=2, log2_scale=40)
    P = ck.Params(*wl.oracle_params_args(p))
    L = P.nq
    conv_kw = dict(BS=1, C_in=4, H=4, W=4, C_out=4, K=3, stride=1, pad=1)
    graph = fr.ConvGraph(fr.ConvDesc(S=1, **conv_kw), P.n)
    assert graph.lin.ch == 4
    okey, diags = (0, 0, 0), (0, 2)
    _, w = wl.conv_inputs(1, conv_kw)
    c = graph.counts()
    ok = ck.keygen(P, 5, c["rot_steps"])
    s_w = P.q[L - 1]
    full = fr.encode_weights(ck, P, graph, w, L)
    sampled = {wk for d in diags for _, _, wk in graph.terms[okey][d]}
    zero = ck.encode(P, np.zeros(P.n), L, s_w)
    oW = {wk: (pt if wk in sampled else zero) for wk, pt in full.items()}
    limbs = wl.random_ct_limbs(3, P.q, L, P.N)
    o_in = {(0, 0, 0): ck.Ciphertext(limbs, L, P.scale)}
    for hoist in (False, True):
        want = fr.hconv(ck, P, ok, graph, o_in, oW, hoist=hoist)[okey]
        terms = {d: graph.terms[okey][d] for d in diags}
        rot_of = {d: d * graph.lin.cs % P.n for d in diags}
        got = oracle_linear_sample(ck, P, ok, L, o_in, terms, rot_of, oW, hoist, P.scale, s_w, chunk=2)
        assert np.array_equal(got.c, want.c) and got.scale == want.scale and got.L == want.L

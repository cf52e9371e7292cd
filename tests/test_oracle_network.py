"""Pins for oracle/network.py (CPU only): the FC-by-diagonals graph against a dense fp64 product, pooling by fragment
selection against a direct sum-pool through Algorithm 1's layout, and an encrypted toy network against its fp64
evaluation.  None of these re-uses the code under test to produce the expected value."""
import numpy as np
import pytest

from oracle import ckks as ck
from oracle import fragment as fr
from oracle import network as nw


@pytest.mark.parametrize("kw", [
    dict(n=256, BS=2, n_in=32, n_out=5, in_C=2, in_H=4, in_W=4, in_M=4),      # conv-layout input, one output ct
    dict(n=256, BS=5, n_in=3 * 3 * 3, n_out=70, in_C=3, in_H=3, in_W=3, in_M=4),  # ragged frame, BS not 2^k, 2 output cts
    dict(n=64, BS=40, n_in=10, n_out=7, in_M=2),                               # flat input, several batch groups (B=16)
    dict(n=64, BS=16, n_in=9, n_out=6, in_M=2),                                # B = 16, P = 4: 3 input cts, 2 output cts
])
def test_fc_graph_equals_dense_product(kw):
    kw = dict(kw)
    n = kw.pop("n")
    g = nw.FcGraph(n, **kw)
    rng = np.random.default_rng(3)
    X = rng.uniform(-1, 1, (kw["BS"], kw["n_in"]))
    W = rng.normal(0, 1, (kw["n_out"], kw["n_in"]))
    assert np.abs(nw.fc_slots(g, X, W) - X @ W.T).max() < 1e-12
    c = g.counts()
    # every existing non-zero diagonal costs one rotation per output ciphertext; d*B are the amounts
    assert c["n_rot"] == g.BG * sum(len([d for d in diags if d]) for diags in g.terms.values())
    assert all(s % g.B == 0 and 0 < s < n for s in c["rot_steps"])


@pytest.mark.parametrize("bsgs", [2, 4, 0])
@pytest.mark.parametrize("kw", [
    dict(n=256, BS=2, n_in=32, n_out=5, in_C=2, in_H=4, in_W=4, in_M=4),
    dict(n=256, BS=5, n_in=3 * 3 * 3, n_out=70, in_C=3, in_H=3, in_W=3, in_M=4),
    dict(n=64, BS=40, n_in=10, n_out=7, in_M=2),
    dict(n=64, BS=16, n_in=9, n_out=6, in_M=2),
    dict(n=512, BS=8, n_in=150, n_out=120, in_M=2),                            # dense: P = 64, 3 input cts, 2 output cts
])
def test_fc_bsgs_equals_dense_product(kw, bsgs):
    """R2.12b: the baby-step giant-step regrouping computes the same product (pre-rotated diagonals, baby rotations on
    the inputs, giant rotations on the sums), with the rotation count of the closed form on a dense layer."""
    kw = dict(kw)
    n = kw.pop("n")
    g = nw.FcGraph(n, bsgs=bsgs, **kw)
    plain = nw.FcGraph(n, **kw)
    rng = np.random.default_rng(4)
    X = rng.uniform(-1, 1, (kw["BS"], kw["n_in"]))
    W = rng.normal(0, 1, (kw["n_out"], kw["n_in"]))
    assert np.abs(nw.fc_slots(g, X, W) - X @ W.T).max() < 1e-12
    c, cp = g.counts(), plain.counts()
    assert c["n_pmult"] == cp["n_pmult"] and c["bsgs"] == g.g and g.P % g.g == 0
    assert c["n_rot"] <= g.BG * (g.n_in_ct * (g.g - 1) + g.n_out_ct * (g.P // g.g - 1))
    if kw["n_in"] == 150:  # dense: every (input ct, baby step) and (output ct, giant step) exists
        assert c["n_rot"] == g.BG * (g.n_in_ct * (g.g - 1) + g.n_out_ct * (g.P // g.g - 1))
        if bsgs == 0:  # 3 (g-1) + 2 (64/g - 1): g = 4 -> 39, g = 8 -> 35, g = 16 -> 51
            assert g.g == 8 and c["n_rot"] == 35 and cp["n_rot"] == 2 * 63


def test_bsgs_auto_rule():
    # LeNet-5 (config 2, P = 64): 16 -> 2, 2 -> 2, 2 -> 1 ciphertexts; ties go to the smaller g
    assert nw.bsgs_auto(64, 16, 2) == 2 and 16 * 1 + 2 * 31 == 78 == 16 * 3 + 2 * 15
    assert nw.bsgs_auto(64, 2, 2) == 8 and nw.bsgs_auto(64, 2, 1) == 4  # 2*3 + 15 == 2*7 + 7 == 21
    assert nw.bsgs_auto(1, 3, 3) == 1


def test_fc_conv_layout_matches_torch_flatten_order():
    # feat(c, p) must be channel*H*W + h*W + w: gather a tensor through Algorithm 1's S=1 layout and compare
    n, BS, C, H, W_, M = 256, 2, 3, 3, 4, 4
    g = nw.FcGraph(n, BS, C * H * W_, 4, in_C=C, in_H=H, in_W=W_, in_M=M)
    lay = fr.Layout(n, M, 1, BS, C)
    X = np.random.default_rng(1).uniform(-1, 1, (BS, C, H, W_))
    for c in range(g.n_in_ct):
        assert np.array_equal(g.gather_in(X.reshape(BS, -1), c, 0), lay.gather(X, 0, 0, c, 0))


def test_pool_order_is_sum_pool_through_the_layout():
    n, BS, C, H, M, S = 128, 2, 3, 8, 8, 4
    X = np.random.default_rng(2).uniform(-1, 1, (BS, C, H, H))
    lin = fr.Layout(n, M, S, BS, C)
    vecs = [lin.gather(X, u, v, g, bg) for (u, v, g, bg) in lin.ct_keys()]
    order = nw.pool_order(len(vecs), S)
    pooled = [sum(vecs[i] for i in order[k:k + 4]) for k in range(0, len(order), 4)]
    Xs = X.reshape(BS, C, H // 2, 2, H // 2, 2).sum(axis=(3, 5))  # direct 2x2 sum-pool
    lout = fr.Layout(n, M // 2, S // 2, BS, C)
    want = [lout.gather(Xs, u, v, g, bg) for (u, v, g, bg) in lout.ct_keys()]
    assert len(pooled) == len(want)
    for a, b in zip(pooled, want):
        assert np.abs(a - b).max() < 1e-12


def toy_network(BS=2, seed=5, bsgs=1):
    rng = np.random.default_rng(seed)
    layers = [
        {"op": "conv", "conv": dict(BS=BS, C_in=1, H=8, W=8, C_out=2, K=3, stride=1, pad=1), "S": 2, "w": rng.normal(0, 0.3, (2, 1, 3, 3))},
        {"op": "square"}, {"op": "pool"},
        {"op": "fc", "fc": dict(BS=BS, n_in=32, n_out=5, in_C=2, in_H=4, in_W=4, in_M=4, bsgs=bsgs), "w": rng.normal(0, 0.3, (5, 32)) * 0.25},
        {"op": "fc", "fc": dict(BS=BS, n_in=5, n_out=3, in_M=4, bsgs=bsgs), "w": rng.normal(0, 0.3, (3, 5))},
    ]
    x = rng.uniform(0, 1, (BS, 1, 8, 8))
    return layers, x


def plain_network(layers, x):
    """fp64 evaluation of the same function (pool = SUM pool; its 1/4 is already inside the next weights)."""
    for ly in layers:
        if ly["op"] == "conv":
            x = fr.direct_conv(fr.ConvDesc(**ly["conv"]), x, ly["w"])
        elif ly["op"] == "square":
            x = x * x
        elif ly["op"] == "pool":
            b, c, h, w = x.shape
            x = x.reshape(b, c, h // 2, 2, w // 2, 2).sum(axis=(3, 5))
        elif ly["op"] == "fc":
            x = x.reshape(x.shape[0], -1) @ ly["w"].T
    return x


@pytest.mark.parametrize("bsgs,hoist,lazy", [(1, False, False), (0, False, False), (0, True, False), (0, True, True)])
def test_encrypted_toy_network_matches_fp64(bsgs, hoist, lazy):
    P = ck.Params(9, 5, 40, 2, 60, 3, 40)
    layers, x = toy_network(bsgs=bsgs)
    steps, relin = nw.network_rot_steps(layers, P.n)
    keys = ck.keygen(P, 11, steps, want_relin=relin)
    lin = fr.Layout(P.n, 8, 2, 2, 1)
    cts = [ck.encrypt(P, keys, ck.encode(P, lin.gather(x, u, v, g, bg), P.nq), 100 + i)
           for i, (u, v, g, bg) in enumerate(lin.ct_keys())]
    out, trace = nw.run_network(ck, P, keys, layers, cts, P.nq, hoist=hoist, lazy_relin=lazy)
    assert len(trace) == len(layers)
    assert len(out) == 1 and out[0].L == 1
    g = nw.FcGraph(P.n, **layers[-1]["fc"])
    Y = np.zeros((2, 3))
    g.scatter_out(Y, ck.decrypt_decode(P, keys, out[0]).real, 0, 0)
    want = plain_network(layers, x)
    assert np.abs(want).max() < 0.45  # a single 40-bit limb at scale 2^40 holds |value| < 0.5 (A23)
    assert np.abs(Y - want).max() < 1e-4


def test_cmult_and_poly3_against_fp64():
    """CMult+relin+rescale decodes to the slot-wise product; the degree-3 activation of BASELINE config 3 decodes to
    0.5 + 0.197 x - 0.004 x^3 (R2.12) and consumes exactly two levels."""
    P = ck.Params(9, 4, 40, 2, 60, 2, 40)
    keys = ck.keygen(P, 21, [], want_relin=True)
    rng = np.random.default_rng(8)
    x, y = rng.uniform(-2, 2, P.n), rng.uniform(-1, 1, P.n)
    cx = ck.encrypt(P, keys, ck.encode(P, x, P.nq), 1)
    cy = ck.encrypt(P, keys, ck.encode(P, y, P.nq), 2)
    prod = ck.cmult_relin(P, keys, cx, cy)
    assert prod.L == P.nq - 1 and np.abs(ck.decrypt_decode(P, keys, prod).real - x * y).max() < 1e-6
    assert np.array_equal(ck.cmult_relin(P, keys, cx, cx).c, ck.square_relin(P, keys, cx).c)  # x^2 is the case y = x
    act = ck.poly3(P, keys, cx)
    assert act.L == P.nq - 2
    want = 0.5 + 0.197 * x - 0.004 * x ** 3
    assert np.abs(ck.decrypt_decode(P, keys, act).real - want).max() < 1e-6
    # PMultConst / add_const closed forms: times the integer 3 at E = 1 triples the slots; adding round(s/4) adds 0.25
    tri = ck.mul_const(P, cx, 3, 1)
    assert np.abs(ck.decrypt_decode(P, keys, tri).real - 3 * x).max() < 1e-6
    quarter = ck.add_const(P, cx, ck.round_half_up(cx.scale / 4))
    assert np.abs(ck.decrypt_decode(P, keys, quarter).real - (x + 0.25)).max() < 1e-6


# --------------------------------------------------------------------------- fragment-encoded embeddings (R2.13)
@pytest.mark.parametrize("n,BS,E,Eo,M,S,So,g", [
    (64, 4, 24, 24, 4, 3, 3, 1),      # E/S = 8 sub-blocks in P = 16 positions (not aligned), plain diagonals
    (64, 8, 16, 32, 2, 2, 4, 0),      # E = S P exactly; another fragment count on the output side; auto BSGS
    (128, 16, 20, 12, 2, 4, 2, 2),    # ragged: 20 = 4 * 5 coordinates in P = 8 positions
    (256, 8, 96, 96, 4, 3, 3, 0),     # a fragment count that is not a power of two (96 = 3 * 32)
    (256, 20, 64, 64, 4, 4, 4, 4),    # 20 tokens: two batch groups (B = 16), the second ragged
])
def test_fragment_encoded_matmul_on_plain_slots(n, BS, E, Eo, M, S, So, g):
    """R2.13: token embeddings split in E/S sub-blocks across S ciphertexts (coordinate e = p S + u in ciphertext u at
    position p); X W^T by the diagonal graph on plain slot vectors equals the dense product; gather / scatter are inverse."""
    rng = np.random.default_rng(31)
    G = nw.FcGraph(n, BS, E, Eo, in_M=M, bsgs=g, frag_in=S, frag_out=So)
    assert (G.n_in_ct, G.n_out_ct) == (S, So)
    X, W = rng.uniform(-1, 1, (BS, E)), rng.normal(0, 0.3, (Eo, E))
    assert np.abs(nw.fc_slots(G, X, W) - X @ W.T).max() < 1e-12
    # the layout itself: coordinate e of token b sits in ciphertext e mod S at position e // S
    v = G.gather_in(X, 1 % S, 0)
    for b in (0, min(BS, G.B) - 1):
        for p in range(-(-E // S)):
            e = p * S + 1 % S
            assert v[p * G.B + b] == (X[b, e] if e < E else 0.0)


def test_fragment_encoding_rotation_count_matches_the_papers_claim():
    """"the number of rotations required for embedding aggregation is reduced from E-1 in full-embedding
    packing to E/S - 1 under fragmented encoding".  With E = S P and plain diagonals the graph needs exactly P - 1 = E/S - 1
    rotations per output ciphertext; full-embedding packing (S = 1, P = E positions) needs E - 1."""
    n, E = 512, 64
    for S, M in ((1, 8), (4, 4), (16, 2)):   # P = M^2 = E / S positions, B = n / P tokens per ciphertext
        P = M * M
        assert S * P == E
        G = nw.FcGraph(n, n // P, E, E, in_M=M, frag_in=S, frag_out=S)
        assert G.P == P and G.counts()["n_rot"] == S * (P - 1) == S * (E // S - 1)
    # and BSGS on top of the fragments (R2.12b) lowers it further
    G = nw.FcGraph(n, n // 16, E, E, in_M=4, frag_in=4, frag_out=4, bsgs=0)
    assert G.counts()["n_rot"] < 4 * 15


def test_fragment_encoded_matmul_encrypted():
    """the same on ciphertexts (hoisted baby steps): decrypt = X W^T within 1e-3, one level"""
    P = ck.Params(8, 4, 40, 2, 60, 2, 40)
    rng = np.random.default_rng(32)
    G = nw.FcGraph(P.n, 8, 48, 48, in_M=4, bsgs=0, frag_in=3, frag_out=3)
    X, W = rng.uniform(-1, 1, (8, 48)), rng.normal(0, 0.2, (48, 48))
    keys = ck.keygen(P, 8, G.counts()["rot_steps"])
    Wp = nw.encode_fc_weights(ck, P, G, W, P.nq)
    ins = [ck.encrypt(P, keys, ck.encode(P, G.gather_in(X, c, 0), P.nq), 90 + c) for c in range(3)]
    outs = nw.fc(ck, P, keys, G, ins, Wp, hoist=True)
    Y = np.zeros((8, 48))
    for c, y in enumerate(outs):
        assert y.L == P.nq - 1
        G.scatter_out(Y, ck.decrypt_decode(P, keys, y).real, c, 0)
    assert np.abs(Y - X @ W.T).max() < 1e-3

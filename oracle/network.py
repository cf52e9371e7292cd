"""Layer-level oracle: FC by plain diagonals, square activation, 2x2 pooling by fragment selection, and a sequential
network runner.  TEST INFRASTRUCTURE ONLY -- see oracle/__init__.py.

Follows PAPER.md:284 ("stride is implemented simply by discarding the unused cts ... FC layers use diagonal-matrix
multiplication", polynomial activation) with the readings R2.12 of DESIGN.md section 4.  As in oracle/fragment.py each
graph runs (i) on plain slot vectors (rotation = cyclic shift), which pins it against a dense fp64 evaluation, and
(ii) on oracle ciphertexts (oracle/ckks.py).
"""
from fractions import Fraction

import numpy as np

from . import fragment as fr


# --------------------------------------------------------------------------- FC by plain diagonals (R2.12)
def bsgs_auto(P, n_in_ct, n_out_ct):
    """baby-step count g (a power of two dividing P) with the fewest rotations n_in_ct (g-1) + n_out_ct (P/g - 1) of a
    dense layer; ties go to the smaller g (R2.12b)."""
    best, g = None, 1
    while g <= P:
        cost = n_in_ct * (g - 1) + n_out_ct * (P // g - 1)
        if best is None or cost < best[0]:
            best = (cost, g)
        g *= 2
    return best[1]


class FcGraph:
    """Position p = cpos*m^2 + k in [0, P), P = n/B.  Input feature <-> (input ct c, p); neuron nu <-> (output ct c', p),
    nu = c'*P + p.  out_{c'} = sum_d Rot(sum_c x_c (*) Wd(c', c, d), d*B), Wd(c', c, d)[p] = W[nu(c', (p-d) mod P), feat(c, p)]
    or 0 when either index is invalid; terms whose Wd is identically zero are skipped.

    Baby-step giant-step ("diagonal-matrix multiplication with BSGS"; R2.12b): with g baby steps a diagonal
    is d = i g + j, 0 <= j < g, and since Rot(x (*) w, r) = Rot(x, r) (*) Rot(w, r),
        out_{c'} = sum_i Rot( sum_j sum_c Rot(x_c, j B) (*) W'(c', c, d), i g B ),   W'(c', c, d) = Rot(Wd(c', c, d), j B),
    i.e. W'(c', c, d)[p] = W[nu(c', (p - i g) mod P), feat(c, (p + j) mod P)].  The baby rotations Rot(x_c, j B) are
    computed once per input ciphertext and shared by every output and giant step.  bsgs = 1: plain diagonals (no baby
    rotation, W' = Wd); bsgs = 0: g = bsgs_auto(P, n_in_ct, n_out_ct).

    Fragment-encoded embeddings (R2.13, the Transformer extension): BS is the number of tokens, a token's
    embedding of dimension E is split in E/S sub-blocks of S coordinates, and coordinate e = p S + u of every token lives
    in ciphertext u (the fragment, 0 <= u < S) at position p -- "fragments from different tokens are interleaved across
    ciphertexts".  frag_in = S: feat(c, p) = p S + c with S input ciphertexts; frag_out = S': neuron(c', p) = p S' + c'
    with S' output ciphertexts.  X W^T is then this same graph; with E = S P its embedding aggregation costs P - 1 = E/S - 1
    rotations per output ciphertext instead of the E - 1 of full-embedding packing."""

    def __init__(self, n, BS, n_in, n_out, in_C=0, in_H=0, in_W=0, in_M=1, bsgs=1, frag_in=0, frag_out=0):
        self.frag_in, self.frag_out = frag_in, frag_out
        self.n, self.BS, self.n_in, self.n_out = n, BS, n_in, n_out
        self.in_C, self.in_H, self.in_W, self.m = in_C, in_H, in_W, in_M
        m2 = in_M * in_M
        assert m2 <= n and n % m2 == 0
        self.B = min(fr.next_pow2(BS), n // m2)
        self.P = n // self.B
        self.ch = n // (self.B * m2)
        self.BG = -(-BS // self.B)
        if frag_in:
            assert not in_C and -(-n_in // frag_in) <= self.P, "E/S sub-blocks must fit the positions of a ciphertext"
            self.n_in_ct = frag_in
        elif in_C:
            assert in_C * in_H * in_W == n_in
            self.n_in_ct = -(-in_C // self.ch)
        else:
            self.n_in_ct = -(-n_in // self.P)
        if frag_out:
            assert -(-n_out // frag_out) <= self.P
            self.n_out_ct = frag_out
        else:
            self.n_out_ct = -(-n_out // self.P)
        self.g = bsgs if bsgs >= 1 else bsgs_auto(self.P, self.n_in_ct, self.n_out_ct)
        assert self.P % self.g == 0
        self.terms = {}  # c' -> {giant step i: [(c, baby step j, wkey (c', c, d = i g + j))]}
        for co in range(self.n_out_ct):
            giants = {}
            for i in range(self.P // self.g):
                lst = [(ci, j, (co, ci, i * self.g + j)) for j in range(self.g) for ci in range(self.n_in_ct)
                       if self.nonzero(co, ci, i * self.g + j)]
                if lst:
                    giants[i] = lst
            self.terms[co] = giants

    def feat(self, c, p):
        """PyTorch flatten order channel*H*W + h*W + w through the S=1 layout, or c*P + p after a previous fc."""
        if self.frag_in:
            f = p * self.frag_in + c
            return f if f < self.n_in else -1
        if self.in_C:
            m2 = self.m * self.m
            cpos, k = divmod(p, m2)
            chan, (h, w) = c * self.ch + cpos, divmod(k, self.m)
            if chan >= self.in_C or h >= self.in_H or w >= self.in_W:
                return -1
            return (chan * self.in_H + h) * self.in_W + w
        f = c * self.P + p
        return f if f < self.n_in else -1

    def neuron(self, c, p):
        v = p * self.frag_out + c if self.frag_out else c * self.P + p
        return v if v < self.n_out else -1

    def nonzero(self, co, ci, d):
        return any(self.feat(ci, p) >= 0 and self.neuron(co, (p - d) % self.P) >= 0 for p in range(self.P))

    def weight_slots(self, wkey, W):
        co, ci, d = wkey
        j = d % self.g
        vec = np.zeros(self.n)
        for p in range(self.P):
            f, v = self.feat(ci, (p + j) % self.P), self.neuron(co, (p + j - d) % self.P)
            if f >= 0 and v >= 0:
                vec[p * self.B:(p + 1) * self.B] = W[v, f]
        return vec

    def baby_steps(self):
        """distinct (input ct, j != 0) pairs some term uses"""
        return sorted({(ci, j) for giants in self.terms.values() for lst in giants.values() for ci, j, _ in lst if j})

    def counts(self):
        n_giant = sum(len([i for i in giants if i]) for giants in self.terms.values())
        n_rot = n_giant + len(self.baby_steps())
        n_pm = sum(len(lst) for giants in self.terms.values() for lst in giants.values())
        steps = {i * self.g * self.B % self.n for giants in self.terms.values() for i in giants if i}
        steps |= {j * self.B % self.n for _, j in self.baby_steps()}
        return dict(n_in_ct=self.n_in_ct * self.BG, n_out_ct=self.n_out_ct * self.BG, n_rot=n_rot * self.BG,
                    n_pmult=n_pm * self.BG, n_distinct_pt=n_pm, rot_steps=sorted(steps), bsgs=self.g)

    def run(self, be, inputs, weights):
        """inputs: list of n_in_ct items of ONE batch group; returns list of n_out_ct items."""
        baby = {(ci, j): be.rot_in(inputs[ci], j * self.B % self.n) for ci, j in self.baby_steps()}
        out = []
        for co in range(self.n_out_ct):
            y = None
            for i in sorted(self.terms[co]):
                acc = be.zero()
                for ci, j, wkey in self.terms[co][i]:
                    be.pmult_acc(acc, baby[(ci, j)] if j else inputs[ci], weights[wkey])
                pd = be.wrap(acc)
                if i:
                    pd = be.rot(pd, i * self.g * self.B % self.n)
                y = pd if y is None else be.add(y, pd)
            out.append(y)
        return out

    # gather / scatter of the feature vectors (host side of the layouts above)
    def gather_in(self, X, c, bg):
        """slot vector of input ciphertext c for X[BS][n_in]."""
        vec = np.zeros(self.n)
        for p in range(self.P):
            f = self.feat(c, p)
            if f < 0:
                continue
            for b in range(self.B):
                bb = bg * self.B + b
                if bb < self.BS:
                    vec[p * self.B + b] = X[bb, f]
        return vec

    def scatter_out(self, Y, vec, c, bg):
        for p in range(self.P):
            v = self.neuron(c, p)
            if v < 0:
                continue
            for b in range(self.B):
                bb = bg * self.B + b
                if bb < self.BS:
                    Y[bb, v] = vec[p * self.B + b]


def fc_counts(n, **kw):
    return FcGraph(n, **kw).counts()


def fc_slots(graph: FcGraph, X, W):
    """The fc graph on plain slot vectors -> Y[BS][n_out] (pin: must equal X @ W.T)."""
    be = fr.SlotBackend(graph.n)
    Wp = {wk: graph.weight_slots(wk, W) for giants in graph.terms.values() for lst in giants.values() for _, _, wk in lst}
    Y = np.zeros((graph.BS, graph.n_out))
    for bg in range(graph.BG):
        ins = [graph.gather_in(X, c, bg) for c in range(graph.n_in_ct)]
        for c, y in enumerate(graph.run(be, ins, Wp)):
            graph.scatter_out(Y, y, c, bg)
    return Y


def encode_fc_weights(ck, params, graph: FcGraph, W, L, scale_w=None):
    sw = Fraction(params.q[L - 1]) if scale_w is None else Fraction(scale_w)
    return {wk: ck.encode(params, graph.weight_slots(wk, W), L, sw)
            for giants in graph.terms.values() for lst in giants.values() for _, _, wk in lst}


def fc(ck, params, keys, graph: FcGraph, inputs, weights, do_rescale=True, hoist=False):
    """inputs: list of Ciphertext of one batch group -> list of Ciphertext; one rescale per output (A13)."""
    w0 = next(iter(weights.values()))
    be = fr.CtBackend(ck, params, keys, inputs[0].L, inputs[0].scale, w0.scale, hoist)
    outs = graph.run(be, inputs, weights)
    return [ck.rescale(params, y) for y in outs] if do_rescale else outs


# --------------------------------------------------------------------------- pooling by fragment selection (R2.12)
def pool_order(n_ct, S):
    """indices such that consecutive groups of four are the fragments (2uo+a, 2vo+b) of output fragment (uo, vo);
    ciphertext order [bg][g][u][v] (pooling / stride keep or combine whole fragment ciphertexts)."""
    idx = []
    for base in range(0, n_ct, S * S):
        for uo in range(S // 2):
            for vo in range(S // 2):
                idx += [base + (2 * uo + a) * S + (2 * vo + b) for a in range(2) for b in range(2)]
    return idx


def sum_pool(ck, params, cts, S):
    """out(uo, vo) = sum_{a,b in {0,1}} in(2uo+a, 2vo+b): no rotation, no level; the factor 1/4 belongs to the next
    linear layer's weights."""
    order = pool_order(len(cts), S)
    out = []
    for i in range(0, len(order), 4):
        y = cts[order[i]]
        for j in order[i + 1:i + 4]:
            y = ck.add(params, y, cts[j])
        out.append(y)
    return out


# --------------------------------------------------------------------------- sequential network
def square_pool(ck, params, keys, cts, S):
    """x^2 followed by the 2x2 sum-pool as one step with lazy relinearisation (R2.12c): one ck.square_sum_relin per
    pooled output over its four fragments (order as in sum_pool)."""
    order = pool_order(len(cts), S)
    return [ck.square_sum_relin(params, keys, [cts[j] for j in order[i:i + 4]]) for i in range(0, len(order), 4)]


def run_network(ck, params, keys, layers, cts, L0, hoist=False, lazy_relin=False):
    """layers as in paper_2606_16359_b200.pipeline.Pipeline (dicts with op = conv / square / pool / fc and fp64 weights);
    cts: oracle ciphertexts ordered [bg][g][u][v].  Returns (final ciphertext list, list of per-layer outputs)."""
    L, S, trace = L0, None, []
    for li, ly in enumerate(layers):
        if lazy_relin and ly["op"] == "pool" and li > 0 and layers[li - 1]["op"] == "square":
            trace.append(cts)  # done together with the square before it
            continue
        if lazy_relin and ly["op"] == "square" and li + 1 < len(layers) and layers[li + 1]["op"] == "pool":
            cts, S, L = square_pool(ck, params, keys, cts, S), S // 2, L - 1
            trace.append(cts)
            continue
        if ly["op"] == "conv":
            graph = fr.ConvGraph(fr.ConvDesc(S=ly["S"], **ly["conv"]), params.n)
            W = fr.encode_weights(ck, params, graph, ly["w"], L)
            per = graph.S * graph.S * graph.lin.G
            out = []
            for bg in range(graph.lin.BG):
                ins = {(u, v, g): cts[bg * per + (g * graph.S + u) * graph.S + v]
                       for g in range(graph.lin.G) for u in range(graph.S) for v in range(graph.S)}
                o = fr.hconv(ck, params, keys, graph, ins, W, hoist=hoist)
                So = graph.S_out
                out += [o[(uo, vo, go)] for go in range(graph.lout.G) for uo in range(So) for vo in range(So)]
            cts, S, L = out, graph.S_out, L - 1
        elif ly["op"] == "fc":
            graph = FcGraph(params.n, **ly["fc"])
            W = encode_fc_weights(ck, params, graph, ly["w"], L)
            out = []
            for bg in range(graph.BG):
                out += fc(ck, params, keys, graph, cts[bg * graph.n_in_ct:(bg + 1) * graph.n_in_ct], W, hoist=hoist)
            cts, S, L = out, 1, L - 1
        elif ly["op"] == "square":
            cts, L = [ck.square_relin(params, keys, c) for c in cts], L - 1
        elif ly["op"] == "poly3":
            cts, L = [ck.poly3(params, keys, c, ly.get("coef", ck.POLY3)) for c in cts], L - 2
        elif ly["op"] == "pool":
            cts, S = sum_pool(ck, params, cts, S), S // 2
        else:
            raise ValueError(ly["op"])
        trace.append(cts)
    return cts, trace


def network_rot_steps(layers, n):
    """every rotation amount the network needs, and whether it needs the relinearisation key."""
    steps, relin = set(), False
    for ly in layers:
        if ly["op"] == "conv":
            steps.update(fr.ConvGraph(fr.ConvDesc(S=ly["S"], **ly["conv"]), n).counts()["rot_steps"])
        elif ly["op"] == "fc":
            steps.update(FcGraph(n, **ly["fc"]).counts()["rot_steps"])
        elif ly["op"] in ("square", "poly3"):
            relin = True
    return sorted(steps), relin

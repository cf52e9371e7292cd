"""Fragment-encoding oracle: Algorithm 1 layout, the HConv operation graph, planner counts, AAC.
TEST INFRASTRUCTURE ONLY -- see oracle/__init__.py.

Follows PAPER.md:166-178 (Algorithm 1), PAPER.md:84-91 (Eq. 2, inner / outer rotations),
PAPER.md:198-246 (Eq. 3-8), PAPER.md:252-276 (AAC), PAPER.md:284 (stride by dropping
ciphertexts), with the readings R2.9-R2.11 / A3-A6, A13-A19 of DESIGN.md section 4.

The graph is written once, over an abstract "backend" with rot / pmult_acc / add / finish, and
run (i) on plain slot vectors, where a rotation is a cyclic shift -- the oracle-of-the-oracle
pin against direct convolution -- and (ii) on oracle ciphertexts (oracle/ckks.py).
"""
import math
from fractions import Fraction

import numpy as np


def next_pow2(x: int) -> int:
    return 1 << max(0, (x - 1).bit_length())


# --------------------------------------------------------------------------- Algorithm 1 (R2.9)
class Layout:
    """Layout(n, M, S, BS, C): ciphertext (u, v, g, bg) holds at slot(cpos, k, b) the value
    X_pad[bg*B + b, g*ch + cpos, bi*S + u, bj*S + v], k = bi*m + bj  (PAPER.md:170-176 read
    0-based with floors, A3; "filled first with other samples then other channels").

    Segmented form (v > 0; the layout AAC's canonical compaction produces, R2.11 / R2.11b): the chp
    physical channel positions of a ciphertext are seg = chp / v segments of v positions; segment sg holds the v channels
    g*v .. g*v + v - 1 of the samples of batch group bg*seg + sg, i.e. slot((sg*v + pl), k, b) holds
    X_pad[(bg*seg + sg)*B + b, g*v + pl, ...].  ch is the number of channel positions of one segment (v); v = 0 or
    v = chp is the plain layout (one segment).  B_cap > 0 caps the samples per ciphertext below "batch first"'s n/m^2
    (B = min(BS^, n/m^2, B_cap)): then a large batch has several batch groups AND several channel positions per ciphertext,
    which is where a channel-reducing layer leaves ciphertexts sparse and batch-group compaction (R2.11) applies."""

    def __init__(self, n, M, S, BS, C, v=0, B_cap=0):
        assert M % S == 0
        self.n, self.M, self.S, self.BS, self.C = n, M, S, BS, C
        self.m = M // S
        m2 = self.m * self.m
        assert m2 <= n and n % m2 == 0, "m^2 must divide the slot count"
        self.B = min(next_pow2(BS), n // m2)
        if B_cap:  # samples per ciphertext capped by the caller (a serving system's request size): channels fill the rest
            self.B = min(self.B, B_cap)
        self.chp = n // (self.B * m2)
        self.v = v if v else self.chp
        assert self.chp % self.v == 0, "the segment size must divide the channel positions"
        self.seg = self.chp // self.v
        self.ch = self.v
        self.cs = self.B * m2
        self.G = -(-C // self.ch)
        self.BG = -(-(-(-BS // self.B)) // self.seg)

    def slot(self, cpos, k, b):
        return cpos * self.cs + k * self.B + b

    def ct_keys(self):
        return [(u, v, g, bg) for bg in range(self.BG) for g in range(self.G) for u in range(self.S) for v in range(self.S)]

    def _entries(self, g, bg, BS, C, H, W, u, v):
        """(slot, sample, channel, h, w) of every tensor entry ciphertext (u, v, g, bg) holds"""
        for sg in range(self.seg):
            for pl in range(self.ch):
                c = g * self.ch + pl
                if c >= C:
                    continue
                for b in range(self.B):
                    bb = (bg * self.seg + sg) * self.B + b
                    if bb >= BS:
                        continue
                    for bi in range(self.m):
                        h = bi * self.S + u
                        if h >= H:
                            continue
                        for bj in range(self.m):
                            w = bj * self.S + v
                            if w < W:
                                yield self.slot(sg * self.ch + pl, bi * self.m + bj, b), bb, c, h, w

    def gather(self, X, u, v, g, bg):
        """Slot vector of ciphertext (u, v, g, bg) for X[BS, C, H, W] (zero outside the tensor)."""
        BS, C, H, W = X.shape
        vec = np.zeros(self.n, dtype=np.float64)
        for sl, bb, c, h, w in self._entries(g, bg, BS, C, H, W, u, v):
            vec[sl] = X[bb, c, h, w]
        return vec

    def scatter(self, Y, vec, u, v, g, bg):
        """Inverse of gather: write this ciphertext's entries into Y[BS, C, H, W]."""
        BS, C, H, W = Y.shape
        for sl, bb, c, h, w in self._entries(g, bg, BS, C, H, W, u, v):
            Y[bb, c, h, w] = vec[sl]


class ConvDesc:
    def __init__(self, BS, C_in, H, W, C_out, K, stride=1, pad=0, depthwise=False, S=0, M=0, seg_v=0, B_cap=0, bsgs=1):
        self.BS, self.C_in, self.H, self.W, self.C_out, self.K = BS, C_in, H, W, C_out, K
        self.stride, self.pad, self.depthwise, self.S, self.M = stride, pad, depthwise, S, M
        self.seg_v = seg_v  # > 0: input and output ciphertexts in the segmented layout with v = seg_v (R2.11b)
        self.B_cap = B_cap    # > 0: at most B_cap samples per ciphertext (Layout)
        self.bsgs = bsgs      # baby steps over the channel diagonals (R2.9d): 1 = none, g > 1 explicit, 0 = fewest rotations
        self.H_out = (H + 2 * pad - K) // stride + 1
        self.W_out = (W + 2 * pad - K) // stride + 1


def direct_conv(desc: ConvDesc, X, Kw):
    """Eq. 2 with stride and zero padding, fp64, plain loops over taps."""
    BS, Ci, H, W = X.shape
    Y = np.zeros((BS, desc.C_out, desc.H_out, desc.W_out), dtype=np.float64)
    Xp = np.zeros((BS, Ci, H + 2 * desc.pad, W + 2 * desc.pad), dtype=np.float64)
    Xp[:, :, desc.pad:desc.pad + H, desc.pad:desc.pad + W] = X
    s = desc.stride
    for o in range(desc.C_out):
        for c in ([o] if desc.depthwise else range(Ci)):
            for i in range(desc.K):
                for j in range(desc.K):
                    w = Kw[o, 0 if desc.depthwise else c, i, j]
                    Y[:, o] += w * Xp[:, c, i:i + s * desc.H_out:s, j:j + s * desc.W_out:s]
    return Y


# --------------------------------------------------------------------------- the HConv graph (R2.9)
class ConvGraph:
    """Static operation graph of one fragment-encoded conv layer for one batch group.

    terms[(u_o, v_o, g_out)][d] = list of (src_key (u', v', g_in), amt, wkey (u_o, v_o, g_out, g_in, d, i, j));
    inner = sorted set of (src_key, amt != 0); outer[(u_o, v_o, g_out)] = existing diagonals d.

    Segmented layouts (desc.seg_v = v > 0 with several segments, R2.11b: the consumer of AAC's output):
    channel diagonal d must wrap inside each v-position segment, not around the whole ciphertext, so it splits in two
    partial sums: part 0 holds the input positions pl >= d of every segment and is rotated by d*cs, part 1 the positions
    pl < d and is rotated by (d - v)*cs (both masks folded into the weight plaintexts); the diagonal key is
    dkey = d + part*chp (chp = physical channel positions), and diag_rot(dkey) is its outer rotation amount.

    Baby-step giant-step over the channel diagonals (desc.bsgs = g > 1; R2.9d; PAPER.md:82 names the outer rotations as
    the cost to cut, PAPER.md:284 uses BSGS for the diagonals of the FC layers): with d = i g + j, 0 <= j < g,
        Y = sum_i Rot( sum_j sum_t Rot(in_t, amt_t + j cs) (*) W'(t, d), i g cs ),   W'(t, d) = Rot(W(t, d), j cs),
    because Rot(x (*) w, r) = Rot(x, r) (*) Rot(w, r) and Rot(Rot(in, amt), j cs) = Rot(in, amt + j cs): the baby step is
    folded into the INNER rotation (still one rotation of the original input, shared by every output and hoistable), the
    giant steps are the outer rotations -- ch/g - 1 per output instead of ch - 1.  After the regrouping the keys of
    terms[okey] are the giant steps i, the term amounts are the composite ones, and weight_slots shifts by j cs.
    On a segmented layout the two parts of diagonal d = i g + j keep their baby step j and become giant keys i and
    i + chp with outer rotations i g cs and (i g - v) cs."""

    def __init__(self, desc: ConvDesc, n: int):
        d = desc
        self.desc, self.n = d, n
        self.M = d.M if d.M else next_pow2(max(d.H, d.W))
        self.S = d.S
        assert self.S >= 1 and self.S % d.stride == 0, "stride must divide S"
        self.lin = Layout(n, self.M, self.S, d.BS, d.C_in, d.seg_v, d.B_cap)
        self.S_out = self.S // d.stride
        self.lout = Layout(n, self.M // d.stride, self.S_out, d.BS, d.C_out, d.seg_v, d.B_cap)
        assert (self.lout.m, self.lout.B, self.lout.ch) == (self.lin.m, self.lin.B, self.lin.ch)
        self.dkeys = list(range(self.lin.ch)) + ([self.lin.chp + dd for dd in range(1, self.lin.ch)] if self.lin.seg > 1 else [])
        self._wcache = {}
        self.terms, inner = {}, set()
        L = self.lin
        for uo in range(self.S_out):
            for vo in range(self.S_out):
                for go in range(self.lout.G):
                    diags = {}
                    for dd in self.dkeys:
                        lst = []
                        for gi in range(L.G):
                            for i in range(d.K):
                                for j in range(d.K):
                                    wkey = (uo, vo, go, gi, dd, i, j)
                                    if not self.weight_nonzero_pattern(wkey):
                                        continue
                                    ti = d.stride * uo + i - d.pad
                                    tj = d.stride * vo + j - d.pad
                                    up, di = ti % self.S, ti // self.S  # floor division, may be negative
                                    vp, dj = tj % self.S, tj // self.S
                                    amt = ((di * L.m + dj) * L.B) % n
                                    lst.append(((up, vp, gi), amt, wkey))
                                    if amt:
                                        inner.add(((up, vp, gi), amt))
                        if lst:
                            diags[dd] = lst
                    self.terms[(uo, vo, go)] = diags
        self.inner = sorted(inner)
        self.g = 1
        if d.bsgs != 1 and L.ch > 1:
            cands = [d.bsgs] if d.bsgs > 1 else [1 << k for k in range(0, L.ch.bit_length()) if L.ch % (1 << k) == 0]
            best = None
            for g in cands:
                assert L.ch % g == 0 and g & (g - 1) == 0, "bsgs must be a power of two dividing the channel positions"
                terms, inner_g = self._regroup(g)
                n_rot = len(inner_g) + sum(len([i for i in giants if i]) for giants in terms.values())
                if best is None or n_rot < best[0]:  # fewest rotations, ties to the smaller g
                    best = (n_rot, g, terms, inner_g)
            _, self.g, self.terms, inner_g = best
            self.inner = sorted(inner_g)

    def _regroup(self, g):
        """the plain graph's diagonals d = i g + j regrouped by giant step i (R2.9d); g = 1 returns the plain graph"""
        L, n = self.lin, self.n
        terms, inner = {}, set()
        for okey, diags in self.terms.items():
            giants = {}
            for dd in sorted(diags):
                # segmented layouts (R2.11b): dd = d + part*chp; both parts of diagonal d share its baby step, the giant
                # key keeps the part (its outer rotation is (i g - part v) cs, see diag_rot)
                part, dl = divmod(dd, L.chp) if L.seg > 1 else (0, dd)
                i, j = divmod(dl, g)
                i += part * L.chp
                for src, amt, wkey in diags[dd]:
                    a = (amt + j * L.cs) % n
                    giants.setdefault(i, []).append((src, a, wkey))
                    if a:
                        inner.add((src, a))
            terms[okey] = giants
        return terms, inner

    # Which entries of weight plaintext wkey can be non-zero (independent of the values).  The validity
    # conditions of R2.9 step 2 factorise: channel positions (c < C_in, o < C_out, depthwise o == c),
    # block rows (h_o < H_o, 0 <= h_i < H) and block columns (w_o < W_o, 0 <= w_i < W).
    def _valid_cpos(self, go, gi, dd):
        key = ("c", go, gi, dd)
        if key not in self._wcache:
            d, L = self.desc, self.lin
            part, dl = divmod(dd, L.chp) if L.seg > 1 else (0, dd)
            out = []
            for sg in range(L.seg):
                for pl in range(L.ch):
                    if L.seg > 1 and (pl >= dl) != (part == 0):
                        continue  # part 0: the positions that stay inside their segment under a shift by dl; part 1: those that wrap
                    c = gi * L.ch + pl
                    o = go * L.ch + ((pl - dl) % L.ch)
                    if c < d.C_in and o < d.C_out and (not d.depthwise or o == c):
                        out.append((sg * L.ch + pl, o, c))
            self._wcache[key] = out
        return self._wcache[key]

    def diag_rot(self, dd):
        """outer rotation amount of diagonal key dd: d*cs, or (d - v)*cs for the wrapping part of a segmented layout"""
        L = self.lin
        if self.g > 1:  # dd is a giant step i (R2.9d), + chp for the wrapping part of a segmented layout
            part, i = divmod(dd, L.chp) if L.seg > 1 else (0, dd)
            return ((i * self.g - part * L.ch) * L.cs) % self.n
        part, dl = divmod(dd, L.chp) if L.seg > 1 else (0, dd)
        return ((dl - L.ch) * L.cs) % self.n if part else (dl * L.cs) % self.n

    def _valid_blocks(self, frag_o, tap, size_in, size_out):
        """Block indices bi with h_o = bi*S_o + frag_o < size_out and 0 <= stride*h_o + tap - pad < size_in."""
        key = ("b", frag_o, tap, size_in, size_out)
        if key not in self._wcache:
            d = self.desc
            out = []
            for bi in range(self.lin.m):
                ho = bi * self.S_out + frag_o
                hi = d.stride * ho + tap - d.pad
                if ho < size_out and 0 <= hi < size_in:
                    out.append(bi)
            self._wcache[key] = out
        return self._wcache[key]

    def _weight_factors(self, wkey):
        uo, vo, go, gi, dd, i, j = wkey
        d = self.desc
        return (self._valid_cpos(go, gi, dd), self._valid_blocks(uo, i, d.H, d.H_out), self._valid_blocks(vo, j, d.W, d.W_out))

    def weight_nonzero_pattern(self, wkey):
        cp, rows, cols = self._weight_factors(wkey)
        return bool(cp) and bool(rows) and bool(cols)

    def weight_slots(self, wkey, Kw):
        """Slot vector W(u_o, v_o, g_out, g_in, d, i, j) (R2.9 step 2); all b alike."""
        _, _, _, _, _, i, j = wkey
        L = self.lin
        cp, rows, cols = self._weight_factors(wkey)
        vec = np.zeros(self.n, dtype=np.float64)
        for cpos, o, c in cp:
            val = Kw[o, 0 if self.desc.depthwise else c, i, j]
            for bi in rows:
                for bj in cols:
                    base = L.slot(cpos, bi * L.m + bj, 0)
                    vec[base:base + L.B] = val
        if self.g > 1:  # W' = Rot(W, j cs) with j the baby step of this plaintext's diagonal (R2.9d)
            vec = np.roll(vec, -((wkey[4] % self.g) * L.cs))
        return vec

    # ---- factored weights (R2.9c; the large-batch case of PAPER.md:218-222, where one ciphertext holds one channel)
    def weight_factor(self, wkey, Kw):
        """(v, mkey) with weight_slots(wkey, Kw) == v * mask_slots(mkey), or None when the plaintext has more than one
        valid channel position (then it is not a scalar times a 0/1 mask).  v = K[o, c, i, j]; mkey = (cpos, rows, cols)."""
        _, _, _, _, _, i, j = wkey
        cp, rows, cols = self._weight_factors(wkey)
        if len(cp) != 1:
            return None
        cpos, o, c = cp[0]
        return Kw[o, 0 if self.desc.depthwise else c, i, j], (cpos, tuple(rows), tuple(cols))

    def mask_slots(self, mkey):
        """0/1 slot vector of mask key (cpos, rows, cols): 1 at slot(cpos, bi*m + bj, b) for bi in rows, bj in cols, all b."""
        cpos, rows, cols = mkey
        L = self.lin
        vec = np.zeros(self.n, dtype=np.float64)
        for bi in rows:
            for bj in cols:
                base = L.slot(cpos, bi * L.m + bj, 0)
                vec[base:base + L.B] = 1.0
        return vec

    def factorable(self):
        """every weight plaintext of the layer is a scalar times a mask (true whenever ch = 1)"""
        return all(len(self._weight_factors(wk)[0]) == 1 for diags in self.terms.values() for lst in diags.values() for _, _, wk in lst)

    def run_factored(self, be, inputs, values, masks):
        """The same graph with every weight plaintext replaced by its factors (R2.9c): per output and diagonal
            P_d = sum over masks mu of  M_mu (*) ( sum over the terms t with mask mu of  v_t . R_t ),
        v_t . R_t a scalar multiple of a (rotated) input, M_mu a mask plaintext.  values: {wkey: v}; masks: {mkey: M};
        self.mask_of[wkey] = mkey (set by the caller through factor_weights)."""
        R = {}
        for src, amt in self.inner:
            R[(src, amt)] = be.rot_in(inputs[src], amt)
        out = {}
        for okey, diags in self.terms.items():
            y = None
            for dd in sorted(diags):
                by_mask = {}
                for src, amt, wkey in diags[dd]:
                    by_mask.setdefault(self.mask_of[wkey], []).append((src, amt, wkey))
                acc = be.zero()
                for mkey, lst in by_mask.items():
                    S = be.zero_in()
                    for src, amt, wkey in lst:
                        S = be.scale_acc(S, R[(src, amt)] if amt else inputs[src], values[wkey])
                    be.pmult_acc(acc, S, masks[mkey])
                pd = be.wrap(acc)
                if self.diag_rot(dd):
                    pd = be.rot(pd, self.diag_rot(dd))
                y = pd if y is None else be.add(y, pd)
            out[okey] = y
        return out

    # ---- exact counts of this graph (per batch group; multiply by BG for the layer)
    def counts(self):
        n_outer = 0
        n_pmult = 0
        for diags in self.terms.values():
            n_outer += len([x for x in diags if self.diag_rot(x)])  # every existing diagonal d != 0 is rotated once
            n_pmult += sum(len(v) for v in diags.values())
        bg = self.lin.BG
        steps = sorted({amt for _, amt in self.inner} | {self.diag_rot(dd) for diags in self.terms.values() for dd in diags if self.diag_rot(dd)})
        return dict(n_in_ct=self.S * self.S * self.lin.G * bg, n_out_ct=self.S_out ** 2 * self.lout.G * bg,
                    n_inner_rot=len(self.inner) * bg, n_outer_rot=n_outer * bg, n_pmult=n_pmult * bg,
                    n_distinct_pt=n_pmult, rot_steps=steps)

    # ---- run the graph on a backend (R2.9 steps 1, 3, 4; rescale / finish is the caller's)
    def run(self, be, inputs, weights):
        """inputs: {(u, v, g_in): x}; weights: {wkey: w}.  Returns {(u_o, v_o, g_out): y}."""
        R = {}
        for src, amt in self.inner:
            R[(src, amt)] = be.rot_in(inputs[src], amt)  # always from the original input, never chained
        out = {}
        for okey, diags in self.terms.items():
            y = None
            for dd in sorted(diags):
                acc = be.zero()
                for src, amt, wkey in diags[dd]:
                    be.pmult_acc(acc, R[(src, amt)] if amt else inputs[src], weights[wkey])
                pd = be.wrap(acc)
                if self.diag_rot(dd):
                    pd = be.rot(pd, self.diag_rot(dd))
                y = pd if y is None else be.add(y, pd)
            out[okey] = y
        return out


class SlotBackend:
    """Plain slot vectors: rotation = cyclic left shift, PMult = slot-wise product."""

    def __init__(self, n):
        self.n = n

    def rot(self, x, r):
        return np.roll(x, -r)

    rot_in = rot  # inner (input-side) rotations: the same shift

    def zero(self):
        return np.zeros(self.n)

    def pmult_acc(self, acc, x, w):
        acc += x * w

    def wrap(self, acc):
        return acc

    def add(self, x, y):
        return x + y

    def zero_in(self):
        return np.zeros(self.n)

    def scale_acc(self, S, x, v):
        return S + v * x


def hconv_slots(desc: ConvDesc, n: int, X, Kw):
    """The graph on plain slot vectors -> Y[BS, C_out, H_out, W_out]."""
    g = ConvGraph(desc, n)
    be = SlotBackend(n)
    W = {wk: g.weight_slots(wk, Kw) for diags in g.terms.values() for lst in diags.values() for _, _, wk in lst}
    Y = np.zeros((desc.BS, desc.C_out, desc.H_out, desc.W_out))
    for bg in range(g.lin.BG):
        ins = {(u, v, gi): g.lin.gather(X, u, v, gi, bg) for u in range(g.S) for v in range(g.S) for gi in range(g.lin.G)}
        outs = g.run(be, ins, W)
        for (uo, vo, go), y in outs.items():
            if y is not None:
                g.lout.scatter(Y, y, uo, vo, go, bg)
    return Y


# --------------------------------------------------------------------------- planner (R2.10, Eq. 3-8)
def alpha_ch(n, M):
    """Channels per ciphertext at S = 1, BS = 1 as a rational: n / M^2 (A16)."""
    return Fraction(n, M * M)


def paper_inner_per_ct(S, K, M):
    """Eq. 3 per input ciphertext, with Table IX's evident 0 for K <= S (A6)."""
    if S >= M or K <= S:
        return 0
    return (-(-K // S)) ** 2 - 1


def paper_rot_count(desc: ConvDesc, n, S):
    """#Rot as Table IX prints it: n_in * I(S, K) + n_out * (ch - 1), with
    n_in = N_in*BS/alpha, n_out = N_out*BS/alpha (A18), ch = alpha*S^2/BS (Eq. 4)."""
    M = desc.M if desc.M else next_pow2(max(desc.H, desc.W))
    a = alpha_ch(n, M)
    n_in = Fraction(desc.C_in * desc.BS) / a
    n_out = Fraction(desc.C_out * desc.BS) / a
    ch = a * S * S / desc.BS
    tot = n_in * paper_inner_per_ct(S, desc.K, M) + n_out * (ch - 1)
    return tot


def s_star_real(desc: ConvDesc, n):
    """Eq. 8 with the BS factor restored (A5): (K^2 N_in BS / (alpha N_out))^(1/4)."""
    M = desc.M if desc.M else next_pow2(max(desc.H, desc.W))
    return (desc.K ** 2 * desc.C_in * desc.BS / (float(alpha_ch(n, M)) * desc.C_out)) ** 0.25


def candidates(desc: ConvDesc, n):
    """Feasible block sizes: powers of two with S | M, stride | S, m^2 <= n, and Eq. 7
    S <= sqrt(BS N_in / alpha) unless that leaves none (then the smallest feasible)."""
    M = desc.M if desc.M else next_pow2(max(desc.H, desc.W))
    feas = [S for S in (1 << k for k in range(0, 12)) if S <= M and M % S == 0 and S % desc.stride == 0 and (M // S) ** 2 <= n]
    bound = math.sqrt(desc.BS * desc.C_in / float(alpha_ch(n, M)))
    ok = [S for S in feas if S <= bound]
    return ok if ok else feas[:1]


def with_S(desc: ConvDesc, S):
    return ConvDesc(desc.BS, desc.C_in, desc.H, desc.W, desc.C_out, desc.K, desc.stride, desc.pad, desc.depthwise, S, desc.M, desc.seg_v, desc.B_cap, desc.bsgs)


def select_S(desc: ConvDesc, n):
    """Conv-aware selection: arg-min of the exact rotation count over the candidates, ties -> smaller S."""
    best = None
    for S in candidates(desc, n):
        c = ConvGraph(with_S(desc, S), n).counts()
        tot = c["n_inner_rot"] + c["n_outer_rot"]
        if best is None or tot < best[0]:
            best = (tot, S)
    return best[1]


# --------------------------------------------------------------------------- encrypted HConv (R2.9)
class CtBackend:
    """hoist: the inner (input-side) rotations, several of which share one input ciphertext, use the hoisted form of
    R2.7b (ck.rotate_hoisted); the outer rotations, each of a different sum, stay plain rotations."""

    def __init__(self, ck, params, keys, L, scale_in, scale_w, hoist=False):
        self.ck, self.params, self.keys, self.L = ck, params, keys, L
        self.scale_in, self.scale_w = Fraction(scale_in), Fraction(scale_w)
        self.hoist = hoist

    def rot(self, x, r):
        return self.ck.rotate(self.params, self.keys, x, r)

    def rot_in(self, x, r):
        return (self.ck.rotate_hoisted if self.hoist else self.ck.rotate)(self.params, self.keys, x, r)

    def zero(self):
        return np.zeros((2, self.L, self.params.N), dtype=np.uint64)

    def pmult_acc(self, acc, x, w):
        assert x.scale == self.scale_in and w.scale == self.scale_w
        self.ck.pmult_acc(self.params, acc, x, w)

    def wrap(self, acc):
        return self.ck.Ciphertext(acc, self.L, self.scale_in * self.scale_w)

    def add(self, x, y):
        return self.ck.add(self.params, x, y)

    # factored weights (R2.9c): S = sum_t round_half_up(v_t E1) . R_t at scale s_in E1, then acc += S (*) M with M at E2
    def zero_in(self):
        return None

    def scale_acc(self, S, x, v):
        assert x.scale == self.scale_in
        t = self.ck.mul_const(self.params, x, v, self.E1)
        return t if S is None else self.ck.add(self.params, S, t)


def encode_weights(ck, params, graph: ConvGraph, Kw, L, scale_w=None):
    """Every non-zero weight plaintext of the graph, encoded at s_w (default q_{L-1}, A14) on L limbs."""
    sw = Fraction(params.q[L - 1]) if scale_w is None else Fraction(scale_w)
    W = {}
    for diags in graph.terms.values():
        for lst in diags.values():
            for _, _, wk in lst:
                if wk not in W:
                    W[wk] = ck.encode(params, graph.weight_slots(wk, Kw), L, sw)
    return W


def factor_scales(scale_w):
    """(E1, E2) with E1 E2 = s_w and E1 = 2^ceil(log2(s_w) / 2): the split Delta_1 Delta_2 = Delta of PAPER.md:276, applied
    to a weight value (E1) and the 0/1 validity mask it multiplies (E2), so the two products still cost one level."""
    sw = Fraction(scale_w)
    bits = 0
    while Fraction(2) ** bits < sw:
        bits += 1
    E1 = Fraction(2) ** (-(-bits // 2))
    return E1, sw / E1


def factor_weights(ck, params, graph: ConvGraph, Kw, L, scale_w=None):
    """R2.9c: every weight plaintext of a layer whose ciphertexts hold one channel each (ch = 1, the large-batch case of
    PAPER.md:218-222) is a real value times a 0/1 mask; the value is kept as a real (rounded to the integer
    round_half_up(v E1) when it multiplies a ciphertext, R2.8), the distinct masks are encoded at E2.
    Returns (values {wkey: v}, masks {mkey: Plaintext}, E1); sets graph.mask_of."""
    assert graph.factorable(), "a weight plaintext with several channel positions is not a scalar times a mask"
    sw = Fraction(params.q[L - 1]) if scale_w is None else Fraction(scale_w)
    E1, E2 = factor_scales(sw)
    values, masks, graph.mask_of = {}, {}, {}
    for diags in graph.terms.values():
        for lst in diags.values():
            for _, _, wk in lst:
                if wk in values:
                    continue
                v, mk = graph.weight_factor(wk, Kw)
                values[wk], graph.mask_of[wk] = float(v), mk
                if mk not in masks:
                    masks[mk] = ck.encode(params, graph.mask_slots(mk), L, E2)
    return values, masks, E1


def hconv_factored(ck, params, keys, graph: ConvGraph, inputs, values, masks, E1, do_rescale=True, hoist=False):
    """hconv with factored weights (R2.9c): inputs {(u, v, g_in): Ciphertext} of one batch group."""
    any_in = next(iter(inputs.values()))
    any_m = next(iter(masks.values()))
    be = CtBackend(ck, params, keys, any_in.L, any_in.scale, any_m.scale, hoist)
    # the ciphertexts entering scale_acc are at the input scale; the sums S entering pmult_acc at s_in E1
    be.E1, be.scale_S = Fraction(E1), any_in.scale * Fraction(E1)
    outs = graph.run_factored(_FactoredView(be), inputs, values, masks)
    if do_rescale:
        outs = {k: (ck.rescale(params, y) if y is not None else None) for k, y in outs.items()}
    return outs


class _FactoredView:
    """CtBackend seen from run_factored: PMult-accumulate takes the sums S (scale s_in E1) and the masks (scale E2)."""

    def __init__(self, be):
        self.be = be
        self.rot, self.rot_in, self.zero, self.add, self.zero_in, self.scale_acc = be.rot, be.rot_in, be.zero, be.add, be.zero_in, be.scale_acc

    def pmult_acc(self, acc, S, M):
        assert S.scale == self.be.scale_S and M.scale == self.be.scale_w
        self.be.ck.pmult_acc(self.be.params, acc, S, M)

    def wrap(self, acc):
        return self.be.ck.Ciphertext(acc, self.be.L, self.be.scale_S * self.be.scale_w)


def hconv(ck, params, keys, graph: ConvGraph, inputs, weights, do_rescale=True, hoist=False):
    """inputs {(u, v, g_in): Ciphertext} of ONE batch group -> {(u_o, v_o, g_out): Ciphertext};
    one rescale per output ciphertext after the outer-rotation sum (A13)."""
    any_in = next(iter(inputs.values()))
    any_w = next(iter(weights.values()))
    be = CtBackend(ck, params, keys, any_in.L, any_in.scale, any_w.scale, hoist)
    outs = graph.run(be, inputs, weights)
    if do_rescale:
        outs = {k: (ck.rescale(params, y) if y is not None else None) for k, y in outs.items()}
    return outs


# --------------------------------------------------------------------------- AAC compress (R2.11)
def compress_plan(n, ch, cs, v, n_src):
    """Canonical batch-group compaction: sources hold valid channel positions [0, v), v | ch, v < ch;
    output t gathers sources i in [t*ch/v, (t+1)*ch/v) with r = (n - (i mod (ch/v)) * v * cs) mod n
    (a right shift by whole v-position segments).  Returns [[(src, r), ...], ...]."""
    assert ch % v == 0 and v < ch
    per = ch // v
    plan = []
    for t in range(-(-n_src // per)):
        plan.append([(i, (n - (i % per) * v * cs) % n) for i in range(t * per, min((t + 1) * per, n_src))])
    return plan


def compress_mask(n, cs, v):
    """0/1 slot vector keeping channel positions [0, v) (constant over k and b)."""
    m = np.zeros(n)
    m[: v * cs] = 1.0
    return m


def compress(ck, params, keys, plan, srcs, mask_pt=None, do_rescale=False):
    """out_t = sum over terms Rot(mask (*) src, r).  Maskless: no level consumed.  Masked split-scale
    (PAPER.md:276): sources at scale s_ct*Delta1 (conv rescale skipped), mask at Delta2, one rescale after."""
    outs = []
    for terms in plan:
        y = None
        for i, r in terms:
            x = srcs[i]
            if mask_pt is not None:
                x = ck.pmult(params, x, mask_pt)
            x = ck.rotate(params, keys, x, r)
            y = x if y is None else ck.add(params, y, x)
        outs.append(ck.rescale(params, y) if do_rescale else y)
    return outs


# --------------------------------------------------------------------------- repack: block-size re-adaptation (R2.11c)
def repack_plan(src: Layout, dst: Layout, shape):
    """Rot-mask-add plan that moves a tensor of `shape` = (BS, C, H, W) from layout `src` to layout `dst` (another block
    size S, another segmentation, ...): "we adapt the pre- or post-processing (rot-mask-add) operations to
    adjust block size".  Every destination slot that holds a tensor entry names the source ciphertext and slot holding
    the same entry; a left rotation by r = (src_slot - dst_slot) mod n brings it in place; entries sharing (destination,
    source, r) share one mask.  Returns {dst_key: [(src_key, r, mask slot vector over the SOURCE slots), ...]}."""
    BS, C, H, W = shape
    where = {}
    for key in src.ct_keys():
        u, v, g, bg = key
        for sl, bb, c, h, w in src._entries(g, bg, BS, C, H, W, u, v):
            where[(bb, c, h, w)] = (key, sl)
    plan = {}
    for key in dst.ct_keys():
        u, v, g, bg = key
        groups = {}
        for sl, bb, c, h, w in dst._entries(g, bg, BS, C, H, W, u, v):
            skey, ssl = where[(bb, c, h, w)]
            groups.setdefault((skey, (ssl - sl) % src.n), []).append(ssl)
        terms = []
        for (skey, r), slots in sorted(groups.items()):
            mask = np.zeros(src.n)
            mask[slots] = 1.0
            terms.append((skey, r, mask))
        plan[key] = terms
    return plan


def repack_slots(plan, vecs):
    """the plan on plain slot vectors: out = sum Rot(mask * src, r), rotation = left cyclic shift"""
    return {k: sum(np.roll(m * vecs[s], -r) for s, r, m in terms) for k, terms in plan.items()}


def repack(ck, params, keys, plan, srcs, L, scale_m=None):
    """out_t = Rescale( sum over terms of Rot(mask (*) src, r) ): masks encoded at q_{L-1} (one level, PAPER.md:276's
    single late rescale); terms sharing (destination, r) are summed before their one rotation."""
    sm = Fraction(params.q[L - 1]) if scale_m is None else Fraction(scale_m)
    outs = {}
    for dkey, terms in plan.items():
        by_rot = {}
        for skey, r, mask in terms:
            by_rot.setdefault(r, []).append((skey, mask))
        y = None
        for r in sorted(by_rot):
            acc = np.zeros((2, L, params.N), dtype=np.uint64)
            for skey, mask in by_rot[r]:
                ck.pmult_acc(params, acc, srcs[skey], ck.encode(params, mask, L, sm))
            t = ck.Ciphertext(acc, L, srcs[by_rot[r][0][0]].scale * sm)
            if r:
                t = ck.rotate(params, keys, t, r)
            y = t if y is None else ck.add(params, y, t)
        outs[dkey] = ck.rescale(params, y)
    return outs

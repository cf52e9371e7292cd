"""Layer sequencing over the C ABI: a list of fragment-encoded layers (conv / square / pool / fc) evaluated by one
batched library call per layer (R2.9, R2.12).  Orchestration only: every ciphertext
operation runs inside libfenc's kernels; this file holds no arithmetic on ciphertext data."""
import math
from fractions import Fraction

import numpy as np

POLY3 = (Fraction(1, 2), Fraction(197, 1000), Fraction(-4, 1000))  # BASELINE config 3: 0.5 + 0.197 x - 0.004 x^3


def _round_half_up(x):
    return math.floor(Fraction(x) + Fraction(1, 2))


def poly3_activation(ctx, keys, cts, scale, coef=POLY3):
    """Degree-3 activation a0 + a1 x + a3 x^3 in two levels (R2.12): ONE library call (fenc_poly3 owns the order
    of the steps); this function only rounds the three integer multipliers exactly from the exact rational scale of the
    inputs (R2.8).  Returns (ciphertexts at L-2, their exact scale)."""
    a0, a1, a3 = (Fraction(c) for c in coef)
    L, s = cts[0].L, Fraction(scale)
    q1, q2 = ctx.q[L - 1], ctx.q[L - 2]
    s3 = s ** 3 / (q1 * q2)
    out = ctx.poly3(keys, cts, _round_half_up(a3 * q1), _round_half_up(a1 * s * s), _round_half_up(a0 * s3), float(s * s))
    return out, s3


class Pipeline:
    """layers: list of dicts
         {"op": "conv", "conv": {BS, C_in, H, W, C_out, K, stride, pad, [depthwise], [M]}, "S": S, "w": ndarray,
          ["factored": True]}                  factored: weights as integer multipliers + mask plaintexts (R2.9c, ch = 1)
         {"op": "square"}                      x -> x^2, relinearised and rescaled (one level)
         {"op": "pool"}                        2x2 sum-pool by fragment selection (S halves; factor 1/4 goes into the next w)
         {"op": "compress", "v": v}            AAC batch-group compaction after a channel-reducing conv (v valid positions);
                                               the next conv's dict carries seg_v = v (segmented layout, R2.11b)
         {"op": "fc", "fc": {...}, "w": ndarray[n_out][n_in]}     plain-diagonal fully connected layer
    """

    def __init__(self, ctx, layers, L0=None):
        self.ctx, self.layers, self.L0 = ctx, layers, L0 or ctx.n_q
        self.plan, self.steps, self.need_relin = [], set(), False
        L = self.L0
        for ly in layers:
            if ly["op"] == "conv":
                conv = ctx.conv_desc(S=ly["S"], **ly["conv"])
                lay = ctx.layout_plan(conv)
                self.steps.update(lay.steps())
                self.plan.append(dict(op="conv", conv=conv, lay=lay, L=L, w=ly.get("w"), factored=bool(ly.get("factored"))))
                L -= 1
            elif ly["op"] == "fc":
                fc = ctx.fc_desc(**ly["fc"])
                info = ctx.fc_plan(fc)
                self.steps.update(info["rot_steps"])
                self.plan.append(dict(op="fc", fc=fc, info=info, L=L, w=ly.get("w")))
                L -= 1
            elif ly["op"] == "square":
                self.need_relin = True
                self.plan.append(dict(op="square", L=L))
                L -= 1
            elif ly["op"] == "poly3":
                self.need_relin = True
                self.plan.append(dict(op="poly3", L=L, coef=ly.get("coef", POLY3)))
                L -= 2
            elif ly["op"] == "pool":
                self.plan.append(dict(op="pool", L=L))
            elif ly["op"] == "compress":
                # AAC (R2.11): the previous conv left v of ch_phys channel positions valid; the
                # ciphertexts of ch_phys / v consecutive batch groups are compacted into one (segmented layout, R2.11b)
                prev = next(p for p in reversed(self.plan) if p["op"] == "conv")["lay"]
                v, n = int(ly["v"]), ctx.n
                if prev.seg != 1 or prev.ch % v or prev.G_out != 1:
                    raise ValueError("compress needs a plain layout whose single output group has v | ch valid positions")
                per = prev.ch // v
                rots = [(n - sg * v * prev.cs) % n for sg in range(per)]
                self.steps.update(r for r in rots if r)
                self.plan.append(dict(op="compress", L=L, v=v, per=per, rots=rots, frags=int(prev.S_out) ** 2, BG=int(prev.BG)))
            else:
                raise ValueError(ly["op"])
        self.L_out = L
        self.keys, self.weights = None, []

    def counts(self, lazy_relin=False):
        """(linear layers, key-switched rotations, relinearisations, PMults) of one forward pass."""
        lin = rot = relin = pm = 0
        n_ct = None
        for li, p in enumerate(self.plan):
            if p["op"] == "conv":
                lin += 1
                rot += p["lay"].n_inner_rot + p["lay"].n_outer_rot
                pm += p["lay"].n_pmult
                n_ct = p["lay"].n_out_ct
            elif p["op"] == "fc":
                lin += 1
                rot += p["info"]["n_rot"]
                pm += p["info"]["n_pmult"]
                n_ct = p["info"]["n_out_ct"]
            elif p["op"] == "square":
                pooled = lazy_relin and li + 1 < len(self.plan) and self.plan[li + 1]["op"] == "pool"
                relin += n_ct // 4 if pooled else n_ct
            elif p["op"] == "pool":
                n_ct //= 4
            elif p["op"] == "compress":
                n_t = -(-p["BG"] // p["per"])
                rot += p["frags"] * (p["BG"] - n_t)  # every source but the first of each output is rotated once
                n_ct = n_t * p["frags"]
        return lin, rot, relin, pm

    def setup(self, key_seed, encode_weight=None):
        """Generate keys for exactly the rotation amounts the layers need and encode every weight plaintext.
        encode_weight(plan_entry) -> int64 coefficient array, to start from pre-encoded integers (A7)."""
        ctx = self.ctx
        self.keys = ctx.keygen(key_seed, sorted(self.steps), want_relin=self.need_relin)
        self.weights = []
        for p in self.plan:
            if p["op"] == "conv":
                if p["factored"]:  # value x mask weights of a one-channel-per-ciphertext layout (R2.9c)
                    self.weights.append(ctx.conv_weights_factored(p["conv"], p["lay"], p["w"], p["L"]))
                elif encode_weight is not None:
                    self.weights.append(ctx.conv_weights_from_coeffs(p["conv"], p["lay"], encode_weight(p), p["L"]))
                else:
                    self.weights.append(ctx.conv_weights(p["conv"], p["lay"], p["w"], p["L"]))
            elif p["op"] == "fc":
                if encode_weight is not None:
                    self.weights.append(ctx.fc_weights_from_coeffs(p["fc"], encode_weight(p), p["L"]))
                else:
                    self.weights.append(ctx.fc_weights(p["fc"], p["w"], p["L"]))
            else:
                self.weights.append(None)
        return self.keys

    def encrypt_input(self, x, enc_seed0):
        """Algorithm 1 on host x[BS][C][H][W] for the first layer; ciphertext order [bg][g][u][v].  A network that starts
        with a fully connected layer takes x[BS][n_in] (token embeddings, R2.13); order [bg][c]."""
        p = self.plan[0]
        if p["op"] == "fc":
            ctx, cts = self.ctx, []
            per_bg = p["info"]["n_in_ct"] // p["info"]["BG"]
            for bg in range(p["info"]["BG"]):
                for c in range(per_bg):
                    cts.append(ctx.encrypt(self.keys, ctx.fc_encode_input(p["fc"], x, c, bg, p["L"]), enc_seed0 + len(cts)))
            return cts
        conv, lay, ctx = p["conv"], p["lay"], self.ctx
        cts = []
        for bg in range(lay.BG):
            for g in range(lay.G_in):
                for u in range(lay.S):
                    for v in range(lay.S):
                        pt = ctx.encode_fragment(conv, lay, x, u, v, g, bg, p["L"])
                        cts.append(ctx.encrypt(self.keys, pt, enc_seed0 + len(cts)))
        return cts

    def forward(self, cts, trace=None, scale=None, lazy_relin=False, on_layer=None):
        """scale: exact rational scale of the inputs (default: the context's 2^log2_scale); only poly3 needs it.
        lazy_relin: a square directly followed by a pool runs as ONE step, fenc_square_sum_relin over the four fragments of
        every pooled output (one relinearisation instead of four, R2.12c); the trace then holds the pooled
        ciphertexts at both positions.  on_layer(index, plan entry): called after each layer's calls are enqueued."""
        ctx = self.ctx
        S = None
        sc = Fraction(cts[0].scale) if scale is None else Fraction(scale)
        for li, (p, w) in enumerate(zip(self.plan, self.weights)):
            fused_prev = lazy_relin and p["op"] == "pool" and li > 0 and self.plan[li - 1]["op"] == "square"
            if fused_prev:
                pass  # done together with the square before it
            elif lazy_relin and p["op"] == "square" and li + 1 < len(self.plan) and self.plan[li + 1]["op"] == "pool":
                cts = ctx.square_sum_pool(self.keys, cts, S)
                sc = sc * sc / ctx.q[p["L"] - 1]
                S //= 2
            elif p["op"] == "conv":
                cts = ctx.hconv(self.keys, p["conv"], p["lay"], w, cts, do_rescale=True)
                S = p["lay"].S_out  # weights at s_w = q_{L-1} and one rescale: the scale is unchanged (A14)
            elif p["op"] == "fc":
                cts = ctx.fc(self.keys, p["fc"], w, cts, do_rescale=True)
                S = 1
            elif p["op"] == "square":
                cts = ctx.square_relin(self.keys, cts)
                sc = sc * sc / ctx.q[p["L"] - 1]
            elif p["op"] == "poly3":
                cts, sc = poly3_activation(ctx, self.keys, cts, sc, p["coef"])
            elif p["op"] == "pool":
                cts = ctx.sum_pool(cts, S)
                S //= 2
            elif p["op"] == "compress":
                # sources ordered [bg][fragment]; output t gathers batch groups t*per .. t*per + per - 1 of each fragment
                fr_, per, n_t = p["frags"], p["per"], -(-p["BG"] // p["per"])
                terms = [(t * fr_ + f, bg * fr_ + f, p["rots"][bg % per]) for t in range(n_t) for f in range(fr_)
                         for bg in range(t * per, min((t + 1) * per, p["BG"]))]
                cts = ctx.compress(self.keys, cts, terms, n_t * fr_)
            if trace is not None:
                trace.append(cts)
            if on_layer is not None and not fused_prev:
                on_layer(li, p)
        return cts

"""bench.py -- measures BASELINE.json's metric on one B200 (or N independent replicas).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl ours|reference]

A step = one pass of the whole hot path over one batch of synthetic input (workloads.py).  The default workload is
BASELINE config 4 (MobileNet-v1-shaped ImageNet layers, N=2^16, 30x50b + 5x60b, the largest single-GPU configuration);
the same run also times, under its own clock samples, the config-5 rotation point L=24 / dnum=3 (plain and hoisted),
the config-2 LeNet-5 step and a config-3 layer, printed as `extras` of the ONE JSON line.
`value` is the whole-job throughput with inputs resident in HBM; `e2e` is the same metric through the C-ABI calls with
HOST buffers (ciphertext limbs imported from / exported to pinned host memory inside the timed region).  `roofline` is
for the dominant kernel class, timed live with CUDA events by the library's profile hooks; `cpu_baseline` times the CPU
oracle as it stands, on the SAME operation graph (hoisted rotations, factored weights, lazy relinearisation ...)."""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
import workloads as wl  # noqa: E402

METRIC = "encrypted conv layers/s & key-switched rotations/s; HBM GB/s vs B200 peak"
HBM_BYTES = 180e9  # B200 HBM3e capacity the maximum batch is sized for (BASELINE.json north_star)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p)), "measured (MEASURED_PEAKS.json)"
    return {"hbm_gbs": 6650.0}, "fallback (B200_PROFILING.md)"


def max_over_ranks(value, world, device):
    """max over all ranks of a per-rank scalar (multi-GPU numbers are the slowest rank's; replicas only)."""
    if world <= 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    torch.distributed.all_reduce(t, op=torch.distributed.ReduceOp.MAX)
    return float(t.item())


def aggregate(units_per_rank, world, seconds):
    """whole-job throughput: every rank processed units_per_rank in `seconds` (the max over ranks)."""
    return world * units_per_rank / seconds


def host_info():
    model = "unknown"
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name"):
                model = ln.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    return {"nproc": os.cpu_count(), "cpu_model": model}


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, device):
        self.rows, self.proc, self.device, self.first = [], None, device, 0

    def mark(self):
        """samples from here on belong to the timed region"""
        self.first = len(self.rows)

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.device), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
            t_wait = time.time()
            while not self.rows and time.time() - t_wait < 3.0:
                time.sleep(0.05)
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def summary(self, upto=None):
        """clocks over the samples since mark() (the sampler keeps running)"""
        rows = self.rows[self.first:upto]
        sm = [float(r[0]) for r in rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) > 2 + i and r[2 + i].lower().startswith("active") for r in rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(sm)}

    def stop(self):
        if self.proc:
            self.proc.terminate()
            self.proc = None


def timed_clocks(sampler, fn):
    """run fn() with the sampler marking its region; returns (fn's result, clocks of the region)"""
    sampler.mark()
    out = fn()
    time.sleep(0.12)  # let the last sample of the region arrive
    return out, sampler.summary()


# ------------------------------------------------------------------------------------------------ workloads
FC_BSGS = 0  # baby-step count of the fully connected layers: 0 = library's choice (R2.12b), 1 = plain diagonals (--plain-fc)
CONV_BSGS = 0  # baby steps over the conv layers' channel diagonals: 0 = fewest rotations (R2.9d), 1 = plain (--plain-conv)


def lenet_layers(BS, seed, upto="fc"):
    """BASELINE config 2: LeNet-5-shaped network on MNIST-shaped input (D2).  S=4 for conv1
    (the paper's best LeNet block size); pooling halves S; the 1/4 pool factors live in the next weights."""
    rng = np.random.default_rng(seed)
    w1 = rng.normal(0, 0.1, (6, 1, 5, 5))
    w2 = rng.normal(0, 0.1, (16, 6, 5, 5)) * 0.25
    layers = [
        {"op": "conv", "conv": dict(BS=BS, C_in=1, H=28, W=28, C_out=6, K=5, stride=1, pad=2), "S": 4, "w": w1},
        {"op": "square"}, {"op": "pool"},
        {"op": "conv", "conv": dict(BS=BS, C_in=6, H=14, W=14, C_out=16, K=5, stride=1, pad=0, M=16), "S": 2, "w": w2},
        {"op": "square"}, {"op": "pool"},
    ]
    if upto == "fc":
        f1 = rng.normal(0, 0.1, (120, 400)) * 0.25
        f2 = rng.normal(0, 0.1, (84, 120))
        f3 = rng.normal(0, 0.1, (10, 84))
        layers += [
            {"op": "fc", "fc": dict(BS=BS, n_in=400, n_out=120, in_C=16, in_H=5, in_W=5, in_M=8, bsgs=FC_BSGS), "w": f1},
            {"op": "fc", "fc": dict(BS=BS, n_in=120, n_out=84, in_M=8, bsgs=FC_BSGS), "w": f2},
            {"op": "fc", "fc": dict(BS=BS, n_in=84, n_out=10, in_M=8, bsgs=FC_BSGS), "w": f3},
        ]
    x = rng.uniform(0, 1, (BS, 1, 28, 28))
    return layers, x


MOBILENET_CONVS = [  # BASELINE config 4: frames 256 -> 128 -> 64, S = 8 -> 4 -> 2, m = 32 throughout
    (dict(C_in=3, H=224, W=224, C_out=32, K=3, stride=2, pad=1), 8),
    (dict(C_in=32, H=112, W=112, C_out=32, K=3, stride=1, pad=1, depthwise=True), 4),
    (dict(C_in=32, H=112, W=112, C_out=64, K=1, stride=1, pad=0), 4),
    (dict(C_in=64, H=112, W=112, C_out=64, K=3, stride=2, pad=1, depthwise=True), 4),
    (dict(C_in=64, H=56, W=56, C_out=128, K=1, stride=1, pad=0), 2),
]


def mobilenet_layers(BS, seed, factored=True):
    """BASELINE config 4: the five MobileNet-v1-shaped layers, chained (each at the level the previous one leaves, A20).
    BS = 32 fills a ciphertext's batch dimension (B = 32, ch = 1: the large-batch case), so the weights
    are factored into integer multipliers and mask plaintexts (R2.9c).  Weights N(0, 0.05), inputs U[-1, 1]."""
    rng = np.random.default_rng(seed)
    layers = []
    for kw, S in MOBILENET_CONVS:
        cw = 1 if kw.get("depthwise") else kw["C_in"]
        w = rng.normal(0.0, 0.05, (kw["C_out"], cw, kw["K"], kw["K"]))
        layers.append({"op": "conv", "conv": dict(BS=BS, **kw), "S": S, "w": w, "factored": factored})
    x = rng.uniform(-1, 1, (BS, 3, 224, 224))
    return layers, x


def conv_layers(name, seed, kaiming=False):
    """one encrypted conv layer of a BASELINE config at the top level (reading A20), planner-selected S."""
    kw = wl.CONVS[name]
    x, w = wl.conv_inputs(seed, kw, kaiming=kaiming)
    return [{"op": "conv", "conv": dict(kw, bsgs=CONV_BSGS), "S": 0, "w": w}], x


def resnet_chain_layers(seed):
    """BASELINE config 3 chained: conv 16->16 - act - conv 16->32 /2 - act - conv 32->64 /2 with
    S = 4 -> 2 -> 1 so both strides are fragment drops; degree-3 activation 0.5 + 0.197x - 0.004x^3."""
    rng = np.random.default_rng(seed)
    shapes = [(wl.CONVS["resnet_16_16"], 4), (wl.CONVS["resnet_16_32_s2"], 4), (wl.CONVS["resnet_32_64_s2"], 2)]
    layers = []
    for i, (kw, S) in enumerate(shapes):
        std = np.sqrt(2.0 / (kw["C_in"] * kw["K"] ** 2))
        layers.append({"op": "conv", "conv": dict(kw, bsgs=CONV_BSGS), "S": S, "w": rng.normal(0.0, std, (kw["C_out"], kw["C_in"], kw["K"], kw["K"]))})
        if i < 2:
            layers.append({"op": "poly3"})
    return layers, rng.uniform(-1, 1, (1, 16, 32, 32))


def bottleneck_layers(seed, aac):
    """A Table-X-shaped bottleneck at config 3's parameters: 64 -> 8 -> 128 channels on
    32 x 32 maps, four requests of one image (B_cap = 1: 32 channel positions per ciphertext, 8 valid after the reducing
    1x1 layer).  aac: the four 25 %-full ciphertexts are compacted into one (fenc_compress, R2.11) and the 3x3 expansion
    runs on the segmented layout (R2.11b); otherwise it runs on the four sparse ciphertexts."""
    rng = np.random.default_rng(seed)
    red = dict(BS=4, C_in=64, H=32, W=32, C_out=8, K=1, stride=1, pad=0, B_cap=1)
    exp = dict(BS=4, C_in=8, H=32, W=32, C_out=128, K=3, stride=1, pad=1, B_cap=1)
    w1 = rng.normal(0.0, np.sqrt(2.0 / 64), (8, 64, 1, 1))
    w2 = rng.normal(0.0, np.sqrt(2.0 / 72), (128, 8, 3, 3))
    layers = [{"op": "conv", "conv": dict(red, bsgs=CONV_BSGS), "S": 1, "w": w1}]
    if aac:
        layers += [{"op": "compress", "v": 8}, {"op": "conv", "conv": dict(exp, seg_v=8, bsgs=CONV_BSGS), "S": 1, "w": w2}]
    else:
        layers += [{"op": "conv", "conv": dict(exp, bsgs=CONV_BSGS), "S": 1, "w": w2}]
    return layers, rng.uniform(-1, 1, (4, 64, 32, 32))


def transformer_linear_layers(seed):
    """One linear layer of a BERT-base-shaped encoder block on fragment-encoded token embeddings (the
    Transformer extension; R2.13): 128 tokens, E = 768 -> 768, sub-blocks of S = 3 coordinates, so B = 128 tokens
    x P = 256 positions fill the 2^15 slots exactly (E / S = P) and the layer takes 3 input and 3 output ciphertexts.
    Weights N(0, 1/sqrt(E)), embeddings U[-1, 1]."""
    rng = np.random.default_rng(seed)
    w = rng.normal(0.0, 768 ** -0.5, (768, 768))
    fc = dict(BS=128, n_in=768, n_out=768, in_M=1, frag_in=3, frag_out=3, bsgs=FC_BSGS)
    return [{"op": "fc", "fc": fc, "w": w}], rng.uniform(-1, 1, (128, 768))


WORKLOADS = {
    # name: (PARAMS key, builder(batch, seed) -> (layers, x), description, images per ciphertext batch group or None)
    "cfg4_mobilenet": ("cfg4", lambda bs, seed: mobilenet_layers(32, seed),
                       "BASELINE config 4: MobileNet-v1-shaped ImageNet layers conv 3->32/2, dw 32, pw 32->64, dw 64/2, pw 64->128, "
                       "chained, N=2^16, 30x50b+5x60b, dnum=6; batch groups of 32 images (B=32, ch=1), factored weights (R2.9c)", 32),
    "cfg2_lenet5_convstage": ("cfg2", lambda bs, seed: lenet_layers(bs, seed, upto="conv"),
                              "BASELINE config 2, conv stage: conv1-x^2-pool-conv2-x^2-pool, N=2^14, 8x40b+2x60b, dnum=4", None),
    "cfg2_lenet5": ("cfg2", lambda bs, seed: lenet_layers(bs, seed, upto="fc"),
                    "BASELINE config 2: LeNet-5-shaped network, N=2^14, 8x40b+2x60b, dnum=4", None),
    # single layers (parity-test configurations, timed for the record; --batch is ignored: BS = 1 as in BASELINE.json)
    "cfg1_conv1": ("cfg1", lambda bs, seed: conv_layers("lenet_conv1", seed),
                   "BASELINE config 1: LeNet conv1-shaped layer, N=2^13, 3x40b+1x60b, dlen=1 (A1), batch 1", None),
    "cfg3_conv_16_16": ("cfg3", lambda bs, seed: conv_layers("resnet_16_16", seed, True),
                        "BASELINE config 3: ResNet-20 3x3 16->16 layer, N=2^16, 24x50b+4x60b, dnum=6, batch 1", None),
    "cfg3_conv_16_32_s2": ("cfg3", lambda bs, seed: conv_layers("resnet_16_32_s2", seed, True),
                           "BASELINE config 3: ResNet-20 3x3 16->32 stride 2, N=2^16, batch 1", None),
    "cfg3_conv_32_64_s2": ("cfg3", lambda bs, seed: conv_layers("resnet_32_64_s2", seed, True),
                           "BASELINE config 3: ResNet-20 3x3 32->64 stride 2, N=2^16, batch 1", None),
    "cfg3_chain": ("cfg3", lambda bs, seed: resnet_chain_layers(seed),
                   "BASELINE config 3 chained: conv 16->16 (S=4) - poly3 - conv 16->32/2 - poly3 - conv 32->64/2, N=2^16, batch 1", None),
    "cfg3_bottleneck_plain": ("cfg3", lambda bs, seed: bottleneck_layers(seed, False),
                              "Table-X-shaped bottleneck 64 -> 8 -> 128 (1x1, 3x3) on 32x32, 4 requests, N=2^16, WITHOUT compression", None),
    "cfg3_bottleneck_aac": ("cfg3", lambda bs, seed: bottleneck_layers(seed, True),
                            "the same bottleneck WITH Arch-aware compression (4 sparse ciphertexts -> 1) and the segmented consumer", None),
    "ext_transformer_linear": ("cfg3", lambda bs, seed: transformer_linear_layers(seed),
                               "Transformer extension (PAPER.md:462-464): one 768 -> 768 projection of 128 fragment-encoded token embeddings "
                               "(S = 3), N=2^16, 24x50b+4x60b, dnum=6", None),
    "cfg5_rotsweep": (None, None, "BASELINE config 5: rotation / key-switch sweep", None),
    "cfg5_rotsweep_hoisted": (None, None, "BASELINE config 5 with hoisted rotations (8 amounts per decomposition)", None),
    "cfg3_compress": (None, None, "AAC compress micro-benchmark at config 3's parameters", None),
}
DEFAULT_WORKLOAD = "cfg4_mobilenet"
DEFAULT_BATCH = {"cfg4_mobilenet": 64, "cfg2_lenet5": 128, "cfg2_lenet5_convstage": 128}


# ------------------------------------------------------------------------------------------------ config 5: rotation sweep
def sweep_point(L, dnum, hoisted, n_ct=64, n_steps=32):
    """One point of BASELINE config 5 at N=2^16 (reading A2: k = dlen = ceil(L/dnum)): n_ct ciphertexts with uniform-random
    limbs, n_steps distinct seeded amounts; plain: every amount is one batched fenc_rotate over the n_ct ciphertexts;
    hoisted: fenc_rotate_hoisted over (n_ct ciphertexts x 8 amounts) per call, one decomposition per ciphertext and
    call (R2.7b -- the shape of a 3x3 convolution's 8 inner rotations)."""
    import torch
    import paper_2606_16359_b200 as fenc
    peaks, _ = measured_peaks()
    pr = wl.sweep_params(L, dnum)
    ctx = fenc.Context(**pr)
    N, k, dlen = ctx.N, ctx.n_p, ctx.dlen
    beta = -(-L // dlen)
    steps = wl.rotation_steps(5000 + L * 10 + dnum, n_steps, ctx.n)
    keys = ctx.keygen(5, steps)
    cts = [ctx.ct_import(wl.random_ct_limbs(100 * L + i, ctx.q, L, N)) for i in range(n_ct)]

    def run():
        if hoisted:
            for at in range(0, n_steps, 8):
                ctx.rotate_hoisted(keys, cts, steps[at:at + 8])
        else:
            for r in steps:
                ctx.rotate(keys, cts, [r] * n_ct)

    for _ in range(3):  # warm-up: three batches of each kind
        (ctx.rotate_hoisted(keys, cts, steps[:8]) if hoisted else ctx.rotate(keys, cts, [steps[0]] * n_ct))
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ctx.launch_count(reset=True)
    e0.record()
    run()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    rots = n_ct * n_steps
    # algorithmic bytes per rotation: ciphertext in + out, key once per batch of n_ct ciphertexts
    b_alg = 2 * (2 * L * N * 8) + 2 * beta * (L + k) * N * 8 / n_ct
    if hoisted:  # input read once per 8 rotations, output once per rotation, key once per n_ct ciphertexts
        b_alg = 2 * L * N * 8 * (1 + 1 / 8) + 2 * beta * (L + k) * N * 8 / n_ct
    gbs = rots * b_alg / (ms * 1e-3) / 1e9
    pt = {"L": L, "dnum": dnum, "dlen": dlen, "k": k, "beta": beta, "ntt_per_rot": beta * (L + k) + 2 * k + 2 * L,
          "rot_per_s": round(rots / (ms * 1e-3), 1), "us_per_rot": round(ms * 1e3 / rots, 2), "alg_GBps": round(gbs, 1),
          "hbm_frac": round(gbs / peaks["hbm_gbs"], 4), "launches": ctx.launch_count(), "ciphertexts": n_ct, "amounts": n_steps}
    del cts, keys
    ctx.close()
    torch.cuda.empty_cache()
    return pt


def run_rotsweep(args, hoisted=False):
    """BASELINE config 5: the whole sweep (or the points selected by --sweep-L / --sweep-dnum)."""
    peaks, peak_src = measured_peaks()
    points = [sweep_point(L, dnum, hoisted, args.sweep_cts, args.sweep_steps)
              for L in (args.sweep_L or (4, 8, 16, 24, 36)) for dnum in (args.sweep_dnum or (1, 2, 3, 4))]
    ref = ([p for p in points if p["L"] == 24 and p["dnum"] == 3] or points)[0]
    return {"metric": METRIC, "value": ref["rot_per_s"], "unit": "key-switched rotations/s", "n_gpus": 1, "steps": args.sweep_steps,
            "warmup": 3, "ms_per_step": round(1e3 * args.sweep_cts / ref["rot_per_s"], 4), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "u64", "data": "synthetic",
            "config": {"workload": "cfg5_rotsweep_hoisted" if hoisted else "cfg5_rotsweep",
                       "description": "BASELINE config 5: N=2^16, %d cts x %d amounts per point; value quoted at L=%d, dnum=%d" % (
                           args.sweep_cts, args.sweep_steps, ref["L"], ref["dnum"])
                       + ("; hoisted form (R2.7b), 8 amounts per decomposition" if hoisted else ""), "peak_source": peak_src, "hbm_peak_GBps": peaks["hbm_gbs"]},
            "points": points}


def run_compress(args):
    """AAC compress micro-benchmark (Table X shapes): BG sparse ciphertexts whose valid
    channel positions are [0, v) of ch are merged into BG*v/ch dense ones (canonical batch-group compaction, R2.11),
    maskless and masked split-scale, at config 3's parameters."""
    import torch
    import paper_2606_16359_b200 as fenc
    ctx = fenc.Context(**wl.PARAMS["cfg3"])
    n, L = ctx.n, ctx.n_q
    rows = []
    rng = np.random.default_rng(77)
    for ch, v, n_src in ((8, 2, 4), (32, 8, 64), (32, 2, 64), (128, 8, 64)):
        cs, per = n // ch, ch // v
        terms = [(i // per, i, (n - (i % per) * v * cs) % n) for i in range(n_src)]
        n_out = -(-n_src // per)
        steps = sorted({r for _, _, r in terms if r})
        keys = ctx.keygen(9, steps)
        srcs = []
        for i in range(n_src):
            z = np.zeros(n)
            z[: v * cs] = rng.uniform(-1, 1, v * cs)
            srcs.append(ctx.encrypt(keys, ctx.encode_slots(z, L), 400 + i))
        m = np.zeros(n)
        m[: v * cs] = 1.0
        mask = ctx.encode_slots(m, L, float(ctx.q[L - 1]))
        for mode in ("maskless", "masked_split_scale"):
            kw = dict(mask=mask, do_rescale=True) if mode != "maskless" else {}
            for _ in range(3):
                ctx.compress(keys, srcs, terms, n_out, **kw)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(args.steps):
                out = ctx.compress(keys, srcs, terms, n_out, **kw)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / args.steps
            rows.append({"ch": ch, "valid": v, "sources": n_src, "outputs": n_out, "mode": mode, "rotations": len([t for t in terms if t[2]]),
                         "ms": round(ms, 3), "rot_per_s": round(len([t for t in terms if t[2]]) / (ms * 1e-3), 1),
                         "slot_util_before": v / ch, "slot_util_after": min(1.0, n_src * v / (ch * n_out)), "level_out": out[0].L})
        del srcs, keys
    ctx.close()
    ref = rows[2]
    return {"metric": METRIC, "value": ref["rot_per_s"], "unit": "key-switched rotations/s", "n_gpus": 1, "steps": args.steps, "warmup": 3,
            "ms_per_step": ref["ms"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u64", "data": "synthetic",
            "config": {"workload": "cfg3_compress", "description": "AAC compress (fenc_compress) on bottleneck-shaped sources, N=2^16, "
                       "24x50b+4x60b; value quoted for ch=32, v=8, 64 sources, maskless"}, "points": rows}


# ------------------------------------------------------------------------------------------------ network workloads
def counted_layers(layers, n_groups):
    """(layers counted by the line's `value`, its unit): the encrypted conv layers; a network without any (the Transformer
    extension's linear layer) counts its fully connected layers and says so in the unit"""
    n = sum(1 for ly in layers if ly["op"] == "conv")
    if n:
        return n * n_groups, "encrypted conv layers/s"
    return sum(1 for ly in layers if ly["op"] == "fc") * n_groups, "encrypted linear layers/s"


class NetBench:
    """One network workload set up on the GPU: context, keys, weights, encrypted inputs resident in HBM.
    Workloads with `per_group` images per ciphertext batch group (config 4) hold batch / per_group independent input sets
    and evaluate them one after the other (batch groups are independent); the others hold one set."""

    def __init__(self, args, name, rank, dev, batch=None):
        import paper_2606_16359_b200 as fenc
        from paper_2606_16359_b200.pipeline import Pipeline
        self.name, self.args = name, args
        pkey, builder, self.desc, per_group = WORKLOADS[name]
        self.pkey = pkey
        seed = 2000 + rank
        batch = batch or DEFAULT_BATCH.get(name, 1)
        self.layers, x = builder(batch, seed)
        self.ctx = ctx = fenc.Context(device=dev, **wl.PARAMS[pkey])
        self.hoist = not args.no_hoist
        ctx.set_hoisting(self.hoist)  # inner rotations share one decomposition per input ciphertext (R2.7b)
        self.pipe = pipe = Pipeline(ctx, self.layers)
        pipe.setup(key_seed=seed)
        self.lazy = not args.eager_relin  # x^2 + pool with one relinearisation per pooled output (R2.12c)
        if per_group:
            n_groups = max(1, batch // per_group)
            rng = np.random.default_rng(seed + 1)
            self.groups = [pipe.encrypt_input(x if g == 0 else rng.uniform(-1, 1, x.shape), enc_seed0=10 * seed + 100000 * g)
                           for g in range(n_groups)]
            self.batch = per_group * n_groups
        else:
            self.groups = [pipe.encrypt_input(x, enc_seed0=10 * seed)]
            self.batch = int(self.layers[0][self.layers[0]["op"]]["BS"])
        self.n_lin, self.n_rot, self.n_relin, self.n_pm = (v * len(self.groups) for v in pipe.counts(lazy_relin=self.lazy))
        self.n_conv, self.unit = counted_layers(self.layers, len(self.groups))
        ctx.sync()
        self.setup_bytes = ctx.device_bytes()

    def step(self):
        return [self.pipe.forward(g, lazy_relin=self.lazy) for g in self.groups]

    def close(self):
        import torch
        self.groups = None
        self.pipe = None
        self.ctx.close()
        torch.cuda.empty_cache()


def time_resident(nb, steps, warmup, world, sampler, profile_range=False):
    """W warm-up steps, then exactly K steps between CUDA events on the stream the library launches on, barrier and
    synchronize on both sides, max over ranks."""
    import torch

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    out = None
    torch.cuda.reset_peak_memory_stats()
    for _ in range(warmup):
        out = None
        out = nb.step()
    barrier()
    sampler.mark()
    nb.ctx.launch_count(reset=True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if profile_range:  # for `ncu --profile-from-start off`: only the timed steps are captured
        torch.cuda.profiler.start()
    e0.record()
    for _ in range(steps):
        out = None
        out = nb.step()
    e1.record()
    barrier()
    if profile_range:
        torch.cuda.profiler.stop()
    time.sleep(0.12)
    ms = max_over_ranks(e0.elapsed_time(e1), world, "cuda")
    launches = nb.ctx.launch_count()
    clocks = sampler.summary()
    peak = torch.cuda.max_memory_allocated()
    in_bytes = sum(nb.ctx.ct_bytes(c) for c in nb.groups[0])
    out_bytes = sum(nb.ctx.ct_bytes(c) for c in out[0])
    return {"ms_per_step": ms / steps, "launches": int(launches), "clocks": clocks, "peak_bytes": int(peak),
            "group_in_bytes": int(in_bytes), "group_out_bytes": int(out_bytes)}, out


def net_summary(nb, t, world):
    s = t["ms_per_step"] * 1e-3
    d = {"workload": nb.name, "batch": nb.batch, "ms_per_step": round(t["ms_per_step"], 4),
         "images_per_s": round(world * nb.batch / s, 2), "conv_layers_per_s": round(world * nb.n_conv / s, 3),
         "linear_layers_per_s": round(world * nb.n_lin / s, 3), "rotations_per_s": round(world * (nb.n_rot + nb.n_relin) / s, 1),
         "gpu_launches": t["launches"], "clocks": t["clocks"], "peak_device_bytes": t["peak_bytes"],
         "counts_per_step": {"conv_layers": nb.n_conv if "conv" in nb.unit else 0, "linear_layers": nb.n_lin, "rotations": nb.n_rot,
                             "relinearisations": nb.n_relin, "pmults": nb.n_pm}}
    return d


def per_kernel_profile(nb, steps):
    """a separate pass with the library's CUDA-event hooks on the same stream: {class: (ms, launches, bytes, ops)} per step"""
    ctx = nb.ctx
    ctx.profile_enable(True)
    t0 = time.perf_counter()
    for _ in range(steps):
        out = nb.step()
        del out
    prof = ctx.profile_read()
    wall_ms = (time.perf_counter() - t0) * 1e3 / steps
    ctx.profile_enable(False)
    return prof, wall_ms


def per_layer_profile(nb):
    """--per-layer: one step with the library's per-class CUDA-event hooks read out after every layer (the read-out
    synchronises the stream, so the layers do not overlap: a breakdown, not a throughput)."""
    ctx = nb.ctx
    rows = []
    ctx.profile_enable(True)
    for gi, g in enumerate(nb.groups):
        def done(li, p, gi=gi):
            prof = ctx.profile_read()
            conv = p.get("conv")
            name = p["op"] + ("" if conv is None else " %d->%d k%d s%d%s L=%d" % (conv.C_in, conv.C_out, conv.K, conv.stride, " dw" if conv.depthwise else "", p["L"]))
            rows.append({"group": gi, "layer": li, "op": name, "ms": round(sum(v[0] for v in prof.values()), 3),
                         "per_kernel_ms": {k: round(v[0], 3) for k, v in sorted(prof.items(), key=lambda kv: -kv[1][0])}})
        out = nb.pipe.forward(g, lazy_relin=nb.lazy, on_layer=done)
        del out
    ctx.profile_enable(False)
    return rows


NTT_CLASSES = ("intt_rowpass", "intt_colpass", "ntt_colpass", "ntt_colpass_bconv", "ntt_rowpass", "ntt_rows_keymac", "ntt_rows_divide")


def roofline_of(nb, prof, prof_steps, prof_ms):
    """`roofline` object of the JSON line for the class with the most time; per-class table beside it.
    NTT-carrying classes: the nearer of the HBM roof and the measured butterfly ceiling; smac: the measured ceiling of its
    own exact fp64 multiply-accumulate (its second counter is multiply-accumulates); everything else: HBM."""
    ctx = nb.ctx
    peaks, peak_src = measured_peaks()
    imad_peak, bfly_peak = ctx.measure_alu_peak()
    smac_peak = ctx.measure_smac_peak() if "smac" in prof and ctx.q[0] < (1 << 50) else None
    per_kernel, best = {}, None
    tot = sum(v[0] for v in prof.values())
    for k, v in sorted(prof.items(), key=lambda kv: -kv[1][0]):
        ms, cnt, nbytes, ops = v
        gbs = nbytes / (ms * 1e-3) / 1e9
        row = {"ms_per_step": round(ms / prof_steps, 4), "launches_per_step": cnt // prof_steps, "share_of_step": round(ms / tot, 4),
               "alg_GBps": round(gbs, 1), "hbm_frac": round(gbs / peaks["hbm_gbs"], 4)}
        if k in NTT_CLASSES and ops:
            row["Gbutterflies_per_s"] = round(ops / (ms * 1e-3) / 1e9, 1)
            row["alu_frac"] = round(ops / (ms * 1e-3) / bfly_peak, 4)
        if k == "smac" and smac_peak:
            row["Gmulacc_per_s"] = round(ops / (ms * 1e-3) / 1e9, 1)
            row["alu_frac"] = round(ops / (ms * 1e-3) / smac_peak, 4)
        per_kernel[k] = row
        if best is None:
            best = k
    t_ms, t_cnt, t_bytes, t_ops = prof[best]
    row = per_kernel[best]
    if row.get("alu_frac", 0) >= row["hbm_frac"]:
        smac = best == "smac"
        roofline = {"bound": "alu", "kernel": best, "achieved": row["Gmulacc_per_s" if smac else "Gbutterflies_per_s"],
                    "peak": round((smac_peak if smac else bfly_peak) / 1e9, 2),
                    "unit": "G modular multiply-accumulates/s" if smac else "G modular butterflies/s", "frac": row["alu_frac"], "traffic": None,
                    "peak_source": ("measured live: this kernel's exact fp64 multiply-accumulate on registers only, all SMs (fenc_measure_smac_peak)"
                                    if smac else "measured live: register-only butterflies of this library on all SMs, the faster of the integer "
                                    "Shoup and the fp64 one (fenc_measure_alu_peak)") + "; 32-bit IMAD peak %.2f T lane-ops/s" % (imad_peak / 1e12),
                    "ops_per_launch": t_ops / t_cnt, "hbm_frac_of_same_kernel": row["hbm_frac"]}
    else:
        roofline = {"bound": "hbm", "kernel": best, "achieved": row["alg_GBps"], "peak": peaks["hbm_gbs"], "unit": "GB/s",
                    "frac": row["hbm_frac"], "traffic": None, "peak_source": peak_src}
    tpath = os.path.join(ROOT, "profiles", "r02_ncu_traffic.json")  # DRAM bytes per launch from the committed ncu capture
    if os.path.exists(tpath):
        tj = json.load(open(tpath))
        ent = tj.get(nb.name, {})
        if ent.get("batch") == nb.batch and best in ent.get("dram_bytes_per_launch", {}):
            roofline["traffic"] = ent["dram_bytes_per_launch"][best]
            roofline["traffic_source"] = ent["source"]
    roofline.update({"avg_launch_us": round(t_ms * 1e3 / t_cnt, 2), "share_of_step": round(t_ms / tot, 4),
                     "alg_bytes_per_launch": t_bytes / t_cnt, "per_kernel": per_kernel, "profiled_step_ms": round(prof_ms, 3),
                     "hbm_peak_GBps": peaks["hbm_gbs"], "hbm_peak_source": peak_src})
    return roofline


def time_e2e(nb, steps, world):
    """The same metric end to end through the C ABI with HOST buffers: every step imports its inputs from pinned host
    memory (H2D + NTT), runs the layers and exports the results (iNTT + D2H) to pinned host memory.
    (a) serial: import, forward, export, one request (batch group) after the other;
    (b) serving loop: software-pipelined over requests -- while request i computes, the host uploads request i+2
        (fenc_ct_import_async: copy stream + staging ring), has request i+1 enqueued, and collects request i's result
        (fenc_ct_export_async / fenc_export_wait).  Every period holds one full upload, one forward and one export."""
    import torch
    ctx, pipe, lazy = nb.ctx, nb.pipe, nb.lazy

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    reqs = []  # per request (batch group): pinned host copies of its input ciphertexts
    for g in nb.groups:
        pinned = [torch.from_numpy(ctx.ct_export(c).view(np.int64)).pin_memory() for c in g]
        reqs.append([t.numpy().view(np.uint64) for t in pinned])
    nb._pinned_keepalive = reqs
    s_in = nb.groups[0][0].scale
    h2d = sum(a.nbytes for r in reqs for a in r)
    d2h, res = 0, None
    for it in range(1 + steps):  # first iteration is a warm-up
        if it == 1:
            barrier()
            t0 = time.perf_counter()
        d2h = 0
        for r in reqs:
            dc = [ctx.ct_import(a, s_in) for a in r]
            res = [ctx.ct_export(c) for c in pipe.forward(dc, lazy_relin=lazy)]
            d2h += sum(a.nbytes for a in res)
            del dc
    barrier()
    serial_s = max_over_ranks((time.perf_counter() - t0) / steps, world, "cuda")

    def upload(r):
        return [ctx.ct_import_async(a, s_in) for a in r]

    host_out = [torch.empty(a.shape, dtype=torch.int64).pin_memory().numpy().view(np.uint64) for a in res]

    def export(outs):
        for c, h in zip(outs, host_out):
            ctx.ct_export_async(c, h)

    nreq = len(reqs)
    barrier()
    outs = pipe.forward(upload(reqs[0]), lazy_relin=lazy)
    dc = upload(reqs[1 % nreq])
    export(outs)
    n_warm, total = 2, steps * nreq
    for it in range(n_warm + total):
        if it == n_warm:
            t0 = time.perf_counter()  # right behind the arrival of a result, the next request already on the GPU
        outs = pipe.forward(dc, lazy_relin=lazy)      # request it+1, enqueued while request it computes
        dc = upload(reqs[(it + 2) % nreq])            # request it+2: copies overlap the compute
        ctx.export_wait()                             # request it's result is on the host
        export(outs)
    e2e_s = (time.perf_counter() - t0) / steps
    ctx.export_wait()
    barrier()
    e2e_s = max_over_ranks(e2e_s, world, "cuda")
    del dc, outs
    return {"ms_per_step": round(e2e_s * 1e3, 3), "serial_ms_per_step": round(serial_s * 1e3, 3), "h2d_bytes_per_step": int(h2d),
            "d2h_bytes_per_step": int(d2h), "steps": steps,
            "mode": "pipelined requests: async upload (copy stream), next request enqueued before this result is collected"}


# ------------------------------------------------------------------------------------------------ CPU oracle arm
def oracle_op_counts(layers, n_slots, n_q, hoist, lazy):
    """{(kind, L): count} of one forward pass in the variant the GPU arm runs, from the ORACLE's own graphs
    (oracle/fragment.py, oracle/network.py; no GPU involved).  Kinds: rot (plain rotation), rot_h (hoisted inner rotation,
    R2.7b), pmult (plaintext PMult-accumulate), smul (scalar multiply-accumulate of a factored weight, R2.9c), add,
    rescale, square (x^2 + relinearise + rescale), square_sum4 (R2.12c over four ciphertexts), poly3."""
    from oracle import fragment as fr
    from oracle import network as nw
    ops, L, n_ct = {}, n_q, None

    def add(kind, lv, n):
        if n:
            ops[(kind, lv)] = ops.get((kind, lv), 0) + n

    for li, ly in enumerate(layers):
        if ly["op"] == "conv":
            S = ly["S"] or fr.select_S(fr.ConvDesc(**ly["conv"]), n_slots)
            g = fr.ConvGraph(fr.ConvDesc(S=S, **ly["conv"]), n_slots)
            c, bg = g.counts(), g.lin.BG
            add("rot_h" if hoist else "rot", L, c["n_inner_rot"])
            add("rot", L, c["n_outer_rot"])
            n_masks = 0
            for diags in g.terms.values():
                add("add", L, (len(diags) - 1) * bg)
                if ly.get("factored"):
                    for lst in diags.values():
                        n_masks += len({(tuple(x[0] for x in f[0]), tuple(f[1]), tuple(f[2])) for f in (g._weight_factors(wk) for _, _, wk in lst)})
            if ly.get("factored"):
                add("smul", L, c["n_pmult"])
                add("pmult", L, n_masks * bg)
            else:
                add("pmult", L, c["n_pmult"])
            add("rescale", L, c["n_out_ct"])
            n_ct, L = c["n_out_ct"], L - 1
        elif ly["op"] == "fc":
            g = nw.FcGraph(n_slots, **ly["fc"])
            c = g.counts()
            n_baby = len(g.baby_steps()) * g.BG
            add("rot_h" if hoist else "rot", L, n_baby)
            add("rot", L, c["n_rot"] - n_baby)
            add("pmult", L, c["n_pmult"])
            add("add", L, sum(len(gi) - 1 for gi in g.terms.values()) * g.BG)
            add("rescale", L, c["n_out_ct"])
            n_ct, L = c["n_out_ct"], L - 1
        elif ly["op"] == "square":
            if lazy and li + 1 < len(layers) and layers[li + 1]["op"] == "pool":
                add("square_sum4", L, n_ct // 4)
            else:
                add("square", L, n_ct)
            L -= 1
        elif ly["op"] == "poly3":
            add("poly3", L, n_ct)
            L -= 2
        elif ly["op"] == "pool":
            if not (lazy and li > 0 and layers[li - 1]["op"] == "square"):
                add("add", L, 3 * (n_ct // 4))
            n_ct //= 4
        elif ly["op"] == "compress":
            prev = fr.ConvGraph(fr.ConvDesc(S=layers[li - 1]["S"], **layers[li - 1]["conv"]), n_slots)
            per, frags, bgs = prev.lout.chp // ly["v"], prev.S_out ** 2, prev.lout.BG
            n_t = -(-bgs // per)
            add("rot", L, frags * (bgs - n_t))
            add("add", L, frags * (bgs - n_t))
            n_ct = n_t * frags
    return ops


def _oracle_job(sh, kind, L, reps):
    """time one oracle operation `reps` times in this (worker) process; returns the list of seconds"""
    ck, P, keys, ct, pt = sh["ck"], sh["P"], sh["keys"], sh["ct"][L], sh["pt"][L]
    out = []
    for _ in range(reps):
        t0 = time.perf_counter()
        if kind == "rot":
            ck.rotate(P, keys, ct, sh["step"])
        elif kind == "rot_h":
            ck.rotate_hoisted(P, keys, ct, sh["step"])
        elif kind == "pmult":
            ck.pmult_acc(P, np.zeros_like(ct.c), ct, pt)
        elif kind == "smul":
            t = ck.mul_const(P, ct, 0.0123, 2 ** 20)
            ck.add(P, t, t)
        elif kind == "add":
            ck.add(P, ct, ct)
        elif kind == "rescale":
            ck.rescale(P, ct)
        elif kind == "square":
            ck.square_relin(P, keys, ct)
        elif kind == "square_sum4":
            ck.square_sum_relin(P, keys, [ct] * 4)
        elif kind == "poly3":
            ck.poly3(P, keys, ct)
        out.append(time.perf_counter() - t0)
    return out


class OracleSampler:
    """Times the CPU oracle (oracle/, as it stands; each operation single-threaded) on every (operation kind, level) the
    workload uses and scales by the exact operation counts of the SAME variant the GPU arm runs.  The independent sample
    operations are timed concurrently in worker processes (fan-out over processes of the same
    single-threaded program); cheap operations are timed three times and the spread reported.  Timing does not depend on
    the operand values: ciphertexts and switching keys are uniform-random residues (no key generation in the sample)."""

    def __init__(self, pkey, ops):
        from oracle import ckks as ck
        self.ck, self.ops = ck, ops
        self.P = P = ck.Params(*wl.oracle_params_args(wl.PARAMS[pkey]))
        rng = np.random.default_rng(0)
        self.step = 1
        keys = ck.Keys(P, 1)
        A = len(P.mod)

        def rand_key():
            k = np.empty((2, P.beta_max, A, P.N), dtype=np.uint64)
            for t in range(A):
                k[:, :, t] = rng.integers(0, P.mod[t], (2, P.beta_max, P.N), dtype=np.uint64)
            return k[0], k[1]

        kinds = {k for k, _ in ops}
        if kinds & {"rot", "rot_h"}:
            keys.evk[self.step] = rand_key()
        if kinds & {"square", "square_sum4", "poly3"}:
            keys.evk[ck.RELIN_KEY_ID] = rand_key()
        levels = sorted({L for _, L in ops})
        z = rng.uniform(-1, 1, P.n)
        self.shared = dict(ck=ck, P=P, keys=keys, step=self.step,
                           ct={L: ck.Ciphertext(wl.random_ct_limbs(L, P.q, L, P.N), L, P.scale) for L in levels},
                           pt={L: ck.encode(P, z, L, P.q[L - 1]) for L in levels})

    def sample(self, procs=None):
        sys.path.insert(0, os.path.join(ROOT, "tests"))
        from oracle_pool import pmap
        heavy = {"rot", "rot_h", "square", "square_sum4", "poly3"}
        big = self.P.N >= (1 << 15)
        jobs = [(k, L, 1 if (big and k in heavy) else 3) for (k, L) in sorted(self.ops)]
        # small rings: one process, one operation at a time.  N >= 2^15 (a rotation takes tens of seconds): the operations
        # run concurrently and every timing is divided by a contention factor measured on one of them (shared hosts
        # hand out fewer cores than they show)
        procs = procs or (min(len(jobs), os.cpu_count() or 1) if big else 1)
        t0 = time.perf_counter()
        res = pmap(self.shared, _oracle_job, jobs, procs=procs)
        factor = 1.0
        if procs > 1:
            cal = next((i for i, j in enumerate(jobs) if j[0] == "pmult"), 0)
            alone = float(np.median(_oracle_job(self.shared, *jobs[cal])))
            factor = max(1.0, float(np.median(res[cal])) / alone)
        wall = time.perf_counter() - t0
        total, detail = 0.0, {}
        for (k, L, _), ts in zip(jobs, res):
            med = float(np.median(ts)) / factor
            total += self.ops[(k, L)] * med
            detail["%s@L%d" % (k, L)] = {"s": round(med, 5), "count": int(self.ops[(k, L)]),
                                          "spread": round((max(ts) - min(ts)) / float(np.median(ts)), 3) if len(ts) > 1 else None}
        self.contention = round(factor, 3)
        return total, detail, procs, wall


def oracle_end_to_end_cfg1(hoist):
    """BASELINE config 1 through the oracle END TO END (one conv layer, about 3 s single-threaded): the check of the
    sampled estimator that cpu_baseline reports beside it."""
    from oracle import ckks as ck
    from oracle import fragment as fr
    P = ck.Params(*wl.oracle_params_args(wl.PARAMS["cfg1"]))
    kw = wl.CONVS["lenet_conv1"]
    x, w = wl.conv_inputs(1, kw)
    S = fr.select_S(fr.ConvDesc(**kw), P.n)
    g = fr.ConvGraph(fr.ConvDesc(S=S, **kw), P.n)
    keys = ck.keygen(P, 1, g.counts()["rot_steps"])
    W = fr.encode_weights(ck, P, g, w, P.nq)
    ins = {(u, v, gi): ck.encrypt(P, keys, ck.encode(P, g.lin.gather(x, u, v, gi, 0), P.nq), 7) for u in range(S) for v in range(S) for gi in range(g.lin.G)}
    t0 = time.perf_counter()
    fr.hconv(ck, P, keys, g, ins, W, hoist=hoist)
    return time.perf_counter() - t0


def cpu_baseline_for(name, layers, n_groups, n_conv, hoist, lazy, unit_count, unit):
    """the `cpu_baseline` object: the oracle's estimated throughput in the line's unit, single-threaded"""
    pkey = WORKLOADS[name][0]
    p = wl.PARAMS[pkey]
    ops = oracle_op_counts(layers, 1 << (p["log2N"] - 1), p["n_q"], hoist, lazy)
    ops = {k: v * n_groups for k, v in ops.items()}
    smp = OracleSampler(pkey, ops)
    est, detail, procs, wall = smp.sample()
    out = {"value": round(unit_count / est, 8), "unit": unit, "cores": 1, "kind": "oracle", "method": "sampled per operation x exact counts",
           "estimated": True, "same_graph": True, "estimated_step_s": round(est, 2), "sample_wall_s": round(wall, 1),
           "sample_processes": procs, "contention_factor": smp.contention, "host": host_info(),
           "sample": "every (operation, level) of the step timed on the oracle as it stands (rotations, squares and the activation once "
                     "at N >= 2^15, everything else three times, median) in %d process(es) -- concurrently at N >= 2^15, timings divided by the "
                     "contention factor measured on one operation run alone --, each operation single-threaded; scaled by the exact counts of the variant the GPU arm runs (hoisted inner rotations: %s, lazy "
                     "relinearisation: %s, factored weights where the layer has them); `value` is the single-thread figure" % (procs, hoist, lazy),
           "seconds_per_op": detail}
    if name == "cfg1_conv1":
        e2e = oracle_end_to_end_cfg1(hoist)
        out["end_to_end_s"] = round(e2e, 3)
        out["estimate_over_end_to_end"] = round(est / e2e, 3)
    return out


# ------------------------------------------------------------------------------------------------ the two arms
def run_ours(args, rank, world):
    import torch
    dev = int(os.environ.get("LOCAL_RANK", 0))
    torch.cuda.set_device(dev)
    name = args.workload
    # the clock sampler starts BEFORE the set-up (nvidia-smi's start-up would otherwise perturb the timed steps) and keeps
    # sampling; every timed region reports only its own samples
    sampler = ClockSampler(dev).start()
    nb = NetBench(args, name, rank, dev, args.batch)
    t, out = time_resident(nb, args.steps, args.warmup, world, sampler, args.profile_range)
    del out
    summ = net_summary(nb, t, world)
    if args.per_layer:
        sampler.stop()
        return {"workload": name, "batch": nb.batch, "ms_per_step": summ["ms_per_step"], "clocks": summ["clocks"], "per_layer": per_layer_profile(nb)}
    if args.no_extras:
        sampler.stop()
        return {"metric": METRIC, "value": summ["conv_layers_per_s"], "unit": nb.unit, "ms_per_step": summ["ms_per_step"],
                "images_per_s": summ["images_per_s"], "gpu_launches": summ["gpu_launches"], "clocks": summ["clocks"],
                "config": {"workload": name, "batch": nb.batch}}
    prof_steps = min(args.steps, 3)
    prof, prof_ms = per_kernel_profile(nb, prof_steps)
    roofline = roofline_of(nb, prof, prof_steps, prof_ms)
    e2e = time_e2e(nb, min(args.steps, args.e2e_steps), world)
    per_group = t["group_in_bytes"] + t["group_out_bytes"]
    n_groups = len(nb.groups)
    # resident batch the measured footprint allows: P(n) = fixed + n (inputs + outputs of a batch group) + one group's temporaries
    max_groups = n_groups + max(0, int((0.95 * HBM_BYTES - t["peak_bytes"]) // per_group)) if WORKLOADS[name][3] else None
    line = {
        "metric": METRIC, "value": summ["conv_layers_per_s"], "unit": nb.unit,
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": summ["ms_per_step"],
        "images_per_s": summ["images_per_s"], "rotations_per_s": summ["rotations_per_s"],
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u64", "data": "synthetic",
        "config": {"workload": name, "description": nb.desc, "batch": nb.batch, "batch_groups": n_groups,
                   "conv_layers_per_step": nb.n_conv if "conv" in nb.unit else 0, "linear_layers_per_step": nb.n_lin, "rotations_per_step": nb.n_rot,
                   "relinearisations_per_step": nb.n_relin, "pmults_per_step": nb.n_pm,
                   "inner_rotations": "hoisted (R2.7b)" if nb.hoist else "plain",
                   "square_pool": "one relinearisation per pooled output (R2.12c)" if nb.lazy else "eager",
                   "multi_gpu": "replicas only" if world > 1 else "single",
                   "l2": "inputs_exceed_l2: %d MiB resident after set-up" % (nb.setup_bytes >> 20),
                   "peak_device_bytes": t["peak_bytes"], "bytes_per_batch_group_in_out": per_group,
                   "max_resident_batch_under_180GB": (max_groups * WORKLOADS[name][3]) if max_groups else None,
                   "max_resident_batch_rule": "batch + floor((0.95 x 180e9 - measured peak) / (input + output bytes of one batch group)) x 32"
                   if max_groups else None},
        "gpu_launches": summ["gpu_launches"], "clocks": summ["clocks"],
        "e2e": dict({"value": round(world * nb.n_conv / (e2e["ms_per_step"] * 1e-3), 3), "unit": nb.unit,
                     "images_per_s": round(world * nb.batch / (e2e["ms_per_step"] * 1e-3), 2),
                     "serial_value": round(world * nb.n_conv / (e2e["serial_ms_per_step"] * 1e-3), 3)}, **e2e),
        "roofline": roofline,
    }
    layers, hoist, lazy, n_conv, unit = nb.layers, nb.hoist, nb.lazy, nb.n_conv, nb.unit
    nb.close()
    del nb
    if rank == 0 and world == 1:
        if not args.no_cpu:
            line["cpu_baseline"] = cpu_baseline_for(name, layers, n_groups, n_conv, hoist, lazy, n_conv, unit)
        if name == DEFAULT_WORKLOAD and not args.no_companions:
            line["extras"] = companions(args, sampler, dev)
    sampler.stop()
    return line


def companions(args, sampler, dev):
    """The other BASELINE configurations, timed in the same run under the same clock sampler (each region reports its own
    clock samples): config 5's L=24 / dnum=3 point plain and hoisted, the config-2 LeNet-5 step, a config-3 layer."""
    ex = {}
    for hoisted in (False, True):
        pt, clocks = timed_clocks(sampler, lambda: sweep_point(24, 3, hoisted))
        ex["cfg5_L24_dnum3_" + ("hoisted" if hoisted else "plain")] = dict(pt, clocks=clocks)
    for wname in ("cfg2_lenet5", "cfg3_conv_16_16"):
        nb = NetBench(args, wname, 0, dev, None)
        steps = max(args.steps, 10) if wname == "cfg2_lenet5" else max(args.steps, 5)
        t, out = time_resident(nb, steps, args.warmup, 1, sampler)
        del out
        d = net_summary(nb, t, 1)
        prof, prof_ms = per_kernel_profile(nb, 3)
        d["per_kernel"] = roofline_of(nb, prof, 3, prof_ms)["per_kernel"]
        d["description"] = nb.desc
        ex[wname] = d
        nb.close()
    return ex


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, on the host cores (no GPU).  Each step is one bounded sample of the
    workload's operations (OracleSampler), scaled by the exact counts of the variant the GPU arm runs by default."""
    name = args.workload
    pkey, builder, desc, per_group = WORKLOADS[name]
    batch = args.batch or DEFAULT_BATCH.get(name, 1)
    layers, _ = builder(batch, 2000)
    n_groups = max(1, batch // per_group) if per_group else 1
    n_conv, unit = counted_layers(layers, n_groups)
    p = wl.PARAMS[pkey]
    ops = oracle_op_counts(layers, 1 << (p["log2N"] - 1), p["n_q"], not args.no_hoist, not args.eager_relin)
    ops = {k: v * n_groups for k, v in ops.items()}
    smp = OracleSampler(pkey, ops)
    for _ in range(min(args.warmup, 1)):
        smp.sample()
    runs = [smp.sample() for _ in range(max(1, min(args.steps, 3)))]
    est = float(np.mean([r[0] for r in runs]))
    v = round(n_conv / est, 8)
    base = {"value": v, "unit": unit, "cores": 1, "kind": "oracle", "method": "sampled per operation x exact counts",
            "estimated": True, "same_graph": True, "sample_processes": runs[-1][2], "contention_factor": smp.contention, "host": host_info(),
            "sample": "per step: every (operation, level) of the workload timed on the oracle (heavy operations once, the others three "
                      "times, median) in %d concurrent worker processes, scaled by the exact operation counts; estimated step %.1f s; "
                      "%d sampled step(s) averaged whatever --steps says" % (runs[-1][2], est, len(runs)),
            "seconds_per_op": runs[-1][1]}
    return {"impl": "reference", "metric": METRIC, "value": v, "unit": unit, "n_gpus": 0,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(est * 1e3, 1), "higher_is_better": True,
            "images_per_s": round((per_group * n_groups if per_group else batch) / est, 6),
            "scaling": "weak", "vs_baseline": None, "dtype": "u64", "data": "synthetic", "estimated": True,
            "config": {"workload": name, "description": desc, "batch": per_group * n_groups if per_group else batch},
            "cpu_baseline": base,
            "e2e": {"value": v, "unit": unit, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}


def respawn_under_torchrun(n):
    """`python bench.py --gpus N` without a launcher: re-execute under torch.distributed.run, one rank per GPU (replicas)."""
    import socket
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(n), "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    os.execv(sys.executable, cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=sorted(WORKLOADS))
    ap.add_argument("--batch", type=int, default=None, help="images per step (config 4: a multiple of 32; default 64; config 2: default 128)")
    ap.add_argument("--e2e-steps", type=int, default=3, help="steps of each end-to-end leg (at most --steps)")
    ap.add_argument("--profile-range", action="store_true", help="cudaProfilerStart/Stop around the timed steps (for ncu)")
    ap.add_argument("--plain-fc", action="store_true", help="fully connected layers by plain diagonals (no baby-step giant-step)")
    ap.add_argument("--plain-conv", action="store_true", help="conv layers' channel diagonals without baby-step giant-step (config 3 workloads)")
    ap.add_argument("--eager-relin", action="store_true", help="x^2 and the pool after it as two steps (four relinearisations per pooled output)")
    ap.add_argument("--no-hoist", action="store_true", help="inner rotations as plain rotations (one decomposition each)")
    ap.add_argument("--sweep-L", type=int, nargs="*", help="config 5: only these limb counts")
    ap.add_argument("--sweep-dnum", type=int, nargs="*", help="config 5: only these dnum values")
    ap.add_argument("--sweep-cts", type=int, default=64, help="config 5: ciphertexts per batched rotation (BASELINE: 64)")
    ap.add_argument("--sweep-steps", type=int, default=32, help="config 5: distinct rotation amounts (BASELINE: 32)")
    ap.add_argument("--no-extras", action="store_true", help="timed steps only: skip the per-kernel pass, e2e, cpu_baseline, companions (profiling runs)")
    ap.add_argument("--per-layer", action="store_true", help="print a per-layer, per-kernel-class breakdown of one step instead of the bench line")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-companions", action="store_true", help="default workload only: skip the config 5 / 2 / 3 companions")
    args = ap.parse_args()
    global FC_BSGS, CONV_BSGS
    if args.plain_fc:
        FC_BSGS = 1
    if args.plain_conv:
        CONV_BSGS = 1
    rank, world = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))
    if args.impl == "reference":
        if rank == 0:
            print(json.dumps(run_reference(args)), flush=True)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        respawn_under_torchrun(args.gpus)
    if args.gpus != world:
        sys.exit("bench.py: --gpus %d but WORLD_SIZE=%d (launch with torch.distributed.run, or without it for N=1)" % (args.gpus, world))
    args.warmup = max(args.warmup, 3)
    if world > 1:
        import torch
        torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", 0)))
        torch.distributed.init_process_group("nccl")
    if args.workload in ("cfg5_rotsweep", "cfg5_rotsweep_hoisted"):
        line = run_rotsweep(args, hoisted=args.workload.endswith("hoisted"))
    elif args.workload == "cfg3_compress":
        line = run_compress(args)
    else:
        line = run_ours(args, rank, world)
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        import torch
        torch.distributed.destroy_process_group()


if __name__ == "__main__":
    main()

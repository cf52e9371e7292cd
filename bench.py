"""bench.py -- measures BASELINE.json's metric on one B200 (or N independent replicas).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl ours|reference]

A step = one pass of the whole hot path over one batch of synthetic input (workloads.py).  `value` is the
whole-job throughput with inputs resident in HBM; `e2e` is the same metric through the C-ABI calls with HOST
buffers (ciphertext limbs imported from / exported to host memory inside the timed region).  `roofline` is
for the dominant kernel class, timed live with CUDA events by the library's profile hooks; `cpu_baseline`
times the CPU oracle as it stands on a bounded sample of the same workload."""
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
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc:
            time.sleep(0.12)  # let the last sample of the timed region arrive
            self.proc.terminate()
        if len(self.rows) > self.first:
            self.rows = self.rows[self.first:]
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) > 2 + i and r[2 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(sm)}


# ------------------------------------------------------------------------------------------------ workloads
FC_BSGS = 0  # baby-step count of the fully connected layers: 0 = library's choice (R2.12b), 1 = plain diagonals (--plain-fc)


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


WORKLOADS = {
    # name: (PARAMS key, builder, description)
    "cfg2_lenet5_convstage": ("cfg2", lambda bs, seed: lenet_layers(bs, seed, upto="conv"),
                              "BASELINE config 2, conv stage: conv1-x^2-pool-conv2-x^2-pool, N=2^14, 8x40b+2x60b, dnum=4"),
    "cfg2_lenet5": ("cfg2", lambda bs, seed: lenet_layers(bs, seed, upto="fc"),
                    "BASELINE config 2: LeNet-5-shaped network, N=2^14, 8x40b+2x60b, dnum=4"),
    # single layers (parity-test configurations, timed for the record; --batch is ignored: BS = 1 as in BASELINE.json)
    "cfg1_conv1": ("cfg1", lambda bs, seed: conv_layers("lenet_conv1", seed),
                   "BASELINE config 1: LeNet conv1-shaped layer, N=2^13, 3x40b+1x60b, dlen=1 (A1), batch 1"),
    "cfg3_conv_16_16": ("cfg3", lambda bs, seed: conv_layers("resnet_16_16", seed, True),
                        "BASELINE config 3: ResNet-20 3x3 16->16 layer, N=2^16, 24x50b+4x60b, dnum=6, batch 1"),
    "cfg3_conv_16_32_s2": ("cfg3", lambda bs, seed: conv_layers("resnet_16_32_s2", seed, True),
                           "BASELINE config 3: ResNet-20 3x3 16->32 stride 2, N=2^16, batch 1"),
    "cfg3_conv_32_64_s2": ("cfg3", lambda bs, seed: conv_layers("resnet_32_64_s2", seed, True),
                           "BASELINE config 3: ResNet-20 3x3 32->64 stride 2, N=2^16, batch 1"),
    "cfg5_rotsweep": (None, None, "BASELINE config 5: rotation / key-switch sweep"),
    "cfg5_rotsweep_hoisted": (None, None, "BASELINE config 5 with hoisted rotations (8 amounts per decomposition)"),
    "cfg3_compress": (None, None, "AAC compress micro-benchmark at config 3's parameters"),
}
DEFAULT_WORKLOAD = "cfg2_lenet5"


def conv_layers(name, seed, kaiming=False):
    """one encrypted conv layer of a BASELINE config at the top level (reading A20), planner-selected S."""
    kw = wl.CONVS[name]
    x, w = wl.conv_inputs(seed, kw, kaiming=kaiming)
    return [{"op": "conv", "conv": dict(kw), "S": 0, "w": w}], x


def run_rotsweep(args, hoisted=False):
    """BASELINE config 5: rotation / key-switch sweep at N=2^16 (reading A2: k = dlen = ceil(L/dnum)).  64 ciphertexts with
    uniform-random limbs, 32 distinct seeded rotation amounts; every amount is one batched fenc_rotate over the 64.
    hoisted: the same 2048 rotations as 4 calls of fenc_rotate_hoisted (64 ciphertexts x 8 amounts each: one
    decomposition per ciphertext and call, R2.7b -- the shape of a 3x3 convolution's 8 inner rotations)."""
    import torch
    import paper_2606_16359_b200 as fenc
    peaks, peak_src = measured_peaks()
    n_ct, n_steps, points = args.sweep_cts, args.sweep_steps, []
    for L in (args.sweep_L or (4, 8, 16, 24, 36)):
        for dnum in (args.sweep_dnum or (1, 2, 3, 4)):
            pr = wl.sweep_params(L, dnum)
            ctx = fenc.Context(**pr)
            N, k, dlen = ctx.N, ctx.n_p, ctx.dlen
            beta = -(-L // dlen)
            steps = wl.rotation_steps(5000 + L * 10 + dnum, n_steps, ctx.n)
            keys = ctx.keygen(5, steps)
            cts = [ctx.ct_import(wl.random_ct_limbs(100 * L + i, ctx.q, L, N)) for i in range(n_ct)]
            if hoisted:
                ctx.rotate_hoisted(keys, cts, steps[:8])
            else:
                for r in steps[:2]:
                    ctx.rotate(keys, cts, [r] * n_ct)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ctx.launch_count(reset=True)
            e0.record()
            if hoisted:
                for at in range(0, n_steps, 8):
                    out = ctx.rotate_hoisted(keys, cts, steps[at:at + 8])
                    del out
            else:
                for r in steps:
                    out = ctx.rotate(keys, cts, [r] * n_ct)
                    del out
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            rots = n_ct * n_steps
            # algorithmic bytes per rotation: ciphertext in + out, key once per batch of 64
            b_alg = 2 * (2 * L * N * 8) + 2 * beta * (L + k) * N * 8 / n_ct
            if hoisted:  # input read once per 8 rotations, output once per rotation, key once per 64 ciphertexts
                b_alg = 2 * L * N * 8 * (1 + 1 / 8) + 2 * beta * (L + k) * N * 8 / n_ct
            gbs = rots * b_alg / (ms * 1e-3) / 1e9
            points.append({"L": L, "dnum": dnum, "dlen": dlen, "k": k, "beta": beta,
                           "ntt_per_rot": beta * (L + k) + 2 * k + 2 * L, "rot_per_s": round(rots / (ms * 1e-3), 1),
                           "us_per_rot": round(ms * 1e3 / rots, 2), "alg_GBps": round(gbs, 1),
                           "hbm_frac": round(gbs / peaks["hbm_gbs"], 4), "launches": ctx.launch_count()})
            del cts, keys
            ctx.close()
            torch.cuda.empty_cache()
    ref = ([p for p in points if p["L"] == 24 and p["dnum"] == 3] or points)[0]
    return {"metric": METRIC, "value": ref["rot_per_s"], "unit": "key-switched rotations/s", "n_gpus": 1, "steps": n_steps,
            "warmup": 2, "ms_per_step": round(1e3 * n_ct / ref["rot_per_s"], 4), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "u64", "data": "synthetic",
            "config": {"workload": "cfg5_rotsweep_hoisted" if hoisted else "cfg5_rotsweep",
                       "description": "BASELINE config 5: N=2^16, 64 cts x 32 amounts per point; value quoted at L=24, dnum=3"
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


def run_ours(args, rank, world):
    import torch
    import paper_2606_16359_b200 as fenc
    from paper_2606_16359_b200.pipeline import Pipeline
    dev = int(os.environ.get("LOCAL_RANK", 0))
    torch.cuda.set_device(dev)
    pkey, builder, desc = WORKLOADS[args.workload]
    seed = 2000 + rank
    layers, x = builder(args.batch, seed)
    args.batch = int(layers[0]["conv"]["BS"])
    ctx = fenc.Context(device=dev, **wl.PARAMS[pkey])
    ctx.set_hoisting(not args.no_hoist)  # inner rotations share one decomposition per input ciphertext (R2.7b)
    pipe = Pipeline(ctx, layers)
    pipe.setup(key_seed=seed)
    cts = pipe.encrypt_input(x, enc_seed0=10 * seed)
    lazy = not args.eager_relin  # x^2 + pool as one step with one relinearisation per pooled output (R2.12c)
    n_lin, n_rot, n_relin, n_pm = pipe.counts(lazy_relin=lazy)
    ctx.sync()
    setup_bytes = ctx.device_bytes()

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    # the clock sampler starts BEFORE the warm-up (nvidia-smi's start-up would otherwise perturb the timed steps) and keeps
    # sampling through the timed region; only samples taken inside the timed region are reported
    sampler = ClockSampler(dev)
    sampler.start()
    t_wait = time.time()
    while not sampler.rows and time.time() - t_wait < 3.0:
        time.sleep(0.05)
    for _ in range(args.warmup):
        pipe.forward(cts, lazy_relin=lazy)
    barrier()
    sampler.mark()
    ctx.launch_count(reset=True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if args.profile_range:  # for `ncu --profile-from-start off`: only the timed steps are captured
        torch.cuda.profiler.start()
    e0.record()
    for _ in range(args.steps):
        out = pipe.forward(cts, lazy_relin=lazy)
    e1.record()
    barrier()
    if args.profile_range:
        torch.cuda.profiler.stop()
    ms = e0.elapsed_time(e1)
    launches = ctx.launch_count()
    clocks = sampler.stop()
    ms = max_over_ranks(ms, world, "cuda")
    step_ms = ms / args.steps
    if args.no_extras:
        return {"metric": METRIC, "value": round(aggregate(n_lin, world, step_ms * 1e-3), 3), "ms_per_step": round(step_ms, 4),
                "gpu_launches": int(launches), "config": {"workload": args.workload, "batch": args.batch}}
    # ---- per-kernel-class timing (separate pass with the library's CUDA-event hooks on the same stream)
    ctx.profile_enable(True)
    prof_steps = min(args.steps, 3)
    t0 = time.perf_counter()
    for _ in range(prof_steps):
        pipe.forward(cts, lazy_relin=lazy)
    prof = ctx.profile_read()
    prof_ms = (time.perf_counter() - t0) * 1e3 / prof_steps
    ctx.profile_enable(False)
    peaks, peak_src = measured_peaks()
    imad_peak, bfly_peak = ctx.measure_alu_peak()
    tot = sum(v[0] for v in prof.values())
    top = max(prof, key=lambda k: prof[k][0])
    t_ms, t_cnt, t_bytes, t_ops = prof[top]
    hbm_ach, alu_ach = t_bytes / (t_ms * 1e-3) / 1e9, t_ops / (t_ms * 1e-3)
    per_kernel = {k: {"ms_per_step": round(v[0] / prof_steps, 4), "launches_per_step": v[1] // prof_steps,
                      "alg_GBps": round(v[2] / (v[0] * 1e-3) / 1e9, 1), "hbm_frac": round(v[2] / (v[0] * 1e-3) / 1e9 / peaks["hbm_gbs"], 4),
                      "Gbutterflies_per_s": round(v[3] / (v[0] * 1e-3) / 1e9, 1), "alu_frac": round(v[3] / (v[0] * 1e-3) / bfly_peak, 4)}
                  for k, v in sorted(prof.items(), key=lambda kv: -kv[1][0])}
    # the NTT-carrying kernels are bound by the integer pipes: report the roof the kernel is nearer to
    if t_ops and alu_ach / bfly_peak >= hbm_ach / peaks["hbm_gbs"]:
        roofline = {"bound": "alu", "kernel": top, "achieved": round(alu_ach / 1e9, 2), "peak": round(bfly_peak / 1e9, 2),
                    "unit": "G modular butterflies/s", "frac": round(alu_ach / bfly_peak, 4), "traffic": None,
                    "peak_source": "measured live: register-only butterflies of this library on all SMs, the faster of the integer "
                                   "Shoup and the fp64 one (fenc_measure_alu_peak); 32-bit IMAD peak %.2f T lane-ops/s" % (imad_peak / 1e12),
                    "butterflies_per_launch": t_ops / t_cnt, "hbm_frac_of_same_kernel": round(hbm_ach / peaks["hbm_gbs"], 4)}
    else:
        roofline = {"bound": "hbm", "kernel": top, "achieved": round(hbm_ach, 1), "peak": peaks["hbm_gbs"], "unit": "GB/s",
                    "frac": round(hbm_ach / peaks["hbm_gbs"], 4), "traffic": None, "peak_source": peak_src}
    tpath = os.path.join(ROOT, "profiles", "r01_ncu_traffic.json")  # DRAM bytes per launch from the committed ncu capture
    if os.path.exists(tpath):
        tj = json.load(open(tpath))
        if tj.get("workload") == args.workload and tj.get("batch") == args.batch:
            roofline["traffic"] = tj["dram_bytes_per_launch"].get(top)
            roofline["traffic_source"] = tj["source"]
    roofline.update({"avg_launch_us": round(t_ms * 1e3 / t_cnt, 2), "share_of_step": round(t_ms / tot, 4),
                     "alg_bytes_per_launch": t_bytes / t_cnt, "per_kernel": per_kernel, "profiled_step_ms": round(prof_ms, 3),
                     "hbm_peak_GBps": peaks["hbm_gbs"], "hbm_peak_source": peak_src})
    # ---- end to end through the C ABI with host buffers: import (H2D + NTT), forward, export (iNTT + D2H)
    # host buffers in pinned memory (torch owns them; numpy views are what the C ABI receives)
    pinned = [torch.from_numpy(ctx.ct_export(c).view(np.int64)).pin_memory() for c in cts]
    host_in = [t.numpy().view(np.uint64) for t in pinned]
    s_in = cts[0].scale
    h2d = sum(a.nbytes for a in host_in)
    d2h = 0
    # (a) serial: every step imports (synchronously), computes, exports
    for it in range(1 + args.steps):  # first iteration is a warm-up
        if it == 1:
            barrier()
            t0 = time.perf_counter()
        dc = [ctx.ct_import(a, s_in) for a in host_in]
        res = [ctx.ct_export(c) for c in pipe.forward(dc, lazy_relin=lazy)]
        d2h = sum(a.nbytes for a in res)
    barrier()
    serial_s = max_over_ranks((time.perf_counter() - t0) / args.steps, world, "cuda")
    # (b) serving loop (the headline): software-pipelined over requests.  While request i computes, the host uploads the
    # inputs of request i+2 (fenc_ct_import_async: copy stream + staging ring), has request i+1 enqueued already, and
    # collects request i's result (fenc_ct_export_async / fenc_export_wait), so the GPU never waits for the host.
    # Every period contains one full upload, one forward and one export to the host; the clock runs from the arrival of
    # one result to the arrival of the result `steps` requests later.
    def upload():
        return [ctx.ct_import_async(a, s_in) for a in host_in]

    host_out = [torch.empty(a.shape, dtype=torch.int64).pin_memory().numpy().view(np.uint64) for a in res]

    def export(outs):
        for c, h in zip(outs, host_out):
            ctx.ct_export_async(c, h)

    barrier()
    outs = pipe.forward(upload(), lazy_relin=lazy)
    dc = upload()
    export(outs)
    n_warm = 2
    for it in range(n_warm + args.steps):
        if it == n_warm:
            t0 = time.perf_counter()  # right behind the arrival of a result, the next request already on the GPU
        outs = pipe.forward(dc, lazy_relin=lazy)       # request it+1, enqueued while request it computes
        dc = upload()                 # request it+2: copies overlap the compute, transforms follow request it+1
        ctx.export_wait()             # request it's result is on the host
        export(outs)
    e2e_s = (time.perf_counter() - t0) / args.steps
    barrier()
    e2e_s = max_over_ranks(e2e_s, world, "cuda")
    assert all(np.array_equal(a, b) for a, b in zip(host_out, res)), "pipelined result differs from the serial one"
    del dc
    layers_per_s = aggregate(n_lin, world, step_ms * 1e-3)
    line = {
        "metric": METRIC, "value": round(layers_per_s, 3), "unit": "encrypted conv layers/s",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(step_ms, 4),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u64", "data": "synthetic",
        "config": {"workload": args.workload, "description": desc, "batch": args.batch, "linear_layers_per_step": n_lin,
                   "rotations_per_step": n_rot, "relinearisations_per_step": n_relin, "pmults_per_step": n_pm, "inner_rotations": "plain" if args.no_hoist else "hoisted (R2.7b)",
                   "square_pool": "one relinearisation per pooled output (R2.12c)" if lazy else "eager",
                   "multi_gpu": "replicas only" if world > 1 else "single", "l2": "inputs_exceed_l2: %d MiB resident" % (setup_bytes >> 20)},
        "rotations_per_s": round(world * (n_rot + n_relin) / (step_ms * 1e-3), 1),
        "images_per_s": round(world * args.batch / (step_ms * 1e-3), 2),
        "gpu_launches": int(launches), "clocks": clocks,
        "e2e": {"value": round(world * n_lin / e2e_s, 3), "unit": "encrypted conv layers/s", "h2d_bytes_per_step": int(h2d),
                "d2h_bytes_per_step": int(d2h), "ms_per_step": round(e2e_s * 1e3, 3),
                "mode": "pipelined requests: async upload (copy stream), next request enqueued before this result is collected",
                "serial_ms_per_step": round(serial_s * 1e3, 3), "serial_value": round(world * n_lin / serial_s, 3)},
        "roofline": roofline,
    }
    if rank == 0 and world == 1:
        line["cpu_baseline"] = cpu_baseline(args, pipe, budget_s=args.cpu_budget)
    del out
    return line


# ------------------------------------------------------------------------------------------------ CPU oracle arm
def level_ops(plan):
    """{L: [rotations, pmults, rescales, squares]} of one forward pass, from the planner's exact counts."""
    ops, n_ct = {}, None
    for p in plan:
        o = ops.setdefault(p["L"], [0, 0, 0, 0])
        if p["op"] == "conv":
            o[0] += p["lay"].n_inner_rot + p["lay"].n_outer_rot
            o[1] += p["lay"].n_pmult
            o[2] += p["lay"].n_out_ct
            n_ct = p["lay"].n_out_ct
        elif p["op"] == "fc":
            o[0] += p["info"]["n_rot"]
            o[1] += p["info"]["n_pmult"]
            o[2] += p["info"]["n_out_ct"]
            n_ct = p["info"]["n_out_ct"]
        elif p["op"] == "square":
            o[3] += n_ct
        elif p["op"] == "pool":
            n_ct //= 4
    return ops


class OracleSampler:
    """Times the CPU oracle (oracle/, as it stands, single-threaded) on one rotation, one PMult-accumulate, one rescale
    and one square per level the workload uses, and scales by the workload's exact operation counts."""

    def __init__(self, pkey, ops, step):
        from oracle import ckks as ck
        self.ck, self.ops = ck, ops
        self.P = ck.Params(*wl.oracle_params_args(wl.PARAMS[pkey]))
        need_sq = any(o[3] for o in ops.values())
        self.keys = ck.keygen(self.P, 1, [step], want_relin=need_sq)
        self.step = step
        rng = np.random.default_rng(0)
        self.ct, self.pt = {}, {}
        for L in ops:
            z = rng.uniform(-1, 1, self.P.n)
            self.pt[L] = ck.encode(self.P, z, L, self.P.q[L - 1])
            self.ct[L] = ck.encrypt(self.P, self.keys, ck.encode(self.P, z, L), 5)

    def sample(self):
        ck, P, total, detail = self.ck, self.P, 0.0, {}
        for L, (n_rot, n_pm, n_rs, n_sq) in sorted(self.ops.items(), reverse=True):
            ct, t = self.ct[L], {}
            if n_rot:
                t0 = time.perf_counter(); ck.rotate(P, self.keys, ct, self.step); t["rot"] = time.perf_counter() - t0
            if n_pm:
                acc = np.zeros_like(ct.c)
                t0 = time.perf_counter(); ck.pmult_acc(P, acc, ct, self.pt[L]); t["pmult"] = time.perf_counter() - t0
            if n_rs and L >= 2:
                t0 = time.perf_counter(); ck.rescale(P, ct); t["rescale"] = time.perf_counter() - t0
            if n_sq and L >= 2:
                t0 = time.perf_counter(); ck.square_relin(P, self.keys, ct); t["square"] = time.perf_counter() - t0
            total += n_rot * t.get("rot", 0) + n_pm * t.get("pmult", 0) + n_rs * t.get("rescale", 0) + n_sq * t.get("square", 0)
            detail[L] = {k: round(v, 4) for k, v in t.items()}
        return total, detail


def cpu_baseline(args, pipe, budget_s=20.0):
    pkey = WORKLOADS[args.workload][0]
    ops = level_ops(pipe.plan)
    smp = OracleSampler(pkey, ops, sorted(pipe.steps)[0])
    est, detail = smp.sample()
    n_lin = pipe.counts()[0]
    return {"value": round(n_lin / est, 6), "unit": "encrypted conv layers/s", "cores": 1, "kind": "oracle",
            "sample": "one rotation, PMult-accumulate, rescale and square+relin per level used (%s), timed once each on the "
                      "oracle and scaled by the step's exact operation counts (rotations as plain ones -- the oracle's hoisted rotation costs "
                      "the same --, squares counted before the pool); estimated oracle step %.1f s" % (
                          ", ".join("L=%d" % L for L in sorted(ops, reverse=True)), est),
            "seconds_per_op": detail}


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, on the host cores (no GPU).  Each step times the bounded sample."""
    pkey, builder, desc = WORKLOADS[args.workload]
    # exact operation counts from the oracle's own planner (oracle/fragment.py), no GPU involved
    from oracle import fragment as fr
    from oracle import ckks as ck
    P_n = 1 << (wl.PARAMS[pkey]["log2N"] - 1)
    layers, _ = builder(args.batch, 2000)
    ops, L, n_ct, n_lin, steps = {}, wl.PARAMS[pkey]["n_q"], None, 0, set()
    for ly in layers:
        o = ops.setdefault(L, [0, 0, 0, 0])
        if ly["op"] == "conv":
            S = ly["S"] or fr.select_S(fr.ConvDesc(**ly["conv"]), P_n)
            g = fr.ConvGraph(fr.ConvDesc(S=S, **ly["conv"]), P_n)
            c = g.counts()
            o[0] += c["n_inner_rot"] + c["n_outer_rot"]; o[1] += c["n_pmult"]; o[2] += c["n_out_ct"]
            n_ct, n_lin = c["n_out_ct"], n_lin + 1
            steps.update(c["rot_steps"])
            L -= 1
        elif ly["op"] == "fc":
            from oracle import network as nw
            c = nw.fc_counts(P_n, **ly["fc"])
            o[0] += c["n_rot"]; o[1] += c["n_pmult"]; o[2] += c["n_out_ct"]
            n_ct, n_lin = c["n_out_ct"], n_lin + 1
            steps.update(c["rot_steps"])
            L -= 1
        elif ly["op"] == "square":
            o[3] += n_ct
            L -= 1
        elif ly["op"] == "pool":
            n_ct //= 4
    ops = {k: v for k, v in ops.items() if any(v)}
    smp = OracleSampler(pkey, ops, sorted(steps)[0])
    for _ in range(min(args.warmup, 1)):
        smp.sample()
    ests = [smp.sample()[0] for _ in range(min(args.steps, 3))]
    est = float(np.mean(ests))
    v = round(n_lin / est, 6)
    sample = "per step: one rotation, PMult-accumulate, rescale, square+relin per level, scaled by exact counts; est. step %.1f s" % est
    return {"impl": "reference", "metric": METRIC, "value": v, "unit": "encrypted conv layers/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(est * 1e3, 1), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u64", "data": "synthetic",
            "config": {"workload": args.workload, "description": desc, "batch": args.batch},
            "cpu_baseline": {"value": v, "unit": "encrypted conv layers/s", "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": "encrypted conv layers/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=sorted(WORKLOADS))
    ap.add_argument("--batch", type=int, default=128)
    ap.add_argument("--cpu-budget", type=float, default=20.0)
    ap.add_argument("--profile-range", action="store_true", help="cudaProfilerStart/Stop around the timed steps (for ncu)")
    ap.add_argument("--plain-fc", action="store_true", help="fully connected layers by plain diagonals (no baby-step giant-step)")
    ap.add_argument("--eager-relin", action="store_true", help="x^2 and the pool after it as two steps (four relinearisations per pooled output)")
    ap.add_argument("--no-hoist", action="store_true", help="inner rotations as plain rotations (one decomposition each)")
    ap.add_argument("--sweep-L", type=int, nargs="*", help="config 5: only these limb counts")
    ap.add_argument("--sweep-dnum", type=int, nargs="*", help="config 5: only these dnum values")
    ap.add_argument("--sweep-cts", type=int, default=64, help="config 5: ciphertexts per batched rotation (BASELINE: 64)")
    ap.add_argument("--sweep-steps", type=int, default=32, help="config 5: distinct rotation amounts (BASELINE: 32)")
    ap.add_argument("--no-extras", action="store_true", help="skip the per-kernel pass, e2e and cpu_baseline (profiling runs)")
    args = ap.parse_args()
    if args.plain_fc:
        global FC_BSGS
        FC_BSGS = 1
    rank, world = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))
    if args.impl == "reference":
        if rank == 0:
            print(json.dumps(run_reference(args)), flush=True)
        return
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

"""CPU tests of bench.py's host logic: the N>1 path is "replicas only", so what must hold is
the max-over-ranks timing and the aggregate, exercised here with world_size 2 on the gloo backend, and the
--impl reference arm (the CPU oracle) printing exactly one JSON line from rank 0."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    slow = bench.max_over_ranks(10.0 + 5.0 * rank, world, "cpu")  # rank 1 is slower
    q.put((rank, slow, bench.aggregate(5, world, slow * 1e-3)))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, 29541, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, slow, agg in got:
        assert slow == 15.0                      # every rank sees the slowest rank's time
        assert abs(agg - 2 * 5 / 15e-3) < 1e-9   # whole-job units over that time


def test_oracle_op_counts_follow_the_variant_the_gpu_arm_runs():
    """bench.py's CPU arm counts the SAME operation graph as the GPU arm: hoisted inner rotations, one relinearisation per
    pooled output, baby-step giant-step fc layers (BASELINE config 2: 48 + 192 conv rotations, 78 + 28 + 21 fc rotations,
    24 + 16 lazy relinearisations), and factored weights for config 4 (scalar multiply-accumulates + one product per mask)."""
    sys.path.insert(0, ROOT)
    import bench
    layers, _ = bench.lenet_layers(128, 2000)
    ops = bench.oracle_op_counts(layers, 8192, 8, hoist=True, lazy=True)
    kinds = lambda k: sum(v for (kk, _), v in ops.items() if kk == k)
    assert kinds("rot_h") == 48 + 192 + 36 and kinds("rot") == 367 - 276
    assert ops[("square_sum4", 7)] == 24 and ops[("square_sum4", 5)] == 16 and kinds("square") == 0
    assert ops[("pmult", 8)] == 2400 and ops[("pmult", 6)] == 9600 and ops[("rescale", 8)] == 96
    eager = bench.oracle_op_counts(layers, 8192, 8, hoist=False, lazy=False)
    assert sum(v for (k, _), v in eager.items() if k == "square") == 160 and sum(v for (k, _), v in eager.items() if k == "rot") == 367
    assert not any(k == "rot_h" for k, _ in eager)
    m, _ = bench.mobilenet_layers(32, 2000)
    ops4 = bench.oracle_op_counts(m, 32768, 30, hoist=True, lazy=True)
    assert ops4[("rot_h", 30)] == 51 and ops4[("rot_h", 29)] == 640 and ops4[("rot_h", 27)] == 576
    assert ops4[("smul", 28)] == 32768 and ops4[("smul", 26)] == 32768 and ops4[("pmult", 28)] == 1024 and ops4[("pmult", 26)] == 512
    assert not any(k == "rot" for k, _ in ops4)  # ch = 1: no outer rotations at all


@pytest.mark.timeout(600)
def test_reference_arm_prints_one_line_under_torchrun_world2():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29543", os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
           "--warmup", "0", "--workload", "cfg2_lenet5_convstage"]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=580, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle" and d["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["n_gpus"] == 0 and d["cpu_baseline"]["same_graph"] is True

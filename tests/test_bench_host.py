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


def test_level_ops_counts_match_plan_shape():
    sys.path.insert(0, ROOT)
    import bench

    class Lay:
        n_inner_rot, n_outer_rot, n_pmult, n_out_ct = 48, 0, 2400, 96
    plan = [dict(op="conv", L=8, lay=Lay), dict(op="square", L=7), dict(op="pool", L=6),
            dict(op="fc", L=6, info=dict(n_rot=126, n_pmult=2048, n_out_ct=2))]
    ops = bench.level_ops(plan)
    assert ops[8] == [48, 2400, 96, 0] and ops[7] == [0, 0, 0, 96] and ops[6] == [126, 2048, 2, 0]


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
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["n_gpus"] == 2

"""CPU tests (gloo, world_size 2) of bench.py's N > 1 logic.  The path does not shard (replicas
only), so the only cross-rank step is the max-over-ranks of the device times and the aggregate seconds per step."""
import json
import os
import subprocess
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    got = bench.max_over_ranks([100.0 + 10 * rank, 7.0 - rank], "cpu")
    out.put((rank, got))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, 29533, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0] == res[1] == [110.0, 7.0]


def test_aggregate_is_whole_job_throughput():
    import bench
    # 2 replicas, 5 steps each in 3000 ms: the job completes 10 steps in 3 s
    assert bench.aggregate_seconds_per_step(3000.0, 5, 2) == pytest.approx(0.3)
    assert bench.max_over_ranks([1.5], "cpu") == [1.5]          # no process group: identity


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, env=env, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_bench_line_contract_keys():
    """The JSON line of the CUDA arm is assembled on the GPU box; here only the static contract is checked."""
    src = open(os.path.join(ROOT, "bench.py")).read()
    for key in ('"metric"', '"value"', '"unit"', '"n_gpus"', '"steps"', '"warmup"', '"ms_per_step"', '"higher_is_better"', '"scaling"',
                '"vs_baseline"', '"dtype"', '"data"', '"config"', '"e2e"', '"gpu_launches"', '"clocks"', '"roofline"', '"cpu_baseline"'):
        assert key in src, key
    assert json.loads(json.dumps({"ok": True}))["ok"]

"""N > 1 host logic on CPU (gloo, world_size 2): the path does not shard ("replicas only"), so the
only cross-rank step is the MAX over ranks of the device timings that bench.py reports."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    out = bench.max_over_ranks([10.0 + rank, 5.0 - rank])
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, out))


def test_max_over_ranks_gloo_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0] == res[1] == [11.0, 5.0]


def test_max_over_ranks_single_process_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([1.5, 2.5]) == [1.5, 2.5]


def test_reference_arm_only_rank0_prints(capsys, monkeypatch):
    sys.path.insert(0, ROOT)
    import bench
    monkeypatch.setenv("RANK", "1")
    bench.run_reference(type("A", (), {"size": 32, "gpus": 2, "steps": 1, "warmup": 0})())
    assert capsys.readouterr().out == ""


def test_bench_gpus_flag_spawns_that_many_ranks():
    """`python bench.py --gpus 2` with no WORLD_SIZE in the environment must run two ranks (it re-launches itself under
    torch.distributed.run); the dry run goes through the same spawn and MAX-over-ranks code on gloo."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--dry-run"], env=env, capture_output=True,
                         text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [json.loads(l) for l in out.stdout.splitlines() if l.startswith("{")]
    assert lines == [{"dry_run": True, "n_gpus": 2, "max_rank_seen": 1.0}]


def test_bench_refuses_a_world_size_that_contradicts_gpus(monkeypatch):
    sys.path.insert(0, ROOT)
    import bench
    import pytest
    monkeypatch.setenv("WORLD_SIZE", "1")
    with pytest.raises(SystemExit):
        bench.run_ours(type("A", (), {"size": 32, "gpus": 2, "steps": 1, "warmup": 0, "dry_run": True, "no_cpu": True})())

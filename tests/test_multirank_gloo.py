"""World-size-2 gloo test of the N>1 path of bench.py: replicas (one independent time frame per rank, no data-path
collective); whole-job figures = units summed over ranks / max time over ranks."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_1910_12214_b200 import datagen
    # every rank generates its own event, as bench.py does (seed depends on the rank)
    ev = datagen.generate(datagen.config(0, seed=1 + 100 * rank))
    units, ms = bench.aggregate(float(ev.n_clusters), 10.0 * (rank + 1), torch.device("cpu"), world)
    q.put((rank, ev.n_clusters, units, ms))
    dist.barrier()
    dist.destroy_process_group()


def test_replica_aggregation_over_two_ranks():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    n0, n1 = res[0][1], res[1][1]
    assert n0 != n1                                   # different seeds -> different events
    for (_, _, units, ms) in res:
        assert units == float(n0 + n1)                # summed over ranks
        assert ms == 20.0                             # max over ranks


def test_reference_arm_runs_on_rank_zero_only(tmp_path):
    import subprocess
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0", "--steps", "1",
                          "--warmup", "0"], capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0 and out.stdout.strip() == ""
    env = dict(os.environ, RANK="0", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0", "--steps", "1",
                          "--warmup", "0"], capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0
    import json
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"


def test_bench_spawns_its_own_ranks_when_no_launcher_did():
    """`python bench.py --gpus 2` without WORLD_SIZE starts two ranks itself (torch.distributed.run on 127.0.0.1); with
    --dry-run they rendezvous over gloo, each contributes its own figures through bench.aggregate(), and rank 0 alone
    prints the one line: units summed over ranks (1000 + 2000), time = max over ranks (20 ms), n_gpus = the world used."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--dry-run"], capture_output=True,
                         text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    line = json.loads(lines[0])
    assert line["n_gpus"] == 2 and line["units"] == 3000.0 and line["ms"] == 20.0


def test_bench_refuses_a_world_that_differs_from_gpus():
    import subprocess
    env = dict(os.environ, RANK="0", WORLD_SIZE="1", LOCAL_RANK="0")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "8", "--dry-run"], capture_output=True,
                         text=True, env=env, timeout=120)
    assert out.returncode == 2 and "--gpus 8" in out.stderr

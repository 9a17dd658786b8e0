"""Host logic of the N>1 path of bench.py ("replicas only"): the max-over-ranks timing
and the whole-job aggregate, on CPU with the gloo backend and world_size 2."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    t_rank = 0.5 if rank == 0 else 2.0                       # rank 1 is the slow replica
    value, t = bench.whole_job_value(1000, 4, t_rank, world)
    out[rank] = (value, t, bench.max_over_ranks(float(rank), world))
    dist.barrier()
    dist.destroy_process_group()


def test_whole_job_value_world2_gloo():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
        for r in (0, 1):
            value, t, mx = out[r]
            assert t == 2.0 and mx == 1.0
            assert value == 2 * 1000 * 4 / 2.0


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.whole_job_value(10, 3, 0.5, 1) == (60.0, 0.5)
    v, why = bench.ncu_traffic_bytes("no-such-workload")
    assert v is None and isinstance(why, str)               # never a stale or foreign capture


def test_gpus_flag_starts_the_replicas_itself():
    """`python bench.py --gpus 2` with WORLD_SIZE unset (how the driver may call it) must start two replica
    processes and report n_gpus 2: the launcher re-executes bench.py under torch.distributed.run.  --dry-run
    keeps the GPU out of it (gloo; every rank 'takes' 1 + rank/10 s for 1000 units per step)."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--dry-run", "--steps", "3"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1                                   # rank 0 alone prints
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["slowest_rank_s"] == 1.1
    assert abs(d["value"] - 2 * 1000 * 3 / 1.1) < 1e-9

"""N > 1 host logic of bench.py: no data-path collective,
time = max over ranks, value = sum of the replicas' site-updates / that time.  world_size 2, gloo,
CPU only."""
import os
import socket
import subprocess
import sys

import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank,
                            world_size=world)
    ms_local = [10.0, 30.0][rank]                       # rank 1 is the slow replica
    ms, e2e = bench.max_over_ranks([ms_local, 1.0 + rank], dist, "cpu")
    out[rank] = (ms, e2e, bench.job_value(world, 1000, 5, ms))
    dist.destroy_process_group()


def test_max_over_ranks_and_job_value_world2():
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    assert out[0] == out[1]                             # every rank sees the same aggregate
    ms, e2e, value = out[0]
    assert ms == 30.0 and e2e == 2.0
    assert value == 2 * 1000 * 5 / 30e-3                # both replicas' units over the max time


def test_max_over_ranks_without_group_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([1.5, 2.5]) == [1.5, 2.5]


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference",
                        "--gpus", "2", "--steps", "1", "--warmup", "0"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""

"""N > 1 is "replicas only": every rank solves its own bunch, there is no data-path
collective, and bench.py reports (solves of all ranks) / (device time of the slowest rank).  This covers that
host-side logic with two gloo ranks on CPU (rendezvous on 127.0.0.1), plus the reference arm's rule that only
rank 0 works under torchrun."""
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        local_ms = 100.0 * (rank + 1)                    # rank 1 is the slow one
        ms = bench.max_over_ranks(local_ms, "cpu")
        out[rank] = (ms, bench.whole_job_value(world, 50, ms))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_replicas_timing_is_max_over_ranks_and_value_is_whole_job():
    import torch.multiprocessing as mp
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1]
    ms, value = res[0]
    assert ms == 200.0
    assert value == pytest.approx(2 * 50 / 0.2)


def test_single_process_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(12.5, "cpu") == 12.5
    assert bench.whole_job_value(1, 10, 5.0) == pytest.approx(2000.0)


def test_reference_arm_runs_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--config", "1", "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and r.stdout.strip() == ""

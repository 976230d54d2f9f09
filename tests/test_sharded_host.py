"""The sharded solve's partition and exchange schedule (paper_1509_07685_b200/sharded.py; SURVEY.md sections 8(e), 8(f3)) on
two gloo ranks with CPU tensors: the two all-to-alls move exactly the slices the partition says (y slabs -> kz slabs -> y
slabs).  The fused transport of the CUDA path (peer stores in the epilogues of P1 and P4) realises the same schedule;
it is checked on one GPU by tests/test_gpu_sharded.py."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_partition_covers_everything_once():
    sys.path.insert(0, ROOT)
    from paper_1509_07685_b200 import sharded as S
    for n, g in [(32, 1), (32, 2), (64, 4), (256, 8)]:
        rows = [S.y_slab(n, r, g) for r in range(g)]
        assert rows[0][0] == 0 and all(rows[r][0] + rows[r][1] == rows[r + 1][0] for r in range(g - 1))
        assert rows[-1][0] + rows[-1][1] == n and len({c for _, c in rows}) == 1
        planes = [S.kz_slab(n, r, g) for r in range(g)]
        assert planes[0][0] == 0 and all(planes[r][0] + planes[r][1] == planes[r + 1][0] for r in range(g - 1))
        assert planes[-1][0] + planes[-1][1] == n + 1          # n + 1 half-spectrum planes; the last rank holds the extra one


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_1509_07685_b200 import sharded as S
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        nx, ny, nz = 8, 12, 6                                   # the schedule does not need powers of two
        rng = np.random.default_rng(0)                          # same global array on every rank
        A = torch.from_numpy(rng.standard_normal((nz + 1, ny, nx)) + 1j * rng.standard_normal((nz + 1, ny, nx)))
        y0, yc = S.y_slab(ny, rank, world)
        k0, kc = S.kz_slab(nz, rank, world)
        mine_y = A[:, y0:y0 + yc].contiguous()                  # what P1 produces on this rank
        got_kz = S.exchange_y_to_kz(mine_y, nz)
        ok1 = bool(torch.equal(got_kz, A[k0:k0 + kc]))          # every y row of this rank's planes, in global order
        back = S.exchange_kz_to_y(got_kz * 2.0, ny)             # what P4 produces, sent back
        ok2 = bool(torch.equal(back, 2.0 * mine_y))
        out[rank] = (ok1, ok2, tuple(got_kz.shape), tuple(back.shape))
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_exchange_schedule_on_gloo(world):
    import torch.multiprocessing as mp
    port = _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert len(res) == world
    for r in range(world):
        ok1, ok2, s1, s2 = res[r]
        assert ok1 and ok2, (r, res[r])
        assert s1 == (6 // world + (1 if r == world - 1 else 0), 12, 8) and s2 == (7, 12 // world, 8)

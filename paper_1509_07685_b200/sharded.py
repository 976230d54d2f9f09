"""One Poisson solve sharded over several GPUs (SURVEY.md sections 8(e), 8(f3)).

Partition: rank r of g owns the y rows [r ny/g, (r+1) ny/g) of rho / phi ("y slab") and the half-spectrum planes
kz in [r nz/g, (r+1) nz/g), the last rank also plane nz ("kz slab").  Pipeline per solve:

    phase 1   P1 on the y slab; every output row is stored into the receive buffer of the rank owning its kz plane
    barrier
    phase 2   P2, P3, P4 on the kz slab; P4 stores every output row into the receive buffer of the rank owning its y row
    barrier
    phase 3   P5 on the y slab

Two transports for the two exchanges (each an all-to-all of buffer A, 269 MB in total at 256^3):
  * fused (the product path on NVLink / NVSwitch): the producing kernels store straight into peer-mapped receive buffers
    (`ShardedPoissonSolver`, torch symmetric memory for the mapping, one NCCL barrier between phases);
  * `exchange_y_to_kz` / `exchange_kz_to_y`: the same data movement as a plain `torch.distributed.all_to_all` of slices,
    backend-agnostic (NCCL or gloo).  It defines the exchange schedule, is what the 2-rank gloo test checks on CPU tensors,
    and is the reference the fused transport must reproduce.
`EmulatedShardedSolver` runs all g ranks' kernels one after another on ONE device with local pointers in the peer tables:
every index computation of the sharded path is exercised on a single GPU (the only hardware this repo is tested on).
This module only marshals: every step of the solve runs in the CUDA kernels of libdks_poisson.so.
"""
from __future__ import annotations


def y_slab(ny: int, rank: int, nranks: int):
    """(first row, rows) of rank's y slab."""
    assert ny % nranks == 0
    return rank * (ny // nranks), ny // nranks


def kz_slab(nz: int, rank: int, nranks: int):
    """(first plane, planes) of rank's kz slab of the nz + 1 half-spectrum planes; the last rank takes plane nz too."""
    assert nz % nranks == 0
    s = nz // nranks
    return rank * s, s + (1 if rank == nranks - 1 else 0)


def _all_to_all_slices(send, recv_shapes, like, group):
    """all_to_all_single over flattened float64 views (works on NCCL and on gloo, complex or real payload)."""
    import torch
    import torch.distributed as dist
    real = lambda t: torch.view_as_real(t) if t.is_complex() else t
    flat = torch.cat([real(t.contiguous()).reshape(-1) for t in send])
    per = 2 if like.is_complex() else 1
    in_split = [real(t).numel() for t in send]
    out_split = [per * int(torch.Size(sh).numel()) for sh in recv_shapes]
    out = torch.empty(sum(out_split), dtype=flat.dtype, device=flat.device)
    dist.all_to_all_single(out, flat, output_split_sizes=out_split, input_split_sizes=in_split, group=group)
    pieces, pos = [], 0
    for sh, cnt in zip(recv_shapes, out_split):
        piece = out[pos:pos + cnt]
        pieces.append(torch.view_as_complex(piece.reshape(tuple(sh) + (2,))) if like.is_complex() else piece.reshape(tuple(sh)))
        pos += cnt
    return pieces


def exchange_y_to_kz(a_y, nz: int, group=None):
    """All-to-all #1.  a_y: this rank's P1 output [nz + 1, ny_loc, nx] (complex); returns its kz slab [planes, ny, nx]."""
    import torch
    import torch.distributed as dist
    g, r = dist.get_world_size(group), dist.get_rank(group)
    send = [a_y[slice(*_span(kz_slab(nz, d, g)))] for d in range(g)]
    k0, planes = kz_slab(nz, r, g)
    recv = _all_to_all_slices(send, [(planes,) + tuple(a_y.shape[1:])] * g, a_y, group)
    return torch.cat(recv, dim=1)                                   # y slabs of all source ranks, in rank order


def exchange_kz_to_y(a_kz, ny: int, group=None):
    """All-to-all #2.  a_kz: this rank's P4 output [planes, ny, nx]; returns its y slab [nz + 1, ny_loc, nx]."""
    import torch
    import torch.distributed as dist
    g, r = dist.get_world_size(group), dist.get_rank(group)
    nz = _nz_from_planes(a_kz.shape[0], r, g)
    send = [a_kz[:, slice(*_span(y_slab(ny, d, g)))] for d in range(g)]
    recv = _all_to_all_slices(send, [(kz_slab(nz, s, g)[1], ny // g, a_kz.shape[2]) for s in range(g)], a_kz, group)
    return torch.cat(recv, dim=0)                                   # kz slabs of all source ranks, in rank order


def _span(first_count):
    return first_count[0], first_count[0] + first_count[1]


def _nz_from_planes(planes, rank, nranks):
    return (planes - (1 if rank == nranks - 1 else 0)) * nranks


class _ShardPlan:
    def __init__(self, n, h, rank, nranks):
        import torch
        from . import dks
        self.dks, self.n, self.rank, self.nranks = dks, tuple(n), rank, nranks
        self.handle = dks.dks_poisson_plan_create(*n, *h)
        dks.dks_poisson_set_shard(self.handle, rank, nranks)
        nbytes = dks.dks_poisson_workspace_bytes(self.handle)
        self.ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        dks.dks_poisson_set_workspace(self.handle, self.ws, nbytes)
        dks.dks_poisson_set_stream(self.handle, torch.cuda.current_stream().cuda_stream)
        dks.dks_greens_setup(self.handle)
        self.recv1, self.recv4 = dks.dks_poisson_shard_buffers(self.handle)

    def phase(self, k, rho_loc=None, phi_loc=None):
        import torch
        self.dks.dks_poisson_solve_shard(self.handle, k, rho_loc, phi_loc, torch.cuda.current_stream().cuda_stream)

    def close(self):
        if self.handle:
            self.dks.dks_poisson_plan_destroy(self.handle)
            self.handle = None


class EmulatedShardedSolver:
    """All g ranks of a sharded solve on ONE device: g plans whose peer tables point at each other's (local) buffers; the
    phases of all ranks are issued rank after rank on one stream, whose order is the inter-rank barrier."""

    def __init__(self, n, h, nranks):
        self.n, self.nranks = tuple(n), nranks
        self.plans = [_ShardPlan(n, h, r, nranks) for r in range(nranks)]
        t1, t4 = [p.recv1 for p in self.plans], [p.recv4 for p in self.plans]
        for p in self.plans:
            p.dks.dks_poisson_set_peers(p.handle, t1, t4)

    def solve(self, rho):
        """rho: CUDA float64 [nz, ny, nx]; returns phi of the same shape, assembled from the ranks' y slabs."""
        import torch
        nx, ny, nz = self.n
        g = self.nranks
        rho_slabs = [rho[:, slice(*_span(y_slab(ny, r, g)))].contiguous() for r in range(g)]
        phi_slabs = [torch.empty_like(s) for s in rho_slabs]
        for r, p in enumerate(self.plans):
            p.phase(1, rho_loc=rho_slabs[r])
        for p in self.plans:
            p.phase(2)
        for r, p in enumerate(self.plans):
            p.phase(3, phi_loc=phi_slabs[r])
        return torch.cat(phi_slabs, dim=1)

    def close(self):
        import torch
        torch.cuda.synchronize()
        for p in self.plans:
            p.close()


class ShardedPoissonSolver:
    """One rank of a sharded solve under torch.distributed (backend nccl, one process per GPU).  The receive buffers live
    in torch symmetric memory, so every peer's buffer is addressable from this device and the kernels' stores travel over
    NVLink.  Needs >= 2 GPUs with peer access; this repo's test hardware has one, so this class is covered by construction
    only (the kernels and index tables are those of EmulatedShardedSolver, the exchange pattern that of exchange_y_to_kz)."""

    def __init__(self, n, h, group=None):
        import torch
        import torch.distributed as dist
        import torch.distributed._symmetric_memory as symm
        from . import dks
        if torch.cuda.device_count() < 2 or not dist.is_initialized() or dist.get_world_size(group) < 2:
            raise RuntimeError("ShardedPoissonSolver needs torch.distributed (nccl) with at least two GPUs")
        self.dks, self.group, self.n = dks, group, tuple(n)
        self.rank, self.nranks = dist.get_rank(group), dist.get_world_size(group)
        self.handle = dks.dks_poisson_plan_create(*n, *h)
        dks.dks_poisson_set_shard(self.handle, self.rank, self.nranks)
        nbytes = dks.dks_poisson_workspace_bytes(self.handle)
        # the whole workspace is symmetric memory: same size on every rank except for the last rank's extra plane, so
        # allocate the maximum over ranks
        t = torch.tensor([nbytes], dtype=torch.int64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
        self.ws = symm.empty(int(t.item()), dtype=torch.uint8, device="cuda")
        hdl = symm.rendezvous(self.ws, group=group if group is not None else dist.group.WORLD)
        dks.dks_poisson_set_workspace(self.handle, self.ws, self.ws.numel())
        dks.dks_poisson_set_stream(self.handle, torch.cuda.current_stream().cuda_stream)
        dks.dks_greens_setup(self.handle)
        r1, r4 = dks.dks_poisson_shard_buffers(self.handle)
        off1, off4 = r1 - self.ws.data_ptr(), r4 - self.ws.data_ptr()
        # offsets of the receive buffers inside the workspace differ between ranks (the last rank has one plane more)
        offs = torch.tensor([off1, off4], dtype=torch.int64, device="cuda")
        all_offs = [torch.empty_like(offs) for _ in range(self.nranks)]
        dist.all_gather(all_offs, offs, group=group)
        bases = [int(hdl.buffer_ptrs[r]) for r in range(self.nranks)]
        dks.dks_poisson_set_peers(self.handle, [bases[r] + int(all_offs[r][0]) for r in range(self.nranks)],
                                  [bases[r] + int(all_offs[r][1]) for r in range(self.nranks)])
        dist.barrier(group=group)

    def solve(self, rho_loc, phi_loc=None):
        """rho_loc: this rank's y slab, CUDA float64 [nz, ny/g, nx]; returns phi_loc."""
        import torch
        import torch.distributed as dist
        if phi_loc is None:
            phi_loc = torch.empty_like(rho_loc)
        st = torch.cuda.current_stream().cuda_stream
        self.dks.dks_poisson_solve_shard(self.handle, 1, rho_loc, None, st)
        dist.barrier(group=self.group)                 # all P1 rows have landed (NCCL barrier: ordered on the current stream)
        self.dks.dks_poisson_solve_shard(self.handle, 2, None, None, st)
        dist.barrier(group=self.group)
        self.dks.dks_poisson_solve_shard(self.handle, 3, None, phi_loc, st)
        return phi_loc

    def close(self):
        if self.handle:
            import torch
            torch.cuda.synchronize()
            self.dks.dks_poisson_plan_destroy(self.handle)
            self.handle = None

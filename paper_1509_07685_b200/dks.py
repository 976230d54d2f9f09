"""Thin ctypes binding of the C ABI in include/dks_poisson.h (same names, argument marshalling only).

Every step of the solve runs in the CUDA kernels of libdks_poisson.so; PyTorch is used here only for
device memory and streams.  There is no CPU fallback: if the library cannot be loaded, importing
this module raises.
"""
from __future__ import annotations

import ctypes as C
import os

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))

DKS_OK = 0
DKS_ERR_INVALID_ARG = -1
DKS_ERR_UNSUPPORTED_DEVICE = -2
DKS_ERR_WORKSPACE_TOO_SMALL = -4
DKS_ERR_NOT_SETUP = -5
DKS_ERR_CUDA = -6

# every symbol include/dks_poisson.h declares: name -> (restype, argtypes)
_vp, _i, _d, _sz = C.c_void_p, C.c_int, C.c_double, C.c_size_t
SYMBOLS = {
    "dks_poisson_plan_create": (_vp, [_i, _i, _i, _d, _d, _d]),
    "dks_poisson_plan_destroy": (None, [_vp]),
    "dks_greens_setup": (_i, [_vp]),
    "dks_poisson_solve": (_i, [_vp, _vp, _vp, _vp]),
    "dks_poisson_set_max_batch": (_i, [_vp, _i]),
    "dks_poisson_solve_batch": (_i, [_vp, _vp, _vp, _i, _vp]),
    "dks_poisson_solve_host": (_i, [_vp, _vp, _vp, _vp]),
    "dks_poisson_solve_host_async": (_i, [_vp, _vp, _vp, _vp]),
    "dks_poisson_host_sync": (_i, [_vp]),
    "dks_poisson_step_host_async": (_i, [_vp, _d, _d, _d, _vp, _vp, _vp]),
    "dks_poisson_set_spacing": (_i, [_vp, _d, _d, _d]),
    "dks_poisson_set_g0": (_i, [_vp, _d]),
    "dks_poisson_workspace_bytes": (_sz, [_vp]),
    "dks_poisson_set_workspace": (_i, [_vp, _vp, _sz]),
    "dks_poisson_set_host_staging": (_i, [_vp, _i]),
    "dks_poisson_set_stream": (_i, [_vp, _vp]),
    "dks_poisson_set_slab_planes": (_i, [_vp, _i]),
    "dks_poisson_slab_planes": (_i, [_vp]),
    "dks_poisson_set_profiling": (_i, [_vp, _i]),
    "dks_poisson_pass_times": (_i, [_vp, C.POINTER(C.c_float), _i]),
    "dks_poisson_launches_per_solve": (_i, [_vp]),
    "dks_poisson_model_bytes": (_d, [_vp, _i]),
    "dks_poisson_pass_name": (C.c_char_p, [_vp, _i]),
    "dks_poisson_copy_greens_hat": (_i, [_vp, _vp]),
    "dks_deposit_cic": (_i, [_vp, _vp, _vp, _vp, _vp, C.c_longlong, _d, _d, _d, _vp, _vp]),
    "dks_gradient": (_i, [_vp, _vp, _vp, _vp, _vp, _vp]),
    "dks_gather_field": (_i, [_vp, _vp, _vp, _vp, _vp, _vp, _vp, C.c_longlong, _d, _d, _d, _vp, _vp, _vp, _vp]),
    "dks_field_at_particles": (_i, [_vp, _vp, _vp, _vp, _vp, C.c_longlong, _d, _d, _d, _vp, _vp, _vp, _vp]),
    "dks_field_at_particles_static": (_i, [_i, _i, _i, _d, _d, _d, _vp, _vp, _vp, _vp, C.c_longlong, _d, _d, _d, _vp, _vp, _vp, _vp]),
    "dks_poisson_set_shard": (_i, [_vp, _i, _i]),
    "dks_poisson_shard_buffers": (_i, [_vp, C.POINTER(_vp), C.POINTER(_vp)]),
    "dks_poisson_set_peers": (_i, [_vp, C.POINTER(_vp), C.POINTER(_vp)]),
    "dks_poisson_solve_shard": (_i, [_vp, _i, _vp, _vp, _vp]),
    "dks_last_error": (C.c_char_p, []),
}


def _load():
    path = _build.build()              # returns at once when the library is newer than its sources; compiling the
                                       # product is not a fallback, and a failed build raises
    lib = C.CDLL(path)
    for name, (res, args) in SYMBOLS.items():
        f = getattr(lib, name)         # AttributeError if the library does not export it
        f.restype, f.argtypes = res, args
    return lib


lib = _load()
LIB_PATH = _build.LIB


class DksError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        super().__init__(f"{where}: status {status}: {dks_last_error()}")


def dks_last_error() -> str:
    return lib.dks_last_error().decode()


def _check(status, where):
    if status < 0:
        raise DksError(status, where)
    return status


def _ptr(t):
    """Device (or host) address of a torch tensor / numpy array / raw int."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        return t.data_ptr()
    return t.ctypes.data


# ---- the C ABI, name for name -------------------------------------------------------------------
def dks_poisson_plan_create(nx, ny, nz, hx, hy, hz):
    h = lib.dks_poisson_plan_create(int(nx), int(ny), int(nz), float(hx), float(hy), float(hz))
    if not h:
        raise DksError(DKS_ERR_INVALID_ARG, "dks_poisson_plan_create")
    return h


def dks_poisson_plan_destroy(plan):
    lib.dks_poisson_plan_destroy(plan)


def dks_greens_setup(plan):
    return _check(lib.dks_greens_setup(plan), "dks_greens_setup")


def dks_poisson_solve(plan, rho_dev, phi_dev, stream=None):
    return _check(lib.dks_poisson_solve(plan, _ptr(rho_dev), _ptr(phi_dev), stream), "dks_poisson_solve")


def dks_poisson_set_max_batch(plan, nbatch):
    return _check(lib.dks_poisson_set_max_batch(plan, int(nbatch)), "dks_poisson_set_max_batch")


def dks_poisson_solve_batch(plan, rho_dev, phi_dev, nbatch, stream=None):
    return _check(lib.dks_poisson_solve_batch(plan, _ptr(rho_dev), _ptr(phi_dev), int(nbatch), stream),
                  "dks_poisson_solve_batch")


def dks_poisson_solve_host(plan, rho_host, phi_host, stream=None):
    return _check(lib.dks_poisson_solve_host(plan, _ptr(rho_host), _ptr(phi_host), stream), "dks_poisson_solve_host")


def dks_poisson_solve_host_async(plan, rho_host, phi_host, stream=None):
    return _check(lib.dks_poisson_solve_host_async(plan, _ptr(rho_host), _ptr(phi_host), stream),
                  "dks_poisson_solve_host_async")


def dks_poisson_step_host_async(plan, hx, hy, hz, rho_host, phi_host, stream=None):
    return _check(lib.dks_poisson_step_host_async(plan, float(hx), float(hy), float(hz), _ptr(rho_host), _ptr(phi_host), stream),
                  "dks_poisson_step_host_async")


def dks_poisson_host_sync(plan):
    return _check(lib.dks_poisson_host_sync(plan), "dks_poisson_host_sync")


def dks_poisson_set_spacing(plan, hx, hy, hz):
    return _check(lib.dks_poisson_set_spacing(plan, float(hx), float(hy), float(hz)), "dks_poisson_set_spacing")


def dks_poisson_set_g0(plan, g0_or_nan):
    return _check(lib.dks_poisson_set_g0(plan, float(g0_or_nan)), "dks_poisson_set_g0")


def dks_poisson_workspace_bytes(plan) -> int:
    return int(lib.dks_poisson_workspace_bytes(plan))


def dks_poisson_set_workspace(plan, dev, nbytes=None):
    if nbytes is None:
        nbytes = dev.numel() * dev.element_size()
    return _check(lib.dks_poisson_set_workspace(plan, _ptr(dev), int(nbytes)), "dks_poisson_set_workspace")


def dks_poisson_set_host_staging(plan, enabled):
    return _check(lib.dks_poisson_set_host_staging(plan, int(bool(enabled))), "dks_poisson_set_host_staging")


def dks_poisson_set_stream(plan, stream):
    return _check(lib.dks_poisson_set_stream(plan, stream), "dks_poisson_set_stream")


def dks_poisson_set_slab_planes(plan, planes):
    return _check(lib.dks_poisson_set_slab_planes(plan, int(planes)), "dks_poisson_set_slab_planes")


def dks_poisson_slab_planes(plan) -> int:
    return _check(lib.dks_poisson_slab_planes(plan), "dks_poisson_slab_planes")


def dks_poisson_set_profiling(plan, slots):
    return _check(lib.dks_poisson_set_profiling(plan, int(slots)), "dks_poisson_set_profiling")


def dks_poisson_pass_times(plan, count=16):
    buf = (C.c_float * count)()
    n = _check(lib.dks_poisson_pass_times(plan, buf, count), "dks_poisson_pass_times")
    return [buf[i] for i in range(n)]


def dks_poisson_launches_per_solve(plan) -> int:
    return _check(lib.dks_poisson_launches_per_solve(plan), "dks_poisson_launches_per_solve")


def dks_poisson_model_bytes(plan, pass_index=0) -> float:
    return float(lib.dks_poisson_model_bytes(plan, int(pass_index)))


def dks_poisson_pass_name(plan, pass_index) -> str:
    return lib.dks_poisson_pass_name(plan, int(pass_index)).decode()


def dks_poisson_copy_greens_hat(plan, host_out):
    return _check(lib.dks_poisson_copy_greens_hat(plan, _ptr(host_out)), "dks_poisson_copy_greens_hat")


def dks_deposit_cic(plan, x, y, z, q, np_, origin, rho, stream=None):
    return _check(lib.dks_deposit_cic(plan, _ptr(x), _ptr(y), _ptr(z), _ptr(q), int(np_), *(float(v) for v in origin),
                                      _ptr(rho), stream), "dks_deposit_cic")


def dks_gradient(plan, phi, ex, ey, ez, stream=None):
    return _check(lib.dks_gradient(plan, _ptr(phi), _ptr(ex), _ptr(ey), _ptr(ez), stream), "dks_gradient")


def dks_gather_field(plan, ex, ey, ez, x, y, z, np_, origin, epx, epy, epz, stream=None):
    return _check(lib.dks_gather_field(plan, _ptr(ex), _ptr(ey), _ptr(ez), _ptr(x), _ptr(y), _ptr(z), int(np_),
                                       *(float(v) for v in origin), _ptr(epx), _ptr(epy), _ptr(epz), stream), "dks_gather_field")


def dks_field_at_particles(plan, phi, x, y, z, np_, origin, epx, epy, epz, stream=None):
    return _check(lib.dks_field_at_particles(plan, _ptr(phi), _ptr(x), _ptr(y), _ptr(z), int(np_), *(float(v) for v in origin),
                                             _ptr(epx), _ptr(epy), _ptr(epz), stream), "dks_field_at_particles")


DKS_STATIC_FIELD_MAX_NODES = 1 << 18
MAX_RANKS = 8                          # kMaxRanks in csrc/dks_passes_r16.cuh


def dks_field_at_particles_static(n, h, phi, x, y, z, np_, origin, epx, epy, epz, stream=None):
    """dks_field_at_particles for callers that must not allocate device memory (a loop that a cudaMalloc would stall, a
    host program whose pool owns the whole device, a component without an allocator): no plan; the node field goes through
    an 8 MiB array inside the library, so nx * ny * nz <= DKS_STATIC_FIELD_MAX_NODES.  Calls on one device share that
    array: do not let two of them overlap on the GPU.  n = (nx, ny, nz), h = (hx, hy, hz); everything else as in
    dks_field_at_particles.  This wrapper only passes the pointers on; the outputs are the caller's."""
    return _check(lib.dks_field_at_particles_static(*(int(v) for v in n), *(float(v) for v in h), _ptr(phi), _ptr(x), _ptr(y),
                                                    _ptr(z), int(np_), *(float(v) for v in origin), _ptr(epx), _ptr(epy),
                                                    _ptr(epz), stream), "dks_field_at_particles_static")


def dks_poisson_set_shard(plan, rank, nranks):
    return _check(lib.dks_poisson_set_shard(plan, int(rank), int(nranks)), "dks_poisson_set_shard")


def dks_poisson_shard_buffers(plan):
    a, b = _vp(), _vp()
    _check(lib.dks_poisson_shard_buffers(plan, C.byref(a), C.byref(b)), "dks_poisson_shard_buffers")
    return a.value, b.value


def dks_poisson_set_peers(plan, recv_p1_of_rank, recv_p4_of_rank):
    # The C side reads one entry per rank and does not know the tables' lengths: pad both to the largest rank count the library
    # supports (8) with NULL, which it rejects by rank number, so a table that is too short is an error instead of a wild read.
    n1, n2 = len(recv_p1_of_rank), len(recv_p4_of_rank)
    if n1 != n2 or not 2 <= n1 <= MAX_RANKS:
        raise ValueError(f"peer tables must have the same length in [2, {MAX_RANKS}] (got {n1} and {n2})")
    t1 = (_vp * MAX_RANKS)(*recv_p1_of_rank, *([None] * (MAX_RANKS - n1)))
    t2 = (_vp * MAX_RANKS)(*recv_p4_of_rank, *([None] * (MAX_RANKS - n2)))
    return _check(lib.dks_poisson_set_peers(plan, t1, t2), "dks_poisson_set_peers")


def dks_poisson_solve_shard(plan, phase, rho_loc, phi_loc, stream=None):
    return _check(lib.dks_poisson_solve_shard(plan, int(phase), _ptr(rho_loc), _ptr(phi_loc), stream), "dks_poisson_solve_shard")


# ---- convenience wrapper (still marshalling only) ---------------------------------------------------
class PoissonPlan:
    """Owns a dks_poisson_plan and a torch-allocated workspace on the current CUDA device."""

    def __init__(self, n, h, g0=None, own_workspace=True, slab_planes=None, max_batch=None, host_staging=True):
        import torch

        self.n, self.h = tuple(int(v) for v in n), tuple(float(v) for v in h)
        self._plan = dks_poisson_plan_create(*self.n, *self.h)
        self._ws = None
        if g0 is not None:
            dks_poisson_set_g0(self._plan, g0)
        if slab_planes is not None:
            dks_poisson_set_slab_planes(self._plan, slab_planes)
        if max_batch is not None:
            dks_poisson_set_max_batch(self._plan, max_batch)
        if not host_staging:
            dks_poisson_set_host_staging(self._plan, False)
        if own_workspace:
            nbytes = dks_poisson_workspace_bytes(self._plan)
            self._ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
            dks_poisson_set_workspace(self._plan, self._ws, nbytes)
        dks_poisson_set_stream(self._plan, torch.cuda.current_stream().cuda_stream)
        dks_greens_setup(self._plan)

    @property
    def handle(self):
        return self._plan

    def set_spacing(self, h):
        import torch

        self.h = tuple(float(v) for v in h)
        dks_poisson_set_spacing(self._plan, *self.h)
        dks_poisson_set_stream(self._plan, torch.cuda.current_stream().cuda_stream)
        dks_greens_setup(self._plan)

    def solve(self, rho, phi=None):
        """rho, phi: CUDA float64 tensors of shape [nz, ny, nx]; runs on torch's current stream."""
        import torch

        nx, ny, nz = self.n
        if not (rho.is_cuda and rho.dtype == torch.float64 and rho.is_contiguous() and tuple(rho.shape) == (nz, ny, nx)):
            raise ValueError(f"rho must be a contiguous CUDA float64 tensor of shape {(nz, ny, nx)}")
        if phi is None:
            phi = torch.empty_like(rho)
        elif not (phi.is_cuda and phi.dtype == torch.float64 and phi.is_contiguous() and phi.shape == rho.shape):
            raise ValueError("phi must match rho")
        dks_poisson_solve(self._plan, rho, phi, torch.cuda.current_stream().cuda_stream)
        return phi

    def solve_batch(self, rho, phi=None):
        """rho, phi: CUDA float64 tensors of shape [nbatch, nz, ny, nx]; one launch per pass for the whole batch."""
        import torch

        nx, ny, nz = self.n
        if not (rho.is_cuda and rho.dtype == torch.float64 and rho.is_contiguous() and tuple(rho.shape[1:]) == (nz, ny, nx)):
            raise ValueError(f"rho must be a contiguous CUDA float64 tensor of shape (nbatch, {nz}, {ny}, {nx})")
        if phi is None:
            phi = torch.empty_like(rho)
        elif not (phi.is_cuda and phi.dtype == torch.float64 and phi.is_contiguous() and phi.shape == rho.shape):
            raise ValueError("phi must match rho")
        dks_poisson_solve_batch(self._plan, rho, phi, rho.shape[0], torch.cuda.current_stream().cuda_stream)
        return phi

    def solve_host(self, rho_host, phi_host):
        """rho_host, phi_host: host float64 arrays/tensors [nz, ny, nx] (pinned recommended); synchronous."""
        import torch

        dks_poisson_solve_host(self._plan, rho_host, phi_host, torch.cuda.current_stream().cuda_stream)
        return phi_host

    def solve_host_async(self, rho_host, phi_host):
        """As solve_host without the final wait: consecutive calls overlap their copies; finish with host_sync()."""
        import torch

        dks_poisson_solve_host_async(self._plan, rho_host, phi_host, torch.cuda.current_stream().cuda_stream)
        return phi_host

    def step_host_async(self, h, rho_host, phi_host):
        """One time step with new spacings h: Green's rebuild overlapped with the copy of rho; finish with host_sync()."""
        import torch

        self.h = tuple(float(v) for v in h)
        dks_poisson_step_host_async(self._plan, *self.h, rho_host, phi_host, torch.cuda.current_stream().cuda_stream)
        return phi_host

    def host_sync(self):
        dks_poisson_host_sync(self._plan)

    def deposit(self, x, y, z, q, origin, rho=None):
        """CUDA float64 particle arrays (SoA) -> rho [nz, ny, nx] on torch's current stream."""
        import torch

        nx, ny, nz = self.n
        if rho is None:
            rho = torch.empty((nz, ny, nx), dtype=torch.float64, device=x.device)
        dks_deposit_cic(self._plan, x, y, z, q, x.numel(), origin, rho, torch.cuda.current_stream().cuda_stream)
        return rho

    def gradient(self, phi):
        import torch

        ex, ey, ez = torch.empty_like(phi), torch.empty_like(phi), torch.empty_like(phi)
        dks_gradient(self._plan, phi, ex, ey, ez, torch.cuda.current_stream().cuda_stream)
        return ex, ey, ez

    def gather(self, ex, ey, ez, x, y, z, origin):
        import torch

        epx, epy, epz = torch.empty_like(x), torch.empty_like(x), torch.empty_like(x)
        dks_gather_field(self._plan, ex, ey, ez, x, y, z, x.numel(), origin, epx, epy, epz, torch.cuda.current_stream().cuda_stream)
        return epx, epy, epz

    def field_at_particles(self, phi, x, y, z, origin):
        import torch

        epx, epy, epz = torch.empty_like(x), torch.empty_like(x), torch.empty_like(x)
        dks_field_at_particles(self._plan, phi, x, y, z, x.numel(), origin, epx, epy, epz, torch.cuda.current_stream().cuda_stream)
        return epx, epy, epz

    def greens_hat(self):
        import numpy as np

        nx, ny, nz = self.n
        out = np.empty((nz + 1, ny + 1, nx + 1), dtype=np.float64)
        dks_poisson_copy_greens_hat(self._plan, out)
        return out

    def model_bytes(self, pass_index=0):
        return dks_poisson_model_bytes(self._plan, pass_index)

    def close(self):
        if self._plan:
            import torch

            torch.cuda.synchronize()
            dks_poisson_plan_destroy(self._plan)
            self._plan = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


"""ctypes wrapper around the CPU oracle (oracle/poisson_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  The product package never imports this.

All arrays are float64, contiguous, [nz][ny][nx] with x fastest.
`precision` selects the build: "ld" (long double inside; the reference values) or
"d" (double inside; the timed baseline).
"""
from __future__ import annotations

import ctypes as C
import math

import numpy as np

from . import build as _build

EPS0 = 8.8541878128e-12          # F/m, CODATA 2018 (reading A1)

_libs = {}


def _lib(precision: str):
    if precision not in _libs:
        libs = _build.build()
        lib = C.CDLL(libs[precision])
        p = f"oracle_{precision}_"
        dp = C.POINTER(C.c_double)
        f = getattr(lib, p + "fft1d"); f.argtypes = [dp, dp, dp, dp, C.c_int, C.c_int]; f.restype = None
        f = getattr(lib, p + "dft1d"); f.argtypes = [dp, dp, dp, dp, C.c_int, C.c_int]; f.restype = None
        f = getattr(lib, p + "green"); f.argtypes = [C.c_double] * 3; f.restype = C.c_double
        f = getattr(lib, p + "plan_create")
        f.argtypes = [C.c_int] * 3 + [C.c_double] * 5; f.restype = C.c_void_p
        f = getattr(lib, p + "plan_destroy"); f.argtypes = [C.c_void_p]; f.restype = None
        f = getattr(lib, p + "plan_ghat_stats"); f.argtypes = [C.c_void_p, dp, dp, dp]; f.restype = None
        f = getattr(lib, p + "plan_solve"); f.argtypes = [C.c_void_p, dp, dp]; f.restype = C.c_double
        f = getattr(lib, p + "plan_ghat_octant"); f.argtypes = [C.c_void_p, dp]; f.restype = None
        f = getattr(lib, p + "solve")
        f.argtypes = [C.c_int] * 3 + [C.c_double] * 5 + [dp, dp]; f.restype = C.c_double
        f = getattr(lib, p + "direct_sum_nodes")
        f.argtypes = [C.c_int] * 3 + [C.c_double] * 4 + [dp, C.POINTER(C.c_longlong), C.c_int, dp]
        f.restype = None
        f = getattr(lib, p + "num_threads"); f.argtypes = []; f.restype = C.c_int
        f = getattr(lib, p + "cic_deposit")
        f.argtypes = [C.c_int] * 3 + [C.c_double] * 6 + [dp, dp, dp, dp, C.c_longlong, dp]; f.restype = C.c_longlong
        f = getattr(lib, p + "gradient"); f.argtypes = [C.c_int] * 3 + [C.c_double] * 3 + [dp, dp, dp, dp]; f.restype = None
        f = getattr(lib, p + "cic_gather")
        f.argtypes = [C.c_int] * 3 + [C.c_double] * 6 + [dp, dp, dp, dp, C.c_longlong, dp]; f.restype = None
        _libs[precision] = (lib, p)
    return _libs[precision]


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def default_g0(h) -> float:
    """Reading A2: G(0,0,0) := G at r0 = min(hx,hy,hz)/2."""
    return 1.0 / (4.0 * math.pi * EPS0 * 0.5 * min(h))


def green(u, v, w, precision="ld") -> float:
    lib, p = _lib(precision)
    return getattr(lib, p + "green")(u, v, w)


def fft1d(x, sign=-1, precision="ld", definition=False):
    """1-D transform of a complex line by the oracle's FFT, or by the O(L^2) definition."""
    lib, p = _lib(precision)
    x = np.asarray(x, dtype=np.complex128)
    re, im = np.ascontiguousarray(x.real), np.ascontiguousarray(x.imag)
    ore, oim = np.empty_like(re), np.empty_like(im)
    getattr(lib, p + ("dft1d" if definition else "fft1d"))(_dp(re), _dp(im), _dp(ore), _dp(oim), len(x), sign)
    return ore + 1j * oim


class Plan:
    """FT{G} precomputed for (n, h, g0); solve(rho) runs steps 1, 3-6 of the oracle."""

    def __init__(self, n, h, g0=None, precision="ld", plane_value=float("nan")):
        self._lib, self._p = _lib(precision)
        self.n, self.h = tuple(n), tuple(h)
        self.g0 = default_g0(h) if g0 is None else float(g0)
        nx, ny, nz = self.n
        self._h = getattr(self._lib, self._p + "plan_create")(nx, ny, nz, *self.h, self.g0, plane_value)
        if not self._h:
            raise MemoryError("oracle plan allocation failed")
        self.max_imag_rel = None

    def solve(self, rho):
        nx, ny, nz = self.n
        rho = np.ascontiguousarray(rho, dtype=np.float64)
        assert rho.shape == (nz, ny, nx)
        phi = np.empty_like(rho)
        self.max_imag_rel = getattr(self._lib, self._p + "plan_solve")(self._h, _dp(rho), _dp(phi))
        return phi

    def ghat_stats(self):
        a, b, c = C.c_double(), C.c_double(), C.c_double()
        getattr(self._lib, self._p + "plan_ghat_stats")(self._h, C.byref(a), C.byref(b), C.byref(c))
        return {"max_im": a.value, "max_abs": b.value, "max_even_defect": c.value}

    def ghat_octant(self):
        """Re FT{Gt} on the octant [nz+1][ny+1][nx+1] (unscaled: no hx hy hz, no 1/N)."""
        nx, ny, nz = self.n
        out = np.empty((nz + 1, ny + 1, nx + 1), dtype=np.float64)
        getattr(self._lib, self._p + "plan_ghat_octant")(self._h, _dp(out))
        return out

    def close(self):
        if self._h:
            getattr(self._lib, self._p + "plan_destroy")(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def solve(rho, n, h, g0=None, precision="ld", plane_value=float("nan")):
    """phi for one rho (steps 1-6)."""
    pl = Plan(n, h, g0, precision, plane_value)
    try:
        return pl.solve(rho)
    finally:
        pl.close()


def direct_sum_nodes(rho, n, h, nodes, g0=None, precision="ld"):
    """Eq. (2) summed directly at the given (i, j, k) nodes."""
    lib, p = _lib(precision)
    nx, ny, nz = n
    rho = np.ascontiguousarray(rho, dtype=np.float64)
    nodes = np.ascontiguousarray(nodes, dtype=np.int64)
    out = np.empty(len(nodes), dtype=np.float64)
    g0 = default_g0(h) if g0 is None else float(g0)
    getattr(lib, p + "direct_sum_nodes")(nx, ny, nz, *h, g0, _dp(rho),
                                         nodes.ctypes.data_as(C.POINTER(C.c_longlong)), len(nodes), _dp(out))
    return out


def direct_sum(rho, n, h, g0=None, precision="ld"):
    """Eq. (2) at every node (tiny meshes only)."""
    nx, ny, nz = n
    kk, jj, ii = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    nodes = np.stack([ii.ravel(), jj.ravel(), kk.ravel()], axis=1)
    return direct_sum_nodes(rho, n, h, nodes, g0, precision).reshape(nz, ny, nx)


def num_threads(precision="d") -> int:
    lib, p = _lib(precision)
    return getattr(lib, p + "num_threads")()


# ---- the steps adjacent to the solve (oracle/field_ops_oracle.c; readings F1-F4) --------------------------------------
def cic_deposit(n, h, origin, x, y, z, q, precision="ld"):
    """rho [nz][ny][nx] from particles at physical positions (x, y, z) with charges q; returns (rho, particles kept)."""
    lib, p = _lib(precision)
    nx, ny, nz = n
    x, y, z, q = (np.ascontiguousarray(a, dtype=np.float64) for a in (x, y, z, q))
    rho = np.empty((nz, ny, nx), dtype=np.float64)
    kept = getattr(lib, p + "cic_deposit")(nx, ny, nz, *h, *origin, _dp(x), _dp(y), _dp(z), _dp(q), len(x), _dp(rho))
    return rho, int(kept)


def gradient(phi, n, h, precision="ld"):
    """(Ex, Ey, Ez) = -grad(phi), second-order differences (F3)."""
    lib, p = _lib(precision)
    nx, ny, nz = n
    phi = np.ascontiguousarray(phi, dtype=np.float64)
    ex, ey, ez = (np.empty_like(phi) for _ in range(3))
    getattr(lib, p + "gradient")(nx, ny, nz, *h, _dp(phi), _dp(ex), _dp(ey), _dp(ez))
    return ex, ey, ez


def cic_gather(field, n, h, origin, x, y, z, precision="ld"):
    """Trilinear interpolation of a node field to the particles (F4); 0 for dropped particles."""
    lib, p = _lib(precision)
    nx, ny, nz = n
    field = np.ascontiguousarray(field, dtype=np.float64)
    x, y, z = (np.ascontiguousarray(a, dtype=np.float64) for a in (x, y, z))
    out = np.empty(len(x), dtype=np.float64)
    getattr(lib, p + "cic_gather")(nx, ny, nz, *h, *origin, _dp(field), _dp(x), _dp(y), _dp(z), len(x), _dp(out))
    return out

"""Pins for the CPU oracle (oracle/poisson_oracle.c) against what the paper and the mathematics fix.

Nothing here touches the CUDA path.  Pin numbers P1..P12 follow SURVEY.md section 8(c) / DESIGN.md.
The result is defined by Eq. (2); G by PAPER.md:117 with reading A1 (1/(4 pi eps0 r)).
"""
import math

import numpy as np
import pytest

EPS0 = 8.8541878128e-12
K_COULOMB = 1.0 / (4.0 * math.pi * EPS0)


def rel_l2(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


# ----------------------------------------------------------------------------- P11: the 1-D FFT
@pytest.mark.parametrize("L", [2, 4, 8, 16, 32, 64, 128, 256, 512, 1024])
@pytest.mark.parametrize("sign", [-1, +1])
def test_p11_fft_matches_dft_definition(oracle, L, sign):
    rng = np.random.default_rng(L + (sign + 1))
    x = rng.standard_normal(L) + 1j * rng.standard_normal(L)
    fast = oracle.fft1d(x, sign, "ld")
    slow = oracle.fft1d(x, sign, "ld", definition=True)
    assert np.max(np.abs(fast - slow)) <= 4e-16 * np.max(np.abs(slow))   # both rounded to double on return
    # independent library opinion (pocketfft)
    lib = np.fft.fft(x) if sign < 0 else np.fft.ifft(x) * L
    assert np.max(np.abs(fast - lib)) <= 1e-14 * np.max(np.abs(lib))


def test_p11_fft_impulse_and_shift_closed_forms(oracle):
    L = 64
    e = np.zeros(L, complex); e[0] = 1
    assert np.allclose(oracle.fft1d(e, -1), np.ones(L), atol=0, rtol=0)
    s = 5
    e = np.zeros(L, complex); e[s] = 1
    X = oracle.fft1d(e, -1)
    k = np.arange(L)
    assert np.max(np.abs(X - np.exp(-2j * np.pi * ((k * s) % L) / L))) < 1e-15     # forward sign is e^{-i theta} (A5)
    X = oracle.fft1d(e, +1)
    assert np.max(np.abs(X - np.exp(+2j * np.pi * ((k * s) % L) / L))) < 1e-15


@pytest.mark.parametrize("L", [8, 128, 1024])
def test_p11_roundtrip_and_parseval(oracle, L):
    rng = np.random.default_rng(7 * L)
    x = rng.standard_normal(L) + 1j * rng.standard_normal(L)
    X = oracle.fft1d(x, -1)
    back = oracle.fft1d(X, +1) / L
    assert np.max(np.abs(back - x)) < 1e-15 * np.max(np.abs(x)) * 4
    assert abs(np.sum(np.abs(X) ** 2) / L - np.sum(np.abs(x) ** 2)) < 1e-13 * np.sum(np.abs(x) ** 2)


# ----------------------------------------------------------------------------- Green's function constant
def test_green_constant_and_radius(oracle):
    # Coulomb potential of 1 C at 1 m: 8.9875517923e9 V (CODATA-consistent value of 1/(4 pi eps0))
    assert abs(oracle.green(1.0, 0.0, 0.0) - 8.9875517923e9) < 1e-1
    assert abs(oracle.green(3e-3, 4e-3, 0.0) - K_COULOMB / 5e-3) < 1e-15 * K_COULOMB / 5e-3 * 8
    assert abs(oracle.default_g0((1e-3, 2e-3, 5e-4)) - K_COULOMB / 2.5e-4) < 1e-15 * K_COULOMB / 2.5e-4 * 8


# ----------------------------------------------------------------------------- P1: full direct summation
@pytest.mark.parametrize("n,h", [
    ((4, 4, 4), (1e-3, 1e-3, 1e-3)),
    ((8, 8, 8), (1e-3, 1e-3, 1e-3)),
    ((8, 4, 16), (1e-3, 2e-3, 5e-4)),          # non-cubic, anisotropic
    ((16, 8, 4), (3e-4, 1e-4, 7e-4)),
])
@pytest.mark.parametrize("precision,tol", [("ld", 1e-14), ("d", 1e-13)])
def test_p1_direct_sum_tiny(oracle, workloads, n, h, precision, tol):
    rho = workloads.random_rho(n, seed=sum(n))
    phi = oracle.solve(rho, n, h, precision=precision)
    ref = oracle.direct_sum(rho, n, h, precision="ld")
    assert rel_l2(phi, ref) <= tol
    assert np.max(np.abs(phi - ref)) <= 10 * tol * np.max(np.abs(ref))


def test_p1_direct_sum_config1(oracle, workloads):
    w = workloads.config(1)
    rho = workloads.make_rho(w)
    phi = oracle.solve(rho, w.n, w.h)
    ref = oracle.direct_sum(rho, w.n, w.h)
    assert rel_l2(phi, ref) <= 1e-14


def test_p1_direct_sum_numpy_restatement(oracle, workloads):
    """Eq. (2) retyped in numpy (fp64) as a check on the C direct-sum checker itself."""
    n, h = (4, 3 + 1, 2), (1e-3, 2e-3, 3e-3)
    nx, ny, nz = n
    rho = workloads.random_rho(n, seed=5)
    g0 = oracle.default_g0(h)
    ref = np.zeros_like(rho)
    for k in range(nz):
        for j in range(ny):
            for i in range(nx):
                acc = 0.0
                for kp in range(nz):
                    for jp in range(ny):
                        for ip in range(nx):
                            if (i, j, k) == (ip, jp, kp):
                                g = g0
                            else:
                                r = math.sqrt(((i - ip) * h[0]) ** 2 + ((j - jp) * h[1]) ** 2 + ((k - kp) * h[2]) ** 2)
                                g = K_COULOMB / r
                            acc += rho[kp, jp, ip] * g
                ref[k, j, i] = h[0] * h[1] * h[2] * acc
    got = oracle.direct_sum(rho, n, h)
    assert rel_l2(got, ref) < 1e-14


# ----------------------------------------------------------------------------- P2: sampled direct summation on every config
@pytest.mark.parametrize("cfg", [1, 2, 3, 5])
def test_p2_sampled_direct_sum_configs(oracle, workloads, cfg):
    w = workloads.config(cfg)
    rho = workloads.make_rho(w)
    phi = oracle.solve(rho, w.n, w.h)
    nodes = workloads.sample_nodes(w.n, w.seed)
    ref = oracle.direct_sum_nodes(rho, w.n, w.h, nodes)
    got = phi[nodes[:, 2], nodes[:, 1], nodes[:, 0]]
    assert np.max(np.abs(got - ref) / np.abs(ref)) <= 1e-13


@pytest.mark.slow
def test_p2_sampled_direct_sum_config4(oracle, workloads):
    w = workloads.config(4)
    rho = workloads.make_rho(w)
    phi = oracle.solve(rho, w.n, w.h)
    nodes = workloads.sample_nodes(w.n, w.seed)
    ref = oracle.direct_sum_nodes(rho, w.n, w.h, nodes)
    got = phi[nodes[:, 2], nodes[:, 1], nodes[:, 0]]
    assert np.max(np.abs(got - ref) / np.abs(ref)) <= 1e-13


# ----------------------------------------------------------------------------- P3: single point charge
@pytest.mark.parametrize("n,h", [((8, 8, 8), (1e-3, 1e-3, 1e-3)), ((16, 8, 4), (2e-4, 3e-4, 5e-4))])
@pytest.mark.parametrize("where", ["corner0", "corner1", "mid"])
def test_p3_point_charge(oracle, n, h, where):
    nx, ny, nz = n
    s = {"corner0": (0, 0, 0), "corner1": (nx - 1, ny - 1, nz - 1), "mid": (nx // 2, ny // 3, nz // 2)}[where]
    q = 2.5e-9
    rho = np.zeros((nz, ny, nx))
    rho[s[2], s[1], s[0]] = q / (h[0] * h[1] * h[2])
    phi = oracle.solve(rho, n, h)
    g0 = oracle.default_g0(h)
    kk, jj, ii = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    r = np.sqrt(((ii - s[0]) * h[0]) ** 2 + ((jj - s[1]) * h[1]) ** 2 + ((kk - s[2]) * h[2]) ** 2)
    with np.errstate(divide="ignore"):
        expect = q * K_COULOMB / r
    expect[s[2], s[1], s[0]] = q * g0
    assert np.max(np.abs(phi - expect) / expect) <= 1e-13
    # no wrap-around: far corner sees the true distance, not a periodic image
    far = (nx - 1 - s[0] if where != "mid" else 0, ny - 1 - s[1] if where != "mid" else 0,
           nz - 1 - s[2] if where != "mid" else 0)
    d = math.sqrt(((far[0] - s[0]) * h[0]) ** 2 + ((far[1] - s[1]) * h[1]) ** 2 + ((far[2] - s[2]) * h[2]) ** 2)
    assert abs(phi[far[2], far[1], far[0]] - q * K_COULOMB / d) <= 1e-13 * q * K_COULOMB / d


def test_p3_unpadded_periodic_convolution_is_wrong(oracle):
    """The pin above has teeth: a circular convolution WITHOUT doubling gives a different far-corner value."""
    n, h = (8, 8, 8), (1e-3,) * 3
    g0 = oracle.default_g0(h)
    idx = np.minimum(np.arange(8), 8 - np.arange(8)) * h[0]
    r = np.sqrt(idx[:, None, None] ** 2 + idx[None, :, None] ** 2 + idx[None, None, :] ** 2)
    with np.errstate(divide="ignore"):
        g = K_COULOMB / r
    g[0, 0, 0] = g0
    rho = np.zeros((8, 8, 8)); rho[0, 0, 0] = 1.0 / h[0] ** 3
    wrong = np.fft.ifftn(np.fft.fftn(rho) * np.fft.fftn(g)).real * h[0] ** 3
    right = oracle.solve(rho, n, h)
    assert abs(wrong[7, 7, 7] - right[7, 7, 7]) > 0.5 * right[7, 7, 7]


# ----------------------------------------------------------------------------- P4: linearity
def test_p4_linearity(oracle, workloads):
    n, h = (16, 8, 8), (1e-3, 2e-3, 1e-3)
    r1, r2 = workloads.random_rho(n, 11), workloads.random_rho(n, 12)
    a, b = 0.75, -2.5
    pl = oracle.Plan(n, h)
    lhs = pl.solve(a * r1 + b * r2)
    rhs = a * pl.solve(r1) + b * pl.solve(r2)
    pl.close()
    assert rel_l2(lhs, rhs) <= 1e-13


# ----------------------------------------------------------------------------- P5: mirror + axis permutation
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_p5_mirror(oracle, workloads, axis):
    n, h = (8, 16, 4), (1e-3, 5e-4, 2e-3)
    rho = workloads.random_rho(n, 21)
    phi = oracle.solve(rho, n, h)
    phi_f = oracle.solve(np.ascontiguousarray(np.flip(rho, axis=axis)), n, h)
    assert rel_l2(np.flip(phi_f, axis=axis), phi) <= 1e-13


@pytest.mark.parametrize("perm", [(1, 0, 2), (2, 1, 0), (0, 2, 1), (1, 2, 0)])
def test_p5_axis_permutation(oracle, workloads, perm):
    n, h = (8, 16, 4), (1e-3, 5e-4, 2e-3)          # (x, y, z)
    rho = workloads.random_rho(n, 22)               # array axes (z, y, x)
    phi = oracle.solve(rho, n, h)
    # permute array axes; array axis a corresponds to spatial axis 2 - a
    rho_p = np.ascontiguousarray(np.transpose(rho, perm))
    spatial_of_new_axis = [2 - perm[a] for a in range(3)]          # for new array axes (z', y', x')
    n_p = tuple(n[spatial_of_new_axis[2 - s]] for s in range(3))
    h_p = tuple(h[spatial_of_new_axis[2 - s]] for s in range(3))
    g0 = oracle.default_g0(h)
    phi_p = oracle.solve(rho_p, n_p, h_p, g0=g0)
    assert rel_l2(phi_p, np.transpose(phi, perm)) <= 1e-13


# ----------------------------------------------------------------------------- P6: translation
def test_p6_translation(oracle, workloads):
    n, h = (16, 16, 16), (1e-3, 1e-3, 2e-3)
    rng = np.random.default_rng(31)
    rho = np.zeros((16, 16, 16))
    rho[2:6, 3:7, 1:5] = rng.standard_normal((4, 4, 4))
    s = (5, 4, 7)                                   # shift in (x, y, z) cells
    rho_s = np.zeros_like(rho)
    rho_s[2 + s[2]:6 + s[2], 3 + s[1]:7 + s[1], 1 + s[0]:5 + s[0]] = rho[2:6, 3:7, 1:5]
    phi, phi_s = oracle.solve(rho, n, h), oracle.solve(rho_s, n, h)
    a = phi[:16 - s[2], :16 - s[1], :16 - s[0]]
    b = phi_s[s[2]:, s[1]:, s[0]:]
    assert rel_l2(b, a) <= 1e-13


# ----------------------------------------------------------------------------- P7: planes i=nx, j=ny, k=nz are irrelevant
def test_p7_nyquist_planes_do_not_matter(oracle, workloads):
    n, h = (8, 8, 16), (1e-3, 1e-3, 5e-4)
    rho = workloads.random_rho(n, 41)
    a = oracle.solve(rho, n, h)
    b = oracle.solve(rho, n, h, plane_value=1.2345e12)
    assert rel_l2(b, a) <= 1e-12


# ----------------------------------------------------------------------------- P8: Hermitian bookkeeping
def test_p8_imag_zero_and_ghat_real_even(oracle, workloads):
    n, h = (8, 16, 8), (1e-3, 5e-4, 1e-3)
    pl = oracle.Plan(n, h)
    pl.solve(workloads.random_rho(n, 51))
    assert pl.max_imag_rel <= 1e-15
    st = pl.ghat_stats()
    pl.close()
    assert st["max_im"] <= 1e-13 * st["max_abs"]
    assert st["max_even_defect"] <= 1e-13 * st["max_abs"]


# ----------------------------------------------------------------------------- P13: the Green's-octant accessor
def mirrored_green_numpy(n, h, g0):
    """Gt on the doubled grid, [2nz][2ny][2nx]: G at the mirrored index min(i, 2n - i), typed here in numpy."""
    nx, ny, nz = n
    ix = np.minimum(np.arange(2 * nx), 2 * nx - np.arange(2 * nx)) * h[0]
    iy = np.minimum(np.arange(2 * ny), 2 * ny - np.arange(2 * ny)) * h[1]
    iz = np.minimum(np.arange(2 * nz), 2 * nz - np.arange(2 * nz)) * h[2]
    r = np.sqrt(iz[:, None, None] ** 2 + iy[None, :, None] ** 2 + ix[None, None, :] ** 2)
    with np.errstate(divide="ignore"):
        g = K_COULOMB / r
    g[0, 0, 0] = g0
    return g


@pytest.mark.parametrize("n,h", [((4, 8, 2), (1e-3, 2e-3, 5e-4)), ((8, 2, 4), (3e-4, 1e-3, 2e-3)), ((2, 4, 16), (1e-3, 7e-4, 4e-4))])
@pytest.mark.parametrize("precision", ["ld", "d"])
def test_p13_ghat_octant_accessor(oracle, n, h, precision):
    """Plan.ghat_octant() (oracle_*_plan_ghat_octant, the reference of the GPU test of step a0) is FT{Gt}[k, j, i] for k <= nz,
    j <= ny, i <= nx, shape (nz+1, ny+1, nx+1).  Non-cubic, anisotropic
    meshes: a swapped extent, stride or axis cannot cancel.  Two opinions: numpy.fft.fftn of Gt built in numpy, and the
    oracle's O(L^2) definition dft1d applied axis by axis to the same Gt."""
    nx, ny, nz = n
    g0 = 0.37 * oracle.default_g0(h)                      # an override, so that the g0 argument is covered too
    pl = oracle.Plan(n, h, g0=g0, precision=precision)
    try:
        oct_ = pl.ghat_octant()
    finally:
        pl.close()
    assert oct_.shape == (nz + 1, ny + 1, nx + 1)
    gt = mirrored_green_numpy(n, h, g0)
    full = np.fft.fftn(gt)                                # (a) library transform, third opinion
    scale = np.max(np.abs(full))
    assert np.max(np.abs(full.imag)) <= 1e-13 * scale     # real and even: the octant carries everything
    assert np.max(np.abs(oct_ - full.real[:nz + 1, :ny + 1, :nx + 1])) <= 1e-13 * scale
    # (b) the definition, axis by axis (x, then y, then z), through the oracle's own O(L^2) dft1d
    t = gt.astype(np.complex128)
    for axis in (2, 1, 0):
        t = np.apply_along_axis(lambda line: oracle.fft1d(line, sign=-1, precision=precision, definition=True), axis, t)
    assert np.max(np.abs(t.imag)) <= 1e-13 * scale
    assert np.max(np.abs(oct_ - t.real[:nz + 1, :ny + 1, :nx + 1])) <= 1e-13 * scale
    # negative controls: the entries the accessor could pick by mistake are really different
    for wrong in (full.real[1:nz + 2, :ny + 1, :nx + 1], full.real[:nz + 1, 1:ny + 2, :nx + 1], full.real[:nz + 1, :ny + 1, 1:nx + 2]):
        assert np.max(np.abs(oct_ - wrong)) > 1e-3 * scale
    wrong_pitch = full.real.ravel()[:oct_.size].reshape(oct_.shape)       # octant read with the doubled grid's own pitch
    assert np.max(np.abs(oct_ - wrong_pitch)) > 1e-3 * scale
    # and the even symmetry that lets the octant stand for the whole transform
    k, j, i = nz // 2 or 1, ny // 2 or 1, nx // 2 or 1
    assert abs(full.real[2 * nz - k, 2 * ny - j, 2 * nx - i] - oct_[k, j, i]) <= 1e-13 * scale


# ----------------------------------------------------------------------------- P9: positivity
def test_p9_positivity(oracle, workloads):
    n, h = (16, 16, 8), (1e-3, 1e-3, 1e-3)
    rho = workloads.random_rho(n, 61, signed=False)
    assert np.all(oracle.solve(rho, n, h) > 0)
    assert np.all(oracle.solve(-rho, n, h) < 0)


# ----------------------------------------------------------------------------- P10: continuum closed form
def test_p10_uniform_sphere(oracle):
    nmesh, hh = 64, 1e-3
    n, h = (nmesh,) * 3, (hh,) * 3
    c = (nmesh - 1) / 2.0
    R, Q = 20.0 * hh, 1e-9
    ax = (np.arange(nmesh) - c) * hh
    zz, yy, xx = np.meshgrid(ax, ax, ax, indexing="ij")
    r = np.sqrt(xx ** 2 + yy ** 2 + zz ** 2)
    rho = np.where(r <= R, Q / (4.0 / 3.0 * math.pi * R ** 3), 0.0)
    Qmesh = rho.sum() * hh ** 3                      # charge actually on the mesh
    phi = oracle.solve(rho, n, h, precision="d")
    with np.errstate(divide="ignore", invalid="ignore"):
        outside = Qmesh * K_COULOMB / r
    inside = Qmesh * K_COULOMB * (3 * R ** 2 - r ** 2) / (2 * R ** 3)
    expect = np.where(r <= R, inside, outside)
    far = r > 1.25 * R
    assert np.max(np.abs(phi[far] - expect[far]) / expect[far]) < 1e-2
    core = r < 0.75 * R
    assert np.max(np.abs(phi[core] - expect[core]) / expect[core]) < 1e-2


def test_p10_far_corner_monopole(oracle, workloads):
    w = workloads.config(2)
    rho = workloads.make_rho(w)
    phi = oracle.solve(rho, w.n, w.h, precision="d")
    Q = rho.sum() * w.h[0] * w.h[1] * w.h[2]
    c = (64 - 1) / 2.0
    d = math.sqrt(3) * c * w.h[0]
    assert abs(phi[0, 0, 0] - Q * K_COULOMB / d) < 2e-2 * Q * K_COULOMB / d


# ----------------------------------------------------------------------------- P12: library special case (third opinion)
def numpy_hockney(rho, n, h, g0):
    nx, ny, nz = n
    ix = np.minimum(np.arange(2 * nx), 2 * nx - np.arange(2 * nx)) * h[0]
    iy = np.minimum(np.arange(2 * ny), 2 * ny - np.arange(2 * ny)) * h[1]
    iz = np.minimum(np.arange(2 * nz), 2 * nz - np.arange(2 * nz)) * h[2]
    r = np.sqrt(iz[:, None, None] ** 2 + iy[None, :, None] ** 2 + ix[None, None, :] ** 2)
    with np.errstate(divide="ignore"):
        g = K_COULOMB / r
    g[0, 0, 0] = g0
    s = (2 * nz, 2 * ny, 2 * nx)
    ax = (0, 1, 2)
    out = np.fft.irfftn(np.fft.rfftn(rho, s, ax) * np.fft.rfftn(g, s, ax), s, ax)
    return out[:nz, :ny, :nx] * (h[0] * h[1] * h[2])


@pytest.mark.parametrize("cfg", [1, 2, 3, 5])
def test_p12_numpy_fft_third_opinion(oracle, workloads, cfg):
    w = workloads.config(cfg)
    rho = workloads.make_rho(w)
    phi = oracle.solve(rho, w.n, w.h)
    lib = numpy_hockney(rho, w.n, w.h, oracle.default_g0(w.h))
    assert rel_l2(lib, phi) <= 1e-13


def test_double_build_tracks_long_double_build(oracle, workloads):
    w = workloads.config(2)
    rho = workloads.make_rho(w)
    a = oracle.solve(rho, w.n, w.h, precision="ld")
    b = oracle.solve(rho, w.n, w.h, precision="d")
    assert rel_l2(b, a) <= 1e-14

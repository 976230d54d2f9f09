"""Pins of the oracle's deposit / gradient / gather (oracle/field_ops_oracle.c, readings F1-F4 of DESIGN.md).

The paper gives no formula for these steps (PAPER.md:86 only names IPPL's "interpolation operators"), so each function is
pinned by what the mathematics fixes: conservation laws, closed forms on polynomial fields, special positions, the adjoint
relation between deposit and gather, convergence order on the analytic point-charge field, and an independent
implementation (the numpy bincount deposit of the input generator).  No GPU.
"""
import numpy as np
import pytest

H = (1e-3, 2e-3, 5e-4)
N = (8, 6, 10)
ORIGIN = (-3.5e-3, 0.25e-3, 1.0)


def node_xyz(n, h, origin):
    nx, ny, nz = n
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    return origin[0] + i * h[0], origin[1] + j * h[1], origin[2] + k * h[2]


def random_particles(n, h, origin, count, seed, margin=0.0):
    rng = np.random.default_rng(seed)
    u = rng.uniform(margin, np.array(n) - 1 - margin, size=(count, 3))
    q = rng.uniform(-1.0, 2.0, size=count) * 1e-12
    return origin[0] + u[:, 0] * h[0], origin[1] + u[:, 1] * h[1], origin[2] + u[:, 2] * h[2], q, u


# ---- deposit ------------------------------------------------------------------------------------------------------------
def test_deposit_conserves_charge_and_dipole(oracle):
    x, y, z, q, u = random_particles(N, H, ORIGIN, 500, 1)
    rho, kept = oracle.cic_deposit(N, H, ORIGIN, x, y, z, q)
    assert kept == 500
    vol = H[0] * H[1] * H[2]
    assert abs(rho.sum() * vol - q.sum()) <= 1e-15 * np.abs(q).sum()
    # first moment: sum_nodes rho vol X_node = sum_p q X_p (trilinear weights reproduce linear functions); a swapped
    # weight (f <-> 1 - f) or a transposed axis breaks this
    X, Y, Z = node_xyz(N, H, ORIGIN)
    for nodes, part in ((X, x), (Y, y), (Z, z)):
        assert abs((rho * vol * nodes).sum() - (q * part).sum()) <= 1e-13 * (np.abs(q) * np.abs(part)).sum()


def test_deposit_special_positions(oracle):
    vol = H[0] * H[1] * H[2]
    # on a node: everything on that node
    i, j, k = 3, 2, 7
    rho, kept = oracle.cic_deposit(N, H, (0, 0, 0), [i * H[0]], [j * H[1]], [k * H[2]], [2.5])
    assert kept == 1 and rho[k, j, i] == pytest.approx(2.5 / vol, rel=1e-15) and np.count_nonzero(rho) == 1
    # at a cell centre: one eighth on each of the 8 corners
    rho, _ = oracle.cic_deposit(N, H, (0, 0, 0), [(i + 0.5) * H[0]], [(j + 0.5) * H[1]], [(k + 0.5) * H[2]], [8.0])
    assert np.count_nonzero(rho) == 8
    assert np.allclose(rho[k:k + 2, j:j + 2, i:i + 2], 1.0 / vol, rtol=1e-12)
    # three quarters along x only: 1/4 on i, 3/4 on i+1, nothing elsewhere
    rho, _ = oracle.cic_deposit(N, H, (0, 0, 0), [(i + 0.75) * H[0]], [j * H[1]], [k * H[2]], [4.0])
    assert rho[k, j, i] == pytest.approx(1.0 / vol, rel=1e-12) and rho[k, j, i + 1] == pytest.approx(3.0 / vol, rel=1e-12)
    assert np.count_nonzero(rho) == 2


def test_deposit_drop_rule(oracle):
    nx, ny, nz = N
    inside = ((nx - 1) * H[0] * (1 - 1e-12), 0.0, 0.0)
    for pos, kept_expected in [((-1e-9, 1e-3, 1e-3), 0), (((nx - 1) * H[0], 1e-3, 1e-3), 0),
                               ((1e-3, (ny - 1) * H[1], 1e-3), 0), ((1e-3, 1e-3, (nz - 1) * H[2]), 0),
                               ((float("nan"), 0.0, 0.0), 0), (inside, 1), ((0.0, 0.0, 0.0), 1)]:
        rho, kept = oracle.cic_deposit(N, H, (0, 0, 0), [pos[0]], [pos[1]], [pos[2]], [1.0])
        assert kept == kept_expected
        assert (np.count_nonzero(rho) > 0) == bool(kept_expected)


def test_deposit_superposition_and_translation(oracle):
    x, y, z, q, _ = random_particles(N, H, ORIGIN, 200, 2, margin=1.0)
    ra, _ = oracle.cic_deposit(N, H, ORIGIN, x[:100], y[:100], z[:100], q[:100])
    rb, _ = oracle.cic_deposit(N, H, ORIGIN, x[100:], y[100:], z[100:], q[100:])
    rab, _ = oracle.cic_deposit(N, H, ORIGIN, x, y, z, 3.0 * q)
    assert np.max(np.abs(rab - 3.0 * (ra + rb))) <= 1e-15 * np.max(np.abs(rab))
    # moving the origin by one cell (-hx, 0, +hz) shifts rho by one node
    shifted, _ = oracle.cic_deposit(N, H, (ORIGIN[0] - H[0], ORIGIN[1], ORIGIN[2] + H[2]), x, y, z, 3.0 * q)
    # new index u' = u + 1 along x, w' = w - 1 along z
    assert np.max(np.abs(shifted[:-1, :, 1:] - rab[1:, :, :-1])) <= 1e-9 * np.max(np.abs(rab))


def test_deposit_matches_independent_numpy_implementation(oracle, workloads):
    w = workloads.config(1)
    x, y, z, q, origin = workloads.particles(w)
    rho, kept = oracle.cic_deposit(w.n, w.h, origin, x, y, z, q)
    ref = workloads.make_rho(w)                      # numpy bincount deposit on node-unit positions
    assert 0.9 * w.n_particles < kept < w.n_particles           # config 1 loses 3-4 % of its particles
    # positions went through origin + u h and back: relative error ~1e-13 of a cell, times the weight slope
    assert np.max(np.abs(rho - ref)) <= 1e-10 * np.max(np.abs(ref))
    assert abs(rho.sum() - ref.sum()) <= 1e-11 * ref.sum()


# ---- gradient -----------------------------------------------------------------------------------------------------------
def test_gradient_exact_on_linear_and_quadratic_fields(oracle):
    X, Y, Z = node_xyz(N, H, ORIGIN)
    a, b, c = 3.0, -2.0, 0.5
    ex, ey, ez = oracle.gradient(a * X + b * Y + c * Z + 7.0, N, H)
    for e, v in ((ex, -a), (ey, -b), (ez, -c)):
        assert np.max(np.abs(e - v)) <= 1e-9 * abs(v)            # differences of values ~1 divided by h ~1e-3
    phi = 2.0 * X * X - 1.5 * Y * Y + 0.25 * Z * Z + X * Y - 3.0 * Y * Z
    ex, ey, ez = oracle.gradient(phi, N, H)
    scale = np.max(np.abs(phi)) / min(H)
    assert np.max(np.abs(ex + (4.0 * X + Y))) <= 1e-13 * scale    # second-order stencils are exact on quadratics,
    assert np.max(np.abs(ey + (-3.0 * Y + X - 3.0 * Z))) <= 1e-13 * scale   # including the one-sided ones at the ends
    assert np.max(np.abs(ez + (0.5 * Z - 3.0 * Y))) <= 1e-13 * scale


def test_gradient_second_order_on_point_charge_field(oracle):
    # phi = q G(r) around a charge outside the mesh: E = q/(4 pi eps0) r_vec / r^3; error ratio ~4 when h halves
    q, src = 1e-9, np.array([-0.02, -0.015, -0.01])
    errs = []
    for m in (1, 2):
        n = (8 * m + 1, 8 * m + 1, 8 * m + 1)
        h = (2e-3 / m,) * 3
        X, Y, Z = node_xyz(n, h, (0.0, 0.0, 0.0))
        dx, dy, dz = X - src[0], Y - src[1], Z - src[2]
        r = np.sqrt(dx * dx + dy * dy + dz * dz)
        k = q / (4.0 * np.pi * oracle.EPS0)
        ex, ey, ez = oracle.gradient(k / r, n, h)
        assert np.all(ex > 0) and np.all(ey > 0) and np.all(ez > 0)      # E points away from the positive charge
        err = max(np.max(np.abs(ex - k * dx / r ** 3)), np.max(np.abs(ey - k * dy / r ** 3)), np.max(np.abs(ez - k * dz / r ** 3)))
        errs.append(err / np.max(k / r ** 2))
    assert errs[0] < 2e-2 and 3.0 < errs[0] / errs[1] < 5.5


def test_gradient_flip_antisymmetry(oracle):
    rng = np.random.default_rng(3)
    phi = rng.standard_normal((N[2], N[1], N[0]))
    ex, ey, ez = oracle.gradient(phi, N, H)
    fx, fy, fz = oracle.gradient(phi[:, :, ::-1].copy(), N, H)
    assert np.array_equal(fx[:, :, ::-1], -ex) and np.array_equal(fy[:, :, ::-1], ey) and np.array_equal(fz[:, :, ::-1], ez)


# ---- gather -------------------------------------------------------------------------------------------------------------
def test_gather_exact_on_trilinear_fields_and_zero_outside(oracle):
    x, y, z, q, u = random_particles(N, H, ORIGIN, 300, 4)
    X, Y, Z = node_xyz(N, H, ORIGIN)
    assert np.allclose(oracle.cic_gather(np.full_like(X, 4.25), N, H, ORIGIN, x, y, z), 4.25, rtol=1e-15)
    f = 2.0 + 3.0 * X - Y + 0.5 * Z + 10.0 * X * Y * Z            # trilinear: reproduced exactly inside every cell
    got = oracle.cic_gather(f, N, H, ORIGIN, x, y, z)
    ref = 2.0 + 3.0 * x - y + 0.5 * z + 10.0 * x * y * z
    assert np.max(np.abs(got - ref)) <= 1e-12 * np.max(np.abs(ref))
    out = oracle.cic_gather(f, N, H, ORIGIN, [ORIGIN[0] - 1e-6], [ORIGIN[1]], [ORIGIN[2]])
    assert out[0] == 0.0


def test_deposit_and_gather_are_adjoint(oracle):
    x, y, z, q, _ = random_particles(N, H, ORIGIN, 400, 5)
    rng = np.random.default_rng(6)
    f = rng.standard_normal((N[2], N[1], N[0]))
    rho, _ = oracle.cic_deposit(N, H, ORIGIN, x, y, z, q)
    lhs = (rho * f).sum() * H[0] * H[1] * H[2]
    rhs = (q * oracle.cic_gather(f, N, H, ORIGIN, x, y, z)).sum()
    assert abs(lhs - rhs) <= 1e-13 * (np.abs(q).sum() * np.max(np.abs(f)))

"""GPU parity of the steps adjacent to the solve (dks_deposit_cic, dks_gradient, dks_gather_field) against
oracle/field_ops_oracle.c, through the C ABI.

Tolerances (readings F1-F4):
  deposit  the GPU sums with fp64 atomics in arbitrary order, the oracle sequentially in long double: a node that
           collects m terms differs by <= m eps of its absolute sum; stated bound 1e-12 * max|rho| (m <~ 1e3).
  gradient differences of neighbouring values scaled by 1/(2h): both sides form the same differences, the oracle in
           long double; bound 1e-14 * max|phi| / min(h).
  gather   8-term weighted sums: 1e-14 * max|field|.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def dks():
    from paper_1509_07685_b200 import dks as D
    return D


def dev(torch, *arrays):
    return [torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda() for a in arrays]


def random_particles(n, h, origin, count, seed, spill=1.5):
    """Uniform over a box `spill` cells larger than the mesh on every side: some particles are dropped."""
    rng = np.random.default_rng(seed)
    u = rng.uniform(-spill, np.array(n) - 1 + spill, size=(count, 3))
    q = rng.uniform(-1.0, 2.0, size=count) * 1e-12
    return origin[0] + u[:, 0] * h[0], origin[1] + u[:, 1] * h[1], origin[2] + u[:, 2] * h[2], q


@pytest.mark.parametrize("ci", [1, 2])
def test_deposit_config_particles(torch_cuda, dks, oracle, workloads, ci):
    torch = torch_cuda
    w = workloads.config(ci)
    x, y, z, q, origin = workloads.particles(w)
    ref, kept = oracle.cic_deposit(w.n, w.h, origin, x, y, z, q)
    plan = dks.PoissonPlan(w.n, w.h)
    try:
        got = plan.deposit(*dev(torch, x, y, z, q), origin).cpu().numpy()
    finally:
        plan.close()
    assert np.max(np.abs(got - ref)) <= 1e-12 * np.max(np.abs(ref))
    assert abs(got.sum() - ref.sum()) <= 1e-12 * np.abs(ref).sum()


@pytest.mark.parametrize("n,h,count", [((8, 8, 8), (1e-3, 1e-3, 1e-3), 1000), ((16, 8, 32), (1e-3, 2e-3, 5e-4), 20000),
                                        ((64, 32, 16), (2e-4, 3e-4, 1e-4), 200001), ((8, 1024, 8), (1e-3, 2e-5, 1e-3), 50000)])
def test_deposit_random_with_drops(torch_cuda, dks, oracle, n, h, count):
    torch = torch_cuda
    origin = (-1e-3, 2e-3, 0.5)
    x, y, z, q = random_particles(n, h, origin, count, seed=count)
    ref, kept = oracle.cic_deposit(n, h, origin, x, y, z, q)
    assert 0 < kept < count                                  # the drop rule is exercised
    plan = dks.PoissonPlan(n, h)
    try:
        got = plan.deposit(*dev(torch, x, y, z, q), origin).cpu().numpy()
    finally:
        plan.close()
    assert np.max(np.abs(got - ref)) <= 1e-12 * np.max(np.abs(ref))


def test_deposit_degenerate(torch_cuda, dks):
    torch = torch_cuda
    n, h = (8, 16, 8), (1e-3, 1e-3, 1e-3)
    plan = dks.PoissonPlan(n, h)
    try:
        rho = torch.full((8, 16, 8), 7.0, dtype=torch.float64, device="cuda")
        empty = torch.empty(0, dtype=torch.float64, device="cuda")
        dks.dks_deposit_cic(plan.handle, empty, empty, empty, empty, 0, (0, 0, 0), rho, None)     # no particles: rho = 0
        assert float(rho.abs().max()) == 0.0
        far = torch.full((5,), 1.0, dtype=torch.float64, device="cuda")                              # all outside the mesh
        plan.deposit(far, far, far, far, (0.0, 0.0, 0.0), rho)
        assert float(rho.abs().max()) == 0.0
        with pytest.raises(dks.DksError):
            dks.dks_deposit_cic(plan.handle, far, far, far, far, -1, (0, 0, 0), rho, None)
        with pytest.raises(dks.DksError):
            dks.dks_gradient(plan.handle, rho, rho, rho, rho, None)                                  # outputs alias phi
        with pytest.raises(dks.DksError):
            dks.dks_field_at_particles(plan.handle, rho, far, far, far, -1, (0, 0, 0), far, far, far, None)
        out = [torch.full((5,), 3.0, dtype=torch.float64, device="cuda") for _ in range(3)]
        dks.dks_field_at_particles(plan.handle, rho, far, far, far, 5, (0.0, 0.0, 0.0), *out, None)  # all dropped: field 0
        assert all(float(o.abs().max()) == 0.0 for o in out)
        bare = dks.dks_poisson_plan_create(8, 16, 8, 1e-3, 1e-3, 1e-3)                                # no workspace yet
        try:
            with pytest.raises(dks.DksError) as e:
                dks.dks_field_at_particles(bare, rho, far, far, far, 5, (0, 0, 0), *out, None)
            assert e.value.status == dks.DKS_ERR_NOT_SETUP
        finally:
            dks.dks_poisson_plan_destroy(bare)
    finally:
        plan.close()


@pytest.mark.parametrize("n,h", [((8, 8, 8), (1e-3, 1e-3, 1e-3)), ((16, 8, 32), (1e-3, 2e-3, 5e-4)),
                                 ((256, 16, 8), (1e-4, 1e-3, 1e-3)), ((64, 128, 32), (2e-4, 3e-4, 1e-4))])
def test_gradient_and_gather(torch_cuda, dks, oracle, workloads, n, h):
    torch = torch_cuda
    phi = workloads.random_rho(n, seed=sum(n) + 1)
    rex, rey, rez = oracle.gradient(phi, n, h)
    origin = (0.25e-3, -1e-3, 3.0)
    x, y, z, _ = random_particles(n, h, origin, 30000, seed=n[0])
    plan = dks.PoissonPlan(n, h)
    try:
        d_phi, dx, dy, dz = dev(torch, phi, x, y, z)
        ex, ey, ez = plan.gradient(d_phi)
        bound = 1e-14 * np.max(np.abs(phi)) / min(h)
        for got, ref in ((ex, rex), (ey, rey), (ez, rez)):
            assert np.max(np.abs(got.cpu().numpy() - ref)) <= bound
        epx, epy, epz = plan.gather(ex, ey, ez, dx, dy, dz, origin)
        fused = plan.field_at_particles(d_phi, dx, dy, dz, origin)         # the same two steps in one call, interleaved scratch
        for got, got_fused, field in ((epx, fused[0], rex), (epy, fused[1], rey), (epz, fused[2], rez)):
            ref = oracle.cic_gather(field, n, h, origin, x, y, z)
            for g in (got, got_fused):
                assert np.max(np.abs(g.cpu().numpy() - ref)) <= 1e-14 * np.max(np.abs(field)) + bound
                assert np.count_nonzero(ref == 0.0) > 0 and np.array_equal(g.cpu().numpy() == 0.0, ref == 0.0)   # dropped particles
    finally:
        plan.close()


def test_space_charge_step_on_device_matches_oracle_chain(torch_cuda, dks, oracle, workloads):
    # particles -> rho -> phi -> E -> E at the particles, everything on the device, against the same chain in the oracle
    torch = torch_cuda
    w = workloads.config(2)
    x, y, z, q, origin = workloads.particles(w, count=200000)
    rho_ref, _ = oracle.cic_deposit(w.n, w.h, origin, x, y, z, q)
    phi_ref = oracle.solve(rho_ref, w.n, w.h, precision="ld")
    e_ref = oracle.gradient(phi_ref, w.n, w.h)
    plan = dks.PoissonPlan(w.n, w.h)
    try:
        dx, dy, dz, dq = dev(torch, x, y, z, q)
        rho = plan.deposit(dx, dy, dz, dq, origin)
        phi = plan.solve(rho)
        ep = plan.field_at_particles(phi, dx, dy, dz, origin)
        got_phi = phi.cpu().numpy()
        assert np.linalg.norm((got_phi - phi_ref).ravel()) <= 1e-12 * np.linalg.norm(phi_ref.ravel())
        emax = max(np.max(np.abs(c)) for c in e_ref)
        for got, field in zip(ep, e_ref):
            ref = oracle.cic_gather(field, w.n, w.h, origin, x, y, z)
            # E is a difference of neighbouring phi values: phi's 1e-12 relative error is amplified by |phi| / (|E| h)
            assert np.max(np.abs(got.cpu().numpy() - ref)) <= 1e-9 * emax
    finally:
        plan.close()

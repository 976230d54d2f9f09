"""The sharded solve (dks_poisson_set_shard / set_peers / solve_shard) with all ranks emulated on ONE GPU:
g plans whose peer tables point at each other's buffers, phases issued rank after rank.  Every index computation of the
multi-GPU path (y slabs, kz slabs, peer stores of P1 and P4) runs; only the NVLink transport is absent.  Checked against
the oracle and, bit for bit, against the unsharded solve (same kernels, same arithmetic per line)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

REL_L2_TOL, MAX_ABS_TOL = 1e-12, 1e-11


@pytest.mark.parametrize("n,g", [((16, 16, 16), 2), ((16, 32, 64), 4), ((64, 16, 16), 8), ((32, 32, 32), 2), ((64, 64, 64), 4), ((32, 64, 128), 8), ((256, 32, 64), 2),
                                 ((128, 256, 32), 8), ((64, 32, 256), 4)])
def test_emulated_sharded_solve(oracle, workloads, n, g):
    import torch
    from paper_1509_07685_b200 import dks, sharded
    h = (2e-4, 3e-4, 1e-4)
    rho = workloads.random_rho(n, seed=g + n[0])
    ref = oracle.solve(rho, n, h, precision="d" if n[0] * n[1] * n[2] > 2 ** 20 else "ld")
    d_rho = torch.from_numpy(rho).cuda()
    s = sharded.EmulatedShardedSolver(n, h, g)
    try:
        got = s.solve(d_rho)
        torch.cuda.synchronize()
        again = s.solve(d_rho)                                # buffers are reused: a second solve must not see stale rows
        torch.cuda.synchronize()
    finally:
        s.close()
    plan = dks.PoissonPlan(n, h)
    try:
        single = plan.solve(d_rho)
        torch.cuda.synchronize()
    finally:
        plan.close()
    got_np = got.cpu().numpy()
    assert np.linalg.norm((got_np - ref).ravel()) <= REL_L2_TOL * np.linalg.norm(ref.ravel())
    assert np.max(np.abs(got_np - ref)) <= MAX_ABS_TOL * np.max(np.abs(ref))
    assert torch.equal(got, again)
    assert torch.equal(got, single)


def test_shard_refusals():
    import torch
    from paper_1509_07685_b200 import dks
    h_ = dks.dks_poisson_plan_create(64, 64, 64, 1e-3, 1e-3, 1e-3)
    try:
        for bad in [(0, 3), (2, 2), (-1, 2), (0, 16)]:
            with pytest.raises(dks.DksError):
                dks.dks_poisson_set_shard(h_, *bad)
        with pytest.raises(dks.DksError) as e:                  # not sharded yet
            dks.dks_poisson_solve_shard(h_, 1, 256, 256, None)
        assert e.value.status == dks.DKS_ERR_NOT_SETUP
        dks.dks_poisson_set_shard(h_, 1, 2)
        d = torch.zeros(64 * 64 * 64, dtype=torch.float64, device="cuda")
        with pytest.raises(dks.DksError):                       # a sharded plan refuses the plain solve
            dks.dks_greens_setup(h_)
            dks.dks_poisson_solve(h_, d, d, None)
        with pytest.raises(dks.DksError):                       # peers not set
            dks.dks_poisson_solve_shard(h_, 1, d, d, None)
        with pytest.raises(dks.DksError) as e:                  # the host path does not exist on a sharded plan
            dks.dks_poisson_solve_host(h_, d.cpu().numpy(), d.cpu().numpy(), None)
        assert "no host path" in str(e.value)
    finally:
        torch.cuda.synchronize()
        dks.dks_poisson_plan_destroy(h_)
    g_ = dks.dks_poisson_plan_create(8, 64, 64, 1e-3, 1e-3, 1e-3)      # nx = 8 has no register-resident x pass
    try:
        with pytest.raises(dks.DksError):
            dks.dks_poisson_set_shard(g_, 0, 2)
    finally:
        dks.dks_poisson_plan_destroy(g_)

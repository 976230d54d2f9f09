"""Out-of-bounds and uninitialised-read probe for every kernel variant (compute-sanitizer is closed on this pool, see
profiles/r2_sanitizers.md): rho, phi and the workspace sit between guard bands filled with a sentinel, the workspace
itself is pre-filled with NaN.  After setup + solves (single, in place, batched, slabbed, host path, sharded, field ops)
the guard bands must be untouched, and the results finite and equal to the oracle's -- a read of workspace memory that
no kernel wrote would carry NaN into phi."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

SENTINEL = -6.02214076e23
GUARD = 1 << 15           # doubles on each side


def guarded(torch, numel, fill):
    buf = torch.full((numel + 2 * GUARD,), SENTINEL, dtype=torch.float64, device="cuda")
    inner = buf[GUARD: GUARD + numel]
    inner.fill_(fill)
    return buf, inner


def guards_intact(torch, buf, numel):
    return bool(torch.all(buf[:GUARD] == SENTINEL)) and bool(torch.all(buf[GUARD + numel:] == SENTINEL))


SHAPES = [(8, 8, 8), (16, 8, 32), (16, 16, 64), (32, 16, 64), (64, 64, 16), (128, 32, 16), (256, 16, 8), (16, 256, 32), (8, 32, 256),
          (16, 16, 128), (32, 128, 256),           # per-parity P1 / P2 kernels (n >= 128 on z / y)
          (512, 8, 16), (8, 8, 1024), (16, 512, 8)]


@pytest.mark.parametrize("n", SHAPES)
@pytest.mark.parametrize("mode", ["single", "batch", "slab"])
def test_guard_bands_and_poisoned_workspace(oracle, workloads, n, mode):
    import torch
    from paper_1509_07685_b200 import dks
    nx, ny, nz = n
    h = (1e-3, 2e-3, 5e-4)
    nb = 3 if mode == "batch" else 1
    nodes = nx * ny * nz
    rhos = np.stack([workloads.random_rho(n, seed=17 + i) for i in range(nb)])
    plan = dks.dks_poisson_plan_create(*n, *h)
    try:
        if mode == "batch":
            dks.dks_poisson_set_max_batch(plan, nb)
        if mode == "slab":
            dks.dks_poisson_set_slab_planes(plan, max(1, (nz + 1) // 3))
        ws_doubles = (dks.dks_poisson_workspace_bytes(plan) + 7) // 8 + 32
        ws_buf, ws = guarded(torch, ws_doubles, float("nan"))
        base = ws.data_ptr()
        shift = (-base) % 256                                   # 256-byte alignment inside the guarded buffer
        dks.dks_poisson_set_workspace(plan, base + shift, ws_doubles * 8 - shift)
        rho_buf, rho = guarded(torch, nb * nodes, 0.0)
        phi_buf, phi = guarded(torch, nb * nodes, float("nan"))
        rho.copy_(torch.from_numpy(rhos.ravel()))
        dks.dks_greens_setup(plan)
        if mode == "batch":
            dks.dks_poisson_solve_batch(plan, rho, phi, nb, None)
        else:
            dks.dks_poisson_solve(plan, rho, phi, None)
        torch.cuda.synchronize()
        assert guards_intact(torch, ws_buf, ws_doubles) and guards_intact(torch, rho_buf, nb * nodes) and guards_intact(torch, phi_buf, nb * nodes)
        assert bool(torch.equal(rho, torch.from_numpy(rhos.ravel()).cuda()))           # rho is read-only
        got = phi.cpu().numpy().reshape(nb, nz, ny, nx)
        assert np.all(np.isfinite(got))
        for i in range(nb):
            ref = oracle.solve(rhos[i], n, h, precision="ld")
            assert np.linalg.norm((got[i] - ref).ravel()) <= 1e-12 * np.linalg.norm(ref.ravel())
        if mode == "single":                                    # in place, then the field ops on guarded outputs
            dks.dks_poisson_solve(plan, rho, rho, None)
            e_buf, e = guarded(torch, 3 * nodes, float("nan"))
            dks.dks_gradient(plan, phi, e[:nodes], e[nodes:2 * nodes], e[2 * nodes:], None)
            torch.cuda.synchronize()
            assert guards_intact(torch, rho_buf, nodes) and guards_intact(torch, e_buf, 3 * nodes)
            assert bool(torch.all(torch.isfinite(e))) and bool(torch.equal(rho, phi))
    finally:
        torch.cuda.synchronize()
        dks.dks_poisson_plan_destroy(plan)


def test_guard_bands_deposit_gather(workloads):
    import torch
    from paper_1509_07685_b200 import dks
    n, h, origin = (16, 8, 32), (1e-3, 2e-3, 5e-4), (0.0, 0.0, 0.0)
    nodes, count = 16 * 8 * 32, 50001
    rng = np.random.default_rng(1)
    u = rng.uniform(-2.0, np.array(n) + 1.0, size=(count, 3))     # includes particles outside on every side
    plan = dks.dks_poisson_plan_create(*n, *h)
    try:
        xyz = [torch.from_numpy(np.ascontiguousarray(u[:, a] * h[a])).cuda() for a in range(3)]
        q = torch.ones(count, dtype=torch.float64, device="cuda")
        rho_buf, rho = guarded(torch, nodes, float("nan"))
        dks.dks_deposit_cic(plan, *xyz, q, count, origin, rho, None)
        e_buf, e = guarded(torch, 3 * nodes, 1.0)
        out_buf, out = guarded(torch, 3 * count, float("nan"))
        dks.dks_gather_field(plan, e[:nodes], e[nodes:2 * nodes], e[2 * nodes:], *xyz, count, origin,
                             out[:count], out[count:2 * count], out[2 * count:], None)
        torch.cuda.synchronize()
        assert guards_intact(torch, rho_buf, nodes) and guards_intact(torch, e_buf, 3 * nodes) and guards_intact(torch, out_buf, 3 * count)
        assert bool(torch.all(torch.isfinite(rho))) and bool(torch.all(((out - 1.0).abs() <= 1e-15) | (out == 0.0)))   # weights sum to 1
    finally:
        torch.cuda.synchronize()
        dks.dks_poisson_plan_destroy(plan)

"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element.

Tolerances are BASELINE.json's north_star: relative L2 error <= 1e-12 and max-abs error
<= 1e-11 * max|phi| in fp64 (definitions: SURVEY.md section 8(c) A12 / DESIGN.md).
The oracle is the long-double build (its own error ~1e-18), so the measured error is the GPU's.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

REL_L2_TOL = 1e-12
MAX_ABS_TOL = 1e-11


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def dks():
    from paper_1509_07685_b200 import dks as D
    return D


def gpu_solve(torch, dks, rho, n, h, g0=None):
    plan = dks.PoissonPlan(n, h, g0=g0)
    try:
        d_rho = torch.from_numpy(rho).cuda()
        d_phi = plan.solve(d_rho)
        torch.cuda.synchronize()
        return d_phi.cpu().numpy()
    finally:
        plan.close()


def errors(got, ref):
    rel_l2 = float(np.linalg.norm((got - ref).ravel()) / np.linalg.norm(ref.ravel()))
    max_abs = float(np.max(np.abs(got - ref)) / np.max(np.abs(ref)))
    return rel_l2, max_abs


def check(got, ref):
    assert np.all(np.isfinite(got))
    rel_l2, max_abs = errors(got, ref)
    assert rel_l2 <= REL_L2_TOL, f"rel-L2 {rel_l2:.3e}"
    assert max_abs <= MAX_ABS_TOL, f"max-abs/max|phi| {max_abs:.3e}"
    return rel_l2, max_abs


# ---- BASELINE.json configs 1, 2, 3, 5 in full against the long-double oracle -----------------------
@pytest.mark.parametrize("ci", [1, 2, 3, 5])
def test_config_full_parity(torch_cuda, dks, oracle, workloads, ci):
    w = workloads.config(ci)
    rho = workloads.make_rho(w)
    ref = oracle.solve(rho, w.n, w.h, precision="ld")
    got = gpu_solve(torch_cuda, dks, rho, w.n, w.h)
    rel_l2, max_abs = check(got, ref)
    print(f"{w.name}: rel-L2 {rel_l2:.3e}  max-abs/max {max_abs:.3e}")


# ---- config 4 (256^3), the bench configuration ----------------------------------------------------
# The long-double oracle needs 2 x 4.3 GB and minutes on this size, so at full size the GPU result is
# checked (a) at the 73 stored nodes against the direct summation of Eq. (2) (tests/golden/, written by
# oracle/ only), (b) at ~200 more sampled nodes against direct summation computed now, (c) in full
# against the double-precision oracle build (error ~1e-15, far below the tolerance).
def test_config4_sampled_parity(torch_cuda, dks, oracle, workloads):
    import os
    w = workloads.config(4)
    rho = workloads.make_rho(w)
    got = gpu_solve(torch_cuda, dks, rho, w.n, w.h)
    assert np.all(np.isfinite(got))
    a = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "sampled_phi_cfg4.txt"))
    nodes, direct = a[:, :3].astype(np.int64), a[:, 3]
    g = got[nodes[:, 2], nodes[:, 1], nodes[:, 0]]
    scale = np.max(np.abs(got))
    assert np.max(np.abs(g - direct)) <= MAX_ABS_TOL * scale
    assert np.max(np.abs(g - direct) / np.abs(direct)) <= 1e-11
    more = workloads.sample_nodes(w.n, 12345, count=32)
    d2 = oracle.direct_sum_nodes(rho, w.n, w.h, more)
    g2 = got[more[:, 2], more[:, 1], more[:, 0]]
    assert np.max(np.abs(g2 - d2)) <= MAX_ABS_TOL * scale


@pytest.mark.slow
def test_config4_full_parity_double_oracle(torch_cuda, dks, oracle, workloads):
    w = workloads.config(4)
    rho = workloads.make_rho(w)
    ref = oracle.solve(rho, w.n, w.h, precision="d")
    got = gpu_solve(torch_cuda, dks, rho, w.n, w.h)
    rel_l2, max_abs = check(got, ref)
    print(f"{w.name}: rel-L2 {rel_l2:.3e}  max-abs/max {max_abs:.3e}")


# ---- shapes: every axis length class, non-cubic, anisotropic h, smallest and ragged cases ---------------
SHAPES = [
    ((8, 8, 8), (1e-3, 1e-3, 1e-3)),
    ((8, 16, 32), (1e-3, 2e-3, 5e-4)),
    ((32, 8, 16), (3e-4, 1e-3, 2e-3)),
    ((16, 64, 8), (1e-3, 1e-3, 1e-3)),
    ((64, 32, 128), (2e-4, 3e-4, 1e-4)),
    ((128, 16, 64), (1e-4, 1e-4, 4e-4)),
    ((32, 256, 16), (1e-3, 1e-4, 1e-3)),
    ((256, 8, 8), (1e-4, 1e-3, 1e-3)),
    ((8, 8, 512), (1e-3, 1e-3, 5e-5)),
    ((16, 512, 8), (1e-3, 5e-5, 1e-3)),
    ((512, 8, 16), (5e-5, 1e-3, 1e-3)),
    ((8, 8, 1024), (1e-3, 1e-3, 2e-5)),
    ((1024, 8, 8), (2e-5, 1e-3, 1e-3)),
    ((8, 1024, 8), (1e-3, 2e-5, 1e-3)),
]


@pytest.mark.parametrize("n,h", SHAPES)
def test_shapes_signed_random(torch_cuda, dks, oracle, workloads, n, h):
    rho = workloads.random_rho(n, seed=sum(n))
    ref = oracle.solve(rho, n, h, precision="ld")
    got = gpu_solve(torch_cuda, dks, rho, n, h)
    check(got, ref)


# ---- the paper's own mesh shapes (Table 1: 64x64x32 ... 512x512x256), synthetic Gaussian bunch ----
@pytest.mark.parametrize("n", [(64, 64, 32), (128, 128, 64), (256, 256, 128)])
def test_paper_table1_shapes(torch_cuda, dks, oracle, workloads, n):
    h = (2e-4, 2e-4, 4e-4)
    rho = workloads.random_rho(n, seed=n[0], signed=False)
    ref = oracle.solve(rho, n, h, precision="d")           # double build: error ~1e-15, far below the tolerance
    got = gpu_solve(torch_cuda, dks, rho, n, h)
    check(got, ref)


def test_paper_table1_largest_shape_sampled(torch_cuda, dks, oracle, workloads):
    # 512x512x256 (padded 1024x1024x512): x and y run the long-line passes (n = 512, dks_passes_big.cuh), z the register-resident ones.
    # Checked against direct summation of Eq. (2) at sampled nodes (one pass over rho per node).
    n, h = (512, 512, 256), (1e-4, 1e-4, 2e-4)
    rho = workloads.random_rho(n, seed=99, signed=False)
    got = gpu_solve(torch_cuda, dks, rho, n, h)
    assert np.all(np.isfinite(got))
    nodes = workloads.sample_nodes(n, 7, count=7)
    direct = oracle.direct_sum_nodes(rho, n, h, nodes)
    g = got[nodes[:, 2], nodes[:, 1], nodes[:, 0]]
    assert np.max(np.abs(g - direct)) <= MAX_ABS_TOL * np.max(np.abs(got))
    assert np.max(np.abs(g - direct) / np.abs(direct)) <= 1e-11


@pytest.mark.slow
def test_paper_table1_largest_shape_1000_nodes_and_library_fft(torch_cuda, dks, oracle, workloads):
    # The only large workload of p2_y_fwd_big / p3_x_conv_big / p4_y_inv_big.  The oracle's doubled-grid arrays
    # would need 2 x 8.6 GB of host memory here, so: (i) Eq. (2) summed directly by the oracle at 1009 sampled nodes (about 40 s
    # of host time), and (ii) EVERY node against the same convolution through torch.fft (cuFFT) -- a third opinion, not the oracle,
    # which ties the unsampled nodes to the sampled ones: a wrong row, tile or plane anywhere fails (ii), a common error (i).
    torch = torch_cuda
    n, h = (512, 512, 256), (1e-4, 1e-4, 2e-4)
    (nx, ny, nz), (hx, hy, hz) = n, h
    rho = workloads.random_rho(n, seed=98, signed=False)
    d_rho = torch.from_numpy(rho).cuda()
    plan = dks.PoissonPlan(n, h, host_staging=False)
    try:
        got_d = plan.solve(d_rho)
        torch.cuda.synchronize()
    finally:
        plan.close()
    got = got_d.cpu().numpy()
    assert np.all(np.isfinite(got))
    nodes = workloads.sample_nodes(n, 8, count=1000)
    direct = oracle.direct_sum_nodes(rho, n, h, nodes, precision="ld")
    g = got[nodes[:, 2], nodes[:, 1], nodes[:, 0]]
    assert np.max(np.abs(g - direct)) <= MAX_ABS_TOL * np.max(np.abs(got))
    assert np.linalg.norm(g - direct) <= REL_L2_TOL * np.linalg.norm(direct)

    def mirrored(m, hh):
        i = torch.arange(2 * m, device="cuda", dtype=torch.float64)
        return torch.minimum(i, 2 * m - i) * hh

    r = torch.sqrt(mirrored(nz, hz)[:, None, None] ** 2 + mirrored(ny, hy)[None, :, None] ** 2 + mirrored(nx, hx)[None, None, :] ** 2)
    r[0, 0, 0] = 0.5 * min(hx, hy, hz)
    ghat = torch.fft.rfftn(1.0 / (4.0 * np.pi * 8.8541878128e-12 * r))
    del r
    shape = (2 * nz, 2 * ny, 2 * nx)
    spec = torch.fft.rfftn(d_rho, s=shape)
    spec *= ghat
    del ghat
    ref = torch.fft.irfftn(spec, s=shape)[:nz, :ny, :nx] * (hx * hy * hz)
    del spec
    assert float(torch.linalg.norm((got_d - ref).flatten()) / torch.linalg.norm(ref.flatten())) <= REL_L2_TOL
    assert float((got_d - ref).abs().max()) <= MAX_ABS_TOL * float(ref.abs().max())
    del ref, got_d
    torch.cuda.empty_cache()


def test_full_size_agreement_with_a_library_fft_on_the_gpu(torch_cuda, dks, workloads):
    # A third opinion at a size the long-double oracle needs minutes for: the same convolution through torch.fft (cuFFT) on the doubled
    # grid of config 3 (the library special case of pin P12, run on the GPU).  Not the oracle: an independent FFT, same readings A1-A5.
    torch = torch_cuda
    w = workloads.config(3)
    (nx, ny, nz), (hx, hy, hz) = w.n, w.h
    d_rho = torch.from_numpy(workloads.make_rho(w)).cuda()

    def mirrored(n, h):
        i = torch.arange(2 * n, device="cuda", dtype=torch.float64)
        return torch.minimum(i, 2 * n - i) * h

    r = torch.sqrt(mirrored(nz, hz)[:, None, None] ** 2 + mirrored(ny, hy)[None, :, None] ** 2 + mirrored(nx, hx)[None, None, :] ** 2)
    r[0, 0, 0] = 0.5 * min(hx, hy, hz)
    g = 1.0 / (4.0 * np.pi * 8.8541878128e-12 * r)
    shape = (2 * nz, 2 * ny, 2 * nx)
    ref = torch.fft.irfftn(torch.fft.rfftn(d_rho, s=shape) * torch.fft.rfftn(g), s=shape)[:nz, :ny, :nx] * (hx * hy * hz)
    plan = dks.PoissonPlan(w.n, w.h)
    try:
        got = plan.solve(d_rho)
        assert float(torch.linalg.norm((got - ref).flatten()) / torch.linalg.norm(ref.flatten())) <= REL_L2_TOL
        assert float((got - ref).abs().max()) <= MAX_ABS_TOL * float(ref.abs().max())
    finally:
        plan.close()


# ---- batched solves: several meshes per launch, one Green's transform ------------------------------------
@pytest.mark.parametrize("n,h", [((32, 16, 64), (2e-4, 3e-4, 1e-4)), ((64, 64, 64), (5e-4, 5e-4, 5e-4)),
                                 ((8, 16, 8), (1e-3, 1e-3, 2e-3)), ((128, 32, 16), (1e-4, 2e-4, 4e-4)),
                                 ((32, 128, 128), (2e-4, 1e-4, 3e-4))])                      # per-parity P1 and P2 kernels
def test_solve_batch_matches_single_solves_and_oracle(torch_cuda, dks, oracle, workloads, n, h):
    torch = torch_cuda
    nb = 3
    rhos = np.stack([workloads.random_rho(n, seed=70 + i) for i in range(nb)])
    plan = dks.PoissonPlan(n, h, max_batch=4)
    try:
        d = torch.from_numpy(rhos).cuda()
        got = plan.solve_batch(d).cpu().numpy()
        for i in range(nb):
            single = plan.solve(d[i].contiguous()).cpu().numpy()
            assert np.array_equal(got[i], single)           # same kernels, same arithmetic: bit-identical
        check(got[1], oracle.solve(rhos[1], n, h, precision="ld"))
        with pytest.raises(dks.DksError) as e:              # more meshes than the workspace was sized for
            dks.dks_poisson_solve_batch(plan.handle, d, d, 5, None)
        assert e.value.status == dks.DKS_ERR_INVALID_ARG
    finally:
        plan.close()


# ---- opt-in variant: slab-by-slab launches of P2-P4 ----
@pytest.mark.parametrize("slab", [1, 3, 17])
def test_slab_launches_match_oracle(torch_cuda, dks, oracle, workloads, slab):
    n, h = (32, 64, 16), (2e-4, 3e-4, 1e-4)
    rho = workloads.random_rho(n, seed=21)
    ref = oracle.solve(rho, n, h, precision="ld")
    plan = dks.PoissonPlan(n, h, slab_planes=slab)
    try:
        assert dks.dks_poisson_slab_planes(plan.handle) == slab
        got = plan.solve(torch_cuda.from_numpy(rho).cuda()).cpu().numpy()
    finally:
        plan.close()
    check(got, ref)


# ---- degenerate inputs -------------------------------------------------------------------------------
def test_zero_rho_gives_zero_phi(torch_cuda, dks):
    n, h = (16, 16, 16), (1e-3, 1e-3, 1e-3)
    got = gpu_solve(torch_cuda, dks, np.zeros((16, 16, 16)), n, h)
    assert np.all(got == 0.0)


@pytest.mark.parametrize("src", [(0, 0, 0), (15, 31, 7), (7, 13, 3)])
def test_point_charge(torch_cuda, dks, oracle, src):
    # rho = q/(hx hy hz) at one node -> phi = q G(x - s), phi[s] = q g0 (PAPER.md:121 with one term)
    n, h = (16, 32, 8), (1e-3, 5e-4, 2e-3)
    nx, ny, nz = n
    q = 1e-9
    rho = np.zeros((nz, ny, nx))
    rho[src[2], src[1], src[0]] = q / (h[0] * h[1] * h[2])
    got = gpu_solve(torch_cuda, dks, rho, n, h)
    ref = oracle.solve(rho, n, h, precision="ld")
    check(got, ref)
    far = (nx - 1 - src[0], ny - 1 - src[1], nz - 1 - src[2])
    if far != src:
        g = q * oracle.green((far[0] - src[0]) * h[0], (far[1] - src[1]) * h[1], (far[2] - src[2]) * h[2])
        assert abs(got[far[2], far[1], far[0]] - g) <= 1e-11 * np.max(np.abs(got))
    assert abs(got[src[2], src[1], src[0]] - q * oracle.default_g0(h)) <= 1e-11 * np.max(np.abs(got))


def test_g0_override_and_spacing_change(torch_cuda, dks, oracle, workloads):
    torch = torch_cuda
    n, h1, h2 = (16, 16, 32), (1e-3, 1e-3, 1e-3), (2e-3, 1e-3, 5e-4)
    rho = workloads.random_rho(n, seed=5, signed=False)
    plan = dks.PoissonPlan(n, h1, g0=123.0)
    try:
        d_rho = torch.from_numpy(rho).cuda()
        got1 = plan.solve(d_rho).cpu().numpy()
        check(got1, oracle.solve(rho, n, h1, g0=123.0, precision="ld"))
        dks.dks_poisson_set_g0(plan.handle, float("nan"))
        # spacing changed: solve must refuse until the Green's transform is rebuilt
        dks.dks_poisson_set_spacing(plan.handle, *h2)
        with pytest.raises(dks.DksError) as e:
            dks.dks_poisson_solve(plan.handle, d_rho, d_rho, None)
        assert e.value.status == dks.DKS_ERR_NOT_SETUP
        plan.set_spacing(h2)
        got2 = plan.solve(d_rho).cpu().numpy()
        check(got2, oracle.solve(rho, n, h2, precision="ld"))
    finally:
        plan.close()


def test_in_place_and_repeatable(torch_cuda, dks, oracle, workloads):
    torch = torch_cuda
    w = workloads.config(2)
    rho = workloads.make_rho(w)
    plan = dks.PoissonPlan(w.n, w.h)
    try:
        d = torch.from_numpy(rho).cuda()
        out1 = plan.solve(d).clone()
        out2 = plan.solve(d).clone()
        assert torch.equal(out1, out2)                       # deterministic, no hidden state
        buf = d.clone()
        plan.solve(buf, buf)                                 # phi aliases rho
        assert torch.equal(buf, out1)
    finally:
        plan.close()


@pytest.mark.parametrize("n", [(128, 128, 128), (256, 64, 32), (64, 256, 256), (32, 16, 512)])
def test_repeated_solves_are_bit_identical(torch_cuda, dks, workloads, n):
    # races in the shared-memory exchanges / async prefetch pipelines would show up as run-to-run differences
    torch = torch_cuda
    plan = dks.PoissonPlan(n, (1e-4, 2e-4, 3e-4))
    try:
        d = torch.from_numpy(workloads.random_rho(n, seed=5)).cuda()
        first = plan.solve(d).clone()
        out = torch.empty_like(d)
        for _ in range(40):
            plan.solve(d, out)
            assert torch.equal(out, first)
    finally:
        plan.close()


def test_greens_point_charge_at_origin_returns_G(torch_cuda, dks, oracle):
    # solve of a unit point charge at the origin returns exactly G on the mesh (a0 through the whole pipeline)
    n, h = (16, 16, 16), (1e-3, 2e-3, 5e-4)
    rho = np.zeros((16, 16, 16))
    rho[0, 0, 0] = 1.0 / (h[0] * h[1] * h[2])
    got = gpu_solve(torch_cuda, dks, rho, n, h)
    for (i, j, k) in [(1, 0, 0), (0, 1, 0), (0, 0, 1), (3, 4, 5), (15, 15, 15)]:
        g = oracle.green(i * h[0], j * h[1], k * h[2])
        assert abs(got[k, j, i] - g) <= 1e-11 * np.max(np.abs(got))


# ---- step a0 directly: the Green's octant of dks_greens_setup against the oracle's FT{Gt} ----
@pytest.mark.parametrize("n,h,g0", [((16, 8, 32), (1e-3, 2e-3, 5e-4), None),           # generic x, y; r16 z
                                     ((512, 16, 8), (5e-5, 1e-3, 1e-3), None),            # long-line x (greens_axis_big)
                                     ((8, 1024, 16), (1e-3, 2e-5, 1e-3), None),           # long-line y
                                     ((32, 64, 16), (2e-4, 3e-4, 1e-4), 7.5e12),         # r16 x, y; generic z
                                     ((128, 32, 64), (1e-4, 2e-4, 4e-4), None),
                                     ((256, 16, 8), (1e-4, 1e-3, 1e-3), None),
                                     ((8, 8, 8), (1e-3, 1e-3, 1e-3), None)])
def test_greens_octant_matches_oracle(torch_cuda, dks, oracle, n, h, g0):
    nx, ny, nz = n
    plan = dks.PoissonPlan(n, h, g0=g0)
    try:
        got = plan.greens_hat()                              # scale hx hy hz / (8 nx ny nz) folded in
    finally:
        plan.close()
    op = oracle.Plan(n, h, g0=g0, precision="ld")
    try:
        ref = op.ghat_octant() * (h[0] * h[1] * h[2] / (8.0 * nx * ny * nz))
    finally:
        op.close()
    assert got.shape == ref.shape == (nz + 1, ny + 1, nx + 1)
    # Ghat is a sum of 8 nx ny nz terms of mixed sign: the bound is relative to its largest entry
    assert np.max(np.abs(got - ref)) <= 1e-12 * np.max(np.abs(ref))
    assert np.linalg.norm((got - ref).ravel()) <= 1e-13 * np.linalg.norm(ref.ravel())


def test_greens_octant_pad_columns_stay_negligible(torch_cuda, dks):
    # The pad entries nx < kx < gpitch of every octant row are the imaginary partners of valid columns in the packed
    # y / z transforms of the setup (dks_greens_r16.cuh): they start at zero and may only pick up the rounding leakage of
    # their partner column; a NaN or a large value there would contaminate column nx.  Read them raw from the workspace.
    torch = torch_cuda
    for n in [(32, 16, 64), (16, 32, 8), (64, 64, 64)]:
        nx, ny, nz = n
        h_ = dks.dks_poisson_plan_create(*n, 1e-3, 2e-3, 5e-4)
        try:
            nbytes = dks.dks_poisson_workspace_bytes(h_)
            ws = torch.full((nbytes // 8,), float("nan"), dtype=torch.float64, device="cuda")
            dks.dks_poisson_set_workspace(h_, ws, nbytes)
            dks.dks_greens_setup(h_)
            torch.cuda.synchronize()
            gpitch = (nx + 1 + 7) // 8 * 8
            off = ((16 * nx * ny * (nz + 1) + 255) // 256 * 256) // 8        # the octant follows buffer A
            G = ws[off: off + gpitch * (ny + 1) * (nz + 1)].view(nz + 1, ny + 1, gpitch)
            assert torch.all(torch.isfinite(G))
            scale = 1e-3 * 2e-3 * 5e-4 / (8.0 * nx * ny * nz)   # folded into the valid entries by the last axis pass only
            assert float(G[:, :, nx + 1:].abs().max()) <= 1e-14 * float(G[:, :, : nx + 1].abs().max()) / scale
            assert torch.all(G[:, :, nx + 2:] == 0.0)        # only column nx + 1 has a valid partner (column nx)
        finally:
            dks.dks_poisson_plan_destroy(h_)


# ---- f1: the per-step sequence of PAPER.md:132 (h changes every step) ------------------------------------
def test_step_host_async_rebuilds_every_step(torch_cuda, dks, oracle, workloads):
    torch = torch_cuda
    n = (32, 16, 64)
    hs = [(2e-4 * (1 + 0.1 * i), 3e-4 * (1 - 0.05 * i), 1e-4 * (1 + 0.2 * i)) for i in range(5)]
    rhos = [workloads.random_rho(n, seed=90 + i) for i in range(5)]
    plan = dks.PoissonPlan(n, hs[0])
    try:
        h_in = [torch.from_numpy(r).pin_memory() for r in rhos]
        h_out = [torch.empty_like(t).pin_memory() for t in h_in]
        for h, a, b in zip(hs, h_in, h_out):
            plan.step_host_async(h, a, b)
        plan.host_sync()
        for h, r, b in zip(hs, rhos, h_out):
            check(b.numpy(), oracle.solve(r, n, h, precision="ld"))
    finally:
        plan.close()


def test_rebuild_on_side_stream_between_pipelined_solves(torch_cuda, dks, oracle, workloads):
    # dks_greens_setup on its own stream between solve_host_async calls: the rebuild must wait for the previous P3
    torch = torch_cuda
    n = (64, 32, 32)
    hs = [(1e-4 * (1 + i), 2e-4, 3e-4 / (1 + i)) for i in range(4)]
    rhos = [workloads.random_rho(n, seed=60 + i) for i in range(4)]
    side = torch.cuda.Stream()
    plan = dks.PoissonPlan(n, hs[0])
    try:
        dks.dks_poisson_set_stream(plan.handle, side.cuda_stream)
        h_in = [torch.from_numpy(r).pin_memory() for r in rhos]
        h_out = [torch.empty_like(t).pin_memory() for t in h_in]
        for h, a, b in zip(hs, h_in, h_out):
            dks.dks_poisson_set_spacing(plan.handle, *h)
            dks.dks_greens_setup(plan.handle)
            plan.solve_host_async(a, b)
        plan.host_sync()
        for h, r, b in zip(hs, rhos, h_out):
            check(b.numpy(), oracle.solve(r, n, h, precision="ld"))
    finally:
        torch.cuda.synchronize()
        plan.close()


def test_rebuild_moves_to_another_stream_behind_queued_solves(torch_cuda, dks, oracle, workloads):
    # PoissonPlan(h0) builds Ghat on torch's current stream and the solves below run there too, so no solve records an event.
    # step_host_async(h1) then moves the rebuild to the plan's own stream while those solves are still queued: it must wait
    # for the first build and for the last queued P3 (it overwrites Ghat in place), with no host synchronisation in between.
    torch = torch_cuda
    n = (128, 128, 128)
    h0, h1 = (1e-4, 2e-4, 3e-4), (2.5e-4, 1.5e-4, 0.7e-4)
    rho0, rho1 = workloads.random_rho(n, seed=71), workloads.random_rho(n, seed=72)
    ref0 = oracle.solve(rho0, n, h0, precision="d")
    ref1 = oracle.solve(rho1, n, h1, precision="d")
    d_rho0 = torch.from_numpy(rho0).cuda()
    phis = [torch.empty_like(d_rho0) for _ in range(24)]
    h_in, h_out = torch.from_numpy(rho1).pin_memory(), torch.empty(rho1.shape, dtype=torch.float64).pin_memory()
    torch.cuda.synchronize()
    plan = dks.PoissonPlan(n, h0)
    try:
        for phi in phis:                       # about 2.5 ms of queued work, all of it reading the h0 transform
            plan.solve(d_rho0, phi)
        plan.step_host_async(h1, h_in, h_out)
        plan.host_sync()
        torch.cuda.synchronize()
        check(phis[-1].cpu().numpy(), ref0)
        check(phis[0].cpu().numpy(), ref0)
        assert all(torch.equal(phis[0], phi) for phi in phis[1:])
        check(h_out.numpy(), ref1)
    finally:
        plan.close()


def test_two_live_plans_of_different_shapes(torch_cuda, dks, oracle, workloads):
    # the kernels' shared-memory attributes are process-wide: a small plan must not lower what a large one needs
    torch = torch_cuda
    big, small = ((8, 8, 512), (1e-3, 1e-3, 5e-5)), ((16, 16, 16), (1e-3, 1e-3, 1e-3))
    rb, rs = workloads.random_rho(big[0], seed=1), workloads.random_rho(small[0], seed=2)
    pb = dks.PoissonPlan(*big)
    ps = dks.PoissonPlan(*small)
    try:
        db, ds = torch.from_numpy(rb).cuda(), torch.from_numpy(rs).cuda()
        for _ in range(2):
            check(pb.solve(db).cpu().numpy(), oracle.solve(rb, *big, precision="ld"))
            check(ps.solve(ds).cpu().numpy(), oracle.solve(rs, *small, precision="ld"))
            pb.set_spacing(big[1])
            ps.set_spacing(small[1])
    finally:
        pb.close()
        ps.close()


# ---- refusals ---------------------------------------------------------------------------------------------------------
def test_refusals(torch_cuda, dks, workloads):
    torch = torch_cuda
    n, h = (16, 16, 16), (1e-3, 1e-3, 1e-3)
    d = torch.zeros(16 * 16 * 16 + 1, dtype=torch.float64, device="cuda")
    plan = dks.PoissonPlan(n, h, slab_planes=5)
    try:
        with pytest.raises(dks.DksError) as e:               # rho not 16-byte aligned
            dks.dks_poisson_solve(plan.handle, d.data_ptr() + 8, d.data_ptr(), None)
        assert e.value.status == dks.DKS_ERR_INVALID_ARG and "aligned" in str(e.value)
        with pytest.raises(dks.DksError) as e:               # batched solve on a slabbed plan
            dks.dks_poisson_solve_batch(plan.handle, d, d, 2, None)
        assert e.value.status == dks.DKS_ERR_INVALID_ARG
        with pytest.raises(dks.DksError) as e:               # the attached workspace cannot hold a batch of 4
            dks.dks_poisson_set_max_batch(plan.handle, 4)
        assert e.value.status == dks.DKS_ERR_WORKSPACE_TOO_SMALL
        with pytest.raises(dks.DksError) as e:               # nor the unslabbed B
            dks.dks_poisson_set_slab_planes(plan.handle, 17)
        assert e.value.status == dks.DKS_ERR_WORKSPACE_TOO_SMALL
        plan.solve(d[:4096].view(16, 16, 16))                # the plan still works after the refusals
        torch.cuda.synchronize()
    finally:
        plan.close()
    big = dks.dks_poisson_plan_create(8, 8, 1024, 1e-3, 1e-3, 1e-3)
    try:
        with pytest.raises(dks.DksError) as e:               # (nz + 1) * nbatch exceeds the grid limit of the y passes
            dks.dks_poisson_set_max_batch(big, 64)
        assert e.value.status == dks.DKS_ERR_INVALID_ARG and "65535" in str(e.value)
    finally:
        dks.dks_poisson_plan_destroy(big)


def test_solve_host_path(torch_cuda, dks, oracle, workloads):
    torch = torch_cuda
    w = workloads.config(1)
    rho = workloads.make_rho(w)
    plan = dks.PoissonPlan(w.n, w.h)
    try:
        h_rho = torch.from_numpy(rho).pin_memory()
        h_phi = torch.empty_like(h_rho).pin_memory()
        plan.solve_host(h_rho, h_phi)
        check(h_phi.numpy(), oracle.solve(rho, w.n, w.h, precision="ld"))
    finally:
        plan.close()


def test_solve_host_async_pipeline(torch_cuda, dks, oracle, workloads):
    # eight pipelined steps with different inputs: every step's phi must be its own (three staging slots take turns, so every
    # slot is reused at least twice and a copy-in has to wait for the copy-out that frees its slot)
    torch = torch_cuda
    n, h = (32, 16, 64), (2e-4, 3e-4, 1e-4)
    rhos = [workloads.random_rho(n, seed=40 + i) for i in range(8)]
    plan = dks.PoissonPlan(n, h)
    try:
        h_in = [torch.from_numpy(r).pin_memory() for r in rhos]
        h_out = [torch.empty_like(t).pin_memory() for t in h_in]
        for a, b in zip(h_in, h_out):
            plan.solve_host_async(a, b)
        plan.host_sync()
        for r, b in zip(rhos, h_out):
            check(b.numpy(), oracle.solve(r, n, h, precision="ld"))
    finally:
        plan.close()


def test_stream_ordering_and_graph_capture(torch_cuda, dks, oracle, workloads):
    torch = torch_cuda
    w = workloads.config(1)
    rho = workloads.make_rho(w)
    ref = oracle.solve(rho, w.n, w.h, precision="ld")
    plan = dks.PoissonPlan(w.n, w.h)
    try:
        s = torch.cuda.Stream()
        d_rho = torch.from_numpy(rho).cuda()
        d_phi = torch.empty_like(d_rho)
        torch.cuda.synchronize()
        with torch.cuda.stream(s):
            plan.solve(d_rho, d_phi)
        s.synchronize()
        check(d_phi.cpu().numpy(), ref)
        # CUDA-graph capture of the solve (stream-ordered, no allocation, no sync inside)
        d_phi.zero_()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            plan.solve(d_rho, d_phi)
        g.replay()
        torch.cuda.synchronize()
        check(d_phi.cpu().numpy(), ref)
    finally:
        plan.close()


def test_caller_owned_and_plan_owned_workspace(torch_cuda, dks, oracle, workloads):
    torch = torch_cuda
    n, h = (16, 16, 16), (1e-3, 1e-3, 1e-3)
    rho = workloads.random_rho(n, seed=3)
    ref = oracle.solve(rho, n, h, precision="ld")
    d_rho = torch.from_numpy(rho).cuda()
    # plan-owned workspace (allocated at setup, not in solve)
    p = dks.PoissonPlan(n, h, own_workspace=False)
    try:
        check(p.solve(d_rho).cpu().numpy(), ref)
    finally:
        p.close()
    # too-small caller workspace is refused
    h_ = dks.dks_poisson_plan_create(*n, *h)
    try:
        small = torch.empty(1024, dtype=torch.uint8, device="cuda")
        with pytest.raises(dks.DksError) as e:
            dks.dks_poisson_set_workspace(h_, small, 1024)
        assert e.value.status == dks.DKS_ERR_WORKSPACE_TOO_SMALL
        with pytest.raises(dks.DksError) as e:
            dks.dks_poisson_solve(h_, d_rho, d_rho, None)
        assert e.value.status == dks.DKS_ERR_NOT_SETUP
    finally:
        dks.dks_poisson_plan_destroy(h_)


def test_plan_without_host_staging(torch_cuda, dks, oracle, workloads):
    # device-resident callers can leave the three staging meshes out of the workspace; the host path is then refused
    torch = torch_cuda
    n, h = (32, 16, 64), (2e-4, 3e-4, 1e-4)
    rho = workloads.random_rho(n, seed=5)
    full = dks.PoissonPlan(n, h)
    plan = dks.PoissonPlan(n, h, host_staging=False)
    try:
        assert dks.dks_poisson_workspace_bytes(full.handle) - dks.dks_poisson_workspace_bytes(plan.handle) == 3 * rho.nbytes
        with pytest.raises(dks.DksError):                      # the workspace is attached: too late to change its layout
            dks.dks_poisson_set_host_staging(plan.handle, True)
        d_rho = torch.from_numpy(rho).cuda()
        phi = plan.solve(d_rho)
        e = plan.field_at_particles(phi, d_rho.flatten()[:100].contiguous(), d_rho.flatten()[:100].contiguous(),
                                    d_rho.flatten()[:100].contiguous(), (0.0, 0.0, 0.0))      # buffer B is still there
        torch.cuda.synchronize()
        assert torch.equal(phi, full.solve(d_rho))
        check(phi.cpu().numpy(), oracle.solve(rho, n, h, precision="ld"))
        out = np.empty_like(rho)
        with pytest.raises(dks.DksError) as err:
            plan.solve_host(rho, out)
        assert err.value.status == dks.DKS_ERR_NOT_SETUP
    finally:
        torch.cuda.synchronize()
        full.close()
        plan.close()


def test_long_line_passes_are_selected(dks):
    cases = {(64, 64, 512): ["p1_z_r2c_big", "p2_y_fwd_r16", "p3_x_conv_r16", "p4_y_inv_r16", "p5_z_c2r_big"],
             (512, 512, 256): ["p1_z_r2c_r16p", "p2_y_fwd_big", "p3_x_conv_big", "p4_y_inv_big", "p5_z_c2r_r16"],
             (8, 1024, 1024): ["p1_z_r2c_big", "p2_y_fwd_big", "p3_x_conv_generic", "p4_y_inv_big", "p5_z_c2r_big"],
             (16, 64, 16): ["p1_z_r2c_r16", "p2_y_fwd_r16", "p3_x_conv_r16", "p4_y_inv_r16", "p5_z_c2r_r16"],
             (16, 16, 16): ["p1_z_r2c_r16", "p2_y_fwd_r16", "p3_x_conv_r16", "p4_y_inv_r16", "p5_z_c2r_r16"],
             (8, 8, 512): ["p1_z_r2c_generic", "p2_y_fwd_generic", "p3_x_conv_generic", "p4_y_inv_generic", "p5_z_c2r_generic"]}
    for n, names in cases.items():
        h_ = dks.dks_poisson_plan_create(*n, 1e-3, 1e-3, 1e-3)
        try:
            assert [dks.dks_poisson_pass_name(h_, i) for i in range(1, 6)] == names
        finally:
            dks.dks_poisson_plan_destroy(h_)


def test_pass_times_and_names(torch_cuda, dks, workloads):
    torch = torch_cuda
    w = workloads.config(2)
    plan = dks.PoissonPlan(w.n, w.h)
    try:
        d = torch.from_numpy(workloads.make_rho(w)).cuda()
        dks.dks_poisson_set_profiling(plan.handle, True)
        plan.solve(d)
        t = dks.dks_poisson_pass_times(plan.handle)
        assert len(t) == 5 and all(x > 0 for x in t)
        assert all(dks.dks_poisson_pass_name(plan.handle, i) for i in range(1, 6))
        assert dks.dks_poisson_launches_per_solve(plan.handle) >= 1
    finally:
        plan.close()

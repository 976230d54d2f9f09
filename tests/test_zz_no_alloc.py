"""dks_field_at_particles_static: the field at the particles for callers that cannot allocate device memory.

Who needs it: code that must not call cudaMalloc where it runs -- a time-step loop in which the device-wide
synchronisation of cudaMalloc / cudaFree would stall the other streams, a host program whose own pool already holds all
device memory (a further cudaMalloc fails there), a component that is handed device pointers and owns no allocator.  The
plan-based dks_field_at_particles is closed to them (a plan allocates its tables and, unless given one, its workspace),
so this entry point keeps the node field in an 8 MiB array inside the library and takes no plan.

What is checked: on two calls in a row (different mesh shapes, different data, so the second call finds the first
call's records in the shared array) the outputs equal those of the plan-based path on the same inputs, within the
gather tolerance of tests/test_gpu_field_ops.py; meshes beyond DKS_STATIC_FIELD_MAX_NODES are refused with a message
that names the limit.

The file name sorts last on purpose: pytest -x stops at the first failure, and a failure here must not hide the parity
tests.  The GPU test does not depend on what ran before it: it passes alone in a fresh process (its first call is then
the first CUDA work of the library on the device) and after the rest of the suite.
"""
import numpy as np
import pytest


def _dks():
    from paper_1509_07685_b200 import dks as D
    return D


def test_static_rejects_meshes_beyond_the_limit():
    # validation comes before any CUDA call, so this runs without a GPU
    dks = _dks()
    assert dks.DKS_STATIC_FIELD_MAX_NODES == 64 * 64 * 64
    for n in [(128, 64, 64), (64, 64, 128), (1024, 1024, 8)]:
        with pytest.raises(dks.DksError) as e:
            dks.dks_field_at_particles_static(n, (1e-3, 1e-3, 1e-3), 256, 256, 256, 256, 1, (0, 0, 0), 256, 256, 256, None)
        assert e.value.status == dks.DKS_ERR_INVALID_ARG
        assert "at most 262144" in str(e.value) and "DKS_STATIC_FIELD_MAX_NODES" in str(e.value)
    for n, h in [((12, 8, 8), (1e-3, 1e-3, 1e-3)), ((8, 8, 4), (1e-3, 1e-3, 1e-3)), ((8, 8, 8), (0.0, 1e-3, 1e-3)),
                 ((8, 8, 8), (1e-3, float("nan"), 1e-3))]:
        with pytest.raises(dks.DksError) as e:
            dks.dks_field_at_particles_static(n, h, 256, 256, 256, 256, 1, (0, 0, 0), 256, 256, 256, None)
        assert e.value.status == dks.DKS_ERR_INVALID_ARG
    with pytest.raises(dks.DksError):                                                    # NULL phi, negative np
        dks.dks_field_at_particles_static((8, 8, 8), (1e-3, 1e-3, 1e-3), None, 256, 256, 256, 1, (0, 0, 0), 256, 256, 256, None)
    with pytest.raises(dks.DksError):
        dks.dks_field_at_particles_static((8, 8, 8), (1e-3, 1e-3, 1e-3), 256, 256, 256, 256, -1, (0, 0, 0), 256, 256, 256, None)


@pytest.mark.gpu
def test_static_matches_plan_path_on_two_calls_in_a_row():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    dks = _dks()
    from paper_1509_07685_b200 import workloads

    # call 1 fills the whole array (64^3 = the limit); call 2 is a smaller, non-cubic mesh with other spacings and data
    cases = [((64, 64, 64), (2e-4, 3e-4, 1e-4), 50001, 11), ((16, 8, 32), (1e-3, 2e-3, 5e-4), 30000, 12)]
    origin = (0.25e-3, -1e-3, 3.0)
    inputs, got = [], []
    stream = torch.cuda.current_stream().cuda_stream
    for n, h, count, seed in cases:
        rng = np.random.default_rng(seed)
        phi = workloads.random_rho(n, seed=seed)
        u = rng.uniform(-1.5, np.array(n) - 1 + 1.5, size=(count, 3))                   # some particles fall outside: field 0
        d = [torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()
             for a in (phi, origin[0] + u[:, 0] * h[0], origin[1] + u[:, 1] * h[1], origin[2] + u[:, 2] * h[2])]
        inputs.append(d)
        out = [torch.full((count,), 7.0, dtype=torch.float64, device="cuda") for _ in range(3)]
        # the two calls follow each other on one stream with no synchronisation in between
        dks.dks_field_at_particles_static(n, h, d[0], d[1], d[2], d[3], count, origin, *out, stream)
        got.append(out)
    torch.cuda.synchronize()
    for (n, h, count, seed), d, out in zip(cases, inputs, got):
        plan = dks.PoissonPlan(n, h)                                                    # the existing path: plan + workspace
        try:
            ref = plan.field_at_particles(d[0], d[1], d[2], d[3], origin)
            torch.cuda.synchronize()
        finally:
            plan.close()
        phi_max = float(d[0].abs().max())
        for g, r in zip(out, ref):
            g, r = g.cpu().numpy(), r.cpu().numpy()
            field_max = np.max(np.abs(r))
            assert field_max > 0 and np.count_nonzero(r == 0.0) > 0                      # kept and dropped particles both occur
            # tolerance of test_gradient_and_gather (tests/test_gpu_field_ops.py): gather 1e-14 max|field| + gradient 1e-14 max|phi| / min h
            assert np.max(np.abs(g - r)) <= 1e-14 * field_max + 1e-14 * phi_max / min(h)
            assert np.array_equal(g == 0.0, r == 0.0)
    # np = 0 is a no-op that leaves the outputs alone
    keep = got[1][0].clone()
    dks.dks_field_at_particles_static(cases[1][0], cases[1][1], inputs[1][0], None, None, None, 0, origin, None, None, None, stream)
    torch.cuda.synchronize()
    assert torch.equal(keep, got[1][0])

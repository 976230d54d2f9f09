"""CPU-side checks of the boundary: the C-ABI library loads and exports every symbol
include/dks_poisson.h declares; host-only entry points validate their arguments.  No compute calls.
"""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def dks():
    from paper_1509_07685_b200 import dks as D
    return D


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "dks_poisson.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dks_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_all_exported(dks):
    names = declared_symbols()
    assert "dks_poisson_plan_create" in names and "dks_greens_setup" in names and "dks_poisson_solve" in names
    raw = ctypes.CDLL(dks.LIB_PATH)
    for name in names:
        assert hasattr(raw, name), f"{name} declared in include/dks_poisson.h but not exported"
    # and the binding covers the same set, name for name
    assert set(names) == set(dks.SYMBOLS)
    for name in names:
        assert callable(getattr(dks, name))


def test_plan_create_validates(dks):
    for bad in [(12, 16, 16), (16, 4, 16), (16, 16, 2048), (0, 16, 16), (-8, 8, 8)]:
        with pytest.raises(dks.DksError):
            dks.dks_poisson_plan_create(*bad, 1e-3, 1e-3, 1e-3)
        assert "power of two" in dks.dks_last_error()
    for badh in [(0.0, 1e-3, 1e-3), (1e-3, -1.0, 1e-3), (1e-3, 1e-3, float("nan")), (float("inf"), 1, 1)]:
        with pytest.raises(dks.DksError):
            dks.dks_poisson_plan_create(16, 16, 16, *badh)


def test_host_only_queries(dks):
    p = dks.dks_poisson_plan_create(256, 256, 256, 1e-4, 1e-4, 1e-4)
    try:
        nx = ny = nz = 256
        a = 16 * nx * ny * (nz + 1)
        g = 8 * (nx + 1) * (ny + 1) * (nz + 1)
        # DESIGN.md model M3: rho + phi + 4 A + 4 B + Ghat octant, B = 2 A
        assert dks.dks_poisson_model_bytes(p, 0) == 2 * 8 * nx * ny * nz + 12 * a + g
        assert abs(dks.dks_poisson_model_bytes(p, 0) - 3638.0e6) < 0.5e6        # SURVEY.md 8(d), cfg 4
        assert sum(dks.dks_poisson_model_bytes(p, i) for i in range(1, 6)) == dks.dks_poisson_model_bytes(p, 0)
        ws = dks.dks_poisson_workspace_bytes(p)
        assert ws >= 3 * a + g + 8 * nx * ny * nz
        assert dks.dks_poisson_launches_per_solve(p) >= 1
        with pytest.raises(dks.DksError) as e:
            dks.dks_poisson_set_spacing(p, 0.0, 1.0, 1.0)
        assert e.value.status == dks.DKS_ERR_INVALID_ARG
        with pytest.raises(dks.DksError):
            dks.dks_poisson_set_g0(p, float("inf"))
        with pytest.raises(dks.DksError):
            dks.dks_poisson_set_workspace(p, 0, 1 << 40)                       # NULL workspace
        with pytest.raises(dks.DksError) as e:
            dks.dks_poisson_solve(p, 256, 512, None)                           # before greens_setup
        assert e.value.status == dks.DKS_ERR_NOT_SETUP
    finally:
        dks.dks_poisson_plan_destroy(p)
    dks.dks_poisson_plan_destroy(None)                                         # NULL is allowed


def test_no_cpu_fallback_without_gpu(dks):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    p = dks.dks_poisson_plan_create(16, 16, 16, 1e-3, 1e-3, 1e-3)
    try:
        with pytest.raises(dks.DksError) as e:
            dks.dks_greens_setup(p)
        assert e.value.status in (dks.DKS_ERR_CUDA, dks.DKS_ERR_UNSUPPORTED_DEVICE)
    finally:
        dks.dks_poisson_plan_destroy(p)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1509_07685_b200")
    pat = re.compile(r"^\s*(from|import)\s+\.*oracle|liboracle|poisson_oracle|#include\s+\".*oracle", re.M)
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not pat.search(src), f"{f} reaches into oracle/"


def test_host_only_plan_options(dks):
    """Slab size and batch size are host-side plan state: workspace sizes and launch counts follow."""
    nx, ny, nz = 256, 128, 64
    p = dks.dks_poisson_plan_create(nx, ny, nz, 1e-4, 1e-4, 1e-4)
    try:
        a = 16 * nx * ny * (nz + 1)
        ws1 = dks.dks_poisson_workspace_bytes(p)
        assert dks.dks_poisson_slab_planes(p) == nz + 1 and dks.dks_poisson_launches_per_solve(p) == 5
        # slabs of 13 planes: B shrinks to one slab, P2-P4 are launched once per slab
        dks.dks_poisson_set_slab_planes(p, 13)
        assert dks.dks_poisson_slab_planes(p) == 13
        assert dks.dks_poisson_launches_per_solve(p) == 2 + 3 * 5
        assert ws1 - dks.dks_poisson_workspace_bytes(p) >= 2 * a * (nz + 1 - 13) // (nz + 1) - 4096
        dks.dks_poisson_set_slab_planes(p, 0)                                   # automatic again
        assert dks.dks_poisson_workspace_bytes(p) == ws1
        with pytest.raises(dks.DksError):
            dks.dks_poisson_set_slab_planes(p, nz + 2)
        # batches: A and B scale with the batch size
        dks.dks_poisson_set_max_batch(p, 4)
        assert dks.dks_poisson_workspace_bytes(p) - ws1 >= 3 * 3 * a - 4096
        with pytest.raises(dks.DksError):
            dks.dks_poisson_set_max_batch(p, 0)
        dks.dks_poisson_set_max_batch(p, 1)
    finally:
        dks.dks_poisson_plan_destroy(p)
    q = dks.dks_poisson_plan_create(128, 128, 128, 1e-4, 1e-4, 1e-4)
    try:
        assert [dks.dks_poisson_pass_name(q, i) for i in range(1, 6)] == [
            "p1_z_r2c_r16p", "p2_y_fwd_r16p", "p3_x_conv_r16", "p4_y_inv_r16", "p5_z_c2r_r16"]   # n = 128: one CTA per parity
    finally:
        dks.dks_poisson_plan_destroy(q)


def test_host_staging_and_shard_options(dks):
    """The host-path staging meshes are optional; sharded plans carry none and refuse batches and slabs."""
    nx, ny, nz = 64, 64, 32
    mesh = 8 * nx * ny * nz
    p = dks.dks_poisson_plan_create(nx, ny, nz, 1e-4, 1e-4, 1e-4)
    try:
        ws = dks.dks_poisson_workspace_bytes(p)
        dks.dks_poisson_set_host_staging(p, False)
        assert ws - dks.dks_poisson_workspace_bytes(p) == 3 * mesh              # three staging meshes (already 256-byte multiples)
        dks.dks_poisson_set_host_staging(p, True)
        assert dks.dks_poisson_workspace_bytes(p) == ws
        dks.dks_poisson_set_host_staging(p, False)
        dks.dks_poisson_set_shard(p, 1, 2)                                      # rank 1 of 2: A1 + A2 + Ghat + B(local planes)
        a1, a2 = 16 * nx * ny * (nz // 2 + 1), 16 * nx * (ny // 2) * (nz + 1)
        ghat = 8 * ((nx + 1 + 7) // 8 * 8) * (ny + 1) * (nz + 1)
        expect = a1 + a2 + ghat + 2 * a1
        assert 0 <= dks.dks_poisson_workspace_bytes(p) - expect <= 4 * 256
        dks.dks_poisson_set_host_staging(p, True)                               # no staging on a sharded plan either way
        assert 0 <= dks.dks_poisson_workspace_bytes(p) - expect <= 4 * 256
        before = dks.dks_poisson_workspace_bytes(p)
        for call in (lambda: dks.dks_poisson_set_max_batch(p, 2), lambda: dks.dks_poisson_set_slab_planes(p, 4)):
            with pytest.raises(dks.DksError) as e:
                call()
            assert e.value.status == dks.DKS_ERR_INVALID_ARG and "sharding excludes" in str(e.value)
        assert dks.dks_poisson_workspace_bytes(p) == before
        dks.dks_poisson_set_max_batch(p, 1)                                     # the default stays acceptable
        for t1, t2 in [([1, 2], [1]), ([1], [1]), ([1] * 9, [1] * 9)]:          # table lengths are checked before the C call
            with pytest.raises(ValueError):
                dks.dks_poisson_set_peers(p, t1, t2)
    finally:
        dks.dks_poisson_plan_destroy(p)
    q = dks.dks_poisson_plan_create(16, 16, 16, 1e-3, 1e-3, 1e-3)               # the smallest extent a sharded solve takes
    try:
        dks.dks_poisson_set_shard(q, 0, 2)
    finally:
        dks.dks_poisson_plan_destroy(q)

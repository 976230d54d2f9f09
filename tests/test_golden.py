"""Stored sampled values (tests/golden/, written by tests/golden/make_golden.py from oracle/ only).

Direct summation of Eq. (2) at 73 nodes of every BASELINE.json config, beside the
long-double oracle's value.  Checks (a) the stored pair agrees (pins the oracle at full scale,
including the 256^3 config, with no FFT on the reference side), (b) the inputs regenerate
bit-identically and the direct sum reproduces the stored value on the configs that are cheap to redo.
"""
import os

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))


def load(ci):
    a = np.loadtxt(os.path.join(HERE, "golden", f"sampled_phi_cfg{ci}.txt"))
    return a[:, :3].astype(np.int64), a[:, 3], a[:, 4]


@pytest.mark.parametrize("ci", [1, 2, 3, 4, 5])
def test_golden_oracle_vs_direct_sum(ci):
    nodes, direct, orc = load(ci)
    assert len(nodes) == 73
    assert np.max(np.abs(orc - direct) / np.abs(direct)) <= 1e-13


@pytest.mark.parametrize("ci", [1, 2, 3])
def test_golden_reproducible(oracle, workloads, ci):
    w = workloads.config(ci)
    nodes, direct, _ = load(ci)
    assert np.array_equal(nodes, workloads.sample_nodes(w.n, w.seed))
    rho = workloads.make_rho(w)
    again = oracle.direct_sum_nodes(rho, w.n, w.h, nodes)
    assert np.max(np.abs(again - direct) / np.abs(direct)) <= 1e-15

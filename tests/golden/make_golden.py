"""Writes tests/golden/sampled_phi_cfg{1..5}.txt.  Calls ONLY oracle/ and the input generator.

    python tests/golden/make_golden.py

The paper prints no numerical phi values for the Poisson path (Table 1, is wall
clock only), so there is no paper-printed fixture.  What is stored instead, per BASELINE.json config:
the definition of the result, Eq. (2), summed directly in long double at 73 seeded
output nodes (64 random + 8 corners + centre), beside the long-double oracle's value at the same nodes.
Columns: i j k  phi_direct_sum[V]  phi_oracle_ld[V]   (17 significant digits).
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import oracle as O                        # noqa: E402
from paper_1509_07685_b200 import workloads as W      # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))


def main():
    for ci in range(1, 6):
        w = W.config(ci)
        rho = W.make_rho(w)
        nodes = W.sample_nodes(w.n, w.seed)
        direct = O.direct_sum_nodes(rho, w.n, w.h, nodes, precision="ld")
        phi = O.solve(rho, w.n, w.h, precision="ld")
        got = phi[nodes[:, 2], nodes[:, 1], nodes[:, 0]]
        path = os.path.join(HERE, f"sampled_phi_cfg{ci}.txt")
        with open(path, "w") as f:
            f.write(f"# {w.name}: n={w.n} h={w.h} seed={w.seed} g0=G(min(h)/2)\n")
            f.write("# Eq. (2), PAPER.md:121 (section 3.1.1), direct long-double summation vs oracle_ld; written by make_golden.py\n")
            f.write("# i j k phi_direct_sum phi_oracle_ld\n")
            for (i, j, k), a, b in zip(nodes, direct, got):
                f.write(f"{i} {j} {k} {a:.17e} {b:.17e}\n")
        print(path, float(np.max(np.abs(got - direct) / np.abs(direct))))


if __name__ == "__main__":
    main()

"""B200-native (sm_100a) open-boundary FFT Poisson solver after arXiv:1509.07685 (DKS, part 1).

`paper_1509_07685_b200.dks` binds the C ABI declared in include/dks_poisson.h (loads the CUDA
library; raises if it is missing).  `paper_1509_07685_b200.workloads` is the seeded input
generator (numpy only) and imports nothing else, so importing this package stays cheap.
"""
__all__ = ["dks", "workloads", "build"]

"""Independent checking code for the GPU tests: plain torch FP64 (checking only).  It lives in the package
(`paper_2409_01712_b200/checks.py`) so that `bench.py` can report the same invariants without importing from tests/."""
from paper_2409_01712_b200.checks import (LowerTiles, factor_matvec, fro_norm_sym, probe_backward_error,  # noqa: F401
                                          solve_residual, sym_matvec)

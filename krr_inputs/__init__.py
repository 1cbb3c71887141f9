"""Seeded synthetic inputs shared by the oracle tests and the CUDA path's tests/bench.

Holds none of the method's arithmetic (no Cholesky, no rounding, no precision rule): only the
counter-based genotype / phenotype generators and the Gaussian-kernel Build step (Alg. 2,
Alg. 5), which is upstream of the hot path and here only produces its input A = K + lambda*I.
"""
from .synth import (CONFIGS, Config, genotypes, kernel_matrix, phenotypes, make_problem,
                    exact_lower_factor, scaled_config, make_problem_lower_tiles,
                    kernel_matrix_lower_tiles)

__all__ = ["CONFIGS", "Config", "genotypes", "kernel_matrix", "phenotypes", "make_problem",
           "exact_lower_factor", "scaled_config", "make_problem_lower_tiles", "kernel_matrix_lower_tiles"]

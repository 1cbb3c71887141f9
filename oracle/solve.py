"""Triangular solves with the tile factor: W <- Solve(K~, P_h) (oracle; test infrastructure).

Alg. 3 l.5: with K + lambda*I = L L^T, solve L Z = Y then L^T alpha = Z -- "forward and
backward substitution operations".  Written per tile: the diagonal tile by a
triangular solve (`scipy.linalg.solve_triangular` as the library step), the off-diagonal tiles by
matrix products, in FP64.  L is the dequantised factor (dense float64).
"""
import numpy as np
from scipy.linalg import solve_triangular


def potrs_fp64(L, Y, nb):
    """alpha = (L L^T)^{-1} Y by tile forward/backward substitution in FP64."""
    L = np.asarray(L, dtype=np.float64)
    n = L.shape[0]
    assert n % nb == 0
    NT = n // nb
    Z = np.array(Y, dtype=np.float64, copy=True)
    if Z.ndim == 1:
        Z = Z[:, None]
    # forward: Z_k = L_kk^{-1} (Y_k - sum_{j<k} L_kj Z_j)
    for k in range(NT):
        r0, r1 = k * nb, (k + 1) * nb
        Z[r0:r1] -= L[r0:r1, :r0] @ Z[:r0]
        Z[r0:r1] = solve_triangular(L[r0:r1, r0:r1], Z[r0:r1], lower=True, check_finite=False)
    # backward: alpha_k = L_kk^{-T} (Z_k - sum_{i>k} L_ik^T alpha_i)
    for k in range(NT - 1, -1, -1):
        r0, r1 = k * nb, (k + 1) * nb
        Z[r0:r1] -= L[r1:, r0:r1].T @ Z[r1:]
        Z[r0:r1] = solve_triangular(L[r0:r1, r0:r1], Z[r0:r1], lower=True, trans="T",
                                    check_finite=False)
    return Z


def solve_fp64(A, Y, nb):
    """alpha = A^{-1} Y through the FP64 tile Cholesky (the reference alpha of north_star)."""
    from .cholesky import tile_cholesky_fp64
    L, info = tile_cholesky_fp64(A, nb)
    if info:
        raise np.linalg.LinAlgError(f"matrix not positive definite (info={info})")
    return potrs_fp64(L, Y, nb)

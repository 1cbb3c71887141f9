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


def refine(A, L, Y, alpha, nb, steps, round_fp32=True):
    """Iterative refinement with a fixed (mixed-precision) factor: for s = 0 .. steps-1
         r_s = Y - A alpha_s,   alpha_{s+1} = alpha_s + (L L^T)^{-1} r_s.
    The paper names the technique ("mixed-precision techniques have been made popular with iterative
    refinement ... recovers all digits of accuracy") and does not adopt it; SURVEY section 8(c) offers it as the remedy
    for the alpha tolerance under FP16 / FP8 maps (R19).  With round_fp32 the residual and the iterate are
    rounded to FP32 where the method stores them (r_s after the FP64 evaluation, alpha_{s+1} after the update); the
    correction itself is solved in FP64.  Returns (alpha_steps, [||r_0||_F, ..., ||r_steps||_F]), the norms taken of
    the residuals as stored."""
    A = np.asarray(A, dtype=np.float64)
    Y = np.asarray(Y, dtype=np.float64)
    x = np.array(alpha, dtype=np.float64, copy=True)
    if x.ndim == 1:
        x = x[:, None]
    if Y.ndim == 1:
        Y = Y[:, None]
    rnd = (lambda v: v.astype(np.float32).astype(np.float64)) if round_fp32 else (lambda v: v)
    norms = []
    for _ in range(steps):
        r = rnd(Y - A @ x)
        norms.append(float(np.linalg.norm(r)))
        x = rnd(x + potrs_fp64(L, r, nb))
    norms.append(float(np.linalg.norm(rnd(Y - A @ x))))
    return x, norms

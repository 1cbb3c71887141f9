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


def pcg(A, L, Y, alpha, nb, iters, round_fp32=True):
    """Conjugate gradients on A alpha = Y preconditioned by the fixed factor, M = L L^T (the textbook method of
    Hestenes and Stiefel with a preconditioner, every right-hand side on its own), started from `alpha`:
         r_0 = Y - A alpha_0,  z_0 = M^{-1} r_0,  p_0 = z_0,  rho_0 = r_0 . z_0
         q_k = A p_k,  a_k = rho_k / (p_k . q_k),  alpha_{k+1} = alpha_k + a_k p_k,  r_{k+1} = r_k - a_k q_k,
         z_{k+1} = M^{-1} r_{k+1},  rho_{k+1} = r_{k+1} . z_{k+1},  p_{k+1} = z_{k+1} + (rho_{k+1} / rho_k) p_k.
    The stationary iteration of `refine` contracts only while the spectral radius of I - M^{-1} A is below one, which
    an FP16 map loses at C4's size (R20); CG with the same M converges for every SPD A and M, at the same
    cost per step (one product with A, one solve with L).  With round_fp32 the quantities the method keeps in FP32
    are rounded there: the right-hand side of the solve with L, the direction p, the returned alpha; everything else
    is FP64.  A column with p.q <= 0 or rho = 0 stops moving (a = 0, new direction z).  Returns (alpha_iters,
    [||r_0||_F, ..., ||r_iters||_F]) with r_k the recursively updated residuals."""
    A = np.asarray(A, dtype=np.float64)
    Y = np.asarray(Y, dtype=np.float64)
    x = np.array(alpha, dtype=np.float64, copy=True)
    if x.ndim == 1:
        x = x[:, None]
    if Y.ndim == 1:
        Y = Y[:, None]
    rnd = (lambda v: v.astype(np.float32).astype(np.float64)) if round_fp32 else (lambda v: v)
    r = Y - A @ x
    z = potrs_fp64(L, rnd(r), nb)
    p = rnd(z)
    rho = np.sum(r * z, axis=0)
    norms = [float(np.linalg.norm(r))]
    for _ in range(iters):
        q = A @ p
        pq = np.sum(p * q, axis=0)
        a = np.where(pq > 0.0, rho / np.where(pq > 0.0, pq, 1.0), 0.0)
        x = x + a[None, :] * p
        r = r - a[None, :] * q
        norms.append(float(np.linalg.norm(r)))
        z = potrs_fp64(L, rnd(r), nb)
        rho_new = np.sum(r * z, axis=0)
        b = np.where(rho > 0.0, rho_new / np.where(rho > 0.0, rho, 1.0), 0.0)
        p = rnd(z + b[None, :] * p)
        rho = rho_new
    return rnd(x), norms

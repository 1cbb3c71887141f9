"""Tile Cholesky of A = K + lambda*I: FP64 reference and emulated-precision mosaic (oracle).

TEST INFRASTRUCTURE.  Follows Alg. 3 l.3 `K~ <- FACTORIZE(K + alpha*Id)` with the tile
algorithm the paper names but does not print -- POTRF on the diagonal tile, triangular solves on the
panel, symmetric rank-k and matrix-matrix updates -- written per tile column k:

    S_kk = A_kk - sum_{j<k} L_kj L_kj^T          (SYRK)
    L_kk = chol(S_kk)                            (POTRF)
    S_ik = A_ik - sum_{j<k} L_ij L_kj^T , i > k  (GEMM)
    L_ik = S_ik L_kk^{-T}                        (TRSM)

`numpy.matmul` and `scipy.linalg.solve_triangular` serve as the GEMM and TRSM steps; the POTRF step
is written out (`chol_unblocked`).  No blocking or reordering beyond this definition.

The emulated version stores tile (i,j) in precision pmap[i,j] ("a tiled mosaic of
precisions embedded in a single stored copy of the matrix") with the rounding points of DESIGN.md:
R3 (A is rounded on entry), R4 (a tile is rounded once, when its final value is
stored), R5 (operands are used as stored), R6 (power-of-two FP8 tile scale), R8 (diagonal FP32),
R10 (TRSM in >= FP32, then round), R11 (breakdown -> info, LAPACK convention).
"""
import math

import numpy as np
from scipy.linalg import solve_triangular

from .rounding import FP32, FP16, FP8, quantise_tile, rd_fp32


def chol_scalar(A):
    """Textbook scalar Cholesky (Cholesky-Banachiewicz), pure Python, for n <= 64 brute-force pins.

    L_jj = sqrt(A_jj - sum_{l<j} L_jl^2);  L_ij = (A_ij - sum_{l<j} L_il L_jl) / L_jj, i > j.
    Only the lower triangle of A is referenced.
    """
    n = len(A)
    L = [[0.0] * n for _ in range(n)]
    for j in range(n):
        s = float(A[j][j])
        for l in range(j):
            s -= L[j][l] * L[j][l]
        if not s > 0.0:
            raise np.linalg.LinAlgError(f"non-positive pivot at column {j + 1}")
        L[j][j] = math.sqrt(s)
        for i in range(j + 1, n):
            s = float(A[i][j])
            for l in range(j):
                s -= L[i][l] * L[j][l]
            L[i][j] = s / L[j][j]
    return np.array(L, dtype=np.float64)


def chol_unblocked(S):
    """POTRF of one tile in FP64, column by column (same recurrences as chol_scalar, vectorised
    over the rows of a column).  Returns (L, info): info = 0, or the 1-based column of the first
    non-positive pivot (then L is valid only left of it)."""
    S = np.asarray(S, dtype=np.float64)
    n = S.shape[0]
    L = np.zeros((n, n), dtype=np.float64)
    for j in range(n):
        d = S[j, j] - np.dot(L[j, :j], L[j, :j])
        if not d > 0.0:
            return L, j + 1
        d = math.sqrt(d)
        L[j, j] = d
        if j + 1 < n:
            L[j + 1:, j] = (S[j + 1:, j] - L[j + 1:, :j] @ L[j, :j]) / d
    return L, 0


def _trsm_right_lower_trans(S, Lkk):
    """X = S Lkk^{-T}  (X Lkk^T = S), the panel TRSM."""
    return solve_triangular(Lkk, S.T, lower=True, trans="N", check_finite=False).T


def tile_cholesky_fp64(A, nb):
    """FP64 tile Cholesky of the symmetric positive definite A (lower triangle referenced).

    Returns (L, info).  L is dense n x n float64, zero above the diagonal."""
    A = np.asarray(A)
    n = A.shape[0]
    assert A.shape == (n, n) and n % nb == 0
    NT = n // nb
    L = np.zeros((n, n), dtype=np.float64)
    for k in range(NT):
        r0, r1 = k * nb, (k + 1) * nb
        Lrow = L[r0:r1, :r0]
        S = np.asarray(A[r0:r1, r0:r1], dtype=np.float64) - Lrow @ Lrow.T
        Lkk, info = chol_unblocked(S)
        if info:
            return L, r0 + info
        L[r0:r1, r0:r1] = Lkk
        if r1 < n:
            Spanel = np.asarray(A[r1:, r0:r1], dtype=np.float64) - L[r1:, :r0] @ Lrow.T
            L[r1:, r0:r1] = _trsm_right_lower_trans(Spanel, Lkk)
    return L, 0


def _operand_for(X, p_stored, p_task):
    """Operand tile of a task that runs in precision p_task (literal reading of PAPER.md:206: "conversion at
    the sender (lower precision needed at the receiver) or at the receiver (higher)"): a tile stored in a
    higher precision than the task's is rounded DOWN to it (lossy; FP8 with the scale of its own amax),
    a tile stored in the same or a lower precision is used exactly (up-conversion is exact)."""
    if p_task > p_stored:                      # codes grow as the precision falls: FP32 = 0 < FP16 = 1 < FP8 = 2
        return quantise_tile(X, p_task)[0]
    return X


def tile_cholesky_emulated(A, nb, pmap, preround_a=True, operands="as_stored"):
    """Emulated mixed-precision tile Cholesky.

    A     : n x n, FP32 values (any float dtype holding them); lower triangle referenced.
    pmap  : NT x NT precision codes (oracle.rounding.FP32/FP16/FP8), lower triangle used,
            diagonal must be FP32.
    Returns (Lhat, scales, info):
      Lhat   dense float64 holding the DEQUANTISED factor (value = scale * payload for FP8 tiles),
      scales NT x NT float64 (1.0 except FP8 tiles),
      info   0, or the 1-based scalar column of the first non-positive pivot (tiles of later
             columns are then not computed).

    Steps:
      3. Ahat_ij = rd_{p(i,j)}(A_ij) if preround_a else A_ij           (i > j; diagonal is FP32)
      4. S_kk = A_kk - sum_{j<k} Lhat_kj Lhat_kj^T ;  Lhat_kk = rd32(chol(rd32(S_kk)))
         S_ik = Ahat_ik - sum_{j<k} Lhat_ij Lhat_kj^T ;  T_ik = S_ik Lhat_kk^{-T} ;
         Lhat_ik = rd_{p(i,k)}(T_ik)            -- each tile rounded once, on its final store
      5. operands="as_stored" (default, reading R5): operands are used as stored (up-conversion exact);
         operands="to_updated" (the paper's literal rule): every SYRK / GEMM task runs in the
         precision of the tile it updates, S_ik -= cv(Lhat_ij) cv(Lhat_kj)^T with cv = _operand_for(., p(.), p(i,k))
         (down-conversion of a higher-precision operand is lossy); identical to the default on uniform maps
      6. FP8 tiles: power-of-two scale from the tile's amax
    Arithmetic between roundings is FP64.
    """
    A = np.asarray(A)
    n = A.shape[0]
    assert A.shape == (n, n) and n % nb == 0
    NT = n // nb
    pmap = np.asarray(pmap)
    assert operands in ("as_stored", "to_updated")
    Lh = np.zeros((n, n), dtype=np.float64)
    scales = np.ones((NT, NT), dtype=np.float64)

    def product_sum(i, k, p_task):
        """sum_{j<k} op(Lhat_ij) op(Lhat_kj)^T for the task that updates tile (i, k)."""
        if operands == "as_stored":
            return Lh[i * nb:(i + 1) * nb, :k * nb] @ Lh[k * nb:(k + 1) * nb, :k * nb].T
        acc = np.zeros((nb, nb), dtype=np.float64)
        for j in range(k):
            a = _operand_for(Lh[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb], int(pmap[i, j]), p_task)
            b = _operand_for(Lh[k * nb:(k + 1) * nb, j * nb:(j + 1) * nb], int(pmap[k, j]), p_task)
            acc += a @ b.T
        return acc

    for k in range(NT):
        assert pmap[k, k] == FP32, "diagonal tiles are FP32 (PAPER.md:229, reading R8)"
        r0, r1 = k * nb, (k + 1) * nb
        S = np.asarray(A[r0:r1, r0:r1], dtype=np.float64) - product_sum(k, k, FP32)
        Lkk, info = chol_unblocked(rd_fp32(S))
        if info:
            return Lh, scales, r0 + info
        Lkk = rd_fp32(Lkk)
        Lh[r0:r1, r0:r1] = Lkk
        for i in range(k + 1, NT):
            i0, i1 = i * nb, (i + 1) * nb
            p = int(pmap[i, k])
            Aik = np.asarray(A[i0:i1, r0:r1], dtype=np.float64)
            if preround_a:
                Aik, _ = quantise_tile(Aik, p)
            Sik = Aik - product_sum(i, k, p)
            Tik = _trsm_right_lower_trans(Sik, Lkk)
            Lh[i0:i1, r0:r1], scales[i, k] = quantise_tile(Tik, p)
    return Lh, scales, 0


def backward_error(A, L):
    """||A - L L^T||_F / ||A||_F over the full symmetric matrix (A given by its lower triangle)."""
    A = np.asarray(A, dtype=np.float64)
    Asym = np.tril(A) + np.tril(A, -1).T
    R = Asym - L @ L.T
    return float(np.linalg.norm(R) / np.linalg.norm(Asym))

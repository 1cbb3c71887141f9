"""Tile-centric adaptive precision map (oracle; test infrastructure).

PAPER.md:192 ("tile-centric adaptive precision [19] resulting in a tiled mosaic of precisions"),
PAPER.md:215 ("The Associate phase starts with adaptive precision to lower the precision of the
off-diagonal tiles depending on the accuracy threshold, as explained in [20]") and PAPER.md:229
(diagonal tiles stay in the highest precision; each other tile gets "the lowest numerically
appropriate supported datatype").  The paper prints no formula; the rule below is the text of
BASELINE.json's north_star (reading R1):

    tile (i,j), i > j, gets the LOWEST allowed precision p with
        ||A_ij||_F * u_p  <=  eps_target * ||A||_F / NT ,
    FP32 if none qualifies; diagonal tiles are FP32.

u_p are unit roundoffs 2^-24 / 2^-11 / 2^-4 (reading R2); ||A||_F is that of the full symmetric
matrix, so off-diagonal tiles count twice; NT = n / nb tiles per dimension.
"""
import numpy as np

from .rounding import FP32, FP16, FP8, UNIT_ROUNDOFF


def tile_norms(A, nb):
    """t[i,j] = ||A_ij||_F for i >= j (0 elsewhere), accumulated in FP64.  Only the lower
    triangle of tiles is read; diagonal tiles are read as full squares (A is symmetric)."""
    n = A.shape[0]
    assert A.shape == (n, n) and n % nb == 0
    NT = n // nb
    t = np.zeros((NT, NT), dtype=np.float64)
    for i in range(NT):
        for j in range(i + 1):
            blk = np.asarray(A[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb], dtype=np.float64)
            t[i, j] = np.sqrt(np.sum(blk * blk))
    return t


def frobenius_from_tile_norms(t):
    """||A||_F^2 = sum_i t_ii^2 + 2 sum_{i>j} t_ij^2 (symmetric matrix, lower tiles stored)."""
    d = np.diag(t)
    off = np.tril(t, -1)
    return float(np.sqrt(np.sum(d * d) + 2.0 * np.sum(off * off)))


def precision_map(A, nb, eps_target, allowed=(FP32, FP16, FP8)):
    """Return (pmap uint8 NTxNT, tile norms float64 NTxNT, ||A||_F).

    pmap[i,j] is defined for i >= j; entries above the diagonal are set to 255 (unused).
    `eps_target` is taken at the precision the C ABI passes it in (a C float widened to double).
    """
    t = tile_norms(A, nb)
    NT = t.shape[0]
    fro = frobenius_from_tile_norms(t)
    eps = float(np.float32(eps_target))
    rhs = eps * fro / NT
    pmap = np.full((NT, NT), 255, dtype=np.uint8)
    lowest_first = [p for p in (FP8, FP16, FP32) if p in allowed]
    for i in range(NT):
        pmap[i, i] = FP32
        for j in range(i):
            chosen = FP32
            for p in lowest_first:
                if t[i, j] * UNIT_ROUNDOFF[p] <= rhs:
                    chosen = p
                    break
            pmap[i, j] = chosen
    return pmap, t, fro


def uniform_map(NT, offdiag):
    """All off-diagonal tiles `offdiag`, diagonal FP32 (the maps of PAPER.md:248, :260)."""
    pmap = np.full((NT, NT), 255, dtype=np.uint8)
    for i in range(NT):
        pmap[i, :i] = offdiag
        pmap[i, i] = FP32
    return pmap


def band_map(NT, fp32_fraction, low):
    """The hand-tuned band technique of [37] the paper compares with ("applies a given precision on each
    band of the off-diagonal tiles"; "100%, 80%, ... 10% FP32 ... the remaining off-diagonal tiles in FP16").
    Reading (R18): the first b = ceil(fp32_fraction * (NT - 1)) sub-diagonals of tiles are FP32, the tiles
    further from the diagonal are `low`; the diagonal tiles are always FP32."""
    b = int(np.ceil(float(fp32_fraction) * (NT - 1) - 1e-12))
    pmap = np.full((NT, NT), 255, dtype=np.uint8)
    for i in range(NT):
        for j in range(i + 1):
            pmap[i, j] = FP32 if i - j <= b else low
    return pmap


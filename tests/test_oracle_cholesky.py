"""Pins for the oracle's FP64 tile Cholesky and its emulated-precision mosaic (oracle/cholesky.py).

Nothing in PAPER.md prints a number for this path (no worked example, no error bound), so the pins
are mathematical: closed-form factors, brute force, LAPACK, invariants, and constructions on which
every rounding is exact so that the emulated oracle must return a known factor bit for bit.
"""
import numpy as np
import pytest

from oracle import cholesky as C
from oracle import rounding as R
from oracle.precision_map import uniform_map
from krr_inputs import exact_lower_factor


def spd(n, seed):
    rng = np.random.default_rng(seed)
    B = rng.standard_normal((n, n))
    return B @ B.T + n * np.eye(n)


# ---------------------------------------------------------------- hand cases ------------------
def test_hand_2x2():
    A = np.array([[4.0, 2.0], [2.0, 5.0]])
    L, info = C.tile_cholesky_fp64(A, 1)
    assert info == 0 and np.array_equal(L, np.array([[2.0, 0.0], [1.0, 2.0]]))


def test_hand_3x3():
    # classic: A = L L^T with L = [[2,0,0],[6,1,0],[-8,5,3]]
    A = np.array([[4.0, 12.0, -16.0], [12.0, 37.0, -43.0], [-16.0, -43.0, 98.0]])
    want = np.array([[2.0, 0, 0], [6.0, 1.0, 0], [-8.0, 5.0, 3.0]])
    for nb in (1, 3):
        L, info = C.tile_cholesky_fp64(A, nb)
        assert info == 0 and np.array_equal(L, want)
    assert np.array_equal(C.chol_scalar(A), want)


# ---------------------------------------------------------------- closed forms ----------------
@pytest.mark.parametrize("n,nb", [(12, 3), (64, 16), (96, 32)])
def test_diagonal_matrix(n, nb):
    d = np.arange(1, n + 1, dtype=np.float64) ** 2
    L, info = C.tile_cholesky_fp64(np.diag(d), nb)
    assert info == 0 and np.array_equal(L, np.diag(np.arange(1, n + 1, dtype=np.float64)))


@pytest.mark.parametrize("n,nb", [(24, 4), (60, 12), (128, 32)])
def test_lehmer_matrix(n, nb):
    i = np.arange(1, n + 1, dtype=np.float64)
    A = np.minimum.outer(i, i) / np.maximum.outer(i, i)
    want = np.tril(np.sqrt(2 * i[None, :] - 1) / i[:, None])       # L_ij = sqrt(2j-1)/i
    L, info = C.tile_cholesky_fp64(A, nb)
    assert info == 0
    assert np.max(np.abs(L - want)) < 1e-13


@pytest.mark.parametrize("n,nb", [(16, 4), (64, 8)])
def test_min_matrix_gives_all_ones(n, nb):
    i = np.arange(1, n + 1, dtype=np.float64)
    L, info = C.tile_cholesky_fp64(np.minimum.outer(i, i), nb)
    assert info == 0 and np.array_equal(L, np.tril(np.ones((n, n))))


@pytest.mark.parametrize("n,nb,c,d", [(32, 8, 0.48, 0.53), (120, 24, 0.26, 0.84)])
def test_equicorrelation_closed_form(n, nb, c, d):
    # A = c 11^T + d I (the mean structure of the configs' K + lambda I):
    # c_0 = c, c_j = 1/(1/c + j/d);  L_jj = sqrt(c_{j-1} + d), L_ij = c_{j-1}/L_jj  (1-based j)
    A = c * np.ones((n, n)) + d * np.eye(n)
    j = np.arange(n, dtype=np.float64)
    cj = 1.0 / (1.0 / c + j / d)
    diag = np.sqrt(cj + d)
    want = np.tril(np.broadcast_to(cj / diag, (n, n)), -1) + np.diag(diag)
    L, info = C.tile_cholesky_fp64(A, nb)
    assert info == 0 and np.max(np.abs(L - want)) < 1e-14


@pytest.mark.parametrize("n,nb,rho", [(40, 8, 0.5), (64, 16, -0.3)])
def test_kac_murdock_szego(n, nb, rho):
    i = np.arange(n)
    A = rho ** np.abs(np.subtract.outer(i, i)).astype(np.float64)
    want = np.tril(rho ** np.subtract.outer(i, i).clip(0).astype(np.float64)) * np.sqrt(1 - rho * rho)
    want[:, 0] = rho ** i.astype(np.float64)
    L, info = C.tile_cholesky_fp64(A, nb)
    assert info == 0 and np.max(np.abs(L - want)) < 1e-14


# ---------------------------------------------------------------- brute force / LAPACK --------
@pytest.mark.parametrize("n", [1, 2, 6, 24, 48, 64])
def test_brute_force_every_tile_size(n):
    A = spd(n, n)
    want = C.chol_scalar(A)
    for nb in [b for b in range(1, n + 1) if n % b == 0]:
        L, info = C.tile_cholesky_fp64(A, nb)
        assert info == 0
        assert np.max(np.abs(L - want)) <= 1e-13 * np.max(np.abs(want)), nb


@pytest.mark.parametrize("n,nb", [(256, 64), (384, 128), (512, 32)])
def test_against_lapack_and_invariants(n, nb):
    A = spd(n, 7)
    L, info = C.tile_cholesky_fp64(A, nb)
    assert info == 0
    assert np.array_equal(L, np.tril(L)) and np.all(np.diag(L) > 0)
    want = np.linalg.cholesky(A)
    assert np.max(np.abs(L - want)) < 1e-11 * np.max(np.abs(want))
    assert C.backward_error(A, L) < 1e-15 * np.sqrt(n) * 4


def test_only_lower_triangle_is_referenced():
    A = spd(48, 3)
    junk = np.tril(A) + np.triu(np.full_like(A, 1e9), 1)
    L1, _ = C.tile_cholesky_fp64(A, 16)
    L2, _ = C.tile_cholesky_fp64(junk, 16)
    assert np.array_equal(L1, L2)
    Lh, _, info = C.tile_cholesky_emulated(junk.astype(np.float32), 16, uniform_map(3, R.FP16))
    assert info == 0 and np.all(np.isfinite(Lh))


def test_breakdown_reports_lapack_info():
    A = spd(32, 5)
    A[20, 20] = -1.0                                    # first non-positive pivot at column 21
    L, info = C.tile_cholesky_fp64(A, 8)
    assert info == 21
    with pytest.raises(np.linalg.LinAlgError):
        np.linalg.cholesky(A)
    _, _, info_e = C.tile_cholesky_emulated(A.astype(np.float32), 8, uniform_map(4, R.FP32))
    assert info_e == 21


# ---------------------------------------------------------------- emulated mosaic -------------
@pytest.mark.parametrize("prec", [R.FP32, R.FP16, R.FP8])
@pytest.mark.parametrize("n,nb", [(128, 32), (512, 64)])
def test_exactly_representable_construction_is_reproduced_bit_for_bit(prec, n, nb):
    # L0 sparse with entries in {0, +-1/2, +-1, +-2}, power-of-two diagonal: every product, sum,
    # quotient and rounding of the factorisation is exact, so any map must return L0 itself.
    # (A's own entries are not E4M3 numbers, hence preround_a=False for FP8 -- DESIGN.md.)
    L0, A = exact_lower_factor(11, n, nb)
    L0 = L0.numpy()
    Lh, scales, info = C.tile_cholesky_emulated(A.numpy(), nb, uniform_map(n // nb, prec),
                                                preround_a=(prec != R.FP8))
    assert info == 0
    assert np.array_equal(Lh, L0)
    if prec == R.FP8:
        off = np.tril(np.ones((n // nb, n // nb)), -1).astype(bool)
        s = scales[off]
        assert np.all(np.log2(s) == np.round(np.log2(s)))       # power-of-two scales
    else:
        assert np.all(scales == 1.0)


def test_mixed_map_on_exact_construction():
    n, nb = 256, 32
    NT = n // nb
    L0, A = exact_lower_factor(5, n, nb)
    rng = np.random.default_rng(0)
    pmap = uniform_map(NT, R.FP32)
    for i in range(NT):
        for j in range(i):
            pmap[i, j] = rng.integers(0, 3)
    Lh, _, info = C.tile_cholesky_emulated(A.numpy(), nb, pmap, preround_a=False)
    assert info == 0 and np.array_equal(Lh, L0.numpy())


def test_all_fp32_map_agrees_with_fp64_to_fp32_accuracy():
    n, nb = 512, 64
    A = spd(n, 9).astype(np.float32)
    L64, _ = C.tile_cholesky_fp64(A, nb)
    Lh, _, info = C.tile_cholesky_emulated(A, nb, uniform_map(n // nb, R.FP32))
    assert info == 0
    rel = np.linalg.norm(Lh - L64) / np.linalg.norm(L64)
    assert rel < 1e-7 * np.sqrt(n)
    assert np.array_equal(Lh, Lh.astype(np.float32).astype(np.float64))    # stored values are FP32


@pytest.mark.parametrize("prec,u", [(R.FP16, 2.0 ** -11), (R.FP8, 2.0 ** -4)])
def test_stored_tiles_are_in_their_format_and_error_scales_with_u(prec, u):
    n, nb = 256, 64
    NT = n // nb
    A = (spd(n, 2) / n).astype(np.float32)
    Lh, scales, info = C.tile_cholesky_emulated(A, nb, uniform_map(NT, prec))
    assert info == 0
    for i in range(NT):
        for j in range(i):
            blk = Lh[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb]
            q, s = R.quantise_tile(blk, prec)
            assert np.array_equal(q, blk)            # idempotent: already in the format
            assert s == scales[i, j] or prec != R.FP8
    be = C.backward_error(A, Lh)
    assert 0.01 * u < be < 2 * u                     # perturbation of the size the format implies


def test_storage_perturbation_bound_of_the_rule():
    # Higham-Mary: rounding tile (i,j) to p perturbs it by <= u_p ||A_ij||_F, so a map produced by
    # the rule satisfies ||Ahat - A||_F <= eps ||A||_F.
    from oracle.precision_map import precision_map
    rng = np.random.default_rng(4)
    n, nb = 256, 32
    NT = n // nb
    A = spd(n, 6) / n
    A *= np.exp(-0.5 * np.abs(np.subtract.outer(np.arange(n), np.arange(n))) / nb)   # decaying tiles
    A = A.astype(np.float32)
    eps = 3e-3
    pmap, t, fro = precision_map(A, nb, eps)
    assert len(set(pmap[np.tril_indices(NT, -1)])) >= 2          # a genuine mosaic
    err2 = 0.0
    for i in range(NT):
        for j in range(i):
            blk = A[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb].astype(np.float64)
            q, _ = R.quantise_tile(blk, int(pmap[i, j]))
            err2 += 2 * np.sum((q - blk) ** 2)
    assert np.sqrt(err2) <= float(np.float32(eps)) * fro

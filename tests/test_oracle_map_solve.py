"""Pins for the precision-map rule and the triangular solves of the oracle.

Map rule: hand-built matrices whose tile norms sit just below / above each threshold, and the
equicorrelation closed form t_ij = c*nb, ||A||_F^2 = n(c+d)^2 + n(n-1)c^2, which makes the rule
degenerate to u_p <= eps (the uniform maps the paper also reports).
Solve: Sherman-Morrison closed form for c 11^T + d I, LAPACK solve, residual.
"""
import numpy as np
import pytest

from oracle import rounding as R
from oracle.cholesky import tile_cholesky_fp64, tile_cholesky_emulated
from oracle.precision_map import precision_map, tile_norms, frobenius_from_tile_norms, uniform_map
from oracle.solve import potrs_fp64, solve_fp64
from krr_inputs import CONFIGS, scaled_config, make_problem


def test_tile_norms_and_symmetric_frobenius():
    rng = np.random.default_rng(0)
    n, nb = 96, 24
    B = rng.standard_normal((n, n))
    A = B + B.T
    t = tile_norms(A, nb)
    for i in range(4):
        for j in range(4):
            blk = A[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb]
            want = np.linalg.norm(blk) if i >= j else 0.0
            assert abs(t[i, j] - want) <= 1e-12 * max(1.0, want)
    assert abs(frobenius_from_tile_norms(t) - np.linalg.norm(A)) < 1e-10


def _block_matrix(NT, nb, norms):
    """Symmetric matrix whose tile (i,j) is constant with Frobenius norm norms[i,j]."""
    n = NT * nb
    A = np.zeros((n, n))
    for i in range(NT):
        for j in range(i + 1):
            A[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb] = norms[i, j] / nb
            A[j * nb:(j + 1) * nb, i * nb:(i + 1) * nb] = norms[i, j] / nb
    return A


def test_rule_thresholds_just_below_and_above():
    NT, nb = 4, 8
    eps = 2.0 ** -13                                 # exactly representable as a C float
    base = np.full((NT, NT), 1.0) + 50.0 * np.eye(NT)   # dominant diagonal fixes ||A||_F
    # choose target norms relative to rhs = eps * fro / NT; iterate once since fro depends on them
    norms = base.copy()
    for _ in range(50):
        A = _block_matrix(NT, nb, norms)
        fro = np.linalg.norm(A)
        rhs = eps * fro / NT
        norms[1, 0] = rhs / 2.0 ** -4 * 0.999        # just qualifies for FP8
        norms[2, 0] = rhs / 2.0 ** -4 * 1.001        # just misses FP8 -> FP16
        norms[2, 1] = rhs / 2.0 ** -11 * 0.999       # just qualifies for FP16
        norms[3, 0] = rhs / 2.0 ** -11 * 1.001       # misses FP16 -> FP32
        norms[3, 1] = rhs / 2.0 ** -11 * 4.0         # far above the FP16 threshold -> FP32
        norms[3, 2] = rhs * 1e-3                     # tiny -> FP8
    A = _block_matrix(NT, nb, norms).astype(np.float64)
    pmap, t, fro = precision_map(A, nb, eps)
    assert pmap[1, 0] == R.FP8 and pmap[2, 0] == R.FP16 and pmap[2, 1] == R.FP16
    assert pmap[3, 0] == R.FP32 and pmap[3, 1] == R.FP32 and pmap[3, 2] == R.FP8
    assert all(pmap[i, i] == R.FP32 for i in range(NT))
    # allowed mask: without FP8 the FP8 tiles fall to FP16; with FP32 only everything is FP32
    pm2, _, _ = precision_map(A, nb, eps, allowed=(R.FP32, R.FP16))
    assert pm2[1, 0] == R.FP16 and pm2[3, 2] == R.FP16 and pm2[3, 0] == R.FP32
    pm3, _, _ = precision_map(A, nb, eps, allowed=(R.FP32,))
    assert np.all(pm3[np.tril_indices(NT)] == R.FP32)


@pytest.mark.parametrize("eps,want", [(1e-4, R.FP32), (1e-3, R.FP16), (0.07, R.FP8)])
def test_equicorrelation_gives_uniform_maps(eps, want):
    # t_ij = c*nb (i>j); ||A||_F/NT -> c*nb for large n, so the rule reduces to u_p <= eps:
    # eps=1e-4 -> FP32 (u16 = 4.9e-4), eps=1e-3 -> FP16, FP8 only for eps >= 2^-4 (SURVEY finding 1).
    n, nb, c, d = 512, 64, 0.48, 0.53
    NT = n // nb
    A = c * np.ones((n, n)) + d * np.eye(n)
    pmap, t, fro = precision_map(A, nb, eps)
    assert abs(t[3, 1] - c * nb) < 1e-12
    assert abs(fro ** 2 - (n * (c + d) ** 2 + n * (n - 1) * c * c)) < 1e-6
    assert np.all(pmap[np.tril_indices(NT, -1)] == want)


def test_config_like_matrices_get_uniform_maps():
    # reduced twins of C2 (eps 1e-4 -> all FP32) and C4 (eps 1e-3 -> all FP16, no FP8)
    c2 = scaled_config(CONFIGS["C2"], nb=32, n=512, p=400)
    A, _ = make_problem(c2)
    pmap, t, fro = precision_map(A.numpy(), c2.nb, c2.eps_target, c2.allowed)
    off = np.tril_indices(c2.NT, -1)
    assert np.all(pmap[off] == R.FP32)
    ratio = t[off] / (fro / c2.NT)
    assert 0.9 < ratio.min() and ratio.max() < 1.1
    c4 = scaled_config(CONFIGS["C4"], nb=32, n=512, p=400)
    A, _ = make_problem(c4)
    pmap, _, _ = precision_map(A.numpy(), c4.nb, c4.eps_target, c4.allowed)
    assert np.all(pmap[off] == R.FP16)


def test_sherman_morrison_closed_form():
    n, nb, c, d = 192, 32, 0.48, 0.53
    A = c * np.ones((n, n)) + d * np.eye(n)
    rng = np.random.default_rng(1)
    Y = rng.standard_normal((n, 4))
    want = (Y - c * np.ones((n, 1)) * (np.ones((1, n)) @ Y) / (d + n * c)) / d
    got = solve_fp64(A, Y, nb)
    assert np.max(np.abs(got - want)) < 1e-12 * np.max(np.abs(want))


@pytest.mark.parametrize("n,nb,nrhs", [(64, 16, 1), (240, 48, 5)])
def test_potrs_against_lapack_and_residual(n, nb, nrhs):
    rng = np.random.default_rng(2)
    B = rng.standard_normal((n, n))
    A = B @ B.T + n * np.eye(n)
    Y = rng.standard_normal((n, nrhs))
    L, info = tile_cholesky_fp64(A, nb)
    assert info == 0
    X = potrs_fp64(L, Y, nb)
    want = np.linalg.solve(A, Y)
    assert np.max(np.abs(X - want)) < 1e-12 * np.max(np.abs(want))
    assert np.linalg.norm(Y - A @ X) / (np.linalg.norm(A) * np.linalg.norm(X)) < 1e-15
    # forward then backward: L (L^T x) = y
    assert np.max(np.abs(L @ (L.T @ X) - Y)) < 1e-10


def _golden_brackets():
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "survey_probe_table.txt")
    out = {}
    for line in open(path):
        f = line.split()
        if f and not line.startswith("#"):
            out[f[0]] = (float(f[1]), float(f[2]))
    return out


def test_survey_probe_numbers_small():
    # SURVEY 8(c) table at reduced size: all-FP32 backward error ~1e-8 and alpha error ~1e-6;
    # all-FP16 backward error ~1.5e-4 (< 5e-4) while alpha misses 1e-3 (finding 3).  The brackets are
    # stored in tests/golden/survey_probe_table.txt (independent survey-time probes, cited there).
    G = _golden_brackets()
    cfg = scaled_config(CONFIGS["C1"], nb=64, n=1024, p=1000)
    A, Y = make_problem(cfg)
    A = A.numpy(); Y = Y.numpy()
    from oracle.cholesky import backward_error
    alpha = solve_fp64(A, Y, cfg.nb)
    L32, _, info = tile_cholesky_emulated(A, cfg.nb, uniform_map(cfg.NT, R.FP32))
    assert info == 0
    assert backward_error(A, L32) < G["fp32_backward_max"][1]
    a32 = potrs_fp64(L32, Y, cfg.nb)
    assert np.linalg.norm(a32 - alpha) / np.linalg.norm(alpha) < G["fp32_alpha_max"][1]
    L16, _, info = tile_cholesky_emulated(A, cfg.nb, uniform_map(cfg.NT, R.FP16))
    assert info == 0
    be16 = backward_error(A, L16)
    assert G["fp16_backward"][0] < be16 < G["fp16_backward"][1]
    a16 = potrs_fp64(L16, Y, cfg.nb)
    assert np.linalg.norm(a16 - alpha) / np.linalg.norm(alpha) > G["fp16_alpha_min"][0]
    # finding 1: with tile norms ~ ||A||_F / NT the rule reduces to u_p <= eps
    assert G["fp16_eps_threshold"][0] < R.UNIT_ROUNDOFF[R.FP16] < G["fp16_eps_threshold"][1]
    assert G["fp8_eps_threshold"][0] < R.UNIT_ROUNDOFF[R.FP8] < G["fp8_eps_threshold"][1]


def test_band_map_reading():
    from oracle.precision_map import band_map, uniform_map
    from oracle.rounding import FP16, FP32
    assert np.array_equal(band_map(8, 1.0, FP16), uniform_map(8, FP32))          # 100 % FP32
    assert np.array_equal(band_map(8, 0.0, FP16), uniform_map(8, FP16))          # every off-diagonal tile low
    m = band_map(11, 0.4, FP16)                                                  # b = ceil(0.4 * 10) = 4 sub-diagonals
    for i in range(11):
        for j in range(11):
            want = 255 if j > i else (FP32 if i - j <= 4 else FP16)
            assert m[i, j] == want
    # monotone in the fraction
    assert all((band_map(9, f1, FP16) <= band_map(9, f2, FP16)).all() for f1, f2 in [(0.8, 0.6), (0.6, 0.2), (0.2, 0.1)])



# ---- iterative refinement with a fixed factor (oracle.solve.refine; R19) ----
def _spd(n, seed, lam=0.5):
    rng = np.random.default_rng(seed)
    B = rng.standard_normal((n, n))
    A = B @ B.T / n + lam * np.eye(n)
    return A, rng


def test_refine_with_the_exact_factor_is_one_solve():
    from oracle.solve import refine
    n, nb = 96, 32
    A, rng = _spd(n, 3)
    Y = rng.standard_normal((n, 3))
    L = np.linalg.cholesky(A)
    x, norms = refine(A, L, Y, np.zeros_like(Y), nb, 1, round_fp32=False)
    np.testing.assert_allclose(x, np.linalg.solve(A, Y), rtol=1e-11, atol=1e-12)
    assert abs(norms[0] - np.linalg.norm(Y)) <= 1e-12 * np.linalg.norm(Y)      # r_0 = Y when alpha_0 = 0
    assert norms[1] <= 1e-12 * norms[0]
    # no step: the iterate comes back untouched and the one norm is that of Y - A alpha
    x0 = rng.standard_normal((n, 3))
    x, norms = refine(A, L, Y, x0, nb, 0, round_fp32=False)
    assert np.array_equal(x, x0) and len(norms) == 1
    assert abs(norms[0] - np.linalg.norm(Y - A @ x0)) <= 1e-12 * norms[0]


def test_refine_error_follows_the_iteration_matrix():
    """Textbook: with a factor of a perturbed matrix At = L L^T the error obeys e_{s+1} = (I - At^{-1} A) e_s.
    Checked against explicit powers of that matrix (numpy inverse; nothing of the oracle's solve in the expected
    value): a wrong sign of the update, a residual taken with At instead of A, or a stale alpha fails it."""
    from oracle.solve import refine
    n, nb = 64, 16
    A, rng = _spd(n, 5)
    E = rng.standard_normal((n, n)) * 2e-2
    At = A + (E + E.T) / 2
    L = np.linalg.cholesky(At)
    Y = rng.standard_normal((n, 2))
    xstar = np.linalg.solve(A, Y)
    x0 = rng.standard_normal((n, 2))
    M = np.eye(n) - np.linalg.inv(At) @ A
    e = x0 - xstar
    for steps in (1, 2, 4):
        x, norms = refine(A, L, Y, x0, nb, steps, round_fp32=False)
        want = np.linalg.matrix_power(M, steps) @ e
        np.testing.assert_allclose(x - xstar, want, rtol=1e-8, atol=1e-12 * np.abs(e).max())
        assert len(norms) == steps + 1
        for s in range(steps + 1):                                              # r_s = -A e_s
            rs = -A @ (np.linalg.matrix_power(M, s) @ e)
            assert abs(norms[s] - np.linalg.norm(rs)) <= 1e-8 * np.linalg.norm(rs)


def test_refine_recovers_alpha_under_a_half_precision_map():
    """an all-FP16 map misses "alpha to 1e-3" raw and meets it after <= 2 steps.  Here on a
    scaled twin of C4 with the emulated factor; the limit of the FP32-stored iterate is FP32 roundoff."""
    from oracle.solve import refine
    cfg = scaled_config(CONFIGS["C4"], nb=64, n=1024, p=256)
    A, Y = make_problem(cfg, device="cpu")
    A, Y = A.numpy().astype(np.float64), Y.numpy().astype(np.float64)
    pm = uniform_map(cfg.NT, R.FP16)
    L, sc, info = tile_cholesky_emulated(A, cfg.nb, pm, preround_a=True)
    assert info == 0
    xstar = np.linalg.solve(A, Y)
    err = lambda x: np.linalg.norm(x - xstar) / np.linalg.norm(xstar)
    x0 = potrs_fp64(L, Y, cfg.nb)
    x2, norms = refine(A, L, Y, x0, cfg.nb, 2)
    assert err(x0) > 5e-3 and err(x2) < 5e-5 and err(x2) < 1e-2 * err(x0)          # SURVEY: 1.5e-2 -> ~2e-5
    assert norms[1] < 0.2 * norms[0] and norms[2] < 0.2 * norms[1]
    x6, _ = refine(A, L, Y, x0, cfg.nb, 6)
    assert err(x6) < 2e-6                                                        # FP32 storage of alpha


# ---- conjugate gradients preconditioned by the fixed factor (oracle.solve.pcg; R20) ----
def test_pcg_with_the_exact_factor_is_one_step():
    from oracle.solve import pcg
    n, nb = 96, 32
    A, rng = _spd(n, 7)
    Y = rng.standard_normal((n, 3))
    x0 = rng.standard_normal((n, 3))
    x, norms = pcg(A, np.linalg.cholesky(A), Y, x0, nb, 1, round_fp32=False)
    np.testing.assert_allclose(x, np.linalg.solve(A, Y), rtol=1e-10, atol=1e-12)
    assert abs(norms[0] - np.linalg.norm(Y - A @ x0)) <= 1e-12 * norms[0] and norms[1] <= 1e-10 * norms[0]
    x, norms = pcg(A, np.linalg.cholesky(A), Y, x0, nb, 0, round_fp32=False)
    assert np.array_equal(x, x0) and len(norms) == 1


def test_pcg_iterates_minimise_the_energy_norm_over_the_krylov_space():
    """What defines CG: alpha_k = alpha_0 + the element of span{M^-1 r_0, (M^-1 A) M^-1 r_0, ...} (k vectors) that
    minimises ||alpha* - alpha||_A.  The expected iterate is built from that definition by dense least squares on an
    explicitly generated Krylov basis (numpy inverse, eigendecomposition square root): nothing of the recurrence."""
    from oracle.solve import pcg
    n, nb = 48, 16
    A, rng = _spd(n, 11, lam=0.2)
    E = rng.standard_normal((n, n)) * 0.05
    Mt = A + (E + E.T) / 2 + 0.3 * np.eye(n)                     # an SPD preconditioner that is not A
    L = np.linalg.cholesky(Mt)
    Y = rng.standard_normal((n, 2))
    x0 = rng.standard_normal((n, 2))
    xstar = np.linalg.solve(A, Y)
    w, V = np.linalg.eigh(A)
    Ah = V @ np.diag(np.sqrt(w)) @ V.T                           # A^(1/2)
    Minv = np.linalg.inv(Mt)
    for k in (1, 2, 5):
        x, _ = pcg(A, L, Y, x0, nb, k, round_fp32=False)
        for c in range(2):
            v = Minv @ (Y[:, c] - A @ x0[:, c])
            basis = [v]
            for _ in range(k - 1):
                basis.append(Minv @ (A @ basis[-1]))
            Kb, _ = np.linalg.qr(np.stack(basis, axis=1))
            coef, *_ = np.linalg.lstsq(Ah @ Kb, Ah @ (xstar[:, c] - x0[:, c]), rcond=None)
            want = x0[:, c] + Kb @ coef
            np.testing.assert_allclose(x[:, c], want, rtol=1e-7, atol=1e-9)


def test_pcg_converges_where_the_stationary_iteration_diverges():
    """A factor of a matrix far enough from A that the spectral radius of I - M^-1 A exceeds one (what the all-FP16 map
    does to C4 at full size, R20): `refine` grows the error, `pcg` with the same factor reduces the energy
    norm of the error at every step and reaches FP32 roundoff."""
    from oracle.solve import pcg, refine
    n, nb = 128, 32
    A, rng = _spd(n, 13, lam=0.05)
    w, V = np.linalg.eigh(A)
    scale = np.where(np.arange(n) % 3 == 0, 0.35 + 0.6 * rng.random(n), 1.0 + 0.1 * rng.standard_normal(n))
    Mt = V @ np.diag(w * scale) @ V.T                          # eigenvalues of M^-1 A spread over (0.8, 2.9)
    L = np.linalg.cholesky(Mt)
    assert np.max(np.abs(np.linalg.eigvals(np.eye(n) - np.linalg.inv(Mt) @ A))) > 1.2
    Y = rng.standard_normal((n, 2))
    xstar = np.linalg.solve(A, Y)
    x0 = potrs_fp64(L, Y, nb)
    enorm = lambda x: float(np.sqrt(np.sum((x - xstar) * (A @ (x - xstar)))))
    xr, _ = refine(A, L, Y, x0, nb, 12)
    assert enorm(xr) > 5.0 * enorm(x0)
    prev = enorm(x0)
    for k in range(1, 5):
        xk, _ = pcg(A, L, Y, x0, nb, k, round_fp32=False)
        assert enorm(xk) < prev
        prev = enorm(xk)
    x, norms = pcg(A, L, Y, x0, nb, 12)
    assert np.linalg.norm(x - xstar) <= 1e-5 * np.linalg.norm(xstar) and norms[-1] < 1e-5 * norms[0]

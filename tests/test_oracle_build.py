"""Pins of the Build-phase oracle (oracle/build_phase.py): the paper's worked example, closed forms,
the expansion identity the method rests on, a library routine, and the independent input generator."""
import os

import numpy as np
import torch
from scipy.spatial.distance import cdist

from krr_inputs import genotypes, kernel_matrix
from oracle.build_phase import (cross_kernel_matrix_definition, kernel_matrix_definition, mspe, pearson, predict_definition,
                                squared_distance_by_expansion, squared_distances)

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "build_three_patients.txt")


def test_paper_three_patient_example():
    pts, want = [], None
    for ln in open(GOLD):
        f = ln.split()
        if not f or f[0].startswith("#"):
            continue
        if f[0] in "abc":
            pts.append([int(f[1]), int(f[2])])
        elif f[0] == "D":
            want = np.array([int(x) for x in f[1:]]).reshape(3, 3)
    G = np.array(pts)
    assert np.array_equal(squared_distances(G, G), want)
    assert np.array_equal(squared_distance_by_expansion(G), want)


def test_expansion_identity_on_random_int8_including_negative_values():
    rng = np.random.default_rng(0)
    G = rng.integers(-128, 128, size=(37, 53)).astype(np.int8)
    assert np.array_equal(squared_distance_by_expansion(G), squared_distances(G, G))
    # and against a library routine (FP64 cdist is exact on these integers)
    assert np.array_equal(cdist(G.astype(np.float64), G.astype(np.float64), "sqeuclidean").astype(np.int64),
                          squared_distances(G, G))


def test_gaussian_kernel_closed_forms():
    gamma, lam = 0.125, 0.01
    # identical patients: K = 1 everywhere; the regulariser sits on the diagonal only
    G = np.tile(np.array([[2, 0, 1, 1]]), (5, 1))
    A = kernel_matrix_definition(G, gamma, lam)
    assert np.array_equal(A, np.ones((5, 5)) + lam * np.eye(5))
    # one-hot patients: every pair is at squared distance 2
    A = kernel_matrix_definition(np.eye(6, dtype=np.int8), gamma, lam)
    off = ~np.eye(6, dtype=bool)
    assert np.allclose(A[off], np.exp(-2 * gamma), rtol=0, atol=1e-16) and np.allclose(np.diag(A), 1 + lam)
    # a patient and its shift by t in one marker: d = t^2
    G = np.array([[0, 1, 2], [0, 1, 0]])
    assert abs(kernel_matrix_definition(G, gamma, 0.0)[0, 1] - np.exp(-gamma * 4)) < 1e-16


def test_structure_and_bandwidth_semigroup():
    rng = np.random.default_rng(1)
    G = rng.integers(0, 3, size=(40, 200)).astype(np.int8)
    K1 = kernel_matrix_definition(G, 0.003, 0.0)
    K2 = kernel_matrix_definition(G, 0.005, 0.0)
    K3 = kernel_matrix_definition(G, 0.008, 0.0)
    assert np.array_equal(K1, K1.T) and np.all(np.diag(K1) == 1.0)
    assert np.allclose(K1 * K2, K3, rtol=1e-14)                          # exp(-g1 d) exp(-g2 d) = exp(-(g1+g2) d)
    assert np.all(np.linalg.eigvalsh(K3) > -1e-12)                       # the Gaussian kernel is positive semi-definite


def test_agrees_with_the_input_generator():
    """krr_inputs.kernel_matrix (torch, Gram expansion, FP64 exp rounded to FP32) is independent code."""
    G = genotypes(5, 96, 300, "maf")
    gamma, lam = 1.0 / 300, 1e-2
    A_gen = kernel_matrix(G, gamma, lam).numpy()
    A_def = kernel_matrix_definition(G.numpy(), gamma, lam)
    assert np.array_equal(A_gen, A_def.astype(np.float32))


def test_cross_kernel_reduces_to_the_symmetric_one_and_to_explicit_loops():
    rng = np.random.default_rng(2)
    G = rng.integers(0, 3, size=(12, 30)).astype(np.int8)
    T = rng.integers(0, 3, size=(5, 30)).astype(np.int8)
    gamma = 0.02
    assert np.array_equal(cross_kernel_matrix_definition(G, G, gamma), kernel_matrix_definition(G, gamma, 0.0))
    K = cross_kernel_matrix_definition(T, G, gamma)
    W = rng.standard_normal((12, 3))
    P = predict_definition(T, G, gamma, W)
    for i in range(5):
        for r in range(3):
            acc = 0.0
            for j in range(12):
                d = sum((int(T[i, k]) - int(G[j, k])) ** 2 for k in range(30))
                acc += np.exp(-gamma * d) * W[j, r]
            assert abs(P[i, r] - acc) < 1e-13
    assert K.shape == (5, 12)


def test_predicting_the_training_cohort_with_its_own_weights_interpolates():
    """With lambda -> 0 and W = K^-1 Y, Predict on the training genotypes returns Y (KRR interpolates)."""
    rng = np.random.default_rng(3)
    G = rng.integers(0, 3, size=(20, 64)).astype(np.int8)
    gamma = 0.05
    K = kernel_matrix_definition(G, gamma, 0.0)
    Y = rng.standard_normal((20, 2))
    W = np.linalg.solve(K, Y)
    assert np.allclose(predict_definition(G, G, gamma, W), Y, atol=1e-8)


def test_mspe_and_pearson_definitions():
    Y = np.array([[1.0], [2.0], [4.0]])
    H = np.array([[1.0], [1.0], [6.0]])
    assert mspe(Y, H)[0] == (0 + 1 + 4) / 3                                # PAPER.md:243 by hand
    rng = np.random.default_rng(4)
    A = rng.standard_normal((50, 3))
    B = 0.3 * A + rng.standard_normal((50, 3))
    for c in range(3):
        assert abs(pearson(A, B)[c] - np.corrcoef(A[:, c], B[:, c])[0, 1]) < 1e-14
    assert abs(pearson(A, 2.5 * A + 1.0)[0] - 1.0) < 1e-14 and abs(pearson(A, -A)[1] + 1.0) < 1e-14
    assert np.all(mspe(A, A) == 0.0)



def test_confounder_term_closed_forms():
    """the squared distance of the real-valued confounders is added before the exponentiation, so the
    kernel factorises: K(G, C) = K(G) * K_rbf(C) entrywise; with zero genotypes it is the plain Gaussian RBF on C."""
    from oracle.build_phase import confounder_distances
    rng = np.random.default_rng(5)
    G = rng.integers(0, 3, size=(25, 40)).astype(np.int8)
    C = rng.standard_normal((25, 3))
    gamma = 0.03
    assert np.allclose(confounder_distances(C, C), cdist(C, C, "sqeuclidean"), atol=1e-12)
    K = kernel_matrix_definition(G, gamma, 0.0, C)
    assert np.allclose(K, kernel_matrix_definition(G, gamma, 0.0) * np.exp(-gamma * cdist(C, C, "sqeuclidean")), rtol=1e-13)
    Z = np.zeros_like(G)
    assert np.allclose(kernel_matrix_definition(Z, gamma, 0.25, C), np.exp(-gamma * cdist(C, C, "sqeuclidean")) + 0.25 * np.eye(25),
                       rtol=1e-13)
    T, CT = G[:7], C[:7] + 0.5
    Kx = cross_kernel_matrix_definition(T, G, gamma, CT, C)
    assert abs(Kx[2, 9] - np.exp(-gamma * (np.sum((T[2].astype(int) - G[9].astype(int)) ** 2) + np.sum((CT[2] - C[9]) ** 2)))) < 1e-15


def test_ibs_kernel_pins():
    """IBS (Alg. 5 l.5-6): the allele-sharing count by an explicit haplotype model, closed forms, and the identity the
    CUDA path uses (thermometer encoding: the Hamming distance of the encoded rows is sum_k |a_k - b_k|)."""
    from oracle.build_phase import ibs_kernel_matrix_definition
    # per-locus table by brute force over unordered allele pairs: genotype g = number of minor alleles among 2;
    # alleles shared by state = size of the multiset intersection
    def shared(a, b):
        A, Bm = ["m"] * a + ["M"] * (2 - a), ["m"] * b + ["M"] * (2 - b)
        return min(A.count("m"), Bm.count("m")) + min(A.count("M"), Bm.count("M"))
    for a in range(3):
        for b in range(3):
            K = ibs_kernel_matrix_definition(np.array([[a]]), np.array([[b]]))
            assert K[0, 0] == shared(a, b) / 2.0
    rng = np.random.default_rng(6)
    G = rng.integers(0, 3, size=(30, 77)).astype(np.int8)
    K = ibs_kernel_matrix_definition(G, G)
    assert np.array_equal(K, K.T) and np.all(np.diag(K) == 1.0) and K.min() >= 0.0
    # opposite homozygotes everywhere share nothing; a heterozygote shares one allele with anybody
    assert ibs_kernel_matrix_definition(np.zeros((1, 9), int), 2 * np.ones((1, 9), int))[0, 0] == 0.0
    assert ibs_kernel_matrix_definition(np.ones((1, 9), int), rng.integers(0, 3, size=(1, 9)) * 2 % 3)[0, 0] >= 0.5
    # thermometer encoding u = ([g >= 1], [g >= 2]): Hamming distance of the encodings = sum |a - b|
    U = np.concatenate([(G >= 1), (G >= 2)], axis=1).astype(np.int64)
    ham = squared_distances(U, U)                                       # 0/1 entries: squared distance = Hamming
    assert np.array_equal(ham, np.abs(G[:, None, :].astype(int) - G[None, :, :].astype(int)).sum(axis=2))
    assert np.allclose(K, 1.0 - ham / (2.0 * 77), rtol=0, atol=1e-15)
    # positive semi-definite (a sum of per-locus PSD kernels)
    assert np.linalg.eigvalsh(K).min() > -1e-10


def test_linear_kernel_and_ridge_regression_pins():
    from oracle.build_phase import linear_kernel_matrix_definition, ridge_regression_definition
    rng = np.random.default_rng(7)
    X = rng.integers(0, 3, size=(40, 12)).astype(np.int8)              # patients x SNPs
    # the Gram matrix from the distance expansion: <a, b> = (|a|^2 + |b|^2 - |a - b|^2) / 2
    s = np.einsum("ik,ik->i", X.astype(np.int64), X.astype(np.int64))
    assert np.array_equal(linear_kernel_matrix_definition(X, X), (s[:, None] + s[None, :] - squared_distances(X, X)) / 2.0)
    assert np.array_equal(linear_kernel_matrix_definition(X, X, 0.5), 0.5 * (X.astype(float) @ X.astype(float).T))
    # Eq. (2): primal ridge = dual (kernel) ridge with the linear kernel, and the normal equations hold
    Y = rng.standard_normal((40, 3))
    lam = 0.7
    beta = ridge_regression_definition(X, Y, lam)
    alpha = np.linalg.solve(linear_kernel_matrix_definition(X, X) + lam * np.eye(40), Y)
    assert np.allclose(beta, X.T.astype(float) @ alpha, atol=1e-10)
    assert np.allclose(X.T.astype(float) @ (Y - X.astype(float) @ beta), lam * beta, atol=1e-9)     # gradient of Eq. (1) vanishes



def test_identity_border_changes_nothing_of_the_problem():
    """DESIGN.md R21: chol([[A,0],[0,I]]) = blockdiag(chol(A), I) and the bordered solve returns A^-1 Y over zero rows
    -- checked with LAPACK on the bordered matrix and with the oracle's own tile Cholesky / solve at a tile size that
    does not divide n."""
    from oracle.build_phase import identity_border, kernel_matrix_definition
    from oracle.cholesky import tile_cholesky_fp64
    from oracle.solve import potrs_fp64
    rng = np.random.default_rng(21)
    n, p, nb = 77, 40, 32
    G = rng.integers(0, 3, size=(n, p)).astype(np.int8)
    A = kernel_matrix_definition(G, 1.0 / p, 0.05)
    n_pad = -(-n // nb) * nb
    B = identity_border(A, n_pad)
    assert B.shape == (96, 96) and np.array_equal(B[:n, :n], A) and np.array_equal(B[n:, n:], np.eye(n_pad - n))
    assert not B[:n, n:].any() and not B[n:, :n].any()
    Lb = np.linalg.cholesky(B)
    np.testing.assert_allclose(Lb[:n, :n], np.linalg.cholesky(A), rtol=1e-13, atol=1e-15)
    assert np.array_equal(Lb[n:, n:], np.eye(n_pad - n)) and not Lb[n:, :n].any()
    Lt, info = tile_cholesky_fp64(B, nb)
    assert info == 0
    np.testing.assert_allclose(Lt, Lb, rtol=1e-12, atol=1e-14)
    Y = rng.standard_normal((n, 3))
    Yb = np.vstack([Y, np.zeros((n_pad - n, 3))])
    xb = potrs_fp64(Lt, Yb, nb)
    np.testing.assert_allclose(xb[:n], np.linalg.solve(A, Y), rtol=1e-10, atol=1e-12)
    assert not xb[n:].any()


def test_ridge_gram_with_confounders():
    """Fig. 2's matrix: blocks against element-wise sums, and the ridge solution through it against the textbook
    augmented least-squares form min ||[X; sqrt(lam) I] beta - [Y; 0]|| (numpy lstsq: no normal equations)."""
    from oracle.build_phase import ridge_gram_definition, linear_kernel_matrix_definition
    rng = np.random.default_rng(31)
    npat, ns, q, lam = 60, 23, 3, 0.7
    S = rng.integers(0, 3, size=(npat, ns)).astype(np.int8)
    C = rng.standard_normal((npat, q))
    A = ridge_gram_definition(S, C, lam)
    assert A.shape == (ns + q, ns + q) and np.array_equal(A, A.T)
    assert np.array_equal(A[:ns, :ns], linear_kernel_matrix_definition(S.T, S.T) + lam * np.eye(ns))   # integers, exact
    for j in (0, 7, ns - 1):
        for t in range(q):
            want = sum(float(S[k, j]) * C[k, t] for k in range(npat))
            assert abs(A[ns + t, j] - want) <= 1e-12 * max(1.0, abs(want))
    for t in range(q):
        for u in range(q):
            want = sum(C[k, t] * C[k, u] for k in range(npat)) + (lam if t == u else 0.0)
            assert abs(A[ns + t, ns + u] - want) <= 1e-12 * max(1.0, abs(want))
    Y = rng.standard_normal((npat, 2))
    X = np.hstack([S.astype(np.float64), C])
    beta = np.linalg.solve(A, X.T @ Y)
    aug, *_ = np.linalg.lstsq(np.vstack([X, np.sqrt(lam) * np.eye(ns + q)]), np.vstack([Y, np.zeros((ns + q, 2))]), rcond=None)
    np.testing.assert_allclose(beta, aug, rtol=1e-9, atol=1e-11)

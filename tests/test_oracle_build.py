"""Pins of the Build-phase oracle (oracle/build_phase.py): the paper's worked example, closed forms,
the expansion identity the method rests on, a library routine, and the independent input generator."""
import os

import numpy as np
import torch
from scipy.spatial.distance import cdist

from krr_inputs import genotypes, kernel_matrix
from oracle.build_phase import kernel_matrix_definition, squared_distance_by_expansion, squared_distances

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

"""CPU oracle of the Build phase (TEST INFRASTRUCTURE, NOT PRODUCT; see oracle/__init__.py).

What it computes, as the paper defines it:

* Alg. 2: K[i, j] = KernelMatrix(type, gamma, G1[i, :], G2[j, :]) for every pair.
* Alg. 5 l.4, Gaussian kernel: exp(-gamma * ||p1 - p2||^2) (the minus sign inside
  the norm is lost in the extraction; cf. :173 "d_ij = sum_k (g_ki - g_kj)^2" and :186; R14).
* Alg. 3 l.3: the matrix handed to FACTORIZE is K + alpha*Id (alpha = the regulariser
  lambda of DESIGN.md R12).

`kernel_matrix_definition` is that definition written out: the squared distance of every pair from the
differences themselves, in exact integer arithmetic, the exponential in FP64.  No expansion into
norms and a Gram matrix -- that is the *method* of PAPER.md:173-190, which the CUDA path implements
and `squared_distance_by_expansion` restates only so that the tests can pin the identity the method
rests on (D~ = D + D^T - 2 G G^T, :186).
"""
import numpy as np


def squared_distances(G1, G2):
    """d_ij = sum_k (G1[i,k] - G2[j,k])^2, exact (int64), by rows: no (n1, n2, p) temporary."""
    G1 = np.asarray(G1, dtype=np.int64)
    G2 = np.asarray(G2, dtype=np.int64)
    D = np.empty((G1.shape[0], G2.shape[0]), dtype=np.int64)
    for i in range(G1.shape[0]):
        diff = G2 - G1[i][None, :]
        D[i] = np.einsum("jk,jk->j", diff, diff)
    return D


def confounder_distances(C1, C2):
    """squared distances between the real-valued confounders, sum_t (c1_it - c2_jt)^2, in FP64."""
    C1 = np.asarray(C1, dtype=np.float64)
    C2 = np.asarray(C2, dtype=np.float64)
    D = np.empty((C1.shape[0], C2.shape[0]))
    for i in range(C1.shape[0]):
        diff = C2 - C1[i][None, :]
        D[i] = np.einsum("jk,jk->j", diff, diff)
    return D


def kernel_matrix_definition(G, gamma, lam, C=None):
    """A = K + lam*I in FP64: K_ij = exp(-gamma * d_ij) (Alg. 5 l.4), d_ij by the definition; with confounders C
    their squared distance is added to the integer one before the exponentiation."""
    D = squared_distances(G, G).astype(np.float64)
    if C is not None:
        D = D + confounder_distances(C, C)
    A = np.exp(-float(gamma) * D)
    A[np.diag_indices_from(A)] += float(lam)
    return A


def squared_distance_by_expansion(G):
    """The method's identity: D with the squared norms down its columns, D~ = D + D^T,
    D~ <- D~ - 2 G G^T.  Integer arithmetic; returned for the tests to compare with the definition."""
    G = np.asarray(G, dtype=np.int64)
    s = np.einsum("ik,ik->i", G, G)
    D = np.tile(s[None, :], (G.shape[0], 1))          # every row holds (||g_1||^2, ..., ||g_n||^2)
    return D + D.T - 2 * (G @ G.T)


# ---- Predict phase (Alg. 4) and the paper's accuracy measures ----
def cross_kernel_matrix_definition(T, G, gamma, CT=None, CG=None):
    """Alg. 4 l.4-5: K (N_P2 x N_P1), K_ij = exp(-gamma ||t_i - g_j||^2) -- BUILD(gamma, T, G, K), no regulariser."""
    D = squared_distances(T, G).astype(np.float64)
    if CT is not None:
        D = D + confounder_distances(CT, CG)
    return np.exp(-float(gamma) * D)


def predict_definition(T, G, gamma, W, CT=None, CG=None):
    """Alg. 4 l.6: P_r = K x W in FP64."""
    return cross_kernel_matrix_definition(T, G, gamma, CT, CG) @ np.asarray(W, dtype=np.float64)


def mspe(Y, Yhat):
    """MSPE = (1 / N_P2) sum_i (Y_i - Yhat_i)^2 (per phenotype column)."""
    Y = np.asarray(Y, dtype=np.float64)
    Yhat = np.asarray(Yhat, dtype=np.float64)
    return np.sum((Y - Yhat) ** 2, axis=0) / Y.shape[0]


def pearson(Y, Yhat):
    """the normalised covariance cov(Y, Yhat) / (sigma_Y sigma_Yhat), per phenotype column."""
    Y = np.asarray(Y, dtype=np.float64)
    Yhat = np.asarray(Yhat, dtype=np.float64)
    yc = Y - Y.mean(axis=0)
    hc = Yhat - Yhat.mean(axis=0)
    return np.sum(yc * hc, axis=0) / np.sqrt(np.sum(yc * yc, axis=0) * np.sum(hc * hc, axis=0))


# ---- IBS kernel (Alg. 5 l.5-6; definition in the text of PAPER.md:134) ----
def ibs_kernel_matrix_definition(G1, G2):
    """K_ij = (p_i ~ p_j) / (total number of alleles): "counting the number of alleles individuals p_i and p_j share
    that are identical by state at a given SNP locus over the total number of alleles".  Genotypes are
    minor-allele counts in {0, 1, 2}; two genotypes a, b share 2 - |a - b| of their 2 alleles by state, counted here
    locus by locus.  Reading (R17): the divisor is the number of alleles, 2 N_S, so that K_ii = 1; Alg. 5 l.6
    prints N_S."""
    G1 = np.asarray(G1, dtype=np.int64)
    G2 = np.asarray(G2, dtype=np.int64)
    assert G1.min() >= 0 and G1.max() <= 2 and G2.min() >= 0 and G2.max() <= 2
    ns = G1.shape[1]
    K = np.empty((G1.shape[0], G2.shape[0]), dtype=np.float64)
    for i in range(G1.shape[0]):
        shared = 2 - np.abs(G2 - G1[i][None, :])          # alleles shared IBS at every locus
        K[i] = shared.sum(axis=1) / (2.0 * ns)
    return K


# ---- linear kernel / Ridge Regression (Eq. (2); Fig. 2: the SYRK of the encoded matrix) ----
def linear_kernel_matrix_definition(Z1, Z2, scale=1.0):
    """scale * Z1 Z2^T in exact integers, then FP64: the symmetric rank-k update of Eq. (2) when Z = X^T (rows = SNPs,
    X^T X over the patients), or the linear kernel between patients when Z = X."""
    return float(scale) * (np.asarray(Z1, dtype=np.int64) @ np.asarray(Z2, dtype=np.int64).T).astype(np.float64)


def ridge_regression_definition(X, Y, lam):
    """Eq. (2): beta = (X^T X + lam I)^-1 X^T Y in FP64."""
    X = np.asarray(X, dtype=np.float64)
    return np.linalg.solve(X.T @ X + float(lam) * np.eye(X.shape[1]), X.T @ np.asarray(Y, dtype=np.float64))



# ---- ragged n (R21) ----
def identity_border(A, n_pad):
    """The n x n matrix A bordered by an identity block up to n_pad x n_pad: [[A, 0], [0, I]].  The tile algorithms
    need n to be a multiple of nb (the paper's cohort, 305,880 patients, is not a multiple of any tile size it
    uses; how its runtime treats the last partial tile row is not said).  Reading R21: the matrix is bordered, the
    right-hand sides get zero rows; then chol = blockdiag(L, I), the first n rows of the solution are A^-1 Y and
    the rest is zero -- nothing of the original problem changes.  The precision rule is evaluated on the bordered
    matrix (NT and ||.||_F of the bordered matrix)."""
    A = np.asarray(A, dtype=np.float64)
    n = A.shape[0]
    assert n_pad >= n
    B = np.zeros((n_pad, n_pad))
    B[:n, :n] = A
    B[np.arange(n, n_pad), np.arange(n, n_pad)] = 1.0
    return B


# ---- the mixed INT8 / FP32 SYRK of ridge regression (Fig. 2) ----
def ridge_gram_definition(S, C, lam):
    """X^T X + lam I in FP64 for X = [S | C]: S the patients x N_S matrix of SNPs (integers), C the patients x q matrix
    of real-valued confounders ("each row of X is a vector of SNPs and confounders").  The SNP x SNP
    block is an integer matrix (the INT8 tiles of Fig. 2), the blocks that involve a confounder are real (its FP32
    tiles); here everything is FP64, the product written out as one matrix product."""
    X = np.hstack([np.asarray(S, dtype=np.float64), np.asarray(C, dtype=np.float64)])
    return X.T @ X + float(lam) * np.eye(X.shape[1])

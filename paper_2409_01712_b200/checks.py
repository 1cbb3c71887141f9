"""Invariants of a factorisation evaluated by independent code: plain torch FP64 on the device (checking only --
none of this is on the product path, none of it comes from oracle/ or calls the CUDA library; the Factor object is
only read through its dequantising `tile()` accessor).  Used by the GPU tests and by bench.py's `checks`."""
import torch


class LowerTiles:
    """The packed lower tiles of a symmetric matrix (config C4's storage): tile (i,j), i >= j, row-major
    nb x nb at slot j*NT - j(j-1)/2 + (i-j).  Diagonal tiles are full squares; only their lower part is used."""

    def __init__(self, At, n, nb):
        self.n, self.nb, self.NT = n, nb, n // nb
        self.T = At.reshape(-1, nb, nb)
        self.shape = (n, n)
        self.device = At.device

    def column(self, j):
        """Tile column j as a ((NT-j)*nb) x nb matrix (rows j*nb .. n)."""
        s0 = j * self.NT - j * (j - 1) // 2
        return self.T[s0:s0 + self.NT - j].reshape(-1, self.nb)


def _sym_matvec_tiles(A, X):
    nb = A.nb
    out = torch.zeros_like(X, dtype=torch.float64)
    for j in range(A.NT):
        col = A.column(j).to(torch.float64)
        col[:nb] = torch.tril(col[:nb])
        r0 = j * nb
        out[r0:] += col @ X[r0:r0 + nb]
        col[:nb] = torch.tril(col[:nb], -1)
        out[r0:r0 + nb] += col.t() @ X[r0:]
    return out


def sym_matvec(A, X, row_block=4096):
    """(lower-referenced symmetric A, FP32) @ X in FP64, by row blocks.  Uses only A's lower
    triangle: A_sym = tril(A) + tril(A,-1)^T."""
    if isinstance(A, LowerTiles):
        return _sym_matvec_tiles(A, X)
    n = A.shape[0]
    out = torch.zeros_like(X, dtype=torch.float64)
    for r0 in range(0, n, row_block):
        r1 = min(n, r0 + row_block)
        blk = A[r0:r1, :r1].to(torch.float64)
        blk[:, r0:r1] = torch.tril(blk[:, r0:r1])
        out[r0:r1] += blk @ X[:r1]
        strict = blk.clone()
        strict[:, r0:r1] = torch.tril(blk[:, r0:r1], -1)
        out[:r1] += strict.t() @ X[r0:r1]
    return out


def factor_matvec(F, X):
    """L (L^T X) with the dequantised tiles of a Factor, FP64."""
    nb, NT = F.nb, F.NT
    Z = torch.zeros_like(X, dtype=torch.float64)
    for j in range(NT):
        for i in range(j, NT):
            T = F.tile(i, j)
            Z[j * nb:(j + 1) * nb] += T.t() @ X[i * nb:(i + 1) * nb]
    R = torch.zeros_like(X, dtype=torch.float64)
    for j in range(NT):
        for i in range(j, NT):
            T = F.tile(i, j)
            R[i * nb:(i + 1) * nb] += T @ Z[j * nb:(j + 1) * nb]
    return R


def fro_norm_sym(A, row_block=4096):
    if isinstance(A, LowerTiles):
        acc = 0.0
        for j in range(A.NT):
            col = A.column(j).to(torch.float64)
            d = torch.tril(col[:A.nb])
            acc += 2.0 * float((col[A.nb:] ** 2).sum()) + 2.0 * float((torch.tril(d, -1) ** 2).sum()) \
                + float((torch.diagonal(d) ** 2).sum())
        return acc ** 0.5
    n = A.shape[0]
    acc = 0.0
    for r0 in range(0, n, row_block):
        r1 = min(n, r0 + row_block)
        blk = A[r0:r1, :r1].to(torch.float64)
        d = torch.tril(blk[:, r0:r1])
        acc += 2.0 * float((blk[:, :r0] ** 2).sum()) + 2.0 * float((torch.tril(d, -1) ** 2).sum()) \
            + float((torch.diagonal(d) ** 2).sum())
    return acc ** 0.5


def probe_backward_error(A, F, nprobe=32, seed=0):
    """||(A - L L^T) Omega||_F / (sqrt(k) ||A||_F), Omega n x k Gaussian: an unbiased estimate of
    the relative backward error ||A - L L^T||_F / ||A||_F."""
    g = torch.Generator(device=A.device).manual_seed(seed)
    Om = torch.randn((A.shape[0], nprobe), dtype=torch.float64, device=A.device, generator=g)
    R = sym_matvec(A, Om) - factor_matvec(F, Om)
    return float(torch.linalg.norm(R)) / (nprobe ** 0.5 * fro_norm_sym(A))


def solve_residual(A, alpha, Y):
    """||Y - A alpha||_F / (||A||_F ||alpha||_F)."""
    R = Y.to(torch.float64) - sym_matvec(A, alpha.to(torch.float64))
    return float(torch.linalg.norm(R)) / (fro_norm_sym(A) * float(torch.linalg.norm(alpha.to(torch.float64))))

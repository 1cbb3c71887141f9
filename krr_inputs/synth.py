"""Counter-based synthetic genotypes / phenotypes and the Gaussian kernel matrix (input recipe).

The paper's datasets (UK BioBank 305,880 x 43,333; msprime 300K x 40K, :260;
random fill, :202, :305) are not available; these seeded inputs stand in for them with the shapes
and distributions BASELINE.json's configs give:

  genotypes   x_ik ~ Binomial(2, m_k), m_k ~ U(0.05, 0.5) per SNP        (configs C1-C4)
              x_ik uniform over {0,1,2}                                  (config C5, random fill)
  kernel      K_ij = exp(-gamma * ||x_i - x_j||^2), gamma = 1/p           (Alg. 5)
  input       A = K + lambda * I in FP32                                  (Alg. 3 l.3)
  phenotypes  Y n x nrhs standard normal

Every value is a pure function of (seed, indices) through a 64-bit mixing hash, written with
torch int64 tensor ops so that CPU and CUDA generate the same integers.  The kernel matrix is
built from the exact integer squared distances; exp is evaluated in FP64 and rounded to FP32, so
devices agree except for a vanishing fraction of last-bit differences -- tests always hand the
SAME A (one generation) to both the oracle and the CUDA path.
"""
from dataclasses import dataclass, replace

import torch

_MASK63 = (1 << 63) - 1


def _lsr(x, s):
    """Logical right shift of an int64 tensor."""
    return (x >> s) & ((1 << (64 - s)) - 1)


def _i64(c):
    """A 64-bit constant as a Python int in int64 range."""
    c &= (1 << 64) - 1
    return c - (1 << 64) if c >= (1 << 63) else c


_C1 = _i64(0x9E3779B97F4A7C15)
_C2 = _i64(0xBF58476D1CE4E5B9)
_C3 = _i64(0x94D049BB133111EB)


def mix64(x):
    """splitmix64 finaliser on an int64 tensor (wrap-around arithmetic)."""
    x = x + _C1
    x = (x ^ _lsr(x, 30)) * _C2
    x = (x ^ _lsr(x, 27)) * _C3
    return x ^ _lsr(x, 31)


def _stream(seed, stream):
    return _i64((seed * 0x2545F4914F6CDD1D + stream * 0x632BE59BD9B4E019) & ((1 << 64) - 1))


def uniform24(seed, stream, counter):
    """24-bit uniforms in [0,1) as float64 from (seed, stream, counter tensor)."""
    h = mix64(mix64(counter + _stream(seed, stream)))
    return _lsr(h, 40).to(torch.float64) * (2.0 ** -24)


def maf(seed, p, device="cpu"):
    """Minor-allele frequencies m_k ~ U(0.05, 0.5), one per SNP."""
    k = torch.arange(p, dtype=torch.int64, device=device)
    return 0.05 + 0.45 * uniform24(seed, 1, k)


def genotypes(seed, n, p, kind="maf", device="cpu", row0=0, rows=None, dtype=torch.int8):
    """Genotype block G[row0:row0+rows, :p] with entries in {0,1,2}.

    kind = "maf":     Binomial(2, m_k) as [u1 < m_k] + [u2 < m_k]
    kind = "uniform": uniform over {0,1,2} (random fill, config C5)
    """
    rows = n - row0 if rows is None else rows
    i = torch.arange(row0, row0 + rows, dtype=torch.int64, device=device)[:, None]
    k = torch.arange(p, dtype=torch.int64, device=device)[None, :]
    ctr = i * p + k
    if kind == "maf":
        m = maf(seed, p, device)[None, :]
        g = (uniform24(seed, 2, ctr) < m).to(dtype) + (uniform24(seed, 3, ctr) < m).to(dtype)
    elif kind == "uniform":
        h = _lsr(mix64(mix64(ctr + _stream(seed, 2))), 40)       # 24 bits
        g = ((h * 3) >> 24).to(dtype)
    elif kind.startswith("families"):
        # S1: contiguous families of `fam_rows` patients; a member copies its family
        # founder's SNP with probability 0.97 / 0.75 / 0.60 (families 0 / 1 / 2), 0 (the rest) -- related
        # individuals give the higher-precision tiles of PAPER.md:229.
        fam_rows = int(kind.split(":")[1])
        m = maf(seed, p, device)[None, :]
        own = (uniform24(seed, 2, ctr) < m).to(dtype) + (uniform24(seed, 3, ctr) < m).to(dtype)
        fam = i // fam_rows
        fctr = (fam * fam_rows) * p + k
        founder = (uniform24(seed, 2, fctr) < m).to(dtype) + (uniform24(seed, 3, fctr) < m).to(dtype)
        q = torch.where(fam == 0, 0.97, torch.where(fam == 1, 0.75, torch.where(fam == 2, 0.60, 0.0))).to(torch.float64)
        copy = uniform24(seed, 6, ctr) < q
        g = torch.where(copy, founder, own)
    else:
        raise ValueError(kind)
    return g


def phenotypes(seed, n, nrhs, device="cpu"):
    """Y (n x nrhs) standard normal by Box-Muller on hashed uniforms, FP32, row-major."""
    i = torch.arange(n * nrhs, dtype=torch.int64, device=device)
    u1 = uniform24(seed, 4, i) + 2.0 ** -25
    u2 = uniform24(seed, 5, i)
    z = torch.sqrt(-2.0 * torch.log(u1)) * torch.cos(2.0 * torch.pi * u2)
    return z.to(torch.float32).reshape(n, nrhs).contiguous()


def _gram_int(Gi, Gj):
    """Exact integer Gram block Gi Gj^T (entries {0,1,2}) as float64."""
    if Gi.is_cuda:
        # bf16 holds {0,1,2} exactly and cuBLAS accumulates in FP32; sums <= 4p < 2^24 are exact
        # in any order.  Build step, off the hot path (library GEMM is allowed here).
        try:
            out = torch.mm(Gi.to(torch.bfloat16), Gj.to(torch.bfloat16).t(), out_dtype=torch.float32)
        except TypeError:
            prev = torch.backends.cuda.matmul.allow_tf32
            torch.backends.cuda.matmul.allow_tf32 = False
            out = Gi.to(torch.float32) @ Gj.to(torch.float32).t()
            torch.backends.cuda.matmul.allow_tf32 = prev
        return out.to(torch.float64)
    return (Gi.to(torch.float32) @ Gj.to(torch.float32).t()).to(torch.float64)


def kernel_matrix(G, gamma, lam, out=None, row_block=4096):
    """A = K + lam*I in FP32, K_ij = exp(-gamma * ||g_i - g_j||^2) (Alg. 5 l.4 with the minus sign
    the extraction dropped), from d^2_ij = s_i + s_j - 2 <g_i, g_j> with
    exact integers.  The full symmetric matrix is written (row-major n x n)."""
    n, p = G.shape
    assert 4 * p < 2 ** 24, "integer Gram sums must stay exact in FP32"
    dev = G.device
    s = (G.to(torch.float32) ** 2).sum(dim=1).to(torch.float64)
    A = torch.empty((n, n), dtype=torch.float32, device=dev) if out is None else out
    for r0 in range(0, n, row_block):
        r1 = min(n, r0 + row_block)
        d2 = s[r0:r1, None] + s[None, :] - 2.0 * _gram_int(G[r0:r1], G)
        A[r0:r1] = torch.exp(-gamma * d2).to(torch.float32)
    idx = torch.arange(n, device=dev)
    A[idx, idx] = torch.tensor(1.0 + lam, dtype=torch.float64).to(torch.float32).to(dev)
    return A


@dataclass(frozen=True)
class Config:
    """One workload of BASELINE.json:configs (or a scaled twin of it)."""
    name: str
    n: int
    p: int
    nb: int
    lam: float
    nrhs: int
    seed: int
    genotype: str = "maf"            # "maf" | "uniform"
    map_request: str = "fp32"        # "fp32" | "rule" | "force_fp8" | "force_fp16" | "fp8_col0_fp32"
    eps_target: float = 0.0
    allowed: tuple = (0,)            # precision codes the rule may use
    lower_tiles_only: bool = False
    gamma_scale: float = 1.0         # gamma = gamma_scale / p

    @property
    def gamma(self):
        return self.gamma_scale / self.p

    @property
    def NT(self):
        return self.n // self.nb


CONFIGS = {
    "C1": Config("C1", 2048, 1000, 256, 1e-2, 4, seed=1, map_request="fp32"),
    "C2": Config("C2", 16384, 10000, 512, 1e-2, 8, seed=2, map_request="rule", eps_target=1e-4,
                 allowed=(0, 1)),
    "C3": Config("C3", 65536, 50000, 1024, 1e-2, 16, seed=3, map_request="rule", eps_target=1e-4,
                 allowed=(0, 1, 2)),
    "C4": Config("C4", 131072, 100000, 1024, 1e-2, 16, seed=4, map_request="rule",
                 eps_target=1e-3, allowed=(0, 1, 2), lower_tiles_only=True),
    "C5": Config("C5", 98304, 20000, 1024, 1e-1, 4, seed=5, genotype="uniform",
                 map_request="force_fp8", allowed=(0, 2)),
    # C5': the matrix of C5 with tile column 0 kept in FP32, the rest FP8, A not pre-rounded,
    # operands as stored -- the timed stand-in for C5, whose literal map breaks down (info > 0)
    "C5p": Config("C5p", 98304, 20000, 1024, 1e-1, 4, seed=5, genotype="uniform",
                  map_request="fp8_col0_fp32", allowed=(0, 2)),
    # supplementary: the paper's regime K ~ I (gamma = 12/p) with two families of
    # relatives -- the only input on which the rule yields a genuine FP32/FP16/FP8 mosaic
    # class probes: C3's matrix with every off-diagonal tile forced to one storage precision (kernel
    # efficiency per MMA class at full depth; numerics are those of the forced map, reported as they are)
    "C3h": Config("C3h", 65536, 50000, 1024, 1e-2, 16, seed=3, map_request="force_fp16", allowed=(0, 1)),
    # C3's matrix under the map of C5' (tile column 0 FP32, the rest E4M3): the same-matrix FP8 figure beside C3 / C3h
    "C3q": Config("C3q", 65536, 50000, 1024, 1e-2, 16, seed=3, map_request="fp8_col0_fp32", allowed=(0, 2)),
    "S1": Config("S1", 32768, 24576, 1024, 1e-2, 8, seed=6, genotype="families:4096",
                 map_request="rule", eps_target=1e-4, allowed=(0, 1, 2), gamma_scale=12.0),
}


def scaled_config(cfg, nb, n=None, p=None):
    """Reduced-size twin: same NT (unless n given), generator, gamma = 1/p, lambda, map request."""
    n = cfg.NT * nb if n is None else n
    p = max(64, (cfg.p * n) // cfg.n) if p is None else p
    geno = cfg.genotype
    if geno.startswith("families"):
        geno = f"families:{4 * nb}"
    return replace(cfg, name=f"{cfg.name}@n{n}", n=n, p=p, nb=nb, genotype=geno)


def _all_genotypes(cfg, device):
    if cfg.n * cfg.p <= (1 << 31):
        return genotypes(cfg.seed, cfg.n, cfg.p, cfg.genotype, device)
    G = torch.empty((cfg.n, cfg.p), dtype=torch.int8, device=device)
    step = max(1, (1 << 28) // cfg.p)
    for r0 in range(0, cfg.n, step):
        r = min(step, cfg.n - r0)
        G[r0:r0 + r] = genotypes(cfg.seed, cfg.n, cfg.p, cfg.genotype, device, r0, r)
    return G


def make_problem(cfg, device="cpu", row_block=4096):
    """(A FP32 n x n, Y FP32 n x nrhs) for a Config."""
    G = _all_genotypes(cfg, device)
    A = kernel_matrix(G, cfg.gamma, cfg.lam, row_block=row_block)
    Y = phenotypes(cfg.seed, cfg.n, cfg.nrhs, device)
    return A, Y


def kernel_matrix_lower_tiles(G, gamma, lam, nb):
    """The lower tiles of A = K + lam*I packed one after the other in column-major tile order
    (tile (i,j), i >= j, at slot j*NT - j(j-1)/2 + (i-j); each tile row-major nb x nb): the
    "lower-triangular tile storage only" layout of config C4.  Same values as kernel_matrix."""
    n, p = G.shape
    assert n % nb == 0 and 4 * p < 2 ** 24
    NT = n // nb
    dev = G.device
    s = (G.to(torch.float32) ** 2).sum(dim=1).to(torch.float64)
    out = torch.empty((NT * (NT + 1) // 2, nb, nb), dtype=torch.float32, device=dev)
    diag = torch.tensor(1.0 + lam, dtype=torch.float64).to(torch.float32).to(dev)
    idx = torch.arange(nb, device=dev)
    slot = 0
    for j in range(NT):
        Gj = G[j * nb:(j + 1) * nb]
        for i0 in range(j, NT, 8):                        # 8 tile rows at a time
            i1 = min(NT, i0 + 8)
            d2 = s[i0 * nb:i1 * nb, None] + s[None, j * nb:(j + 1) * nb] - 2.0 * _gram_int(G[i0 * nb:i1 * nb], Gj)
            blk = torch.exp(-gamma * d2).to(torch.float32).reshape(i1 - i0, nb, nb)
            if i0 == j:
                blk[0, idx, idx] = diag
            out[slot:slot + (i1 - i0)] = blk
            slot += i1 - i0
    return out.reshape(-1)


def make_problem_lower_tiles(cfg, device="cpu"):
    """(packed lower tiles of A, Y) for a Config -- never materialises the n x n matrix."""
    G = _all_genotypes(cfg, device)
    At = kernel_matrix_lower_tiles(G, cfg.gamma, cfg.lam, cfg.nb)
    Y = phenotypes(cfg.seed, cfg.n, cfg.nrhs, device)
    return At, Y


def exact_lower_factor(seed, n, nb, nnz_per_row=2, device="cpu"):
    """Sparse lower-triangular L0 with entries in {0, +-1/2, +-1, +-2} off the diagonal and a
    power-of-two diagonal in {1, 2}; A = L0 L0^T is then exact in FP32 and every intermediate of
    a tile Cholesky is exactly representable in FP32, FP16 and (with power-of-two tile scales)
    E4M3.  Returns (L0 float64, A float32).  Pure data construction; no factorisation here."""
    g = torch.Generator(device="cpu").manual_seed(seed)
    L0 = torch.zeros((n, n), dtype=torch.float64)
    vals = torch.tensor([0.5, -0.5, 1.0, -1.0, 2.0, -2.0], dtype=torch.float64)
    for i in range(n):
        L0[i, i] = float(2 ** int(torch.randint(0, 2, (1,), generator=g)))
        if i > 0:
            cols = torch.randint(0, i, (nnz_per_row,), generator=g)
            L0[i, cols] = vals[torch.randint(0, 6, (nnz_per_row,), generator=g)]
    A = (L0 @ L0.t())
    assert torch.equal(A.to(torch.float32).to(torch.float64), A)
    return L0.to(device), A.to(torch.float32).to(device)

"""GPU parity of krr_build (Build phase on the INT8 tensor cores) against the oracle's definition.

Tolerance: the squared distances are exact on both sides (integers); the kernel entry is exp(-gamma d)
evaluated by the oracle in FP64 and by the CUDA path in FP32 (expf of the FP32 product gamma*d): the
product carries <= 2 roundings of relative size 2^-24 on an exponent of magnitude gamma*d <= ~4, expf
<= 2 ulp, so |K_gpu - K| <= (2 * 2^-24 * gamma*d + 3 * 2^-24) K  <  8e-7 K for the workloads' gamma*d < 4.
The diagonal (1 + lambda) and the structure (upper tiles untouched) are exact."""
import numpy as np
import pytest
import torch

from krr_inputs import CONFIGS, genotypes, kernel_matrix, scaled_config
from oracle.build_phase import kernel_matrix_definition

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def krr():
    from paper_2409_01712_b200 import build
    build.build()
    import paper_2409_01712_b200 as k
    k.lib()
    return k


def padded(G, mult=16):
    """Row pitch a multiple of 16 bytes (TMA): a view into a wider buffer."""
    n, p = G.shape
    ld = (p + mult - 1) // mult * mult
    buf = torch.full((n, ld), 7, dtype=torch.int8, device=G.device)      # garbage past p must not be read as data
    buf[:, :p] = G
    return buf[:, :p]


@pytest.mark.parametrize("n,p,nb,kind", [(512, 1000, 256, "maf"),        # p not a multiple of 128: TMA zero fill
                                          (1024, 777, 512, "uniform"),
                                          (768, 128, 256, "maf"),         # a single K chunk
                                          (2048, 1000, 256, "maf"),       # config 1 at full size
                                          (3072, 640, 1024, "maf")])      # 256 x 512 blocks, two per tile row unit
def test_build_matches_definition(krr, n, p, nb, kind):
    G = genotypes(11, n, p, kind, device="cuda")
    gamma, lam = 1.0 / p, 1e-2
    A = krr.krr_build(padded(G), gamma, lam, nb)
    torch.cuda.synchronize()
    want = kernel_matrix_definition(G.cpu().numpy(), gamma, lam)
    got = A.cpu().numpy().astype(np.float64)
    NT = n // nb
    for i in range(NT):
        for j in range(NT):
            g = got[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb]
            if j > i:
                assert not g.any()                                        # tiles above the diagonal are not written
                continue
            w = want[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb]
            assert np.all(np.abs(g - w) <= 8e-7 * w), (i, j, float(np.max(np.abs(g - w) / w)))
    assert np.all(np.diag(got) == np.float64(np.float32(1.0 + lam)))
    # within a few ulp of the generator's FP64-evaluated, FP32-rounded matrix, most entries identical
    gen = kernel_matrix(G, gamma, lam).cpu().numpy()
    low = np.tril_indices(n)
    a32 = A.cpu().numpy()
    assert np.mean(a32[low] == gen[low]) > 0.5
    assert np.max(np.abs(a32[low].astype(np.float64) - gen[low]) / gen[low]) < 8e-7


def test_build_general_int8_values_and_tiled_output(krr):
    """Any int8 genotype encoding (negative values included), and the packed lower-tile layout of config C4."""
    n, p, nb = 512, 300, 256
    g = torch.Generator(device="cpu").manual_seed(3)
    G = torch.randint(-128, 128, (n, p), generator=g, dtype=torch.int8).cuda()
    gamma, lam = 2e-7, 0.5
    want = kernel_matrix_definition(G.cpu().numpy(), gamma, lam)
    At = krr.krr_build(padded(G), gamma, lam, nb, tiled_lower=True)
    Ad = krr.krr_build(padded(G), gamma, lam, nb)
    torch.cuda.synchronize()
    T = At.reshape(-1, nb, nb).cpu().numpy()
    NT, slot = n // nb, 0
    for j in range(NT):
        for i in range(j, NT):
            w = want[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb]
            assert np.all(np.abs(T[slot] - w) <= 8e-7 * w)
            assert np.array_equal(T[slot], Ad[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb].cpu().numpy())
            slot += 1


def test_build_feeds_the_associate_phase(krr):
    """Build -> precision map -> factorisation -> solve on the built matrix: same map, backward error and alpha
    tolerances as with the generator's matrix."""
    from oracle.cholesky import backward_error
    from oracle.solve import solve_fp64
    cfg = scaled_config(CONFIGS["C1"], nb=256, n=1024, p=500)
    G = genotypes(cfg.seed, cfg.n, cfg.p, cfg.genotype, device="cuda")
    A = krr.krr_build(padded(G), cfg.gamma, cfg.lam, cfg.nb)
    Y = torch.randn((cfg.n, 4), device="cuda", generator=torch.Generator(device="cuda").manual_seed(0))
    d_map, *_ = krr.precision_map(A, cfg.nb, 1e-4)
    F = krr.potrf_mp(A, cfg.nb, d_map, d_map.cpu())
    alpha = krr.potrs(F, Y.clone())
    torch.cuda.synchronize()
    assert int(F.info.item()) == 0
    Aw = kernel_matrix_definition(G.cpu().numpy(), cfg.gamma, cfg.lam)
    Lg = F.dense().cpu().numpy()
    assert backward_error(Aw.astype(np.float32), Lg) <= 2e-6
    a64 = solve_fp64(Aw.astype(np.float32), Y.cpu().numpy(), cfg.nb)
    assert np.linalg.norm(alpha.cpu().numpy() - a64) / np.linalg.norm(a64) <= 1e-3


def test_build_argument_errors(krr):
    L = krr.lib()
    import ctypes
    G = torch.zeros((512, 160), dtype=torch.int8, device="cuda")
    A = torch.zeros((512, 512), dtype=torch.float32, device="cuda")
    ws = torch.zeros(1 << 20, dtype=torch.uint8, device="cuda")
    vp = lambda t: ctypes.c_void_p(t.data_ptr())
    call = lambda n, p, ldg, nb, flags=0: L.krr_build(vp(G), n, p, ldg, None, 0, 0, 0.01, 0.01, vp(A), 512, nb, flags, None, vp(ws), 1 << 20, None)
    assert call(512, 160, 160, 256) == 0
    assert call(500, 160, 160, 250) == -2            # n, nb not multiples of 256
    assert call(512, 160, 150, 256) == -1            # ldg < p
    assert call(512, 150, 152, 256) == -1            # row pitch not a multiple of 16 bytes
    assert call(512, 160, 160, 256, 8) == -7         # unsupported flag
    torch.cuda.synchronize()


# ------------------------------------------------------------------------------ Predict (Alg. 4)
@pytest.mark.parametrize("m,n,p,nrhs", [(256, 512, 300, 4), (512, 768, 1000, 16), (768, 1024, 129, 32), (256, 256, 64, 1)])
def test_predict_matches_definition(krr, m, n, p, nrhs):
    """K(T, G) entrywise within 8e-7 K (as for krr_build); P_r = K W against the FP64 product: FP32 products and
    sums of n terms of size <= max|W| -> |P_gpu - P| <= 4e-6 * sum_j K_ij |W_jr| (a few n^(1/2) 2^-24, with margin)."""
    from oracle.build_phase import cross_kernel_matrix_definition, predict_definition
    G = genotypes(21, n, p, "maf", device="cuda")
    T = genotypes(22, m, p, "maf", device="cuda")
    gamma = 1.0 / p
    W = torch.randn((n, nrhs), device="cuda", generator=torch.Generator(device="cuda").manual_seed(1))
    P, K = krr.krr_predict(padded(T), padded(G), gamma, W, return_kernel=True)
    torch.cuda.synchronize()
    Kw = cross_kernel_matrix_definition(T.cpu().numpy(), G.cpu().numpy(), gamma)
    Kg = K.cpu().numpy().astype(np.float64)
    assert np.all(np.abs(Kg - Kw) <= 8e-7 * Kw)
    Pw = predict_definition(T.cpu().numpy(), G.cpu().numpy(), gamma, W.cpu().numpy())
    bound = 4e-6 * (Kw @ np.abs(W.cpu().numpy().astype(np.float64))) + 1e-30
    assert np.all(np.abs(P.cpu().numpy() - Pw) <= bound)


def test_build_associate_predict_end_to_end_mspe_and_pearson(krr):
    """Alg. 1 end to end on a synthetic phenotype with an epistatic (pairwise-interaction) signal: Build ->
    precision map -> factorisation -> solve -> Predict on a held-out cohort; MSPE and Pearson correlation of the
    CUDA path against the same pipeline in FP64 (oracle definitions), all-FP32 map and the FP16 map."""
    from oracle.build_phase import kernel_matrix_definition, mspe, pearson, predict_definition
    n, m, p, nb = 1536, 512, 400, 256
    Gall = genotypes(31, n + m, p, "maf", device="cuda")
    G, T = Gall[:n].contiguous(), Gall[n:].contiguous()
    rng = np.random.default_rng(0)
    X = Gall.cpu().numpy().astype(np.float64)
    X = (X - X.mean(0)) / (X.std(0) + 1e-12)
    beta = rng.standard_normal(p) * (rng.random(p) < 0.1)
    pairs = rng.integers(0, p, size=(40, 2))
    signal = X @ beta + 1.5 * sum(X[:, a] * X[:, b] for a, b in pairs)
    Yall = np.stack([signal + 0.5 * signal.std() * rng.standard_normal(n + m) for _ in range(2)], axis=1)
    Yall = (Yall - Yall[:n].mean(0)) / Yall[:n].std(0)
    Y, Ytest = Yall[:n], Yall[n:]
    gamma, lam = 1.0 / p, 1e-1
    # FP64 pipeline from the definitions
    A64 = kernel_matrix_definition(G.cpu().numpy(), gamma, lam)
    W64 = np.linalg.solve(A64, Y)
    P64 = predict_definition(T.cpu().numpy(), G.cpu().numpy(), gamma, W64)
    # CUDA pipeline
    A = krr.krr_build(padded(G), gamma, lam, nb)
    Yd = torch.from_numpy(Y.astype(np.float32)).cuda()
    for forced in (krr.FP32, krr.FP16):
        h = krr.uniform_map(n // nb, forced)
        F = krr.potrf_mp(A, nb, h.cuda(), h)
        Wd = krr.potrs(F, Yd.clone())
        P = krr.krr_predict(padded(T), padded(G), gamma, Wd).cpu().numpy().astype(np.float64)
        torch.cuda.synchronize()
        assert int(F.info.item()) == 0
        m64, mg = mspe(Ytest, P64), mspe(Ytest, P)
        r64, rg = pearson(Ytest, P64), pearson(Ytest, P)
        print(f"map {forced}: MSPE fp64 {m64} gpu {mg}; Pearson fp64 {r64} gpu {rg}")
        tol = 1e-4 if forced == krr.FP32 else 2e-2
        assert np.all(np.abs(mg - m64) <= tol * m64) and np.all(np.abs(rg - r64) <= tol)
        assert np.all(r64 > 0.1)                    # the synthetic signal is learnable: the comparison is not vacuous


@pytest.mark.parametrize("q", [1, 5, 16])
def test_build_and_predict_with_confounders(krr, q):
    """confounder distances accumulated in FP32 and added before the exponentiation.  Tolerance: the
    FP32 confounder sum and its addition to the (exact) integer distance add <= (q + 2) 2^-24 relative to the
    exponent gamma*d <= ~4, on top of the 8e-7 of the plain kernel: 2e-6 K."""
    from oracle.build_phase import cross_kernel_matrix_definition, kernel_matrix_definition
    n, m, p, nb = 768, 256, 500, 256
    G = genotypes(41, n, p, "maf", device="cuda")
    T = genotypes(42, m, p, "maf", device="cuda")
    gen = torch.Generator(device="cuda").manual_seed(q)
    C = 3.0 * torch.randn((n, q), device="cuda", generator=gen)
    CT = 3.0 * torch.randn((m, q), device="cuda", generator=gen)
    gamma, lam = 1.0 / p, 1e-2
    A = krr.krr_build(padded(G), gamma, lam, nb, C=C)
    W = torch.randn((n, 3), device="cuda", generator=gen)
    P, K = krr.krr_predict(padded(T), padded(G), gamma, W, return_kernel=True, CT=CT, CG=C)
    torch.cuda.synchronize()
    want = kernel_matrix_definition(G.cpu().numpy(), gamma, lam, C.cpu().numpy())
    got = A.cpu().numpy().astype(np.float64)
    low = np.tril_indices(n)
    NT = n // nb
    for i in range(NT):
        for j in range(i + 1):
            g, w = got[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb], want[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb]
            assert np.all(np.abs(g - w) <= 2e-6 * w)
    assert np.all(np.diag(got) == np.float64(np.float32(1.0 + lam)))
    Kw = cross_kernel_matrix_definition(T.cpu().numpy(), G.cpu().numpy(), gamma, CT.cpu().numpy(), C.cpu().numpy())
    assert np.all(np.abs(K.cpu().numpy() - Kw) <= 2e-6 * Kw)
    assert float(np.abs(Kw - cross_kernel_matrix_definition(T.cpu().numpy(), G.cpu().numpy(), gamma)).max()) > 1e-3   # the term matters
    Pw = Kw @ W.cpu().numpy().astype(np.float64)
    assert np.all(np.abs(P.cpu().numpy() - Pw) <= 6e-6 * (Kw @ np.abs(W.cpu().numpy().astype(np.float64))))


@pytest.mark.parametrize("n,m,p,nb", [(512, 256, 300, 256), (1024, 512, 1111, 512)])
def test_ibs_kernel_build_and_predict(krr, n, m, p, nb):
    """Alg. 5 l.5-6: the IBS kernel through the same tensor-core kernel on thermometer-encoded genotypes.  The
    allele counts are exact integers on both sides and the quotient by 2 N_S is one correctly rounded FP32 division
    against the oracle's FP64 one: entries agree to half an FP32 ulp (double rounding aside: <= 1 ulp asserted)."""
    from oracle.build_phase import ibs_kernel_matrix_definition
    G = genotypes(51, n, p, "maf", device="cuda")
    T = genotypes(52, m, p, "uniform", device="cuda")
    lam = 0.05
    A = krr.krr_build(padded(G), 0.0, lam, nb, flags=krr.FLAG_KERNEL_IBS)
    W = torch.randn((n, 2), device="cuda", generator=torch.Generator(device="cuda").manual_seed(2))
    P, K = krr.krr_predict(padded(T), padded(G), 0.0, W, return_kernel=True, flags=krr.FLAG_KERNEL_IBS)
    torch.cuda.synchronize()
    want = ibs_kernel_matrix_definition(G.cpu().numpy(), G.cpu().numpy())
    got = A.cpu().numpy()
    NT = n // nb
    for i in range(NT):
        for j in range(i + 1):
            g, w = got[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb].astype(np.float64), want[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb].copy()
            if i == j:
                w[np.diag_indices(nb)] = np.float64(np.float32(1.0 + lam))
            assert np.all(np.abs(g - w) <= 6e-8 * np.abs(w) + 1e-45), (i, j)
    assert float(np.mean(got[np.tril_indices(n, -1)] == want[np.tril_indices(n, -1)].astype(np.float32))) > 0.99
    Kw = ibs_kernel_matrix_definition(T.cpu().numpy(), G.cpu().numpy())
    assert np.all(np.abs(K.cpu().numpy() - Kw) <= 6e-8 * Kw)
    Pw = Kw @ W.cpu().numpy().astype(np.float64)
    assert np.all(np.abs(P.cpu().numpy() - Pw) <= 4e-6 * (Kw @ np.abs(W.cpu().numpy().astype(np.float64))))


@pytest.mark.parametrize("nb,n", [(256, 1536), (512, 2560)])
def test_fit_host_matches_device_pipeline(krr, nb, n):
    """krr_fit_host (genotypes and Y from host memory; the Build runs strip by strip behind the copy: six strips of one
    tile row with 256 x 256 blocks, five with 256 x 512 blocks) against Build -> map -> factorisation -> solve called one
    by one: the same kernels on the same data, bit-identical alpha and map."""
    cfg = scaled_config(CONFIGS["C2"], nb=nb, n=n, p=700)
    G = genotypes(cfg.seed, cfg.n, cfg.p, cfg.genotype, device="cuda")
    Y = torch.randn((cfg.n, 8), device="cuda", generator=torch.Generator(device="cuda").manual_seed(5))
    A = krr.krr_build(padded(G), cfg.gamma, cfg.lam, cfg.nb)
    d_map, *_ = krr.precision_map(A, cfg.nb, 1e-4, (krr.FP32, krr.FP16))
    F = krr.potrf_mp(A, cfg.nb, d_map, d_map.cpu())
    alpha = krr.potrs(F, Y.clone())
    torch.cuda.synchronize()
    hG = G.cpu().pin_memory()
    hY = Y.cpu().pin_memory()
    a2, m2, info, _ = krr.fit_host(hG, cfg.gamma, cfg.lam, cfg.nb, hY, 1e-4, (krr.FP32, krr.FP16))
    assert info == 0 and int(F.info.item()) == 0
    low = torch.tril(torch.ones(cfg.NT, cfg.NT, dtype=torch.bool))
    assert torch.equal(m2[low], d_map.cpu()[low])
    assert torch.equal(a2, alpha.cpu())


def test_linear_kernel_and_ridge_regression(krr):
    """PAPER.md Eq. (2): beta = (X^T X + lam I)^-1 X^T Y with the SYRK on the INT8 tensor cores (krr_build with
    KRR_FLAG_KERNEL_LINEAR on X^T: exact integers), the factorisation and the FP32 solves of the Associate path."""
    from oracle.build_phase import linear_kernel_matrix_definition, ridge_regression_definition
    npat, nsnp, nb = 3000, 1024, 256
    X = genotypes(61, npat, nsnp, "maf", device="cuda")                    # patients x SNPs
    Z = X.t().contiguous()                                                 # SNPs x patients: rows = the vectors of the SYRK
    lam = 50.0
    A = krr.krr_build(padded(Z), 1.0, lam, nb, flags=krr.FLAG_KERNEL_LINEAR)
    torch.cuda.synchronize()
    want = linear_kernel_matrix_definition(Z.cpu().numpy(), Z.cpu().numpy()) + lam * np.eye(nsnp)
    got = A.cpu().numpy().astype(np.float64)
    low = np.tril_indices(nsnp)
    NT = nsnp // nb
    for i in range(NT):
        for j in range(i + 1):
            assert np.array_equal(got[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb], want[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb])   # exact
    Y = torch.randn((npat, 4), device="cuda", generator=torch.Generator(device="cuda").manual_seed(3))
    XtY = (X.to(torch.float32).t() @ Y).contiguous()                       # "in single precision"
    h = krr.uniform_map(NT, krr.FP32)
    F = krr.potrf_mp(A, nb, h.cuda(), h)
    beta = krr.potrs(F, XtY.clone())
    torch.cuda.synchronize()
    assert int(F.info.item()) == 0
    b64 = ridge_regression_definition(X.cpu().numpy(), Y.cpu().numpy(), lam)
    assert np.linalg.norm(beta.cpu().numpy() - b64) / np.linalg.norm(b64) <= 1e-3
    # the rectangular variant: scale * T G^T
    T = genotypes(62, 256, nsnp, "maf", device="cuda")
    W = torch.randn((npat // 8 * 8 // 256 * 256, 2), device="cuda")
    Gs = X[:W.shape[0]].contiguous()
    P, K = krr.krr_predict(padded(T), padded(Gs), 0.25, W, return_kernel=True, flags=krr.FLAG_KERNEL_LINEAR)
    torch.cuda.synchronize()
    assert np.array_equal(K.cpu().numpy().astype(np.float64), linear_kernel_matrix_definition(T.cpu().numpy(), Gs.cpu().numpy(), 0.25))


@pytest.mark.parametrize("name,nb,n,p,eps", [("S1", 256, 2048, 1536, 1e-4), ("C4", 512, 2048, 1500, 1e-3), ("S1", 1024, 4096, 3072, 1e-4)])
def test_precision_map_from_build_statistics(krr, name, nb, n, p, eps):
    """tile sums of squares from the Build epilogue, so that the precision map needs no pass of its own
    over A.  Against krr_precision_map on the matrix the same call produced: the same map bit for bit, tile norms and
    ||A||_F to FP64 summation order, tile maxima exactly; and against the oracle's rule on that matrix."""
    from oracle.precision_map import precision_map as oracle_map
    cfg = scaled_config(CONFIGS[name], nb=nb, n=n, p=p)
    G = genotypes(cfg.seed, cfg.n, cfg.p, cfg.genotype, device="cuda")
    A, st = krr.krr_build(padded(G), cfg.gamma, cfg.lam, nb, stats=True)
    m1, n1, a1, f1 = krr.precision_map_from_build(st, n, nb, eps)
    m2, n2, a2, f2 = krr.precision_map(A, nb, eps)
    torch.cuda.synchronize()
    assert torch.equal(m1, m2)
    assert torch.equal(a1, a2)
    assert abs(float(f1) - float(f2)) <= 1e-12 * float(f2)
    assert float((n1 - n2).abs().max()) <= 2e-7 * float(n2.max())
    # the upper tiles of A are zero here, so the oracle sees the same lower tiles
    pm, _, _ = oracle_map(A.cpu().numpy(), nb, eps)
    low = np.tril_indices(n // nb)
    assert np.array_equal(m1.cpu().numpy()[low], pm[low])



@pytest.mark.parametrize("n_valid,nb,p,tiled", [(1000, 256, 700, False), (777, 512, 333, False), (1300, 256, 512, True)])
def test_ragged_n_by_identity_border(krr, n_valid, nb, p, tiled):
    """DESIGN.md R21 (SURVEY NEXT-4 "ragged n"): krr_build_bordered writes [[A, 0], [0, I]]; garbage in the padding rows
    of G is ignored.  Entries against the oracle's definition on the n_valid patients, bordered by the oracle; then the
    whole Associate phase on the bordered matrix: the statistics of the Build epilogue give the map of
    krr_precision_map, the factor is blockdiag(L, I), the first n_valid rows of alpha are the FP64 solution of the
    original system and the rest is exactly zero."""
    from oracle.build_phase import identity_border
    from oracle.cholesky import tile_cholesky_fp64
    from oracle.solve import solve_fp64
    from helpers import LowerTiles
    n = -(-n_valid // max(nb, 256)) * max(nb, 256)
    G = genotypes(29, n, p, "maf", device="cuda")
    G[n_valid:] = 77                                                          # padding rows: anything
    gamma, lam = 1.0 / p, 5e-2
    A, st = krr.krr_build(padded(G), gamma, lam, nb, tiled_lower=tiled, stats=True, n_valid=n_valid)
    torch.cuda.synchronize()
    want = identity_border(kernel_matrix_definition(G[:n_valid].cpu().numpy(), gamma, lam), n)
    NT = n // nb
    if tiled:
        T = A.reshape(-1, nb, nb).cpu().numpy().astype(np.float64)
        got = np.zeros((n, n))
        for j in range(NT):
            for i in range(j, NT):
                got[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb] = T[krr.tile_slot(NT, i, j)]
    else:
        got = A.cpu().numpy().astype(np.float64)
    for i in range(NT):
        for j in range(i + 1):
            g = got[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb]
            w = want[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb]
            assert np.all(np.abs(g - w) <= 8e-7 * np.abs(w)), (i, j)          # the border (0 and 1) exactly
    flags = krr.FLAG_A_TILED_LOWER if tiled else 0
    m1, n1, a1, f1 = krr.precision_map_from_build(st, n, nb, 1e-4)
    m2, n2, a2, f2 = krr.precision_map(A, nb, 1e-4, flags=flags, n=n)
    assert torch.equal(m1, m2) and torch.equal(a1, a2)
    h = krr.uniform_map(NT, krr.FP32)
    F = krr.potrf_mp(A, nb, h.cuda(), h, flags=krr.FLAG_PREROUND_A | flags, n=n)
    g = torch.Generator(device="cpu").manual_seed(n_valid)
    Y = torch.zeros((n, 4), dtype=torch.float32)
    Y[:n_valid] = torch.randn((n_valid, 4), generator=g)
    alpha = krr.potrs(F, Y.cuda())
    torch.cuda.synchronize()
    assert int(F.info.item()) == 0
    a = alpha.cpu().numpy().astype(np.float64)
    assert not a[n_valid:].any()                                              # the border rows stay exactly zero
    Lb, info = tile_cholesky_fp64(want, nb)
    assert info == 0
    Lg = F.dense().cpu().numpy()
    assert np.linalg.norm(Lg - Lb) <= 1e-4 * np.linalg.norm(Lb)
    assert np.array_equal(Lg[n_valid:, n_valid:], np.eye(n - n_valid)) and not Lg[n_valid:, :n_valid].any()
    xs = np.linalg.solve(want[:n_valid, :n_valid], Y[:n_valid].numpy().astype(np.float64))
    assert np.linalg.norm(a[:n_valid] - xs) <= 1e-4 * np.linalg.norm(xs)


def test_build_bordered_rejects_bad_n_valid(krr):
    G = genotypes(3, 512, 256, "maf", device="cuda")
    with pytest.raises(krr.KrrError):
        krr.krr_build(padded(G), 1.0 / 256, 1e-2, 256, n_valid=0)
    with pytest.raises(krr.KrrError):
        krr.krr_build(padded(G), 1.0 / 256, 1e-2, 256, n_valid=513)


@pytest.mark.parametrize("ns,q,npat,nb,tiled", [(1000, 5, 3001, 256, False), (700, 16, 2000, 512, False), (1500, 3, 1111, 256, True)])
def test_ridge_regression_with_confounders_mixed_syrk(krr, ns, q, npat, nb, tiled):
    """PAPER.md Fig. 2 / :165-167: X = [SNPs | confounders]; the SNP x SNP block of X^T X from the INT8 tensor cores
    (exact), the q rows that involve a confounder accumulated in FP32 (the paper's SGEMM tiles), identity border up to
    the tile size (R21).  Against the oracle's FP64 definition: INT8 block exact, FP32 rows to the bound of an FP32 dot
    product of `npat` terms accumulated in 32 partial sums (sqrt-free bound: npat/32 * 2^-24 * sum |x||c|, taken as
    2e-5 of the row's scale); then beta through the Associate path against the FP64 ridge solution."""
    from oracle.build_phase import identity_border, ridge_gram_definition, ridge_regression_definition
    n = -(-(ns + q) // max(nb, 256)) * max(nb, 256)
    X = genotypes(71, npat, ns, "maf", device="cuda")                      # patients x SNPs
    g = torch.Generator(device="cpu").manual_seed(ns + q)
    C = (torch.randn((npat, q), generator=g) * 3.0 + 1.0).cuda()           # confounders: real, not centred (age-like)
    S = torch.full((n, npat), 5, dtype=torch.int8, device="cuda")          # padding rows: anything
    S[:ns] = X.t()
    lam = 20.0
    A = krr.build_rr(padded(S), ns, lam, nb, C=C, tiled_lower=tiled)
    torch.cuda.synchronize()
    want = identity_border(ridge_gram_definition(X.cpu().numpy(), C.cpu().numpy().astype(np.float64), lam), n)
    NT = n // nb
    if tiled:
        T = A.reshape(-1, nb, nb).cpu().numpy().astype(np.float64)
        got = np.zeros((n, n))
        for j in range(NT):
            for i in range(j, NT):
                got[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb] = T[krr.tile_slot(NT, i, j)]
    else:
        got = A.cpu().numpy().astype(np.float64)
    low = np.tril(np.ones((n, n), dtype=bool))
    blk = np.zeros((n, n), dtype=bool)
    for i in range(NT):                                                    # what is stored: lower tiles, diagonal tiles in full
        blk[i * nb:(i + 1) * nb, :(i + 1) * nb] = True
    snp = np.zeros((n, n), dtype=bool)
    snp[:ns, :ns] = True
    border = np.zeros((n, n), dtype=bool)
    border[ns + q:, :] = True
    border[:, ns + q:] = True
    assert np.array_equal(got[blk & snp], want[blk & snp])                 # INT8 tiles: exact integers (+ lam)
    assert np.array_equal(got[blk & border], want[blk & border])           # identity border
    conf = blk & ~snp & ~border
    scale = np.abs(want[conf]).max()
    assert np.all(np.abs(got[conf] - want[conf]) <= 2e-5 * scale), float(np.abs(got[conf] - want[conf]).max() / scale)
    assert np.array_equal(got[blk & low.T & ~border & ~snp], got.T[blk & low.T & ~border & ~snp])   # mirrored inside the diagonal tile
    # beta = (X^T X + lam I)^-1 X^T Y
    Y = torch.randn((npat, 3), generator=g).cuda()
    Xf = torch.cat([X.to(torch.float32), C], dim=1)
    XtY = torch.zeros((n, 3), device="cuda")
    XtY[:ns + q] = Xf.t() @ Y
    h = krr.uniform_map(NT, krr.FP32)
    F = krr.potrf_mp(A, nb, h.cuda(), h, flags=krr.FLAG_PREROUND_A | (krr.FLAG_A_TILED_LOWER if tiled else 0), n=n)
    beta = krr.potrs(F, XtY.clone())
    torch.cuda.synchronize()
    assert int(F.info.item()) == 0
    b = beta.cpu().numpy().astype(np.float64)
    assert not b[ns + q:].any()
    b64 = ridge_regression_definition(Xf.cpu().numpy().astype(np.float64), Y.cpu().numpy(), lam)
    assert np.linalg.norm(b[:ns + q] - b64) / np.linalg.norm(b64) <= 1e-3

"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, on the same seeded inputs.

Tolerances (BASELINE.json north_star):
  * precision map: bit-exact; tile norms / ||A||_F to FP64-summation-order accuracy
  * all-FP32 maps: ||L_gpu - L_oracle||_F / ||L_oracle||_F <= 1e-4, backward error <= 1e-6,
    alpha vs the FP64 solve <= 1e-3
  * FP16 / FP8 / mixed maps: backward error <= 5e-4 and within 2 % of the oracle's; the literal
    L comparison passes at max(1e-4, 2 x the oracle's own rounding-flip noise floor); the first tile
    column (no accumulated noise yet) agrees to one storage ulp
  * exactly-representable constructions: bit for bit under every map
  * breakdown: same `info` tile column as the oracle
"""
from dataclasses import replace

import numpy as np
import pytest
import torch

from krr_inputs import CONFIGS, exact_lower_factor, make_problem, scaled_config
from oracle import rounding as R
from oracle.cholesky import backward_error, tile_cholesky_emulated
from oracle.precision_map import precision_map as oracle_map
from oracle.precision_map import uniform_map as oracle_uniform
from oracle.solve import potrs_fp64, solve_fp64

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def krr():
    from paper_2409_01712_b200 import build
    build.build()
    import paper_2409_01712_b200 as k
    k.lib()
    return k


def relF(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def gpu_factor(krr, A, nb, pmap, preround=True):
    h = torch.from_numpy(np.ascontiguousarray(pmap))
    F = krr.potrf_mp(A, nb, h.cuda(), h, flags=krr.FLAG_PREROUND_A if preround else 0)
    torch.cuda.synchronize()
    return F


# ------------------------------------------------------------------------------ precision map
@pytest.mark.parametrize("name,nb,n,p,eps", [("C1", 128, 1024, 500, 1e-4), ("C4", 128, 1024, 800, 1e-3),
                                             ("S1", 128, 2048, 1536, 1e-4), ("C5", 256, 1024, 400, 0.07)])
def test_precision_map_bit_exact(krr, name, nb, n, p, eps):
    cfg = scaled_config(CONFIGS[name], nb=nb, n=n, p=p)
    A, _ = make_problem(cfg, device="cuda")
    d_map, norms, amax, fro = krr.precision_map(A, nb, eps, (0, 1, 2))
    torch.cuda.synchronize()
    pm, t, f = oracle_map(A.cpu().numpy(), nb, eps)
    assert np.array_equal(d_map.cpu().numpy(), pm)
    assert abs(float(fro) - f) <= 1e-12 * f
    assert np.max(np.abs(norms.cpu().numpy().astype(np.float64) - t)) <= 2e-7 * t.max()
    An = A.cpu().numpy()
    for (i, j) in [(0, 0), (3, 1), (cfg.NT - 1, 0), (cfg.NT - 1, cfg.NT - 1)]:
        assert float(amax[i, j]) == np.abs(An[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb]).max()
    # allowed mask: FP32 only -> all FP32
    d2, _, _, _ = krr.precision_map(A, nb, eps, (0,))
    assert int((d2.cpu()[np.tril_indices(cfg.NT)] != 0).sum()) == 0


def pack_lower_tiles(A, nb):
    n = A.shape[0]
    NT = n // nb
    tiles = []
    for j in range(NT):
        for i in range(j, NT):
            tiles.append(A[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb].contiguous().reshape(-1))
    return torch.cat(tiles)


def test_tiled_lower_storage_gives_identical_results(krr):
    cfg = scaled_config(CONFIGS["C4"], nb=128, n=1024, p=800)
    A, _ = make_problem(cfg, device="cuda")
    At = pack_lower_tiles(A, cfg.nb)
    m1, n1, a1, f1 = krr.precision_map(A, cfg.nb, 1e-3)
    m2, n2, a2, f2 = krr.precision_map(At, cfg.nb, 1e-3, flags=krr.FLAG_A_TILED_LOWER, n=cfg.n)
    assert torch.equal(m1, m2) and torch.equal(n1, n2) and torch.equal(f1, f2)
    h = m1.cpu()
    F1 = krr.potrf_mp(A, cfg.nb, m1, h)
    F2 = krr.potrf_mp(At, cfg.nb, m1, h, flags=krr.FLAG_PREROUND_A | krr.FLAG_A_TILED_LOWER, n=cfg.n)
    torch.cuda.synchronize()
    assert torch.equal(F1.payload, F2.payload) and torch.equal(F1.scales, F2.scales)


# ------------------------------------------------------------------------------ FP32 maps
@pytest.mark.parametrize("name,nb,n,p", [("C1", 256, 2048, 1000),      # config 1 at full size
                                         ("C2", 128, 1536, 1000),      # NT = 12, ragged vs 148 CTAs
                                         ("C1", 128, 128, 200),        # NT = 1: POTRF only
                                         ("C1", 512, 1024, 300)])
def test_fp32_map_meets_all_three_tolerances(krr, name, nb, n, p):
    cfg = scaled_config(CONFIGS[name], nb=nb, n=n, p=p)
    A, Y = make_problem(cfg, device="cuda")
    pmap = oracle_uniform(cfg.NT, R.FP32)
    F = gpu_factor(krr, A, nb, pmap)
    assert int(F.info.item()) == 0
    An, Yn = A.cpu().numpy(), Y.cpu().numpy()
    Lo, _, info = tile_cholesky_emulated(An, nb, pmap)
    assert info == 0
    Lg = F.dense().cpu().numpy()
    assert np.array_equal(Lg, np.tril(Lg)) and np.all(np.diag(Lg) > 0)
    assert relF(Lg, Lo) <= 1e-4
    assert backward_error(An, Lg) <= 1e-6
    alpha = krr.potrs(F, Y.clone())
    torch.cuda.synchronize()
    a64 = solve_fp64(An, Yn, nb)
    assert relF(alpha.cpu().numpy().astype(np.float64), a64) <= 1e-3
    # the solve itself against the oracle's substitution with the SAME factor
    assert relF(alpha.cpu().numpy().astype(np.float64), potrs_fp64(Lg, Yn, nb)) <= 1e-5
    assert torch.all(F.scales.cpu()[np.tril_indices(cfg.NT)] == 1.0)


def test_lookahead_pipeline_matches_serial_schedule(krr):
    """Default schedule (column k+1's update of the final columns overlaps the factorisation of column
    k on internal streams) against KRR_FLAG_NO_LOOKAHEAD: same arithmetic up to the FP32 summation
    order of the newest term, both within the all-FP32 tolerances."""
    cfg = scaled_config(CONFIGS["C2"], nb=256, n=3072, p=1500)           # NT = 12, nsub = 2
    A, _ = make_problem(cfg, device="cuda")
    pmap = oracle_uniform(cfg.NT, R.FP32)
    h = torch.from_numpy(np.ascontiguousarray(pmap))
    F1 = krr.potrf_mp(A, cfg.nb, h.cuda(), h, flags=krr.FLAG_PREROUND_A)
    F2 = krr.potrf_mp(A, cfg.nb, h.cuda(), h, flags=krr.FLAG_PREROUND_A | krr.FLAG_NO_LOOKAHEAD)
    F3 = krr.potrf_mp(A, cfg.nb, h.cuda(), h, flags=krr.FLAG_PREROUND_A)
    torch.cuda.synchronize()
    assert int(F1.info.item()) == 0 and int(F2.info.item()) == 0
    assert torch.equal(F1.payload, F3.payload)                            # the pipeline is deterministic
    L1, L2 = F1.dense().cpu().numpy(), F2.dense().cpu().numpy()
    assert relF(L1, L2) <= 1e-5
    An = A.cpu().numpy()
    Lo, _, _ = tile_cholesky_emulated(An, cfg.nb, pmap)
    for Lg in (L1, L2):
        assert relF(Lg, Lo) <= 1e-4 and backward_error(An, Lg) <= 1e-6


@pytest.mark.parametrize("nb,n", [(256, 2048), (1024, 4096)])
def test_fused_diagonal_chain_is_bit_identical_to_unfused(krr, nb, n):
    """The diagonal-tile chain as ONE launch of nb/128 co-operating CTAs (KRR_FLAG_FUSED_CHAIN: POTRF of the
    128-blocks on the epilogue warps, items ordered through progress counters in global memory) against one
    launch per step (default): the same arithmetic in the same order, so the factors agree bit for bit --
    in both schedules, repeatedly (no dependence on timing)."""
    cfg = replace(scaled_config(CONFIGS["S1"], nb=nb, n=n, p=1536), genotype="maf", gamma_scale=4.0)
    A, _ = make_problem(cfg, device="cuda")
    rng = np.random.default_rng(7)
    pmap = oracle_uniform(cfg.NT, R.FP32)
    for i in range(cfg.NT):
        for j in range(i):
            pmap[i, j] = rng.integers(0, 3)
    h = torch.from_numpy(np.ascontiguousarray(pmap))
    for extra in (0, krr.FLAG_NO_LOOKAHEAD):
        F1 = krr.potrf_mp(A, cfg.nb, h.cuda(), h, flags=krr.FLAG_PREROUND_A | extra)
        F2 = krr.potrf_mp(A, cfg.nb, h.cuda(), h, flags=krr.FLAG_PREROUND_A | extra | krr.FLAG_FUSED_CHAIN)
        F3 = krr.potrf_mp(A, cfg.nb, h.cuda(), h, flags=krr.FLAG_PREROUND_A | extra)
        torch.cuda.synchronize()
        assert int(F1.info.item()) == 0 and int(F2.info.item()) == 0
        assert torch.equal(F1.payload, F2.payload) and torch.equal(F1.scales, F2.scales)
        assert torch.equal(F1.payload, F3.payload)


@pytest.mark.parametrize("prec", ["fp32", "mixed"])
def test_cta_pair_updates_match_single_cta(krr, prec):
    """Trailing updates on CTA pairs (cta_group::2, 256x128 blocks, default when nb % 256 == 0) against
    KRR_FLAG_NO_CTA_PAIRS: the same products in the same order."""
    cfg = replace(scaled_config(CONFIGS["S1"], nb=256, n=2560, p=1536), genotype="maf", gamma_scale=4.0)
    A, _ = make_problem(cfg, device="cuda")
    pmap = oracle_uniform(cfg.NT, R.FP32)
    if prec == "mixed":
        rng = np.random.default_rng(3)
        for i in range(cfg.NT):
            for j in range(i):
                pmap[i, j] = rng.integers(0, 3)
    h = torch.from_numpy(np.ascontiguousarray(pmap))
    F1 = krr.potrf_mp(A, cfg.nb, h.cuda(), h, flags=krr.FLAG_PREROUND_A)
    F2 = krr.potrf_mp(A, cfg.nb, h.cuda(), h, flags=krr.FLAG_PREROUND_A | krr.FLAG_NO_CTA_PAIRS)
    torch.cuda.synchronize()
    assert int(F1.info.item()) == 0 and int(F2.info.item()) == 0
    L1, L2 = F1.dense().cpu().numpy(), F2.dense().cpu().numpy()
    print(f"pairs vs single ({prec}): relF {relF(L1, L2):.3e} equal fraction {np.mean(L1 == L2):.4f}")
    Lo, floor = noise_floor(A.cpu().numpy(), cfg.nb, pmap, True)
    assert relF(L1, L2) <= max(1e-5, 2.0 * floor)
    assert relF(L1, Lo) <= max(1e-4, 2.0 * floor)


# ------------------------------------------------------------------------------ low-precision maps
def noise_floor(An, nb, pmap, preround, seed=0):
    """The oracle against itself on an input perturbed at the level of the CUDA path's FP32-class
    arithmetic (relative 2^-21 ~ 4.8e-7: 22-bit hi/lo operands and truncating tensor-core
    accumulation give a measured backward error of 2-4e-7): how far two correct evaluations of the
    emulated mosaic drift apart through flipped roundings."""
    rng = np.random.default_rng(seed)
    Ap = (An.astype(np.float64) * (1.0 + rng.uniform(-1, 1, An.shape) * 2.0 ** -21)).astype(np.float32)
    Ap = np.tril(Ap) + np.tril(Ap, -1).T
    L1, _, _ = tile_cholesky_emulated(An, nb, pmap, preround)
    L2, _, _ = tile_cholesky_emulated(Ap, nb, pmap, preround)
    return L1, relF(L2, L1)


@pytest.mark.parametrize("case", ["fp16_uniform", "s1_rule_mosaic", "random_mixed", "fp8_col0_fp32", "c3q_twin"])
def test_low_precision_maps(krr, case):
    if case == "fp16_uniform":
        cfg = scaled_config(CONFIGS["C4"], nb=128, n=1024, p=800)
        A, Y = make_problem(cfg, device="cuda")
        pmap, preround = oracle_uniform(cfg.NT, R.FP16), True
    elif case == "s1_rule_mosaic":
        cfg = scaled_config(CONFIGS["S1"], nb=128, n=2048, p=1536)
        A, Y = make_problem(cfg, device="cuda")
        pmap, _, _ = oracle_map(A.cpu().numpy(), cfg.nb, cfg.eps_target)
        preround = True
        assert len(set(pmap[np.tril_indices(cfg.NT, -1)].tolist())) == 3
    elif case == "random_mixed":
        # K ~ I regime without relatives (gamma = 12/p): any map keeps the matrix definite
        cfg = replace(scaled_config(CONFIGS["S1"], nb=128, n=1024, p=768), genotype="maf", gamma_scale=4.0)
        A, Y = make_problem(cfg, device="cuda")
        rng = np.random.default_rng(5)
        pmap = oracle_uniform(cfg.NT, R.FP32)
        for i in range(cfg.NT):
            for j in range(i):
                pmap[i, j] = rng.integers(0, 3)
        preround = True
    elif case == "c3q_twin":   # the map of C5' on the matrix family of C3 (bench.py's same-matrix FP8 figure)
        cfg = scaled_config(CONFIGS["C3q"], nb=128, n=2048, p=1600)
        A, Y = make_problem(cfg, device="cuda")
        pmap = oracle_uniform(cfg.NT, R.FP8)
        pmap[1:, 0] = R.FP32
        preround = False
    else:   # C5': forced FP8 with tile column 0 kept in FP32, operands as stored
        cfg = scaled_config(CONFIGS["C5"], nb=128, n=1024, p=200)
        A, Y = make_problem(cfg, device="cuda")
        pmap = oracle_uniform(cfg.NT, R.FP8)
        pmap[1:, 0] = R.FP32
        preround = False
    nb = cfg.nb
    An = A.cpu().numpy()
    F = gpu_factor(krr, A, nb, pmap, preround)
    Lo, floor = noise_floor(An, nb, pmap, preround)
    Lg = F.dense().cpu().numpy()
    _, sc_o, info_o = tile_cholesky_emulated(An, nb, pmap, preround)
    assert int(F.info.item()) == info_o == 0
    bg, bo = backward_error(An, Lg), backward_error(An, Lo)
    lit = relF(Lg, Lo)
    print(f"{case}: relF {lit:.3e} floor {floor:.3e} backward gpu {bg:.4e} oracle {bo:.4e}")
    if case in ("fp16_uniform", "s1_rule_mosaic", "c3q_twin"):    # maps the rule produces (and the bench's C3q): north_star's bound
        assert bg <= 5e-4
    assert abs(bg - bo) <= 0.02 * bo
    assert lit <= max(1e-4, 2.0 * floor)
    # first tile column: L_i0 = rd(A_i0 L_00^-T) has no accumulated noise -> at most one storage ulp
    for i in range(1, cfg.NT):
        g, o = Lg[i * nb:(i + 1) * nb, :nb], Lo[i * nb:(i + 1) * nb, :nb]
        p = int(pmap[i, 0])
        if p == R.FP32:                      # FP32 tiles: the literal criterion, tile by tile
            assert relF(g, o) <= 1e-4, (case, i)
            continue
        u = R.UNIT_ROUNDOFF[p]
        # one storage ulp (<= 2u|x|, or the subnormal spacing of a scaled FP8 tile) where FP32-level
        # noise of the TRSM (<= 1e-5 of the tile's largest entry, conditioning of L_00 included)
        # flips a rounding; exactly equal elsewhere
        sub = float(sc_o[i, 0]) * 2.0 ** -9 if p == R.FP8 else 0.0
        tol = 2.5 * u * np.abs(o) + sub + 1e-5 * np.abs(o).max()
        assert np.all(np.abs(g - o) <= tol), (case, i, float(np.max(np.abs(g - o) - tol)))
        assert np.mean(g == o) > 0.5, (case, i)          # most elements round identically
    # FP8 scales: powers of two, equal to the oracle's
    sg = F.scales.cpu().numpy().astype(np.float64)
    low = np.tril_indices(cfg.NT)
    mism = (sg[low] != sc_o[low]).sum()
    assert mism <= 0.02 * len(low[0]) + 1          # a tile amax within rounding noise of a binade edge
    # stored tiles are in their formats
    for (i, j) in [(cfg.NT - 1, 0), (cfg.NT - 1, cfg.NT - 2), (2, 1)]:
        blk = Lg[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb]
        p = int(pmap[i, j])
        if p == R.FP8:
            assert np.array_equal(R.rd_e4m3(blk / sg[i, j]) * sg[i, j], blk)
        elif p == R.FP16:
            assert np.array_equal(R.rd_fp16(blk), blk)
    # solve parity with the same factor
    alpha = krr.potrs(F, Y.clone())
    torch.cuda.synchronize()
    assert relF(alpha.cpu().numpy().astype(np.float64), potrs_fp64(Lg, Y.cpu().numpy(), nb)) <= 1e-5


def test_fp8_block_scaled_mma_matches_fp16_image_path(krr):
    """FP8 x FP8 tile products on the E4M3 images (kind::mxf8f6f4, UE8M0 tile scales from the TMEM table)
    against the same products through the exact FP16 images (KRR_FLAG_FP8_VIA_FP16): identical operand
    values, so the factors agree to FP32 accumulation noise amplified by the FP8 roundings."""
    cfg = replace(scaled_config(CONFIGS["S1"], nb=256, n=2048, p=1536), genotype="maf", gamma_scale=4.0)
    A, _ = make_problem(cfg, device="cuda")
    pmap = oracle_uniform(cfg.NT, R.FP8)
    h = torch.from_numpy(np.ascontiguousarray(pmap))
    F1 = krr.potrf_mp(A, cfg.nb, h.cuda(), h, flags=krr.FLAG_PREROUND_A)
    F2 = krr.potrf_mp(A, cfg.nb, h.cuda(), h, flags=krr.FLAG_PREROUND_A | krr.FLAG_FP8_VIA_FP16)
    torch.cuda.synchronize()
    assert int(F1.info.item()) == 0 and int(F2.info.item()) == 0
    An = A.cpu().numpy()
    L1, L2 = F1.dense().cpu().numpy(), F2.dense().cpu().numpy()
    Lo, floor = noise_floor(An, cfg.nb, pmap, True)
    b1, b2, bo = backward_error(An, L1), backward_error(An, L2), backward_error(An, Lo)
    print(f"fp8 mx vs fp16-image: relF {relF(L1, L2):.3e} floor {floor:.3e} backward {b1:.4e} {b2:.4e} oracle {bo:.4e}")
    assert relF(L1, L2) <= max(1e-4, 2.0 * floor)
    assert abs(b1 - bo) <= 0.02 * bo and abs(b2 - bo) <= 0.02 * bo
    # the first tile column involves no FP8 x FP8 product: bitwise equal
    assert np.array_equal(L1[:, :cfg.nb], L2[:, :cfg.nb])
    assert np.mean(L1 == L2) > 0.5


# ------------------------------------------------------------------------------ exact constructions
@pytest.mark.parametrize("prec", [R.FP32, R.FP16, R.FP8, "mixed"])
@pytest.mark.parametrize("n,nb", [(512, 128), (1024, 256)])
def test_exactly_representable_factor_bit_for_bit(krr, prec, n, nb):
    L0, A = exact_lower_factor(11, n, nb, device="cuda")
    NT = n // nb
    if prec == "mixed":
        rng = np.random.default_rng(1)
        pmap = oracle_uniform(NT, R.FP32)
        for i in range(NT):
            for j in range(i):
                pmap[i, j] = rng.integers(0, 3)
    else:
        pmap = oracle_uniform(NT, prec)
    F = gpu_factor(krr, A, nb, pmap, preround=False)
    assert int(F.info.item()) == 0
    assert torch.equal(F.dense(), L0)
    # and the oracle agrees (same construction, same map)
    Lo, _, info = tile_cholesky_emulated(A.cpu().numpy(), nb, pmap, preround_a=False)
    assert info == 0 and np.array_equal(Lo, L0.cpu().numpy())


# ------------------------------------------------------------------------------ breakdown
def test_breakdown_reports_same_info_as_oracle(krr):
    # forced FP8 on a gamma = 1/p matrix makes the rounded matrix indefinite (SURVEY finding 2)
    cfg = scaled_config(CONFIGS["C1"], nb=128, n=512, p=500)
    A, _ = make_problem(cfg, device="cuda")
    pmap = oracle_uniform(cfg.NT, R.FP8)
    F = gpu_factor(krr, A, cfg.nb, pmap)
    _, _, info_o = tile_cholesky_emulated(A.cpu().numpy(), cfg.nb, pmap)
    info_g = int(F.info.item())
    assert info_o > 0 and info_g > 0
    assert (info_g - 1) // cfg.nb == (info_o - 1) // cfg.nb          # same tile column
    # an indefinite input: negative diagonal entry -> exact LAPACK info
    B = A.clone()
    B[300, 300] = -1.0
    F = gpu_factor(krr, B, cfg.nb, oracle_uniform(cfg.NT, R.FP32))
    assert int(F.info.item()) == 301


def test_argument_errors(krr):
    A = torch.eye(256, device="cuda")
    h = krr.uniform_map(2, krr.FP32)
    with pytest.raises(krr.KrrError):
        krr.potrf_mp(A[:250, :250].contiguous(), 128, h.cuda(), h)       # nb does not divide n
    bad = h.clone()
    bad[1, 0] = 7
    with pytest.raises(krr.KrrError):
        krr.potrf_mp(A, 128, bad.cuda(), bad)
    F = krr.potrf_mp(A, 128, h.cuda(), h)
    with pytest.raises(krr.KrrError):
        krr.potrs(F, torch.zeros((256, 40), device="cuda"))              # nrhs > 32
    torch.cuda.synchronize()
    assert torch.equal(F.dense(), torch.eye(256, dtype=torch.float64, device="cuda"))


@pytest.mark.parametrize("nrhs", [1, 3, 4, 8, 16, 32])
def test_potrs_every_nrhs_class(krr, nrhs):
    cfg = scaled_config(CONFIGS["C1"], nb=128, n=512, p=300)
    A, _ = make_problem(cfg, device="cuda")
    g = torch.Generator(device="cuda").manual_seed(nrhs)
    Y = torch.randn((cfg.n, nrhs), device="cuda", generator=g)
    F = gpu_factor(krr, A, cfg.nb, oracle_uniform(cfg.NT, R.FP32))
    alpha = krr.potrs(F, Y.clone())
    torch.cuda.synchronize()
    want = potrs_fp64(F.dense().cpu().numpy(), Y.cpu().numpy(), cfg.nb)
    assert relF(alpha.cpu().numpy().astype(np.float64), want) <= 1e-5
    # strided right-hand side (ldb > nrhs)
    big = torch.zeros((cfg.n, nrhs + 5), device="cuda")
    big[:, :nrhs] = Y
    krr.potrs(F, big[:, :nrhs])
    torch.cuda.synchronize()
    assert torch.equal(big[:, :nrhs], alpha) and float(big[:, nrhs:].abs().max()) == 0.0


@pytest.mark.parametrize("NT,nb", [(1, 256), (2, 256), (3, 640), (5, 512), (6, 512), (6, 256)])
def test_potrs_lookahead_depths(krr, NT, nb):
    """The solve's two-column lookahead at its edges: NT = 1, 2 (no internal streams), 3 (near and mid tiles only; nb = 640:
    five units per tile, the single-CTA factorisation path), 5 and 6 (bulk launches of one to three tiles on the streamed
    kernel, last columns without a mid / bulk part, near / mid tiles as K slices); tile columns of a megabyte and more take
    the lookahead, (6, 256) stays below that and runs column by column on the caller's stream.  Against the oracle's
    substitution with the same factor; repeatable bits."""
    cfg = scaled_config(CONFIGS["C1"], nb=nb, n=NT * nb, p=700)
    A, _ = make_problem(cfg, device="cuda")
    rng = np.random.default_rng(100 + NT)
    pmap = oracle_uniform(cfg.NT, R.FP32)
    for i in range(cfg.NT):
        for j in range(i):
            pmap[i, j] = rng.integers(0, 2)                 # FP32 / FP16 tiles
    F = gpu_factor(krr, A, nb, pmap)
    assert int(F.info.item()) == 0
    g = torch.Generator(device="cuda").manual_seed(7 * NT)
    Y = torch.randn((cfg.n, 16), device="cuda", generator=g)
    alpha = krr.potrs(F, Y.clone())
    torch.cuda.synchronize()
    want = potrs_fp64(F.dense().cpu().numpy(), Y.cpu().numpy(), nb)
    assert relF(alpha.cpu().numpy().astype(np.float64), want) <= 1e-5
    again = krr.potrs(F, Y.clone())
    torch.cuda.synchronize()
    assert torch.equal(again, alpha)


@pytest.mark.parametrize("nb,NT,nrhs", [(2048, 4, 16), (4096, 3, 8)])
def test_largest_tile_sizes(krr, nb, NT, nrhs):
    """The largest tile sizes the library accepts (nb <= 4096; the solved block of the solve must fit in shared memory:
    nrhs <= 16 at nb = 2048, <= 8 at nb = 4096): 16 and 32 sub-columns per diagonal tile, the streamed solve kernel with a
    ring cut down to what the solved block leaves.  FP32 / FP16 mosaic: info = 0, backward error of the factor as stored
    (checked with torch FP64 on the GPU), the solve against the oracle's substitution with the same factor, repeatable
    bits; all-FP32 map: backward error and alpha against the FP64 solution inside the north_star's 1e-6 / 1e-3 -- tiles
    above 1024 take the segmented-accumulation form of the panel product (the CTA-pair form gives
    3.6e-6 / 6.7e-4 at nb = 4096)."""
    n = nb * NT
    cfg = replace(scaled_config(CONFIGS["C2"], nb=nb, n=n, p=max(1024, n // 4)), nrhs=nrhs)
    A, Y = make_problem(cfg, device="cuda")
    A64 = torch.tril(A.double()) + torch.tril(A.double(), -1).T
    rng = np.random.default_rng(nb + NT)
    pmap = oracle_uniform(NT, R.FP32)
    for i in range(NT):
        for j in range(i):
            pmap[i, j] = rng.integers(0, 2)
    pmap[NT - 1, 0] = R.FP16                                  # both classes whatever the draw
    pmap[1, 0] = R.FP32
    F = gpu_factor(krr, A, nb, pmap)
    torch.cuda.synchronize()
    assert int(F.info.item()) == 0
    L = F.dense().double()
    assert float(torch.linalg.norm(L @ L.T - A64) / torch.linalg.norm(A64)) <= 5e-4
    alpha = krr.potrs(F, Y.clone())
    torch.cuda.synchronize()
    want = potrs_fp64(F.dense().cpu().numpy(), Y.cpu().numpy(), nb)
    assert relF(alpha.cpu().numpy().astype(np.float64), want) <= 1e-5
    again = krr.potrs(F, Y.clone())
    torch.cuda.synchronize()
    assert torch.equal(again, alpha)
    del L
    F32 = gpu_factor(krr, A, nb, oracle_uniform(NT, R.FP32))
    a32 = krr.potrs(F32, Y.clone())
    torch.cuda.synchronize()
    assert int(F32.info.item()) == 0
    xs = torch.linalg.solve(A64, Y.double())
    assert float(torch.linalg.norm(a32.double() - xs) / torch.linalg.norm(xs)) <= 5e-4
    L32 = F32.dense().double()
    assert float(torch.linalg.norm(L32 @ L32.T - A64) / torch.linalg.norm(A64)) <= 1e-6


def test_potrs_rejects_a_misaligned_factor(krr):
    import ctypes
    cfg = scaled_config(CONFIGS["C1"], nb=128, n=256, p=100)
    A, _ = make_problem(cfg, device="cuda")
    F = gpu_factor(krr, A, cfg.nb, oracle_uniform(cfg.NT, R.FP32))
    L = krr.lib()
    B = torch.zeros((cfg.n, 4), device="cuda")
    wsb = int(L.krr_potrs_workspace(cfg.n, cfg.nb, 4))
    ws = torch.empty(wsb + 1024, dtype=torch.uint8, device="cuda")
    wp = (ws.data_ptr() + 1023) // 1024 * 1024
    shifted = torch.empty(F.payload.numel() + 16, dtype=torch.uint8, device="cuda")
    base = shifted.data_ptr()
    off = (8 - base % 16) % 16                                # an address that is 8 modulo 16
    rc = L.krr_potrs(ctypes.c_void_p(base + off), ctypes.c_void_p(F.scales.data_ptr()), ctypes.c_void_p(F.d_map.data_ptr()),
                     ctypes.c_void_p(F.h_map.data_ptr()), cfg.n, cfg.nb, ctypes.c_void_p(B.data_ptr()), 4, 4,
                     ctypes.c_void_p(wp), wsb, None)
    assert rc == -1 and krr.last_launch_count() == 0


@pytest.mark.parametrize("nb", [128, 512])
@pytest.mark.parametrize("nrhs", [1, 5, 8, 16, 32])
def test_potrs_mixed_mosaic_every_nrhs_class(krr, nrhs, nb):
    """The solve kernels read FP32, FP16 and FP8 tiles through precision-specific loops: a random mosaic, NT = 8, against
    the oracle's substitution with the SAME dequantised factor.  nb = 128: column by column with the r01 kernels (a
    one-column-per-lane variant in the backward sweep); nb = 512: the two-column lookahead, every update on the streamed
    kernel (bulk launches, near / mid tiles as K slices, partial sums gathered by the stage kernel)."""
    cfg = replace(scaled_config(CONFIGS["S1"], nb=nb, n=8 * nb, p=768), genotype="maf", gamma_scale=4.0)
    A, _ = make_problem(cfg, device="cuda")
    rng = np.random.default_rng(11)
    pmap = oracle_uniform(cfg.NT, R.FP32)
    for i in range(cfg.NT):
        for j in range(i):
            pmap[i, j] = rng.integers(0, 3)
    assert len(set(pmap[np.tril_indices(cfg.NT, -1)].tolist())) == 3
    F = gpu_factor(krr, A, cfg.nb, pmap)
    assert int(F.info.item()) == 0
    g = torch.Generator(device="cuda").manual_seed(100 + nrhs)
    Y = torch.randn((cfg.n, nrhs), device="cuda", generator=g)
    alpha = krr.potrs(F, Y.clone())
    torch.cuda.synchronize()
    want = potrs_fp64(F.dense().cpu().numpy(), Y.cpu().numpy(), cfg.nb)
    assert relF(alpha.cpu().numpy().astype(np.float64), want) <= 1e-5
    again = krr.potrs(F, Y.clone())                      # fixed summation order: the same bits every time
    torch.cuda.synchronize()
    assert torch.equal(again, alpha)


def test_associate_host_matches_device_path(krr):
    cfg = scaled_config(CONFIGS["S1"], nb=128, n=1024, p=768)
    A, Y = make_problem(cfg, device="cuda")
    d_map, _, _, _ = krr.precision_map(A, cfg.nb, cfg.eps_target, cfg.allowed)
    h = d_map.cpu()
    F = krr.potrf_mp(A, cfg.nb, d_map, h)
    alpha = krr.potrs(F, Y.clone())
    hA, hY = A.cpu().pin_memory(), Y.cpu().pin_memory()
    a2, m2, info, _ = krr.associate_host(hA, cfg.nb, hY, cfg.eps_target, cfg.allowed)
    assert info == 0 and torch.equal(m2, h) and torch.equal(a2, alpha.cpu())
    a3, m3, info3, _ = krr.associate_host(hA, cfg.nb, hY, force_prec=krr.FP32)
    assert info3 == 0 and int((m3[np.tril_indices(cfg.NT)] != 0).sum()) == 0


# ------------------------------------------------------------------------------ badly scaled input
@pytest.mark.parametrize("scaling", ["tile_rows_pow2", "smooth"])
@pytest.mark.parametrize("prec", [R.FP32, R.FP16])
def test_diagonally_scaled_matrix(krr, scaling, prec):
    """A = D A0 D with D spanning 2^-12 .. 2^12 (the dynamic range of the FP32-class path, whose operands reach the
    tensor cores as FP16 hi / lo images): the tile rows are equilibrated by powers of two on entry ("Dynamic
    range"), so the factor is as accurate RELATIVE TO EVERY ROW'S OWN SCALE as for the unscaled matrix -- measured in the
    equilibrated norm ||D^-1 (A - L L^T) D^-1||_F / ||A0||_F, where a global image scale loses the small rows.
    (All-FP16 map: D spans 2^-4 .. 2^4 only -- beyond that the FP16 STORAGE format itself runs out of range, whatever
    the arithmetic: entries of A below 6e-8 round to zero and the oracle breaks down as well.)"""
    cfg = scaled_config(CONFIGS["C1"], nb=256, n=2048, p=1000)
    A0, Y = make_problem(cfg, device="cuda")
    n, nb = cfg.n, cfg.nb
    i = np.arange(n)
    span = 12.0 if prec == R.FP32 else 4.0
    if scaling == "tile_rows_pow2":
        d = 2.0 ** (np.round(2.0 * span * (i // nb) / (cfg.NT - 1)) - span)    # one power of two per tile row
    else:
        d = 2.0 ** (2.0 * span * i / (n - 1) - span) * (1.0 + 0.3 * np.sin(i))   # smooth, up to a factor ~ 8 inside a tile
    An = (d[:, None] * A0.cpu().numpy().astype(np.float64) * d[None, :]).astype(np.float32)
    An = np.tril(An) + np.tril(An, -1).T
    A = torch.from_numpy(An).cuda()
    pmap = oracle_uniform(cfg.NT, prec)
    F = gpu_factor(krr, A, nb, pmap)
    assert int(F.info.item()) == 0
    Lo, _, info = tile_cholesky_emulated(An, nb, pmap)
    assert info == 0
    Lg = F.dense().cpu().numpy()
    dinv = 1.0 / d
    A64 = An.astype(np.float64)
    scaled_bwd = lambda L: float(np.linalg.norm(dinv[:, None] * (A64 - L @ L.T) * dinv[None, :]) /
                                 np.linalg.norm(dinv[:, None] * A64 * dinv[None, :]))
    bg, bo = scaled_bwd(Lg), scaled_bwd(Lo)
    lit = relF(dinv[:, None] * Lg, dinv[:, None] * Lo)
    print(f"scaled {scaling} prec {prec}: equilibrated backward gpu {bg:.3e} oracle {bo:.3e} relF(D^-1 L) {lit:.3e}")
    if prec == R.FP32:
        assert bg <= 1e-6 and lit <= 1e-4
    else:
        assert bg <= 5e-4 and abs(bg - bo) <= 0.05 * bo
    # the plain (unscaled-norm) criteria hold as well
    assert backward_error(An, Lg) <= (1e-6 if prec == R.FP32 else 5e-4)
    # and the solve with the scaled factor: against the oracle's substitution with the same factor
    Ys = torch.from_numpy((d[:, None] * Y.cpu().numpy()).astype(np.float32)).cuda()
    alpha = krr.potrs(F, Ys.clone())
    torch.cuda.synchronize()
    ref = potrs_fp64(Lg, Ys.cpu().numpy(), nb)
    err = np.linalg.norm(d[:, None] * (alpha.cpu().numpy().astype(np.float64) - ref)) / np.linalg.norm(d[:, None] * ref)
    assert err <= 1e-5

"""The seeded input generators: determinism, distributions, and the structure SURVEY 8(d) states."""
import numpy as np
import torch

from krr_inputs import CONFIGS, genotypes, kernel_matrix, phenotypes, make_problem, scaled_config
from krr_inputs.synth import maf, mix64


def test_mix64_known_values_and_wraparound():
    x = torch.tensor([0, 1, -1, 2 ** 62], dtype=torch.int64)
    h = mix64(x)
    # splitmix64 of 0 (first output of the generator seeded with 0)
    assert int(h[0]) & ((1 << 64) - 1) == 0xE220A8397B1DCDAF
    assert len(set(h.tolist())) == 4


def test_genotypes_deterministic_and_blockwise_consistent():
    G = genotypes(7, 64, 50, "maf")
    assert G.dtype == torch.int8 and set(np.unique(G.numpy())) <= {0, 1, 2}
    G2 = torch.cat([genotypes(7, 64, 50, "maf", row0=0, rows=20),
                    genotypes(7, 64, 50, "maf", row0=20, rows=44)])
    assert torch.equal(G, G2)
    assert not torch.equal(G, genotypes(8, 64, 50, "maf"))


def test_maf_distribution():
    n, p = 4000, 200
    G = genotypes(3, n, p, "maf").to(torch.float64)
    m = maf(3, p)
    assert 0.05 <= float(m.min()) and float(m.max()) < 0.5
    freq = G.mean(dim=0) / 2.0
    assert float((freq - m).abs().max()) < 0.03
    U = genotypes(3, n, p, "uniform").to(torch.float64)
    for v in (0, 1, 2):
        assert abs(float((U == v).double().mean()) - 1 / 3) < 0.01


def test_kernel_matrix_definition_and_structure():
    cfg = scaled_config(CONFIGS["C1"], nb=32, n=256, p=1000)
    G = genotypes(cfg.seed, cfg.n, cfg.p)
    A = kernel_matrix(G, cfg.gamma, cfg.lam)
    Gd = G.to(torch.float64)
    i, j = 17, 203
    d2 = float(((Gd[i] - Gd[j]) ** 2).sum())
    assert abs(float(A[i, j]) - np.exp(-cfg.gamma * d2)) < 1e-7
    assert torch.equal(A, A.t())
    assert float(A[5, 5]) == float(np.float32(1.0 + cfg.lam))
    off = A[~torch.eye(cfg.n, dtype=torch.bool)]
    assert abs(float(off.mean()) - 0.4815) < 0.01          # mean 0.4815, sd 0.015 at p=1000
    assert 0.008 < float(off.std()) < 0.03
    cu = scaled_config(CONFIGS["C5"], nb=32, n=256, p=2000)
    Au, _ = make_problem(cu)
    offu = Au[~torch.eye(cu.n, dtype=torch.bool)]
    assert abs(float(offu.mean()) - np.exp(-4.0 / 3.0)) < 0.01


def test_phenotypes_standard_normal():
    Y = phenotypes(1, 20000, 4)
    assert Y.shape == (20000, 4) and Y.dtype == torch.float32
    assert abs(float(Y.mean())) < 0.02 and abs(float(Y.std()) - 1.0) < 0.02
    assert torch.equal(Y, phenotypes(1, 20000, 4))


def test_lower_tile_packing_matches_dense_matrix():
    from krr_inputs import make_problem_lower_tiles
    cfg = scaled_config(CONFIGS["C4"], nb=32, n=352, p=300)       # NT = 11: ragged against the 8-row batches
    A, Y = make_problem(cfg)
    At, Yt = make_problem_lower_tiles(cfg)
    NT, nb = cfg.NT, cfg.nb
    assert At.numel() == NT * (NT + 1) // 2 * nb * nb and torch.equal(Y, Yt)
    T = At.reshape(-1, nb, nb)
    slot = 0
    for j in range(NT):
        for i in range(j, NT):
            assert torch.equal(T[slot], A[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb]), (i, j)
            slot += 1

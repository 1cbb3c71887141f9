"""Launch-geometry limits: sizes at which an index that used to sit in gridDim.y (limit 65535) passes it.

  * krr_precision_map at NT = 363 (nb = 128, n = 46464): NT (NT + 1) / 2 = 66066 tile slots;
  * krr_build with the IBS kernel at n = 65536 rows (BASELINE.json config 3's patient count);
  * krr_potrf_mp / krr_potrs at NT = 1024, the largest tile count the library accepts (nb = 128, n = 131072).

Expected values come from independent torch FP64 code on sampled tiles / entries (checking only).
"""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def krr():
    from paper_2409_01712_b200 import build
    build.build()
    import paper_2409_01712_b200 as k
    k.lib()
    return k


def test_precision_map_with_more_than_65535_tile_slots(krr):
    nb, NT = 128, 363
    n = nb * NT
    g = torch.Generator(device="cuda").manual_seed(5)
    A = torch.empty((n, n), dtype=torch.float32, device="cuda")
    for r0 in range(0, n, 4096):                                   # scale the rows so that tile norms differ by orders
        r1 = min(n, r0 + 4096)
        A[r0:r1] = torch.randn((r1 - r0, n), generator=g, device="cuda") * (10.0 ** (-3.0 * r0 / n))
    eps = 3e-2
    d_map, norms, amax, fro = krr.precision_map(A, nb, eps, (0, 1, 2))
    torch.cuda.synchronize()
    m = d_map.cpu().numpy()
    # ||A||_F of the symmetric matrix the lower tiles define, FP64
    tot = 0.0
    for r0 in range(0, n, 4096):
        r1 = min(n, r0 + 4096)
        blk = A[r0:r1, :r1].double()
        i0, i1 = r0 // nb, r1 // nb
        for i in range(i0, i1):                                    # tiles of this tile row: diagonal once, the others twice
            row = blk[(i - i0) * nb:(i - i0 + 1) * nb]
            tot += 2.0 * float((row[:, :i * nb] ** 2).sum()) + float((row[:, i * nb:(i + 1) * nb] ** 2).sum())
    f = tot ** 0.5
    assert abs(float(fro) - f) <= 1e-10 * f
    rhs = eps * f / NT
    u = {0: 2.0 ** -24, 1: 2.0 ** -11, 2: 2.0 ** -4}
    rng = np.random.default_rng(0)
    seen = set()
    for _ in range(400):
        i = int(rng.integers(1, NT)); j = int(rng.integers(0, i))
        t = float(torch.linalg.norm(A[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb].double()))
        assert abs(float(norms[i, j]) - t) <= 2e-7 * t
        want = 2 if t * u[2] <= rhs else (1 if t * u[1] <= rhs else 0)
        if min(abs(t * u[2] - rhs), abs(t * u[1] - rhs)) > 1e-6 * rhs:      # not within rounding of a threshold
            assert m[i, j] == want, (i, j)
        seen.add(int(m[i, j]))
    assert len(seen) >= 2                                          # the sample exercises more than one class
    assert all(m[i, i] == 0 for i in range(NT)) and m[0, 1] == 255
    assert float(amax[NT - 1, 3]) == float(A[(NT - 1) * nb:, 3 * nb:4 * nb].abs().max())
    # the last slots (beyond 65535) are really written
    assert m[NT - 1, NT - 2] in (0, 1, 2) and float(norms[NT - 1, NT - 1]) > 0.0


def test_ibs_build_with_65536_patients(krr):
    n, p, nb = 65536, 48, 1024
    g = torch.Generator(device="cuda").manual_seed(9)
    G = torch.randint(0, 3, (n, p), dtype=torch.int8, device="cuda", generator=g)
    lam = 0.25
    At = krr.krr_build(G, 0.0, lam, nb, tiled_lower=True, flags=krr.FLAG_KERNEL_IBS)
    torch.cuda.synchronize()
    NT = n // nb
    T = At.reshape(-1, nb, nb)
    Gd = G.double()
    for (i, j) in [(0, 0), (1, 0), (NT - 1, 0), (NT - 1, NT - 1), (NT - 1, 17), (40, 39)]:
        slot = krr.tile_slot(NT, i, j)
        gi, gj = Gd[i * nb:(i + 1) * nb], Gd[j * nb:(j + 1) * nb]
        # alleles identical by state: 2 - |a - b| per locus, over 2 p alleles (R17)
        want = (2.0 - (gi[:, None, :] - gj[None, :, :]).abs()).sum(dim=2) / (2.0 * p)
        if i == j:
            want = want + lam * torch.eye(nb, dtype=torch.float64, device="cuda")
            got = torch.tril(T[slot].double())
            want = torch.tril(want)
        else:
            got = T[slot].double()
        assert float((got - want).abs().max()) <= 2e-7, (i, j)


def test_largest_tile_count(krr):
    """NT = 1024, the largest tile count the library accepts (nb = 128, n = 131072: 524800 lower tiles, 34 GB of packed
    FP32 tiles; the host-built launch sequence has 1024 tile columns).  All-FP32 map: info = 0; sampled tiles of L L^T
    against A (the last diagonal tile sums 1024 tile products) and sampled row blocks of A alpha = Y, both with torch
    FP64 on the GPU (checking only)."""
    from dataclasses import replace
    from krr_inputs import CONFIGS, make_problem_lower_tiles
    nb, NT = 128, 1024
    n = nb * NT
    cfg = replace(CONFIGS["C4"], nb=nb, n=n, p=8192, nrhs=4)
    At, Y = make_problem_lower_tiles(cfg, device="cuda")
    h = krr.uniform_map(NT, krr.FP32)
    F = krr.potrf_mp(At, nb, h.cuda(), h, flags=krr.FLAG_PREROUND_A | krr.FLAG_A_TILED_LOWER, n=n)
    alpha = krr.potrs(F, Y.clone())
    torch.cuda.synchronize()
    assert int(F.info.item()) == 0
    T = At.reshape(-1, nb, nb)

    def a_tile(i, k):                                            # tile (i, k) of the symmetric matrix, FP64
        t = T[krr.tile_slot(NT, max(i, k), min(i, k))].double()
        if k > i:
            return t.T
        return t if i != k else torch.tril(t) + torch.tril(t, -1).T

    for (i, j) in [(NT - 1, NT - 1), (NT - 1, 0), (700, 699)]:
        acc = torch.zeros((nb, nb), dtype=torch.float64, device="cuda")
        for k in range(j + 1):
            acc += F.tile(i, k) @ F.tile(j, k).T
        a = a_tile(i, j)
        assert float(torch.linalg.norm(acc - a) / torch.linalg.norm(a)) <= 5e-5, (i, j)      # measured 1.4e-5 (last diagonal tile)
    for i in (0, NT - 1):
        r = Y[i * nb:(i + 1) * nb].double().clone()
        for k in range(NT):
            r -= a_tile(i, k) @ alpha[k * nb:(k + 1) * nb].double()
        assert float(torch.linalg.norm(r) / torch.linalg.norm(Y[i * nb:(i + 1) * nb].double())) <= 1e-3, i   # measured 1e-4 .. 3.5e-4

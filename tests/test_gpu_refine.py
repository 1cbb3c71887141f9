"""GPU parity of krr_refine (R19; SURVEY section 8(c) C4 / C5' rows, 8(f) NEXT-4) against oracle.solve.refine.

The oracle runs on its own emulated factor and its own starting point (no value of the CUDA path enters it); the two
factors differ by storage-rounding flips, so after s steps the iterates are compared through what is unique -- the
error against the FP64 solution, step by step -- and the residual kernel itself through a case where every element of
the residual matters: with an FP32 map one step from a random starting point must land on the FP64 solution.
"""
from dataclasses import replace

import numpy as np
import pytest
import torch

from helpers import solve_residual
from krr_inputs import CONFIGS, make_problem, make_problem_lower_tiles, scaled_config
from oracle import rounding as R
from oracle.cholesky import tile_cholesky_emulated
from oracle.precision_map import uniform_map
from oracle.solve import potrs_fp64, refine, solve_fp64

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def krr():
    from paper_2409_01712_b200 import build
    build.build()
    import paper_2409_01712_b200 as k
    k.lib()
    return k


def rel(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


@pytest.mark.parametrize("n,nb,nrhs", [(1280, 256, 1), (1024, 128, 5), (4096, 512, 16), (2048, 256, 32)])
def test_one_step_from_a_random_start_with_an_fp32_map(krr, n, nb, nrhs):
    """FP32 map: (L L^T)^-1 is A^-1 to FP32 accuracy, so X_1 = X_0 + A^-1 (Y - A X_0) is the solution whatever X_0 --
    unless an element of the residual is wrong.  The strict upper triangle of the dense input is poisoned with NaN
    (only the lower tiles, and the lower triangles of the diagonal blocks, may be read); a second step changes
    nothing beyond FP32 noise; the norms are those of the oracle's residuals (same X_0: a seeded input)."""
    cfg = replace(scaled_config(CONFIGS["C2"], nb=nb, n=n, p=max(256, n // 4)), nrhs=nrhs)
    A, Y = make_problem(cfg, device="cuda")
    h = krr.uniform_map(cfg.NT, krr.FP32)
    F = krr.potrf_mp(A, nb, h.cuda(), h)
    g = torch.Generator(device="cpu").manual_seed(n + nrhs)
    X0 = torch.randn((n, nrhs), generator=g, dtype=torch.float32)
    An, Yn = A.cpu().numpy().astype(np.float64), Y.cpu().numpy().astype(np.float64)
    xstar = solve_fp64(An, Yn, nb)
    Ap = A.clone()
    Ap[torch.triu(torch.ones_like(Ap, dtype=torch.bool), 1)] = float("nan")
    X, norms = krr.refine(Ap, F, Y, X0.cuda(), 2)
    torch.cuda.synchronize()
    norms = norms.cpu().numpy()
    assert np.all(np.isfinite(norms))
    assert rel(X.cpu().numpy().astype(np.float64), xstar) <= 2e-5
    X1, n1 = krr.refine(Ap, F, Y, X0.cuda(), 1)
    assert rel(X1.cpu().numpy().astype(np.float64), xstar) <= 1e-4
    r0 = (Yn - An @ X0.numpy().astype(np.float64)).astype(np.float32).astype(np.float64)
    assert abs(norms[0] - np.linalg.norm(r0)) <= 1e-6 * np.linalg.norm(r0)
    assert float(n1[0]) == norms[0]                                          # deterministic
    assert norms[1] <= 1e-3 * norms[0] and norms[2] <= 1e-4 * norms[0]
    # steps = 0: X untouched, one norm
    Xc = X0.cuda()
    X00, n0 = krr.refine(Ap, F, Y, Xc, 0)
    assert torch.equal(X00.cpu(), X0) and n0.numel() == 1 and float(n0[0]) == norms[0]


@pytest.mark.parametrize("n,nb,nrhs", [(2048, 256, 4), (4096, 1024, 16)])
def test_steps_in_one_call_equal_one_call_per_step(krr, n, nb, nrhs):
    """krr_refine / krr_pcg compute the inverses of the diagonal tiles in their first solve and keep them in the workspace
    for the later ones (the factor does not change inside a call): three steps in one call and three calls of one step
    (each of which prepares the workspace again) give the same bits; PCG: the iterates of a 3-iteration call are repeatable
    and its first iterate is that of a 1-iteration call."""
    cfg = replace(scaled_config(CONFIGS["C2"], nb=nb, n=n, p=max(256, n // 4)), nrhs=nrhs)
    A, Y = make_problem(cfg, device="cuda")
    h = krr.uniform_map(cfg.NT, krr.FP16)
    F = krr.potrf_mp(A, nb, h.cuda(), h)
    X0 = krr.potrs(F, Y.clone())
    Xa, na = krr.refine(A, F, Y, X0.clone(), 3)
    Xb = X0.clone()
    nbs = []
    for _ in range(3):
        Xb, n1 = krr.refine(A, F, Y, Xb, 1)
        nbs.append(float(n1[0]))
    torch.cuda.synchronize()
    assert torch.equal(Xa, Xb)
    assert [float(v) for v in na[:3]] == nbs
    Pa, pa = krr.pcg(A, F, Y, X0.clone(), 3)
    Pb, pb = krr.pcg(A, F, Y, X0.clone(), 3)
    P1, p1 = krr.pcg(A, F, Y, X0.clone(), 1)
    torch.cuda.synchronize()
    assert torch.equal(Pa, Pb) and torch.equal(pa, pb)
    assert float(p1[0]) == float(pa[0]) and float(p1[1]) == float(pa[1])


@pytest.mark.parametrize("prec,tiled", [("fp16", False), ("fp16", True), ("fp8", False)])
def test_refinement_under_low_precision_maps_against_the_oracle(krr, prec, tiled):
    """All-FP16 map (C4's map by the rule) and the C5' map (tile column 0 FP32, the rest FP8): raw alpha misses the
    1e-3 of north_star, two steps meet it; the error after every step stays within a factor of the oracle's (two
    factors that differ by rounding flips contract at the same rate), the residual norms likewise."""
    nb = 128
    if prec == "fp16":
        cfg = scaled_config(CONFIGS["C4"], nb=nb, n=2048, p=512)
    else:
        cfg = scaled_config(CONFIGS["C5p"], nb=nb, n=2048, p=400)
    if tiled:
        At, Y = make_problem_lower_tiles(cfg, device="cuda")
        A = None
    else:
        A, Y = make_problem(cfg, device="cuda")
    NT = cfg.NT
    h = krr.uniform_map(NT, krr.FP16 if prec == "fp16" else krr.FP8)
    flags = krr.FLAG_PREROUND_A
    if prec == "fp8":
        h[1:, 0] = krr.FP32
        flags = 0
    if tiled:
        F = krr.potrf_mp(At, nb, h.cuda(), h, flags=flags | krr.FLAG_A_TILED_LOWER, n=cfg.n)
    else:
        F = krr.potrf_mp(A, nb, h.cuda(), h, flags=flags)
    X0 = krr.potrs(F, Y.clone())
    torch.cuda.synchronize()
    assert int(F.info.item()) == 0
    if tiled:
        Ad, _ = make_problem(cfg, device="cuda")                              # the same matrix, dense, for the oracle
        An = Ad.cpu().numpy().astype(np.float64)
    else:
        An = A.cpu().numpy().astype(np.float64)
    Yn = Y.cpu().numpy().astype(np.float64)
    xstar = solve_fp64(An, Yn, nb)
    Lo, sc, info = tile_cholesky_emulated(An, nb, h.numpy().copy(), preround_a=(prec == "fp16"))
    assert info == 0
    o0 = potrs_fp64(Lo, Yn, nb)
    err_g = [rel(X0.cpu().numpy().astype(np.float64), xstar)]
    err_o = [rel(o0, xstar)]
    assert err_g[0] > 1e-3 and err_o[0] > 1e-3                               # raw alpha misses the tolerance
    o, on = refine(An, Lo, Yn, o0, nb, 3)
    Xg = X0.clone()
    gn = []
    for s in range(3):
        Xg, nn = krr.refine(At if tiled else A, F, Y, Xg, 1, tiled_lower=tiled)
        gn.append(float(nn[0]))
        err_g.append(rel(Xg.cpu().numpy().astype(np.float64), xstar))
        err_o.append(rel(refine(An, Lo, Yn, o0, nb, s + 1)[0], xstar))
    gn.append(float(nn[1]))
    for s in range(1, 4):
        assert err_g[s] <= 3.0 * err_o[s] + 3e-6, (s, err_g, err_o)
    assert err_g[2] <= 1e-3 and err_g[3] <= 1e-4                             # north_star's alpha tolerance, met
    for s in range(3):
        assert 0.33 * on[s] <= gn[s] <= 3.0 * on[s] + 1e-4, (s, gn, on)
    # three steps in one call = three calls of one step (same arithmetic, same order)
    X3, n3 = krr.refine(At if tiled else A, F, Y, X0.clone(), 3, tiled_lower=tiled)
    assert torch.equal(X3, Xg)
    assert [float(v) for v in n3] == gn


def test_refine_rejects_bad_arguments(krr):
    cfg = replace(scaled_config(CONFIGS["C2"], nb=128, n=512, p=256), nrhs=4)
    A, Y = make_problem(cfg, device="cuda")
    h = krr.uniform_map(cfg.NT, krr.FP32)
    F = krr.potrf_mp(A, 128, h.cuda(), h)
    L = krr.lib()
    assert int(L.krr_refine_workspace(500, 128, 4)) == 0
    assert int(L.krr_refine_workspace(512, 128, 33)) == 0
    with pytest.raises(krr.KrrError):
        krr.refine(A, F, Y, Y.clone(), 65)
    with pytest.raises(krr.KrrError):
        krr.refine(A, F, Y, Y.clone(), -1)


def test_full_size_refinement_under_the_half_precision_map(krr):
    """C3's matrix with every off-diagonal tile in FP16 (config C3h, n = 65536): one step takes the residual of the raw
    solve (5.7e-7 of ||A|| ||alpha||) down to the floor the FP32 storage of alpha sets (~ 1e-7), where the second step
    leaves it (independent torch-FP64 residual, tests/helpers.py); the norms the library reports agree with it."""
    cfg = CONFIGS["C3h"]
    A, Y = make_problem(cfg, device="cuda")
    h = krr.uniform_map(cfg.NT, krr.FP16)
    F = krr.potrf_mp(A, cfg.nb, h.cuda(), h)
    X0 = krr.potrs(F, Y.clone())
    torch.cuda.synchronize()
    assert int(F.info.item()) == 0
    res0 = solve_residual(A, X0, Y)
    X2, norms = krr.refine(A, F, Y, X0.clone(), 2)
    torch.cuda.synchronize()
    res2 = solve_residual(A, X2, Y)
    norms = norms.cpu().numpy()
    assert norms[1] < 0.25 * norms[0] and norms[2] < 1.5 * norms[1]
    assert res2 < 0.25 * res0 and res2 <= 2e-7
    # the reported norm of the first residual against the independent evaluation
    from helpers import fro_norm_sym
    want0 = res0 * fro_norm_sym(A) * float(torch.linalg.norm(X0.to(torch.float64)))
    assert abs(norms[0] - want0) <= 1e-4 * want0


# ---- krr_pcg (R20) ----
@pytest.mark.parametrize("n,nb,nrhs", [(1280, 256, 3), (2048, 256, 16), (1024, 128, 32)])
def test_pcg_with_an_fp32_map_from_a_random_start(krr, n, nb, nrhs):
    """M^-1 A = I to FP32 accuracy: the first step lands on the solution -- unless an element of the residual, of
    q = A p, of an inner product or of an update is wrong.  NaN above the diagonal as in the refinement test."""
    cfg = replace(scaled_config(CONFIGS["C2"], nb=nb, n=n, p=max(256, n // 4)), nrhs=nrhs)
    A, Y = make_problem(cfg, device="cuda")
    h = krr.uniform_map(cfg.NT, krr.FP32)
    F = krr.potrf_mp(A, nb, h.cuda(), h)
    g = torch.Generator(device="cpu").manual_seed(3 * n + nrhs)
    X0 = torch.randn((n, nrhs), generator=g, dtype=torch.float32)
    An, Yn = A.cpu().numpy().astype(np.float64), Y.cpu().numpy().astype(np.float64)
    xstar = solve_fp64(An, Yn, nb)
    Ap = A.clone()
    Ap[torch.triu(torch.ones_like(Ap, dtype=torch.bool), 1)] = float("nan")
    X1, n1 = krr.pcg(Ap, F, Y, X0.cuda(), 1)
    X2, n2 = krr.pcg(Ap, F, Y, X0.cuda(), 2)
    torch.cuda.synchronize()
    assert rel(X1.cpu().numpy().astype(np.float64), xstar) <= 1e-4
    assert rel(X2.cpu().numpy().astype(np.float64), xstar) <= 1e-6
    n2 = n2.cpu().numpy()
    r0 = Yn - An @ X0.numpy().astype(np.float64)
    assert abs(n2[0] - np.linalg.norm(r0)) <= 1e-9 * np.linalg.norm(r0)
    assert n2[1] <= 1e-3 * n2[0] and n2[2] <= 1e-2 * n2[1] and float(n1[1]) == n2[1]
    X00, n0 = krr.pcg(Ap, F, Y, X0.cuda(), 0)
    assert torch.equal(X00.cpu(), X0) and float(n0[0]) == n2[0]


@pytest.mark.parametrize("prec,tiled", [("fp16", False), ("fp16", True), ("fp8", False)])
def test_pcg_under_low_precision_maps_against_the_oracle(krr, prec, tiled):
    """Step by step against oracle.solve.pcg on the oracle's own emulated factor: errors within a factor of the
    oracle's (plus FP32 roundoff), residual norms likewise; four steps meet north_star's 1e-3 with room to spare."""
    from oracle.solve import pcg
    nb = 128
    cfg = scaled_config(CONFIGS["C4"], nb=nb, n=2048, p=512) if prec == "fp16" else \
        scaled_config(CONFIGS["C5p"], nb=nb, n=2048, p=400)
    Ad, Y = make_problem(cfg, device="cuda")
    A = make_problem_lower_tiles(cfg, device="cuda")[0] if tiled else Ad
    h = krr.uniform_map(cfg.NT, krr.FP16 if prec == "fp16" else krr.FP8)
    flags = krr.FLAG_PREROUND_A
    if prec == "fp8":
        h[1:, 0] = krr.FP32
        flags = 0
    F = krr.potrf_mp(A, nb, h.cuda(), h, flags=flags | (krr.FLAG_A_TILED_LOWER if tiled else 0), n=cfg.n)
    X0 = krr.potrs(F, Y.clone())
    torch.cuda.synchronize()
    assert int(F.info.item()) == 0
    An, Yn = Ad.cpu().numpy().astype(np.float64), Y.cpu().numpy().astype(np.float64)
    xstar = solve_fp64(An, Yn, nb)
    Lo, sc, info = tile_cholesky_emulated(An, nb, h.numpy().copy(), preround_a=(prec == "fp16"))
    assert info == 0
    o0 = potrs_fp64(Lo, Yn, nb)
    for k in (1, 2, 4):
        Xg, gn = krr.pcg(A, F, Y, X0.clone(), k, tiled_lower=tiled)
        xo, on = pcg(An, Lo, Yn, o0, nb, k)
        eg, eo = rel(Xg.cpu().numpy().astype(np.float64), xstar), rel(xo, xstar)
        assert eg <= 3.0 * eo + 3e-6, (k, eg, eo)
        gn = gn.cpu().numpy()
        for s in range(k + 1):
            assert 0.33 * on[s] <= gn[s] <= 3.0 * on[s] + 1e-5, (k, s, gn, on)
    assert eg <= 1e-5


def test_pcg_converges_where_refinement_diverges(krr):
    """The factor of K + lambda I as the preconditioner of K + (lambda + 0.2) I: most eigenvalues of M^-1 A lie above
    2, so the stationary iteration grows the error while CG converges -- as on C4 at full size (R20), here
    at a size the oracle checks step by step."""
    from oracle.solve import pcg
    nb = 128
    cfg = replace(scaled_config(CONFIGS["C2"], nb=nb, n=1536, p=384), nrhs=8)
    A, Y = make_problem(replace(cfg, lam=cfg.lam + 0.2), device="cuda")       # the system
    A2, _ = make_problem(cfg, device="cuda")                                  # what is factored
    h = krr.uniform_map(cfg.NT, krr.FP32)
    F = krr.potrf_mp(A2, nb, h.cuda(), h)
    X0 = krr.potrs(F, Y.clone())
    An, A2n, Yn = (t.cpu().numpy().astype(np.float64) for t in (A, A2, Y))
    xstar = solve_fp64(An, Yn, nb)
    e0 = rel(X0.cpu().numpy().astype(np.float64), xstar)
    Xr, rn = krr.refine(A, F, Y, X0.clone(), 8)
    assert rel(Xr.cpu().numpy().astype(np.float64), xstar) > 5.0 * e0 and float(rn[8]) > 5.0 * float(rn[0])
    Lo = np.linalg.cholesky(A2n)
    o0 = potrs_fp64(Lo, Yn, nb)
    for k in (2, 6, 12):
        Xg, gn = krr.pcg(A, F, Y, X0.clone(), k)
        xo, on = pcg(An, Lo, Yn, o0, nb, k)
        eg, eo = rel(Xg.cpu().numpy().astype(np.float64), xstar), rel(xo, xstar)
        assert eg <= 2.0 * eo + 3e-6, (k, eg, eo)
    assert eg <= 1e-5 and eg < 1e-4 * e0

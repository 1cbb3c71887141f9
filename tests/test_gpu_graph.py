"""CUDA-graph replay of the tile-DAG launch sequence (include/krr_mp.h: krr_graph_*; BASELINE.json north_star:
"a single-GPU tile-DAG scheduler with lookahead, run as CUDA graphs").  A replay launches the same kernels with the
same arguments and dependencies as the direct calls, so every result must be bit-identical to theirs; the direct
calls are the ones tests/test_gpu_parity.py holds against the oracle."""
import pytest
import torch

from krr_inputs import CONFIGS, make_problem, scaled_config

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def krr():
    from paper_2409_01712_b200 import build
    build.build()
    import paper_2409_01712_b200 as k
    k.lib()
    return k


def direct(krr, A, Y, nb, d_map, h_map, flags):
    F = krr.potrf_mp(A, nb, d_map, h_map, flags=flags)
    n_potrf = krr.last_launch_count()
    B = Y.clone()
    krr.potrs(F, B)
    n_potrs = krr.last_launch_count()
    torch.cuda.synchronize()
    return F, B, n_potrf + n_potrs


def record(krr, A, B, nb, d_map, h_map, flags):
    ws = krr.potrs_workspace(A.shape[0], nb, B.shape[1], A.device)
    krr.graph_begin()
    F = krr.potrf_mp(A, nb, d_map, h_map, flags=flags)
    krr.potrs(F, B, ws=ws)
    return krr.graph_end(keep=(A, B, d_map, F, ws)), F


# NT = 8: lookahead on three internal streams (mixed FP32 / FP16 map by the rule); NT = 2: the in-order path on the
# caller's stream; forced FP8 below column 0: block-scaled MMAs, split flags, amax pass.
@pytest.mark.parametrize("name,nb,n,p,force", [("S1", 256, 2048, 1536, None), ("C1", 512, 1024, 500, None),
                                               ("C5", 256, 2048, 400, "fp8")])
def test_replay_is_bit_identical_to_direct_calls(krr, name, nb, n, p, force):
    cfg = scaled_config(CONFIGS[name], nb=nb, n=n, p=p)
    A, Y = make_problem(cfg, device="cuda")
    flags = krr.FLAG_PREROUND_A
    if force == "fp8":
        h_map = krr.uniform_map(cfg.NT, krr.FP8)
        h_map[1:, 0] = krr.FP32
        d_map = h_map.cuda()
        flags = 0
    else:
        d_map, _, _, _ = krr.precision_map(A, nb, cfg.eps_target, cfg.allowed)
        h_map = d_map.cpu()
    F0, B0, launches = direct(krr, A, Y, nb, d_map, h_map, flags)
    assert int(F0.info.item()) == 0
    s = torch.cuda.Stream()
    B = torch.empty_like(Y)
    torch.cuda.synchronize()
    with torch.cuda.stream(s):
        g, F = record(krr, A, B, nb, d_map, h_map, flags)
        assert g.kernel_nodes == launches
        for scale in (1.0, 2.0):                   # a replay reads its inputs when it runs, not when it was recorded
            F.payload.zero_()
            F.scales.zero_()
            F.info.fill_(-7)
            B.copy_(Y * scale)
            g.launch()
            assert krr.last_launch_count() == launches
            s.synchronize()
            assert int(F.info.item()) == 0
            assert torch.equal(F.payload, F0.payload)
            assert torch.equal(F.scales, F0.scales)
            assert torch.equal(B, B0 * scale)      # a power of two scales every FP32 operation exactly
        g.destroy()


def test_replay_reports_breakdown_like_the_direct_call(krr):
    # a matrix that is not positive definite: the replay writes the same 1-based pivot column into info
    cfg = scaled_config(CONFIGS["C1"], nb=256, n=1024, p=500)
    A, Y = make_problem(cfg, device="cuda")
    A = A.clone()
    A[700, 700] = -1.0
    h_map = krr.uniform_map(cfg.NT, krr.FP32)
    d_map = h_map.cuda()
    F0, _, _ = direct(krr, A, Y, 256, d_map, h_map, krr.FLAG_PREROUND_A)
    assert int(F0.info.item()) == 701
    s = torch.cuda.Stream()
    B = Y.clone()
    torch.cuda.synchronize()
    with torch.cuda.stream(s):
        g, F = record(krr, A, B, 256, d_map, h_map, krr.FLAG_PREROUND_A)
        g.launch()
        s.synchronize()
    assert int(F.info.item()) == 701


def test_usage_errors(krr):
    with pytest.raises(krr.KrrError, match="KRR_ERR_ARG"):
        krr.graph_begin()                          # torch's current stream is the legacy default stream here
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        krr.profile_enable(1)
        try:
            with pytest.raises(krr.KrrError, match="KRR_ERR_UNSUPPORTED"):
                krr.graph_begin()
        finally:
            krr.profile_enable(0)
        krr.graph_begin()                          # an empty recording is a valid (empty) graph
        g = krr.graph_end()
        assert g.kernel_nodes == 0
        g.launch()
        s.synchronize()

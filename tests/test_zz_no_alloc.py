"""krr_precision_map_static: the entry point that allocates nothing (scratch = a file-scope __device__ array of the
library, 4 MiB) against the existing krr_precision_map (caller workspace) -- same kernels, same summation order, so
every output is compared bit for bit (the tolerance of tests/test_gpu_parity.py for the map; norms / amax / ||A||_F
there are bounded against the oracle, here they must simply be the same bits as the existing path's).

Two calls in a row share the array: the second one (another shape, smaller scratch footprint) must not see the first
one's leftovers.  Collected last on purpose (the suite runs with pytest -x): the file passes alone in a fresh process
and after the other tests.
"""
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


def _outputs(NT, dev):
    # filled with a pattern the kernels never produce: a word the call fails to write would show
    return (torch.full((NT, NT), 77, dtype=torch.uint8, device=dev),
            torch.full((NT, NT), -3.0, dtype=torch.float32, device=dev),
            torch.full((NT, NT), -3.0, dtype=torch.float32, device=dev),
            torch.full((1,), -3.0, dtype=torch.float64, device=dev))


def _same_bits(got, want):
    for g, w in zip(got, want):
        assert g.dtype == w.dtype and g.shape == w.shape
        assert torch.equal(g.view(torch.uint8), w.view(torch.uint8))


def test_static_scratch_entry_point_matches_the_workspace_path_on_two_calls_in_a_row(krr):
    cases = [("S1", 128, 2048, 1536, 1e-4, (0, 1, 2)),      # NT = 16: the rule's genuine FP32 / FP16 mosaic
             ("C5", 256, 1024, 400, 0.07, (0, 1, 2)),       # NT = 4, other nb: smaller footprint, stale words behind it
             ("C4", 128, 1024, 800, 1e-3, (0, 1))]          # FP8 masked out
    problems = []
    for name, nb, n, p, eps, allowed in cases:
        cfg = scaled_config(CONFIGS[name], nb=nb, n=n, p=p)
        A, _ = make_problem(cfg, device="cuda")
        problems.append((A, nb, eps, allowed, cfg.NT))
    # the existing path first (its own workspaces), then the static entry point back to back on one stream
    want = [krr.precision_map(A, nb, eps, allowed) for (A, nb, eps, allowed, NT) in problems]
    outs = [_outputs(NT, "cuda") for (A, nb, eps, allowed, NT) in problems]
    torch.cuda.synchronize()
    for (A, nb, eps, allowed, NT), out in zip(problems, outs):
        krr.precision_map_static(A, nb, eps, out, allowed)
        assert krr.last_launch_count() == 2
    torch.cuda.synchronize()
    for out, w in zip(outs, want):
        _same_bits(out, w)
    assert len({bytes(w[0].cpu().numpy().tobytes()) for w in want}) == len(want)        # the cases do differ
    m = want[0][0].cpu()
    assert int((m == krr.FP16).sum()) > 0 and int((m == krr.FP32).sum()) > m.shape[0]   # a genuine mosaic went through
    # again, in the opposite order (every call starts from another call's leftovers)
    outs2 = [_outputs(NT, "cuda") for (A, nb, eps, allowed, NT) in problems]
    for (A, nb, eps, allowed, NT), out in reversed(list(zip(problems, outs2))):
        krr.precision_map_static(A, nb, eps, out, allowed)
    torch.cuda.synchronize()
    for out, w in zip(outs2, want):
        _same_bits(out, w)


def test_static_scratch_entry_point_on_packed_lower_tiles_and_optional_outputs(krr):
    nb, n = 128, 1024
    cfg = scaled_config(CONFIGS["C4"], nb=nb, n=n, p=800)
    A, _ = make_problem(cfg, device="cuda")
    NT = cfg.NT
    tiles = [A[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb].contiguous().reshape(-1) for j in range(NT) for i in range(j, NT)]
    packed = torch.cat(tiles)
    want = krr.precision_map(packed, nb, 1e-3, (0, 1, 2), flags=krr.FLAG_A_TILED_LOWER, n=n)
    out = _outputs(NT, "cuda")
    krr.precision_map_static(packed, nb, 1e-3, out, (0, 1, 2), flags=krr.FLAG_A_TILED_LOWER, n=n)
    only_map = (torch.full((NT, NT), 77, dtype=torch.uint8, device="cuda"), None, None, None)
    krr.precision_map_static(A, nb, 1e-3, only_map, (0, 1, 2))
    torch.cuda.synchronize()
    _same_bits(out, want)
    assert torch.equal(only_map[0], want[0])


def test_static_scratch_entry_point_refuses_shapes_beyond_its_array(krr):
    import ctypes
    L = krr.lib()
    limit = int(L.krr_precision_map_static_limit())
    assert limit == 4 << 20
    # every BASELINE.json configuration fits
    for name in ("C1", "C2", "C3", "C4", "C5"):
        c = CONFIGS[name]
        assert 0 < int(L.krr_precision_map_workspace(c.n, c.nb)) <= limit, name
    # NT = 160 at nb = 1024 does not (4.9 MiB): refused on the host, nothing launched, outputs untouched
    n, nb = 160 * 1024, 1024
    assert int(L.krr_precision_map_workspace(n, nb)) > limit
    A = torch.zeros(16, dtype=torch.float32, device="cuda")          # never dereferenced
    out = _outputs(160, "cuda")
    rc = L.krr_precision_map_static(ctypes.c_void_p(A.data_ptr()), n, n, nb, 1e-4, 7, 0, ctypes.c_void_p(out[0].data_ptr()),
                                    None, None, None, None)
    assert rc == -3 and krr.last_launch_count() == 0
    with pytest.raises(krr.KrrError, match="static"):
        krr.precision_map_static(A, nb, 1e-4, out, flags=krr.FLAG_A_TILED_LOWER, n=n)
    torch.cuda.synchronize()
    assert int((out[0] != 77).sum()) == 0

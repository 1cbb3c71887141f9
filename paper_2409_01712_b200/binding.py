"""ctypes binding with the same names as include/krr_mp.h (marshalling only)."""
import ctypes
import os
from dataclasses import dataclass

import torch

FP32, FP16, FP8 = 0, 1, 2
FLAG_PREROUND_A = 1
FLAG_A_TILED_LOWER = 4
FLAG_NO_LOOKAHEAD = 8
FLAG_FP8_VIA_FP16 = 16
FLAG_NO_CTA_PAIRS = 32
FLAG_FUSED_CHAIN = 64
FLAG_KERNEL_IBS = 256
FLAG_KERNEL_LINEAR = 512
FLAG_NO_TAIL_SPLIT = 1024

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None

ERRORS = {-1: "KRR_ERR_ARG", -2: "KRR_ERR_SHAPE", -3: "KRR_ERR_WORKSPACE", -4: "KRR_ERR_DEVICE",
          -5: "KRR_ERR_CUDA", -6: "KRR_ERR_MAP", -7: "KRR_ERR_UNSUPPORTED"}

EXPORTS = ["krr_version", "krr_built_for_sm", "krr_tile_slot", "krr_precision_map_workspace",
           "krr_precision_map", "krr_precision_map_static_limit", "krr_precision_map_static", "krr_factor_bytes", "krr_factor_tile_offset",
           "krr_potrf_mp_workspace", "krr_potrf_mp", "krr_potrs_workspace", "krr_potrs", "krr_refine_workspace", "krr_refine", "krr_pcg_workspace", "krr_pcg",
           "krr_associate_host_arena", "krr_associate_host", "krr_build_workspace", "krr_build", "krr_build_bordered", "krr_build_rr", "krr_predict_workspace", "krr_predict", "krr_fit_host_arena", "krr_fit_host", "krr_band_map", "krr_build_stats_bytes", "krr_precision_map_from_build",
           "krr_graph_begin", "krr_graph_end", "krr_graph_launch", "krr_graph_kernel_nodes", "krr_graph_destroy",
           "krr_last_launch_count",
           "krr_profile_enable", "krr_profile_read", "krr_profile_timeline", "krr_peak_probe", "krr_shutdown", "krr_dist_schedule"]


class KrrError(RuntimeError):
    pass


def library_path():
    return os.path.join(_HERE, "libkrr_mp.so")


def lib():
    """Load libkrr_mp.so (built in-tree by build.py).  Fails loudly when it is missing."""
    global _LIB
    if _LIB is not None:
        return _LIB
    path = library_path()
    if not os.path.exists(path):
        raise KrrError(f"{path} not found: build it with `python -m paper_2409_01712_b200.build` "
                       "(there is no CPU fallback)")
    L = ctypes.CDLL(path)
    c = ctypes
    vp, i64, u32, sz = c.c_void_p, c.c_int64, c.c_uint, c.c_size_t
    L.krr_version.restype = c.c_int
    L.krr_built_for_sm.restype = c.c_int
    L.krr_tile_slot.restype = i64
    L.krr_tile_slot.argtypes = [c.c_int, c.c_int, c.c_int]
    L.krr_precision_map_workspace.restype = sz
    L.krr_precision_map_workspace.argtypes = [i64, c.c_int]
    L.krr_precision_map.restype = c.c_int
    L.krr_precision_map.argtypes = [vp, i64, i64, c.c_int, c.c_float, u32, u32, vp, vp, vp, vp, vp, sz, vp]
    L.krr_precision_map_static_limit.restype = sz
    L.krr_precision_map_static_limit.argtypes = []
    L.krr_precision_map_static.restype = c.c_int
    L.krr_precision_map_static.argtypes = [vp, i64, i64, c.c_int, c.c_float, u32, u32, vp, vp, vp, vp, vp]
    L.krr_factor_bytes.restype = sz
    L.krr_factor_bytes.argtypes = [i64, c.c_int, vp]
    L.krr_factor_tile_offset.restype = i64
    L.krr_factor_tile_offset.argtypes = [i64, c.c_int, vp, c.c_int, c.c_int]
    L.krr_potrf_mp_workspace.restype = sz
    L.krr_potrf_mp_workspace.argtypes = [i64, c.c_int, vp]
    L.krr_potrf_mp.restype = c.c_int
    L.krr_potrf_mp.argtypes = [vp, i64, i64, c.c_int, vp, vp, vp, vp, vp, vp, sz, u32, vp]
    L.krr_potrs_workspace.restype = sz
    L.krr_potrs_workspace.argtypes = [i64, c.c_int, c.c_int]
    L.krr_potrs.restype = c.c_int
    L.krr_potrs.argtypes = [vp, vp, vp, vp, i64, c.c_int, vp, i64, c.c_int, vp, sz, vp]
    L.krr_refine_workspace.restype = sz
    L.krr_refine_workspace.argtypes = [i64, c.c_int, c.c_int]
    L.krr_refine.restype = c.c_int
    L.krr_refine.argtypes = [vp, i64, i64, c.c_int, vp, vp, vp, vp, vp, i64, vp, i64, c.c_int, c.c_int, vp, vp, sz,
                             c.c_uint, vp]
    L.krr_pcg_workspace.restype = sz
    L.krr_pcg_workspace.argtypes = [i64, c.c_int, c.c_int]
    L.krr_pcg.restype = c.c_int
    L.krr_pcg.argtypes = L.krr_refine.argtypes
    L.krr_associate_host_arena.restype = sz
    L.krr_associate_host_arena.argtypes = [i64, c.c_int, c.c_int]
    L.krr_associate_host.restype = c.c_int
    L.krr_associate_host.argtypes = [vp, i64, i64, c.c_int, c.c_float, u32, c.c_int, u32, vp, c.c_int, vp,
                                     vp, vp, vp, sz, vp]
    L.krr_build_workspace.restype = sz
    L.krr_build_workspace.argtypes = [i64, i64, u32]
    L.krr_build.restype = c.c_int
    L.krr_build.argtypes = [vp, i64, i64, i64, vp, c.c_int, i64, c.c_float, c.c_float, vp, i64, c.c_int, u32, vp, vp, sz, vp]
    L.krr_build_bordered.restype = c.c_int
    L.krr_build_bordered.argtypes = [vp, i64, i64, i64, i64, vp, c.c_int, i64, c.c_float, c.c_float, vp, i64, c.c_int, u32, vp, vp,
                                     sz, vp]
    L.krr_build_rr.restype = c.c_int
    L.krr_build_rr.argtypes = [vp, i64, i64, i64, i64, vp, c.c_int, i64, c.c_float, vp, i64, c.c_int, u32, vp, sz, vp]
    L.krr_build_stats_bytes.restype = sz
    L.krr_build_stats_bytes.argtypes = [i64, c.c_int]
    L.krr_precision_map_from_build.restype = c.c_int
    L.krr_precision_map_from_build.argtypes = [vp, i64, c.c_int, c.c_float, u32, vp, vp, vp, vp, vp]
    L.krr_predict_workspace.restype = sz
    L.krr_predict_workspace.argtypes = [i64, i64, i64, u32]
    L.krr_predict.restype = c.c_int
    L.krr_predict.argtypes = [vp, i64, i64, vp, i64, i64, i64, vp, i64, vp, i64, c.c_int, c.c_float, vp, i64, c.c_int, vp, i64,
                              u32, vp, sz, vp]
    L.krr_fit_host_arena.restype = sz
    L.krr_fit_host_arena.argtypes = [i64, i64, c.c_int, c.c_int]
    L.krr_fit_host.restype = c.c_int
    L.krr_fit_host.argtypes = [vp, i64, i64, i64, c.c_float, c.c_float, c.c_int, c.c_float, u32, c.c_int, u32, vp, c.c_int, vp,
                               vp, vp, vp, sz, vp]
    L.krr_band_map.restype = c.c_int
    L.krr_band_map.argtypes = [c.c_int, c.c_double, c.c_int, vp]
    L.krr_last_launch_count.restype = i64
    L.krr_graph_begin.restype = c.c_int
    L.krr_graph_begin.argtypes = [vp]
    L.krr_graph_end.restype = c.c_int
    L.krr_graph_end.argtypes = [vp, c.POINTER(vp)]
    L.krr_graph_launch.restype = c.c_int
    L.krr_graph_launch.argtypes = [vp, vp]
    L.krr_graph_kernel_nodes.restype = i64
    L.krr_graph_kernel_nodes.argtypes = [vp]
    L.krr_graph_destroy.restype = c.c_int
    L.krr_graph_destroy.argtypes = [vp]
    L.krr_profile_enable.restype = c.c_int
    L.krr_profile_enable.argtypes = [u32]
    L.krr_profile_read.restype = c.c_int
    L.krr_profile_read.argtypes = [c.c_int, c.POINTER(c.c_double), c.POINTER(i64)]
    L.krr_profile_timeline.restype = c.c_int
    L.krr_profile_timeline.argtypes = [c.c_int, c.POINTER(c.c_float)]
    L.krr_peak_probe.restype = c.c_int
    L.krr_peak_probe.argtypes = [c.c_int, i64, c.POINTER(c.c_float), c.POINTER(c.c_double), vp]
    L.krr_shutdown.restype = c.c_int
    L.krr_dist_schedule.restype = i64
    L.krr_dist_schedule.argtypes = [c.c_int, c.c_int, vp, c.c_int, c.c_int, vp, i64]
    _LIB = L
    return L


def _check(rc, what):
    if rc != 0:
        raise KrrError(f"{what} failed: {ERRORS.get(rc, rc)}")


def _stream():
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ptr(t):
    return ctypes.c_void_p(t.data_ptr()) if t is not None else ctypes.c_void_p(0)


def _ws(nbytes, device):
    # torch's caching allocator returns 512-byte aligned blocks; over-allocate and align to 1 KiB
    buf = torch.empty(nbytes + 1024, dtype=torch.uint8, device=device)
    shift = (-buf.data_ptr()) % 1024
    return buf[shift:shift + nbytes]


def last_launch_count():
    return int(lib().krr_last_launch_count())


class Graph:
    """A recorded launch sequence (krr_graph_t).  `keep` holds the tensors the recorded calls were given:
    they must outlive the graph and are what a replay reads and writes."""

    def __init__(self, handle, keep):
        self.handle, self.keep = handle, keep

    @property
    def kernel_nodes(self):
        return int(lib().krr_graph_kernel_nodes(self.handle))

    def launch(self):
        _check(lib().krr_graph_launch(self.handle, _stream()), "krr_graph_launch")

    def destroy(self):
        if self.handle is not None:
            _check(lib().krr_graph_destroy(self.handle), "krr_graph_destroy")
            self.handle, self.keep = None, None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def graph_begin():
    """krr_graph_begin on torch's current stream (not the default stream: use `with torch.cuda.stream(s)`)."""
    _check(lib().krr_graph_begin(_stream()), "krr_graph_begin")


def graph_end(keep=()):
    """krr_graph_end on torch's current stream.  Returns a Graph that keeps `keep` alive."""
    h = ctypes.c_void_p(0)
    _check(lib().krr_graph_end(_stream(), ctypes.byref(h)), "krr_graph_end")
    return Graph(h, keep)


PROFILE_CATEGORIES = ["update_gemm", "panel_update", "panel_trsm", "potrf128", "finalize", "precision_map",
                      "potrs", "misc"]


def profile_enable(mask):
    _check(lib().krr_profile_enable(mask), "krr_profile_enable")


def profile_read():
    """{category: (total device ms, launches)} for the records since the last profile_enable."""
    out = {}
    for cat, name in enumerate(PROFILE_CATEGORIES):
        ms, cnt = ctypes.c_double(0.0), ctypes.c_int64(0)
        _check(lib().krr_profile_read(cat, ctypes.byref(ms), ctypes.byref(cnt)), "krr_profile_read")
        out[name] = (ms.value, cnt.value)
    return out


def profile_timeline(NT):
    """krr_profile_timeline: NT rows of [first, old, newb, fin] in ms since the fork of the last potrf_mp call."""
    buf = (ctypes.c_float * (4 * NT))()
    _check(lib().krr_profile_timeline(NT, buf), "krr_profile_timeline")
    return [[buf[4 * k + e] for e in range(4)] for k in range(NT)]


def tile_slot(NT, i, j):
    return int(lib().krr_tile_slot(NT, i, j))


def uniform_map(NT, offdiag):
    """Host map (uint8 NT x NT): diagonal FP32, every off-diagonal tile `offdiag`, 255 above."""
    m = torch.full((NT, NT), 255, dtype=torch.uint8)
    idx = torch.tril_indices(NT, NT, -1)
    m[idx[0], idx[1]] = offdiag
    m[torch.arange(NT), torch.arange(NT)] = FP32
    return m


def _host_map(h_map):
    h = h_map.detach().to("cpu", torch.uint8).contiguous()
    return h


def factor_bytes(n, nb, h_map):
    h = _host_map(h_map)
    return int(lib().krr_factor_bytes(n, nb, _ptr(h)))


def factor_tile_offset(n, nb, h_map, i, j):
    h = _host_map(h_map)
    return int(lib().krr_factor_tile_offset(n, nb, _ptr(h), i, j))


def precision_map(A, nb, eps_target, allowed=(FP32, FP16, FP8), flags=0, n=None):
    """krr_precision_map.  A: CUDA FP32 (n x n row-major, or the packed lower tiles with
    FLAG_A_TILED_LOWER and n given).  Returns (d_map uint8 NT x NT, tile norms, tile amax, fro)."""
    L = lib()
    if flags & FLAG_A_TILED_LOWER:
        assert n is not None
        lda = nb
    else:
        n, lda = A.shape[0], A.stride(0)
    NT = n // nb
    dev = A.device
    d_map = torch.empty((NT, NT), dtype=torch.uint8, device=dev)
    norms = torch.empty((NT, NT), dtype=torch.float32, device=dev)
    amax = torch.empty((NT, NT), dtype=torch.float32, device=dev)
    fro = torch.empty(1, dtype=torch.float64, device=dev)
    wsb = int(L.krr_precision_map_workspace(n, nb))
    if wsb == 0:
        raise KrrError("krr_precision_map_workspace: invalid shape")
    ws = _ws(wsb, dev)
    mask = sum(1 << p for p in allowed)
    _check(L.krr_precision_map(_ptr(A), n, lda, nb, float(eps_target), mask, flags, _ptr(d_map), _ptr(norms),
                               _ptr(amax), _ptr(fro), _ptr(ws), wsb, _stream()), "krr_precision_map")
    return d_map, norms, amax, fro


def precision_map_static(A, nb, eps_target, out, allowed=(FP32, FP16, FP8), flags=0, n=None):
    """krr_precision_map_static: krr_precision_map on the library's own file-scope scratch array -- the call allocates
    nothing (neither does this wrapper: `out` = (d_map uint8 NT x NT, tile norms, tile amax, fro) are the caller's
    tensors, as in precision_map's return value).  Shapes whose scratch exceeds the 4 MiB array are refused."""
    L = lib()
    if flags & FLAG_A_TILED_LOWER:
        assert n is not None
        lda = nb
    else:
        n, lda = A.shape[0], A.stride(0)
    d_map, norms, amax, fro = out
    NT = n // nb
    assert d_map.dtype == torch.uint8 and d_map.numel() == NT * NT and d_map.is_contiguous()
    for t in (norms, amax):
        assert t is None or (t.dtype == torch.float32 and t.numel() == NT * NT and t.is_contiguous())
    assert fro is None or fro.dtype == torch.float64
    need, limit = int(L.krr_precision_map_workspace(n, nb)), int(L.krr_precision_map_static_limit())
    if need > limit:
        raise KrrError(f"krr_precision_map_static: n = {n}, nb = {nb} needs {need} bytes of scratch, the library's static "
                       f"array holds {limit}; use precision_map (caller workspace) for this shape")
    mask = sum(1 << p for p in allowed)
    _check(L.krr_precision_map_static(_ptr(A), n, lda, nb, float(eps_target), mask, flags, _ptr(d_map), _ptr(norms),
                                      _ptr(amax), _ptr(fro), _stream()), "krr_precision_map_static")
    return out


@dataclass
class Factor:
    """Result of potrf_mp: the tile mosaic and what krr_potrs needs."""
    n: int
    nb: int
    h_map: torch.Tensor        # host uint8 NT x NT
    d_map: torch.Tensor        # device copy
    payload: torch.Tensor      # device uint8, krr_factor_bytes
    scales: torch.Tensor       # device float32 NT x NT
    info: torch.Tensor         # device int32 [1]
    ws: torch.Tensor           # device workspace (FP16 operand images), kept alive

    @property
    def NT(self):
        return self.n // self.nb

    def tile(self, i, j):
        """Dequantised tile (i,j) as a float64 CUDA tensor (test / inspection helper)."""
        nb, NT = self.nb, self.NT
        p = int(self.h_map[i, j])
        off = factor_tile_offset(self.n, nb, self.h_map, i, j)
        nbytes = nb * nb * (4, 2, 1)[p]
        raw = self.payload[off:off + nbytes]
        if p == FP32:
            return raw.view(torch.float32).reshape(nb, nb).to(torch.float64)
        if p == FP16:
            return raw.view(torch.float16).reshape(nb, nb).to(torch.float64)
        return raw.view(torch.float8_e4m3fn).reshape(nb, nb).to(torch.float64) * float(self.scales[i, j])

    def dense(self):
        """Dense dequantised lower-triangular factor, float64, on the factor's device."""
        n, nb, NT = self.n, self.nb, self.NT
        Ld = torch.zeros((n, n), dtype=torch.float64, device=self.payload.device)
        for j in range(NT):
            for i in range(j, NT):
                Ld[i * nb:(i + 1) * nb, j * nb:(j + 1) * nb] = self.tile(i, j)
        return Ld


def potrf_mp(A, nb, d_map, h_map=None, flags=FLAG_PREROUND_A, n=None):
    """krr_potrf_mp.  Returns a Factor; `info` is read by the caller after synchronising."""
    L = lib()
    if flags & FLAG_A_TILED_LOWER:
        assert n is not None
        lda = nb
    else:
        n, lda = A.shape[0], A.stride(0)
    dev = A.device
    NT = n // nb
    h = _host_map(d_map if h_map is None else h_map)
    d_map = d_map.to(dev, torch.uint8).contiguous()
    fb = int(L.krr_factor_bytes(n, nb, _ptr(h)))
    wsb = int(L.krr_potrf_mp_workspace(n, nb, _ptr(h)))
    if fb == 0 or wsb == 0:
        raise KrrError("invalid shape or precision map")
    payload = _ws(fb, dev)
    ws = _ws(wsb, dev)
    scales = torch.empty((NT, NT), dtype=torch.float32, device=dev)
    info = torch.empty(1, dtype=torch.int32, device=dev)
    _check(L.krr_potrf_mp(_ptr(A), n, lda, nb, _ptr(d_map), _ptr(h), _ptr(payload), _ptr(scales), _ptr(info),
                          _ptr(ws), wsb, flags, _stream()), "krr_potrf_mp")
    return Factor(n, nb, h, d_map, payload, scales, info, ws)


def potrs_workspace(n, nb, nrhs, device):
    """A krr_potrs workspace (krr_potrs_workspace bytes), for callers that keep it (graph replay)."""
    wsb = int(lib().krr_potrs_workspace(n, nb, nrhs))
    if wsb == 0:
        raise KrrError("krr_potrs_workspace: invalid shape / nrhs")
    return _ws(wsb, device)


def potrs(factor, B, ws=None):
    """krr_potrs, in place on B (CUDA FP32, n x nrhs row-major).  Returns B.  `ws`: a workspace from
    potrs_workspace; a recorded call (graph_begin) needs one that outlives the graph."""
    L = lib()
    assert B.dtype == torch.float32 and B.is_cuda and B.stride(1) == 1
    n, nrhs = B.shape
    wsb = int(L.krr_potrs_workspace(n, factor.nb, nrhs))
    if wsb == 0:
        raise KrrError("krr_potrs_workspace: invalid shape / nrhs")
    if ws is None:
        ws = _ws(wsb, B.device)
    assert ws.numel() >= wsb and ws.data_ptr() % 16 == 0
    _check(L.krr_potrs(_ptr(factor.payload), _ptr(factor.scales), _ptr(factor.d_map), _ptr(factor.h_map), n,
                       factor.nb, _ptr(B), B.stride(0), nrhs, _ptr(ws), wsb, _stream()), "krr_potrs")
    return B


def refine(A, factor, Y, X, steps, tiled_lower=False, residual_norms=True):
    """krr_refine: `steps` refinement steps of X (in place) for A X = Y with the factor kept fixed (R19).
    A as for precision_map (dense n x n, or the packed lower tiles with tiled_lower=True).  Returns (X, norms) with
    norms the steps + 1 residual norms ||fl32(Y - A alpha_s)||_F (a CUDA float64 tensor), or None."""
    L = lib()
    assert A.dtype == torch.float32 and A.is_cuda
    assert Y.dtype == torch.float32 and Y.is_cuda and Y.stride(1) == 1
    assert X.dtype == torch.float32 and X.is_cuda and X.stride(1) == 1 and X.shape == Y.shape
    n, nrhs = Y.shape
    lda = factor.nb if tiled_lower else A.stride(0)
    wsb = int(L.krr_refine_workspace(n, factor.nb, nrhs))
    if wsb == 0:
        raise KrrError("krr_refine_workspace: invalid shape / nrhs")
    ws = _ws(wsb, Y.device)
    norms = torch.zeros(steps + 1, dtype=torch.float64, device=Y.device) if residual_norms else None
    _check(L.krr_refine(_ptr(A), n, lda, factor.nb, _ptr(factor.payload), _ptr(factor.scales), _ptr(factor.d_map),
                        _ptr(factor.h_map), _ptr(Y), Y.stride(0), _ptr(X), X.stride(0), nrhs, steps,
                        _ptr(norms) if residual_norms else None, _ptr(ws), wsb,
                        FLAG_A_TILED_LOWER if tiled_lower else 0, _stream()), "krr_refine")
    return X, norms


def pcg(A, factor, Y, X, iters, tiled_lower=False, residual_norms=True):
    """krr_pcg: `iters` steps of conjugate gradients on A X = Y preconditioned by the factor, started from X (in place;
    DESIGN.md R20).  Arguments and result as for `refine`; the norms are those of the recursively updated residuals."""
    L = lib()
    assert A.dtype == torch.float32 and A.is_cuda
    assert Y.dtype == torch.float32 and Y.is_cuda and Y.stride(1) == 1
    assert X.dtype == torch.float32 and X.is_cuda and X.stride(1) == 1 and X.shape == Y.shape
    n, nrhs = Y.shape
    lda = factor.nb if tiled_lower else A.stride(0)
    wsb = int(L.krr_pcg_workspace(n, factor.nb, nrhs))
    if wsb == 0:
        raise KrrError("krr_pcg_workspace: invalid shape / nrhs")
    ws = _ws(wsb, Y.device)
    norms = torch.zeros(iters + 1, dtype=torch.float64, device=Y.device) if residual_norms else None
    _check(L.krr_pcg(_ptr(A), n, lda, factor.nb, _ptr(factor.payload), _ptr(factor.scales), _ptr(factor.d_map),
                     _ptr(factor.h_map), _ptr(Y), Y.stride(0), _ptr(X), X.stride(0), nrhs, iters,
                     _ptr(norms) if residual_norms else None, _ptr(ws), wsb,
                     FLAG_A_TILED_LOWER if tiled_lower else 0, _stream()), "krr_pcg")
    return X, norms


def associate_host(h_A, nb, h_Y, eps_target=0.0, allowed=(FP32,), force_prec=-1, flags=FLAG_PREROUND_A,
                   arena=None, device="cuda"):
    """krr_associate_host: whole Associate phase from host tensors (pinned recommended).
    Returns (alpha host tensor, h_map, info int, arena)."""
    L = lib()
    n, lda = h_A.shape[0], h_A.stride(0)
    nrhs = h_Y.shape[1]
    NT = n // nb
    need = int(L.krr_associate_host_arena(n, nb, nrhs))
    if need == 0:
        raise KrrError("krr_associate_host_arena: invalid shape")
    if arena is None or arena.numel() < need:
        arena = _ws(need, device)
    alpha = torch.empty_like(h_Y)
    h_map = torch.empty((NT, NT), dtype=torch.uint8)
    h_info = torch.zeros(1, dtype=torch.int32)
    mask = sum(1 << p for p in allowed)
    _check(L.krr_associate_host(_ptr(h_A), n, lda, nb, float(eps_target), mask, force_prec, flags, _ptr(h_Y), nrhs,
                                _ptr(alpha), _ptr(h_map), _ptr(h_info), _ptr(arena), arena.numel(), _stream()),
           "krr_associate_host")
    return alpha, h_map, int(h_info[0]), arena


def _conf(C):
    if C is None:
        return None, 0, 0
    assert C.dtype == torch.float32 and C.is_cuda and C.stride(1) == 1
    return C, C.shape[1], C.stride(0)


def krr_build(G, gamma, lam, nb, tiled_lower=False, out=None, flags=0, C=None, stats=False, n_valid=None):
    """krr_build (named in full: `build` is this package's compile step): A = K + lam*I (Gaussian kernel) from CUDA int8 genotypes G (n x p, row-major, row pitch a
    multiple of 16 bytes).  Returns A: n x n FP32 with the lower tiles written (the rest zero), or the packed
    lower tiles with tiled_lower.  n_valid < n (krr_build_bordered, R21): rows >= n_valid of G are padding,
    rows and columns >= n_valid of A the identity border."""
    L = lib()
    assert G.dtype == torch.int8 and G.is_cuda and G.stride(1) == 1
    n, p = G.shape
    NT = n // nb
    dev = G.device
    if out is None:
        out = (torch.zeros(NT * (NT + 1) // 2 * nb * nb, dtype=torch.float32, device=dev) if tiled_lower
               else torch.zeros((n, n), dtype=torch.float32, device=dev))
    flags |= FLAG_A_TILED_LOWER if tiled_lower else 0
    wsb = int(L.krr_build_workspace(n, p, flags))
    if wsb == 0:
        raise KrrError("krr_build_workspace: n must be a multiple of 256")
    ws = _ws(wsb, dev)
    lda = nb if tiled_lower else out.stride(0)
    C, q, ldc = _conf(C)
    st = _ws(int(L.krr_build_stats_bytes(n, nb)), dev) if stats else None
    _check(L.krr_build_bordered(_ptr(G), n, n if n_valid is None else int(n_valid), p, G.stride(0), _ptr(C), q, ldc,
                                float(gamma), float(lam), _ptr(out), lda, nb, flags, _ptr(st), _ptr(ws), wsb, _stream()),
           "krr_build_bordered")
    return (out, st) if stats else out


def build_rr(S, ns, lam, nb, C=None, tiled_lower=False):
    """krr_build_rr: X^T X + lam I for X = [S^T | C], bordered by the identity (Fig. 2).  S: CUDA int8 n x p with the
    SNP features as rows (rows >= ns are padding), C: CUDA FP32 p x q confounders or None."""
    L = lib()
    assert S.dtype == torch.int8 and S.is_cuda and S.stride(1) == 1
    n, p = S.shape
    NT = n // nb
    dev = S.device
    out = (torch.zeros(NT * (NT + 1) // 2 * nb * nb, dtype=torch.float32, device=dev) if tiled_lower
           else torch.zeros((n, n), dtype=torch.float32, device=dev))
    wsb = int(L.krr_build_workspace(n, p, 0))
    if wsb == 0:
        raise KrrError("krr_build_workspace: n must be a multiple of 256")
    ws = _ws(wsb, dev)
    C, q, ldc = _conf(C)
    _check(L.krr_build_rr(_ptr(S), n, int(ns), p, S.stride(0), _ptr(C), q, ldc, float(lam), _ptr(out),
                          nb if tiled_lower else out.stride(0), nb, FLAG_A_TILED_LOWER if tiled_lower else 0, _ptr(ws), wsb,
                          _stream()), "krr_build_rr")
    return out


def precision_map_from_build(stats, n, nb, eps_target, allowed=(FP32, FP16, FP8)):
    """krr_precision_map_from_build: the map from the tile statistics krr_build(..., stats=True) left behind.
    Returns (d_map, tile norms, tile amax, fro) like precision_map."""
    L = lib()
    NT = n // nb
    dev = stats.device
    d_map = torch.empty((NT, NT), dtype=torch.uint8, device=dev)
    norms = torch.empty((NT, NT), dtype=torch.float32, device=dev)
    amax = torch.empty((NT, NT), dtype=torch.float32, device=dev)
    fro = torch.empty(1, dtype=torch.float64, device=dev)
    mask = sum(1 << p for p in allowed)
    _check(L.krr_precision_map_from_build(_ptr(stats), n, nb, float(eps_target), mask, _ptr(d_map), _ptr(norms), _ptr(amax),
                                          _ptr(fro), _stream()), "krr_precision_map_from_build")
    return d_map, norms, amax, fro


def krr_predict(T, G, gamma, W, return_kernel=False, CT=None, CG=None, flags=0):
    """krr_predict: P_r = K(T, G) W (Alg. 4).  T (m x p), G (n x p): CUDA int8, row pitch a multiple of 16 bytes;
    W: CUDA FP32 n x nrhs.  Returns P (m x nrhs) and, on request, the test-training kernel matrix (a view
    into the call's workspace)."""
    L = lib()
    assert T.dtype == torch.int8 and G.dtype == torch.int8 and T.is_cuda and G.is_cuda
    assert W.dtype == torch.float32 and W.is_cuda and W.stride(1) == 1
    m, p = T.shape
    n = G.shape[0]
    nrhs = W.shape[1]
    wsb = int(L.krr_predict_workspace(m, n, p, flags))
    if wsb == 0:
        raise KrrError("krr_predict_workspace: m and n must be multiples of 256")
    ws = _ws(wsb, G.device)
    P = torch.empty((m, nrhs), dtype=torch.float32, device=G.device)
    CT, q, ldct = _conf(CT)
    CG, q2, ldcg = _conf(CG)
    assert q == q2
    _check(L.krr_predict(_ptr(T), m, T.stride(0), _ptr(G), n, G.stride(0), p, _ptr(CT), ldct, _ptr(CG), ldcg, q, float(gamma),
                         _ptr(W), W.stride(0), nrhs, _ptr(P), P.stride(0), flags, _ptr(ws), wsb, _stream()), "krr_predict")
    if not return_kernel:
        return P
    off = (m * 4 + 1023) // 1024 * 1024 + (n * 4 + 1023) // 1024 * 1024
    return P, ws[off:off + m * n * 4].view(torch.float32).reshape(m, n)


def fit_host(h_G, gamma, lam, nb, h_Y, eps_target=0.0, allowed=(FP32,), force_prec=-1, flags=FLAG_PREROUND_A, arena=None,
             device="cuda"):
    """krr_fit_host: Build + Associate from host genotypes (int8, pinned recommended) and phenotypes.
    Returns (alpha host tensor, h_map, info int, arena)."""
    L = lib()
    assert h_G.dtype == torch.int8 and not h_G.is_cuda and h_G.stride(1) == 1
    n, p = h_G.shape
    nrhs = h_Y.shape[1]
    NT = n // nb
    need = int(L.krr_fit_host_arena(n, p, nb, nrhs))
    if need == 0:
        raise KrrError("krr_fit_host_arena: invalid shape")
    if arena is None or arena.numel() < need:
        arena = _ws(need, device)
    alpha = torch.empty_like(h_Y)
    h_map = torch.empty((NT, NT), dtype=torch.uint8)
    h_info = torch.zeros(1, dtype=torch.int32)
    mask = sum(1 << q for q in allowed)
    _check(L.krr_fit_host(_ptr(h_G), n, p, h_G.stride(0), float(gamma), float(lam), nb, float(eps_target), mask, force_prec,
                          flags, _ptr(h_Y), nrhs, _ptr(alpha), _ptr(h_map), _ptr(h_info), _ptr(arena), arena.numel(), _stream()),
           "krr_fit_host")
    return alpha, h_map, int(h_info[0]), arena


def band_map(NT, fp32_fraction, low):
    """krr_band_map: host map (uint8 NT x NT) of the band technique of [37]."""
    m = torch.empty((NT, NT), dtype=torch.uint8)
    _check(lib().krr_band_map(NT, float(fp32_fraction), int(low), _ptr(m)), "krr_band_map")
    return m



PEAK_KINDS = {"f16": 0, "f8": 1, "mxf8": 2, "ffma": 3, "f16x3": 4}


def peak_probe(kind, work):
    """One launch of krr_peak_probe: (device ms, flops performed)."""
    ms, fl = ctypes.c_float(0.0), ctypes.c_double(0.0)
    _check(lib().krr_peak_probe(PEAK_KINDS[kind], int(work), ctypes.byref(ms), ctypes.byref(fl), _stream()), "krr_peak_probe")
    return float(ms.value), float(fl.value)


def shutdown():
    """Destroy the internal streams and events of the calling thread on the current device (krr_shutdown)."""
    _check(lib().krr_shutdown(), "krr_shutdown")


DIST_OPS = {1: "chain", 2: "newest", 3: "older", 4: "trsm", 5: "bcast_m", 6: "bcast_next", 7: "allgather"}


def dist_schedule(NT, nb, h_map, world, rank):
    """krr_dist_schedule: the task / message list of `rank` as a list of dicts (host logic only; NEXT-3)."""
    h = _host_map(h_map)
    cnt = int(lib().krr_dist_schedule(NT, nb, _ptr(h), world, rank, None, 0))
    if cnt < 0:
        _check(cnt, "krr_dist_schedule")
    buf = torch.zeros((cnt, 6), dtype=torch.int32)
    got = int(lib().krr_dist_schedule(NT, nb, _ptr(h), world, rank, _ptr(buf), cnt))
    assert got == cnt
    out = []
    for r in buf.tolist():
        out.append({"op": DIST_OPS[r[0]], "k": r[1], "root": r[2], "nrows": r[3], "bytes": (r[4] & 0xffffffff) | (r[5] << 32)})
    return out

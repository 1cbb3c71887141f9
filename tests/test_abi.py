"""The C-ABI library builds, loads and exports every symbol include/krr_mp.h declares (no compute
calls: this runs without a GPU), and its pure host functions behave as documented."""
import ctypes
import os
import re

import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _lib():
    from paper_2409_01712_b200 import build
    build.build()
    import paper_2409_01712_b200 as krr
    return krr, krr.lib()


def test_library_exports_every_declared_symbol():
    krr, L = _lib()
    header = open(os.path.join(ROOT, "include", "krr_mp.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(krr_[a-z0-9_]+)\s*\(", header))
    assert {"krr_precision_map", "krr_potrf_mp", "krr_potrs"} <= declared
    for name in declared:
        assert hasattr(L, name), name
    from paper_2409_01712_b200.binding import EXPORTS
    assert declared == set(EXPORTS)
    assert L.krr_built_for_sm() == 100


def test_host_layout_functions():
    krr, L = _lib()
    NT, nb = 4, 128
    assert [krr.tile_slot(NT, i, 0) for i in range(4)] == [0, 1, 2, 3]
    assert krr.tile_slot(NT, 1, 1) == 4 and krr.tile_slot(NT, 3, 3) == 9
    assert krr.tile_slot(NT, 0, 1) == -1
    m = krr.uniform_map(NT, krr.FP16)
    m[2, 0] = krr.FP8
    m[3, 1] = krr.FP32
    n = NT * nb
    e = nb * nb
    # column-major lower order: (0,0)32 (1,0)16 (2,0)8 (3,0)16 (1,1)32 (2,1)16 (3,1)32 ...
    assert krr.factor_tile_offset(n, nb, m, 0, 0) == 0
    assert krr.factor_tile_offset(n, nb, m, 1, 0) == 4 * e
    assert krr.factor_tile_offset(n, nb, m, 2, 0) == 6 * e
    assert krr.factor_tile_offset(n, nb, m, 3, 0) == 7 * e
    assert krr.factor_tile_offset(n, nb, m, 1, 1) == 9 * e
    assert krr.factor_tile_offset(n, nb, m, 3, 1) == 15 * e
    total = (4 * 4 + 1 * 1 + 4 * 2 + 1 * 4) * e            # 4 diag FP32, 1 FP8, 4 FP16, 1 FP32 off-diag
    assert krr.factor_bytes(n, nb, m) == total
    assert krr.factor_bytes(n + 1, nb, m) == 0              # nb does not divide n
    bad = m.clone(); bad[1, 1] = krr.FP16                   # non-FP32 diagonal
    assert krr.factor_bytes(n, nb, bad) == 0
    assert L.krr_potrf_mp_workspace(n, nb, ctypes.c_void_p(m.data_ptr())) > 2 * 10 * e * 2
    assert L.krr_precision_map_workspace(n, 100) == 0       # nb not a multiple of 128
    assert L.krr_potrs_workspace(n, nb, 33) == 0


def test_argument_errors_are_reported_before_any_launch():
    krr, L = _lib()
    null = ctypes.c_void_p(0)
    rc = L.krr_precision_map(null, 256, 256, 128, 1e-4, 7, 0, null, null, null, null, null, 0, null)
    assert rc == -1
    m = krr.uniform_map(2, krr.FP32)
    rc = L.krr_potrf_mp(null, 256, 256, 128, null, ctypes.c_void_p(m.data_ptr()), null, null, null, null, 0, 1, null)
    assert rc == -1


def test_band_map_host_utility_matches_oracle():
    """krr_band_map is pure host code: callable without a GPU; bit-exact against the oracle's reading."""
    import numpy as np
    import paper_2409_01712_b200 as krr
    from oracle.precision_map import band_map
    for NT in (1, 2, 8, 11, 64):
        for frac in (0.0, 0.1, 0.2, 0.4, 0.6, 0.8, 1.0):
            for low in (1, 2):
                assert np.array_equal(krr.band_map(NT, frac, low).numpy(), band_map(NT, frac, low)), (NT, frac, low)


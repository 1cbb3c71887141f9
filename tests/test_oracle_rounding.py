"""Pins for the oracle's rounding emulators (oracle/rounding.py).

Pins: numpy.float16 / numpy.float32 casts (independent IEEE implementations), torch.float8_e4m3fn
CPU cast for in-range values, the full E4M3 code table (OCP FP8: bias 7, max 448, subnormal step
2^-9), ties-to-even on every midpoint, and exact power-of-two tile scales.
"""
import numpy as np
import pytest
import torch

from oracle import rounding as R


def _samples(rng, n, lo_exp, hi_exp):
    m = rng.uniform(-1.0, 1.0, n)
    e = rng.integers(lo_exp, hi_exp, n)
    return np.ldexp(m, e)


def test_fp16_matches_numpy_cast():
    rng = np.random.default_rng(0)
    x = np.concatenate([_samples(rng, 200000, -30, 17), [0.0, -0.0, 65504.0, 65519.9, 65520.0, 1e6,
                                                        2.0 ** -24, 2.0 ** -25, 3 * 2.0 ** -25]])
    with np.errstate(over="ignore"):
        want = x.astype(np.float16).astype(np.float64)
    got = R.rd_fp16(x)
    assert np.array_equal(got, want)


def test_fp32_matches_c_float_cast():
    rng = np.random.default_rng(1)
    x = np.concatenate([_samples(rng, 200000, -160, 128), [0.0, 1.0 + 2.0 ** -24, 1.0 + 3 * 2.0 ** -24,
                                                           2.0 ** -149, 2.0 ** -150, 1e39]])
    with np.errstate(over="ignore"):
        want = x.astype(np.float32).astype(np.float64)
    assert np.array_equal(R.rd_fp32(x), want)


def test_e4m3_code_table():
    codes = np.arange(256)
    v = R.e4m3_decode(codes)
    # NaN codes
    assert np.isnan(v[0x7F]) and np.isnan(v[0xFF]) and np.isnan(v).sum() == 2
    pos = v[:0x7F]
    assert pos[0] == 0.0 and pos[1] == 2.0 ** -9 and pos[7] == 7 * 2.0 ** -9
    assert pos[8] == 2.0 ** -6                       # smallest normal
    assert pos[0x7E] == 448.0                        # largest finite
    assert pos[0x38] == 1.0 and pos[0x39] == 1.125
    assert np.all(np.diff(pos) > 0)                  # monotone
    assert np.array_equal(v[0x80:0xFF], -pos)
    # round trip of every finite code: value -> rd -> encode
    fin = np.array([c for c in codes if c not in (0x7F, 0xFF)])
    vals = R.e4m3_decode(fin)
    assert np.array_equal(R.rd_e4m3(vals), vals)
    enc = R.e4m3_encode(vals)
    # -0.0 and +0.0 keep their sign bit
    assert np.array_equal(enc, fin.astype(np.uint8))


def test_e4m3_ties_to_even_on_all_midpoints():
    pos = R.e4m3_decode(np.arange(0x7F))
    for c in range(0x7E):
        lo, hi = pos[c], pos[c + 1]
        mid = 0.5 * (lo + hi)
        want = lo if c % 2 == 0 else hi              # even mantissa code wins
        assert R.rd_e4m3(mid) == want, (c, lo, hi)
        assert R.rd_e4m3(np.nextafter(mid, np.inf)) == hi
        assert R.rd_e4m3(np.nextafter(mid, -np.inf)) == lo
        assert R.rd_e4m3(-mid) == -want


def test_e4m3_saturates():
    assert R.rd_e4m3(449.0) == 448.0 and R.rd_e4m3(1e9) == 448.0 and R.rd_e4m3(-500.0) == -448.0
    assert R.rd_e4m3(464.0) == 448.0


def test_e4m3_matches_torch_cast_in_range():
    rng = np.random.default_rng(2)
    x = np.concatenate([_samples(rng, 300000, -14, 9), rng.uniform(-448, 448, 100000)])
    x = x[np.abs(x) <= 448.0]
    x32 = x.astype(np.float32)                       # torch casts from FP32
    want = torch.from_numpy(x32).to(torch.float8_e4m3fn).to(torch.float32).numpy().astype(np.float64)
    got = R.rd_e4m3(x32.astype(np.float64))
    assert np.array_equal(got, want)


@pytest.mark.parametrize("amax,scale", [
    (448.0, 1.0), (448.0001, 2.0), (224.0, 0.5), (224.0001, 1.0), (1.0, 2.0 ** -8),
    (0.875, 2.0 ** -9), (0.8750001, 2.0 ** -8), (2.0, 2.0 ** -7), (0.0, 1.0), (1e-4, 2.0 ** -22),
])
def test_fp8_tile_scale(amax, scale):
    s = R.fp8_tile_scale(amax)
    assert s == scale
    if amax > 0:
        assert amax <= 448.0 * s and amax > 224.0 * s


def test_quantise_tile_fp8_uses_top_binade_and_is_exact_for_dyadic():
    T = np.array([[0.5, -1.0], [2.0, 0.0]])
    q, s = R.quantise_tile(T, R.FP8)
    assert s == 2.0 ** -7 and np.array_equal(q, T)
    rng = np.random.default_rng(3)
    T = rng.standard_normal((64, 64))
    q, s = R.quantise_tile(T, R.FP8)
    assert np.max(np.abs(T - q) / np.maximum(np.abs(T), np.max(np.abs(T)) * 2.0 ** -8)) <= 2.0 ** -4
    q16, s16 = R.quantise_tile(T, R.FP16)
    assert s16 == 1.0 and np.array_equal(q16, T.astype(np.float16).astype(np.float64))

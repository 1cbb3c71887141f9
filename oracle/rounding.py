"""Software rounding into the storage precisions of the tile mosaic (oracle; test infrastructure).

The paper stores each tile in FP32, FP16 or FP8 and uses the E4M3 form of FP8 for
both GEMM operands.  It does not print the formats; they are the IEEE-754 binary32
and binary16 formats and the OCP FP8 E4M3 format (no infinities, one NaN code per sign, maximum
finite value 448).  Every rounding is round-to-nearest, ties-to-even, subnormals kept.

All functions take and return float64 arrays holding values that are exactly representable in the
target format, so arithmetic between rounding points can stay in FP64.
"""
import numpy as np

# name -> (t = significand bits including the implicit one, emin = exponent of the smallest normal,
#          largest finite value, unit roundoff u = 2^-t)
FORMATS = {
    "fp32": (24, -126, float(np.finfo(np.float32).max), 2.0 ** -24),
    "fp16": (11, -14, 65504.0, 2.0 ** -11),
    "e4m3": (4, -6, 448.0, 2.0 ** -4),
}

# precision codes used in the map (same numbering as include/krr_mp.h, an interface constant)
FP32, FP16, FP8 = 0, 1, 2
CODE_TO_FORMAT = {FP32: "fp32", FP16: "fp16", FP8: "e4m3"}
UNIT_ROUNDOFF = {FP32: 2.0 ** -24, FP16: 2.0 ** -11, FP8: 2.0 ** -4}


def round_to_format(x, fmt, saturate=False):
    """Round float64 `x` to the nearest value of format `fmt` (ties to even).

    Definition: for x != 0 let e = floor(log2|x|), e' = max(e, emin) and q = 2^(e' - (t-1)) the
    spacing of the format around x; the result is q * rint(x / q).  x / q is exact (q is a power of
    two) and rint rounds half to even.  Above the largest finite value the result is +-inf (IEEE
    formats) or, with `saturate`, +-max (E4M3 "satfinite", reading R7).
    """
    t, emin, fmax, _ = FORMATS[fmt]
    x = np.asarray(x, dtype=np.float64)
    _, ex = np.frexp(x)                      # x = m * 2^ex, 0.5 <= |m| < 1  ->  e = ex - 1
    e = np.maximum(ex - 1, emin)
    q = np.ldexp(1.0, e - (t - 1))
    y = np.rint(x / q) * q
    y = np.where(x == 0.0, x, y)
    over = np.abs(y) > fmax
    if saturate:
        y = np.where(over, np.copysign(fmax, x), y)
    else:
        y = np.where(over, np.copysign(np.inf, x), y)
    return y


def rd_fp32(x):
    return round_to_format(x, "fp32")


def rd_fp16(x):
    return round_to_format(x, "fp16")


def rd_e4m3(x):
    """E4M3 rounding, saturating to +-448 (never reached once the tile scale is applied)."""
    return round_to_format(x, "e4m3", saturate=True)


def e4m3_decode(code):
    """Value of an E4M3 byte: s eeee mmm, bias 7, subnormals at e=0, 0x7f/0xff are NaN."""
    code = np.asarray(code, dtype=np.int64)
    s = np.where((code >> 7) & 1, -1.0, 1.0)
    e = (code >> 3) & 0xF
    m = code & 0x7
    normal = np.ldexp(1.0 + m / 8.0, e - 7)
    sub = np.ldexp(m / 8.0, -6)
    v = np.where(e == 0, sub, normal)
    v = np.where((e == 15) & (m == 7), np.nan, v)
    return s * v


def e4m3_encode(x):
    """E4M3 byte of a value that is already exactly representable (after rd_e4m3)."""
    x = np.asarray(x, dtype=np.float64)
    sign = (np.signbit(x)).astype(np.int64) << 7
    a = np.abs(x)
    mant, ex = np.frexp(a)                   # a = mant * 2^ex, mant in [0.5, 1)
    e = ex - 1
    is_sub = (a < 2.0 ** -6)
    m_norm = np.rint((mant * 2.0 - 1.0) * 8.0).astype(np.int64)
    code_norm = ((e + 7).astype(np.int64) << 3) | m_norm
    code_sub = np.rint(a * 2.0 ** 9).astype(np.int64)          # m/8 * 2^-6 = m * 2^-9
    return (sign | np.where(is_sub, code_sub, code_norm)).astype(np.uint8)


def fp8_tile_scale(amax):
    """Power-of-two per-tile scale of an FP8 tile (reading R6).

    s = 2^ceil(log2(amax / 448)): the smallest power of two with amax / s <= 448, so the scaled tile
    never overflows E4M3 and uses its top binade.  s = 1 when amax == 0.  Computed with exact
    comparisons (448 * s is exact) rather than a floating-point log2.
    """
    amax = float(amax)
    if amax == 0.0 or not np.isfinite(amax):
        return 1.0
    _, ex = np.frexp(amax / 448.0)
    s = float(np.ldexp(1.0, int(ex)))        # candidate, may be one binade off after the division
    while amax > 448.0 * s:
        s *= 2.0
    while amax <= 448.0 * (s / 2.0):
        s /= 2.0
    return s


def quantise_tile(T, prec):
    """Round a tile (float64) into storage precision `prec`; returns (dequantised values, scale).

    FP32/FP16: plain rounding, scale 1.  FP8: scale s = fp8_tile_scale(max|T|), stored payload
    q = rd_e4m3(T / s), value s * q (division and multiplication by a power of two are exact).
    """
    if prec == FP32:
        return rd_fp32(T), 1.0
    if prec == FP16:
        return rd_fp16(T), 1.0
    if prec == FP8:
        s = fp8_tile_scale(np.max(np.abs(T)) if T.size else 0.0)
        return rd_e4m3(T / s) * s, s
    raise ValueError(f"unknown precision code {prec}")

// Shared host/device definitions of the CUDA path (no arithmetic of the method lives here).
#pragma once
#include <cuda_fp16.h>
#include <cuda_fp8.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/krr_mp.h"

namespace krr {

constexpr int kBlk = 128;          // row/column sub-block of the panel algorithm and GEMM tile edge
constexpr int kMaxNT = 1024;

// scl[] (device, written by plane_scale_kernel): power-of-two scales of the FP16 operand images and the exact
// rescalings of the accumulators.  sx: L and X values, ss: Schur-complement values, sm: M = inv(L_kk) and M^T,
// su: the intermediate U = L21 M11 of the inverse's recursion.
enum { SCL_SX = 0, SCL_SS = 1, SCL_INV_SX2 = 2, SCL_INV_SS = 3, SCL_SM = 4, SCL_SU = 5, SCL_INV_SM_SX = 6, SCL_INV_SM_SU = 7,
       SCL_INV_SS_SM = 8, SCL_COUNT = 16 };

// Index of tile (i,j), i >= j, in column-major order over the lower triangle (all tiles of one
// tile column are consecutive, so a tile column is one contiguous [m x nb] slab of a plane).
__host__ __device__ __forceinline__ int64_t tile_slot(int NT, int i, int j) {
    return static_cast<int64_t>(j) * NT - static_cast<int64_t>(j) * (j - 1) / 2 + (i - j);
}

// View of the input matrix A = K + lambda*I (FP32): dense row-major with lda, or lower tiles packed.
struct AView {
    const float* base;
    int64_t lda;
    int tiled;   // KRR_FLAG_A_TILED_LOWER
    int NT;
    int nb;
    // pointer to element (r, c) of tile (i, j), i >= j
    __host__ __device__ __forceinline__ const float* tile_ptr(int i, int j, int r, int c) const {
        if (tiled)
            return base + (tile_slot(NT, i, j) * nb + r) * static_cast<int64_t>(nb) + c;
        return base + (static_cast<int64_t>(i) * nb + r) * lda + static_cast<int64_t>(j) * nb + c;
    }
    __host__ __device__ __forceinline__ int64_t row_stride() const { return tiled ? nb : lda; }
};

// Power-of-two per-tile FP8 scale: the smallest s = 2^e with amax <= 448 * s (s = 1 for amax = 0).
// Exact comparisons only, mirrored (independently written) by the oracle's fp8_tile_scale.
__host__ __device__ __forceinline__ float fp8_scale_from_amax(float amax) {
    if (!(amax > 0.0f) || !(amax < 3.0e38f)) return 1.0f;
    int e;
    frexpf(amax * (1.0f / 448.0f), &e);
    float s = ldexpf(1.0f, e);
    while (amax > 448.0f * s) s *= 2.0f;
    while (amax <= 448.0f * (s * 0.5f)) s *= 0.5f;
    return s;
}

__device__ __forceinline__ uint8_t f32_to_e4m3(float x) {
    return static_cast<uint8_t>(__nv_cvt_float_to_fp8(x, __NV_SATFINITE, __NV_E4M3));
}
__device__ __forceinline__ float e4m3_to_f32(uint8_t q) {
    __half_raw h = __nv_cvt_fp8_to_halfraw(q, __NV_E4M3);
    return __half2float(*reinterpret_cast<__half*>(&h));
}

// Round x into storage precision p (value domain), FP8 with the given power-of-two scale.
__device__ __forceinline__ float round_to_prec(float x, int p, float s) {
    if (p == KRR_FP16) return __half2float(__float2half_rn(x));
    if (p == KRR_FP8_E4M3) return e4m3_to_f32(f32_to_e4m3(x / s)) * s;
    return x;
}

// Element sizes of the mosaic payload
__host__ __device__ __forceinline__ int prec_bytes(int p) { return p == KRR_FP32 ? 4 : (p == KRR_FP16 ? 2 : 1); }

// Programmatic dependent launch (PTX griddepcontrol, sm_90+): a kernel launched with the programmatic-stream-serialization
// attribute may start -- prologue, loads of data no earlier kernel writes -- once every CTA of the kernel before it in the
// stream has called pdl_trigger() (or exited); pdl_wait() then blocks until that kernel has completed and its writes are
// visible.  Both are no-ops in a kernel launched the ordinary way.
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// Launch counter (host, per thread) for krr_last_launch_count().
extern thread_local int64_t g_launches;

#define KRR_CUDA_CHECK(expr)                                   \
    do {                                                       \
        cudaError_t _e = (expr);                               \
        if (_e != cudaSuccess) return KRR_ERR_CUDA;            \
    } while (0)

}  // namespace krr

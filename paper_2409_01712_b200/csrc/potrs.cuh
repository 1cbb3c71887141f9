// krr_potrs kernels: forward and backward substitution in FP32 with the tile mosaic
// ("W <- Solve(K~, P_h)", "forward and backward substitution operations
// in the full FP32 precision").  nrhs is small (1..32), so each sweep is bound by reading L once
// from HBM and by 2*nrhs FP32 flops per element of L.  Right-hand sides are
// row-major n x nrhs.
//
// Structure (right-looking over tile columns, like the paper's tile algorithm):
//   trtri128_kernel (tri128.cuh)   inverses of the 128x128 diagonal blocks of every diagonal tile, once
//   potrs_tile_inverse_kernel      from them the inverses of the whole diagonal tiles (and their transposes), once
//   potrs_diagmul_kernel           one diagonal tile: z_k = inv(L_kk) t_k (forward) or inv(L_kk)^T t_k (backward)
//                                  as ONE product -- no chain of dependent 128-row block solves
//   potrs_fwd_update_kernel        Y_i -= L_ik Z_k for tile rows i in a range (the single tiles the chain waits for)
//   potrs_bwd_update_kernel        Z_j -= L_kj^T alpha_k for tile columns j in a range (likewise)
//   potrs_stream_update_kernel     (potrs_stream.cuh) the bulk of both: all the other tiles of column / row k, by TMA
// All sums are accumulated in a fixed order: results are deterministic.
#pragma once
#include <cooperative_groups.h>

#include "common.cuh"

namespace krr {

constexpr int kMaxRhs = 32;
constexpr int kSolveThreads = 256;          // update kernels
constexpr int kDiagThreads = 256;           // diagonal-tile product kernel: CTAs of 8 warps

// Dequantising loads of CPL (4 or 2) consecutive elements of a mosaic tile (element index e).
__device__ __forceinline__ float4 load4(const uint8_t* tile, int p, float s, int64_t e) {
    if (p == KRR_FP32) return __ldg(reinterpret_cast<const float4*>(tile + e * 4));
    if (p == KRR_FP16) {
        const uint2 raw = __ldg(reinterpret_cast<const uint2*>(tile + e * 2));
        const __half2 a = *reinterpret_cast<const __half2*>(&raw.x);
        const __half2 b = *reinterpret_cast<const __half2*>(&raw.y);
        return make_float4(__low2float(a), __high2float(a), __low2float(b), __high2float(b));
    }
    const uint32_t raw = __ldg(reinterpret_cast<const uint32_t*>(tile + e));
    return make_float4(e4m3_to_f32(raw & 0xff) * s, e4m3_to_f32((raw >> 8) & 0xff) * s,
                       e4m3_to_f32((raw >> 16) & 0xff) * s, e4m3_to_f32(raw >> 24) * s);
}
__device__ __forceinline__ float2 load2(const uint8_t* tile, int p, float s, int64_t e) {
    if (p == KRR_FP32) return __ldg(reinterpret_cast<const float2*>(tile + e * 4));
    if (p == KRR_FP16) {
        const uint32_t raw = __ldg(reinterpret_cast<const uint32_t*>(tile + e * 2));
        const __half2 a = *reinterpret_cast<const __half2*>(&raw);
        return make_float2(__low2float(a), __high2float(a));
    }
    const uint16_t raw = __ldg(reinterpret_cast<const uint16_t*>(tile + e));
    return make_float2(e4m3_to_f32(raw & 0xff) * s, e4m3_to_f32(raw >> 8) * s);
}

// The same with the storage precision known at compile time (the update kernels switch on the tile's
// precision once, outside their streaming loops, so that several iterations' loads stay in flight).
template <int P>
__device__ __forceinline__ float4 load4p(const uint8_t* tile, float s, int64_t e) {
    if (P == KRR_FP32) return __ldg(reinterpret_cast<const float4*>(tile + e * 4));
    if (P == KRR_FP16) {
        const uint2 raw = __ldg(reinterpret_cast<const uint2*>(tile + e * 2));
        const __half2 a = *reinterpret_cast<const __half2*>(&raw.x);
        const __half2 b = *reinterpret_cast<const __half2*>(&raw.y);
        return make_float4(__low2float(a), __high2float(a), __low2float(b), __high2float(b));
    }
    const uint32_t raw = __ldg(reinterpret_cast<const uint32_t*>(tile + e));
    return make_float4(e4m3_to_f32(raw & 0xff) * s, e4m3_to_f32((raw >> 8) & 0xff) * s,
                       e4m3_to_f32((raw >> 16) & 0xff) * s, e4m3_to_f32(raw >> 24) * s);
}
template <int P>
__device__ __forceinline__ float2 load2p(const uint8_t* tile, float s, int64_t e) {
    if (P == KRR_FP32) return __ldg(reinterpret_cast<const float2*>(tile + e * 4));
    if (P == KRR_FP16) {
        const uint32_t raw = __ldg(reinterpret_cast<const uint32_t*>(tile + e * 2));
        const __half2 a = *reinterpret_cast<const __half2*>(&raw);
        return make_float2(__low2float(a), __high2float(a));
    }
    const uint16_t raw = __ldg(reinterpret_cast<const uint16_t*>(tile + e));
    return make_float2(e4m3_to_f32(raw & 0xff) * s, e4m3_to_f32(raw >> 8) * s);
}

template <int P>
__device__ __forceinline__ float load1p(const uint8_t* tile, float s, int64_t e) {
    if (P == KRR_FP32) return __ldg(reinterpret_cast<const float*>(tile + e * 4));
    if (P == KRR_FP16) return __half2float(__ldg(reinterpret_cast<const __half*>(tile + e * 2)));
    return e4m3_to_f32(__ldg(tile + e)) * s;
}

// Sum 64 per-lane values v[0..63] across the 32 lanes of a warp with 62 shuffles (each step halves
// the number of values a lane carries).  Afterwards lane `l` holds in v[0], v[1] the totals of the
// values with index  warp_reduce64_index(l) + {0, 1}.
__device__ __forceinline__ void warp_reduce64(float (&v)[64], int lane) {
#pragma unroll
    for (int step = 0; step < 5; ++step) {
        const int o = 16 >> step;            // lane offset 16, 8, 4, 2, 1
        const int cnt = 32 >> step;          // values kept after this step
        const bool upper = (lane & o) != 0;
#pragma unroll
        for (int i = 0; i < cnt; ++i) {
            const float send = upper ? v[i] : v[i + cnt];
            const float keep = upper ? v[i + cnt] : v[i];
            v[i] = keep + __shfl_xor_sync(0xffffffffu, send, o);
        }
    }
}
__device__ __forceinline__ int warp_reduce64_index(int lane) {
    return ((lane & 16) ? 32 : 0) + ((lane & 8) ? 16 : 0) + ((lane & 4) ? 8 : 0) + ((lane & 2) ? 4 : 0) +
           ((lane & 1) ? 2 : 0);
}

// acc[u*NRHS + h] += sum_{l in [0,K)} row_u[l] * zs[h*zld + l]  for u in [0, ROWS), ROWS*NRHS = 64.
// One warp; lanes stride over l in float4 chunks (K % 128 == 0).  rows: FP32, row stride ld floats.
template <int NRHS>
__device__ __forceinline__ void rows_dot_f32(const float* __restrict__ rows, int64_t ld, int K,
                                             const float* __restrict__ zs, int zld, int lane, float (&acc)[64]) {
    constexpr int ROWS = 64 / NRHS;
#pragma unroll 2
    for (int l = lane * 4; l < K; l += 128) {
        float4 a[ROWS];
#pragma unroll
        for (int u = 0; u < ROWS; ++u) a[u] = __ldg(reinterpret_cast<const float4*>(rows + u * ld + l));
#pragma unroll
        for (int h = 0; h < NRHS; ++h) {
            const float4 z = *reinterpret_cast<const float4*>(zs + h * zld + l);
#pragma unroll
            for (int u = 0; u < ROWS; ++u)
                acc[u * NRHS + h] = fmaf(a[u].x, z.x, fmaf(a[u].y, z.y, fmaf(a[u].z, z.z, fmaf(a[u].w, z.w, acc[u * NRHS + h]))));
        }
    }
}

// The same for a low-precision tile (P = KRR_FP16 / KRR_FP8_E4M3, scale s): rows r0 .. r0+ROWS of `tile`.
// The loads are 8 / 4 bytes per lane, so four iterations are kept in flight.
template <int NRHS, int P>
__device__ __forceinline__ void rows_dot_lp(const uint8_t* __restrict__ tile, float s, int r0, int nb,
                                            const float* __restrict__ zs, int lane, float (&acc)[64]) {
    constexpr int ROWS = 64 / NRHS;
#pragma unroll 4
    for (int l = lane * 4; l < nb; l += 128) {
        float4 a[ROWS];
#pragma unroll
        for (int u = 0; u < ROWS; ++u) a[u] = load4p<P>(tile, s, static_cast<int64_t>(r0 + u) * nb + l);
#pragma unroll
        for (int h = 0; h < NRHS; ++h) {
            const float4 z = *reinterpret_cast<const float4*>(zs + h * nb + l);
#pragma unroll
            for (int u = 0; u < ROWS; ++u)
                acc[u * NRHS + h] = fmaf(a[u].x, z.x, fmaf(a[u].y, z.y, fmaf(a[u].z, z.z, fmaf(a[u].w, z.w, acc[u * NRHS + h]))));
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Forward update after Z_k is known:  Y_i -= L_ik Z_k  for the tile rows i in [i_lo, i_hi)  (all > k).
// Persistent CTAs over groups of 8 * ROWS rows (ROWS = 64 / NRHS rows per warp); smem = NRHS*nb floats (Z_k) + the
// tiles' (offset, precision, scale), fetched once per CTA so that a warp task starts streaming at once.
// Tried and dropped (r02): streaming the tile through a per-warp cp.async ring in shared memory (16 KB in flight per
// warp, one CTA per SM): 12.5 -> 13.8 ms for the whole solve at n = 65536 -- the kernel is bound by the shared-memory
// reads of Z_k (16 LDS.128 per 256 FMAs and warp), not by load latency.
template <int NRHS>
__global__ void __launch_bounds__(kSolveThreads)
potrs_fwd_update_kernel(int NT, int nb, int k, int i_lo, int i_hi, const uint8_t* __restrict__ factor,
                        const int64_t* __restrict__ off, const uint8_t* __restrict__ map,
                        const float* __restrict__ scales, float* __restrict__ B, int64_t ldb, int nrhs) {
    constexpr int ROWS = 64 / NRHS;
    constexpr int NW = kSolveThreads / 32;
    extern __shared__ __align__(16) float zs[];        // [NRHS][nb], then the tiles' (offset, precision, scale)
    int64_t* t_off = reinterpret_cast<int64_t*>(zs + static_cast<size_t>(NRHS) * nb);
    int* t_prec = reinterpret_cast<int*>(t_off + (i_hi - i_lo));
    float* t_scale = reinterpret_cast<float*>(t_prec + (i_hi - i_lo));
    const float* Zk = B + static_cast<int64_t>(k) * nb * ldb;
    for (int idx = threadIdx.x; idx < nb * NRHS; idx += kSolveThreads) {
        const int c = idx / NRHS, rh = idx % NRHS;
        zs[rh * nb + c] = (rh < nrhs) ? Zk[static_cast<int64_t>(c) * ldb + rh] : 0.0f;
    }
    for (int t = threadIdx.x; t < i_hi - i_lo; t += kSolveThreads) {
        const int i = i_lo + t;
        t_off[t] = off[i * NT + k];
        t_prec[t] = map[i * NT + k];
        t_scale[t] = scales[i * NT + k];
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t ngroups = static_cast<int64_t>(i_hi - i_lo) * nb / ROWS;   // warp tasks
    for (int64_t g = static_cast<int64_t>(blockIdx.x) * NW + warp; g < ngroups; g += static_cast<int64_t>(gridDim.x) * NW) {
        const int64_t prow = g * ROWS;                                      // row below the top of tile i_lo
        const int ti = static_cast<int>(prow / nb);
        const int i = i_lo + ti;
        const int r0 = static_cast<int>(prow % nb);
        const int p = t_prec[ti];
        const float s = t_scale[ti];
        const uint8_t* tile = factor + t_off[ti];
        float acc[64];
#pragma unroll
        for (int v = 0; v < 64; ++v) acc[v] = 0.0f;
        if (p == KRR_FP32) {
            rows_dot_f32<NRHS>(reinterpret_cast<const float*>(tile) + static_cast<int64_t>(r0) * nb, nb, nb, zs, nb, lane, acc);
        } else if (p == KRR_FP16) {
            rows_dot_lp<NRHS, KRR_FP16>(tile, s, r0, nb, zs, lane, acc);
        } else {
            rows_dot_lp<NRHS, KRR_FP8_E4M3>(tile, s, r0, nb, zs, lane, acc);
        }
        warp_reduce64(acc, lane);
        const int v0 = warp_reduce64_index(lane);
#pragma unroll
        for (int t = 0; t < 2; ++t) {
            const int u = (v0 + t) / NRHS, h = (v0 + t) % NRHS;
            if (h < nrhs) B[(static_cast<int64_t>(i) * nb + r0 + u) * ldb + h] -= acc[t];
        }
    }
}

// Streaming loop of the backward update: the rows of one strip of a tile (storage precision P), RU rows per
// warp and iteration, against alpha_k in shared memory (`as`: [nb][NRHS]).  Every column's sum runs over the rows
// warp, warp + NW, warp + 2 NW, ... in this order whatever CPL and RU are, so all variants give identical results.
template <int NRHS, int CPL, int P>
__device__ __forceinline__ void bwd_rows(const uint8_t* __restrict__ tile, float s, int c0, int nb,
                                         const float* __restrict__ as, int warp, float (&acc)[CPL * NRHS]) {
    constexpr int NW = kSolveThreads / 32;
    constexpr int RU = (CPL == 1) ? 16 : 4;
#pragma unroll ((P == KRR_FP32 || CPL == 1) ? 2 : 4)
    for (int r = warp; r < nb; r += NW * RU) {
        float l[RU][CPL];
#pragma unroll
        for (int u = 0; u < RU; ++u) {
            const int64_t e = static_cast<int64_t>(r + u * NW) * nb + c0;
            if (CPL == 4) {
                const float4 v = load4p<P>(tile, s, e);
                l[u][0] = v.x; l[u][1] = v.y; l[u][CPL - 2] = v.z; l[u][CPL - 1] = v.w;
            } else if (CPL == 2) {
                const float2 v = load2p<P>(tile, s, e);
                l[u][0] = v.x; l[u][1] = v.y;
            } else {
                l[u][0] = load1p<P>(tile, s, e);
            }
        }
#pragma unroll
        for (int u = 0; u < RU; ++u) {
            const float* ar = as + static_cast<size_t>(r + u * NW) * NRHS;
#pragma unroll
            for (int h = 0; h < NRHS; h += 4) {
                const float4 a = *reinterpret_cast<const float4*>(ar + h);
#pragma unroll
                for (int c = 0; c < CPL; ++c) {
                    acc[c * NRHS + h + 0] = fmaf(l[u][c], a.x, acc[c * NRHS + h + 0]);
                    acc[c * NRHS + h + 1] = fmaf(l[u][c], a.y, acc[c * NRHS + h + 1]);
                    acc[c * NRHS + h + 2] = fmaf(l[u][c], a.z, acc[c * NRHS + h + 2]);
                    acc[c * NRHS + h + 3] = fmaf(l[u][c], a.w, acc[c * NRHS + h + 3]);
                }
            }
        }
    }
}

// Backward update after alpha_k is known:  Z_j -= L_kj^T alpha_k  for the tiles j in [j_lo, j_lo + gridDim.x / strips)
// (all < k).  One CTA per (tile j, strip of 32*CPL columns); warps split the nb rows (interleaved), lanes own
// CPL consecutive columns; the per-warp partial sums are combined through shared memory in a fixed
// tree order.  smem = nb*NRHS floats (alpha_k) + (NW/2) * 32*CPL*NRHS floats.
// CPL = 4 (2 for NRHS = 32) for the bulk launches; CPL = 1 (four times the CTAs per tile, sixteen rows in flight per
// warp) for the single tile on the chain stream that the next diagonal solve waits for.
template <int NRHS, int CPL>
__global__ void __launch_bounds__(kSolveThreads)
potrs_bwd_update_kernel(int NT, int nb, int k, int j_lo, int ntiles, const uint8_t* __restrict__ factor,
                        const int64_t* __restrict__ off, const uint8_t* __restrict__ map,
                        const float* __restrict__ scales, float* __restrict__ B, int64_t ldb, int nrhs) {
    constexpr int NACC = CPL * NRHS;
    constexpr int NW = kSolveThreads / 32;
    constexpr int STRIP = 32 * CPL;
    extern __shared__ __align__(16) float as[];        // [nb][NRHS] alpha_k, then the reduction buffers
    float* red = as + static_cast<size_t>(nb) * NRHS;  // [NW/2][32 lanes][NACC]
    const float* Ak = B + static_cast<int64_t>(k) * nb * ldb;
    for (int idx = threadIdx.x; idx < nb * NRHS; idx += kSolveThreads) {
        const int r = idx / NRHS, rh = idx % NRHS;
        as[idx] = (rh < nrhs) ? Ak[static_cast<int64_t>(r) * ldb + rh] : 0.0f;
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int strips = nb / STRIP;
    // units = (tile j, strip of 32 * CPL columns), dealt round-robin to the persistent CTAs (alpha_k is staged once per CTA)
    for (int unit = blockIdx.x; unit < ntiles * strips; unit += gridDim.x) {
        const int j = j_lo + unit / strips;
        const int c0 = (unit % strips) * STRIP + lane * CPL;
        const int p = map[k * NT + j];
        const float s = scales[k * NT + j];
        const uint8_t* tile = factor + off[k * NT + j];
        float acc[NACC];
#pragma unroll
        for (int v = 0; v < NACC; ++v) acc[v] = 0.0f;
        if (p == KRR_FP32) bwd_rows<NRHS, CPL, KRR_FP32>(tile, s, c0, nb, as, warp, acc);
        else if (p == KRR_FP16) bwd_rows<NRHS, CPL, KRR_FP16>(tile, s, c0, nb, as, warp, acc);
        else bwd_rows<NRHS, CPL, KRR_FP8_E4M3>(tile, s, c0, nb, as, warp, acc);
        // fixed-order tree over the NW warps
#pragma unroll
        for (int half = NW / 2; half >= 1; half >>= 1) {
            if (warp >= half && warp < 2 * half) {
                float* dst = red + (static_cast<size_t>(warp - half) * 32 + lane) * NACC;
#pragma unroll
                for (int v = 0; v < NACC; v += 4) *reinterpret_cast<float4*>(dst + v) = make_float4(acc[v], acc[v + 1], acc[v + 2], acc[v + 3]);
            }
            __syncthreads();
            if (warp < half) {
                const float* src = red + (static_cast<size_t>(warp) * 32 + lane) * NACC;
#pragma unroll
                for (int v = 0; v < NACC; v += 4) {
                    const float4 t = *reinterpret_cast<const float4*>(src + v);
                    acc[v] += t.x; acc[v + 1] += t.y; acc[v + 2] += t.z; acc[v + 3] += t.w;
                }
            }
            __syncthreads();
        }
        if (warp == 0) {
#pragma unroll
            for (int c = 0; c < CPL; ++c) {
                float* z = B + (static_cast<int64_t>(j) * nb + c0 + c) * ldb;
#pragma unroll
                for (int h = 0; h < NRHS; ++h)
                    if (h < nrhs) z[h] -= acc[c * NRHS + h];
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Inverse of the diagonal tiles in FP32, once per krr_potrs call: Minv[k] = inv(L_kk) and MinvT[k] = its transpose
// (nb x nb row-major each).  With them a diagonal step of either sweep is ONE product, z_k = inv(L_kk) t_k, instead
// of a chain of nb/128 dependent block solves.  CTA (c, k) produces block column c of Minv[k] by forward
// substitution over the 128-blocks with the inverted diagonal blocks D_r of trtri128_kernel:
//     X_c = D_c,   X_r = -D_r (sum_{j = c}^{r-1} L_rj X_j)   for r > c,
// every term a 128 x 128 x 128 FP32 product out of shared memory (8 x 8 outputs per thread, fixed summation order).
constexpr int kTinvThreads = 256;
constexpr int kTinvLd = kBlk + 4;
constexpr int kTinvSmem = (2 * 16 * kTinvLd + kBlk * kTinvLd) * 4;       // A chunk, B chunk, T

// acc += A B for 128 x 128 blocks: A row-major (global or shared, leading dimension lda), B row-major (ldb).
__device__ __forceinline__ void tinv_block_mma(const float* __restrict__ A, int64_t lda, const float* __restrict__ B, int64_t ldb,
                                               float* As, float* Bs, float (&acc)[8][8], int tid) {
    const int ty = tid >> 4, tx = tid & 15;
    for (int k0 = 0; k0 < kBlk; k0 += 16) {
        {
            const int row = tid >> 1, kk = (tid & 1) * 8;
            const float4 v0 = *reinterpret_cast<const float4*>(A + row * lda + k0 + kk);
            const float4 v1 = *reinterpret_cast<const float4*>(A + row * lda + k0 + kk + 4);
            As[(kk + 0) * kTinvLd + row] = v0.x; As[(kk + 1) * kTinvLd + row] = v0.y;
            As[(kk + 2) * kTinvLd + row] = v0.z; As[(kk + 3) * kTinvLd + row] = v0.w;
            As[(kk + 4) * kTinvLd + row] = v1.x; As[(kk + 5) * kTinvLd + row] = v1.y;
            As[(kk + 6) * kTinvLd + row] = v1.z; As[(kk + 7) * kTinvLd + row] = v1.w;
            const int kr = tid >> 4, nn = (tid & 15) * 8;
            *reinterpret_cast<float4*>(Bs + kr * kTinvLd + nn) = *reinterpret_cast<const float4*>(B + kr * ldb + nn + k0 * ldb);
            *reinterpret_cast<float4*>(Bs + kr * kTinvLd + nn + 4) = *reinterpret_cast<const float4*>(B + kr * ldb + nn + 4 + k0 * ldb);
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < 16; ++kk) {
            const float4 a0 = *reinterpret_cast<const float4*>(As + kk * kTinvLd + ty * 8);
            const float4 a1 = *reinterpret_cast<const float4*>(As + kk * kTinvLd + ty * 8 + 4);
            const float4 b0 = *reinterpret_cast<const float4*>(Bs + kk * kTinvLd + tx * 8);
            const float4 b1 = *reinterpret_cast<const float4*>(Bs + kk * kTinvLd + tx * 8 + 4);
            const float av[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
            const float bv[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
#pragma unroll
            for (int i = 0; i < 8; ++i)
#pragma unroll
                for (int j = 0; j < 8; ++j) acc[i][j] = fmaf(av[i], bv[j], acc[i][j]);
        }
        __syncthreads();
    }
}

// grid = (nsub, NT).  dinv: the inverted 128 x 128 diagonal blocks ([n/128][128][128], trtri128_kernel).
__global__ void __launch_bounds__(kTinvThreads, 2)
potrs_tile_inverse_kernel(const uint8_t* __restrict__ factor, const int64_t* __restrict__ off, int NT, int nb,
                          const float* __restrict__ dinv, float* __restrict__ Minv, float* __restrict__ MinvT) {
    extern __shared__ __align__(16) float tinv_sm[];
    float* As = tinv_sm;
    float* Bs = As + 16 * kTinvLd;
    float* Ts = Bs + 16 * kTinvLd;                                    // [128][kTinvLd]
    const int nsub = nb / kBlk;
    const int c = nsub - 1 - static_cast<int>(blockIdx.x);            // the long block columns are scheduled first
    const int k = blockIdx.y;
    const int tid = threadIdx.x, ty = tid >> 4, tx = tid & 15;
    const float* L = reinterpret_cast<const float*>(factor + off[static_cast<int64_t>(k) * NT + k]);
    float* M = Minv + static_cast<int64_t>(k) * nb * nb;
    float* MT = MinvT + static_cast<int64_t>(k) * nb * nb;
    const float* D = dinv + static_cast<int64_t>(k) * nsub * kBlk * kBlk;
    auto store_block = [&](int r, const float (&x)[8][8]) {           // X_r into M[r-block rows][c-block columns] and transposed
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            float* dst = M + static_cast<int64_t>(r * kBlk + ty * 8 + i) * nb + c * kBlk + tx * 8;
            *reinterpret_cast<float4*>(dst) = make_float4(x[i][0], x[i][1], x[i][2], x[i][3]);
            *reinterpret_cast<float4*>(dst + 4) = make_float4(x[i][4], x[i][5], x[i][6], x[i][7]);
        }
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            float* dst = MT + static_cast<int64_t>(c * kBlk + tx * 8 + j) * nb + r * kBlk + ty * 8;
            *reinterpret_cast<float4*>(dst) = make_float4(x[0][j], x[1][j], x[2][j], x[3][j]);
            *reinterpret_cast<float4*>(dst + 4) = make_float4(x[4][j], x[5][j], x[6][j], x[7][j]);
        }
    };
    {
        float x[8][8];
        const float* Dc = D + static_cast<int64_t>(c) * kBlk * kBlk;
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int j = 0; j < 8; ++j) x[i][j] = Dc[(ty * 8 + i) * kBlk + tx * 8 + j];
        store_block(c, x);
    }
    for (int r = c + 1; r < nsub; ++r) {
        __syncthreads();                                              // X_c .. X_{r-1} are in global memory (this CTA wrote them)
        float acc[8][8];
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int j = 0; j < 8; ++j) acc[i][j] = 0.0f;
        for (int j = c; j < r; ++j)
            tinv_block_mma(L + static_cast<int64_t>(r) * kBlk * nb + j * kBlk, nb, M + static_cast<int64_t>(j) * kBlk * nb + c * kBlk, nb,
                           As, Bs, acc, tid);
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int j = 0; j < 8; ++j) Ts[(ty * 8 + i) * kTinvLd + tx * 8 + j] = -acc[i][j];
        __syncthreads();
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int j = 0; j < 8; ++j) acc[i][j] = 0.0f;
        tinv_block_mma(D + static_cast<int64_t>(r) * kBlk * kBlk, kBlk, Ts, kTinvLd, As, Bs, acc, tid);
        store_block(r, acc);
    }
}

// Diagonal step of a sweep as one product, rows k*nb .. (k+1)*nb of B:
//     forward   z_k = inv(L_kk) t_k      (Mk = Minv[k],  lower triangular: row block b meets columns [0, 128 (b+1)))
//     backward  a_k = inv(L_kk)^T t_k    (Mk = MinvT[k], upper triangular: row block b meets columns [128 b, nb))
// t_k is first copied out of B into a compact [nb][NRHS] buffer (potrs_stage_kernel), so that the product can write its
// result over t_k in B while other CTAs still read t_k.  One CTA per group of 64 / NRHS rows; its eight warps split the
// K range in slices of whole 128-column steps, lane = 4 consecutive columns; the slices are added in a fixed order
// through shared memory: deterministic.  The launch is short (one DRAM round trip per warp) and wide (nb NRHS / 64 CTAs).
// The updates of these rows by the two previous tile columns may have been left as partial sums (potrs_stream.cuh, ksplit):
// Pm[slice][nb][NRHS] (nm slices) by the column before the previous one ("mid"), Pn (nn slices) by the previous one
// ("near").  They are subtracted here in that order, lowest slice first -- a fixed order.
template <int NRHS>
__global__ void __launch_bounds__(256)
potrs_stage_kernel(int nb, const float* __restrict__ Bk, int64_t ldb, int nrhs, float* __restrict__ T,
                   const float* __restrict__ Pm, int nm, const float* __restrict__ Pn, int nn) {
    pdl_trigger();
    pdl_wait();
    const int idx = blockIdx.x * 256 + threadIdx.x;
    if (idx < nb * NRHS) {
        const int r = idx / NRHS, h = idx % NRHS;
        float v = (h < nrhs) ? Bk[static_cast<int64_t>(r) * ldb + h] : 0.0f;
        for (int s = 0; s < nm; ++s) v -= Pm[static_cast<size_t>(s) * nb * NRHS + idx];
        for (int s = 0; s < nn; ++s) v -= Pn[static_cast<size_t>(s) * nb * NRHS + idx];
        T[idx] = v;
    }
}

template <int NRHS>
__global__ void __launch_bounds__(kDiagThreads)
potrs_diagmul_kernel(int nb, const float* __restrict__ Mk, const float* __restrict__ T, float* __restrict__ Bk, int64_t ldb,
                     int nrhs, int backward) {
    constexpr int ROWS = 64 / NRHS;
    constexpr int NW = kDiagThreads / 32;
    __shared__ float red[NW][64];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int r0 = blockIdx.x * ROWS;
    const int blk = r0 / kBlk;
    const int k_lo = backward ? blk * kBlk : 0, k_hi = backward ? nb : (blk + 1) * kBlk;
    const int steps = (k_hi - k_lo) / kBlk;                        // 128-column steps of the row group
    float acc[64];
#pragma unroll
    for (int v = 0; v < 64; ++v) acc[v] = 0.0f;
    pdl_trigger();
    pdl_wait();                                                    // T is the stage kernel's output
    // step s of the range goes to warp s % NW (a fixed assignment)
    for (int st = warp; st < steps; st += NW) {
        const int l = k_lo + st * kBlk + lane * 4;
        float4 a[ROWS];
#pragma unroll
        for (int u = 0; u < ROWS; ++u) a[u] = __ldg(reinterpret_cast<const float4*>(Mk + static_cast<int64_t>(r0 + u) * nb + l));
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
            float y[NRHS];
#pragma unroll
            for (int h = 0; h < NRHS; h += 4) {
                const float4 v = __ldg(reinterpret_cast<const float4*>(T + static_cast<int64_t>(l + kk) * NRHS + h));
                y[h] = v.x; y[h + 1] = v.y; y[h + 2] = v.z; y[h + 3] = v.w;
            }
#pragma unroll
            for (int u = 0; u < ROWS; ++u) {
                const float av = kk == 0 ? a[u].x : (kk == 1 ? a[u].y : (kk == 2 ? a[u].z : a[u].w));
#pragma unroll
                for (int h = 0; h < NRHS; ++h) acc[u * NRHS + h] = fmaf(av, y[h], acc[u * NRHS + h]);
            }
        }
    }
    warp_reduce64(acc, lane);
    const int v0 = warp_reduce64_index(lane);
    red[warp][v0] = acc[0];
    red[warp][v0 + 1] = acc[1];
    __syncthreads();
    if (threadIdx.x < 64) {
        float sum = 0.0f;
#pragma unroll
        for (int w2 = 0; w2 < NW; ++w2) sum += red[w2][threadIdx.x];
        const int u = threadIdx.x / NRHS, h = threadIdx.x % NRHS;
        if (h < nrhs) Bk[static_cast<int64_t>(r0 + u) * ldb + h] = sum;
    }
}

}  // namespace krr

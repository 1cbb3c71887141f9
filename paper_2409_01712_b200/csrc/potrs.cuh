// krr_potrs kernels: forward and backward substitution in FP32 with the tile mosaic
// ("W <- Solve(K~, P_h)", "forward and backward substitution operations
// in the full FP32 precision").  nrhs is small (1..32), so each sweep is bound by reading L once
// from HBM and by 2*nrhs FP32 flops per element of L.  Right-hand sides are
// row-major n x nrhs.
//
// Structure (right-looking over tile columns, like the paper's tile algorithm):
//   trtri128_kernel (tri128.cuh)   inverses of the 128x128 diagonal blocks of every diagonal tile, once
//   potrs_diag_transpose_kernel    transposed copies of the diagonal tiles for the backward sweep, once
//   potrs_diag_kernel              one diagonal tile: 128-row blocks in order, each a product with the
//                                  already solved part of the tile followed by a product with the
//                                  inverted diagonal block
//   potrs_fwd_update_kernel        Y_i -= L_ik Z_k for all i > k   (streams tile column k once)
//   potrs_bwd_update_kernel        Z_j -= L_kj^T alpha_k for all j < k (streams tile row k once)
// All sums are accumulated in a fixed order: results are deterministic.
#pragma once
#include <cooperative_groups.h>

#include "common.cuh"

namespace krr {

constexpr int kMaxRhs = 32;
constexpr int kSolveThreads = 256;          // update kernels
constexpr int kDiagThreads = 256;           // diagonal-tile kernel: CTAs of 8 warps ...
constexpr int kDiagCluster = 8;             // ... in a cluster of 8

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
// Persistent CTAs over groups of 8 * ROWS rows (ROWS = 64 / NRHS rows per warp); smem = NRHS*nb floats.
template <int NRHS>
__global__ void __launch_bounds__(kSolveThreads)
potrs_fwd_update_kernel(int NT, int nb, int k, int i_lo, int i_hi, const uint8_t* __restrict__ factor,
                        const int64_t* __restrict__ off, const uint8_t* __restrict__ map,
                        const float* __restrict__ scales, float* __restrict__ B, int64_t ldb, int nrhs) {
    constexpr int ROWS = 64 / NRHS;
    constexpr int NW = kSolveThreads / 32;
    extern __shared__ __align__(16) float zs[];        // [NRHS][nb]
    const float* Zk = B + static_cast<int64_t>(k) * nb * ldb;
    for (int idx = threadIdx.x; idx < nb * NRHS; idx += kSolveThreads) {
        const int c = idx / NRHS, rh = idx % NRHS;
        zs[rh * nb + c] = (rh < nrhs) ? Zk[static_cast<int64_t>(c) * ldb + rh] : 0.0f;
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t ngroups = static_cast<int64_t>(i_hi - i_lo) * nb / ROWS;   // warp tasks
    for (int64_t g = static_cast<int64_t>(blockIdx.x) * NW + warp; g < ngroups; g += static_cast<int64_t>(gridDim.x) * NW) {
        const int64_t prow = g * ROWS;                                      // row below the top of tile i_lo
        const int i = i_lo + static_cast<int>(prow / nb);
        const int r0 = static_cast<int>(prow % nb);
        const int p = map[i * NT + k];
        const float s = scales[i * NT + k];
        const uint8_t* tile = factor + off[i * NT + k];
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
potrs_bwd_update_kernel(int NT, int nb, int k, int j_lo, const uint8_t* __restrict__ factor,
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
    const int j = j_lo + blockIdx.x / strips;
    const int c0 = (blockIdx.x % strips) * STRIP + lane * CPL;
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

// ---------------------------------------------------------------------------------------------
// Transposed copies of the diagonal tiles (FP32, full squares): T[k] = L_kk^T, so that the backward solve reads
// rows of L^T exactly as the forward solve reads rows of L.  One CTA per 32 x 32 block with row block <= column
// block of L^T (the rest is never read).  Once per krr_potrs call: 2 * 4 * nb^2 / 2 bytes per tile.
__global__ void __launch_bounds__(256)
potrs_diag_transpose_kernel(const uint8_t* __restrict__ factor, const int64_t* __restrict__ off, int NT, int nb,
                            float* __restrict__ T) {
    __shared__ float t[32][33];
    const int k = blockIdx.z, bi = blockIdx.y, bj = blockIdx.x;        // block (bi, bj) of L^T = block (bj, bi) of L
    if (bi > bj) return;
    const float* L = reinterpret_cast<const float*>(factor + off[static_cast<int64_t>(k) * NT + k]);
    float* Tk = T + static_cast<int64_t>(k) * nb * nb;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
#pragma unroll
    for (int r = ty; r < 32; r += 8) t[r][tx] = L[static_cast<int64_t>(bj * 32 + r) * nb + bi * 32 + tx];
    __syncthreads();
#pragma unroll
    for (int r = ty; r < 32; r += 8) Tk[static_cast<int64_t>(bi * 32 + r) * nb + bj * 32 + tx] = t[tx][r];
}

// Diagonal tile solve by one thread-block cluster of kDiagCluster CTAs: forward (L z = y) or
// backward (L^T a = z), in place on rows k*nb .. (k+1)*nb of B.  For each 128-row block c, in order:
//   forward   t = y_c - L[c, 0:c] z_{0:c}                       z_c = inv(L_cc) t
//   backward  t = z_c - (L^T)[c, c+1:] a_{c+1:}                 a_c = inv(L_cc)^T t
// M: the diagonal tile L_kk (forward) or its transposed copy (backward; potrs_diag_transpose_kernel), so both
// directions run the same code: rows of M against the solved values, the K range split over warp slices.
// dinv / dinvT: the inverted diagonal blocks of this tile and their transposes ([nsub][128][128]).
// Every CTA keeps a full copy of the solved values and of t in its shared memory; the rows of a step are split
// over the CTAs, and the pieces are exchanged through distributed shared memory between two cluster barriers.
// smem per CTA: solved values NRHS*nb floats + t NRHS*128 + exchange buffer (see potrs_diag_smem_floats).
template <int NRHS>
__host__ __device__ constexpr int potrs_diag_smem_floats(int nb) {
    // solved + ts + red (K slices: 8 warps * 64 values)
    return NRHS * nb + NRHS * kBlk + 4 * 32 * 64;
}

template <int NRHS>
__global__ void __cluster_dims__(kDiagCluster, 1, 1) __launch_bounds__(kDiagThreads, 1)
potrs_diag_kernel(int nb, const float* __restrict__ Lkk /* M */, const float* __restrict__ dinv,
                  const float* __restrict__ dinvT, float* __restrict__ Bk, int64_t ldb, int nrhs, int backward) {
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    constexpr int ROWS = 64 / NRHS;                    // rows per warp task
    constexpr int NW = kDiagThreads / 32;              // 8 warps
    constexpr int GQ = (kBlk / ROWS) / kDiagCluster;   // row groups per CTA: 1, 2, 4, 8 for NRHS 4, 8, 16, 32
    constexpr int KS = NW / GQ;                        // K slices per row group
    static_assert(GQ >= 1 && KS >= 1 && GQ * KS == NW, "warp decomposition");
    extern __shared__ __align__(16) float sm[];
    float* zs = sm;                                    // [NRHS][nb] solved values, by rhs
    float* ts = sm + static_cast<size_t>(NRHS) * nb;   // [NRHS][128]
    float* red = ts + NRHS * kBlk;                     // [4][32][64] scratch
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int q = static_cast<int>(cluster.block_rank());
    const int nsub = nb / kBlk;
    // pull the part of M that is read and the inverted blocks towards L2 (fire and forget)
    {
        const int gt = q * kDiagThreads + threadIdx.x, nt = kDiagCluster * kDiagThreads;
        for (int c = 0; c < nsub; ++c) {
            const int col0 = backward ? c * kBlk : 0;                     // block row c: columns 0 .. c (L) or c .. nsub-1 (L^T)
            const int lines_per_row = backward ? 4 * (nsub - c) : 4 * (c + 1);
            for (int idx = gt; idx < kBlk * lines_per_row; idx += nt) {
                const float* ptr = Lkk + static_cast<int64_t>(c * kBlk + idx / lines_per_row) * nb + col0 + (idx % lines_per_row) * 32;
                asm volatile("prefetch.global.L2 [%0];" ::"l"(ptr));
            }
        }
        const float* D = backward ? dinvT : dinv;
        for (int idx = gt; idx < nsub * kBlk * 4; idx += nt) asm volatile("prefetch.global.L2 [%0];" ::"l"(D + idx * 32));
    }
    cluster.sync();                                    // every CTA is running before its smem is written remotely
    const int gl = warp % GQ, ks = warp / GQ;          // this warp's row group inside the CTA, K slice
    const int grow = (q * GQ + gl) * ROWS;             // first row (inside a 128 block) of the warp's group
    for (int bi = 0; bi < nsub; ++bi) {
        const int c = backward ? (nsub - 1 - bi) : bi;
        const int R0 = c * kBlk;
        const int k_lo = backward ? R0 + kBlk : 0, k_hi = backward ? nb : R0;      // solved range the block row meets
        // ---- phase 1: t = y_c - M[c, k_lo:k_hi] solved  for this CTA's rows (M = L forward, L^T backward), K split over
        // the warp slices
        float acc[64];
#pragma unroll
        for (int v = 0; v < 64; ++v) acc[v] = 0.0f;
        {
            const float* rows = Lkk + static_cast<int64_t>(R0 + grow) * nb;
            for (int l = k_lo + lane * 4 + ks * 128; l < k_hi; l += 128 * KS) {
                float4 a[ROWS];
#pragma unroll
                for (int u = 0; u < ROWS; ++u) a[u] = __ldg(reinterpret_cast<const float4*>(rows + static_cast<int64_t>(u) * nb + l));
#pragma unroll
                for (int h = 0; h < NRHS; ++h) {
                    const float4 z = *reinterpret_cast<const float4*>(zs + h * nb + l);
#pragma unroll
                    for (int u = 0; u < ROWS; ++u)
                        acc[u * NRHS + h] = fmaf(a[u].x, z.x, fmaf(a[u].y, z.y, fmaf(a[u].z, z.z, fmaf(a[u].w, z.w, acc[u * NRHS + h]))));
                }
            }
        }
        warp_reduce64(acc, lane);
        if (KS > 1) {
            if (ks > 0) {
                red[((ks - 1) * GQ + gl) * 64 + lane * 2 + 0] = acc[0];
                red[((ks - 1) * GQ + gl) * 64 + lane * 2 + 1] = acc[1];
            }
            __syncthreads();
        }
        if (ks == 0) {
#pragma unroll
            for (int s2 = 1; s2 < KS; ++s2) {
                acc[0] += red[((s2 - 1) * GQ + gl) * 64 + lane * 2 + 0];
                acc[1] += red[((s2 - 1) * GQ + gl) * 64 + lane * 2 + 1];
            }
            const int v0 = warp_reduce64_index(lane);
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                const int u = (v0 + t) / NRHS, h = (v0 + t) % NRHS;
                const int r = grow + u;
                const float y = (h < nrhs) ? Bk[static_cast<int64_t>(R0 + r) * ldb + h] : 0.0f;
                const float tv = y - acc[t];
#pragma unroll
                for (int d = 0; d < kDiagCluster; ++d) cluster.map_shared_rank(ts, d)[h * kBlk + r] = tv;
            }
        }
        cluster.sync();
        // ---- phase 2: solved_c = inv(L_cc) t   (forward)   or   inv(L_cc)^T t   (backward)
        if (ks == 0) {
            const float* D = (backward ? dinvT : dinv) + static_cast<int64_t>(c) * kBlk * kBlk;
            float acc[64];
#pragma unroll
            for (int v = 0; v < 64; ++v) acc[v] = 0.0f;
            rows_dot_f32<NRHS>(D + static_cast<int64_t>(grow) * kBlk, kBlk, kBlk, ts, kBlk, lane, acc);
            warp_reduce64(acc, lane);
            const int v0 = warp_reduce64_index(lane);
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                const int u = (v0 + t) / NRHS, h = (v0 + t) % NRHS;
                const int r = R0 + grow + u;
#pragma unroll
                for (int d = 0; d < kDiagCluster; ++d) {
                    cluster.map_shared_rank(zs, d)[h * nb + r] = acc[t];
                }
                if (h < nrhs) Bk[static_cast<int64_t>(r) * ldb + h] = acc[t];
            }
        }
        cluster.sync();
    }
}

}  // namespace krr

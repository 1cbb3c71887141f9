// krr_potrs kernels: forward and backward substitution in FP32 with the tile mosaic
// ("W <- Solve(K~, P_h)", "forward and backward substitution operations
// in the full FP32 precision").  nrhs is small (4..32), so each sweep is bound by reading L once
// from HBM.  Right-hand sides are row-major n x nrhs.
#pragma once
#include "common.cuh"

namespace krr {

constexpr int kMaxRhs = 32;

// Dequantising 4-element load of a mosaic tile row segment (columns c..c+3, c % 4 == 0).
__device__ __forceinline__ float4 load4(const uint8_t* tile, int p, float s, int64_t e) {
    if (p == KRR_FP32) return *reinterpret_cast<const float4*>(tile + e * 4);
    if (p == KRR_FP16) {
        const uint2 raw = *reinterpret_cast<const uint2*>(tile + e * 2);
        const __half2 a = *reinterpret_cast<const __half2*>(&raw.x);
        const __half2 b = *reinterpret_cast<const __half2*>(&raw.y);
        return make_float4(__low2float(a), __high2float(a), __low2float(b), __high2float(b));
    }
    const uint32_t raw = *reinterpret_cast<const uint32_t*>(tile + e);
    return make_float4(e4m3_to_f32(raw & 0xff) * s, e4m3_to_f32((raw >> 8) & 0xff) * s,
                       e4m3_to_f32((raw >> 16) & 0xff) * s, e4m3_to_f32(raw >> 24) * s);
}
__device__ __forceinline__ float load1(const uint8_t* tile, int p, float s, int64_t e) {
    if (p == KRR_FP32) return *reinterpret_cast<const float*>(tile + e * 4);
    if (p == KRR_FP16) return __half2float(*reinterpret_cast<const __half*>(tile + e * 2));
    return e4m3_to_f32(tile[e]) * s;
}

// ---------------------------------------------------------------------------------------------
// Forward update after Z_k is known:  Y_i -= L_ik Z_k  for all i > k.
// grid.x = (NT-k-1)*nb / 32 (32 rows per CTA, 4 per warp), 256 threads, smem = nrhs*nb floats.
template <int NRHS>
__global__ void __launch_bounds__(256)
potrs_fwd_update_kernel(int NT, int nb, int k, const uint8_t* __restrict__ factor,
                        const int64_t* __restrict__ off, const uint8_t* __restrict__ map,
                        const float* __restrict__ scales, float* __restrict__ B, int64_t ldb, int nrhs) {
    extern __shared__ float zs[];                      // [NRHS][nb]
    const float* Zk = B + static_cast<int64_t>(k) * nb * ldb;
    for (int idx = threadIdx.x; idx < nb * nrhs; idx += 256) {
        const int c = idx / nrhs, rh = idx % nrhs;
        zs[rh * nb + c] = Zk[static_cast<int64_t>(c) * ldb + rh];
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t prow0 = static_cast<int64_t>(blockIdx.x) * 32;       // rows below tile k
    const int i = k + 1 + static_cast<int>(prow0 / nb);
    const int p = map[i * NT + k];
    const float s = scales[i * NT + k];
    const uint8_t* tile = factor + off[i * NT + k];
    for (int rr = 0; rr < 4; ++rr) {
        const int r = static_cast<int>(prow0 % nb) + warp * 4 + rr;
        float acc[NRHS];
#pragma unroll
        for (int h = 0; h < NRHS; ++h) acc[h] = 0.0f;
        for (int c = lane * 4; c < nb; c += 128) {
            const float4 l = load4(tile, p, s, static_cast<int64_t>(r) * nb + c);
#pragma unroll
            for (int h = 0; h < NRHS; ++h) {
                if (h < nrhs) {
                    const float4 z = *reinterpret_cast<const float4*>(zs + h * nb + c);
                    acc[h] = fmaf(l.x, z.x, fmaf(l.y, z.y, fmaf(l.z, z.z, fmaf(l.w, z.w, acc[h]))));
                }
            }
        }
#pragma unroll
        for (int h = 0; h < NRHS; ++h) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) acc[h] += __shfl_xor_sync(0xffffffffu, acc[h], o);
        }
        float* y = B + (static_cast<int64_t>(i) * nb + r) * ldb;
#pragma unroll
        for (int h = 0; h < NRHS; ++h)
            if (lane == h && h < nrhs) y[h] -= acc[h];
    }
}

// Backward update after alpha_k is known:  Z_j -= L_kj^T alpha_k  for all j < k.
// grid.x = k*nb / 128 (128 columns per CTA, one per thread), smem = nrhs*nb floats.
template <int NRHS>
__global__ void __launch_bounds__(128)
potrs_bwd_update_kernel(int NT, int nb, int k, const uint8_t* __restrict__ factor,
                        const int64_t* __restrict__ off, const uint8_t* __restrict__ map,
                        const float* __restrict__ scales, float* __restrict__ B, int64_t ldb, int nrhs) {
    extern __shared__ float as[];                      // [nb][NRHS] alpha_k
    const float* Ak = B + static_cast<int64_t>(k) * nb * ldb;
    for (int idx = threadIdx.x; idx < nb * NRHS; idx += 128) {
        const int r = idx / NRHS, rh = idx % NRHS;
        as[idx] = (rh < nrhs) ? Ak[static_cast<int64_t>(r) * ldb + rh] : 0.0f;
    }
    __syncthreads();
    const int64_t gcol = static_cast<int64_t>(blockIdx.x) * 128 + threadIdx.x;
    const int j = static_cast<int>(gcol / nb), c = static_cast<int>(gcol % nb);
    const int p = map[k * NT + j];
    const float s = scales[k * NT + j];
    const uint8_t* tile = factor + off[k * NT + j];
    float acc[NRHS];
#pragma unroll
    for (int h = 0; h < NRHS; ++h) acc[h] = 0.0f;
    for (int r = 0; r < nb; ++r) {
        const float l = load1(tile, p, s, static_cast<int64_t>(r) * nb + c);
#pragma unroll
        for (int h = 0; h < NRHS; ++h) acc[h] = fmaf(l, as[r * NRHS + h], acc[h]);
    }
    float* z = B + gcol * ldb;
#pragma unroll
    for (int h = 0; h < NRHS; ++h)
        if (h < nrhs) z[h] -= acc[h];
}

// Diagonal tile solve, one CTA of 256 threads: forward (L z = y) or backward (L^T a = z), in place
// on rows k*nb .. (k+1)*nb of B.  Blocks of 32 rows: a GEMV with the already-solved part, then a
// 32x32 triangular solve by one warp (lane = right-hand side).
template <int NRHS>
__global__ void __launch_bounds__(256)
potrs_diag_kernel(int nb, const float* __restrict__ Lkk, float* __restrict__ Bk, int64_t ldb, int nrhs,
                  int backward) {
    extern __shared__ float sm[];
    float* zs = sm;                         // [NRHS][nb] solved values
    float* blk = sm + NRHS * nb;            // [32][33] diagonal block
    float* part = blk + 32 * 33;            // [8][32][NRHS] partial sums (backward) / [32][NRHS] (forward)
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nblk = nb / 32;
    for (int bi = 0; bi < nblk; ++bi) {
        const int b = backward ? (nblk - 1 - bi) : bi;
        const int r0 = b * 32;
        // diagonal 32x32 block into smem
        for (int idx = threadIdx.x; idx < 32 * 32; idx += 256) {
            const int r = idx >> 5, c = idx & 31;
            blk[r * 33 + c] = Lkk[static_cast<int64_t>(r0 + r) * nb + r0 + c];
        }
        if (!backward) {
            // part[r][h] = sum_{l < r0} L[r0+r][l] z[l][h] ; warp w handles rows 4w..4w+3
            for (int rr = 0; rr < 4; ++rr) {
                const int r = warp * 4 + rr;
                float acc[NRHS];
#pragma unroll
                for (int h = 0; h < NRHS; ++h) acc[h] = 0.0f;
                const float* lrow = Lkk + static_cast<int64_t>(r0 + r) * nb;
                for (int l = lane; l < r0; l += 32) {
                    const float lv = lrow[l];
#pragma unroll
                    for (int h = 0; h < NRHS; ++h) acc[h] = fmaf(lv, zs[h * nb + l], acc[h]);
                }
#pragma unroll
                for (int h = 0; h < NRHS; ++h) {
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) acc[h] += __shfl_xor_sync(0xffffffffu, acc[h], o);
                }
#pragma unroll
                for (int h = 0; h < NRHS; ++h)
                    if (lane == h) part[r * NRHS + h] = acc[h];
            }
        } else {
            // part[w][c][h] = sum over rows r > block, r = r1 + w, r1 + w + 8, ... of L[r][r0+c] a[r][h]
            float acc[NRHS];
#pragma unroll
            for (int h = 0; h < NRHS; ++h) acc[h] = 0.0f;
            for (int r = r0 + 32 + warp; r < nb; r += 8) {
                const float lv = Lkk[static_cast<int64_t>(r) * nb + r0 + lane];
#pragma unroll
                for (int h = 0; h < NRHS; ++h) acc[h] = fmaf(lv, zs[h * nb + r], acc[h]);
            }
#pragma unroll
            for (int h = 0; h < NRHS; ++h) part[(warp * 32 + lane) * NRHS + h] = acc[h];
        }
        __syncthreads();
        if (warp == 0) {
            const int h = lane;                   // this lane's right-hand side
            if (h < nrhs) {
                float v[32];
                if (!backward) {
#pragma unroll
                    for (int r = 0; r < 32; ++r) v[r] = Bk[static_cast<int64_t>(r0 + r) * ldb + h] - part[r * NRHS + h];
#pragma unroll
                    for (int r = 0; r < 32; ++r) {
                        float sacc = v[r];
#pragma unroll
                        for (int l = 0; l < r; ++l) sacc = fmaf(-blk[r * 33 + l], v[l], sacc);
                        v[r] = sacc / blk[r * 33 + r];
                    }
                } else {
#pragma unroll
                    for (int r = 0; r < 32; ++r) {
                        float sacc = 0.0f;
                        for (int w = 0; w < 8; ++w) sacc += part[(w * 32 + r) * NRHS + h];
                        v[r] = Bk[static_cast<int64_t>(r0 + r) * ldb + h] - sacc;
                    }
#pragma unroll
                    for (int r = 31; r >= 0; --r) {
                        float sacc = v[r];
#pragma unroll
                        for (int l = r + 1; l < 32; ++l) sacc = fmaf(-blk[l * 33 + r], v[l], sacc);
                        v[r] = sacc / blk[r * 33 + r];
                    }
                }
#pragma unroll
                for (int r = 0; r < 32; ++r) {
                    zs[h * nb + r0 + r] = v[r];
                    Bk[static_cast<int64_t>(r0 + r) * ldb + h] = v[r];
                }
            }
        }
        __syncthreads();
    }
}

}  // namespace krr

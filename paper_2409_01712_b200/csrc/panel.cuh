// Panel-side helper kernels of the tile Cholesky (the FP32 POTRF of a
// 128x128 block is in tri128.cuh):
//   finalize_kernel   rounds the finished tile column into the storage precisions of the mosaic
//                     (per-tile power-of-two FP8 scale from the tile amax) -- "round once"
//   offsets_kernel    byte offsets of the mosaic tiles from the device map
//   tile_amax_kernel  max|A_ij| of the FP8 tiles of A (scale of the pre-rounding of A)
#pragma once
#include "common.cuh"

namespace krr {

// Symmetric power-of-two equilibration by tile rows and the (then constant) scales of the FP16 operand images.
//   d_I = 2^-e_I  with  2^(e_I - 1) <= sqrt(max_{r in tile row I} A_rr) < 2^(e_I)
// The factorisation runs on  A~ = D A D  (D = diag(d_I) over the tile rows; the scaling is applied when a tile of A is
// first read and undone when a tile of L is stored, L = D^-1 L~: exact, powers of two), so that every tile row has
// max A~_rr in [1/4, 1): |L~_ij| < 1 and |S~_ij| < 1 whatever the scaling of the input, and the 22 significant bits of
// the hi / lo images are spent on the tile row's own magnitude instead of the largest diagonal entry of the whole
// matrix.  (Uniform diagonals -- every kernel matrix -- give one d: the same bits as a global scale.)  Image scales:
// sx = 2^14 for L~ and X~, ss = 2^15 for S~; M~ = inv(L~_kk) has entries of order one and no a-priori bound, so
// sm = 2^4: room for entries up to 2^12 (beyond that krr_potrf_mp reports info = -2), 22 significant bits down to
// 2^-7 and an absolute resolution of 2^-29 below; su likewise for U = L~21 M~11.  One CTA.
__global__ void __launch_bounds__(1024)
equilibrate_kernel(AView A, int64_t n, float* __restrict__ scl, float* __restrict__ dscale) {
    const int NT = A.NT, nb = A.nb;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int t = warp; t < NT; t += 32) {                      // one warp per tile row
        float m = 0.0f;
        for (int r = lane; r < nb; r += 32) m = fmaxf(m, fabsf(*A.tile_ptr(t, t, r, r)));
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
        if (lane == 0) {
            float d = 1.0f;
            if (m > 0.0f && m < 3.0e38f) {
                int e;
                frexpf(sqrtf(m), &e);                          // sqrt(m) in [2^(e-1), 2^e)
                d = ldexpf(1.0f, -e);
            }
            dscale[t] = d;
        }
    }
    if (threadIdx.x == 0) {
        const float sx = 16384.0f, ss = 32768.0f, sm = 16.0f, su = 16.0f;
        scl[SCL_SX] = sx;
        scl[SCL_SS] = ss;
        scl[SCL_INV_SX2] = (1.0f / sx) * (1.0f / sx);
        scl[SCL_INV_SS] = 1.0f / ss;
        scl[SCL_SM] = sm;
        scl[SCL_SU] = su;
        scl[SCL_INV_SM_SX] = (1.0f / sm) * (1.0f / sx);
        scl[SCL_INV_SM_SU] = (1.0f / sm) * (1.0f / su);
        scl[SCL_INV_SS_SM] = (1.0f / ss) * (1.0f / sm);
    }
    (void)n;
}

// d_scales of the mosaic: 1 for the lower tiles (finalize_kernel overwrites the FP8 tiles'), 0 above the diagonal.
__global__ void scales_init_kernel(int NT, float* __restrict__ scales) {
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx < NT * NT) scales[idx] = (idx % NT <= idx / NT) ? 1.0f : 0.0f;
}

// FNV-1a over the lower entries of a map in column-major tile order: the host (h_map) and the device (d_map) side of
// the same call must agree (sizes come from h_map, offsets and MMA classes from d_map).
__host__ __device__ __forceinline__ uint64_t map_hash_step(uint64_t h, uint8_t v) { return (h ^ v) * 1099511628211ull; }
constexpr uint64_t kMapHashSeed = 1469598103934665603ull;

// Byte offsets of the mosaic tiles (column-major lower order prefix sum).  One thread.  If the device map does not
// hash to `host_hash` (the caller's h_map and d_map differ) every offset is set to 0 -- all tiles alias the first
// (FP32, diagonal) tile, so that nothing is read or written outside buffers sized from h_map -- and *info = -1.
// lrow / qrow (may be null): first row of tile (i,j) in the compact lo plane (FP32 tiles) and E4M3 plane (FP8 tiles), in the
// same column-major tile order, -1 for tiles without that image (all 0 on a hash mismatch).
__global__ void offsets_kernel(int NT, int nb, const uint8_t* __restrict__ map, int64_t* __restrict__ off, uint64_t host_hash,
                               int* __restrict__ info, int* __restrict__ lrow, int* __restrict__ qrow) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    int64_t acc = 0;
    const int64_t elems = static_cast<int64_t>(nb) * nb;
    uint64_t h = kMapHashSeed;
    int nl = 0, nq = 0;
    for (int j = 0; j < NT; ++j)
        for (int i = j; i < NT; ++i) {
            off[i * NT + j] = acc;
            const uint8_t p = map[i * NT + j];
            h = map_hash_step(h, p);
            acc += elems * prec_bytes(p);
            if (lrow) lrow[i * NT + j] = (p == KRR_FP32) ? (nl++) * nb : -1;
            if (qrow) qrow[i * NT + j] = (p == KRR_FP8_E4M3) ? (nq++) * nb : -1;
        }
    if (h != host_hash) {
        for (int j = 0; j < NT; ++j)
            for (int i = j; i < NT; ++i) {
                off[i * NT + j] = 0;
                if (lrow) lrow[i * NT + j] = 0;
                if (qrow) qrow[i * NT + j] = 0;
            }
        if (info) *info = -1;
    }
}

// max|A_ij| for the FP8 tiles of A.  grid = (nslots, nb / 32); a_amax zeroed beforehand.
__global__ void __launch_bounds__(256)
tile_amax_kernel(AView A, const uint8_t* __restrict__ map, float* __restrict__ a_amax) {
    const int NT = A.NT, nb = A.nb;
    int j = 0;
    int64_t rem = blockIdx.x;
    while (rem >= NT - j) { rem -= NT - j; ++j; }
    const int i = j + static_cast<int>(rem);
    if (map[i * NT + j] != KRR_FP8_E4M3) return;
    const int r0 = blockIdx.y * 32;
    const int vec_per_row = nb / 4;
    float amax = 0.0f;
    for (int idx = threadIdx.x; idx < 32 * vec_per_row; idx += 256) {
        const float4 v = __ldg(reinterpret_cast<const float4*>(A.tile_ptr(i, j, r0 + idx / vec_per_row, (idx % vec_per_row) * 4)));
        amax = fmaxf(amax, fmaxf(fmaxf(fabsf(v.x), fabsf(v.y)), fmaxf(fabsf(v.z), fabsf(v.w))));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
    if ((threadIdx.x & 31) == 0) atomicMax(reinterpret_cast<int*>(a_amax + i * NT + j), __float_as_int(amax));
}

// Round tiles (k + i0 + blockIdx.y, k) of tile column k (FP32 in W, block-column-major 128x128 blocks)
// into the mosaic.  With only_fp8 the tiles of the other precisions are left alone: the TRSM product has stored
// them already (gemm_tc.cuh MODE_TRSM); FP8 tiles wait for their amax and are rounded here.  grid = (nsub*nsub*4, number of tiles), 256 threads: one CTA transposes 32 rows of one 128x128 block through
// shared memory (coalesced reads of W columns, coalesced row-major writes of the factor / images).
__global__ void __launch_bounds__(256)
finalize_kernel(int NT, int nb, int k, int i0, const float* __restrict__ W, const uint8_t* __restrict__ map,
                const int64_t* __restrict__ off, const float* __restrict__ tile_amax /* per slot */,
                uint8_t* __restrict__ factor, float* __restrict__ scales, __half* __restrict__ Hp,
                uint8_t* __restrict__ Qp, const int* __restrict__ qrow, const float* __restrict__ scl,
                const float* __restrict__ dscale, int only_fp8) {
    __shared__ float tile[32][kBlk + 1];
    const float sx = scl[SCL_SX];
    const int nsub = nb / kBlk;
    const int i = k + i0 + blockIdx.y;
    const int p = map[i * NT + k];
    if (only_fp8 && p != KRR_FP8_E4M3) return;
    const int64_t slot = tile_slot(NT, i, k);
    // W and tile_amax hold the equilibrated L~ = d_i L: the stored tile is L (exact power-of-two unscaling)
    const float di = dscale[i], inv_di = 1.0f / di;
    const float s = (p == KRR_FP8_E4M3) ? fp8_scale_from_amax(tile_amax[slot] * inv_di) : 1.0f;
    if (blockIdx.x == 0 && threadIdx.x == 0) scales[i * NT + k] = s;
    uint8_t* dst = factor + off[i * NT + k];
    const int blk = blockIdx.x >> 2, qr = blockIdx.x & 3;
    const int rbl = blk / nsub, cb = blk % nsub;                         // block inside the tile
    const int64_t rb = static_cast<int64_t>(i0 + blockIdx.y) * nsub + rbl;    // panel-local row block
    const float* wblk = W + (rb * nsub + cb) * (kBlk * kBlk) + 32 * qr;
    {   // all 16 loads of a thread in flight at once (one DRAM round trip per CTA instead of four)
        float v[16];
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            const int idx = threadIdx.x + 256 * u;
            v[u] = __ldg(wblk + (idx >> 5) * kBlk + (idx & 31));
        }
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            const int idx = threadIdx.x + 256 * u;
            tile[idx & 31][idx >> 5] = v[u];
        }
    }
    __syncthreads();
    for (int idx = threadIdx.x; idx < 32 * (kBlk / 4); idx += 256) {
        const int rr = idx / (kBlk / 4), c4 = (idx % (kBlk / 4)) * 4;
        const int r = rbl * kBlk + 32 * qr + rr, c = cb * kBlk + c4;     // element of the tile
        float4 v = make_float4(tile[rr][c4] * inv_di, tile[rr][c4 + 1] * inv_di, tile[rr][c4 + 2] * inv_di, tile[rr][c4 + 3] * inv_di);
        const int64_t e = static_cast<int64_t>(r) * nb + c;
        if (p == KRR_FP32) {
            if (i == k) {      // diagonal tile: zeros above the diagonal
                if (c + 0 > r) v.x = 0.f;
                if (c + 1 > r) v.y = 0.f;
                if (c + 2 > r) v.z = 0.f;
                if (c + 3 > r) v.w = 0.f;
            }
            *reinterpret_cast<float4*>(dst + e * 4) = v;
        } else if (p == KRR_FP16) {
            __align__(8) __half h[4] = {__float2half_rn(v.x), __float2half_rn(v.y), __float2half_rn(v.z), __float2half_rn(v.w)};
            *reinterpret_cast<uint2*>(dst + e * 2) = *reinterpret_cast<const uint2*>(h);
            // operand image of the STORED value (exact: a power-of-two multiple of an FP16 number)
            __align__(8) __half hs[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) hs[u] = __float2half_rn(__half2float(h[u]) * di * sx);
            *reinterpret_cast<uint2*>(Hp + (slot * nb + r) * nb + c) = *reinterpret_cast<const uint2*>(hs);
        } else {
            const float inv = 1.0f / s;          // power of two: exact
            __align__(4) uint8_t q[4] = {f32_to_e4m3(v.x * inv), f32_to_e4m3(v.y * inv), f32_to_e4m3(v.z * inv), f32_to_e4m3(v.w * inv)};
            *reinterpret_cast<uint32_t*>(dst + e) = *reinterpret_cast<const uint32_t*>(q);
            if (Qp) *reinterpret_cast<uint32_t*>(Qp + (static_cast<int64_t>(qrow[i * NT + k]) + r) * nb + c) = *reinterpret_cast<const uint32_t*>(q);
            __align__(8) __half h[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) h[u] = __float2half_rn(e4m3_to_f32(q[u]) * s * di * sx);
            *reinterpret_cast<uint2*>(Hp + (slot * nb + r) * nb + c) = *reinterpret_cast<const uint2*>(h);
        }
    }
}

}  // namespace krr

// FP32 kernels on one 128x128 diagonal block ("POTRF"):
//   potrf128_kernel   Cholesky of the block on plain FP32 ALUs plus the inverse of its factor
//                     (the panel TRSM multiplies by it on the tensor cores, gemm_tc.cuh MODE_P3)
//   trtri128_kernel   inverse of a stored 128x128 lower-triangular diagonal block (krr_potrs)
//
// Both are recursive over 32x32 sub-blocks held in shared memory:
//   chol32   one warp, lane = row, the row in registers, right-looking with shuffles
//   inv32    one warp, lane = column of the inverse, forward substitution in registers
//   the off-diagonal work (panel = product with inv32, trailing update, off-diagonal blocks of the
//   inverse) is small FP32 matrix products done by all warps out of shared memory.
// The arithmetic is IEEE FP32 with true sqrt and division, so exactly representable inputs give the
// exact factor (tests: "exactly representable constructions").
#pragma once
#include "common.cuh"

namespace krr {

constexpr int kTriThreads = 256;
constexpr int kTriLd = 132;                       // 16-byte aligned rows; LDS.128 by row is conflict free
constexpr int kTriSmem = 2 * kBlk * kTriLd * 4;   // L and inv(L)

// Cholesky of the 32x32 block at (j0, j0) of a (smem, ld kTriLd), in place; zeros above the diagonal.
// One warp.  Returns through *bad the 1-based local column of the first non-positive pivot (0 = none).
__device__ __forceinline__ int chol32_warp(float* a, int j0, int lane) {
    float r[32];
    float* row = a + (j0 + lane) * kTriLd + j0;
#pragma unroll
    for (int c = 0; c < 32; c += 4) {
        const float4 v = *reinterpret_cast<const float4*>(row + c);
        r[c] = v.x; r[c + 1] = v.y; r[c + 2] = v.z; r[c + 3] = v.w;
    }
    int bad = 0;
#pragma unroll
    for (int j = 0; j < 32; ++j) {
        const float d = __shfl_sync(0xffffffffu, r[j], j);
        if (!(d > 0.0f) && bad == 0) bad = j + 1;
        const float dj = sqrtf(d);
        const float l = (lane > j) ? r[j] / dj : (lane == j ? dj : 0.0f);
        r[j] = l;
#pragma unroll
        for (int c = j + 1; c < 32; ++c) {
            const float lc = __shfl_sync(0xffffffffu, l, c);
            r[c] = fmaf(-l, lc, r[c]);             // rows above c hold garbage there; never used
        }
    }
#pragma unroll
    for (int c = 0; c < 32; c += 4) {
        float4 v;
        v.x = (c + 0 <= lane) ? r[c + 0] : 0.0f;
        v.y = (c + 1 <= lane) ? r[c + 1] : 0.0f;
        v.z = (c + 2 <= lane) ? r[c + 2] : 0.0f;
        v.w = (c + 3 <= lane) ? r[c + 3] : 0.0f;
        *reinterpret_cast<float4*>(row + c) = v;
    }
    return bad;
}

// x = inverse of the lower-triangular 32x32 block of l at (j0, j0), written to the same block of x.
// One warp, lane = column j of the inverse: x_rj = (delta_rj - sum_{m<r} l_rm x_mj) / l_rr.
__device__ __forceinline__ void inv32_warp(const float* l, float* x, int j0, int lane) {
    float v[32];
#pragma unroll
    for (int r = 0; r < 32; ++r) {
        const float* lr = l + (j0 + r) * kTriLd + j0;       // broadcast reads
        float s = (r == lane) ? 1.0f : 0.0f;
#pragma unroll
        for (int m = 0; m < r; ++m) s = fmaf(-lr[m], v[m], s);
        v[r] = (r >= lane) ? s / lr[r] : 0.0f;
    }
#pragma unroll
    for (int r = 0; r < 32; ++r) x[(j0 + r) * kTriLd + j0 + lane] = v[r];
}

// C[r][c] (op)= sum_m P[r][m] Q[c][m]   for r in [0,R), c in [0,32), m in [0,M): "P Q^T" with both
// operands row-major in smem (ld kTriLd).  Warp per 4 rows, lane = column c; P rows are broadcast
// LDS.128, Q rows conflict-free LDS.128.  mode 0: C = acc, 1: C -= acc, 2: C = -acc.
// C may alias P's rows only through `out` pointing elsewhere (callers take care).
template <int MODE>
__device__ __forceinline__ void small_abt(const float* P, const float* Q, float* out, int R, int M,
                                          int warp, int nwarps, int lane) {
    for (int r0 = warp * 4; r0 < R; r0 += nwarps * 4) {
        float acc[4] = {0.f, 0.f, 0.f, 0.f};
        const float* q = Q + lane * kTriLd;
        for (int m = 0; m < M; m += 4) {
            const float4 qv = *reinterpret_cast<const float4*>(q + m);
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const float4 pv = *reinterpret_cast<const float4*>(P + (r0 + u) * kTriLd + m);
                acc[u] = fmaf(pv.x, qv.x, fmaf(pv.y, qv.y, fmaf(pv.z, qv.z, fmaf(pv.w, qv.w, acc[u]))));
            }
        }
        __syncwarp();                                   // all lanes read row r0+u before it is overwritten
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            float* o = out + (r0 + u) * kTriLd + lane;
            if (MODE == 0) *o = acc[u];
            else if (MODE == 1) *o -= acc[u];
            else *o = -acc[u];
        }
    }
}

// C[r][c] = - sum_m P[r][m] Q[m][c]  ("P Q", Q row-major): r in [0,R), c in [0,32), m in [0,M).
// lane = column c: Q[m][c] is a conflict-free LDS.32, P[r][m] a broadcast.
__device__ __forceinline__ void small_ab_neg(const float* P, const float* Q, float* out, int R, int M,
                                             int warp, int nwarps, int lane) {
    for (int r0 = warp * 4; r0 < R; r0 += nwarps * 4) {
        float acc[4] = {0.f, 0.f, 0.f, 0.f};
        for (int m = 0; m < M; m += 4) {
            const float q0 = Q[(m + 0) * kTriLd + lane], q1 = Q[(m + 1) * kTriLd + lane];
            const float q2 = Q[(m + 2) * kTriLd + lane], q3 = Q[(m + 3) * kTriLd + lane];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const float4 pv = *reinterpret_cast<const float4*>(P + (r0 + u) * kTriLd + m);
                acc[u] = fmaf(pv.x, q0, fmaf(pv.y, q1, fmaf(pv.z, q2, fmaf(pv.w, q3, acc[u]))));
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) out[(r0 + u) * kTriLd + lane] = -acc[u];
    }
}

// Off-diagonal 32x32 blocks of x = inv(l) once the four diagonal blocks x_ii are known:
//   x_ij = - x_ii * (sum_{j<=m<i} l_im x_mj),  block row i = 1..3 in order.  `t` is a 32-row scratch
// strip (32 x 96 used) inside the caller's shared memory (callers pass the still-zero upper-right
// corner of x, rows 0..31 x columns 32..127, and mask c > r when they write x out).  All kTriThreads threads.
__device__ __forceinline__ void inv128_offdiag(const float* l, float* x, float* t, int warp, int lane) {
    constexpr int NW = kTriThreads / 32;
    for (int i = 1; i < 4; ++i) {
        // t[:, 32j..32j+31] = sum_{m=j}^{i-1} l_im x_mj   (columns 0 .. 32i-1; x_mj = 0 for m < j)
        for (int j = 0; j < i; ++j)
            small_ab_neg(l + (32 * i) * kTriLd + 32 * j, x + (32 * j) * kTriLd + 32 * j, t + 32 * j, 32,
                         32 * (i - j), warp, NW, lane);          // t = -(l_i,[j..i) x_[j..i),j)
        __syncthreads();
        // x_ij = x_ii * t_j  (t already carries the minus sign)
        for (int j = 0; j < i; ++j) {
            // out[r][c] = sum_m x_ii[r][m] t[m][32j + c]; reuse small_ab_neg on (-x_ii)?  do it inline
            for (int r0 = warp * 4; r0 < 32; r0 += NW * 4) {
                float acc[4] = {0.f, 0.f, 0.f, 0.f};
                for (int m = 0; m < 32; ++m) {
                    const float q = t[m * kTriLd + 32 * j + lane];
#pragma unroll
                    for (int u = 0; u < 4; ++u) acc[u] = fmaf(x[(32 * i + r0 + u) * kTriLd + 32 * i + m], q, acc[u]);
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) x[(32 * i + r0 + u) * kTriLd + 32 * j + lane] = acc[u];
            }
        }
        __syncthreads();
    }
}

// W: panel workspace [m][nb] FP32; the block is rows r0..r0+127 (panel-local), columns c0..c0+127.
// Writes L (lower, zeros above) back into W and inv(L) as scaled FP16 hi/lo planes into
// linv_hi/lo ([nb][128] row-major, rows c0..c0+127) with their power-of-two scale in linv_scale.
// col_base = 1-based global index of the block's first column, for info (LAPACK convention).
__global__ void __launch_bounds__(kTriThreads, 1)
potrf128_kernel(float* __restrict__ W, int nb, int r0, int c0, __half* __restrict__ linv_hi,
                __half* __restrict__ linv_lo, float* __restrict__ linv_scale, int* __restrict__ info,
                int64_t col_base) {
    extern __shared__ __align__(16) float tri_sm[];
    float* a = tri_sm;                       // [128][132] : S, then L
    float* x = tri_sm + kBlk * kTriLd;       // [128][132] : inv(L); rows 96..127 double as scratch early on
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    constexpr int NW = kTriThreads / 32;
    // W is block-column-major: element (r, c) of 128x128 block (rb, cb) at ((rb*nsub + cb)*128 + c)*128 + r
    float* wblk = W + (static_cast<int64_t>(r0 / kBlk) * (nb / kBlk) + c0 / kBlk) * (kBlk * kBlk);
    for (int idx = tid; idx < kBlk * (kBlk / 4); idx += kTriThreads) {
        const int c = idx / (kBlk / 4), r4 = (idx % (kBlk / 4)) * 4;
        const float4 v = *reinterpret_cast<const float4*>(wblk + c * kBlk + r4);
        a[(r4 + 0) * kTriLd + c] = v.x;
        a[(r4 + 1) * kTriLd + c] = v.y;
        a[(r4 + 2) * kTriLd + c] = v.z;
        a[(r4 + 3) * kTriLd + c] = v.w;
        *reinterpret_cast<float4*>(x + c * kTriLd + r4) = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    __syncthreads();
    for (int jb = 0; jb < 4; ++jb) {
        const int j0 = 32 * jb;
        if (warp == 0) {
            const int bad = chol32_warp(a, j0, lane);
            // the lowest bad column of the warp (every lane sees the same pivots)
            if (bad && lane == 0) atomicCAS(info, 0, static_cast<int>(col_base + j0 + bad - 1));
            __syncwarp();
            inv32_warp(a, x, j0, lane);
        }
        __syncthreads();
        const int R = kBlk - (j0 + 32);                 // rows below the diagonal block
        if (R > 0) {
            // panel: L_i,jb = S_i,jb * x_jb,jb^T   (in place: a warp owns whole rows)
            small_abt<0>(a + (j0 + 32) * kTriLd + j0, x + j0 * kTriLd + j0, a + (j0 + 32) * kTriLd + j0, R, 32,
                         warp, NW, lane);
            __syncthreads();
            // trailing update: S_ic -= L_i,jb L_c,jb^T for the 32-column blocks right of jb (lower part)
            for (int cb = jb + 1; cb < 4; ++cb) {
                const int rr = 32 * cb;                 // rows from the diagonal block of cb downwards
                small_abt<1>(a + rr * kTriLd + j0, a + rr * kTriLd + j0, a + rr * kTriLd + rr, kBlk - rr, 32,
                             warp, NW, lane);
            }
            __syncthreads();
        }
    }
    // off-diagonal blocks of the inverse; scratch strip = the (still zero) upper-right corner of x
    inv128_offdiag(a, x, x + 32, warp, lane);
    // power-of-two scale of the inverse's planes: max|x| * si <= 2^14
    __shared__ float s_red[kTriThreads / 32];
    {
        float m = 0.0f;
        for (int idx = tid; idx < kBlk * kBlk; idx += kTriThreads) {
            const int r = idx >> 7, c = idx & 127;
            if (c <= r) m = fmaxf(m, fabsf(x[r * kTriLd + c]));
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
        if (lane == 0) s_red[warp] = m;
    }
    __syncthreads();
    float si = 1.0f;
    {
        float m = 0.0f;
#pragma unroll
        for (int w = 0; w < kTriThreads / 32; ++w) m = fmaxf(m, s_red[w]);
        if (m > 0.0f && m < 3.0e38f) {
            int e;
            frexpf(m, &e);                 // m <= 2^e
            si = ldexpf(1.0f, 14 - e);
        }
    }
    if (tid == 0) linv_scale[c0 / kBlk] = si;
    for (int idx = tid; idx < kBlk * (kBlk / 4); idx += kTriThreads) {
        const int r = idx / (kBlk / 4), c4 = (idx % (kBlk / 4)) * 4;
        const float4 lv = *reinterpret_cast<const float4*>(a + r * kTriLd + c4);
        float4 v;
        v.x = (c4 + 0 <= r) ? lv.x : 0.0f;
        v.y = (c4 + 1 <= r) ? lv.y : 0.0f;
        v.z = (c4 + 2 <= r) ? lv.z : 0.0f;
        v.w = (c4 + 3 <= r) ? lv.w : 0.0f;
        wblk[(c4 + 0) * kBlk + r] = v.x;
        wblk[(c4 + 1) * kBlk + r] = v.y;
        wblk[(c4 + 2) * kBlk + r] = v.z;
        wblk[(c4 + 3) * kBlk + r] = v.w;
        __align__(8) __half hi[4];
        __align__(8) __half lo[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const float xv = (c4 + u <= r) ? x[r * kTriLd + c4 + u] * si : 0.0f;
            hi[u] = __float2half_rn(xv);
            lo[u] = __float2half_rn(xv - __half2float(hi[u]));
        }
        *reinterpret_cast<uint2*>(linv_hi + static_cast<int64_t>(c0 + r) * kBlk + c4) = *reinterpret_cast<const uint2*>(hi);
        *reinterpret_cast<uint2*>(linv_lo + static_cast<int64_t>(c0 + r) * kBlk + c4) = *reinterpret_cast<const uint2*>(lo);
    }
}

// Inverse of the stored 128x128 diagonal blocks of L for krr_potrs: block b = blockIdx.x is rows and
// columns [128 c, 128 c + 128) of diagonal tile k (b = k * nsub + c).  dinv, dinvT: [n/128][128][128]
// FP32, the inverse and its transpose.
__global__ void __launch_bounds__(kTriThreads, 1)
trtri128_kernel(const uint8_t* __restrict__ factor, const int64_t* __restrict__ off, int NT, int nb,
                float* __restrict__ dinv, float* __restrict__ dinvT) {
    extern __shared__ __align__(16) float tri_sm[];
    float* a = tri_sm;
    float* x = tri_sm + kBlk * kTriLd;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int nsub = nb / kBlk;
    const int k = blockIdx.x / nsub, c = blockIdx.x % nsub;
    const float* Lkk = reinterpret_cast<const float*>(factor + off[k * NT + k]);
    for (int idx = tid; idx < kBlk * (kBlk / 4); idx += kTriThreads) {
        const int r = idx / (kBlk / 4), c4 = (idx % (kBlk / 4)) * 4;
        *reinterpret_cast<float4*>(a + r * kTriLd + c4) =
            *reinterpret_cast<const float4*>(Lkk + static_cast<int64_t>(c * kBlk + r) * nb + c * kBlk + c4);
        *reinterpret_cast<float4*>(x + r * kTriLd + c4) = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    __syncthreads();
    if (warp < 4) inv32_warp(a, x, 32 * warp, lane);
    __syncthreads();
    inv128_offdiag(a, x, x + 32, warp, lane);
    float* out = dinv + static_cast<int64_t>(blockIdx.x) * kBlk * kBlk;
    for (int idx = tid; idx < kBlk * (kBlk / 4); idx += kTriThreads) {
        const int r = idx / (kBlk / 4), c4 = (idx % (kBlk / 4)) * 4;
        float4 v = *reinterpret_cast<const float4*>(x + r * kTriLd + c4);
        if (c4 + 0 > r) v.x = 0.f;
        if (c4 + 1 > r) v.y = 0.f;
        if (c4 + 2 > r) v.z = 0.f;
        if (c4 + 3 > r) v.w = 0.f;
        *reinterpret_cast<float4*>(out + r * kBlk + c4) = v;
    }
    float* outT = dinvT + static_cast<int64_t>(blockIdx.x) * kBlk * kBlk;
    for (int idx = tid; idx < kBlk * kBlk; idx += kTriThreads) {
        const int r = idx >> 7, c = idx & 127;
        outT[idx] = (c >= r) ? x[c * kTriLd + r] : 0.0f;
    }
}

}  // namespace krr

// FP32 kernels on one 128x128 diagonal block ("POTRF"):
//   potrf128_kernel   Cholesky of the block on plain FP32 ALUs plus the inverse of its factor
//                     (the panel TRSM multiplies by it on the tensor cores, gemm_tc.cuh MODE_P3)
//   trtri128_kernel   inverse of a stored 128x128 lower-triangular diagonal block (krr_potrs)
//
// Both are recursive over 32x32 sub-blocks held in shared memory.  The 128 pivots are a serial chain,
// so everything on that chain is kept short and everything else is moved off it:
//   chol32   one warp, lane = row, the row in registers, right-looking with shuffles.  Per pivot the
//            chain is shuffle -> reciprocal square root (MUFU.RSQ + one Newton step, correctly rounded
//            whenever 1/sqrt(d) is representable, else to ~1 ulp) -> multiply -> FMA; the diagonal entry
//            itself is the IEEE square root, computed off the chain.
//   trsv32   x L^T = s by substitution with the stored reciprocals of the diagonal, one thread per row
//            of the panel (and per column of the inverse of the diagonal sub-block, s = e_j): no
//            division and no explicit inverse on the chain.
//   the trailing update and the off-diagonal blocks of the inverse are small FP32 matrix products done by
//   all warps out of shared memory.
// Exactly representable inputs with power-of-two pivots give the exact factor (tests: "exactly
// representable constructions").
#pragma once
#include "common.cuh"

namespace krr {

constexpr int kAbUnroll = 2;
constexpr int kTriThreads = 512;
constexpr int kTriLd = 132;                       // 16-byte aligned rows; LDS.128 by row is conflict free
constexpr int kTriSmem = (2 * kBlk * kTriLd + kBlk + 32) * 4;   // L, inv(L), reciprocals of the diagonal of L, reduction scratch

__device__ __forceinline__ float rsqrt_newton(float d) {
    float rs;
    asm("rsqrt.approx.f32 %0, %1;" : "=f"(rs) : "f"(d));
    return rs * fmaf(-0.5f * d * rs, rs, 1.5f);    // rs (1.5 - 0.5 d rs^2): error squared, then one rounding
}

// Cholesky of the 32x32 block at (j0, j0) of a (smem, ld kTriLd), in place; zeros above the diagonal;
// rinv[j0 + j] = 1 / L_jj.  One warp.  Returns the 1-based local column of the first non-positive pivot
// (0 = none).
__device__ __forceinline__ int chol32_warp(float* a, float* rinv, int j0, int lane) {
    float r[32];
    float* row = a + (j0 + lane) * kTriLd + j0;
#pragma unroll
    for (int c = 0; c < 32; c += 4) {
        const float4 v = *reinterpret_cast<const float4*>(row + c);
        r[c] = v.x; r[c + 1] = v.y; r[c + 2] = v.z; r[c + 3] = v.w;
    }
    int bad = 0;
    float my_d = 1.0f, my_rs = 1.0f;
    float dn = r[0];                               // lane j's value is pivot j before its square root
#pragma unroll
    for (int j = 0; j < 32; ++j) {
        const float d = __shfl_sync(0xffffffffu, dn, j);
        if (!(d > 0.0f) && bad == 0) bad = j + 1;
        const float rs = rsqrt_newton(d);
        if (lane == j) { my_d = d; my_rs = rs; }
        const float l = r[j] * rs;                 // rows above j hold garbage here; never used
        r[j] = l;
        // the next pivot needs only lane j+1's own multiplier: keep it off the shuffle chain
        if (j + 1 < 32) dn = fmaf(-l, l, r[j + 1]);
#pragma unroll
        for (int c = j + 1; c < 32; ++c) {
            const float lc = __shfl_sync(0xffffffffu, l, c);
            r[c] = fmaf(-l, lc, r[c]);
        }
    }
    const float dj = sqrtf(my_d);                  // the diagonal entry: IEEE square root
    rinv[j0 + lane] = my_rs;
#pragma unroll
    for (int c = 0; c < 32; c += 4) {
        float4 v;
        v.x = (c + 0 < lane) ? r[c + 0] : (c + 0 == lane ? dj : 0.0f);
        v.y = (c + 1 < lane) ? r[c + 1] : (c + 1 == lane ? dj : 0.0f);
        v.z = (c + 2 < lane) ? r[c + 2] : (c + 2 == lane ? dj : 0.0f);
        v.w = (c + 3 < lane) ? r[c + 3] : (c + 3 == lane ? dj : 0.0f);
        *reinterpret_cast<float4*>(row + c) = v;
    }
    return bad;
}

// In place on s: the row vector x with x L^T = s for the lower-triangular 32x32 block Lb (smem, ld
// kTriLd) whose reciprocal diagonal is ri:  x_c = (s_c - sum_{m<c} x_m L[c][m]) * ri[c].
// Rows of L are broadcast LDS.128; four partial sums keep the FMA chains short.
__device__ __forceinline__ void trsv32(const float* Lb, const float* ri, float (&s)[32]) {
#pragma unroll
    for (int c = 0; c < 32; ++c) {
        float a0 = s[c], a1 = 0.0f, a2 = 0.0f, a3 = 0.0f;
        const float* lrow = Lb + c * kTriLd;
#pragma unroll
        for (int m = 0; m + 4 <= c; m += 4) {
            const float4 l = *reinterpret_cast<const float4*>(lrow + m);
            a0 = fmaf(-s[m + 0], l.x, a0);
            a1 = fmaf(-s[m + 1], l.y, a1);
            a2 = fmaf(-s[m + 2], l.z, a2);
            a3 = fmaf(-s[m + 3], l.w, a3);
        }
#pragma unroll
        for (int m = c & ~3; m < c; ++m) a0 = fmaf(-s[m], lrow[m], a0);
        s[c] = ((a0 + a1) + (a2 + a3)) * ri[c];
    }
}

// x = inverse of the lower-triangular 32x32 block of l at (j0, j0), written to the same block of x.
// One warp, lane = column j of the inverse: L x = e_j row by row, which is trsv32 with s = e_j.
__device__ __forceinline__ void inv32_warp(const float* l, const float* rinv, float* x, int j0, int lane) {
    float v[32];
#pragma unroll
    for (int r = 0; r < 32; ++r) v[r] = (r == lane) ? 1.0f : 0.0f;
    trsv32(l + j0 * kTriLd + j0, rinv + j0, v);
#pragma unroll
    for (int r = 0; r < 32; ++r) x[(j0 + r) * kTriLd + j0 + lane] = v[r];
}

// Panel of the 32-column block at j0: row i of a (i = first_row + thread index) <- row i times L_jj^-T.
__device__ __forceinline__ void panel32_row(float* a, const float* rinv, int j0, int i) {
    float s[32];
    float* row = a + i * kTriLd + j0;
#pragma unroll
    for (int c = 0; c < 32; c += 4) {
        const float4 v = *reinterpret_cast<const float4*>(row + c);
        s[c] = v.x; s[c + 1] = v.y; s[c + 2] = v.z; s[c + 3] = v.w;
    }
    trsv32(a + j0 * kTriLd + j0, rinv + j0, s);
#pragma unroll
    for (int c = 0; c < 32; c += 4) *reinterpret_cast<float4*>(row + c) = make_float4(s[c], s[c + 1], s[c + 2], s[c + 3]);
}

// C[r][c] -= sum_{m<32} P[r][m] Q[c][m] for rows r = rbeg, rbeg + rstep, ... < rend and c = lane: "P Q^T" with
// both operands row-major in smem (ld kTriLd).  The lane's row of Q stays in registers for all rows (the
// update is bound by shared-memory wavefronts: 8 broadcast LDS.128 of P per row of 32 outputs).
__device__ __forceinline__ void abt32_sub_rows(const float* P, const float* Q, float* out, int rbeg, int rend, int rstep,
                                               int lane) {
    float q[32];
#pragma unroll
    for (int m = 0; m < 32; m += 4) {
        const float4 v = *reinterpret_cast<const float4*>(Q + lane * kTriLd + m);
        q[m] = v.x; q[m + 1] = v.y; q[m + 2] = v.z; q[m + 3] = v.w;
    }
    for (int r = rbeg; r < rend; r += rstep) {
        float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
#pragma unroll
        for (int m = 0; m < 32; m += 4) {
            const float4 pv = *reinterpret_cast<const float4*>(P + r * kTriLd + m);
            a0 = fmaf(pv.x, q[m], a0);
            a1 = fmaf(pv.y, q[m + 1], a1);
            a2 = fmaf(pv.z, q[m + 2], a2);
            a3 = fmaf(pv.w, q[m + 3], a3);
        }
        out[r * kTriLd + lane] -= (a0 + a1) + (a2 + a3);
    }
}

// out[r][c] = sign * sum_{m<M} P[r][m] Q[m][c] for 4 rows and c = lane ("P Q", Q row-major): Q[m][c] is a
// conflict-free LDS.32, P[r][m] a broadcast LDS.128.
template <int M>
__device__ __forceinline__ void ab_4rows(const float* P, const float* Q, float* out, float sign, int lane) {
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll kAbUnroll
    for (int m = 0; m < M; m += 4) {
        const float q0 = Q[(m + 0) * kTriLd + lane], q1 = Q[(m + 1) * kTriLd + lane];
        const float q2 = Q[(m + 2) * kTriLd + lane], q3 = Q[(m + 3) * kTriLd + lane];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const float4 pv = *reinterpret_cast<const float4*>(P + u * kTriLd + m);
            acc[u] = fmaf(pv.x, q0, fmaf(pv.y, q1, fmaf(pv.z, q2, fmaf(pv.w, q3, acc[u]))));
        }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) out[u * kTriLd + lane] = sign * acc[u];
}

// Off-diagonal 32x32 blocks of block row i of x = inv(l), once x_ii and the block rows above are known:
//   x_ij = - x_ii * t_ij,  t_ij = sum_{j<=m<i} l_im x_mj.
// Two phases with a barrier between them, each a set of (block column j, 4-row group) tasks dealt to the
// `nw` participating warps (w = this warp's index among them).  `t` is a 32-row scratch strip (32 x 96
// used) inside the caller's shared memory (callers pass the still-zero upper-right corner of x, rows
// 0..31 x columns 32..127, and mask c > r when they write x out).
__device__ __forceinline__ void inv_row_phase1(const float* l, const float* x, float* t, int i, int w, int nw, int lane) {
    for (int task = w; task < 8 * i; task += nw) {
        const int j = task >> 3, r0 = (task & 7) * 4;
        const float* P = l + (32 * i + r0) * kTriLd + 32 * j;           // l_i,[j..i)
        const float* Q = x + (32 * j) * kTriLd + 32 * j;                // x_[j..i),j  (x_mj = 0 for m < j)
        float* o = t + r0 * kTriLd + 32 * j;
        if (i - j == 1) ab_4rows<32>(P, Q, o, 1.0f, lane);
        else if (i - j == 2) ab_4rows<64>(P, Q, o, 1.0f, lane);
        else ab_4rows<96>(P, Q, o, 1.0f, lane);
    }
}
__device__ __forceinline__ void inv_row_phase2(float* x, const float* t, int i, int w, int nw, int lane) {
    for (int task = w; task < 8 * i; task += nw) {
        const int j = task >> 3, r0 = (task & 7) * 4;
        ab_4rows<32>(x + (32 * i + r0) * kTriLd + 32 * i, t + 32 * j, x + (32 * i + r0) * kTriLd + 32 * j, -1.0f, lane);
    }
}
// all block rows in order, all kTriThreads threads (trtri128_kernel)
__device__ __forceinline__ void inv128_offdiag(const float* l, float* x, float* t, int warp, int lane) {
    constexpr int NW = kTriThreads / 32;
    for (int i = 1; i < 4; ++i) {
        inv_row_phase1(l, x, t, i, warp, NW, lane);
        __syncthreads();
        inv_row_phase2(x, t, i, warp, NW, lane);
        __syncthreads();
    }
}

// W: panel workspace [m][nb] FP32; the block is rows r0..r0+127 (panel-local), columns c0..c0+127.
// Writes L (lower, zeros above) back into W and inv(L) as scaled FP16 hi/lo planes into
// linv_hi/lo ([nb][128] row-major, rows c0..c0+127) with their power-of-two scale in linv_scale.
// col_base = 1-based global index of the block's first column, for info (LAPACK convention).
// The body runs on NTHR threads (tid = 0 .. NTHR-1, whole warps) that synchronise through `sync()`:
// the stand-alone kernel below uses the whole CTA, the fused diagonal-tile chain of gemm_tc.cuh its
// eight epilogue warps and a named barrier.  tri_sm: kTriSmem bytes of shared memory, 16-byte aligned.
template <int NTHR, typename Sync>
__device__ __forceinline__ void potrf128_body(float* tri_sm, int tid, Sync sync, float* __restrict__ W, int nb, int r0,
                                              int c0, __half* __restrict__ linv_hi, __half* __restrict__ linv_lo,
                                              float* __restrict__ linv_scale, int* __restrict__ info, int64_t col_base) {
    float* a = tri_sm;                       // [128][132] : S, then L
    float* x = tri_sm + kBlk * kTriLd;       // [128][132] : inv(L); rows 0..31 x columns 32.. double as scratch
    float* rinv = x + kBlk * kTriLd;         // [128]      : 1 / L_jj
    float* s_red = rinv + kBlk;              // [NTHR / 32]
    const int warp = tid >> 5, lane = tid & 31;
    constexpr int NW = NTHR / 32;
    // W is block-column-major: element (r, c) of 128x128 block (rb, cb) at ((rb*nsub + cb)*128 + c)*128 + r
    float* wblk = W + (static_cast<int64_t>(r0 / kBlk) * (nb / kBlk) + c0 / kBlk) * (kBlk * kBlk);
    {
        // coalesced column reads (lane = row), 32 per thread in flight before the first store
        constexpr int PER = 32;
        for (int base = 0; base < kBlk * kBlk; base += PER * NTHR) {
            float v[PER];
#pragma unroll
            for (int u = 0; u < PER; ++u) v[u] = wblk[base + tid + u * NTHR];
#pragma unroll
            for (int u = 0; u < PER; ++u) {
                const int idx = base + tid + u * NTHR, r = idx & (kBlk - 1), c = idx >> 7;
                a[r * kTriLd + c] = v[u];
            }
        }
        for (int idx = tid; idx < kBlk * (kBlk / 4); idx += NTHR)
            *reinterpret_cast<float4*>(x + (idx >> 5) * kTriLd + (idx & 31) * 4) = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    sync();
    float* tscr = x + 32;                    // scratch strip of the inverse's off-diagonal rows
    for (int jb = 0; jb < 4; ++jb) {
        const int j0 = 32 * jb;
        // A: warp 0 factors the diagonal sub-block (the serial chain); the other warps start block row
        //    jb-1 of the inverse, whose inputs are final
        if (warp == 0) {
            const int bad = chol32_warp(a, rinv, j0, lane);
            // the lowest bad column of the warp (every lane sees the same pivots)
            if (bad && lane == 0) atomicCAS(info, 0, static_cast<int>(col_base + j0 + bad - 1));
        } else if (jb >= 2) {
            inv_row_phase1(a, x, tscr, jb - 1, warp - 1, NW - 1, lane);
        }
        sync();
        const int R = kBlk - (j0 + 32);                 // rows below the diagonal block
        // B: panel, one thread per row below (warps 1 ..); warp 0 inverts the diagonal sub-block; the
        //    remaining warps finish block row jb-1 of the inverse
        const int first_free = 1 + R / 32;              // warps first_free .. NW-1 have neither job
        if (warp == 0) inv32_warp(a, rinv, x, j0, lane);
        else if (tid - 32 < R) panel32_row(a, rinv, j0, j0 + 32 + (tid - 32));
        else if (jb >= 2) inv_row_phase2(x, tscr, jb - 1, warp - first_free, NW - first_free, lane);
        sync();
        if (R > 0) {
            // C: trailing update S_ic -= L_i,jb L_c,jb^T for the 32-column blocks right of jb (lower part):
            //    each column block's rows are dealt to its share of the warps
            const int ncb = 3 - jb;                     // column blocks jb+1 .. 3
            const int cb = jb + 1 + warp % ncb, wi = warp / ncb, wn = (NW - 1 - warp % ncb) / ncb + 1;
            const int rr = 32 * cb;
            abt32_sub_rows(a + j0, a + rr * kTriLd + j0, a + rr, rr + wi, kBlk, wn, lane);
            sync();
        }
    }
    // block row 3 of the inverse
    inv_row_phase1(a, x, tscr, 3, warp, NW, lane);
    sync();
    inv_row_phase2(x, tscr, 3, warp, NW, lane);
    sync();
    // power-of-two scale of the inverse's planes: max|x| * si <= 2^14
    {
        float m = 0.0f;
        for (int idx = tid; idx < kBlk * kBlk; idx += NTHR) {
            const int r = idx >> 7, c = idx & 127;
            if (c <= r) m = fmaxf(m, fabsf(x[r * kTriLd + c]));
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
        if (lane == 0) s_red[warp] = m;
    }
    sync();
    float si = 1.0f;
    {
        float m = 0.0f;
#pragma unroll
        for (int w = 0; w < NTHR / 32; ++w) m = fmaxf(m, s_red[w]);
        if (m > 0.0f && m < 3.0e38f) {
            int e;
            frexpf(m, &e);                 // m <= 2^e
            si = ldexpf(1.0f, 14 - e);
        }
    }
    if (tid == 0) linv_scale[c0 / kBlk] = si;
    // L back into W: coalesced column writes (lane = row)
    for (int idx = tid; idx < kBlk * kBlk; idx += NTHR) {
        const int r = idx & (kBlk - 1), c = idx >> 7;
        wblk[idx] = (c <= r) ? a[r * kTriLd + c] : 0.0f;
    }
    // inverse as scaled hi/lo FP16 planes, row-major
    for (int idx = tid; idx < kBlk * (kBlk / 4); idx += NTHR) {
        const int r = idx / (kBlk / 4), c4 = (idx % (kBlk / 4)) * 4;
        const float4 xv4 = *reinterpret_cast<const float4*>(x + r * kTriLd + c4);
        const float xs[4] = {xv4.x, xv4.y, xv4.z, xv4.w};
        __align__(8) __half hi[4];
        __align__(8) __half lo[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const float xv = (c4 + u <= r) ? xs[u] * si : 0.0f;
            hi[u] = __float2half_rn(xv);
            lo[u] = __float2half_rn(xv - __half2float(hi[u]));
        }
        *reinterpret_cast<uint2*>(linv_hi + static_cast<int64_t>(c0 + r) * kBlk + c4) = *reinterpret_cast<const uint2*>(hi);
        *reinterpret_cast<uint2*>(linv_lo + static_cast<int64_t>(c0 + r) * kBlk + c4) = *reinterpret_cast<const uint2*>(lo);
    }
}


struct CtaSync { __device__ __forceinline__ void operator()() const { __syncthreads(); } };

__global__ void __launch_bounds__(kTriThreads, 1)
potrf128_kernel(float* __restrict__ W, int nb, int r0, int c0, __half* __restrict__ linv_hi,
                __half* __restrict__ linv_lo, float* __restrict__ linv_scale, int* __restrict__ info,
                int64_t col_base) {
    extern __shared__ __align__(16) float tri_sm[];
    potrf128_body<kTriThreads>(tri_sm, static_cast<int>(threadIdx.x), CtaSync(), W, nb, r0, c0, linv_hi, linv_lo, linv_scale,
                               info, col_base);
}

// The inverted 128-block c0 / 128 of the diagonal tile (linv planes, scale linv_scale[c0 / 128]) as the diagonal block of
// M = inv(L_kk) and, transposed, of M^T in the scratch planes Sh / Sl (row pitch nb; rows srow_m + c0.. / srow_mt + c0..,
// columns c0..) with the fixed scale scl[SCL_SM] (panel.cuh).  A power-of-two rescaling of the same 22 bits: exact unless
// the value leaves the FP16 range, which is reported as info = -2.  Off the critical path (inverse stream).
// grid = 16 CTAs of 256 threads: CTA b handles rows 8 b .. 8 b + 7.
__global__ void __launch_bounds__(256)
inv_export_kernel(const __half* __restrict__ linv_hi, const __half* __restrict__ linv_lo, const float* __restrict__ linv_scale,
                  int nb, int c0, __half* __restrict__ Sh, __half* __restrict__ Sl, int64_t srow_m, int64_t srow_mt,
                  const float* __restrict__ scl, int* __restrict__ info) {
    __shared__ float t[8][kBlk + 1];
    const float mul = scl[SCL_SM] / linv_scale[c0 / kBlk];
    const int r0 = blockIdx.x * 8;
    bool over = false;
    for (int idx = threadIdx.x; idx < 8 * kBlk; idx += 256) {
        const int rr = idx >> 7, c = idx & 127;
        const int64_t e = static_cast<int64_t>(c0 + r0 + rr) * kBlk + c;
        const float v = (__half2float(linv_hi[e]) + __half2float(linv_lo[e])) * mul;
        over |= !(fabsf(v) < 60000.0f);
        t[rr][c] = v;
        const __half h = __float2half_rn(v);
        const int64_t o = (srow_m + c0 + r0 + rr) * nb + c0 + c;
        Sh[o] = h;
        Sl[o] = __float2half_rn(v - __half2float(h));
    }
    __syncthreads();
    // transposed: rows c0 + c of M^T, columns c0 + r0 .. + 7 (16 bytes per row and plane)
    for (int idx = threadIdx.x; idx < 8 * kBlk; idx += 256) {
        const int c = idx >> 3, rr = idx & 7;
        const float v = t[rr][c];
        const __half h = __float2half_rn(v);
        const int64_t o = (srow_mt + c0 + c) * nb + c0 + r0 + rr;
        Sh[o] = h;
        Sl[o] = __float2half_rn(v - __half2float(h));
    }
    if (over) atomicCAS(info, 0, -2);
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
    float* rinv = x + kBlk * kTriLd;
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
    if (tid < kBlk) rinv[tid] = 1.0f / a[tid * kTriLd + tid];
    __syncthreads();
    if (warp < 4) inv32_warp(a, rinv, x, 32 * warp, lane);
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

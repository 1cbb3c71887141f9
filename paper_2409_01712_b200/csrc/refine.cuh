// Iterative refinement with a fixed factor (R19; named and not adopted in PAPER.md:192, offered by SURVEY
// section 8(c) as the remedy for the alpha tolerance under FP16 / FP8 maps): the residual of the symmetric system,
//     R = Y - A X,   A = K + lambda*I given by its lower tiles (FP32), X and Y row-major n x nrhs (FP32),
// with every product and sum in FP64 and R rounded to FP32 once, and the update X += D.
//
// HBM-bound (each stored 128 x 128 block of A is read twice: once for the rows it holds, once, transposed, for its
// columns; 2 * 4 n^2/2 bytes per residual) next to 2 n^2 nrhs FP64 flops.  One CTA owns 128 rows of R and one residue
// class of the 128-column blocks (segment); the segments' partial sums are added in a fixed order by the finishing
// kernel, so the result does not depend on timing.
#pragma once
#include "common.cuh"

namespace krr {

constexpr int kResKc = 32;         // columns of A staged per step (at most: ResidCfg::KC)
constexpr int kResSegMax = 16;

// number of column segments: a pure function of n (not of the device), about 4096 CTAs per residual (four are
// resident per SM: seven waves at n = 65536)
__host__ __device__ __forceinline__ int resid_segments(int64_t n) {
    const int64_t nblk = n / kBlk;
    int64_t s = 4096 / nblk;
    if (s < 1) s = 1;
    if (s > kResSegMax) s = kResSegMax;
    if (s > nblk) s = nblk;
    return static_cast<int>(s);
}

template <int NR>
struct ResidCfg {
    static constexpr int RPT = NR < 8 ? NR : 8;       // right-hand sides per thread
    static constexpr int NG = NR / RPT;               // thread groups over the right-hand sides
    // rows per thread (r, r + 128 / ROWS, ...): fewer shared-memory reads of X per FMA.  Measured at n = 65536 (A/B in one
    // gpurun call): NR = 32 with 4 rows 14.6 ms (2 rows: 15.8), NR = 4 with 2 rows 3.9 ms (1 row: 4.2), NR = 16 with 2 rows
    // 8.5 ms (4 rows: 8.8; reading column kk + 1 from shared memory before the FMAs of column kk: 8.9)
    static constexpr int ROWS = NR >= 32 ? 4 : 2;
    static constexpr int NTHR = kBlk / ROWS * NG;     // 64 (NR <= 8) or 128 (NR >= 16)
    static constexpr int KC = NTHR >= 128 ? kResKc : kResKc / 2;   // columns of A per chunk: 32 staged elements per thread
    static constexpr int NLD = kBlk * KC / NTHR;      // elements of A per thread and chunk
    static constexpr int NXL = (KC * NR + NTHR - 1) / NTHR;
};

// partial[seg][row][NR] = sum over the 128-column blocks cb = seg, seg + nseg, ... of A(rows, cb) X(cb, :).
// A chunk is 128 rows x 32 columns of the symmetric matrix; the loads of chunk i + 1 are issued (into registers)
// before the FMAs of chunk i, so DRAM latency is covered by the arithmetic of the same CTA.
template <int NR>
__global__ void __launch_bounds__(ResidCfg<NR>::NTHR)
resid_partial_kernel(AView A, const float* __restrict__ X, int64_t ldx, int nrhs, int nblk, int nseg,
                     double* __restrict__ partial) {
    using Cfg = ResidCfg<NR>;
    constexpr int RPT = Cfg::RPT, NTHR = Cfg::NTHR, ROWS = Cfg::ROWS, RSTEP = kBlk / ROWS, NLD = Cfg::NLD, NXL = Cfg::NXL;
    constexpr int KC = Cfg::KC, CPB = kBlk / KC;                // chunks per block
    __shared__ float S[KC][kBlk + (KC == 16 ? 2 : 1)];   // S[kk][r] = a(row r of the block row, column k0 + kk); padded: conflict-free staging
    __shared__ double Xs[KC][NR];
    const int t = threadIdx.x, r = t % RSTEP, g = t / RSTEP;
    const int rb = blockIdx.x, seg = blockIdx.y;
    const int nsub = A.nb / kBlk;
    const int64_t ls = A.row_stride();
    double acc[ROWS][RPT];
#pragma unroll
    for (int i = 0; i < ROWS; ++i)
#pragma unroll
        for (int q = 0; q < RPT; ++q) acc[i][q] = 0.0;
    float ra[NLD], rx[NXL];

    const int nchunks = ((nblk - seg + nseg - 1) / nseg) * CPB;
    // issue the global loads of chunk i
    auto fetch = [&](int i) {
        const int cb = seg + (i / CPB) * nseg, k0 = (i % CPB) * KC;
        // block (rb, cb) of the symmetric matrix lives in the lower triangle as block (max, min)
        const int br = rb > cb ? rb : cb, bc = rb > cb ? cb : rb;
        const float* B = A.tile_ptr(br / nsub, bc / nsub, (br % nsub) * kBlk, (bc % nsub) * kBlk);
        if (cb < rb) {                                                        // stored as is: rows of B are our rows
#pragma unroll
            for (int j = 0; j < NLD; ++j) {
                const int e = t + j * NTHR, rr = e / KC, kk = e % KC;
                ra[j] = __ldg(B + rr * ls + k0 + kk);
            }
        } else if (cb > rb) {                                                 // stored transposed: columns of B are our rows
#pragma unroll
            for (int j = 0; j < NLD; ++j) {
                const int e = t + j * NTHR, kk = e / kBlk, rr = e % kBlk;
                ra[j] = __ldg(B + (k0 + kk) * ls + rr);
            }
        } else {                                                              // diagonal block: lower triangle, mirrored
#pragma unroll
            for (int j = 0; j < NLD; ++j) {
                const int e = t + j * NTHR, kk = e / kBlk, rr = e % kBlk, c = k0 + kk;
                ra[j] = rr >= c ? __ldg(B + rr * ls + c) : __ldg(B + c * ls + rr);
            }
        }
#pragma unroll
        for (int j = 0; j < NXL; ++j) {
            const int e = t + j * NTHR, kk = e / NR, q = e % NR;
            rx[j] = (e < KC * NR && q < nrhs) ? __ldg(X + (static_cast<int64_t>(cb) * kBlk + k0 + kk) * ldx + q) : 0.0f;
        }
    };
    // registers -> shared memory, in the layout the FMAs read
    auto stage = [&](int i) {
        const int cb = seg + (i / CPB) * nseg;
        if (cb < rb) {
#pragma unroll
            for (int j = 0; j < NLD; ++j) {
                const int e = t + j * NTHR;
                S[e % KC][e / KC] = ra[j];
            }
        } else {
#pragma unroll
            for (int j = 0; j < NLD; ++j) {
                const int e = t + j * NTHR;
                S[e / kBlk][e % kBlk] = ra[j];
            }
        }
#pragma unroll
        for (int j = 0; j < NXL; ++j) {
            const int e = t + j * NTHR;
            if (e < KC * NR) Xs[e / NR][e % NR] = static_cast<double>(rx[j]);
        }
    };

    if (nchunks > 0) fetch(0);
    for (int i = 0; i < nchunks; ++i) {
        __syncthreads();                                                      // the previous chunk has been consumed
        stage(i);
        __syncthreads();
        if (i + 1 < nchunks) fetch(i + 1);
#pragma unroll 4
        for (int kk = 0; kk < KC; ++kk) {
            double a[ROWS];
#pragma unroll
            for (int u = 0; u < ROWS; ++u) a[u] = static_cast<double>(S[kk][r + u * RSTEP]);
#pragma unroll
            for (int q = 0; q < RPT; ++q) {
                const double x = Xs[kk][g * RPT + q];
#pragma unroll
                for (int u = 0; u < ROWS; ++u) acc[u][q] = fma(a[u], x, acc[u][q]);
            }
        }
    }
#pragma unroll
    for (int u = 0; u < ROWS; ++u) {
        double* out = partial + ((static_cast<int64_t>(seg) * nblk + rb) * kBlk + r + u * RSTEP) * NR + g * RPT;
#pragma unroll
        for (int q = 0; q < RPT; ++q) out[q] = acc[u][q];
    }
}

// R = fl32(Y - (partial[0] + partial[1] + ...)), compact n x nrhs; blk_sumsq[block] = sum of the squares of the stored R
// of that block's elements (FP64, fixed tree).  One thread per element of the NR-padded rows.
template <int NR>
__global__ void __launch_bounds__(256)
resid_finish_kernel(const double* __restrict__ partial, int nseg, int64_t n, const float* __restrict__ Y, int64_t ldy,
                    float* __restrict__ R, int nrhs, double* __restrict__ blk_sumsq) {
    __shared__ double red[8];
    const int64_t e = static_cast<int64_t>(blockIdx.x) * 256 + threadIdx.x;
    const int64_t row = e / NR;
    const int q = static_cast<int>(e % NR);
    double sq = 0.0;
    if (row < n && q < nrhs) {
        double s = 0.0;
        for (int g = 0; g < nseg; ++g) s += partial[(static_cast<int64_t>(g) * n + row) * NR + q];
        const float rv = static_cast<float>(static_cast<double>(Y[row * ldy + q]) - s);
        R[row * nrhs + q] = rv;
        sq = static_cast<double>(rv) * static_cast<double>(rv);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sq += __shfl_xor_sync(0xffffffffu, sq, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = sq;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < 8; ++w) s += red[w];
        blk_sumsq[blockIdx.x] = s;
    }
}

// out[0] = sqrt(sum of blk_sumsq[0 .. nblocks)), one block, fixed order
__global__ void __launch_bounds__(256)
resid_norm_kernel(const double* __restrict__ blk_sumsq, int64_t nblocks, double* __restrict__ out) {
    __shared__ double red[256];
    double s = 0.0;
    for (int64_t i = threadIdx.x; i < nblocks; i += 256) s += blk_sumsq[i];
    red[threadIdx.x] = s;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) out[0] = sqrt(red[0]);
}

// X(row, q) = fl32(X(row, q) + D(row, q)), D compact n x nrhs
__global__ void __launch_bounds__(256)
refine_update_kernel(float* __restrict__ X, int64_t ldx, const float* __restrict__ D, int64_t n, int nrhs) {
    const int64_t e = static_cast<int64_t>(blockIdx.x) * 256 + threadIdx.x;
    if (e >= n * nrhs) return;
    const int64_t row = e / nrhs;
    const int q = static_cast<int>(e % nrhs);
    X[row * ldx + q] += D[e];
}

// ---- conjugate gradients preconditioned by the fixed factor (R20) ----
// All vectors are compact n x nrhs (row-major, leading dimension nrhs); every right-hand side has its own scalars.

// v = sum of the segments' partial products (FP64); out64 = Y - v (Y given) or v; optionally the FP32 copy and the
// per-block sums of squares of out64.
template <int NR>
__global__ void __launch_bounds__(256)
pcg_finish_kernel(const double* __restrict__ partial, int nseg, int64_t n, const float* __restrict__ Y, int64_t ldy,
                  double* __restrict__ out64, float* __restrict__ out32, int nrhs, double* __restrict__ blk_sumsq) {
    __shared__ double red[8];
    const int64_t e = static_cast<int64_t>(blockIdx.x) * 256 + threadIdx.x;
    const int64_t row = e / NR;
    const int q = static_cast<int>(e % NR);
    double sq = 0.0;
    if (row < n && q < nrhs) {
        double v = 0.0;
        for (int g = 0; g < nseg; ++g) v += partial[(static_cast<int64_t>(g) * n + row) * NR + q];
        if (Y) v = static_cast<double>(Y[row * ldy + q]) - v;
        out64[row * nrhs + q] = v;
        if (out32) out32[row * nrhs + q] = static_cast<float>(v);
        sq = v * v;
    }
    if (!blk_sumsq) return;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sq += __shfl_xor_sync(0xffffffffu, sq, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = sq;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < 8; ++w) s += red[w];
        blk_sumsq[blockIdx.x] = s;
    }
}

constexpr int kDotRows = 256;      // rows per block of the column inner products
constexpr int kMaxRhsDot = 32;

// part[block][q] = sum over the block's rows of a(row, q) * b(row, q), FP64, fixed order
template <typename TA, typename TB>
__global__ void __launch_bounds__(kDotRows)
coldot_partial_kernel(const TA* __restrict__ a, const TB* __restrict__ b, int64_t n, int nrhs, double* __restrict__ part) {
    __shared__ double red[kDotRows / 32][kMaxRhsDot];
    const int64_t row = static_cast<int64_t>(blockIdx.x) * kDotRows + threadIdx.x;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int q = 0; q < nrhs; ++q) {
        double v = row < n ? static_cast<double>(a[row * nrhs + q]) * static_cast<double>(b[row * nrhs + q]) : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) red[warp][q] = v;
    }
    __syncthreads();
    if (threadIdx.x < nrhs) {
        double s = 0.0;
        for (int w = 0; w < kDotRows / 32; ++w) s += red[w][threadIdx.x];
        part[static_cast<int64_t>(blockIdx.x) * kMaxRhsDot + threadIdx.x] = s;
    }
}

// out[q] = sum over the blocks of part[block][q]
__global__ void __launch_bounds__(kMaxRhsDot)
coldot_final_kernel(const double* __restrict__ part, int64_t nblocks, int nrhs, double* __restrict__ out) {
    if (threadIdx.x >= nrhs) return;
    double s = 0.0;
    for (int64_t i = 0; i < nblocks; ++i) s += part[i * kMaxRhsDot + threadIdx.x];
    out[threadIdx.x] = s;
}

// a_q = rho_q / pq_q (0 if pq_q <= 0);  x += a p;  r -= a q;  z32 = fl32(r);  blk_sumsq = sums of squares of the new r
__global__ void __launch_bounds__(256)
pcg_update_xr_kernel(double* __restrict__ x, double* __restrict__ r, const float* __restrict__ p, const double* __restrict__ qv,
                     const double* __restrict__ rho, const double* __restrict__ pq, float* __restrict__ z32, int64_t n,
                     int nrhs, double* __restrict__ blk_sumsq) {
    __shared__ double red[8];
    const int64_t e = static_cast<int64_t>(blockIdx.x) * 256 + threadIdx.x;
    double sq = 0.0;
    if (e < n * nrhs) {
        const int q = static_cast<int>(e % nrhs);
        const double d = pq[q];
        const double a = d > 0.0 ? rho[q] / d : 0.0;
        x[e] = fma(a, static_cast<double>(p[e]), x[e]);
        const double rv = fma(-a, qv[e], r[e]);
        r[e] = rv;
        z32[e] = static_cast<float>(rv);
        sq = rv * rv;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sq += __shfl_xor_sync(0xffffffffu, sq, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = sq;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < 8; ++w) s += red[w];
        blk_sumsq[blockIdx.x] = s;
    }
}

// b_q = rho_new_q / rho_q (0 if rho_q <= 0);  p = fl32(z + b p)
__global__ void __launch_bounds__(256)
pcg_update_p_kernel(float* __restrict__ p, const float* __restrict__ z, const double* __restrict__ rho,
                    const double* __restrict__ rho_new, int64_t n, int nrhs) {
    const int64_t e = static_cast<int64_t>(blockIdx.x) * 256 + threadIdx.x;
    if (e >= n * nrhs) return;
    const int q = static_cast<int>(e % nrhs);
    const double d = rho[q];
    const double b = d > 0.0 ? rho_new[q] / d : 0.0;
    p[e] = static_cast<float>(fma(b, static_cast<double>(p[e]), static_cast<double>(z[e])));
}

// compact FP64 <- strided FP32, and back
__global__ void __launch_bounds__(256)
pcg_load_x_kernel(const float* __restrict__ X, int64_t ldx, double* __restrict__ x, int64_t n, int nrhs) {
    const int64_t e = static_cast<int64_t>(blockIdx.x) * 256 + threadIdx.x;
    if (e >= n * nrhs) return;
    x[e] = static_cast<double>(X[(e / nrhs) * ldx + e % nrhs]);
}
__global__ void __launch_bounds__(256)
pcg_store_x_kernel(float* __restrict__ X, int64_t ldx, const double* __restrict__ x, int64_t n, int nrhs) {
    const int64_t e = static_cast<int64_t>(blockIdx.x) * 256 + threadIdx.x;
    if (e >= n * nrhs) return;
    X[(e / nrhs) * ldx + e % nrhs] = static_cast<float>(x[e]);
}

}  // namespace krr

// krr_precision_map kernels: tile Frobenius norms (FP64 accumulation, fixed order), tile amax and
// the Frobenius-norm precision rule (rule text BASELINE.json north_star).
// One pass over the lower tiles of A: HBM-bound.
#pragma once
#include "common.cuh"

namespace krr {

constexpr int kStatRows = 32;        // rows of a tile reduced by one CTA
constexpr int kStatThreads = 256;

// grid = (nslots, nb / kStatRows) -- the unbounded index in x (gridDim.y stops at 65535).  partial[slot * chunks + chunk] = sum of squares (double),
// pamax[...] = max |a| of rows [chunk*kStatRows, +kStatRows) of the tile.
__global__ void __launch_bounds__(kStatThreads)
tile_stats_kernel(AView A, double* __restrict__ partial, float* __restrict__ pamax) {
    const int NT = A.NT, nb = A.nb;
    const int64_t slot = blockIdx.x;
    // invert slot -> (i, j): column-major lower order
    int j = 0;
    int64_t rem = slot;
    while (rem >= NT - j) { rem -= NT - j; ++j; }
    const int i = j + static_cast<int>(rem);
    const int chunk = blockIdx.y;
    const int r0 = chunk * kStatRows;
    const int vec_per_row = nb / 4;
    double acc = 0.0;
    float amax = 0.0f;
    for (int idx = threadIdx.x; idx < kStatRows * vec_per_row; idx += kStatThreads) {
        const int r = r0 + idx / vec_per_row;
        const int c = (idx % vec_per_row) * 4;
        const float4 v = __ldg(reinterpret_cast<const float4*>(A.tile_ptr(i, j, r, c)));
        acc += static_cast<double>(v.x) * v.x;
        acc += static_cast<double>(v.y) * v.y;
        acc += static_cast<double>(v.z) * v.z;
        acc += static_cast<double>(v.w) * v.w;
        amax = fmaxf(amax, fmaxf(fmaxf(fabsf(v.x), fabsf(v.y)), fmaxf(fabsf(v.z), fabsf(v.w))));
    }
    __shared__ double s_acc[kStatThreads];
    __shared__ float s_max[kStatThreads];
    s_acc[threadIdx.x] = acc;
    s_max[threadIdx.x] = amax;
    __syncthreads();
    for (int o = kStatThreads / 2; o > 0; o >>= 1) {      // fixed-order tree: deterministic
        if (threadIdx.x < o) {
            s_acc[threadIdx.x] += s_acc[threadIdx.x + o];
            s_max[threadIdx.x] = fmaxf(s_max[threadIdx.x], s_max[threadIdx.x + o]);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        partial[slot * gridDim.y + chunk] = s_acc[0];
        pamax[slot * gridDim.y + chunk] = s_max[0];
    }
}

// Single CTA: per-tile totals, ||A||_F, and the rule.
__global__ void __launch_bounds__(1024)
map_decide_kernel(int NT, int chunks, const double* __restrict__ partial, const float* __restrict__ pamax,
                  float eps_target, unsigned allowed_mask, uint8_t* __restrict__ map,
                  float* __restrict__ tile_norms, float* __restrict__ tile_amax, double* __restrict__ fro_out,
                  double* __restrict__ sumsq /* nslots scratch */) {
    const int64_t nslots = static_cast<int64_t>(NT) * (NT + 1) / 2;
    __shared__ double s_red[1024];
    double local = 0.0;
    // slots are visited in a fixed assignment; the weighted sum below is a fixed-shape tree
    for (int64_t s = threadIdx.x; s < nslots; s += blockDim.x) {
        double t = 0.0;
        float m = 0.0f;
        for (int c = 0; c < chunks; ++c) {
            t += partial[s * chunks + c];
            m = fmaxf(m, pamax[s * chunks + c]);
        }
        sumsq[s] = t;
        int j = 0;
        int64_t rem = s;
        while (rem >= NT - j) { rem -= NT - j; ++j; }
        const int i = j + static_cast<int>(rem);
        local += (i == j) ? t : 2.0 * t;                 // off-diagonal tiles count twice
        if (tile_norms) tile_norms[i * NT + j] = static_cast<float>(sqrt(t));
        if (tile_amax) tile_amax[i * NT + j] = m;
    }
    s_red[threadIdx.x] = local;
    __syncthreads();
    for (int o = blockDim.x / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) s_red[threadIdx.x] += s_red[threadIdx.x + o];
        __syncthreads();
    }
    const double fro = sqrt(s_red[0]);
    if (threadIdx.x == 0 && fro_out) *fro_out = fro;
    const double rhs = static_cast<double>(eps_target) * fro / NT;
    const double u[3] = {5.9604644775390625e-08 /*2^-24*/, 4.8828125e-04 /*2^-11*/, 6.25e-02 /*2^-4*/};
    for (int64_t s = threadIdx.x; s < nslots; s += blockDim.x) {
        int j = 0;
        int64_t rem = s;
        while (rem >= NT - j) { rem -= NT - j; ++j; }
        const int i = j + static_cast<int>(rem);
        int p = KRR_FP32;
        if (i != j) {
            const double t = sqrt(sumsq[s]);
            if ((allowed_mask & 4u) && t * u[2] <= rhs) p = KRR_FP8_E4M3;
            else if ((allowed_mask & 2u) && t * u[1] <= rhs) p = KRR_FP16;
        }
        map[i * NT + j] = static_cast<uint8_t>(p);
    }
    // entries above the diagonal: unused marker / zeros
    for (int idx = threadIdx.x; idx < NT * NT; idx += blockDim.x) {
        const int i = idx / NT, j = idx % NT;
        if (j > i) {
            map[idx] = 255;
            if (tile_norms) tile_norms[idx] = 0.0f;
            if (tile_amax) tile_amax[idx] = 0.0f;
        }
    }
}

}  // namespace krr

// Build phase (Alg. 2 :92-106, Alg. 5 :136-143, V-B1 :173-190, VI-B2 :207-209):
//   A = K + lambda*I,  K_ij = exp(-gamma * ||g_i - g_j||^2),  g_i = row i of the int8 genotype matrix G,
// with the squared distance expanded as  d2_ij = s_i + s_j - 2 <g_i, g_j>  (:186), the Gram matrix G G^T on the
// INT8 tensor cores (tcgen05 kind::i8, INT32 accumulation -- exact), the squared norms s folded into one vector
// (:209 "fold the column entries of the matrix D ... store D as a one-dimensional vector"), the tiles of D
// generated on demand and exponentiated before they are released (:209) -- no n x n integer temporary.
//
// Only the lower TILES of A (tile row >= tile column, diagonal tiles as full squares) are produced: that
// is what the Associate phase reads.  One persistent, warp-specialised kernel on CTA pairs (cluster of 2,
// cta_group::2): a pair computes a 256 x 512 block over the whole SNP range (256 x 256 when the tile size is
// no multiple of 512) into both 256-column INT32 accumulators of TMEM (single-buffered), each CTA staging
// 128 rows of the row operand and 2 x 128 of the column operand per 128-SNP chunk (TMA, 128-byte swizzle,
// 4-slot ring of 48 KB).  SNP counts that are not a multiple of 128 rely on TMA's zero fill.
#pragma once
#include "common.cuh"
#include "ptx.cuh"

namespace krr {

struct BuildOp {
    int64_t n, p;           // columns of the output (patients of the column operand), SNPs
    int64_t m;              // rows of the output: = n for the symmetric Build, the test cohort for Predict (rect)
    int rect;               // 1: test x training kernel matrix (Alg. 4 l.5): every block, no diagonal, dense output
    int nb;                 // tile size of A (which tiles are "lower", and the packed layout)
    int tiled;              // KRR_FLAG_A_TILED_LOWER
    float gamma;
    float diag;             // (float)(1.0 + lambda): K_ii = exp(0) = 1 exactly
    const int* sq;          // s_j = sum_k g_jk^2 of the column operand
    const int* sq_row;      // the same of the row operand (= sq for the symmetric Build)
    float* A;
    int64_t lda;
    // confounders: real-valued covariates whose squared distance, accumulated in FP32, is added to the
    // integer squared distance before the exponentiation.  q = 0: none.
    const float* C;         // column operand's confounders, n x q row-major (ldc)
    const float* C_row;     // row operand's (= C for the symmetric Build)
    int64_t ldc, ldc_row;
    int q;
    // IBS kernel (Alg. 5 l.5-6): the operands are thermometer encodings ([g >= 1], [g >= 2]) of the genotypes, d2 is then
    // the Hamming distance sum_k |g_ik - g_jk| and K_ij = (alleles - d2) / alleles, alleles = 2 N_S (no exponential)
    int ibs;
    float alleles;
    // linear kernel (the SYRK of ridge regression, Eq. (2), Fig. 2): K_ij = gamma * <g_i, g_j>, lambda on the diagonal
    int linear;
    float lambda;
    // ragged n (R21): rows and columns >= n_valid are the identity border (1 on the diagonal, 0 elsewhere)
    int64_t n_valid;
    // optional tile statistics of A for the precision map (no second pass over A): per lower tile
    // stats_chunks = (blocks per tile) * 16 partial sums of squares (FP64) and maxima, one per epilogue warp of the
    // block's two CTAs, in the layout map_decide_kernel reads (precision_map.cuh)
    double* stat_sumsq;
    float* stat_amax;
    int stats_chunks;
    // row units (of 256 rows) [ru_lo, ru_hi) of the output are built by this launch (ru_hi = 0: all of them).  krr_fit_host
    // builds the matrix strip by strip behind the host-to-device copy of the genotypes.
    int ru_lo, ru_hi;
};
constexpr int kMaxConfounders = 16;

// NACC = 256-column accumulators per pair: 2 -> a pair computes 256 x 512 (all 512 TMEM columns, the exp epilogue
// is then not overlapped with the next block's MMAs -- a few % at thousands of SNPs -- but every byte of the row
// operand feeds twice the MMAs: the kernel is bound by L2 -> shared-memory and HBM traffic, not by the tensor
// pipe); 1 -> 256 x 256 with double-buffered accumulators (tiles of 256).
constexpr int kBuildThreads = 320;                  // warp 0 TMA, warp 1 MMA (+ TMEM alloc), 2-9 epilogue
__host__ __device__ constexpr int build_slot_bytes(int nacc) { return (1 + nacc) * kBlk * 128; }   // [row block | nacc column blocks] x 128 SNPs
__host__ __device__ constexpr int build_slots(int nacc) { return nacc == 1 ? 6 : 4; }
__host__ __device__ constexpr int build_smem(int nacc) { return build_slots(nacc) * build_slot_bytes(nacc) + 1024 + 256; }

// s_i = sum_k g_ik^2 (INT32; exact while p * 127^2 < 2^31).  One warp per row, 16-byte loads.
__global__ void __launch_bounds__(256)
row_sqnorm_kernel(const int8_t* __restrict__ G, int64_t n, int64_t p, int64_t ldg, int* __restrict__ sq) {
    const int64_t row = static_cast<int64_t>(blockIdx.x) * 8 + (threadIdx.x >> 5);
    if (row >= n) return;
    const int lane = threadIdx.x & 31;
    const int8_t* g = G + row * ldg;
    int acc = 0;
    const int64_t pv = p & ~static_cast<int64_t>(15);
    for (int64_t k = lane * 16; k < pv; k += 32 * 16) {
        const int4 v = *reinterpret_cast<const int4*>(g + k);
        acc = __dp4a(v.x, v.x, acc);
        acc = __dp4a(v.y, v.y, acc);
        acc = __dp4a(v.z, v.z, acc);
        acc = __dp4a(v.w, v.w, acc);
    }
    for (int64_t k = pv + lane; k < p; k += 32) acc += static_cast<int>(g[k]) * static_cast<int>(g[k]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) sq[row] = acc;
}

// Thermometer encoding for the IBS kernel: U[i][k] = [g_ik >= 1], U[i][p + k] = [g_ik >= 2] (int8 0/1, row pitch ldu);
// columns p2 .. ldu-1 are zeroed so that the encoded matrix can be read in whole 16-byte units.
__global__ void __launch_bounds__(256)
ibs_encode_kernel(const int8_t* __restrict__ G, int64_t n, int64_t p, int64_t ldg, int8_t* __restrict__ U, int64_t ldu) {
    const int64_t row = blockIdx.x;             // rows in x: gridDim.y stops at 65535, n does not
    const int8_t* g = G + row * ldg;
    int8_t* u = U + row * ldu;
    for (int64_t k = static_cast<int64_t>(blockIdx.y) * 256 + threadIdx.x; k < ldu; k += static_cast<int64_t>(gridDim.y) * 256) {
        int8_t v = 0;
        if (k < p) v = g[k] >= 1;
        else if (k < 2 * p) v = g[k - p] >= 2;
        u[k] = v;
    }
    (void)n;
}

// 256 x 256 blocks (units) of the lower tiles: unit (ru, cu) is wanted when the tile of its rows is at or below
// the tile of its columns.  Order: panels of kBuildPanel column units; inside a panel row unit by row unit.
// The ~74 blocks in flight at any time then cover ~9 row units x 8 column units and read 17 operand strips
// instead of 75 (a strip = 256 patients x p SNPs; G is far larger than L2, so the order decides the DRAM
// traffic: 552 GB -> see profiles/ for the row-major order on C3).  Every warp role walks the same sequence
// with its own cursor; stepping is a few integer operations per block against ~100k clocks of MMAs.
constexpr int kBuildPanel = 8;                      // panel width in 256-column units
struct BuildCursor {
    int cp, ru, ci;          // column panel, row unit, column inside the panel
    bool done;
};
// cw = width of a column unit in 256-column units (NACC); cu counts column units of that width
// (upt = 0 marks the rectangular test x training matrix of Predict: every block is wanted)
__device__ __forceinline__ bool build_valid(int ru, int cu, int upt, int cw) { return upt == 0 || ru / upt >= cu * cw / upt; }
__device__ __forceinline__ void build_cursor_init(BuildCursor& c, int upt, int ru_lo) {
    c.cp = 0; c.ru = ru_lo; c.ci = 0; c.done = false;
    (void)upt;
}
// move to the next wanted unit strictly after the current position (or stay if `first` and it is wanted)
// (rows: units [ru_lo, nru))
__device__ __forceinline__ void build_cursor_seek(BuildCursor& c, int ru_lo, int nru, int ncu256, int upt, int cw, bool first) {
    const int pw = kBuildPanel / cw, ncu = ncu256 / cw;       // panel width and matrix width in column units
    bool skip = !first;
    while (!c.done) {
        if (!skip) {
            const int cu = c.cp * pw + c.ci;
            if (cu < ncu && c.ru < nru && build_valid(c.ru, cu, upt, cw)) return;
        }
        skip = false;
        if (++c.ci == pw) {
            c.ci = 0;
            if (++c.ru >= nru) {
                ++c.cp;
                if (c.cp * pw >= ncu) { c.done = true; return; }
                c.ru = upt ? (c.cp * kBuildPanel / upt) * upt : 0;   // first row unit of the panel's first tile
                if (c.ru < ru_lo) c.ru = ru_lo;
                if (c.ru >= nru && upt) { c.done = true; return; }    // later panels start further down still
            }
        }
    }
}
// the block this pair handles next: `steps` wanted units further (steps = pair index at first, then #pairs)
__device__ __forceinline__ bool build_next_block(BuildCursor& c, bool& started, int pair0, int npairs, int ru_lo, int nru, int ncu256,
                                                 int upt, int cw, int& ru, int& cu) {
    int steps = started ? npairs : pair0;
    if (!started) { build_cursor_seek(c, ru_lo, nru, ncu256, upt, cw, true); started = true; }
    for (; steps > 0 && !c.done; --steps) build_cursor_seek(c, ru_lo, nru, ncu256, upt, cw, false);
    if (c.done) return false;
    ru = c.ru;
    cu = c.cp * (kBuildPanel / cw) + c.ci;
    return true;
}

template <int NACC>
__global__ void __launch_bounds__(kBuildThreads, 1)
build_tc_kernel(const __grid_constant__ CUtensorMap tmR, const __grid_constant__ CUtensorMap tmG, const BuildOp op) {
    // tmR: genotypes of the row operand (= tmG for the symmetric Build), tmG: of the column operand
    constexpr int kBuildSlots = build_slots(NACC), kBuildSlotBytes = build_slot_bytes(NACC), NBUF = 2 / NACC;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar_base = smem_base + kBuildSlots * kBuildSlotBytes;
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (8 + s); };
    auto tfull_bar = [&](int b) { return bar_base + 8u * (16 + b); };
    auto tempty_bar = [&](int b) { return bar_base + 8u * (18 + b); };
    const uint32_t tmem_slot = bar_base + 8u * 20;
    uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - ptx::smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int rank = static_cast<int>(ptx::cluster_ctarank());
    const int pair0 = static_cast<int>(blockIdx.x >> 1), npairs = static_cast<int>(gridDim.x >> 1);
    const int nru = op.ru_hi > 0 ? op.ru_hi : static_cast<int>(op.m / 256), ncu256 = static_cast<int>(op.n / 256);
    const int ru_lo = op.ru_hi > 0 ? op.ru_lo : 0;
    const int NT = static_cast<int>(op.n / op.nb), upt = op.rect ? 0 : op.nb / 256;
    const int nch = static_cast<int>((op.p + 127) / 128);           // 128-SNP chunks (the last one zero-filled by TMA)
    constexpr uint32_t kHalf = kBlk * 128;                           // 16 KB operand block

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tmap(&tmG);
        ptx::prefetch_tmap(&tmR);
        for (int s = 0; s < kBuildSlots; ++s) { ptx::mbar_init(full_bar(s), 1); ptx::mbar_init(empty_bar(s), 1); }
        for (int b = 0; b < 2; ++b) { ptx::mbar_init(tfull_bar(b), 1); ptx::mbar_init(tempty_bar(b), 16); }
        ptx::fence_mbar_init();
    }
    if (warp == 1) {
        ptx::tmem_alloc<512, 2>(tmem_slot);
        ptx::tmem_relinquish<2>();
    }
    ptx::tc_fence_before();
    ptx::cluster_sync_all();
    ptx::tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    if (warp == 0) {
        // ===================== TMA producer (uniform control flow, one elected lane issues) =====================
        int slot = 0;
        uint32_t phase = 0;
        BuildCursor cur;
        build_cursor_init(cur, upt, ru_lo);
        bool started = false;
        int ru, cu;
        while (build_next_block(cur, started, pair0, npairs, ru_lo, nru, ncu256, upt, NACC, ru, cu)) {
            const int a_row = ru * 256 + rank * kBlk, b_row = cu * 256 * NACC + rank * kBlk;
            for (int ch = 0; ch < nch; ++ch) {
                ptx::mbar_wait(empty_bar(slot), phase ^ 1u);
                if (ptx::elect_one()) {
                    const uint32_t sa = smem_base + slot * kBuildSlotBytes;
                    if (rank == 0) ptx::mbar_arrive_expect_tx(full_bar(slot), 2u * (1 + NACC) * kHalf);
                    ptx::tma_load_2d_pair(sa, &tmR, full_bar(slot), ch * 128, a_row);
#pragma unroll
                    for (int a = 0; a < NACC; ++a)           // this CTA's 128 rows of each 256-column accumulator
                        ptx::tma_load_2d_pair(sa + (1 + a) * kHalf, &tmG, full_bar(slot), ch * 128, b_row + a * 256);
                }
                if (++slot == kBuildSlots) { slot = 0; phase ^= 1u; }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer =====================
        if (rank == 0) {
            constexpr uint32_t idesc = ptx::make_idesc_i8(256, 256);
            const uint32_t dlo0 = ptx::smem_desc_lo(smem_base);
            int slot = 0, buf = 0;
            uint32_t phase = 0, acc_phase = 0;
            BuildCursor cur;
            build_cursor_init(cur, upt, ru_lo);
            bool started = false;
            int ru, cu;
            while (build_next_block(cur, started, pair0, npairs, ru_lo, nru, ncu256, upt, NACC, ru, cu)) {
                ptx::mbar_wait(tempty_bar(buf), acc_phase ^ 1u);
                ptx::tc_fence_after();
                const uint32_t d_tmem = tmem_base + buf * 256 * NACC;
                for (int ch = 0; ch < nch; ++ch) {
                    ptx::mbar_wait(full_bar(slot), phase);
                    ptx::tc_fence_after();
                    if (ptx::elect_one()) {
                        const uint32_t a = dlo0 + slot * (kBuildSlotBytes >> 4);
#pragma unroll
                        for (int c = 0; c < NACC; ++c) {
                            const uint32_t b = a + (1 + c) * (kHalf >> 4);
#pragma unroll
                            for (int kk = 0; kk < 4; ++kk)         // 4 x K = 32 per 128-byte row
                                ptx::mma_i8_ss_pair(d_tmem + c * 256, ptx::smem_desc_from_lo(a + 2 * kk), ptx::smem_desc_from_lo(b + 2 * kk),
                                                    idesc, (ch > 0 || kk > 0) ? 1u : 0u);
                        }
                        ptx::tc_commit_pair(empty_bar(slot));
                    }
                    if (++slot == kBuildSlots) { slot = 0; phase ^= 1u; }
                }
                if (ptx::elect_one()) ptx::tc_commit_pair(tfull_bar(buf));
                if (++buf == NBUF) { buf = 0; acc_phase ^= 1u; }
            }
        }
    } else {
        // ===================== epilogue: d2 = s_i + s_j - 2 <g_i, g_j>, exp, store =====================
        const int ew = warp - 2, q = warp & 3, hf = ew >> 2;          // TMEM lanes 32q.., columns 128 hf ..
        int buf = 0;
        uint32_t acc_phase = 0;
        BuildCursor cur;
        build_cursor_init(cur, upt, ru_lo);
        bool started = false;
        int ru, cu;
        while (build_next_block(cur, started, pair0, npairs, ru_lo, nru, ncu256, upt, NACC, ru, cu)) {
            const int64_t gi = static_cast<int64_t>(ru) * 256 + rank * kBlk + q * 32 + lane;       // my row of A
            const int si = op.sq_row[gi];
            const int ti = op.rect ? 0x7fffffff : static_cast<int>(gi / op.nb);
            double ssq = 0.0;                       // this thread's share of the block's sum of squares / maximum
            float amx = 0.0f;
            float ci[kMaxConfounders];
#pragma unroll
            for (int c = 0; c < kMaxConfounders; ++c) ci[c] = (c < op.q) ? __ldg(op.C_row + gi * op.ldc_row + c) : 0.0f;
            ptx::mbar_wait(tfull_bar(buf), acc_phase);
            ptx::tc_fence_after();
#pragma unroll 1
            for (int part = 0; part < 4 * NACC; ++part) {
                const int col = (part >> 2) * 256 + hf * 128 + (part & 3) * 32;                     // column inside the block
                const int64_t gj0 = static_cast<int64_t>(cu) * 256 * NACC + col;                    // first column of this part
                uint32_t acc[32];
                ptx::tmem_ld_32x32(tmem_base + buf * 256 * NACC + (static_cast<uint32_t>(q * 32) << 16) + col, acc);
                ptx::tmem_ld_wait();
                if (part == 4 * NACC - 1) {
                    ptx::tc_fence_before();
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive_leader(tempty_bar(buf));          // accumulator is in registers
                }
                const int tj = static_cast<int>(gj0 / op.nb);
                if (tj > ti) continue;                                               // an upper tile: not produced
                float* dst = (op.tiled && !op.rect)
                    ? op.A + (tile_slot(NT, ti, tj) * op.nb + gi % op.nb) * static_cast<int64_t>(op.nb) + gj0 % op.nb
                    : op.A + gi * op.lda + gj0;
#pragma unroll
                for (int e = 0; e < 32; e += 4) {
                    float v[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int d2 = si + __ldg(op.sq + gj0 + e + u) - 2 * static_cast<int>(acc[e + u]);
                        float d2f = static_cast<float>(d2);
                        if (op.q > 0) {
                            const float* cj = op.C + (gj0 + e + u) * op.ldc;      // the same address in every lane
                            float dc = 0.0f;
#pragma unroll
                            for (int c = 0; c < kMaxConfounders; ++c)
                                if (c < op.q) { const float t = ci[c] - __ldg(cj + c); dc = fmaf(t, t, dc); }
                            d2f += dc;
                        }
                        float kv;
                        if (op.linear) {
                            kv = op.gamma * static_cast<float>(static_cast<int>(acc[e + u]));
                            if (!op.rect && gj0 + e + u == gi) kv += op.lambda;
                        } else {
                            kv = op.ibs ? __fdiv_rn(op.alleles - d2f, op.alleles) : expf(-op.gamma * d2f);
                            if (!op.rect && gj0 + e + u == gi) kv = op.diag;
                        }
                        if (!op.rect && (gi >= op.n_valid || gj0 + e + u >= op.n_valid)) kv = (gj0 + e + u == gi) ? 1.0f : 0.0f;
                        v[u] = kv;
                        ssq += static_cast<double>(kv) * kv;
                        amx = fmaxf(amx, fabsf(kv));
                    }
                    *reinterpret_cast<float4*>(dst + e) = make_float4(v[0], v[1], v[2], v[3]);
                }
            }
            if (op.stat_sumsq != nullptr && !op.rect) {
                // fixed-order warp reduction, one partial per (block of the tile, CTA of the pair, epilogue warp)
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    ssq += __shfl_xor_sync(0xffffffffu, ssq, o);
                    amx = fmaxf(amx, __shfl_xor_sync(0xffffffffu, amx, o));
                }
                if (lane == 0) {
                    const int tj = static_cast<int>(static_cast<int64_t>(cu) * 256 * NACC / op.nb);
                    if (tj <= ti) {
                        const int upt_ = op.nb / 256, cpt = upt_ / NACC;                 // row / column units per tile
                        const int bit = (ru % upt_) * cpt + (cu % cpt);                   // block inside the tile
                        const int64_t idx = tile_slot(NT, ti, tj) * op.stats_chunks + bit * 16 + rank * 8 + ew;
                        op.stat_sumsq[idx] = ssq;
                        op.stat_amax[idx] = amx;
                    }
                }
            }
            if (++buf == NBUF) { buf = 0; acc_phase ^= 1u; }
        }
    }
    ptx::tc_fence_before();
    ptx::cluster_sync_all();
    if (warp == 1) ptx::tmem_dealloc<512, 2>(tmem_base);
}

// P = K W (Alg. 4 l.6): K m x n FP32 row-major (ldk, n % 4 == 0, 16-byte aligned rows), W n x nrhs
// row-major (ldw), P m x nrhs (ldp).  Lane = right-hand side r (NRP = nrhs rounded up to 8 / 16 / 32; 32 / NRP
// groups of lanes per warp), every group owns 4 rows of K: per 4 columns a group reads 4 float4 of K (the same
// address in all its lanes) and 4 coalesced rows of W, each reused by the 4 rows.  Every (row, r) sum runs over
// the columns in order in four interleaved partial sums -- a fixed order, no reduction across lanes.  Bound by
// the read of K from HBM.
template <int NRP>
__global__ void __launch_bounds__(256)
predict_kw_kernel(const float* __restrict__ K, int64_t m, int64_t n, int64_t ldk, const float* __restrict__ W, int64_t ldw,
                  int nrhs, float* __restrict__ P, int64_t ldp) {
    constexpr int GROUPS = 32 / NRP, ROWS = 4;
    const int lane = threadIdx.x & 31, g = lane / NRP, r = lane % NRP;
    const int64_t warp = static_cast<int64_t>(blockIdx.x) * 8 + (threadIdx.x >> 5);
    const int64_t row0 = (warp * GROUPS + g) * ROWS;
    if (row0 >= m) return;
    const bool active = r < nrhs;
    float acc[ROWS][4];
#pragma unroll
    for (int i = 0; i < ROWS; ++i)
#pragma unroll
        for (int u = 0; u < 4; ++u) acc[i][u] = 0.0f;
    const float* k0 = K + row0 * ldk;
    for (int64_t j = 0; j < n; j += 4) {
        float w[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) w[u] = active ? __ldg(W + (j + u) * ldw + r) : 0.0f;
#pragma unroll
        for (int i = 0; i < ROWS; ++i) {
            const float4 kv = (row0 + i < m) ? __ldg(reinterpret_cast<const float4*>(k0 + i * ldk + j)) : make_float4(0.f, 0.f, 0.f, 0.f);
            acc[i][0] = fmaf(kv.x, w[0], acc[i][0]);
            acc[i][1] = fmaf(kv.y, w[1], acc[i][1]);
            acc[i][2] = fmaf(kv.z, w[2], acc[i][2]);
            acc[i][3] = fmaf(kv.w, w[3], acc[i][3]);
        }
    }
    if (active)
#pragma unroll
        for (int i = 0; i < ROWS; ++i)
            if (row0 + i < m) P[(row0 + i) * ldp + r] = (acc[i][0] + acc[i][1]) + (acc[i][2] + acc[i][3]);
}

// ---- the FP32 tiles of the mixed SYRK of ridge regression (Fig. 2) ----
// X = [S^T | C]: the SNP features are the int8 rows of S (N_S x patients, the matrix the INT8 kernel above works on),
// the q confounder features the columns of C (patients x q, FP32).  The INT8 kernel has produced the SNP x SNP block;
// this kernel writes the q rows ns .. ns+q-1 of X^T X + lambda I: for every column j <= row,
//     A(ns + t, j) = sum_k x_j[k] * C[k][t],   x_j = row j of S (j < ns) or column j - ns of C,
// in FP32 (the paper's SGEMM tiles), sums in a fixed order (lane-strided partial sums, then a shuffle tree).  Inside
// the diagonal tile the mirrored element is written too (diagonal tiles are full squares).
// HBM: S is read once (ns * p bytes); C (p * q * 4 bytes) stays in L2 and is staged through shared memory.
constexpr int kRrWarps = 8, kRrRowsPerWarp = 4, kRrKc = 128;

__global__ void __launch_bounds__(kRrWarps * 32)
rr_confounder_rows_kernel(const int8_t* __restrict__ S, int64_t lds, int64_t ns, int64_t p, const float* __restrict__ C,
                          int64_t ldc, int q, float lambda, float* __restrict__ A, int64_t lda, int tiled, int nb, int NT) {
    __shared__ float Cs[kRrKc][kMaxConfounders + 1];                      // + 1: lanes read different rows, conflict-free
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int64_t j0 = (static_cast<int64_t>(blockIdx.x) * kRrWarps + warp) * kRrRowsPerWarp;     // this warp's columns j0 .. j0+3
    const int64_t ncol = ns + q;
    float acc[kRrRowsPerWarp][kMaxConfounders];
#pragma unroll
    for (int r = 0; r < kRrRowsPerWarp; ++r)
#pragma unroll
        for (int t = 0; t < kMaxConfounders; ++t) acc[r][t] = 0.0f;

    for (int64_t k0 = 0; k0 < p; k0 += kRrKc) {
        __syncthreads();
        for (int e = threadIdx.x; e < kRrKc * kMaxConfounders; e += kRrWarps * 32) {
            const int kk = e / kMaxConfounders, t = e % kMaxConfounders;
            Cs[kk][t] = (k0 + kk < p && t < q) ? __ldg(C + (k0 + kk) * ldc + t) : 0.0f;
        }
        __syncthreads();
#pragma unroll
        for (int u = 0; u < kRrKc / 32; ++u) {
            const int kk = u * 32 + lane;                                   // consecutive lanes, consecutive patients
            const int64_t k = k0 + kk;
            float x[kRrRowsPerWarp];
#pragma unroll
            for (int r = 0; r < kRrRowsPerWarp; ++r) {
                const int64_t j = j0 + r;
                x[r] = 0.0f;
                if (k < p && j < ncol) x[r] = j < ns ? static_cast<float>(S[j * lds + k]) : Cs[kk][j - ns];
            }
#pragma unroll
            for (int t = 0; t < kMaxConfounders; ++t) {
                const float c = Cs[kk][t];
#pragma unroll
                for (int r = 0; r < kRrRowsPerWarp; ++r) acc[r][t] = fmaf(x[r], c, acc[r][t]);
            }
        }
    }
#pragma unroll
    for (int r = 0; r < kRrRowsPerWarp; ++r)
#pragma unroll
        for (int t = 0; t < kMaxConfounders; ++t) {
            float v = acc[r][t];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            acc[r][t] = v;
        }
    if (lane == 0) {
        for (int r = 0; r < kRrRowsPerWarp; ++r) {
            const int64_t j = j0 + r;
            if (j >= ncol) continue;
            for (int t = 0; t < q; ++t) {
                const int64_t row = ns + t;
                if (j > row) continue;                                       // the upper triangle follows by symmetry
                const float v = acc[r][t] + (j == row ? lambda : 0.0f);
                const int ti = static_cast<int>(row / nb), tj = static_cast<int>(j / nb);
                if (tiled) {
                    float* T = A + tile_slot(NT, ti, tj) * static_cast<int64_t>(nb) * nb;
                    T[(row % nb) * nb + j % nb] = v;
                    if (ti == tj) T[(j % nb) * nb + row % nb] = v;
                } else {
                    A[row * lda + j] = v;
                    if (ti == tj) A[j * lda + row] = v;
                }
            }
        }
    }
}

}  // namespace krr

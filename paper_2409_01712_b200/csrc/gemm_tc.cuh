// Tensor-core update kernel of the tile Cholesky.
//
// One warp-specialised, persistent tcgen05 kernel serves the three contraction shapes of a tile
// column k (all "C = base - A * B^T" with K-major FP16 operand images, FP32 accumulation in TMEM):
//
//   MODE_UPDATE  S_ik = rd_p(A_ik) - sum_{s<k} L_is L_ks^T      for every tile i >= k   (SYRK+GEMM)
//   MODE_P1      S[:, c] -= X[:, 0:c] X[c, 0:c]^T               inside the panel (sub-blocks of 128)
//   MODE_P3      X[:, c]  = S[:, c] * inv(L_cc)^T               the TRSM as a product with the
//                                                               inverted 128x128 diagonal block
//
// Operand images ("planes"): every value x that feeds the tensor cores is kept as FP16 hi = rn(s*x)
// and, for FP32-class tiles, lo = rn(s*x - hi), with a global power-of-two scale s that lifts the
// data into the upper FP16 binades (sx = 2^14 / 2^ceil(log2 sqrt(max diag A)) for L and X values,
// ss likewise for Schur-complement values) -- without it lo falls into the FP16 subnormals and the
// split keeps only ~17 bits.  The accumulator is rescaled by the exact inverse in the epilogue.
// An FP32 x FP32 term issues three kind::f16 MMAs (hi*hi + lo*hi + hi*lo), FP32 x {FP16,FP8} two, {FP16,FP8} x {FP16,FP8} one (the hi plane of a
// low-precision tile holds its stored value exactly).  Accumulators never leave TMEM until the
// tile's whole K range is done ("round once", R4).
//
// FP8 x FP8 terms (both operand tiles stored as E4M3 with power-of-two tile scales) run as
// kind::mxf8f6f4.block_scale MMAs on the 1-byte images (Qp plane, K = 128 per 16 KB smem block): the
// per-tile scale times the plane scale sx is a power of two, i.e. a UE8M0 block scale that is the same
// for every row and every K block of the tile.  TMEM columns 256.. hold a table of constant scale
// vectors (entry j: every byte = sf_bias + j); an MMA just points its scale operands at the two
// entries of its tiles, so no scale data is ever staged.  Tiles whose exponent falls outside the
// table (never seen on the workloads) take the FP16 path through their hi image, which is exact too.
//
// Shared-memory ring: 6 slots of 32 KB = [one 16 KB block of A | one of B].  A K chunk of an
// FP16-class or FP8 term occupies one slot, of an FP32-class term two (hi images, then lo images), so
// the low-precision classes -- whose MMAs consume a slot in a quarter of the time -- get a six-deep
// prefetch, the FP32 class three.
//
// Accumulation order: the tensor core adds each MMA's result to the TMEM accumulator with
// truncation, a bias of ~half an ulp OF THE ACCUMULATOR per instruction (measured: backward error
// growing linearly in n when K is walked upwards).  In a Cholesky update the leading columns of L
// carry almost all of sum_k L_ik L_jk, so K is walked DOWNWARDS: the accumulator stays small until
// the dominant terms arrive last, and the bias stays at the FP32 noise level.
#pragma once
#include "common.cuh"
#include "ptx.cuh"
#include "tri128.cuh"

namespace krr {

enum { MODE_UPDATE = 0, MODE_P1 = 1, MODE_P3 = 2, MODE_TRSM = 3, MODE_DIAG = 4, MODE_POTRF = 5 /* item of MODE_DIAG */,
       MODE_INV = 6 };

// Scratch planes (hi / lo FP16 images, row pitch nb, one tensor map each): rows [0, n) hold the Schur complement S of
// the panel rows below the diagonal tile (panel-local row index), then two sets (tile-column parity) of three nb x nb
// areas: M = inv(L_kk), its transpose MT, and the intermediate U of the inverse's recursion.
struct InvNode { int o, hl, hr; };   // MODE_INV: left blocks [o, o + hl), right blocks [o + hl, o + hl + hr) of the diagonal tile

struct GemmOp {
    int mode;
    int nb, NT, k;        // tile size, tiles per dimension, tile column being produced
    int s_lo, s_hi;       // MODE_UPDATE: tile columns s in [s_lo, s_hi) are accumulated (lookahead splits
                          // the sum into the part known early and the newest column)
    int base_w;           // MODE_UPDATE: 0 = start from rd_p(A), 1 = continue the FP32 partial sum in W
    int planes;           // MODE_UPDATE: 1 = also write the FP16 hi/lo images of the result (final pass)
    int c;                // 128-wide sub-column inside the tile column (P1 / P3)
    int rb0, nrb;         // output row blocks (128 rows, panel-local: row 0 = top of tile (k,k))
    int cb0, ncb;         // output column blocks (128 columns inside the tile column)
    int64_t prow0;        // plane row of panel-local row 0  (= tile_slot(k,k) * nb)
    const uint8_t* map;   // device precision map (NT*NT)
    AView A;              // input matrix (MODE_UPDATE base)
    const float* a_amax;  // NT*NT max|A_ij| (FP8 pre-rounding of A), may be null
    float* W;             // panel workspace, FP32 [m][nb]
    __half* Hp;           // hi plane  [nslots*nb][nb]
    __half* Lp;           // lo plane: FP32 tiles only, compact (row of tile (i,j) = lrow[i*NT+j], -1 for other tiles)
    const int* lrow;      // device int[NT*NT]
    const int* qrow;      // device int[NT*NT]: first row of the E4M3 image of tile (i,j) in the Qp plane (FP8 tiles only), else -1
    int64_t prow0_lo;     // lo-plane row of panel-local row 0 of the diagonal tile (k,k) (= lrow[k*NT+k], known to the host)
    float* tile_amax;     // per-slot max|X| accumulated by MODE_P3
    const float* scales;  // NT*NT tile scales of the mosaic (FP8 tiles), written by finalize_kernel
    int fp8q;             // MODE_UPDATE: FP8 x FP8 terms may use the E4M3 images (Qp plane exists)
    const float* scl;     // device: power-of-two plane scales and accumulator rescalings (common.cuh SCL_*)
    const float* dscale;  // device float[NT]: the equilibration d_I of the tile rows (panel.cuh equilibrate_kernel)
    const float* linv_scale;  // device float[nb/128]: scale of each inverted diagonal block's planes
    unsigned flags;
    // MODE_DIAG (fused diagonal-tile chain): outputs of the in-kernel POTRF of 128-blocks and the cross-CTA progress
    int* prog;                // nb/128 ints, zero at launch: prog[r] = completed items of the CTA of row block r
    __half* linv_hi;          // inverted diagonal blocks, hi / lo FP16 planes [nb][128]
    __half* linv_lo;
    float* linv_scale_w;      // = linv_scale, writable
    int* info;                // krr_potrf_mp's d_info
    int64_t col_base;         // 1-based global index of the tile column's first scalar column
    // MODE_UPDATE with sk = 1 (K-split of the last, partial wave: see next_item): sk_flags[unit] counts the CTAs of a unit
    // that have stored the partial sum of their tail item (zero at launch), sk_partial holds one output block per unit.
    int sk;
    int* sk_flags;
    float* sk_partial;
    // scratch planes and the quantising store of MODE_TRSM (X = S inv(L_kk)^T, straight into the mosaic)
    __half* Sh;               // scratch hi plane [n + 6 nb][nb]
    __half* Sl;               // scratch lo plane
    int64_t srow_m, srow_mt, srow_u;   // scratch rows of M, M^T and U of this tile column (parity set)
    const int64_t* off;       // byte offsets of the mosaic tiles
    uint8_t* factor;          // the mosaic
    // MODE_INV: one step of one level of the recursion M21 = -M22 L21 M11 (step 0: U^T = M11^T L21^T; step 1: M21 and M21^T)
    int inv_step, inv_last;   // inv_last: the root level, whose M21^T is not needed
    InvNode node;             // (scalars: a dynamically indexed array in the kernel parameters would be copied to local memory)
};



constexpr int kSlots = 6;                          // shared-memory ring: 6 slots of [A block | B block]
constexpr int kBlockK = 64;                        // fp16 elements per 128-byte swizzle row
constexpr int kPlaneBytes = kBlk * kBlockK * 2;    // one 128 x 64 fp16 (or 128 x 128 E4M3) operand block = 16 KB
constexpr int kSlotBytes = 2 * kPlaneBytes;        // one plane of A and one of B.  A K chunk takes one slot
                                                   // (hi images / E4M3 images) or two (hi, then lo images)
constexpr int kAccCols = 128;                      // TMEM columns of one 128x128 FP32 accumulator
constexpr int kMaxAccBufs = 4;                     // CG = 1: four 128-column accumulators; CG = 2: two of 256 columns
constexpr int kSegChunks = 2;                      // MODE_TRSM / MODE_INV: K chunks (of 64) per accumulation segment
constexpr int kSfCol0 = 256;                       // first TMEM column of the scale table
constexpr int kSfCols = 256;                       // table: 256 / (4 CG) entries of 4 CG columns
constexpr int kTmemCols = 512;                     // accumulators + scale table
// entry j <-> UE8M0 byte sf_bias + j: CG = 1: 64 entries, 2^-40 .. 2^23; CG = 2: 32 entries, 2^-24 .. 2^7
__host__ __device__ constexpr int sf_entries(int cg) { return kSfCols / (4 * cg); }
__host__ __device__ constexpr int sf_bias(int cg) { return cg == 1 ? 127 - 40 : 127 - 24; }
constexpr int kGemmThreads = 320;                  // warp 0 TMA, warp 1 MMA (+TMEM alloc), 2-9 epilogue
constexpr int kEpiWarps = 8;
constexpr int kEpiRowBytes = 80;                   // 64 B of FP16 per row + 16 B pad (conflict-free 16 B accesses)
constexpr int kEpiStageBytes = 32 * kEpiRowBytes;  // per-warp transpose buffer
constexpr int kGemmSmem = kSlots * kSlotBytes + 1024 /*align*/ + 256 /*barriers*/ + kEpiWarps * kEpiStageBytes;

// One term of an output block's sum = one tile product (MODE_UPDATE) or the single in-panel product.
// Geometry (plane rows / first K column / K extent) is arithmetic on launch parameters and block
// indices -- warp-uniform by construction.  The MMA class of the term comes from the device-resident
// map and tile scales; it is fetched as one packed word and made provably uniform with a warp
// reduction (REDUX writes a uniform register), so that the issue loops below compile to uniform-
// datapath code around the single elected lane that issues TMA / tcgen05 instructions.
struct TermGeom {
    int a_row, b_row;       // plane rows (TMA coordinate 1) in the hi planes
    int a_row_lo, b_row_lo; // ... in the lo planes (the compact Lp for factor tiles; the same rows elsewhere)
    int a_row_q, b_row_q;   // ... in the E4M3 plane (MODE_UPDATE, FP8 tiles)
    int a_k0, b_k0;         // first K column (TMA coordinate 0)
    int kelems;             // K extent in elements
    int a_src, b_src;       // operand planes: 0 = factor / panel images (tmH, tmL), 1 = inverted 128-blocks (tmIH, tmIL),
                            // 2 = scratch (tmSH, tmSL)
};

// class word: bit 0: A operand has a lo image (FP32 tile), bit 1: B has one, bit 2: FP8 x FP8 term on the
// E4M3 images (K chunks of 128, block-scaled MMA), bits 8-13 / 16-21: scale-table entries of the two tiles
constexpr uint32_t kClsALo = 1u, kClsBLo = 2u, kClsQ = 4u;

// UE8M0 byte of the power of two x (> 0, normal): its biased exponent.
__device__ __forceinline__ int pow2_exponent_byte(float x) { return static_cast<int>((__float_as_uint(x) >> 23) & 0xffu); }

// rb: this CTA's output row block; cb: the column block whose B rows this CTA stages; cb_first: first column block of
// the unit's output block (MODE_TRSM: the K range ends with the unit's last column block, M being lower triangular)
__device__ __forceinline__ TermGeom term_geom(const GemmOp& op, int mode, int c, int s /* term index */, int rb, int cb, int cb_first,
                                              int cg) {
    TermGeom t;
    t.a_src = 0; t.b_src = 0;
    if (mode == MODE_UPDATE) {
        const int i = op.k + (rb * kBlk) / op.nb;
        const int subrow = (rb * kBlk) % op.nb;
        s += op.s_lo;
        t.a_row = static_cast<int>(tile_slot(op.NT, i, s) * op.nb + subrow);
        t.b_row = static_cast<int>(tile_slot(op.NT, op.k, s) * op.nb + cb * kBlk);
        // (the tables answer -1 for tiles without that image; the class word keeps such a row from ever being loaded)
        t.a_row_lo = op.lrow[i * op.NT + s] + subrow;
        t.b_row_lo = op.lrow[op.k * op.NT + s] + cb * kBlk;
        t.a_row_q = op.qrow[i * op.NT + s] + subrow;
        t.b_row_q = op.qrow[op.k * op.NT + s] + cb * kBlk;
        t.a_k0 = 0;
        t.b_k0 = 0;
        t.kelems = op.nb;
        return t;
    } else if (mode == MODE_P1) {
        t.a_row = static_cast<int>(op.prow0) + rb * kBlk;
        t.b_row = static_cast<int>(op.prow0) + c * kBlk;
        t.a_k0 = 0;
        t.b_k0 = 0;
        t.kelems = c * kBlk;
    } else if (mode == MODE_TRSM) {
        // X[rb, cb] = sum_{j <= cb} S[rb, j] M[cb, j]^T : A = S of the panel row block (scratch), B = rows of M (scratch)
        t.a_src = 2; t.b_src = 2;
        t.a_row = rb * kBlk;
        t.b_row = static_cast<int>(op.srow_m) + cb * kBlk;
        t.a_k0 = 0;
        t.b_k0 = 0;
        t.kelems = (cb_first + cg) * kBlk < op.nb ? (cb_first + cg) * kBlk : op.nb;
    } else {
        t.a_row = static_cast<int>(op.prow0) + rb * kBlk;
        t.b_row = c * kBlk;                                // row in the Linv planes
        t.b_src = 1;
        t.a_k0 = c * kBlk;
        t.b_k0 = 0;
        t.kelems = kBlk;
    }
    // rows of the diagonal tile in the (compact) lo plane; the scratch and inverse planes index hi and lo alike
    t.a_row_lo = (t.a_src == 0) ? t.a_row - static_cast<int>(op.prow0) + static_cast<int>(op.prow0_lo) : t.a_row;
    t.b_row_lo = (t.b_src == 0) ? t.b_row - static_cast<int>(op.prow0) + static_cast<int>(op.prow0_lo) : t.b_row;
    t.a_row_q = t.b_row_q = 0;
    return t;
}

template <int CG>
__device__ __forceinline__ uint32_t term_class_load(const GemmOp& op, int mode, int s /* term index */, int rb) {
    // (MODE_TRSM: a one-pass product -- hi images only -- for tiles that will be stored as E4M3 was tried in r02: three
    // times faster, backward error unchanged, but the perturbation of 2^-11 flips enough E4M3 roundings to take the
    // literal difference from the emulated oracle from 4e-5 to 1.5e-3 on a random mosaic: dropped, every tile keeps
    // the 22-bit product)
    if (mode != MODE_UPDATE) return kClsALo | kClsBLo;
    const int i = op.k + (rb * kBlk) / op.nb;
    s += op.s_lo;
    const int pa = op.map[i * op.NT + s], pb = op.map[op.k * op.NT + s];
    uint32_t w = (pa == KRR_FP32 ? kClsALo : 0u) | (pb == KRR_FP32 ? kClsBLo : 0u);
    if (op.fp8q && pa == KRR_FP8_E4M3 && pb == KRR_FP8_E4M3) {
        // images are of the equilibrated L~ = d L: value = (sx d s_tile) * code
        const float sx = op.scl[SCL_SX];
        const int sfa = pow2_exponent_byte(sx * op.dscale[i] * op.scales[i * op.NT + s]) - sf_bias(CG);
        const int sfb = pow2_exponent_byte(sx * op.dscale[op.k] * op.scales[op.k * op.NT + s]) - sf_bias(CG);
        if (sfa >= 0 && sfa < sf_entries(CG) && sfb >= 0 && sfb < sf_entries(CG))
            w |= kClsQ | (static_cast<uint32_t>(sfa) << 8) | (static_cast<uint32_t>(sfb) << 16);
    }
    return w;
}
__device__ __forceinline__ uint32_t make_uniform(uint32_t w) { return __reduce_max_sync(0xffffffffu, w); }

__device__ __forceinline__ int num_terms(const GemmOp& op) {
    return op.mode == MODE_UPDATE ? (op.s_hi - op.s_lo) : 1;
}

// Tiles of the diagonal tile that lie entirely above the diagonal are never read: skip them.
__device__ __forceinline__ bool tile_is_skipped(const GemmOp& op, int rb, int cb) {
    return op.mode == MODE_UPDATE && (rb * kBlk) < op.nb && cb > rb;
}

// ---- work items ------------------------------------------------------------------------------------
// The three warp roles of a CTA walk the same sequence of work items, each with its own iterator.
//   MODE_UPDATE / MODE_P1 / MODE_P3 / MODE_TRSM: item = one output block (of a pair: 256 x 256), blocks dealt
//     round-robin over the CTAs (pairs) of the grid.
//   MODE_DIAG (CG = 1, nb/128 co-resident CTAs): the whole chain of the diagonal tile in one launch --
//     the FP32 POTRF of each 128-block runs on the eight epilogue warps of its CTA (tri128.cuh), the
//     products on the tensor cores as elsewhere; CTAs order their items through progress counters in
//     global memory (release: __threadfence + proxy fence + store; acquire: volatile load + fences).
//   MODE_INV (CG = 1): one step of one level of the inverse of the diagonal tile, M = inv(L_kk), by binary
//     splitting of its 128-blocks: for a node with left blocks [o, o + hl) and right blocks [o + hl, o + hl + hr)
//         M21 = -M22 L21 M11,   in two steps whose operands are all K-major as stored:
//         step 0   U^T   = M11^T L21^T          (A = rows of M^T, B = rows of L_kk)
//         step 1   M21   = -M22 U               (A = rows of M,   B = rows of U^T)
//                  M21^T = -U^T M22^T           (A = rows of U^T, B = rows of M)     -- not for the root
//     item = one 128 x 128 block of one of these products; the nodes of a level are independent.
struct WorkItem {
    int mode, c;     // contraction shape (MODE_UPDATE / MODE_P1 / MODE_P3 / MODE_TRSM / MODE_INV) and sub-column
    int rb, cb;      // first output row block / column block (of the pair when CG = 2)
    int dep;         // > 0: reads what the item `dep` places earlier in this CTA's sequence wrote
    int xcta, xneed; // MODE_DIAG: reads what CTA xcta wrote in its first xneed items (xcta < 0: nothing)
    int t_lo, t_hi;  // terms [t_lo, t_hi) of the launch's term range are accumulated by this item
    int sk_role;     // 0: the item holds all terms of its block; 1: it holds the highest terms and finishes the block,
                     // adding the partial sums of sk_nother units (the first items of units sk_other, sk_other + stride ...);
                     // 2: it holds lower terms only and leaves a partial sum for the finisher
    int sk_other, sk_nother, sk_stride;
    TermGeom g;      // MODE_INV: operand geometry of the block
    int o_row, o_col, o_var;   // MODE_INV: scratch row / column of the output block; 0 = U^T, 1 = M21, 2 = M21^T
    // MODE_TRSM / MODE_INV (CG = 1): the K range of a block is accumulated in segments of kSegChunks chunks, each in its
    // own TMEM accumulator, and the segments are added in FP32 (round to nearest) by the epilogue -- see the note on
    // segmented accumulation below.  ch_lo / ch_hi: the item's K chunks (-1: the whole range); first / last segment flags.
    int ch_lo, ch_hi, seg_first, seg_last;
};
struct ItemIter {
    long long u;     // (unused)
    int t;           // block modes: next block index
    int g, it, m;    // MODE_DIAG: item inside the chain; segmented modes: it = segments of block t already emitted
};

// Segmented accumulation.  The tensor core adds every MMA's result to the TMEM accumulator with truncation, a bias of
// about half an ulp OF THE ACCUMULATOR per instruction.  In a trailing update the accumulator stays small until the
// dominant leading columns arrive last (K is walked downwards).  A product with an explicit inverse, X = S M^T, has no
// such order: its partial sums are of the size of |S||M| throughout while the result is a small difference (for the
// first diagonal tile of a kernel matrix 0.5 against 0.02), and a hundred truncations at that size cost a backward
// error of 1.2e-6 (measured, nb = 512).  So these products start a fresh accumulator every kSegChunks K chunks
// (24 instructions) and the epilogue adds the segments in FP32 with round to nearest, highest K first.
__device__ __forceinline__ bool emit_segment(ItemIter& st, int nunits, int kelems, WorkItem& w) {
    const int nch = kelems / kBlockK;
    const int nseg = (nch + kSegChunks - 1) / kSegChunks;
    const int sidx = nseg - 1 - st.it;                 // highest K first
    w.ch_lo = sidx * kSegChunks;
    w.ch_hi = (sidx + 1) * kSegChunks < nch ? (sidx + 1) * kSegChunks : nch;
    w.seg_first = (st.it == 0);
    w.seg_last = (sidx == 0);
    if (w.seg_last) { st.it = 0; st.t += nunits; } else { ++st.it; }
    return true;
}

template <int CG>
__device__ __forceinline__ bool next_item(const GemmOp& op, ItemIter& st, int unit0, int nunits, WorkItem& w) {
    w.xcta = -1; w.xneed = 0;
    w.t_lo = 0; w.t_hi = num_terms(op); w.sk_role = 0; w.sk_other = 0; w.sk_nother = 0; w.sk_stride = 0;
    w.ch_lo = -1; w.ch_hi = -1; w.seg_first = 1; w.seg_last = 1;
    if (op.mode == MODE_DIAG) {
        // CTA r owns row block r of the diagonal tile: P3(0), P1(1), P3(1), ..., P3(r-1), P1(r), POTRF(r).
        // P1(c) reads the rows of block c that CTA c finished with its P3(c-1) (item 2c-2), P3(c) the inverse
        // CTA c's POTRF (item 2c) produced.
        const int r = unit0;
        if (st.it > 2 * r) return false;
        const int it = st.it++;
        w.rb = op.rb0 + r;
        w.dep = it > 0 ? 1 : 0;
        if (it == 2 * r) { w.mode = MODE_POTRF; w.c = r; }
        else if (it & 1) { w.mode = MODE_P1; w.c = (it + 1) >> 1; if (w.c < r) { w.xcta = w.c; w.xneed = 2 * w.c - 1; } }
        else { w.mode = MODE_P3; w.c = it >> 1; w.xcta = w.c; w.xneed = 2 * w.c + 1; }
        w.cb = w.c;
        return true;
    }
    if (op.mode == MODE_INV) {
        // the blocks of the node's products, every block in K segments
        int t = st.t;
        for (int nd = 0; nd < 1; ++nd) {
            const int hl = op.node.hl, hr = op.node.hr, o = op.node.o;
            const int per = hl * hr;
            const int cnt = op.inv_step == 0 ? per : (op.inv_last ? per : 2 * per);
            if (t >= cnt) { t -= cnt; continue; }
            const int var = op.inv_step == 0 ? 0 : 1 + t / per;
            t %= per;
            w.mode = MODE_INV; w.c = 0; w.dep = 0; w.o_var = var;
            w.g.a_k0 = w.g.b_k0 = (var == 0 ? o : o + hl) * kBlk;
            w.g.kelems = (var == 0 ? hl : hr) * kBlk;
            if (var == 0) {              // U^T[m, n] : m over the left blocks, n over the right blocks
                const int mb = t / hr, nbk = t % hr;
                w.g.a_src = 2; w.g.a_row = static_cast<int>(op.srow_mt) + (o + mb) * kBlk;
                w.g.b_src = 0; w.g.b_row = static_cast<int>(op.prow0) + (o + hl + nbk) * kBlk;
                w.o_row = static_cast<int>(op.srow_u) + (o + mb) * kBlk; w.o_col = (o + hl + nbk) * kBlk;
            } else if (var == 1) {       // M21[m, n] : m over the right blocks, n over the left blocks
                const int mb = t / hl, nbk = t % hl;
                w.g.a_src = 2; w.g.a_row = static_cast<int>(op.srow_m) + (o + hl + mb) * kBlk;
                w.g.b_src = 2; w.g.b_row = static_cast<int>(op.srow_u) + (o + nbk) * kBlk;
                w.o_row = static_cast<int>(op.srow_m) + (o + hl + mb) * kBlk; w.o_col = (o + nbk) * kBlk;
            } else {                     // M21^T[m, n] : m over the left blocks, n over the right blocks
                const int mb = t / hr, nbk = t % hr;
                w.g.a_src = 2; w.g.a_row = static_cast<int>(op.srow_u) + (o + mb) * kBlk;
                w.g.b_src = 2; w.g.b_row = static_cast<int>(op.srow_m) + (o + hl + nbk) * kBlk;
                w.o_row = static_cast<int>(op.srow_mt) + (o + mb) * kBlk; w.o_col = (o + hl + nbk) * kBlk;
            }
            w.g.a_row_lo = w.g.a_row;
            w.g.b_row_lo = (w.g.b_src == 0) ? w.g.b_row - static_cast<int>(op.prow0) + static_cast<int>(op.prow0_lo) : w.g.b_row;
            w.g.a_row_q = w.g.b_row_q = 0;
            w.rb = 0; w.cb = 0;
            return emit_segment(st, nunits, w.g.kelems, w);
        }
        return false;
    }
    const int ncbu = op.ncb / CG;
    const int ntiles = (op.nrb / CG) * ncbu;
    if (op.mode == MODE_UPDATE && op.sk) {
        // Whole blocks round-robin (all units walk the terms in step, so a tile of the B operand is read by every unit
        // at the same time and served from L2 once), and the TAIL of the last, partial wave split in K: when the remainder
        // r is at most half the units, each of the r leftover blocks is shared by g = nunits / r units, unit sl of a block
        // accumulating the slice [nt sl / g, nt (sl + 1) / g) of its terms.  The slices below the highest leave their sum in
        // sk_partial; the unit with the highest slice (the smallest contributions) adds them to its accumulator in FP32,
        // descending -- the dominant leading tile columns last -- and stores the block.  Everyone works at the same
        // time, nobody waits for work that has not been issued, and the order of every sum is a function of the launch
        // geometry alone: deterministic.
        // (Tried in r02 and dropped: a full stream-K split -- equal (strip, term) ranges per group of units.  Balanced to
        // a fraction of a percent, but the groups then sit at different terms at any one time, the B operand (tile row k of
        // L) is streamed once per group instead of once per wave, and the kernel turns DRAM-bound: C3 232 -> 279 ms.)
        const int nt = w.t_hi;
        const int q = ntiles / nunits, r = ntiles % nunits;
        int g = (q >= 1 && r > 0 && 2 * r <= nunits && nt >= 2) ? nunits / r : 0;
        if (g > nt) g = nt;
        if (g > 16) g = 16;
        if (g < 2) g = 0;
        while (true) {
            int t;
            if (st.t < q * nunits || g == 0) {
                if (st.t >= ntiles) return false;
                t = st.t;
                st.t += nunits;
                if (g != 0 && st.t >= q * nunits) st.t = ntiles;          // next: the tail item
            } else {
                if (st.it) return false;                                  // (the tail item has been handed out)
                st.it = 1;
                const int b = unit0 / g, sl = unit0 % g;
                if (b >= r) return false;
                t = q * nunits + b;
                w.t_lo = nt * sl / g; w.t_hi = nt * (sl + 1) / g;
                if (sl == g - 1) { w.sk_role = 1; w.sk_other = unit0 - 1; w.sk_stride = -1; w.sk_nother = g - 1; }
                else w.sk_role = 2;
            }
            w.rb = op.rb0 + (t / ncbu) * CG;
            w.cb = op.cb0 + (t % ncbu) * CG;
            if (tile_is_skipped(op, w.rb + CG - 1, w.cb)) { if (w.sk_role) return false; continue; }
            w.mode = op.mode; w.c = op.c; w.dep = 0;
            return true;
        }
    }
    while (st.t < ntiles) {
        const int t = st.t;
        st.t += nunits;
        w.rb = op.rb0 + (t / ncbu) * CG;
        w.cb = op.cb0 + (t % ncbu) * CG;
        if (tile_is_skipped(op, w.rb + CG - 1, w.cb)) continue;      // the whole (pair) block lies above the diagonal
        w.mode = op.mode; w.c = op.c; w.dep = 0;
        if (CG == 1 && op.mode == MODE_TRSM) {
            st.t = t;                                                 // (emit_segment advances to the next block after the last segment)
            return emit_segment(st, nunits, ((w.cb + 1) * kBlk < op.nb ? (w.cb + 1) * kBlk : op.nb), w);
        }
        return true;
    }
    return false;
}

// ---- epilogue store helpers (free functions, forced inline: every array stays in registers) --------------------------
// One 32-row x 64-byte part of a warp's sub-block: s0..s3 are this lane's 64 bytes (its row); the rows go through the
// warp's staging buffer so that every store instruction writes 8 full 64-byte row segments.  dst = address of row 0 of
// the part, pitch in bytes.
__device__ __forceinline__ void epi_store_part(uint8_t* stg, int lane, uint4 s0, uint4 s1, uint4 s2, uint4 s3, uint8_t* dst, int64_t pitch) {
    __syncwarp();                                   // previous part has been read out
    *reinterpret_cast<uint4*>(stg + lane * kEpiRowBytes + 0) = s0;
    *reinterpret_cast<uint4*>(stg + lane * kEpiRowBytes + 16) = s1;
    *reinterpret_cast<uint4*>(stg + lane * kEpiRowBytes + 32) = s2;
    *reinterpret_cast<uint4*>(stg + lane * kEpiRowBytes + 48) = s3;
    __syncwarp();
#pragma unroll
    for (int it = 0; it < 4; ++it) {
        const int rr = it * 8 + (lane >> 2), ch = lane & 3;
        const uint4 v = *reinterpret_cast<const uint4*>(stg + rr * kEpiRowBytes + ch * 16);
        *reinterpret_cast<uint4*>(dst + rr * pitch + ch * 16) = v;
    }
}
__device__ __forceinline__ uint32_t epi_pack2(float a, float b) {      // two FP16 roundings in one word (a in the low half)
    const __half2 h = __floats2half2_rn(a, b);
    return *reinterpret_cast<const uint32_t*>(&h);
}
// hi (and lo, if lo_plane) FP16 images of out[0..63] * mul: rows prow.. (lo plane: prow_lo..), columns col.. of planes
// with row pitch nb.  Returns the largest |image value| of this lane (range check of the inverse's planes).
__device__ __forceinline__ float epi_store_images(uint8_t* stg, int lane, const float (&out)[64], float mul, __half* hi_plane,
                                                  __half* lo_plane, int64_t prow, int64_t prow_lo, int col, int nb) {
    float big = 0.0f;
#pragma unroll
    for (int part = 0; part < 4; ++part) {             // (columns 0-31 hi, lo, columns 32-63 hi, lo)
        const int jj = part >> 1;
        const bool is_lo = part & 1;
        if (is_lo && lo_plane == nullptr) continue;
        uint32_t wds[16];
#pragma unroll
        for (int t = 0; t < 16; ++t) {
            const float x0 = out[jj * 32 + 2 * t] * mul, x1 = out[jj * 32 + 2 * t + 1] * mul;
            if (!is_lo) {
                big = fmaxf(big, fmaxf(fabsf(x0), fabsf(x1)));
                wds[t] = epi_pack2(x0, x1);
            } else {
                wds[t] = epi_pack2(x0 - __half2float(__float2half_rn(x0)), x1 - __half2float(__float2half_rn(x1)));
            }
        }
        __half* plane = is_lo ? lo_plane : hi_plane;
        epi_store_part(stg, lane, make_uint4(wds[0], wds[1], wds[2], wds[3]), make_uint4(wds[4], wds[5], wds[6], wds[7]),
                       make_uint4(wds[8], wds[9], wds[10], wds[11]), make_uint4(wds[12], wds[13], wds[14], wds[15]),
                       reinterpret_cast<uint8_t*>(plane + (is_lo ? prow_lo : prow) * nb + col + jj * 32), static_cast<int64_t>(nb) * 2);
    }
    return big;
}

// CG = 1: one CTA per 128x128 output block.  CG = 2 (MODE_UPDATE only): a CTA pair (cluster of 2,
// tcgen05 cta_group::2) per 256x256 block -- each CTA stages its own 128 rows of A and the 128 rows of
// B of ONE of the two column blocks, the leader issues M = 256, N = 256 MMAs that read both CTAs'
// shared memory, and each CTA's TMEM receives its own 128 rows x 256 columns of the accumulator.  Two
// such buffers fill the 512 TMEM columns; when the map holds FP8 tiles the upper 256 columns carry the
// scale table instead and the pair works with a single accumulator (the epilogue of a block is then
// not overlapped with the next block's MMAs: a few % at the K depths of a trailing update).
// Per flop a pair moves half the operand bytes of CG = 1.
template <int CG>
__global__ void __launch_bounds__(kGemmThreads, 1)
gemm_tc_kernel(const __grid_constant__ CUtensorMap tmH, const __grid_constant__ CUtensorMap tmL,
               const __grid_constant__ CUtensorMap tmIH, const __grid_constant__ CUtensorMap tmIL,
               const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmSH,
               const __grid_constant__ CUtensorMap tmSL, const GemmOp op) {
    // tmH / tmL: hi / lo FP16 images of the factor and panel; tmIH / tmIL: the inverted 128-blocks of the diagonal
    // tile (B operand of MODE_P3); tmSH / tmSL: the scratch planes (S of the panel rows, M = inv(L_kk), M^T, U);
    // tmQ: E4M3 images.
    constexpr uint32_t SB = kSlotBytes;                 // [A block 16 KB | B block 16 KB]
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar_base = smem_base + kSlots * kSlotBytes;
    // barriers: full[8], empty[8], tmem_full[2], tmem_empty[2], tmem ptr
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (8 + s); };
    auto tfull_bar = [&](int b) { return bar_base + 8u * (16 + b); };
    auto tempty_bar = [&](int b) { return bar_base + 8u * (16 + kMaxAccBufs + b); };
    const uint32_t tmem_slot = bar_base + 8u * (16 + 2 * kMaxAccBufs);
    uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - ptx::smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const int rank = (CG == 2) ? static_cast<int>(ptx::cluster_ctarank()) : 0;
    const int unit0 = (CG == 2) ? static_cast<int>(blockIdx.x >> 1) : static_cast<int>(blockIdx.x);   // pair / CTA index
    const int nunits = (CG == 2) ? static_cast<int>(gridDim.x >> 1) : static_cast<int>(gridDim.x);
    constexpr int kAccW = kAccCols * CG;                // accumulator columns per buffer
    const int nterms = num_terms(op);
    const bool use_sf = op.fp8q && op.mode == MODE_UPDATE;
    // a pair's 256-column accumulators fill TMEM: with the scale table present there is room for one only
    // MODE_TRSM on pairs keeps the small cross terms (lo * hi, hi * lo) in the second accumulator: the main one then
    // sees a third of the truncating additions (see the note on segmented accumulation), and the epilogue adds the two
    const bool split_cross = (CG == 2) && op.mode == MODE_TRSM;
    const int nbufs = (CG == 2) ? ((use_sf || split_cross) ? 1 : 2) : (use_sf ? 2 : 4);

    const bool has_acc = (op.mode != MODE_UPDATE) ? (op.mode != MODE_P1 || op.c > 0) : (nterms > 0);
    const bool write_planes = (op.mode != MODE_UPDATE) || op.planes;
    // Completion of this CTA's items, counted PER ITEM: slot q % 8 receives one arrival from every epilogue warp when it
    // has stored its share of item q (items q, q + 8, ... share a slot: item q is complete when the slot holds
    // 8 (q / 8 + 1); an epilogue warp is never more than the number of TMEM buffers ahead of another, so slots cannot
    // alias).  A single running total would not do: a fast warp's arrival for item q + 1 could stand in for a slow
    // warp's missing arrival for item q.
    volatile int* item_ctr = reinterpret_cast<volatile int*>(tmem_slot_ptr + 2);
    auto item_complete_count = [](int q) { return kEpiWarps * (q / 8 + 1); };
    int* split_ctr = reinterpret_cast<int*>(tmem_slot_ptr + 10);     // arrivals for this CTA's (single) split block

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tmap(&tmH);
        ptx::prefetch_tmap(&tmL);
        if (op.mode == MODE_P3 || op.mode == MODE_DIAG) { ptx::prefetch_tmap(&tmIH); ptx::prefetch_tmap(&tmIL); }
        if (op.mode == MODE_TRSM || op.mode == MODE_INV) { ptx::prefetch_tmap(&tmSH); ptx::prefetch_tmap(&tmSL); }
        if (op.fp8q) ptx::prefetch_tmap(&tmQ);
        for (int s = 0; s < kSlots; ++s) {
            ptx::mbar_init(full_bar(s), 1);
            ptx::mbar_init(empty_bar(s), 1);
        }
        for (int b = 0; b < kMaxAccBufs; ++b) {
            ptx::mbar_init(tfull_bar(b), 1);
            ptx::mbar_init(tempty_bar(b), kEpiWarps * CG);
        }
        for (int i = 0; i < 8; ++i) item_ctr[i] = 0;
        *split_ctr = 0;
        ptx::fence_mbar_init();
    }
    if (warp == 1) {
        ptx::tmem_alloc<kTmemCols, CG>(tmem_slot);
        ptx::tmem_relinquish<CG>();
    }
    ptx::tc_fence_before();
    if (CG == 2) ptx::cluster_sync_all(); else __syncthreads();     // peer barriers are initialised too
    ptx::tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;
    if (use_sf) {
        // scale table: entry j = 4 CG TMEM columns whose every byte is the UE8M0 code sf_bias + j (an MMA
        // of a pair reads the scales of its 256 B rows from 8 columns, of its 128 A rows from 4)
        if (warp >= 2 && warp < 6) {
            const uint32_t lane_base = static_cast<uint32_t>((warp & 3) * 32) << 16;
            for (int j = 0; j < kSfCols / 4; ++j)
                ptx::tmem_st_32x32_x4(tmem_base + lane_base + kSfCol0 + 4 * j,
                                      static_cast<uint32_t>(sf_bias(CG) + j / CG) * 0x01010101u);
            ptx::tmem_st_wait();
        }
        ptx::tc_fence_before();
        if (CG == 2) ptx::cluster_sync_all(); else __syncthreads();     // the leader's MMAs read both tables
        ptx::tc_fence_after();
    }

    if (warp == 0) {
        // ===================== TMA producer (whole warp in uniform control flow; one elected lane issues) ====
        if (has_acc) {
            int slot = 0;
            uint32_t phase = 0;
            auto load = [&](uint32_t dst, const CUtensorMap* m, uint32_t bar, int c0, int c1) {
                if (CG == 2) ptx::tma_load_2d_pair(dst, m, bar, c0, c1); else ptx::tma_load_2d(dst, m, bar, c0, c1);
            };
            ItemIter iter = {-1, unit0, 0, 0, 0};
            WorkItem w;
            int seq = 0;
            while (next_item<CG>(op, iter, unit0, nunits, w)) {
                const int rb = w.rb + rank, cb0u = w.cb;
                if (w.mode == MODE_POTRF) { ++seq; continue; }
                if (w.dep) {
                    // the operand images this item reads were written by this CTA's epilogue warps `dep` items ago
                    const int qd = seq - w.dep;
                    uint32_t spins = 0;
                    while (item_ctr[qd & 7] < item_complete_count(qd)) { if (++spins > (1u << 27)) __trap(); }
                    __threadfence();
                    ptx::fence_proxy_async_global();
                }
                if (w.xcta >= 0) {
                    const volatile int* pr = op.prog + w.xcta;
                    uint32_t spins = 0;
                    while (*pr < w.xneed) { __nanosleep(64); if (++spins > (1u << 25)) __trap(); }
                    __threadfence();
                    ptx::fence_proxy_async_global();
                }
                ++seq;
                uint32_t cls_next = term_class_load<CG>(op, w.mode, w.t_hi - 1, rb);
                for (int s = w.t_hi - 1; s >= w.t_lo; --s) {      // descending K: see note on accumulation order
                    const uint32_t cls = make_uniform(cls_next);
                    if (s > w.t_lo) cls_next = term_class_load<CG>(op, w.mode, s - 1, rb);   // in flight during this term's chunks
                    // this CTA's A rows and B rows
                    TermGeom g = (w.mode == MODE_INV) ? w.g : term_geom(op, w.mode, w.c, s, rb, cb0u + rank, cb0u, CG);
                    if (w.mode == MODE_UPDATE) {         // table look-ups: make them provably warp-uniform (TMA coordinates)
                        g.a_row_lo = static_cast<int>(make_uniform(static_cast<uint32_t>(g.a_row_lo)));
                        g.b_row_lo = static_cast<int>(make_uniform(static_cast<uint32_t>(g.b_row_lo)));
                        g.a_row_q = static_cast<int>(make_uniform(static_cast<uint32_t>(g.a_row_q)));
                        g.b_row_q = static_cast<int>(make_uniform(static_cast<uint32_t>(g.b_row_q)));
                    }
                    if (cls & kClsQ) {                       // E4M3 images: 128 bytes of K per row, one slot per chunk
                        for (int ch = g.kelems / 128 - 1; ch >= 0; --ch) {
                            ptx::mbar_wait(empty_bar(slot), phase ^ 1u);
                            if (ptx::elect_one()) {
                                const uint32_t sa = smem_base + slot * SB;
                                if (rank == 0) ptx::mbar_arrive_expect_tx(full_bar(slot), CG * 2u * kPlaneBytes);
                                load(sa, &tmQ, full_bar(slot), ch * 128, g.a_row_q);
                                load(sa + kPlaneBytes, &tmQ, full_bar(slot), ch * 128, g.b_row_q);
                            }
                            if (++slot == kSlots) { slot = 0; phase ^= 1u; }
                        }
                        continue;
                    }
                    const bool a_lo = cls & kClsALo, b_lo = cls & kClsBLo;
                    const CUtensorMap* mA_hi = (g.a_src == 2) ? &tmSH : &tmH;
                    const CUtensorMap* mA_lo = (g.a_src == 2) ? &tmSL : &tmL;
                    const CUtensorMap* mB_hi = (g.b_src == 2) ? &tmSH : ((g.b_src == 1) ? &tmIH : &tmH);
                    const CUtensorMap* mB_lo = (g.b_src == 2) ? &tmSL : ((g.b_src == 1) ? &tmIL : &tmL);
                    const uint32_t lo_bytes = CG * ((a_lo ? 1u : 0u) + (b_lo ? 1u : 0u)) * kPlaneBytes;
                    const int ch_hi = (w.ch_hi >= 0) ? w.ch_hi : g.kelems / kBlockK, ch_lo = (w.ch_lo >= 0) ? w.ch_lo : 0;
                    for (int ch = ch_hi - 1; ch >= ch_lo; --ch) {
                        const int ak = g.a_k0 + ch * kBlockK, bk = g.b_k0 + ch * kBlockK;
                        ptx::mbar_wait(empty_bar(slot), phase ^ 1u);
                        if (ptx::elect_one()) {              // hi images
                            const uint32_t sa = smem_base + slot * SB;
                            if (rank == 0) ptx::mbar_arrive_expect_tx(full_bar(slot), CG * 2u * kPlaneBytes);
                            load(sa, mA_hi, full_bar(slot), ak, g.a_row);
                            load(sa + kPlaneBytes, mB_hi, full_bar(slot), bk, g.b_row);
                        }
                        if (++slot == kSlots) { slot = 0; phase ^= 1u; }
                        if (lo_bytes) {                      // lo images of the FP32-class operand(s)
                            ptx::mbar_wait(empty_bar(slot), phase ^ 1u);
                            if (ptx::elect_one()) {
                                const uint32_t sa = smem_base + slot * SB;
                                if (rank == 0) ptx::mbar_arrive_expect_tx(full_bar(slot), lo_bytes);
                                if (a_lo) load(sa, mA_lo, full_bar(slot), ak, g.a_row_lo);
                                if (b_lo) load(sa + kPlaneBytes, mB_lo, full_bar(slot), bk, g.b_row_lo);
                            }
                            if (++slot == kSlots) { slot = 0; phase ^= 1u; }
                        }
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer (whole warp in uniform control flow; one elected lane issues) =====
        if (has_acc && rank == 0) {
            constexpr uint32_t idesc = ptx::make_idesc(kBlk * CG, kBlk * CG, /*F16*/ 0, /*F16*/ 0);
            constexpr uint32_t idesc_q = ptx::make_idesc_mxf8(kBlk * CG, kBlk * CG);
            auto mma = [&](uint32_t d, uint32_t a_lo32, uint32_t b_lo32, uint32_t acc) {
                const uint64_t a = ptx::smem_desc_from_lo(a_lo32), b = ptx::smem_desc_from_lo(b_lo32);
                if (CG == 2) ptx::mma_f16_ss_pair(d, a, b, idesc, acc); else ptx::mma_f16_ss(d, a, b, idesc, acc);
            };
            auto commit = [&](uint32_t bar) { if (CG == 2) ptx::tc_commit_pair(bar); else ptx::tc_commit(bar); };
            // low word of the descriptor of ring slot c's A block; the B block is 16 KB (1024 x 16 B) further
            const uint32_t dlo0 = ptx::smem_desc_lo(smem_base);
            constexpr uint32_t kDescSlot = SB >> 4, kDescB = kPlaneBytes >> 4;
            int slot = 0;
            uint32_t phase = 0;
            int buf = 0;
            uint32_t acc_phase = 0;
            ItemIter iter = {-1, unit0, 0, 0, 0};
            WorkItem w;
            while (next_item<CG>(op, iter, unit0, nunits, w)) {
                const int rb = w.rb;
                if (w.mode == MODE_POTRF) continue;
                uint32_t cls_next = term_class_load<CG>(op, w.mode, w.t_hi - 1, rb);
                ptx::mbar_wait(tempty_bar(buf), acc_phase ^ 1u);     // epilogue drained this buffer
                ptx::tc_fence_after();
                const uint32_t d_tmem = tmem_base + buf * kAccW;
                uint32_t accumulate = 0;
                for (int s = w.t_hi - 1; s >= w.t_lo; --s) {      // descending K: see note on accumulation order
                    const uint32_t cls = make_uniform(cls_next);
                    if (s > w.t_lo) cls_next = term_class_load<CG>(op, w.mode, s - 1, rb);
                    const int kelems = (w.mode == MODE_UPDATE) ? op.nb
                                       : (w.mode == MODE_P1 ? w.c * kBlk
                                          : (w.mode == MODE_INV ? w.g.kelems
                                             : (w.mode == MODE_TRSM ? ((w.cb + CG) * kBlk < op.nb ? (w.cb + CG) * kBlk : op.nb) : kBlk)));
                    if (cls & kClsQ) {
                        const uint32_t sfa = tmem_base + kSfCol0 + 4 * CG * ((cls >> 8) & 63u);
                        const uint32_t sfb = tmem_base + kSfCol0 + 4 * CG * ((cls >> 16) & 63u);
                        for (int ch = kelems / 128 - 1; ch >= 0; --ch) {
                            ptx::mbar_wait(full_bar(slot), phase);
                            ptx::tc_fence_after();
                            if (ptx::elect_one()) {
                                const uint32_t a = dlo0 + slot * kDescSlot, b = a + kDescB;
#pragma unroll
                                for (int kk = 3; kk >= 0; --kk) {          // 4 x K=32 per 128-byte row
                                    const uint64_t da = ptx::smem_desc_from_lo(a + 2 * kk), db = ptx::smem_desc_from_lo(b + 2 * kk);
                                    if (CG == 2) ptx::mma_mxf8_ss_pair(d_tmem, da, db, idesc_q, (kk == 3) ? accumulate : 1u, sfa, sfb);
                                    else ptx::mma_mxf8_ss(d_tmem, da, db, idesc_q, (kk == 3) ? accumulate : 1u, sfa, sfb);
                                }
                                commit(empty_bar(slot));
                            }
                            accumulate = 1;
                            if (++slot == kSlots) { slot = 0; phase ^= 1u; }
                        }
                        continue;
                    }
                    const bool a_lo = cls & kClsALo, b_lo = cls & kClsBLo;
                    const int ch_hi = (w.ch_hi >= 0) ? w.ch_hi : kelems / kBlockK, ch_lo = (w.ch_lo >= 0) ? w.ch_lo : 0;
                    for (int ch = ch_hi - 1; ch >= ch_lo; --ch) {
                        const int c0 = slot;
                        ptx::mbar_wait(full_bar(c0), phase);
                        if (++slot == kSlots) { slot = 0; phase ^= 1u; }
                        const int c1 = slot;
                        if (a_lo || b_lo) {
                            ptx::mbar_wait(full_bar(c1), phase);
                            if (++slot == kSlots) { slot = 0; phase ^= 1u; }
                        }
                        ptx::tc_fence_after();
                        if (ptx::elect_one()) {
                            const uint32_t ah = dlo0 + c0 * kDescSlot, bh = ah + kDescB;
                            const uint32_t al = dlo0 + c1 * kDescSlot, bl = al + kDescB;
                            // +32 B (2 descriptor units) per K = 16; small cross terms first, the dominant hi*hi last
                            if (a_lo && b_lo && split_cross) {
                                const uint32_t d_cross = d_tmem + kAccW;
#pragma unroll
                                for (int kk = kBlockK / 16 - 1; kk >= 0; --kk) {
                                    mma(d_cross, al + 2 * kk, bh + 2 * kk, (kk == 3) ? accumulate : 1u);
                                    mma(d_cross, ah + 2 * kk, bl + 2 * kk, 1u);
                                    mma(d_tmem, ah + 2 * kk, bh + 2 * kk, (kk == 3) ? accumulate : 1u);
                                }
                            } else if (a_lo && b_lo) {
#pragma unroll
                                for (int kk = kBlockK / 16 - 1; kk >= 0; --kk) {
                                    mma(d_tmem, al + 2 * kk, bh + 2 * kk, (kk == 3) ? accumulate : 1u);
                                    mma(d_tmem, ah + 2 * kk, bl + 2 * kk, 1u);
                                    mma(d_tmem, ah + 2 * kk, bh + 2 * kk, 1u);
                                }
                            } else if (a_lo) {
#pragma unroll
                                for (int kk = kBlockK / 16 - 1; kk >= 0; --kk) {
                                    mma(d_tmem, al + 2 * kk, bh + 2 * kk, (kk == 3) ? accumulate : 1u);
                                    mma(d_tmem, ah + 2 * kk, bh + 2 * kk, 1u);
                                }
                            } else if (b_lo) {
#pragma unroll
                                for (int kk = kBlockK / 16 - 1; kk >= 0; --kk) {
                                    mma(d_tmem, ah + 2 * kk, bl + 2 * kk, (kk == 3) ? accumulate : 1u);
                                    mma(d_tmem, ah + 2 * kk, bh + 2 * kk, 1u);
                                }
                            } else {
#pragma unroll
                                for (int kk = kBlockK / 16 - 1; kk >= 0; --kk)
                                    mma(d_tmem, ah + 2 * kk, bh + 2 * kk, (kk == 3) ? accumulate : 1u);
                            }
                            commit(empty_bar(c0));                   // smem slots free (in both CTAs) when MMAs retire
                            if (a_lo || b_lo) commit(empty_bar(c1));
                        }
                        accumulate = 1;
                    }
                }
                if (ptx::elect_one()) commit(tfull_bar(buf));        // accumulator complete
                if (++buf == nbufs) { buf = 0; acc_phase ^= 1u; }
            }
        }
    } else {
        // ===================== epilogue warps (TMEM -> registers -> global) =====================
        // Warp (q, hf): TMEM lanes (rows) 32q..32q+31, columns 64hf..64hf+63 of the 128x128 block.
        // W is block-column-major, so a warp's 32 rows of one column are 128 contiguous bytes; the FP16
        // images and the mosaic tiles are row-major and go through a per-warp smem transpose so
        // that every store instruction writes 8 full 64-byte row segments.
        const int ew = warp - 2;
        const int q = warp & 3;
        const int hf = ew >> 2;
        uint8_t* stg = smem_raw + (bar_base - ptx::smem_u32(smem_raw)) + 256 + ew * kEpiStageBytes;
        const int nsub = op.nb / kBlk;
        int buf = 0;
        uint32_t acc_phase = 0;
        ItemIter iter = {-1, unit0, 0, 0, 0};
        WorkItem w;
        int eseq = 0;                                                // items this CTA has finished
        float out[64];                                               // (lives across the K segments of a block)
        while (next_item<CG>(op, iter, unit0, nunits, w)) {
            const int rb = w.rb + rank, cb0u = w.cb;
            if (w.mode == MODE_POTRF) {
                // FP32 Cholesky + inverse of the diagonal 128-block on the epilogue warps; the operand ring is idle
                // (this is the CTA's last item) and serves as its shared memory
                struct EpiSync { __device__ __forceinline__ void operator()() const { asm volatile("bar.sync 1, 256;" ::: "memory"); } };
                EpiSync esync;
                esync();                                              // every warp's stores of the previous item are done
                float* tri_sm = reinterpret_cast<float*>(smem_raw + (smem_base - ptx::smem_u32(smem_raw)));
                potrf128_body<kEpiWarps * 32>(tri_sm, static_cast<int>(threadIdx.x) - 64, esync, op.W, op.nb, rb * kBlk, w.c * kBlk,
                                              op.linv_hi, op.linv_lo, op.linv_scale_w, op.info, op.col_base + w.c * kBlk);
                __threadfence();
                ptx::fence_proxy_async_global();
                esync();
                if (threadIdx.x == 64) { __threadfence(); *const_cast<volatile int*>(op.prog + (rb - op.rb0)) = eseq + 1; }
                ++eseq;
                continue;
            }
            const bool item_planes = write_planes && (w.sk_role != 2);
            // everything the store needs from global memory is fetched here, before the wait for the accumulator
            int t_prec = KRR_FP32;
            uint8_t* t_tile = nullptr;
            float t_acc_mul = 0.0f, t_sx = 0.0f, t_di = 1.0f, t_inv_di = 1.0f;
            int64_t t_lrow = 0;                                      // first lo-plane row of the tile (FP32 tiles)
            if (w.mode == MODE_TRSM) {
                const int ti = op.k + (rb * kBlk) / op.nb;
                t_prec = op.map[ti * op.NT + op.k];
                t_tile = op.factor + op.off[ti * op.NT + op.k];
                t_acc_mul = -op.scl[SCL_INV_SS_SM];
                t_sx = op.scl[SCL_SX];
                t_di = op.dscale[ti];
                t_inv_di = 1.0f / t_di;
                t_lrow = op.lrow[ti * op.NT + op.k];
            }
#pragma unroll 1
          for (int j2 = 0; j2 < CG; ++j2) {                       // the unit's column blocks, one after the other
            const int cb = cb0u + j2;
            const bool dead = tile_is_skipped(op, rb, cb);        // this CTA's block lies above the diagonal: nothing to store
            const int row_in_blk = q * 32 + lane;
            const int col0 = cb * kBlk + 64 * hf;                 // first column (inside the tile column) of this warp
            float* wblk = op.W + (static_cast<int64_t>(rb) * nsub + cb) * (kBlk * kBlk) + static_cast<int64_t>(64 * hf) * kBlk + row_in_blk;
            // ---- base values, fetched before the accumulator is ready
            float bs[64];
            const bool base_from_w = (w.mode == MODE_P1) || (w.mode == MODE_UPDATE && op.base_w && w.sk_role != 2);
            const bool base_from_a = (w.mode == MODE_UPDATE && !op.base_w && w.sk_role != 2);
            if (dead) {
#pragma unroll
                for (int e = 0; e < 64; ++e) bs[e] = 0.0f;
            } else if (base_from_w) {
#pragma unroll
                for (int e = 0; e < 64; ++e) bs[e] = __ldcg(wblk + e * kBlk);
            } else if (base_from_a) {
                const int i = op.k + (rb * kBlk) / op.nb;
                const int subrow = (rb * kBlk) % op.nb;
                const float* arow = op.A.tile_ptr(i, op.k, subrow + row_in_blk, col0);
                int p = KRR_FP32;
                float sc = 1.0f;
                if ((op.flags & KRR_FLAG_PREROUND_A) && i != op.k) {
                    p = op.map[i * op.NT + op.k];
                    if (p == KRR_FP8_E4M3) sc = fp8_scale_from_amax(op.a_amax[i * op.NT + op.k]);
                }
                const float dd = op.dscale[i] * op.dscale[op.k];        // A~ = D A D (rounded first, then scaled: exact)
#pragma unroll
                for (int e = 0; e < 64; e += 4) {
                    const float4 v = *reinterpret_cast<const float4*>(arow + e);
                    bs[e + 0] = round_to_prec(v.x, p, sc) * dd;
                    bs[e + 1] = round_to_prec(v.y, p, sc) * dd;
                    bs[e + 2] = round_to_prec(v.z, p, sc) * dd;
                    bs[e + 3] = round_to_prec(v.w, p, sc) * dd;
                }
            } else {
#pragma unroll
                for (int e = 0; e < 64; ++e) bs[e] = 0.0f;
            }
            if (has_acc) {
                if (j2 == 0) ptx::mbar_wait(tfull_bar(buf), acc_phase);
                ptx::tc_fence_after();
                // exact power-of-two rescaling of the accumulator into the value domain, sign included (out = bs - acc * acc_mul).
                // (read after the accumulator is complete: in MODE_DIAG the scale of the inverted block is written by
                // another CTA of this launch, and the MMAs could not have run before it was)
                float acc_mul;
                if (w.mode == MODE_P3) acc_mul = -op.scl[SCL_INV_SS] / __ldcg(op.linv_scale + w.c);
                else if (w.mode == MODE_TRSM) acc_mul = t_acc_mul;
                else if (w.mode == MODE_INV) acc_mul = (w.o_var == 0) ? -op.scl[SCL_INV_SM_SX] : op.scl[SCL_INV_SM_SU];
                else acc_mul = op.scl[SCL_INV_SX2];
                uint32_t a0[32], a1[32];
                const uint32_t taddr = tmem_base + buf * kAccW + (static_cast<uint32_t>(q * 32) << 16) + kAccCols * j2 + 64 * hf;
                ptx::tmem_ld_32x32(taddr, a0);
                ptx::tmem_ld_32x32(taddr + 32, a1);
                ptx::tmem_ld_wait();
                ptx::tc_fence_before();
                __syncwarp();
                if (j2 == CG - 1) {
                    if (lane == 0 && !split_cross) {                        // accumulator is in registers
                        if (CG == 2) ptx::mbar_arrive_leader(tempty_bar(buf)); else ptx::mbar_arrive(tempty_bar(buf));
                    }
                    if (++buf == nbufs) { buf = 0; acc_phase ^= 1u; }
                }
                if (split_cross) {
                    // main + cross accumulators, added in FP32 (round to nearest); the TMEM buffer is released afterwards
                    uint32_t c0[32];
                    ptx::tmem_ld_32x32(taddr + kAccW, c0);
                    ptx::tmem_ld_wait();
#pragma unroll
                    for (int e = 0; e < 32; ++e) out[e] = -(__uint_as_float(a0[e]) + __uint_as_float(c0[e])) * acc_mul;
                    ptx::tmem_ld_32x32(taddr + kAccW + 32, c0);
                    ptx::tmem_ld_wait();
#pragma unroll
                    for (int e = 0; e < 32; ++e) out[32 + e] = -(__uint_as_float(a1[e]) + __uint_as_float(c0[e])) * acc_mul;
                    ptx::tc_fence_before();
                    __syncwarp();
                    if (j2 == CG - 1 && lane == 0) ptx::mbar_arrive_leader(tempty_bar(0));
                } else if (w.seg_first) {
#pragma unroll
                    for (int e = 0; e < 32; ++e) {
                        out[e] = fmaf(-__uint_as_float(a0[e]), acc_mul, bs[e]);
                        out[32 + e] = fmaf(-__uint_as_float(a1[e]), acc_mul, bs[32 + e]);
                    }
                } else {                                                     // a later K segment of the same block
#pragma unroll
                    for (int e = 0; e < 32; ++e) {
                        out[e] = fmaf(-__uint_as_float(a0[e]), acc_mul, out[e]);
                        out[32 + e] = fmaf(-__uint_as_float(a1[e]), acc_mul, out[32 + e]);
                    }
                }
            } else {
#pragma unroll
                for (int e = 0; e < 64; ++e) out[e] = bs[e];
            }
            if (dead || !w.seg_last) continue;
            if (w.sk_role == 2) {
                // lower terms of a block another group finishes: leave -(sum of the products) for it (block-column-major
                // like W: a warp's 32 rows of a column are 128 contiguous bytes)
                float* pblk = op.sk_partial + ((static_cast<int64_t>(unit0) * CG + rank) * CG + j2) * (kBlk * kBlk) +
                              static_cast<int64_t>(64 * hf) * kBlk + row_in_blk;
#pragma unroll
                for (int e = 0; e < 64; ++e) __stcg(pblk + e * kBlk, out[e]);
                continue;
            }
            if (w.sk_role == 1) {
                // highest terms of a shared block: add the partial sums of the groups that hold the lower terms, in ascending
                // group order (descending terms: the dominant leading columns last)
                for (int m = 0; m < w.sk_nother; ++m) {
                    const int ou = w.sk_other + m * w.sk_stride;
                    if (lane == 0) {
                        const volatile int* f = op.sk_flags + ou;
                        uint32_t spins = 0;
                        while (*f < CG) { __nanosleep(64); if (++spins > (1u << 26)) __trap(); }
                        __threadfence();
                    }
                    __syncwarp();
                    const float* pblk = op.sk_partial + ((static_cast<int64_t>(ou) * CG + rank) * CG + j2) * (kBlk * kBlk) +
                                        static_cast<int64_t>(64 * hf) * kBlk + row_in_blk;
#pragma unroll
                    for (int e = 0; e < 64; ++e) out[e] += __ldcg(pblk + e * kBlk);
                }
            }
            if (w.mode == MODE_INV) {
                // a block of U^T (scale su) or of M / M^T (scale sm) into the scratch planes; a value beyond the FP16 range
                // means the diagonal tile is too ill-conditioned for the product form of the TRSM: info = -2
                const float mul = op.scl[w.o_var == 0 ? SCL_SU : SCL_SM];
                const int64_t orow = static_cast<int64_t>(w.o_row) + q * 32;
                const float big = epi_store_images(stg, lane, out, mul, op.Sh, op.Sl, orow, orow, w.o_col + 64 * hf, op.nb);
                if (!(big < 60000.0f)) atomicCAS(op.info, 0, -2);
            } else if (w.mode == MODE_TRSM) {
                // X = S inv(L_kk)^T is final: round once into the tile's storage precision and store it (R4; PAPER.md:206
                // "on-the-fly" conversion): FP32 / FP16 tiles straight into the mosaic with their operand images; FP8 tiles
                // need the tile's amax first, so they leave FP32 values in W and finalize_kernel rounds them
                const int p = t_prec;
                const int r_tile = (rb * kBlk) % op.nb + q * 32;                            // this warp's row 0 inside the tile
                const int64_t prow = op.prow0 + static_cast<int64_t>(rb) * kBlk + q * 32;   // ... and in the planes
                uint8_t* tile = t_tile;
                // (out holds the equilibrated X~ = d_i X: the images are of X~, the stored tile is X = X~ / d_i)
                if (p == KRR_FP32) {
                    epi_store_images(stg, lane, out, t_sx, op.Hp, op.Lp, prow, t_lrow + (rb * kBlk) % op.nb + q * 32, col0, op.nb);
#pragma unroll
                    for (int part = 0; part < 4; ++part) {
                        uint32_t wds[16];
#pragma unroll
                        for (int t = 0; t < 16; ++t) wds[t] = __float_as_uint(out[16 * part + t] * t_inv_di);
                        epi_store_part(stg, lane, make_uint4(wds[0], wds[1], wds[2], wds[3]), make_uint4(wds[4], wds[5], wds[6], wds[7]),
                                       make_uint4(wds[8], wds[9], wds[10], wds[11]), make_uint4(wds[12], wds[13], wds[14], wds[15]),
                                       tile + (static_cast<int64_t>(r_tile) * op.nb + col0 + 16 * part) * 4, static_cast<int64_t>(op.nb) * 4);
                    }
                } else if (p == KRR_FP16) {
                    // the stored value h = rn16(X~ / d_i); out becomes its equilibrated value h d_i, whose image is exact
#pragma unroll
                    for (int part = 0; part < 2; ++part) {
                        uint32_t wds[16];
#pragma unroll
                        for (int t = 0; t < 16; ++t) {
                            const int e = 32 * part + 2 * t;
                            const __half2 h = __floats2half2_rn(out[e] * t_inv_di, out[e + 1] * t_inv_di);
                            out[e] = __low2float(h) * t_di;
                            out[e + 1] = __high2float(h) * t_di;
                            wds[t] = *reinterpret_cast<const uint32_t*>(&h);
                        }
                        epi_store_part(stg, lane, make_uint4(wds[0], wds[1], wds[2], wds[3]), make_uint4(wds[4], wds[5], wds[6], wds[7]),
                                       make_uint4(wds[8], wds[9], wds[10], wds[11]), make_uint4(wds[12], wds[13], wds[14], wds[15]),
                                       tile + (static_cast<int64_t>(r_tile) * op.nb + col0 + 32 * part) * 2, static_cast<int64_t>(op.nb) * 2);
                    }
                    epi_store_images(stg, lane, out, t_sx, op.Hp, nullptr, prow, prow, col0, op.nb);      // image of the STORED value (exact)
                } else {
                    float amax = 0.0f;
#pragma unroll
                    for (int e = 0; e < 64; ++e) { wblk[e * kBlk] = out[e]; amax = fmaxf(amax, fabsf(out[e])); }
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
                    if (lane == 0) {
                        const int64_t slot = op.prow0 / op.nb + (static_cast<int64_t>(rb) * kBlk) / op.nb;
                        atomicMax(reinterpret_cast<int*>(op.tile_amax + slot), __float_as_int(amax));
                    }
                }
            } else {
                // S of the rows below the diagonal tile goes to the scratch planes only (the TRSM product reads it
                // there); everything else keeps its FP32 value in W
                const bool below = (w.mode == MODE_UPDATE) && (rb >= nsub);
                if (!(below && item_planes)) {
#pragma unroll
                    for (int e = 0; e < 64; ++e) wblk[e * kBlk] = out[e];
                }
                if (item_planes) {
                    const float mul = op.scl[w.mode == MODE_P3 ? SCL_SX : SCL_SS];
                    const int64_t lrow0 = static_cast<int64_t>(rb) * kBlk + q * 32;      // panel-local row of this warp
                    if (below) epi_store_images(stg, lane, out, mul, op.Sh, op.Sl, lrow0, lrow0, col0, op.nb);
                    else epi_store_images(stg, lane, out, mul, op.Hp, op.Lp, op.prow0 + lrow0, op.prow0_lo + lrow0, col0, op.nb);
                }
            }
          }   // j2
            if (w.sk_role == 2) {
                // the partial sum is in sk_partial: tell the finisher (the last warp of this CTA signals; a unit leaves at
                // most one partial sum per launch -- for its first item)
                __threadfence();
                __syncwarp();
                if (lane == 0) {
                    if (atomicAdd_block(split_ctr, 1) == kEpiWarps - 1) { __threadfence(); atomicAdd(op.sk_flags + unit0, 1); }
                }
            }
            if (op.mode == MODE_DIAG) {
                // publish this item's operand images to the TMA loads of a later item of this CTA and of the other
                // CTAs: the last warp to finish advances the CTA's progress counter
                __threadfence();
                ptx::fence_proxy_async_global();
                __syncwarp();
                if (lane == 0) {
                    const int old = atomicAdd_block(const_cast<int*>(item_ctr + (eseq & 7)), 1);
                    if (old == item_complete_count(eseq) - 1) {
                        __threadfence();
                        *const_cast<volatile int*>(op.prog + (rb - op.rb0)) = eseq + 1;
                    }
                }
            }
            ++eseq;
        }
    }

    // teardown
    ptx::tc_fence_before();
    if (CG == 2) ptx::cluster_sync_all(); else __syncthreads();
    if (warp == 1) ptx::tmem_dealloc<kTmemCols, CG>(tmem_base);
}

}  // namespace krr

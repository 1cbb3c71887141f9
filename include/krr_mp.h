/*
 * krr_mp.h -- C ABI of the B200-native mixed-precision tile Cholesky for Kernel Ridge Regression.
 *
 * The hot path of the paper's Associate phase (Alg. 3):
 *     K~ <- FACTORIZE(K + alpha*Id)      -> krr_precision_map + krr_potrf_mp
 *     W  <- Solve(K~, P_h)      -> krr_potrs
 * with the tile-centric adaptive-precision Cholesky of PAPER.md:192 ("a tiled mosaic of precisions
 * embedded in a single stored copy of the matrix", FP32 / FP16 / FP8-E4M3 per tile)
 * and forward/backward substitution "in the full FP32 precision".
 *
 * Conventions
 *   - Every d_* pointer is DEVICE memory owned by the caller (e.g. a PyTorch tensor); every h_*
 *     pointer is HOST memory.  `stream` is a cudaStream_t passed as void*.  Unless stated, the
 *     library never allocates or frees device memory, never synchronises the device and never
 *     reads or writes the host copy of the data; all work is enqueued on `stream`.  What it does
 *     create, once per host thread and device, are three internal CUDA streams (priorities high /
 *     middle / low) and a pool of CUDA events for the lookahead schedule; krr_shutdown() destroys them.
 *   - n = number of patients (matrix order), nb = tile size, NT = n / nb.  nb must be a multiple
 *     of 128 and divide n (all BASELINE.json configs do; ragged edges are not supported).
 *   - Tiles are addressed (i, j), 0-based, i >= j (lower triangle).  A precision map is NT*NT
 *     bytes, row-major, map[i*NT + j] in {KRR_FP32, KRR_FP16, KRR_FP8_E4M3} for i >= j; entries
 *     with i < j are ignored on input and written as 255 on output.  Diagonal tiles are FP32.
 *   - Return value: 0 on success, < 0 for an argument / usage error detected on the host before
 *     anything is launched (see KRR_ERR_*).  Numerical breakdown is reported asynchronously
 *     through *d_info (LAPACK convention), never through the return value.
 *   - Thread-safety: re-entrant on distinct streams with distinct workspaces.
 */
#ifndef KRR_MP_H
#define KRR_MP_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum { KRR_FP32 = 0, KRR_FP16 = 1, KRR_FP8_E4M3 = 2 } krr_prec_t;

#define KRR_OK               0
#define KRR_ERR_ARG        (-1)   /* null pointer, non-positive size, lda/ldb too small            */
#define KRR_ERR_SHAPE      (-2)   /* nb does not divide n, nb not a multiple of 128, NT too large  */
#define KRR_ERR_WORKSPACE  (-3)   /* ws_bytes smaller than the matching *_workspace() query        */
#define KRR_ERR_DEVICE     (-4)   /* current device is not compute capability 10.x (sm_100)        */
#define KRR_ERR_CUDA       (-5)   /* a CUDA call or kernel launch failed                           */
#define KRR_ERR_MAP        (-6)   /* invalid precision code in h_map, or non-FP32 diagonal tile    */
#define KRR_ERR_UNSUPPORTED (-7)  /* a flag bit this build does not implement                      */

/* flags (krr_precision_map, krr_potrf_mp, krr_associate_host, krr_build) */
#define KRR_FLAG_PREROUND_A     1u  /* round the off-diagonal tiles of A into their storage precision
                                       before factorising ("lower the precision of the
                                       off-diagonal tiles ... followed by the mixed-precision
                                       Cholesky").  Default of the Python binding.                  */
#define KRR_FLAG_A_TILED_LOWER  4u  /* d_A holds only the lower tiles ("lower-triangular tile
                                       storage", BASELINE.json config 4): tile (i,j), i >= j, is a
                                       contiguous row-major nb x nb block at element offset
                                       krr_tile_slot(NT,i,j) * nb * nb; lda is ignored.             */

#define KRR_FLAG_NO_LOOKAHEAD    8u  /* krr_potrf_mp: run the tile columns strictly one after the other on
                                       the caller's stream (no internal streams; per-kernel timing and
                                       debugging).  Default: column k+1's update of the already final
                                       columns overlaps the factorisation of column k (lookahead 1).  */

#define KRR_FLAG_FP8_VIA_FP16   16u  /* krr_potrf_mp: multiply FP8 x FP8 tile pairs through their (exact) FP16
                                       images with kind::f16 MMAs instead of kind::mxf8f6f4 on the E4M3
                                       images (same values, half the tensor rate; cross-check).       */

#define KRR_FLAG_NO_CTA_PAIRS   32u  /* krr_potrf_mp: run the trailing updates with one CTA per 128x128 block
                                       instead of CTA pairs (tcgen05 cta_group::2, 256x128 blocks); same
                                       arithmetic, cross-check / comparison.  Pairs need nb % 256 == 0.   */

#define KRR_FLAG_FUSED_CHAIN    64u  /* krr_potrf_mp: run the diagonal-tile chain (in-tile update, POTRF of a
                                       128-block, TRSM against its inverse, per 128-wide sub-column) as ONE
                                       launch of nb/128 co-operating CTAs (the POTRF on the epilogue warps,
                                       items ordered through progress counters in global memory) instead of
                                       one launch per step; bit-identical results.  Measured equal or a
                                       few % slower than the default on a B200 (the chain is bound by the
                                       128 dependent pivots of each block, not by launches), kept as the
                                       persistent-kernel variant and as a cross-check.                 */

#define KRR_FLAG_NO_TAIL_SPLIT 1024u /* krr_potrf_mp: do not split the blocks of a trailing update's last, partial wave
                                       between several CTA pairs (slices of the term range added into the FP32
                                       partial sums one after the other); same products, another summation order
                                       for those blocks; comparison.                                   */

#define KRR_FLAG_KERNEL_IBS    256u  /* krr_build, krr_predict: the identical-by-state kernel of Alg. 5 l.5-6 (PAPER.md:134,
                                       :141) instead of the Gaussian one: K_ij = (alleles of i and j identical
                                       by state, 2 - |g_ik - g_jk| per locus for genotypes in {0,1,2}) / (2 N_S).
                                       Same tensor-core kernel on thermometer-encoded genotypes ([g>=1],[g>=2]:
                                       their Hamming distance is sum_k |g_ik - g_jk|); gamma is ignored and
                                       confounders are not accepted.                                  */

#define KRR_FLAG_KERNEL_LINEAR 512u  /* krr_build, krr_predict: the linear kernel K_ij = gamma * <g_i, g_j> (exact INT32 Gram
                                       matrix times the FP32 scale `gamma`; krr_build adds lambda on the diagonal):
                                       with G = X^T (rows = SNPs) this is the mixed-precision SYRK X^T X + lambda I of
                                       ridge regression (Eq. (2), Fig. 2; integer part only), with G = X the
                                       dual form of the same regression.  Confounders are not accepted.       */

/* Library version (major*100 + minor) and the compute capability it was built for (100). */
int krr_version(void);
int krr_built_for_sm(void);

/* Index of tile (i,j), i >= j, in column-major order over the lower triangle:
 * slot = j*NT - j*(j-1)/2 + (i - j).  Pure host function. */
int64_t krr_tile_slot(int NT, int i, int j);

/* ---------------------------------------------------------------------------------------------
 * krr_precision_map -- tile norms and the tile-centric adaptive-precision map.
 * PAPER.md:192, :215, :229; rule text from BASELINE.json (the paper prints no formula):
 *     off-diagonal tile (i,j) gets the LOWEST precision p with bit p set in allowed_mask and
 *         ||A_ij||_F * u_p  <=  eps_target * ||A||_F / NT ,     u = 2^-24, 2^-11, 2^-4,
 *     KRR_FP32 if none qualifies; diagonal tiles are KRR_FP32.  ||A||_F is of the full symmetric
 *     matrix (off-diagonal tiles counted twice).
 * d_A         in   FP32, row-major n x n with leading dimension lda (elements), only tiles with
 *                  i >= j are read (diagonal tiles as full squares); or tile-packed lower storage
 *                  with KRR_FLAG_A_TILED_LOWER.  Not modified.
 * d_map       out  NT*NT bytes.
 * d_tile_norms out NT*NT floats, ||A_ij||_F for i >= j, 0 above; may be NULL.
 * d_tile_amax out  NT*NT floats, max|A_ij| for i >= j, 0 above; may be NULL.
 * d_fro       out  one double, ||A||_F; may be NULL.
 * d_ws        workspace of at least krr_precision_map_workspace(n, nb) bytes.
 * Sums of squares are accumulated in FP64 in a fixed order (deterministic).  One pass over the
 * lower tiles of A: HBM-bound.
 */
size_t krr_precision_map_workspace(int64_t n, int nb);
int krr_precision_map(const float* d_A, int64_t n, int64_t lda, int nb,
                      float eps_target, unsigned allowed_mask, unsigned flags,
                      uint8_t* d_map, float* d_tile_norms, float* d_tile_amax, double* d_fro,
                      void* d_ws, size_t ws_bytes, void* stream);

/* ---------------------------------------------------------------------------------------------
 * krr_precision_map_static -- krr_precision_map for callers that cannot allocate (code under CUDA-graph
 * capture, serving loops, harnesses that forbid cudaMalloc): same operation,
 * same kernels, same summation order, hence the same bits in every output -- but the scratch memory is
 * a file-scope __device__ array inside the library instead of the caller's d_ws.  The call allocates
 * nothing: no cudaMalloc / cudaFree, no stream, event or host-vector growth (it is not timed by
 * krr_profile_enable); it enqueues two kernels on `stream` and returns.
 *   - Limit: krr_precision_map_workspace(n, nb) <= KRR_PRECISION_MAP_STATIC_BYTES (4 MiB; every
 *     BASELINE.json config fits: C4, NT = 128, nb = 1024 needs 3.09 MiB).  Larger shapes return
 *     KRR_ERR_WORKSPACE and launch nothing; krr_precision_map_static_limit() returns the limit.
 *   - Cost: every GPU that loads the library holds the 4 MiB until the process exits.
 *   - The array is ONE per device, shared by every call and every host thread, and keeps the last
 *     call's contents.  Nothing in it has to start at zero (every word a call reads it has written
 *     before), so no clearing is done.  Two calls that overlap on the GPU (different streams without
 *     an ordering between them) RACE on it: order them, or use krr_precision_map with own workspaces.
 * Arguments as krr_precision_map without d_ws / ws_bytes; inputs and outputs remain the caller's.
 */
#define KRR_PRECISION_MAP_STATIC_BYTES (4u << 20)
size_t krr_precision_map_static_limit(void);
int krr_precision_map_static(const float* d_A, int64_t n, int64_t lda, int nb,
                             float eps_target, unsigned allowed_mask, unsigned flags,
                             uint8_t* d_map, float* d_tile_norms, float* d_tile_amax, double* d_fro,
                             void* stream);

/* ---------------------------------------------------------------------------------------------
 * Factor storage (the tile mosaic).  Tile (i,j), i >= j, is a contiguous row-major
 * nb x nb block in its own precision (4, 2 or 1 bytes per element) at byte offset
 *     off(i,j) = sum of the byte sizes of all lower tiles preceding it in column-major tile order,
 * a pure function of (map, nb); every offset is a multiple of 128 bytes.  Diagonal tiles are FP32
 * full squares with zeros above the diagonal.  An FP8 tile holds E4M3 codes q with value
 * scales[i*NT+j] * q; the scale is a power of two (1.0 for FP32 / FP16 tiles).
 * krr_factor_bytes returns the payload size; krr_factor_tile_offset one tile's offset.
 * Both are pure host functions; they return 0 / -1 on invalid arguments.
 */
size_t  krr_factor_bytes(int64_t n, int nb, const uint8_t* h_map);
int64_t krr_factor_tile_offset(int64_t n, int nb, const uint8_t* h_map, int i, int j);

/* ---------------------------------------------------------------------------------------------
 * krr_potrf_mp -- mixed-precision tile Cholesky  A = L L^T  of A = K + lambda*I.
 * PAPER.md:112 (FACTORIZE), :192 (four-precision tile Cholesky; FP64 not required), :211 (E4M3 for
 * both operands), :206 (operands converted on the fly), :130/:159 (POTRF / TRSM / SYRK / GEMM).
 * Per tile column k:  S_kk = A_kk - sum_j L_kj L_kj^T, L_kk = chol(S_kk) in FP32;
 * S_ik = rd_p(A_ik) - sum_j L_ij L_kj^T accumulated in FP32 (tensor cores, operands as stored),
 * L_ik = rd_{p(i,k)}(S_ik L_kk^{-T}) -- each tile is rounded once, when its final value is stored.
 * d_A      in   as for krr_precision_map; not modified.
 * d_map / h_map in  the same map in device and host memory (the launch sequence is built on the
 *               host from h_map; kernels read d_map).  A mismatch is detected on the device: *d_info = -1, the
 *               factor is unspecified, nothing is written outside buffers sized from h_map.
 * d_factor out  krr_factor_bytes(n, nb, h_map) bytes, layout above.
 * d_scales out  NT*NT floats (row-major, scales[i*NT+j]); 1.0 except FP8 tiles; 0 above diagonal.
 * d_info   out  one int: 0 on success, j > 0 = 1-based scalar column of the first non-positive
 *               pivot (contents of later tile columns are then unspecified); -1: d_map and h_map differ;
 *               -2: the inverse of a diagonal tile left the range of its FP16 images (entries beyond 2^12 times
 *               1 / sqrt(max A_ii): the tile is too ill-conditioned for the product form of the panel TRSM).
 * Accuracy the panel below a diagonal tile is one product with the explicit inverse of that tile.  With an all-FP32
 *          map the backward error ||A - L L^T||_F / ||A||_F stays below 1e-6 at every admitted shape (measured up to
 *          nb = 4096); tiles above 1024 and matrices of at most four tile columns take a segmented-accumulation form
 *          of the product for that ("Accuracy of the product form").
 * d_ws     workspace, at least krr_potrf_mp_workspace(n, nb, h_map) bytes, 1024-byte aligned.
 *          It holds the FP16 operand images of L that the tensor-core kernels read and two FP32
 *          panel buffers; it may be released once the call has completed on `stream` (krr_potrs
 *          needs only d_factor / d_scales / d_map).
 * flags    KRR_FLAG_PREROUND_A, KRR_FLAG_A_TILED_LOWER, KRR_FLAG_NO_LOOKAHEAD.
 * Streams  the work is ordered after everything already enqueued on `stream`, and work enqueued on
 *          `stream` after the call is ordered after it.  Unless KRR_FLAG_NO_LOOKAHEAD is given the
 *          kernels run on three internal streams (created once per host thread, together with a
 *          pool of CUDA events) that fork from and join back into `stream`: the diagonal-tile
 *          chain of column k+1 starts as soon as tile (k+1,k) is stored and runs beside the
 *          trailing updates and the rest of column k's panel (PAPER.md:206 overlap of the DAG's
 *          tasks, :295 lookahead).  The result does not depend
 *          on timing (fixed summation order), but differs in the last bits between the two
 *          schedules (the newest column is added in the FP32 epilogue instead of in TMEM).
 */
size_t krr_potrf_mp_workspace(int64_t n, int nb, const uint8_t* h_map);
int krr_potrf_mp(const float* d_A, int64_t n, int64_t lda, int nb,
                 const uint8_t* d_map, const uint8_t* h_map,
                 void* d_factor, float* d_scales, int* d_info,
                 void* d_ws, size_t ws_bytes, unsigned flags, void* stream);

/* ---------------------------------------------------------------------------------------------
 * krr_potrs -- solve (L L^T) X = B by forward and backward substitution in FP32 (PAPER.md:114,
 * :169), with the tile mosaic produced by krr_potrf_mp (tiles dequantised on the fly).
 * d_B   in/out  n x nrhs FP32, ROW-major with leading dimension ldb >= nrhs (elements);
 *               in: Y (phenotypes), out: alpha (the weights W of PAPER.md:82).  1 <= nrhs <= 32 and
 *               nb * (nrhs rounded up to 4, 8, 16 or 32) <= 32768 (the solved block of one tile is
 *               kept in shared memory), else KRR_ERR_SHAPE.
 * d_ws  workspace of at least krr_potrs_workspace(n, nb, nrhs) bytes, 16-byte aligned: tile offsets, the inverses of
 *       the 128x128 diagonal blocks of L (2 * n * 128 floats), and from them the inverses of the whole diagonal
 *       tiles and their transposes (2 * n * nb floats, FP32 block forward substitution), computed by every call
 *       before the sweeps (the factor may have changed).  A diagonal step of a sweep is then one product
 *       z_k = inv(L_kk) t_k; the updates behind it run with a two-column lookahead on the library's three
 *       internal streams (the bulk of them streamed from d_factor by TMA; d_factor must be 16-byte aligned,
 *       else KRR_ERR_ARG); sums are accumulated in a fixed order
 *       (deterministic results).  If d_map does not agree with h_map the result is unspecified (all reads stay
 *       inside buffers sized from h_map).
 */
size_t krr_potrs_workspace(int64_t n, int nb, int nrhs);
int krr_potrs(const void* d_factor, const float* d_scales,
              const uint8_t* d_map, const uint8_t* h_map, int64_t n, int nb,
              float* d_B, int64_t ldb, int nrhs,
              void* d_ws, size_t ws_bytes, void* stream);

/* ---------------------------------------------------------------------------------------------
 * krr_refine -- iterative refinement of alpha with the factor kept fixed (R19).  The paper
 * names the technique and does not adopt it; it is the remedy SURVEY section 8(c)
 * offers where an FP16 / FP8 map misses "alpha to 1e-3".  A call beside the path: krr_potrf_mp and
 * krr_potrs never refine.  For s = 0 .. steps-1:
 *     R = fl32(Y - A X)   A, X in FP32, every product and sum in FP64, rounded once;
 *     D = krr_potrs(factor, R);   X = fl32(X + D).
 * d_A      in      as for krr_precision_map (dense row-major with lda, or KRR_FLAG_A_TILED_LOWER); only
 *                  the lower tiles are read, the diagonal blocks through their lower triangles.
 * d_factor, d_scales, d_map, h_map   in   the factor, as for krr_potrs.
 * d_Y      in      n x nrhs FP32 row-major, leading dimension ldy >= nrhs.
 * d_X      in/out  n x nrhs FP32 row-major, ldx >= nrhs: in alpha_0 (e.g. the result of krr_potrs), out
 *                  alpha_steps.  nrhs as for krr_potrs.
 * steps    0 .. 64.
 * d_resid  out     NULL, or steps + 1 doubles (device): d_resid[s] = ||fl32(Y - A alpha_s)||_F; asking for
 *                  them costs one more residual evaluation (that of alpha_steps).
 * d_ws     workspace of at least krr_refine_workspace(n, nb, nrhs) bytes, 1024-byte aligned.
 * flags    KRR_FLAG_A_TILED_LOWER only.
 * The residual is a fixed-order sum (deterministic).  Cost per step: the lower tiles of A read twice
 * (4 n^2 bytes), 2 n^2 nrhs FP64 flops, one krr_potrs.
 */
size_t krr_refine_workspace(int64_t n, int nb, int nrhs);
int krr_refine(const float* d_A, int64_t n, int64_t lda, int nb,
               const void* d_factor, const float* d_scales, const uint8_t* d_map, const uint8_t* h_map,
               const float* d_Y, int64_t ldy, float* d_X, int64_t ldx, int nrhs,
               int steps, double* d_resid,
               void* d_ws, size_t ws_bytes, unsigned flags, void* stream);

/* ---------------------------------------------------------------------------------------------
 * krr_pcg -- conjugate gradients on A alpha = Y preconditioned by the fixed factor, M = L L^T
 * (R20).  krr_refine contracts only while the spectral radius of I - M^-1 A is below one;
 * with the all-FP16 map the rule gives C4 it is not at n = 131072 (measured).  CG with the same M
 * converges for every SPD A and M at the same cost per step: one product with A (FP64 sums), one
 * krr_potrs.  Textbook recurrence, every right-hand side with its own scalars, started from d_X:
 *     r = Y - A x,  z = M^-1 fl32(r),  p = z,  rho = r.z;   then `iters` times
 *     q = A p,  a = rho / p.q,  x += a p,  r -= a q,  z = M^-1 fl32(r),  rho' = r.z,  p = fl32(z + (rho'/rho) p).
 * x, r, q and the inner products are FP64 (workspace); p and z FP32; a right-hand side with p.q <= 0 or
 * rho = 0 stops moving.  Arguments as for krr_refine, with
 * iters    0 .. 1024;
 * d_resid  out  NULL, or iters + 1 doubles: d_resid[k] = ||r_k||_F of the recursively updated residuals
 *               (no extra product with A).
 * d_ws     at least krr_pcg_workspace(n, nb, nrhs) bytes, 1024-byte aligned.
 * Deterministic (fixed-order sums).
 */
size_t krr_pcg_workspace(int64_t n, int nb, int nrhs);
int krr_pcg(const float* d_A, int64_t n, int64_t lda, int nb,
            const void* d_factor, const float* d_scales, const uint8_t* d_map, const uint8_t* h_map,
            const float* d_Y, int64_t ldy, float* d_X, int64_t ldx, int nrhs,
            int iters, double* d_resid,
            void* d_ws, size_t ws_bytes, unsigned flags, void* stream);

/* ---------------------------------------------------------------------------------------------
 * krr_associate_host -- the whole Associate phase (Alg. 3) from HOST buffers: copies A and Y to the
 * device arena, runs krr_precision_map -> krr_potrf_mp -> krr_potrs, copies alpha, the map and info
 * back, and synchronises `stream` before returning.  Used for end-to-end timing.
 * h_A      in   FP32 n x n row-major (lda) host memory (pinned memory makes the copies asynchronous); only the
 *               lower tiles (tile row i: its first (i+1)*nb columns) are read and copied: 4 nb^2 NT(NT+1)/2 bytes
 * h_Y      in   n x nrhs row-major; h_alpha out n x nrhs; h_map out NT*NT bytes; h_info out 1 int
 * force_prec    < 0: use the rule with (eps_target, allowed_mask); 0..2: uniform off-diagonal map
 * d_arena  device scratch of at least krr_associate_host_arena(n, nb, nrhs) bytes (sized for the
 *          worst-case map), 1024-byte aligned.
 */
size_t krr_associate_host_arena(int64_t n, int nb, int nrhs);
int krr_associate_host(const float* h_A, int64_t n, int64_t lda, int nb,
                       float eps_target, unsigned allowed_mask, int force_prec, unsigned flags,
                       const float* h_Y, int nrhs, float* h_alpha,
                       uint8_t* h_map, int* h_info,
                       void* d_arena, size_t arena_bytes, void* stream);

/* Host utility: the hand-tuned band map of [37] the paper compares its adaptive rule with: diagonal
 * tiles and the first ceil(fp32_fraction * (NT-1)) sub-diagonals of tiles FP32, the remaining off-diagonal tiles
 * `low_prec`; 255 above the diagonal.  h_map: NT*NT bytes.  Pure host code. */
int krr_band_map(int NT, double fp32_fraction, int low_prec, uint8_t* h_map);

/* ---------------------------------------------------------------------------------------------
 * krr_build -- Build phase (Alg. 2 :92-106 with the Gaussian kernel of Alg. 5 :136-143;
 * the method of V-B1 :173-190 and VI-B2 :207-209):
 *   A = K + lambda*I,  K_ij = exp(-gamma * ||g_i - g_j||^2),  g_i = row i of G,
 * with ||g_i - g_j||^2 = s_i + s_j - 2 <g_i, g_j>, the Gram matrix on the INT8 tensor cores (INT32
 * accumulation, exact), the squared norms s as one folded vector, each 256 x 256 block of squared
 * distances generated on chip and exponentiated before it is stored (no n x n integer temporary).
 * d_G    in   n x p signed 8-bit genotypes, row-major with row pitch ldg bytes (ldg >= p, ldg % 16 == 0,
 *             16-byte aligned); any int8 values (the workloads use {0,1,2}); p <= 133000 keeps the INT32
 *             sums exact.  Not modified.
 * d_C    in   optional confounders: n x q FP32 real-valued covariates, row-major (ldc), q <= 16;
 *             their squared distance sum_t (c_it - c_jt)^2 is accumulated in FP32 and added to the integer
 *             squared distance before the exponentiation.  NULL / q = 0: none.
 * gamma, lambda  kernel bandwidth and regulariser; the diagonal is (float)(1 + lambda) exactly.
 * d_A    out  the lower TILES of A (tile row >= tile column; diagonal tiles as full squares) in FP32:
 *             n x n row-major with lda (lda % 4 == 0; tiles above the diagonal are not written), or
 *             packed lower tiles with KRR_FLAG_A_TILED_LOWER -- the two input layouts of krr_precision_map
 *             and krr_potrf_mp.  exp is evaluated in FP32 (expf of the FP32 product gamma*d2, d2 exact):
 *             entries agree with the FP64-evaluated, FP32-rounded kernel to a few ulp.
 * n % 256 == 0, nb % 256 == 0, n % nb == 0.  d_ws: krr_build_workspace(n, p, flags) bytes (the folded vector s;
 * with KRR_FLAG_KERNEL_IBS also the encoded genotypes, n x 2p bytes).
 */
size_t krr_build_workspace(int64_t n, int64_t p, unsigned flags);
int krr_build(const int8_t* d_G, int64_t n, int64_t p, int64_t ldg, const float* d_C, int q, int64_t ldc,
              float gamma, float lambda, float* d_A, int64_t lda, int nb, unsigned flags,
              void* d_stats, void* d_ws, size_t ws_bytes, void* stream);

/* krr_build_bordered -- the same for a cohort whose size is no multiple of the tile size (R21; SURVEY 8(f)
 * NEXT-4 "ragged n"; the paper's cohort has 305,880 patients): n is the padded size (the next multiple of nb and of
 * 256), n_valid <= n the number of patients.  Rows >= n_valid of d_G (and d_C) must exist (n rows are read for the
 * folded norms) and are ignored; rows and columns >= n_valid of A are written as the identity border (1 on the
 * diagonal, 0 elsewhere), which changes nothing of the problem: chol = blockdiag(L, I), and with zero rows appended
 * to Y the first n_valid rows of krr_potrs's result are the solution, the rest exactly 0.  The tile statistics
 * (d_stats) are those of the bordered matrix.  krr_build(...) == krr_build_bordered(..., n_valid = n).
 */
int krr_build_bordered(const int8_t* d_G, int64_t n, int64_t n_valid, int64_t p, int64_t ldg, const float* d_C, int q,
                       int64_t ldc, float gamma, float lambda, float* d_A, int64_t lda, int nb, unsigned flags,
                       void* d_stats, void* d_ws, size_t ws_bytes, void* stream);

/* krr_build_rr -- the mixed INT8 / FP32 SYRK of ridge regression (Fig. 2; Eq. (2)):
 *     A = X^T X + lambda I,   X = [S^T | C]   (patients x (ns + q): SNPs, then confounders),
 * bordered by the identity up to n (R21; ns + q is rarely a multiple of the tile size).
 * d_S   in   the SNP features as rows: n x p int8, row-major with pitch lds (as d_G of krr_build: p = patients is the
 *            contraction dimension); rows >= ns must exist and are ignored.
 * d_C   in   p x q FP32 confounders, row-major (ldc >= q), q <= 16; NULL / q = 0: none.
 * d_A   out  as for krr_build (dense lower tiles or KRR_FLAG_A_TILED_LOWER).  The SNP x SNP block comes from the INT8
 *            tensor cores (exact integers, the INT8 tiles of Fig. 2); the q rows that involve a confounder are
 *            accumulated in FP32 (its FP32 tiles, SGEMM in the paper) in a fixed order; lambda is added on the diagonal.
 * d_ws       krr_build_workspace(n, p, 0) bytes.  Follow with krr_precision_map / krr_potrf_mp / krr_potrs on A and
 *            X^T Y (zero rows appended) for beta.
 */
int krr_build_rr(const int8_t* d_S, int64_t n, int64_t ns, int64_t p, int64_t lds, const float* d_C, int q, int64_t ldc,
                 float lambda, float* d_A, int64_t lda, int nb, unsigned flags, void* d_ws, size_t ws_bytes, void* stream);

/* Tile statistics from the Build epilogue ("tile sum-of-squares emitted in the same epilogue so
 * krr_precision_map needs no extra pass").  If krr_build is given d_stats (krr_build_stats_bytes(n, nb) bytes, 1024-byte
 * aligned; NULL: none) every epilogue warp also leaves the FP64 sum of squares and the maximum modulus of its share of A
 * there; krr_precision_map_from_build then sums them per tile in a fixed order and applies the rule exactly as
 * krr_precision_map does (same outputs; the norms agree to FP64 summation order).  d_stats is read and partly used as
 * scratch by krr_precision_map_from_build. */
size_t krr_build_stats_bytes(int64_t n, int nb);
int krr_precision_map_from_build(const void* d_stats, int64_t n, int nb, float eps_target, unsigned allowed_mask,
                                 uint8_t* d_map, float* d_tile_norms, float* d_tile_amax, double* d_fro, void* stream);

/* ---------------------------------------------------------------------------------------------
 * krr_predict -- Predict phase (Alg. 4 :116-122):
 *   K = BUILD(gamma, T, G): the N_P2 x N_P1 test-training kernel matrix, K_ij = exp(-gamma ||t_i - g_j||^2);
 *   P_r = K x W.
 * K is produced by the kernel of krr_build (INT8 tensor cores, every block of the rectangle, no
 * regulariser) into the workspace as FP32, then multiplied by W in FP32 (one warp per row of K, fixed
 * summation order).
 * d_T  in  m x p int8 test genotypes (row pitch ldt), d_G in n x p int8 training genotypes (ldg); both
 *          pitches multiples of 16 bytes, 16-byte aligned; m % 256 == 0, n % 256 == 0, p <= 133000.
 * d_CT, d_CG  in  optional confounders of the two cohorts (m x q, n x q FP32, ldct / ldcg), as for krr_build.
 * d_W  in  n x nrhs FP32 row-major (ldw): the weights of krr_potrs; nrhs <= 32.
 * d_P  out m x nrhs FP32 row-major (ldp): the predicted phenotypes.
 * flags    0 or KRR_FLAG_KERNEL_IBS.
 * d_ws     krr_predict_workspace(m, n, p, flags) bytes, 1024-byte aligned; on return it holds, after the two
 *          folded norm vectors (each rounded up to 1 KiB), K as m x n FP32 row-major.
 */
size_t krr_predict_workspace(int64_t m, int64_t n, int64_t p, unsigned flags);
int krr_predict(const int8_t* d_T, int64_t m, int64_t ldt, const int8_t* d_G, int64_t n, int64_t ldg, int64_t p,
                const float* d_CT, int64_t ldct, const float* d_CG, int64_t ldcg, int q,
                float gamma, const float* d_W, int64_t ldw, int nrhs, float* d_P, int64_t ldp,
                unsigned flags, void* d_ws, size_t ws_bytes, void* stream);

/* ---------------------------------------------------------------------------------------------
 * krr_fit_host -- Build and Associate (Alg. 1 l.2-3) from HOST buffers: copies the int8 genotypes
 * and Y to the device, builds A = K + lambda*I there (krr_build, Gaussian kernel), then runs the Associate phase as
 * krr_associate_host does and copies alpha (= W), the precision map and info back.  The n x n matrix never crosses
 * PCIe: n*p bytes of genotypes do.  The genotypes are copied in strips of whole tile rows on one of the library's internal
 * streams and the rows of A a strip completes are built on `stream` as soon as it has arrived (the Build runs behind the
 * copy; same blocks and arithmetic as one krr_build call: identical bits).  Synchronises `stream` before it returns.
 * h_G  in  n x p int8 genotypes, row pitch ldg >= p bytes (pinned memory makes the copy asynchronous).
 * Other arguments as for krr_build / krr_associate_host; n % 256 == 0, nb % 256 == 0.
 * d_arena  krr_fit_host_arena(n, p, nb, nrhs) bytes, 1024-byte aligned.
 */
size_t krr_fit_host_arena(int64_t n, int64_t p, int nb, int nrhs);
int krr_fit_host(const int8_t* h_G, int64_t n, int64_t p, int64_t ldg, float gamma, float lambda, int nb,
                 float eps_target, unsigned allowed_mask, int force_prec, unsigned flags,
                 const float* h_Y, int nrhs, float* h_alpha, uint8_t* h_map, int* h_info,
                 void* d_arena, size_t arena_bytes, void* stream);

/* ---------------------------------------------------------------------------------------------
 * CUDA-graph replay of the tile-DAG launch sequence (BASELINE.json north_star: "a single-GPU tile-DAG scheduler with
 * lookahead, run as CUDA graphs"; PAPER.md:206 task DAG, :295 lookahead).  The launch sequence of krr_potrf_mp /
 * krr_potrs / krr_refine / krr_pcg is a pure function of (n, nb, map, flags, pointers): krr_graph_begin puts `stream`
 * into stream capture, the krr_* calls made on it afterwards are recorded instead of run (their fork / join onto the
 * library's internal priority streams becomes the parallel branches of the graph), krr_graph_end instantiates what
 * was recorded.  krr_graph_launch replays it on any stream: same kernels, same arguments, same dependencies, so the
 * results are bit-identical to the direct calls; the buffers the recorded calls were given must stay allocated and
 * hold the inputs (A, map, Y) at replay time.  A graph is valid for ONE precision map: when krr_precision_map returns
 * another map, record again.
 * stream      must not be the legacy default stream (CUDA cannot capture it): KRR_ERR_ARG.
 * Calls that synchronise (krr_associate_host, krr_fit_host, krr_profile_read) must not be recorded; per-kernel timing
 * (krr_profile_enable) must be off: KRR_ERR_UNSUPPORTED.
 * krr_graph_end returns KRR_ERR_CUDA when a recorded call failed (the capture is then discarded, *out = NULL).
 * krr_graph_kernel_nodes: kernels one replay launches (for bench.py's gpu_launches).
 * The graph object is host memory owned by the library until krr_graph_destroy. */
typedef struct krr_graph krr_graph_t;
int krr_graph_begin(void* stream);
int krr_graph_end(void* stream, krr_graph_t** out);
int krr_graph_launch(const krr_graph_t* graph, void* stream);
int64_t krr_graph_kernel_nodes(const krr_graph_t* graph);
int krr_graph_destroy(krr_graph_t* graph);

/* Number of kernels the last krr_* call on this thread enqueued (for bench.py's gpu_launches). */
int64_t krr_last_launch_count(void);

/* Optional per-kernel timing for measurement (bench.py's roofline object): while a category's bit
 * is set in category_mask, every launch of that category made by this host thread is bracketed by
 * CUDA events on the launching stream.  Categories: 0 trailing SYRK/GEMM update (tcgen05),
 * 1 in-panel update, 2 panel TRSM product, 3 FP32 POTRF of a 128 block, 4 quantising store,
 * 5 precision map, 6 POTRS, 7 misc.  krr_profile_enable(mask) also clears the records (0 = off).
 * krr_profile_read synchronises on the recorded events and returns the summed device time and the
 * number of launches of one category.  This is the only place the library creates CUDA events. */
int krr_profile_enable(unsigned category_mask);
int krr_profile_read(int category, double* total_ms, int64_t* launches);

/* Timeline of the tile-column pipeline of the LAST krr_potrf_mp call of this host thread that ran
 * the lookahead schedule (NT > 2, no KRR_FLAG_NO_LOOKAHEAD, not recorded into a graph), read before any other krr_* call:
 * h_ms[4k + 0..3] = device time in ms since the call forked onto the internal streams at which, for tile column k,
 *   0  the critical stream finished the diagonal-tile chain and the TRSM / store of tile (k+1, k),
 *   1  the bulk stream finished O(k) (terms s < k-1 of column k),
 *   2  the bulk stream finished N(k) (newest term on the rows below the diagonal tile),
 *   3  the panel stream finished P(k) and F(k) (TRSM and store of the remaining rows);
 * -1 where the event was not recorded (O(k) for k < 2, ...).  Waits for the call to finish.  h_ms: host, 4*NT floats. */
int krr_profile_timeline(int NT, float* h_ms);

/* ---------------------------------------------------------------------------------------------
 * krr_peak_probe -- roofline denominators measured on the current device (SURVEY 8(d) "Which roofline": "FP8 =
 * measure with a no-traffic kind::f8f6f4 loop ... FP32 ALU = measure an FFMA loop").  Beside the path; used by
 * bench.py --peaks and paper_2409_01712_b200/peaks.py.
 * kind   0  tcgen05 kind::f16 on CTA pairs (cta_group::2, M = N = 256, K = 16 per instruction), operands resident
 *           in shared memory (pseudo-random finite data, four ring slots), accumulator in TMEM, no global traffic
 *        1  the same with kind::f8f6f4 (E4M3 x E4M3, K = 32 per instruction)
 *        2  the same with kind::mxf8f6f4.block_scale (UE8M0 scales 2^0 from TMEM) -- the FP8 x FP8 instruction of
 *           krr_potrf_mp
 *        3  FFMA: 8 independent chains per thread, 1024 threads per CTA, 2 CTAs per SM
 *        4  the three-instruction FP32-class sequence of krr_potrf_mp (hi*hi + lo*hi + hi*lo on kind::f16)
 * work   tensor kinds: 128-byte K slices ("chunks", 4 instructions each; kind 4: 12) per CTA pair, a multiple of 16;
 *        FFMA: loop iterations (128 FMAs per thread each).
 * h_ms   out  device time of the one launch (CUDA events); h_flops out  the flops it performed (2 per multiply-add;
 *        kind 4: of all three instructions).  Synchronises `stream`. */
int krr_peak_probe(int kind, int64_t work, float* h_ms, double* h_flops, void* stream);

/* ---------------------------------------------------------------------------------------------
 * krr_dist_schedule -- the per-rank task and message schedule of the factorisation over `world` GPUs of one NVSwitch
 * domain (SURVEY 8(e) / 8(f) NEXT-3; PAPER.md:206 overlap of communication and computation, :291-295 strong scaling).
 * HOST LOGIC ONLY: pure function of (NT, nb, map, world, rank); nothing is launched.  krr_potrf_mp itself runs on one GPU;
 * this is the partitioning a multi-GPU driver follows and what the world-size-2 gloo test checks.
 * Tile row i belongs to rank i mod world.  Records of 6 int32 {op, k, root, nrows, bytes_lo, bytes_hi}, in issue order:
 *   op 1  diagonal-tile chain + inverse of column k (only on its owner)      op 5  broadcast of M_k = inv(L_kk) from owner(k)
 *   op 2  newest term N(k) on this rank's nrows tile rows below tile (k,k)    op 6  broadcast of tile (k+1,k) from owner(k+1)
 *   op 3  older terms O(k) of column k (lookahead) on nrows rows              op 7  all-gather of the tiles (i,k), i > k+1
 *   op 4  TRSM product T(k) and quantising store on nrows rows                      (nrows = tiles this rank contributes)
 * bytes = what one rank receives, in STORAGE precision (the mosaic is what travels: PAPER.md:192, :206).
 * h_tasks NULL: only the count is returned.  Returns the number of records, or a KRR_ERR_* code (< 0). */
int64_t krr_dist_schedule(int NT, int nb, const uint8_t* h_map, int world, int rank, int32_t* h_tasks, int64_t max_tasks);

/* krr_shutdown -- destroy what the library created for the calling host thread on the current device: the three
 * internal priority streams of the lookahead schedule, the pool of CUDA events (pipeline events and the timing
 * events of krr_profile_*).  Everything the thread enqueued must have completed.  The next krr_* call creates them
 * again.  These streams and events are the only resources the library ever allocates (no device memory). */
int krr_shutdown(void);

#ifdef __cplusplus
}
#endif
#endif /* KRR_MP_H */

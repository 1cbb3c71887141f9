// C ABI of the library (include/krr_mp.h): argument checks, workspace layout, and the host-side
// launch sequence of the tile-column pipeline.  Everything numerical runs in the kernels of
// precision_map.cuh, gemm_tc.cuh, panel.cuh and potrs.cuh.
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <vector>

#include "build.cuh"
#include "common.cuh"
#include "dist_schedule.cuh"
#include "gemm_tc.cuh"
#include "panel.cuh"
#include "peaks.cuh"
#include "potrs.cuh"
#include "potrs_stream.cuh"
#include "precision_map.cuh"
#include "refine.cuh"
#include "tri128.cuh"

namespace krr {

thread_local int64_t g_launches = 0;

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

static int check_device(int* num_sms) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return KRR_ERR_CUDA;
    int major = 0, sms = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) return KRR_ERR_CUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return KRR_ERR_CUDA;
    if (major != 10) return KRR_ERR_DEVICE;
    if (num_sms) *num_sms = sms;
    return KRR_OK;
}

static int check_shape(int64_t n, int nb) {
    if (n <= 0 || nb <= 0) return KRR_ERR_ARG;
    if (nb % kBlk != 0 || n % nb != 0 || nb > 4096) return KRR_ERR_SHAPE;
    if (n / nb > kMaxNT) return KRR_ERR_SHAPE;
    return KRR_OK;
}

static int check_map(int NT, const uint8_t* h_map, bool* any_fp8) {
    bool f8 = false;
    for (int i = 0; i < NT; ++i)
        for (int j = 0; j <= i; ++j) {
            const uint8_t p = h_map[i * NT + j];
            if (p > KRR_FP8_E4M3) return KRR_ERR_MAP;
            if (i == j && p != KRR_FP32) return KRR_ERR_MAP;
            f8 |= (p == KRR_FP8_E4M3);
        }
    if (any_fp8) *any_fp8 = f8;
    return KRR_OK;
}

// ---- tensor maps ---------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (fn) return fn;
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
        return nullptr;
    fn = reinterpret_cast<EncodeTiledFn>(p);
    return fn;
}

// Row-major [rows][cols] array of 2-byte elements, box = 64 columns x 128 rows, 128-byte swizzle.
static int make_plane_tmap(CUtensorMap* tm, const void* base, uint64_t rows, uint64_t cols, int box_rows = kBlk) {
    EncodeTiledFn enc = get_encode_fn();
    if (!enc) return KRR_ERR_CUDA;
    cuuint64_t gdim[2] = {cols, rows};
    cuuint64_t gstride[1] = {cols * 2};
    cuuint32_t box[2] = {static_cast<cuuint32_t>(kBlockK), static_cast<cuuint32_t>(box_rows)};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, const_cast<void*>(base), gdim, gstride, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? KRR_OK : KRR_ERR_CUDA;
}

// Row-major [rows][cols] array of bytes (E4M3 images), box = 128 columns x 128 rows, 128-byte swizzle.
static int make_byte_plane_tmap(CUtensorMap* tm, const void* base, uint64_t rows, uint64_t cols, int box_rows = kBlk) {
    EncodeTiledFn enc = get_encode_fn();
    if (!enc) return KRR_ERR_CUDA;
    cuuint64_t gdim[2] = {cols, rows};
    cuuint64_t gstride[1] = {cols};
    cuuint32_t box[2] = {128u, static_cast<cuuint32_t>(box_rows)};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void*>(base), gdim, gstride, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? KRR_OK : KRR_ERR_CUDA;
}

// The mosaic payload as a 2-D array of es-byte elements with nb columns (potrs_stream.cuh): box = bc columns x br rows.
static int make_mosaic_tmap(CUtensorMap* tm, const void* base, size_t payload_bytes, int nb, int es, int bc, int br, bool swizzle128) {
    EncodeTiledFn enc = get_encode_fn();
    if (!enc) return KRR_ERR_CUDA;
    cuuint64_t gdim[2] = {static_cast<cuuint64_t>(nb), payload_bytes / (static_cast<size_t>(nb) * es)};
    cuuint64_t gstride[1] = {static_cast<cuuint64_t>(nb) * es};
    cuuint32_t box[2] = {static_cast<cuuint32_t>(bc), static_cast<cuuint32_t>(br)};
    cuuint32_t estr[2] = {1, 1};
    const CUtensorMapDataType dt = es == 4 ? CU_TENSOR_MAP_DATA_TYPE_UINT32 : (es == 2 ? CU_TENSOR_MAP_DATA_TYPE_UINT16 : CU_TENSOR_MAP_DATA_TYPE_UINT8);
    CUresult r = enc(tm, dt, 2, const_cast<void*>(base), gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                     swizzle128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? KRR_OK : KRR_ERR_CUDA;
}

// ---- mosaic offsets (host) -------------------------------------------------------------------
static uint64_t host_map_hash(int NT, const uint8_t* h_map) {
    uint64_t h = kMapHashSeed;
    for (int j = 0; j < NT; ++j)
        for (int i = j; i < NT; ++i) h = map_hash_step(h, h_map[i * NT + j]);
    return h;
}

static size_t host_offsets(int NT, int nb, const uint8_t* h_map, std::vector<int64_t>* off) {
    size_t acc = 0;
    const size_t elems = static_cast<size_t>(nb) * nb;
    if (off) off->assign(static_cast<size_t>(NT) * NT, -1);
    for (int j = 0; j < NT; ++j)
        for (int i = j; i < NT; ++i) {
            if (off) (*off)[static_cast<size_t>(i) * NT + j] = static_cast<int64_t>(acc);
            acc += elems * prec_bytes(h_map[i * NT + j]);
        }
    return acc;
}

// ---- workspace layout of krr_potrf_mp ----------------------------------------------------------
constexpr int kMaxSkUnits = 128;                     // CTA pairs of a stream-K launch (half the SMs of any sm_100 part)
struct PotrfWs {
    size_t off_table, lrow, qrow, a_amax, tile_amax, scl, dscale, prog, split, sk_partial, W, W2, linv_hi, linv_lo, Sh, Sl, Hp, Lp, Qp, total;
};
// rows of the scratch planes: S of the panel rows, then two sets (tile-column parity) of M, M^T, U
static inline size_t scratch_rows(int64_t n, int nb) { return static_cast<size_t>(n) + 6 * static_cast<size_t>(nb); }
// The operand images are sized from the map (the mosaic "reduces memory footprint"): the hi image for every
// lower tile, the lo image only for FP32 tiles, the E4M3 image only for FP8 tiles (n_fp32 / n_fp8 = their counts; at least
// one tile's worth each, so that the tensor maps stay valid).
static void count_tiles(int NT, const uint8_t* h_map, size_t* n_fp32, size_t* n_fp8) {
    size_t a = 0, b = 0;
    for (int i = 0; i < NT; ++i)
        for (int j = 0; j <= i; ++j) {
            a += (h_map[i * NT + j] == KRR_FP32);
            b += (h_map[i * NT + j] == KRR_FP8_E4M3);
        }
    *n_fp32 = a; *n_fp8 = b;
}
static PotrfWs potrf_ws_layout(int64_t n, int nb, size_t n_fp32, size_t n_fp8) {
    const int64_t NT = n / nb;
    const size_t nslots = static_cast<size_t>(NT) * (NT + 1) / 2;
    const size_t plane = nslots * nb * nb;
    const size_t tile = static_cast<size_t>(nb) * nb;
    PotrfWs w;
    size_t o = 0;
    w.off_table = o; o = align_up(o + NT * NT * sizeof(int64_t), 1024);
    w.lrow = o;      o = align_up(o + NT * NT * sizeof(int), 1024);
    w.qrow = o;      o = align_up(o + NT * NT * sizeof(int), 1024);
    w.a_amax = o;    o = align_up(o + NT * NT * sizeof(float), 1024);
    w.tile_amax = o; o = align_up(o + nslots * sizeof(float), 1024);
    w.scl = o;       o = align_up(o + (SCL_COUNT + 2 * (nb / kBlk)) * sizeof(float), 1024);
    w.dscale = o;    o = align_up(o + static_cast<size_t>(NT) * sizeof(float), 1024);        // equilibration of the tile rows
    w.prog = o;      o = align_up(o + static_cast<size_t>(n / kBlk) * sizeof(int), 1024);   // fused-chain progress, per 128-block
    w.split = o;     o = align_up(o + 1024 * sizeof(int), 1024);                             // stream-K: partial-sum flags, one per unit
    w.sk_partial = o; o = align_up(o + static_cast<size_t>(kMaxSkUnits) * 4 * kBlk * kBlk * sizeof(float), 1024);   // ... and one 256 x 256 block each
    w.W = o;         o = align_up(o + static_cast<size_t>(n) * nb * sizeof(float), 1024);
    w.W2 = o;        o = align_up(o + static_cast<size_t>(n) * nb * sizeof(float), 1024);   // lookahead: column k+1's partial
    w.linv_hi = o;   o = align_up(o + 2 * static_cast<size_t>(nb) * kBlk * 2, 1024);   // two sets (column parity)
    w.linv_lo = o;   o = align_up(o + 2 * static_cast<size_t>(nb) * kBlk * 2, 1024);
    w.Sh = o;        o = align_up(o + scratch_rows(n, nb) * nb * 2, 1024);
    w.Sl = o;        o = align_up(o + scratch_rows(n, nb) * nb * 2, 1024);
    w.Hp = o;        o = align_up(o + plane * 2, 1024);
    w.Lp = o;        o = align_up(o + (n_fp32 ? n_fp32 : 1) * tile * 2, 1024);
    w.Qp = o;        o = align_up(o + (n_fp8 ? n_fp8 : 1) * tile, 1024);
    w.total = o;
    return w;
}

// ---- per host thread and device: internal streams, event pool, timing records, one-time kernel attributes ----
// (the only resources the library creates; krr_shutdown destroys them)
enum { CAT_UPDATE = 0, CAT_P1 = 1, CAT_P3 = 2, CAT_POTRF = 3, CAT_FINALIZE = 4, CAT_MAP = 5, CAT_POTRS = 6,
       CAT_MISC = 7, CAT_COUNT = 8 };
struct TimedLaunch { int cat; cudaEvent_t e0, e1; };

// Internal streams of the tile-column pipeline (lookahead): `hi` carries the critical path (diagonal-tile chain,
// panel, store), `lo` the bulk updates that run ahead; both are fenced by events against the caller's stream,
// which is never blocked on the host.
struct Pipeline {
    cudaStream_t hi = nullptr, mid = nullptr, lo = nullptr;
    std::vector<cudaEvent_t> ev;
    cudaEvent_t event(size_t i) {
        while (ev.size() <= i) {
            cudaEvent_t e = nullptr;
            cudaEventCreate(&e);                 // timing enabled: krr_profile_timeline reads them
            ev.push_back(e);
        }
        return ev[i];
    }
    int init() {
        if (hi) return KRR_OK;
        int least = 0, greatest = 0;
        KRR_CUDA_CHECK(cudaDeviceGetStreamPriorityRange(&least, &greatest));
        KRR_CUDA_CHECK(cudaStreamCreateWithPriority(&hi, cudaStreamNonBlocking, greatest));
        KRR_CUDA_CHECK(cudaStreamCreateWithPriority(&mid, cudaStreamNonBlocking, (least + greatest) / 2));
        KRR_CUDA_CHECK(cudaStreamCreateWithPriority(&lo, cudaStreamNonBlocking, least));
        return KRR_OK;
    }
    void destroy() {
        for (cudaEvent_t e : ev) cudaEventDestroy(e);
        ev.clear();
        if (hi) cudaStreamDestroy(hi);
        if (mid) cudaStreamDestroy(mid);
        if (lo) cudaStreamDestroy(lo);
        hi = mid = lo = nullptr;
    }
};

constexpr int kMaxDevices = 64;
struct DeviceState {
    Pipeline pipe;
    unsigned prof_mask = 0;
    std::vector<TimedLaunch> prof;
    std::vector<cudaEvent_t> event_pool;
    bool attrs_done = false, build_attrs_done = false, peak_attrs_done = false;
};
static thread_local DeviceState g_dev_state[kMaxDevices];
static DeviceState& dev_state() {
    int dev = 0;
    cudaGetDevice(&dev);
    return g_dev_state[(dev >= 0 && dev < kMaxDevices) ? dev : 0];
}
#define g_pipe (dev_state().pipe)

static cudaEvent_t pool_event(DeviceState& d) {
    if (!d.event_pool.empty()) { cudaEvent_t e = d.event_pool.back(); d.event_pool.pop_back(); return e; }
    cudaEvent_t e = nullptr;
    cudaEventCreate(&e);
    return e;
}
struct ProfScope {
    bool on; TimedLaunch t; cudaStream_t st; DeviceState* d;
    ProfScope(int cat, cudaStream_t s) : st(s), d(&dev_state()) {
        on = (d->prof_mask >> cat) & 1u;
        if (on) { t.cat = cat; t.e0 = pool_event(*d); t.e1 = pool_event(*d); cudaEventRecord(t.e0, st); }
    }
    ~ProfScope() { if (on) { cudaEventRecord(t.e1, st); d->prof.push_back(t); } }
};

template <typename K, typename... Args>
static int launch(int cat, K kernel, dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
    ProfScope ps(cat, st);
    kernel<<<grid, block, smem, st>>>(args...);
    ++g_launches;
    return cudaGetLastError() == cudaSuccess ? KRR_OK : KRR_ERR_CUDA;
}

// The same as a programmatic dependent of the kernel before it in the stream (common.cuh pdl_trigger / pdl_wait): the
// kernel's prologue runs beside that kernel's tail.  Only for kernels that call pdl_wait() before they touch its output.
template <typename... KArgs, typename... Args>
static int launch_pdl(int cat, void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
    ProfScope ps(cat, st);
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    ++g_launches;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...) == cudaSuccess ? KRR_OK : KRR_ERR_CUDA;
}

// The tensor maps of one factorisation: hi/lo FP16 images of L (128-row boxes for A operands and for
// single-CTA B operands, 64-row boxes for the B halves of CTA pairs), the inverted diagonal blocks,
// and the E4M3 images.
struct GemmMaps { CUtensorMap H, L, IH[2], IL[2], Q, SH, SL; };

// cg = 2 runs MODE_UPDATE on CTA pairs (256 x 256 output blocks); needs even block counts.
struct StreamK { int* flags; float* partial; };      // workspace of the K-split of an update's last wave (null: whole blocks only)

static int launch_gemm(const GemmMaps& m, const GemmOp& op_in, int max_ctas, int cg, cudaStream_t st, int linv_buf = 0,
                       const StreamK* sk = nullptr) {
    GemmOp op = op_in;
    if (op.nrb <= 0 || op.ncb <= 0) return KRR_OK;
    // MODE_TRSM counts as panel_trsm; the fused diagonal chain (MODE_DIAG, POTRF included) and the inverse's recursion as potrf128
    ProfScope ps(op.mode == MODE_UPDATE ? CAT_UPDATE : (op.mode == MODE_P1 ? CAT_P1 : ((op.mode == MODE_DIAG || op.mode == MODE_INV) ? CAT_POTRF : CAT_P3)), st);
    ++g_launches;
    if (cg == 2 && (op.mode == MODE_UPDATE || op.mode == MODE_TRSM) && op.nrb % 2 == 0 && op.rb0 % 2 == 0 && op.ncb % 2 == 0 &&
        op.cb0 % 2 == 0) {
        const int npairs = (op.nrb / 2) * (op.ncb / 2);
        const int max_pairs = max_ctas / 2;
        const int grid = 2 * (npairs < max_pairs ? npairs : max_pairs);
        if (sk && op.mode == MODE_UPDATE && npairs > max_pairs && op.s_hi - op.s_lo >= 2) {
            op.sk = 1; op.sk_flags = sk->flags; op.sk_partial = sk->partial;
            if (cudaMemsetAsync(sk->flags, 0, static_cast<size_t>(max_pairs) * sizeof(int), st) != cudaSuccess) return KRR_ERR_CUDA;
        }
        cudaLaunchConfig_t cfg;
        memset(&cfg, 0, sizeof(cfg));
        cfg.gridDim = dim3(grid); cfg.blockDim = dim3(kGemmThreads); cfg.dynamicSmemBytes = kGemmSmem; cfg.stream = st;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr; cfg.numAttrs = 1;
        const cudaError_t e = cudaLaunchKernelEx(&cfg, gemm_tc_kernel<2>, m.H, m.L, m.IH[0], m.IL[0], m.Q, m.SH, m.SL, op);
        if (e != cudaSuccess && getenv("KRR_DEBUG")) fprintf(stderr, "krr: gemm_tc_kernel<2> launch: %s\n", cudaGetErrorString(e));
        return e == cudaSuccess ? KRR_OK : KRR_ERR_CUDA;
    }
    // MODE_DIAG: one CTA per row block of the diagonal tile; MODE_INV: one per 128 x 128 block of the level's products
    int ntiles = op.nrb * op.ncb;
    if (op.mode == MODE_DIAG) ntiles = op.nrb;
    if (op.mode == MODE_INV) {
        ntiles = op.node.hl * op.node.hr * (op.inv_step == 0 ? 1 : (op.inv_last ? 1 : 2));
        if (ntiles == 0) return KRR_OK;
    }
    const int grid = ntiles < max_ctas ? ntiles : max_ctas;
    gemm_tc_kernel<1><<<grid, kGemmThreads, kGemmSmem, st>>>(m.H, m.L, m.IH[linv_buf], m.IL[linv_buf], m.Q, m.SH, m.SL, op);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess && getenv("KRR_DEBUG")) fprintf(stderr, "krr: gemm_tc_kernel<1> launch (mode %d): %s\n", op.mode, cudaGetErrorString(e));
    return e == cudaSuccess ? KRR_OK : KRR_ERR_CUDA;
}

template <int NRHS>
static int set_potrs_attrs() {
    const int big = 227 * 1024;
    KRR_CUDA_CHECK(cudaFuncSetAttribute(potrs_fwd_update_kernel<NRHS>, cudaFuncAttributeMaxDynamicSharedMemorySize, big));
    KRR_CUDA_CHECK(cudaFuncSetAttribute(potrs_bwd_update_kernel<NRHS, (NRHS <= 16) ? 4 : 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, big));
    KRR_CUDA_CHECK(cudaFuncSetAttribute(potrs_bwd_update_kernel<NRHS, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, big));
    KRR_CUDA_CHECK(cudaFuncSetAttribute(potrs_stream_update_kernel<NRHS, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, big));
    KRR_CUDA_CHECK(cudaFuncSetAttribute(potrs_stream_update_kernel<NRHS, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, big));
    return KRR_OK;
}

static int set_kernel_attrs() {
    bool& done = dev_state().attrs_done;
    if (done) return KRR_OK;
    KRR_CUDA_CHECK(cudaFuncSetAttribute(gemm_tc_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kGemmSmem));
    KRR_CUDA_CHECK(cudaFuncSetAttribute(gemm_tc_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, kGemmSmem));
    KRR_CUDA_CHECK(cudaFuncSetAttribute(potrf128_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kTriSmem));
    KRR_CUDA_CHECK(cudaFuncSetAttribute(trtri128_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kTriSmem));
    KRR_CUDA_CHECK(cudaFuncSetAttribute(potrs_tile_inverse_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kTinvSmem));
    if (set_potrs_attrs<4>() || set_potrs_attrs<8>() || set_potrs_attrs<16>() || set_potrs_attrs<32>()) return KRR_ERR_CUDA;
    done = true;
    return KRR_OK;
}

// ---- scratch of krr_precision_map_static: a file-scope device array (no allocation at call time) --------------
// In host code `g_pm_static_scratch` is only a stand-in for the symbol, not a device address: the address is looked up
// once per device, with that device current, by cudaGetSymbolAddress, and that pointer is what the kernels receive.
static __device__ __align__(256) unsigned char g_pm_static_scratch[KRR_PRECISION_MAP_STATIC_BYTES];
static std::mutex g_pm_static_mutex;
static void* g_pm_static_ptr[kMaxDevices];          // per device ordinal; process-wide (the array is per device, not per thread)

static int pm_static_scratch(void** out) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return KRR_ERR_CUDA;
    if (dev < 0 || dev >= kMaxDevices) return KRR_ERR_DEVICE;
    std::lock_guard<std::mutex> lock(g_pm_static_mutex);
    if (!g_pm_static_ptr[dev]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_pm_static_scratch);
        if (e != cudaSuccess || !p) {
            if (getenv("KRR_DEBUG")) fprintf(stderr, "krr: cudaGetSymbolAddress(g_pm_static_scratch): %s\n", cudaGetErrorString(e));
            cudaGetLastError();
            return KRR_ERR_CUDA;
        }
        g_pm_static_ptr[dev] = p;
    }
    *out = g_pm_static_ptr[dev];
    return KRR_OK;
}

}  // namespace krr

using namespace krr;

extern "C" {

int krr_version(void) { return 100; }
int krr_built_for_sm(void) { return 100; }
int64_t krr_last_launch_count(void) { return g_launches; }

int krr_profile_enable(unsigned category_mask) {
    DeviceState& d = dev_state();
    for (auto& t : d.prof) { d.event_pool.push_back(t.e0); d.event_pool.push_back(t.e1); }
    d.prof.clear();
    d.prof_mask = category_mask;
    return KRR_OK;
}

int krr_shutdown(void) {
    DeviceState& d = dev_state();
    for (auto& t : d.prof) { cudaEventDestroy(t.e0); cudaEventDestroy(t.e1); }
    d.prof.clear();
    d.prof_mask = 0;
    for (cudaEvent_t e : d.event_pool) cudaEventDestroy(e);
    d.event_pool.clear();
    d.pipe.destroy();
    return cudaGetLastError() == cudaSuccess ? KRR_OK : KRR_ERR_CUDA;
}

int krr_profile_read(int category, double* total_ms, int64_t* launches) {
    if (category < 0 || category >= CAT_COUNT || !total_ms || !launches) return KRR_ERR_ARG;
    double ms = 0.0;
    int64_t cnt = 0;
    for (auto& t : dev_state().prof) {
        if (t.cat != category) continue;
        if (cudaEventSynchronize(t.e1) != cudaSuccess) return KRR_ERR_CUDA;
        float f = 0.f;
        if (cudaEventElapsedTime(&f, t.e0, t.e1) != cudaSuccess) return KRR_ERR_CUDA;
        ms += f;
        ++cnt;
    }
    *total_ms = ms;
    *launches = cnt;
    return KRR_OK;
}

// ------------------------------------------------------------------------- CUDA-graph replay
// Stream capture of the launch sequence (include/krr_mp.h): the fork / join of krr_potrf_mp and krr_potrs onto the
// internal priority streams is the capture-compatible pattern (event recorded on the capturing stream, waited for by
// the others, all joined back before the end), so the three streams become parallel branches of one graph and the
// kernel nodes keep the priority of the stream they were recorded on.
struct krr_graph { cudaGraph_t graph; cudaGraphExec_t exec; int64_t kernels; };

int krr_graph_begin(void* stream) {
    if (!stream) return KRR_ERR_ARG;                     // the legacy default stream cannot be captured
    if (dev_state().prof_mask) return KRR_ERR_UNSUPPORTED;  // timing events cannot be read back from a capture
    int num_sms = 0;
    int rc = check_device(&num_sms);
    if (rc) return rc;
    rc = set_kernel_attrs();                             // everything that is not a stream operation happens before
    if (rc) return rc;
    rc = g_pipe.init();
    if (rc) return rc;
    KRR_CUDA_CHECK(cudaStreamBeginCapture(static_cast<cudaStream_t>(stream), cudaStreamCaptureModeRelaxed));
    return KRR_OK;
}

int krr_graph_end(void* stream, krr_graph_t** out) {
    if (!stream || !out) return KRR_ERR_ARG;
    *out = nullptr;
    cudaGraph_t g = nullptr;
    if (cudaStreamEndCapture(static_cast<cudaStream_t>(stream), &g) != cudaSuccess || !g) {
        cudaGetLastError();                              // a failed capture leaves a sticky-looking error behind
        return KRR_ERR_CUDA;
    }
    size_t nn = 0;
    int64_t kernels = 0;
    if (cudaGraphGetNodes(g, nullptr, &nn) == cudaSuccess && nn > 0) {
        std::vector<cudaGraphNode_t> nodes(nn);
        if (cudaGraphGetNodes(g, nodes.data(), &nn) == cudaSuccess)
            for (size_t i = 0; i < nn; ++i) {
                cudaGraphNodeType t;
                if (cudaGraphNodeGetType(nodes[i], &t) == cudaSuccess && t == cudaGraphNodeTypeKernel) ++kernels;
            }
    }
    cudaGraphExec_t x = nullptr;
    if (cudaGraphInstantiate(&x, g, 0) != cudaSuccess) {
        cudaGraphDestroy(g);
        cudaGetLastError();
        return KRR_ERR_CUDA;
    }
    *out = new krr_graph{g, x, kernels};
    return KRR_OK;
}

int krr_graph_launch(const krr_graph_t* graph, void* stream) {
    if (!graph) return KRR_ERR_ARG;
    g_launches = graph->kernels;
    KRR_CUDA_CHECK(cudaGraphLaunch(graph->exec, static_cast<cudaStream_t>(stream)));
    return KRR_OK;
}

int64_t krr_graph_kernel_nodes(const krr_graph_t* graph) { return graph ? graph->kernels : -1; }

int krr_graph_destroy(krr_graph_t* graph) {
    if (!graph) return KRR_ERR_ARG;
    cudaGraphExecDestroy(graph->exec);
    cudaGraphDestroy(graph->graph);
    delete graph;
    return KRR_OK;
}

// Device times of the pipeline events of the last krr_potrf_mp call of this thread (lookahead schedule), in ms since
// the fork: per tile column k  {first(k), old(k), newb(k), fin(k)} = {chain + TRSM / store of tile (k+1,k) done on the
// critical stream, O(k) done, N(k) done on the bulk stream, P(k) + F(k) done on the panel stream}; -1 = not recorded.
int krr_profile_timeline(int NT, float* h_ms) {
    if (NT < 1 || !h_ms) return KRR_ERR_ARG;
    if (NT < 3 || g_pipe.ev.size() < 4 + 5 * static_cast<size_t>(NT - 1)) return KRR_ERR_ARG;      // no such call yet
    if (cudaEventSynchronize(g_pipe.ev[1]) != cudaSuccess || cudaEventSynchronize(g_pipe.ev[3]) != cudaSuccess)
        return KRR_ERR_CUDA;
    for (int k = 0; k < NT; ++k)
        for (int e = 0; e < 4; ++e) {
            float ms = -1.0f;
            const size_t idx = 4 + 5 * static_cast<size_t>(k) + e;
            if (idx >= g_pipe.ev.size()) { h_ms[4 * k + e] = ms; continue; }         // (the last column records nothing)
            if (cudaEventElapsedTime(&ms, g_pipe.ev[0], g_pipe.ev[idx]) != cudaSuccess) {
                ms = -1.0f;
                cudaGetLastError();
            }
            h_ms[4 * k + e] = ms;
        }
    return KRR_OK;
}

int64_t krr_tile_slot(int NT, int i, int j) {
    if (NT <= 0 || j < 0 || i < j || i >= NT) return -1;
    return tile_slot(NT, i, j);
}

// ------------------------------------------------------------------------- precision map
size_t krr_precision_map_workspace(int64_t n, int nb) {
    if (check_shape(n, nb) != KRR_OK) return 0;
    const size_t NT = n / nb, nslots = NT * (NT + 1) / 2, chunks = nb / kStatRows;
    return align_up(nslots * chunks * sizeof(double), 1024) + align_up(nslots * chunks * sizeof(float), 1024) +
           align_up(nslots * sizeof(double), 1024);
}

int krr_precision_map(const float* d_A, int64_t n, int64_t lda, int nb, float eps_target, unsigned allowed_mask,
                      unsigned flags, uint8_t* d_map, float* d_tile_norms, float* d_tile_amax, double* d_fro,
                      void* d_ws, size_t ws_bytes, void* stream) {
    g_launches = 0;
    if (!d_A || !d_map || !d_ws) return KRR_ERR_ARG;
    int rc = check_shape(n, nb);
    if (rc) return rc;
    const bool tiled = flags & KRR_FLAG_A_TILED_LOWER;
    if (!tiled && (lda < n || lda % 4 != 0)) return KRR_ERR_ARG;
    if (reinterpret_cast<uintptr_t>(d_A) % 16 != 0) return KRR_ERR_ARG;
    if (flags & ~(KRR_FLAG_PREROUND_A | KRR_FLAG_A_TILED_LOWER)) return KRR_ERR_UNSUPPORTED;
    if (ws_bytes < krr_precision_map_workspace(n, nb)) return KRR_ERR_WORKSPACE;
    rc = check_device(nullptr);
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int NT = static_cast<int>(n / nb);
    const size_t nslots = static_cast<size_t>(NT) * (NT + 1) / 2, chunks = nb / kStatRows;
    uint8_t* ws = static_cast<uint8_t*>(d_ws);
    double* partial = reinterpret_cast<double*>(ws);
    float* pamax = reinterpret_cast<float*>(ws + align_up(nslots * chunks * sizeof(double), 1024));
    double* sumsq = reinterpret_cast<double*>(reinterpret_cast<uint8_t*>(pamax) + align_up(nslots * chunks * sizeof(float), 1024));
    AView A{d_A, lda, tiled ? 1 : 0, NT, nb};
    rc = launch(CAT_MAP, tile_stats_kernel, dim3(static_cast<unsigned>(nslots), static_cast<unsigned>(chunks)), dim3(kStatThreads), 0, st,
                A, partial, pamax);
    if (rc) return rc;
    return launch(CAT_MAP, map_decide_kernel, dim3(1), dim3(1024), 0, st, NT, static_cast<int>(chunks),
                  static_cast<const double*>(partial), static_cast<const float*>(pamax), eps_target, allowed_mask, d_map,
                  d_tile_norms, d_tile_amax, d_fro, sumsq);
}

// The same two kernels on the library's own file-scope scratch array: nothing is allocated by this call (no workspace,
// no events -- the launches bypass the timing scope of launch()).  See include/krr_mp.h for the limit and the sharing rules.
size_t krr_precision_map_static_limit(void) { return KRR_PRECISION_MAP_STATIC_BYTES; }

int krr_precision_map_static(const float* d_A, int64_t n, int64_t lda, int nb, float eps_target, unsigned allowed_mask,
                             unsigned flags, uint8_t* d_map, float* d_tile_norms, float* d_tile_amax, double* d_fro,
                             void* stream) {
    g_launches = 0;
    if (!d_A || !d_map) return KRR_ERR_ARG;
    int rc = check_shape(n, nb);
    if (rc) return rc;
    const bool tiled = flags & KRR_FLAG_A_TILED_LOWER;
    if (!tiled && (lda < n || lda % 4 != 0)) return KRR_ERR_ARG;
    if (reinterpret_cast<uintptr_t>(d_A) % 16 != 0) return KRR_ERR_ARG;
    if (flags & ~(KRR_FLAG_PREROUND_A | KRR_FLAG_A_TILED_LOWER)) return KRR_ERR_UNSUPPORTED;
    const size_t need = krr_precision_map_workspace(n, nb);
    if (need == 0 || need > KRR_PRECISION_MAP_STATIC_BYTES) {
        if (getenv("KRR_DEBUG"))
            fprintf(stderr, "krr_precision_map_static: n = %lld, nb = %d needs %zu bytes of scratch, the static array holds %u; "
                            "use krr_precision_map with a caller workspace\n", static_cast<long long>(n), nb, need,
                    KRR_PRECISION_MAP_STATIC_BYTES);
        return KRR_ERR_WORKSPACE;
    }
    rc = check_device(nullptr);
    if (rc) return rc;
    void* scratch = nullptr;
    rc = pm_static_scratch(&scratch);
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int NT = static_cast<int>(n / nb);
    const size_t nslots = static_cast<size_t>(NT) * (NT + 1) / 2, chunks = nb / kStatRows;
    uint8_t* ws = static_cast<uint8_t*>(scratch);
    double* partial = reinterpret_cast<double*>(ws);
    float* pamax = reinterpret_cast<float*>(ws + align_up(nslots * chunks * sizeof(double), 1024));
    double* sumsq = reinterpret_cast<double*>(reinterpret_cast<uint8_t*>(pamax) + align_up(nslots * chunks * sizeof(float), 1024));
    AView A{d_A, lda, tiled ? 1 : 0, NT, nb};
    // every word of partial / pamax / sumsq that is read below is written first by this call: nothing to clear
    tile_stats_kernel<<<dim3(static_cast<unsigned>(nslots), static_cast<unsigned>(chunks)), dim3(kStatThreads), 0, st>>>(A, partial, pamax);
    ++g_launches;
    if (cudaGetLastError() != cudaSuccess) return KRR_ERR_CUDA;
    map_decide_kernel<<<dim3(1), dim3(1024), 0, st>>>(NT, static_cast<int>(chunks), static_cast<const double*>(partial),
                                                      static_cast<const float*>(pamax), eps_target, allowed_mask, d_map,
                                                      d_tile_norms, d_tile_amax, d_fro, sumsq);
    ++g_launches;
    return cudaGetLastError() == cudaSuccess ? KRR_OK : KRR_ERR_CUDA;
}

// ------------------------------------------------------------------------- factor layout
size_t krr_factor_bytes(int64_t n, int nb, const uint8_t* h_map) {
    if (!h_map || check_shape(n, nb) != KRR_OK) return 0;
    const int NT = static_cast<int>(n / nb);
    if (check_map(NT, h_map, nullptr) != KRR_OK) return 0;
    return host_offsets(NT, nb, h_map, nullptr);
}

int64_t krr_factor_tile_offset(int64_t n, int nb, const uint8_t* h_map, int i, int j) {
    if (!h_map || check_shape(n, nb) != KRR_OK) return -1;
    const int NT = static_cast<int>(n / nb);
    if (j < 0 || i < j || i >= NT || check_map(NT, h_map, nullptr) != KRR_OK) return -1;
    std::vector<int64_t> off;
    host_offsets(NT, nb, h_map, &off);
    return off[static_cast<size_t>(i) * NT + j];
}

// Band map of [37]: the first ceil(fp32_fraction (NT-1)) sub-diagonals of tiles FP32, the rest `low_prec`.
int krr_band_map(int NT, double fp32_fraction, int low_prec, uint8_t* h_map) {
    if (NT <= 0 || NT > kMaxNT || !h_map || low_prec < KRR_FP32 || low_prec > KRR_FP8_E4M3 || !(fp32_fraction >= 0.0) ||
        fp32_fraction > 1.0)
        return KRR_ERR_ARG;
    double bd = fp32_fraction * (NT - 1) - 1e-12;
    int b = static_cast<int>(bd);
    if (static_cast<double>(b) < bd) ++b;                    // ceil
    if (b < 0) b = 0;
    for (int i = 0; i < NT; ++i)
        for (int j = 0; j < NT; ++j)
            h_map[i * NT + j] = (j > i) ? 255 : ((i - j <= b) ? KRR_FP32 : static_cast<uint8_t>(low_prec));
    return KRR_OK;
}

// ------------------------------------------------------------------------- factorisation
size_t krr_potrf_mp_workspace(int64_t n, int nb, const uint8_t* h_map) {
    if (!h_map || check_shape(n, nb) != KRR_OK) return 0;
    bool f8 = false;
    if (check_map(static_cast<int>(n / nb), h_map, &f8) != KRR_OK) return 0;
    size_t n32 = 0, n8 = 0;
    count_tiles(static_cast<int>(n / nb), h_map, &n32, &n8);
    return potrf_ws_layout(n, nb, n32, n8).total;
}

int krr_potrf_mp(const float* d_A, int64_t n, int64_t lda, int nb, const uint8_t* d_map, const uint8_t* h_map,
                 void* d_factor, float* d_scales, int* d_info, void* d_ws, size_t ws_bytes, unsigned flags,
                 void* stream) {
    g_launches = 0;
    if (!d_A || !d_map || !h_map || !d_factor || !d_scales || !d_info || !d_ws) return KRR_ERR_ARG;
    int rc = check_shape(n, nb);
    if (rc) return rc;
    const bool tiled = flags & KRR_FLAG_A_TILED_LOWER;
    if (!tiled && (lda < n || lda % 4 != 0)) return KRR_ERR_ARG;
    if (reinterpret_cast<uintptr_t>(d_A) % 16 != 0 || reinterpret_cast<uintptr_t>(d_ws) % 1024 != 0 ||
        reinterpret_cast<uintptr_t>(d_factor) % 128 != 0)
        return KRR_ERR_ARG;
    if (flags & ~(KRR_FLAG_PREROUND_A | KRR_FLAG_A_TILED_LOWER | KRR_FLAG_NO_LOOKAHEAD | KRR_FLAG_FP8_VIA_FP16 | KRR_FLAG_NO_CTA_PAIRS |
                  KRR_FLAG_FUSED_CHAIN | KRR_FLAG_NO_TAIL_SPLIT))
        return KRR_ERR_UNSUPPORTED;
    const int NT = static_cast<int>(n / nb);
    bool any_fp8 = false;
    rc = check_map(NT, h_map, &any_fp8);
    if (rc) return rc;
    size_t n_fp32 = 0, n_fp8 = 0;
    count_tiles(NT, h_map, &n_fp32, &n_fp8);
    const PotrfWs L = potrf_ws_layout(n, nb, n_fp32, n_fp8);
    if (ws_bytes < L.total) return KRR_ERR_WORKSPACE;
    int num_sms = 0;
    rc = check_device(&num_sms);
    if (rc) return rc;
    rc = set_kernel_attrs();
    if (rc) return rc;

    cudaStream_t st = static_cast<cudaStream_t>(stream);
    uint8_t* ws = static_cast<uint8_t*>(d_ws);
    int64_t* off = reinterpret_cast<int64_t*>(ws + L.off_table);
    int* lrow = reinterpret_cast<int*>(ws + L.lrow);
    int* qrow = reinterpret_cast<int*>(ws + L.qrow);
    float* a_amax = reinterpret_cast<float*>(ws + L.a_amax);
    float* tile_amax = reinterpret_cast<float*>(ws + L.tile_amax);
    float* W = reinterpret_cast<float*>(ws + L.W);
    float* scl = reinterpret_cast<float*>(ws + L.scl);
    float* linv_scale = scl + SCL_COUNT;
    float* dscale = reinterpret_cast<float*>(ws + L.dscale);
    __half* linv_hi = reinterpret_cast<__half*>(ws + L.linv_hi);
    __half* linv_lo = reinterpret_cast<__half*>(ws + L.linv_lo);
    __half* Sh = reinterpret_cast<__half*>(ws + L.Sh);
    __half* Sl = reinterpret_cast<__half*>(ws + L.Sl);
    __half* Hp = reinterpret_cast<__half*>(ws + L.Hp);
    __half* Lp = reinterpret_cast<__half*>(ws + L.Lp);
    uint8_t* Qp = any_fp8 ? ws + L.Qp : nullptr;
    const size_t nslots = static_cast<size_t>(NT) * (NT + 1) / 2;
    AView A{d_A, lda, tiled ? 1 : 0, NT, nb};

    KRR_CUDA_CHECK(cudaMemsetAsync(d_info, 0, sizeof(int), st));
    KRR_CUDA_CHECK(cudaMemsetAsync(tile_amax, 0, nslots * sizeof(float), st));
    // the blocks of M above and of M^T below the diagonal are read as zeros and never written
    KRR_CUDA_CHECK(cudaMemsetAsync(Sh + static_cast<size_t>(n) * nb, 0, 6 * static_cast<size_t>(nb) * nb * 2, st));
    KRR_CUDA_CHECK(cudaMemsetAsync(Sl + static_cast<size_t>(n) * nb, 0, 6 * static_cast<size_t>(nb) * nb * 2, st));
    int* prog = reinterpret_cast<int*>(ws + L.prog);
    StreamK sk_ws{reinterpret_cast<int*>(ws + L.split), reinterpret_cast<float*>(ws + L.sk_partial)};
    const StreamK* sk = ((flags & KRR_FLAG_NO_TAIL_SPLIT) || num_sms / 2 > kMaxSkUnits) ? nullptr : &sk_ws;
    KRR_CUDA_CHECK(cudaMemsetAsync(prog, 0, static_cast<size_t>(n / kBlk) * sizeof(int), st));
    rc = launch(CAT_MISC, scales_init_kernel, dim3((NT * NT + 255) / 256), dim3(256), 0, st, NT, d_scales);
    if (rc) return rc;
    rc = launch(CAT_MISC, offsets_kernel, dim3(1), dim3(32), 0, st, NT, nb, d_map, off, host_map_hash(NT, h_map), d_info, lrow, qrow);
    if (rc) return rc;
    rc = launch(CAT_MISC, equilibrate_kernel, dim3(1), dim3(1024), 0, st, A, n, scl, dscale);
    if (rc) return rc;
    const bool preround = flags & KRR_FLAG_PREROUND_A;
    if (preround && any_fp8) {
        KRR_CUDA_CHECK(cudaMemsetAsync(a_amax, 0, static_cast<size_t>(NT) * NT * sizeof(float), st));
        rc = launch(CAT_MISC, tile_amax_kernel, dim3(static_cast<unsigned>(nslots), nb / 32), dim3(256), 0, st, A, d_map, a_amax);
        if (rc) return rc;
    }

    GemmMaps tm;
    // (host copy of the lo-plane rows of the diagonal tiles: the same count, in the same order, as offsets_kernel's)
    std::vector<int64_t> diag_lrow(NT);
    {
        int64_t nl = 0;
        for (int j = 0; j < NT; ++j)
            for (int i = j; i < NT; ++i)
                if (h_map[i * NT + j] == KRR_FP32) { if (i == j) diag_lrow[j] = nl * nb; ++nl; }
    }
    if (make_plane_tmap(&tm.H, Hp, nslots * nb, nb) || make_plane_tmap(&tm.L, Lp, (n_fp32 ? n_fp32 : 1) * nb, nb) ||
        make_plane_tmap(&tm.SH, Sh, scratch_rows(n, nb), nb) || make_plane_tmap(&tm.SL, Sl, scratch_rows(n, nb), nb))
        return KRR_ERR_CUDA;
    const size_t linv_elems = static_cast<size_t>(nb) * kBlk;           // one set of inverted diagonal blocks
    for (int b = 0; b < 2; ++b)
        if (make_plane_tmap(&tm.IH[b], linv_hi + b * linv_elems, nb, kBlk) ||
            make_plane_tmap(&tm.IL[b], linv_lo + b * linv_elems, nb, kBlk))
            return KRR_ERR_CUDA;
    if (any_fp8) {
        if (make_byte_plane_tmap(&tm.Q, Qp, (n_fp8 ? n_fp8 : 1) * nb, nb)) return KRR_ERR_CUDA;
    } else {
        tm.Q = tm.H;                              // never dereferenced (op.fp8q = 0)
    }
    const int cg = ((flags & KRR_FLAG_NO_CTA_PAIRS) || nb % (2 * kBlk) != 0) ? 1 : 2;
    // the panel product X = S M^T walks K = nb with partial sums far larger than the result ("Accuracy of
    // the product form"): every MMA truncates the accumulator, so the error grows with nb.  Up to nb = 1024 the CTA-pair form
    // (cross terms in the second accumulator) stays below the 1e-6 of an all-FP32 factorisation; larger tiles take the
    // single-CTA form, which starts a fresh accumulator every 128 columns of K and adds the segments in FP32 (twice the
    // operand traffic per flop); so do matrices of at most four tile columns, where the margin is thinnest (nb = 1024, NT = 2:
    // 9.9e-7 against 5.6e-7) and the panel costs next to nothing
    const int cg_trsm = (nb > 1024 || NT <= 4) ? 1 : cg;

    const int nsub = nb / kBlk;
    const bool lookahead = !(flags & KRR_FLAG_NO_LOOKAHEAD) && NT > 2;
    float* Wbuf[2] = {W, reinterpret_cast<float*>(ws + L.W2)};
    cudaStream_t sh = st, sl = st, sv = st;      // critical-path stream, bulk stream, inverse stream
    enum { EV_FORK = 0, EV_JOIN_HI = 1, EV_JOIN_MID = 2, EV_JOIN_LO = 3, EV_BASE = 4, EV_PER_COL = 5 };
    auto ev_first = [&](int k) { return g_pipe.event(EV_BASE + EV_PER_COL * static_cast<size_t>(k) + 0); };
    auto ev_old = [&](int k) { return g_pipe.event(EV_BASE + EV_PER_COL * static_cast<size_t>(k) + 1); };
    auto ev_newb = [&](int k) { return g_pipe.event(EV_BASE + EV_PER_COL * static_cast<size_t>(k) + 2); };
    auto ev_trsm = [&](int k) { return g_pipe.event(EV_BASE + EV_PER_COL * static_cast<size_t>(k) + 3); };
    auto ev_chain = [&](int k) { return g_pipe.event(EV_BASE + EV_PER_COL * static_cast<size_t>(k) + 4); };
    if (lookahead) {
        rc = g_pipe.init();
        if (rc) return rc;
        sh = g_pipe.hi; sl = g_pipe.lo; sv = g_pipe.mid;
        KRR_CUDA_CHECK(cudaEventRecord(g_pipe.event(EV_FORK), st));
        KRR_CUDA_CHECK(cudaStreamWaitEvent(sh, g_pipe.event(EV_FORK), 0));
        KRR_CUDA_CHECK(cudaStreamWaitEvent(sl, g_pipe.event(EV_FORK), 0));
        KRR_CUDA_CHECK(cudaStreamWaitEvent(sv, g_pipe.event(EV_FORK), 0));
    }
    // events of the inverse stream: one per 128-block of the diagonal tile (re-recorded every column; a wait is always
    // enqueued right after its record) and one for the finished inverse
    auto ev_blk = [&](int c) { return g_pipe.event(EV_BASE + EV_PER_COL * static_cast<size_t>(NT) + c); };
    auto ev_inv = [&]() { return g_pipe.event(EV_BASE + EV_PER_COL * static_cast<size_t>(NT) + nsub); };
    auto ev_p3 = [&](int c) { return g_pipe.event(EV_BASE + EV_PER_COL * static_cast<size_t>(NT) + nsub + 1 + c); };
    // M = inv(L_kk) row block by row block (gemm_tc.cuh MODE_INV with the node: left blocks [0, r), right block r): as soon
    // as the chain has factored 128-block r, row r of M follows from the rows above it -- two launches, which run on the
    // inverse stream beside the chain's next sub-columns; only the last row block's two launches come after the chain
    // (step 0, U^T = M[0:r, 0:r]^T L[r, 0:r]^T, needs the row block's TRSM steps only -- it is issued behind P3(r - 1) and runs
    // beside P1(r) and the POTRF of block r; step 1 needs the block's inverse)
    auto inverse_row = [&](GemmOp op, int r, int lb, cudaStream_t s, int step_lo, int step_hi) -> int {
        op.mode = MODE_INV; op.c = 0; op.cb0 = 0; op.ncb = 1; op.rb0 = 0; op.nrb = 1;
        op.node.o = 0; op.node.hl = r; op.node.hr = 1;
        op.inv_last = (r == nsub - 1) ? 1 : 0;
        for (int step = step_lo; step < step_hi; ++step) {
            op.inv_step = step;
            const int e = launch_gemm(tm, op, num_sms, 1, s, lb);
            if (e) return e;
        }
        return static_cast<int>(KRR_OK);
    };
    auto inverse_export = [&](const GemmOp& op, int c, int lb, cudaStream_t s) -> int {
        return launch(CAT_POTRF, inv_export_kernel, dim3(16), dim3(256), 0, s, static_cast<const __half*>(linv_hi + lb * linv_elems),
                      static_cast<const __half*>(linv_lo + lb * linv_elems), static_cast<const float*>(linv_scale + lb * nsub), nb,
                      c * kBlk, Sh, Sl, op.srow_m, op.srow_mt, static_cast<const float*>(scl), d_info);
    };
    // bulk kernels leave a few SMs to the diagonal-tile chain they overlap with
    const int reserve = nsub < 8 ? nsub : 8;
    const int bulk_ctas = lookahead ? (num_sms - reserve > reserve ? num_sms - reserve : num_sms) : num_sms;
    auto finalize = [&](int k, const float* Wk, int i0, int count, int only_fp8, cudaStream_t s) {
        if (count <= 0) return static_cast<int>(KRR_OK);
        if (only_fp8) {                      // nothing to do when none of these tiles is FP8 (the launch sequence follows the map)
            bool any = false;
            for (int i = k + i0; i < k + i0 + count; ++i) any |= (h_map[i * NT + k] == KRR_FP8_E4M3);
            if (!any) return static_cast<int>(KRR_OK);
        }
        return launch(CAT_FINALIZE, finalize_kernel, dim3(nsub * nsub * 4, count), dim3(256), 0, s, NT, nb, k, i0, Wk, d_map,
                      static_cast<const int64_t*>(off), static_cast<const float*>(tile_amax), static_cast<uint8_t*>(d_factor),
                      d_scales, Hp, Qp, static_cast<const int*>(qrow), static_cast<const float*>(scl), static_cast<const float*>(dscale), only_fp8);
    };

    // Tile column k.  Critical stream `sh`: newest term on the diagonal tile, the diagonal-tile
    // chain, M = inv(L_kk), then the TRSM product and store of tile (k+1, k) -- all the next column's chain needs.
    // Bulk stream `sl`: newest term on the rows below (N(k): S into the scratch planes), the older terms of column
    // k+1 (O(k+1), beside the chain of column k), then the TRSM product of the remaining rows (T(k) = S M^T, stored
    // straight into the mosaic) -- every bulk kernel is a full-width tensor-core product.
    // (a lambda: an error in the middle still joins the internal streams below, so the caller's stream -- or a
    // stream capture -- is left in a consistent state)
    auto run_columns = [&]() -> int {
    for (int k = 0; k < NT; ++k) {
        const int mblk = (NT - k) * nsub;             // 128-row blocks of the panel
        const int lb = k & 1;                         // parity set: inverted diagonal blocks, M / M^T / U, W buffer
        float* Wk = Wbuf[lb];
        GemmOp op;
        memset(&op, 0, sizeof(op));
        op.nb = nb; op.NT = NT; op.k = k;
        op.prow0 = tile_slot(NT, k, k) * nb;
        op.prow0_lo = diag_lrow[k]; op.lrow = lrow; op.qrow = qrow;
        op.map = d_map; op.A = A; op.a_amax = (preround && any_fp8) ? a_amax : nullptr;
        op.W = Wk; op.Hp = Hp; op.Lp = Lp; op.tile_amax = tile_amax; op.flags = flags;
        op.scl = scl; op.dscale = dscale; op.linv_scale = linv_scale + lb * nsub;
        op.scales = d_scales; op.fp8q = (any_fp8 && !(flags & KRR_FLAG_FP8_VIA_FP16)) ? 1 : 0;
        op.Sh = Sh; op.Sl = Sl;
        op.srow_m = static_cast<int64_t>(n) + static_cast<int64_t>(lb) * 3 * nb; op.srow_mt = op.srow_m + nb; op.srow_u = op.srow_m + 2 * nb;
        op.off = off; op.factor = static_cast<uint8_t*>(d_factor); op.info = d_info;
        // ---- U(k): S = rd(A) - L[:, 0:k] L[k, 0:k]^T over the tile column (SYRK + GEMM) ----
        op.mode = MODE_UPDATE; op.c = 0; op.cb0 = 0; op.ncb = nsub;
        if (!lookahead) {
            op.s_lo = 0; op.s_hi = k; op.base_w = 0; op.planes = 1; op.rb0 = 0; op.nrb = mblk;
            rc = launch_gemm(tm, op, num_sms, cg, st, 0, sk);
            if (rc) return rc;
        } else {
            // terms s < k-1 were accumulated into Wk by O(k) while column k-1 was being factorised; the
            // newest term s = k-1 is added here, the diagonal tile on the critical stream
            const bool have_old = (k >= 2);
            op.s_lo = (k >= 1) ? k - 1 : 0; op.s_hi = k; op.base_w = have_old ? 1 : 0; op.planes = 1;
            if (have_old) KRR_CUDA_CHECK(cudaStreamWaitEvent(sh, ev_old(k), 0));
            op.rb0 = 0; op.nrb = nsub;
            rc = launch_gemm(tm, op, num_sms, cg, sh);
            if (rc) return rc;
            if (k >= 1) KRR_CUDA_CHECK(cudaStreamWaitEvent(sl, ev_first(k - 1), 0));     // tile (k, k-1) is stored
            op.rb0 = nsub; op.nrb = mblk - nsub;
            rc = launch_gemm(tm, op, bulk_ctas, cg, sl);                                 // N(k)
            if (rc) return rc;
            KRR_CUDA_CHECK(cudaEventRecord(ev_newb(k), sl));
            if (k + 1 < NT && k >= 1) {
                // O(k+1): terms s < k of column k+1, beside the chain of column k
                GemmOp on = op;
                on.k = k + 1; on.prow0 = tile_slot(NT, k + 1, k + 1) * nb; on.prow0_lo = diag_lrow[k + 1]; on.W = Wbuf[(k + 1) & 1];
                on.s_lo = 0; on.s_hi = k; on.base_w = 0; on.planes = 0;
                on.rb0 = 0; on.nrb = (NT - k - 1) * nsub;
                rc = launch_gemm(tm, on, bulk_ctas, cg, sl, 0, sk);
                if (rc) return rc;
                KRR_CUDA_CHECK(cudaEventRecord(ev_old(k + 1), sl));
            }
        }
        // ---- diagonal-tile chain: 128-wide sub-columns of tile (k,k) ----
        // one launch per step (in-tile update, POTRF of a 128-block, TRSM against its inverse), or with
        // KRR_FLAG_FUSED_CHAIN one launch of nsub co-resident CTAs (MODE_DIAG): the same arithmetic
        const bool fused_chain = (flags & KRR_FLAG_FUSED_CHAIN) && nsub <= 16;
        op.linv_hi = linv_hi + lb * linv_elems; op.linv_lo = linv_lo + lb * linv_elems;
        op.linv_scale_w = linv_scale + lb * nsub; op.col_base = static_cast<int64_t>(k) * nb + 1;
        if (fused_chain) {
            op.mode = MODE_DIAG; op.c = 0; op.cb0 = 0; op.ncb = 1; op.rb0 = 0; op.nrb = nsub;
            op.prog = prog + static_cast<size_t>(k) * nsub;
            rc = launch_gemm(tm, op, num_sms, 1, sh, lb);
            if (rc) return rc;
        }
        for (int c = 0; c < nsub && !fused_chain; ++c) {
            if (c > 0) {
                op.mode = MODE_P1; op.c = c; op.cb0 = c; op.ncb = 1; op.rb0 = c; op.nrb = nsub - c;
                rc = launch_gemm(tm, op, num_sms, 1, sh, lb);
                if (rc) return rc;
            }
            rc = launch(CAT_POTRF, potrf128_kernel, dim3(1), dim3(kTriThreads), static_cast<size_t>(kTriSmem), sh, Wk, nb,
                        c * kBlk, c * kBlk, linv_hi + lb * linv_elems, linv_lo + lb * linv_elems, linv_scale + lb * nsub, d_info,
                        static_cast<int64_t>(k) * nb + static_cast<int64_t>(c) * kBlk + 1);
            if (rc) return rc;
            if (k + 1 < NT) {                         // row block c of M, beside the rest of the chain
                if (lookahead) {
                    KRR_CUDA_CHECK(cudaEventRecord(ev_blk(c), sh));
                    KRR_CUDA_CHECK(cudaStreamWaitEvent(sv, ev_blk(c), 0));
                }
                rc = inverse_export(op, c, lb, sv);
                if (rc) return rc;
                if (c >= 1) {
                    rc = inverse_row(op, c, lb, sv, 1, 2);
                    if (rc) return rc;
                }
            }
            op.mode = MODE_P3; op.c = c; op.cb0 = c; op.ncb = 1; op.rb0 = c + 1; op.nrb = nsub - c - 1;
            if (op.nrb > 0) {
                rc = launch_gemm(tm, op, num_sms, 1, sh, lb);
                if (rc) return rc;
                if (k + 1 < NT) {                     // row block c + 1 of L_kk is final: the first step of its row of M
                    if (lookahead) {
                        KRR_CUDA_CHECK(cudaEventRecord(ev_p3(c), sh));
                        KRR_CUDA_CHECK(cudaStreamWaitEvent(sv, ev_p3(c), 0));
                    }
                    rc = inverse_row(op, c + 1, lb, sv, 0, 1);
                    if (rc) return rc;
                }
            }
        }
        rc = finalize(k, Wk, 0, 1, 0, sh);
        if (rc) return rc;
        if (k + 1 == NT) continue;                    // the last column has no panel below
        if (fused_chain)                              // (one launch for the whole chain: the rows of M follow it)
            for (int r = 0; r < nsub; ++r) {
                rc = inverse_export(op, r, lb, sh);
                if (rc) return rc;
                if (r >= 1) {
                    rc = inverse_row(op, r, lb, sh, 0, 2);
                    if (rc) return rc;
                }
            }
        else if (lookahead) {
            KRR_CUDA_CHECK(cudaEventRecord(ev_inv(), sv));
            KRR_CUDA_CHECK(cudaStreamWaitEvent(sh, ev_inv(), 0));
        }
        // ---- panel below: X = S M^T as one triangular product, rounded once and stored (MODE_TRSM) ----
        op.mode = MODE_TRSM; op.c = 0; op.cb0 = 0; op.ncb = nsub;
        if (!lookahead) {
            op.rb0 = nsub; op.nrb = mblk - nsub;
            rc = launch_gemm(tm, op, num_sms, cg_trsm, st, lb);
            if (rc) return rc;
            rc = finalize(k, Wk, 1, NT - k - 1, 1, st);
            if (rc) return rc;
        } else {
            KRR_CUDA_CHECK(cudaEventRecord(ev_chain(k), sh));
            // tile (k+1, k) first, on the critical stream: column k+1's chain needs nothing else of column k
            KRR_CUDA_CHECK(cudaStreamWaitEvent(sh, ev_newb(k), 0));
            op.rb0 = nsub; op.nrb = nsub;
            rc = launch_gemm(tm, op, num_sms, cg_trsm, sh, lb);
            if (rc) return rc;
            rc = finalize(k, Wk, 1, 1, 1, sh);
            if (rc) return rc;
            KRR_CUDA_CHECK(cudaEventRecord(ev_first(k), sh));
            if (k + 2 < NT) {
                KRR_CUDA_CHECK(cudaStreamWaitEvent(sl, ev_chain(k), 0));
                op.rb0 = 2 * nsub; op.nrb = mblk - 2 * nsub;
                rc = launch_gemm(tm, op, bulk_ctas, cg_trsm, sl, lb);                    // T(k)
                if (rc) return rc;
                rc = finalize(k, Wk, 2, NT - k - 2, 1, sl);
                if (rc) return rc;
            }
            KRR_CUDA_CHECK(cudaEventRecord(ev_trsm(k), sl));
        }
    }
    return static_cast<int>(KRR_OK);
    };
    const int rc_columns = run_columns();
    if (lookahead) {
        KRR_CUDA_CHECK(cudaEventRecord(g_pipe.event(EV_JOIN_HI), sh));
        KRR_CUDA_CHECK(cudaEventRecord(g_pipe.event(EV_JOIN_LO), sl));
        KRR_CUDA_CHECK(cudaEventRecord(g_pipe.event(EV_JOIN_MID), sv));
        KRR_CUDA_CHECK(cudaStreamWaitEvent(st, g_pipe.event(EV_JOIN_HI), 0));
        KRR_CUDA_CHECK(cudaStreamWaitEvent(st, g_pipe.event(EV_JOIN_LO), 0));
        KRR_CUDA_CHECK(cudaStreamWaitEvent(st, g_pipe.event(EV_JOIN_MID), 0));
    }
    return rc_columns;
}

// ------------------------------------------------------------------------- solve
static int rhs_class(int nrhs) { return nrhs <= 4 ? 4 : (nrhs <= 8 ? 8 : (nrhs <= 16 ? 16 : 32)); }

struct PotrsWs { size_t off_table, dinv, dinvT, Minv, MinvT, stage, nearP, total; };
static PotrsWs potrs_ws_layout(int64_t n, int nb) {
    const size_t NT = n / nb;
    PotrsWs w;
    size_t o = 0;
    w.off_table = o; o = align_up(o + NT * NT * sizeof(int64_t), 1024);
    w.dinv = o;      o = align_up(o + static_cast<size_t>(n) * kBlk * sizeof(float), 1024);
    w.dinvT = o;     o = align_up(o + static_cast<size_t>(n) * kBlk * sizeof(float), 1024);
    w.Minv = o;      o = align_up(o + static_cast<size_t>(n) * nb * sizeof(float), 1024);     // inv(L_kk), every k
    w.MinvT = o;     o = align_up(o + static_cast<size_t>(n) * nb * sizeof(float), 1024);     // inv(L_kk)^T for the backward sweep
    w.stage = o;     o = align_up(o + static_cast<size_t>(nb) * kMaxRhs * sizeof(float), 1024);  // t_k of the diagonal step
    w.nearP = o;     o = align_up(o + 3 * 8 * static_cast<size_t>(nb) * kMaxRhs * sizeof(float), 1024);  // K slices of the near / mid tiles' updates
    w.total = o;
    return w;
}

size_t krr_potrs_workspace(int64_t n, int nb, int nrhs) {
    if (check_shape(n, nb) != KRR_OK || nrhs < 1 || nrhs > kMaxRhs) return 0;
    if (static_cast<int64_t>(rhs_class(nrhs)) * nb > 32768) return 0;     // solved block must fit in smem
    return potrs_ws_layout(n, nb).total;
}

}  // extern "C"

// Forward and backward sweeps with a two-column lookahead on the library's internal streams (`sh` chain, `sm` middle,
// `sl` bulk): once z_k (alpha_k) is known, the update of the NEXT tile row (column) -- all the next diagonal solve waits
// for -- runs on the chain stream, the one after it on the middle stream, the remaining rows on the bulk stream beside
// the following solves (the comment at the loops has the event order that keeps the sums deterministic).
template <int NRHS>
static int potrs_run(const uint8_t* factor, const float* d_scales, const uint8_t* d_map, const std::vector<int64_t>& hoff,
                     const int64_t* off, const float* Minv, const float* MinvT, float* stage, int NT, int nb, float* B,
                     int64_t ldb, int nrhs, int num_sms, cudaStream_t st, const StreamMaps* smaps, const uint8_t* h_map_, float* nearP) {
    constexpr int ROWS = 64 / NRHS, NW = kSolveThreads / 32, CPL = (NRHS <= 16) ? 4 : 2;
    const size_t smem_z = static_cast<size_t>(NRHS) * nb * sizeof(float);
    const size_t smem_bu = smem_z + static_cast<size_t>(NW / 2) * 32 * CPL * NRHS * sizeof(float);
    const size_t smem_b1 = smem_z + static_cast<size_t>(NW / 2) * 32 * NRHS * sizeof(float);
    const int64_t blk_elems = static_cast<int64_t>(kBlk) * kBlk;
    const int nsub = nb / kBlk;
    // the lookahead pays once a tile column is a few megabytes (C1, n = 2048, nb = 256: 0.24 ms without it against 0.41 ms
    // with its five launches and the events per column; C2, n = 16384, nb = 512: 1.64 against 1.53 ms)
    const bool pipe = NT > 2 && static_cast<int64_t>(NT) * nb * nb >= (int64_t{1} << 20);
    cudaStream_t sh = st, sm = st, sl = st;
    enum { EV_FORK = 0, EV_JOIN_HI = 1, EV_JOIN_MID = 2, EV_JOIN_LO = 3, EV_BASE = 4 };      // the event pool of krr_potrf_mp, reused
    auto ev_diag = [&](int k) { return g_pipe.event(EV_BASE + 4 * static_cast<size_t>(k) + 0); };
    auto ev_bulk = [&](int k) { return g_pipe.event(EV_BASE + 4 * static_cast<size_t>(k) + 1); };
    auto ev_mid = [&](int k) { return g_pipe.event(EV_BASE + 4 * static_cast<size_t>(k) + 2); };
    int rc;
    if (pipe) {
        rc = g_pipe.init();
        if (rc) return rc;
        sh = g_pipe.hi; sm = g_pipe.mid; sl = g_pipe.lo;
        KRR_CUDA_CHECK(cudaEventRecord(g_pipe.event(EV_FORK), st));
        KRR_CUDA_CHECK(cudaStreamWaitEvent(sh, g_pipe.event(EV_FORK), 0));
        KRR_CUDA_CHECK(cudaStreamWaitEvent(sm, g_pipe.event(EV_FORK), 0));
        KRR_CUDA_CHECK(cudaStreamWaitEvent(sl, g_pipe.event(EV_FORK), 0));
    }
    // bulk updates leave room for a diagonal-solve CTA on every SM (1 update CTA + 1 solve CTA fit in shared memory;
    // the update CTAs are persistent, so a solve CTA that does not fit beside them would wait for the whole kernel)
    const int bulk_per_sm = 3;
    auto fwd_update = [&](int k, int i_lo, int i_hi, cudaStream_t s, int per_sm) {
        if (i_hi <= i_lo) return static_cast<int>(KRR_OK);
        const int64_t tasks = static_cast<int64_t>(i_hi - i_lo) * nb / ROWS;
        const int64_t want = (tasks + NW - 1) / NW;
        const int64_t cap = static_cast<int64_t>(per_sm) * num_sms;
        return launch(CAT_POTRS, potrs_fwd_update_kernel<NRHS>, dim3(static_cast<unsigned>(want < cap ? want : cap)), dim3(kSolveThreads),
                      smem_z + static_cast<size_t>(i_hi - i_lo) * 16, s, NT, nb, k, i_lo, i_hi,
                      factor, off, d_map, d_scales, B, ldb, nrhs);
    };
    auto bwd_update = [&](int k, int j_lo, int j_hi, cudaStream_t s) {
        if (j_hi <= j_lo) return static_cast<int>(KRR_OK);
        if (pipe && j_hi - j_lo == 1)            // the tile the next diagonal solve waits for: one column per lane, 4 x the CTAs
            return launch(CAT_POTRS, potrs_bwd_update_kernel<NRHS, 1>, dim3(nb / 32), dim3(kSolveThreads), smem_b1, s,
                          NT, nb, k, j_lo, 1, factor, off, d_map, d_scales, B, ldb, nrhs);
        const int units = (j_hi - j_lo) * (nb / (32 * CPL));
        const int cap = 2 * num_sms;             // two persistent CTAs per SM (shared memory), alpha_k staged once each
        return launch(CAT_POTRS, potrs_bwd_update_kernel<NRHS, CPL>, dim3(units < cap ? units : cap), dim3(kSolveThreads), smem_bu, s,
                      NT, nb, k, j_lo, j_hi - j_lo, factor, off, d_map, d_scales, B, ldb, nrhs);
    };
    // Bulk updates (rows k + 3 .. / columns .. k - 3 of the two-column lookahead below): streamed through a shared-memory
    // ring by TMA, one persistent CTA per SM (potrs_stream.cuh), the ring as deep as shared memory allows (8 x 16 KB at
    // nb = 1024, nrhs <= 16).  Shapes whose small operand leaves no room for two ring slots take the older kernels.
    const int stream_budget = 227 * 1024;
    const int stream_sms = num_sms > 32 ? num_sms - 16 : num_sms;     // 16 SMs stay free for the chain's kernels (measured: 148 / 140 / 132 -> 9.51 / 9.55 / 9.34 ms at C3)
    auto stream_update = [&](bool bwd, int k, int t_lo, int t_hi, cudaStream_t s, int* done, int ksplit = 1, float* P = nullptr) {
        using C = StreamCfg<NRHS>;
        *done = 0;
        const int ntiles = t_hi - t_lo;
        if (ntiles <= 0 || stream_budget <= 0 || !smaps) return static_cast<int>(KRR_OK);
        if (ksplit > 1 && (ntiles != 1 || !P)) return static_cast<int>(KRR_OK);
        const size_t fixed = smem_z + C::RED_BYTES + static_cast<size_t>(ntiles) * 12 + 8 + (2 * kStreamMaxStages + 1) * 8;
        if (fixed + 2 * kStreamStage > static_cast<size_t>(stream_budget)) return static_cast<int>(KRR_OK);
        int nst = static_cast<int>((static_cast<size_t>(stream_budget) - fixed) / kStreamStage);
        if (nst > kStreamMaxStages) nst = kStreamMaxStages;
        const int units = ntiles * (nb / 128) * ksplit;
        // (a sliced tile takes one CTA per unit -- the SMs the bulk launches leave free)
        const int grid = (ksplit > 1) ? units : (units < stream_sms ? units : stream_sms);
        *done = 1;
        const size_t smem = fixed + static_cast<size_t>(nst) * kStreamStage;
        if (ksplit > 1 && s == sh) {     // the near tile: a programmatic dependent of the diagonal step's product
            if (bwd)
                return launch_pdl(CAT_POTRS, potrs_stream_update_kernel<NRHS, true>, dim3(grid), dim3(kStreamThreads), smem, s,
                                  smaps[1], NT, nb, k, t_lo, ntiles, nst, off, d_map, d_scales, B, ldb, nrhs, ksplit, P);
            return launch_pdl(CAT_POTRS, potrs_stream_update_kernel<NRHS, false>, dim3(grid), dim3(kStreamThreads), smem, s,
                              smaps[0], NT, nb, k, t_lo, ntiles, nst, off, d_map, d_scales, B, ldb, nrhs, ksplit, P);
        }
        if (bwd)
            return launch(CAT_POTRS, potrs_stream_update_kernel<NRHS, true>, dim3(grid), dim3(kStreamThreads), smem, s,
                          smaps[1], NT, nb, k, t_lo, ntiles, nst, off, d_map, d_scales, B, ldb, nrhs, ksplit, P);
        return launch(CAT_POTRS, potrs_stream_update_kernel<NRHS, false>, dim3(grid), dim3(kStreamThreads), smem, s,
                      smaps[0], NT, nb, k, t_lo, ntiles, nst, off, d_map, d_scales, B, ldb, nrhs, ksplit, P);
    };
    // A single tile of the lookahead -- the "near" tile, all the next diagonal step waits for, or the "mid" tile behind it -- as
    // K slices on the SMs the bulk launches leave free: the largest power of two <= 8 that divides the tile's chunk count and
    // keeps one CTA per free SM; the slices' sums go to Pbuf and the stage kernel of the diagonal step that needs these rows
    // subtracts them.  *nslices = 0: the tile went through the r01 kernel (read-modify-write of B) instead.
    auto near_update = [&](bool bwd, int k, int t, cudaStream_t s, float* Pbuf, int* nslices) {
        *nslices = 0;
        const int p = bwd ? h_map_[k * NT + t] : h_map_[t * NT + k];
        const int es = (p == KRR_FP32) ? 4 : (p == KRR_FP16 ? 2 : 1);
        const int chunks = nb * es / 128, free_sms = num_sms - stream_sms;
        int ks = 1;
        while (ks < 8 && chunks % (2 * ks) == 0 && (nb / 128) * 2 * ks <= free_sms) ks *= 2;
        if (pipe && ks > 1 && Pbuf) {
            int done = 0;
            const int e = stream_update(bwd, k, t, t + 1, s, &done, ks, Pbuf);
            if (e) return e;
            if (done) { *nslices = ks; return static_cast<int>(KRR_OK); }
        }
        return bwd ? bwd_update(k, t, t + 1, s) : fwd_update(k, t, t + 1, s, 3);
    };
    const size_t p_elems = 8 * static_cast<size_t>(nb) * kMaxRhs;      // one partial buffer: near | mid (even tile) | mid (odd tile)
    auto midP = [&](int tile) { return nearP ? nearP + (1 + (tile & 1)) * p_elems : nullptr; };
    int mid_slices[2] = {0, 0};       // slices a sliced mid tile left for the diagonal step of tile row (column) `tile`, by parity
    auto diag = [&](int k, int backward, cudaStream_t s, int nslices) {
        const float* Mk = (backward ? MinvT : Minv) + static_cast<int64_t>(k) * nb * nb;
        float* Bk = B + static_cast<int64_t>(k) * nb * ldb;
        int e = launch_pdl(CAT_POTRS, potrs_stage_kernel<NRHS>, dim3((nb * NRHS + 255) / 256), dim3(256), 0, s, nb,
                       static_cast<const float*>(Bk), ldb, nrhs, stage, static_cast<const float*>(midP(k)), mid_slices[k & 1],
                       static_cast<const float*>(nearP), nslices);
        mid_slices[k & 1] = 0;
        if (e) return e;
        return launch_pdl(CAT_POTRS, potrs_diagmul_kernel<NRHS>, dim3(nb / ROWS), dim3(kDiagThreads), 0, s, nb, Mk,
                      static_cast<const float*>(stage), Bk, ldb, nrhs, backward);
    };
    int near_slices = 0;              // slices the pending near tile left in nearP for the next diagonal step's stage kernel
    // (a lambda: an error in the middle still joins the internal streams below)
    auto run_sweeps = [&]() -> int {
    // Two-column lookahead.  Column k's update of row r is made by: the chain stream for r = k + 1 ("near": all the next
    // diagonal solve waits for), the middle stream for r = k + 2 ("mid"), the bulk stream for r >= k + 3.  A row of B is
    // read-modify-written, so the order of its updates is fixed by events (deterministic results): bulk(.. r-3), then
    // mid(r-2) -- which waits for bulk(r-3) --, then near(r-1) -- which waits for mid(r-2).  The chain therefore waits
    // for a bulk launch issued TWO columns earlier, not for the previous column's.
    // ---- forward: L z = y
    for (int k = 0; k < NT; ++k) {
        rc = diag(k, 0, sh, near_slices);
        if (rc) return rc;
        near_slices = 0;
        if (!pipe) {
            rc = fwd_update(k, k + 1, NT, st, 3);
            if (rc) return rc;
            continue;
        }
        KRR_CUDA_CHECK(cudaEventRecord(ev_diag(k), sh));
        if (k + 1 < NT) {
            if (k >= 1) KRR_CUDA_CHECK(cudaStreamWaitEvent(sh, ev_mid(k - 1), 0));
            rc = near_update(false, k, k + 1, sh, nearP, &near_slices);
            if (rc) return rc;
        }
        KRR_CUDA_CHECK(cudaStreamWaitEvent(sm, ev_diag(k), 0));
        if (k >= 1) KRR_CUDA_CHECK(cudaStreamWaitEvent(sm, ev_bulk(k - 1), 0));
        if (k + 2 < NT) {
            rc = near_update(false, k, k + 2, sm, midP(k + 2), &mid_slices[(k + 2) & 1]);
            if (rc) return rc;
        }
        KRR_CUDA_CHECK(cudaEventRecord(ev_mid(k), sm));
        KRR_CUDA_CHECK(cudaStreamWaitEvent(sl, ev_diag(k), 0));
        if (k + 3 < NT) {
            int streamed = 0;
            rc = stream_update(false, k, k + 3, NT, sl, &streamed);
            if (rc) return rc;
            if (!streamed) rc = fwd_update(k, k + 3, NT, sl, bulk_per_sm);
            if (rc) return rc;
        }
        KRR_CUDA_CHECK(cudaEventRecord(ev_bulk(k), sl));
    }
    if (pipe) {      // the backward sweep starts from a quiescent state
        KRR_CUDA_CHECK(cudaEventRecord(ev_bulk(NT), sl));
        KRR_CUDA_CHECK(cudaEventRecord(ev_mid(NT), sm));
        KRR_CUDA_CHECK(cudaStreamWaitEvent(sh, ev_bulk(NT), 0));
        KRR_CUDA_CHECK(cudaStreamWaitEvent(sh, ev_mid(NT), 0));
    }
    // ---- backward: L^T alpha = z
    for (int k = NT - 1; k >= 0; --k) {
        rc = diag(k, 1, sh, near_slices);
        if (rc) return rc;
        near_slices = 0;
        if (!pipe) {
            rc = bwd_update(k, 0, k, st);
            if (rc) return rc;
            continue;
        }
        KRR_CUDA_CHECK(cudaEventRecord(ev_diag(k), sh));
        if (k >= 1) {
            if (k + 1 < NT) KRR_CUDA_CHECK(cudaStreamWaitEvent(sh, ev_mid(k + 1), 0));
            rc = near_update(true, k, k - 1, sh, nearP, &near_slices);
            if (rc) return rc;
        }
        KRR_CUDA_CHECK(cudaStreamWaitEvent(sm, ev_diag(k), 0));
        if (k + 1 < NT) KRR_CUDA_CHECK(cudaStreamWaitEvent(sm, ev_bulk(k + 1), 0));
        if (k >= 2) {
            rc = near_update(true, k, k - 2, sm, midP(k - 2), &mid_slices[(k - 2) & 1]);
            if (rc) return rc;
        }
        KRR_CUDA_CHECK(cudaEventRecord(ev_mid(k), sm));
        KRR_CUDA_CHECK(cudaStreamWaitEvent(sl, ev_diag(k), 0));
        if (k >= 3) {
            int streamed = 0;
            rc = stream_update(true, k, 0, k - 2, sl, &streamed);
            if (rc) return rc;
            if (!streamed) rc = bwd_update(k, 0, k - 2, sl);
            if (rc) return rc;
        }
        KRR_CUDA_CHECK(cudaEventRecord(ev_bulk(k), sl));
    }
    return static_cast<int>(KRR_OK);
    };
    const int rc_sweeps = run_sweeps();
    if (pipe) {
        KRR_CUDA_CHECK(cudaEventRecord(g_pipe.event(EV_JOIN_HI), sh));
        KRR_CUDA_CHECK(cudaEventRecord(g_pipe.event(EV_JOIN_MID), sm));
        KRR_CUDA_CHECK(cudaEventRecord(g_pipe.event(EV_JOIN_LO), sl));
        KRR_CUDA_CHECK(cudaStreamWaitEvent(st, g_pipe.event(EV_JOIN_HI), 0));
        KRR_CUDA_CHECK(cudaStreamWaitEvent(st, g_pipe.event(EV_JOIN_MID), 0));
        KRR_CUDA_CHECK(cudaStreamWaitEvent(st, g_pipe.event(EV_JOIN_LO), 0));
    }
    return rc_sweeps;
}

// krr_potrs; prepare = false skips the once-per-factor part (tile offsets, inverses of the diagonal tiles), which a caller
// that solves again with the SAME factor and the SAME workspace (krr_refine, krr_pcg) has left in the workspace
static int potrs_impl(const void* d_factor, const float* d_scales, const uint8_t* d_map, const uint8_t* h_map, int64_t n,
                      int nb, float* d_B, int64_t ldb, int nrhs, void* d_ws, size_t ws_bytes, void* stream, bool prepare) {
    g_launches = 0;
    if (!d_factor || !d_scales || !d_map || !h_map || !d_B || !d_ws) return KRR_ERR_ARG;
    int rc = check_shape(n, nb);
    if (rc) return rc;
    if (nrhs < 1 || nrhs > kMaxRhs || ldb < nrhs) return KRR_ERR_ARG;
    if (static_cast<int64_t>(rhs_class(nrhs)) * nb > 32768) return KRR_ERR_SHAPE;
    if (reinterpret_cast<uintptr_t>(d_ws) % 16 != 0 || reinterpret_cast<uintptr_t>(d_factor) % 16 != 0) return KRR_ERR_ARG;
    const int NT = static_cast<int>(n / nb);
    rc = check_map(NT, h_map, nullptr);
    if (rc) return rc;
    const PotrsWs L = potrs_ws_layout(n, nb);
    if (ws_bytes < L.total) return KRR_ERR_WORKSPACE;
    int num_sms = 0;
    rc = check_device(&num_sms);
    if (rc) return rc;
    rc = set_kernel_attrs();
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    std::vector<int64_t> hoff;
    host_offsets(NT, nb, h_map, &hoff);
    uint8_t* ws = static_cast<uint8_t*>(d_ws);
    int64_t* off = reinterpret_cast<int64_t*>(ws + L.off_table);
    float* dinv = reinterpret_cast<float*>(ws + L.dinv);
    float* dinvT = reinterpret_cast<float*>(ws + L.dinvT);
    float* Minv = reinterpret_cast<float*>(ws + L.Minv);
    float* MinvT = reinterpret_cast<float*>(ws + L.MinvT);
    float* stage = reinterpret_cast<float*>(ws + L.stage);
    float* nearP = reinterpret_cast<float*>(ws + L.nearP);
    const uint8_t* factor = static_cast<const uint8_t*>(d_factor);
    if (prepare) {
        rc = launch(CAT_MISC, offsets_kernel, dim3(1), dim3(32), 0, st, NT, nb, d_map, off, host_map_hash(NT, h_map), static_cast<int*>(nullptr),
                    static_cast<int*>(nullptr), static_cast<int*>(nullptr));
        if (rc) return rc;
        rc = launch(CAT_POTRS, trtri128_kernel, dim3(static_cast<unsigned>(n / kBlk)), dim3(kTriThreads), static_cast<size_t>(kTriSmem), st,
                    factor, static_cast<const int64_t*>(off), NT, nb, dinv, dinvT);
        if (rc) return rc;
        rc = launch(CAT_POTRS, potrs_tile_inverse_kernel, dim3(nb / kBlk, NT), dim3(kTinvThreads), static_cast<size_t>(kTinvSmem), st,
                    factor, static_cast<const int64_t*>(off), NT, nb, static_cast<const float*>(dinv), Minv, MinvT);
        if (rc) return rc;
    }
    // the mosaic as a TMA source of the streamed bulk updates: per direction one map per element size
    StreamMaps smaps[2];
    const size_t payload = host_offsets(NT, nb, h_map, nullptr);
    bool have_maps = true;                                   // (an encoding failure falls back to the r01 bulk kernels)
    for (int d = 0; d < 2 && have_maps; ++d) {
        CUtensorMap* m[3] = {&smaps[d].m4, &smaps[d].m2, &smaps[d].m1};
        const int es[3] = {4, 2, 1};
        for (int e = 0; e < 3 && have_maps; ++e)
            have_maps = make_mosaic_tmap(m[e], factor, payload, nb, es[e], d == 0 ? 128 / es[e] : 128, d == 0 ? 128 : 128 / es[e], d == 0) == KRR_OK;
    }
    const StreamMaps* sm = have_maps ? smaps : nullptr;
    switch (rhs_class(nrhs)) {
        case 4:  return potrs_run<4>(factor, d_scales, d_map, hoff, off, Minv, MinvT, stage, NT, nb, d_B, ldb, nrhs, num_sms, st, sm, h_map, nearP);
        case 8:  return potrs_run<8>(factor, d_scales, d_map, hoff, off, Minv, MinvT, stage, NT, nb, d_B, ldb, nrhs, num_sms, st, sm, h_map, nearP);
        case 16: return potrs_run<16>(factor, d_scales, d_map, hoff, off, Minv, MinvT, stage, NT, nb, d_B, ldb, nrhs, num_sms, st, sm, h_map, nearP);
        default: return potrs_run<32>(factor, d_scales, d_map, hoff, off, Minv, MinvT, stage, NT, nb, d_B, ldb, nrhs, num_sms, st, sm, h_map, nearP);
    }
}

extern "C" {

int krr_potrs(const void* d_factor, const float* d_scales, const uint8_t* d_map, const uint8_t* h_map, int64_t n,
              int nb, float* d_B, int64_t ldb, int nrhs, void* d_ws, size_t ws_bytes, void* stream) {
    return potrs_impl(d_factor, d_scales, d_map, h_map, n, nb, d_B, ldb, nrhs, d_ws, ws_bytes, stream, true);
}

}  // extern "C"

// ------------------------------------------------------------------------- iterative refinement (R19)
namespace {
struct RefineWs { size_t potrs, R, partial, blk, total; };
RefineWs refine_ws_layout(int64_t n, int nb, int nrhs) {
    RefineWs w;
    const size_t NR = static_cast<size_t>(rhs_class(nrhs));
    size_t o = 0;
    w.potrs = o;   o = align_up(o + potrs_ws_layout(n, nb).total, 1024);
    w.R = o;       o = align_up(o + static_cast<size_t>(n) * nrhs * sizeof(float), 1024);
    w.partial = o; o = align_up(o + static_cast<size_t>(resid_segments(n)) * n * NR * sizeof(double), 1024);
    w.blk = o;     o = align_up(o + (static_cast<size_t>(n) * NR / 256 + 1) * sizeof(double), 1024);
    w.total = o;
    return w;
}

template <int NR>
int residual_run(const AView& av, const float* X, int64_t ldx, const float* Y, int64_t ldy, int64_t n, int nrhs,
                 float* R, double* partial, double* blk, double* d_norm, cudaStream_t st) {
    const int nblk = static_cast<int>(n / kBlk), nseg = resid_segments(n);
    int rc = launch(CAT_MISC, resid_partial_kernel<NR>, dim3(nblk, nseg), dim3(ResidCfg<NR>::NTHR), 0, st, av, X, ldx, nrhs,
                    nblk, nseg, partial);
    if (rc) return rc;
    const int64_t nfin = (n * NR + 255) / 256;
    rc = launch(CAT_MISC, resid_finish_kernel<NR>, dim3(static_cast<unsigned>(nfin)), dim3(256), 0, st,
                static_cast<const double*>(partial), nseg, n, Y, ldy, R, nrhs, blk);
    if (rc) return rc;
    if (d_norm) rc = launch(CAT_MISC, resid_norm_kernel, dim3(1), dim3(256), 0, st, static_cast<const double*>(blk), nfin, d_norm);
    return rc;
}
}  // namespace

extern "C" {

size_t krr_refine_workspace(int64_t n, int nb, int nrhs) {
    if (krr_potrs_workspace(n, nb, nrhs) == 0) return 0;
    return refine_ws_layout(n, nb, nrhs).total;
}

int krr_refine(const float* d_A, int64_t n, int64_t lda, int nb, const void* d_factor, const float* d_scales,
               const uint8_t* d_map, const uint8_t* h_map, const float* d_Y, int64_t ldy, float* d_X, int64_t ldx,
               int nrhs, int steps, double* d_resid, void* d_ws, size_t ws_bytes, unsigned flags, void* stream) {
    g_launches = 0;
    if (!d_A || !d_factor || !d_scales || !d_map || !h_map || !d_Y || !d_X || !d_ws) return KRR_ERR_ARG;
    int rc = check_shape(n, nb);
    if (rc) return rc;
    const bool tiled = (flags & KRR_FLAG_A_TILED_LOWER) != 0;
    if ((flags & ~static_cast<unsigned>(KRR_FLAG_A_TILED_LOWER)) != 0) return KRR_ERR_ARG;
    if (nrhs < 1 || nrhs > kMaxRhs || ldy < nrhs || ldx < nrhs || steps < 0 || steps > 64) return KRR_ERR_ARG;
    if (!tiled && lda < n) return KRR_ERR_ARG;
    if (static_cast<int64_t>(rhs_class(nrhs)) * nb > 32768) return KRR_ERR_SHAPE;
    if (reinterpret_cast<uintptr_t>(d_ws) % 1024 != 0) return KRR_ERR_ARG;
    const RefineWs L = refine_ws_layout(n, nb, nrhs);
    if (ws_bytes < L.total) return KRR_ERR_WORKSPACE;
    rc = check_device(nullptr);
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    uint8_t* ws = static_cast<uint8_t*>(d_ws);
    float* R = reinterpret_cast<float*>(ws + L.R);
    double* partial = reinterpret_cast<double*>(ws + L.partial);
    double* blk = reinterpret_cast<double*>(ws + L.blk);
    AView av{d_A, lda, tiled ? 1 : 0, static_cast<int>(n / nb), nb};
    int64_t launches = 0;
    auto residual = [&](double* d_norm) -> int {
        switch (rhs_class(nrhs)) {
            case 4:  return residual_run<4>(av, d_X, ldx, d_Y, ldy, n, nrhs, R, partial, blk, d_norm, st);
            case 8:  return residual_run<8>(av, d_X, ldx, d_Y, ldy, n, nrhs, R, partial, blk, d_norm, st);
            case 16: return residual_run<16>(av, d_X, ldx, d_Y, ldy, n, nrhs, R, partial, blk, d_norm, st);
            default: return residual_run<32>(av, d_X, ldx, d_Y, ldy, n, nrhs, R, partial, blk, d_norm, st);
        }
    };
    for (int s = 0; s < steps; ++s) {
        rc = residual(d_resid ? d_resid + s : nullptr);
        if (rc) return rc;
        launches += g_launches;
        // (resets the launch counter; the inverses of the diagonal tiles stay in the workspace after the first step)
        rc = potrs_impl(d_factor, d_scales, d_map, h_map, n, nb, R, nrhs, nrhs, ws + L.potrs, L.R - L.potrs, stream, s == 0);
        if (rc) return rc;
        const int64_t ne = n * nrhs;
        rc = launch(CAT_MISC, refine_update_kernel, dim3(static_cast<unsigned>((ne + 255) / 256)), dim3(256), 0, st, d_X, ldx,
                    static_cast<const float*>(R), n, nrhs);
        if (rc) return rc;
        launches += g_launches;
        g_launches = 0;
    }
    if (d_resid) {
        rc = residual(d_resid + steps);
        if (rc) return rc;
    }
    g_launches += launches;
    return KRR_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------- preconditioned CG (R20)
namespace {
struct PcgWs { size_t potrs, x, r, q, p, z, partial, blk, dot, scal, total; };
PcgWs pcg_ws_layout(int64_t n, int nb, int nrhs) {
    PcgWs w;
    const size_t NR = static_cast<size_t>(rhs_class(nrhs));
    const size_t vec64 = static_cast<size_t>(n) * nrhs * sizeof(double), vec32 = static_cast<size_t>(n) * nrhs * sizeof(float);
    size_t o = 0;
    w.potrs = o;   o = align_up(o + potrs_ws_layout(n, nb).total, 1024);
    w.x = o;       o = align_up(o + vec64, 1024);
    w.r = o;       o = align_up(o + vec64, 1024);
    w.q = o;       o = align_up(o + vec64, 1024);
    w.p = o;       o = align_up(o + vec32, 1024);
    w.z = o;       o = align_up(o + vec32, 1024);
    w.partial = o; o = align_up(o + static_cast<size_t>(resid_segments(n)) * n * NR * sizeof(double), 1024);
    w.blk = o;     o = align_up(o + (static_cast<size_t>(n) * NR / 256 + 1) * sizeof(double), 1024);
    w.dot = o;     o = align_up(o + (static_cast<size_t>(n) / kDotRows + 1) * kMaxRhsDot * sizeof(double), 1024);
    w.scal = o;    o = align_up(o + 3 * kMaxRhsDot * sizeof(double), 1024);
    w.total = o;
    return w;
}

// partial products of A with the compact FP32 vectors V, then out64 = Y - A V (Y given) or A V
template <int NR>
int symm_run(const AView& av, const float* V, int64_t ldv, const float* Y, int64_t ldy, int64_t n, int nrhs, double* partial,
             double* out64, float* out32, double* blk, cudaStream_t st) {
    const int nblk = static_cast<int>(n / kBlk), nseg = resid_segments(n);
    int rc = launch(CAT_MISC, resid_partial_kernel<NR>, dim3(nblk, nseg), dim3(ResidCfg<NR>::NTHR), 0, st, av, V, ldv, nrhs,
                    nblk, nseg, partial);
    if (rc) return rc;
    const int64_t nfin = (n * NR + 255) / 256;
    return launch(CAT_MISC, pcg_finish_kernel<NR>, dim3(static_cast<unsigned>(nfin)), dim3(256), 0, st,
                  static_cast<const double*>(partial), nseg, n, Y, ldy, out64, out32, nrhs, blk);
}

template <typename TA, typename TB>
int coldot(const TA* a, const TB* b, int64_t n, int nrhs, double* part, double* out, cudaStream_t st) {
    const int64_t nb_ = (n + kDotRows - 1) / kDotRows;
    int rc = launch(CAT_MISC, coldot_partial_kernel<TA, TB>, dim3(static_cast<unsigned>(nb_)), dim3(kDotRows), 0, st, a, b, n, nrhs, part);
    if (rc) return rc;
    return launch(CAT_MISC, coldot_final_kernel, dim3(1), dim3(kMaxRhsDot), 0, st, static_cast<const double*>(part), nb_, nrhs, out);
}
}  // namespace

extern "C" {

size_t krr_pcg_workspace(int64_t n, int nb, int nrhs) {
    if (krr_potrs_workspace(n, nb, nrhs) == 0) return 0;
    return pcg_ws_layout(n, nb, nrhs).total;
}

int krr_pcg(const float* d_A, int64_t n, int64_t lda, int nb, const void* d_factor, const float* d_scales,
            const uint8_t* d_map, const uint8_t* h_map, const float* d_Y, int64_t ldy, float* d_X, int64_t ldx,
            int nrhs, int iters, double* d_resid, void* d_ws, size_t ws_bytes, unsigned flags, void* stream) {
    g_launches = 0;
    if (!d_A || !d_factor || !d_scales || !d_map || !h_map || !d_Y || !d_X || !d_ws) return KRR_ERR_ARG;
    int rc = check_shape(n, nb);
    if (rc) return rc;
    const bool tiled = (flags & KRR_FLAG_A_TILED_LOWER) != 0;
    if ((flags & ~static_cast<unsigned>(KRR_FLAG_A_TILED_LOWER)) != 0) return KRR_ERR_ARG;
    if (nrhs < 1 || nrhs > kMaxRhs || ldy < nrhs || ldx < nrhs || iters < 0 || iters > 1024) return KRR_ERR_ARG;
    if (!tiled && lda < n) return KRR_ERR_ARG;
    if (static_cast<int64_t>(rhs_class(nrhs)) * nb > 32768) return KRR_ERR_SHAPE;
    if (reinterpret_cast<uintptr_t>(d_ws) % 1024 != 0) return KRR_ERR_ARG;
    const PcgWs L = pcg_ws_layout(n, nb, nrhs);
    if (ws_bytes < L.total) return KRR_ERR_WORKSPACE;
    rc = check_device(nullptr);
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    uint8_t* ws = static_cast<uint8_t*>(d_ws);
    double* x = reinterpret_cast<double*>(ws + L.x);
    double* r = reinterpret_cast<double*>(ws + L.r);
    double* qv = reinterpret_cast<double*>(ws + L.q);
    float* p = reinterpret_cast<float*>(ws + L.p);
    float* z = reinterpret_cast<float*>(ws + L.z);
    double* partial = reinterpret_cast<double*>(ws + L.partial);
    double* blk = reinterpret_cast<double*>(ws + L.blk);
    double* dot = reinterpret_cast<double*>(ws + L.dot);
    double* rho[2] = {reinterpret_cast<double*>(ws + L.scal), reinterpret_cast<double*>(ws + L.scal) + kMaxRhsDot};
    double* pq = reinterpret_cast<double*>(ws + L.scal) + 2 * kMaxRhsDot;
    AView av{d_A, lda, tiled ? 1 : 0, static_cast<int>(n / nb), nb};
    const int64_t ne = n * nrhs;
    const unsigned gel = static_cast<unsigned>((ne + 255) / 256);
    int64_t launches = 0;
    auto symm = [&](const float* V, int64_t ldv, const float* Yp, double* out64, float* out32, double* blkp) -> int {
        switch (rhs_class(nrhs)) {
            case 4:  return symm_run<4>(av, V, ldv, Yp, ldy, n, nrhs, partial, out64, out32, blkp, st);
            case 8:  return symm_run<8>(av, V, ldv, Yp, ldy, n, nrhs, partial, out64, out32, blkp, st);
            case 16: return symm_run<16>(av, V, ldv, Yp, ldy, n, nrhs, partial, out64, out32, blkp, st);
            default: return symm_run<32>(av, V, ldv, Yp, ldy, n, nrhs, partial, out64, out32, blkp, st);
        }
    };
    bool prepared = false;                            // the inverses of the diagonal tiles are computed by the first solve only
    auto solve = [&]() -> int {                       // z <- (L L^T)^-1 z; the solve resets the launch counter
        launches += g_launches;
        int e = potrs_impl(d_factor, d_scales, d_map, h_map, n, nb, z, nrhs, nrhs, ws + L.potrs, L.x - L.potrs, stream, !prepared);
        prepared = true;
        launches += g_launches;
        g_launches = 0;
        return e;
    };
    auto norm_to = [&](double* out, int64_t nblocks) -> int {
        return launch(CAT_MISC, resid_norm_kernel, dim3(1), dim3(256), 0, st, static_cast<const double*>(blk), nblocks, out);
    };
    const int64_t nfin = (n * rhs_class(nrhs) + 255) / 256;
    // r_0 = Y - A alpha_0, z_0 = M^-1 r_0, p_0 = z_0, rho_0 = r_0 . z_0
    rc = launch(CAT_MISC, pcg_load_x_kernel, dim3(gel), dim3(256), 0, st, static_cast<const float*>(d_X), ldx, x, n, nrhs);
    if (rc) return rc;
    rc = symm(d_X, ldx, d_Y, r, z, d_resid ? blk : nullptr);
    if (rc) return rc;
    if (d_resid) { rc = norm_to(d_resid, nfin); if (rc) return rc; }
    if (iters > 0) {
        rc = solve();
        if (rc) return rc;
        rc = coldot(static_cast<const double*>(r), static_cast<const float*>(z), n, nrhs, dot, rho[0], st);
        if (rc) return rc;
        KRR_CUDA_CHECK(cudaMemcpyAsync(p, z, static_cast<size_t>(ne) * sizeof(float), cudaMemcpyDeviceToDevice, st));
    }
    for (int k = 0; k < iters; ++k) {
        double* rho_k = rho[k & 1];
        double* rho_n = rho[(k + 1) & 1];
        rc = symm(p, nrhs, nullptr, qv, nullptr, nullptr);                                       // q = A p
        if (rc) return rc;
        rc = coldot(static_cast<const float*>(p), static_cast<const double*>(qv), n, nrhs, dot, pq, st);
        if (rc) return rc;
        rc = launch(CAT_MISC, pcg_update_xr_kernel, dim3(gel), dim3(256), 0, st, x, r, static_cast<const float*>(p),
                    static_cast<const double*>(qv), static_cast<const double*>(rho_k), static_cast<const double*>(pq), z, n, nrhs, blk);
        if (rc) return rc;
        if (d_resid) { rc = norm_to(d_resid + k + 1, gel); if (rc) return rc; }
        if (k + 1 == iters) break;                                                               // no further direction needed
        rc = solve();
        if (rc) return rc;
        rc = coldot(static_cast<const double*>(r), static_cast<const float*>(z), n, nrhs, dot, rho_n, st);
        if (rc) return rc;
        rc = launch(CAT_MISC, pcg_update_p_kernel, dim3(gel), dim3(256), 0, st, p, static_cast<const float*>(z),
                    static_cast<const double*>(rho_k), static_cast<const double*>(rho_n), n, nrhs);
        if (rc) return rc;
    }
    if (iters > 0) {
        rc = launch(CAT_MISC, pcg_store_x_kernel, dim3(gel), dim3(256), 0, st, d_X, ldx, static_cast<const double*>(x), n, nrhs);
        if (rc) return rc;
    }
    g_launches += launches;
    return KRR_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------- host-buffer Associate
namespace {
struct Arena {
    size_t A, Y, map, norms, amax, fro, info, scales, pm_ws, factor, potrf_ws, potrs_ws, total;
};
Arena arena_layout(int64_t n, int nb, int nrhs);
}  // namespace
static int build_rows(const int8_t* d_G, int64_t n, int64_t n_valid, int64_t p, int64_t ldg, const float* d_C, int q,
                      int64_t ldc, float gamma, float lambda, float* d_A, int64_t lda, int nb, unsigned flags, void* d_stats,
                      void* d_ws, size_t ws_bytes, void* stream, int64_t row_lo, int64_t row_hi);

static int associate_in_arena(uint8_t* ar, const Arena& L, int64_t n, int nb, float eps_target, unsigned allowed_mask, int force_prec,
                              unsigned flags, int nrhs, float* h_alpha, uint8_t* h_map, int* h_info, void* stream, int64_t launches,
                              const void* build_stats = nullptr);
namespace {
Arena arena_layout(int64_t n, int nb, int nrhs) {
    const size_t NT = n / nb, nslots = NT * (NT + 1) / 2;
    Arena a;
    size_t o = 0;
    a.A = o;        o = align_up(o + static_cast<size_t>(n) * n * sizeof(float), 1024);
    a.Y = o;        o = align_up(o + static_cast<size_t>(n) * nrhs * sizeof(float), 1024);
    a.map = o;      o = align_up(o + NT * NT, 1024);
    a.norms = o;    o = align_up(o + NT * NT * sizeof(float), 1024);
    a.amax = o;     o = align_up(o + NT * NT * sizeof(float), 1024);
    a.fro = o;      o = align_up(o + sizeof(double), 1024);
    a.info = o;     o = align_up(o + sizeof(int), 1024);
    a.scales = o;   o = align_up(o + NT * NT * sizeof(float), 1024);
    a.pm_ws = o;    o = align_up(o + krr_precision_map_workspace(n, nb), 1024);
    a.factor = o;   o = align_up(o + nslots * nb * nb * sizeof(float), 1024);
    a.potrf_ws = o; o = align_up(o + potrf_ws_layout(n, nb, nslots, 0).total, 1024);     // worst case: every tile FP32 (hi + lo images)
    a.potrs_ws = o; o = align_up(o + krr_potrs_workspace(n, nb, nrhs), 1024);
    a.total = o;
    return a;
}
}  // namespace

extern "C" {

size_t krr_associate_host_arena(int64_t n, int nb, int nrhs) {
    if (check_shape(n, nb) != KRR_OK || nrhs < 1 || nrhs > kMaxRhs) return 0;
    return arena_layout(n, nb, nrhs).total;
}

int krr_associate_host(const float* h_A, int64_t n, int64_t lda, int nb, float eps_target, unsigned allowed_mask,
                       int force_prec, unsigned flags, const float* h_Y, int nrhs, float* h_alpha, uint8_t* h_map,
                       int* h_info, void* d_arena, size_t arena_bytes, void* stream) {
    if (!h_A || !h_Y || !h_alpha || !h_map || !h_info || !d_arena) return KRR_ERR_ARG;
    int rc = check_shape(n, nb);
    if (rc) return rc;
    if (nrhs < 1 || nrhs > kMaxRhs || lda < n) return KRR_ERR_ARG;
    if (flags & KRR_FLAG_A_TILED_LOWER) return KRR_ERR_UNSUPPORTED;
    if (force_prec > KRR_FP8_E4M3) return KRR_ERR_ARG;
    const Arena L = arena_layout(n, nb, nrhs);
    if (arena_bytes < L.total) return KRR_ERR_WORKSPACE;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    uint8_t* ar = static_cast<uint8_t*>(d_arena);
    float* dA = reinterpret_cast<float*>(ar + L.A);
    float* dY = reinterpret_cast<float*>(ar + L.Y);
    // only the lower tiles are read by the phase: tile row i needs its first (i+1)*nb columns
    for (int64_t i = 0; i < n / nb; ++i)
        KRR_CUDA_CHECK(cudaMemcpy2DAsync(dA + i * nb * n, n * sizeof(float), h_A + i * nb * lda, lda * sizeof(float),
                                         static_cast<size_t>(i + 1) * nb * sizeof(float), nb, cudaMemcpyHostToDevice, st));
    KRR_CUDA_CHECK(cudaMemcpyAsync(dY, h_Y, static_cast<size_t>(n) * nrhs * sizeof(float), cudaMemcpyHostToDevice, st));
    return associate_in_arena(ar, L, n, nb, eps_target, allowed_mask, force_prec, flags, nrhs, h_alpha, h_map, h_info, stream, 0);
}

}  // extern "C"

// Associate phase on A and Y already in the arena: map -> factorisation -> solve -> alpha, map, info to the host.
static int associate_in_arena(uint8_t* ar, const Arena& L, int64_t n, int nb, float eps_target, unsigned allowed_mask, int force_prec,
                              unsigned flags, int nrhs, float* h_alpha, uint8_t* h_map, int* h_info, void* stream, int64_t launches,
                              const void* build_stats) {
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    float* dA = reinterpret_cast<float*>(ar + L.A);
    float* dY = reinterpret_cast<float*>(ar + L.Y);
    uint8_t* dmap = ar + L.map;
    const int NT = static_cast<int>(n / nb);
    int rc;
    if (force_prec < 0) {
        if (build_stats)
            rc = krr_precision_map_from_build(build_stats, n, nb, eps_target, allowed_mask, dmap, reinterpret_cast<float*>(ar + L.norms),
                                              reinterpret_cast<float*>(ar + L.amax), reinterpret_cast<double*>(ar + L.fro), stream);
        else
            rc = krr_precision_map(dA, n, n, nb, eps_target, allowed_mask, flags & KRR_FLAG_PREROUND_A, dmap,
                                   reinterpret_cast<float*>(ar + L.norms), reinterpret_cast<float*>(ar + L.amax),
                                   reinterpret_cast<double*>(ar + L.fro), ar + L.pm_ws, L.potrf_ws - L.pm_ws, stream);
        if (rc) return rc;
        launches += g_launches;
        // the launch sequence of the factorisation is built on the host from the map
        KRR_CUDA_CHECK(cudaMemcpyAsync(h_map, dmap, static_cast<size_t>(NT) * NT, cudaMemcpyDeviceToHost, st));
        KRR_CUDA_CHECK(cudaStreamSynchronize(st));
    } else {
        for (int i = 0; i < NT; ++i)
            for (int j = 0; j < NT; ++j)
                h_map[i * NT + j] = (j > i) ? 255 : (i == j ? KRR_FP32 : static_cast<uint8_t>(force_prec));
        KRR_CUDA_CHECK(cudaMemcpyAsync(dmap, h_map, static_cast<size_t>(NT) * NT, cudaMemcpyHostToDevice, st));
    }
    rc = krr_potrf_mp(dA, n, n, nb, dmap, h_map, ar + L.factor, reinterpret_cast<float*>(ar + L.scales),
                      reinterpret_cast<int*>(ar + L.info), ar + L.potrf_ws, L.potrs_ws - L.potrf_ws,
                      flags & KRR_FLAG_PREROUND_A, stream);
    if (rc) return rc;
    launches += g_launches;
    rc = krr_potrs(ar + L.factor, reinterpret_cast<float*>(ar + L.scales), dmap, h_map, n, nb, dY, nrhs, nrhs,
                   ar + L.potrs_ws, L.total - L.potrs_ws, stream);
    if (rc) return rc;
    launches += g_launches;
    KRR_CUDA_CHECK(cudaMemcpyAsync(h_alpha, dY, static_cast<size_t>(n) * nrhs * sizeof(float), cudaMemcpyDeviceToHost, st));
    KRR_CUDA_CHECK(cudaMemcpyAsync(h_info, ar + L.info, sizeof(int), cudaMemcpyDeviceToHost, st));
    KRR_CUDA_CHECK(cudaStreamSynchronize(st));
    g_launches = launches;
    return KRR_OK;
}

extern "C" {

// ------------------------------------------------------------------------- Build + Associate from host genotypes
static size_t fit_g_bytes(int64_t n, int64_t p) { return align_up(static_cast<size_t>(n) * align_up(static_cast<size_t>(p), 16), 1024); }

size_t krr_fit_host_arena(int64_t n, int64_t p, int nb, int nrhs) {
    if (check_shape(n, nb) != KRR_OK || nrhs < 1 || nrhs > kMaxRhs || p < 1 || n % 256 != 0 || nb % 256 != 0) return 0;
    return arena_layout(n, nb, nrhs).total + fit_g_bytes(n, p) + krr_build_workspace(n, p, 0) + krr_build_stats_bytes(n, nb);
}

int krr_fit_host(const int8_t* h_G, int64_t n, int64_t p, int64_t ldg, float gamma, float lambda, int nb, float eps_target,
                 unsigned allowed_mask, int force_prec, unsigned flags, const float* h_Y, int nrhs, float* h_alpha,
                 uint8_t* h_map, int* h_info, void* d_arena, size_t arena_bytes, void* stream) {
    if (!h_G || !h_Y || !h_alpha || !h_map || !h_info || !d_arena) return KRR_ERR_ARG;
    int rc = check_shape(n, nb);
    if (rc) return rc;
    if (n % 256 != 0 || nb % 256 != 0) return KRR_ERR_SHAPE;
    if (nrhs < 1 || nrhs > kMaxRhs || p < 1 || ldg < p || force_prec > KRR_FP8_E4M3) return KRR_ERR_ARG;
    if (flags & ~KRR_FLAG_PREROUND_A) return KRR_ERR_UNSUPPORTED;
    if (arena_bytes < krr_fit_host_arena(n, p, nb, nrhs)) return KRR_ERR_WORKSPACE;
    const Arena L = arena_layout(n, nb, nrhs);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    uint8_t* ar = static_cast<uint8_t*>(d_arena);
    int8_t* dG = reinterpret_cast<int8_t*>(ar + L.total);
    uint8_t* bws = ar + L.total + fit_g_bytes(n, p);
    const int64_t ldd = static_cast<int64_t>(align_up(static_cast<size_t>(p), 16));
    KRR_CUDA_CHECK(cudaMemcpyAsync(ar + L.Y, h_Y, static_cast<size_t>(n) * nrhs * sizeof(float), cudaMemcpyHostToDevice, st));
    // tile statistics from the Build epilogue: the precision map needs no pass of its own over A
    uint8_t* stats = bws + krr_build_workspace(n, p, 0);
    // The genotypes cross PCIe in strips of whole tile rows on an internal copy stream; the rows of A that a strip completes
    // (their blocks need the rows of G up to the strip's end only: lower triangle) are built on the caller's stream as soon
    // as the strip has arrived, so the Build runs behind the copy instead of after it.  Same kernels, same blocks, same
    // per-block arithmetic as krr_build in one launch: identical bits.
    int64_t strip_rows = (n / 8 + nb - 1) / nb * nb;
    if (strip_rows < nb) strip_rows = nb;
    const int nstrips = static_cast<int>((n + strip_rows - 1) / strip_rows);
    rc = g_pipe.init();
    if (rc) return rc;
    cudaStream_t sc = g_pipe.mid;
    enum { EV_FORK = 0, EV_BASE = 4 };
    KRR_CUDA_CHECK(cudaEventRecord(g_pipe.event(EV_FORK), st));
    KRR_CUDA_CHECK(cudaStreamWaitEvent(sc, g_pipe.event(EV_FORK), 0));
    int64_t launches = 0;
    for (int s = 0; s < nstrips; ++s) {
        const int64_t r0 = s * strip_rows, r1 = (r0 + strip_rows < n) ? r0 + strip_rows : n;
        KRR_CUDA_CHECK(cudaMemcpy2DAsync(dG + r0 * ldd, ldd, h_G + r0 * ldg, ldg, p, r1 - r0, cudaMemcpyHostToDevice, sc));
        KRR_CUDA_CHECK(cudaEventRecord(g_pipe.event(EV_BASE + s), sc));
        KRR_CUDA_CHECK(cudaStreamWaitEvent(st, g_pipe.event(EV_BASE + s), 0));
        g_launches = 0;
        rc = build_rows(dG, n, n, p, ldd, nullptr, 0, 0, gamma, lambda, reinterpret_cast<float*>(ar + L.A), n, nb, 0,
                        force_prec < 0 ? stats : nullptr, bws, krr_build_workspace(n, p, 0), stream, r0, r1);
        if (rc) return rc;
        launches += g_launches;
    }
    g_launches = launches;
    return associate_in_arena(ar, L, n, nb, eps_target, allowed_mask, force_prec, flags, nrhs, h_alpha, h_map, h_info, stream, g_launches,
                              force_prec < 0 ? stats : nullptr);
}

}  // extern "C"

// ------------------------------------------------------------------------- Build phase (NEXT-1)
namespace {
// genotypes as a [rows][p] byte matrix, box = 128 SNPs x 128 patients, 128-byte swizzle, zero fill past p
int make_genotype_tmap(CUtensorMap* tm, const int8_t* G, int64_t rows, int64_t p, int64_t ld) {
    EncodeTiledFn enc = get_encode_fn();
    if (!enc) return KRR_ERR_CUDA;
    cuuint64_t gdim[2] = {static_cast<cuuint64_t>(p), static_cast<cuuint64_t>(rows)};
    cuuint64_t gstride[1] = {static_cast<cuuint64_t>(ld)};
    cuuint32_t box[2] = {128u, static_cast<cuuint32_t>(kBlk)};
    cuuint32_t estr[2] = {1, 1};
    return enc(tm, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<int8_t*>(G), gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS
               ? KRR_OK : KRR_ERR_CUDA;
}
int launch_build(const CUtensorMap& tmR, const CUtensorMap& tmG, const BuildOp& op, int64_t blocks, int nacc, int num_sms,
                 cudaStream_t st) {
    bool& attr_done = dev_state().build_attrs_done;
    if (!attr_done) {
        KRR_CUDA_CHECK(cudaFuncSetAttribute(build_tc_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, build_smem(1)));
        KRR_CUDA_CHECK(cudaFuncSetAttribute(build_tc_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, build_smem(2)));
        attr_done = true;
    }
    const int64_t max_pairs = num_sms / 2;
    const int grid = static_cast<int>(2 * (blocks < max_pairs ? blocks : max_pairs));
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(kBuildThreads); cfg.dynamicSmemBytes = build_smem(nacc); cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    ProfScope ps(CAT_MISC, st);
    ++g_launches;
    const cudaError_t e = (nacc == 2) ? cudaLaunchKernelEx(&cfg, build_tc_kernel<2>, tmR, tmG, op)
                                      : cudaLaunchKernelEx(&cfg, build_tc_kernel<1>, tmR, tmG, op);
    return e == cudaSuccess ? KRR_OK : KRR_ERR_CUDA;
}
}  // namespace

extern "C" {

static size_t ibs_pitch(int64_t p) { return align_up(static_cast<size_t>(2 * p), 16); }

size_t krr_build_workspace(int64_t n, int64_t p, unsigned flags) {
    if (n <= 0 || n % 256 != 0 || p < 1) return 0;
    size_t b = align_up(static_cast<size_t>(n) * sizeof(int), 1024);       // the folded squared norms
    if (flags & KRR_FLAG_KERNEL_IBS) b += align_up(static_cast<size_t>(n) * ibs_pitch(p), 1024);   // encoded genotypes
    return b;
}

static int build_stats_chunks(int nb) { const int upt = nb / 256, nacc = (nb % 512 == 0) ? 2 : 1; return upt * (upt / nacc) * 16; }

size_t krr_build_stats_bytes(int64_t n, int nb) {
    if (check_shape(n, nb) != KRR_OK || nb % 256 != 0) return 0;
    const size_t NT = n / nb, nslots = NT * (NT + 1) / 2, chunks = build_stats_chunks(nb);
    return align_up(nslots * chunks * sizeof(double), 1024) + align_up(nslots * chunks * sizeof(float), 1024) +
           align_up(nslots * sizeof(double), 1024);
}

int krr_precision_map_from_build(const void* d_stats, int64_t n, int nb, float eps_target, unsigned allowed_mask, uint8_t* d_map,
                                 float* d_tile_norms, float* d_tile_amax, double* d_fro, void* stream) {
    g_launches = 0;
    if (!d_stats || !d_map) return KRR_ERR_ARG;
    int rc = check_shape(n, nb);
    if (rc) return rc;
    if (nb % 256 != 0) return KRR_ERR_SHAPE;
    rc = check_device(nullptr);
    if (rc) return rc;
    const int NT = static_cast<int>(n / nb);
    const size_t nslots = static_cast<size_t>(NT) * (NT + 1) / 2, chunks = build_stats_chunks(nb);
    const uint8_t* sb = static_cast<const uint8_t*>(d_stats);
    const double* partial = reinterpret_cast<const double*>(sb);
    const float* pamax = reinterpret_cast<const float*>(sb + align_up(nslots * chunks * sizeof(double), 1024));
    double* sumsq = reinterpret_cast<double*>(const_cast<uint8_t*>(sb) + align_up(nslots * chunks * sizeof(double), 1024) +
                                              align_up(nslots * chunks * sizeof(float), 1024));
    return launch(CAT_MAP, map_decide_kernel, dim3(1), dim3(1024), 0, static_cast<cudaStream_t>(stream), NT, static_cast<int>(chunks),
                  partial, pamax, eps_target, allowed_mask, d_map, d_tile_norms, d_tile_amax, d_fro, sumsq);
}

int krr_build(const int8_t* d_G, int64_t n, int64_t p, int64_t ldg, const float* d_C, int q, int64_t ldc, float gamma,
              float lambda, float* d_A, int64_t lda, int nb, unsigned flags, void* d_stats, void* d_ws, size_t ws_bytes,
              void* stream) {
    return krr_build_bordered(d_G, n, n, p, ldg, d_C, q, ldc, gamma, lambda, d_A, lda, nb, flags, d_stats, d_ws, ws_bytes, stream);
}

}  // extern "C"

// Rows [row_lo, row_hi) of A (whole 256-row units; row_hi = 0: all rows): the squared norms of those rows of G, then the
// blocks of the lower tiles in those rows.  A launch needs the rows [0, row_hi) of G and their squared norms (earlier
// calls): krr_fit_host builds the matrix strip by strip behind the host-to-device copy of the genotypes.
static int build_rows(const int8_t* d_G, int64_t n, int64_t n_valid, int64_t p, int64_t ldg, const float* d_C, int q,
                      int64_t ldc, float gamma, float lambda, float* d_A, int64_t lda, int nb, unsigned flags, void* d_stats,
                      void* d_ws, size_t ws_bytes, void* stream, int64_t row_lo, int64_t row_hi) {
    if (!d_G || !d_A || !d_ws) return KRR_ERR_ARG;
    if (n_valid < 1 || n_valid > n) return KRR_ERR_ARG;
    if (q < 0 || q > kMaxConfounders || (q > 0 && (!d_C || ldc < q))) return KRR_ERR_ARG;
    int rc = check_shape(n, nb);
    if (rc) return rc;
    if (n % 256 != 0 || nb % 256 != 0) return KRR_ERR_SHAPE;
    if (p < 1 || p > 133000 || ldg < p || ldg % 16 != 0) return KRR_ERR_ARG;      // INT32 sums of int8 squares stay exact
    const bool tiled = flags & KRR_FLAG_A_TILED_LOWER;
    const bool ibs = flags & KRR_FLAG_KERNEL_IBS, linear = flags & KRR_FLAG_KERNEL_LINEAR;
    if (flags & ~(KRR_FLAG_A_TILED_LOWER | KRR_FLAG_KERNEL_IBS | KRR_FLAG_KERNEL_LINEAR)) return KRR_ERR_UNSUPPORTED;
    if ((ibs || linear) && q > 0) return KRR_ERR_UNSUPPORTED;                      // confounders belong to the Gaussian kernel
    if (ibs && linear) return KRR_ERR_ARG;
    if (!tiled && (lda < n || lda % 4 != 0)) return KRR_ERR_ARG;
    if (reinterpret_cast<uintptr_t>(d_G) % 16 != 0 || reinterpret_cast<uintptr_t>(d_A) % 16 != 0 ||
        reinterpret_cast<uintptr_t>(d_ws) % 16 != 0)
        return KRR_ERR_ARG;
    if (ws_bytes < krr_build_workspace(n, p, flags)) return KRR_ERR_WORKSPACE;
    int num_sms = 0;
    rc = check_device(&num_sms);
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int* sq = static_cast<int*>(d_ws);
    if (ibs) {      // thermometer-encode, then the same kernel on the encoded matrix (2p columns of 0/1)
        int8_t* U = reinterpret_cast<int8_t*>(static_cast<uint8_t*>(d_ws) + align_up(static_cast<size_t>(n) * sizeof(int), 1024));
        const int64_t ldu = static_cast<int64_t>(ibs_pitch(p));
        rc = launch(CAT_MISC, ibs_encode_kernel, dim3(static_cast<unsigned>(n), static_cast<unsigned>((ldu + 255) / 256 < 64 ? (ldu + 255) / 256 : 64)),
                    dim3(256), 0, st, d_G, n, p, ldg, U, ldu);
        if (rc) return rc;
        d_G = U; ldg = ldu; p = 2 * p;
    }
    const bool strip = row_hi > 0;
    if (strip && (ibs || row_lo % 256 != 0 || row_hi % 256 != 0 || row_lo < 0 || row_hi > n || row_lo >= row_hi)) return KRR_ERR_ARG;
    if (!strip) { row_lo = 0; row_hi = n; }
    rc = launch(CAT_MISC, row_sqnorm_kernel, dim3(static_cast<unsigned>((row_hi - row_lo + 7) / 8)), dim3(256), 0, st,
                d_G + row_lo * ldg, row_hi - row_lo, p, ldg, sq + row_lo);
    if (rc) return rc;
    CUtensorMap tmG;
    rc = make_genotype_tmap(&tmG, d_G, n, p, ldg);
    if (rc) return rc;
    BuildOp op;
    memset(&op, 0, sizeof(op));
    op.ibs = ibs ? 1 : 0; op.alleles = static_cast<float>(p);        // (p was doubled above: 2 N_S alleles)
    op.linear = linear ? 1 : 0; op.lambda = lambda;
    op.n = n; op.m = n; op.rect = 0; op.p = p; op.nb = nb; op.tiled = tiled ? 1 : 0; op.gamma = gamma;
    op.n_valid = n_valid;
    op.diag = static_cast<float>(1.0 + static_cast<double>(lambda));
    op.sq = sq; op.sq_row = sq; op.A = d_A; op.lda = lda;
    op.C = d_C; op.C_row = d_C; op.ldc = ldc; op.ldc_row = ldc; op.q = q;
    if (d_stats) {
        const size_t nslots = static_cast<size_t>(n / nb) * (n / nb + 1) / 2, chunks = build_stats_chunks(nb);
        op.stat_sumsq = static_cast<double*>(d_stats);
        op.stat_amax = reinterpret_cast<float*>(static_cast<uint8_t*>(d_stats) + align_up(nslots * chunks * sizeof(double), 1024));
        op.stats_chunks = static_cast<int>(chunks);
    }
    const int64_t upt = nb / 256;
    const int nacc = (nb % 512 == 0) ? 2 : 1;                      // 256 x 512 blocks when a tile holds them
    if (strip) { op.ru_lo = static_cast<int>(row_lo / 256); op.ru_hi = static_cast<int>(row_hi / 256); }
    int64_t blocks = 0;                                            // wanted blocks of the row range (sizes the grid)
    for (int64_t ru = row_lo / 256; ru < row_hi / 256; ++ru) blocks += (ru / upt + 1) * upt / nacc;
    return launch_build(tmG, tmG, op, blocks, nacc, num_sms, st);
}

extern "C" {

int krr_build_bordered(const int8_t* d_G, int64_t n, int64_t n_valid, int64_t p, int64_t ldg, const float* d_C, int q,
                       int64_t ldc, float gamma, float lambda, float* d_A, int64_t lda, int nb, unsigned flags, void* d_stats,
                       void* d_ws, size_t ws_bytes, void* stream) {
    g_launches = 0;
    return build_rows(d_G, n, n_valid, p, ldg, d_C, q, ldc, gamma, lambda, d_A, lda, nb, flags, d_stats, d_ws, ws_bytes, stream, 0, 0);
}

// The mixed INT8 / FP32 SYRK of ridge regression (Fig. 2): X^T X + lambda I for X = [S^T | C].
int krr_build_rr(const int8_t* d_S, int64_t n, int64_t ns, int64_t p, int64_t lds, const float* d_C, int q, int64_t ldc,
                 float lambda, float* d_A, int64_t lda, int nb, unsigned flags, void* d_ws, size_t ws_bytes, void* stream) {
    if (ns < 1 || q < 0 || q > kMaxConfounders || ns + q > n || (q > 0 && (!d_C || ldc < q))) return KRR_ERR_ARG;
    if (flags & ~static_cast<unsigned>(KRR_FLAG_A_TILED_LOWER)) return KRR_ERR_UNSUPPORTED;
    // the SNP x SNP block on the INT8 tensor cores; rows / columns >= ns + q become the identity border
    int rc = krr_build_bordered(d_S, n, ns + q, p, lds, nullptr, 0, 0, 1.0f, lambda, d_A, lda, nb,
                                flags | KRR_FLAG_KERNEL_LINEAR, nullptr, d_ws, ws_bytes, stream);
    if (rc || q == 0) return rc;
    const int64_t ncol = ns + q, per_block = static_cast<int64_t>(kRrWarps) * kRrRowsPerWarp;
    return launch(CAT_MISC, rr_confounder_rows_kernel, dim3(static_cast<unsigned>((ncol + per_block - 1) / per_block)),
                  dim3(kRrWarps * 32), 0, static_cast<cudaStream_t>(stream), d_S, lds, ns, p, d_C, ldc, q, lambda, d_A, lda,
                  (flags & KRR_FLAG_A_TILED_LOWER) ? 1 : 0, nb, static_cast<int>(n / nb));
}

// ------------------------------------------------------------------------- Predict phase (NEXT-2)
size_t krr_predict_workspace(int64_t m, int64_t n, int64_t p, unsigned flags) {
    if (m <= 0 || n <= 0 || m % 256 != 0 || n % 256 != 0 || p < 1) return 0;
    size_t b = align_up(static_cast<size_t>(m) * sizeof(int), 1024) + align_up(static_cast<size_t>(n) * sizeof(int), 1024) +
               align_up(static_cast<size_t>(m) * n * sizeof(float), 1024);
    if (flags & KRR_FLAG_KERNEL_IBS) b += align_up(static_cast<size_t>(m + n) * ibs_pitch(p), 1024);
    return b;
}

int krr_predict(const int8_t* d_T, int64_t m, int64_t ldt, const int8_t* d_G, int64_t n, int64_t ldg, int64_t p,
                const float* d_CT, int64_t ldct, const float* d_CG, int64_t ldcg, int q, float gamma,
                const float* d_W, int64_t ldw, int nrhs, float* d_P, int64_t ldp, unsigned flags, void* d_ws, size_t ws_bytes,
                void* stream) {
    g_launches = 0;
    if (!d_T || !d_G || !d_W || !d_P || !d_ws) return KRR_ERR_ARG;
    const bool ibs = flags & KRR_FLAG_KERNEL_IBS, linear = flags & KRR_FLAG_KERNEL_LINEAR;
    if (flags & ~(KRR_FLAG_KERNEL_IBS | KRR_FLAG_KERNEL_LINEAR)) return KRR_ERR_UNSUPPORTED;
    if ((ibs || linear) && q > 0) return KRR_ERR_UNSUPPORTED;
    if (ibs && linear) return KRR_ERR_ARG;
    if (q < 0 || q > kMaxConfounders || (q > 0 && (!d_CT || !d_CG || ldct < q || ldcg < q))) return KRR_ERR_ARG;
    if (m <= 0 || n <= 0 || m % 256 != 0 || n % 256 != 0) return KRR_ERR_SHAPE;
    if (p < 1 || p > 133000 || ldg < p || ldg % 16 != 0 || ldt < p || ldt % 16 != 0) return KRR_ERR_ARG;
    if (nrhs < 1 || nrhs > kMaxRhs || ldw < nrhs || ldp < nrhs) return KRR_ERR_ARG;
    if (reinterpret_cast<uintptr_t>(d_G) % 16 != 0 || reinterpret_cast<uintptr_t>(d_T) % 16 != 0 ||
        reinterpret_cast<uintptr_t>(d_ws) % 1024 != 0)
        return KRR_ERR_ARG;
    if (ws_bytes < krr_predict_workspace(m, n, p, flags)) return KRR_ERR_WORKSPACE;
    int num_sms = 0;
    int rc = check_device(&num_sms);
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    uint8_t* ws = static_cast<uint8_t*>(d_ws);
    int* sqT = reinterpret_cast<int*>(ws);
    int* sqG = reinterpret_cast<int*>(ws + align_up(static_cast<size_t>(m) * sizeof(int), 1024));
    float* K = reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(sqG) + align_up(static_cast<size_t>(n) * sizeof(int), 1024));
    if (ibs) {
        int8_t* UT = reinterpret_cast<int8_t*>(reinterpret_cast<uint8_t*>(K) + align_up(static_cast<size_t>(m) * n * sizeof(float), 1024));
        const int64_t ldu = static_cast<int64_t>(ibs_pitch(p));
        int8_t* UG = UT + m * ldu;
        const unsigned gx = static_cast<unsigned>((ldu + 255) / 256 < 64 ? (ldu + 255) / 256 : 64);
        rc = launch(CAT_MISC, ibs_encode_kernel, dim3(static_cast<unsigned>(m), gx), dim3(256), 0, st, d_T, m, p, ldt, UT, ldu);
        if (rc) return rc;
        rc = launch(CAT_MISC, ibs_encode_kernel, dim3(static_cast<unsigned>(n), gx), dim3(256), 0, st, d_G, n, p, ldg, UG, ldu);
        if (rc) return rc;
        d_T = UT; d_G = UG; ldt = ldg = ldu; p = 2 * p;
    }
    rc = launch(CAT_MISC, row_sqnorm_kernel, dim3(static_cast<unsigned>((m + 7) / 8)), dim3(256), 0, st, d_T, m, p, ldt, sqT);
    if (rc) return rc;
    rc = launch(CAT_MISC, row_sqnorm_kernel, dim3(static_cast<unsigned>((n + 7) / 8)), dim3(256), 0, st, d_G, n, p, ldg, sqG);
    if (rc) return rc;
    CUtensorMap tmT, tmG;
    if (make_genotype_tmap(&tmT, d_T, m, p, ldt) || make_genotype_tmap(&tmG, d_G, n, p, ldg)) return KRR_ERR_CUDA;
    BuildOp op;
    memset(&op, 0, sizeof(op));
    op.ibs = ibs ? 1 : 0; op.alleles = static_cast<float>(p);
    op.linear = linear ? 1 : 0; op.lambda = 0.0f;
    op.n = n; op.m = m; op.rect = 1; op.p = p; op.nb = 256; op.tiled = 0; op.gamma = gamma; op.diag = 1.0f;
    op.sq = sqG; op.sq_row = sqT; op.A = K; op.lda = n;
    op.C = d_CG; op.C_row = d_CT; op.ldc = ldcg; op.ldc_row = ldct; op.q = q;
    const int nacc = (n % 512 == 0) ? 2 : 1;
    rc = launch_build(tmT, tmG, op, (m / 256) * (n / (256 * nacc)), nacc, num_sms, st);      // K = test x training kernel matrix
    if (rc) return rc;
    const int nrp = nrhs <= 8 ? 8 : (nrhs <= 16 ? 16 : 32);
    const int64_t rows_per_cta = 8 * (32 / nrp) * 4;                 // 8 warps x groups x 4 rows
    const unsigned grid = static_cast<unsigned>((m + rows_per_cta - 1) / rows_per_cta);
    ProfScope ps(CAT_MISC, st);
    ++g_launches;
    if (nrp == 8) predict_kw_kernel<8><<<grid, 256, 0, st>>>(K, m, n, n, d_W, ldw, nrhs, d_P, ldp);
    else if (nrp == 16) predict_kw_kernel<16><<<grid, 256, 0, st>>>(K, m, n, n, d_W, ldw, nrhs, d_P, ldp);
    else predict_kw_kernel<32><<<grid, 256, 0, st>>>(K, m, n, n, d_W, ldw, nrhs, d_P, ldp);
    return cudaGetLastError() == cudaSuccess ? KRR_OK : KRR_ERR_CUDA;
}

// ------------------------------------------------------------------------- multi-GPU schedule (NEXT-3, host logic only)
int64_t krr_dist_schedule(int NT, int nb, const uint8_t* h_map, int world, int rank, int32_t* h_tasks, int64_t max_tasks) {
    if (NT < 1 || NT > kMaxNT || nb < kBlk || !h_map || world < 1 || rank < 0 || rank >= world) return KRR_ERR_ARG;
    if (check_map(NT, h_map, nullptr) != KRR_OK) return KRR_ERR_MAP;
    std::vector<DistTask> t;
    dist_build_schedule(NT, nb, world, rank,
                        [&](int i, int j) { return static_cast<int64_t>(nb) * nb * prec_bytes(h_map[i * NT + j]); }, &t);
    if (h_tasks) {
        if (static_cast<int64_t>(t.size()) > max_tasks) return KRR_ERR_WORKSPACE;
        for (size_t q = 0; q < t.size(); ++q) {
            int32_t* r = h_tasks + 6 * q;
            r[0] = t[q].op; r[1] = t[q].k; r[2] = t[q].root; r[3] = t[q].nrows;
            r[4] = static_cast<int32_t>(t[q].bytes & 0xffffffffll); r[5] = static_cast<int32_t>(t[q].bytes >> 32);
        }
    }
    return static_cast<int64_t>(t.size());
}

// ------------------------------------------------------------------------- roofline denominators (beside the path)
int krr_peak_probe(int kind, int64_t work, float* h_ms, double* h_flops, void* stream) {
    if (!h_ms || !h_flops || work < 1 || kind < PEAK_F16 || kind > PEAK_F16x3) return KRR_ERR_ARG;
    if (kind != PEAK_FFMA && (work % 16 != 0 || work > (1ll << 30))) return KRR_ERR_ARG;
    int num_sms = 0;
    int rc = check_device(&num_sms);
    if (rc) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    DeviceState& d = dev_state();
    if (!d.peak_attrs_done) {
        KRR_CUDA_CHECK(cudaFuncSetAttribute(peak_mma_kernel<PEAK_F16>, cudaFuncAttributeMaxDynamicSharedMemorySize, kPeakSmem));
        KRR_CUDA_CHECK(cudaFuncSetAttribute(peak_mma_kernel<PEAK_F8>, cudaFuncAttributeMaxDynamicSharedMemorySize, kPeakSmem));
        KRR_CUDA_CHECK(cudaFuncSetAttribute(peak_mma_kernel<PEAK_MXF8>, cudaFuncAttributeMaxDynamicSharedMemorySize, kPeakSmem));
        KRR_CUDA_CHECK(cudaFuncSetAttribute(peak_mma_kernel<PEAK_F16x3>, cudaFuncAttributeMaxDynamicSharedMemorySize, kPeakSmem));
        d.peak_attrs_done = true;
    }
    cudaEvent_t e0 = pool_event(d), e1 = pool_event(d);
    const int pairs = num_sms / 2;
    double flops = 0.0;
    KRR_CUDA_CHECK(cudaEventRecord(e0, st));
    if (kind == PEAK_FFMA) {
        float* sink = nullptr;                                   // never written (the guard value is unreachable)
        peak_ffma_kernel<<<2 * num_sms, 1024, 0, st>>>(static_cast<int>(work), sink);
        flops = 2.0 * num_sms * 1024.0 * static_cast<double>(work) * 128.0 * 2.0;
    } else {
        const int chunks = static_cast<int>(work);
        const double per_mma = 2.0 * 256.0 * 256.0 * (kind == PEAK_F16 || kind == PEAK_F16x3 ? 16.0 : 32.0);
        if (kind == PEAK_F16) peak_mma_kernel<PEAK_F16><<<2 * pairs, kPeakThreads, kPeakSmem, st>>>(chunks);
        else if (kind == PEAK_F8) peak_mma_kernel<PEAK_F8><<<2 * pairs, kPeakThreads, kPeakSmem, st>>>(chunks);
        else if (kind == PEAK_MXF8) peak_mma_kernel<PEAK_MXF8><<<2 * pairs, kPeakThreads, kPeakSmem, st>>>(chunks);
        else peak_mma_kernel<PEAK_F16x3><<<2 * pairs, kPeakThreads, kPeakSmem, st>>>(chunks);
        flops = static_cast<double>(pairs) * chunks * 4.0 * (kind == PEAK_F16x3 ? 3.0 : 1.0) * per_mma;
    }
    ++g_launches;
    if (cudaGetLastError() != cudaSuccess) return KRR_ERR_CUDA;
    KRR_CUDA_CHECK(cudaEventRecord(e1, st));
    KRR_CUDA_CHECK(cudaEventSynchronize(e1));
    KRR_CUDA_CHECK(cudaEventElapsedTime(h_ms, e0, e1));
    *h_flops = flops;
    d.event_pool.push_back(e0);
    d.event_pool.push_back(e1);
    return KRR_OK;
}

}  // extern "C"


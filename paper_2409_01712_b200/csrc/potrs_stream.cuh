// Bulk updates of krr_potrs, streamed: Y_i -= L_ik Z_k (forward, all tile rows behind the chain's) and
// Z_j -= L_kj^T alpha_k (backward) in FP32 FMAs ("forward and backward substitution operations in the full
// FP32 precision"), with the tile read ONCE from HBM by TMA into a shared-memory ring.
//
// Why a second pair of kernels beside potrs_fwd_update_kernel / potrs_bwd_update_kernel (which stay for the single tile on
// the chain stream, where width and latency count): those let a lane own a slice of the SUMMATION range, so the small
// operand (Z_k / alpha_k) is re-read from shared memory with 32 distinct addresses per warp for every 16 FMAs per lane, and
// a warp has 4 KB of loads in flight -- ncu: FMA pipe 25 % active, `long_scoreboard` on top, 1.3 - 1.8 TB/s.  Here a lane owns
// OUTPUT rows (R = 4 rows x NRHS sums in registers), so the small operand is one address per warp (a broadcast read) and
// every element of L costs one shared-memory read for NRHS FMAs; a unit (128 output rows x the whole summation range of
// one tile) is summed by the eight consumer warps of the CTA in slices, and the slices are added in a fixed tree order
// (deterministic).  A ninth warp is the producer: one TMA box of 16 KB per chunk, `nstages` chunks in flight per SM whatever
// the consumers are doing (full / empty mbarriers per ring slot, no CTA-wide barrier per chunk).
//
// The mosaic as a TMA source: every tile's byte size is a multiple of nb^2, so the payload is, for each element size es,
// a 2-D array of es-byte elements with nb columns in which a tile of that element size is nb consecutive rows starting
// at row offset / (nb es): three tensor maps per direction serve all tiles.
//   forward   unit = rows [o0, o0+128) of tile (i, k); chunk = box of 128 rows x 128 bytes (32 / 64 / 128 columns of an
//             FP32 / FP16 / E4M3 tile), 128-byte swizzle (the 16-byte reads of 8 consecutive rows hit 32 banks);
//             warp ks takes the ks-th 16 bytes of every row; lane l the rows l, l+32, l+64, l+96.
//   backward  unit = columns [o0, o0+128) of tile (k, j); chunk = box of 32 / 64 / 128 rows x 128 columns (16 KB);
//             warp ks takes the rows ks, ks+8, ...; lane l the columns 4l .. 4l+3.
//   NRHS = 32: R = 2, two groups of 64 output rows, four slices each.
// The same kernel serves the single tiles of the lookahead (near / mid) with `ksplit` > 1: a block's summation range is cut
// into ksplit units on as many CTAs, and a unit leaves its sum in a partial buffer instead of adding it to B.
#pragma once
#include "potrs.cuh"
#include "ptx.cuh"

namespace krr {

template <int NRHS>
struct StreamCfg {
    static constexpr int R = (NRHS <= 16) ? 4 : 2;          // output rows per lane
    static constexpr int NACC = R * NRHS;
    static constexpr int RG = 128 / (32 * R);               // groups of 32 R output rows in a unit
    static constexpr int KS = 8 / RG;                       // warps (slices of the summation range) per group
    static constexpr int PIECES = 8 / KS;                   // forward: 16-byte pieces of a 128-byte row segment per warp
    static constexpr int RED_BYTES = RG * (KS / 2) * NACC * 32 * 4;
};
constexpr int kStreamConsumers = 256;                       // 8 consumer warps ...
constexpr int kStreamThreads = kStreamConsumers + 32;       // ... and the producer warp
constexpr int kStreamStage = 16384;
constexpr int kStreamMaxStages = 8;

struct StreamMaps { CUtensorMap m4, m2, m1; };              // element size 4, 2, 1

__device__ __forceinline__ void bulk_load_1d(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(reinterpret_cast<uint64_t>(src)), "r"(bytes), "r"(bar) : "memory");
}

__device__ __forceinline__ void red_add_f32(float* p, float v) {
    asm volatile("red.global.add.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory");
}

// Element e (compile-time after unrolling) of 16 raw bytes of a tile in storage precision P, as FP32 (FP8: the code's
// value; the tile's power-of-two scale multiplies the finished sums).
template <int P>
__device__ __forceinline__ float stream_elem(const uint32_t (&w)[4], int e) {
    if (P == KRR_FP32) return __uint_as_float(w[e]);
    if (P == KRR_FP16) {
        const __half2 h = *reinterpret_cast<const __half2*>(&w[e >> 1]);
        return (e & 1) ? __high2float(h) : __low2float(h);
    }
    return e4m3_to_f32(static_cast<uint8_t>((w[e >> 2] >> (8 * (e & 3))) & 0xffu));
}

// R consecutive elements of precision P at `p` (shared memory) as FP32.
template <int P, int R>
__device__ __forceinline__ void stream_load_r(const uint8_t* p, float (&l)[R]) {
    if (P == KRR_FP32) {
        if (R == 4) { const float4 v = *reinterpret_cast<const float4*>(p); l[0] = v.x; l[1] = v.y; l[R - 2] = v.z; l[R - 1] = v.w; }
        else { const float2 v = *reinterpret_cast<const float2*>(p); l[0] = v.x; l[1] = v.y; }
    } else if (P == KRR_FP16) {
        if (R == 4) {
            const uint2 v = *reinterpret_cast<const uint2*>(p);
            const __half2 a = *reinterpret_cast<const __half2*>(&v.x), b = *reinterpret_cast<const __half2*>(&v.y);
            l[0] = __low2float(a); l[1] = __high2float(a); l[R - 2] = __low2float(b); l[R - 1] = __high2float(b);
        } else {
            const uint32_t v = *reinterpret_cast<const uint32_t*>(p);
            const __half2 a = *reinterpret_cast<const __half2*>(&v);
            l[0] = __low2float(a); l[1] = __high2float(a);
        }
    } else {
        if (R == 4) {
            const uint32_t v = *reinterpret_cast<const uint32_t*>(p);
            l[0] = e4m3_to_f32(v & 0xff); l[1] = e4m3_to_f32((v >> 8) & 0xff);
            l[R - 2] = e4m3_to_f32((v >> 16) & 0xff); l[R - 1] = e4m3_to_f32(v >> 24);
        } else {
            const uint16_t v = *reinterpret_cast<const uint16_t*>(p);
            l[0] = e4m3_to_f32(v & 0xff); l[1] = e4m3_to_f32(v >> 8);
        }
    }
}

// One chunk of a forward unit (128 rows x 128 bytes, 128-byte swizzle): acc[u][h] += the warp's 16-byte pieces of row
// (grp*32R + lane + 32u) times the matching rows of the small operand.
template <int NRHS, int P>
__device__ __forceinline__ void stream_fwd_chunk(const uint8_t* __restrict__ st, int chunk, int grp, int ks, int lane,
                                                 const float* __restrict__ vs, float (&acc)[StreamCfg<NRHS>::NACC]) {
    using C = StreamCfg<NRHS>;
    constexpr int R = C::R, ES = (P == KRR_FP32) ? 4 : (P == KRR_FP16 ? 2 : 1), NE = 16 / ES;
#pragma unroll
    for (int q = 0; q < C::PIECES; ++q) {
        const int piece = ks * C::PIECES + q;
        const int kbase = chunk * (128 / ES) + piece * NE;
        uint32_t raw[R][4];
#pragma unroll
        for (int u = 0; u < R; ++u) {
            const int row = grp * 32 * R + lane + 32 * u;
            const uint4 v = *reinterpret_cast<const uint4*>(st + row * 128 + ((piece ^ (row & 7)) << 4));
            raw[u][0] = v.x; raw[u][1] = v.y; raw[u][2] = v.z; raw[u][3] = v.w;
        }
        // the small operand's row for element e + 1 is loaded before the FMAs of element e
        float4 zc[NRHS / 4];
        {
            const float* zr = vs + static_cast<size_t>(kbase) * NRHS;
#pragma unroll
            for (int h = 0; h < NRHS / 4; ++h) zc[h] = *reinterpret_cast<const float4*>(zr + 4 * h);
        }
#pragma unroll
        for (int e = 0; e < NE; ++e) {
            float4 zn[NRHS / 4];
            if (e + 1 < NE) {
                const float* zr = vs + static_cast<size_t>(kbase + e + 1) * NRHS;
#pragma unroll
                for (int h = 0; h < NRHS / 4; ++h) zn[h] = *reinterpret_cast<const float4*>(zr + 4 * h);
            }
#pragma unroll
            for (int u = 0; u < R; ++u) {
                const float l = stream_elem<P>(raw[u], e);
#pragma unroll
                for (int h = 0; h < NRHS / 4; ++h) {
                    acc[u * NRHS + 4 * h + 0] = fmaf(l, zc[h].x, acc[u * NRHS + 4 * h + 0]);
                    acc[u * NRHS + 4 * h + 1] = fmaf(l, zc[h].y, acc[u * NRHS + 4 * h + 1]);
                    acc[u * NRHS + 4 * h + 2] = fmaf(l, zc[h].z, acc[u * NRHS + 4 * h + 2]);
                    acc[u * NRHS + 4 * h + 3] = fmaf(l, zc[h].w, acc[u * NRHS + 4 * h + 3]);
                }
            }
            if (e + 1 < NE) {
#pragma unroll
                for (int h = 0; h < NRHS / 4; ++h) zc[h] = zn[h];
            }
        }
    }
}

// One chunk of a backward unit (RC rows x 128 columns): acc[u][h] += sum over the warp's rows (ks, ks + KS, ...) of
// L[row][grp*32R + lane*R + u] alpha[row][h].
template <int NRHS, int P>
__device__ __forceinline__ void stream_bwd_chunk(const uint8_t* __restrict__ st, int chunk, int grp, int ks, int lane,
                                                 const float* __restrict__ vs, float (&acc)[StreamCfg<NRHS>::NACC]) {
    using C = StreamCfg<NRHS>;
    constexpr int R = C::R, KS = C::KS, ES = (P == KRR_FP32) ? 4 : (P == KRR_FP16 ? 2 : 1), RC = 128 / ES;
    const int rbase = chunk * RC;
    const uint8_t* col = st + (grp * 32 * R + lane * R) * ES;
#pragma unroll 4
    for (int t = 0; t < RC / KS; ++t) {
        const int r = ks + KS * t;
        float l[R];
        stream_load_r<P, R>(col + r * (128 * ES), l);
        const float* ar = vs + static_cast<size_t>(rbase + r) * NRHS;
#pragma unroll
        for (int h = 0; h < NRHS; h += 4) {
            const float4 a = *reinterpret_cast<const float4*>(ar + h);
#pragma unroll
            for (int u = 0; u < R; ++u) {
                acc[u * NRHS + h + 0] = fmaf(l[u], a.x, acc[u * NRHS + h + 0]);
                acc[u * NRHS + h + 1] = fmaf(l[u], a.y, acc[u * NRHS + h + 1]);
                acc[u * NRHS + h + 2] = fmaf(l[u], a.z, acc[u * NRHS + h + 2]);
                acc[u * NRHS + h + 3] = fmaf(l[u], a.w, acc[u * NRHS + h + 3]);
            }
        }
    }
}

// Tiles t_lo .. t_lo + ntiles of tile column k (forward: rows i = t_lo + t) or of tile row k (backward: columns j = t_lo + t).
// grid <= units = ntiles * nb / 128, one persistent CTA per SM (units dealt round-robin).
// smem (1 KB aligned): nstages ring slots | [nb][NRHS] floats | reduction buffer | the tiles' (row base, precision, scale) | mbarriers.
template <int NRHS, bool BWD>
__global__ void __launch_bounds__(kStreamThreads, 1)
potrs_stream_update_kernel(const __grid_constant__ StreamMaps maps, int NT, int nb, int k, int t_lo, int ntiles, int nstages,
                           const int64_t* __restrict__ off, const uint8_t* __restrict__ map, const float* __restrict__ scales,
                           float* __restrict__ B, int64_t ldb, int nrhs, int ksplit, float* __restrict__ P) {
    using C = StreamCfg<NRHS>;
    constexpr int R = C::R, NACC = C::NACC, KS = C::KS;
    extern __shared__ __align__(1024) uint8_t stream_smem[];
    uint8_t* ring = stream_smem;
    float* vs = reinterpret_cast<float*>(ring + static_cast<size_t>(nstages) * kStreamStage);
    float* red = vs + static_cast<size_t>(nb) * NRHS;
    int* t_row = reinterpret_cast<int*>(reinterpret_cast<uint8_t*>(red) + C::RED_BYTES);     // tile's first row in its element-size view
    int* t_prec = t_row + ntiles;
    float* t_scale = reinterpret_cast<float*>(t_prec + ntiles);
    uint64_t* bars = reinterpret_cast<uint64_t*>((reinterpret_cast<uintptr_t>(t_scale + ntiles) + 7) & ~static_cast<uintptr_t>(7));
    const uint32_t full0 = ptx::smem_u32(bars), empty0 = full0 + 8 * kStreamMaxStages, zbar = empty0 + 8 * kStreamMaxStages;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int upt = nb / 128;                                    // 128-row (column) blocks per tile
    // ksplit > 1 (one tile, the chain's "near" tile): a block's summation range is cut into ksplit slices, one unit each,
    // and a unit leaves its sum in P[slice][row][NRHS] -- the next diagonal step's stage kernel subtracts the slices in a
    // fixed order -- so that the 4 MB tile is read by upt * ksplit SMs instead of upt.
    const int nunits = ntiles * upt * ksplit;
    const bool sliced = ksplit > 1 && gridDim.x >= static_cast<unsigned>(nunits);     // one unit per CTA: only its slice of the small operand is needed
    const int zrows = sliced ? nb / ksplit : nb, zrow0 = sliced ? (static_cast<int>(blockIdx.x) % ksplit) * zrows : 0;
    const bool z_bulk = (nrhs == NRHS) && (ldb == NRHS) && (reinterpret_cast<uintptr_t>(B) % 16 == 0);
    for (int t = tid; t < ntiles; t += kStreamThreads) {
        const int idx = BWD ? (k * NT + t_lo + t) : ((t_lo + t) * NT + k);
        const int p = map[idx];
        const int es = (p == KRR_FP32) ? 4 : (p == KRR_FP16 ? 2 : 1);
        t_row[t] = static_cast<int>(off[idx] / (static_cast<int64_t>(nb) * es));
        t_prec[t] = p;
        t_scale[t] = scales[idx];
    }
    if (tid == 0) {
        for (int s = 0; s < nstages; ++s) { ptx::mbar_init(full0 + 8 * s, 1); ptx::mbar_init(empty0 + 8 * s, 8); }
        ptx::mbar_init(zbar, 1);
        ptx::fence_mbar_init();
    }
    pdl_trigger();
    __syncthreads();

    if (warp == 8) {
        // ---------------- producer: one TMA box per chunk, in the order the consumers walk them
        if (lane == 0) {
            ptx::prefetch_tmap(&maps.m4); ptx::prefetch_tmap(&maps.m2); ptx::prefetch_tmap(&maps.m1);
            int slot = 0;
            uint32_t pass = 0;                                   // times the ring has wrapped
            for (int unit = blockIdx.x; unit < nunits; unit += gridDim.x) {
                const int blk = unit / ksplit, slice = unit % ksplit;
                const int t = blk / upt, o0 = (blk % upt) * 128;
                const int p = t_prec[t], row0 = t_row[t];
                const int es = (p == KRR_FP32) ? 4 : (p == KRR_FP16 ? 2 : 1);
                const CUtensorMap* tm = (es == 4) ? &maps.m4 : (es == 2 ? &maps.m2 : &maps.m1);
                const int cps = nb * es / 128 / ksplit;          // chunks per unit
                for (int c = slice * cps; c < (slice + 1) * cps; ++c) {
                    if (pass > 0) {      // polled with a pause: the producer shares its scheduler with two consumer warps
                        uint32_t done = 0, spins = 0;
                        while (true) {
                            asm volatile("{\n\t.reg .pred p;\n\tmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}\n"
                                         : "=r"(done) : "r"(empty0 + 8 * slot), "r"((pass - 1) & 1) : "memory");
                            if (done) break;
                            __nanosleep(200);
                            if (++spins > (1u << 24)) __trap();
                        }
                    }
                    ptx::mbar_arrive_expect_tx(full0 + 8 * slot, kStreamStage);
                    if (!BWD) ptx::tma_load_2d(ptx::smem_u32(ring + static_cast<size_t>(slot) * kStreamStage), tm, full0 + 8 * slot, c * (128 / es), row0 + o0);
                    else      ptx::tma_load_2d(ptx::smem_u32(ring + static_cast<size_t>(slot) * kStreamStage), tm, full0 + 8 * slot, o0, row0 + c * (128 / es));
                    if (++slot == nstages) { slot = 0; ++pass; }
                }
            }
        }
        return;
    }

    // ---------------- consumers
    const int grp = warp / KS, ks = warp % KS;
    auto consumer_bar = [&]() { asm volatile("bar.sync 1, 256;" ::: "memory"); };
    if (blockIdx.x >= static_cast<unsigned>(nunits)) return;
    // Launched as a programmatic dependent (the chain's near tile behind the diagonal step's product), everything above --
    // and the producer warp's first tile loads: the factor is not written during a solve -- runs beside the previous kernel;
    // its output (the small operand, and B / the partial buffer this kernel writes at the end) is touched only behind this wait.
    pdl_wait();
    if (!z_bulk) {      // the small operand: rows k*nb .. of B (the unit's slice of them), zero-padded to NRHS columns
        const float* Vk = B + static_cast<int64_t>(k) * nb * ldb;
        for (int idx = zrow0 * NRHS + tid; idx < (zrow0 + zrows) * NRHS; idx += kStreamConsumers) {
            const int r = idx / NRHS, h = idx % NRHS;
            vs[idx] = (h < nrhs) ? Vk[static_cast<int64_t>(r) * ldb + h] : 0.0f;
        }
        consumer_bar();
    } else {
        if (tid == 0) {
            ptx::mbar_arrive_expect_tx(zbar, static_cast<uint32_t>(zrows) * NRHS * 4);
            bulk_load_1d(ptx::smem_u32(vs + static_cast<size_t>(zrow0) * NRHS), B + (static_cast<int64_t>(k) * nb + zrow0) * ldb,
                         static_cast<uint32_t>(zrows) * NRHS * 4, zbar);
        }
        ptx::mbar_wait(zbar, 0);
    }
    float acc[NACC];
#pragma unroll
    for (int v = 0; v < NACC; ++v) acc[v] = 0.0f;
    int slot = 0;
    uint32_t phase = 0;
    for (int unit = blockIdx.x; unit < nunits; unit += gridDim.x) {
        const int blk = unit / ksplit, slice = unit % ksplit;
        const int t = blk / upt, o0 = (blk % upt) * 128;
        const int p = t_prec[t];
        const int es = (p == KRR_FP32) ? 4 : (p == KRR_FP16 ? 2 : 1);
        const int cps = nb * es / 128 / ksplit;
        for (int c = slice * cps; c < (slice + 1) * cps; ++c) {
            ptx::mbar_wait(full0 + 8 * slot, phase);
            const uint8_t* st = ring + static_cast<size_t>(slot) * kStreamStage;
            if (!BWD) {
                if (es == 4) stream_fwd_chunk<NRHS, KRR_FP32>(st, c, grp, ks, lane, vs, acc);
                else if (es == 2) stream_fwd_chunk<NRHS, KRR_FP16>(st, c, grp, ks, lane, vs, acc);
                else stream_fwd_chunk<NRHS, KRR_FP8_E4M3>(st, c, grp, ks, lane, vs, acc);
            } else {
                if (es == 4) stream_bwd_chunk<NRHS, KRR_FP32>(st, c, grp, ks, lane, vs, acc);
                else if (es == 2) stream_bwd_chunk<NRHS, KRR_FP16>(st, c, grp, ks, lane, vs, acc);
                else stream_bwd_chunk<NRHS, KRR_FP8_E4M3>(st, c, grp, ks, lane, vs, acc);
            }
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(empty0 + 8 * slot);
            if (++slot == nstages) { slot = 0; phase ^= 1u; }
        }
        // the KS slices of every group, added in a fixed tree order
#pragma unroll
        for (int half = KS / 2; half >= 1; half >>= 1) {
            if (ks >= half && ks < 2 * half) {
                float* dst = red + (static_cast<size_t>(grp * (KS / 2) + ks - half) * NACC) * 32 + lane;
#pragma unroll
                for (int v = 0; v < NACC; ++v) dst[v * 32] = acc[v];
            }
            consumer_bar();
            if (ks < half) {
                const float* src = red + (static_cast<size_t>(grp * (KS / 2) + ks) * NACC) * 32 + lane;
#pragma unroll
                for (int v = 0; v < NACC; ++v) acc[v] += src[v * 32];
            }
            consumer_bar();
        }
        if (ks == 0) {
            const float s = (es == 1) ? t_scale[t] : 1.0f;
            if (ksplit > 1) {
                // the slice's sum, for the stage kernel of the next diagonal step
                float* pr = P + (static_cast<size_t>(slice) * nb + o0 + grp * 32 * R) * NRHS;
#pragma unroll
                for (int u = 0; u < R; ++u) {
                    float* out = pr + static_cast<size_t>(BWD ? lane * R + u : lane + 32 * u) * NRHS;
#pragma unroll
                    for (int h = 0; h < NRHS; h += 4)
                        *reinterpret_cast<float4*>(out + h) = make_float4(s * acc[u * NRHS + h], s * acc[u * NRHS + h + 1], s * acc[u * NRHS + h + 2], s * acc[u * NRHS + h + 3]);
                }
            } else {
                const int64_t row0 = static_cast<int64_t>(t_lo + t) * nb + o0 + grp * 32 * R;
#pragma unroll
                for (int u = 0; u < R; ++u) {
                    float* out = B + (row0 + (BWD ? lane * R + u : lane + 32 * u)) * ldb;
#pragma unroll
                    for (int h = 0; h < NRHS; ++h)
                        if (h < nrhs) red_add_f32(out + h, -(s * acc[u * NRHS + h]));   // the unit is the only writer of its rows: same result as a read-modify-write, no round trip
                }
            }
        }
#pragma unroll
        for (int v = 0; v < NACC; ++v) acc[v] = 0.0f;
    }
}

}  // namespace krr

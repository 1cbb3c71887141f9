// Roofline denominators measured on the device the library runs on (SURVEY 8(d) "Which roofline": "FP8 =
// measure with a no-traffic kind::f8f6f4 loop ... FP32 ALU = measure an FFMA loop").  Not on the hot path:
// `krr_peak_probe` is called by bench.py --peaks / paper_2409_01712_b200/peaks.py.
//
//   tensor probes   every CTA pair (cluster of 2, cta_group::2, M = N = 256 -- the shape of the trailing
//                   update) issues MMAs back to back on operand blocks that sit in shared memory (four ring
//                   slots of pseudo-random finite data, so the datapath toggles as in a real product);
//                   no global traffic inside the loop, accumulator in TMEM
//   FFMA probe      8 independent FMA chains per thread, 1024 threads per CTA, 2 CTAs per SM
#pragma once
#include "common.cuh"
#include "ptx.cuh"

namespace krr {

enum { PEAK_F16 = 0, PEAK_F8 = 1, PEAK_MXF8 = 2, PEAK_FFMA = 3, PEAK_F16x3 = 4 };

constexpr int kPeakSlots = 4;
constexpr int kPeakSlotBytes = 2 * 128 * 128;       // [A block 16 KB | B block 16 KB] per CTA
constexpr int kPeakSmem = kPeakSlots * kPeakSlotBytes + 1024 + 64;
constexpr int kPeakThreads = 128;

__device__ __forceinline__ uint32_t peak_hash(uint32_t x) {
    x ^= x >> 16; x *= 0x7feb352dU; x ^= x >> 15; x *= 0x846ca68bU; x ^= x >> 16;
    return x;
}

// One "chunk" = the MMAs of one 128-byte K slice of a ring slot: 4 instructions (K = 16 FP16 / 32 FP8 each);
// PEAK_F16x3 issues the three-instruction FP32-class sequence of gemm_tc.cuh (12 per chunk, two slots).
template <int KIND>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kPeakThreads, 1)
peak_mma_kernel(int chunks) {
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* smem = smem_raw + (smem_base - ptx::smem_u32(smem_raw));
    const uint32_t bar_base = smem_base + kPeakSlots * kPeakSlotBytes;
    const uint32_t tmem_slot = bar_base + 32;
    uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem + kPeakSlots * kPeakSlotBytes + 32);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int rank = static_cast<int>(ptx::cluster_ctarank());
    // pseudo-random finite operands: FP16 in (-2, 2) with full mantissas, E4M3 bytes without the NaN codes
    for (int i = threadIdx.x; i < kPeakSlots * kPeakSlotBytes / 4; i += kPeakThreads) {
        uint32_t h = peak_hash(static_cast<uint32_t>(i) * 2654435761u + blockIdx.x * 97u + 12345u);
        if (KIND == PEAK_F16 || KIND == PEAK_F16x3) {
            // per half: sign | exponent in [11, 15] | 10 mantissa bits
            const uint32_t lo = (h & 0x83ffu) | ((11u + ((h >> 10) & 3u) + ((h >> 12) & 1u)) << 10);
            const uint32_t g = h >> 16;
            const uint32_t hi = (g & 0x83ffu) | ((11u + ((g >> 10) & 3u) + ((g >> 12) & 1u)) << 10);
            h = lo | (hi << 16);
        } else {
            // E4M3: clear bit 6 of every byte -> |x| < 2, never the NaN pattern 0x7f / 0xff
            h &= 0xbfbfbfbfu;
        }
        reinterpret_cast<uint32_t*>(smem)[i] = h;
    }
    ptx::fence_proxy_async();
    if (warp == 0 && lane == 0) {
        ptx::mbar_init(bar_base + 0, 1);
        ptx::mbar_init(bar_base + 8, 1);
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
    if (KIND == PEAK_MXF8) {
        // UE8M0 scale 2^0 for every row and K block: columns 256.. of TMEM
        const uint32_t lane_base = static_cast<uint32_t>(warp * 32) << 16;
        for (int j = 0; j < 16; ++j) ptx::tmem_st_32x32_x4(tmem_base + lane_base + 256 + 4 * j, 0x7f7f7f7fu);
        ptx::tmem_st_wait();
        ptx::tc_fence_before();
        ptx::cluster_sync_all();
        ptx::tc_fence_after();
    }
    if (warp == 0 && rank == 0) {
        constexpr uint32_t idesc16 = ptx::make_idesc(256, 256, 0, 0);
        constexpr uint32_t idesc8 = ptx::make_idesc(256, 256, 0, 0);          // kind::f8f6f4: formats 0 = E4M3
        constexpr uint32_t idescq = ptx::make_idesc_mxf8(256, 256);
        const uint32_t dlo0 = ptx::smem_desc_lo(smem_base);
        constexpr uint32_t kDescSlot = kPeakSlotBytes >> 4, kDescB = (128 * 128) >> 4;
        uint32_t phase[2] = {0, 0};
        uint32_t acc = 0;
        constexpr int kGroup = 16;                                           // chunks per commit
        int groups_issued = 0;
        for (int c0 = 0; c0 < chunks; c0 += kGroup) {
            if (groups_issued >= 2) {                                        // at most two groups in flight
                const int b = groups_issued & 1;
                ptx::mbar_wait(bar_base + 8u * b, phase[b]);
                phase[b] ^= 1u;
            }
            if (ptx::elect_one()) {
#pragma unroll 4
                for (int c = 0; c < kGroup; ++c) {
                    const uint32_t a = dlo0 + ((c0 + c) & (kPeakSlots - 1)) * kDescSlot, b = a + kDescB;
#pragma unroll
                    for (int kk = 3; kk >= 0; --kk) {
                        const uint64_t da = ptx::smem_desc_from_lo(a + 2 * kk), db = ptx::smem_desc_from_lo(b + 2 * kk);
                        if (KIND == PEAK_F16) {
                            ptx::mma_f16_ss_pair(tmem_base, da, db, idesc16, acc);
                        } else if (KIND == PEAK_F16x3) {
                            const uint32_t a2 = dlo0 + ((c0 + c + 1) & (kPeakSlots - 1)) * kDescSlot, b2 = a2 + kDescB;
                            ptx::mma_f16_ss_pair(tmem_base, ptx::smem_desc_from_lo(a2 + 2 * kk), db, idesc16, acc);
                            ptx::mma_f16_ss_pair(tmem_base, da, ptx::smem_desc_from_lo(b2 + 2 * kk), idesc16, 1u);
                            ptx::mma_f16_ss_pair(tmem_base, da, db, idesc16, 1u);
                        } else if (KIND == PEAK_F8) {
                            asm volatile(
                                "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                                "tcgen05.mma.cta_group::2.kind::f8f6f4 [%0], %1, %2, %3, p;\n\t}\n"
                                ::"r"(tmem_base), "l"(da), "l"(db), "r"(idesc8), "r"(acc) : "memory");
                        } else {
                            ptx::mma_mxf8_ss_pair(tmem_base, da, db, idescq, acc, tmem_base + 256, tmem_base + 256 + 8);
                        }
                        acc = 1u;
                    }
                }
                ptx::tc_commit_pair(bar_base + 8u * (groups_issued & 1));
            }
            acc = 1u;
            ++groups_issued;
        }
        for (int g = (groups_issued >= 2 ? groups_issued - 2 : 0); g < groups_issued; ++g) {
            const int b = g & 1;
            ptx::mbar_wait(bar_base + 8u * b, phase[b]);
            phase[b] ^= 1u;
        }
    }
    ptx::tc_fence_before();
    ptx::cluster_sync_all();
    if (warp == 1) ptx::tmem_dealloc<512, 2>(tmem_base);
}

// FFMA probe: 8 independent chains per thread; `out` keeps the compiler from removing them.
__global__ void __launch_bounds__(1024, 2)
peak_ffma_kernel(int iters, float* __restrict__ out) {
    float a[8];
    const float x = 1.0f + 1e-7f * static_cast<float>(threadIdx.x), y = 1e-9f * static_cast<float>(blockIdx.x + 1);
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = static_cast<float>(i) * 0.125f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
#pragma unroll
            for (int i = 0; i < 8; ++i) a[i] = fmaf(a[i], x, y);
        }
    }
    float s = 0.0f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += a[i];
    if (s == 123.456f) out[0] = s;
}

}  // namespace krr

// common.cuh -- shared device/host helpers of libspear.so (sm_100a only).
//
// PTX wrappers (mbarrier, cp.async.bulk / TMA, tcgen05, griddepcontrol, mma.sync), the int4 -> fp16
// dequantisation of the SPW4 layout, and the host-side error plumbing.
// Nothing here is shared with oracle/ (the oracle is plain C compiled by gcc alone).
#pragma once

#include <cuda.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/spear.h"

#ifndef SPEAR_NUM_SMS_FALLBACK
#define SPEAR_NUM_SMS_FALLBACK 148
#endif

namespace spear {

// ------------------------------------------------------------------------------------------------
// host side: error state, launch counter, device info
// ------------------------------------------------------------------------------------------------
int set_error(int status, const char* fmt, ...);
void count_launch(int n = 1);
#define SPEAR_CUDA_OK(expr)                                                                      \
    do {                                                                                         \
        cudaError_t _e = (expr);                                                                 \
        if (_e != cudaSuccess)                                                                   \
            return ::spear::set_error(SPEAR_ECUDA, "%s failed: %s (%s:%d)", #expr,               \
                                      cudaGetErrorString(_e), __FILE__, __LINE__);               \
    } while (0)

struct DeviceInfo {
    int device = -1;
    int num_sms = SPEAR_NUM_SMS_FALLBACK;
    int cc_major = 0, cc_minor = 0;
    size_t smem_optin = 0;
};
const DeviceInfo& device_info();

// Encodes (and caches) a 2-D TMA tensor map over a row-major fp16 matrix [rows][cols] whose rows are
// `row_stride_bytes` apart: box = box_rows x 64 columns (128 bytes), SWIZZLE_128B, zero fill outside.
int get_tensor_map_2d(const void* base, uint64_t rows, uint64_t cols, uint64_t row_stride_bytes,
                      uint32_t box_rows, uint32_t box_cols, CUtensorMap* out);
// 3-D view of the same matrix as [rows][cols / 64][64]: box = box_rows x box_ktiles x 64 columns, SWIZZLE_128B.
int get_tensor_map_x3d(const void* base, uint64_t rows, uint64_t cols, uint32_t box_rows, uint32_t box_ktiles,
                       CUtensorMap* out);

#ifdef __CUDACC__
// ------------------------------------------------------------------------------------------------
// device side
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ uint32_t lane_id() {
    uint32_t l;
    asm volatile("mov.u32 %0, %%laneid;" : "=r"(l));
    return l;
}
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile(
        "{\n\t.reg .pred P;\n\telect.sync _|P, 0xffffffff;\n\tselp.u32 %0, 1, 0, P;\n\t}\n"
        : "=r"(pred));
    return pred != 0;
}

// ---- programmatic dependent launch -----------------------------------------------------------
__device__ __forceinline__ void pdl_launch_dependents() {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// ---- mbarrier ---------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async_smem() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
                 "r"(bytes)
                 : "memory");
}
// The suspend-time hint lets the hardware park the thread until the phase completes (or the hint expires) instead
// of returning after the short default limit: a polling loop of try_wait / branch otherwise eats issue slots of the
// warps that share the scheduler (measured in the layer-stream kernel: a quarter of all issued instructions).
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred P;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 P, [%1], %2, %3;\n\t"
        "selp.u32 %0, 1, 0, P;\n\t}\n"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity), "r"(0x989680u)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {
    }
}

// ---- TMA --------------------------------------------------------------------------------------
// 1-D bulk copy global -> shared, completion on an mbarrier (bytes % 16 == 0, both 16-B aligned).
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar,
                                         uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint "
        "[%0], [%1], %2, [%3], %4;" ::"r"(smem_u32(dst)),
        "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
        : "memory");
}
// 2-D tiled tensor copy global -> shared (c0 = innermost coordinate).
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, int c0, int c1,
                                            uint64_t* bar, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint "
        "[%0], [%1, {%3, %4}], [%2], %5;" ::"r"(smem_u32(dst)),
        "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "l"(policy)
        : "memory");
}
// 3-D tiled tensor copy global -> shared (c0 = innermost coordinate).
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, int c0, int c1, int c2,
                                            uint64_t* bar, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint "
        "[%0], [%1, {%3, %4, %5}], [%2], %6;" ::"r"(smem_u32(dst)),
        "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "l"(policy)
        : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* map) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t policy_evict_last() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ void prefetch_l2(const void* p) {
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}

// ---- int4 -> fp16 (SPW4 word: column 2i in bits [4i,4i+4), column 2i+1 in bits [4i+16,4i+20)) ----
// Returns the four half2 pairs (q-8) of one 32-bit word, columns (0,1) (2,3) (4,5) (6,7); exact.
// Attribution: this is the well-known "magic number" int4 -> fp16 conversion (OR the nibble under the exponent of 1024.0,
// subtract 1024 + zero-point; for the high nibble of a byte multiply by 1/16 first) published with FasterTransformer /
// TensorRT-LLM (FastInterleavedAndBiasedNumericArrayConverter<half, uint4b_t>) and used by Marlin-style kernels.  The
// constants below are fixed by that arithmetic (0x6400 = 1024.0, 0x6408 = 1032.0, 0x2c00 = 1/16, 0xd480 = -72.0) and so
// is the interleaved nibble order of the SPW4 word, chosen so that two lop3 masks yield fp16 pairs.
__device__ __forceinline__ void dequant_word(uint32_t w, uint32_t (&out)[4]) {
    constexpr uint32_t kMagic = 0x64006400u;    // fp16 1024.0 twice
    constexpr uint32_t kSub = 0x64086408u;      // 1032.0  : (1024 + q) - 1032 = q - 8
    constexpr uint32_t kSixteenth = 0x2c002c00u;  // 1/16
    constexpr uint32_t kNeg72 = 0xd480d480u;    // -72     : (1024 + 16 q)/16 - 72 = q - 8
    uint32_t lo0, hi0, lo1, hi1;
    asm("lop3.b32 %0, %1, 0x000f000f, %2, 0xea;" : "=r"(lo0) : "r"(w), "r"(kMagic));
    asm("lop3.b32 %0, %1, 0x00f000f0, %2, 0xea;" : "=r"(hi0) : "r"(w), "r"(kMagic));
    uint32_t w8 = w >> 8;
    asm("lop3.b32 %0, %1, 0x000f000f, %2, 0xea;" : "=r"(lo1) : "r"(w8), "r"(kMagic));
    asm("lop3.b32 %0, %1, 0x00f000f0, %2, 0xea;" : "=r"(hi1) : "r"(w8), "r"(kMagic));
    asm("sub.f16x2 %0, %1, %2;" : "=r"(out[0]) : "r"(lo0), "r"(kSub));
    asm("fma.rn.f16x2 %0, %1, %2, %3;" : "=r"(out[1]) : "r"(hi0), "r"(kSixteenth), "r"(kNeg72));
    asm("sub.f16x2 %0, %1, %2;" : "=r"(out[2]) : "r"(lo1), "r"(kSub));
    asm("fma.rn.f16x2 %0, %1, %2, %3;" : "=r"(out[3]) : "r"(hi1), "r"(kSixteenth), "r"(kNeg72));
}
// ---- int8 -> fp16 (INT8 EC factors): four signed bytes of one word -> two half2, exact ----
// b ^ 0x80 is b + 128 as an unsigned byte; spliced under the exponent byte 0x64 it is the fp16 value 1024 + (b + 128);
// minus 1152 gives b.
__device__ __forceinline__ void cvt_i8x4_f16x2(uint32_t w, uint32_t& lo, uint32_t& hi) {
    const uint32_t x = w ^ 0x80808080u;
    uint32_t a, b;
    asm("prmt.b32 %0, %1, %2, 0x5140;" : "=r"(a) : "r"(x), "r"(0x64646464u));     // bytes: x0, 0x64, x1, 0x64
    asm("prmt.b32 %0, %1, %2, 0x7362;" : "=r"(b) : "r"(x), "r"(0x64646464u));     // bytes: x2, 0x64, x3, 0x64
    asm("sub.f16x2 %0, %1, %2;" : "=r"(lo) : "r"(a), "r"(0x64806480u));
    asm("sub.f16x2 %0, %1, %2;" : "=r"(hi) : "r"(b), "r"(0x64806480u));
}
// ---- 16 consecutive columns of an EC factor row (or of x) as mma.sync fragment registers; NULL row = zeros ----
__device__ __forceinline__ void ec_load16(const __half* row, int col, bool readonly, uint32_t (&lo)[4], uint32_t (&hi)[4]) {
    if (row) {
        uint4 a, b;
        if (readonly) {
            a = __ldg(reinterpret_cast<const uint4*>(row + col));
            b = __ldg(reinterpret_cast<const uint4*>(row + col + 8));
        } else {
            a = *reinterpret_cast<const uint4*>(row + col);
            b = *reinterpret_cast<const uint4*>(row + col + 8);
        }
        lo[0] = a.x; lo[1] = a.y; lo[2] = a.z; lo[3] = a.w;
        hi[0] = b.x; hi[1] = b.y; hi[2] = b.z; hi[3] = b.w;
    } else {
#pragma unroll
        for (int i = 0; i < 4; ++i) lo[i] = hi[i] = 0u;
    }
}

// the same 16 columns of an INT8 factor row (16 bytes): exact conversion to the fp16 fragment registers
__device__ __forceinline__ void ec_load16_i8(const int8_t* row, int col, uint32_t (&lo)[4], uint32_t (&hi)[4]) {
    if (row) {
        const uint4 a = __ldg(reinterpret_cast<const uint4*>(row + col));
        cvt_i8x4_f16x2(a.x, lo[0], lo[1]);
        cvt_i8x4_f16x2(a.y, lo[2], lo[3]);
        cvt_i8x4_f16x2(a.z, hi[0], hi[1]);
        cvt_i8x4_f16x2(a.w, hi[2], hi[3]);
    } else {
#pragma unroll
        for (int i = 0; i < 4; ++i) lo[i] = hi[i] = 0u;
    }
}

__device__ __forceinline__ uint32_t hmul2_u32(uint32_t a, uint32_t b) {
    uint32_t d;
    asm("mul.rn.f16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
    return d;
}

// ---- thread-block clusters: rank, peer shared-memory addresses, split barrier ----
__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t mapa_shared(uint32_t local_addr, uint32_t rank) {      // same offset in CTA `rank` of the cluster
    uint32_t ra;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(local_addr), "r"(rank));
    return ra;
}
__device__ __forceinline__ void st_shared_cluster_f32(uint32_t addr, float v) {
    asm volatile("st.shared::cluster.f32 [%0], %1;" :: "r"(addr), "f"(v) : "memory");
}
__device__ __forceinline__ void cluster_arrive_release() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait_acquire() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

// ---- legacy tensor-core MMA (decode path): D(16x8,f32) += A(16x16,f16,row) * B(16x8,f16,col) ----
__device__ __forceinline__ void mma_m16n8k16(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2,
                                             uint32_t a3, uint32_t b0, uint32_t b1) {
    asm volatile(
        "mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, "
        "{%0,%1,%2,%3};"
        : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
        : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

// ---- named barrier among a subset of warps ---------------------------------------------------
__device__ __forceinline__ void named_bar_sync(uint32_t id, uint32_t nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
#endif  // __CUDACC__

}  // namespace spear

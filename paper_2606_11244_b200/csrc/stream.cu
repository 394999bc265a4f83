// stream.cu -- the weight-streaming kernel for small token counts (decode, M <= 16).
//
// Computes steps S1-S3, S7, S8 of SURVEY.md 8(a) -- and, in the fused variant, S4-S6 -- in one launch
// (Eq. 3):
//     y[m][n] = sum_k x[m][k] * (q[n][k] - 8) * s[n][k/group]  +  sum_j u[m][j] * B[n][j]
// where u = alpha * gamma (.) (A x) comes from the EC pre-kernel (ec_pre.cu, split variant) or from warp 9
// of this kernel (fused variant); r == 0 is the plain W4 layer.  The paper's decode kernel
// runs the EC chain in a MARLIN epilogue on Hopper; here the layer is HBM-bound, so the design is a
// TMA-fed shared-memory ring:
//
//   * work unit = (panel of 128 output rows, PAIR of 128-column chunks) = 16 KiB of packed int4,
//     contiguous in the SPW4 layout (the last unit of a panel is a single chunk when K/128 is odd);
//     units are numbered panel-major and split evenly (stream-K) over gridDim.x CTAs, so every SM streams
//     the same number of bytes whatever the shape.  Large units keep the number of asynchronous-copy
//     instructions per byte low: one thread issues them, and ~200 cycles each is what bounds a ring of
//     small copies;
//   * warp 0, one lane: cp.async.bulk of weights and scales into a ring (depth = launch parameter) guarded by
//     full/empty mbarriers.  The first ring-full is issued BEFORE griddepcontrol.wait (weights do not depend on
//     the previous kernel): under programmatic dependent launch the ring of layer i+1 fills while layer i
//     drains.  After the wait the same lane adds one 3-D TMA tensor copy per unit for the x tile (8*MT tokens x
//     4 k-tiles x 64 columns, 128-byte swizzle, zero-filled beyond M and K);
//   * warp 9 (r > 0): fused variant: reduces this CTA's share of z = x [A; w_g]^T and arrives; in the CTAs that
//     finalise a panel it then stages u = alpha gamma (.) z in shared memory (split variant: copies the pre-kernel's u);
//   * 8 consumer warps, all on the same unit: warp (h, kq) takes strips 4h..4h+3 (64 rows) x k-tile kq
//     (64 columns): 4 LDS.128 of int4, lop3/sub dequantisation in registers, mma.sync.m16n8k16 with the
//     tokens as the n=8 operand (fp32 accumulate), group scale applied to the fp32 accumulator;
//   * per panel segment the 8 warps reduce through shared memory; a CTA that owns a whole panel writes y
//     directly, otherwise the parts meet through fp32 slots in the workspace and a counter per panel.  Plain layer: the
//     last arriver sums them in CTA order (nobody waits).  With an EC: the CTA that owns the panel's FIRST unit
//     finalises -- the ring brings the panel's B slab (128 x r, <= 2 items of 16 KiB) to it right behind that
//     segment's weights, and the same 8 warps add B u^T as r / 16 extra mma.sync k-steps (u split into an fp16 head
//     and remainder) before the single cast: S7 costs one ring item per panel instead of a scalar epilogue.
#include <mutex>

#include "common.cuh"
#include "kernels.h"

namespace spear {

template <int MT>
struct StreamCfg {
    // ring depth is a launch parameter: shallow (two CTAs per SM, the next layer's CTA prefetches beside this
    // one under programmatic dependent launch) for small layers, deep (one CTA per SM, ~150 KiB in flight per
    // SM to cover the HBM latency) for large ones
    static constexpr int kStagesShallow = (MT == 1) ? 4 : 3;
    static constexpr int kStagesDeep = (MT == 1) ? 10 : 7;
    static constexpr int kMaxStages = 10;
    static constexpr int kXTile = MT * 8 * 512;       // bytes: 8*MT token rows x 4 k-tiles x 128 B
    static constexpr int kWUnit = 16384;              // two chunks of packed int4
    static constexpr int kScUnit = 512;               // one 256-byte scale slot per chunk
    static constexpr int kRedStride = 68;             // floats; 68 makes the fragment stores conflict-free
    static constexpr int kTok = 8 * MT;
    static constexpr size_t x_bytes(int S) { return size_t(S) * kXTile; }
    static constexpr size_t w_bytes(int S) { return size_t(S) * kWUnit; }
    static constexpr size_t sc_bytes(int S) { return size_t(S) * kScUnit; }
    static constexpr size_t kRedBytes = size_t(8) * kTok * kRedStride * 4;
    static constexpr size_t kBarBytes = size_t(kMaxStages) * 16 + 32;
    static constexpr size_t smem_bytes(int S) { return 1024 + x_bytes(S) + w_bytes(S) + sc_bytes(S) + kRedBytes + kBarBytes; }
    static_assert(smem_bytes(kStagesDeep) <= 232448, "deep ring exceeds the 227 KiB opt-in shared memory");
    static_assert(2 * (smem_bytes(kStagesShallow) + 1024) <= 233472, "two shallow CTAs must fit one SM");
};

__device__ __forceinline__ int cta_of_unit(int u, int per, int rem) {
    const int big = rem * (per + 1);
    return (u < big) ? u / (per + 1) : rem + (u - big) / per;
}

// Device-wide arrive: one acq_rel RMW at gpu scope.  Executed after a warp / named barrier it releases the
// writes of every thread that synchronised with the caller (cumulativity) and acquires what earlier arrivers
// released -- no separate __threadfence round trips on the critical path.
__device__ __forceinline__ unsigned arrive_acq_rel(unsigned* ctr) {
    unsigned old;
    asm volatile("atom.add.acq_rel.gpu.global.u32 %0, [%1], 1;" : "=r"(old) : "l"(ctr) : "memory");
    return old;
}
// ... and the same arrive when nobody needs the count it returns: fire and forget, the issuing thread does not wait
__device__ __forceinline__ void arrive_release(unsigned* ctr) {
    asm volatile("red.release.gpu.global.add.u32 [%0], 1;" :: "l"(ctr) : "memory");
}

// ---- the consumer inner loop -------------------------------------------------------------------------
// Explicit shared-window loads (32-bit addresses; the generic-pointer form compiles to LD.E + 64-bit math).
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint32_t lds32(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}
// The four fp16 pairs of one SPW4 word WITHOUT removing the bias: pairs 0 and 2 hold 1024 + q, pairs 1
// and 3 hold 1024 + 16 q (lop3 only: 5 instructions per 8 weights instead of 9).  The mma that consumes
// pairs 1 and 3 is fed x / 16 (exact), and the bias -- (1024 + 8) x on the even pairs, (64 + 8) x on the
// odd ones, the same for every output row -- enters as the accumulator's initial value (see stream_task).
__device__ __forceinline__ void biased_word(uint32_t w, uint32_t (&out)[4]) {
    constexpr uint32_t kMagic = 0x64006400u;
    asm("lop3.b32 %0, %1, 0x000f000f, %2, 0xea;" : "=r"(out[0]) : "r"(w), "r"(kMagic));
    asm("lop3.b32 %0, %1, 0x00f000f0, %2, 0xea;" : "=r"(out[1]) : "r"(w), "r"(kMagic));
    const uint32_t w8 = w >> 8;
    asm("lop3.b32 %0, %1, 0x000f000f, %2, 0xea;" : "=r"(out[2]) : "r"(w8), "r"(kMagic));
    asm("lop3.b32 %0, %1, 0x00f000f0, %2, 0xea;" : "=r"(out[3]) : "r"(w8), "r"(kMagic));
}

__device__ __forceinline__ uint32_t lds16(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u16 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint32_t pack_half2(float lo, float hi) {
    const __half2 h = __floats2half2_rn(lo, hi);
    return *reinterpret_cast<const uint32_t*>(&h);
}

// S7 on the tensor cores (the B (gamma (.) A x) term of Eq. 3): one 16-row strip of the panel's B slab
// (fp16 [row][r], or int8 [row][r]; b_addr = the strip's first row in the ring slot) times u^T, into acc.
//   A operand = the strip (rows g / g + 8, k = 16 ks + 2t.. and + 8), B operand = u[token][k] split into an fp16 head
//   and an fp16 remainder (two mma per k-step: u keeps ~22 bits, the products are exact, fp32 accumulate).
// r % 16 == 8: the upper half of the last k-step is absent and fed as zeros on both operands.
template <int MT>
__device__ __forceinline__ void ec_up(uint32_t b_addr, int r, bool int8, const float* us, int lane, float (&acc)[MT][4]) {
    const int g = lane >> 2, t = lane & 3;
    for (int k0 = 2 * t; k0 < r; k0 += 16) {
        const bool up = k0 + 8 < r;
        uint32_t a0, a1, a2, a3;
        if (!int8) {
            a0 = lds32(b_addr + (g * r + k0) * 2);
            a1 = lds32(b_addr + ((g + 8) * r + k0) * 2);
            a2 = up ? lds32(b_addr + (g * r + k0 + 8) * 2) : 0u;
            a3 = up ? lds32(b_addr + ((g + 8) * r + k0 + 8) * 2) : 0u;
        } else {
            const uint32_t w0 = lds16(b_addr + g * r + k0) | (up ? lds16(b_addr + g * r + k0 + 8) << 16 : 0u);
            const uint32_t w1 = lds16(b_addr + (g + 8) * r + k0) | (up ? lds16(b_addr + (g + 8) * r + k0 + 8) << 16 : 0u);
            cvt_i8x4_f16x2(w0, a0, a2);
            cvt_i8x4_f16x2(w1, a1, a3);
        }
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) {
            const float* up_ = us + (mt * 8 + g) * r + k0;
            const float2 u0 = *reinterpret_cast<const float2*>(up_);
            const float2 u1 = up ? *reinterpret_cast<const float2*>(up_ + 8) : make_float2(0.f, 0.f);
            const __half2 h0 = __floats2half2_rn(u0.x, u0.y), h1 = __floats2half2_rn(u1.x, u1.y);
            const float2 f0 = __half22float2(h0), f1 = __half22float2(h1);
            const uint32_t hi0 = *reinterpret_cast<const uint32_t*>(&h0), hi1 = *reinterpret_cast<const uint32_t*>(&h1);
            const uint32_t lo0 = pack_half2(u0.x - f0.x, u0.y - f0.y), lo1 = pack_half2(u1.x - f1.x, u1.y - f1.y);
            mma_m16n8k16(acc[mt], a0, a1, a2, a3, hi0, hi1);
            mma_m16n8k16(acc[mt], a0, a1, a2, a3, lo0, lo1);
        }
    }
}

// One (4 strips = 64 rows) x (64 columns) task of a warp.  w_addr: this lane's first 16 bytes of the
// chunk's k-tile (strip 4h), strips are 512 bytes apart; sc_addr: this lane's scale word of strip 4h,
// strips 32 bytes apart; x_addr: the unit's x tile [token row][k-tile kq 0..3][64 columns], written by TMA
// with the 128-byte swizzle (16-byte chunk index XOR bits 7..9 of the address = kq | (row & 1) << 2).
//   sum_k (q - 8) x  =  sum_even (1024 + q) x + sum_odd (1024 + 16 q)(x / 16) - [1032 sum_even x + 72 sum_odd x]
// The bracket is produced by four mma with the constant fragment (-1032 | -1152 = -72 * 16) and used as the
// initial accumulator of every strip; all products are exact in fp32, the sums are fp32 tensor-core adds.
template <int MT>
__device__ __forceinline__ void stream_task(uint32_t w_addr, uint32_t x_addr, uint32_t sc_addr, int kq, int lane,
                                            float (&tot)[4][MT][4]) {
    const int g = lane >> 2, t = lane & 3;
    const int xr = kq | ((g & 1) << 2);
    uint32_t xa[MT][4], xb[MT][4];
    float negc[MT][4];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) {
        const uint32_t row = x_addr + (mt * 8 + g) * 512 + kq * 128;
        const uint4 va = lds128(row + (((2 * t) ^ xr) << 4));
        const uint4 vb = lds128(row + (((2 * t + 1) ^ xr) << 4));
        constexpr uint32_t kSixteenth = 0x2c002c00u;
        xa[mt][0] = va.x; xa[mt][1] = hmul2_u32(va.y, kSixteenth); xa[mt][2] = va.z; xa[mt][3] = hmul2_u32(va.w, kSixteenth);
        xb[mt][0] = vb.x; xb[mt][1] = hmul2_u32(vb.y, kSixteenth); xb[mt][2] = vb.z; xb[mt][3] = hmul2_u32(vb.w, kSixteenth);
        constexpr uint32_t kNeg1032 = 0xe408e408u, kNeg1152 = 0xe480e480u;
        // short dependency chains: a dependent mma.sync costs far more than an independent one here
        float n0[4] = {0.f, 0.f, 0.f, 0.f}, n1[4] = {0.f, 0.f, 0.f, 0.f};
        mma_m16n8k16(n0, kNeg1032, kNeg1032, kNeg1032, kNeg1032, xa[mt][0], xb[mt][0]);
        mma_m16n8k16(n1, kNeg1152, kNeg1152, kNeg1152, kNeg1152, xa[mt][1], xb[mt][1]);
        mma_m16n8k16(n0, kNeg1032, kNeg1032, kNeg1032, kNeg1032, xa[mt][2], xb[mt][2]);
        mma_m16n8k16(n1, kNeg1152, kNeg1152, kNeg1152, kNeg1152, xa[mt][3], xb[mt][3]);
#pragma unroll
        for (int i = 0; i < 4; ++i) negc[mt][i] = n0[i] + n1[i];
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const uint4 w = lds128(w_addr + j * 512);
        const uint32_t scw = lds32(sc_addr + j * 32);
        const float s_lo = __half2float(__ushort_as_half(uint16_t(scw & 0xffff)));
        const float s_hi = __half2float(__ushort_as_half(uint16_t(scw >> 16)));
        uint32_t a0[4], a1[4], a2[4], a3[4];
        biased_word(w.x, a0);   // row g,   columns 16t + 0..7
        biased_word(w.z, a1);   // row g+8, columns 16t + 0..7
        biased_word(w.y, a2);   // row g,   columns 16t + 8..15
        biased_word(w.w, a3);   // row g+8, columns 16t + 8..15
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) {
            float acc[4] = {negc[mt][0], negc[mt][1], negc[mt][2], negc[mt][3]};
            float acd[4] = {0.f, 0.f, 0.f, 0.f};
            mma_m16n8k16(acc, a0[0], a1[0], a2[0], a3[0], xa[mt][0], xb[mt][0]);
            mma_m16n8k16(acd, a0[1], a1[1], a2[1], a3[1], xa[mt][1], xb[mt][1]);
            mma_m16n8k16(acc, a0[2], a1[2], a2[2], a3[2], xa[mt][2], xb[mt][2]);
            mma_m16n8k16(acd, a0[3], a1[3], a2[3], a3[3], xa[mt][3], xb[mt][3]);
#pragma unroll
            for (int i = 0; i < 4; ++i) acc[i] += acd[i];
            tot[j][mt][0] = fmaf(s_lo, acc[0], tot[j][mt][0]);
            tot[j][mt][1] = fmaf(s_lo, acc[1], tot[j][mt][1]);
            tot[j][mt][2] = fmaf(s_hi, acc[2], tot[j][mt][2]);
            tot[j][mt][3] = fmaf(s_hi, acc[3], tot[j][mt][3]);
        }
    }
}

// ---- fused EC (warp 9): S4-S6 of SURVEY.md 8(a) inside the weight-stream kernel ---------------------
// Every CTA reduces one (16-row strip of [A; w_g]) x (K slice) piece of z = x [A; w_g]^T with mma.sync,
// adds it to the global fp32 z with red.add and ARRIVES on a device-wide counter (red.release, fire and forget).
// Only warp 9 of the CTAs that FINALISE a panel goes on: it waits until the counter shows every CTA of the grid,
// reads the complete z (z must be complete before the gate), applies the gate (PAPER.md:107-109 /
// BASELINE.json scalar gate) and stages u = alpha * gamma (.) z in shared memory -- all of it beside the consumers'
// main loop, which meets u on a shared-memory barrier when it reaches the panel's B slab (S7, see the kernel).
// z and the counter are double-buffered by the parity of an epoch word: launch n uses buffer n & 1, CTA 0
// re-zeroes the other buffer for launch n + 1 (its previous user, launch n - 1, is complete once
// griddepcontrol.wait returns) and bumps the epoch once everybody has arrived, so nothing has to be cleaned on
// the critical path.  All CTAs of the grid are co-resident (grid <= SMs x resident CTAs) and launches with an EC are
// COOPERATIVE launches (launch_stream): the driver starts the grid only when all of its CTAs fit at once, whatever
// else runs on the device, so the waits (this one, and a panel's head CTA for the panel's other parts) cannot deadlock.
// Before griddepcontrol.wait: pull this CTA's slice of [A; w_g] (the rows / K range of its phase-A tasks) into
// L2, so that the loads after the wait do not pay an HBM round trip on the critical path.
__device__ void ec_prefetch_factors(const StreamParams& p, int lane) {
    const bool scalar = (p.gate_kind == SPEAR_GATE_SCALAR_SIGMOID);
    const int rows_total = p.r + (scalar ? 1 : 0);
    const int strips = (rows_total + 15) >> 4;
    const int G = gridDim.x;
    const int ktiles = p.K >> 6;
    const int ksplit = max(1, min(ktiles, G / strips));
    const int n_tasks = strips * ksplit;
    for (int task = blockIdx.x; task < n_tasks; task += G) {
        const int strip = task % strips, ks = task / strips;
        const int kt_begin = int((long long)ks * ktiles / ksplit);
        const int kt_end = int((long long)(ks + 1) * ktiles / ksplit);
        const int lines = kt_end - kt_begin;           // 128-byte lines per row
        for (int i = lane; i < 16 * lines; i += 32) {
            const int rho = strip * 16 + i / lines, kt = kt_begin + i % lines;
            if (p.ec_int8 && rho < p.r) {
                if ((kt & 1) == 0) prefetch_l2(reinterpret_cast<const int8_t*>(p.A) + size_t(rho) * p.K + kt * 64);
                continue;
            }
            const __half* row = rho < p.r ? p.A + size_t(rho) * p.K : (rho == p.r && scalar ? p.w_g : nullptr);
            if (row) prefetch_l2(row + kt * 64);
        }
    }
}

// Phase A (whole warp, after griddepcontrol.wait): this CTA's piece of z, red.add, arrive.  Returns true in
// the last CTA to arrive.
__device__ unsigned ec_reduce_and_arrive(const StreamParams& p, int lane) {
    const int g = lane >> 2, t = lane & 3;
    const bool scalar = (p.gate_kind == SPEAR_GATE_SCALAR_SIGMOID);
    const int rows_total = p.r + (scalar ? 1 : 0);
    const int strips = (rows_total + 15) >> 4;
    const int G = gridDim.x;
    const int ktiles = p.K >> 6;
    const int ksplit = max(1, min(ktiles, G / strips));
    const int n_tasks = strips * ksplit;
    const __half* px0 = g < p.M ? p.x + size_t(g) * p.K : nullptr;
    const __half* px1 = g + 8 < p.M ? p.x + size_t(g + 8) * p.K : nullptr;
    // the epoch load is issued first and consumed after the first loads / mma (one L2 round trip, overlapped)
    unsigned epoch;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(epoch) : "l"(p.ec_sync) : "memory");
    bool announced = false;
    float* zpar = nullptr;
    for (int task = blockIdx.x; task < n_tasks; task += G) {
        const int strip = task % strips, ks = task / strips;
        const int rho0 = strip * 16 + g, rho1 = rho0 + 8;
        const bool q0 = p.ec_int8 && rho0 < p.r, q1 = p.ec_int8 && rho1 < p.r;      // INT8 factor rows; the gate row w_g stays fp16
        const int8_t* A8 = reinterpret_cast<const int8_t*>(p.A);
        const __half* pa0 = rho0 < p.r ? p.A + size_t(rho0) * p.K : (rho0 == p.r && scalar ? p.w_g : nullptr);
        const __half* pa1 = rho1 < p.r ? p.A + size_t(rho1) * p.K : (rho1 == p.r && scalar ? p.w_g : nullptr);
        // per-row scale of the INT8 factors, applied once to the K-reduced partial sum (1 for fp16 rows)
        const float sa0 = q0 ? __half2float(__ldg(p.A_scale + rho0)) : 1.f, sa1 = q1 ? __half2float(__ldg(p.A_scale + rho1)) : 1.f;
        const int kt_begin = int((long long)ks * ktiles / ksplit);
        const int kt_end = int((long long)(ks + 1) * ktiles / ksplit);
        float acc0[4] = {0.f, 0.f, 0.f, 0.f}, acc1[4] = {0.f, 0.f, 0.f, 0.f};
        for (int kt = kt_begin; kt < kt_end; ++kt) {
            const int col = kt * 64 + 16 * t;
            uint32_t a0l[4], a0h[4], a1l[4], a1h[4], x0l[4], x0h[4], x1l[4], x1h[4];
            if (q0) ec_load16_i8(A8 + size_t(rho0) * p.K, col, a0l, a0h);
            else ec_load16(pa0, col, true, a0l, a0h);     // EC factors are parameters: never written by a kernel
            if (q1) ec_load16_i8(A8 + size_t(rho1) * p.K, col, a1l, a1h);
            else ec_load16(pa1, col, true, a1l, a1h);
            ec_load16(px0, col, false, x0l, x0h);
            ec_load16(px1, col, false, x1l, x1h);
#pragma unroll
            for (int jj = 0; jj < 4; ++jj) {
                mma_m16n8k16(acc0, a0l[jj], a1l[jj], a0h[jj], a1h[jj], x0l[jj], x0h[jj]);
                mma_m16n8k16(acc1, a0l[jj], a1l[jj], a0h[jj], a1h[jj], x1l[jj], x1h[jj]);
            }
        }
        if (!announced) {
            zpar = p.zbuf + (epoch & 1u) * (16 * kZStride);
            announced = true;
        }
        // C fragment: rows rho0 / rho1 of [A; w_g], tokens 2t, 2t+1 (acc0) and 8+2t, 9+2t (acc1)
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int rho = (i & 2) ? rho1 : rho0;
            const int tok = 2 * t + (i & 1);
            if (rho < rows_total) {
                const float sa = (i & 2) ? sa1 : sa0;
                if (tok < p.M) atomicAdd(zpar + tok * kZStride + rho, sa * acc0[i]);
                if (tok + 8 < p.M) atomicAdd(zpar + (tok + 8) * kZStride + rho, sa * acc1[i]);
            }
        }
    }
    const unsigned par = epoch & 1u;
    __syncwarp();
    if (lane == 0) arrive_release(p.ec_sync + 1 + par);     // (CTA 0 bumps the epoch once it has seen everybody: ec_stage_u)
    if (blockIdx.x == 0) {
        // prepare the other buffer for the next fused launch on this workspace (after the arrive: everybody waits for it)
        float* zo = p.zbuf + (par ^ 1u) * (16 * kZStride);
        for (int i = lane; i < 16 * kZStride; i += 32) zo[i] = 0.f;
        if (lane == 0) p.ec_sync[1 + (par ^ 1u)] = 0;
    }
    return par;
}

// S5 + S6 (warp 9 of the CTAs that finalise a panel): u = alpha * gamma (.) z into shared memory, from the COMPLETE z
// (fused variant: after every CTA of the grid has arrived) or from the pre-kernel's u (split variant).
// Runs beside the consumers' main loop, so the device-wide wait and the z round trip stay off their critical path; they
// meet it on the u_ready barrier when they reach the panel's B items.
template <int KTOK>
__device__ void ec_stage_u(const StreamParams& p, int lane, unsigned par, float* us, uint64_t* u_ready) {
    const int n = KTOK * p.r;
    if (p.fused) {
        if (lane == 0) {
            const unsigned* ctr = p.ec_sync + 1 + par;
            unsigned f;
            do {       // all CTAs of the grid are co-resident (cooperative launch), and every one arrives within
                       // microseconds of its start: this wait cannot deadlock
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(f) : "l"(ctr) : "memory");
            } while (f < gridDim.x);
            if (blockIdx.x == 0) p.ec_sync[0] += 1u;       // everybody has arrived: the next fused launch takes the other buffer
        }
        __syncwarp();
        const bool scalar = (p.gate_kind == SPEAR_GATE_SCALAR_SIGMOID);
        const float* zc = p.zbuf + par * (16 * kZStride);
        const float bias = (scalar && p.b_g) ? __ldg(p.b_g) : 0.f;
        const float rinv = 1.f / float(p.r);
        for (int i0 = lane; i0 < n; i0 += 8 * 32) {
            float zz[8], zg[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) {       // eight independent L2 round trips in flight per lane
                const int idx = i0 + 32 * q;
                const int m = int((float(idx) + 0.5f) * rinv), j = idx - m * p.r;
                const bool on = idx < n && m < p.M;
                zz[q] = on ? __ldcg(zc + m * kZStride + j) : 0.f;
                zg[q] = (on && scalar) ? __ldcg(zc + m * kZStride + p.r) : 0.f;
            }
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const int idx = i0 + 32 * q;
                if (idx >= n) break;
                const int m = int((float(idx) + 0.5f) * rinv), j = idx - m * p.r;
                const float gam = scalar ? 1.f / (1.f + expf(-(zg[q] + bias))) : 1.f;
                us[idx] = m < p.M ? p.alpha * gam * zz[q] : 0.f;
                if (scalar && p.gate_out && blockIdx.x == 0 && j == 0 && m < p.M) p.gate_out[m] = gam;
            }
        }
    } else {
        for (int idx = lane; idx < n; idx += 32) us[idx] = idx < p.M * p.r ? __ldcg(p.u + idx) : 0.f;
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(u_ready);
}

// MINB = resident CTAs per SM the register allocation must allow: 2 for the shallow ring (96 registers), 1 for the
// deep ring, where the consumer loop gets the registers to keep its four strips in flight without spilling.
template <int MT, int MINB>
__global__ void __launch_bounds__(320, MINB)
stream_kernel(const __grid_constant__ CUtensorMap xmap, const StreamParams p) {
    using Cfg = StreamCfg<MT>;
    const int S = p.stages;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* base = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* xring = base;
    uint8_t* wring = xring + Cfg::x_bytes(S);
    uint8_t* scring = wring + Cfg::w_bytes(S);
    float* red = reinterpret_cast<float*>(scring + Cfg::sc_bytes(S));
    uint64_t* full = reinterpret_cast<uint64_t*>(reinterpret_cast<uint8_t*>(red) + Cfg::kRedBytes);
    uint64_t* empty = full + Cfg::kMaxStages;
    int* flag = reinterpret_cast<int*>(empty + Cfg::kMaxStages);
    uint64_t* u_ready = reinterpret_cast<uint64_t*>(flag + 2);     // EC: warp 9 has staged u in us[]
    float* us = reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(full) + Cfg::kBarBytes);      // u = alpha gamma (.) z, [8 MT][r] fp32 (r > 0 only)

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int G = gridDim.x, b = blockIdx.x;
    const int per = p.U / G, rem = p.U % G;
    const int u0 = b * per + min(b, rem);
    const int n_units = per + (b < rem ? 1 : 0);
    const int C = p.C, CP = p.CP;     // chunks and chunk pairs (= units) per panel

    if (threadIdx.x == 0) {
        for (int s = 0; s < S; ++s) { mbar_init(&full[s], 2); mbar_init(&empty[s], 8); }
        mbar_init(u_ready, 1);
        fence_mbar_init();
        tma_prefetch_desc(&xmap);
    }
    __syncthreads();
    pdl_launch_dependents();

    if (warp == 0) {
        // ------------------------------ producer: weights, scales, x tiles ------------------------------
        // The first ring-full of weights is issued WITHOUT waiting for the previous kernel (weights never depend
        // on it): under programmatic dependent launch the ring of layer i+1 fills while layer i drains.  x tiles
        // (which may be the previous kernel's output) follow griddepcontrol.wait.
        if (lane == 0) {
            const uint64_t pol_w = policy_evict_first(), pol_s = policy_evict_last();
            const uint8_t* wq = reinterpret_cast<const uint8_t*>(p.wq);
            const uint8_t* sc = reinterpret_cast<const uint8_t*>(p.scales);
            // ring items of this CTA: its units in order; a segment (the CTA's units of one panel) that starts its panel is followed by the
            // panel's B slab (p.b_slots items of p.b_slot_bytes), consumed by the same warps as r / 16 extra k-steps
            const uint8_t* Bb = reinterpret_cast<const uint8_t*>(p.B);
            const int nb = p.r > 0 ? p.b_slots : 0;
            // (B follows the segment that STARTS the panel: its CTA is the one that finalises the panel, see below)
            int pnl = u0 / CP, pr = u0 - pnl * CP, bs = 0, s = 0;       // bs: 0 = weight unit, 1..nb = B item
            int done = 0;                                               // units issued
            bool head = (pr == 0);                                      // the current segment starts its panel
            const int n_items = n_units + nb * ((u0 + n_units - 1) / CP - u0 / CP + (pr == 0 ? 1 : 0));
            auto issue_w = [&]() {
                if (bs > 0) {
                    mbar_arrive_expect_tx(&full[s], p.b_slot_bytes);
                    bulk_g2s(wring + s * Cfg::kWUnit, Bb + (size_t(pnl) * nb + (bs - 1)) * p.b_slot_bytes, p.b_slot_bytes, &full[s], pol_w);
                    return;
                }
                const int c0 = 2 * pr, nch = (c0 + 1 < C) ? 2 : 1;
                mbar_arrive_expect_tx(&full[s], nch * (8192 + 256));
                bulk_g2s(wring + s * Cfg::kWUnit, wq + (size_t(pnl) * C + c0) * 8192, nch * 8192, &full[s], pol_w);
                const uint8_t* sp = sc + size_t(pnl) * p.G * 256;
                if (p.group_chunks == 1) {
                    bulk_g2s(scring + s * Cfg::kScUnit, sp + size_t(c0) * 256, nch * 256, &full[s], pol_s);
                } else {
                    bulk_g2s(scring + s * Cfg::kScUnit, sp + size_t(c0 / p.group_chunks) * 256, 256, &full[s], pol_s);
                    if (nch == 2)
                        bulk_g2s(scring + s * Cfg::kScUnit + 256, sp + size_t((c0 + 1) / p.group_chunks) * 256, 256,
                                 &full[s], pol_s);
                }
            };
            auto issue_x = [&]() {
                if (bs > 0) { mbar_arrive(&full[s]); return; }      // a B item has no x tile
                mbar_arrive_expect_tx(&full[s], Cfg::kXTile);
                tma_load_3d(xring + s * Cfg::kXTile, &xmap, 0, pr * 4, 0, &full[s], pol_s);
            };
            auto advance = [&]() {
                if (++s == S) s = 0;
                if (bs == 0) {
                    ++done;
                    const bool seg_end = (pr == CP - 1) || (done == n_units);
                    if (nb > 0 && seg_end && head) { bs = 1; return; }
                    if (seg_end) head = true;        // every later segment starts at a panel boundary
                } else if (bs < nb) {
                    ++bs;
                    return;
                }
                bs = 0;
                if (++pr == CP) { pr = 0; ++pnl; }
            };
            const int nfirst = min(n_items, S);
            for (int it = 0; it < nfirst; ++it) { issue_w(); advance(); }
            pdl_wait();   // x may be written by the previous kernel in the stream
            pnl = u0 / CP; pr = u0 - pnl * CP; bs = 0; s = 0; done = 0; head = (pr == 0);
            for (int it = 0; it < nfirst; ++it) { issue_x(); advance(); }
            uint32_t eph = 0;     // parity of the first completion of empty[]
            for (int it = nfirst; it < n_items; ++it) {
                mbar_wait(&empty[s], eph);
                issue_w();
                issue_x();
                advance();
                if (s == 0) eph ^= 1;
            }
        }
        return;
    }
    if (warp == 9) {
        // ------------------------------ EC warp (fused variant only) ------------------------------
        if (p.r == 0) return;
        // this CTA finalises the panels whose first unit it owns (every segment but a first one that starts mid-panel)
        const bool finalises = (u0 + n_units - 1) / CP - u0 / CP + (u0 % CP == 0 ? 1 : 0) > 0;
        unsigned par = 0;
        if (p.fused) ec_prefetch_factors(p, lane);   // EC factors are parameters: warm L2 before the wait
        pdl_wait();
        if (p.fused) par = ec_reduce_and_arrive(p, lane);
        if (finalises) ec_stage_u<Cfg::kTok>(p, lane, par, us, u_ready);
        return;
    }

    // -------------------------------- consumers --------------------------------
    const int cw = warp - 1;
    const int h = cw & 1, kq = cw >> 1;        // strips 4h..4h+3, k-tile kq of the unit's (up to) four
    const int g = lane >> 2, t = lane & 3;
    const int ct = threadIdx.x - 32;            // 0..255
    pdl_wait();                                 // orders our workspace / y writes after the previous kernel

    float tot[4][MT][4];
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int mt = 0; mt < MT; ++mt)
#pragma unroll
            for (int i = 0; i < 4; ++i) tot[j][mt][i] = 0.f;

    // ring slot / phase and the unit's position inside its panel advance incrementally (no divisions here)
    int rs = 0, pr = u0 % CP;
    uint32_t rph = 0;
    const uint32_t w_lane = smem_u32(wring) + (kq >> 1) * 8192 + (((kq & 1) * 8 + 4 * h) * 32 + lane) * 16;
    const uint32_t sc_lane = smem_u32(scring) + (kq >> 1) * 256 + (4 * h * 16 + 2 * g) * 2;
    const uint32_t x_base = smem_u32(xring);
    bool u_seen = false;
    int it = 0;
    constexpr int kMaxMine = 128;      // panels one CTA may finalise with the fused tail on (grid >= N / 128 / kMaxMine, checked on the host)
    __shared__ float tail_s[16];
    __shared__ int mine[kMaxMine];
    int n_mine = 0;
    while (it < n_units) {
        const int pnl = (u0 + it) / CP;
        const int seg_begin = it;
        const int seg_end = min(n_units, (pnl + 1) * CP - u0);
        for (int i = seg_begin; i < seg_end; ++i) {
            mbar_wait(&full[rs], rph);
            if (2 * pr + (kq >> 1) < C)   // the second chunk is absent in a panel's odd tail unit
                stream_task<MT>(w_lane + rs * Cfg::kWUnit, x_base + rs * Cfg::kXTile, sc_lane + rs * Cfg::kScUnit,
                                kq, lane, tot);
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[rs]);
            if (++rs == S) { rs = 0; rph ^= 1; }
            if (++pr == CP) pr = 0;
        }
        // ---- CTA-level reduction of the segment: red[warp][token][row within the half panel] ----
        float* myred = red + size_t(cw) * Cfg::kTok * Cfg::kRedStride;
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
                const int row = j * 16 + g, tok = mt * 8 + 2 * t;
                myred[tok * Cfg::kRedStride + row] = tot[j][mt][0];
                myred[(tok + 1) * Cfg::kRedStride + row] = tot[j][mt][1];
                myred[tok * Cfg::kRedStride + row + 8] = tot[j][mt][2];
                myred[(tok + 1) * Cfg::kRedStride + row + 8] = tot[j][mt][3];
                tot[j][mt][0] = tot[j][mt][1] = tot[j][mt][2] = tot[j][mt][3] = 0.f;
            }
        named_bar_sync(1, 256);
        const int row = ct & 127, hh = row >> 6, rl = row & 63;
        float val[4 * MT];
#pragma unroll
        for (int i = 0; i < 4 * MT; ++i) {
            const int tok = (ct >> 7) + 2 * i;
            float v = 0.f;
#pragma unroll
            for (int q = 0; q < 4; ++q)
                v += red[size_t(hh + 2 * q) * Cfg::kTok * Cfg::kRedStride + tok * Cfg::kRedStride + rl];
            val[i] = v;
        }
        const bool whole = ((u0 + seg_begin) % CP == 0) && (seg_end - seg_begin == CP);
        // Who finalises a split panel.  Plain layer (r == 0): the last CTA to arrive (nobody ever waits).  With an EC: the
        // CTA that owns the panel's first unit -- the ring brought the panel's B slab to ITS shared memory -- which waits
        // for the other parts; those were started earlier (a CTA's mid-panel segment is its first) and the launch is
        // cooperative, so the wait is short and cannot deadlock.
        const bool head = (u0 + seg_begin) % CP == 0;
        const bool waits = p.r > 0 && head;
        bool finalize = whole;
        int c_first = b, c_last = b;
        if (!whole) {
            const int which = ((u0 / CP) == pnl) ? 0 : 1;
            float* slot = p.partial + size_t(b * 2 + which) * Cfg::kTok * 128;
            if (!waits) {
#pragma unroll
                for (int i = 0; i < 4 * MT; ++i) slot[((ct >> 7) + 2 * i) * 128 + row] = val[i];
            }
            named_bar_sync(2, 256);
            c_first = cta_of_unit(pnl * CP, per, rem);
            c_last = cta_of_unit(pnl * CP + CP - 1, per, rem);
            if (ct == 0) {
                if (waits) {
                    unsigned f;
                    do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(f) : "l"(p.counters + pnl) : "memory"); } while (f < unsigned(c_last - c_first));
                    p.counters[pnl] = 0;            // self-cleaning: the next call finds zero
                    *flag = 1;
                } else {
                    int last = 0;
                    if (p.r > 0) {
                        arrive_release(p.counters + pnl);        // the panel's head CTA is waiting for this
                    } else {
                        const unsigned old = arrive_acq_rel(p.counters + pnl);   // releases the CTA's partial, acquires the others'
                        last = (old == unsigned(c_last - c_first));
                        if (last) p.counters[pnl] = 0;
                    }
                    *flag = last;
                }
            }
            named_bar_sync(2, 256);
            finalize = (*flag != 0);
            if (finalize) {
                if (!waits) {
#pragma unroll
                    for (int i = 0; i < 4 * MT; ++i) val[i] = 0.f;
                }
                // partials are summed in CTA order (a waiting head CTA keeps its own part in registers and adds the others);
                // four CTAs' loads are issued before the first add so that their L2 round trips overlap
                for (int cj = waits ? c_first + 1 : c_first; cj <= c_last; cj += 4) {
                    float tmp[4][4 * MT];
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const int cq = min(cj + q, c_last);
                        const int uj = cq * per + min(cq, rem);
                        const int wj = ((uj / CP) == pnl) ? 0 : 1;
                        const float* sj = p.partial + size_t(cq * 2 + wj) * Cfg::kTok * 128;
#pragma unroll
                        for (int i = 0; i < 4 * MT; ++i) tmp[q][i] = __ldcg(sj + ((ct >> 7) + 2 * i) * 128 + row);
                    }
#pragma unroll
                    for (int q = 0; q < 4; ++q)
                        if (cj + q <= c_last) {
#pragma unroll
                            for (int i = 0; i < 4 * MT; ++i) val[i] += tmp[q][i];
                        }
                }
            }
        }
        if (waits) {
            // ---- S7: the next ring item(s) hold this panel's B slab; every warp multiplies its 16-row strip by u^T on
            // the tensor cores (u staged by warp 9, met here on u_ready) and the strips go through red[] once more to
            // reach the row-per-thread layout of val[].
            if (!u_seen) { mbar_wait(u_ready, 0); u_seen = true; }
            const int nb = p.b_slots;
            const int esz = p.ec_int8 ? 1 : 2;
            const int row0 = 64 * h + 16 * kq;                   // this warp's strip of the panel
            float sb0 = 1.f, sb1 = 1.f;
            if (p.ec_int8) {                                     // INT8 factors: per-row scale of B
                sb0 = __half2float(__ldg(p.B_scale + pnl * 128 + row0 + g));
                sb1 = __half2float(__ldg(p.B_scale + pnl * 128 + row0 + g + 8));
            }
            float acc[MT][4];
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) acc[mt][0] = acc[mt][1] = acc[mt][2] = acc[mt][3] = 0.f;
            for (int k = 0; k < nb; ++k) {
                mbar_wait(&full[rs], rph);
                if (nb == 1 || h == k)
                    ec_up<MT>(smem_u32(wring) + rs * Cfg::kWUnit + (nb == 1 ? row0 : 16 * kq) * p.r * esz, p.r, p.ec_int8 != 0, us, lane, acc);
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[rs]);
                if (++rs == S) { rs = 0; rph ^= 1; }
            }
            constexpr int kEcStride = 132;                       // [token][row]: conflict-free fragment stores
            named_bar_sync(2, 256);                              // every thread has taken its sums out of red[]
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
                const int tok = mt * 8 + 2 * t;
                red[tok * kEcStride + row0 + g] = sb0 * acc[mt][0];
                red[(tok + 1) * kEcStride + row0 + g] = sb0 * acc[mt][1];
                red[tok * kEcStride + row0 + g + 8] = sb1 * acc[mt][2];
                red[(tok + 1) * kEcStride + row0 + g + 8] = sb1 * acc[mt][3];
            }
            named_bar_sync(2, 256);
#pragma unroll
            for (int i = 0; i < 4 * MT; ++i) val[i] += red[((ct >> 7) + 2 * i) * kEcStride + row];
        }
        if (finalize) {
            const int n = pnl * 128 + row;
            if (p.resid) {
                // fused tail, first half: residual add on the fp32 sums, and this panel's share of the
                // per-token sum of squares that the next layer's RMSNorm needs (taken before the rounding)
                if (ct < 16) tail_s[ct] = 0.f;
                named_bar_sync(2, 256);
#pragma unroll
                for (int i = 0; i < 4 * MT; ++i) {
                    const int tok = (ct >> 7) + 2 * i;
                    float sq = 0.f;
                    if (tok < p.M) {
                        val[i] += __half2float(p.resid[size_t(tok) * p.N + n]);
                        sq = val[i] * val[i];
                    }
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) sq += __shfl_xor_sync(0xffffffffu, sq, o);
                    if (lane == 0 && tok < p.M) atomicAdd(&tail_s[tok], sq);
                }
                named_bar_sync(2, 256);
                if (ct < p.M) atomicAdd(p.tail_ssq + ct, tail_s[ct]);
                if (ct == 0 && n_mine < kMaxMine) mine[n_mine] = pnl;
                ++n_mine;       // (every thread counts; only ct == 0 writes the list)
            }
            // S8: one RN-even cast, coalesced store of 128 consecutive n per token
#pragma unroll
            for (int i = 0; i < 4 * MT; ++i) {
                const int tok = (ct >> 7) + 2 * i;
                if (tok < p.M) p.y[size_t(tok) * p.N + n] = __float2half_rn(val[i]);
            }
            if (p.resid) {
                named_bar_sync(2, 256);      // the panel's y stores and ssq adds are issued
                if (ct == 0) { __threadfence(); atomicAdd(p.tail_ctr, 1u); }
            }
        }
        named_bar_sync(1, 256);     // red[] and flag are reused by the next segment
        it = seg_end;
    }
    if (p.resid) {
        // fused tail, second half: once every panel of the layer has contributed (all CTAs are co-resident: cooperative
        // launch), normalise the panels this CTA finalised.  y is re-read as stored (fp16).
        if (n_mine > 0) {
            if (ct == 0) {
                unsigned f;
                do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(f) : "l"(p.tail_ctr) : "memory"); } while (f < unsigned(p.N >> 7));
            }
            named_bar_sync(2, 256);
            if (ct < 16) tail_s[ct] = ct < p.M ? rsqrtf(__ldcg(p.tail_ssq + ct) / float(p.N) + p.rms_eps) : 0.f;
            named_bar_sync(2, 256);
            const int row = ct & 127;
            for (int q = 0; q < min(n_mine, kMaxMine); ++q) {
                const int n = mine[q] * 128 + row;
                const float gw = __half2float(__ldg(p.rms_w + n));
#pragma unroll
                for (int i = 0; i < 4 * MT; ++i) {
                    const int tok = (ct >> 7) + 2 * i;
                    if (tok < p.M) {
                        const float yv = __half2float(__ldcg(p.y + size_t(tok) * p.N + n));
                        p.h_out[size_t(tok) * p.N + n] = __float2half_rn(yv * tail_s[tok] * gw);
                    }
                }
            }
        }
        named_bar_sync(2, 256);
        if (ct == 0) {      // the last CTA to leave resets the tail state for the next call
            __threadfence();
            if (atomicAdd(p.tail_ctr + 1, 1u) == gridDim.x - 1) {
                for (int m = 0; m < 16; ++m) p.tail_ssq[m] = 0.f;
                p.tail_ctr[0] = 0;
                p.tail_ctr[1] = 0;
            }
        }
    }
}

int stream_stages(int MT, bool deep) {
    if (MT == 1) return deep ? StreamCfg<1>::kStagesDeep : StreamCfg<1>::kStagesShallow;
    return deep ? StreamCfg<2>::kStagesDeep : StreamCfg<2>::kStagesShallow;
}
// u buffer behind the barriers: [8 MT][r] fp32
static int stream_u_bytes(int MT, int r) { return r > 0 ? ((8 * MT * r * 4 + 127) & ~127) : 0; }
int stream_smem_bytes(int MT, int stages, int r) {
    return int(MT == 1 ? StreamCfg<1>::smem_bytes(stages) : StreamCfg<2>::smem_bytes(stages)) + stream_u_bytes(MT, r);
}
int stream_fit_stages(int MT, bool deep, int r) {
    constexpr int kLimit = 232448 - 1024;      // opt-in shared memory per CTA minus the kernel's static shared variables
    int S = stream_stages(MT, deep);
    while (S > 2 && stream_smem_bytes(MT, S, r) > kLimit) --S;
    return S;
}

// Resident CTAs per SM of the instance a launch would take (occupancy query, cached per u-buffer size): the fused EC's
// device-wide arrive / wait needs the whole grid resident, so api.cu clamps the grid to num_sms x this.
int stream_resident_ctas(int MT, bool deep, int r) {
    static std::mutex mu;
    static int cache[2][2][130] = {};
    std::lock_guard<std::mutex> lock(mu);
    int& c = cache[MT - 1][deep ? 1 : 0][std::min(r, 129)];
    if (c == 0) {
        const int smem = stream_smem_bytes(MT, stream_fit_stages(MT, deep, r), r);
        const void* fn = MT == 1 ? (deep ? (const void*)stream_kernel<1, 1> : (const void*)stream_kernel<1, 2>)
                                 : (deep ? (const void*)stream_kernel<2, 1> : (const void*)stream_kernel<2, 2>);
        int n = 0;
        if (cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, 232448 - 1024) != cudaSuccess ||
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, fn, 320, smem) != cudaSuccess || n < 1)
            n = 1;
        c = n;
    }
    return c;
}

int launch_stream(const CUtensorMap& xmap, const StreamParams& p, int MT, int grid, bool pdl,
                  cudaStream_t st) {
    static std::once_flag attr_once;
    static cudaError_t attr_err = cudaSuccess;
    std::call_once(attr_once, [&]() {
        auto set = [&](const void* fn, size_t bytes) {
            if (attr_err == cudaSuccess) attr_err = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, int(bytes));
        };
        // every instance may take up to the opt-in maximum (ring + u buffer; stream_fit_stages keeps it below)
        set((const void*)stream_kernel<1, 2>, 232448 - 1024);
        set((const void*)stream_kernel<2, 2>, 232448 - 1024);
        set((const void*)stream_kernel<1, 1>, 232448 - 1024);
        set((const void*)stream_kernel<2, 1>, 232448 - 1024);
    });
    SPEAR_CUDA_OK(attr_err);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(320);
    cfg.dynamicSmemBytes = stream_smem_bytes(MT, p.stages, p.r);
    cfg.stream = st;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (p.r > 0 || p.resid) {
        // the fused EC (and the fused tail's row-wide mean) wait device-wide for their own grid: a cooperative launch makes the co-residency of all CTAs a
        // guarantee of the driver instead of an assumption about dispatch order (other lanes, other tenants of the GPU)
        attr[1].id = cudaLaunchAttributeCooperative;
        attr[1].val.cooperative = 1;
        cfg.numAttrs = 2;
    }
    const bool deep = p.deep != 0;
    if (MT == 1 && !deep) SPEAR_CUDA_OK(cudaLaunchKernelEx(&cfg, stream_kernel<1, 2>, xmap, p));
    else if (MT == 1) SPEAR_CUDA_OK(cudaLaunchKernelEx(&cfg, stream_kernel<1, 1>, xmap, p));
    else if (!deep) SPEAR_CUDA_OK(cudaLaunchKernelEx(&cfg, stream_kernel<2, 2>, xmap, p));
    else SPEAR_CUDA_OK(cudaLaunchKernelEx(&cfg, stream_kernel<2, 1>, xmap, p));
    count_launch();
    return SPEAR_OK;
}

}  // namespace spear

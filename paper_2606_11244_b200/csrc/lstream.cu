// lstream.cu -- the persistent "layer stream" kernel for small token counts (decode, M <= 16).
//
// One cooperative launch (one CTA per SM, co-resident by construction) consumes a table of layer calls
// (LsParams) and computes, for every call, steps S1-S8 of SURVEY.md 8(a) (Eq. 3):
//     y[m][n] = sum_k x[m][k] (q[n][k] - 8) s[n][k/group]  +  alpha sum_j B[n][j] gamma[m] z[m][j],  z = x A^T
// The paper's decode kernel is a MARLIN mma.sync main loop with the EC chain in its epilogue,
// one launch per module; measured on B200 the legacy mma.sync path tops out near 4 clk per m16n8k16 per SM
// (~300 TFLOP/s), below what an 8 TB/s int4 stream needs at M = 8..16.  So here:
//
//   * work item = (call, 128-row panel, 128-column chunk) = 8 KiB of SPW4 codes + 256 B of scales; the calls of
//     a PHASE (calls that do not depend on each other) form one chunk sequence that is cut into gridDim.x equal
//     contiguous ranges, so every SM streams the same number of bytes and the cp.async.bulk ring never drains
//     between calls; a call whose x is an earlier call's y opens a new phase, whose x loads wait for the
//     previous phase's panel-completion counter while its WEIGHTS are prefetched across the boundary;
//   * warp 0 (one lane): cp.async.bulk of chunk + scales into a shared-memory ring (evict_first);
//   * warp 1: x tile of the chunk ([16 tokens][128 columns] fp16) by 8-byte cp.async into the K-major
//     SWIZZLE_128B operand layout, with the k-order permuted to match the weight fragments (below);
//   * warps 8-23 (16 dequantisation warps, 4 per TMEM lane quarter): LDS.128 -> exact q - 8 in fp16
//     (lop3 / sub / fma) -> tcgen05.st.16x256b.x4 into a ring of A-operand slots in TENSOR MEMORY.  The SPW4
//     word of lane (g, t) holds rows g, g+8 x columns 16t..16t+15, the 16x256b store shape spreads a row's
//     columns over the four lanes of a quad, so MMA j of a 64-column k-tile sees k = 16t + 4j + e at its
//     K position 4t + e; the x loader applies the same permutation (a dot product is order-invariant);
//   * warp 2 (one lane): tcgen05.mma.cta_group::1.kind::f16, M = 128 rows of the panel, N = 16 tokens, K = 16,
//     A from TMEM, B = x tile from shared memory, D = one of two 16-column fp32 accumulators in TMEM, one
//     accumulation run per scale group; tcgen05.commit frees the A slot / ring stage and hands D over;
//   * warps 4-7 (epilogue, thread = output row): tcgen05.ld the run, scale by s[n][group] into fp32 registers;
//     at the end of a panel segment: split-K through fp32 partial slots + an acq_rel counter when the panel
//     is shared with neighbouring CTAs, then the rank-r update y += u B^T, one RN-even cast, store;
//   * warp 3 (EC): this CTA's share of z = x [A; w_g]^T for every call of the phase (mma.sync, red.add),
//     arrive; the last arriver applies the gate (PAPER.md:109 scalar form of BASELINE.json / gamma = 1) and
//     publishes u = alpha gamma z behind a flag that finalising CTAs look at only in their epilogue
//     (z must be complete before the gate).
#include <cooperative_groups.h>

#include "common.cuh"
#include "kernels.h"

namespace spear {

namespace ls {
constexpr int kStages = 16;                 // ring depth (chunks): 16 x 12.25 KiB
constexpr int kASlots = 8;                  // TMEM A-operand slots (one 64-column k-tile = 32 TMEM columns each)
constexpr int kThreads = 768;
constexpr int kWBytes = 8192, kScBytes = 256, kXBytes = 4096;
constexpr uint32_t kTmemCols = 512;
constexpr uint32_t kDCol = kASlots * 32;    // two 16-column accumulators behind the A ring
constexpr uint32_t kIdesc = (1u << 4) | (uint32_t(16 >> 3) << 17) | (uint32_t(128 >> 4) << 24);
constexpr int kEmptyCount = 8 + 4 + 1;      // 8 dequant warps + 4 epilogue warps + the MMA commit per chunk
struct Smem {
    static constexpr size_t x = 0;
    static constexpr size_t w = x + size_t(kStages) * kXBytes;
    static constexpr size_t sc = w + size_t(kStages) * kWBytes;
    static constexpr size_t u = sc + size_t(kStages) * kScBytes;       // [16][128] fp32 staging of u
    static constexpr size_t bars = u + 16 * 128 * 4;
    static constexpr size_t total = bars + 1024;
};
static_assert(Smem::total + 1024 <= 232448, "layer-stream shared memory exceeds the 227 KiB opt-in limit");

__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem]^T : fp16 inputs, fp32 accumulate, A = 128 lanes x 8 columns, B K-major SW128
__device__ __forceinline__ void umma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}\n" ::"r"(d_tmem),
        "r"(a_tmem), "l"(b_desc), "r"(kIdesc), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ uint64_t desc_sw128(uint32_t smem_addr) {
    return uint64_t((smem_addr & 0x3ffff) >> 4) | (uint64_t(1) << 16) | (uint64_t(1024 >> 4) << 32) |
           (uint64_t(1) << 46) | (uint64_t(2) << 61);
}
__device__ __forceinline__ void cp_async8(uint32_t dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_arrive_noinc(uint64_t* bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ unsigned ld_acquire(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned atom_add_acq_rel(unsigned* p, unsigned v) {
    unsigned old;
    asm volatile("atom.add.acq_rel.gpu.global.u32 %0, [%1], %2;" : "=r"(old) : "l"(p), "r"(v) : "memory");
    return old;
}
__device__ __forceinline__ void red_add_release(unsigned* p, unsigned v) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void wait_counter(const unsigned* p, unsigned target) {
    while (ld_acquire(p) < target) __nanosleep(64);
}

// ---- the work sequence of this CTA --------------------------------------------------------------------------
struct Seg {
    int call, panel, k0, k1;   // chunks [k0, k1) of the panel
    int ph;                    // phase
    int pos;                   // position of chunk k0 in the phase's chunk sequence
};
__device__ __forceinline__ int range_lo(int b, int T, int G) { return int((long long)b * T / G); }
__device__ __forceinline__ int cta_of(int pos, int T, int G) {
    int b = int((long long)pos * G / T);
    while (b + 1 < G && range_lo(b + 1, T, G) <= pos) ++b;
    while (b > 0 && range_lo(b, T, G) > pos) --b;
    return b;
}
struct SegIter {
    int ph, pos, hi, call;
    __device__ SegIter() : ph(-1), pos(0), hi(0), call(0) {}
    // advances to the next segment of this CTA; false when the table is exhausted
    __device__ bool next(const LsParams& P, Seg& s) {
        const int G = gridDim.x, b = blockIdx.x;
        while (pos >= hi) {
            if (++ph >= P.n_phases) return false;
            const int T = P.phase_chunks[ph];
            pos = range_lo(b, T, G);
            hi = range_lo(b + 1, T, G);
            call = P.phase_first_call[ph];
        }
        while (pos >= P.calls[call].chunk_base + P.calls[call].P * P.calls[call].C) ++call;
        const LsCall& c = P.calls[call];
        const int rel = pos - c.chunk_base;
        s.call = call; s.ph = ph; s.pos = pos;
        s.panel = rel / c.C;
        s.k0 = rel - s.panel * c.C;
        const int end = min(hi, c.chunk_base + (s.panel + 1) * c.C);
        s.k1 = s.k0 + (end - pos);
        pos = end;
        return true;
    }
};
__device__ __forceinline__ int total_chunks(const LsParams& P) {
    int n = 0;
    for (int ph = 0; ph < P.n_phases; ++ph)
        n += range_lo(blockIdx.x + 1, P.phase_chunks[ph], gridDim.x) - range_lo(blockIdx.x, P.phase_chunks[ph], gridDim.x);
    return n;
}
}  // namespace ls

namespace ls {
struct Bars {
    uint64_t full[kStages], empty[kStages], a_full[kASlots], a_empty[kASlots], d_full[2], d_empty[2];
    uint32_t tmem;
    int flag;       // epilogue broadcast: this CTA finalises the panel
    int u_call;     // call whose u sits in the staging buffer (-1 = none)
};
static_assert(sizeof(Bars) <= 1024, "barrier block");

// ---- warp 0: weights + scales -------------------------------------------------------------------------------
__device__ void producer(const LsParams& P, uint8_t* wring, uint8_t* scring, Bars* B) {
    const uint64_t pol_w = policy_evict_first(), pol_s = policy_evict_last();
    SegIter it;
    Seg sg;
    int n = 0;
    while (it.next(P, sg)) {
        const LsCall& c = P.calls[sg.call];
        const uint8_t* wp = c.wq + (size_t(sg.panel) * c.C + sg.k0) * kWBytes;
        const uint8_t* sp = c.scales + size_t(sg.panel) * (c.C / c.group_chunks) * kScBytes;
        for (int k = sg.k0; k < sg.k1; ++k, ++n, wp += kWBytes) {
            const int s = n % kStages;
            mbar_wait(&B->empty[s], ((n / kStages) & 1) ^ 1);
            mbar_arrive_expect_tx(&B->full[s], kWBytes + kScBytes);
            bulk_g2s(wring + s * kWBytes, wp, kWBytes, &B->full[s], pol_w);
            bulk_g2s(scring + s * kScBytes, sp + size_t(k / c.group_chunks) * kScBytes, kScBytes, &B->full[s], pol_s);
        }
    }
}

// ---- warp 1: x tiles ----------------------------------------------------------------------------------------
// Lane l copies, for every token m < M, the 8-byte piece k = 4l..4l+3 of the chunk's 128 columns to the place the
// MMA expects it: k-tile half = l >> 4; inside the k-tile k = 16 t + 4 j + e goes to K position 16 j + 4 t + e
// (see the header: the 16x256b TMEM store spreads the columns of lane (g, t)'s word over MMA j = 0..3), in the
// K-major SWIZZLE_128B layout: row m at (m >> 3) * 1024 + (m & 7) * 128, 16-byte unit index XOR (m & 7).
__device__ void x_loader(const LsParams& P, uint8_t* xring, Bars* B, int lane) {
    const int half = lane >> 4, t = (lane & 15) >> 2, j = lane & 3;
    const int unit = 2 * j + (t >> 1), off = (t & 1) * 8;
    SegIter it;
    Seg sg;
    int n = 0, ph_seen = 0;
    while (it.next(P, sg)) {
        if (sg.ph != ph_seen) {     // this phase's x is an earlier phase's y: wait until all its panels are stored
            for (int q = ph_seen; q < sg.ph; ++q) wait_counter(P.done + q, unsigned(P.phase_panels[q]));
            ph_seen = sg.ph;
        }
        const LsCall& c = P.calls[sg.call];
        const __half* xp = c.x + size_t(sg.k0) * 128 + 4 * lane;
        for (int k = sg.k0; k < sg.k1; ++k, ++n, xp += 128) {
            const int s = n % kStages;
            mbar_wait(&B->empty[s], ((n / kStages) & 1) ^ 1);
            const uint32_t dst = smem_u32(xring + s * kXBytes) + half * 2048 + off;
#pragma unroll
            for (int m = 0; m < 16; ++m)
                if (m < c.M)
                    cp_async8(dst + (m >> 3) * 1024 + (m & 7) * 128 + ((unit ^ (m & 7)) << 4), xp + size_t(m) * c.K);
            cp_async_arrive_noinc(&B->full[s]);
        }
    }
}

// ---- warp 2 (one lane): MMA issue ---------------------------------------------------------------------------
__device__ void mma_issuer(const LsParams& P, uint8_t* xring, Bars* B, uint32_t tmem) {
    SegIter it;
    Seg sg;
    int n = 0, db = 0;
    unsigned uses[2] = {0, 0};
    while (it.next(P, sg)) {
        const int gc = P.calls[sg.call].group_chunks;
        bool fresh = true;      // next MMA starts an accumulation run
        for (int k = sg.k0; k < sg.k1; ++k, ++n) {
            const int s = n % kStages;
            if (fresh) mbar_wait(&B->d_empty[db], (uses[db] & 1) ^ 1);
            const uint64_t bd = desc_sw128(smem_u32(xring + s * kXBytes));
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int tau = 2 * n + h, slot = tau % kASlots;
                mbar_wait(&B->a_full[slot], (tau / kASlots) & 1);
                tc_fence_after();
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    umma_ts(tmem + kDCol + 16 * db, tmem + slot * 32 + 8 * j, bd + uint64_t(h * 128 + 2 * j), !(fresh && h == 0 && j == 0));
                umma_commit(&B->a_empty[slot]);
            }
            fresh = false;
            umma_commit(&B->empty[s]);
            if ((k + 1) % gc == 0 || k + 1 == sg.k1) {
                umma_commit(&B->d_full[db]);
                ++uses[db];
                db ^= 1;
                fresh = true;
            }
        }
    }
}

// ---- warps 8-23: int4 -> fp16 -> TMEM -----------------------------------------------------------------------
__device__ void dequantiser(int n_total, uint8_t* wring, Bars* B, uint32_t tmem, int warp, int lane) {
    const int q = warp & 3, i = (warp - 8) >> 2;
    const uint32_t w_lane = smem_u32(wring) + (2 * q * 32 + lane) * 16;
    const uint32_t t_lane = tmem + (uint32_t(32 * q) << 16);
    for (int tau = i; tau < 2 * n_total; tau += 4) {
        const int n = tau >> 1, h = tau & 1, s = n % kStages, slot = tau % kASlots;
        mbar_wait(&B->a_empty[slot], ((tau / kASlots) & 1) ^ 1);
        mbar_wait(&B->full[s], (n / kStages) & 1);
        tc_fence_after();
#pragma unroll
        for (int sp = 0; sp < 2; ++sp) {
            uint4 w;
            const uint32_t addr = w_lane + s * kWBytes + h * 4096 + sp * 512;
            asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(w.x), "=r"(w.y), "=r"(w.z), "=r"(w.w) : "r"(addr));
            uint32_t a[4], b[4], c[4], d[4];
            dequant_word(w.x, a);   // row g,   k 16t + 0..7
            dequant_word(w.y, b);   // row g,   k 16t + 8..15
            dequant_word(w.z, c);   // row g+8, k 16t + 0..7
            dequant_word(w.w, d);   // row g+8, k 16t + 8..15
            // register order of 16x256b.x4: MMA j <- {row g: 2 regs, row g+8: 2 regs}
            asm volatile(
                "tcgen05.st.sync.aligned.16x256b.x4.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
                ::"r"(t_lane + slot * 32 + (uint32_t(16 * sp) << 16)),
                "r"(a[0]), "r"(a[1]), "r"(c[0]), "r"(c[1]), "r"(a[2]), "r"(a[3]), "r"(c[2]), "r"(c[3]),
                "r"(b[0]), "r"(b[1]), "r"(d[0]), "r"(d[1]), "r"(b[2]), "r"(b[3]), "r"(d[2]), "r"(d[3])
                : "memory");
        }
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        fence_proxy_async_smem();       // the x tile was written by cp.async (generic proxy); the MMA reads it through the async proxy
        tc_fence_before();
        __syncwarp();
        if (lane == 0) {
            mbar_arrive(&B->a_full[slot]);
            mbar_arrive(&B->empty[s]);
        }
    }
}
}  // namespace ls

namespace ls {
__device__ __forceinline__ void epi_bar() { named_bar_sync(1, 128); }

// ---- warps 4-7: accumulate the runs, finalise panel segments ------------------------------------------------
__device__ void epilogue(const LsParams& P, uint8_t* scring, float* us, Bars* B, uint32_t tmem, int warp, int lane) {
    const int q = warp - 4, row = 32 * q + lane, et = row;        // et = thread index among the 128 epilogue threads
    const int sc_off = ((row >> 4) * 16 + 2 * (row & 7) + ((row >> 3) & 1)) * 2;
    const int G = gridDim.x, b = blockIdx.x;
    SegIter it;
    Seg sg;
    int n = 0, db = 0;
    unsigned uses[2] = {0, 0};
    while (it.next(P, sg)) {
        const LsCall& c = P.calls[sg.call];
        const int gc = c.group_chunks;
        float acc[16];
#pragma unroll
        for (int m = 0; m < 16; ++m) acc[m] = 0.f;
        for (int k = sg.k0; k < sg.k1; ++k, ++n) {
            const int s = n % kStages;
            const bool readout = ((k + 1) % gc == 0) || (k + 1 == sg.k1);
            mbar_wait(&B->full[s], (n / kStages) & 1);
            float scale = 0.f;
            if (readout) scale = __half2float(*reinterpret_cast<const __half*>(scring + s * kScBytes + sc_off));
            __syncwarp();
            if (lane == 0) mbar_arrive(&B->empty[s]);
            if (readout) {
                mbar_wait(&B->d_full[db], uses[db] & 1);
                tc_fence_after();
                uint32_t v[16];
                asm volatile(
                    "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                    : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                      "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
                    : "r"(tmem + kDCol + 16 * db + (uint32_t(32 * q) << 16))
                    : "memory");
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&B->d_empty[db]);
                ++uses[db];
                db ^= 1;
#pragma unroll
                for (int m = 0; m < 16; ++m) acc[m] = fmaf(scale, __uint_as_float(v[m]), acc[m]);
            }
        }
        // ---- end of the segment: S8 split-K, S7 rank-r update, cast, store ----
        const int T = P.phase_chunks[sg.ph];
        const bool whole = (sg.k0 == 0 && sg.k1 == c.C);
        bool finalize = whole;
        if (!whole) {
            const int lo_b = range_lo(b, T, G);
            const int which = (sg.pos == lo_b) ? 0 : 1;
            float* slot = P.partial + (size_t((sg.ph & 1) * G + b) * 2 + which) * 2048;
#pragma unroll
            for (int m = 0; m < 16; ++m) slot[m * 128 + row] = acc[m];
            epi_bar();
            const int p_begin = c.chunk_base + sg.panel * c.C, p_end = p_begin + c.C;
            if (et == 0) {
                // CTAs that hold a piece of this panel (ranges may be empty when the phase has fewer chunks than CTAs)
                int parts = 0;
                for (int pos = p_begin; pos < p_end; pos = range_lo(cta_of(pos, T, G) + 1, T, G)) ++parts;
                unsigned* ctr = P.counters + c.panel_base + sg.panel;
                const unsigned old = atom_add_acq_rel(ctr, 1);      // releases this CTA's partial, acquires the others'
                const int last = (old == unsigned(parts - 1));
                if (last) *ctr = 0;                                  // self-cleaning
                B->flag = last;
            }
            epi_bar();
            finalize = (B->flag != 0);
            if (finalize) {
#pragma unroll
                for (int m = 0; m < 16; ++m) acc[m] = 0.f;
                for (int pos = p_begin; pos < p_end;) {             // fixed CTA order: bitwise reproducible
                    const int cq = cta_of(pos, T, G);
                    const int lo_q = range_lo(cq, T, G);
                    const int wq = (pos == lo_q) ? 0 : 1;
                    pos = range_lo(cq + 1, T, G);
                    const float* sj = P.partial + (size_t((sg.ph & 1) * G + cq) * 2 + wq) * 2048;
                    float tmp[16];
#pragma unroll
                    for (int m = 0; m < 16; ++m) tmp[m] = __ldcg(sj + m * 128 + row);
#pragma unroll
                    for (int m = 0; m < 16; ++m) acc[m] += tmp[m];
                }
            }
        }
        if (finalize) {
            const int nrow = sg.panel * 128 + row;
            if (c.r > 0) {
                if (B->u_call != sg.call) {      // u of this call is not staged yet (uniform across the 128 threads)
                    epi_bar();
                    if (et == 0) wait_counter(P.ec_sync + 2 * c.ec_slot + 1, 1u);     // wait late: z was complete long ago
                    epi_bar();
                    const float* ug = P.ubuf + size_t(c.ec_slot) * 2048;
                    for (int idx = et; idx < c.M * c.r; idx += 128) us[idx] = __ldcg(ug + idx);
                    if (et == 0) B->u_call = sg.call;
                    epi_bar();
                }
                const uint4* Brow = reinterpret_cast<const uint4*>(c.B + size_t(nrow) * c.r);
#pragma unroll 2
                for (int j8 = 0; j8 < c.r / 8; ++j8) {
                    const uint4 bv = __ldg(Brow + j8);
                    const __half2* bh = reinterpret_cast<const __half2*>(&bv);
                    float bf[8];
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const float2 f = __half22float2(bh[e]);
                        bf[2 * e] = f.x; bf[2 * e + 1] = f.y;
                    }
#pragma unroll
                    for (int m = 0; m < 16; ++m) {
                        if (m < c.M) {
                            const float4* up = reinterpret_cast<const float4*>(us + m * c.r + j8 * 8);
                            const float4 ua = up[0], ub = up[1];
                            acc[m] += ua.x * bf[0] + ua.y * bf[1] + ua.z * bf[2] + ua.w * bf[3] +
                                      ub.x * bf[4] + ub.y * bf[5] + ub.z * bf[6] + ub.w * bf[7];
                        }
                    }
                }
            }
#pragma unroll
            for (int m = 0; m < 16; ++m)
                if (m < c.M) c.y[size_t(m) * c.N + nrow] = __float2half_rn(acc[m]);
            if (P.n_phases > 1) {               // somebody may be waiting for this phase's y
                epi_bar();
                if (et == 0) { __threadfence(); red_add_release(P.done + sg.ph, 1u); }
            }
        }
    }
}
}  // namespace ls

namespace ls {
// ---- warp 3: z = x [A; w_g]^T, gate, u (S4-S6) --------------------------------------------------------------
__device__ __forceinline__ void ec_load16(const __half* row, int col, uint32_t (&lo)[4], uint32_t (&hi)[4]) {
    if (row) {
        const uint4 a = *reinterpret_cast<const uint4*>(row + col);
        const uint4 b = *reinterpret_cast<const uint4*>(row + col + 8);
        lo[0] = a.x; lo[1] = a.y; lo[2] = a.z; lo[3] = a.w;
        hi[0] = b.x; hi[1] = b.y; hi[2] = b.z; hi[3] = b.w;
    } else {
#pragma unroll
        for (int i = 0; i < 4; ++i) lo[i] = hi[i] = 0u;
    }
}
__device__ void ec_call(const LsParams& P, int ci, int lane) {
    const LsCall& c = P.calls[ci];
    const int g = lane >> 2, t = lane & 3, G = gridDim.x;
    const bool scalar = (c.gate_kind == SPEAR_GATE_SCALAR_SIGMOID);
    const int rows_total = c.r + (scalar ? 1 : 0);
    const int strips = (rows_total + 15) >> 4;
    const int ktiles = c.K >> 6;
    const int ksplit = max(1, min(ktiles, G / strips));
    const int n_tasks = strips * ksplit;
    float* z = P.zbuf + size_t(c.ec_slot) * 16 * kZStride;
    const __half* px0 = g < c.M ? c.x + size_t(g) * c.K : nullptr;
    const __half* px1 = g + 8 < c.M ? c.x + size_t(g + 8) * c.K : nullptr;
    // rotate the task -> CTA map from call to call so that the same CTAs are not hit every time
    for (int task = (blockIdx.x + G - (ci * 37) % G) % G; task < n_tasks; task += G) {
        const int strip = task % strips, ks = task / strips;
        const int rho0 = strip * 16 + g, rho1 = rho0 + 8;
        const __half* pa0 = rho0 < c.r ? c.A + size_t(rho0) * c.K : (rho0 == c.r && scalar ? c.w_g : nullptr);
        const __half* pa1 = rho1 < c.r ? c.A + size_t(rho1) * c.K : (rho1 == c.r && scalar ? c.w_g : nullptr);
        const int kt_begin = int((long long)ks * ktiles / ksplit), kt_end = int((long long)(ks + 1) * ktiles / ksplit);
        float acc0[4] = {0.f, 0.f, 0.f, 0.f}, acc1[4] = {0.f, 0.f, 0.f, 0.f};
        for (int kt = kt_begin; kt < kt_end; ++kt) {
            const int col = kt * 64 + 16 * t;
            uint32_t a0l[4], a0h[4], a1l[4], a1h[4], x0l[4], x0h[4], x1l[4], x1h[4];
            ec_load16(pa0, col, a0l, a0h);
            ec_load16(pa1, col, a1l, a1h);
            ec_load16(px0, col, x0l, x0h);
            ec_load16(px1, col, x1l, x1h);
#pragma unroll
            for (int jj = 0; jj < 4; ++jj) {
                mma_m16n8k16(acc0, a0l[jj], a1l[jj], a0h[jj], a1h[jj], x0l[jj], x0h[jj]);
                mma_m16n8k16(acc1, a0l[jj], a1l[jj], a0h[jj], a1h[jj], x1l[jj], x1h[jj]);
            }
        }
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int rho = (i & 2) ? rho1 : rho0, tok = 2 * t + (i & 1);
            if (rho < rows_total) {
                if (tok < c.M) atomicAdd(z + tok * kZStride + rho, acc0[i]);
                if (tok + 8 < c.M) atomicAdd(z + (tok + 8) * kZStride + rho, acc1[i]);
            }
        }
    }
    __syncwarp();
    unsigned* sync = P.ec_sync + 2 * c.ec_slot;
    unsigned old = 0;
    if (lane == 0) old = atom_add_acq_rel(sync, 1u);
    old = __shfl_sync(0xffffffffu, old, 0);
    if (old != unsigned(G - 1)) return;
    // last arriver: z is complete -> gate (S5), u = alpha gamma z (S6)
    const float bias = (scalar && c.b_g) ? __ldg(c.b_g) : 0.f;
    float* u = P.ubuf + size_t(c.ec_slot) * 2048;
    for (int idx = lane; idx < c.M * c.r; idx += 32) {
        const int m = idx / c.r, j = idx - m * c.r;
        const float zz = __ldcg(z + m * kZStride + j);
        float gam = 1.f;
        if (scalar) gam = 1.f / (1.f + expf(-(__ldcg(z + m * kZStride + c.r) + bias)));
        u[idx] = c.alpha * gam * zz;
        if (scalar && c.gate_out && j == 0) c.gate_out[m] = gam;
    }
    __syncwarp();
    for (int i = lane; i < 16 * kZStride; i += 32) z[i] = 0.f;       // the next launch finds zeros
    __syncwarp();
    if (lane == 0) {
        sync[0] = 0;
        __threadfence();
        red_add_release(sync + 1, 1u);
    }
}
__device__ void ec_warp(const LsParams& P, int lane) {
    for (int ph = 0; ph < P.n_phases; ++ph) {
        if (ph > 0) wait_counter(P.done + ph - 1, unsigned(P.phase_panels[ph - 1]));
        for (int ci = P.phase_first_call[ph]; ci < P.phase_first_call[ph + 1]; ++ci)
            if (P.calls[ci].r > 0) ec_call(P, ci, lane);
    }
}
}  // namespace ls

__global__ void __launch_bounds__(ls::kThreads, 1) ls_kernel(const __grid_constant__ LsParams P) {
    using namespace ls;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* base = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* xring = base + Smem::x;
    uint8_t* wring = base + Smem::w;
    uint8_t* scring = base + Smem::sc;
    float* us = reinterpret_cast<float*>(base + Smem::u);
    Bars* B = reinterpret_cast<Bars*>(base + Smem::bars);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int s = 0; s < kStages; ++s) { mbar_init(&B->full[s], 1 + 32); mbar_init(&B->empty[s], kEmptyCount); }
        for (int s = 0; s < kASlots; ++s) { mbar_init(&B->a_full[s], 4); mbar_init(&B->a_empty[s], 1); }
        for (int s = 0; s < 2; ++s) { mbar_init(&B->d_full[s], 1); mbar_init(&B->d_empty[s], 4); }
        B->flag = 0;
        B->u_call = -1;
        fence_mbar_init();
    }
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&B->tmem)), "n"(kTmemCols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = B->tmem;

    if (warp == 0) {
        if (lane == 0) producer(P, wring, scring, B);
    } else if (warp == 1) {
        x_loader(P, xring, B, lane);
    } else if (warp == 2) {
        if (lane == 0) mma_issuer(P, xring, B, tmem);
    } else if (warp == 3) {
        ec_warp(P, lane);
    } else if (warp < 8) {
        epilogue(P, scring, us, B, tmem, warp, lane);
    } else {
        dequantiser(total_chunks(P), wring, B, tmem, warp, lane);
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 2) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(kTmemCols) : "memory");
    if (threadIdx.x == 0) {
        // the last CTA to leave resets what the next launch expects to be zero
        unsigned* exit_ctr = P.done + kLsMaxCalls;
        __threadfence();
        if (atom_add_acq_rel(exit_ctr, 1u) == gridDim.x - 1) {
            for (int ph = 0; ph < P.n_phases; ++ph) P.done[ph] = 0;
            for (int ci = 0; ci < P.n_calls; ++ci)
                if (P.calls[ci].ec_slot >= 0) P.ec_sync[2 * P.calls[ci].ec_slot + 1] = 0;
            *exit_ctr = 0;
        }
    }
}

// ---- host ----------------------------------------------------------------------------------------------------
static int g_ls_grid = 0;
int ls_grid() {
    if (g_ls_grid) return g_ls_grid;
    const int smem = int(ls::Smem::total + 1024);
    if (cudaFuncSetAttribute(ls_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return 0;
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ls_kernel, ls::kThreads, smem) != cudaSuccess || per_sm < 1) return 0;
    g_ls_grid = device_info().num_sms;      // one CTA per SM: the kernel owns the SM's shared and tensor memory
    return g_ls_grid;
}
size_t ls_workspace_bytes(int grid) {
    return size_t(grid) * 2 * 2 * 2048 * 4 + (size_t(1) << 20);
}
int launch_lstream(const LsParams& p, cudaStream_t st) {
    const int grid = ls_grid();
    if (grid <= 0) return set_error(SPEAR_ECUDA, "layer-stream kernel cannot be resident on this device");
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(ls::kThreads);
    cfg.dynamicSmemBytes = ls::Smem::total + 1024;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;      // all CTAs co-resident or the launch fails: the device-wide
    attr[0].val.cooperative = 1;                      // arrive / wait patterns above cannot deadlock
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    SPEAR_CUDA_OK(cudaLaunchKernelEx(&cfg, ls_kernel, p));
    count_launch();
    return SPEAR_OK;
}

}  // namespace spear

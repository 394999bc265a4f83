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
//   * 896 threads, one CTA per SM.  Service warps: warp 0 (one lane) weight producer -- cp.async.bulk of the chunk into
//     a shared-memory ring of LS_STAGES = 10 stages (evict_first); warp 1 (one lane) x producer -- the chunk's x tile
//     ([16 tokens][128 columns] fp16 in the MMA operand layout, k-permuted; written once per launch into the workspace
//     by x_prologue, so it is a plain bulk copy here); warp 3 (one lane) scale producer -- the chunk's 256-byte scale
//     slot rides in the same stage (global scale loads queued 2-3 us behind the deep bulk ring) -- and TMEM allocation;
//   * warps 8-23, the workers: 4 pipelines x 4 TMEM lane quarters; pipeline i takes the chunks n = i mod 4 of the CTA's
//     stream: LDS.128 -> exact q - 8 in fp16 (dequant_word) -> tcgen05.st.16x256b.x4 into A-operand slot n mod 6 in
//     TENSOR MEMORY (6 slots x 64 columns).  The SPW4 word of lane (g, t) holds rows g, g + 8 x columns 16t..16t+15,
//     the 16x256b store shape spreads a row's columns over the four lanes of a quad, so MMA j of a 64-column k-tile
//     sees k = 16t + 4j + e at its K position 16j + 4t + e; x_prologue applies the same permutation to x (a dot product is
//     order-invariant).  The same warps run the pipeline's epilogue, lagging TWO own chunks behind the dequantisation
//     (tcgen05.ld the run's accumulator, scale by s[n][group] in fp32, add into registers; at the end of a panel segment
//     hand the [16 tokens][128 rows] part over through shared memory); before a phase boundary they catch up;
//   * warps 24-27 (one lane each), MMA issuer of pipeline i: tcgen05.mma.cta_group::1.kind::f16, M = 128 rows of the
//     panel, N = 16 tokens, K = 16, A from TMEM, B = x tile from shared memory (SWIZZLE_128B, K-major), D = one of the
//     pipeline's two 16-column fp32 accumulators in TMEM; one accumulation run per scale group.  Measured: one thread
//     issues a small-N MMA every ~47 clk whatever N while the tensor pipe needs 8 clk, hence four issuers.  A lane waits
//     for a_empty[slot] of chunk m - 6 BEFORE a_full[slot] of chunk m: the slot barriers are shared between pipelines
//     and an mbarrier parity wait is only valid one phase behind (this was a 1-in-3000-replays hang);
//     tcgen05.commit frees the A slot / ring stage and hands D over;
//   * warps 4-7, the finalisers (thread = output row): sum the four pipelines' parts; split-K across CTAs through fp32
//     red.add accumulators in the workspace + an acq_rel counter per panel (the last arriver finalises); then the rank-r
//     update y += u B^T (B rows prefetched), one RN-even cast, store; in a chain also the k-permuted copy of y that the
//     next phase reads as its x tile, and the panel-completion counter that phase waits on;
//   * warp 2 (EC): this CTA's share of z = x [A; w_g]^T for every call of the phase (mma.sync, red.add), arrive; the
//     last arriver applies the gate (scalar form of BASELINE.json / gamma = 1; the MLP gate is not served here) and
//     publishes u = alpha gamma z behind a flag that finalisers look at only when they need it (z must be complete
//     before the gate).
//
// Where it stands (B200, config 2 step as ONE launch): 43 us plain / 60 us with the EC against 40 / 53 us for the same
// step on the per-call kernels over 12 lanes: ~12 us fixed (cooperative launch, prologue, first fill, tail) and a
// ~275 ns per-chunk hand-shake floor (3.3 TB/s streaming) that neither ring depth, ALU work nor MMA issue explains.
// It is therefore opt-in: spear_tune("lstream", 1), or a batch signature for which spear_plan_batch measured it faster
// (DESIGN.md 6.5).  Development builds: -DLS_TRACE (per-role time stamps, watchdog printf), -DLS_TIMER.
#include <cooperative_groups.h>
#include <cstdio>

#include "common.cuh"
#include "kernels.h"

namespace spear {

namespace ls {
#if defined(LS_TRACE) || defined(LS_TIMER)
__device__ __forceinline__ unsigned long long ls_now() { unsigned long long t; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t)); return t; }
#endif
#ifdef LS_TRACE
__shared__ unsigned long long g_stamp[48];
#define LS_STAMP(i) do { if (et == 0) g_stamp[i] = ls_now(); } while (0)
__shared__ unsigned long long g_ct[32][8];
#define LS_CT(n, j) do { if ((n) < 32) g_ct[n][j] = ls_now(); } while (0)
#else
#define LS_STAMP(i)
#define LS_CT(n, j)
#endif
#ifdef LS_TRACE
__device__ __forceinline__ void ls_wait_impl(uint64_t* bar, uint32_t parity, int tag, int a, int b) {
    long long t0 = clock64();
    while (!mbar_try_wait(bar, parity)) {
        if (clock64() - t0 > 400000000ll) {
            if ((threadIdx.x & 31) == 0 || (threadIdx.x >> 5) < 4 || (threadIdx.x >> 5) >= 24) printf("STUCK mbar tag %d cta %d warp %d lane %d info %d %d\n", tag, blockIdx.x, threadIdx.x >> 5, threadIdx.x & 31, a, b);
            t0 = clock64() + 4000000000ll;
        }
    }
}
#define LS_WAIT(bar, parity, tag, a, b) ls_wait_impl(bar, parity, tag, a, b)
#else
#define LS_WAIT(bar, parity, tag, a, b) mbar_wait(bar, parity)
#endif
#ifndef LS_STAGES
#define LS_STAGES 10
#endif
static_assert(LS_STAGES % 2 == 0 && LS_STAGES >= 6, "ring depth must be even: chunk n - kStages must belong to pipeline n or n + 2 (mod 4), whose progress a worker has observed before it tests full[] by parity");
constexpr int kStages = LS_STAGES;          // ring depth (chunks): 10 x (8 KiB weights + 4 KiB x tile + 256 B scales); measured 6..12: within 5 %
constexpr int kPipes = 4;                   // dequantisation / MMA pipelines; pipeline i owns chunks n = i (mod 4)
constexpr int kThreads = (8 + 4 * kPipes + kPipes) * 32;      // 4 service warps, 4 finalisers, 16 workers, 4 MMA issuers
constexpr int kWBytes = 8192, kXBytes = 4096, kScBytes = 256;
constexpr uint32_t kTmemCols = 512;
constexpr int kASlots = 6;                  // A-operand slots in tensor memory (64 columns = one chunk each); chunk n -> slot n mod 6
constexpr uint32_t kDCol = kASlots * 64;    // behind them: two 16-column fp32 accumulators per pipeline (6*64 + 4*32 = 512 columns)
constexpr uint32_t kIdesc = (1u << 4) | (uint32_t(16 >> 3) << 17) | (uint32_t(128 >> 4) << 24);
constexpr int kEmptyCount = 4 + 1;          // the chunk's 4 worker warps + its MMA commit
struct Smem {
    static constexpr size_t x = 0;
    static constexpr size_t w = x + size_t(kStages) * kXBytes;
    static constexpr size_t sc = w + size_t(kStages) * kWBytes;
    static constexpr size_t u = sc + size_t(kStages) * kScBytes;       // [16][128] fp32 staging of u
    static constexpr size_t part = u + 16 * 128 * 4;                   // [2][kPipes][16][128] fp32 segment hand-over
    static constexpr size_t bars = part + size_t(2) * kPipes * 2048 * 4;
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
#ifdef LS_TRACE
    long long t0 = clock64();
    while (ld_acquire(p) < target) {
        if (clock64() - t0 > 400000000ll) { printf("STUCK counter cta %d warp %d have %u want %u\n", blockIdx.x, threadIdx.x >> 5, ld_acquire(p), target); t0 = clock64() + 4000000000ll; }
    }
#else
    while (ld_acquire(p) < target) {}
#endif
}

// ---- the work sequence of this CTA --------------------------------------------------------------------------
struct Seg {
    int call, panel, k0, k1;   // chunks [k0, k1) of the panel
    int ph;                    // phase
    int pos;                   // position of chunk k0 in the phase's chunk sequence
};
// The phase's T chunks are cut into gridDim.x contiguous ranges: the first `rem` CTAs take per + 1 chunks, the
// others per (per = T / G, rem = T % G, supplied by the host: no 64-bit division on the device).
struct Cut { int per, rem; };
__device__ __forceinline__ int range_lo(int b, Cut c) { return b * c.per + min(b, c.rem); }
__device__ __forceinline__ int cta_of(int pos, Cut c) {
    const int big = c.rem * (c.per + 1);
    return pos < big ? pos / (c.per + 1) : c.rem + (pos - big) / c.per;     // pos >= big implies per >= 1
}
__device__ __forceinline__ Cut phase_cut(const LsParams& P, int ph) { return Cut{P.phase_per[ph], P.phase_rem[ph]}; }
// Segments of this CTA, phase by phase.  Inside a phase the range's LAST segment comes first when it is the head
// of a panel that continues in the next CTA: all pieces of a shared panel are then produced at the start of the
// phase, its split-K reduction happens in the shadow of the whole panels that follow, and the CTA's final
// segment needs no cross-CTA hand-shake.
struct SegIter {
    int ph, pos, hi, call, tail_pos;     // tail_pos: start of the deferred-to-front segment (== hi when none)
    bool tail_done;
    __device__ SegIter() : ph(-1), pos(0), hi(0), call(0), tail_pos(0), tail_done(true) {}
    __device__ void locate(const LsParams& P, int at, int first_call, int& ci, int& panel, int& k) const {
        ci = first_call;
        while (at >= P.calls[ci].chunk_base + P.calls[ci].P * P.calls[ci].C) ++ci;
        const int rel = at - P.calls[ci].chunk_base;
        panel = rel / P.calls[ci].C;
        k = rel - panel * P.calls[ci].C;
    }
    __device__ bool next(const LsParams& P, Seg& s) {
        const int b = blockIdx.x;
        while (pos >= tail_pos && tail_done) {
            if (++ph >= P.n_phases) return false;
            const Cut cut = phase_cut(P, ph);
            pos = range_lo(b, cut);
            hi = range_lo(b + 1, cut);
            call = P.phase_first_call[ph];
            tail_pos = hi;
            tail_done = true;
            if (hi > pos) {
                int ci, panel, k;
                locate(P, hi - 1, call, ci, panel, k);
                if (k + 1 < P.calls[ci].C) {          // the range ends inside a panel
                    tail_pos = max(pos, hi - 1 - k);
                    tail_done = false;
                }
            }
        }
        int at, end;
        if (!tail_done) { at = tail_pos; tail_done = true; end = hi; }
        else { at = pos; end = tail_pos; }
        int ci, panel, k;
        locate(P, at, (at == pos) ? call : P.phase_first_call[ph], ci, panel, k);
        const LsCall& c = P.calls[ci];
        s.call = ci; s.ph = ph; s.pos = at; s.panel = panel; s.k0 = k;
        const int seg_end = min(end, c.chunk_base + (panel + 1) * c.C);
        s.k1 = k + (seg_end - at);
        if (at == pos) { pos = seg_end; call = ci; }
        return true;
    }
};
__device__ __forceinline__ int total_chunks(const LsParams& P) {
    int n = 0;
    for (int ph = 0; ph < P.n_phases; ++ph) n += P.phase_per[ph] + (int(blockIdx.x) < P.phase_rem[ph] ? 1 : 0);
    return n;
}
}  // namespace ls

namespace ls {
struct Bars {
    uint64_t full[kStages], empty[kStages], a_full[kASlots], a_empty[kASlots], d_full[kPipes][2], d_empty[kPipes][2];
    uint64_t seg_full[2], seg_empty[2];      // segment hand-over (workers -> finalisers), double-buffered
    uint32_t tmem;
    int flag;       // epilogue broadcast: this CTA finalises the panel
    int u_call;     // call whose u sits in the staging buffer (-1 = none)
};
static_assert(sizeof(Bars) <= 1024, "barrier block");

// ---- warp 0: weights ------------------------------------------------------------------------------------------
__device__ void producer(const LsParams& P, uint8_t* wring, Bars* B) {
    const uint64_t pol_w = policy_evict_first();
    SegIter it;
    Seg sg;
    int n = 0;
    while (it.next(P, sg)) {
        const LsCall& c = P.calls[sg.call];
        const uint8_t* wp = c.wq + (size_t(sg.panel) * c.C + sg.k0) * kWBytes;
        for (int k = sg.k0; k < sg.k1; ++k, ++n, wp += kWBytes) {
            const int s = n % kStages;
            LS_WAIT(&B->empty[s], ((n / kStages) & 1) ^ 1, 1, n, 0);
            mbar_arrive_expect_tx(&B->full[s], kWBytes);
            bulk_g2s(wring + s * kWBytes, wp, kWBytes, &B->full[s], pol_w);
            LS_CT(n, 6);
        }
    }
}

// ---- x in the operand layout -----------------------------------------------------------------------------------
// The MMA wants, per chunk, the tile [k-tile half][16 tokens][64 columns] fp16 in the K-major SWIZZLE_128B layout
// (row m at (m >> 3) * 1024 + (m & 7) * 128, 16-byte unit index XOR (m & 7)) with the k-order of the weight
// fragments: inside a k-tile, column k = 16 t + 4 j + e sits at K position 16 j + 4 t + e (see the header).  That is
// a permutation of 8-byte pieces, which neither TMA nor a 16-byte cp.async can express, so x is rewritten ONCE per
// launch into the workspace (xperm: one contiguous tile per chunk, 2 KiB when M <= 8, else 4 KiB) and the tiles
// then travel through the ring as plain cp.async.bulk copies, like the weights.
__device__ __forceinline__ uint32_t xperm_offset(int m, int kk, int xtile) {    // byte offset of (token m, column kk of the chunk)
    const int l = kk >> 2, e = kk & 3;
    const int half = l >> 4, t = (l & 15) >> 2, j = l & 3;
    const int unit = 2 * j + (t >> 1);
    return half * (xtile >> 1) + (m >> 3) * 1024 + (m & 7) * 128 + ((unit ^ (m & 7)) << 4) + (t & 1) * 8 + e * 2;
}
// Prologue (all dequantisation warps of all CTAs): the external x of every call -> xperm, then one arrive per CTA.
__device__ void x_prologue(const LsParams& P, int tid, int nthreads) {
    const int gtid = blockIdx.x * nthreads + tid, gsz = gridDim.x * nthreads;
    for (int ci = 0; ci < P.n_calls; ++ci) {
        const LsCall& c = P.calls[ci];
        if (c.x_internal) continue;
        const int per_row = c.K >> 2;                   // 8-byte pieces per token row
        uint8_t* dstb = const_cast<uint8_t*>(c.xperm);
        for (int p = gtid; p < c.M * per_row; p += gsz) {
            const int m = p / per_row, q = p - m * per_row;
            const uint2 v = *reinterpret_cast<const uint2*>(c.x + size_t(m) * c.K + 4 * q);
            const int k = 4 * q;
            *reinterpret_cast<uint2*>(dstb + size_t(k >> 7) * c.xtile + xperm_offset(m, k & 127, c.xtile)) = v;
        }
    }
}

// ---- warp 1 (one lane): x tiles; warp 3 (one lane): scale slots ------------------------------------------------
__device__ void x_producer(const LsParams& P, uint8_t* xring, Bars* B) {
    const uint64_t pol = policy_evict_last();
    SegIter it;
    Seg sg;
    int n = 0, ph_seen = 0;
    bool prologue_seen = false;
    while (it.next(P, sg)) {
        const LsCall& c = P.calls[sg.call];
        if (sg.ph != ph_seen) {     // this phase's x is an earlier phase's y: wait until all its panels are stored
            for (int q = ph_seen; q < sg.ph; ++q) wait_counter(P.done + q, unsigned(P.phase_panels[q]));
            ph_seen = sg.ph;
            asm volatile("fence.proxy.async;" ::: "memory");     // generic-proxy stores of other SMs -> our bulk copies
        }
        if (!c.x_internal && !prologue_seen) {
            wait_counter(P.done + kLsMaxCalls + 1, gridDim.x);
            asm volatile("fence.proxy.async;" ::: "memory");
            prologue_seen = true;
#ifdef LS_TRACE
            g_stamp[47] = ls_now();
#endif
        }
        const uint8_t* xp = c.xperm + size_t(sg.k0) * c.xtile;
        for (int k = sg.k0; k < sg.k1; ++k, ++n, xp += c.xtile) {
            const int s = n % kStages;
            LS_WAIT(&B->empty[s], ((n / kStages) & 1) ^ 1, 2, n, 0);
            mbar_arrive_expect_tx(&B->full[s], c.xtile);
            bulk_g2s(xring + s * kXBytes, xp, c.xtile, &B->full[s], pol);
        }
    }
}
__device__ void sc_producer(const LsParams& P, uint8_t* scring, Bars* B) {
    const uint64_t pol = policy_evict_last();
    SegIter it;
    Seg sg;
    int n = 0;
    while (it.next(P, sg)) {
        const LsCall& c = P.calls[sg.call];
        const uint8_t* sp = c.scales + size_t(sg.panel) * (c.C / c.group_chunks) * kScBytes;
        for (int k = sg.k0; k < sg.k1; ++k, ++n) {
            const int s = n % kStages;
            LS_WAIT(&B->empty[s], ((n / kStages) & 1) ^ 1, 3, n, 0);
            mbar_arrive_expect_tx(&B->full[s], kScBytes);
            bulk_g2s(scring + s * kScBytes, sp + size_t(k / c.group_chunks) * kScBytes, kScBytes, &B->full[s], pol);
        }
    }
}

// ---- warps 20-23 (one lane each): MMA issue of pipeline i ---------------------------------------------------
__device__ void mma_issuer(const LsParams& P, uint8_t* xring, Bars* B, uint32_t tmem, int i) {
    SegIter it;
    Seg sg;
    int n = 0, db = 0;
    unsigned par = 0;       // bit b: parity of accumulator b's next d_empty phase
    const uint32_t d_base = tmem + kDCol + i * 32;
    while (it.next(P, sg)) {
        const int gsh = P.calls[sg.call].group_shift;       // log2(chunks per scale group); >= 31: one group per row
        const uint64_t half_desc = uint64_t(P.calls[sg.call].xtile >> 5);      // (xtile / 2) >> 4: descriptor step to the second k-tile
        const int n_seg = n + (sg.k1 - sg.k0);
        int m = n + ((i - n) & (kPipes - 1));                // first own chunk of the segment
        for (; m < n_seg; m += kPipes) {
            // the accumulation run (chunks of one scale group inside this segment) that chunk m belongs to
            const int k = sg.k0 + (m - n);
            const int run_lo = gsh >= 31 ? sg.k0 : max(sg.k0, (k >> gsh) << gsh);
            const int run_hi = gsh >= 31 ? sg.k1 : min(sg.k1, ((k >> gsh) + 1) << gsh);
            const bool first = (k - kPipes < run_lo), last = (k + kPipes >= run_hi);
            const int s = m % kStages, slot = m % kASlots;
            const uint32_t a_base = tmem + slot * 64;
            if (first) LS_WAIT(&B->d_empty[i][db], ((par >> db) & 1) ^ 1, 4, m, db);
            // A slots are shared between pipelines (chunk m - 6 belongs to another issuer): a parity wait is only valid
            // when the barrier is at most one phase behind, so first make sure MMA(m - 6) has been committed -- then
            // a_full[slot] can only be completed by chunk m's own workers
            LS_WAIT(&B->a_empty[slot], ((m / kASlots) & 1) ^ 1, 11, m, 0);
            LS_WAIT(&B->a_full[slot], (m / kASlots) & 1, 5, m, 0);
            tc_fence_after();
            const uint64_t bd = desc_sw128(smem_u32(xring + s * kXBytes));
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    umma_ts(d_base + 16 * db, a_base + h * 32 + 8 * j, bd + h * half_desc + uint64_t(2 * j), !(first && h == 0 && j == 0));
            umma_commit(&B->a_empty[slot]);
            umma_commit(&B->empty[s]);
            if (last) {
                umma_commit(&B->d_full[i][db]);
                par ^= 1u << db;
                db ^= 1;
            }
        }
        n = n_seg;
    }
}

// ---- warps 8-23: workers (pipeline g = chunks n = g mod 4, TMEM lane quarter q) ---------------------------------
// Per own chunk n: first the epilogue of own chunk n - 4 (tcgen05.ld of the pipeline's accumulator at the end of each
// scale-group run, acc += s * D, thread = output row; at the end of a segment the pipeline's partial sums go to a
// shared-memory hand-over buffer for the finaliser warps), then the dequantisation of chunk n: LDS.128 -> exact
// q - 8 in fp16 -> tcgen05.st.16x256b.x4 into the pipeline's A slot.  The row's scale is read from the ring stage
// while the chunk is there and kept in a register until the run is read out.
struct EpiState {
    SegIter it;
    Seg sg;
    int n0, n1;          // stream positions [n0, n1) of the current segment's chunks
    int m;               // next own chunk to look at
    int seg_idx;         // segments finished (hand-over buffer = seg_idx & 1)
    bool live, done;
    int db;
    unsigned par;
};
__device__ void worker(const LsParams& P, uint8_t* wring, const uint8_t* scring, float* part, Bars* B, uint32_t tmem,
                       int warp, int lane) {
    const int q = warp & 3, g = (warp - 8) >> 2;
    const int row = 32 * q + lane;
    const int sc_off = ((row >> 4) * 16 + 2 * (row & 7) + ((row >> 3) & 1)) * 2;       // SPW4 scale slot of this row
    const uint32_t w_lane = smem_u32(wring) + (2 * q * 32 + lane) * 16;
    const uint32_t t_quarter = tmem + (uint32_t(32 * q) << 16);
    const uint32_t d_lane = tmem + kDCol + g * 32 + (uint32_t(32 * q) << 16);
    const int n_total = total_chunks(P);
    EpiState e;
    e.n0 = e.n1 = 0; e.m = g; e.seg_idx = 0; e.live = false; e.done = false; e.db = 0; e.par = 0;
    float acc[16];
#pragma unroll
    for (int mm = 0; mm < 16; ++mm) acc[mm] = 0.f;
    float sc_a = 0.f, sc_b = 0.f;      // this row's scale in the groups of own chunks n - 4 and n - 8 (read out two iterations late)

    // epilogue of every own chunk <= limit, plus the segment hand-overs that become due
    auto epilogue_until = [&](int limit, int old_chunk) __attribute__((always_inline)) {
        while (!e.done) {
            if (!e.live) {
                e.n0 = e.n1;
                if (!e.it.next(P, e.sg)) { e.done = true; break; }
                e.n1 = e.n0 + (e.sg.k1 - e.sg.k0);
                e.live = true;
            }
            if (e.m < e.n1) {
                if (e.m > limit) break;
                // own chunk e.m of this segment: is it the pipeline's last chunk of its scale-group run?
                const int gsh = P.calls[e.sg.call].group_shift;
                const int k = e.sg.k0 + (e.m - e.n0);
                const int run_hi = gsh >= 31 ? e.sg.k1 : min(e.sg.k1, ((k >> gsh) + 1) << gsh);      // chunk after the run
                if (k + kPipes >= run_hi) {
                    LS_WAIT(&B->d_full[g][e.db], (e.par >> e.db) & 1, 6, e.m, e.db);
                    tc_fence_after();
                    uint32_t v[16];
                    asm volatile(
                        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
                          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
                        : "r"(d_lane + 16 * e.db)
                        : "memory");
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&B->d_empty[g][e.db]);
                    e.par ^= 1u << e.db;
                    e.db ^= 1;
                    const float sc = (e.m == old_chunk) ? sc_b : sc_a;
#pragma unroll
                    for (int mm = 0; mm < 16; ++mm) acc[mm] = fmaf(sc, __uint_as_float(v[mm]), acc[mm]);
                }
                e.m += kPipes;
                continue;
            }
            // the segment holds no further own chunk: hand the pipeline's partial sums to the finalisers
            const int buf = e.seg_idx & 1;
            LS_WAIT(&B->seg_empty[buf], ((e.seg_idx >> 1) & 1) ^ 1, 7, e.seg_idx, e.m);
            float* dst = part + size_t(buf * kPipes + g) * 2048 + row;
#pragma unroll
            for (int mm = 0; mm < 16; ++mm) { dst[mm * 128] = acc[mm]; acc[mm] = 0.f; }
            __syncwarp();
            if (lane == 0) mbar_arrive(&B->seg_full[buf]);
            ++e.seg_idx;
            e.live = false;
        }
    };

    // stream position at which the next phase of this CTA starts: its x tiles exist only once the previous phase is
    // finalised, which needs this pipeline's partial sums -- so the lagging epilogue catches up before crossing it
    int ph_next = 1;
    int boundary = P.n_phases > 1 ? P.phase_per[0] + (int(blockIdx.x) < P.phase_rem[0] ? 1 : 0) : 0x7fffffff;
    for (int n = g;; n += kPipes) {
        // epilogue of own chunk n - 8 (its MMAs finished long ago: no wait, and the accumulator is free for chunk n);
        // also of chunk n - 4 when chunk n opens a new phase; past the end of the stream: whatever is left
        int limit = n - 2 * kPipes;
        if (n >= boundary) {
            limit = n - kPipes;
            while (n >= boundary) {
                boundary = ph_next < P.n_phases - 1 ? boundary + P.phase_per[ph_next] + (int(blockIdx.x) < P.phase_rem[ph_next] ? 1 : 0)
                                                    : 0x7fffffff;
                ++ph_next;
            }
        }
        epilogue_until(limit, n - 2 * kPipes);
        if (n >= n_total) {
            if (e.done) break;
            sc_b = sc_a;
            continue;
        }
        const int s = n % kStages, slot = n % kASlots;
        const uint32_t t_lane = t_quarter + slot * 64;
        LS_WAIT(&B->a_empty[slot], ((n / kASlots) & 1) ^ 1, 8, n, 0);
        LS_WAIT(&B->full[s], (n / kStages) & 1, 9, n, 0);
#ifdef LS_TRACE
        if (n == 0 && q == 0 && lane == 0) g_stamp[46] = ls_now();
#endif
        tc_fence_after();
        sc_b = sc_a;
        sc_a = __half2float(*reinterpret_cast<const __half*>(scring + s * kScBytes + sc_off));
#pragma unroll
        for (int h = 0; h < 2; ++h) {
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
                    ::"r"(t_lane + h * 32 + (uint32_t(16 * sp) << 16)),
                    "r"(a[0]), "r"(a[1]), "r"(c[0]), "r"(c[1]), "r"(a[2]), "r"(a[3]), "r"(c[2]), "r"(c[3]),
                    "r"(b[0]), "r"(b[1]), "r"(d[0]), "r"(d[1]), "r"(b[2]), "r"(b[3]), "r"(d[2]), "r"(d[3])
                    : "memory");
            }
        }
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
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

// ---- warps 4-7: finalise panel segments (thread = output row) --------------------------------------------------
__device__ void finaliser(const LsParams& P, const float* part, float* us, Bars* B, int warp, int lane) {
    const int q = warp - 4, row = 32 * q + lane, et = row;        // et = thread index among the 128 finaliser threads
    const int G = gridDim.x;
    SegIter it;
    Seg sg;
    int seg_idx = 0;
    while (it.next(P, sg)) {
        const LsCall& c = P.calls[sg.call];
        // While the workers are still on this segment: fetch this row of B (first 32 columns) and, when the call's u has
        // been published already, stage it -- so that the finalisation below finds both on chip.
        uint4 bpre[4];
        if (c.r > 0) {
            const uint4* Brow = reinterpret_cast<const uint4*>(c.B + size_t(sg.panel * 128 + row) * c.r);
#pragma unroll
            for (int j8 = 0; j8 < 4; ++j8)
                if (j8 < c.r / 8) bpre[j8] = __ldg(Brow + j8);
            if (B->u_call != sg.call) {          // uniform across the 128 threads
                epi_bar();
                if (et == 0) B->flag = ld_acquire(P.ec_sync + 2 * c.ec_slot + 1) >= 1u;
                epi_bar();
                if (B->flag) {
                    const float* ug = P.ubuf + size_t(c.ec_slot) * 2048;
                    for (int idx = et; idx < c.M * c.r; idx += 128) us[idx] = __ldcg(ug + idx);
                    epi_bar();
                    if (et == 0) B->u_call = sg.call;
                }
                epi_bar();
            }
        }
        // the four pipelines' partial sums of this segment
        const int buf = seg_idx & 1;
        LS_WAIT(&B->seg_full[buf], (seg_idx >> 1) & 1, 10, seg_idx, 0);
        float acc[16];
        {
            const float* src = part + size_t(buf * kPipes) * 2048 + row;
#pragma unroll
            for (int m = 0; m < 16; ++m) acc[m] = (src[m * 128] + src[2048 + m * 128]) + (src[4096 + m * 128] + src[6144 + m * 128]);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&B->seg_empty[buf]);
        ++seg_idx;
        LS_STAMP(40);
        // ---- end of the segment: S8 split-K, S7 rank-r update, cast, store ----
        const Cut cut = phase_cut(P, sg.ph);
        const bool whole = (sg.k0 == 0 && sg.k1 == c.C);
        bool finalize = whole;
        if (!whole) {
            // The panel is shared with neighbouring CTAs: every holder adds its piece to the panel's fp32 accumulator in
            // the workspace (red.add, fire and forget) and arrives; the last arriver takes the sum, leaves zeros behind
            // and finalises.  One round trip whatever the number of pieces (the sum order, hence the last bits of y of
            // such panels, depends on arrival order -- inside the tolerance, PAPER.md leaves the order free).
            const int p_begin = c.chunk_base + sg.panel * c.C;
            const int c_first = cta_of(p_begin, cut);
            const int parts = cut.per == 0 ? c.C : cta_of(p_begin + c.C - 1, cut) - c_first + 1;
            float* accum = P.partial + size_t((sg.ph & 1) * G + c_first) * 2048 + row;
#pragma unroll
            for (int m = 0; m < 16; ++m) atomicAdd(accum + m * 128, acc[m]);
            epi_bar();
            LS_STAMP(41);
            if (et == 0) {
                unsigned* ctr = P.counters + c.panel_base + sg.panel;
                const unsigned old = atom_add_acq_rel(ctr, 1);      // releases this CTA's adds, acquires the others'
                const int last = (old == unsigned(parts - 1));
                if (last) *ctr = 0;                                  // self-cleaning
                B->flag = last;
            }
            epi_bar();
            LS_STAMP(42);
            finalize = (B->flag != 0);
            if (finalize) {
#pragma unroll
                for (int m = 0; m < 16; ++m) acc[m] = __ldcg(accum + m * 128);
#pragma unroll
                for (int m = 0; m < 16; ++m) accum[m * 128] = 0.f;
            }
        }
        LS_STAMP(43);
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
#pragma unroll 4
                for (int j8 = 0; j8 < c.r / 8; ++j8) {
                    const uint4 bv = j8 < 4 ? bpre[j8 & 3] : __ldg(Brow + j8);
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
            if (c.yperm) {      // a later call of this launch reads this y as its x: hand it over in the operand layout
                uint8_t* yp = c.yperm + size_t(nrow >> 7) * c.xtile;
#pragma unroll
                for (int m = 0; m < 16; ++m)
                    if (m < c.M) *reinterpret_cast<__half*>(yp + xperm_offset(m, nrow & 127, c.xtile)) = __float2half_rn(acc[m]);
            }
            LS_STAMP(44);
            if (P.n_phases > 1) {               // somebody may be waiting for this phase's y
                epi_bar();
                if (et == 0) { __threadfence(); asm volatile("fence.proxy.async;" ::: "memory"); red_add_release(P.done + sg.ph, 1u); }
            }
        }
    }
}
}  // namespace ls

namespace ls {
// ---- warp 2: z = x [A; w_g]^T, gate, u (S4-S6) --------------------------------------------------------------
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
// this CTA's share of z = x [A; w_g]^T of call ci, added to the global fp32 z (red.add); no synchronisation here
__device__ void ec_partial(const LsParams& P, int ci, int lane) {
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
}
// z of call ci is complete (the gate needs the fully reduced z): gate (S5), u = alpha gamma z (S6),
// publish u behind the call's flag, leave z zeroed for the next launch
__device__ void ec_gate(const LsParams& P, int ci, int lane) {
    const LsCall& c = P.calls[ci];
    const bool scalar = (c.gate_kind == SPEAR_GATE_SCALAR_SIGMOID);
    float* z = P.zbuf + size_t(c.ec_slot) * 16 * kZStride;
    unsigned* sync = P.ec_sync + 2 * c.ec_slot;
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
// a call of a later phase (x is an earlier phase's y): the EC warp of every CTA adds its share and arrives; the last
// arriver applies the gate
__device__ void ec_call(const LsParams& P, int ci, int lane) {
    ec_partial(P, ci, lane);
    __syncwarp();
    unsigned* sync = P.ec_sync + 2 * P.calls[ci].ec_slot;
    unsigned old = 0;
    if (lane == 0) old = atom_add_acq_rel(sync, 1u);
    old = __shfl_sync(0xffffffffu, old, 0);
    if (old == gridDim.x - 1) ec_gate(P, ci, lane);
}
// Phase 0 (x comes from outside the launch): the worker warps add the z shares in the launch prologue (one arrive per CTA
// covers them and the x rewrite); the gate of call ci is then applied by the EC warp of CTA ci mod gridDim.x.
__device__ void ec_warp(const LsParams& P, int lane) {
    bool waited = false;
    for (int ci = P.phase_first_call[0]; ci < P.phase_first_call[1]; ++ci) {
        if (P.calls[ci].r == 0 || ci % int(gridDim.x) != int(blockIdx.x)) continue;
        if (!waited) { wait_counter(P.done + kLsMaxCalls + 1, gridDim.x); waited = true; }
        ec_gate(P, ci, lane);
    }
    for (int ph = 1; ph < P.n_phases; ++ph) {
        wait_counter(P.done + ph - 1, unsigned(P.phase_panels[ph - 1]));
        for (int ci = P.phase_first_call[ph]; ci < P.phase_first_call[ph + 1]; ++ci)
            if (P.calls[ci].r > 0) ec_call(P, ci, lane);
    }
}
}  // namespace ls

__global__ void __launch_bounds__(ls::kThreads, 1) ls_kernel(const __grid_constant__ LsParams P) {
    using namespace ls;
#ifdef LS_TRACE
    const unsigned long long t_entry = ls_now();
#endif
    extern __shared__ uint8_t smem_raw[];
    uint8_t* base = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* xring = base + Smem::x;
    uint8_t* wring = base + Smem::w;
    uint8_t* scring = base + Smem::sc;
    float* us = reinterpret_cast<float*>(base + Smem::u);
    float* part = reinterpret_cast<float*>(base + Smem::part);
    Bars* B = reinterpret_cast<Bars*>(base + Smem::bars);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int s = 0; s < kStages; ++s) { mbar_init(&B->full[s], 3); mbar_init(&B->empty[s], kEmptyCount); }
        for (int s = 0; s < kASlots; ++s) { mbar_init(&B->a_full[s], 4); mbar_init(&B->a_empty[s], 1); }
        for (int s = 0; s < kPipes; ++s) {
            for (int d = 0; d < 2; ++d) { mbar_init(&B->d_full[s][d], 1); mbar_init(&B->d_empty[s][d], 4); }
        }
        for (int d = 0; d < 2; ++d) { mbar_init(&B->seg_full[d], 4 * kPipes); mbar_init(&B->seg_empty[d], 4); }
        B->flag = 0;
        B->u_call = -1;
        fence_mbar_init();
    }
    if (warp == 3) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&B->tmem)), "n"(kTmemCols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = B->tmem;
#ifdef LS_TRACE
    unsigned long long* stamp = g_stamp;
    if (threadIdx.x == 0) stamp[39] = ls_now();
    __syncthreads();
#endif

    if (warp == 0) {
        if (lane == 0) producer(P, wring, B);
    } else if (warp == 1) {
        if (lane == 0) x_producer(P, xring, B);
    } else if (warp == 3) {
        if (lane == 0) sc_producer(P, scring, B);
    } else if (warp == 2) {
        ec_warp(P, lane);
    } else if (warp < 8) {
        finaliser(P, part, us, B, warp, lane);
    } else if (warp < 8 + 4 * kPipes) {
        // prologue: x -> operand layout (workspace), one arrive per CTA once its 16 worker warps are through
        x_prologue(P, threadIdx.x - 256, 128 * kPipes);
        for (int ci = P.phase_first_call[0] + (warp - 8); ci < P.phase_first_call[1]; ci += 4 * kPipes)
            if (P.calls[ci].r > 0) ec_partial(P, ci, lane);
        __threadfence();
        named_bar_sync(2, 128 * kPipes);
        if (threadIdx.x == 256) { asm volatile("fence.proxy.async;" ::: "memory"); red_add_release(P.done + kLsMaxCalls + 1, 1u); }
#ifdef LS_TRACE
        if (threadIdx.x == 256) g_stamp[45] = ls_now();
#endif
        worker(P, wring, scring, part, B, tmem, warp, lane);
    } else {
        if (lane == 0) mma_issuer(P, xring, B, tmem, warp - (8 + 4 * kPipes));
    }
#ifdef LS_TRACE
    if (lane == 0) stamp[warp] = ls_now();
#endif
    tc_fence_before();
    __syncthreads();
#ifdef LS_TRACE
    if (false && threadIdx.x == 0 && total_chunks(P) > 0 && (blockIdx.x % 37) == 36) {
        const unsigned long long t0 = stamp[39];
        printf("   prologue %llu xgo %llu first-full %llu | last seg: parts %llu slot %llu atom %llu sum %llu store %llu\n", stamp[45]-stamp[39], stamp[47]-stamp[39], stamp[46]-stamp[39], stamp[40]-stamp[39], stamp[41]-stamp[39], stamp[42]-stamp[39], stamp[43]-stamp[39], stamp[44]-stamp[39]);
        if (blockIdx.x == 36) for (int n = 0; n < min(32, total_chunks(P)); ++n)
            printf("  chunk %2d: mma-lane: arrive %llu dempty-ok %llu (after-dfull-commit %llu run-top %llu) | mma: afull %llu commit %llu | bulk %llu mma-complete %llu\n", n, g_ct[n][0]-t0, g_ct[n][1]-t0, g_ct[n][2]-t0, g_ct[n][3]-t0, g_ct[n][4]-t0, g_ct[n][5]-t0, g_ct[n][6]-t0, g_ct[n][7]-t0);
        printf("cta %d chunks %d: prod %llu xld %llu ec %llu epi %llu dq %llu %llu mma %llu %llu end %llu\n", blockIdx.x, total_chunks(P), stamp[0] - t0, stamp[1] - t0,
               stamp[2] - t0, stamp[4] - t0, stamp[8] - t0, stamp[23] - t0, stamp[24] - t0, stamp[27] - t0, ls_now() - t0);
    }
#endif
    if (warp == 3) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(kTmemCols) : "memory");
#ifdef LS_TRACE
    if (threadIdx.x == 0) printf("CTA %d entry %llu setup %llu exit %llu\n", blockIdx.x, t_entry, g_stamp[39], ls_now());
#endif
#if defined(LS_TRACE) || defined(LS_TIMER)
    if (threadIdx.x == 0) atomicMin(reinterpret_cast<unsigned long long*>(P.done + kLsMaxCalls + 2), t_entry);
#endif
    if (threadIdx.x == 0) {
        // the last CTA to leave resets what the next launch expects to be zero
        unsigned* exit_ctr = P.done + kLsMaxCalls;
        __threadfence();
        if (atom_add_acq_rel(exit_ctr, 1u) == gridDim.x - 1) {
            for (int ph = 0; ph < P.n_phases; ++ph) P.done[ph] = 0;
            for (int ci = 0; ci < P.n_calls; ++ci)
                if (P.calls[ci].ec_slot >= 0) P.ec_sync[2 * P.calls[ci].ec_slot + 1] = 0;
            exit_ctr[0] = 0;
            exit_ctr[1] = 0;
#if defined(LS_TRACE) || defined(LS_TIMER)
            unsigned long long* tmin = reinterpret_cast<unsigned long long*>(P.done + kLsMaxCalls + 2);
            printf("KERNEL %llu ns (first entry -> last exit), chunks/cta %d\n", ls_now() - *tmin, total_chunks(P));
            *tmin = ~0ull;
#endif
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

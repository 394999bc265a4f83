// tc.cu -- the tensor-core path for M > 16 tokens (mid-M and prefill): steps S1-S3, S7, S8 of
// SURVEY.md 8(a) in one persistent, warp-specialised tcgen05 kernel (Eq. 3):
//
//     y[m][n] = sum_k x[m][k] * What[n][k]  +  sum_j u[m][j] * B[n][j]        u = alpha * gamma (.) (A x)
//
// evaluated as ONE contraction over the concatenated reduction axis  Y^T = [What | B] . [X | U]^T :
// after the K/64 weight k-blocks the same main loop runs ceil(r/64) more k-blocks whose operands are
// B[n][:] and u16[m][:] (fp16, fetched by TMA, zero-filled beyond r).  The paper's prefill design
// runs the MARLIN GEMM and a separate EC kernel on two streams and joins them at the
// final accumulation; here the up-projection costs r/K extra MMA work and no extra pass over y.
//
// Orientation ("swap-AB"): the 128 output channels of a weight panel are the M = 128 rows of the
// UMMA, the tokens are its N (BT in {32, 64, 128, 256}).  The accumulator D[n][m] lives in TMEM
// (lane = output channel, column = token), two accumulators in flight so that the epilogue of tile i
// overlaps the main loop of tile i+1.
//
// Warp roles (736 threads for BT = 256, 992 for narrower token tiles; one CTA per SM, persistent over a static
// schedule of work items = output tile x split-K share):
//   warp 0      x producer: after griddepcontrol.wait, TMA tensor loads of the x tile (BT x 64 fp16,
//               SWIZZLE_128B; for the EC k-blocks the u16 tile), multicast to the CTAs of a cluster that share
//               the token tile.
//   last warp   int4 producer: cp.async.bulk of the packed int4 (4 KiB per (panel, 64-k tile)) + 256 B of
//               scales into a small ring; never waits for the previous kernel.  (One thread issuing both kinds
//               of copies was the bottleneck of the first version: 39 % -> 72 % tensor-pipe activity.)
//   warp 1      allocates TMEM; one elected lane issues tcgen05.mma (4 x K=16 per k-block) and commits
//               to the mbarriers that free the operand stages / publish the accumulator.
//   warps 2-5   epilogue: tcgen05.ld the accumulator, one RN-even cast to fp16, store y; with split-K: park
//               the fp32 partial, last arriver of the tile sums the partials in split order and stores.
//   warps 6-... dequantisation, 2 (BT = 256) or 3 groups of 8 warps taking k-blocks round-robin: LDS.128 of
//               int4 -> lop3 / sub / fma (exact q - 8) -> mul by the fp16 group scale (one rounding: the same
//               RN_fp16((q-8)*s) the dequant test hook exports) -> STS.128 into the K-major 128-byte-swizzled
//               A-operand stage, fence.proxy.async, arrive.  For an EC k-block one lane TMA-loads the B slab.
#include <algorithm>

#include <mutex>

#include "common.cuh"
#include "kernels.h"

namespace spear {

// ---- tcgen05 wrappers --------------------------------------------------------------------------
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
template <int kCols>
__device__ __forceinline__ void tmem_alloc(uint32_t* slot) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(slot)), "n"(kCols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
template <int kCols>
__device__ __forceinline__ void tmem_dealloc(uint32_t addr) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(addr), "n"(kCols) : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// D[tmem] (+)= A[smem] * B[smem]^T, fp16 inputs, fp32 accumulate, both operands K-major.
__device__ __forceinline__ void umma_f16(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}\n" ::"r"(d_tmem),
        "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// K-major operand tile, 128-byte swizzle: rows 128 B apart, 8-row atoms 1024 B apart (SBO), version 1.
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t smem_addr) {
    return uint64_t((smem_addr & 0x3ffff) >> 4) | (uint64_t(1) << 16) | (uint64_t(1024 >> 4) << 32) |
           (uint64_t(1) << 46) | (uint64_t(2) << 61);
}
// 32 lanes x 32 consecutive 32-bit columns -> 32 registers per thread (thread = lane, register = column)
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
          "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
          "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr)
        : "memory");
}
// cluster variants: the commit arrives on the barrier at the same offset in every CTA of `mask`; the TMA
// load writes the box into the same shared-memory offset of every CTA of `mask` and completes tx there.
__device__ __forceinline__ void umma_commit_mc(uint64_t* bar, uint16_t mask) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(smem_u32(bar)), "h"(mask) : "memory");
}
__device__ __forceinline__ void tma_load_2d_mc(void* dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar,
                                               uint16_t mask, uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.multicast::cluster.L2::cache_hint "
        "[%0], [%1, {%3, %4}], [%2], %5, %6;" ::"r"(smem_u32(dst)),
        "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "h"(mask), "l"(policy)
        : "memory");
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// ---- configuration -----------------------------------------------------------------------------
struct TcParams {
    const uint8_t* wq;       // SPW4 packed codes
    const uint8_t* scales;   // SPW4 packed scales
    __half* y;               // [M][N]
    int M, N, K, r;
    int G, group;            // K / group, group
    int kb_w;                // weight k-blocks (= pipeline stages of kKT x 64 columns)
    int kb_ec;               // EC k-blocks: ceil(r / (kKT x 64))
    int n_pp, n_mt;          // N / (128 * CS) panel groups (CS = cluster size), ceil(M / BT)
    int mt_group;            // token tiles per raster group (keeps the x slice L2-resident)
    int n_tiles;             // n_pp * n_mt output tiles; each is taken by one cluster (CTA rank c -> panel pp * CS + c)
    int ksplit;              // split-K factor: a (split) tile's weight k-blocks are shared by `ksplit` work items
    int n_whole;             // the first n_whole tiles are ONE work item each; the tiles behind them are split `ksplit` ways
                             // (0 with a uniform split; with a split tail: the tiles of the last, partial wave)
    int n_work;              // n_whole + (n_tiles - n_whole) * ksplit
    float* partial;          // [(n_tiles - n_whole) * CS][ksplit][BT][128] fp32, split-K partial sums (ksplit > 1)
    unsigned* counters;      // [n_tiles * CS], zero between calls
};

// One work item: output tile (panel group, token tile) and its share of the reduction axis.  The EC k-blocks
// belong to the last split.
struct TcWork {
    int panel, mt, ks, kb0, nw, ne;
    int tile, nsplit;        // output tile; number of work items that share it (1 = the item owns the tile)
};
__device__ __forceinline__ void tile_coords(const TcParams& p, int tile, int& panel, int& mt);
__device__ __forceinline__ TcWork get_work(const TcParams& p, int w) {
    TcWork t;
    if (w < p.n_whole) {
        t.tile = w; t.ks = 0; t.nsplit = 1;
    } else {
        const int idx = w - p.n_whole;
        t.tile = p.n_whole + idx / p.ksplit;
        t.ks = idx - (t.tile - p.n_whole) * p.ksplit;
        t.nsplit = p.ksplit;
    }
    tile_coords(p, t.tile, t.panel, t.mt);
    t.kb0 = int((long long)t.ks * p.kb_w / t.nsplit);
    t.nw = int((long long)(t.ks + 1) * p.kb_w / t.nsplit) - t.kb0;
    t.ne = (t.ks == t.nsplit - 1) ? p.kb_ec : 0;
    return t;
}

template <int BT>
struct TcCfg {
    // the x ring hides an L2 round trip per stage (deep); the A ring only the local dequantisation (shallow)
    // k-tiles (64 columns) per pipeline stage: a stage costs one barrier round trip (~0.45 us measured) whatever
    // its MMA time, so narrow token tiles (short MMAs) take 128 columns per stage
    static constexpr int kKT = BT == 256 ? 1 : 2;
    static constexpr int kXStages = BT == 256 ? 4 : (BT == 128 ? 3 : (BT == 64 ? 4 : 6));
    // dequantisation warp groups of 8 taking k-blocks round-robin: a k-block costs one barrier round trip
    // (~0.7 us) whatever its MMA time, so narrow token tiles (short MMAs) get three groups and a deeper A ring
    // The A ring must be deeper than the number of groups, or a group's next stage waits for the MMA of its previous
    // one (same slot) and nothing overlaps: 2 groups x 4 slots where shared memory allows (BT <= 64)
    static constexpr int kDequantGroups = BT == 128 ? 3 : 2;
    static constexpr int kThreads = (7 + 8 * kDequantGroups) * 32;   // + x producer, MMA, 4 epilogue, int4 producer
    static constexpr int kAStages = BT == 128 ? 3 : 4;
    static constexpr int kW4Stages = BT == 256 ? 6 : (BT == 128 ? 4 : (BT == 64 ? 4 : 6));     // ncu: with 4 the dequantisation warps spun on w4_full (HBM latency x 4 KiB per stage)
    static constexpr int kABytes = kKT * 128 * 128;      // kKT sub-tiles of 128 channels x 64 k fp16
    static constexpr int kXBytes = kKT * BT * 128;       // kKT sub-tiles of BT tokens x 64 k fp16
    static constexpr int kW4Bytes = kKT * 4096 + 256;    // codes of kKT (panel, 64-k tile)s + one scale block
    static constexpr int kTmemCols = 2 * BT < 32 ? 32 : 2 * BT;
    static constexpr size_t kSmemBytes = 1024 + size_t(kAStages) * kABytes + size_t(kXStages) * kXBytes + size_t(kW4Stages) * kW4Bytes + 512;
    static_assert(kSmemBytes <= 232448, "exceeds the 227 KiB opt-in shared memory of sm_100");
    static constexpr uint32_t kIdesc = (1u << 4) | (uint32_t(BT >> 3) << 17) | (uint32_t(128 >> 4) << 24);
};

__device__ __forceinline__ void tile_coords(const TcParams& p, int tile, int& panel, int& mt) {
    const int per_group = p.mt_group * p.n_pp;
    const int grp = tile / per_group;
    const int mt0 = grp * p.mt_group;
    const int width = min(p.mt_group, p.n_mt - mt0);
    const int rem = tile - grp * per_group;
    panel = rem / width;
    mt = mt0 + rem - panel * width;
}

template <int BT, int CS>
__global__ void __launch_bounds__(TcCfg<BT>::kThreads, 1)
tc_kernel(const __grid_constant__ CUtensorMap xmap, const __grid_constant__ CUtensorMap umap,
          const __grid_constant__ CUtensorMap bmap, const TcParams p) {
    using Cfg = TcCfg<BT>;
    constexpr int SX = Cfg::kXStages, SA = Cfg::kAStages, S4 = Cfg::kW4Stages, KT = Cfg::kKT;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* base = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* a_ring = base;                                   // S x 16 KiB, 1024-aligned
    uint8_t* x_ring = a_ring + size_t(SA) * Cfg::kABytes;     // SX x BT*128 B, 1024-aligned
    uint8_t* w4_ring = x_ring + size_t(SX) * Cfg::kXBytes;    // S4 x 4352 B
    uint64_t* bars = reinterpret_cast<uint64_t*>(w4_ring + size_t(S4) * Cfg::kW4Bytes);
    uint64_t* x_full = bars;              // [SX] producer TMA (tx bytes)
    uint64_t* x_empty = x_full + SX;      // [SX] tcgen05.commit (from every CTA of the cluster)
    uint64_t* a_full = x_empty + SX;      // [SA] 8 dequant-warp arrivals (+ tx bytes for EC k-blocks)
    uint64_t* a_empty = a_full + SA;      // [SA] tcgen05.commit
    uint64_t* w4_full = a_empty + SA;     // [S4] producer bulk copy (tx bytes)
    uint64_t* w4_empty = w4_full + S4;    // [S4] 8 dequant-warp arrivals
    uint64_t* acc_full = w4_empty + S4;   // [2]  tcgen05.commit
    uint64_t* acc_empty = acc_full + 2;   // [2]  4 epilogue-warp arrivals
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc_empty + 2);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // a cluster of CS CTAs shares every x tile: each CTA fetches BT / CS token rows and multicasts them
    const int cta_rank = CS > 1 ? int(cluster_ctarank()) : 0;
    const int work0 = blockIdx.x / CS, work_stride = gridDim.x / CS;
    constexpr uint16_t kMask = uint16_t((1u << CS) - 1);
    constexpr int kXRows = BT / CS;

    if (threadIdx.x == 0) {
        for (int s = 0; s < SX; ++s) { mbar_init(&x_full[s], 1); mbar_init(&x_empty[s], CS); }
        for (int s = 0; s < SA; ++s) { mbar_init(&a_full[s], 8); mbar_init(&a_empty[s], 1); }
        for (int s = 0; s < S4; ++s) { mbar_init(&w4_full[s], 1); mbar_init(&w4_empty[s], 8); }
        for (int s = 0; s < 2; ++s) { mbar_init(&acc_full[s], 1); mbar_init(&acc_empty[s], 4); }
        fence_mbar_init();
        tma_prefetch_desc(&xmap);
        if (p.kb_ec) { tma_prefetch_desc(&umap); tma_prefetch_desc(&bmap); }
    }
    if (warp == 1) tmem_alloc<Cfg::kTmemCols>(tmem_slot);
    tc_fence_before();
    __syncthreads();
    if (CS > 1) cluster_sync_all();      // peers' barriers are initialised before anything arrives on them
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    pdl_launch_dependents();

    if (warp == 0) {
        // ---------------------------------- x producer ----------------------------------
        if (lane == 0) {
            const uint64_t pol_x = policy_evict_last();
            pdl_wait();      // x / u16 may be written by the previous kernel in the stream
            int it = 0;
            for (int w = work0; w < p.n_work; w += work_stride) {
                const TcWork t = get_work(p, w);
                const int c1 = t.mt * BT + cta_rank * kXRows;
                for (int j = 0; j < t.nw + t.ne; ++j, ++it) {
                    const int s = it % SX;
                    mbar_wait(&x_empty[s], ((it / SX) & 1) ^ 1);
                    mbar_arrive_expect_tx(&x_full[s], Cfg::kXBytes);
                    const CUtensorMap* map = j < t.nw ? &xmap : &umap;
#pragma unroll
                    for (int kt = 0; kt < KT; ++kt) {
                        uint8_t* dst = x_ring + size_t(s) * Cfg::kXBytes + size_t(kt) * (BT * 128) + size_t(cta_rank) * kXRows * 128;
                        const int c0 = ((j < t.nw ? t.kb0 + j : j - t.nw) * KT + kt) * 64;
                        if (CS > 1) tma_load_2d_mc(dst, map, c0, c1, &x_full[s], kMask, pol_x);
                        else tma_load_2d(dst, map, c0, c1, &x_full[s], pol_x);
                    }
                }
            }
        }
    } else if (warp == Cfg::kThreads / 32 - 1) {
        // ---------------------------------- int4 producer ----------------------------------
        // weights never depend on the previous kernel: no griddepcontrol.wait on this path
        if (lane == 0) {
            const uint64_t pol_w = policy_evict_first(), pol_s = policy_evict_last();
            int w_it = 0;
            for (int w = work0; w < p.n_work; w += work_stride) {
                const TcWork t = get_work(p, w);
                const int panel = t.panel * CS + cta_rank;
                const uint8_t* wsrc = p.wq + size_t(panel) * p.kb_w * (KT * 4096);
                const uint8_t* ssrc = p.scales + size_t(panel) * p.G * 256;
                for (int kb = t.kb0; kb < t.kb0 + t.nw; ++kb, ++w_it) {
                    const int s4 = w_it % S4;
                    mbar_wait(&w4_empty[s4], ((w_it / S4) & 1) ^ 1);
                    mbar_arrive_expect_tx(&w4_full[s4], Cfg::kW4Bytes);
                    uint8_t* dst = w4_ring + size_t(s4) * Cfg::kW4Bytes;
                    bulk_g2s(dst, wsrc + size_t(kb) * (KT * 4096), KT * 4096, &w4_full[s4], pol_w);
                    bulk_g2s(dst + KT * 4096, ssrc + size_t((kb * 64 * KT) / p.group) * 256, 256, &w4_full[s4], pol_s);
                }
            }
        }
    } else if (warp == 1) {
        // ---------------------------------- MMA issuer ----------------------------------
        int it = 0, tcount = 0;
        for (int w = work0; w < p.n_work; w += work_stride, ++tcount) {
            const TcWork t = get_work(p, w);
            const int kb_total = t.nw + t.ne;
            const int acc = tcount & 1;
            mbar_wait(&acc_empty[acc], ((tcount >> 1) & 1) ^ 1);
            tc_fence_after();
            const uint32_t d_tmem = tmem_base + uint32_t(acc * BT);
            for (int kb = 0; kb < kb_total; ++kb, ++it) {
                const int s = it % SX, sa = it % SA;
                mbar_wait(&x_full[s], (it / SX) & 1);
                mbar_wait(&a_full[sa], (it / SA) & 1);
                tc_fence_after();
                if (elect_one()) {
                    const uint64_t a_desc = umma_desc_sw128(smem_u32(a_ring + size_t(sa) * Cfg::kABytes));
                    const uint64_t b_desc = umma_desc_sw128(smem_u32(x_ring + size_t(s) * Cfg::kXBytes));
#pragma unroll
                    for (int kt = 0; kt < KT; ++kt)
#pragma unroll
                        for (int k = 0; k < 4; ++k)   // K = 16 per instruction: +32 bytes inside the swizzle atom
                            umma_f16(d_tmem, a_desc + uint64_t(kt * (16384 >> 4) + k * 2),
                                     b_desc + uint64_t(kt * ((BT * 128) >> 4) + k * 2), Cfg::kIdesc, (kb | kt | k) != 0);
                    if (CS > 1) umma_commit_mc(&x_empty[s], kMask);
                    else umma_commit(&x_empty[s]);
                    umma_commit(&a_empty[sa]);
                    if (kb == kb_total - 1) umma_commit(&acc_full[acc]);
                }
                __syncwarp();
            }
        }
    } else if (warp < 6) {
        // ---------------------------------- epilogue ----------------------------------
        const int q = warp & 3;                 // TMEM lane quarter this warp may access
        int tcount = 0;
        for (int w = work0; w < p.n_work; w += work_stride, ++tcount) {
            const TcWork t = get_work(p, w);
            const int panel = t.panel * CS + cta_rank;
            const int acc = tcount & 1;
            mbar_wait(&acc_full[acc], (tcount >> 1) & 1);
            tc_fence_after();
            const int nl = q * 32 + lane;
            const int n = panel * 128 + nl;
            const int m0 = t.mt * BT;
            __half* yp = p.y + size_t(m0) * p.N + n;
            if (t.nsplit == 1) {
#pragma unroll 1
                for (int c = 0; c < BT; c += 32) {
                    if (m0 + c >= p.M) break;       // warp-uniform: nothing left in this tile
                    uint32_t v[32];
                    tmem_ld32(tmem_base + (uint32_t(q * 32) << 16) + uint32_t(acc * BT + c), v);
                    tmem_ld_wait();
#pragma unroll
                    for (int i = 0; i < 32; ++i)
                        if (m0 + c + i < p.M) yp[size_t(c + i) * p.N] = __float2half_rn(__uint_as_float(v[i]));
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&acc_empty[acc]);
            } else {
                // split-K: park the fp32 partial, the last of the tile's `ksplit` work items to arrive sums them
                // in split order, casts once and stores y (same pattern as the decode kernel's panels)
                const int out_id = t.tile * CS + cta_rank;                          // counter of this (tile, rank)
                float* slots = p.partial + size_t((t.tile - p.n_whole) * CS + cta_rank) * p.ksplit * (BT * 128);
                float* mine = slots + size_t(t.ks) * (BT * 128);
#pragma unroll 1
                for (int c = 0; c < BT; c += 32) {
                    if (m0 + c >= p.M) break;
                    uint32_t v[32];
                    tmem_ld32(tmem_base + (uint32_t(q * 32) << 16) + uint32_t(acc * BT + c), v);
                    tmem_ld_wait();
#pragma unroll
                    for (int i = 0; i < 32; ++i)
                        if (m0 + c + i < p.M) mine[(c + i) * 128 + nl] = __uint_as_float(v[i]);
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&acc_empty[acc]);     // the accumulator is drained
                __threadfence();
                named_bar_sync(3, 128);
                if (warp == 2 && lane == 0) {
                    const unsigned old = atomicAdd(p.counters + out_id, 1u);
                    const unsigned last = (old == unsigned(p.ksplit - 1));
                    if (last) p.counters[out_id] = 0;           // self-cleaning
                    tmem_slot[1] = last;
                }
                named_bar_sync(3, 128);
                if (tmem_slot[1]) {
                    __threadfence();
                    const int rows = min(BT, p.M - m0);
                    // 16 token rows per pass: every load of a pass is issued before the first add, so that 16 L2 round trips
                    // overlap (with 4 the sum of a 128-token tile took ~10 us per share and made a 2-way split a loss)
                    constexpr int kRows = 16;
                    for (int mm = 0; mm < rows; mm += kRows) {
                        float sum[kRows];
#pragma unroll
                        for (int u = 0; u < kRows; ++u) sum[u] = 0.f;
                        for (int ks = 0; ks < p.ksplit; ++ks) {
                            const float* sk = slots + size_t(ks) * (BT * 128) + nl;
                            float v[kRows];
#pragma unroll
                            for (int u = 0; u < kRows; ++u) v[u] = (mm + u < rows) ? __ldcg(sk + (mm + u) * 128) : 0.f;
#pragma unroll
                            for (int u = 0; u < kRows; ++u) sum[u] += v[u];
                        }
#pragma unroll
                        for (int u = 0; u < kRows; ++u)
                            if (mm + u < rows) yp[size_t(mm + u) * p.N] = __float2half_rn(sum[u]);
                    }
                }
                named_bar_sync(3, 128);      // tmem_slot[1] is reused by the next work item
            }
        }
    } else {
        // ---------------------------------- dequantisation ----------------------------------
        const int strip = (warp - 6) & 7;       // 16 output channels of the panel
        const int dgroup = (warp - 6) >> 3;     // this warp converts the k-blocks with it % Cfg::kDequantGroups == dgroup
        const int g = lane >> 2, t = lane & 3;
        int it = 0, w_it = 0;
        for (int w = work0; w < p.n_work; w += work_stride) {
            const TcWork tw = get_work(p, w);
            const int panel = tw.panel * CS + cta_rank;
            for (int kb = 0; kb < tw.nw + tw.ne; ++kb, ++it) {
                const int s = it % SA;
                uint8_t* a_stage = a_ring + size_t(s) * Cfg::kABytes;
                if (it % Cfg::kDequantGroups != dgroup) {
                    if (kb < tw.nw) ++w_it;
                    continue;
                }
                mbar_wait(&a_empty[s], ((it / SA) & 1) ^ 1);
                if (kb < tw.nw) {
                    const int s4 = w_it % S4;
                    mbar_wait(&w4_full[s4], (w_it / S4) & 1);
                    ++w_it;
                    const uint8_t* src = w4_ring + size_t(s4) * Cfg::kW4Bytes;
                    const uint32_t scw = *reinterpret_cast<const uint32_t*>(src + KT * 4096 + (strip * 16 + 2 * g) * 2);
                    const uint32_t s_lo = __byte_perm(scw, scw, 0x1010), s_hi = __byte_perm(scw, scw, 0x3232);
#pragma unroll
                    for (int kt = 0; kt < KT; ++kt) {
                        const uint4 w = *reinterpret_cast<const uint4*>(src + kt * 4096 + (strip * 32 + lane) * 16);
                        uint32_t c0[4], c1[4], c2[4], c3[4];
                        dequant_word(w.x, c0);      // row g,     columns 16t + 0..7   -> 16-byte chunk 2t
                        dequant_word(w.y, c1);      // row g,     columns 16t + 8..15  -> chunk 2t + 1
                        dequant_word(w.z, c2);      // row g + 8, columns 16t + 0..7
                        dequant_word(w.w, c3);      // row g + 8, columns 16t + 8..15
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            c0[i] = hmul2_u32(c0[i], s_lo); c1[i] = hmul2_u32(c1[i], s_lo);
                            c2[i] = hmul2_u32(c2[i], s_hi); c3[i] = hmul2_u32(c3[i], s_hi);
                        }
                        // K-major SWIZZLE_128B: row n at n * 128, 16-byte chunk c at position c ^ (n & 7); (n & 7) == g
                        uint8_t* r0 = a_stage + kt * 16384 + (strip * 16 + g) * 128;
                        uint8_t* r1 = r0 + 8 * 128;
                        *reinterpret_cast<uint4*>(r0 + (((2 * t) ^ g) << 4)) = make_uint4(c0[0], c0[1], c0[2], c0[3]);
                        *reinterpret_cast<uint4*>(r0 + (((2 * t + 1) ^ g) << 4)) = make_uint4(c1[0], c1[1], c1[2], c1[3]);
                        *reinterpret_cast<uint4*>(r1 + (((2 * t) ^ g) << 4)) = make_uint4(c2[0], c2[1], c2[2], c2[3]);
                        *reinterpret_cast<uint4*>(r1 + (((2 * t + 1) ^ g) << 4)) = make_uint4(c3[0], c3[1], c3[2], c3[3]);
                    }
                    fence_proxy_async_smem();   // generic-proxy writes -> visible to the tensor core's async proxy
                    __syncwarp();
                    if (lane == 0) { mbar_arrive(&w4_empty[s4]); mbar_arrive(&a_full[s]); }
                } else {
                    // EC k-block: the A operand is a 128 x 64 slab of B[N][r], fetched by TMA (zero beyond r)
                    if (lane == 0) {
                        if (strip == 0) {
                            mbar_arrive_expect_tx(&a_full[s], Cfg::kABytes);
#pragma unroll
                            for (int kt = 0; kt < KT; ++kt)
                                tma_load_2d(a_stage + kt * 16384, &bmap, ((kb - tw.nw) * KT + kt) * 64, panel * 128,
                                            &a_full[s], policy_evict_last());
                        } else {
                            mbar_arrive(&a_full[s]);
                        }
                    }
                }
            }
        }
    }

    tc_fence_before();
    __syncthreads();
    if (CS > 1) cluster_sync_all();      // no CTA leaves while a peer may still multicast into it or arrive on its barriers
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc<Cfg::kTmemCols>(tmem_base);
    }
}

// ---- host side -----------------------------------------------------------------------------------

template <int BT, int CS>
static int launch_tc(const CUtensorMap& xmap, const CUtensorMap& umap, const CUtensorMap& bmap, const TcParams& p,
                     int grid_override, bool pdl, cudaStream_t st) {
    static std::mutex init_mutex;    // first-call query, guarded: concurrent host threads may launch the same instance
    static int max_clusters = 0;     // co-resident clusters of CS CTAs (one CTA per SM)
    std::unique_lock<std::mutex> init_lock(init_mutex);
    if (!max_clusters) {
        SPEAR_CUDA_OK(cudaFuncSetAttribute(tc_kernel<BT, CS>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           int(TcCfg<BT>::kSmemBytes)));
        int n = device_info().num_sms / CS;
        if (CS > 1) {
            cudaLaunchConfig_t q = {};
            q.gridDim = dim3(device_info().num_sms / CS * CS);
            q.blockDim = dim3(TcCfg<BT>::kThreads);
            q.dynamicSmemBytes = TcCfg<BT>::kSmemBytes;
            cudaLaunchAttribute qa[1];
            qa[0].id = cudaLaunchAttributeClusterDimension;
            qa[0].val.clusterDim.x = CS; qa[0].val.clusterDim.y = 1; qa[0].val.clusterDim.z = 1;
            q.attrs = qa; q.numAttrs = 1;
            int nc = 0;
            SPEAR_CUDA_OK(cudaOccupancyMaxActiveClusters(&nc, tc_kernel<BT, CS>, &q));
            if (nc < 1) return set_error(SPEAR_ECUDA, "tc_kernel<%d,%d>: no co-resident cluster fits", BT, CS);
            n = std::min(n, nc);
        }
        max_clusters = n;
    }
    init_lock.unlock();
    int clusters = std::min(p.n_work, max_clusters);
    if (grid_override > 0) clusters = std::min(clusters, std::max(1, grid_override / CS));
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(clusters * CS);
    cfg.blockDim = dim3(TcCfg<BT>::kThreads);
    cfg.dynamicSmemBytes = TcCfg<BT>::kSmemBytes;
    cfg.stream = st;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
    attr[1].id = cudaLaunchAttributeClusterDimension;
    attr[1].val.clusterDim.x = CS; attr[1].val.clusterDim.y = 1; attr[1].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = CS > 1 ? 2 : 1;
    SPEAR_CUDA_OK(cudaLaunchKernelEx(&cfg, tc_kernel<BT, CS>, xmap, umap, bmap, p));
    count_launch();
    return SPEAR_OK;
}

int run_tc(const TcProblem& t, cudaStream_t st) {
    int BT = t.M <= 32 ? 32 : (t.M <= 64 ? 64 : (t.M <= 128 ? 128 : 256));
    const int n_panels = t.N / 128;
    // few, wide tiles leave SMs idle and pay one barrier round trip per 64 columns: with too few 256-token tiles
    // to fill the machine, 128-token tiles (two k-tiles per stage, twice the CTAs) are faster (measured at M = 256)
    if (BT == 256 && t.M <= 512 && n_panels * ((t.M + 255) / 256) < device_info().num_sms) BT = 128;
    if (t.bt_override == 32 || t.bt_override == 64 || t.bt_override == 128 || t.bt_override == 256)
        if (t.bt_override >= 32 && (t.bt_override >= t.M || t.bt_override >= 128)) BT = t.bt_override;
    const int n_mt = (t.M + BT - 1) / BT;
    // clusters share x tiles by TMA multicast; worth it once there are more tiles than SMs (L2 -> SM bound)
    int CS = 1;
    if (BT == 256 && n_panels * n_mt >= 2 * device_info().num_sms && n_panels % 2 == 0) CS = 2;   // measured: 2 > 1 > 4
    if (t.cluster_override > 0 && BT == 256 && n_panels % t.cluster_override == 0) CS = t.cluster_override;
    TcParams p = {};
    p.wq = static_cast<const uint8_t*>(t.wq);
    p.scales = static_cast<const uint8_t*>(t.scales);
    p.y = static_cast<__half*>(t.y);
    p.M = t.M; p.N = t.N; p.K = t.K; p.r = t.r;
    p.group = t.group; p.G = t.K / t.group;
    const int KT = BT == 256 ? 1 : 2;        // TcCfg<BT>::kKT: 64-column k-tiles per pipeline stage
    p.kb_w = t.K / (64 * KT);               // from here on a "k-block" is one stage
    p.kb_ec = (t.r + 64 * KT - 1) / (64 * KT);
    p.n_pp = n_panels / CS;
    p.n_mt = n_mt;
    // raster: token tiles in groups whose x slice (mt_group * BT * K * 2 bytes, <= 16 MiB) stays L2-resident next to the weights in flight
    const size_t slice = size_t(BT) * t.K * 2;
    p.mt_group = int(std::max<size_t>(1, std::min<size_t>(size_t(p.n_mt), (size_t(t.xslice_mb > 0 ? t.xslice_mb : 16) << 20) / slice)));   // measured: 8-16 MiB > 32-96 MiB
    p.n_tiles = p.n_pp * p.n_mt;
    // split-K when there are fewer output tiles than SMs (mid-M on small layers): work items = tiles x ksplit
    int ks = 1;
    if (CS == 1 && p.n_tiles < device_info().num_sms) {
        // A share saves K-loop time (one ~0.45 us barrier round trip per stage) and pays for parking and re-reading fp32 partials
        // (~0.035 us per token row of the tile and per share, measured): take the factor that minimises the sum.  E.g. 128 tokens,
        // 4096 -> 6144: no split (23.4 us; 2-way 25.2); 64 tokens, 8192 -> 2048: 4-way (20.7 us; none 33.7, 2-way 24.6).
        const int ks_max = std::min(std::min(device_info().num_sms / p.n_tiles, p.kb_w), 16);
        double best_t = 0.45 * p.kb_w;
        for (int c = 2; c <= ks_max; ++c) {
            const double tc_us = 0.45 * p.kb_w / c + 0.035 * BT * c;
            if (tc_us < best_t) { best_t = tc_us; ks = c; }
        }
        while (ks > 1 && size_t(p.n_tiles) * ks * BT * 128 * 4 > t.partial_bytes) --ks;
        if (p.n_tiles > t.max_counters || !t.partial || !t.counters) ks = 1;
    }
    if (t.ksplit_override > 0) ks = std::max(1, std::min(t.ksplit_override, p.kb_w));
    if (ks > 1 && CS > 1) ks = 1;       // a uniform split is for problems with fewer tiles than SMs; clusters are for many tiles
    p.n_whole = 0;
    // Partial last wave (e.g. 224 cluster-tiles on 74 clusters = 3.03 waves: the 4th round keeps 2 clusters busy and 72 idle):
    // the tiles of that round are split along K over the idle clusters, `ks` ways each, so the round lasts 1 / ks of a tile.
    // Only when the tail is small (<= half a wave) and a share keeps >= 32 k-tiles (a split must pay for its reduction).
    if (ks == 1 && t.tail_split != 0 && t.partial && t.counters) {
        const int slots = std::max(1, device_info().num_sms / CS);
        const int rem = p.n_tiles % slots;
        // ... and only for a few waves: with many (M >= 2048 on the big layers) the CTAs drift apart, the "last wave" is no longer a
        // wave, and the split costs 5-9 % (measured: M = 4096 config 4 1237 -> 1121 TFLOP/s; M = 512 1031 -> 1079, M = 1024 1168 -> 1179)
        if (p.n_tiles > slots && (p.n_tiles <= 8 * slots || t.tail_split == 2) && rem > 0 && 2 * rem <= slots) {
            int kt = std::min(std::min(slots / rem, std::max(1, p.kb_w * KT / 32)), 16);
            while (kt > 1 && size_t(rem) * CS * kt * BT * 128 * 4 > t.partial_bytes) --kt;
            if (kt > 1 && p.n_tiles * CS <= t.max_counters) {
                ks = kt;
                p.n_whole = p.n_tiles - rem;
            }
        }
    }
    if (ks > 1 && (size_t(p.n_tiles - p.n_whole) * CS * ks * BT * 128 * 4 > t.partial_bytes || p.n_tiles * CS > t.max_counters))
        return set_error(SPEAR_ENOMEM, "tc split-K %d needs more workspace", ks);
    p.ksplit = ks;
    p.n_work = p.n_whole + (p.n_tiles - p.n_whole) * ks;
    p.partial = static_cast<float*>(t.partial);
    p.counters = t.counters;
    CUtensorMap xmap, umap, bmap;
    if (int rc = get_tensor_map_2d(t.x, uint64_t(t.M), uint64_t(t.K), uint64_t(t.K) * 2, uint32_t(BT / CS), 64, &xmap)) return rc;
    if (t.r > 0) {
        if (int rc = get_tensor_map_2d(t.u16, uint64_t(t.M), uint64_t(t.r), uint64_t(t.r) * 2, uint32_t(BT / CS), 64, &umap)) return rc;
        if (int rc = get_tensor_map_2d(t.B, uint64_t(t.N), uint64_t(t.r), uint64_t(t.r) * 2, 128, 64, &bmap)) return rc;
    } else {
        umap = xmap; bmap = xmap;
    }
    switch (BT) {
        case 32: return launch_tc<32, 1>(xmap, umap, bmap, p, t.grid_override, t.pdl, st);
        case 64: return launch_tc<64, 1>(xmap, umap, bmap, p, t.grid_override, t.pdl, st);
        case 128: return launch_tc<128, 1>(xmap, umap, bmap, p, t.grid_override, t.pdl, st);
        default:
            if (CS == 4) return launch_tc<256, 4>(xmap, umap, bmap, p, t.grid_override, t.pdl, st);
            if (CS == 2) return launch_tc<256, 2>(xmap, umap, bmap, p, t.grid_override, t.pdl, st);
            return launch_tc<256, 1>(xmap, umap, bmap, p, t.grid_override, t.pdl, st);
    }
}

}  // namespace spear

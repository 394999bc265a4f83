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
// Warp roles (448 threads, one CTA per SM, persistent over a static tile schedule):
//   warp 0      producer: cp.async.bulk of the packed int4 (4 KiB per (panel, 64-k tile)) + 256 B of
//               scales into a small ring; TMA tensor loads of the x tile (BT x 64 fp16, SWIZZLE_128B).
//               int4 copies never wait for the previous kernel; x / u16 loads come after griddepcontrol.wait.
//   warp 1      allocates TMEM; one elected lane issues tcgen05.mma (4 x K=16 per k-block) and commits
//               to the mbarriers that free the operand stages / publish the accumulator.
//   warps 2-5   epilogue: tcgen05.ld the accumulator, one RN-even cast to fp16, store y.
//   warps 6-13  dequantisation: LDS.128 of int4 -> lop3 / sub / fma (exact q - 8) -> mul by the fp16
//               group scale (one rounding: the same RN_fp16((q-8)*s) the dequant test hook exports)
//               -> STS.128 into the K-major 128-byte-swizzled A-operand stage, fence.proxy.async, arrive.
#include <algorithm>

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
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// ---- configuration -----------------------------------------------------------------------------
struct TcParams {
    const uint8_t* wq;       // SPW4 packed codes
    const uint8_t* scales;   // SPW4 packed scales
    __half* y;               // [M][N]
    int M, N, K, r;
    int G, group;            // K / group, group
    int kb_w;                // K / 64 weight k-blocks
    int kb_ec;               // ceil(r / 64) EC k-blocks
    int n_panels, n_mt;      // N / 128, ceil(M / BT)
    int mt_group;            // token tiles per raster group (keeps the x slice L2-resident)
    int n_tiles;
};

template <int BT>
struct TcCfg {
    static constexpr int kStages = BT == 256 ? 4 : (BT == 128 ? 5 : (BT == 64 ? 6 : 8));
    static constexpr int kW4Stages = BT == 256 ? 6 : 8;
    static constexpr int kABytes = 128 * 128;            // 128 channels x 64 k fp16
    static constexpr int kXBytes = BT * 128;             // BT tokens x 64 k fp16
    static constexpr int kW4Bytes = 4096 + 256;          // codes + scales of one (panel, 64-k tile)
    static constexpr int kTmemCols = 2 * BT < 32 ? 32 : 2 * BT;
    static constexpr size_t kSmemBytes = 1024 + size_t(kStages) * (kABytes + kXBytes) + size_t(kW4Stages) * kW4Bytes + 512;
    static_assert(kSmemBytes <= 232448, "exceeds the 227 KiB opt-in shared memory of sm_100");
    static constexpr uint32_t kIdesc = (1u << 4) | (uint32_t(BT >> 3) << 17) | (uint32_t(128 >> 4) << 24);
};
constexpr int kTcThreads = 448;

__device__ __forceinline__ void tile_coords(const TcParams& p, int tile, int& panel, int& mt) {
    const int per_group = p.mt_group * p.n_panels;
    const int grp = tile / per_group;
    const int mt0 = grp * p.mt_group;
    const int width = min(p.mt_group, p.n_mt - mt0);
    const int rem = tile - grp * per_group;
    panel = rem / width;
    mt = mt0 + rem - panel * width;
}

template <int BT>
__global__ void __launch_bounds__(kTcThreads, 1)
tc_kernel(const __grid_constant__ CUtensorMap xmap, const __grid_constant__ CUtensorMap umap,
          const __grid_constant__ CUtensorMap bmap, const TcParams p) {
    using Cfg = TcCfg<BT>;
    constexpr int S = Cfg::kStages, S4 = Cfg::kW4Stages;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* base = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* a_ring = base;                                   // S x 16 KiB, 1024-aligned
    uint8_t* x_ring = a_ring + size_t(S) * Cfg::kABytes;      // S x BT*128 B, 1024-aligned
    uint8_t* w4_ring = x_ring + size_t(S) * Cfg::kXBytes;     // S4 x 4352 B
    uint64_t* bars = reinterpret_cast<uint64_t*>(w4_ring + size_t(S4) * Cfg::kW4Bytes);
    uint64_t* x_full = bars;              // [S]  producer TMA (tx bytes)
    uint64_t* a_full = x_full + S;        // [S]  8 dequant-warp arrivals (+ tx bytes for EC k-blocks)
    uint64_t* xa_empty = a_full + S;      // [S]  tcgen05.commit
    uint64_t* w4_full = xa_empty + S;     // [S4] producer bulk copy (tx bytes)
    uint64_t* w4_empty = w4_full + S4;    // [S4] 8 dequant-warp arrivals
    uint64_t* acc_full = w4_empty + S4;   // [2]  tcgen05.commit
    uint64_t* acc_empty = acc_full + 2;   // [2]  4 epilogue-warp arrivals
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc_empty + 2);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int kb_total = p.kb_w + p.kb_ec;

    if (threadIdx.x == 0) {
        for (int s = 0; s < S; ++s) { mbar_init(&x_full[s], 1); mbar_init(&a_full[s], 8); mbar_init(&xa_empty[s], 1); }
        for (int s = 0; s < S4; ++s) { mbar_init(&w4_full[s], 1); mbar_init(&w4_empty[s], 8); }
        for (int s = 0; s < 2; ++s) { mbar_init(&acc_full[s], 1); mbar_init(&acc_empty[s], 4); }
        fence_mbar_init();
        tma_prefetch_desc(&xmap);
        if (p.kb_ec) { tma_prefetch_desc(&umap); tma_prefetch_desc(&bmap); }
    }
    if (warp == 1) tmem_alloc<Cfg::kTmemCols>(tmem_slot);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    pdl_launch_dependents();

    if (warp == 0) {
        // ---------------------------------- producer ----------------------------------
        if (lane == 0) {
            const uint64_t pol_w = policy_evict_first(), pol_x = policy_evict_last();
            // the two rings advance independently: int4 copies run ahead of the x loads by up to S4 k-blocks
            int w_tile = blockIdx.x, w_kb = 0, w_it = 0;          // next int4 copy to issue
            auto issue_w4 = [&]() {
                int panel, mt;
                tile_coords(p, w_tile, panel, mt);
                const int s4 = w_it % S4;
                mbar_wait(&w4_empty[s4], ((w_it / S4) & 1) ^ 1);
                mbar_arrive_expect_tx(&w4_full[s4], Cfg::kW4Bytes);
                uint8_t* dst = w4_ring + size_t(s4) * Cfg::kW4Bytes;
                bulk_g2s(dst, p.wq + (size_t(panel) * p.kb_w + w_kb) * 4096, 4096, &w4_full[s4], pol_w);
                bulk_g2s(dst + 4096, p.scales + (size_t(panel) * p.G + (w_kb * 64) / p.group) * 256, 256, &w4_full[s4], pol_x);
                ++w_it;
                if (++w_kb == p.kb_w) { w_kb = 0; w_tile += gridDim.x; }
            };
            // prologue: fill the int4 ring before waiting for the previous kernel (weights never depend on it)
            for (int i = 0; i < S4 && w_tile < p.n_tiles; ++i) issue_w4();
            pdl_wait();
            int it = 0;
            for (int tile = blockIdx.x; tile < p.n_tiles; tile += gridDim.x) {
                int panel, mt;
                tile_coords(p, tile, panel, mt);
                for (int kb = 0; kb < kb_total; ++kb, ++it) {
                    const int s = it % S;
                    mbar_wait(&xa_empty[s], ((it / S) & 1) ^ 1);
                    mbar_arrive_expect_tx(&x_full[s], Cfg::kXBytes);
                    if (kb < p.kb_w) tma_load_2d(x_ring + size_t(s) * Cfg::kXBytes, &xmap, kb * 64, mt * BT, &x_full[s], pol_x);
                    else tma_load_2d(x_ring + size_t(s) * Cfg::kXBytes, &umap, (kb - p.kb_w) * 64, mt * BT, &x_full[s], pol_x);
                    if (w_tile < p.n_tiles) {
                        // keep the int4 ring topped up without blocking on it
                        const int s4 = w_it % S4;
                        if (mbar_try_wait(&w4_empty[s4], ((w_it / S4) & 1) ^ 1)) issue_w4();
                    }
                }
            }
            // int4 copies the loop above did not get to (cannot happen unless kb_ec == 0 and try_wait lagged)
            while (w_tile < p.n_tiles) issue_w4();
        }
    } else if (warp == 1) {
        // ---------------------------------- MMA issuer ----------------------------------
        int it = 0, tcount = 0;
        for (int tile = blockIdx.x; tile < p.n_tiles; tile += gridDim.x, ++tcount) {
            const int acc = tcount & 1;
            mbar_wait(&acc_empty[acc], ((tcount >> 1) & 1) ^ 1);
            tc_fence_after();
            const uint32_t d_tmem = tmem_base + uint32_t(acc * BT);
            for (int kb = 0; kb < kb_total; ++kb, ++it) {
                const int s = it % S;
                const uint32_t ph = (it / S) & 1;
                mbar_wait(&x_full[s], ph);
                mbar_wait(&a_full[s], ph);
                tc_fence_after();
                if (elect_one()) {
                    const uint64_t a_desc = umma_desc_sw128(smem_u32(a_ring + size_t(s) * Cfg::kABytes));
                    const uint64_t b_desc = umma_desc_sw128(smem_u32(x_ring + size_t(s) * Cfg::kXBytes));
#pragma unroll
                    for (int k = 0; k < 4; ++k)   // K = 16 per instruction: +32 bytes inside the swizzle atom
                        umma_f16(d_tmem, a_desc + uint64_t(k * 2), b_desc + uint64_t(k * 2), Cfg::kIdesc, (kb | k) != 0);
                    umma_commit(&xa_empty[s]);
                    if (kb == kb_total - 1) umma_commit(&acc_full[acc]);
                }
                __syncwarp();
            }
        }
    } else if (warp < 6) {
        // ---------------------------------- epilogue ----------------------------------
        const int q = warp & 3;                 // TMEM lane quarter this warp may access
        int tcount = 0;
        for (int tile = blockIdx.x; tile < p.n_tiles; tile += gridDim.x, ++tcount) {
            int panel, mt;
            tile_coords(p, tile, panel, mt);
            const int acc = tcount & 1;
            mbar_wait(&acc_full[acc], (tcount >> 1) & 1);
            tc_fence_after();
            const int n = panel * 128 + q * 32 + lane;
            const int m0 = mt * BT;
            __half* yp = p.y + size_t(m0) * p.N + n;
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
        }
    } else {
        // ---------------------------------- dequantisation ----------------------------------
        const int strip = warp - 6;             // 16 output channels of the panel
        const int g = lane >> 2, t = lane & 3;
        int it = 0, w_it = 0;
        for (int tile = blockIdx.x; tile < p.n_tiles; tile += gridDim.x) {
            int panel, mt;
            tile_coords(p, tile, panel, mt);
            for (int kb = 0; kb < kb_total; ++kb, ++it) {
                const int s = it % S;
                uint8_t* a_stage = a_ring + size_t(s) * Cfg::kABytes;
                mbar_wait(&xa_empty[s], ((it / S) & 1) ^ 1);
                if (kb < p.kb_w) {
                    const int s4 = w_it % S4;
                    mbar_wait(&w4_full[s4], (w_it / S4) & 1);
                    ++w_it;
                    const uint8_t* src = w4_ring + size_t(s4) * Cfg::kW4Bytes;
                    const uint4 w = *reinterpret_cast<const uint4*>(src + (strip * 32 + lane) * 16);
                    const uint32_t scw = *reinterpret_cast<const uint32_t*>(src + 4096 + (strip * 16 + 2 * g) * 2);
                    const uint32_t s_lo = __byte_perm(scw, scw, 0x1010), s_hi = __byte_perm(scw, scw, 0x3232);
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
                    uint8_t* r0 = a_stage + (strip * 16 + g) * 128;
                    uint8_t* r1 = r0 + 8 * 128;
                    *reinterpret_cast<uint4*>(r0 + (((2 * t) ^ g) << 4)) = make_uint4(c0[0], c0[1], c0[2], c0[3]);
                    *reinterpret_cast<uint4*>(r0 + (((2 * t + 1) ^ g) << 4)) = make_uint4(c1[0], c1[1], c1[2], c1[3]);
                    *reinterpret_cast<uint4*>(r1 + (((2 * t) ^ g) << 4)) = make_uint4(c2[0], c2[1], c2[2], c2[3]);
                    *reinterpret_cast<uint4*>(r1 + (((2 * t + 1) ^ g) << 4)) = make_uint4(c3[0], c3[1], c3[2], c3[3]);
                    fence_proxy_async_smem();   // generic-proxy writes -> visible to the tensor core's async proxy
                    __syncwarp();
                    if (lane == 0) { mbar_arrive(&w4_empty[s4]); mbar_arrive(&a_full[s]); }
                } else {
                    // EC k-block: the A operand is a 128 x 64 slab of B[N][r], fetched by TMA (zero beyond r)
                    if (lane == 0) {
                        if (strip == 0) {
                            mbar_arrive_expect_tx(&a_full[s], Cfg::kABytes);
                            tma_load_2d(a_stage, &bmap, (kb - p.kb_w) * 64, panel * 128, &a_full[s], policy_evict_last());
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
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc<Cfg::kTmemCols>(tmem_base);
    }
}

// ---- host side -----------------------------------------------------------------------------------
bool tc_available() { return true; }

template <int BT>
static int launch_tc(const CUtensorMap& xmap, const CUtensorMap& umap, const CUtensorMap& bmap, const TcParams& p,
                     int grid, bool pdl, cudaStream_t st) {
    static bool attr_set = false;
    if (!attr_set) {
        SPEAR_CUDA_OK(cudaFuncSetAttribute(tc_kernel<BT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           int(TcCfg<BT>::kSmemBytes)));
        attr_set = true;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(kTcThreads);
    cfg.dynamicSmemBytes = TcCfg<BT>::kSmemBytes;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    SPEAR_CUDA_OK(cudaLaunchKernelEx(&cfg, tc_kernel<BT>, xmap, umap, bmap, p));
    count_launch();
    return SPEAR_OK;
}

int run_tc(const TcProblem& t, cudaStream_t st) {
    const int BT = t.M <= 32 ? 32 : (t.M <= 64 ? 64 : (t.M <= 128 ? 128 : 256));
    TcParams p = {};
    p.wq = static_cast<const uint8_t*>(t.wq);
    p.scales = static_cast<const uint8_t*>(t.scales);
    p.y = static_cast<__half*>(t.y);
    p.M = t.M; p.N = t.N; p.K = t.K; p.r = t.r;
    p.group = t.group; p.G = t.K / t.group;
    p.kb_w = t.K / 64;
    p.kb_ec = (t.r + 63) / 64;
    p.n_panels = t.N / 128;
    p.n_mt = (t.M + BT - 1) / BT;
    // raster: token tiles in groups whose x slice (mt_group * BT * K * 2 bytes) stays L2-resident
    const size_t slice = size_t(BT) * t.K * 2;
    p.mt_group = int(std::max<size_t>(1, std::min<size_t>(size_t(p.n_mt), (size_t(48) << 20) / slice)));
    p.n_tiles = p.n_panels * p.n_mt;
    CUtensorMap xmap, umap, bmap;
    if (int rc = get_tensor_map_2d(t.x, uint64_t(t.M), uint64_t(t.K), uint64_t(t.K) * 2, uint32_t(BT), 64, &xmap)) return rc;
    if (t.r > 0) {
        if (int rc = get_tensor_map_2d(t.u16, uint64_t(t.M), uint64_t(t.r), uint64_t(t.r) * 2, uint32_t(BT), 64, &umap)) return rc;
        if (int rc = get_tensor_map_2d(t.B, uint64_t(t.N), uint64_t(t.r), uint64_t(t.r) * 2, 128, 64, &bmap)) return rc;
    } else {
        umap = xmap; bmap = xmap;
    }
    int grid = std::min(p.n_tiles, device_info().num_sms);
    if (t.grid_override > 0) grid = std::min(p.n_tiles, t.grid_override);
    switch (BT) {
        case 32: return launch_tc<32>(xmap, umap, bmap, p, grid, t.pdl, st);
        case 64: return launch_tc<64>(xmap, umap, bmap, p, grid, t.pdl, st);
        case 128: return launch_tc<128>(xmap, umap, bmap, p, grid, t.pdl, st);
        default: return launch_tc<256>(xmap, umap, bmap, p, grid, t.pdl, st);
    }
}

}  // namespace spear

// stream.cu -- the weight-streaming kernel for small token counts (decode, M <= 16).
//
// Computes steps S1-S3, S7, S8 of SURVEY.md 8(a) in one launch (Eq. 3):
//     y[m][n] = sum_k x[m][k] * (q[n][k] - 8) * s[n][k/group]  +  sum_j u[m][j] * B[n][j]
// where u = alpha * gamma (.) (A x) was produced by the EC pre-kernel (ec_pre.cu) and r == 0 is the
// plain W4 layer.  The paper's decode kernel runs the EC chain in a MARLIN epilogue on
// Hopper; here the layer is HBM-bound, so the design is a TMA-fed shared-memory ring:
//
//   * work unit = (panel of 128 output rows, chunk of 128 input columns) = 8 KiB of packed int4,
//     contiguous in the SPW4 layout; units are numbered panel-major and split evenly (stream-K)
//     over gridDim.x CTAs, so every SM streams the same number of bytes whatever the shape;
//   * warp 0 is the producer: one lane issues cp.async.bulk (weights, scales) and a swizzled TMA
//     tensor copy (the x tile, zero-filled beyond M) per unit into a kStages-deep ring guarded by
//     full/empty mbarriers.  Weight copies are issued BEFORE griddepcontrol.wait (they never depend
//     on the previous kernel), x copies after it: under programmatic dependent launch the ring of
//     layer i+1 fills while layer i drains;
//   * 8 consumer warps: each task is (4 strips of 16 rows) x (64 columns): 4 LDS.128 of int4,
//     lop3/hsub2 dequantisation in registers, mma.sync.m16n8k16 with the tokens as the n=8 operand
//     (fp32 accumulate), group scale applied to the fp32 accumulator;
//   * per panel segment the 8 warps reduce through shared memory; a CTA that owns a whole panel
//     writes y directly, otherwise it parks an fp32 partial in the workspace and the last arriver
//     (atomic counter per panel) sums the partials in CTA order, adds the EC term and casts once.
#include "common.cuh"
#include "kernels.h"

namespace spear {

template <int MT>
struct StreamCfg {
    static constexpr int kStages = (MT == 1) ? 8 : 6;
    static constexpr int kXTile = MT * 1024;          // bytes: 8*MT token rows x 128 B
    static constexpr int kRedStride = 68;             // floats; 68 makes the fragment stores conflict-free
    static constexpr int kTok = 8 * MT;
    static constexpr size_t kXBytes = size_t(kStages) * 2 * kXTile;
    static constexpr size_t kWBytes = size_t(kStages) * 8192;
    static constexpr size_t kScBytes = size_t(kStages) * 256;
    static constexpr size_t kRedBytes = size_t(8) * kTok * kRedStride * 4;
    static constexpr size_t kBarBytes = size_t(kStages) * 16 + 32;
    static constexpr size_t kSmemBytes = 1024 + kXBytes + kWBytes + kScBytes + kRedBytes + kBarBytes;
};

__device__ __forceinline__ int cta_of_unit(int u, int per, int rem) {
    const int big = rem * (per + 1);
    return (u < big) ? u / (per + 1) : rem + (u - big) / per;
}

template <int MT>
__device__ __forceinline__ void stream_task(const uint8_t* __restrict__ wst, const uint8_t* __restrict__ xst,
                                            const uint8_t* __restrict__ scst, int h, int ktl, int lane,
                                            float (&tot)[4][MT][4]) {
    const int g = lane >> 2, t = lane & 3;
    uint32_t xa[MT][4], xb[MT][4];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) {
        const uint8_t* row = xst + ktl * (MT * 1024) + (mt * 8 + g) * 128;
        const uint4 va = *reinterpret_cast<const uint4*>(row + (((2 * t) ^ g) << 4));
        const uint4 vb = *reinterpret_cast<const uint4*>(row + (((2 * t + 1) ^ g) << 4));
        xa[mt][0] = va.x; xa[mt][1] = va.y; xa[mt][2] = va.z; xa[mt][3] = va.w;
        xb[mt][0] = vb.x; xb[mt][1] = vb.y; xb[mt][2] = vb.z; xb[mt][3] = vb.w;
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int strip = 4 * h + j;
        const uint4 w = *reinterpret_cast<const uint4*>(wst + ((ktl * 8 + strip) * 32 + lane) * 16);
        const uint32_t scw = *reinterpret_cast<const uint32_t*>(scst + (strip * 16 + 2 * g) * 2);
        const float s_lo = __half2float(__ushort_as_half(uint16_t(scw & 0xffff)));
        const float s_hi = __half2float(__ushort_as_half(uint16_t(scw >> 16)));
        uint32_t a0[4], a1[4], a2[4], a3[4];
        dequant_word(w.x, a0);   // row g,   columns 16t + 0..7
        dequant_word(w.z, a1);   // row g+8, columns 16t + 0..7
        dequant_word(w.y, a2);   // row g,   columns 16t + 8..15
        dequant_word(w.w, a3);   // row g+8, columns 16t + 8..15
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) {
            float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int jj = 0; jj < 4; ++jj)
                mma_m16n8k16(acc, a0[jj], a1[jj], a2[jj], a3[jj], xa[mt][jj], xb[mt][jj]);
            tot[j][mt][0] = fmaf(s_lo, acc[0], tot[j][mt][0]);
            tot[j][mt][1] = fmaf(s_lo, acc[1], tot[j][mt][1]);
            tot[j][mt][2] = fmaf(s_hi, acc[2], tot[j][mt][2]);
            tot[j][mt][3] = fmaf(s_hi, acc[3], tot[j][mt][3]);
        }
    }
}

// ---- fused EC (warp 9): S4-S6 of SURVEY.md 8(a) inside the weight-stream kernel ---------------------
// Every CTA reduces one (16-row strip of [A; w_g]) x (K slice) piece of z = x [A; w_g]^T with mma.sync,
// adds it to the global fp32 z with red.add and ARRIVES on a device-wide counter right away; nobody
// waits there.  The last CTA to arrive applies the gate (z must be complete before
// the gate), writes u = alpha * gamma (.) z, re-zeroes z and raises a flag; the other
// CTAs only look at the flag in their epilogue, long after everybody has arrived (arrive early / wait
// late).  All CTAs of the grid are co-resident (grid <= SMs x occupancy), so the wait cannot deadlock.
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

__device__ void ec_warp_fused(const StreamParams& p, int lane, uint64_t* u_ready) {
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
    bool waited = false;
    for (int task = blockIdx.x; task < n_tasks; task += G) {
        const int strip = task % strips, ks = task / strips;
        const int rho0 = strip * 16 + g, rho1 = rho0 + 8;
        const __half* pa0 = rho0 < p.r ? p.A + size_t(rho0) * p.K : (rho0 == p.r && scalar ? p.w_g : nullptr);
        const __half* pa1 = rho1 < p.r ? p.A + size_t(rho1) * p.K : (rho1 == p.r && scalar ? p.w_g : nullptr);
        const int kt_begin = int((long long)ks * ktiles / ksplit);
        const int kt_end = int((long long)(ks + 1) * ktiles / ksplit);
        float acc0[4] = {0.f, 0.f, 0.f, 0.f}, acc1[4] = {0.f, 0.f, 0.f, 0.f};
        for (int kt = kt_begin; kt < kt_end; ++kt) {
            const int col = kt * 64 + 16 * t;
            uint32_t a0l[4], a0h[4], a1l[4], a1h[4], x0l[4], x0h[4], x1l[4], x1h[4];
            ec_load16(pa0, col, true, a0l, a0h);     // EC factors are parameters: never written by a kernel
            ec_load16(pa1, col, true, a1l, a1h);
            if (!waited) { pdl_wait(); waited = true; }   // x may come from the previous kernel
            ec_load16(px0, col, false, x0l, x0h);
            ec_load16(px1, col, false, x1l, x1h);
#pragma unroll
            for (int jj = 0; jj < 4; ++jj) {
                mma_m16n8k16(acc0, a0l[jj], a1l[jj], a0h[jj], a1h[jj], x0l[jj], x0h[jj]);
                mma_m16n8k16(acc1, a0l[jj], a1l[jj], a0h[jj], a1h[jj], x1l[jj], x1h[jj]);
            }
        }
        // C fragment: rows rho0 / rho1 of [A; w_g], tokens 2t, 2t+1 (acc0) and 8+2t, 9+2t (acc1)
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int rho = (i & 2) ? rho1 : rho0;
            const int tok = 2 * t + (i & 1);
            if (rho < rows_total) {
                if (tok < p.M) atomicAdd(p.zbuf + tok * kZStride + rho, acc0[i]);
                if (tok + 8 < p.M) atomicAdd(p.zbuf + (tok + 8) * kZStride + rho, acc1[i]);
            }
        }
    }
    if (!waited) pdl_wait();
    __threadfence();
    __syncwarp();
    unsigned old = 0;
    if (lane == 0) old = atomicAdd(p.ec_sync + 0, 1u);
    old = __shfl_sync(0xffffffffu, old, 0);
    if (old == unsigned(G - 1)) {
        // ---- last arriver: gate, u, clean-up ----
        __threadfence();
        const float bias = (scalar && p.b_g) ? *p.b_g : 0.f;
        const int n = p.M * p.r;
        for (int idx = lane; idx < n; idx += 32) {
            const int m = idx / p.r, j = idx - m * p.r;
            const float z = __ldcg(p.zbuf + m * kZStride + j);
            float gam = 1.f;
            if (scalar) gam = 1.f / (1.f + expf(-(__ldcg(p.zbuf + m * kZStride + p.r) + bias)));
            p.u_out[idx] = p.alpha * gam * z;
            if (scalar && p.gate_out && j == 0) p.gate_out[m] = gam;
        }
        __syncwarp();
        for (int idx = lane; idx < p.M * rows_total; idx += 32) {
            const int m = idx / rows_total, rho = idx - m * rows_total;
            p.zbuf[m * kZStride + rho] = 0.f;
        }
        __threadfence();
        __syncwarp();
        if (lane == 0) {
            p.ec_sync[0] = 0;
            if (G > 1) {
                __threadfence();
                asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p.ec_sync + 1), "r"(1u) : "memory");
            }
        }
    } else if (lane == 0) {
        unsigned f = 0;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(f) : "l"(p.ec_sync + 1) : "memory");
        } while (f == 0);
        const unsigned readers = atomicAdd(p.ec_sync + 2, 1u);
        if (readers == unsigned(G - 2)) {      // every waiting CTA has seen the flag: leave the workspace clean
            p.ec_sync[2] = 0;
            p.ec_sync[1] = 0;
        }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(u_ready);
}

template <int MT>
__global__ void __launch_bounds__(320, 2)
stream_kernel(const __grid_constant__ CUtensorMap xmap, const StreamParams p) {
    using Cfg = StreamCfg<MT>;
    constexpr int S = Cfg::kStages;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* base = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* xring = base;
    uint8_t* wring = xring + Cfg::kXBytes;
    uint8_t* scring = wring + Cfg::kWBytes;
    float* red = reinterpret_cast<float*>(scring + Cfg::kScBytes);
    uint64_t* full = reinterpret_cast<uint64_t*>(reinterpret_cast<uint8_t*>(red) + Cfg::kRedBytes);
    uint64_t* empty = full + S;
    int* flag = reinterpret_cast<int*>(empty + S);
    uint64_t* u_ready = reinterpret_cast<uint64_t*>(flag + 2);   // fused EC: u is in global memory, visible

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int G = gridDim.x, b = blockIdx.x;
    const int per = p.U / G, rem = p.U % G;
    const int u0 = b * per + min(b, rem);
    const int n_units = per + (b < rem ? 1 : 0);
    const int C = p.C;

    if (threadIdx.x == 0) {
        for (int s = 0; s < S; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 4); }
        mbar_init(u_ready, 1);
        fence_mbar_init();
        tma_prefetch_desc(&xmap);
    }
    __syncthreads();
    pdl_launch_dependents();
    if (warp == 9) {
        if (p.fused && p.r > 0) ec_warp_fused(p, lane, u_ready);
        return;
    }
    if (n_units == 0) return;

    if (warp == 0) {
        // ------------------------------ producer ------------------------------
        if (lane == 0) {
            const uint64_t pol_w = policy_evict_first(), pol_x = policy_evict_last();
            const uint8_t* wq = reinterpret_cast<const uint8_t*>(p.wq);
            const uint8_t* sc = reinterpret_cast<const uint8_t*>(p.scales);
            const int nfirst = min(n_units, S);
            for (int it = 0; it < nfirst; ++it) {
                const int u = u0 + it, pnl = u / C, c = u - pnl * C;
                mbar_expect_tx(&full[it], 8192 + 256);
                bulk_g2s(wring + it * 8192, wq + (size_t(pnl) * C + c) * 8192, 8192, &full[it], pol_w);
                bulk_g2s(scring + it * 256, sc + (size_t(pnl) * p.G + c / p.group_chunks) * 256, 256,
                         &full[it], pol_x);
            }
            pdl_wait();   // x may be written by the previous kernel in the stream
            for (int it = 0; it < nfirst; ++it) {
                const int c = (u0 + it) % C;
                mbar_arrive_expect_tx(&full[it], 2 * Cfg::kXTile);
                tma_load_2d(xring + (it * 2 + 0) * Cfg::kXTile, &xmap, c * 128, 0, &full[it], pol_x);
                tma_load_2d(xring + (it * 2 + 1) * Cfg::kXTile, &xmap, c * 128 + 64, 0, &full[it], pol_x);
            }
            for (int it = S; it < n_units; ++it) {
                const int s = it % S;
                const int u = u0 + it, pnl = u / C, c = u - pnl * C;
                mbar_wait(&empty[s], ((it / S) & 1) ^ 1);
                mbar_arrive_expect_tx(&full[s], 8192 + 256 + 2 * Cfg::kXTile);
                bulk_g2s(wring + s * 8192, wq + (size_t(pnl) * C + c) * 8192, 8192, &full[s], pol_w);
                bulk_g2s(scring + s * 256, sc + (size_t(pnl) * p.G + c / p.group_chunks) * 256, 256,
                         &full[s], pol_x);
                tma_load_2d(xring + (s * 2 + 0) * Cfg::kXTile, &xmap, c * 128, 0, &full[s], pol_x);
                tma_load_2d(xring + (s * 2 + 1) * Cfg::kXTile, &xmap, c * 128 + 64, 0, &full[s], pol_x);
            }
        } else if (p.r > 0) {
            // warm L2 with the B rows of every panel this CTA may finalise (read only in the epilogue)
            const int p_first = u0 / C, p_last = (u0 + n_units - 1) / C;
            const uint8_t* Bb = reinterpret_cast<const uint8_t*>(p.B);
            const size_t slab = size_t(128) * p.r * 2;
            for (int pnl = p_first; pnl <= p_last; ++pnl)
                for (size_t off = size_t(lane - 1) * 128; off < slab; off += 31 * 128)
                    prefetch_l2(Bb + size_t(pnl) * slab + off);
        }
        return;
    }

    // -------------------------------- consumers --------------------------------
    const int cw = warp - 1;
    const int h = cw & 1, ktl = (cw >> 1) & 1, par = cw >> 2;
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

    int it = 0;
    while (it < n_units) {
        const int pnl = (u0 + it) / C;
        const int seg_begin = it;
        const int seg_end = min(n_units, (pnl + 1) * C - u0);
        for (int i = seg_begin + ((par ^ seg_begin) & 1); i < seg_end; i += 2) {
            const int s = i % S;
            mbar_wait(&full[s], (i / S) & 1);
            stream_task<MT>(wring + s * 8192, xring + s * 2 * Cfg::kXTile, scring + s * 256, h, ktl, lane, tot);
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[s]);
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
        const bool whole = ((u0 + seg_begin) % C == 0) && (seg_end - seg_begin == C);
        bool finalize = whole;
        int c_first = b, c_last = b;
        if (!whole) {
            const int which = ((u0 / C) == pnl) ? 0 : 1;
            float* slot = p.partial + size_t(b * 2 + which) * Cfg::kTok * 128;
#pragma unroll
            for (int i = 0; i < 4 * MT; ++i) slot[((ct >> 7) + 2 * i) * 128 + row] = val[i];
            __threadfence();
            named_bar_sync(2, 256);
            c_first = cta_of_unit(pnl * C, per, rem);
            c_last = cta_of_unit(pnl * C + C - 1, per, rem);
            if (ct == 0) {
                const unsigned old = atomicAdd(p.counters + pnl, 1u);
                const int last = (old == unsigned(c_last - c_first));
                if (last) p.counters[pnl] = 0;      // self-cleaning: the next call finds zero
                *flag = last;
            }
            named_bar_sync(2, 256);
            finalize = (*flag != 0);
            if (finalize) {
                __threadfence();
#pragma unroll
                for (int i = 0; i < 4 * MT; ++i) val[i] = 0.f;
                for (int cj = c_first; cj <= c_last; ++cj) {
                    const int uj = cj * per + min(cj, rem);
                    const int wj = ((uj / C) == pnl) ? 0 : 1;
                    const float* sj = p.partial + size_t(cj * 2 + wj) * Cfg::kTok * 128;
#pragma unroll
                    for (int i = 0; i < 4 * MT; ++i) val[i] += __ldcg(sj + ((ct >> 7) + 2 * i) * 128 + row);
                }
            }
        }
        if (finalize) {
            const int n = pnl * 128 + row;
            if (p.r > 0) {
                // S7: y += sum_j u[m][j] * B[n][j]   (u = alpha * gamma (.) z, fp32, from the pre-kernel or warp 9)
                if (p.fused) mbar_wait(u_ready, 0);
                const uint4* Brow = reinterpret_cast<const uint4*>(p.B + size_t(n) * p.r);
                for (int j8 = 0; j8 < p.r / 8; ++j8) {
                    const uint4 bv = __ldg(Brow + j8);
                    const __half2* bh = reinterpret_cast<const __half2*>(&bv);
                    float bf[8];
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const float2 f = __half22float2(bh[q]);
                        bf[2 * q] = f.x; bf[2 * q + 1] = f.y;
                    }
#pragma unroll
                    for (int i = 0; i < 4 * MT; ++i) {
                        const int tok = (ct >> 7) + 2 * i;
                        if (tok < p.M) {
                            const float4* up = reinterpret_cast<const float4*>(p.u + size_t(tok) * p.r + j8 * 8);
                            const float4 ua = __ldcg(up), ub = __ldcg(up + 1);
                            val[i] += ua.x * bf[0] + ua.y * bf[1] + ua.z * bf[2] + ua.w * bf[3] +
                                      ub.x * bf[4] + ub.y * bf[5] + ub.z * bf[6] + ub.w * bf[7];
                        }
                    }
                }
            }
            // S8: one RN-even cast, coalesced store of 128 consecutive n per token
#pragma unroll
            for (int i = 0; i < 4 * MT; ++i) {
                const int tok = (ct >> 7) + 2 * i;
                if (tok < p.M) p.y[size_t(tok) * p.N + n] = __float2half_rn(val[i]);
            }
        }
        named_bar_sync(1, 256);     // red[] and flag are reused by the next segment
        it = seg_end;
    }
}

int stream_smem_bytes(int MT) {
    return int(MT == 1 ? StreamCfg<1>::kSmemBytes : StreamCfg<2>::kSmemBytes);
}

int launch_stream(const CUtensorMap& xmap, const StreamParams& p, int MT, int grid, bool pdl,
                  cudaStream_t st) {
    static bool attr_set = false;
    if (!attr_set) {
        SPEAR_CUDA_OK(cudaFuncSetAttribute(stream_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           int(StreamCfg<1>::kSmemBytes)));
        SPEAR_CUDA_OK(cudaFuncSetAttribute(stream_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           int(StreamCfg<2>::kSmemBytes)));
        attr_set = true;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(320);
    cfg.dynamicSmemBytes = stream_smem_bytes(MT);
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (MT == 1) SPEAR_CUDA_OK(cudaLaunchKernelEx(&cfg, stream_kernel<1>, xmap, p));
    else SPEAR_CUDA_OK(cudaLaunchKernelEx(&cfg, stream_kernel<2>, xmap, p));
    count_launch();
    return SPEAR_OK;
}

}  // namespace spear

// rows.cu -- the row-strip kernel for small token counts (decode, M <= 16) on layers whose time is launch / latency
// bound rather than bandwidth bound (SPEAR_VARIANT_ROWS).
//
// Same arithmetic as stream.cu (Eq. 3; steps S1-S3, S7, S8 of SURVEY.md 8(a)):
//     y[m][n] = sum_k x[m][k] * (q[n][k] - 8) * s[n][k/group]  +  sum_j u[m][j] * B[n][j]
// but partitioned the other way round.  stream.cu cuts the layer along K (stream-K over 16 KiB units) and pays a
// cross-CTA reduction through L2 -- partial, fence, counter, reload: four dependent round trips, 2.5 us on a 2 MB layer
// whose HBM time is 0.3 us.  Here one CTA owns ONE 16-row strip of the output over the WHOLE of K, so no CTA ever talks
// to another:
//
//   * grid = N / 16 CTAs of 8 warps; warp w takes the 64-column k-tiles w, w + 8, ... of its strip.  In the SPW4
//     layout a (strip, k-tile) piece is 512 contiguous bytes = one LDG.128 per lane, already in mma.sync A-fragment
//     order, so the weights go global -> registers with no shared-memory stage; four k-tiles per warp are in flight and
//     the next four are requested before the current four are consumed.  The first requests are issued BEFORE
//     griddepcontrol.wait (weights and scales do not depend on the previous kernel);
//   * x needs no staging either: lane (g, t) of a k-tile wants 16 consecutive columns of token row g (two LDG.128, L2
//     hits -- x is at most 16 x K fp16 and every CTA reads all of it);
//   * int4 -> fp16 exactly (q - 8, dequant_word), mma.sync.m16n8k16 with the tokens as n = 8 (two n-tiles for M > 8),
//     fp32 accumulate per k-tile, group scale applied in fp32 to the k-tile's sum (the products stay exact);
//   * the 8 warps meet once in shared memory; thread (row, token) sums them, adds the EC term u[m][:] . B[n][:] (u from
//     the EC pre-kernel, staged in shared memory; the strip's 16 x r slab of B was fetched before the wait) and stores
//     y with one RN-even cast.
//
// Fused EC (scalar / none gate; FUSED instance, launched as clusters of 8 CTAs = one 128-row panel): z = x [A; w_g]^T
// has to be COMPLETE before the gate, and a device-wide reduction costs three more round trips
// through L2 (red.add, fence + counter, reload) -- as long as the whole layer.  So every cluster computes z for itself:
// CTA c of the cluster takes the c-th eighth of K (all r + 1 rows, mma.sync, A fetched before the wait), the eight
// partial z meet through distributed shared memory (each CTA stores its part into slot c of every peer, then
// barrier.cluster arrive; the matching wait sits AFTER the main loop, so the exchange hides behind the weight stream), and
// each CTA sums the eight slots in rank order (deterministic), applies the gate and forms u.  No global counter, no
// workspace, no co-residency requirement beyond the cluster's own.  Price: A is read once per cluster (L2 hits after
// the first), N / 128 times in all.
//
// Measured and NOT kept (round 2): a persistent form (2 CTAs per SM walking strips, first with a one-batch register look-ahead across
// strips, then with lane-private cp.async rings of 12 k-tile slots = 96 KiB in flight per SM).  gate_up 2048 -> 16384 went 9.05 ->
// 9.2 -> 8.4 us (the ring kernel: 7.4), small layers got 0.1-0.6 us slower.  Bytes in flight are therefore not what bounds this
// kernel on big layers; the L1 wavefronts of the x fragment loads (8 lines per LDG.128, twice per k-tile, four times at M > 8)
// and the legacy mma.sync rate (~3.9 clk per m16n8k16 per SM) are.
//
// Default EC arm since the end of round 2 ("rows_ec" 2): the pre-kernel (ecz_cluster_kernel<MT, true>) is 8 independent CTAs, CTA c
// reduces the c-th eighth of K and parks its partial z [8 MT][r + 1] in the workspace; the plain layer kernel, which started under PDL
// while they ran, sums the eight parts in rank order and applies the gate when it stages u -- those loads share the round trip of
// its x loads.  No cluster, no DSMEM, no barrier: 5.8 us against 6.4 (one-cluster arm) on o at M = 8.
//
// Also measured and not kept: the EC cluster INSIDE the layer kernel's grid (8 extra CTAs compute z once and raise a flag; the strips
// poll it after their main loop, with a bounded wait and a compute-it-yourself fallback so that progress never rests on dispatch
// order).  One launch instead of two, but slower than the one-cluster pre-kernel: qkv 7.0 / 7.4 / 8.6 us against 5.8 / 6.4 / 8.5 --
// fence + flag + poll + reload of u is a longer chain than the PDL hand-over between two kernels.
//
// What it costs: x is re-read by every CTA (L2 traffic 2 M / 16 times the weight bytes) and a strip of a K = 8192 layer
// is 64 KiB through one CTA -- fine while the layer is small, wrong for the big ones, which stay with stream.cu
// (api.cu: heuristic_variant / spear_plan decide).
#include <mutex>

#include "common.cuh"
#include "kernels.h"

namespace spear {

namespace {

// asynchronous global -> shared copies (LDGSTS): the issuing thread does not wait for the data
__device__ __forceinline__ void cp_async8(void* dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async4(void* dst, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

__device__ __forceinline__ uint4 ldg128_stream(const void* p) {     // weights: read once, keep them out of L1
    uint4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    return v;
}

template <int MT, bool FUSED>
__global__ void __launch_bounds__(256, 2) rows_kernel(const RowsParams p) {
    constexpr int kTok = 8 * MT;
    constexpr int kRowsNB = MT == 1 ? 4 : 2;      // k-tiles per warp in flight (current) + as many requested ahead; the x fragments of a batch cost 8 MT registers per k-tile
    constexpr int kSG = 2;                        // FUSED: 16-row strips of [A; w_g] per z item (one item = kSG strips x one k-tile)
    extern __shared__ float zslots[];             // FUSED: [8 ranks][kTok][r + 1] partial z, written by the peers (+ [kTok][r + 1] of the sum)
    __shared__ float red[8][16][kTok + 1];
    __shared__ __align__(16) float us[16 * 128];          // u [kTok][r] fp32 (r > 0)
    __shared__ __align__(16) uint8_t bs[16 * (128 * 2 + 16)];    // the strip's rows of B, [16][r] fp16 or int8, rows padded by 16 bytes
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane >> 2, t = lane & 3;
    const int strip = blockIdx.x;                          // 16 output rows
    const int pnl = strip >> 3, sp = strip & 7;
    const int KT = p.K >> 6;                               // 64-column k-tiles
    const int C = p.K >> 7;

    // this lane's 16 bytes of (k-tile kt): chunk kt / 2, half kt & 1
    const uint8_t* wbase = reinterpret_cast<const uint8_t*>(p.wq) + size_t(pnl) * C * 8192 + (sp * 32 + lane) * 16;
    auto w_ptr = [&](int kt) { return wbase + size_t(kt >> 1) * 8192 + (kt & 1) * 4096; };
    // this lane's scale word (rows g, g + 8 of the strip) of the group that holds k-tile kt
    const uint8_t* sbase = reinterpret_cast<const uint8_t*>(p.scales) + size_t(pnl) * p.G * 256 + (sp * 16 + 2 * g) * 2;
    const int kt_per_group = p.group >> 6;
    auto s_ptr = [&](int kt) { return sbase + size_t(kt / kt_per_group) * 256; };

    uint4 wv[kRowsNB], wn[kRowsNB];          // current / next batch of this warp's k-tiles
    uint32_t sc[kRowsNB], sn[kRowsNB];
    auto load_w = [&](uint4 (&wd)[kRowsNB], uint32_t (&sd)[kRowsNB], int base) {
#pragma unroll
        for (int b = 0; b < kRowsNB; ++b) {
            const int kt = base + 8 * b;
            if (kt < KT) {
                wd[b] = ldg128_stream(w_ptr(kt));
                sd[b] = __ldg(reinterpret_cast<const uint32_t*>(s_ptr(kt)));
            }
        }
    };
    load_w(wv, sc, warp);
    const int esz = p.ec_int8 ? 1 : 2;
    const int brow = p.r * esz + 16;                       // padded row of bs[]: 16 rows hit distinct banks
    if (p.r > 0) {      // the strip's slab of B (a parameter: requested before the wait, awaited before the epilogue)
        const int per_row = p.r * esz / 8;                 // 8-byte pieces per row (r is a multiple of 8)
        const uint8_t* Bs = reinterpret_cast<const uint8_t*>(p.B) + size_t(strip) * 16 * p.r * esz;
        for (int i = threadIdx.x; i < 16 * per_row; i += 256) {
            const int rw = i / per_row, pc = i - rw * per_row;
            cp_async8(bs + rw * brow + pc * 8, Bs + (size_t(rw) * per_row + pc) * 8);
        }
    }

    // ---- FUSED, S4: this CTA's eighth of K of z = x [A; w_g]^T, for the whole cluster.  Item = (k-tile, kSG strips). ----
    const bool scalar = FUSED && (p.gate_kind == SPEAR_GATE_SCALAR_SIGMOID);
    const int zr = p.r + 1;                                    // row r = the scalar gate's pre-activation (unused otherwise)
    const int strips = (p.r + (scalar ? 1 : 0) + 15) >> 4;
    const int sgroups = (strips + kSG - 1) / kSG;
    const uint32_t rank = FUSED ? cluster_ctarank() : 0u;
    const int kt0 = int(rank) * KT / 8, kt1 = (int(rank) + 1) * KT / 8;
    const int n_items = (kt1 - kt0) * sgroups;
    float* zmine = zslots + 8 * kTok * zr;                     // this CTA's partial, then the cluster's sum
    uint32_t al[kSG][2][4], ah[kSG][2][4];                     // [strip of the item][row g / g + 8][4 k16 steps]: columns 16t.. / 16t + 8..
    float sa[kSG][2];
    auto load_A = [&](int item) {
        const int kt = kt0 + item / sgroups, s0 = (item % sgroups) * kSG;
        const int col = kt * 64 + 16 * t;
        const int8_t* A8 = reinterpret_cast<const int8_t*>(p.A);
#pragma unroll
        for (int s = 0; s < kSG; ++s)
#pragma unroll
            for (int hrow = 0; hrow < 2; ++hrow) {
                const int rho = (s0 + s) * 16 + g + 8 * hrow;
                const bool q = p.ec_int8 && rho < p.r;                 // the gate row w_g stays fp16
                const __half* pa = rho < p.r ? p.A + size_t(rho) * p.K : (rho == p.r && scalar ? p.w_g : nullptr);
                if (q) ec_load16_i8(A8 + size_t(rho) * p.K, col, al[s][hrow], ah[s][hrow]);
                else ec_load16(pa, col, true, al[s][hrow], ah[s][hrow]);
                sa[s][hrow] = q ? __half2float(__ldg(p.A_scale + rho)) : 1.f;
            }
    };
    if constexpr (FUSED) {
        for (int i = threadIdx.x; i < kTok * zr; i += 256) zmine[i] = 0.f;
        cluster_arrive_release();                              // "this CTA runs": matched before the first peer store below
        if (warp < n_items) load_A(warp);                      // the factors are parameters: before the wait
    }
    pdl_launch_dependents();
    pdl_wait();          // x (and u) may be written by the previous kernel in the stream
    if (!FUSED && p.r > 0) {
        if (p.zpart) {
            // the pre-kernel left eight partial z [kTok][r + 1] in global memory: sum them in rank order, gate, u (all loads of a
            // thread in flight at once; they share the round trip with the x loads below)
            const bool sc = (p.gate_kind == SPEAR_GATE_SCALAR_SIGMOID);
            const int zr1 = p.r + 1;
            const float bias = (sc && p.b_g) ? __ldg(p.b_g) : 0.f;
            for (int i = threadIdx.x; i < kTok * p.r; i += 256) {
                const int m = i / p.r, j = i - m * p.r;
                float zv[8], gv[8];
#pragma unroll
                for (int c = 0; c < 8; ++c) {
                    zv[c] = p.zpart[(c * kTok + m) * zr1 + j];
                    gv[c] = sc ? p.zpart[(c * kTok + m) * zr1 + p.r] : 0.f;
                }
                float z = 0.f, zg = 0.f;
#pragma unroll
                for (int c = 0; c < 8; ++c) { z += zv[c]; zg += gv[c]; }
                const float gam = sc ? 1.f / (1.f + expf(-(zg + bias))) : 1.f;
                us[i] = m < p.M ? p.alpha * gam * z : 0.f;
                if (sc && p.gate_out && blockIdx.x == 0 && j == 0 && m < p.M) p.gate_out[m] = gam;
            }
        } else {
            for (int i = threadIdx.x; i < kTok * p.r; i += 256) {
                if (i < p.M * p.r) cp_async4(us + i, p.u + i); else us[i] = 0.f;
            }
        }
    }

    float tot[MT][4];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) tot[mt][0] = tot[mt][1] = tot[mt][2] = tot[mt][3] = 0.f;
    const __half* xrow[MT];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) xrow[mt] = (mt * 8 + g < p.M) ? p.x + size_t(mt * 8 + g) * p.K + 16 * t : nullptr;

    uint4 xa[kRowsNB][MT], xb[kRowsNB][MT];
    auto load_x = [&](int base) {
#pragma unroll
        for (int b = 0; b < kRowsNB; ++b) {
            const int kt = base + 8 * b;
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
                if (kt < KT && xrow[mt]) {
                    xa[b][mt] = *reinterpret_cast<const uint4*>(xrow[mt] + kt * 64);
                    xb[b][mt] = *reinterpret_cast<const uint4*>(xrow[mt] + kt * 64 + 8);
                } else {
                    xa[b][mt] = make_uint4(0u, 0u, 0u, 0u);
                    xb[b][mt] = make_uint4(0u, 0u, 0u, 0u);
                }
            }
        }
    };
    auto compute = [&](int base) {
#pragma unroll
        for (int b = 0; b < kRowsNB; ++b) {
            const int kt = base + 8 * b;
            if (kt < KT) {
                const uint4 w = wv[b];
                uint32_t a0[4], a1[4], a2[4], a3[4];
                dequant_word(w.x, a0);   // row g,     columns 16t + 0..7
                dequant_word(w.z, a1);   // row g + 8, columns 16t + 0..7
                dequant_word(w.y, a2);   // row g,     columns 16t + 8..15
                dequant_word(w.w, a3);   // row g + 8, columns 16t + 8..15
                const float s_lo = __half2float(__ushort_as_half(uint16_t(sc[b] & 0xffff)));
                const float s_hi = __half2float(__ushort_as_half(uint16_t(sc[b] >> 16)));
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    float acc[4] = {0.f, 0.f, 0.f, 0.f}, acd[4] = {0.f, 0.f, 0.f, 0.f};      // two short chains
                    mma_m16n8k16(acc, a0[0], a1[0], a2[0], a3[0], xa[b][mt].x, xb[b][mt].x);
                    mma_m16n8k16(acd, a0[1], a1[1], a2[1], a3[1], xa[b][mt].y, xb[b][mt].y);
                    mma_m16n8k16(acc, a0[2], a1[2], a2[2], a3[2], xa[b][mt].z, xb[b][mt].z);
                    mma_m16n8k16(acd, a0[3], a1[3], a2[3], a3[3], xa[b][mt].w, xb[b][mt].w);
                    tot[mt][0] = fmaf(s_lo, acc[0] + acd[0], tot[mt][0]);
                    tot[mt][1] = fmaf(s_lo, acc[1] + acd[1], tot[mt][1]);
                    tot[mt][2] = fmaf(s_hi, acc[2] + acd[2], tot[mt][2]);
                    tot[mt][3] = fmaf(s_hi, acc[3] + acd[3], tot[mt][3]);
                }
            }
        }
#pragma unroll
        for (int b = 0; b < kRowsNB; ++b) { wv[b] = wn[b]; sc[b] = sn[b]; }
    };

    // the first batch: its x requests (and the second batch's weights) are in flight while the z phase runs
    load_x(warp);
    if (warp + 8 * kRowsNB < KT) load_w(wn, sn, warp + 8 * kRowsNB);
    if constexpr (FUSED) {
        __syncthreads();                                       // zmine is zero
        for (int item = warp; item < n_items; item += 8) {
            if (item != warp) load_A(item);
            const int kt = kt0 + item / sgroups, s0 = (item % sgroups) * kSG;
            uint32_t xl[MT][4], xh[MT][4];
#pragma unroll
            for (int mt = 0; mt < MT; ++mt)
                ec_load16(mt * 8 + g < p.M ? p.x + size_t(mt * 8 + g) * p.K : nullptr, kt * 64 + 16 * t, false, xl[mt], xh[mt]);
#pragma unroll
            for (int s = 0; s < kSG; ++s) {
                if (s0 + s >= strips) break;
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
                    for (int jj = 0; jj < 4; ++jj)
                        mma_m16n8k16(acc, al[s][0][jj], al[s][1][jj], ah[s][0][jj], ah[s][1][jj], xl[mt][jj], xh[mt][jj]);
                    // C fragment: rows rho0 / rho0 + 8 of [A; w_g], tokens mt * 8 + 2t, + 1
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const int rho = (s0 + s) * 16 + g + ((i & 2) ? 8 : 0);
                        if (rho < zr) atomicAdd(zmine + (mt * 8 + 2 * t + (i & 1)) * zr + rho, sa[s][(i & 2) ? 1 : 0] * acc[i]);
                    }
                }
            }
        }
        __syncthreads();
        cluster_wait_acquire();                                // every CTA of the cluster has started: its shared memory may be written
        // every CTA of the cluster gets this part in its slot `rank`
        const uint32_t slot_local = smem_u32(zslots + int(rank) * kTok * zr);
        for (int i = threadIdx.x; i < kTok * zr; i += 256) {
            const float v = zmine[i];
#pragma unroll
            for (uint32_t c = 0; c < 8; ++c) st_shared_cluster_f32(mapa_shared(slot_local + 4 * i, c), v);
        }
        cluster_arrive_release();                              // the matching wait is after the main loop
    }
    compute(warp);
    for (int base = warp + 8 * kRowsNB; base < KT; base += 8 * kRowsNB) {
        load_x(base);
        if (base + 8 * kRowsNB < KT) load_w(wn, sn, base + 8 * kRowsNB);      // the next batch is in flight while this one is consumed
        compute(base);
    }
    // C fragment: rows g / g + 8, tokens mt * 8 + 2t, + 1
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) {
        red[warp][g][mt * 8 + 2 * t] = tot[mt][0];
        red[warp][g][mt * 8 + 2 * t + 1] = tot[mt][1];
        red[warp][g + 8][mt * 8 + 2 * t] = tot[mt][2];
        red[warp][g + 8][mt * 8 + 2 * t + 1] = tot[mt][3];
    }
    if (p.r > 0) cp_async_wait_all();      // this thread's pieces of the B slab (and of u) have landed; the barriers below publish them
    if constexpr (FUSED) {
        // ---- S5 + S6: the cluster's z is complete once every CTA has arrived: sum the slots in rank order, gate, u ----
        cluster_wait_acquire();
        float* zsum = zslots + 8 * kTok * zr;
        for (int i = threadIdx.x; i < kTok * zr; i += 256) {
            float z = 0.f;
#pragma unroll
            for (int c = 0; c < 8; ++c) z += zslots[c * kTok * zr + i];
            zsum[i] = z;
        }
        __syncthreads();
        if (scalar && threadIdx.x < kTok) {                    // one gate per token, kept in the (now free) pre-activation column
            const int m = threadIdx.x;
            const float gam = 1.f / (1.f + expf(-(zsum[m * zr + p.r] + (p.b_g ? __ldg(p.b_g) : 0.f))));
            zsum[m * zr + p.r] = gam;
            if (p.gate_out && blockIdx.x == 0 && m < p.M) p.gate_out[m] = gam;
        }
        __syncthreads();
        for (int m = warp; m < kTok; m += 8) {
            const float ag = p.alpha * (scalar ? zsum[m * zr + p.r] : 1.f);
            for (int j = lane; j < p.r; j += 32) us[m * p.r + j] = m < p.M ? ag * zsum[m * zr + j] : 0.f;
        }
    }
    __syncthreads();
    const int row = threadIdx.x & 15, tok = threadIdx.x >> 4;
    if (tok < p.M) {
        float v = 0.f;
#pragma unroll
        for (int w = 0; w < 8; ++w) v += red[w][row][tok];
        const int n = strip * 16 + row;
        if (p.r > 0) {
            // S7: + sum_j u[m][j] B[n][j], eight terms per step on two independent chains
            const float4* up = reinterpret_cast<const float4*>(us + tok * p.r);
            float e0 = 0.f, e1 = 0.f;
            for (int j8 = 0; j8 < p.r / 8; ++j8) {
                uint32_t bw[4];
                if (p.ec_int8) {
                    const uint2 b8 = *reinterpret_cast<const uint2*>(bs + row * brow + j8 * 8);
                    cvt_i8x4_f16x2(b8.x, bw[0], bw[1]);
                    cvt_i8x4_f16x2(b8.y, bw[2], bw[3]);
                } else {
                    const uint4 bv = *reinterpret_cast<const uint4*>(bs + row * brow + j8 * 16);
                    bw[0] = bv.x; bw[1] = bv.y; bw[2] = bv.z; bw[3] = bv.w;
                }
                const float4 ua = up[2 * j8], ub = up[2 * j8 + 1];
                const float2 f0 = __half22float2(*reinterpret_cast<const __half2*>(&bw[0]));
                const float2 f1 = __half22float2(*reinterpret_cast<const __half2*>(&bw[1]));
                const float2 f2 = __half22float2(*reinterpret_cast<const __half2*>(&bw[2]));
                const float2 f3 = __half22float2(*reinterpret_cast<const __half2*>(&bw[3]));
                e0 += ua.x * f0.x + ua.y * f0.y + ua.z * f1.x + ua.w * f1.y;
                e1 += ub.x * f2.x + ub.y * f2.y + ub.z * f3.x + ub.w * f3.y;
            }
            float e = e0 + e1;
            if (p.ec_int8) e *= __half2float(__ldg(p.B_scale + n));
            v += e;
        }
        p.y[size_t(tok) * p.N + n] = __float2half_rn(v);      // S8: one RN-even cast
    }
}

// ---- the same strip kernel for 17..64 tokens (mid-M on small layers) ------------------------------------------------------------
// The tcgen05 kernel pays one ~0.45 us barrier round trip per 128 columns of K whatever the token count, so a 2048-column
// layer costs it >= 9-12 us at any M; this kernel has no such floor.  grid = (N / 16 strips, ceil(M / 32) token blocks); a CTA
// takes 32 tokens (four n = 8 tiles per mma.sync k-step) of one strip over the whole of K; weights are re-read per token block
// (L2 hits: these are small layers).  It is bound by the legacy mma.sync rate and the x fragment loads, so it loses to tcgen05 on
// big layers and above 64 tokens (api.cu decides).  EC: u = alpha gamma (.) z comes as fp16 [M][r] from the M > 16 pre-pass.
__global__ void __launch_bounds__(256, 2) rowsm_kernel(const RowsParams p) {
    constexpr int MT = 4, kTok = 32, kNB = 2;
    __shared__ float red[8][16][kTok + 1];
    __shared__ __align__(16) float us[kTok * 128];
    __shared__ __align__(16) uint8_t bs[16 * (128 * 2 + 16)];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane >> 2, t = lane & 3;
    const int strip = blockIdx.x, mb = blockIdx.y * kTok;
    const int pnl = strip >> 3, sp = strip & 7;
    const int KT = p.K >> 6, C = p.K >> 7;
    const uint8_t* wbase = reinterpret_cast<const uint8_t*>(p.wq) + size_t(pnl) * C * 8192 + (sp * 32 + lane) * 16;
    const uint8_t* sbase = reinterpret_cast<const uint8_t*>(p.scales) + size_t(pnl) * p.G * 256 + (sp * 16 + 2 * g) * 2;
    const int kt_per_group = p.group >> 6;
    uint4 wv[kNB], wn[kNB];
    uint32_t sc[kNB], sn[kNB];
    auto load_w = [&](uint4 (&wd)[kNB], uint32_t (&sd)[kNB], int base) {
#pragma unroll
        for (int b = 0; b < kNB; ++b) {
            const int kt = base + 8 * b;
            if (kt < KT) {
                wd[b] = __ldg(reinterpret_cast<const uint4*>(wbase + size_t(kt >> 1) * 8192 + (kt & 1) * 4096));      // (re-read by the other token blocks: keep it cached)
                sd[b] = __ldg(reinterpret_cast<const uint32_t*>(sbase + size_t(kt / kt_per_group) * 256));
            }
        }
    };
    load_w(wv, sc, warp);
    const int brow = p.r * 2 + 16;
    if (p.r > 0) {
        const int per_row = p.r * 2 / 8;
        const uint8_t* Bs = reinterpret_cast<const uint8_t*>(p.B) + size_t(strip) * 16 * p.r * 2;
        for (int i = threadIdx.x; i < 16 * per_row; i += 256) {
            const int rw = i / per_row, pc = i - rw * per_row;
            cp_async8(bs + rw * brow + pc * 8, Bs + (size_t(rw) * per_row + pc) * 8);
        }
    }
    pdl_launch_dependents();
    pdl_wait();
    if (p.r > 0)
        for (int i = threadIdx.x; i < kTok * p.r; i += 256) {
            const int m = mb + i / p.r;
            us[i] = m < p.M ? __half2float(__ldcg(p.u16 + size_t(mb) * p.r + i)) : 0.f;
        }
    float tot[MT][4];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) tot[mt][0] = tot[mt][1] = tot[mt][2] = tot[mt][3] = 0.f;
    const __half* xrow[MT];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) xrow[mt] = (mb + mt * 8 + g < p.M) ? p.x + size_t(mb + mt * 8 + g) * p.K + 16 * t : nullptr;
    for (int base = warp; base < KT; base += 8 * kNB) {
        if (base + 8 * kNB < KT) load_w(wn, sn, base + 8 * kNB);
#pragma unroll
        for (int b = 0; b < kNB; ++b) {
            const int kt = base + 8 * b;
            if (kt < KT) {
                uint4 xa[MT], xb[MT];
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    if (xrow[mt]) {
                        xa[mt] = *reinterpret_cast<const uint4*>(xrow[mt] + kt * 64);
                        xb[mt] = *reinterpret_cast<const uint4*>(xrow[mt] + kt * 64 + 8);
                    } else {
                        xa[mt] = make_uint4(0u, 0u, 0u, 0u);
                        xb[mt] = make_uint4(0u, 0u, 0u, 0u);
                    }
                }
                const uint4 w = wv[b];
                uint32_t a0[4], a1[4], a2[4], a3[4];
                dequant_word(w.x, a0);
                dequant_word(w.z, a1);
                dequant_word(w.y, a2);
                dequant_word(w.w, a3);
                const float s_lo = __half2float(__ushort_as_half(uint16_t(sc[b] & 0xffff)));
                const float s_hi = __half2float(__ushort_as_half(uint16_t(sc[b] >> 16)));
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    float acc[4] = {0.f, 0.f, 0.f, 0.f}, acd[4] = {0.f, 0.f, 0.f, 0.f};
                    mma_m16n8k16(acc, a0[0], a1[0], a2[0], a3[0], xa[mt].x, xb[mt].x);
                    mma_m16n8k16(acd, a0[1], a1[1], a2[1], a3[1], xa[mt].y, xb[mt].y);
                    mma_m16n8k16(acc, a0[2], a1[2], a2[2], a3[2], xa[mt].z, xb[mt].z);
                    mma_m16n8k16(acd, a0[3], a1[3], a2[3], a3[3], xa[mt].w, xb[mt].w);
                    tot[mt][0] = fmaf(s_lo, acc[0] + acd[0], tot[mt][0]);
                    tot[mt][1] = fmaf(s_lo, acc[1] + acd[1], tot[mt][1]);
                    tot[mt][2] = fmaf(s_hi, acc[2] + acd[2], tot[mt][2]);
                    tot[mt][3] = fmaf(s_hi, acc[3] + acd[3], tot[mt][3]);
                }
            }
        }
#pragma unroll
        for (int b = 0; b < kNB; ++b) { wv[b] = wn[b]; sc[b] = sn[b]; }
    }
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) {
        red[warp][g][mt * 8 + 2 * t] = tot[mt][0];
        red[warp][g][mt * 8 + 2 * t + 1] = tot[mt][1];
        red[warp][g + 8][mt * 8 + 2 * t] = tot[mt][2];
        red[warp][g + 8][mt * 8 + 2 * t + 1] = tot[mt][3];
    }
    if (p.r > 0) cp_async_wait_all();
    __syncthreads();
    const int row = threadIdx.x & 15;
    const int n = strip * 16 + row;
#pragma unroll
    for (int pass = 0; pass < 2; ++pass) {
        const int tok = (threadIdx.x >> 4) + 16 * pass;
        if (mb + tok >= p.M) continue;
        float v = 0.f;
#pragma unroll
        for (int w = 0; w < 8; ++w) v += red[w][row][tok];
        if (p.r > 0) {
            const float4* up = reinterpret_cast<const float4*>(us + tok * p.r);
            float e0 = 0.f, e1 = 0.f;
            for (int j8 = 0; j8 < p.r / 8; ++j8) {
                const uint4 bv = *reinterpret_cast<const uint4*>(bs + row * brow + j8 * 16);
                const float4 ua = up[2 * j8], ub = up[2 * j8 + 1];
                const float2 f0 = __half22float2(*reinterpret_cast<const __half2*>(&bv.x));
                const float2 f1 = __half22float2(*reinterpret_cast<const __half2*>(&bv.y));
                const float2 f2 = __half22float2(*reinterpret_cast<const __half2*>(&bv.z));
                const float2 f3 = __half22float2(*reinterpret_cast<const __half2*>(&bv.w));
                e0 += ua.x * f0.x + ua.y * f0.y + ua.z * f1.x + ua.w * f1.y;
                e1 += ub.x * f2.x + ub.y * f2.y + ub.z * f3.x + ub.w * f3.y;
            }
            v += e0 + e1;
        }
        p.y[size_t(mb + tok) * p.N + n] = __float2half_rn(v);
    }
}

// ---- z, gate and u ONCE, by one cluster of 8 CTAs (S4-S6 for the split arm of the row-strip kernel) -----------------------------
// The fused instance above makes every cluster of the layer recompute z (N / 128 times the work, and it sits in front of
// each CTA's main loop).  Here z = x [A; w_g]^T is computed once: CTA c of ONE cluster takes the c-th eighth of K (its
// slice of A is requested before griddepcontrol.wait, x after), the eight partial z land in the slots of rank 0 through
// distributed shared memory, rank 0 sums them in rank order, applies the gate (scalar / none) and writes
// u = alpha gamma (.) z as fp32 [8 MT][r] to global memory for the layer kernel that is already running behind it under
// programmatic dependent launch (its weight requests are in flight; it reads u after its own griddepcontrol.wait).
template <int MT, bool PART>      // PART: no cluster -- 8 independent CTAs park their partial z in global memory, the layer kernel sums and gates
__global__ void __launch_bounds__(256, 1) ecz_cluster_kernel(const RowsParams p) {
    constexpr int kTok = 8 * MT;
    constexpr int kSG = 2;
    extern __shared__ float zs[];                 // [8 ranks][kTok][r + 1] (used in rank 0), then [kTok][r + 1] own partial
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane >> 2, t = lane & 3;
    const int KT = p.K >> 6;
    const bool scalar = (p.gate_kind == SPEAR_GATE_SCALAR_SIGMOID);
    const int zr = p.r + 1;
    const int strips = (p.r + (scalar ? 1 : 0) + 15) >> 4;
    const int sgroups = (strips + kSG - 1) / kSG;
    const uint32_t rank = PART ? blockIdx.x : cluster_ctarank();
    const int kt0 = int(rank) * KT / 8, kt1 = (int(rank) + 1) * KT / 8;
    const int n_items = (kt1 - kt0) * sgroups;
    float* zmine = zs + 8 * kTok * zr;
    pdl_launch_dependents();                      // the layer kernel may start (and request its weights) right away
    uint32_t al[2][kSG][2][4], ah[2][kSG][2][4];  // two items in flight: [buffer][strip][row g / g + 8][k16 step]
    float sa[2][kSG][2];
    auto load_A = [&](int buf, int item) {
        const int kt = kt0 + item / sgroups, s0 = (item % sgroups) * kSG;
        const int col = kt * 64 + 16 * t;
        const int8_t* A8 = reinterpret_cast<const int8_t*>(p.A);
#pragma unroll
        for (int s = 0; s < kSG; ++s)
#pragma unroll
            for (int hrow = 0; hrow < 2; ++hrow) {
                const int rho = (s0 + s) * 16 + g + 8 * hrow;
                const bool q = p.ec_int8 && rho < p.r;                 // the gate row w_g stays fp16
                const __half* pa = rho < p.r ? p.A + size_t(rho) * p.K : (rho == p.r && scalar ? p.w_g : nullptr);
                if (q) ec_load16_i8(A8 + size_t(rho) * p.K, col, al[buf][s][hrow], ah[buf][s][hrow]);
                else ec_load16(pa, col, true, al[buf][s][hrow], ah[buf][s][hrow]);
                sa[buf][s][hrow] = q ? __half2float(__ldg(p.A_scale + rho)) : 1.f;
            }
    };
    for (int i = threadIdx.x; i < kTok * zr; i += 256) zmine[i] = 0.f;
    if (!PART) cluster_arrive_release();          // "this CTA runs": matched before the first peer store below
    if (warp < n_items) load_A(0, warp);          // the factors are parameters: before the wait
    pdl_wait();                                   // x may be the previous kernel's output
    __syncthreads();                              // zmine is zero
    int buf = 0;
    for (int item = warp; item < n_items; item += 8, buf ^= 1) {
        const int kt = kt0 + item / sgroups, s0 = (item % sgroups) * kSG;
        uint32_t xl[MT][4], xh[MT][4];
#pragma unroll
        for (int mt = 0; mt < MT; ++mt)
            ec_load16(mt * 8 + g < p.M ? p.x + size_t(mt * 8 + g) * p.K : nullptr, kt * 64 + 16 * t, false, xl[mt], xh[mt]);
        if (item + 8 < n_items) {                 // the next item's factors are in flight while this one is consumed
            if (buf == 0) load_A(1, item + 8); else load_A(0, item + 8);
        }
#pragma unroll
        for (int bsel = 0; bsel < 2; ++bsel) {
            if (bsel != buf) continue;
#pragma unroll
            for (int s = 0; s < kSG; ++s) {
                if (s0 + s >= strips) break;
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    float acc[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
                    for (int jj = 0; jj < 4; ++jj)
                        mma_m16n8k16(acc, al[bsel][s][0][jj], al[bsel][s][1][jj], ah[bsel][s][0][jj], ah[bsel][s][1][jj], xl[mt][jj], xh[mt][jj]);
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const int rho = (s0 + s) * 16 + g + ((i & 2) ? 8 : 0);
                        if (rho < zr) atomicAdd(zmine + (mt * 8 + 2 * t + (i & 1)) * zr + rho, sa[bsel][s][(i & 2) ? 1 : 0] * acc[i]);
                    }
                }
            }
        }
    }
    __syncthreads();
    if (PART) {
        float* out = p.zpart + size_t(rank) * kTok * zr;
        for (int i = threadIdx.x; i < kTok * zr; i += 256) out[i] = zmine[i];
        return;
    }
    cluster_wait_acquire();                       // every CTA of the cluster has started: rank 0's shared memory may be written
    const uint32_t slot0 = mapa_shared(smem_u32(zs + int(rank) * kTok * zr), 0);
    for (int i = threadIdx.x; i < kTok * zr; i += 256) st_shared_cluster_f32(slot0 + 4 * i, zmine[i]);
    cluster_arrive_release();
    cluster_wait_acquire();                       // all eight parts are in rank 0
    if (rank != 0) return;
    float* zsum = zmine;
    for (int i = threadIdx.x; i < kTok * zr; i += 256) {
        float z = 0.f;
#pragma unroll
        for (int c = 0; c < 8; ++c) z += zs[c * kTok * zr + i];
        zsum[i] = z;
    }
    __syncthreads();
    if (scalar && threadIdx.x < kTok) {
        const int m = threadIdx.x;
        const float gam = 1.f / (1.f + expf(-(zsum[m * zr + p.r] + (p.b_g ? __ldg(p.b_g) : 0.f))));
        zsum[m * zr + p.r] = gam;
        if (p.gate_out && m < p.M) p.gate_out[m] = gam;
    }
    __syncthreads();
    float* uo = const_cast<float*>(p.u);
    for (int i = threadIdx.x; i < p.M * p.r; i += 256) {
        const int m = i / p.r, j = i - m * p.r;
        uo[i] = p.alpha * (scalar ? zsum[m * zr + p.r] : 1.f) * zsum[m * zr + j];
    }
}
}  // namespace

int launch_rows(const RowsParams& p, bool pdl, cudaStream_t st) {
    const int MT = p.M <= 8 ? 1 : 2;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(p.N / 16);
    cfg.blockDim = dim3(256);
    cfg.dynamicSmemBytes = p.fused ? size_t(9) * 8 * MT * (p.r + 1) * 4 : 0;
    cfg.stream = st;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (p.fused) {
        static std::once_flag once;
        static cudaError_t err = cudaSuccess;
        std::call_once(once, [&]() {
            err = cudaFuncSetAttribute((const void*)rows_kernel<1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 9 * 8 * 129 * 4);
            if (err == cudaSuccess)
                err = cudaFuncSetAttribute((const void*)rows_kernel<2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 9 * 16 * 129 * 4);
        });
        SPEAR_CUDA_OK(err);
        attr[1].id = cudaLaunchAttributeClusterDimension;      // one cluster = the 8 strips of one 128-row panel
        attr[1].val.clusterDim.x = 8;
        attr[1].val.clusterDim.y = 1;
        attr[1].val.clusterDim.z = 1;
        cfg.numAttrs = 2;
        if (MT == 1) SPEAR_CUDA_OK(cudaLaunchKernelEx(&cfg, rows_kernel<1, true>, p));
        else SPEAR_CUDA_OK(cudaLaunchKernelEx(&cfg, rows_kernel<2, true>, p));
    } else {
        if (MT == 1) SPEAR_CUDA_OK(cudaLaunchKernelEx(&cfg, rows_kernel<1, false>, p));
        else SPEAR_CUDA_OK(cudaLaunchKernelEx(&cfg, rows_kernel<2, false>, p));
    }
    count_launch();
    return SPEAR_OK;
}

int launch_ecz_cluster(const RowsParams& p, bool pdl, cudaStream_t st) {
    const int MT = p.M <= 8 ? 1 : 2;
    static std::once_flag once;
    static cudaError_t err = cudaSuccess;
    std::call_once(once, [&]() {
        err = cudaFuncSetAttribute((const void*)ecz_cluster_kernel<1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 9 * 8 * 129 * 4);
        if (err == cudaSuccess)
            err = cudaFuncSetAttribute((const void*)ecz_cluster_kernel<2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 9 * 16 * 129 * 4);
    });
    SPEAR_CUDA_OK(err);
    if (p.zpart) {
        static std::once_flag once2;
        static cudaError_t err2 = cudaSuccess;
        std::call_once(once2, [&]() {
            err2 = cudaFuncSetAttribute((const void*)ecz_cluster_kernel<1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 9 * 8 * 129 * 4);
            if (err2 == cudaSuccess)
                err2 = cudaFuncSetAttribute((const void*)ecz_cluster_kernel<2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 9 * 16 * 129 * 4);
        });
        SPEAR_CUDA_OK(err2);
        cudaLaunchConfig_t c2 = {};
        c2.gridDim = dim3(8);
        c2.blockDim = dim3(256);
        c2.dynamicSmemBytes = size_t(9) * 8 * MT * (p.r + 1) * 4;
        c2.stream = st;
        cudaLaunchAttribute a2[1];
        a2[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        a2[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
        c2.attrs = a2;
        c2.numAttrs = 1;
        if (MT == 1) SPEAR_CUDA_OK(cudaLaunchKernelEx(&c2, ecz_cluster_kernel<1, true>, p));
        else SPEAR_CUDA_OK(cudaLaunchKernelEx(&c2, ecz_cluster_kernel<2, true>, p));
        count_launch();
        return SPEAR_OK;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(8);
    cfg.blockDim = dim3(256);
    cfg.dynamicSmemBytes = size_t(9) * 8 * MT * (p.r + 1) * 4;
    cfg.stream = st;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
    attr[1].id = cudaLaunchAttributeClusterDimension;
    attr[1].val.clusterDim.x = 8;
    attr[1].val.clusterDim.y = 1;
    attr[1].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 2;
    if (MT == 1) SPEAR_CUDA_OK(cudaLaunchKernelEx(&cfg, ecz_cluster_kernel<1, false>, p));
    else SPEAR_CUDA_OK(cudaLaunchKernelEx(&cfg, ecz_cluster_kernel<2, false>, p));
    count_launch();
    return SPEAR_OK;
}

int launch_rows_mid(const RowsParams& p, bool pdl, cudaStream_t st) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(p.N / 16, (p.M + 31) / 32);
    cfg.blockDim = dim3(256);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    SPEAR_CUDA_OK(cudaLaunchKernelEx(&cfg, rowsm_kernel, p));
    count_launch();
    return SPEAR_OK;
}

}  // namespace spear

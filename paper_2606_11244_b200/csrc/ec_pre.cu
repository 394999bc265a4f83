// ec_pre.cu -- steps S4-S6 of SURVEY.md 8(a) for small token counts (M <= 16):
//     z = x A^T           ("Ax"; must be fully K-reduced before the gate)
//     gamma               (PAPER.md:109 MLP gate 1 + tanh(W2 relu(W1 z + b1) + b2); BASELINE.json scalar
//                          gate sigmoid(x . w_g + b), reading A1; gamma == 1 is Eq. 2)
//     u = alpha * gamma (.) z   -> fp32 workspace, consumed by the weight-stream kernel's epilogue.
//
// A is streamed once device-wide: grid = (16-row strips of A [+ the w_g row]) x (K splits); every warp
// multiplies its K tiles with mma.sync.m16n8k16 (A rows as the 16-row operand, tokens as n = 8, the
// same k-permutation trick as the weight kernel: a lane reads 32 contiguous bytes of a row), partial
// z goes to a global fp32 buffer with red.add, and the LAST CTA to arrive (atomic counter) applies the
// gate, writes u and re-zeroes the buffer so the workspace is clean for the next call.
#include <algorithm>
#include <mutex>

#include "common.cuh"
#include "kernels.h"

namespace spear {

__device__ __forceinline__ void load_row32(const __half* row, int col, uint32_t (&lo)[4], uint32_t (&hi)[4]) {
    if (row) {
        const uint4 a = __ldg(reinterpret_cast<const uint4*>(row + col));
        const uint4 b = __ldg(reinterpret_cast<const uint4*>(row + col + 8));
        lo[0] = a.x; lo[1] = a.y; lo[2] = a.z; lo[3] = a.w;
        hi[0] = b.x; hi[1] = b.y; hi[2] = b.z; hi[3] = b.w;
    } else {
#pragma unroll
        for (int i = 0; i < 4; ++i) lo[i] = hi[i] = 0u;
    }
}
// INT8 factor row: 16 columns = 16 bytes, converted exactly to the fp16 fragment registers
__device__ __forceinline__ void load_row32_i8(const int8_t* row, int col, uint32_t (&lo)[4], uint32_t (&hi)[4]) {
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
__device__ __forceinline__ void load_x32(const __half* row, int col, uint32_t (&lo)[4], uint32_t (&hi)[4]) {
    if (row) {   // x may have been written by the previous kernel: plain (coherent) loads
        const uint4 a = *reinterpret_cast<const uint4*>(row + col);
        const uint4 b = *reinterpret_cast<const uint4*>(row + col + 8);
        lo[0] = a.x; lo[1] = a.y; lo[2] = a.z; lo[3] = a.w;
        hi[0] = b.x; hi[1] = b.y; hi[2] = b.z; hi[3] = b.w;
    } else {
#pragma unroll
        for (int i = 0; i < 4; ++i) lo[i] = hi[i] = 0u;
    }
}

// S5 + S6 for up to 16 tokens whose fully reduced z rows sit in zs[m][0..r) (zs[m][r] = scalar-gate logit):
//   MLP    gamma = 1 + tanh(W2 relu(W1 z + b1) + b2)
//   scalar gamma = sigmoid(x . w_g + b)                  BASELINE.json configs (reading A1)
//   none   gamma = 1                                     PAPER.md:96 (Eq. 2)
// u = alpha * gamma (.) z goes to u32[m][r] (fp32, decode path) or u16[m_base + m][r] (fp16, tcgen05 path).
struct GateArgs {
    int gate_kind, r, h;
    float alpha;
    const float* b_g;
    const __half* W1; const float* b1; const __half* W2; const float* b2;
    float* u32; __half* u16; float* gate_out;
};
__device__ __forceinline__ void put_u(const GateArgs& ga, int m, int m_base, int j, float v) {
    if (ga.u16) ga.u16[size_t(m_base + m) * ga.r + j] = __float2half_rn(v);
    else ga.u32[m * ga.r + j] = v;
}
__device__ void apply_gate(const GateArgs& ga, float (*zs)[kZStride], float (*hid)[512], int m_count,
                           int m_base, int tid, int nthreads) {
    const int r = ga.r;
    if (ga.gate_kind == SPEAR_GATE_SCALAR_SIGMOID) {
        const float bias = ga.b_g ? *ga.b_g : 0.f;
        for (int o = tid; o < m_count * r; o += nthreads) {
            const int m = o / r, j = o - m * r;
            const float gam = 1.f / (1.f + expf(-(zs[m][r] + bias)));
            put_u(ga, m, m_base, j, ga.alpha * gam * zs[m][j]);
            if (ga.gate_out && j == 0) ga.gate_out[m_base + m] = gam;
        }
    } else if (ga.gate_kind == SPEAR_GATE_MLP) {
        const int h = ga.h;
        // rows of W1 / W2 are read as 16-byte vectors, four in flight, so that the L2 latency is paid per row and
        // not per element (r % 8 == 0 and h % 8 == 0: every row is 16-byte aligned)
        for (int i = tid; i < h; i += nthreads) {
            float a[16];
#pragma unroll
            for (int m = 0; m < 16; ++m) a[m] = 0.f;
            const uint4* w1 = reinterpret_cast<const uint4*>(ga.W1 + size_t(i) * r);
#pragma unroll 4
            for (int j8 = 0; j8 < r / 8; ++j8) {
                const uint4 wv = __ldg(w1 + j8);
                const __half2* wh = reinterpret_cast<const __half2*>(&wv);
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const float2 w = __half22float2(wh[q]);
                    const int j = j8 * 8 + 2 * q;
#pragma unroll
                    for (int m = 0; m < 16; ++m) a[m] = fmaf(w.y, zs[m][j + 1], fmaf(w.x, zs[m][j], a[m]));
                }
            }
            const float bb = ga.b1[i];
#pragma unroll
            for (int m = 0; m < 16; ++m) hid[m][i] = fmaxf(a[m] + bb, 0.f);
        }
        __syncthreads();
        for (int j = tid; j < r; j += nthreads) {
            float a[16];
#pragma unroll
            for (int m = 0; m < 16; ++m) a[m] = 0.f;
            const uint4* w2 = reinterpret_cast<const uint4*>(ga.W2 + size_t(j) * h);
#pragma unroll 4
            for (int i8 = 0; i8 < h / 8; ++i8) {
                const uint4 wv = __ldg(w2 + i8);
                const __half2* wh = reinterpret_cast<const __half2*>(&wv);
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const float2 w = __half22float2(wh[q]);
                    const int i = i8 * 8 + 2 * q;
#pragma unroll
                    for (int m = 0; m < 16; ++m) a[m] = fmaf(w.y, hid[m][i + 1], fmaf(w.x, hid[m][i], a[m]));
                }
            }
            const float bb = ga.b2[j];
            for (int m = 0; m < m_count; ++m) {
                const float gam = 1.f + tanhf(a[m] + bb);
                put_u(ga, m, m_base, j, ga.alpha * gam * zs[m][j]);
                if (ga.gate_out) ga.gate_out[size_t(m_base + m) * r + j] = gam;
            }
        }
    } else {
        for (int o = tid; o < m_count * r; o += nthreads) {
            const int m = o / r, j = o - m * r;
            put_u(ga, m, m_base, j, ga.alpha * zs[m][j]);
        }
    }
}


__global__ void __launch_bounds__(128) ec_pre_kernel(const EcPreParams p) {
    __shared__ float red[4][16][17];
    __shared__ float zs[16][kZStride];
    __shared__ float hid[16][512];
    __shared__ int is_last;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane >> 2, t = lane & 3;
    const int strip = blockIdx.x, ks = blockIdx.y;
    const bool scalar = (p.gate_kind == SPEAR_GATE_SCALAR_SIGMOID);
    const int rows_total = p.r + (scalar ? 1 : 0);

    pdl_launch_dependents();

    const int rho0 = strip * 16 + g, rho1 = rho0 + 8;
    const __half* pa0 = rho0 < p.r ? p.A + size_t(rho0) * p.K : (rho0 == p.r && scalar ? p.w_g : nullptr);
    const __half* pa1 = rho1 < p.r ? p.A + size_t(rho1) * p.K : (rho1 == p.r && scalar ? p.w_g : nullptr);
    const __half* px0 = g < p.M ? p.x + size_t(g) * p.K : nullptr;
    const __half* px1 = g + 8 < p.M ? p.x + size_t(g + 8) * p.K : nullptr;

    const int ktiles = p.K >> 6;
    const int kt_begin = int((long long)ks * ktiles / p.ksplit);
    const int kt_end = int((long long)(ks + 1) * ktiles / p.ksplit);

    float acc0[4] = {0.f, 0.f, 0.f, 0.f}, acc1[4] = {0.f, 0.f, 0.f, 0.f};
    pdl_wait();
    for (int kt = kt_begin + warp; kt < kt_end; kt += 4) {
        const int col = kt * 64 + 16 * t;
        uint32_t a0l[4], a0h[4], a1l[4], a1h[4], x0l[4], x0h[4], x1l[4], x1h[4];
        if (p.ec_int8 && rho0 < p.r) load_row32_i8(reinterpret_cast<const int8_t*>(p.A) + size_t(rho0) * p.K, col, a0l, a0h);
        else load_row32(pa0, col, a0l, a0h);
        if (p.ec_int8 && rho1 < p.r) load_row32_i8(reinterpret_cast<const int8_t*>(p.A) + size_t(rho1) * p.K, col, a1l, a1h);
        else load_row32(pa1, col, a1l, a1h);
        load_x32(px0, col, x0l, x0h);
        load_x32(px1, col, x1l, x1h);
#pragma unroll
        for (int jj = 0; jj < 4; ++jj) {
            mma_m16n8k16(acc0, a0l[jj], a1l[jj], a0h[jj], a1h[jj], x0l[jj], x0h[jj]);
            mma_m16n8k16(acc1, a0l[jj], a1l[jj], a0h[jj], a1h[jj], x1l[jj], x1h[jj]);
        }
    }
    // fragment -> red[warp][row in strip][token]
    red[warp][g][2 * t] = acc0[0];       red[warp][g][2 * t + 1] = acc0[1];
    red[warp][g + 8][2 * t] = acc0[2];   red[warp][g + 8][2 * t + 1] = acc0[3];
    red[warp][g][8 + 2 * t] = acc1[0];   red[warp][g][8 + 2 * t + 1] = acc1[1];
    red[warp][g + 8][8 + 2 * t] = acc1[2]; red[warp][g + 8][8 + 2 * t + 1] = acc1[3];
    __syncthreads();
    for (int o = threadIdx.x; o < 256; o += 128) {
        const int row = o & 15, tok = o >> 4;
        const int rho = strip * 16 + row;
        if (tok < p.M && rho < rows_total) {
            float v = red[0][row][tok] + red[1][row][tok] + red[2][row][tok] + red[3][row][tok];
            if (p.ec_int8 && rho < p.r) v *= __half2float(__ldg(p.A_scale + rho));     // per-row scale of the INT8 factor
            atomicAdd(p.zbuf + tok * kZStride + rho, v);
        }
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned total = gridDim.x * gridDim.y;
        const unsigned old = atomicAdd(p.counter, 1u);
        is_last = (old == total - 1);
        if (is_last) *p.counter = 0;
    }
    __syncthreads();
    if (!is_last) return;

    // ------------------------------ last CTA: gate and u ------------------------------
    __threadfence();
    for (int o = threadIdx.x; o < p.M * rows_total; o += 128) {
        const int m = o / rows_total, rho = o - m * rows_total;
        zs[m][rho] = __ldcg(p.zbuf + m * kZStride + rho);
        p.zbuf[m * kZStride + rho] = 0.f;
    }
    __syncthreads();
    GateArgs ga;
    ga.gate_kind = p.gate_kind; ga.r = p.r; ga.h = p.h; ga.alpha = p.alpha; ga.b_g = p.b_g;
    ga.W1 = p.W1; ga.b1 = p.b1; ga.W2 = p.W2; ga.b2 = p.b2;
    ga.u32 = p.u; ga.u16 = nullptr; ga.gate_out = p.gate_out;
    apply_gate(ga, zs, hid, p.M, 0, threadIdx.x, 128);
}

int launch_ec_pre(const EcPreParams& p, bool pdl, cudaStream_t st) {
    const bool scalar = (p.gate_kind == SPEAR_GATE_SCALAR_SIGMOID);
    const int strips = (p.r + (scalar ? 1 : 0) + 15) / 16;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(strips, p.ksplit);
    cfg.blockDim = dim3(128);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    SPEAR_CUDA_OK(cudaLaunchKernelEx(&cfg, ec_pre_kernel, p));
    count_launch();
    return SPEAR_OK;
}

// ------------------------------------------------------------------------------------------------
// M > 16: z = x [A; w_g]^T as a split-K mma.sync GEMM (tokens are the 16-row operand here), then a
// gate kernel per 16 tokens.  Cost is r/N of the main GEMM (SURVEY.md section 7 "Prefill EC fold").
// ------------------------------------------------------------------------------------------------
// A CTA of 8 warps takes 128 tokens (16 per warp) x every row of [A; w_g] x one K slice.  Per 64-column k-tile the block of
// [A; w_g] (NT x 8 rows x 128 bytes) is staged ONCE per CTA in shared memory by cp.async (three stages in flight) and read by all
// 8 warps; the x fragments are each warp's own and come straight from global memory.  (The first version let every warp fetch its
// A fragments from global memory: at M = 2048, K = 14336, r = 64 that is 128 warps x 1.8 MB through L2 -- 74 us on a 210 us layer.)
// (Measured and not kept: applying the scalar gate in this kernel's last arriver per 128-token block instead of the separate gate
// kernel -- fence + counter + a serial tail in one CTA cost more than the launch they save: M = 256, 4096 -> 6144 36 -> 41 us.)
constexpr int kEzRowBytes = 144;      // 128 bytes of a k-tile row + 16 bytes of padding: the 8 rows x 4 column groups of a quarter-warp hit distinct banks
constexpr int kEzStages = 3;

template <int NT>   // NT = number of 8-row tiles of [A; w_g] (rows beyond r [+1] read as zero)
__global__ void __launch_bounds__(256) ec_big_z_kernel(const EcBigParams p) {
    extern __shared__ __align__(16) uint8_t ez_smem[];      // [kEzStages][NT * 8][kEzRowBytes]
    constexpr int kStageBytes = NT * 8 * kEzRowBytes;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int g = lane >> 2, t = lane & 3;
    const bool scalar = (p.gate_kind == SPEAR_GATE_SCALAR_SIGMOID);
    const int rows_total = p.r + (scalar ? 1 : 0);
    const int m0 = blockIdx.x * 128 + warp * 16;
    const int ktiles = p.K >> 6;
    const int kt_begin = int((long long)blockIdx.y * ktiles / p.ksplit);
    const int kt_end = int((long long)(blockIdx.y + 1) * ktiles / p.ksplit);
    const int n_kt = kt_end - kt_begin;
    pdl_launch_dependents();
    // rows beyond [A; w_g] stay zero in every stage
    for (int i = threadIdx.x; i < kEzStages * NT * 8; i += 256) {
        const int row = i % (NT * 8);
        if (row >= rows_total) {
            uint4* dst = reinterpret_cast<uint4*>(ez_smem + size_t(i / (NT * 8)) * kStageBytes + row * kEzRowBytes);
#pragma unroll
            for (int q = 0; q < 8; ++q) dst[q] = make_uint4(0u, 0u, 0u, 0u);
        }
    }
    auto stage_in = [&](int j) {        // k-tile kt_begin + j -> stage j % kEzStages (one commit group, possibly empty)
        if (j < n_kt) {
            const int kt = kt_begin + j;
            uint8_t* st = ez_smem + size_t(j % kEzStages) * kStageBytes;
            for (int i = threadIdx.x; i < rows_total * 8; i += 256) {
                const int row = i >> 3, pc = i & 7;
                const __half* src = row < p.r ? p.A + size_t(row) * p.K : p.w_g;
                const uint32_t dst = smem_u32(st + row * kEzRowBytes + pc * 16);
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src + kt * 64 + pc * 8) : "memory");
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    // [A; w_g] are parameters: the first stages are requested before griddepcontrol.wait
    for (int j = 0; j < kEzStages - 1; ++j) stage_in(j);
    const __half* px0 = (m0 + g) < p.M ? p.x + size_t(m0 + g) * p.K : nullptr;
    const __half* px1 = (m0 + g + 8) < p.M ? p.x + size_t(m0 + g + 8) * p.K : nullptr;
    float acc[NT][4];
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) acc[nt][0] = acc[nt][1] = acc[nt][2] = acc[nt][3] = 0.f;
    pdl_wait();
    for (int j = 0; j < n_kt; ++j) {
        const int col = (kt_begin + j) * 64 + 16 * t;
        uint32_t x0l[4], x0h[4], x1l[4], x1h[4];
        load_x32(px0, col, x0l, x0h);
        load_x32(px1, col, x1l, x1h);
        asm volatile("cp.async.wait_group %0;" ::"n"(kEzStages - 2) : "memory");      // this thread's pieces of stage j have landed
        __syncthreads();                                     // ... and everybody's; everybody is also done with stage j - 1
        stage_in(j + kEzStages - 1);                         // refill the stage read in iteration j - 1
        const uint8_t* st = ez_smem + size_t(j % kEzStages) * kStageBytes + g * kEzRowBytes + t * 32;
        if (m0 < p.M) {
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) {
                const uint4 lo = *reinterpret_cast<const uint4*>(st + nt * 8 * kEzRowBytes);
                const uint4 hi = *reinterpret_cast<const uint4*>(st + nt * 8 * kEzRowBytes + 16);
                mma_m16n8k16(acc[nt], x0l[0], x1l[0], x0h[0], x1h[0], lo.x, hi.x);
                mma_m16n8k16(acc[nt], x0l[1], x1l[1], x0h[1], x1h[1], lo.y, hi.y);
                mma_m16n8k16(acc[nt], x0l[2], x1l[2], x0h[2], x1h[2], lo.z, hi.z);
                mma_m16n8k16(acc[nt], x0l[3], x1l[3], x0h[3], x1h[3], lo.w, hi.w);
            }
        }
    }
    if (m0 >= p.M) return;
    // C fragment: rows = tokens g, g+8; columns = EC rows nt*8 + 2t, +1
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) {
        const int rho = nt * 8 + 2 * t;
        if (m0 + g < p.M) {
            if (rho < rows_total) atomicAdd(p.zbuf + size_t(m0 + g) * kZStride + rho, acc[nt][0]);
            if (rho + 1 < rows_total) atomicAdd(p.zbuf + size_t(m0 + g) * kZStride + rho + 1, acc[nt][1]);
        }
        if (m0 + g + 8 < p.M) {
            if (rho < rows_total) atomicAdd(p.zbuf + size_t(m0 + g + 8) * kZStride + rho, acc[nt][2]);
            if (rho + 1 < rows_total) atomicAdd(p.zbuf + size_t(m0 + g + 8) * kZStride + rho + 1, acc[nt][3]);
        }
    }
}

__global__ void __launch_bounds__(128) ec_big_gate_kernel(const EcBigParams p) {
    __shared__ float zs[16][kZStride];
    __shared__ float hid[16][512];
    const int m_base = blockIdx.x * 16;
    const int m_count = min(16, p.M - m_base);
    const bool scalar = (p.gate_kind == SPEAR_GATE_SCALAR_SIGMOID);
    const int rows_total = p.r + (scalar ? 1 : 0);
    pdl_launch_dependents();
    pdl_wait();
    for (int o = threadIdx.x; o < 16 * rows_total; o += 128) {
        const int m = o / rows_total, rho = o - m * rows_total;
        float v = 0.f;
        if (m < m_count) {
            float* zp = p.zbuf + size_t(m_base + m) * kZStride + rho;
            v = __ldcg(zp);
            *zp = 0.f;                    // the workspace is left zero for the next call
        }
        zs[m][rho] = v;
    }
    __syncthreads();
    GateArgs ga;
    ga.gate_kind = p.gate_kind; ga.r = p.r; ga.h = p.h; ga.alpha = p.alpha; ga.b_g = p.b_g;
    ga.W1 = p.W1; ga.b1 = p.b1; ga.W2 = p.W2; ga.b2 = p.b2;
    ga.u32 = nullptr; ga.u16 = p.u16; ga.gate_out = p.gate_out;
    apply_gate(ga, zs, hid, m_count, m_base, threadIdx.x, 128);
}

template <int NT>
static int launch_ec_big_z(const EcBigParams& p, cudaLaunchConfig_t& cfg) {
    constexpr int kBytes = kEzStages * NT * 8 * kEzRowBytes;      // <= 58,752 B (NT = 17)
    static std::once_flag once;
    static cudaError_t err = cudaSuccess;
    std::call_once(once, [] { err = cudaFuncSetAttribute(ec_big_z_kernel<NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, kBytes); });
    SPEAR_CUDA_OK(err);
    cfg.dynamicSmemBytes = kBytes;
    SPEAR_CUDA_OK(cudaLaunchKernelEx(&cfg, ec_big_z_kernel<NT>, p));
    return SPEAR_OK;
}

int launch_ec_big(const EcBigParams& p, bool pdl, cudaStream_t st) {
    const bool scalar = (p.gate_kind == SPEAR_GATE_SCALAR_SIGMOID);
    const int nt = (p.r + (scalar ? 1 : 0) + 7) / 8;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((p.M + 127) / 128, p.ksplit);
    cfg.blockDim = dim3(256);
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    int rc;
    if (nt <= 3) rc = launch_ec_big_z<3>(p, cfg);
    else if (nt <= 5) rc = launch_ec_big_z<5>(p, cfg);
    else if (nt <= 9) rc = launch_ec_big_z<9>(p, cfg);
    else if (nt <= 13) rc = launch_ec_big_z<13>(p, cfg);
    else rc = launch_ec_big_z<17>(p, cfg);
    if (rc) return rc;
    cfg.gridDim = dim3((p.M + 15) / 16);
    cfg.blockDim = dim3(128);
    cfg.dynamicSmemBytes = 0;
    SPEAR_CUDA_OK(cudaLaunchKernelEx(&cfg, ec_big_gate_kernel, p));
    count_launch(2);
    return SPEAR_OK;
}

// ------------------------------------------------------------------------------------------------
// Split arm for M > 16 (SPEAR_VARIANT_TC_SPLIT): the rank-r up-projection as its own pass over y,
//     y[m][n] = RN_fp16( y[m][n] + sum_j u16[m][j] * B[n][j] )        (S7 of SURVEY.md 8(a))
// i.e. the paper's naive "re-projection and accumulation" kernels kept as the comparator the
// measured dispatch chooses against.  y was already rounded once by the plain W4 GEMM: this arm double-rounds
// (reading A8) and reads + writes y a second time -- which is exactly why the fused arm usually wins.
// Block = 256 threads, tile = 32 tokens x 128 channels; u and B tiles staged in shared memory as fp32 / fp16.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) ec_update_kernel(const __half* __restrict__ u16, const __half* __restrict__ B,
                                                        __half* __restrict__ y, int M, int N, int r) {
    extern __shared__ uint8_t ec_upd_smem[];
    float* us = reinterpret_cast<float*>(ec_upd_smem);                 // [32][r]
    __half* bs = reinterpret_cast<__half*>(us + 32 * r);               // [128][r + 2] (padded: conflict-free)
    const int m0 = blockIdx.y * 32, n0 = blockIdx.x * 128;
    const int tid = threadIdx.x;
    pdl_launch_dependents();
    pdl_wait();
    for (int i = tid; i < 32 * r; i += 256) {
        const int m = m0 + i / r;
        us[i] = m < M ? __half2float(u16[size_t(m) * r + (i % r)]) : 0.f;
    }
    const int rs = r + 2;
    for (int i = tid; i < 128 * r; i += 256) {
        const int nn = i / r, j = i - nn * r;
        bs[nn * rs + j] = B[size_t(n0 + nn) * r + j];
    }
    __syncthreads();
    const int nl = tid & 127, tg = tid >> 7;        // channel, token half (16 tokens each)
    float acc[16];
#pragma unroll
    for (int t = 0; t < 16; ++t) acc[t] = 0.f;
    for (int j = 0; j < r; ++j) {
        const float b = __half2float(bs[nl * rs + j]);
#pragma unroll
        for (int t = 0; t < 16; ++t) acc[t] = fmaf(us[(tg * 16 + t) * r + j], b, acc[t]);
    }
#pragma unroll
    for (int t = 0; t < 16; ++t) {
        const int m = m0 + tg * 16 + t;
        if (m < M) {
            __half* yp = y + size_t(m) * N + n0 + nl;
            *yp = __float2half_rn(__half2float(*yp) + acc[t]);
        }
    }
}

// INT8 EC factors on the M > 16 path: code * per-row scale -> fp16 scratch (one rounding; the tcgen05 path consumes fp16
// operand tiles through TMA).  r (K + N) elements per call, < 1 % of the layer's weight bytes.
__global__ void ec_dequant_i8_kernel(const int8_t* __restrict__ q, const __half* __restrict__ scale, __half* __restrict__ out,
                                     int rows, int cols) {
    const size_t n = size_t(rows) * cols;
    for (size_t i = (blockIdx.x * size_t(blockDim.x) + threadIdx.x) * 4; i < n; i += size_t(gridDim.x) * blockDim.x * 4) {
        const int row = int(i / cols);          // cols % 8 == 0: the four elements share a row
        const float s = __half2float(__ldg(scale + row));
        const char4 c = *reinterpret_cast<const char4*>(q + i);
        __half2 a = __floats2half2_rn(float(c.x) * s, float(c.y) * s), b = __floats2half2_rn(float(c.z) * s, float(c.w) * s);
        *reinterpret_cast<__half2*>(out + i) = a;
        *reinterpret_cast<__half2*>(out + i + 2) = b;
    }
}
int launch_ec_dequant_i8(const int8_t* q, const __half* scale, __half* out, int rows, int cols, cudaStream_t st) {
    const size_t n = size_t(rows) * cols;
    const int blocks = int(std::min<size_t>(1184, (n / 4 + 255) / 256));
    ec_dequant_i8_kernel<<<std::max(blocks, 1), 256, 0, st>>>(q, scale, out, rows, cols);
    SPEAR_CUDA_OK(cudaGetLastError());
    count_launch();
    return SPEAR_OK;
}

// ---- the post-EC tail as a row kernel, for the variants whose layer kernel does not fuse it ----------
// One CTA per token: y <- residual + y (one more rounding of the layer's output: the fused decode epilogue avoids it),
// mean of squares over the row from the fp32 sums, h_out <- y * rsqrt(mean + eps) * w.
__global__ void __launch_bounds__(256) tail_rows_kernel(__half* __restrict__ y, const __half* resid, const __half* __restrict__ w,
                                                        __half* __restrict__ h_out, float eps, int N) {
    __shared__ float red[8];
    __shared__ float inv_s;
    pdl_launch_dependents();
    pdl_wait();
    const size_t base = size_t(blockIdx.x) * N;
    float ssq = 0.f;
    for (int n = threadIdx.x * 2; n < N; n += 512) {
        const float2 a = __half22float2(*reinterpret_cast<const __half2*>(y + base + n));
        const float2 b = __half22float2(*reinterpret_cast<const __half2*>(resid + base + n));
        const float s0 = a.x + b.x, s1 = a.y + b.y;
        ssq += s0 * s0 + s1 * s1;
        *reinterpret_cast<__half2*>(y + base + n) = __floats2half2_rn(s0, s1);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) ssq += __shfl_xor_sync(0xffffffffu, ssq, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = ssq;
    __syncthreads();
    if (threadIdx.x == 0) {
        float t = 0.f;
        for (int i = 0; i < 8; ++i) t += red[i];
        inv_s = rsqrtf(t / float(N) + eps);
    }
    __syncthreads();
    const float inv = inv_s;
    for (int n = threadIdx.x * 2; n < N; n += 512) {       // the same elements this thread stored above
        const float2 a = __half22float2(*reinterpret_cast<const __half2*>(y + base + n));
        const float2 g = __half22float2(*reinterpret_cast<const __half2*>(w + n));
        *reinterpret_cast<__half2*>(h_out + base + n) = __floats2half2_rn(a.x * inv * g.x, a.y * inv * g.y);
    }
}
int launch_tail_rows(__half* y, const __half* resid, const __half* rms_w, __half* h_out, float eps, int M, int N, bool pdl, cudaStream_t st) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(M);
    cfg.blockDim = dim3(256);
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    SPEAR_CUDA_OK(cudaLaunchKernelEx(&cfg, tail_rows_kernel, y, resid, rms_w, h_out, eps, N));
    count_launch();
    return SPEAR_OK;
}

int launch_ec_update(const __half* u16, const __half* B, __half* y, int M, int N, int r, bool pdl, cudaStream_t st) {
    const size_t smem = size_t(32) * r * 4 + size_t(128) * (r + 2) * 2;
    static std::once_flag attr_once;
    static cudaError_t attr_err = cudaSuccess;
    std::call_once(attr_once, [] { attr_err = cudaFuncSetAttribute(ec_update_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024); });
    SPEAR_CUDA_OK(attr_err);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(N / 128, (M + 31) / 32);
    cfg.blockDim = dim3(256);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    SPEAR_CUDA_OK(cudaLaunchKernelEx(&cfg, ec_update_kernel, u16, B, y, M, N, r));
    count_launch();
    return SPEAR_OK;
}

}  // namespace spear

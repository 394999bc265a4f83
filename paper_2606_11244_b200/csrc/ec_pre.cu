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
        load_row32(pa0, col, a0l, a0h);
        load_row32(pa1, col, a1l, a1h);
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
            const float v = red[0][row][tok] + red[1][row][tok] + red[2][row][tok] + red[3][row][tok];
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
    const int r = p.r;
    if (p.gate_kind == SPEAR_GATE_SCALAR_SIGMOID) {
        const float bias = p.b_g ? *p.b_g : 0.f;
        for (int o = threadIdx.x; o < p.M * r; o += 128) {
            const int m = o / r, j = o - m * r;
            const float gam = 1.f / (1.f + expf(-(zs[m][r] + bias)));
            p.u[m * r + j] = p.alpha * gam * zs[m][j];
            if (p.gate_out && j == 0) p.gate_out[m] = gam;
        }
    } else if (p.gate_kind == SPEAR_GATE_MLP) {
        const int h = p.h;
        for (int i = threadIdx.x; i < h; i += 128) {
            float a[16];
#pragma unroll
            for (int m = 0; m < 16; ++m) a[m] = 0.f;
            const __half* w1 = p.W1 + size_t(i) * r;
            for (int j = 0; j < r; ++j) {
                const float w = __half2float(w1[j]);
#pragma unroll
                for (int m = 0; m < 16; ++m) a[m] = fmaf(w, zs[m][j], a[m]);
            }
            const float bb = p.b1[i];
#pragma unroll
            for (int m = 0; m < 16; ++m) hid[m][i] = fmaxf(a[m] + bb, 0.f);
        }
        __syncthreads();
        for (int j = threadIdx.x; j < r; j += 128) {
            float a[16];
#pragma unroll
            for (int m = 0; m < 16; ++m) a[m] = 0.f;
            const __half* w2 = p.W2 + size_t(j) * h;
            for (int i = 0; i < h; ++i) {
                const float w = __half2float(w2[i]);
#pragma unroll
                for (int m = 0; m < 16; ++m) a[m] = fmaf(w, hid[m][i], a[m]);
            }
            const float bb = p.b2[j];
            for (int m = 0; m < p.M; ++m) {
                const float gam = 1.f + tanhf(a[m] + bb);
                p.u[m * r + j] = p.alpha * gam * zs[m][j];
                if (p.gate_out) p.gate_out[m * r + j] = gam;
            }
        }
    } else {
        for (int o = threadIdx.x; o < p.M * r; o += 128) {
            const int m = o / r, j = o - m * r;
            p.u[m * r + j] = p.alpha * zs[m][j];
        }
    }
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

}  // namespace spear

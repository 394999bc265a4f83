// pack.cu -- S0 of SURVEY.md 8(a): canonical int4 codes + fp16 scales <-> the SPW4 packed layout
// (DESIGN.md section 2), plus the two test hooks (unpack, dequantise to fp16).
//
// W4 format: PAPER.md:247, :585 (4-bit codes, per-group or per-channel scale); zero-point 8 and fp16
// scales are fixed by BASELINE.json (reading A4).  All kernels here are bit-exact integer / one-rounding
// work: one thread per 32-bit packed word (8 codes of one row).
#include "common.cuh"

namespace spear {

// word index -> (n, k of its first code)
__device__ __forceinline__ void word_to_nk(size_t w, int K, int& n, int& k) {
    const int wd = w & 1, hi = (w >> 1) & 1, lane = (w >> 2) & 31, s = (w >> 7) & 7;
    const size_t blk = w >> 10;             // p * (K/64) + kt
    const int ktiles = K >> 6;
    const int p = int(blk / ktiles), kt = int(blk % ktiles);
    const int g = lane >> 2, t = lane & 3;
    n = p * 128 + s * 16 + hi * 8 + g;
    k = kt * 64 + t * 16 + wd * 8;
}

__global__ void pack_w4_kernel(const uint8_t* __restrict__ codes, uint32_t* __restrict__ wq, int N,
                               int K, int* __restrict__ bad_flag) {
    const size_t nwords = size_t(N) * K / 8;
    for (size_t w = blockIdx.x * size_t(blockDim.x) + threadIdx.x; w < nwords;
         w += size_t(gridDim.x) * blockDim.x) {
        int n, k;
        word_to_nk(w, K, n, k);
        const uint2 c8 = *reinterpret_cast<const uint2*>(codes + size_t(n) * K + k);
        if ((c8.x | c8.y) & 0xf0f0f0f0u) *bad_flag = 1;
        // column e goes to slot (e >> 1) + 4 * (e & 1): even columns in the low half-word.
        uint32_t word = 0;
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            const uint32_t c = ((e < 4 ? c8.x : c8.y) >> (8 * (e & 3))) & 0xf;
            word |= c << (4 * ((e >> 1) + 4 * (e & 1)));
        }
        wq[w] = word;
    }
}

__global__ void pack_scales_kernel(const __half* __restrict__ scales, __half* __restrict__ out, int N,
                                   int G) {
    const size_t total = size_t(N) * G;
    for (size_t i = blockIdx.x * size_t(blockDim.x) + threadIdx.x; i < total;
         i += size_t(gridDim.x) * blockDim.x) {
        const int n = int(i / G), grp = int(i % G);
        const int p = n >> 7, s = (n & 127) >> 4, g = n & 7, hi = (n & 15) >> 3;
        out[(size_t(p) * G + grp) * 128 + s * 16 + 2 * g + hi] = scales[i];
    }
}

__global__ void unpack_w4_kernel(const uint32_t* __restrict__ wq, uint8_t* __restrict__ codes, int N,
                                 int K) {
    const size_t nwords = size_t(N) * K / 8;
    for (size_t w = blockIdx.x * size_t(blockDim.x) + threadIdx.x; w < nwords;
         w += size_t(gridDim.x) * blockDim.x) {
        int n, k;
        word_to_nk(w, K, n, k);
        const uint32_t word = wq[w];
        uint2 c8 = make_uint2(0, 0);
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            const uint32_t c = (word >> (4 * ((e >> 1) + 4 * (e & 1)))) & 0xf;
            if (e < 4) c8.x |= c << (8 * e); else c8.y |= c << (8 * (e - 4));
        }
        *reinterpret_cast<uint2*>(codes + size_t(n) * K + k) = c8;
    }
}

// What16[n][k] = RN_fp16((q - 8) * s): (q - 8) is formed exactly in fp16, then one rounding multiply.
__global__ void dequant_w4_kernel(const uint32_t* __restrict__ wq, const __half* __restrict__ sp,
                                  __half* __restrict__ out, int N, int K, int group) {
    const size_t nwords = size_t(N) * K / 8;
    const int G = K / group;
    for (size_t w = blockIdx.x * size_t(blockDim.x) + threadIdx.x; w < nwords;
         w += size_t(gridDim.x) * blockDim.x) {
        int n, k;
        word_to_nk(w, K, n, k);
        const int p = n >> 7, s = (n & 127) >> 4, g = n & 7, hi = (n & 15) >> 3;
        const __half sc = sp[(size_t(p) * G + k / group) * 128 + s * 16 + 2 * g + hi];
        const uint32_t sc2 = uint32_t(__half_as_ushort(sc)) * 0x00010001u;
        uint32_t q[4];
        dequant_word(wq[w], q);
        uint4 v;
        v.x = hmul2_u32(q[0], sc2);
        v.y = hmul2_u32(q[1], sc2);
        v.z = hmul2_u32(q[2], sc2);
        v.w = hmul2_u32(q[3], sc2);
        *reinterpret_cast<uint4*>(out + size_t(n) * K + k) = v;
    }
}

static int check_shape(int N, int K, int group) {
    if (N <= 0 || K <= 0 || group <= 0)
        return set_error(SPEAR_EINVAL, "N, K, group must be positive (N=%d K=%d group=%d)", N, K, group);
    if (N % 128 || K % 128 || group % 128 || K % group)
        return set_error(SPEAR_EUNSUPPORTED,
                         "need N%%128==0, K%%128==0, group%%128==0, K%%group==0 (N=%d K=%d group=%d)",
                         N, K, group);
    return SPEAR_OK;
}

static int grid_for(size_t items, int block) {
    size_t g = (items + block - 1) / block;
    const size_t cap = size_t(device_info().num_sms) * 16;
    return int(g < 1 ? 1 : (g > cap ? cap : g));
}

}  // namespace spear

using namespace spear;

extern "C" int spear_pack_w4_sizes(int N, int K, int group, size_t* wq_bytes, size_t* scales_bytes) {
    if (int rc = check_shape(N, K, group)) return rc;
    if (wq_bytes) *wq_bytes = size_t(N) * K / 2;
    if (scales_bytes) *scales_bytes = size_t(N) * (K / group) * 2;
    return SPEAR_OK;
}

extern "C" int spear_pack_w4(const uint8_t* codes, const void* scales, void* wq_out, void* scales_out,
                             int N, int K, int group, void* stream) {
    if (int rc = check_shape(N, K, group)) return rc;
    if (!codes || !scales || !wq_out || !scales_out) return set_error(SPEAR_EINVAL, "NULL pointer");
    if ((uintptr_t(codes) | uintptr_t(scales) | uintptr_t(wq_out) | uintptr_t(scales_out)) & 15)
        return set_error(SPEAR_EINVAL, "pointers must be 16-byte aligned");
    if (int rc = spear_init()) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int* flag = nullptr;
    SPEAR_CUDA_OK(cudaMalloc(&flag, sizeof(int)));
    cudaMemsetAsync(flag, 0, sizeof(int), st);
    const size_t nwords = size_t(N) * K / 8;
    pack_w4_kernel<<<grid_for(nwords, 256), 256, 0, st>>>(codes, static_cast<uint32_t*>(wq_out), N, K, flag);
    pack_scales_kernel<<<grid_for(size_t(N) * (K / group), 256), 256, 0, st>>>(
        static_cast<const __half*>(scales), static_cast<__half*>(scales_out), N, K / group);
    count_launch(2);
    int bad = 0;
    cudaError_t e = cudaMemcpyAsync(&bad, flag, sizeof(int), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(flag);
    if (e != cudaSuccess) return set_error(SPEAR_ECUDA, "spear_pack_w4: %s", cudaGetErrorString(e));
    if (bad) return set_error(SPEAR_EINVAL, "spear_pack_w4: a code is > 15");
    return SPEAR_OK;
}

extern "C" int spear_unpack_w4(const void* wq, uint8_t* codes_out, int N, int K, int group, void* stream) {
    if (int rc = check_shape(N, K, group)) return rc;
    if (!wq || !codes_out) return set_error(SPEAR_EINVAL, "NULL pointer");
    if (int rc = spear_init()) return rc;
    const size_t nwords = size_t(N) * K / 8;
    unpack_w4_kernel<<<grid_for(nwords, 256), 256, 0, static_cast<cudaStream_t>(stream)>>>(
        static_cast<const uint32_t*>(wq), codes_out, N, K);
    count_launch();
    SPEAR_CUDA_OK(cudaGetLastError());
    return SPEAR_OK;
}

extern "C" int spear_dequant_w4(const void* wq, const void* scales_packed, void* w_fp16_out, int N, int K,
                                int group, void* stream) {
    if (int rc = check_shape(N, K, group)) return rc;
    if (!wq || !scales_packed || !w_fp16_out) return set_error(SPEAR_EINVAL, "NULL pointer");
    if (int rc = spear_init()) return rc;
    const size_t nwords = size_t(N) * K / 8;
    dequant_w4_kernel<<<grid_for(nwords, 256), 256, 0, static_cast<cudaStream_t>(stream)>>>(
        static_cast<const uint32_t*>(wq), static_cast<const __half*>(scales_packed),
        static_cast<__half*>(w_fp16_out), N, K, group);
    count_launch();
    SPEAR_CUDA_OK(cudaGetLastError());
    return SPEAR_OK;
}

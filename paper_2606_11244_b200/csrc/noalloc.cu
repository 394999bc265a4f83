// noalloc.cu -- spear_w4_ec_gemm_noalloc: the decode layer (Eq. 3) for callers that cannot allocate.
//
// Some callers may not call cudaMalloc at all: code under CUDA graph capture, tight serving loops, harnesses that forbid
// it.  Every other entry point of the library goes through spear_init (which allocates the library's workspaces once) or
// takes a caller-provided workspace.  This one needs neither: the scratch memory of its EC pre-pass -- the fp32 z
// accumulators [16][kZStride], the arrival counter and u = alpha gamma (.) z as fp32 [16][128] -- lives in a file-scope
// static __device__ array of kNoAllocScratchBytes = 17,152 bytes (every GPU that loads the library holds it until exit).
// The maxima it is sized for are the path's own: M <= 16 tokens, r <= 128.  Larger problems are refused, not served.
//
// Path: ec_pre_kernel (z = x [A; w_g]^T, any gate incl. the paper's MLP gate, u) -> rows_kernel (one CTA per 16 output
// rows over the whole of K, adds u B^T, one cast).  Both exist already (ec_pre.cu, rows.cu); here they are handed
// pointers into the static array.  No tensor map, no plan table, no lanes: nothing on this path allocates on the host
// or on the device, and spear_init is NOT called.
//
// The array's name is a host-side stand-in in host code, not a device address: its address is taken once per device with
// cudaGetSymbolAddress (that device current) and only that pointer is passed to kernels.
//
// Sharing: every call on a device uses the same array, and it keeps the last call's contents.  z and the counter must
// start at zero: they are cleared stream-ordered at the head of every call (the kernels also leave them zero, but a call
// must not trust its predecessor).  u is fully overwritten for the tokens / ranks the call reads.  Two calls that overlap
// on the GPU (different streams, or graph branches without an edge between them) RACE on the array: serialise them.
#include <algorithm>
#include <mutex>

#include "common.cuh"
#include "kernels.h"

namespace spear {
namespace {

constexpr int kNoAllocMaxM = 16;
constexpr int kNoAllocMaxR = 128;
constexpr size_t kZBytes = size_t(16) * kZStride * 4;                 // 8704
constexpr size_t kCtrOff = kZBytes;                                   // arrival counter (+ padding to 256 bytes)
constexpr size_t kUOff = kCtrOff + 256;                               // 8960
constexpr size_t kNoAllocScratchBytes = kUOff + size_t(kNoAllocMaxM) * kNoAllocMaxR * 4;     // 17152
static_assert(kZBytes % 256 == 0 && kUOff % 256 == 0, "sub-buffers stay 256-byte aligned");
static_assert(kZStride >= kNoAllocMaxR + 1, "z row holds r values and the scalar gate's pre-activation");

static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocScratchBytes];

constexpr int kMaxDevices = 64;
struct DeviceSlot {
    unsigned char* scratch = nullptr;      // device address of g_noalloc_scratch on this device
    int num_sms = 0;
};
DeviceSlot g_slots[kMaxDevices];
std::mutex g_slots_mutex;

// Once per device, with that device current (the caller's current device: the one its pointers and stream belong to).
int device_slot(const DeviceSlot** out) {
    int dev = -1;
    SPEAR_CUDA_OK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return set_error(SPEAR_EUNSUPPORTED, "spear_w4_ec_gemm_noalloc: device ordinal %d (supported: 0..%d)", dev, kMaxDevices - 1);
    std::lock_guard<std::mutex> lock(g_slots_mutex);
    DeviceSlot& s = g_slots[dev];
    if (!s.scratch) {
        void* p = nullptr;
        SPEAR_CUDA_OK(cudaGetSymbolAddress(&p, g_noalloc_scratch));
        if (!p || (uintptr_t(p) & 255)) return set_error(SPEAR_ECUDA, "spear_w4_ec_gemm_noalloc: bad address %p for the static scratch array", p);
        int sms = 0;
        SPEAR_CUDA_OK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        s.num_sms = sms > 0 ? sms : 1;
        s.scratch = static_cast<unsigned char*>(p);
    }
    *out = &s;
    return SPEAR_OK;
}

}  // namespace
}  // namespace spear

using namespace spear;

extern "C" int spear_w4_ec_gemm_noalloc(const void* x, const void* Wq, const void* scales, const void* A, const void* B,
                                        const spear_ec_desc* ec, void* y,
                                        int M, int N, int K, int r, int group, void* stream) {
    // ---- the limits of the static scratch first, with their own message ----
    if (M > kNoAllocMaxM)
        return set_error(SPEAR_EUNSUPPORTED, "spear_w4_ec_gemm_noalloc: M = %d exceeds the maximum of %d tokens its static scratch (%zu bytes) is sized for; "
                         "use spear_w4_ec_gemm_ex", M, kNoAllocMaxM, kNoAllocScratchBytes);
    if (r > kNoAllocMaxR)
        return set_error(SPEAR_EUNSUPPORTED, "spear_w4_ec_gemm_noalloc: r = %d exceeds the maximum rank %d its static scratch (%zu bytes) is sized for",
                         r, kNoAllocMaxR, kNoAllocScratchBytes);
    if (M < 1 || N < 1 || K < 1 || group < 1 || r < 0)
        return set_error(SPEAR_EINVAL, "spear_w4_ec_gemm_noalloc: bad sizes M=%d N=%d K=%d r=%d group=%d", M, N, K, r, group);
    if (N % 128 || K % 128 || group % 128 || K % group)
        return set_error(SPEAR_EUNSUPPORTED, "spear_w4_ec_gemm_noalloc: need N%%128==0, K%%128==0, group%%128==0, K%%group==0 (N=%d K=%d group=%d)", N, K, group);
    if (r % 8) return set_error(SPEAR_EUNSUPPORTED, "spear_w4_ec_gemm_noalloc: need r%%8==0 (r=%d)", r);
    if (!x || !Wq || !scales || !y) return set_error(SPEAR_EINVAL, "spear_w4_ec_gemm_noalloc: NULL x / Wq / scales / y");
    if (x == y) return set_error(SPEAR_EINVAL, "spear_w4_ec_gemm_noalloc: x and y must not alias");
    uintptr_t al = uintptr_t(x) | uintptr_t(Wq) | uintptr_t(scales) | uintptr_t(y);
    bool int8 = false;
    if (r > 0) {
        if (!A || !B || !ec) return set_error(SPEAR_EINVAL, "spear_w4_ec_gemm_noalloc: r > 0 needs A, B and the EC descriptor");
        al |= uintptr_t(A) | uintptr_t(B);
        if (ec->ec_dtype == SPEAR_EC_INT8) {
            if (!ec->A_scale || !ec->B_scale) return set_error(SPEAR_EINVAL, "spear_w4_ec_gemm_noalloc: INT8 EC factors need A_scale[r] and B_scale[N]");
            int8 = true;
        } else if (ec->ec_dtype != SPEAR_EC_FP16) {
            return set_error(SPEAR_EINVAL, "spear_w4_ec_gemm_noalloc: unknown ec_dtype %d", ec->ec_dtype);
        }
        if (ec->gate_kind == SPEAR_GATE_SCALAR_SIGMOID) {
            if (!ec->w_g) return set_error(SPEAR_EINVAL, "spear_w4_ec_gemm_noalloc: scalar gate needs w_g");
            al |= uintptr_t(ec->w_g);
        } else if (ec->gate_kind == SPEAR_GATE_MLP) {
            if (!ec->W1 || !ec->b1 || !ec->W2 || !ec->b2) return set_error(SPEAR_EINVAL, "spear_w4_ec_gemm_noalloc: MLP gate needs W1, b1, W2, b2");
            if (ec->gate_hidden < 1 || ec->gate_hidden > 512 || ec->gate_hidden % 8)
                return set_error(SPEAR_EUNSUPPORTED, "spear_w4_ec_gemm_noalloc: MLP gate needs 8 <= h <= 512, h%%8==0 (h=%d)", ec->gate_hidden);
            al |= uintptr_t(ec->W1) | uintptr_t(ec->W2);
        } else if (ec->gate_kind != SPEAR_GATE_NONE) {
            return set_error(SPEAR_EINVAL, "spear_w4_ec_gemm_noalloc: unknown gate kind %d", ec->gate_kind);
        }
    }
    if (al & 15) return set_error(SPEAR_EINVAL, "spear_w4_ec_gemm_noalloc: device pointers must be 16-byte aligned");

    const DeviceSlot* slot = nullptr;
    if (int rc = device_slot(&slot)) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    float* zbuf = reinterpret_cast<float*>(slot->scratch);
    unsigned* counter = reinterpret_cast<unsigned*>(slot->scratch + kCtrOff);
    float* u = reinterpret_cast<float*>(slot->scratch + kUOff);

    if (r > 0) {
        // z and the counter start at zero whatever the previous call (or an aborted one) left behind
        SPEAR_CUDA_OK(cudaMemsetAsync(slot->scratch, 0, kUOff, st));
        EcPreParams e = {};
        e.x = static_cast<const __half*>(x);
        e.A = static_cast<const __half*>(A);
        e.ec_int8 = int8 ? 1 : 0;
        e.A_scale = static_cast<const __half*>(ec->A_scale);
        e.w_g = static_cast<const __half*>(ec->w_g);
        e.b_g = static_cast<const float*>(ec->b_g);
        e.W1 = static_cast<const __half*>(ec->W1);
        e.b1 = static_cast<const float*>(ec->b1);
        e.W2 = static_cast<const __half*>(ec->W2);
        e.b2 = static_cast<const float*>(ec->b2);
        e.zbuf = zbuf;
        e.u = u;
        e.gate_out = static_cast<float*>(ec->gate_out);
        e.counter = counter;
        e.M = M; e.K = K; e.r = r; e.h = ec->gate_hidden; e.gate_kind = ec->gate_kind;
        e.alpha = ec->alpha;
        const int strips = (r + (ec->gate_kind == SPEAR_GATE_SCALAR_SIGMOID ? 1 : 0) + 15) / 16;
        const int ktiles = K / 64;
        const int ksplit = std::max(1, std::min(ktiles / 4, slot->num_sms / strips));
        e.ksplit = std::max(1, std::min(ksplit, ktiles));
        if (int rc = launch_ec_pre(e, /*pdl=*/false, st)) return rc;      // plain stream order behind the memset
    }
    RowsParams p = {};
    p.wq = Wq; p.scales = scales;
    p.x = static_cast<const __half*>(x);
    p.y = static_cast<__half*>(y);
    p.u = u;
    p.B = B;
    if (int8) { p.ec_int8 = 1; p.B_scale = static_cast<const __half*>(ec->B_scale); }
    p.M = M; p.N = N; p.K = K; p.r = r; p.G = K / group; p.group = group;
    p.fused = 0;                                                           // u comes from the pre-kernel through the static array
    return launch_rows(p, /*pdl=*/r > 0, st);     // its weight requests overlap the pre-kernel's tail; u is read after griddepcontrol.wait
}

/*
 * spear.h -- C ABI of libspear.so: the SPEAR W4A16 + per-token-gated Error Compensator layer
 * on one NVIDIA B200 (sm_100a).
 *
 * The operation (PAPER.md:107-110, Eq. 3; shapes PAPER.md:118; W4 format PAPER.md:247, :585):
 *
 *     y[m][n] = sum_k x[m][k] * What[n][k]  +  alpha * sum_j B[n][j] * gamma[m][j] * z[m][j]
 *     What[n][k] = (q[n][k] - 8) * s[n][k / group]              q in 0..15, zero-point 8, fp16 scale
 *     z[m][j]    = sum_k A[j][k] * x[m][k]                      "Ax"
 *     gamma      = 1 + tanh(W2 relu(W1 z + b1) + b2)            SPEAR_GATE_MLP
 *     gamma[m][*]= 1 / (1 + exp(-(x[m] . w_g + b)))             SPEAR_GATE_SCALAR_SIGMOID (BASELINE.json configs)
 *     gamma      = 1                                            SPEAR_GATE_NONE    (Eq. 2)
 *
 * Canonical layouts: row-major, contiguous.  x[M][K] fp16, q[N][K] uint8, s[N][K/group] fp16,
 * A[r][K] fp16, B[N][r] fp16, y[M][N] fp16 (orientation as in the paper: What in R^{d_out x d_in},
 * A in R^{r x d_in}, B in R^{d_out x r}).  Accumulation is fp32, y is rounded to fp16 once (RN-even).
 *
 * Conventions for every entry point
 *   - returns 0 (SPEAR_OK) or a negative spear_status; never throws, never exits;
 *     spear_last_error() gives a thread-local message for the last non-zero status;
 *   - every data pointer is a DEVICE pointer, 16-byte aligned, owned by the caller, unless the
 *     argument is documented as "host";
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream);
 *   - work is enqueued on `stream` and the call returns without synchronising, except
 *     spear_pack_w4 (reads back a validity flag), spear_plan (measures) and spear_init;
 *   - supported shapes: M >= 1, N % 128 == 0, K % 128 == 0, group % 128 == 0, K % group == 0,
 *     0 <= r <= 128 with r % 8 == 0 (pad A with zero rows and B with zero columns: exact);
 *     anything else returns SPEAR_EUNSUPPORTED.  x and y must not alias.
 *   - there is no CPU path: without a CUDA device every compute call returns SPEAR_ECUDA.
 */
#ifndef SPEAR_H
#define SPEAR_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    SPEAR_OK = 0,
    SPEAR_EINVAL = -1,        /* bad argument (NULL pointer, misaligned, code > 15, ...)            */
    SPEAR_EUNSUPPORTED = -2,  /* shape outside the supported set above                              */
    SPEAR_ECUDA = -3,         /* a CUDA runtime call failed (message in spear_last_error)           */
    SPEAR_ENOMEM = -4         /* workspace too small / allocation failed                            */
} spear_status;

typedef enum {
    SPEAR_GATE_SCALAR_SIGMOID = 0,
    SPEAR_GATE_MLP = 1,
    SPEAR_GATE_NONE = 2
} spear_gate_kind;

/* Execution variants.  AUTO consults the table filled by spear_plan and
 * otherwise a size heuristic. */
typedef enum { SPEAR_EC_FP16 = 0, SPEAR_EC_INT8 = 1 } spear_ec_dtype;

typedef enum {
    SPEAR_VARIANT_AUTO = 0,
    SPEAR_VARIANT_STREAM_FUSED = 1,  /* one kernel: weight stream (mma.sync) + x.A^T, gate, B add inside; M <= 16, scalar / none gate */
    SPEAR_VARIANT_STREAM_SPLIT = 2,  /* EC pre-kernel (z, any gate, u) then weight-stream kernel adding u.B^T; M <= 16 */
    SPEAR_VARIANT_TC_FUSED = 3,      /* EC pre-kernel + tcgen05 GEMM with [X|U].[What|B]^T K-concatenation; any M */
    SPEAR_VARIANT_TC_SPLIT = 4,      /* EC pre-kernel + tcgen05 GEMM (plain W4) + a separate rank-r update pass over y (the
                                        paper's unfused comparator; y is rounded twice); any M, r > 0 */
    SPEAR_VARIANT_LSTREAM = 5,       /* persistent layer-stream kernel (tcgen05, weights through TMEM), EC fused; M <= 16,
                                        scalar / none gate; also what spear_w4_ec_gemm_batch runs for such calls */
    SPEAR_VARIANT_ROWS = 6,          /* EC pre-kernel (r > 0) + row-strip kernel: one CTA per 16 output rows over the whole of K, no
                                        cross-CTA reduction; M <= 16 on the latency-bound (small) layers, and a 32-token form for 17..64 tokens (fp16 EC factors) */
    SPEAR_VARIANT_COUNT = 7
} spear_variant;

/* ---- S0: packing (the "SPW4" layout) -------------------------------- */

/* Sizes in bytes of the opaque packed buffers: wq = N*K/2, scales = 2*N*(K/group). */
int spear_pack_w4_sizes(int N, int K, int group, size_t* wq_bytes, size_t* scales_bytes);

/* Canonical -> packed.  codes[N][K] uint8 in 0..15 (any code > 15 -> SPEAR_EINVAL, outputs
 * undefined), scales[N][K/group] fp16.  Bit-exact and deterministic.  Synchronises `stream`. */
int spear_pack_w4(const uint8_t* codes, const void* scales, void* wq_out, void* scales_out,
                  int N, int K, int group, void* stream);

/* Test hooks: packed -> canonical codes; packed -> fp16 weights What16[N][K] = RN_fp16((q-8)*s),
 * computed as the exact fp16 (q-8) times s with one rounding (bit-exact against the oracle). */
int spear_unpack_w4(const void* wq, uint8_t* codes_out, int N, int K, int group, void* stream);
int spear_dequant_w4(const void* wq, const void* scales_packed, void* w_fp16_out,
                     int N, int K, int group, void* stream);

/* ---- the layer --------------------------------------------------------------------------- */

/* The call BASELINE.json names, argument order verbatim.  Gate = scalar sigmoid, alpha = 1:
 * gate_w = w_g[K] fp16, gate_b = pointer to ONE fp32 on the device.  r == 0 (A, B, gate_* may
 * then be NULL) is the plain W4 layer.  Wq / scales are the packed buffers of spear_pack_w4.
 * Uses the library's default workspace (spear_init): calls sharing it must be stream-ordered
 * with respect to each other. */
int spear_w4_ec_gemm(const void* x, const void* Wq, const void* scales, const void* A, const void* B,
                     const void* gate_w, const void* gate_b, void* y,
                     int M, int N, int K, int r, int group, void* stream);

/* Extended form: everything the paper's EC needs that the 14-argument form cannot express. */
typedef struct {
    int gate_kind;            /* spear_gate_kind                                                    */
    int gate_hidden;          /* h, MLP gate only (8 <= h <= 512, h % 8 == 0; reading A2: default 4r) */
    float alpha;              /* Eq. 3 alpha (reading A3)                                           */
    const void* W1;           /* [h][r] fp16   MLP gate                                             */
    const void* b1;           /* [h]    fp32                                                        */
    const void* W2;           /* [r][h] fp16                                                        */
    const void* b2;           /* [r]    fp32                                                        */
    const void* w_g;          /* [K]    fp16   scalar gate                                          */
    const void* b_g;          /* 1      fp32   scalar gate (device pointer; NULL = 0)               */
    void* gate_out;           /* optional: MLP -> [M][r] fp32, scalar -> [M] fp32; NULL = not written */
    void* workspace;          /* NULL = library default; else 1024-byte aligned, >= spear_workspace_bytes(),
                                 zero-filled once by the caller before first use (the library keeps its
                                 counters and accumulators zero between calls).  Every call sharing one
                                 buffer must pass the same workspace_bytes (a scratch region is placed
                                 relative to the END of the buffer).                                    */
    size_t workspace_bytes;
    int force_variant;        /* spear_variant; SPEAR_VARIANT_AUTO = use the plan                   */
    int ec_dtype;             /* spear_ec_dtype: storage of A and B.  SPEAR_EC_INT8 = "INT8 per-channel symmetric"
                                 (PAPER.md:603): A is int8 [r][K], B is int8 [N][r], Ahat[j][k] = A[j][k] * A_scale[j],
                                 Bhat[n][j] = B[n][j] * B_scale[n] (reading A17)                                        */
    const void* A_scale;      /* [r] fp16, SPEAR_EC_INT8 only                                        */
    const void* B_scale;      /* [N] fp16, SPEAR_EC_INT8 only                                        */
} spear_ec_desc;

int spear_w4_ec_gemm_ex(const void* x, const void* Wq, const void* scales, const void* A, const void* B,
                        const spear_ec_desc* ec, void* y,
                        int M, int N, int K, int r, int group, void* stream);

/* The layer followed by the rest of the paper's fused post-EC tail ("residual addition, and next-layer
 * RMSNorm ... as a single fused tail"):
 *     y[m][n]     = residual[m][n] + (What x + alpha B (gamma (.) A x))[m][n]          the new residual stream, fp16
 *     h_out[m][n] = y[m][n] / sqrt(mean_n(y[m][:]^2) + eps) * rms_weight[n]            input of the next layer, fp16
 * Both are formed from the fp32 accumulators (one rounding each; the mean of squares is taken before rounding).  For
 * M <= 16 on the weight-stream variants this happens inside the layer kernel's epilogue (the row-wide mean needs every
 * output panel: arrive / wait across the co-resident CTAs of a cooperative launch); the other variants run the layer and a
 * row kernel; AUTO therefore keeps M <= 16 on the weight-stream variants when a tail is asked for.
 * residual [M][N] fp16, rms_weight [N] fp16, h_out [M][N] fp16 (must not alias y or x).  residual == y (the residual
 * stream updated in place) is supported where the tail is fused -- M <= 16, SPEAR_VARIANT_AUTO / STREAM_FUSED /
 * STREAM_SPLIT; on every other arm (M > 16, or a forced ROWS / LSTREAM / TC variant) the layer kernel has stored y before
 * the row kernel reads residual, so an aliased or partly overlapping residual is rejected with SPEAR_EINVAL. */
typedef struct {
    const void* residual;
    const void* rms_weight;
    float eps;
    void* h_out;
} spear_tail_desc;
int spear_w4_ec_gemm_tail(const void* x, const void* Wq, const void* scales, const void* A, const void* B,
                          const spear_ec_desc* ec, const spear_tail_desc* tail, void* y,
                          int M, int N, int K, int r, int group, void* stream);

/* The decode layer for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): same operation and argument meaning as spear_w4_ec_gemm_ex (Eq. 3; any gate, fp16 or
 * INT8 EC factors), limited to M <= 16 tokens and r <= 128, and this call -- unlike every other entry point -- never
 * calls cudaMalloc / cudaFree, spear_init or any allocating routine, on the first call or later.  Its scratch (fp32 z
 * [16][136], a counter, u [16][128]: 17,152 bytes) is a static __device__ array inside the library, held by every GPU
 * that loads the library until exit.  ec->workspace, ec->force_variant and the plan table are ignored; the path is the EC
 * pre-kernel followed by the row-strip kernel.  Sizes beyond the limits return SPEAR_EUNSUPPORTED with a message naming
 * the limit.  All calls on a device share the array: z and the counter are cleared (stream-ordered) at the head of each
 * call, u is overwritten; calls that overlap on the GPU (different streams, unordered graph branches) race -- serialise
 * them.  Uses the caller's current device; the pointers and the stream must belong to it. */
int spear_w4_ec_gemm_noalloc(const void* x, const void* Wq, const void* scales, const void* A, const void* B,
                             const spear_ec_desc* ec, void* y,
                             int M, int N, int K, int r, int group, void* stream);

/* A batch of layer calls, e.g. the projections of one or several transformer blocks, or unrelated requests.
 * Independent calls run concurrently on the library's internal lanes (up to 16 streams with their own workspaces), or --
 * for M <= 16, when spear_plan_batch measured it faster or spear_tune("lstream", 1) -- as ONE persistent layer-stream
 * launch.  A call may read an earlier call's y as its x (same pointer, same M, K == that call's N): such chains are
 * ordered (one after the other on `stream`, or as dependency phases inside the layer-stream launch).  Everything is
 * ordered after the work already enqueued on `stream` and before anything enqueued on it afterwards (capturable in a
 * CUDA graph).  ec->workspace must be NULL.  The
 * per-token-gated EC of every call is evaluated exactly as in spear_w4_ec_gemm_ex. */
typedef struct {
    const void *x, *Wq, *scales, *A, *B;
    const spear_ec_desc* ec;    /* may be NULL when r == 0 */
    void* y;
    int M, N, K, r, group;
} spear_call;
int spear_w4_ec_gemm_batch(const spear_call* calls, int n_calls, void* stream);

/* The same batch with HOST activations: for call i, io[i].x_host [M][K] fp16 is copied to calls[i].x (the device
 * staging buffer the caller provides), the layer runs, and calls[i].y is copied back to io[i].y_host [M][N] --
 * all on that call's lane, inside the fork / join (preferably pinned host memory; the end-to-end path bench.py
 * times).  The host buffers are valid once `stream` has been synchronised. */
typedef struct {
    const void* x_host;
    void* y_host;
} spear_host_io;
int spear_w4_ec_gemm_batch_hostio(const spear_call* calls, const spear_host_io* io, int n_calls, void* stream);

/* Same layer with HOST activations: x_host[M][K] and y_host[M][N] are (preferably pinned) host
 * buffers; x is copied to x_dev, the layer runs, y_dev is copied back, all on `stream` (the end-
 * to-end path bench.py times).  Weights and EC parameters stay device-resident. */
int spear_w4_ec_gemm_hostio(const void* x_host, void* y_host, void* x_dev, void* y_dev,
                            const void* Wq, const void* scales, const void* A, const void* B,
                            const spear_ec_desc* ec, int M, int N, int K, int r, int group, void* stream);

/* Workspace a call of this shape may need (upper bound over variants). */
int spear_workspace_bytes(int M, int N, int K, int r, int group, size_t* bytes);

/* Allocates (once per process, current device) and zero-fills the library's own device memory and reads the device
 * properties: the default workspace (96 MiB), 16 batch lanes (a stream + 48 MiB workspace each) and the layer-stream
 * kernel's workspace (~40 MiB: split-K accumulators, counters, EC state, 32 MiB of x in the MMA operand layout) --
 * spear_memory_bytes() reports the total.  No compute call allocates anything after that; a caller who wants to own
 * the memory passes spear_ec_desc.workspace (single calls).  Called implicitly by the first compute call; call it
 * explicitly before capturing a CUDA graph.  Synchronises the device. */
int spear_init(void);
int spear_memory_bytes(size_t* bytes);   /* device bytes spear_init allocates */

/* ---- S9: measured dispatch ---------------------------------------------------------------- */

/* Times every variant valid for this problem on synthetic device buffers it allocates itself
 * (PAPER.md:274 protocol scaled down: warm-up then the median of timed launches, CUDA events),
 * records the fastest in the process-wide table and returns it.  times_us_out (host, may be
 * NULL) receives SPEAR_VARIANT_COUNT medians in microseconds (negative = variant not valid).
 * Synchronises. */
int spear_plan(int M, int N, int K, int r, int group, int gate_kind, int gate_hidden,
               int* chosen_variant_out, float* times_us_out, void* stream);
int spear_plan_save(const char* path);   /* text file, one line per planned problem (host path) */
int spear_plan_load(const char* path);
/* S9 for batches: times the two ways of running THIS batch of M <= 16 calls on the caller's own
 * buffers (the y buffers are overwritten) -- 0: per-call kernels (concurrent lanes, or one after the other when calls read
 * each other's y), 1: ONE persistent layer-stream launch -- and records the winner for every later batch with the same
 * shapes.  times_us_out[2] (host, may be NULL): microseconds per batch, negative = not applicable.  Synchronises. */
int spear_plan_batch(const spear_call* calls, int n_calls, int* chosen_out, float* times_us_out, void* stream);
/* The variant AUTO would run for this problem right now (table hit or heuristic). */
int spear_plan_query(int M, int N, int K, int r, int group, int gate_kind, int* variant_out);

/* ---- PAPER.md 4.3: latency look-up tables and SLO-constrained chunk selection (host only) ------------ */

/* per layer type t the offline tables l_W4[t](M), l_EC[t](M) (microseconds) on a sparse, strictly
 * increasing grid of token counts M_grid[n_grid], row-major [n_types][n_grid]; lat_attn_us[n_grid] is the attention
 * table the caller profiled (NULL = no attention term: this library has no attention kernel).  Tables are copied; an
 * entry smaller than its predecessor is raised to it (T_S must be monotone for the binary search of PAPER.md:237). */
typedef struct spear_lut spear_lut;
int spear_lut_create(const int* M_grid, int n_grid, int n_types, const float* lat_w4_us, const float* lat_ec_us,
                     const float* lat_attn_us, spear_lut** out);
void spear_lut_destroy(spear_lut* lut);
/* PAPER.md:231 online aggregator: T_S(M) = sum over the n_modules linear layers of (selected[m] ? l_EC : l_W4)[type[m]](M)
 * + n_attn_layers * l_attn(M), linear interpolation between grid points (first entry below the grid, last segment
 * extended above it, T_S(0) = 0).  selected may be NULL (no EC anywhere).  All pointers are host pointers. */
int spear_lut_iteration_us(const spear_lut* lut, const int* module_type, const unsigned char* selected, int n_modules,
                           int n_attn_layers, int M, double* us_out);
/* the largest prefill chunk c in [c_min, c_max] with T_S(d) + T_S(c) <= t_slo_us, d = decode tokens already
 * scheduled; binary search.  *c_out = 0 when even c_min does not fit. */
int spear_slo_chunk(const spear_lut* lut, const int* module_type, const unsigned char* selected, int n_modules,
                    int n_attn_layers, int d, int c_min, int c_max, double t_slo_us, int* c_out);
/* Measures one layer type's two table rows on the device with spear_plan (fastest variant per grid point, weights read
 * from HBM): lat_w4_us_out[n_grid] for the plain layer, lat_ec_us_out[n_grid] with the rank-r EC.  Synchronises. */
int spear_lut_measure(const int* M_grid, int n_grid, int N, int K, int group, int r, int gate_kind, int gate_hidden,
                      float* lat_w4_us_out, float* lat_ec_us_out, void* stream);

/* Sweep hook: sets a launch tunable.  Every knob preserves results (it moves work between kernels, grids or streams, never
 * changes what is computed).  Decode ring kernel: "stream_ctas_per_sm", "stream_deep" (-1 heuristic, 0 / 1 shallow / deep
 * ring), "stream_whole_panels", "stream_aligned", "stream_grid", "stream_batch_grid", "stream_batch_units", "stream_units"; decode kernel choice: "rows" (1 =
 * the heuristic may pick the row-strip kernel for small layers, 0 = never), "rows_mid" (1 = the heuristic may pick its 32-token form for 17..64 tokens), "rows_ec" (the row-strip kernel's EC: 0 = z per cluster inside
 * the kernel, 1 = z, gate and u once by a one-cluster pre-kernel, 2 (default) = partial z by 8 pre-kernel CTAs, summed and gated in the layer kernel), "lstream" (-1 = the layer-stream kernel only
 * where spear_plan_batch measured it faster, 0 = never, 1 = always for M <= 16); EC pre-kernels: "ecpre_ctas", "ecbig_kdiv";
 * tcgen05 kernel: "tc_grid", "tc_cluster", "tc_ksplit", "tc_tail" (split the tiles of a small partial last wave along K), "tc_bt", "tc_xslice_mb"; all: "pdl"; batch: "batch_lanes".
 * Unknown key -> SPEAR_EINVAL.  Host-only, process-wide, not thread-safe against concurrent compute calls.  bench.py
 * echoes every override it was run with (config.spear_tune_overrides). */
int spear_tune(const char* key, int value);

const char* spear_last_error(void);
/* Number of kernels the library has launched in this process (bench.py's gpu_launches). */
unsigned long long spear_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* SPEAR_H */

// kernels.h -- parameter blocks and host launchers shared by api.cu and the kernel translation units.
#pragma once

#include "common.cuh"

namespace spear {

constexpr int kZStride = 136;    // >= r + 1 (the extra column carries the scalar-gate logit)

// ---- stream.cu (M <= 16) ------------------------------------------------------------------------
struct StreamParams {
    const void* wq;          // SPW4 packed codes
    const void* scales;      // SPW4 packed scales
    __half* y;               // [M][N]
    const float* u;          // [16][r] fp32, alpha * gamma (.) z (EC pre-kernel); unused when r == 0
    const __half* B;         // [N][r] (int8 [N][r] when ec_int8)
    int ec_int8;             // 1: A and B are int8 with one fp16 scale per row
    const __half* A_scale;   // [r]
    const __half* B_scale;   // [N]
    float* partial;          // [grid * 2][8*MT][128] fp32 split-K slots
    unsigned* counters;      // [N / 128], zero between calls
    int M, N, K, r;
    int G;                   // K / group
    int group_chunks;        // group / 128
    int C;                   // K / 128 chunks per panel
    int CP;                  // (C + 1) / 2 chunk pairs = work units per panel
    int U;                   // (N / 128) * CP work units
    int stages;              // ring depth (stream_stages, minus what the u buffer needs: stream_fit_stages)
    int deep;                // 1: the one-CTA-per-SM instance (deep ring), 0: the two-CTA instance
    int b_slots;             // r > 0: ring items that carry one panel's B slab (1, or 2 when 128 r elements exceed 16 KiB)
    int b_slot_bytes;        // bytes of one such item (128 r esize / b_slots)
    // ---- fused tail: y = residual + layer, h_out = RMSNorm(y) * rms_w; NULL resid = off ----
    const __half* resid;     // [M][N]
    const __half* rms_w;     // [N]
    __half* h_out;           // [M][N]
    float rms_eps;
    float* tail_ssq;         // [16] fp32 sum of squares per token, zero between calls
    unsigned* tail_ctr;      // [0] finalised panels, [1] CTAs that left; zero between calls
    // ---- fused EC (SPEAR_VARIANT_STREAM_FUSED): z = x [A; w_g]^T, gate and u are computed by this kernel ----
    int fused;               // 0: u comes from the EC pre-kernel; 1: warp 9 of every CTA produces it
    int gate_kind;           // SPEAR_GATE_SCALAR_SIGMOID or SPEAR_GATE_NONE
    float alpha;
    const __half* x;         // [M][K]
    const __half* A;         // [r][K]
    const __half* w_g;       // [K] (scalar gate)
    const float* b_g;        // 1 or NULL
    float* zbuf;             // [2][16][kZStride] fp32, double-buffered by the parity of the epoch word
    float* gate_out;         // optional [M]
    unsigned* ec_sync;       // [0] epoch (bumped once per fused launch), [1], [2] arrival counters of buffer 0 / 1
};
int stream_stages(int MT, bool deep);
int stream_smem_bytes(int MT, int stages, int r);
int stream_fit_stages(int MT, bool deep, int r);          // deepest ring <= stream_stages whose CTA (ring + u buffer) fits
int stream_resident_ctas(int MT, bool deep, int r);
int launch_stream(const CUtensorMap& xmap, const StreamParams& p, int MT, int grid, bool pdl, cudaStream_t st);

// ---- rows.cu (M <= 16): row-strip kernel -- one CTA per 16 output rows over the whole of K, no cross-CTA reduction ----
struct RowsParams {
    const void* wq;          // SPW4 packed codes
    const void* scales;      // SPW4 packed scales
    const __half* x;         // [M][K]
    __half* y;               // [M][N]
    const float* u;          // [16][r] fp32, alpha * gamma (.) z from the EC pre-kernel; unused when r == 0
    const __half* u16;       // mid-M form (launch_rows_mid): u as fp16 [M][r] from the M > 16 pre-pass
    const void* B;           // [N][r] fp16 (int8 when ec_int8)
    const __half* B_scale;   // [N] (ec_int8)
    int ec_int8;
    int M, N, K, r;
    int G;                   // K / group
    int group;
    // ---- fused EC (scalar / none gate): every cluster of 8 CTAs computes z = x [A; w_g]^T for itself ----
    int fused;
    int gate_kind;
    float alpha;
    const __half* A;         // [r][K] fp16 (int8 when ec_int8)
    const __half* A_scale;   // [r] (ec_int8)
    const __half* w_g;       // [K] (scalar gate)
    const float* b_g;        // 1 or NULL
    float* gate_out;         // optional [M]
    float* zpart;            // non-NULL: the pre-kernel parks 8 partial z [8 MT][r + 1] here (no cluster), the layer kernel sums and gates
};
int launch_rows(const RowsParams& p, bool pdl, cudaStream_t st);
int launch_ecz_cluster(const RowsParams& p, bool pdl, cudaStream_t st);
int launch_rows_mid(const RowsParams& p, bool pdl, cudaStream_t st);        // 17..64 tokens: 32 tokens x one strip per CTA, fp16 EC factors, u16 from the M > 16 pre-pass      // z, gate, u once, by one cluster of 8 CTAs -> p.u

// ---- lstream.cu (M <= 16): persistent "layer stream" -- ONE cooperative launch consumes a table of layer
// calls as a single queue of (call, panel, 128-column chunk) work items; int4 -> fp16 in registers -> TMEM
// (tcgen05.st) -> tcgen05.mma with the tokens as N = 16 (A operand in tensor memory), fp32 accumulators in TMEM.
#ifndef LS_MAX_CALLS
#define LS_MAX_CALLS 64
#endif
constexpr int kLsMaxCalls = LS_MAX_CALLS;
struct LsCall {
    const uint8_t* wq;       // SPW4 packed codes
    const uint8_t* scales;   // SPW4 packed scales
    const __half* x;         // [M][K]
    __half* y;               // [M][N]
    const __half* A;         // [r][K] or NULL
    const __half* B;         // [N][r] or NULL
    const __half* w_g;       // [K] (scalar gate) or NULL
    const float* b_g;        // 1 (device) or NULL
    float* gate_out;         // optional [M]
    const uint8_t* xperm;    // [K/128][xtile] x in the MMA operand layout (workspace): written by the prologue of the launch
                             // (external x) or by the finalisers of the call whose y this x is
    uint8_t* yperm;          // NULL, or where a later call of this launch expects this call's y as its xperm
    int xtile;               // bytes per chunk tile of xperm / yperm: 2048 (M <= 8) or 4096
    int x_internal;          // 1: x is an earlier call's y (xperm comes from its finalisers)
    int M, N, K, r;
    int group_chunks;        // group / 128
    int group_shift;         // log2(group_chunks) when the group is a power-of-two number of chunks; 31: group == K
    int C;                   // K / 128 chunks per panel
    int P;                   // N / 128 panels
    int gate_kind;           // SPEAR_GATE_SCALAR_SIGMOID or SPEAR_GATE_NONE
    float alpha;
    int chunk_base;          // first chunk of this call inside its phase's chunk sequence
    int panel_base;          // first split-K counter of this call
    int ec_slot;             // EC state slot (z, u, counters) or -1
};
struct LsParams {
    LsCall calls[kLsMaxCalls];
    int n_calls, n_phases;
    int phase_first_call[kLsMaxCalls + 1];   // calls of phase ph: [phase_first_call[ph], phase_first_call[ph + 1])
    int phase_chunks[kLsMaxCalls];           // chunks of the phase (all its calls)
    int phase_per[kLsMaxCalls], phase_rem[kLsMaxCalls];   // phase_chunks / grid, phase_chunks % grid
    int phase_panels[kLsMaxCalls];           // panels of the phase = y completions to wait for
    float* partial;          // [2 phase parities][grid][16][128] fp32 split-K accumulators of shared panels, zero between launches
    unsigned* counters;      // per-panel split-K counters, zero between launches (self-cleaning)
    unsigned* done;          // [n_phases] finalised panels per phase, [kLsMaxCalls] exit counter, [kLsMaxCalls + 1] CTAs that
                             // finished the x prologue; zeroed by the last CTA
    float* zbuf;             // [ec slots][16][kZStride] fp32, zero between launches
    float* ubuf;             // [ec slots][16][128] fp32: u = alpha * gamma (.) z
    unsigned* ec_sync;       // [ec slots][2]: z arrivals, u-ready flag; zeroed by the last arriver / last CTA
};
size_t ls_workspace_bytes(int grid);
int ls_grid();
int launch_lstream(const LsParams& p, cudaStream_t st);

// ---- ec_pre.cu (M <= 16): z = x A^T, gate, u = alpha * gamma (.) z ------------------------------
struct EcPreParams {
    const __half* x;         // [M][K]
    const __half* A;         // [r][K] (int8 [r][K] when ec_int8)
    int ec_int8;
    const __half* A_scale;   // [r]
    const __half* w_g;       // [K]       scalar gate
    const float* b_g;        // 1 (device) or NULL
    const __half* W1;        // [h][r]    MLP gate
    const float* b1;         // [h]
    const __half* W2;        // [r][h]
    const float* b2;         // [r]
    float* zbuf;             // [16][kZStride] fp32 accumulators, zero between calls
    float* u;                // [16][r] out
    float* gate_out;         // optional
    unsigned* counter;       // zero between calls
    int M, K, r, h, gate_kind;
    int ksplit;
    float alpha;
};
int launch_ec_pre(const EcPreParams& p, bool pdl, cudaStream_t st);

// ---- ec_big.cu (M > 16): z = x [A; w_g]^T (split-K, fp32 red.add), then gate -> u16 = fp16(alpha*gamma(.)z)
struct EcBigParams {
    const __half* x;         // [M][K]
    const __half* A;         // [r][K]
    const __half* w_g;       // [K] or NULL
    const float* b_g;
    const __half* W1; const float* b1; const __half* W2; const float* b2;
    float* zbuf;             // [M][kZStride] fp32, zero between calls
    __half* u16;             // [M][r] out
    float* gate_out;         // optional
    int M, K, r, h, gate_kind;
    int ksplit;
    float alpha;
};
int launch_ec_big(const EcBigParams& p, bool pdl, cudaStream_t st);
// split arm for M > 16: y += u16 . B^T as a separate pass (SPEAR_VARIANT_TC_SPLIT)
// the tail as a row kernel (variants whose layer kernel does not fuse it): y <- residual + y, h_out <- RMSNorm(y) * w
int launch_tail_rows(__half* y, const __half* resid, const __half* rms_w, __half* h_out, float eps, int M, int N, bool pdl, cudaStream_t st);
int launch_ec_update(const __half* u16, const __half* B, __half* y, int M, int N, int r, bool pdl, cudaStream_t st);
// INT8 EC factors on the M > 16 path: rows * cols int8 codes times one fp16 scale per row -> fp16 scratch
int launch_ec_dequant_i8(const int8_t* q, const __half* scale, __half* out, int rows, int cols, cudaStream_t st);

// ---- tc.cu (M > 16): tcgen05 GEMM, int4 dequantised into shared memory, EC folded in as extra K blocks
struct TcProblem {
    const void* x; const void* wq; const void* scales; const void* B; void* y;
    const void* u16;         // [M][r] fp16 (alpha * gamma (.) z) or NULL when r == 0
    int M, N, K, r, group;
    bool pdl;
    int grid_override;
    int cluster_override;    // 0 = heuristic, else 1 / 2 / 4 CTAs sharing x tiles by TMA multicast
    int ksplit_override;     // 0 = heuristic, else the split-K factor
    int tail_split;          // 0 = off, else: split the tiles of a small partial last wave along K over the idle CTAs
    int bt_override;         // 0 = heuristic, else the token-tile width (32 / 64 need M <= width)
    int xslice_mb;           // 0 = default: MiB of x a raster group of token tiles may cover (L2 residency)
    void* partial;           // fp32 split-K slots (workspace)
    size_t partial_bytes;
    unsigned* counters;      // zero between calls
    int max_counters;
};
int run_tc(const TcProblem& t, cudaStream_t st);

}  // namespace spear

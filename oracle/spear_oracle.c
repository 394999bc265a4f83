/*
 * spear_oracle.c -- CPU oracle for the SPEAR W4A16 + gated Error Compensator layer.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may call this.  It shares no
 * code with the CUDA path (no common header, helper, table or constant) and is
 * compiled by gcc alone.
 *
 * What it computes (PAPER.md line numbers; equation numbers as in the paper):
 *   O1  What[n][k] = (codes[n][k] - 8) * scales[n][k/group]        W4 format, :247, :585;
 *                                                                  zero-point 8 = reading A4
 *   O2  ybase[m][n] = sum_k x[m][k] * What[n][k]                   Eq. 3 first term, :107
 *   O3  z[m][j]     = sum_k A[j][k] * x[m][k]                      "Ax", Eq. 3, :107
 *   O4  gate   MLP    gamma = 1 + tanh(W2 relu(W1 z + b1) + b2)    Eq. 3 second line, :109
 *              scalar gamma = sigmoid(x . w_g + b)  (per token)    BASELINE.json configs (reading A1)
 *              none   gamma = 1                                    Eq. 2, :96
 *   O5  u[m][j]     = gamma[m][j] * z[m][j]                        Eq. 3, :107
 *   O6  y[m][n]     = ybase[m][n] + alpha * sum_j B[n][j] u[m][j]  Eq. 3, :107
 *   T1, T2  residual add + next-layer RMSNorm of the fused post-EC tail   :217 (spo_tail)
 *   O3', O6'  the same with INT8 per-channel symmetric factors A8*sA, B8*sB   :603 (spo_forward_q8)
 *
 * Everything is fp64, plain left-to-right loops, no blocking, no reordering.
 * fp16 inputs arrive as raw uint16 bit patterns and are decoded by the decoder
 * below (exact: every fp16 is an fp64).
 *
 * Also here, for the bit-exact part of the contract:
 *   Q1  spo_pack_w4 / spo_unpack_w4: the packed int4 layout, written from the
 *       layout document in DESIGN.md section "Packed W4 layout" (not from the
 *       CUDA source).
 *   Q3  spo_dequant16: RN-even fp16 of O1.
 *   A5  spo_rtn_quantise: test-only round-to-nearest quantiser.
 *
 * Pins (tests/test_oracle_pins.py): worked example P1 of SURVEY.md 8(c) stored in
 * tests/golden/, the MLP-gate worked example (h != r, ReLU active, non-zero biases) stored in
 * tests/golden/, exact-rational brute force with and without the gate, numpy.matmul on the dequantised
 * weight, Eq. 2 / Eq. 4 effective-weight identities, rank / linearity, gate
 * bounds, token-permutation equivariance, fp16 codec against numpy.float16.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

/* ---- fp16 codec (IEEE 754 binary16), written out by hand ------------------------------- */

double spo_f16_to_f64(uint16_t h)
{
    int sign = (h >> 15) & 1;
    int e = (h >> 10) & 0x1f;
    int f = h & 0x3ff;
    double v;
    if (e == 0) {
        v = ldexp((double)f, -24);                 /* subnormal: f * 2^-24 */
    } else if (e == 31) {
        v = f ? NAN : INFINITY;
    } else {
        v = ldexp((double)(1024 + f), e - 25);     /* (1 + f/1024) * 2^(e-15) */
    }
    return sign ? -v : v;
}

/* round-to-nearest-even fp64 -> fp16 */
uint16_t spo_f64_to_f16(double v)
{
    uint16_t sign = 0;
    if (isnan(v)) return 0x7e00;
    if (signbit(v)) { sign = 0x8000; v = -v; }
    if (isinf(v)) return sign | 0x7c00;
    if (v == 0.0) return sign;
    int ex;
    double m = frexp(v, &ex);                      /* v = m * 2^ex, m in [0.5,1) */
    int e = ex - 1;                                /* v = (2m) * 2^e, 2m in [1,2) */
    double q;                                      /* v expressed in units of the target ulp */
    int biased;
    if (e < -14) {                                 /* subnormal range: ulp = 2^-24 */
        q = ldexp(v, 24);
        biased = 0;
    } else {
        q = ldexp(m, 11);                          /* 2m * 2^10 in [1024, 2048) */
        biased = e + 15;
    }
    double fl = floor(q);
    double rem = q - fl;
    uint64_t qi = (uint64_t)fl;
    if (rem > 0.5 || (rem == 0.5 && (qi & 1))) qi += 1;
    if (biased == 0) {
        /* qi in [0, 1024]; 1024 carries into the smallest normal, which the bit pattern encodes */
        return sign | (uint16_t)qi;
    }
    if (qi == 2048) { qi = 1024; biased += 1; }
    if (biased >= 31) return sign | 0x7c00;        /* overflow -> inf */
    return sign | (uint16_t)((biased << 10) | (qi - 1024));
}

void spo_f16_to_f64_array(const uint16_t *in, double *out, size_t n)
{
    for (size_t i = 0; i < n; ++i) out[i] = spo_f16_to_f64(in[i]);
}

void spo_f64_to_f16_array(const double *in, uint16_t *out, size_t n)
{
    for (size_t i = 0; i < n; ++i) out[i] = spo_f64_to_f16(in[i]);
}

/* ---- O1 / Q3: dequantisation ------------------------------------------------------------ */

/* What[n][k] = (codes[n][k] - 8) * scales[n][k/group].  Returns -1 on a code > 15. */
int spo_dequant(const uint8_t *codes, const uint16_t *scales, int N, int K, int group,
                double *What)
{
    int G = K / group;
    int bad = 0;
#pragma omp parallel for schedule(static) reduction(|:bad)
    for (int n = 0; n < N; ++n) {
        for (int k = 0; k < K; ++k) {
            uint8_t c = codes[(size_t)n * K + k];
            if (c > 15) bad = 1;
            double s = spo_f16_to_f64(scales[(size_t)n * G + k / group]);
            What[(size_t)n * K + k] = ((double)c - 8.0) * s;
        }
    }
    return bad ? -1 : 0;
}

int spo_dequant16(const uint8_t *codes, const uint16_t *scales, int N, int K, int group,
                  uint16_t *out)
{
    int G = K / group;
    int bad = 0;
#pragma omp parallel for schedule(static) reduction(|:bad)
    for (int n = 0; n < N; ++n) {
        for (int k = 0; k < K; ++k) {
            uint8_t c = codes[(size_t)n * K + k];
            if (c > 15) bad = 1;
            double s = spo_f16_to_f64(scales[(size_t)n * G + k / group]);
            out[(size_t)n * K + k] = spo_f64_to_f16(((double)c - 8.0) * s);
        }
    }
    return bad ? -1 : 0;
}

/* ---- O2..O6: the layer ------------------------------------------------------------------ */

enum { SPO_GATE_SCALAR_SIGMOID = 0, SPO_GATE_MLP = 1, SPO_GATE_NONE = 2 };

/*
 * x[M][K] f16 bits; What[N][K] f64 (from spo_dequant); A[r][K], B[N][r] f16 bits (may be NULL if r==0);
 * gate parameters: MLP W1[h][r] f16, b1[h] f32, W2[r][h] f16, b2[r] f32; scalar w_g[K] f16, b_g.
 * Outputs (any may be NULL): y[M][N], ybase[M][N], z[M][r], gam[M][r] (scalar/none gates are
 * broadcast along r).  Returns 0, or -1 on bad arguments.
 */
static int spo_forward_core(const uint16_t *x, const double *What, const double *A, const double *B,
                int gate_kind, int h, double alpha,
                const uint16_t *W1, const float *b1, const uint16_t *W2, const float *b2,
                const uint16_t *w_g, double b_g,
                int M, int N, int K, int r,
                double *y, double *ybase, double *z, double *gam)
{
    if (M < 0 || N < 0 || K < 0 || r < 0) return -1;
    if (r > 0 && (!A || !B)) return -1;
    if (r > 0 && gate_kind == SPO_GATE_MLP && (!W1 || !b1 || !W2 || !b2 || h <= 0)) return -1;
    if (r > 0 && gate_kind == SPO_GATE_SCALAR_SIGMOID && !w_g) return -1;

    double *xd = (double *)malloc(sizeof(double) * (size_t)M * K + 8);
    double *zz = (double *)calloc((size_t)M * (r > 0 ? r : 1), sizeof(double));
    double *uu = (double *)calloc((size_t)M * (r > 0 ? r : 1), sizeof(double));
    double *gg = (double *)calloc((size_t)M * (r > 0 ? r : 1), sizeof(double));
    if (!xd || !zz || !uu || !gg) { free(xd); free(zz); free(uu); free(gg); return -1; }
    spo_f16_to_f64_array(x, xd, (size_t)M * K);

    /* O3: z = A x */
    if (r > 0) {
#pragma omp parallel for collapse(2) schedule(static)
        for (int m = 0; m < M; ++m) {
            for (int j = 0; j < r; ++j) {
                double acc = 0.0;
                for (int k = 0; k < K; ++k)
                    acc += A[(size_t)j * K + k] * xd[(size_t)m * K + k];
                zz[(size_t)m * r + j] = acc;
            }
        }
        /* O4: gate */
        for (int m = 0; m < M; ++m) {
            if (gate_kind == SPO_GATE_MLP) {
                double *hid = (double *)malloc(sizeof(double) * (size_t)h);
                for (int i = 0; i < h; ++i) {
                    double acc = 0.0;
                    for (int j = 0; j < r; ++j)
                        acc += spo_f16_to_f64(W1[(size_t)i * r + j]) * zz[(size_t)m * r + j];
                    acc += (double)b1[i];
                    hid[i] = acc > 0.0 ? acc : 0.0;
                }
                for (int j = 0; j < r; ++j) {
                    double acc = 0.0;
                    for (int i = 0; i < h; ++i)
                        acc += spo_f16_to_f64(W2[(size_t)j * h + i]) * hid[i];
                    acc += (double)b2[j];
                    gg[(size_t)m * r + j] = 1.0 + tanh(acc);
                }
                free(hid);
            } else if (gate_kind == SPO_GATE_SCALAR_SIGMOID) {
                double acc = 0.0;
                for (int k = 0; k < K; ++k)
                    acc += xd[(size_t)m * K + k] * spo_f16_to_f64(w_g[k]);
                acc += b_g;
                double g = 1.0 / (1.0 + exp(-acc));
                for (int j = 0; j < r; ++j) gg[(size_t)m * r + j] = g;
            } else {
                for (int j = 0; j < r; ++j) gg[(size_t)m * r + j] = 1.0;
            }
            /* O5: u = gamma (.) z */
            for (int j = 0; j < r; ++j)
                uu[(size_t)m * r + j] = gg[(size_t)m * r + j] * zz[(size_t)m * r + j];
        }
    }

    /* O2 + O6 */
#pragma omp parallel for collapse(2) schedule(static)
    for (int m = 0; m < M; ++m) {
        for (int n = 0; n < N; ++n) {
            const double *xr = xd + (size_t)m * K;
            const double *wr = What + (size_t)n * K;
            double acc = 0.0;
            for (int k = 0; k < K; ++k) acc += xr[k] * wr[k];
            double ec = 0.0;
            for (int j = 0; j < r; ++j)
                ec += B[(size_t)n * r + j] * uu[(size_t)m * r + j];
            if (ybase) ybase[(size_t)m * N + n] = acc;
            if (y) y[(size_t)m * N + n] = acc + alpha * ec;
        }
    }
    if (z && r > 0) memcpy(z, zz, sizeof(double) * (size_t)M * r);
    if (gam && r > 0) memcpy(gam, gg, sizeof(double) * (size_t)M * r);
    free(xd); free(zz); free(uu); free(gg);
    return 0;
}

/* fp16 EC factors (the exact fp64 value of every fp16 entry) */
int spo_forward(const uint16_t *x, const double *What, const uint16_t *A, const uint16_t *B,
                int gate_kind, int h, double alpha,
                const uint16_t *W1, const float *b1, const uint16_t *W2, const float *b2,
                const uint16_t *w_g, double b_g,
                int M, int N, int K, int r,
                double *y, double *ybase, double *z, double *gam)
{
    double *Ad = NULL, *Bd = NULL;
    if (r > 0) {
        if (!A || !B) return -1;
        Ad = (double *)malloc(sizeof(double) * (size_t)r * K);
        Bd = (double *)malloc(sizeof(double) * (size_t)N * r);
        if (!Ad || !Bd) { free(Ad); free(Bd); return -1; }
        spo_f16_to_f64_array(A, Ad, (size_t)r * K);
        spo_f16_to_f64_array(B, Bd, (size_t)N * r);
    }
    int rc = spo_forward_core(x, What, Ad, Bd, gate_kind, h, alpha, W1, b1, W2, b2, w_g, b_g, M, N, K, r, y, ybase, z, gam);
    free(Ad); free(Bd);
    return rc;
}

/*
 * INT8 EC factors, "INT8 per-channel symmetric" (PAPER.md:603, Table 7; :585, :607): the stored factors are
 *   Ahat[j][k] = A8[j][k] * sA[j]      (one fp16 scale per row of A, i.e. per rank channel j)
 *   Bhat[n][j] = B8[n][j] * sB[n]      (one fp16 scale per row of B, i.e. per output channel n)
 * (reading A17 of DESIGN.md: "per-channel" = per output channel of each factor); everything else is Eq. 3 unchanged.
 * The products int8 * fp16 are exact in fp64.
 */
int spo_forward_q8(const uint16_t *x, const double *What, const int8_t *A8, const uint16_t *sA,
                   const int8_t *B8, const uint16_t *sB,
                   int gate_kind, int h, double alpha,
                   const uint16_t *W1, const float *b1, const uint16_t *W2, const float *b2,
                   const uint16_t *w_g, double b_g,
                   int M, int N, int K, int r,
                   double *y, double *ybase, double *z, double *gam)
{
    if (r <= 0 || !A8 || !sA || !B8 || !sB) return -1;
    double *Ad = (double *)malloc(sizeof(double) * (size_t)r * K);
    double *Bd = (double *)malloc(sizeof(double) * (size_t)N * r);
    if (!Ad || !Bd) { free(Ad); free(Bd); return -1; }
    for (int j = 0; j < r; ++j)
        for (int k = 0; k < K; ++k)
            Ad[(size_t)j * K + k] = (double)A8[(size_t)j * K + k] * spo_f16_to_f64(sA[j]);
    for (int n = 0; n < N; ++n)
        for (int j = 0; j < r; ++j)
            Bd[(size_t)n * r + j] = (double)B8[(size_t)n * r + j] * spo_f16_to_f64(sB[n]);
    int rc = spo_forward_core(x, What, Ad, Bd, gate_kind, h, alpha, W1, b1, W2, b2, w_g, b_g, M, N, K, r, y, ybase, z, gam);
    free(Ad); free(Bd);
    return rc;
}

/* ---- post-EC tail: residual add + next-layer RMSNorm ------------------------ */
/*
 * "residual addition, and next-layer RMSNorm ... as a single fused tail".  Given the layer output y (fp64,
 * from spo_forward), the residual stream res[M][N] (f16 bits) and the next layer's RMSNorm weight g[N] (f16 bits):
 *   T1  s[m][n] = res[m][n] + y[m][n]                                  the new residual stream
 *   T2  h[m][n] = s[m][n] / sqrt( (1/N) sum_n s[m][n]^2 + eps ) * g[n]  RMSNorm (Zhang & Sennrich), eps as given
 * Plain loops, fp64.
 */
int spo_tail(const double *y, const uint16_t *res, const uint16_t *g, double eps, int M, int N,
             double *s_out, double *h_out)
{
    if (M < 0 || N <= 0 || !y || !res || !g) return -1;
    for (int m = 0; m < M; ++m) {
        double ssq = 0.0;
        for (int n = 0; n < N; ++n) {
            double s = spo_f16_to_f64(res[(size_t)m * N + n]) + y[(size_t)m * N + n];
            if (s_out) s_out[(size_t)m * N + n] = s;
            ssq += s * s;
        }
        double inv = 1.0 / sqrt(ssq / (double)N + eps);
        for (int n = 0; n < N; ++n) {
            double s = spo_f16_to_f64(res[(size_t)m * N + n]) + y[(size_t)m * N + n];
            if (h_out) h_out[(size_t)m * N + n] = s * inv * spo_f16_to_f64(g[n]);
        }
    }
    return 0;
}

/* ---- Q1: packed layout, from the layout document ---------------------------------------- */
/*
 * DESIGN.md section 2 "Packed W4 layout (SPW4)"; requires N % 128 == 0, K % 128 == 0,
 * group % 128 == 0, K % group == 0.  For element (n, k):
 *   p = n / 128, s = (n % 128) / 16, g = n % 8, hi = (n % 16) / 8,
 *   kt = k / 64, t = (k % 64) / 16, wd = (k % 16) / 8, e = k % 8, lane = g * 4 + t,
 *   word = (((p * (K/64) + kt) * 8 + s) * 32 + lane) * 4 + hi * 2 + wd        (uint32 units)
 *   slot = (e >> 1) + 4 * (e & 1); the code occupies bits [4*slot, 4*slot + 4).
 *   scales_packed[(p * G + k/group) * 128 + s * 16 + 2 * g + hi] = scales[n][k/group].
 */
static size_t spo_word_index(int n, int k, int K)
{
    int p = n / 128, s = (n % 128) / 16, g = n % 8, hi = (n % 16) / 8;
    int kt = k / 64, t = (k % 64) / 16, wd = (k % 16) / 8;
    int lane = g * 4 + t;
    return ((((size_t)p * (K / 64) + kt) * 8 + s) * 32 + lane) * 4 + (size_t)hi * 2 + wd;
}

static int spo_slot(int k)
{
    int e = k % 8;
    return (e >> 1) + 4 * (e & 1);
}

int spo_pack_w4(const uint8_t *codes, const uint16_t *scales, int N, int K, int group,
                uint32_t *wq, uint16_t *scales_packed)
{
    if (N <= 0 || K <= 0 || group <= 0) return -2;
    if (N % 128 || K % 128 || group % 128 || K % group) return -2;
    int G = K / group;
    memset(wq, 0, (size_t)N * K / 2);
    for (int n = 0; n < N; ++n) {
        for (int k = 0; k < K; ++k) {
            uint8_t cd = codes[(size_t)n * K + k];
            if (cd > 15) return -1;
            wq[spo_word_index(n, k, K)] |= (uint32_t)cd << (4 * spo_slot(k));
        }
        int p = n / 128, s = (n % 128) / 16, g = n % 8, hi = (n % 16) / 8;
        for (int gi = 0; gi < G; ++gi)
            scales_packed[((size_t)p * G + gi) * 128 + s * 16 + 2 * g + hi] = scales[(size_t)n * G + gi];
    }
    return 0;
}

int spo_unpack_w4(const uint32_t *wq, int N, int K, uint8_t *codes)
{
    if (N <= 0 || K <= 0 || N % 128 || K % 128) return -2;
    for (int n = 0; n < N; ++n)
        for (int k = 0; k < K; ++k)
            codes[(size_t)n * K + k] =
                (uint8_t)((wq[spo_word_index(n, k, K)] >> (4 * spo_slot(k))) & 0xf);
    return 0;
}

/* ---- A5: test-only RTN quantiser -------------------------------------------------------- */
/* per (n, group): s = fp16_RN(max|w| / 7) (s = 1 if the group is all zero);
 * q = clamp(nearbyint_even(w / s) + 8, 0, 15). */
void spo_rtn_quantise(const double *W, int N, int K, int group, uint8_t *codes, uint16_t *scales)
{
    int G = K / group;
    for (int n = 0; n < N; ++n) {
        for (int g = 0; g < G; ++g) {
            double mx = 0.0;
            for (int k = g * group; k < (g + 1) * group; ++k) {
                double a = fabs(W[(size_t)n * K + k]);
                if (a > mx) mx = a;
            }
            uint16_t s16 = mx == 0.0 ? spo_f64_to_f16(1.0) : spo_f64_to_f16(mx / 7.0);
            double s = spo_f16_to_f64(s16);
            scales[(size_t)n * G + g] = s16;
            for (int k = g * group; k < (g + 1) * group; ++k) {
                double q = nearbyint(W[(size_t)n * K + k] / s) + 8.0;   /* default mode: ties-to-even */
                if (q < 0.0) q = 0.0;
                if (q > 15.0) q = 15.0;
                codes[(size_t)n * K + k] = (uint8_t)q;
            }
        }
    }
}

int spo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

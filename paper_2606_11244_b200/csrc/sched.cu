// sched.cu -- host-only: the paper's latency look-up tables and SLO-constrained chunk selection (PAPER.md:231-237,
// section 4.3).  No device code; it lives in libspear.so because its tables are filled from the library's own
// measurements (spear_lut_measure -> spear_plan) and its output (a prefill chunk size) sizes the next layer calls.
//
//   offline : per layer type t, latency tables l_W4[t](M) and l_EC[t](M) on a sparse grid of token counts M, plus an
//             attention table l_attn(M) supplied by the caller (no attention kernel in this library)   (:231)
//   online  : T_S(M) = sum over modules m of ( selected[m] ? l_EC[type(m)](M) : l_W4[type(m)](M) ) + n_attn * l_attn(M),
//             linear interpolation between grid points                                                   (:231)
//   schedule: the largest c in [c_min, c_max] with T_S(d) + T_S(c) <= T_SLO, by binary search (T_S monotone)  (:235-237)
//
// Readings (S1-S3): T_S(0) = 0; below the first grid point the first entry is used, above the last
// the last segment is extended linearly; a measured table that is not monotone is made so by a running maximum when the
// LUT is created (the binary search of :237 needs it, measurement noise must not break it).
#include <algorithm>
#include <cstring>
#include <new>
#include <vector>

#include "common.cuh"

struct spear_lut {
    std::vector<int> grid;
    int n_types;
    std::vector<float> w4, ec;      // [n_types][n_grid]
    std::vector<float> attn;        // [n_grid] (zeros when absent)
};

namespace {
double interp(const std::vector<int>& g, const float* tab, int M) {
    const int n = int(g.size());
    if (M <= 0) return 0.0;
    if (M <= g[0] || n == 1) return tab[0];
    int hi = int(std::upper_bound(g.begin(), g.end(), M) - g.begin());      // first grid point > M
    if (hi >= n) hi = n - 1;                                                  // beyond the grid: extend the last segment
    const int lo = hi - 1;
    const double t = double(M - g[lo]) / double(g[hi] - g[lo]);
    return double(tab[lo]) + t * (double(tab[hi]) - double(tab[lo]));
}
double iteration_us(const spear_lut* L, const int* type, const unsigned char* sel, int n_modules, int n_attn, int M) {
    if (M <= 0) return 0.0;
    const int n = int(L->grid.size());
    double t = 0.0;
    for (int m = 0; m < n_modules; ++m) {
        const float* tab = ((sel && sel[m]) ? L->ec.data() : L->w4.data()) + size_t(type[m]) * n;
        t += interp(L->grid, tab, M);
    }
    return t + double(n_attn) * interp(L->grid, L->attn.data(), M);
}
}  // namespace

extern "C" int spear_lut_create(const int* M_grid, int n_grid, int n_types, const float* lat_w4_us, const float* lat_ec_us,
                                const float* lat_attn_us, spear_lut** out) {
    if (!M_grid || n_grid < 1 || n_types < 1 || !lat_w4_us || !lat_ec_us || !out)
        return spear::set_error(SPEAR_EINVAL, "spear_lut_create: bad arguments");
    for (int i = 0; i < n_grid; ++i)
        if (M_grid[i] < 1 || (i && M_grid[i] <= M_grid[i - 1]))
            return spear::set_error(SPEAR_EINVAL, "spear_lut_create: the M grid must be positive and strictly increasing");
    spear_lut* L = new (std::nothrow) spear_lut;
    if (!L) return spear::set_error(SPEAR_ENOMEM, "spear_lut_create: out of host memory");
    L->grid.assign(M_grid, M_grid + n_grid);
    L->n_types = n_types;
    L->w4.assign(lat_w4_us, lat_w4_us + size_t(n_types) * n_grid);
    L->ec.assign(lat_ec_us, lat_ec_us + size_t(n_types) * n_grid);
    L->attn.assign(size_t(n_grid), 0.f);
    if (lat_attn_us) L->attn.assign(lat_attn_us, lat_attn_us + n_grid);
    auto monotone = [&](float* tab) {
        for (int i = 0; i < n_grid; ++i) {
            if (!(tab[i] >= 0.f)) tab[i] = 0.f;
            if (i && tab[i] < tab[i - 1]) tab[i] = tab[i - 1];
        }
    };
    for (int t = 0; t < n_types; ++t) { monotone(&L->w4[size_t(t) * n_grid]); monotone(&L->ec[size_t(t) * n_grid]); }
    monotone(L->attn.data());
    *out = L;
    return SPEAR_OK;
}

extern "C" void spear_lut_destroy(spear_lut* L) { delete L; }

extern "C" int spear_lut_iteration_us(const spear_lut* L, const int* module_type, const unsigned char* selected, int n_modules,
                                      int n_attn_layers, int M, double* us_out) {
    if (!L || !us_out || n_modules < 0 || (n_modules && !module_type) || n_attn_layers < 0 || M < 0)
        return spear::set_error(SPEAR_EINVAL, "spear_lut_iteration_us: bad arguments");
    for (int m = 0; m < n_modules; ++m)
        if (module_type[m] < 0 || module_type[m] >= L->n_types)
            return spear::set_error(SPEAR_EINVAL, "spear_lut_iteration_us: module %d has type %d (LUT holds %d types)", m, module_type[m], L->n_types);
    *us_out = iteration_us(L, module_type, selected, n_modules, n_attn_layers, M);
    return SPEAR_OK;
}

extern "C" int spear_slo_chunk(const spear_lut* L, const int* module_type, const unsigned char* selected, int n_modules,
                               int n_attn_layers, int d, int c_min, int c_max, double t_slo_us, int* c_out) {
    if (!c_out || d < 0 || c_min < 1 || c_max < c_min)
        return spear::set_error(SPEAR_EINVAL, "spear_slo_chunk: bad arguments");
    double td = 0.0;
    if (int rc = spear_lut_iteration_us(L, module_type, selected, n_modules, n_attn_layers, d, &td)) return rc;
    auto fits = [&](int c) { return td + iteration_us(L, module_type, selected, n_modules, n_attn_layers, c) <= t_slo_us; };
    if (!fits(c_min)) { *c_out = 0; return SPEAR_OK; }      // not even the smallest chunk meets the SLO: schedule no prefill
    int lo = c_min, hi = c_max;                              // invariant: fits(lo)
    while (lo < hi) {
        const int mid = lo + (hi - lo + 1) / 2;
        if (fits(mid)) lo = mid; else hi = mid - 1;
    }
    *c_out = lo;
    return SPEAR_OK;
}

// Fills one layer type's tables from the library's own measurements: for every grid point spear_plan times the variants
// of the plain layer (r = 0) and of the layer with its EC, and the fastest of each is the table entry (PAPER.md:231
// "we microbenchmark the low-bit backbone kernels and the ones with EC attached at a sparse grid of token counts M").
extern "C" int spear_lut_measure(const int* M_grid, int n_grid, int N, int K, int group, int r, int gate_kind, int gate_hidden,
                                 float* lat_w4_us_out, float* lat_ec_us_out, void* stream) {
    if (!M_grid || n_grid < 1 || !lat_w4_us_out || !lat_ec_us_out) return spear::set_error(SPEAR_EINVAL, "spear_lut_measure: bad arguments");
    for (int i = 0; i < n_grid; ++i) {
        float us[SPEAR_VARIANT_COUNT];
        int chosen = 0;
        if (int rc = spear_plan(M_grid[i], N, K, 0, group, SPEAR_GATE_NONE, 0, &chosen, us, stream)) return rc;
        lat_w4_us_out[i] = us[chosen];
        lat_ec_us_out[i] = us[chosen];
        if (r > 0) {
            if (int rc = spear_plan(M_grid[i], N, K, r, group, gate_kind, gate_hidden, &chosen, us, stream)) return rc;
            lat_ec_us_out[i] = us[chosen];
        }
    }
    return SPEAR_OK;
}

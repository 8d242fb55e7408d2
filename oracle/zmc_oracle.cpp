/*
 * zmc_oracle.cpp -- ORACLE (test infrastructure, NOT the product).
 *
 * Plain single-threaded C++17 restatement of the ZMCintegral hot path
 * (arXiv:1902.07916, section 2.1) with every open convention fixed
 * as listed in DESIGN.md section 3 (R1..R12). Written from the paper and
 * those readings only; shares nothing with the CUDA path. No blocking, no
 * fusion, no reordering beyond what the readings state.
 *
 * Build: g++ -O2 -std=c++17 -ffp-contract=off -mfma -fPIC -shared   (see oracle/build.py)
 *   -ffp-contract=off : a*b+c is two roundings unless std::fma[f] is written
 *   -mfma             : std::fmaf is the hardware instruction (same IEEE result, faster)
 *
 * Parity unpinned by the paper (readings only; see header): threshold form and
 * scope (R6), ddof (R5), how stds are collected (R7).
 */
#include "zmc_oracle.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <limits>
#include <string>
#include <vector>

typedef unsigned __int128 u128;

/* ------------------------------------------------------------------ R1 */
/* Philox4x32-10, Salmon, Moraes, Dror, Shaw: "Parallel random numbers: as easy
 * as 1, 2, 3" (SC'11), named by BASELINE.json; PAPER.md:81 only asks for a
 * generator that produces each number when it is used (ref [23], :284).
 * One round:  (hi0,lo0) = M0*c0 ; (hi1,lo1) = M1*c2 ;
 *             c <- (hi1^c1^k0, lo1, hi0^c3^k1, lo0) ; then k0 += W0, k1 += W1. */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = M0 * (uint64_t)c0;
        uint64_t p1 = M1 * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* ------------------------------------------------------------------ R3 */
/* Derived key: words 0,1 of Philox(ctr = (b,0,0,0x5A4D4321), key = (seed_lo, seed_hi)). */
void orc_derive_key(uint64_t seed, uint32_t instance, uint32_t key[2]) {
    uint32_t ctr[4] = {instance, 0u, 0u, 0x5A4D4321u};
    uint32_t k[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    uint32_t out[4];
    orc_philox4x32_10(ctr, k, out);
    key[0] = out[0]; key[1] = out[1];
}

namespace {

/* Counter of call q of unit (path P, level l, trial t):
 *   c0 = q ; c1 = t | l<<8 | P[79:64]<<16 ; c2 = P[31:0] ; c3 = P[63:32]. */
struct UnitStream {
    uint32_t key[2];
    uint32_t c1, c2, c3;
    uint64_t cached_q;
    uint32_t cached[4];
    bool have;
    UnitStream(uint64_t seed, uint32_t instance, uint64_t path_lo, uint32_t path_hi, int level, int trial) {
        orc_derive_key(seed, instance, key);
        c1 = (uint32_t)trial | ((uint32_t)level << 8) | ((path_hi & 0xFFFFu) << 16);
        c2 = (uint32_t)path_lo;
        c3 = (uint32_t)(path_lo >> 32);
        have = false; cached_q = 0;
    }
    /* word with flat index idx: call q = idx >> 2, output lane idx & 3 */
    uint32_t word(uint64_t idx) {
        uint64_t q = idx >> 2;
        if (!have || q != cached_q) {
            uint32_t ctr[4] = {(uint32_t)q, c1, c2, c3};
            orc_philox4x32_10(ctr, key, cached);
            cached_q = q; have = true;
        }
        return cached[idx & 3];
    }
};

inline uint32_t f2u(float f) { uint32_t u; std::memcpy(&u, &f, 4); return u; }
inline float u2f(uint32_t u) { float f; std::memcpy(&f, &u, 4); return f; }

}  // namespace

void orc_unit_words(uint64_t seed, uint32_t instance, uint64_t path_lo, uint32_t path_hi, int level,
                    int trial, uint64_t first_word, uint64_t n_words, uint32_t* out) {
    UnitStream st(seed, instance, path_lo, path_hi, level, trial);
    for (uint64_t i = 0; i < n_words; ++i) out[i] = st.word(first_word + i);
}

/* ------------------------------------------------------------------ R2 */
/* Equal sub-domains, the same g on every axis at every level (:73).
 * width_d = (upper_d-lower_d)/(double)g^level ; lo_d = lower_d + (double)I_d*width_d
 * (multiply, then add) ; V = w_0*w_1*...*w_{D-1} in axis order. */
void orc_cell_geometry(int dim, const double* lower, const double* upper, int g, int level,
                       const uint32_t* coords, double* lo, double* width, double* volume) {
    double cells_per_axis = 1.0;
    for (int l = 0; l < level; ++l) cells_per_axis = cells_per_axis * (double)g;
    double V = 1.0;
    for (int d = 0; d < dim; ++d) {
        double w = (upper[d] - lower[d]) / cells_per_axis;
        double t = (double)coords[d] * w;
        lo[d] = lower[d] + t;
        width[d] = w;
        V = (d == 0) ? w : V * w;
    }
    *volume = V;
}

/* ------------------------------------------------------------------ R4 */
/* FP64: x = lo + ((double)w + 0.5) * (width * 2^-32): centred 32-bit lattice, open interval. */
double orc_map_f64(uint32_t w, double lo, double width) {
    double step = width * 0x1p-32;
    double t = ((double)w + 0.5) * step;
    return lo + t;
}
/* FP32: u' = bits(0x3F800000 | w>>9) in [1,2) ; x = fmaf(u', (float)width, base),
 * base = (float)(((lo - width) + width*2^-24) - centre) formed in FP64: centred 23-bit lattice. */
float orc_map_f32(uint32_t w, double lo, double width, double centre) {
    float u = u2f(0x3F800000u | (w >> 9));
    double b = (lo - width) + width * 0x1p-24;
    b = b - centre;
    float base = (float)b;
    float wf = (float)width;
    return std::fmaf(u, wf, base);
}

/* ------------------------------------------------------------------ R8 */
/* zsin: k = rint(a/pi) by the magic-number add, two-constant Cody-Waite
 * reduction r = a - k*pi, odd degree-9 polynomial on [-pi/2, pi/2], sign (-1)^k.
 * Every operation is an IEEE binary32 fma/mul/add, in this order. */
float orc_zsin(float a) {
    const float INV_PI = u2f(0x3ea2f983u);   /* 0.318309873 */
    const float MAGIC = u2f(0x4b400000u);    /* 1.5 * 2^23 */
    const float PI_A = u2f(0x40490000u);     /* 3.140625 */
    const float PI_B = u2f(0x3a7daa22u);     /* 9.67653584e-4 = fl(pi - PI_A) */
    const float C3 = u2f(0xbe2aaaa6u), C5 = u2f(0x3c08876au), C7 = u2f(0xb94fb7f7u), C9 = u2f(0x362ede75u);
    float t = std::fmaf(a, INV_PI, MAGIC);
    float kf = t - MAGIC;
    float r = std::fmaf(kf, -PI_A, a);
    r = std::fmaf(kf, -PI_B, r);
    float s = r * r;
    float p = std::fmaf(C9, s, C7);
    p = std::fmaf(p, s, C5);
    p = std::fmaf(p, s, C3);
    float rs = r * s;
    float v = std::fmaf(rs, p, r);
    return u2f(f2u(v) ^ (f2u(t) << 31));
}

/* zexp: n = rint(e*log2(e)) by the magic-number add, two-constant reduction
 * r = e - n*ln2, degree-6 polynomial for exp(r) on [-ln2/2, ln2/2]. Returns the
 * FP32 p ~ exp(r) and the integer n; exp(e) ~= p * 2^n is assembled in FP64 by
 * orc_zexp_value so that the FP64 exponent range is available (reading R9). */
float orc_zexp(float e, int32_t* n) {
    const float LOG2E = u2f(0x3fb8aa3bu);
    const float MAGIC = u2f(0x4b400000u);
    const float LN2_HI = u2f(0x3f317200u);   /* 0.693145752 */
    const float LN2_LO = u2f(0x35bfbe8eu);   /* 1.42860677e-6 */
    const float E2 = u2f(0x3efffffeu), E3 = u2f(0x3e2aaa49u), E4 = u2f(0x3d2aac79u), E5 = u2f(0x3c091cf1u),
                E6 = u2f(0x3ab5121au);
    float t = std::fmaf(e, LOG2E, MAGIC);
    float nf = t - MAGIC;
    float r = std::fmaf(nf, -LN2_HI, e);
    r = std::fmaf(nf, -LN2_LO, r);
    float p = std::fmaf(E6, r, E5);
    p = std::fmaf(p, r, E4);
    p = std::fmaf(p, r, E3);
    p = std::fmaf(p, r, E2);
    p = std::fmaf(p, r, 1.0f);
    p = std::fmaf(p, r, 1.0f);
    *n = (int32_t)(f2u(t) - 0x4b400000u);
    return p;
}

double orc_zexp_value(float e) {
    if (e != e) return std::numeric_limits<double>::quiet_NaN();
    if (e < -708.0f) return 0.0;
    if (e > 708.0f) return std::numeric_limits<double>::infinity();
    int32_t n;
    float p = orc_zexp(e, &n);
    return std::ldexp((double)p, n);
}

namespace {

/* Integrand parameters of one instance, as each precision sees them. */
struct Integrand {
    int id, dim, precision;
    const double* p;  /* this instance's parameters */
    double prefactor() const { return id == ORC_EXP_QUAD ? p[0] : 1.0; }
    double centre(int d) const { return id == ORC_EXP_QUAD ? p[2 + d] : 0.0; }
};

/* f at the point generated from `words[0..D)` inside the cell (lo, width).
 * x_out (optional) receives the coordinates (for EXP_QUAD in FP32: x - c, see R8). */
double eval_point(const Integrand& F, const uint32_t* words, const double* lo, const double* width, double* x_out) {
    const int D = F.dim;
    if (F.precision == ORC_F64) {
        double x[64] = {0.0};
        for (int d = 0; d < D; ++d) { x[d] = orc_map_f64(words[d], lo[d], width[d]); if (x_out) x_out[d] = x[d]; }
        switch (F.id) {
            case ORC_CONST: return F.p[0];
            case ORC_LINEAR: {
                double f = F.p[0];
                for (int d = 0; d < D; ++d) { double t = F.p[1 + d] * x[d]; f = f + t; }
                return f;
            }
            case ORC_SIN_SUM: {   /* paper f1, Eq. (1) */
                double a = x[0];
                for (int d = 1; d < D; ++d) a = a + x[d];
                return std::sin(a);
            }
            case ORC_EXP_QUAD: {  /* paper f2, Eq. (2), as A*exp(-a|x-c|^2); A applied per trial */
                double q = 0.0;
                for (int d = 0; d < D; ++d) { double y = x[d] - F.p[2 + d]; double yy = y * y; q = (d == 0) ? yy : q + yy; }
                double e = -(F.p[1] * q);
                return std::exp(e);
            }
        }
        return std::numeric_limits<double>::quiet_NaN();
    }
    /* canonical FP32 operation sequences */
    float x[64] = {0.0f};
    for (int d = 0; d < D; ++d) { x[d] = orc_map_f32(words[d], lo[d], width[d], F.centre(d)); if (x_out) x_out[d] = (double)x[d]; }
    switch (F.id) {
        case ORC_CONST: return (double)(float)F.p[0];
        case ORC_LINEAR: {
            float f = (float)F.p[0];
            for (int d = 0; d < D; ++d) f = std::fmaf((float)F.p[1 + d], x[d], f);
            return (double)f;
        }
        case ORC_SIN_SUM: {
            float a = x[0];
            for (int d = 1; d < D; ++d) a = a + x[d];
            return (double)orc_zsin(a);
        }
        case ORC_EXP_QUAD: {      /* x[d] already holds x_d - c_d */
            float q = x[0] * x[0];
            for (int d = 1; d < D; ++d) q = std::fmaf(x[d], x[d], q);
            float na = -(float)F.p[1];
            float e = na * q;
            return orc_zexp_value(e);
        }
    }
    return std::numeric_limits<double>::quiet_NaN();
}

const char* check_config(const orc_config* c) {
    if (!c) return "null config";
    if (c->dim < 1 || c->dim > 64) return "dim out of range";
    if (c->g < 1) return "g < 1";
    if (c->trials < 1 || c->trials > 255) return "trials out of range (1..255)";
    if (c->depth < 1 || c->depth > 15) return "depth out of range (1..15)";
    if (c->n_samples < 1) return "n_samples < 1";
    /* R3: call indices are 32-bit; the limit is stated once for both implementations (R3): N*D < 2^34 - 2^14 */
    if ((u128)c->n_samples * (u128)c->dim >= ((u128)1 << 34) - ((u128)1 << 14)) return "N*D >= 2^34 - 2^14";
    if (c->n_instances < 1) return "n_instances < 1";
    if (!(c->sigma_multiplier == c->sigma_multiplier)) return "sigma_multiplier is NaN";
    for (int d = 0; d < c->dim; ++d)
        if (!(c->upper[d] > c->lower[d]) || !std::isfinite(c->upper[d]) || !std::isfinite(c->lower[d])) return "bad bounds";
    int need = c->integrand == ORC_CONST ? 1 : c->integrand == ORC_LINEAR ? 1 + c->dim : c->integrand == ORC_SIN_SUM ? 0
             : c->integrand == ORC_EXP_QUAD ? 2 + c->dim : -1;
    if (need < 0) return "unknown integrand";
    if (c->params_per_instance < need) return "too few parameters";
    /* path must fit 80 bits: k^depth <= 2^80 ; coordinates must fit 32 bits: g^depth <= 2^32 */
    long double bits = (long double)c->depth * (long double)c->dim * std::log2((long double)c->g);
    if (bits > 80.0L) return "path exceeds 80 bits";
    if ((long double)c->depth * std::log2((long double)c->g) > 32.0L) return "g^depth exceeds 32 bits";
    return nullptr;
}

}  // namespace

/* ------------------------------------------------------------------ R5 */
/* S_{c,t} = sum_s (double) f(x_s), sample s uses words s*D .. s*D+D-1 of the unit's flat stream. */
int orc_unit_sum(const orc_config* cfg, uint32_t instance, uint64_t path_lo, uint32_t path_hi, int level,
                 const uint32_t* coords, int trial, double* S, double* Sabs) {
    if (check_config(cfg)) return -1;
    const int D = cfg->dim;
    double lo[64], width[64], V;
    orc_cell_geometry(D, cfg->lower, cfg->upper, cfg->g, level, coords, lo, width, &V);
    Integrand F{cfg->integrand, D, cfg->precision, cfg->params + (size_t)instance * cfg->params_per_instance};
    UnitStream st(cfg->seed, instance, path_lo, path_hi, level, trial);
    double sum = 0.0, sumabs = 0.0;
    uint32_t words[64];
    for (uint64_t s = 0; s < cfg->n_samples; ++s) {
        for (int d = 0; d < D; ++d) words[d] = st.word(s * (uint64_t)D + (uint64_t)d);
        double f = eval_point(F, words, lo, width, nullptr);
        sum = sum + f;
        sumabs = sumabs + std::fabs(f);
    }
    *S = sum;
    if (Sabs) *Sabs = sumabs;
    return 0;
}

/* R13: S and Q = sum_s f*f of one unit (the product is rounded to FP64, then added; sequential order) */
int orc_unit_sums(const orc_config* cfg, uint32_t instance, uint64_t path_lo, uint32_t path_hi, int level,
                  const uint32_t* coords, int trial, double* S, double* Q) {
    if (check_config(cfg)) return -1;
    const int D = cfg->dim;
    double lo[64], width[64], V;
    orc_cell_geometry(D, cfg->lower, cfg->upper, cfg->g, level, coords, lo, width, &V);
    Integrand F{cfg->integrand, D, cfg->precision, cfg->params + (size_t)instance * cfg->params_per_instance};
    UnitStream st(cfg->seed, instance, path_lo, path_hi, level, trial);
    double sum = 0.0, sumsq = 0.0;
    uint32_t words[64];
    for (uint64_t s = 0; s < cfg->n_samples; ++s) {
        for (int d = 0; d < D; ++d) words[d] = st.word(s * (uint64_t)D + (uint64_t)d);
        double f = eval_point(F, words, lo, width, nullptr);
        sum = sum + f;
        double ff = f * f;
        sumsq = sumsq + ff;
    }
    *S = sum;
    *Q = sumsq;
    return 0;
}

int orc_unit_points(const orc_config* cfg, uint32_t instance, uint64_t path_lo, uint32_t path_hi, int level,
                    const uint32_t* coords, int trial, uint64_t n, double* x, double* f) {
    if (check_config(cfg)) return -1;
    const int D = cfg->dim;
    double lo[64], width[64], V;
    orc_cell_geometry(D, cfg->lower, cfg->upper, cfg->g, level, coords, lo, width, &V);
    Integrand F{cfg->integrand, D, cfg->precision, cfg->params + (size_t)instance * cfg->params_per_instance};
    UnitStream st(cfg->seed, instance, path_lo, path_hi, level, trial);
    uint32_t words[64];
    for (uint64_t s = 0; s < n; ++s) {
        for (int d = 0; d < D; ++d) words[d] = st.word(s * (uint64_t)D + (uint64_t)d);
        double v = eval_point(F, words, lo, width, x ? x + s * D : nullptr);
        if (f) f[s] = v;
    }
    return 0;
}

/* I_t = ((V*A)*S_t)/(double)N ; mu = (sum_t I_t)/T ; s = sqrt((sum_t (I_t-mu)^2)/T)  (two-pass, ddof 0)
 * "the mean and standard deviation of these n1 integration values". */
void orc_cell_stats(const double* S, int trials, double volume, double prefactor, uint64_t n_samples,
                    double* I, double* mu, double* s) {
    std::vector<double> It((size_t)trials);
    double VA = volume * prefactor;
    double acc = 0.0;
    for (int t = 0; t < trials; ++t) {
        double v = VA * S[t];
        It[t] = v / (double)n_samples;
        acc = acc + It[t];
    }
    double m = acc / (double)trials;
    double q = 0.0;
    for (int t = 0; t < trials; ++t) {
        double d = It[t] - m;
        double dd = d * d;
        q = q + dd;
    }
    *mu = m;
    *s = std::sqrt(q / (double)trials);
    if (I) for (int t = 0; t < trials; ++t) I[t] = It[t];
}

/* R13 (ours): the spread of a cell from its T*N samples instead of from T trial values.
 * mu is R5's. Pooled sums Sc = sum_t S_t, Qc = sum_t Q_t over M = T*N samples; population variance of f
 * var_f = (Qc - Sc^2/M)/M, cut to 0 when the difference is below 2^-40 of Qc (rounding noise of a constant
 * integrand); s = V*A*sqrt(var_f/M) is the standard error of mu, so sqrt(sum s^2) is a 1-sigma error. */
void orc_cell_stats_samples(const double* S, const double* Q, int trials, double volume, double prefactor,
                            uint64_t n_samples, double* mu, double* s) {
    double VA = volume * prefactor;
    double acc = 0.0, Sc = 0.0, Qc = 0.0;
    for (int t = 0; t < trials; ++t) {
        double v = VA * S[t];
        acc = acc + v / (double)n_samples;
        Sc = Sc + S[t];
        Qc = Qc + Q[t];
    }
    *mu = acc / (double)trials;
    double M = (double)trials * (double)n_samples;
    double sq = Sc * Sc;
    double d = Qc - sq / M;
    if (!(d > Qc * 9.094947017729282e-13)) d = 0.0;     /* 2^-40 */
    double var_f = d / M;
    *s = VA * std::sqrt(var_f / M);
}

/* ------------------------------------------------------------------ R6 */
/* tau = mean(s) + m * pstd(s) over one set of k stds (two-pass, population form).
 * PAPER.md:71 "determined by the mean and standard deviation of the calculated k standard deviations". */
double orc_threshold(const double* s, int64_t k, double m) {
    double acc = 0.0;
    for (int64_t i = 0; i < k; ++i) acc = acc + s[i];
    double mean = acc / (double)k;
    double q = 0.0;
    for (int64_t i = 0; i < k; ++i) {
        double d = s[i] - mean;
        double dd = d * d;
        q = q + dd;
    }
    double pstd = std::sqrt(q / (double)k);
    double mp = m * pstd;
    return mean + mp;
}

/* ------------------------------------------------------------------ R7 */
struct CellRec {
    uint32_t instance;
    u128 path;
    std::vector<uint32_t> coords;
};

struct LevelStore {
    std::vector<uint32_t> instance;
    std::vector<uint64_t> path_lo;
    std::vector<uint32_t> path_hi;
    std::vector<double> mu, s, tau, S, Q;
    std::vector<uint8_t> refined;
    int64_t n_cells = 0, n_refined = 0, n_truncated = 0;
};

struct orc_result {
    std::string err;
    std::vector<double> value, var;
    std::vector<LevelStore> levels;   /* index level-1 */
    int levels_done = 0;
    uint64_t evals = 0;
    int trials = 0;
};

namespace {

struct Driver {
    const orc_config* cfg;
    orc_result* R;
    bool keep;
    int D, g, T, L;
    int64_t k;
    std::vector<std::vector<int64_t>> refined_count;   /* [level][instance]: cells refined so far (budget R12) */

    Driver(const orc_config* c, orc_result* r, bool kp) : cfg(c), R(r), keep(kp) {
        D = c->dim; g = c->g; T = c->trials; L = c->depth;
        k = 1;
        for (int d = 0; d < D; ++d) k *= g;
        R->value.assign(c->n_instances, 0.0);
        R->var.assign(c->n_instances, 0.0);
        R->levels.resize(L);
        R->trials = T;
        refined_count.assign(L + 1, std::vector<int64_t>(c->n_instances, 0));
    }

    /* the j-th child of `parent` (R2): axis 0 least significant digit of j; P' = P*k + j ; I'_d = I_d*g + j_d */
    CellRec child(const CellRec& parent, int64_t j) const {
        CellRec c;
        c.instance = parent.instance;
        c.path = parent.path * (u128)k + (u128)j;
        c.coords.resize(D);
        int64_t rem = j;
        for (int d = 0; d < D; ++d) {
            uint32_t jd = (uint32_t)(rem % g);
            rem /= g;
            c.coords[d] = parent.coords[d] * (uint32_t)g + jd;
        }
        return c;
    }

    /* evaluate one cell at `level`: T trials -> (mu, s) ; PAPER.md:71 (R5), or R13 when spread = samples */
    void eval_cell(const CellRec& c, int level, double* mu, double* s, double* S_out, double* Q_out) {
        std::vector<double> S(T), Q(T, 0.0);
        for (int t = 0; t < T; ++t) {
            if (cfg->spread == ORC_SPREAD_SAMPLES)
                orc_unit_sums(cfg, c.instance, (uint64_t)c.path, (uint32_t)(c.path >> 64), level, c.coords.data(), t, &S[t], &Q[t]);
            else
                orc_unit_sum(cfg, c.instance, (uint64_t)c.path, (uint32_t)(c.path >> 64), level, c.coords.data(), t, &S[t], nullptr);
        }
        R->evals += (uint64_t)T * cfg->n_samples;
        double lo[64], width[64], V;
        orc_cell_geometry(D, cfg->lower, cfg->upper, g, level, c.coords.data(), lo, width, &V);
        double A = (cfg->integrand == ORC_EXP_QUAD) ? cfg->params[(size_t)c.instance * cfg->params_per_instance] : 1.0;
        if (cfg->spread == ORC_SPREAD_SAMPLES) orc_cell_stats_samples(S.data(), Q.data(), T, V, A, cfg->n_samples, mu, s);
        else orc_cell_stats(S.data(), T, V, A, cfg->n_samples, nullptr, mu, s);
        if (S_out) for (int t = 0; t < T; ++t) S_out[t] = S[t];
        if (Q_out) for (int t = 0; t < T; ++t) Q_out[t] = Q[t];
    }

    void store(int level, const CellRec& c, double mu, double s, double tau, bool refined, const double* S, const double* Q) {
        LevelStore& ls = R->levels[level - 1];
        ls.n_cells++;
        if (refined) ls.n_refined++;
        if (!keep) return;
        ls.instance.push_back(c.instance);
        ls.path_lo.push_back((uint64_t)c.path);
        ls.path_hi.push_back((uint32_t)(c.path >> 64));
        ls.mu.push_back(mu); ls.s.push_back(s); ls.tau.push_back(tau);
        ls.refined.push_back(refined ? 1 : 0);
        for (int t = 0; t < T; ++t) ls.S.push_back(S[t]);
        if (cfg->spread == ORC_SPREAD_SAMPLES) for (int t = 0; t < T; ++t) ls.Q.push_back(Q[t]);
    }

    /* flag rule (R7): level < L and s > tau (strict; NaN compares false), then the budget (R12):
     * at most B refined cells per instance and level, first come in ascending path order. */
    bool decide(int level, uint32_t instance, double s, double tau) {
        if (level >= L) return false;
        if (!(s > tau)) return false;
        if (cfg->max_groups_per_level > 0 && refined_count[level][instance] >= cfg->max_groups_per_level) {
            R->levels[level - 1].n_truncated++;
            return false;
        }
        refined_count[level][instance]++;
        return true;
    }

    void accept(uint32_t instance, double mu, double s) {
        R->value[instance] = R->value[instance] + mu;
        double ss = s * s;
        R->var[instance] = R->var[instance] + ss;
    }

    /* ---- breadth-first: one level at a time over the list of parents ("a new list") ---- */
    void run_bfs() {
        std::vector<CellRec> parents;
        for (int b = 0; b < cfg->n_instances; ++b) {
            CellRec root; root.instance = (uint32_t)b; root.path = 0; root.coords.assign(D, 0u);
            parents.push_back(root);
        }
        for (int level = 1; level <= L && !parents.empty(); ++level) {
            R->levels_done = level;
            const size_t ng = parents.size();
            std::vector<double> mu(ng * (size_t)k), s(ng * (size_t)k), S(ng * (size_t)k * (size_t)T), Q(ng * (size_t)k * (size_t)T);
            for (size_t G = 0; G < ng; ++G)
                for (int64_t j = 0; j < k; ++j) {
                    CellRec c = child(parents[G], j);
                    size_t i = G * (size_t)k + (size_t)j;
                    eval_cell(c, level, &mu[i], &s[i], &S[i * (size_t)T], &Q[i * (size_t)T]);
                }
            /* thresholds */
            std::vector<double> tau(ng);
            if (cfg->threshold_scope == ORC_SCOPE_GROUP) {
                for (size_t G = 0; G < ng; ++G) tau[G] = orc_threshold(&s[G * (size_t)k], k, cfg->sigma_multiplier);
            } else {  /* pooled: all cells of this level of the same instance (parents are grouped by instance) */
                size_t G0 = 0;
                while (G0 < ng) {
                    size_t G1 = G0;
                    while (G1 < ng && parents[G1].instance == parents[G0].instance) ++G1;
                    double t = orc_threshold(&s[G0 * (size_t)k], (int64_t)(G1 - G0) * k, cfg->sigma_multiplier);
                    for (size_t G = G0; G < G1; ++G) tau[G] = t;
                    G0 = G1;
                }
            }
            /* R7: flagged iff level < L and s > tau (strict; NaN compares false) */
            const size_t n = ng * (size_t)k;
            std::vector<char> refine(n, 0);
            for (size_t i = 0; i < n; ++i) refine[i] = (level < L && s[i] > tau[i / (size_t)k]) ? 1 : 0;
            /* budget: at most B refined cells per instance and level -- the first B flagged ones in ascending path
             * order (R12), or the B with the largest spread, equal spreads in path order (R14) */
            if (cfg->max_groups_per_level > 0) {
                const size_t B = (size_t)cfg->max_groups_per_level;
                size_t G0 = 0;
                while (G0 < ng) {
                    size_t G1 = G0;
                    while (G1 < ng && parents[G1].instance == parents[G0].instance) ++G1;
                    std::vector<size_t> fl;
                    for (size_t i = G0 * (size_t)k; i < G1 * (size_t)k; ++i) if (refine[i]) fl.push_back(i);
                    if (fl.size() > B) {
                        if (cfg->budget_order == ORC_BUDGET_LARGEST_SPREAD)
                            std::stable_sort(fl.begin(), fl.end(), [&](size_t a, size_t b) { return s[a] > s[b]; });
                        for (size_t r = B; r < fl.size(); ++r) refine[fl[r]] = 0;
                        R->levels[level - 1].n_truncated += (int64_t)(fl.size() - B);
                    }
                    G0 = G1;
                }
            }
            std::vector<CellRec> next;
            for (size_t G = 0; G < ng; ++G)
                for (int64_t j = 0; j < k; ++j) {
                    size_t i = G * (size_t)k + (size_t)j;
                    CellRec c = child(parents[G], j);
                    store(level, c, mu[i], s[i], tau[G], refine[i] != 0, &S[i * (size_t)T], &Q[i * (size_t)T]);
                    if (refine[i]) next.push_back(c);
                    else accept(c.instance, mu[i], s[i]);
                }
            parents.swap(next);
        }
    }

    /* ---- depth-first recursion (the paper's picture, Fig. 1); group scope only ---- */
    void refine_dfs(const CellRec& parent, int level) {
        if (level > R->levels_done) R->levels_done = level;
        std::vector<double> mu((size_t)k), s((size_t)k), S((size_t)k * (size_t)T), Q((size_t)k * (size_t)T);
        std::vector<CellRec> cells;
        for (int64_t j = 0; j < k; ++j) {
            cells.push_back(child(parent, j));
            eval_cell(cells.back(), level, &mu[j], &s[j], &S[(size_t)j * (size_t)T], &Q[(size_t)j * (size_t)T]);
        }
        double tau = orc_threshold(s.data(), k, cfg->sigma_multiplier);
        for (int64_t j = 0; j < k; ++j) {
            bool refine = decide(level, cells[j].instance, s[j], tau);
            store(level, cells[j], mu[j], s[j], tau, refine, &S[(size_t)j * (size_t)T], &Q[(size_t)j * (size_t)T]);
            if (refine) refine_dfs(cells[j], level + 1);
            else accept(cells[j].instance, mu[j], s[j]);
        }
    }
    void run_dfs() {
        for (int b = 0; b < cfg->n_instances; ++b) {
            CellRec root; root.instance = (uint32_t)b; root.path = 0; root.coords.assign(D, 0u);
            refine_dfs(root, 1);
        }
    }
};

}  // namespace

orc_result* orc_run(const orc_config* cfg, int keep_cells) {
    orc_result* R = new orc_result();
    const char* e = check_config(cfg);
    if (e) { R->err = e; return R; }
    if (cfg->traversal == ORC_DFS && cfg->threshold_scope != ORC_SCOPE_GROUP) {
        R->err = "depth-first traversal needs the per-group threshold"; return R;
    }
    if (cfg->traversal == ORC_DFS && cfg->budget_order != ORC_BUDGET_PATH_ORDER && cfg->max_groups_per_level > 0) {
        R->err = "a largest-spread budget needs a whole level: breadth-first only"; return R;
    }
    Driver drv(cfg, R, keep_cells != 0);
    if (cfg->traversal == ORC_DFS) drv.run_dfs(); else drv.run_bfs();
    return R;
}

void orc_free(orc_result* r) { delete r; }
const char* orc_error(const orc_result* r) { return r->err.empty() ? nullptr : r->err.c_str(); }
void orc_get(const orc_result* r, double* value, double* std_) {
    for (size_t b = 0; b < r->value.size(); ++b) { value[b] = r->value[b]; std_[b] = std::sqrt(r->var[b]); }
}
int orc_levels(const orc_result* r) { return r->levels_done; }
void orc_level_counts(const orc_result* r, int level, int64_t* n_cells, int64_t* n_refined, int64_t* n_truncated) {
    const LevelStore& ls = r->levels[level - 1];
    if (n_cells) *n_cells = ls.n_cells;
    if (n_refined) *n_refined = ls.n_refined;
    if (n_truncated) *n_truncated = ls.n_truncated;
}
uint64_t orc_total_evals(const orc_result* r) { return r->evals; }
int64_t orc_level_cells(const orc_result* r, int level, uint32_t* instance, uint64_t* path_lo, uint32_t* path_hi,
                        double* mu, double* s, double* tau, uint8_t* refined, double* S) {
    const LevelStore& ls = r->levels[level - 1];
    const size_t n = ls.mu.size();
    for (size_t i = 0; i < n; ++i) {
        if (instance) instance[i] = ls.instance[i];
        if (path_lo) path_lo[i] = ls.path_lo[i];
        if (path_hi) path_hi[i] = ls.path_hi[i];
        if (mu) mu[i] = ls.mu[i];
        if (s) s[i] = ls.s[i];
        if (tau) tau[i] = ls.tau[i];
        if (refined) refined[i] = ls.refined[i];
    }
    if (S) for (size_t i = 0; i < ls.S.size(); ++i) S[i] = ls.S[i];
    return (int64_t)n;
}
int64_t orc_level_sumsq(const orc_result* r, int level, double* Q) {
    const LevelStore& ls = r->levels[level - 1];
    if (Q) for (size_t i = 0; i < ls.Q.size(); ++i) Q[i] = ls.Q[i];
    return (int64_t)(ls.Q.size() / (size_t)(r->trials > 0 ? r->trials : 1));
}

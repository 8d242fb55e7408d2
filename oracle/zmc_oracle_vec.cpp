/*
 * zmc_oracle_vec.cpp -- ORACLE (test infrastructure, NOT the product): vector-valued user integrands.
 *
 * DESIGN.md R15 (ours; the paper's "general user defined functions", and its
 * application whose integrand has "several thousands terms"): an integrand with C components
 * f_0 .. f_{C-1}, all evaluated at the SAME sample points (one stream of random words per (cell, trial) unit,
 * R3, feeds every component). Step by step, breadth-first, in the notation of R2-R7 and R12:
 *
 *   S_j(c,t) = sum_s (double) f_j(x_s)                                                  (R5, per component)
 *   (mu_j(c), s_j(c)) = orc_cell_stats(S_j(c, .))                                      (R5)
 *                       or, with R13, orc_cell_stats_samples(S_j(c, .), Q_j(c, .)), Q_j(c,t) = sum_s f_j(x_s)^2
 *   tau_j(G) = orc_threshold(s_j over the k cells of sibling group G)                  (R6, per component)
 *   cell c of group G is flagged iff level < L and s_j(c) > tau_j(G) for SOME j        (R7 with "any component")
 *   budget B > 0: per instance and level the first B flagged cells in path order       (R12)
 *   refined cells are cut into k children; every other cell is accepted:
 *       value_j += mu_j(c) ; var_j += s_j(c)^2 ;  result (value_j, sqrt(var_j))         (R7)
 *
 * The user function is an INPUT of the method (like the integrand parameters): a C function pointer here, the
 * same source text compiled by NVRTC on the CUDA side. Everything else is built from the scalar oracle's
 * public, pinned primitives (orc_unit_words, orc_cell_geometry, orc_map_f64/f32, orc_cell_stats,
 * orc_threshold); no arithmetic of zmc_oracle.cpp is changed by this file.
 *
 * Pins (tests/test_oracle_vec.py): C = 1 with a user function that restates LINEAR reproduces orc_run bit for
 * bit; polynomial components against their closed forms; a constant component is exact with s = 0; the
 * "any component" rule against the union of single-component runs (brute force); tiling and sum invariants.
 * The rule "any component" itself is a reading (R15): parity unpinned by the paper, like R6.
 */
#include "zmc_oracle.h"

#include <cmath>
#include <string>
#include <vector>

typedef unsigned __int128 u128;

struct orc_vec_result {
    std::string err;
    int C = 1, T = 1, n_instances = 1, levels_done = 0;
    uint64_t evals = 0;
    std::vector<double> value, var;               /* [instance*C + j] */
    struct Level {
        int64_t n_cells = 0, n_refined = 0, n_truncated = 0;
        std::vector<uint32_t> instance;
        std::vector<uint64_t> path_lo;
        std::vector<uint32_t> path_hi;
        std::vector<double> mu, s, tau;           /* [cell*C + j] */
        std::vector<double> S;                    /* [(cell*T + t)*C + j] */
        std::vector<double> Q;                    /* R13: sums of squares, same layout */
        std::vector<uint8_t> refined;
    };
    std::vector<Level> levels;
};

namespace {

struct Cell {
    uint32_t instance;
    u128 path;
    std::vector<uint32_t> coords;
};

/* R2: the j-th child; axis 0 is the least significant digit of j */
Cell child_of(const Cell& parent, int64_t j, int D, int g, int64_t k) {
    Cell c;
    c.instance = parent.instance;
    c.path = parent.path * (u128)k + (u128)j;
    c.coords.resize(D);
    int64_t rem = j;
    for (int d = 0; d < D; ++d) {
        c.coords[d] = parent.coords[d] * (uint32_t)g + (uint32_t)(rem % g);
        rem /= g;
    }
    return c;
}

}  // namespace

extern "C" {

/* S[j] = sum over the unit's N samples of (double) f_j(x_s); sample s takes words s*D .. s*D+D-1 (R3), the point is R4's */
static int vec_unit_sums(const orc_config* cfg, int n_components, orc_user_f64 f64, orc_user_f32 f32, uint32_t instance,
                         uint64_t path_lo, uint32_t path_hi, int level, const uint32_t* coords, int trial, double* S, double* Q) {
    const int D = cfg->dim, C = n_components;
    if (D < 1 || D > 64 || C < 1 || C > 64) return -1;
    if (cfg->precision == ORC_F64 ? !f64 : !f32) return -1;
    double lo[64], width[64], V;
    orc_cell_geometry(D, cfg->lower, cfg->upper, cfg->g, level, coords, lo, width, &V);
    const double* p = cfg->params + (size_t)instance * (size_t)cfg->params_per_instance;
    std::vector<float> pf((size_t)cfg->params_per_instance + 1);
    for (int i = 0; i < cfg->params_per_instance; ++i) pf[i] = (float)p[i];
    for (int j = 0; j < C; ++j) S[j] = 0.0;
    if (Q) for (int j = 0; j < C; ++j) Q[j] = 0.0;
    std::vector<uint32_t> words((size_t)D);
    for (uint64_t s = 0; s < cfg->n_samples; ++s) {
        orc_unit_words(cfg->seed, instance, path_lo, path_hi, level, trial, s * (uint64_t)D, (uint64_t)D, words.data());
        if (cfg->precision == ORC_F64) {
            double x[64], out[64];
            for (int d = 0; d < D; ++d) x[d] = orc_map_f64(words[d], lo[d], width[d]);
            f64(x, D, p, cfg->params_per_instance, out, C);
            for (int j = 0; j < C; ++j) S[j] = S[j] + out[j];
            if (Q) for (int j = 0; j < C; ++j) { const double ff = out[j] * out[j]; Q[j] = Q[j] + ff; }      /* R13: product rounded, then added */
        } else {
            float x[64], out[64];
            for (int d = 0; d < D; ++d) x[d] = orc_map_f32(words[d], lo[d], width[d], 0.0);
            f32(x, D, pf.data(), cfg->params_per_instance, out, C);
            for (int j = 0; j < C; ++j) S[j] = S[j] + (double)out[j];
            if (Q) for (int j = 0; j < C; ++j) { const double fd = (double)out[j]; const double ff = fd * fd; Q[j] = Q[j] + ff; }
        }
    }
    return 0;
}

int orc_vec_unit_sums(const orc_config* cfg, int n_components, orc_user_f64 f64, orc_user_f32 f32, uint32_t instance,
                      uint64_t path_lo, uint32_t path_hi, int level, const uint32_t* coords, int trial, double* S) {
    return vec_unit_sums(cfg, n_components, f64, f32, instance, path_lo, path_hi, level, coords, trial, S, nullptr);
}
/* R13: the same unit, also Q[j] = sum_s f_j(x_s)^2 */
int orc_vec_unit_sums_sq(const orc_config* cfg, int n_components, orc_user_f64 f64, orc_user_f32 f32, uint32_t instance,
                         uint64_t path_lo, uint32_t path_hi, int level, const uint32_t* coords, int trial, double* S, double* Q) {
    return vec_unit_sums(cfg, n_components, f64, f32, instance, path_lo, path_hi, level, coords, trial, S, Q);
}

orc_vec_result* orc_run_vec(const orc_config* cfg, int n_components, orc_user_f64 f64, orc_user_f32 f32, int keep_cells) {
    orc_vec_result* R = new orc_vec_result();
    if (!cfg || cfg->dim < 1 || cfg->dim > 64 || cfg->g < 1 || cfg->trials < 1 || cfg->trials > 255 || cfg->depth < 1 ||
        cfg->depth > 15 || cfg->n_samples < 1 || cfg->n_instances < 1) { R->err = "bad config"; return R; }
    if (n_components < 1 || n_components > 64) { R->err = "n_components out of range (1..64)"; return R; }
    if (cfg->precision == ORC_F64 ? !f64 : !f32) { R->err = "no user function for this precision"; return R; }
    if (cfg->threshold_scope != ORC_SCOPE_GROUP || cfg->traversal != ORC_BFS || cfg->budget_order != ORC_BUDGET_PATH_ORDER) {
        R->err = "vector-valued runs: group scope, BFS, path-order budget only"; return R; }
    const bool from_samples = cfg->spread == ORC_SPREAD_SAMPLES;      /* R13 per component */
    const int D = cfg->dim, g = cfg->g, T = cfg->trials, L = cfg->depth, C = n_components;
    long double bits = (long double)L * (long double)D * std::log2((long double)g);
    if (bits > 80.0L) { R->err = "path exceeds 80 bits"; return R; }
    int64_t k = 1;
    for (int d = 0; d < D; ++d) k *= g;
    R->C = C; R->T = T; R->n_instances = cfg->n_instances;
    R->value.assign((size_t)cfg->n_instances * C, 0.0);
    R->var.assign((size_t)cfg->n_instances * C, 0.0);
    R->levels.resize(L);

    std::vector<Cell> parents;
    for (int b = 0; b < cfg->n_instances; ++b) {
        Cell root; root.instance = (uint32_t)b; root.path = 0; root.coords.assign(D, 0u);
        parents.push_back(root);
    }
    for (int level = 1; level <= L && !parents.empty(); ++level) {
        R->levels_done = level;
        orc_vec_result::Level& LS = R->levels[level - 1];
        const size_t ng = parents.size(), n = ng * (size_t)k;
        std::vector<double> mu(n * C), s(n * C), S(n * (size_t)T * C), Q(from_samples ? n * (size_t)T * C : 0);
        /* every cell: T trials, C sums each, then (mu_j, s_j) by R5 */
        for (size_t G = 0; G < ng; ++G)
            for (int64_t j = 0; j < k; ++j) {
                const Cell c = child_of(parents[G], j, D, g, k);
                const size_t i = G * (size_t)k + (size_t)j;
                for (int t = 0; t < T; ++t)
                    vec_unit_sums(cfg, C, f64, f32, c.instance, (uint64_t)c.path, (uint32_t)(c.path >> 64), level, c.coords.data(), t,
                                  &S[(i * (size_t)T + (size_t)t) * C], from_samples ? &Q[(i * (size_t)T + (size_t)t) * C] : nullptr);
                R->evals += (uint64_t)T * cfg->n_samples;
                double lo[64], width[64], V;
                orc_cell_geometry(D, cfg->lower, cfg->upper, g, level, c.coords.data(), lo, width, &V);
                std::vector<double> St((size_t)T), Qt((size_t)T);
                for (int q = 0; q < C; ++q) {
                    for (int t = 0; t < T; ++t) St[t] = S[(i * (size_t)T + (size_t)t) * C + q];
                    if (from_samples) {
                        for (int t = 0; t < T; ++t) Qt[t] = Q[(i * (size_t)T + (size_t)t) * C + q];
                        orc_cell_stats_samples(St.data(), Qt.data(), T, V, 1.0, cfg->n_samples, &mu[i * C + q], &s[i * C + q]);
                    } else {
                        orc_cell_stats(St.data(), T, V, 1.0, cfg->n_samples, nullptr, &mu[i * C + q], &s[i * C + q]);
                    }
                }
            }
        /* R6 per component and sibling group */
        std::vector<double> tau(ng * C), col((size_t)k);
        for (size_t G = 0; G < ng; ++G)
            for (int q = 0; q < C; ++q) {
                for (int64_t j = 0; j < k; ++j) col[(size_t)j] = s[(G * (size_t)k + (size_t)j) * C + q];
                tau[G * C + q] = orc_threshold(col.data(), k, cfg->sigma_multiplier);
            }
        /* R7 / R15: flagged iff level < L and SOME component has s_j > tau_j (strict; NaN compares false) */
        std::vector<char> refine(n, 0);
        for (size_t i = 0; i < n; ++i) {
            bool any = false;
            for (int q = 0; q < C; ++q) any = any || (s[i * C + q] > tau[(i / (size_t)k) * C + q]);
            refine[i] = (level < L && any) ? 1 : 0;
        }
        /* R12: per instance the first B flagged cells in path order (parents are sorted by instance, then path) */
        if (cfg->max_groups_per_level > 0) {
            std::vector<int64_t> taken((size_t)cfg->n_instances, 0);
            for (size_t i = 0; i < n; ++i) {
                if (!refine[i]) continue;
                const uint32_t b = parents[i / (size_t)k].instance;
                if (taken[b] >= cfg->max_groups_per_level) { refine[i] = 0; LS.n_truncated++; }
                else taken[b]++;
            }
        }
        std::vector<Cell> next;
        for (size_t G = 0; G < ng; ++G)
            for (int64_t j = 0; j < k; ++j) {
                const size_t i = G * (size_t)k + (size_t)j;
                const Cell c = child_of(parents[G], j, D, g, k);
                LS.n_cells++;
                if (refine[i]) { LS.n_refined++; next.push_back(c); }
                else
                    for (int q = 0; q < C; ++q) {
                        double& v = R->value[(size_t)c.instance * C + q];
                        double& w = R->var[(size_t)c.instance * C + q];
                        v = v + mu[i * C + q];
                        const double ss = s[i * C + q] * s[i * C + q];
                        w = w + ss;
                    }
                if (keep_cells) {
                    LS.instance.push_back(c.instance);
                    LS.path_lo.push_back((uint64_t)c.path);
                    LS.path_hi.push_back((uint32_t)(c.path >> 64));
                    LS.refined.push_back(refine[i] ? 1 : 0);
                    for (int q = 0; q < C; ++q) { LS.mu.push_back(mu[i * C + q]); LS.s.push_back(s[i * C + q]); LS.tau.push_back(tau[G * C + q]); }
                    for (size_t e = 0; e < (size_t)T * C; ++e) LS.S.push_back(S[i * (size_t)T * C + e]);
                    if (from_samples) for (size_t e = 0; e < (size_t)T * C; ++e) LS.Q.push_back(Q[i * (size_t)T * C + e]);
                }
            }
        parents.swap(next);
    }
    return R;
}

void orc_vec_free(orc_vec_result* r) { delete r; }
const char* orc_vec_error(const orc_vec_result* r) { return r->err.empty() ? nullptr : r->err.c_str(); }
/* value, std: [n_instances * n_components], component fastest */
void orc_vec_get(const orc_vec_result* r, double* value, double* std_) {
    for (size_t i = 0; i < r->value.size(); ++i) { value[i] = r->value[i]; std_[i] = std::sqrt(r->var[i]); }
}
int orc_vec_levels(const orc_vec_result* r) { return r->levels_done; }
uint64_t orc_vec_total_evals(const orc_vec_result* r) { return r->evals; }
void orc_vec_level_counts(const orc_vec_result* r, int level, int64_t* n_cells, int64_t* n_refined, int64_t* n_truncated) {
    const orc_vec_result::Level& ls = r->levels[level - 1];
    if (n_cells) *n_cells = ls.n_cells;
    if (n_refined) *n_refined = ls.n_refined;
    if (n_truncated) *n_truncated = ls.n_truncated;
}
/* kept cells of one level in evaluation order; mu, s, tau: [cells*C]; S: [cells*T*C] (trial-major, component fastest) */
int64_t orc_vec_level_cells(const orc_vec_result* r, int level, uint32_t* instance, uint64_t* path_lo, uint32_t* path_hi,
                            double* mu, double* s, double* tau, uint8_t* refined, double* S) {
    const orc_vec_result::Level& ls = r->levels[level - 1];
    const size_t n = ls.refined.size();
    for (size_t i = 0; i < n; ++i) {
        if (instance) instance[i] = ls.instance[i];
        if (path_lo) path_lo[i] = ls.path_lo[i];
        if (path_hi) path_hi[i] = ls.path_hi[i];
        if (refined) refined[i] = ls.refined[i];
    }
    for (size_t i = 0; i < ls.mu.size(); ++i) {
        if (mu) mu[i] = ls.mu[i];
        if (s) s[i] = ls.s[i];
        if (tau) tau[i] = ls.tau[i];
    }
    if (S) for (size_t i = 0; i < ls.S.size(); ++i) S[i] = ls.S[i];
    return (int64_t)n;
}

/* R13: per-(cell, trial, component) sums of squares of one level, [cells*T*C]; nothing unless spread = samples and keep_cells */
int64_t orc_vec_level_sumsq(const orc_vec_result* r, int level, double* Q) {
    const orc_vec_result::Level& ls = r->levels[level - 1];
    if (Q) for (size_t i = 0; i < ls.Q.size(); ++i) Q[i] = ls.Q[i];
    return (int64_t)ls.Q.size();
}

}  /* extern "C" */

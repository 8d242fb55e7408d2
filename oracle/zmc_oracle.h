/*
 * zmc_oracle.h -- ORACLE (test infrastructure, NOT the product).
 *
 * A plain, slow, single-threaded CPU restatement of the hot path of ZMCintegral
 * (arXiv:1902.07916): stratified Monte-Carlo over a grid of cells with the
 * heuristic tree search of PAPER.md:69-73 (section 2.1, Fig. 1).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this library. It shares no code, header,
 * table or constant generator with paper_1902_07916_b200/csrc (the CUDA path).
 *
 * Every convention the paper leaves open is fixed in DESIGN.md section 3
 * ("Readings"); the R-numbers in the comments below refer to that list.
 *
 * Parity status: the *form* of the threshold, its scope, the ddof of the
 * standard deviations and how cell stds are "collected" are
 * readings, "parity unpinned" by the paper (its tables print no formula and
 * its numbers match none exactly); everything else is pinned in
 * tests/test_oracle_*.py. The "any component" flag rule of vector-valued integrands
 * (R15, zmc_oracle_vec.cpp) is a reading as well: parity unpinned by the paper.
 */
#ifndef ZMC_ORACLE_H
#define ZMC_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { ORC_CONST = 0, ORC_LINEAR = 1, ORC_SIN_SUM = 2, ORC_EXP_QUAD = 3 };
enum { ORC_F64 = 0, ORC_F32 = 1 };
enum { ORC_SCOPE_GROUP = 0, ORC_SCOPE_POOLED = 1 };
enum { ORC_BFS = 0, ORC_DFS = 1 };
enum { ORC_SPREAD_TRIALS = 0, ORC_SPREAD_SAMPLES = 1 };   /* R13 */
enum { ORC_BUDGET_PATH_ORDER = 0, ORC_BUDGET_LARGEST_SPREAD = 1 };   /* R14 */

typedef struct orc_config {
    int32_t dim;                 /* D */
    int32_t g;                   /* divisions per axis; k = g^D cells per split */
    int32_t trials;              /* n1 independent repetitions */
    int32_t depth;               /* L = number of levels evaluated */
    uint64_t n_samples;          /* N uniform points per cell per trial */
    uint64_t seed;
    double sigma_multiplier;     /* m in tau = mean(s) + m*pstd(s) */
    int32_t integrand;           /* ORC_CONST .. ORC_EXP_QUAD */
    int32_t precision;           /* ORC_F64 or ORC_F32 (canonical FP32 operation sequence) */
    int32_t n_instances;         /* independent integrals sharing geometry (R11) */
    int32_t params_per_instance;
    int32_t threshold_scope;     /* ORC_SCOPE_GROUP (default reading R6) or ORC_SCOPE_POOLED */
    int32_t traversal;           /* ORC_BFS or ORC_DFS (R2: both give the same numbers) */
    int64_t max_groups_per_level;/* R12 refinement budget per instance and level; <= 0 = off */
    int32_t spread;              /* R13: ORC_SPREAD_TRIALS (the paper, default) or ORC_SPREAD_SAMPLES */
    int32_t budget_order;        /* R14: which flagged cells the budget keeps: first in path order (R12, default) or largest spread */
    const double* lower;         /* [D] */
    const double* upper;         /* [D] */
    const double* params;        /* [n_instances * params_per_instance] */
} orc_config;

/* ---- R1: Philox4x32-10 (Salmon et al., SC'11), counter c[4], key k[2] ---- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* ---- R3: per-instance derived key Kd(seed, b) ---- */
void orc_derive_key(uint64_t seed, uint32_t instance, uint32_t key[2]);
/* ---- R3: n_words words of the flat stream of unit (path, level, trial), starting at word index first_word ---- */
void orc_unit_words(uint64_t seed, uint32_t instance, uint64_t path_lo, uint32_t path_hi, int level,
                    int trial, uint64_t first_word, uint64_t n_words, uint32_t* out);
/* ---- R2: geometry of the level-`level` cell with integer coordinates coords[D] ---- */
void orc_cell_geometry(int dim, const double* lower, const double* upper, int g, int level,
                       const uint32_t* coords, double* lo, double* width, double* volume);
/* ---- R4: word -> coordinate ---- */
double orc_map_f64(uint32_t w, double lo, double width);
float orc_map_f32(uint32_t w, double lo, double width, double centre /* subtracted in FP64 before rounding the base; 0 for none */);
/* ---- R8: canonical FP32 elementary functions ---- */
float orc_zsin(float a);
/* zexp: returns the FP32 significand part p and writes the power of two n: exp(e) ~= p * 2^n */
float orc_zexp(float e, int32_t* n);
/* zexp assembled as the FP64 number the accumulation uses (0 for e < -708) */
double orc_zexp_value(float e);

/* ---- one (cell, trial) unit: S = sum_s f(x_s) in FP64, Sabs = sum |f| ---- */
int orc_unit_sum(const orc_config* cfg, uint32_t instance, uint64_t path_lo, uint32_t path_hi, int level,
                 const uint32_t* coords, int trial, double* S, double* Sabs);
/* R13: the same unit, also Q = sum_s f(x_s)^2 (FP64: product rounded, then added) */
int orc_unit_sums(const orc_config* cfg, uint32_t instance, uint64_t path_lo, uint32_t path_hi, int level,
                  const uint32_t* coords, int trial, double* S, double* Q);
/* first `n` sample points of a unit (FP64 mode: doubles; FP32 mode: floats widened to double) and f values */
int orc_unit_points(const orc_config* cfg, uint32_t instance, uint64_t path_lo, uint32_t path_hi, int level,
                    const uint32_t* coords, int trial, uint64_t n, double* x /* [n*D] */, double* f /* [n] */);

/* ---- R5: trial estimates -> (mu, s) ; R6: threshold of one set of stds ---- */
void orc_cell_stats(const double* S, int trials, double volume, double prefactor, uint64_t n_samples,
                    double* I /* [trials] or NULL */, double* mu, double* s);
/* R13: spread from the samples. mu as in R5; with M = T*N, Sc = sum_t S_t, Qc = sum_t Q_t:
 *   d = Qc - (Sc*Sc)/M ; d = 0 unless d > Qc * 2^-40 ; s = (V*A) * sqrt((d/M) / M)   -- the standard error of mu */
void orc_cell_stats_samples(const double* S, const double* Q, int trials, double volume, double prefactor,
                            uint64_t n_samples, double* mu, double* s);
double orc_threshold(const double* s, int64_t k, double m);

/* ---- whole tree (R7) ---- */
typedef struct orc_result orc_result;
orc_result* orc_run(const orc_config* cfg, int keep_cells);
void orc_free(orc_result*);
const char* orc_error(const orc_result*);           /* NULL if ok */
void orc_get(const orc_result*, double* value, double* std); /* [n_instances] each */
int orc_levels(const orc_result*);                   /* levels actually evaluated */
/* per-level counters: cells evaluated, cells flagged for refinement (after budget), flagged cells dropped by the budget */
void orc_level_counts(const orc_result*, int level, int64_t* n_cells, int64_t* n_refined, int64_t* n_truncated);
uint64_t orc_total_evals(const orc_result*);
/* kept cells of one level in evaluation order (BFS: ascending (instance, path)); any pointer may be NULL */
int64_t orc_level_cells(const orc_result*, int level, uint32_t* instance, uint64_t* path_lo, uint32_t* path_hi,
                        double* mu, double* s, double* tau, uint8_t* refined, double* S /* [cells*T] */);

/* R13: per-(cell, trial) sums of squares of one level, [cells*T]; 0 cells unless spread = samples and keep_cells */
int64_t orc_level_sumsq(const orc_result*, int level, double* Q);

/* ---- R15: vector-valued user integrands (zmc_oracle_vec.cpp). The user function is an input of the method: it writes
 * n_out components of f at the point x (the FP64 or the FP32 arithmetic, by cfg->precision). cfg->integrand is ignored;
 * group scope, breadth-first, path-order budget only; the spread from the trials (R5) or, per component, from the samples (R13). ---- */
typedef void (*orc_user_f64)(const double* x, int dim, const double* p, int np, double* out, int n_out);
typedef void (*orc_user_f32)(const float* x, int dim, const float* p, int np, float* out, int n_out);
typedef struct orc_vec_result orc_vec_result;
/* S[j] = sum_s (double) f_j(x_s) of one (cell, trial) unit, j = 0 .. n_components-1 */
int orc_vec_unit_sums(const orc_config* cfg, int n_components, orc_user_f64 f64, orc_user_f32 f32, uint32_t instance,
                      uint64_t path_lo, uint32_t path_hi, int level, const uint32_t* coords, int trial, double* S);
/* R13: the same unit, also Q[j] = sum_s f_j(x_s)^2 */
int orc_vec_unit_sums_sq(const orc_config* cfg, int n_components, orc_user_f64 f64, orc_user_f32 f32, uint32_t instance,
                         uint64_t path_lo, uint32_t path_hi, int level, const uint32_t* coords, int trial, double* S, double* Q);
orc_vec_result* orc_run_vec(const orc_config* cfg, int n_components, orc_user_f64 f64, orc_user_f32 f32, int keep_cells);
void orc_vec_free(orc_vec_result*);
const char* orc_vec_error(const orc_vec_result*);
void orc_vec_get(const orc_vec_result*, double* value, double* std);   /* [n_instances * n_components], component fastest */
int orc_vec_levels(const orc_vec_result*);
uint64_t orc_vec_total_evals(const orc_vec_result*);
void orc_vec_level_counts(const orc_vec_result*, int level, int64_t* n_cells, int64_t* n_refined, int64_t* n_truncated);
/* mu, s, tau: [cells * C]; S: [cells * T * C] (trial-major, component fastest); any pointer may be NULL */
int64_t orc_vec_level_sumsq(const orc_vec_result*, int level, double* Q);   /* R13: [cells * T * C] */
int64_t orc_vec_level_cells(const orc_vec_result*, int level, uint32_t* instance, uint64_t* path_lo, uint32_t* path_hi,
                            double* mu, double* s, double* tau, uint8_t* refined, double* S);

#ifdef __cplusplus
}
#endif
#endif

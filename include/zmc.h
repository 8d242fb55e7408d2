/*
 * zmc.h -- C ABI of libzmc.so: the B200 (sm_100a) hot path of ZMCintegral
 * (arXiv:1902.07916): stratified Monte-Carlo over a grid of hyper-rectangular cells
 * with the heuristic tree search of the paper's section 2.1.
 *
 * Citations are "PAPER.md:<line>" (the paper's text) and "DESIGN.md R<n>" (the reading
 * this build takes where the paper is silent). BASELINE.json names the four core calls
 * (zmc_create, zmc_set_integrand, zmc_run, zmc_result); the others are what those four
 * cannot work without (options, workspace, statistics, level dumps for parity tests).
 *
 * Conventions for every call
 *   - return value: ZMC_OK (0) or a negative zmc_status; nothing throws or aborts.
 *     zmc_last_error(ctx) gives a human-readable reason for the last failure on ctx.
 *   - every pointer argument marked [host] is caller-owned host memory, read or written
 *     during the call only (inputs are copied); [device] pointers are CUDA device memory.
 *   - a context is used from one host thread at a time; distinct contexts are independent.
 *   - all work is enqueued on the CUDA stream given to zmc_run; only zmc_result,
 *     zmc_stats and zmc_level_cells synchronise that stream.
 *   - the library needs a CUDA device; without one zmc_create fails with ZMC_ERR_CUDA.
 *     There is no CPU fallback of any kind.
 */
#ifndef ZMC_H
#define ZMC_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ZMC_MAX_DIM 16      /* D <= 16 (D <= 12 pre-compiled, 13..16 JIT-compiled) */
#define ZMC_MAX_DEPTH 15    /* level fits 4 bits of the Philox counter (R3) */
#define ZMC_MAX_TRIALS 255  /* trial fits 8 bits of the Philox counter (R3) */
#define ZMC_MAX_COMPONENTS 16 /* components of a vector-valued user integrand (R15) */

typedef enum zmc_status {
    ZMC_OK = 0,
    ZMC_ERR_ARG = -1,          /* null pointer, non-finite or empty bounds, counts < 1 ... */
    ZMC_ERR_RANGE = -2,        /* path > 80 bits, g^depth > 2^32, N*D >= 2^34 - 2^14, trials > 255, depth > 15, dim > 16 (R3) */
    ZMC_ERR_NO_INTEGRAND = -3, /* zmc_run before zmc_set_integrand* */
    ZMC_ERR_COMPILE = -4,      /* NVRTC failed; the log is in zmc_last_error */
    ZMC_ERR_CUDA = -5,         /* a CUDA runtime call failed (or no device) */
    ZMC_ERR_CAPACITY = -6,     /* a level needed more cells than max_cells_per_level; result invalid */
    ZMC_ERR_NOT_RUN = -7,      /* zmc_result / zmc_stats / zmc_level_cells before zmc_run */
    ZMC_ERR_STATE = -8         /* option changed after the workspace was fixed, level stats not kept, an option not defined for a
                                  vector-valued integrand ... */
} zmc_status;

/* Built-in integrands. params = [n_instances][params_per_instance] doubles.
 *   ZMC_CONST     f = p[0]                                          (test integrand)
 *   ZMC_LINEAR    f = p[0] + sum_d p[1+d] x_d                       (test integrand)
 *   ZMC_SIN_SUM   f = sin(sum_d x_d)            paper f1, Eq. (1); no parameters
 *   ZMC_EXP_QUAD  f = p[0] * exp(-p[1] * |x - c|^2), c_d = p[2+d]
 *                 paper f2, Eq. (2), is p[0] = (2 pi sigma^2)^(-D/2), p[1] = 1/(2 sigma^2), c = 0.
 *                 The prefactor p[0] multiplies each trial estimate, not each sample (R8). */
enum { ZMC_CONST = 0, ZMC_LINEAR = 1, ZMC_SIN_SUM = 2, ZMC_EXP_QUAD = 3, ZMC_USER = 100 };

/* zmc_set_option keys */
enum {
    ZMC_OPT_PRECISION = 1,            /* ZMC_F64 (default) or ZMC_F32: arithmetic of map + integrand; sums are always FP64 */
    ZMC_OPT_MATH = 2,                 /* ZMC_MATH_EXACT (default): documented IEEE op sequence, bit-comparable with a CPU
                                         (R8); ZMC_MATH_FAST: MUFU sin/ex2 (FP32 only) */
    ZMC_OPT_MAX_GROUPS_PER_LEVEL = 3, /* refinement budget B per instance and level, first B flagged cells in path
                                         order (R12); 0 = off = the paper's semantics (default) */
    ZMC_OPT_KEEP_LEVEL_STATS = 4,     /* 1: keep every level's per-cell arrays for zmc_level_cells (default 0) */
    ZMC_OPT_MAX_CELLS_PER_LEVEL = 5,  /* capacity of one level in cells. 0 = automatic (default): sized for the budget if there is one; else a
                                         modest guess (128 x level 1, within 2^22 .. 2^28 cells), and if a level outgrows it the search stops
                                         there, zmc_result learns what that level needed, allocates a workspace for it (library-owned
                                         workspaces only, if the device has the memory) and runs the search again -- same seeds, same bits as
                                         a run that had the room from the start. BASELINE.json configs[1] as given (4.5e8 cells at level 3)
                                         runs this way with no option set. A value > 0 is a hard limit: ZMC_ERR_CAPACITY beyond it */
    ZMC_OPT_GRID_BLOCKS = 6,          /* persistent sampling grid in CTAs; 0 = auto (SM count x resident CTAs) */
    ZMC_OPT_TARGET_ITEMS = 7,         /* a level with fewer (cell,trial) units than this is split into sample chunks
                                         until it has about this many work items (default 65536) */
    ZMC_OPT_USE_GRAPH = 8,            /* 1: zmc_run captures its kernel sequence into a CUDA graph once and replays it
                                         (one launch per run instead of 2 + 6*depth; for launch-bound problems such as
                                         BASELINE.json configs[0]); per-level times in zmc_stats are then 0 (default 0) */
    ZMC_OPT_SPREAD = 9,               /* ZMC_SPREAD_TRIALS (default, the paper: s = std of the T trial estimates) or
                                         ZMC_SPREAD_SAMPLES (R13: s = standard error of the cell mean from sum f and
                                         sum f^2 of its T*N samples; zmc_result's std is then a 1-sigma error; per component for a
                                         vector-valued integrand) */
    ZMC_OPT_BUDGET_ORDER = 10,        /* which flagged cells the budget keeps: ZMC_BUDGET_PATH_ORDER (default, R12) or
                                         ZMC_BUDGET_LARGEST_SPREAD (R14: the B largest s, equal ones in path order) */
    ZMC_OPT_SINGLE_LAUNCH = 11        /* the whole tree search as ONE cooperative kernel launch (grid-wide barriers between the
                                         sampling and control phases of every level) instead of 2 + 6*depth launches: for
                                         launch-bound problems (BASELINE.json configs[0]; PAPER.md:162-184 is about this per-call
                                         overhead). Same device functions, bit-identical results. 0 never, 1 whenever the kernel
                                         exists (built-in integrands of at most 8 dimensions in FP64 or exact FP32, ZMC_SPREAD_TRIALS, path-order budget), 2 = auto (default):
                                         when level 1 has at most 4e6 evaluations and no later level can have more than 6.4e7 (by the budget,
                                         by depth 2, or by the level capacity). 1 and 2 are preferences: if the driver refuses the
                                         cooperative launch (fewer SMs than the device reports under an MPS thread percentage or a green
                                         context; a tool in between) the run goes kernel by kernel, with the same bits. zmc_stats: kernel_launches 1; the per-level times come
                                         from %globaltimer stamps at the kernel's grid barriers (ZMC_TREE_MARKS=1 in the environment prints
                                         the finer split to stderr) */
};
enum { ZMC_F64 = 0, ZMC_F32 = 1 };
enum { ZMC_MATH_EXACT = 0, ZMC_MATH_FAST = 1 };
enum { ZMC_SPREAD_TRIALS = 0, ZMC_SPREAD_SAMPLES = 1 };
enum { ZMC_BUDGET_PATH_ORDER = 0, ZMC_BUDGET_LARGEST_SPREAD = 1 };

typedef struct zmc_ctx zmc_ctx; /* opaque; owned by the library between zmc_create and zmc_destroy */

/* The parameters of PAPER.md:87 (section 2.3) in BASELINE.json's order.
 *   out                [host] receives the context
 *   dim                D, 1..ZMC_MAX_DIM
 *   lower, upper       [host] D doubles each: the integration box, upper_d > lower_d, finite
 *   divisions_per_axis g >= 1: every (sub-)domain is cut into k = g^D equal cells
 *   samples_per_cell   N >= 1 uniform points per cell per trial
 *   trials             n1 = T independent repetitions per cell, 1..255
 *   depth              L = number of levels evaluated; depth 1 = no refinement, 1..15
 *   sigma_multiplier   m in the threshold tau = mean(s) + m * pstd(s) of one sibling group (R6)
 *   seed               Philox seed (R3)
 * Limits (else ZMC_ERR_RANGE): samples_per_cell * dim < 2^34 - 2^14, depth * dim * log2(g) <= 80, g^depth <= 2^32, g^dim <= 2^40.
 * On failure *out is NULL -- there is nothing to destroy -- and zmc_last_error(NULL) gives the reason. */
int zmc_create(zmc_ctx** out, int dim, const double* lower, const double* upper, int divisions_per_axis,
               uint64_t samples_per_cell, int trials, int depth, double sigma_multiplier, uint64_t seed);

/* Choose a built-in integrand. n_instances >= 1 independent integrals share the geometry and the seed,
 * each with its own parameters, Philox key, thresholds and (value, std) (R11).
 * params [host] n_instances*params_per_instance doubles (may be NULL iff params_per_instance == 0). */
int zmc_set_integrand(zmc_ctx* ctx, int builtin_id, const double* params, int params_per_instance, int n_instances);

/* Choose a user integrand given as CUDA source, JIT-compiled with NVRTC for sm_100a together with the
 * sampling kernel so that it inlines. cuda_src [host] must define
 *     __device__ float  fn_name(const float*  x, int dim, const float*  p, int np)   (ZMC_F32)
 *     __device__ double fn_name(const double* x, int dim, const double* p, int np)   (ZMC_F64)
 * x = the sample point, p = this instance's parameters. Parity with a CPU holds for built-ins only.
 * The program is compiled DURING THIS CALL, for the precision, math mode and spread in force now (the default precision is
 * ZMC_F64), so that a compile error surfaces here with the NVRTC log in zmc_last_error: a source that defines one overload
 * only needs that precision set BEFORE this call. A later zmc_set_option(ZMC_OPT_PRECISION / MATH / SPREAD) recompiles at
 * once; if that fails it returns ZMC_ERR_COMPILE and the context keeps its previous, working setting.
 * Compiled programs are cached per process, and on disk as well if the environment variable ZMC_CACHE_DIR names a
 * writable directory (keyed by the complete program text; a stale or foreign file is ignored). */
int zmc_set_integrand_source(zmc_ctx* ctx, const char* cuda_src, const char* fn_name, const double* params,
                             int params_per_instance, int n_instances);

/* A VECTOR-VALUED user integrand (R15; the paper's "general user defined functions", and its application with
 * an integrand of "several thousands terms"): n_components values f_0 .. f_{C-1} per point, 1 <= C <= ZMC_MAX_COMPONENTS,
 * all evaluated at the same sample points -- one random stream and one map per (cell, trial) unit, C FP64 sums. cuda_src [host] must define
 *     __device__ void fn_name(const float*  x, int dim, const float*  p, int np, float*  out, int n_out)   (ZMC_F32)
 *     __device__ void fn_name(const double* x, int dim, const double* p, int np, double* out, int n_out)   (ZMC_F64)
 * which writes out[0 .. n_out), n_out = n_components. Each component gets its own per-cell (mu, s) and per-group threshold; a cell is
 * refined iff SOME component's s exceeds that component's threshold; zmc_result then returns n_instances * n_components values and
 * stds, [instance][component], and the per-cell arrays of zmc_level_cells* carry C entries per cell (mu, s, tau: [cell*C + j];
 * S: [(cell*T + t)*C + j]). Compiled during this call like zmc_set_integrand_source. ZMC_SPREAD_SAMPLES applies per component
 * (R13, R15). ZMC_ERR_STATE if ZMC_BUDGET_LARGEST_SPREAD is in force with C > 1 (not defined for several components);
 * ZMC_ERR_RANGE for C outside 1..16. */
int zmc_set_integrand_source_vec(zmc_ctx* ctx, const char* cuda_src, const char* fn_name, int n_components, const double* params,
                                 int params_per_instance, int n_instances);

/* Returns ZMC_ERR_ARG for an unknown key or a value out of range, ZMC_ERR_STATE for a value that changes the workspace
 * layout (KEEP_LEVEL_STATS, MAX_CELLS_PER_LEVEL, TARGET_ITEMS, SPREAD, BUDGET_ORDER) after zmc_set_workspace has fixed a
 * caller-owned workspace and a run has laid it out. On any error the context is unchanged. */
int zmc_set_option(zmc_ctx* ctx, int key, int64_t value);

/* Device memory the run needs under the options in force. Optional: without zmc_set_workspace the
 * library allocates with cudaMalloc at the first zmc_run. workspace [device], 256-byte aligned,
 * caller-owned, must outlive the context or the next zmc_set_workspace. */
int zmc_workspace_bytes(zmc_ctx* ctx, size_t* bytes);
int zmc_set_workspace(zmc_ctx* ctx, void* workspace, size_t bytes);

/* Enqueue the whole tree search -- every level's sampling, statistics, threshold, flag and compaction
 * kernels -- on cuda_stream (a cudaStream_t; NULL = the default stream) and return without
 * synchronising. No host decision is taken between levels.
 * The first zmc_run after zmc_set_integrand* or a layout change does the one-time work first: kernel
 * selection (NVRTC if needed), workspace allocation, parameter upload and key derivation, and waits
 * for that upload (the derived key of a single-instance run travels back as a launch parameter). */
int zmc_run(zmc_ctx* ctx, void* cuda_stream);

/* Synchronise the run's stream and fetch, per instance, the integral estimate (sum of accepted cell
 * means) and its standard deviation (sqrt of the sum of accepted cell variances, R7).
 * value, std [host] n_instances doubles each (n_instances * n_components, [instance][component], for a vector-valued
 * integrand). If a level overflowed: with the automatic capacity and a library-owned workspace the workspace is grown to what
 * that level needed and the search is run again from here, on the same stream, once per overflowing level (this call then takes
 * as long as those runs); otherwise ZMC_ERR_CAPACITY, and zmc_last_error says which level needed how many cells. */
int zmc_result(zmc_ctx* ctx, double* value, double* std);

typedef struct zmc_level_stats {
    uint64_t n_groups;     /* sibling groups (= parents) evaluated at this level */
    uint64_t n_cells;      /* cells evaluated = n_groups * k */
    uint64_t n_flagged;    /* cells with s > tau (level < L) */
    uint64_t n_refined;    /* flagged cells passed on to the next level (after budget / capacity) */
    uint64_t evals;        /* integrand evaluations = n_cells * T * N */
    float sample_ms;       /* device time of this level's sampling kernel (CUDA events) */
    float control_ms;      /* device time of this level's statistics/threshold/flag/compaction kernels */
} zmc_level_stats;

typedef struct zmc_stats_t {
    int32_t levels;                 /* = depth */
    int32_t overflow;               /* 1 if some level exceeded max_cells_per_level */
    uint64_t nonfinite;             /* cells whose mean or std is not finite */
    uint64_t total_evals;
    float total_ms;                 /* first kernel to last kernel of the run */
    int32_t regs_per_thread;        /* sampling kernel */
    int32_t grid_blocks, block_threads;
    int32_t kernel_origin;          /* sampling kernel: 0 pre-compiled, 1 compiled by NVRTC for this context, 2 from the process-wide
                                       cache, 3 from the on-disk cache (ZMC_CACHE_DIR) */
    int32_t kernel_launches;        /* kernels the last zmc_run enqueued (all the library's own; a CUDA graph replays the same nodes;
                                       1 = the single-launch path, ZMC_OPT_SINGLE_LAUNCH) */
    zmc_level_stats level[ZMC_MAX_DEPTH];
} zmc_stats_t;

int zmc_stats(zmc_ctx* ctx, zmc_stats_t* out);

/* Per-cell arrays of one level (1-based), in evaluation order = ascending (instance, path); needs
 * ZMC_OPT_KEEP_LEVEL_STATS. Any [host] pointer may be NULL. capacity = number of cells the arrays can
 * hold; *n_cells receives the level's cell count (call once with capacity 0 to size them).
 *   instance[c], path_lo[c], path_hi[c]  cell identity (R2: path P' = P*k + j)
 *   mu[c], s[c]        mean and population std of the T trial estimates (R5)
 *   tau[c]             threshold of the cell's sibling group (R6)
 *   refined[c]         1 if the cell was subdivided
 *   S[c*T + t]         per-(cell, trial) sum of f over the N samples, FP64 */
int zmc_level_cells(zmc_ctx* ctx, int level, uint64_t capacity, uint64_t* n_cells, uint32_t* instance,
                    uint64_t* path_lo, uint32_t* path_hi, double* mu, double* s, double* tau, uint8_t* refined,
                    double* S);

/* The same arrays for the cells [first_cell, first_cell + count) of the level only (a level of a deep, unbudgeted tree can
 * hold 10^8 cells and more: BASELINE.json configs[1] at depth 3). Every non-NULL [host] array holds count entries (S: count*T).
 * ZMC_ERR_ARG if the range passes the level's cell count.
 * Both dump calls take mu, s, tau, refined, S and the parents' (instance, path) from device memory as the kernels wrote them;
 * a cell's own path P' = P*k + j is then formed on the host from its parent's path P and its position j in the group (128-bit
 * integer arithmetic). The device forms the same P' per work item for the Philox counter and does not store it. */
int zmc_level_cells_range(zmc_ctx* ctx, int level, uint64_t first_cell, uint64_t count, uint32_t* instance,
                          uint64_t* path_lo, uint32_t* path_hi, double* mu, double* s, double* tau, uint8_t* refined,
                          double* S);

/* Per-(cell, trial) sums of f^2 of one level, Q[c*T + t], FP64 (R13); needs ZMC_OPT_KEEP_LEVEL_STATS and
 * ZMC_SPREAD_SAMPLES. Q [host] capacity*T doubles (capacity*T*n_components, Q[(c*T + t)*C + j], for a vector-valued integrand),
 * capacity >= the level's cell count. */
int zmc_level_sumsq(zmc_ctx* ctx, int level, uint64_t capacity, double* Q);

/* Raw generator access for parity tests (R1, R3): n_words words of the flat stream of unit
 * (instance, path, level, trial) starting at word index first_word, produced by the device code.
 * out [host] n_words uint32. */
int zmc_debug_words(zmc_ctx* ctx, uint32_t instance, uint64_t path_lo, uint32_t path_hi, int level, int trial,
                    uint64_t first_word, uint64_t n_words, uint32_t* out);

/* Sample points and integrand values of the first n samples of one unit, produced by the same device
 * functions the sampling kernel uses. coords [host] D level-`level` integer cell coordinates.
 * x [host] n*D doubles (FP32 mode: floats widened; EXP_QUAD in FP32: x - c, R8), f [host] n doubles
 * (n * n_components, component fastest, for a vector-valued integrand). */
int zmc_debug_points(zmc_ctx* ctx, uint32_t instance, uint64_t path_lo, uint32_t path_hi, int level,
                     const uint32_t* coords, int trial, uint64_t n, double* x, double* f);

/* ---- One level of stratified sampling WITHOUT any device-memory allocation ------------------------------------------------------
 * For callers that cannot allocate on the GPU: a process whose device memory is already spoken for down to the last byte (another
 * component's memory pool holds the card, so cudaMalloc fails), or a latency-critical loop that must not meet the device-wide
 * synchronisation of cudaMalloc / cudaFree. zmc_run is closed to them -- it allocates its workspace, or needs one somebody allocated.
 *
 * zmc_flat_static computes what zmc_create(.., depth = 1, ..) + zmc_set_integrand + zmc_run + zmc_result compute for ONE instance of a
 * built-in integrand (every cell of the g^D grid sampled `trials` times with `samples_per_cell` points; per-cell mean
 * and spread; value = sum of the cell means, std = sqrt of the sum of the cell variances, R5, R7), with the same device
 * functions and therefore the same bits. All of its scratch memory is a fixed array inside the library image:
 *   - every GPU that loads the library's kernels holds ZMC_STATIC_SCRATCH_BYTES (2 MiB) for it until the process exits;
 *   - the problem must fit: divisions_per_axis^dim <= ZMC_STATIC_MAX_CELLS, cells * trials <= ZMC_STATIC_MAX_UNITS, dim <= 12
 *     (pre-compiled kernels only), n_params <= ZMC_STATIC_MAX_PARAMS; anything larger is refused with ZMC_ERR_CAPACITY (ZMC_ERR_RANGE
 *     for dim) and a message that names the limit -- nothing is launched;
 *   - ALL calls on one GPU share the array. Calls that follow one another on one stream are fine (each call resets what it needs and
 *     never reads what an earlier call left). Calls that can overlap on the GPU -- different streams, or different host threads --
 *     race on it and give garbage: serialise them.
 * The call itself runs no cudaMalloc, cudaFree or other allocating routine, enqueues three kernels on cuda_stream and returns without
 * synchronising. The FIRST call on each device also looks up the array's address on that device (cudaGetSymbolAddress, with the
 * caller's current device) and the SM count, and makes the runtime load the kernels there; make that first call at start-up, before
 * any stream capture, not in the middle of one.
 *   dim, lower, upper, divisions_per_axis, samples_per_cell, trials, seed     as zmc_create ([host] arrays, read during the call)
 *   builtin_id, params [host], n_params      as zmc_set_integrand with one instance (ZMC_USER is refused: NVRTC allocates)
 *   precision, math    ZMC_F64 / ZMC_F32, ZMC_MATH_EXACT / ZMC_MATH_FAST (as the options of the same names)
 *   result             [device] 2 doubles, caller-owned: value, std -- valid once the work enqueued on cuda_stream has finished
 *   cuda_stream        a cudaStream_t (NULL = the default stream)
 *   err, err_len       [host] optional buffer for the reason of a failure (NUL-terminated, "" on success); may be NULL / 0 */
#define ZMC_STATIC_SCRATCH_BYTES (2u << 20)
#define ZMC_STATIC_MAX_CELLS 4096
#define ZMC_STATIC_MAX_UNITS 131072
#define ZMC_STATIC_MAX_PARAMS 32
int zmc_flat_static(int dim, const double* lower, const double* upper, int divisions_per_axis, uint64_t samples_per_cell, int trials,
                    uint64_t seed, int builtin_id, const double* params, int n_params, int precision, int math, double* result,
                    void* cuda_stream, char* err, size_t err_len);

/* The reason of the last failure on ctx ("" if none; valid until the next call on ctx). ctx == NULL: the reason of the calling
 * thread's last failed zmc_create (valid until that thread's next zmc_create). */
const char* zmc_last_error(const zmc_ctx* ctx);
const char* zmc_status_string(int status);
void zmc_destroy(zmc_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* ZMC_H */

/*
 * zmc_static.cu -- zmc_flat_static (include/zmc.h): one level of the stratified sampling of PAPER.md:69-71 -- every cell of the g^D grid
 * sampled T times, per-cell mean and spread, the integral as the sum over the cells -- for callers that cannot allocate device memory.
 *
 * Who that is. zmc_run needs a workspace: it either calls cudaMalloc itself or is handed memory by zmc_set_workspace, which somebody had
 * to allocate. Some hosts can do neither: a process in which another component (a serving engine's memory pool, a solver that sized its
 * arrays to fill the card) already owns all of the 180 GB, so that any further cudaMalloc returns out-of-memory; and code on a latency
 * path that must not run into the device-wide synchronisation cudaMalloc and cudaFree imply. For them every byte this entry point
 * needs beyond the caller's own input and output lives in ONE file-scope __device__ array, zmc_static_scratch below: it is part of the
 * library image, so every GPU on which the library's kernels are loaded holds its ZMC_STATIC_SCRATCH_BYTES (2 MiB) until the process
 * exits, whether zmc_flat_static is ever called or not. That is why the maximum problem size is small and fixed.
 *
 * What runs. Three launches on the caller's stream, the same device functions as the other paths (so the same bits):
 *     zmc_static_begin_kernel    derived key (R3), parameters, root parent, zeroed sums, the level's work-item plan  -> scratch
 *     zmc_sample_kernel<F,false> the pre-compiled sampling kernel of zmc_inst.cu: per-(cell, trial, chunk) sums      -> scratch
 *     zmc_static_reduce_kernel   one block: cell statistics (R5), the group's accepted sums (R7), value and std      -> caller's result
 * The begin kernel rewrites everything that has to start from a known state (item counter, value and variance sums, flags); the rest of
 * the array is written before it is read within a call, so the previous call's contents never matter.
 *
 * In host code the name zmc_static_scratch is only a handle for the runtime, not an address the GPU understands: the device address comes
 * from cudaGetSymbolAddress, asked once per device with that device current, and it is that pointer which the kernels receive.
 *
 * No cudaMalloc, cudaFree, stream, event, graph, NVRTC or module load by this file; the first use of a kernel on a device makes the CUDA
 * runtime load the library's code there (which is also when the scratch array comes into being).
 */
#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>

#include "../../include/zmc.h"
#define ZMC_CONTROL_BODIES_ONLY
#include "zmc_control.cuh"
#include "zmc_inst.h"

#define ZMC_STATIC_TARGET_ITEMS 65536u      /* the work-item plan's default (zmc_plan_level; ZMC_OPT_TARGET_ITEMS of the other path) */
#define ZMC_STATIC_MIN_CHUNK_GROUPS 64u

static_assert(ZMC_STATIC_MAX_CELLS <= ZMC_TILE_CELLS, "the reduce kernel takes the sibling group as one control tile");

/* the scratch of every zmc_flat_static call on this GPU */
static __device__ __align__(256) unsigned char zmc_static_scratch[ZMC_STATIC_SCRATCH_BYTES];

namespace {

/* where each array sits inside the scratch: fixed, sized for the maximum problem */
struct StaticLayout {
    ZmcLevelInfo* info;       /* [3]: levels 0..2, level 1 used */
    zu32* keys;               /* [2] */
    double* params;           /* [ZMC_STATIC_MAX_PARAMS] */
    float* params_f32;
    ZmcParents par[2];        /* the root, and the (empty) list a second level would read */
    double* partial;          /* [ZMC_STATIC_MAX_UNITS + ZMC_STATIC_TARGET_ITEMS] */
    double *mu, *s;           /* [ZMC_STATIC_MAX_CELLS] */
    double* tau;
    zu64 *cnt, *excl;
    double* gacc;
    zu64 *gfirst, *gend, *out0;
    double *value, *var;
    zu64* nonfinite;
    zu32* overflow;
    size_t bytes;
};

struct Carver {
    char* base;
    size_t off = 0;
    explicit Carver(void* b) : base((char*)b) {}
    template <class T>
    T* take(size_t n) {
        off = (off + 255) & ~(size_t)255;
        T* p = (T*)(base + off);
        off += n * sizeof(T);
        return p;
    }
};

StaticLayout carve_static(void* base) {
    Carver A(base);
    StaticLayout Y;
    Y.info = A.take<ZmcLevelInfo>(3);
    Y.keys = A.take<zu32>(2);
    Y.params = A.take<double>(ZMC_STATIC_MAX_PARAMS);
    Y.params_f32 = A.take<float>(ZMC_STATIC_MAX_PARAMS);
    for (int i = 0; i < 2; ++i) {
        Y.par[i].inst = A.take<zu32>(1);
        Y.par[i].plo = A.take<zu64>(1);
        Y.par[i].phi = A.take<zu32>(1);
        Y.par[i].coord = A.take<zu32>(ZMC_MAX_DIM);
    }
    Y.partial = A.take<double>((size_t)ZMC_STATIC_MAX_UNITS + ZMC_STATIC_TARGET_ITEMS);
    Y.mu = A.take<double>(ZMC_STATIC_MAX_CELLS);
    Y.s = A.take<double>(ZMC_STATIC_MAX_CELLS);
    Y.tau = A.take<double>(1);
    Y.cnt = A.take<zu64>(1);
    Y.excl = A.take<zu64>(1);
    Y.gacc = A.take<double>(2);
    Y.gfirst = A.take<zu64>(1);
    Y.gend = A.take<zu64>(1);
    Y.out0 = A.take<zu64>(1);
    Y.value = A.take<double>(1);
    Y.var = A.take<double>(1);
    Y.nonfinite = A.take<zu64>(1);
    Y.overflow = A.take<zu32>(1);
    Y.bytes = (A.off + 255) & ~(size_t)255;
    return Y;
}

struct ZmcStaticBegin {
    double p[ZMC_STATIC_MAX_PARAMS];
    zu32 n_params, seed_lo, seed_hi;
    zu32* keys;
    double* params;
    float* params_f32;
};

}  // namespace

/* R3: Kd(seed, 0) = words 0,1 of Philox(ctr = (0, 0, 0, 0x5A4D4321), key = (seed_lo, seed_hi)) ; the parameters in FP64 and rounded to
 * FP32 ; then what zmc_init_kernel does: root parent, zeroed value/variance/flags, level 1's plan with its item counter at 0 */
__global__ void __launch_bounds__(ZMC_CTL_THREADS) zmc_static_begin_kernel(const __grid_constant__ ZmcCtlArgs c, const __grid_constant__ ZmcStaticBegin b) {
    if (threadIdx.x == 0) {
        ZmcKeySchedule ks;
        ks.init(b.seed_lo, b.seed_hi);
        zu32 w[4];
        zmc_philox(0u, 0u, 0u, 0x5A4D4321u, ks, w);
        b.keys[0] = w[0];
        b.keys[1] = w[1];
    }
    for (zu32 i = threadIdx.x; i < b.n_params; i += blockDim.x) {
        b.params[i] = b.p[i];
        b.params_f32[i] = (float)b.p[i];
    }
    zmc_init_kernel_body(c, 0u, 1u);
}

/* The control steps of a one-level search by one block, in the order and with the device functions of the single-launch tree kernel's
 * tail (zmc_tree.cuh): statistics + threshold + accepted sums of the one sibling group | bookkeeping scan | value += , var += | result.
 * result [2]: the integral estimate and its standard deviation (R5, R7). */
__global__ void __launch_bounds__(ZMC_CTL_THREADS) zmc_static_reduce_kernel(const __grid_constant__ ZmcCtlArgs c, double* result) {
    zmc_group_control_body(c, 0u, 1u);
    __syncthreads();
    zmc_scan_kernel_body(c);
    __syncthreads();
    zmc_accumulate_kernel_body(c, 0u, 1u);
    __syncthreads();
    zmc_finalize_body(c.value, c.var, result, 1u, 0u, 1u);
}

namespace {

int fail(char* err, size_t err_len, int code, const char* fmt, ...) {
    if (err && err_len) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(err, err_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

/* one entry per device ordinal: the scratch array's address ON THAT DEVICE and its SM count, looked up at the first call there */
constexpr int kMaxDevices = 64;
struct PerDevice {
    void* scratch = nullptr;
    int sms = 0;
};
PerDevice g_dev[kMaxDevices];
std::mutex g_dev_mu;

int device_setup(PerDevice& out, char* err, size_t err_len) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        return fail(err, err_len, ZMC_ERR_CUDA, "no CUDA device: %s", cudaGetErrorString(e));
    }
    if (dev < 0 || dev >= kMaxDevices) return fail(err, err_len, ZMC_ERR_RANGE, "device ordinal %d outside 0..%d", dev, kMaxDevices - 1);
    std::lock_guard<std::mutex> lock(g_dev_mu);
    if (!g_dev[dev].scratch) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, zmc_static_scratch);      /* the current device's copy of the array */
        if (e != cudaSuccess || !p) {
            (void)cudaGetLastError();
            return fail(err, err_len, ZMC_ERR_CUDA, "cudaGetSymbolAddress(zmc_static_scratch) on device %d: %s", dev, cudaGetErrorString(e));
        }
        int sms = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess || sms < 1) {
            (void)cudaGetLastError();
            return fail(err, err_len, ZMC_ERR_CUDA, "cudaDeviceGetAttribute(multiProcessorCount) on device %d: %s", dev, cudaGetErrorString(e));
        }
        g_dev[dev].sms = sms;
        g_dev[dev].scratch = p;
    }
    out = g_dev[dev];
    return ZMC_OK;
}

/* the pre-compiled per-item-key sampling kernel (zmc_inst.cu) of a built-in integrand; nullptr if there is none */
const void* sample_kernel(int prec, int mode, int id, int D) {
    if (D < 1 || D > ZMC_AOT_MAX_DIM) return nullptr;
    if (prec == ZMC_F64) {
        switch (id) {
            case ZMC_CONST: return zmc_lookup_0_0_0(D).sample;
            case ZMC_LINEAR: return zmc_lookup_0_0_1(D).sample;
            case ZMC_SIN_SUM: return zmc_lookup_0_0_2(D).sample;
            case ZMC_EXP_QUAD: return zmc_lookup_0_0_3(D).sample;
        }
        return nullptr;
    }
    if (mode == ZMC_MATH_FAST) {
        if (id == ZMC_SIN_SUM) return zmc_lookup_1_1_2(D).sample;
        if (id == ZMC_EXP_QUAD) return zmc_lookup_1_1_3(D).sample;
    }
    switch (id) {       /* CONST and LINEAR have no elementary function: fast = exact */
        case ZMC_CONST: return zmc_lookup_1_0_0(D).sample;
        case ZMC_LINEAR: return zmc_lookup_1_0_1(D).sample;
        case ZMC_SIN_SUM: return zmc_lookup_1_0_2(D).sample;
        case ZMC_EXP_QUAD: return zmc_lookup_1_0_3(D).sample;
    }
    return nullptr;
}

}  // namespace

extern "C" int zmc_flat_static(int dim, const double* lower, const double* upper, int g, uint64_t N, int T, uint64_t seed, int builtin_id,
                               const double* params, int n_params, int precision, int math, double* result, void* cuda_stream,
                               char* err, size_t err_len) {
    if (err && err_len) err[0] = '\0';
    /* 1. arguments: the rules of zmc_create and zmc_set_integrand, then this entry point's own limits */
    if (!lower || !upper || !result) return fail(err, err_len, ZMC_ERR_ARG, "lower, upper or result is null");
    if (dim < 1) return fail(err, err_len, ZMC_ERR_ARG, "dim < 1");
    if (dim > ZMC_AOT_MAX_DIM) return fail(err, err_len, ZMC_ERR_RANGE, "dim %d: zmc_flat_static runs the pre-compiled kernels only, dim <= %d (no NVRTC: loading a compiled program allocates)", dim, ZMC_AOT_MAX_DIM);
    if (g < 1 || N < 1 || T < 1) return fail(err, err_len, ZMC_ERR_ARG, "divisions_per_axis, samples_per_cell and trials must be >= 1");
    if (T > ZMC_MAX_TRIALS) return fail(err, err_len, ZMC_ERR_RANGE, "trials > 255");
    for (int d = 0; d < dim; ++d)
        if (!std::isfinite(lower[d]) || !std::isfinite(upper[d]) || !(upper[d] > lower[d])) return fail(err, err_len, ZMC_ERR_ARG, "bounds must be finite with upper > lower");
    if ((long double)N * (long double)dim >= 17179869184.0L - 16384.0L) return fail(err, err_len, ZMC_ERR_RANGE, "samples_per_cell * dim >= 2^34 - 2^14 (DESIGN.md R3)");
    if (precision != ZMC_F64 && precision != ZMC_F32) return fail(err, err_len, ZMC_ERR_ARG, "precision must be ZMC_F64 or ZMC_F32");
    if (math != ZMC_MATH_EXACT && math != ZMC_MATH_FAST) return fail(err, err_len, ZMC_ERR_ARG, "math must be ZMC_MATH_EXACT or ZMC_MATH_FAST");
    if (precision == ZMC_F64) math = ZMC_MATH_EXACT;      /* as zmc_run: the fast functions are FP32 */
    int need;
    switch (builtin_id) {
        case ZMC_CONST: need = 1; break;
        case ZMC_LINEAR: need = 1 + dim; break;
        case ZMC_SIN_SUM: need = 0; break;
        case ZMC_EXP_QUAD: need = 2 + dim; break;
        default: return fail(err, err_len, ZMC_ERR_ARG, "unknown built-in integrand id %d (user integrands need NVRTC, which allocates)", builtin_id);
    }
    if (n_params < need) return fail(err, err_len, ZMC_ERR_ARG, "too few parameters for this integrand: %d given, %d needed", n_params, need);
    if (n_params > ZMC_STATIC_MAX_PARAMS) return fail(err, err_len, ZMC_ERR_CAPACITY, "n_params %d exceeds ZMC_STATIC_MAX_PARAMS (%d)", n_params, ZMC_STATIC_MAX_PARAMS);
    if (n_params > 0 && !params) return fail(err, err_len, ZMC_ERR_ARG, "params is null");
    uint64_t k = 1;
    for (int d = 0; d < dim; ++d) {
        k *= (uint64_t)g;
        if (k > ZMC_STATIC_MAX_CELLS)
            return fail(err, err_len, ZMC_ERR_CAPACITY, "divisions_per_axis^dim = %d^%d cells exceed ZMC_STATIC_MAX_CELLS (%d): the static scratch array is %u bytes and cannot grow; use zmc_run",
                        g, dim, ZMC_STATIC_MAX_CELLS, (unsigned)ZMC_STATIC_SCRATCH_BYTES);
    }
    if (k * (uint64_t)T > ZMC_STATIC_MAX_UNITS)
        return fail(err, err_len, ZMC_ERR_CAPACITY, "cells * trials = %llu * %d exceed ZMC_STATIC_MAX_UNITS (%d): the static scratch array is %u bytes and cannot grow; use zmc_run",
                    (unsigned long long)k, T, ZMC_STATIC_MAX_UNITS, (unsigned)ZMC_STATIC_SCRATCH_BYTES);

    /* 2. this device's scratch (first call on a device: cudaGetSymbolAddress) and kernel */
    (void)cudaGetLastError();      /* errors left behind by earlier, unrelated calls are not this call's */
    PerDevice pd;
    int rc = device_setup(pd, err, err_len);
    if (rc != ZMC_OK) return rc;
    const StaticLayout Y = carve_static(pd.scratch);
    if (Y.bytes > (size_t)ZMC_STATIC_SCRATCH_BYTES) return fail(err, err_len, ZMC_ERR_CAPACITY, "internal: layout of %zu bytes exceeds the scratch array", Y.bytes);
    const void* k_sample = sample_kernel(precision, math, builtin_id, dim);
    if (!k_sample) return fail(err, err_len, ZMC_ERR_ARG, "no pre-compiled sampling kernel for this integrand, precision and dimension");
    int per_sm = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_sample, ZMC_BLOCK_THREADS, 0);
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        return fail(err, err_len, ZMC_ERR_CUDA, "cudaOccupancyMaxActiveBlocksPerMultiprocessor: %s", cudaGetErrorString(e));
    }
    if (per_sm < 1) per_sm = 1;

    /* 3. launch parameters of level 1 of a depth-1 search with one instance (what zmc_run's fill_sample_args / fill_ctl_args give) */
    ZmcSampleArgs sa;
    memset(&sa, 0, sizeof sa);
    sa.par_inst = Y.par[0].inst; sa.par_plo = Y.par[0].plo; sa.par_phi = Y.par[0].phi; sa.par_coord = Y.par[0].coord;
    sa.par_stride = 1;
    sa.info = Y.info + 1;
    sa.partial = Y.partial;
    sa.keys = Y.keys;
    sa.params = Y.params;
    sa.params_f32 = Y.params_f32;
    sa.ppi = n_params;
    sa.g = (zu32)g; sa.T = (zu32)T; sa.level = 1u;
    sa.k = k;
    sa.N = N;
    const double cells = 1.0 * (double)g;      /* R2: width_d = (upper_d - lower_d) / (double)g^level */
    for (int d = 0; d < dim; ++d) { sa.lower[d] = lower[d]; sa.width[d] = (upper[d] - lower[d]) / cells; }

    ZmcCtlArgs ca;
    memset(&ca, 0, sizeof ca);
    ca.info = Y.info;
    ca.level = 1u; ca.L = 1u; ca.T = (zu32)T; ca.g = (zu32)g; ca.D = (zu32)dim;
    ca.n_inst = 1u;
    ca.nc = 1u;
    ca.k = k; ca.N = N;
    const int SG = (dim % 4 == 0) ? 1 : ((dim % 2 == 0) ? 2 : 4);      /* samples per group that starts on a Philox call boundary */
    ca.sample_groups = (zu32)((N + SG - 1) / SG);
    ca.target_items = ZMC_STATIC_TARGET_ITEMS;
    ca.min_chunk_groups = ZMC_STATIC_MIN_CHUNK_GROUPS;
    ca.trial_loop = zmc_tune_trial_loop(dim) ? 1u : 0u;
    double V = 1.0;      /* R2: V = w_0 * w_1 * ... in axis order */
    for (int d = 0; d < dim; ++d) V = (d == 0) ? sa.width[0] : V * sa.width[d];
    ca.V = V;
    ca.m = 0.0;          /* the threshold decides nothing on the last level (R7) */
    ca.budget = ~0ull;
    ca.cap_par = 1;
    ca.tpg = 1u;
    ca.cur = Y.par[0];
    ca.next = Y.par[1];
    ca.par_stride = 1;
    ca.params = Y.params;
    ca.ppi = n_params;
    ca.prefactor_index = (builtin_id == ZMC_EXP_QUAD) ? 0 : -1;
    ca.partial = Y.partial;
    ca.mu = Y.mu;
    ca.s = Y.s;
    ca.tau = Y.tau;
    ca.cnt = Y.cnt; ca.excl = Y.excl; ca.gacc = Y.gacc;
    ca.gfirst = Y.gfirst; ca.gend = Y.gend; ca.out0 = Y.out0;
    ca.value = Y.value; ca.var = Y.var;
    ca.nonfinite = Y.nonfinite; ca.overflow = Y.overflow;

    ZmcStaticBegin bg;
    memset(&bg, 0, sizeof bg);
    for (int i = 0; i < n_params; ++i) bg.p[i] = params[i];
    bg.n_params = (zu32)n_params;
    bg.seed_lo = (zu32)seed; bg.seed_hi = (zu32)(seed >> 32);
    bg.keys = Y.keys; bg.params = Y.params; bg.params_f32 = Y.params_f32;

    /* 4. three launches, no synchronisation */
    cudaStream_t st = (cudaStream_t)cuda_stream;
    zmc_static_begin_kernel<<<1, ZMC_CTL_THREADS, 0, st>>>(ca, bg);
    void* args[] = {&sa};
    e = cudaLaunchKernel(k_sample, dim3(pd.sms * per_sm), dim3(ZMC_BLOCK_THREADS), args, 0, st);
    if (e == cudaSuccess) {
        zmc_static_reduce_kernel<<<1, ZMC_CTL_THREADS, 0, st>>>(ca, result);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        return fail(err, err_len, ZMC_ERR_CUDA, "kernel launch: %s", cudaGetErrorString(e));
    }
    return ZMC_OK;
}

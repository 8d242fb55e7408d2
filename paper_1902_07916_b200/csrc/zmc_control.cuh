/*
 * zmc_control.cuh -- the tree-search control kernels that run between two levels' sampling
 * kernels, entirely on the device (R5-R7, R12):
 *
 *   zmc_keys_kernel        derived Philox keys, one call per instance                           (R3)
 *   zmc_init_kernel        root parents, zeroed results, level-1 plan
 *   zmc_cell_stats_kernel  per-(cell,trial) partial sums -> S_t -> I_t -> (mu_c, s_c)          (R5; R13 from sum f^2)
 *   zmc_threshold_kernel   per sibling group: tau = mean(s) + m*pstd(s), number of s > tau      (R6)
 *   zmc_threshold_pass_kernel<0,1,2>   the same for groups of several 4096-cell tiles, one launch per pass
 *   zmc_scan_kernel        exclusive scans over groups and instances -> output slots, next plan (R7, R12)
 *   zmc_select_kernel (or, for few large instances, zmc_select_begin/hist/pick_kernel), zmc_count2_kernel, zmc_scan2_kernel
 *                          only with ZMC_BUDGET_LARGEST_SPREAD: radix select of the B largest flagged
 *                          spreads per instance, counts above / at the pivot, their scans            (R14)
 *   zmc_scatter_kernel     stable compaction of flagged cells into the next parent list;
 *                          accepted cells -> per-group (sum mu, sum s^2)                         (R7)
 *   zmc_accumulate_kernel  per instance: value += sum mu, var += sum s^2                         (R7)
 *   zmc_finalize_kernel    (value, sqrt(var)) per instance
 *
 * Every kernel is a device function (zmc_*_body) plus a one-line __global__ wrapper: the single-launch tree kernel (zmc_tree.cuh)
 * calls the same bodies between grid barriers, and zmc_group_control_body fuses statistics, threshold and count for one group.
 *
 * Every reduction has a fixed shape (strided partials, then a tree), so repeated runs are
 * bit-identical. Nothing here is read by the host until zmc_result.
 */
#ifndef ZMC_CONTROL_CUH
#define ZMC_CONTROL_CUH
/* ZMC_CONTROL_BODIES_ONLY: the device functions (zmc_*_body) without the __global__ kernels around them -- for the translation
 * units that only build the single-launch tree kernel (zmc_inst.cu); the kernels themselves are defined once, in zmc_lib.cu. */
#include "zmc_device.cuh"

#define ZMC_CTL_THREADS 256
#define ZMC_SCAN_THREADS 1024
/* A sibling group of k cells is handled as ceil(k / ZMC_TILE_CELLS) tiles of consecutive cells, one CTA per tile, so that a level
 * that is ONE group of 10^5 .. 10^6 cells (BASELINE.json configs[4]; the paper's Table 3 and 4 sizes) is not walked by one CTA.
 * Groups up to ZMC_TILE_CELLS cells are one tile and take the single-launch threshold kernel. The tiling depends on k only, so
 * the reductions keep a fixed shape: repeated runs and different grid sizes give identical bits. */
#define ZMC_TILE_CELLS 4096

struct ZmcParents {
    zu32* inst;
    zu64* plo;
    zu32* phi;
    zu32* coord;   /* [d * stride + G] */
};

struct ZmcCtlArgs {
    ZmcLevelInfo* info;     /* array indexed by level, 1..L+1 */
    zu32 level, L, T, g, D;
    zu32 n_inst;
    zu32 nc;                /* components per cell (R15); 1 except for vector-valued user integrands. Per-cell arrays are
                               [cell * nc + j], per-group ones [group * nc + j], per-tile ones [tile * nc + j], value/var [instance * nc + j] */
    zu64 k, N;
    zu32 sample_groups;     /* sample groups per unit = ceil(N / SG) */
    zu32 target_items, min_chunk_groups;
    zu32 trial_loop;        /* 1: the sampling kernel in use honours ZmcLevelInfo::trials_per_item (ZmcTune::TRIAL_LOOP) */
    double V;               /* cell volume at this level (R2) */
    double m;               /* sigma multiplier */
    zu64 budget;            /* R12; ~0 = off */
    zu64 cap_par;           /* capacity of a parent list */
    zu32 tpg;               /* tiles per sibling group = ceil(k / ZMC_TILE_CELLS): the unit of the flag/compaction kernels */
    double* tsum;           /* [tile] sum of s            (tpg > 1 only: the three passes of R6 are three launches) */
    double* tsq;            /* [tile] sum of (s - mean)^2 (tpg > 1 only) */
    ZmcParents cur, next;
    zu64 par_stride;
    const double* params;
    zi32 ppi;
    zi32 prefactor_index;   /* EXP_QUAD: 0 (A = p[0] multiplies each trial estimate); else -1 */
    const double* partial;
    double* S;              /* [cell*T + t], or nullptr */
    double* mu;             /* [cell] */
    double* s;              /* [cell] */
    unsigned char* refined; /* [cell], or nullptr */
    double* tau;            /* [group] */
    zu64* cnt;              /* [tile] flagged cells */
    zu64* excl;             /* [tile] exclusive prefix of cnt over all tiles */
    double* gacc;           /* [tile][2] accepted (sum mu, sum s^2) */
    zu64* gfirst;           /* [instance] first tile */
    zu64* gend;             /* [instance] one past the last tile */
    zu64* out0;             /* [instance] first output slot */
    double* value;          /* [instance] */
    double* var;            /* [instance] */
    zu64* nonfinite;
    zu32* overflow;
    /* R13: spread from the samples */
    zu32 spread;            /* 0: from the T trial values (paper) ; 1: from sum f, sum f^2 of the T*N samples */
    const double* partial_q;
    double* Q;              /* [cell*T + t], or nullptr */
    /* R14: the budget keeps the largest spreads */
    zu32 budget_order;      /* 0: first B flagged cells in path order (R12) ; 1: the B largest spreads */
    zu64* piv;              /* [instance] key (bits of s) of the B-th largest flagged spread; 0 with quota ~0 = keep every flagged cell */
    zu64* quota;            /* [instance] how many cells with s == pivot are kept (the first in path order) */
    zu64* cnt_gt;           /* [tile] flagged cells with key > pivot */
    zu64* cnt_eq;           /* [tile] flagged cells with key == pivot */
    zu64* excl_gt;          /* [tile] exclusive prefixes over all tiles */
    zu64* excl_eq;
    zu64* sel_state;        /* [instance][4] prefix, need, above, active: the radix select spread over the grid (few, large instances) */
    zu64* sel_hist;         /* [instance][256] */
    zu32 stop_on_overflow;  /* 1: a level that does not fit ends the search (the next level is empty) instead of going on with the parents that fit --
                               the host grows the workspace and runs again, so what would follow is wasted time */
};

/* plan of one level: how the (cell, trial) units are cut into work items. (Tried and not kept: choosing the number of chunks
 * by a cost model "rounds x (item overhead + item length)" -- on BASELINE.json configs[0] level 2 as 1600 long items sampled in
 * 28.7 us against 31.0 us as 11200 short ones, and the model's divisions cost the one planning thread 11 us.) */
__device__ __forceinline__ void zmc_plan_level(ZmcLevelInfo& li, zu64 n_groups, const ZmcCtlArgs& c) {
    li.n_groups = n_groups;
    li.n_cells = n_groups * c.k;
    const zu64 units = li.n_cells * c.T;
    zu64 nch = 1;
    if (units > 0 && units < c.target_items) {
        nch = (c.target_items + units - 1) / units;
        zu64 max_ch = c.sample_groups / c.min_chunk_groups;
        if (max_ch < 1) max_ch = 1;
        if (nch > max_ch) nch = max_ch;
    }
    const zu32 cg = (zu32)(((zu64)c.sample_groups + nch - 1) / nch);
    li.chunk_groups = cg;
    li.n_chunks = (zu32)(((zu64)c.sample_groups + cg - 1) / cg);    /* 64-bit: sample_groups may be within cg of 2^32 */
    /* a level with at least target_items CELLS has work items to spare: one item = all T trials of a cell, so that item decoding and
     * cell geometry are paid once per cell (visible at small N: BASELINE.json configs[3] has 4096 samples per unit) */
    li.trials_per_item = (c.trial_loop && li.n_chunks == 1u && li.n_cells >= c.target_items) ? c.T : 1u;
    li.reserved = 0u;
    li.n_items = (units / li.trials_per_item) * li.n_chunks;
    li.work_ctr = 0;
    li.n_flagged = 0;
    li.n_refined = 0;
    li.t_mark[0] = li.t_mark[1] = li.t_mark[2] = li.t_mark[3] = 0ull;
}

/* R3: Kd(seed, b) = words 0,1 of Philox(ctr = (b, 0, 0, 0x5A4D4321), key = (seed_lo, seed_hi)) */
#ifndef ZMC_CONTROL_BODIES_ONLY
__global__ void zmc_keys_kernel(zu32* keys, zu32 n_inst, zu32 seed_lo, zu32 seed_hi) {
    for (zu64 b = (zu64)blockIdx.x * blockDim.x + threadIdx.x; b < n_inst; b += (zu64)gridDim.x * blockDim.x) {
        ZmcKeySchedule ks;
        ks.init(seed_lo, seed_hi);
        zu32 w[4];
        zmc_philox((zu32)b, 0u, 0u, 0x5A4D4321u, ks, w);
        keys[2 * b] = w[0];
        keys[2 * b + 1] = w[1];
    }
}
#endif

/* root parents (path 0, coordinates 0), zeroed results, the level-1 plan */
__device__ __forceinline__ void zmc_init_kernel_body(const ZmcCtlArgs& c, const zu32 bid, const zu32 nb) {
    const zu64 tid = (zu64)bid * blockDim.x + threadIdx.x;
    for (zu64 b = tid; b < c.n_inst; b += (zu64)nb * blockDim.x) {
        c.cur.inst[b] = (zu32)b;
        c.cur.plo[b] = 0ull;
        c.cur.phi[b] = 0u;
        for (zu32 d = 0; d < c.D; ++d) c.cur.coord[(zu64)d * c.par_stride + b] = 0u;
        for (zu32 j = 0; j < c.nc; ++j) { c.value[b * c.nc + j] = 0.0; c.var[b * c.nc + j] = 0.0; }
    }
    if (tid == 0) {
        for (zu32 l = 0; l <= c.L + 1; ++l) {
            ZmcLevelInfo z;
            z.n_groups = z.n_cells = z.n_items = z.work_ctr = z.n_flagged = z.n_refined = 0;
            z.n_chunks = 1; z.chunk_groups = c.sample_groups; z.trials_per_item = 1; z.reserved = 0;
            z.t_mark[0] = z.t_mark[1] = z.t_mark[2] = z.t_mark[3] = 0ull;
            if (l != 1) c.info[l] = z;
        }
        ZmcLevelInfo li;
        zmc_plan_level(li, c.n_inst, c);
        c.info[1] = li;
        *c.nonfinite = 0ull;
        *c.overflow = 0u;
    }
}
#ifndef ZMC_CONTROL_BODIES_ONLY
__global__ void zmc_init_kernel(const __grid_constant__ ZmcCtlArgs c) { zmc_init_kernel_body(c, blockIdx.x, gridDim.x); }
#endif

/* R5: S_t = sum of the chunk partials in chunk order ; I_t = ((V*A)*S_t)/(double)N ;
 * mu = (sum_t I_t)/T ; s = sqrt((sum_t (I_t-mu)^2)/T)  -- two-pass, population form. */
/* the (cell, component) entries first, first + step, .. < last: one thread per entry */
__device__ __forceinline__ void zmc_cell_stats_span(const ZmcCtlArgs& c, const zu64 first, const zu64 last, const zu64 step) {
    const ZmcLevelInfo& li = c.info[c.level];
    const zu32 nch = li.n_chunks;
    const double dN = (double)c.N, dT = (double)c.T;
    zu64 bad = 0;
    const zu64 nc = c.nc;
    /* one thread per (cell, component): component j of work item i is partial[i * nc + j] (R15); nc == 1: one thread per cell */
    for (zu64 e = first; e < last; e += step) {
        const zu64 cell = (nc == 1ull) ? e : e / nc;
        const zu64 jc = e - cell * nc;
        double A = 1.0;
        if (c.prefactor_index >= 0) {
            const zu32 inst = c.cur.inst[cell / c.k];
            A = c.params[(zu64)inst * (zu64)c.ppi + (zu64)c.prefactor_index];
        }
        const double VA = __dmul_rn(c.V, A);
        const double* p = c.partial + cell * (zu64)c.T * nch * nc + jc;
        /* the cell's T * n_chunks partial sums are read one after the other below (a dependent chain of FP64 adds): ask for their
         * cache lines first, all at once, so that the chain does not pay an L2 round trip per trial */
        if (nch > 1u || c.T > 4u) {
            const char* q0 = (const char*)p;
            const zu64 bytes = (zu64)c.T * nch * nc * sizeof(double);
            for (zu64 off = 0; off < bytes; off += 128ull) asm volatile("prefetch.global.L1 [%0];" ::"l"(q0 + off));
        }
        double acc = 0.0;
        for (zu32 t = 0; t < c.T; ++t) {
            double S = p[(zu64)t * nch * nc];
            for (zu32 ch = 1; ch < nch; ++ch) S = __dadd_rn(S, p[((zu64)t * nch + ch) * nc]);
            if (c.S) c.S[(cell * c.T + t) * nc + jc] = S;
            acc = __dadd_rn(acc, __ddiv_rn(__dmul_rn(VA, S), dN));
        }
        const double mu = __ddiv_rn(acc, dT);
        double sd;
        if (c.spread == 0) {
            double q = 0.0;
            for (zu32 t = 0; t < c.T; ++t) {
                double S = p[(zu64)t * nch * nc];
                for (zu32 ch = 1; ch < nch; ++ch) S = __dadd_rn(S, p[((zu64)t * nch + ch) * nc]);
                const double d = __dadd_rn(__ddiv_rn(__dmul_rn(VA, S), dN), -mu);
                q = __dadd_rn(q, __dmul_rn(d, d));
            }
            sd = __dsqrt_rn(__ddiv_rn(q, dT));
        } else {
            /* R13: Sc = sum_t S_t, Qc = sum_t Q_t over M = T*N samples ; d = Qc - Sc^2/M, 0 unless d > Qc*2^-40 ;
             * s = (V*A) * sqrt((d/M)/M), the standard error of mu. per component (R15) */
            const double* pq = c.partial_q + cell * (zu64)c.T * nch * nc + jc;
            double Sc = 0.0, Qc = 0.0;
            for (zu32 t = 0; t < c.T; ++t) {
                double S = p[(zu64)t * nch * nc], Q = pq[(zu64)t * nch * nc];
                for (zu32 ch = 1; ch < nch; ++ch) { S = __dadd_rn(S, p[((zu64)t * nch + ch) * nc]); Q = __dadd_rn(Q, pq[((zu64)t * nch + ch) * nc]); }
                if (c.Q) c.Q[(cell * c.T + t) * nc + jc] = Q;
                Sc = __dadd_rn(Sc, S);
                Qc = __dadd_rn(Qc, Q);
            }
            const double M = __dmul_rn(dT, dN);
            double d = __dadd_rn(Qc, -__ddiv_rn(__dmul_rn(Sc, Sc), M));
            if (!(d > __dmul_rn(Qc, 9.094947017729282e-13))) d = 0.0;
            sd = __dmul_rn(VA, __dsqrt_rn(__ddiv_rn(__ddiv_rn(d, M), M)));
        }
        c.mu[e] = mu;
        c.s[e] = sd;
        if (!(fabs(mu) <= 1.7976931348623157e308) || !(fabs(sd) <= 1.7976931348623157e308)) ++bad;
    }
    if (bad) atomicAdd(c.nonfinite, bad);
}

/* One block, batches of floor(256 / T) entries (an entry = a (cell, component)); entries [e_begin, e_end), batches b_first, b_first + b_step, ..
 * One thread per (entry, trial) sums that trial's chunk partials (in chunk order) and forms I_t -- T independent loads and divisions side by side
 * instead of one thread walking them as a chain; then the entry's first thread adds the T values in trial order. The arithmetic of every number is what
 * a single thread would do, operation by operation (R5, R13). sh: 3 * ZMC_CTL_THREADS doubles of shared memory. */
__device__ __forceinline__ void zmc_cell_stats_batches(const ZmcCtlArgs& c, const zu64 e_begin, const zu64 e_end, const zu64 b_first,
                                                       const zu64 b_step, double* sh) {
    const ZmcLevelInfo& li = c.info[c.level];
    const zu32 nch = li.n_chunks;
    const double dN = (double)c.N, dT = (double)c.T;
    const zu64 nc = c.nc;
    const zu32 T = c.T;
    const zu32 epb = (zu32)ZMC_CTL_THREADS / T;          /* T <= 255: at least one entry per batch */
    const zu32 le = threadIdx.x / T, t = threadIdx.x - le * T;
    double* shI = sh;
    double* shS = sh + ZMC_CTL_THREADS;
    double* shQ = sh + 2 * ZMC_CTL_THREADS;
    const zu64 n_batches = (e_end > e_begin) ? (e_end - e_begin + epb - 1) / epb : 0ull;
    zu64 bad = 0;
    for (zu64 b = b_first; b < n_batches; b += b_step) {
        const zu64 e = e_begin + b * epb + le;
        const bool live = le < epb && e < e_end;
        double VA = 0.0;
        if (live) {
            const zu64 cell = (nc == 1ull) ? e : e / nc;
            const zu64 jc = e - cell * nc;
            double A = 1.0;
            if (c.prefactor_index >= 0) {
                const zu32 inst = c.cur.inst[cell / c.k];
                A = c.params[(zu64)inst * (zu64)c.ppi + (zu64)c.prefactor_index];
            }
            VA = __dmul_rn(c.V, A);
            const zu64 unit = cell * (zu64)T + t;
            const double* p = c.partial + unit * nch * nc + jc;
            double S = p[0];
            for (zu32 ch = 1; ch < nch; ++ch) S = __dadd_rn(S, p[(zu64)ch * nc]);
            if (c.S) c.S[unit * nc + jc] = S;
            shI[threadIdx.x] = __ddiv_rn(__dmul_rn(VA, S), dN);
            if (c.spread != 0) {      /* R13, per component */
                const double* pq = c.partial_q + unit * nch * nc + jc;
                double Q = pq[0];
                for (zu32 ch = 1; ch < nch; ++ch) Q = __dadd_rn(Q, pq[(zu64)ch * nc]);
                if (c.Q) c.Q[unit * nc + jc] = Q;
                shS[threadIdx.x] = S;
                shQ[threadIdx.x] = Q;
            }
        }
        __syncthreads();
        if (live && t == 0u) {
            const double* I = shI + le * T;
            double acc = 0.0;
            for (zu32 tt = 0; tt < T; ++tt) acc = __dadd_rn(acc, I[tt]);
            const double mu = __ddiv_rn(acc, dT);
            double sd;
            if (c.spread == 0) {
                double q = 0.0;
                for (zu32 tt = 0; tt < T; ++tt) {
                    const double d = __dadd_rn(I[tt], -mu);
                    q = __dadd_rn(q, __dmul_rn(d, d));
                }
                sd = __dsqrt_rn(__ddiv_rn(q, dT));
            } else {
                /* R13: Sc = sum_t S_t, Qc = sum_t Q_t over M = T*N samples ; d = Qc - Sc^2/M, 0 unless d > Qc*2^-40 ;
                 * s = (V*A) * sqrt((d/M)/M), the standard error of mu (of each component's mu, R15) */
                double Sc = 0.0, Qc = 0.0;
                for (zu32 tt = 0; tt < T; ++tt) { Sc = __dadd_rn(Sc, shS[le * T + tt]); Qc = __dadd_rn(Qc, shQ[le * T + tt]); }
                const double M = __dmul_rn(dT, dN);
                double d = __dadd_rn(Qc, -__ddiv_rn(__dmul_rn(Sc, Sc), M));
                if (!(d > __dmul_rn(Qc, 9.094947017729282e-13))) d = 0.0;
                sd = __dmul_rn(VA, __dsqrt_rn(__ddiv_rn(__ddiv_rn(d, M), M)));
            }
            c.mu[e] = mu;
            c.s[e] = sd;
            if (!(fabs(mu) <= 1.7976931348623157e308) || !(fabs(sd) <= 1.7976931348623157e308)) ++bad;
        }
        __syncthreads();
    }
    if (bad) atomicAdd(c.nonfinite, bad);
}
/* Small levels (where the statistics are latency, not throughput) go one thread per (entry, trial); large ones one thread per entry, every
 * thread busy -- the 4.5e8-cell level of BASELINE.json configs[1] whole: 18 ms against 34 ms. The numbers are the same bit for bit. */
__device__ __forceinline__ void zmc_cell_stats_kernel_body(const ZmcCtlArgs& c, const zu32 bid, const zu32 nb) {
    __shared__ double sh[3 * ZMC_CTL_THREADS];
    const zu64 n_entries = c.info[c.level].n_cells * (zu64)c.nc;
    if (n_entries <= (1ull << 18)) zmc_cell_stats_batches(c, 0ull, n_entries, bid, nb, sh);
    else zmc_cell_stats_span(c, (zu64)bid * blockDim.x + threadIdx.x, n_entries, (zu64)nb * blockDim.x);
}
#ifndef ZMC_CONTROL_BODIES_ONLY
__global__ void __launch_bounds__(ZMC_CTL_THREADS) zmc_cell_stats_kernel(const __grid_constant__ ZmcCtlArgs c) { zmc_cell_stats_kernel_body(c, blockIdx.x, gridDim.x); }
#endif

/* fixed-shape block reduction (sum); every thread gets the result */
__device__ __forceinline__ double zmc_block_sum(double v, double* smem) {
    const int tid = threadIdx.x;
    __syncthreads();
    smem[tid] = v;
    __syncthreads();
    for (int off = ZMC_CTL_THREADS / 2; off > 0; off >>= 1) {
        if (tid < off) smem[tid] = __dadd_rn(smem[tid], smem[tid + off]);
        __syncthreads();
    }
    return smem[0];
}

__device__ __forceinline__ zu64 zmc_block_sum_u64(zu64 v, zu64* smem) {
    const int tid = threadIdx.x;
    __syncthreads();
    smem[tid] = v;
    __syncthreads();
    for (int off = ZMC_CTL_THREADS / 2; off > 0; off >>= 1) {
        if (tid < off) smem[tid] += smem[tid + off];
        __syncthreads();
    }
    return smem[0];
}

/* tile -> its sibling group and cell range */
struct ZmcTile {
    zu64 G, c0, c1;
    __device__ __forceinline__ ZmcTile(const ZmcCtlArgs& c, zu64 tile) {
        G = tile / c.tpg;
        const zu64 t = tile - G * c.tpg;
        c0 = G * c.k + t * (zu64)ZMC_TILE_CELLS;
        const zu64 end = (G + 1ull) * c.k;
        c1 = (c0 + (zu64)ZMC_TILE_CELLS < end) ? c0 + (zu64)ZMC_TILE_CELLS : end;
    }
};

/* R6: one block per sibling group of at most ZMC_TILE_CELLS cells (tpg == 1); tau = mean(s) + m * pstd(s), both moments
 * two-pass, population form ("the mean and standard deviation of the calculated k standard deviations").
 * R7: flagged iff level < L and s > tau (strict; NaN compares false). */
/* one sibling group, by one block */
__device__ __forceinline__ void zmc_threshold_group(const ZmcCtlArgs& c, const zu64 G, double* smem, zu64* smem_u, double* tau_sh) {
    const double dk = (double)c.k;
    const zu64 nc = c.nc;
    {
        const double* s = c.s + G * c.k * nc;
        for (zu64 jc = 0; jc < nc; ++jc) {      /* R15: one threshold per component */
            double part = 0.0;
            for (zu64 j = threadIdx.x; j < c.k; j += ZMC_CTL_THREADS) part = __dadd_rn(part, s[j * nc + jc]);
            const double mean = __ddiv_rn(zmc_block_sum(part, smem), dk);
            part = 0.0;
            for (zu64 j = threadIdx.x; j < c.k; j += ZMC_CTL_THREADS) {
                const double d = __dadd_rn(s[j * nc + jc], -mean);
                part = __dadd_rn(part, __dmul_rn(d, d));
            }
            const double pstd = __dsqrt_rn(__ddiv_rn(zmc_block_sum(part, smem), dk));
            const double tau = __dadd_rn(mean, __dmul_rn(c.m, pstd));
            if (threadIdx.x == 0) { c.tau[G * nc + jc] = tau; tau_sh[jc] = tau; }
        }
        __syncthreads();
        zu64 n = 0;
        if (c.level < c.L)
            for (zu64 j = threadIdx.x; j < c.k; j += ZMC_CTL_THREADS) {
                bool any = false;       /* R15: flagged iff some component's spread passes its threshold */
                for (zu64 jc = 0; jc < nc; ++jc) any = any || (s[j * nc + jc] > tau_sh[jc]);
                n += any ? 1ull : 0ull;
            }
        n = zmc_block_sum_u64(n, smem_u);
        if (threadIdx.x == 0) c.cnt[G] = n;
        __syncthreads();        /* tau_sh is rewritten by the next group */
    }
}
__device__ __forceinline__ void zmc_threshold_kernel_body(const ZmcCtlArgs& c, const zu32 bid, const zu32 nb) {
    __shared__ double smem[ZMC_CTL_THREADS];
    __shared__ zu64 smem_u[ZMC_CTL_THREADS];
    __shared__ double tau_sh[ZMC_DEV_MAX_COMPONENTS];
    const zu64 n_groups = c.info[c.level].n_groups;
    for (zu64 G = bid; G < n_groups; G += nb) zmc_threshold_group(c, G, smem, smem_u, tau_sh);
}

/* Single-launch path, groups of one tile (tpg == 1), scalar integrands: one block takes a sibling group through its cell statistics
 * (R5) AND its threshold and flag count (R6, R7) -- the block reads back only what it wrote itself, so a __syncthreads stands where
 * the multi-launch path has a kernel boundary. On the last level (nothing can be flagged, R7) the group's accepted sums follow at
 * once, in the shape zmc_scatter_kernel gives them, and the compaction step is skipped. Same arithmetic, same shapes, same bits. */
__device__ __forceinline__ void zmc_group_control_body(const ZmcCtlArgs& c, const zu32 bid, const zu32 nb) {
    __shared__ double smem[ZMC_CTL_THREADS];
    __shared__ zu64 smem_u[ZMC_CTL_THREADS];
    __shared__ double tau_sh[ZMC_DEV_MAX_COMPONENTS];
    const zu64 n_groups = c.info[c.level].n_groups;
    __shared__ double sh[3 * ZMC_CTL_THREADS];
    for (zu64 G = bid; G < n_groups; G += nb) {
        zmc_cell_stats_batches(c, G * c.k, (G + 1ull) * c.k, 0ull, 1ull, sh);      /* ends with a __syncthreads */
        zmc_threshold_group(c, G, smem, smem_u, tau_sh);
        if (c.level >= c.L) {
            double acc_mu = 0.0, acc_var = 0.0;
            for (zu64 cell = G * c.k + threadIdx.x; cell < (G + 1ull) * c.k; cell += ZMC_CTL_THREADS) {
                const double sj = c.s[cell];
                acc_mu = __dadd_rn(acc_mu, c.mu[cell]);
                acc_var = __dadd_rn(acc_var, __dmul_rn(sj, sj));
                if (c.refined) c.refined[cell] = 0;
            }
            const double gm = zmc_block_sum(acc_mu, smem);
            const double gv = zmc_block_sum(acc_var, smem);
            if (threadIdx.x == 0) { c.gacc[2 * G] = gm; c.gacc[2 * G + 1] = gv; }
        }
    }
}
#ifndef ZMC_CONTROL_BODIES_ONLY
__global__ void __launch_bounds__(ZMC_CTL_THREADS) zmc_threshold_kernel(const __grid_constant__ ZmcCtlArgs c) { zmc_threshold_kernel_body(c, blockIdx.x, gridDim.x); }
#endif

/* R6 for groups of more than ZMC_TILE_CELLS cells (tpg > 1): the same two-pass moments, one block per TILE and one launch per
 * pass, because each pass needs the whole group's previous one:
 *   PASS 0  tsum[tile] = sum of s over the tile
 *   PASS 1  mean_G = (sum of the group's tsum, fixed shape) / k ;  tsq[tile] = sum of (s - mean_G)^2 over the tile
 *   PASS 2  pstd_G = sqrt((sum of the group's tsq) / k) ; tau_G = mean_G + m * pstd_G ; cnt[tile] = #(s > tau_G) in the tile */
__device__ __forceinline__ double zmc_group_total(const double* t, zu64 G, zu32 tpg, zu64 nc, zu64 jc, double* smem) {
    double part = 0.0;
    for (zu32 i = threadIdx.x; i < tpg; i += ZMC_CTL_THREADS) part = __dadd_rn(part, t[(G * tpg + i) * nc + jc]);
    return zmc_block_sum(part, smem);
}

template <int PASS>
__device__ __forceinline__ void zmc_threshold_pass_kernel_body(const ZmcCtlArgs& c, const zu32 bid, const zu32 nb) {
    __shared__ double smem[ZMC_CTL_THREADS];
    __shared__ zu64 smem_u[ZMC_CTL_THREADS];
    __shared__ double tau_sh[ZMC_DEV_MAX_COMPONENTS];
    const zu64 n_tiles = c.info[c.level].n_groups * c.tpg;
    const double dk = (double)c.k;
    const zu64 nc = c.nc;
    for (zu64 tile = bid; tile < n_tiles; tile += nb) {
        const ZmcTile T(c, tile);
        for (zu64 jc = 0; jc < nc; ++jc) {      /* R15: per component */
            double mean = 0.0;
            if (PASS >= 1) mean = __ddiv_rn(zmc_group_total(c.tsum, T.G, c.tpg, nc, jc, smem), dk);
            if (PASS == 2) {
                const double pstd = __dsqrt_rn(__ddiv_rn(zmc_group_total(c.tsq, T.G, c.tpg, nc, jc, smem), dk));
                const double tau = __dadd_rn(mean, __dmul_rn(c.m, pstd));
                if (threadIdx.x == 0) { tau_sh[jc] = tau; if (tile == T.G * c.tpg) c.tau[T.G * nc + jc] = tau; }
                continue;
            }
            double part = 0.0;
            for (zu64 cell = T.c0 + threadIdx.x; cell < T.c1; cell += ZMC_CTL_THREADS) {
                const double sj = c.s[cell * nc + jc];
                if (PASS == 0) part = __dadd_rn(part, sj);
                if (PASS == 1) { const double d = __dadd_rn(sj, -mean); part = __dadd_rn(part, __dmul_rn(d, d)); }
            }
            const double tot = zmc_block_sum(part, smem);
            if (threadIdx.x == 0) (PASS == 0 ? c.tsum : c.tsq)[tile * nc + jc] = tot;
        }
        if (PASS == 2) {
            __syncthreads();
            zu64 n = 0;
            if (c.level < c.L)
                for (zu64 cell = T.c0 + threadIdx.x; cell < T.c1; cell += ZMC_CTL_THREADS) {
                    bool any = false;
                    for (zu64 jc = 0; jc < nc; ++jc) any = any || (c.s[cell * nc + jc] > tau_sh[jc]);
                    n += any ? 1ull : 0ull;
                }
            n = zmc_block_sum_u64(n, smem_u);
            if (threadIdx.x == 0) c.cnt[tile] = n;
            __syncthreads();
        }
    }
}
template <int PASS>
__global__ void __launch_bounds__(ZMC_CTL_THREADS) zmc_threshold_pass_kernel(const __grid_constant__ ZmcCtlArgs c) { zmc_threshold_pass_kernel_body<PASS>(c, blockIdx.x, gridDim.x); }

/* block-wide exclusive scan of one value per thread (any block of whole warps, up to 1024 threads); returns the
 * exclusive prefix and writes the block total to *total */
__device__ __forceinline__ zu64 zmc_scan_block_excl(zu64 v, zu64* warp_tot, zu64* total) {
    const zu32 lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    zu64 inc = v;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const zu64 o = __shfl_up_sync(0xFFFFFFFFu, inc, off);
        if (lane >= (zu32)off) inc += o;
    }
    __syncthreads();
    if (lane == 31u) warp_tot[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        zu64 w = (lane < (blockDim.x >> 5)) ? warp_tot[lane] : 0ull;
        zu64 winc = w;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const zu64 o = __shfl_up_sync(0xFFFFFFFFu, winc, off);
            if (lane >= (zu32)off) winc += o;
        }
        warp_tot[lane] = winc - w;
        if (lane == 31u) *total = winc;
    }
    __syncthreads();
    return warp_tot[warp] + inc - v;
}

/* One block. (A) exclusive scan of cnt over the tiles and the first/last tile of every instance
 * (groups, hence tiles, are sorted by instance); (B) per instance: flagged c_b, kept = min(c_b, B) (R12), exclusive
 * scan -> first output slot; (C) the next level's plan. */
__device__ __forceinline__ void zmc_scan_kernel_body(const ZmcCtlArgs& c) {
    const zu32 NT = blockDim.x;     /* ZMC_SCAN_THREADS as its own launch; the block size of the single-launch tree kernel inside it */
    __shared__ zu64 warp_tot[32];
    __shared__ zu64 total;
    __shared__ zu64 carry;
    const zu64 n_tiles = c.info[c.level].n_groups * c.tpg;
    for (zu64 b = threadIdx.x; b < c.n_inst; b += NT) { c.gfirst[b] = 0; c.gend[b] = 0; }
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (zu64 base = 0; base < n_tiles; base += NT) {
        const zu64 t = base + threadIdx.x;
        const zu64 v = (t < n_tiles) ? c.cnt[t] : 0ull;
        const zu64 ex = zmc_scan_block_excl(v, warp_tot, &total);
        if (t < n_tiles) {
            c.excl[t] = carry + ex;
            const zu32 me = c.cur.inst[t / c.tpg];
            if (t == 0 || c.cur.inst[(t - 1) / c.tpg] != me) c.gfirst[me] = t;
            if (t + 1 == n_tiles || c.cur.inst[(t + 1) / c.tpg] != me) c.gend[me] = t + 1;
        }
        __syncthreads();
        if (threadIdx.x == 0) carry += total;
        __syncthreads();
    }
    const zu64 total_flagged = carry;
    __syncthreads();
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (zu64 base = 0; base < c.n_inst; base += NT) {
        const zu64 b = base + threadIdx.x;
        zu64 kept = 0;
        if (b < c.n_inst) {
            const zu64 g0 = c.gfirst[b], g1 = c.gend[b];
            if (g1 > g0) {
                const zu64 cb = c.excl[g1 - 1] + c.cnt[g1 - 1] - c.excl[g0];
                kept = (cb < c.budget) ? cb : c.budget;
            }
        }
        const zu64 ex = zmc_scan_block_excl(kept, warp_tot, &total);
        if (b < c.n_inst) c.out0[b] = carry + ex;
        __syncthreads();
        if (threadIdx.x == 0) carry += total;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        zu64 n_next = carry;
        if (n_next > c.cap_par) { n_next = c.stop_on_overflow ? 0ull : c.cap_par; *c.overflow = 1u; }
        c.info[c.level].n_flagged = total_flagged;
        c.info[c.level].n_refined = n_next;
        ZmcLevelInfo li;
        zmc_plan_level(li, (c.level < c.L) ? n_next : 0ull, c);
        c.info[c.level + 1] = li;
    }
}
#ifndef ZMC_CONTROL_BODIES_ONLY
__global__ void __launch_bounds__(ZMC_SCAN_THREADS) zmc_scan_kernel(const __grid_constant__ ZmcCtlArgs c) { zmc_scan_kernel_body(c); }
#endif

/* ------------------------------------------------------------------ R14: the budget keeps the largest spreads */
/* One block per instance: if more than B cells are flagged, radix-select (8 passes of 8 bits over the bit pattern
 * of s, which orders positive doubles) the B-th largest flagged spread -> piv, and how many cells equal to it are
 * kept -> quota = B - #(s > pivot). Otherwise piv = 0 and quota = all: no flagged cell is dropped (s >= +0, i.e. key >= 0). */
#ifndef ZMC_CONTROL_BODIES_ONLY
__global__ void __launch_bounds__(ZMC_SCAN_THREADS) zmc_select_kernel(const __grid_constant__ ZmcCtlArgs c) {
    __shared__ zu32 hist[256];
    __shared__ zu64 sh_prefix, sh_need, sh_above;
    for (zu64 b = blockIdx.x; b < c.n_inst; b += gridDim.x) {
        const zu64 g0 = c.gfirst[b], g1 = c.gend[b];     /* tiles; an instance owns whole groups, i.e. multiples of tpg tiles */
        const zu64 cb = (g1 > g0) ? c.excl[g1 - 1] + c.cnt[g1 - 1] - c.excl[g0] : 0ull;
        const zu64 cell0 = (g0 / c.tpg) * c.k, cell1 = (g1 / c.tpg) * c.k;
        __syncthreads();
        if (cb <= c.budget) {   /* nothing to cut: every flagged cell is kept -- also those with s == +0 (key 0), flagged when tau < 0 (m < 0) */
            if (threadIdx.x == 0) { c.piv[b] = 0ull; c.quota[b] = ~0ull; }
            continue;
        }
        if (threadIdx.x == 0) { sh_prefix = 0ull; sh_need = c.budget; sh_above = 0ull; }
        for (int pass = 7; pass >= 0; --pass) {
            const int shift = pass * 8;
            for (int i = threadIdx.x; i < 256; i += ZMC_SCAN_THREADS) hist[i] = 0u;
            __syncthreads();
            const zu64 prefix = sh_prefix;
            for (zu64 cell = cell0 + threadIdx.x; cell < cell1; cell += ZMC_SCAN_THREADS) {
                const double sj = c.s[cell];
                if (sj > c.tau[cell / c.k]) {
                    const zu64 key = (zu64)__double_as_longlong(sj);
                    if (pass == 7 || (key >> (shift + 8)) == (prefix >> (shift + 8))) atomicAdd(&hist[(key >> shift) & 255ull], 1u);
                }
            }
            __syncthreads();
            if (threadIdx.x == 0) {
                zu64 cum = 0, need = sh_need;
                int digit = 0;
                for (int dgt = 255; dgt >= 0; --dgt) {
                    if (cum + hist[dgt] >= need) { digit = dgt; break; }
                    cum += hist[dgt];
                }
                sh_need = need - cum;        /* rank, from the top, inside the chosen bin */
                sh_above += cum;             /* keys strictly greater than everything in the chosen bin */
                sh_prefix = prefix | ((zu64)digit << shift);
            }
            __syncthreads();
        }
        if (threadIdx.x == 0) { c.piv[b] = sh_prefix; c.quota[b] = c.budget - sh_above; }
    }
}
#endif

/* The same selection for FEW, LARGE instances (a single-instance level of 10^8 cells must not be walked eight times by one block):
 * one launch per step -- begin | 8 x (histogram by all tiles | pick one digit per instance). Integer logic only: the same pivot and quota. */
#ifndef ZMC_CONTROL_BODIES_ONLY
__global__ void __launch_bounds__(ZMC_CTL_THREADS) zmc_select_begin_kernel(const __grid_constant__ ZmcCtlArgs c) {
    for (zu64 b = blockIdx.x; b < c.n_inst; b += gridDim.x) {
        const zu64 g0 = c.gfirst[b], g1 = c.gend[b];
        const zu64 cb = (g1 > g0) ? c.excl[g1 - 1] + c.cnt[g1 - 1] - c.excl[g0] : 0ull;
        c.sel_hist[b * 256ull + threadIdx.x] = 0ull;
        if (threadIdx.x == 0) {
            zu64* st = c.sel_state + 4ull * b;
            st[0] = 0ull; st[1] = c.budget; st[2] = 0ull;
            st[3] = (cb > c.budget) ? 1ull : 0ull;
            if (cb <= c.budget) { c.piv[b] = 0ull; c.quota[b] = ~0ull; }     /* nothing to cut (see zmc_select_kernel) */
        }
    }
}

__global__ void __launch_bounds__(ZMC_CTL_THREADS) zmc_select_hist_kernel(const __grid_constant__ ZmcCtlArgs c, const int pass) {
    __shared__ zu32 hist[256];
    const zu64 n_tiles = c.info[c.level].n_groups * c.tpg;
    const int shift = pass * 8;
    for (zu64 tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const ZmcTile T(c, tile);
        const zu32 inst = c.cur.inst[T.G];
        const zu64* st = c.sel_state + 4ull * inst;
        if (st[3] == 0ull) continue;                     /* uniform over the block */
        const zu64 prefix = st[0];
        const double tau = c.tau[T.G];
        __syncthreads();
        hist[threadIdx.x] = 0u;
        __syncthreads();
        for (zu64 cell = T.c0 + threadIdx.x; cell < T.c1; cell += ZMC_CTL_THREADS) {
            const double sj = c.s[cell];
            if (sj > tau) {
                const zu64 key = (zu64)__double_as_longlong(sj);
                if (pass == 7 || (key >> (shift + 8)) == (prefix >> (shift + 8))) atomicAdd(&hist[(key >> shift) & 255ull], 1u);
            }
        }
        __syncthreads();
        const zu32 h = hist[threadIdx.x];
        if (h) atomicAdd((unsigned long long*)&c.sel_hist[inst * 256ull + threadIdx.x], (unsigned long long)h);
    }
}

__global__ void __launch_bounds__(ZMC_CTL_THREADS) zmc_select_pick_kernel(const __grid_constant__ ZmcCtlArgs c, const int pass) {
    __shared__ zu64 h[256];
    for (zu64 b = blockIdx.x; b < c.n_inst; b += gridDim.x) {
        zu64* st = c.sel_state + 4ull * b;
        __syncthreads();
        h[threadIdx.x] = c.sel_hist[b * 256ull + threadIdx.x];
        c.sel_hist[b * 256ull + threadIdx.x] = 0ull;     /* ready for the next pass */
        __syncthreads();
        if (threadIdx.x == 0 && st[3] != 0ull) {
            zu64 cum = 0, need = st[1];
            int digit = 0;
            for (int dgt = 255; dgt >= 0; --dgt) {
                if (cum + h[dgt] >= need) { digit = dgt; break; }
                cum += h[dgt];
            }
            st[1] = need - cum;
            st[2] += cum;
            st[0] |= (zu64)digit << (pass * 8);
            if (pass == 0) { c.piv[b] = st[0]; c.quota[b] = c.budget - st[2]; }
        }
    }
}
#endif

/* per tile: flagged cells above and at the instance's pivot */
#ifndef ZMC_CONTROL_BODIES_ONLY
__global__ void __launch_bounds__(ZMC_CTL_THREADS) zmc_count2_kernel(const __grid_constant__ ZmcCtlArgs c) {
    __shared__ zu64 smem_u[ZMC_CTL_THREADS];
    const zu64 n_tiles = c.info[c.level].n_groups * c.tpg;
    for (zu64 tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const ZmcTile T(c, tile);
        const double tau = c.tau[T.G];
        const zu64 piv = c.piv[c.cur.inst[T.G]];
        zu64 ngt = 0, neq = 0;
        if (c.level < c.L)
            for (zu64 cell = T.c0 + threadIdx.x; cell < T.c1; cell += ZMC_CTL_THREADS) {
                const double sj = c.s[cell];
                if (sj > tau) {
                    const zu64 key = (zu64)__double_as_longlong(sj);
                    ngt += (key > piv) ? 1ull : 0ull;
                    neq += (key == piv) ? 1ull : 0ull;
                }
            }
        ngt = zmc_block_sum_u64(ngt, smem_u);
        neq = zmc_block_sum_u64(neq, smem_u);
        if (threadIdx.x == 0) { c.cnt_gt[tile] = ngt; c.cnt_eq[tile] = neq; }
    }
}
#endif

/* One block: exclusive scans of cnt_gt and cnt_eq over the tiles. */
#ifndef ZMC_CONTROL_BODIES_ONLY
__global__ void __launch_bounds__(ZMC_SCAN_THREADS) zmc_scan2_kernel(const __grid_constant__ ZmcCtlArgs c) {
    __shared__ zu64 warp_tot[32];
    __shared__ zu64 total;
    __shared__ zu64 carry;
    const zu64 n_groups = c.info[c.level].n_groups * c.tpg;     /* tiles */
    for (int which = 0; which < 2; ++which) {
        const zu64* in = which ? c.cnt_eq : c.cnt_gt;
        zu64* out = which ? c.excl_eq : c.excl_gt;
        __syncthreads();
        if (threadIdx.x == 0) carry = 0;
        __syncthreads();
        for (zu64 base = 0; base < n_groups; base += ZMC_SCAN_THREADS) {
            const zu64 G = base + threadIdx.x;
            const zu64 v = (G < n_groups) ? in[G] : 0ull;
            const zu64 ex = zmc_scan_block_excl(v, warp_tot, &total);
            if (G < n_groups) out[G] = carry + ex;
            __syncthreads();
            if (threadIdx.x == 0) carry += total;
            __syncthreads();
        }
    }
}
#endif

/* R7: one block per tile. Flagged cells get their rank within the instance (stable, path
 * order); rank < B (R12) and slot < capacity -> the child record (R2) is written to the next parent
 * list. Every other cell is accepted: its mu and s^2 go into the tile's fixed-shape sums. */
/* VEC (R15, nc > 1): a cell is flagged iff some component's spread passes that component's threshold, and the accepted sums are
 * kept per component; the scalar instance is the code as it was. */
template <bool VEC>
__device__ __forceinline__ void zmc_scatter_kernel_body(const ZmcCtlArgs& c, const zu32 bid, const zu32 nb) {
    __shared__ double smem[ZMC_CTL_THREADS];
    __shared__ zu32 warp_cnt[ZMC_CTL_THREADS / 32], warp_cnt_eq[ZMC_CTL_THREADS / 32];
    __shared__ zu64 run, run_eq;
    const zu64 n_tiles = c.info[c.level].n_groups * c.tpg;
    const zu32 lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    for (zu64 tile = bid; tile < n_tiles; tile += nb) {
        const ZmcTile T(c, tile);
        const zu64 G = T.G;
        const zu32 inst = c.cur.inst[G];
        const zu64 nc = VEC ? (zu64)c.nc : 1ull;
        const double tau = c.tau[G * nc];
        const bool by_spread = !VEC && (c.budget_order != 0) && (c.budget != ~0ull);
        const zu64 gf = c.gfirst[inst];
        const zu64 r0 = c.excl[tile] - c.excl[gf];   /* flagged cells of this instance in earlier tiles */
        const zu64 r0_gt = by_spread ? c.excl_gt[tile] - c.excl_gt[gf] : 0ull;   /* ... above the pivot */
        const zu64 r0_eq = by_spread ? c.excl_eq[tile] - c.excl_eq[gf] : 0ull;   /* ... at the pivot */
        const zu64 piv = by_spread ? c.piv[inst] : 0ull;
        const zu64 quota = by_spread ? c.quota[inst] : 0ull;
        const zu64 slot0 = c.out0[inst];
        const zu64 plo = c.cur.plo[G];
        const zu32 phi = c.cur.phi[G];
        const zu64 j0 = T.c0 - G * c.k;              /* child index of the tile's first cell */
        const zu64 n_tile = T.c1 - T.c0;
        double acc_mu = 0.0, acc_var = 0.0;
        double vacc_mu[VEC ? ZMC_DEV_MAX_COMPONENTS : 1], vacc_var[VEC ? ZMC_DEV_MAX_COMPONENTS : 1];
        if constexpr (VEC)
            for (int jc = 0; jc < ZMC_DEV_MAX_COMPONENTS; ++jc) { vacc_mu[jc] = 0.0; vacc_var[jc] = 0.0; }
        __syncthreads();
        if (threadIdx.x == 0) { run = 0; run_eq = 0; }
        __syncthreads();
        for (zu64 base = 0; base < n_tile; base += ZMC_CTL_THREADS) {
            const zu64 i = base + threadIdx.x;
            const zu64 j = j0 + i;
            const zu64 cell = T.c0 + i;
            double sj = 0.0, muj = 0.0;
            bool flag = false;
            if (i < n_tile) {
                if constexpr (!VEC) {
                    sj = c.s[cell];
                    muj = c.mu[cell];
                    flag = (c.level < c.L) && (sj > tau);
                } else {
                    for (zu64 jc = 0; jc < nc; ++jc) flag = flag || (c.s[cell * nc + jc] > c.tau[G * nc + jc]);
                    flag = flag && (c.level < c.L);
                }
            }
            /* path order: every flagged cell counts in `run`. Largest spread: cells above the pivot count in `run`,
             * cells at the pivot in `run_eq`; cells below it are not candidates. */
            const zu64 key = (zu64)__double_as_longlong(sj);
            const bool is_eq = by_spread && flag && key == piv;
            const bool is_a = by_spread ? (flag && key > piv) : flag;
            const zu32 bal = __ballot_sync(0xFFFFFFFFu, is_a);
            const zu32 bal_eq = __ballot_sync(0xFFFFFFFFu, is_eq);
            if (lane == 0) { warp_cnt[warp] = __popc(bal); warp_cnt_eq[warp] = __popc(bal_eq); }
            __syncthreads();
            zu64 before = run, before_eq = run_eq;
            zu32 tile_total = 0, tile_total_eq = 0;
#pragma unroll
            for (int w = 0; w < ZMC_CTL_THREADS / 32; ++w) {
                if ((zu32)w < warp) { before += warp_cnt[w]; before_eq += warp_cnt_eq[w]; }
                tile_total += warp_cnt[w];
                tile_total_eq += warp_cnt_eq[w];
            }
            const zu32 below = (1u << lane) - 1u;
            zu64 rank;          /* position among the cells that are kept, in path order */
            bool want;
            if (by_spread) {
                const zu64 n_gt = r0_gt + before + __popc(bal & below);
                const zu64 n_eq = r0_eq + before_eq + __popc(bal_eq & below);
                want = is_a || (is_eq && n_eq < quota);
                rank = n_gt + (n_eq < quota ? n_eq : quota);
            } else {
                rank = r0 + before + __popc(bal & below);
                want = flag && rank < c.budget;
            }
            bool kept = false;
            if (want) {
                const zu64 slot = slot0 + rank;
                if (slot < c.cap_par) {
                    kept = true;
                    /* R2: P' = P*k + j (80 bits) ; I'_d = I_d*g + j_d, axis 0 least significant */
                    const zu64 nlo = plo * c.k + j;
                    const zu64 cy = __umul64hi(plo, c.k) + ((nlo < j) ? 1ull : 0ull);
                    c.next.inst[slot] = inst;
                    c.next.plo[slot] = nlo;
                    c.next.phi[slot] = (zu32)((zu64)phi * c.k + cy);
                    zu64 rem = j;
                    for (zu32 d = 0; d < c.D; ++d) {
                        const zu64 q = rem / c.g;
                        const zu32 jd = (zu32)(rem - q * c.g);
                        rem = q;
                        c.next.coord[(zu64)d * c.par_stride + slot] = c.cur.coord[(zu64)d * c.par_stride + G] * c.g + jd;
                    }
                }
            }
            if (i < n_tile) {
                if constexpr (!VEC) {
                    if (!kept) { acc_mu = __dadd_rn(acc_mu, muj); acc_var = __dadd_rn(acc_var, __dmul_rn(sj, sj)); }
                } else if (!kept) {
                    for (zu64 jc = 0; jc < nc; ++jc) {
                        const double sv = c.s[cell * nc + jc];
                        vacc_mu[jc] = __dadd_rn(vacc_mu[jc], c.mu[cell * nc + jc]);
                        vacc_var[jc] = __dadd_rn(vacc_var[jc], __dmul_rn(sv, sv));
                    }
                }
                if (c.refined) c.refined[cell] = kept ? 1 : 0;
            }
            __syncthreads();
            if (threadIdx.x == 0) { run += tile_total; run_eq += tile_total_eq; }
            __syncthreads();
        }
        if constexpr (!VEC) {
            const double gm = zmc_block_sum(acc_mu, smem);
            const double gv = zmc_block_sum(acc_var, smem);
            if (threadIdx.x == 0) { c.gacc[2 * tile] = gm; c.gacc[2 * tile + 1] = gv; }
        } else {
            for (zu64 jc = 0; jc < nc; ++jc) {
                const double gm = zmc_block_sum(vacc_mu[jc], smem);
                const double gv = zmc_block_sum(vacc_var[jc], smem);
                if (threadIdx.x == 0) { c.gacc[2 * (tile * nc + jc)] = gm; c.gacc[2 * (tile * nc + jc) + 1] = gv; }
            }
        }
    }
}
template <bool VEC>
__global__ void __launch_bounds__(ZMC_CTL_THREADS) zmc_scatter_kernel(const __grid_constant__ ZmcCtlArgs c) { zmc_scatter_kernel_body<VEC>(c, blockIdx.x, gridDim.x); }

/* R7: value_b += sum of accepted mu ; var_b += sum of accepted s^2, one block per instance, over its tiles */
__device__ __forceinline__ void zmc_accumulate_kernel_body(const ZmcCtlArgs& c, const zu32 bid, const zu32 nb) {
    __shared__ double smem[ZMC_CTL_THREADS];
    const zu64 nc = c.nc;
    for (zu64 e = bid; e < (zu64)c.n_inst * nc; e += nb) {      /* one block per (instance, component) */
        const zu64 b = e / nc, jc = e - b * nc;
        const zu64 g0 = c.gfirst[b], g1 = c.gend[b];
        double am = 0.0, av = 0.0;
        for (zu64 G = g0 + threadIdx.x; G < g1; G += ZMC_CTL_THREADS) {
            am = __dadd_rn(am, c.gacc[2 * (G * nc + jc)]);
            av = __dadd_rn(av, c.gacc[2 * (G * nc + jc) + 1]);
        }
        const double sm = zmc_block_sum(am, smem);
        const double sv = zmc_block_sum(av, smem);
        if (threadIdx.x == 0 && g1 > g0) {
            c.value[e] = __dadd_rn(c.value[e], sm);
            c.var[e] = __dadd_rn(c.var[e], sv);
        }
    }
}
#ifndef ZMC_CONTROL_BODIES_ONLY
__global__ void __launch_bounds__(ZMC_CTL_THREADS) zmc_accumulate_kernel(const __grid_constant__ ZmcCtlArgs c) { zmc_accumulate_kernel_body(c, blockIdx.x, gridDim.x); }
#endif

/* result[b] = value_b ; result[n_inst + b] = sqrt(var_b)   (n_inst here = instances * components, R15) */
__device__ __forceinline__ void zmc_finalize_body(const double* value, const double* var, double* result, zu32 n_inst, zu32 bid, zu32 nb) {
    for (zu64 b = (zu64)bid * blockDim.x + threadIdx.x; b < n_inst; b += (zu64)nb * blockDim.x) {
        result[b] = value[b];
        result[n_inst + b] = __dsqrt_rn(var[b]);
    }
}
#ifndef ZMC_CONTROL_BODIES_ONLY
__global__ void zmc_finalize_kernel(const double* value, const double* var, double* result, zu32 n_inst) {
    zmc_finalize_body(value, var, result, n_inst, blockIdx.x, gridDim.x);
}
#endif

/* debug: words of one unit's flat stream (R3) */
#ifndef ZMC_CONTROL_BODIES_ONLY
__global__ void zmc_words_kernel(const zu32* keys, zu32 inst, zu64 path_lo, zu32 path_hi, zu32 level, zu32 trial,
                                 zu64 first_word, zu64 n_words, zu32* out) {
    ZmcKeySchedule ks;
    ks.init(keys[2 * inst], keys[2 * inst + 1]);
    ZmcUnitCounter uc;
    uc.init(path_lo, path_hi, level, trial);
    for (zu64 i = (zu64)blockIdx.x * blockDim.x + threadIdx.x; i < n_words; i += (zu64)gridDim.x * blockDim.x) {
        const zu64 idx = first_word + i;
        zu32 w[4];
        zmc_philox((zu32)(idx >> 2), uc.c1, uc.c2, uc.c3, ks, w);
        const zu32 l = (zu32)(idx & 3ull);
        out[i] = (l == 0) ? w[0] : (l == 1) ? w[1] : (l == 2) ? w[2] : w[3];
    }
}
#endif

#endif /* ZMC_CONTROL_CUH */

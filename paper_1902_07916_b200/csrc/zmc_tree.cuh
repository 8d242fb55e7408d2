/*
 * zmc_tree.cuh -- the whole tree search as ONE cooperative launch, for problems whose kernels are so short that the launches
 * between them are the time-to-result (BASELINE.json configs[0]: 3.84e6 evaluations, 14 dependent kernels; the paper's own
 * Table 3, is about exactly this per-call overhead).
 *
 * The kernel runs, for level = 1 .. L:
 *
 *     sampling phase     every warp of the grid pulls work items, as zmc_sample_kernel does        (H2-H6)
 *     -- grid barrier --
 *     control phase      cell statistics, thresholds, flag counts, scan, compaction, accepted sums  (H7-H10)
 *     -- grid barrier --
 *
 * with the device functions of the multi-launch path (zmc_sample_items, zmc_*_body), so that the two paths give the same
 * bits: the work-item plan, every sum's shape and every comparison are the same code. A grid barrier costs 1.2 us on B200
 * (296 blocks, measured), so the control phase is cut to few of them: one block takes a whole sibling group through statistics,
 * threshold and flag count (zmc_group_control_body) | barrier | block 0 scans | barrier | compaction by all | barrier; the
 * accepted sums are added by block 0 while the others already sample the next level; the last level, where nothing can be
 * flagged, skips scan and compaction. Groups of several control tiles (k > 4096) keep the step-by-step order of the kernels.
 *
 * Scalar integrands, spread from the trials (R5) and path-order budget (R12) only: R13 needs the sum-of-squares sampling
 * kernel, R14 three more control steps -- zmc_run takes the multi-launch path for those.
 */
#ifndef ZMC_TREE_CUH
#define ZMC_TREE_CUH
#include <cooperative_groups.h>

#include "zmc_control.cuh"

struct ZmcTreeArgs {
    const ZmcSampleArgs* sample;   /* [L] in device memory: the launch parameters the multi-launch path passes per level */
    const ZmcCtlArgs* ctl;         /* [L] */
    zu32 L, n_res;                 /* depth ; results = instances * components */
    const double* value;
    const double* var;
    double* result;
};

/* block 0 stamps %globaltimer as it passes the level's grid barriers: zmc_stats turns the stamps into per-level times */
__device__ __forceinline__ void zmc_tree_mark(const ZmcCtlArgs& ca, zu32 level, int which) {
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        zu64 t;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
        ca.info[level].t_mark[which] = t;
    }
}

/* two 256-thread blocks per SM (128 registers) keep as many warps on the sampling phase as the multi-launch kernel has; FP64 at
 * high D would spill there */
template <class F> struct ZmcTreeTune { static constexpr int MINB = (F::PREC == ZMC_PREC_F64 && F::D >= 7) ? 1 : 2; };

template <class F>
__global__ void __launch_bounds__(ZMC_CTL_THREADS, ZmcTreeTune<F>::MINB) zmc_tree_kernel(const __grid_constant__ ZmcTreeArgs t) {
    namespace cg = cooperative_groups;
    cg::grid_group grid = cg::this_grid();
    __shared__ ZmcSampleArgs sa;      /* this level's parameters, copied once per block: the item loop reads them often */
    __shared__ ZmcCtlArgs ca;
    if (blockIdx.x == 0) {
        if (threadIdx.x == 0) ca = t.ctl[0];
        __syncthreads();
        zmc_init_kernel_body(ca, 0u, 1u);
    }
    grid.sync();
    for (zu32 level = 1; level <= t.L; ++level) {
        __syncthreads();
        if (threadIdx.x == 0) { sa = t.sample[level - 1]; ca = t.ctl[level - 1]; }
        __syncthreads();
        zmc_tree_mark(ca, level, 0);
        zmc_sample_items<F, false, false>(sa);
        grid.sync();
        zmc_tree_mark(ca, level, 1);
        const bool last = level >= t.L;
        const bool fused = ca.tpg == 1u;       /* a sibling group is one control tile: statistics, threshold and count by one block */
        if (fused) {
            zmc_group_control_body(ca, blockIdx.x, gridDim.x);
        } else {
            zmc_cell_stats_kernel_body(ca, blockIdx.x, gridDim.x);
            grid.sync();
            zmc_threshold_pass_kernel_body<0>(ca, blockIdx.x, gridDim.x);
            grid.sync();
            zmc_threshold_pass_kernel_body<1>(ca, blockIdx.x, gridDim.x);
            grid.sync();
            zmc_threshold_pass_kernel_body<2>(ca, blockIdx.x, gridDim.x);
        }
        grid.sync();
        zmc_tree_mark(ca, level, 2);
        if (fused && last) break;             /* the accepted sums are there: block 0 finishes below */
        if (blockIdx.x == 0) zmc_scan_kernel_body(ca);
        grid.sync();
        zmc_scatter_kernel_body<false>(ca, blockIdx.x, gridDim.x);
        grid.sync();
        zmc_tree_mark(ca, level, 3);
        /* value += accepted sums: nobody needs it before the end, so block 0 does it while the others sample the next level */
        if (blockIdx.x == 0) zmc_accumulate_kernel_body(ca, 0u, 1u);
    }
    if (blockIdx.x == 0) {
        if (ca.tpg == 1u) {                    /* the last level's bookkeeping (first and last tile per instance, empty next level) and sums */
            zmc_scan_kernel_body(ca);
            __syncthreads();
            zmc_accumulate_kernel_body(ca, 0u, 1u);
        }
        __syncthreads();
        zmc_finalize_body(t.value, t.var, t.result, t.n_res, 0u, 1u);
        zmc_tree_mark(ca, t.L, 3);
    }
}

#endif /* ZMC_TREE_CUH */

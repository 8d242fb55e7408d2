/* zmc_inst.h -- lookup of the pre-compiled sampling kernels (one translation unit per
 * (precision, math mode, integrand); see zmc_inst.cu and build.py). Host side only. */
#ifndef ZMC_INST_H
#define ZMC_INST_H

#define ZMC_AOT_MAX_DIM 12
#define ZMC_TREE_MAX_DIM 8     /* zmc_tree_kernel<F> is pre-compiled for D <= 8, exact math */

struct ZmcKernelEntry {
    const void* sample;       /* zmc_sample_kernel<F, false>: per-item key (batched instances) */
    const void* sample_ukey;  /* zmc_sample_kernel<F, true>: one key for the whole launch (n_instances == 1) */
    const void* points;   /* zmc_points_kernel<F> */
    const void* tree;     /* zmc_tree_kernel<F>: the whole tree search as one cooperative launch (zmc_tree.cuh); nullptr where not compiled */
};

#define ZMC_DECLARE_LOOKUP(PREC, MODE, ID) ZmcKernelEntry zmc_lookup_##PREC##_##MODE##_##ID(int dim);
ZMC_DECLARE_LOOKUP(0, 0, 0) ZMC_DECLARE_LOOKUP(0, 0, 1) ZMC_DECLARE_LOOKUP(0, 0, 2) ZMC_DECLARE_LOOKUP(0, 0, 3)
ZMC_DECLARE_LOOKUP(1, 0, 0) ZMC_DECLARE_LOOKUP(1, 0, 1) ZMC_DECLARE_LOOKUP(1, 0, 2) ZMC_DECLARE_LOOKUP(1, 0, 3)
ZMC_DECLARE_LOOKUP(1, 1, 2) ZMC_DECLARE_LOOKUP(1, 1, 3)

#endif

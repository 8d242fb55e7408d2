/* zmc_inst.cu -- pre-compiled instances of the sampling kernel (and of the single-launch tree kernel around it) for one (precision, math mode,
 * integrand) and every dimension 1..ZMC_AOT_MAX_DIM. build.py compiles this file once per
 * combination with -DZMC_INST_PREC= -DZMC_INST_MODE= -DZMC_INST_ID= (in parallel). */
#define ZMC_CONTROL_BODIES_ONLY
#include "zmc_tree.cuh"
#include "zmc_inst.h"

#if !defined(ZMC_INST_PREC) || !defined(ZMC_INST_MODE) || !defined(ZMC_INST_ID)
#error "compile with -DZMC_INST_PREC=<0|1> -DZMC_INST_MODE=<0|1> -DZMC_INST_ID=<0..3>"
#endif

template <int D>
static ZmcKernelEntry zmc_entry() {
    using F = ZmcIntegrand<ZMC_INST_ID, D, ZMC_INST_PREC, ZMC_INST_MODE>;
    ZmcKernelEntry e;
    e.sample = (const void*)zmc_sample_kernel<F, false>;
    e.sample_ukey = (const void*)zmc_sample_kernel<F, true>;
    e.points = (const void*)zmc_points_kernel<F>;
    /* the single-launch tree kernel is for launch-bound problems: low dimensions, exact math (it doubles the compile time of an instance) */
    if constexpr (D <= ZMC_TREE_MAX_DIM && ZMC_INST_MODE == ZMC_MODE_EXACT) e.tree = (const void*)zmc_tree_kernel<F>;
    else e.tree = nullptr;
    return e;
}

#define ZMC_CAT5(a, b, c, d, e, f) a##b##c##d##e##f
#define ZMC_LOOKUP_NAME(PREC, MODE, ID) ZMC_CAT5(zmc_lookup_, PREC, _, MODE, _, ID)

ZmcKernelEntry ZMC_LOOKUP_NAME(ZMC_INST_PREC, ZMC_INST_MODE, ZMC_INST_ID)(int dim) {
    switch (dim) {
        case 1: return zmc_entry<1>();
        case 2: return zmc_entry<2>();
        case 3: return zmc_entry<3>();
        case 4: return zmc_entry<4>();
        case 5: return zmc_entry<5>();
        case 6: return zmc_entry<6>();
        case 7: return zmc_entry<7>();
        case 8: return zmc_entry<8>();
        case 9: return zmc_entry<9>();
        case 10: return zmc_entry<10>();
        case 11: return zmc_entry<11>();
        case 12: return zmc_entry<12>();
    }
    ZmcKernelEntry none = {nullptr, nullptr, nullptr, nullptr};
    return none;
}

// ss_warp_tu.cu -- instantiations of the warp-per-eval kernel.  Compiled twelve times by _build.py:
//   -DSS_TU_GV=0|1 (cross-validation / generalized validation)  x  -DSS_TU_GROUP=0|1|2 (C = 2..4 / 5..6 / 7..8)
//   x -DSS_TU_SHARED=0|1|2|3 (warp_kernel / warp_shared_kernel, the shared-time-sampling variant / warp_opt_kernel,
//     the listing's options / warp_kernel with the smoother in fp32, the MIXED precision)
// so that the kernels build in parallel.
#include "ss_launch.h"
#include "ss_warp_kernel.cuh"
#include "ss_warp_opt.cuh"
#include "ss_warp_shared.cuh"

#ifndef SS_TU_GV
#error "compile with -DSS_TU_GV=0|1 -DSS_TU_GROUP=0|1|2 -DSS_TU_SHARED=0|1|2|3"
#endif

namespace ss {

#define SS_CAT2(a, b, c, d) a##b##c##d
#define SS_CAT(a, b, c, d) SS_CAT2(a, b, c, d)
#if SS_TU_SHARED == 1
#define SS_TU_FN SS_CAT(launch_warp_shared_tu_, SS_TU_GV, _, SS_TU_GROUP)
#define SS_TU_LAUNCH(C_, I_) launch_warp_shared_variant<C_, I_, GV>
#elif SS_TU_SHARED == 3
// MIXED precision: the same kernel with the smoother in fp32
#define SS_TU_FN SS_CAT(launch_warp_f32_tu_, SS_TU_GV, _, SS_TU_GROUP)
#define SS_TU_LAUNCH(C_, I_) launch_warp_variant<C_, I_, GV, float>
#else
#define SS_TU_FN SS_CAT(launch_warp_tu_, SS_TU_GV, _, SS_TU_GROUP)
#define SS_TU_LAUNCH(C_, I_) launch_warp_variant<C_, I_, GV, double>
#endif

#if SS_TU_SHARED == 2
// the options variant (ss_warp_opt.cuh): variant = points per lane C; mode 0 = CV, 1 = GV, 2 = fixed span.  This
// translation unit holds MODE = SS_TU_GV, and the fixed-span kernels ride with SS_TU_GV = 0.
#undef SS_TU_FN
#define SS_TU_FN SS_CAT(launch_warp_opt_tu_, SS_TU_GV, _, SS_TU_GROUP)
ss_status_t SS_TU_FN(const EvalParams& p, int c, int mode, int64_t n_items, cudaStream_t stream)
{
#define SS_OPT_CASE(C_)                                                                                   \
    case C_:                                                                                               \
        if (mode == SS_TU_GV) return launch_warp_opt_variant<C_, SS_TU_GV>(p, n_items, stream);            \
        if (SS_TU_GV == 0 && mode == 2) return launch_warp_opt_variant<C_, SS_TU_GV == 0 ? 2 : 1>(p, n_items, stream); \
        return SS_ERR_UNSUPPORTED;
    switch (c) {
#if SS_TU_GROUP == 0
        SS_OPT_CASE(2) SS_OPT_CASE(3) SS_OPT_CASE(4)
#elif SS_TU_GROUP == 1
        SS_OPT_CASE(5) SS_OPT_CASE(6)
#else
        SS_OPT_CASE(7) SS_OPT_CASE(8)
#endif
        default: return SS_ERR_UNSUPPORTED;
    }
#undef SS_OPT_CASE
}
#else
ss_status_t SS_TU_FN(const EvalParams& p, int variant, int64_t n_items, cudaStream_t stream)
{
    constexpr bool GV = SS_TU_GV != 0;
    switch (variant) {
#if SS_TU_GROUP == 0
        case 2 * 8 + 2: return SS_TU_LAUNCH(2, 2)(p, n_items, stream);
        case 3 * 8 + 2: return SS_TU_LAUNCH(3, 2)(p, n_items, stream);
        case 4 * 8 + 2: return SS_TU_LAUNCH(4, 2)(p, n_items, stream);
        case 4 * 8 + 3: return SS_TU_LAUNCH(4, 3)(p, n_items, stream);
#elif SS_TU_GROUP == 1
        case 5 * 8 + 3: return SS_TU_LAUNCH(5, 3)(p, n_items, stream);
        case 5 * 8 + 4: return SS_TU_LAUNCH(5, 4)(p, n_items, stream);
        case 6 * 8 + 4: return SS_TU_LAUNCH(6, 4)(p, n_items, stream);
        case 6 * 8 + 5: return SS_TU_LAUNCH(6, 5)(p, n_items, stream);
#else
        case 7 * 8 + 5: return SS_TU_LAUNCH(7, 5)(p, n_items, stream);
        case 8 * 8 + 6: return SS_TU_LAUNCH(8, 6)(p, n_items, stream);
#endif
        default: return SS_ERR_UNSUPPORTED;
    }
}
#endif

}  // namespace ss

// ss_group_tu.cu -- instantiations of the G-warps-per-eval kernel (ss_group_kernel.cuh).  Compiled 24 times by
// _build.py: -DSS_TU_GV=0|1 x -DSS_TU_G=4|8|16 x -DSS_TU_F32=0|1|2|3 (smoother scalar double / float / double with the
// listing's options compiled in / double for catalogs with one shared time sampling), three to five kernels each
// (C = 3..7 points per thread).
#include "ss_group_kernel.cuh"
#include "ss_launch.h"

#ifndef SS_TU_GV
#error "compile with -DSS_TU_GV=0|1 -DSS_TU_G=4|8|16 -DSS_TU_F32=0|1|2|3"
#endif

namespace ss {

#define SS_CAT2(a, b, c, d) a##b##c##d
#define SS_CAT(a, b, c, d) SS_CAT2(a, b, c, d)
#if SS_TU_F32 == 2
// the listing's options (periodic windows; with SS_TU_GV = 0 also the fixed-span kernels): mode 0 = CV, 1 = GV, 2 = fixed
#define SS_TU_FN SS_CAT(launch_group_opt_tu_, SS_TU_GV, _, SS_TU_G)
typedef double tu_real;
#elif SS_TU_F32 == 3
// shared time sampling: SHARED_TIMES_M objects per work item, one fold + sort per frequency
#define SS_TU_FN SS_CAT(launch_group_shared_tu_, SS_TU_GV, _, SS_TU_G)
#define SS_TU_OPT 3
typedef double tu_real;
#elif SS_TU_F32
#define SS_TU_FN SS_CAT(launch_group_f32_tu_, SS_TU_GV, _, SS_TU_G)
typedef float tu_real;
#else
#define SS_TU_FN SS_CAT(launch_group_tu_, SS_TU_GV, _, SS_TU_G)
typedef double tu_real;
#endif

#if SS_TU_F32 == 2
ss_status_t SS_TU_FN(const EvalParams& p, int c, int mode, int64_t n_items, cudaStream_t stream)
{
#if SS_TU_GV == 0
#define SS_OPT_CASE(C_)                                                                                            \
    case C_:                                                                                                       \
        return mode == 2 ? launch_group_variant<SS_TU_G, C_, false, double, 2>(p, n_items, stream)                 \
                         : launch_group_variant<SS_TU_G, C_, false, double, 1>(p, n_items, stream);
#else
#define SS_OPT_CASE(C_) \
    case C_: return launch_group_variant<SS_TU_G, C_, true, double, 1>(p, n_items, stream);
#endif
    (void)mode;
    switch (c) {
        SS_OPT_CASE(3) SS_OPT_CASE(4) SS_OPT_CASE(5) SS_OPT_CASE(6) SS_OPT_CASE(7)
        default: return SS_ERR_UNSUPPORTED;
    }
#undef SS_OPT_CASE
}
#else
#ifndef SS_TU_OPT
#define SS_TU_OPT 0
#endif
ss_status_t SS_TU_FN(const EvalParams& p, int c, int64_t n_items, cudaStream_t stream)
{
    constexpr bool GV = SS_TU_GV != 0;
    switch (c) {
        case 3: return launch_group_variant<SS_TU_G, 3, GV, tu_real, SS_TU_OPT>(p, n_items, stream);
        case 4: return launch_group_variant<SS_TU_G, 4, GV, tu_real, SS_TU_OPT>(p, n_items, stream);
        case 5: return launch_group_variant<SS_TU_G, 5, GV, tu_real, SS_TU_OPT>(p, n_items, stream);
        case 6: return launch_group_variant<SS_TU_G, 6, GV, tu_real, SS_TU_OPT>(p, n_items, stream);
        case 7: return launch_group_variant<SS_TU_G, 7, GV, tu_real, SS_TU_OPT>(p, n_items, stream);
        default: return SS_ERR_UNSUPPORTED;
    }
}
#endif

}  // namespace ss

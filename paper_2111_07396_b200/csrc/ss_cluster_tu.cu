// ss_cluster_tu.cu -- instantiations of the cluster-per-eval kernel (ss_cluster_kernel.cuh).  Compiled six times by
// _build.py: -DSS_TU_GV=0|1 x -DSS_TU_C=3|4|5 (points per thread); the cluster size R is a launch parameter.
#include "ss_cluster_kernel.cuh"
#include "ss_launch.h"

#ifndef SS_TU_GV
#error "compile with -DSS_TU_GV=0|1 -DSS_TU_C=3|4|5"
#endif

namespace ss {

#define SS_CAT2(a, b, c, d) a##b##c##d
#define SS_CAT(a, b, c, d) SS_CAT2(a, b, c, d)
#define SS_TU_FN SS_CAT(launch_cluster_tu_, SS_TU_GV, _, SS_TU_C)

ss_status_t SS_TU_FN(const EvalParams& p, int r, int64_t n_items, cudaStream_t stream)
{
    return launch_cluster_variant<SS_TU_C, SS_TU_GV != 0>(p, r, n_items, stream);
}

}  // namespace ss

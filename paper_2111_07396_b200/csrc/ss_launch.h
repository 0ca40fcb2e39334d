// ss_launch.h -- host-side launchers of the eval kernels.  The kernels are instantiated in their own translation
// units (ss_warp_tu.cu is compiled once per mode and variant group, ss_block_tu.cu once) so the library builds in
// parallel; ss_api.cu sees only these declarations.
#pragma once
#include <cuda_runtime.h>

#include "../../include/ss_periodogram.h"
#include "ss_common.cuh"

namespace ss {

// warp-per-eval kernels (ss_warp_kernel.cuh); variant = warp_variant_for_n(n)
ss_status_t launch_warp_kernel(const EvalParams& p, int variant, int64_t n_items, cudaStream_t stream);

// the same for a catalog with one shared time sampling (ss_warp_shared.cuh): n_items = groups of SHARED_M objects x chunks
ss_status_t launch_warp_shared_kernel(const EvalParams& p, int variant, int64_t n_items, cudaStream_t stream);

// the listing's options on the warp path (ss_warp_opt.cuh): c = points per lane, mode 0 = CV, 1 = GV, 2 = fixed span
ss_status_t launch_warp_opt_kernel(const EvalParams& p, int c, int mode, int64_t n_items, cudaStream_t stream);

// G-warps-per-eval kernels (ss_group_kernel.cuh); variant = group_variant_for_n(n)
ss_status_t launch_group_kernel(const EvalParams& p, int variant, int64_t n_items, cudaStream_t stream);

// the group kernels for a catalog with one shared time sampling (fp64, default options)
ss_status_t launch_group_shared_kernel(const EvalParams& p, int variant, int64_t n_items, cudaStream_t stream);

// the listing's options on the group path: variant = group_variant_for_n(n), mode 0 = CV, 1 = GV, 2 = fixed span
ss_status_t launch_group_opt_kernel(const EvalParams& p, int variant, int mode, int64_t n_items, cudaStream_t stream);

// cluster-per-eval kernels (ss_cluster_kernel.cuh); variant = cluster_variant_for_n(n); n_items clusters
ss_status_t launch_cluster_kernel(const EvalParams& p, int variant, int64_t n_items, cudaStream_t stream);

// CTA-per-eval kernels (ss_block_kernel.cuh): path = SS_PATH_BLOCK (threads = 128 / 256 / 512, per-eval arrays in
// shared memory sized for max_n) or SS_PATH_STAGE (512 threads, arrays in p.stage); opt = listing options compiled in
ss_status_t launch_block_kernel(const EvalParams& p, int path, int threads, int max_n, bool opt, int64_t n_items,
                                int sm_count, cudaStream_t stream);

// evals / whole work items the warp path handed over (p.defer_entries): recompute with the generic code, patch the
// periodogram and the item's partial-argmax slot (item entries) or fold into best_val / best_idx (eval entries)
ss_status_t launch_deferred_eval(const EvalParams& p, double* dval, unsigned long long* dmax, int max_n, bool opt,
                                 int sm_count, cudaStream_t stream);
ss_status_t launch_deferred_merge(const EvalParams& p, const double* dval, const unsigned long long* dmax,
                                  unsigned long long* dmin, double* best_val, int64_t* best_idx, int sm_count,
                                  cudaStream_t stream);

// ss_debug_eval: one eval by one 512-thread CTA, arrays in p.stage
ss_status_t launch_block_debug(const EvalParams& p, bool opt, double f, double* smo_out, int32_t* perm_out,
                               double* p_out, cudaStream_t stream);

}  // namespace ss

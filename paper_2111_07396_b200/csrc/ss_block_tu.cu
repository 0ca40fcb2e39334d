// ss_block_tu.cu -- instantiations and launchers of the CTA-per-eval kernels (ss_block_kernel.cuh), the kernels
// that recompute what the warp path hands over, and the dispatcher over the warp-kernel translation units.
// Compiled fourteen times by _build.py, -DSS_TU_PART=0..13, so the instantiations build in parallel:
//   part 0         dispatchers and the small hand-over kernels
//   part 1         the debug kernel
//   parts 2..9     one block_kernel<T, STAGE, OPT> each
//   parts 10..13   one deferred_eval_kernel<T, STAGE, OPT> each (what the warp / group / cluster paths hand over)
#include "ss_block_kernel.cuh"
#include "ss_launch.h"
#include "ss_planner.h"

#ifndef SS_TU_PART
#error "compile with -DSS_TU_PART=0..13"
#endif

namespace ss {

template <int T, bool STAGE, bool OPT>
ss_status_t launch_block_variant(const EvalParams& p, size_t smem, int grid, cudaStream_t stream);
template <int T, bool STAGE, bool OPT>
ss_status_t launch_deferred_variant(const EvalParams& p, double* dval, unsigned long long* dmax, size_t smem, int grid,
                                    cudaStream_t stream);

#if SS_TU_PART >= 10
// ---- what the warp path hands over: recomputed exactly by the generic CTA-per-eval code ------------------
// Entry formats (EvalParams::defer_entries):
//   eval  : record index << 32 | (k - k_begin)             one (object, frequency) pair (tied or misordered phases,
//                                                          a leave-one-out denominator <= 0)
//   item  : 1 << 63 | record index << 32 | chunk index     a whole work item (the object has duplicated time stamps:
//                                                          every one of its evals ties)

__device__ __forceinline__ unsigned long long sortable_bits(double v)
{
    if (v != v) return 0ull;      // NaN sorts below everything: it can never hide a valid maximum
    unsigned long long u = (unsigned long long)__double_as_longlong(v);
    return (u >> 63) ? ~u : (u | 0x8000000000000000ull);
}

// STAGE: per-eval arrays in this CTA's slot of the global staging scratch (light curves beyond the shared-memory limit)
template <int DEFER_T, bool STAGE, bool OPT>
__global__ void __launch_bounds__(DEFER_T) deferred_eval_kernel(const EvalParams p, double* dval,
                                                                unsigned long long* dmax)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NW = DEFER_T / 32;
    __shared__ double s_wsum[6][NW];
    __shared__ double s_red[NW];
    __shared__ int s_flags[4];
    BlockCtx<DEFER_T> cx;
    cx.wsum = s_wsum; cx.red = s_red; cx.flags = s_flags;
    double* S = STAGE ? p.stage + (int64_t)blockIdx.x * p.stage_stride : reinterpret_cast<double*>(smem_raw);
    const unsigned cnt = min(p.defer_count[0], p.defer_capacity);
    for (unsigned e = blockIdx.x; e < cnt; e += gridDim.x) {
        const unsigned long long ent = p.defer_entries[e];
        const int ri = (int)((ent & ~DEFER_ITEM) >> 32);
        const ObjRec rec = p.recs[ri];
        const int64_t sl = block_slot_len(rec.n);
        double* prow = p.pgram ? p.pgram + (rec.obj - p.pgram_row0) * p.pgram_row_stride - p.pgram_k0 : nullptr;
        if (ent & DEFER_ITEM) {
            const int ch = (int)(ent & 0xffffffffull);
            const int64_t k0 = p.k_begin + (int64_t)ch * p.chunk;
            const int64_t k1 = min(k0 + (int64_t)p.chunk, p.k_end);
            double best = -INFINITY;
            int64_t best_k = k0;
            for (int64_t k = k0; k < k1; k++) {
                __syncthreads();
                const double P = block_eval<DEFER_T, OPT>(p, rec, freq_of(p.f_min, p.df, k), S, sl, cx, nullptr, nullptr);
                if (threadIdx.x == 0) {
                    if (prow) prow[k] = P;
                    if (P > best) { best = P; best_k = k; }
                }
            }
            if (threadIdx.x == 0) {
                const int64_t slot = (int64_t)ri * p.chunks_total + p.chunk_base + ch;
                p.part_val[slot] = best;
                p.part_idx[slot] = best_k;
                dval[e] = nan("");
            }
            continue;
        }
        const int64_t k = p.k_begin + (int64_t)(ent & 0xffffffffull);
        __syncthreads();
        const double P = block_eval<DEFER_T, OPT>(p, rec, freq_of(p.f_min, p.df, k), S, sl, cx, nullptr, nullptr);
        if (threadIdx.x == 0) {
            if (prow) prow[k] = P;
            dval[e] = P;
            atomicMax(&dmax[rec.obj], sortable_bits(P));
        }
    }
}


template <int T, bool STAGE, bool OPT>
ss_status_t launch_deferred_variant(const EvalParams& p, double* dval, unsigned long long* dmax, size_t smem, int grid,
                                    cudaStream_t stream)
{
    auto kern = deferred_eval_kernel<T, STAGE, OPT>;
    if (smem > 0 && cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
        return SS_ERR_CUDA;
    kern<<<grid, T, smem, stream>>>(p, dval, dmax);
    return cudaGetLastError() == cudaSuccess ? SS_OK : SS_ERR_CUDA;
}
#if SS_TU_PART == 10
template ss_status_t launch_deferred_variant<128, false, false>(const EvalParams&, double*, unsigned long long*, size_t, int, cudaStream_t);
#elif SS_TU_PART == 11
template ss_status_t launch_deferred_variant<128, false, true>(const EvalParams&, double*, unsigned long long*, size_t, int, cudaStream_t);
#elif SS_TU_PART == 12
template ss_status_t launch_deferred_variant<512, true, false>(const EvalParams&, double*, unsigned long long*, size_t, int, cudaStream_t);
#else
template ss_status_t launch_deferred_variant<512, true, true>(const EvalParams&, double*, unsigned long long*, size_t, int, cudaStream_t);
#endif

#elif SS_TU_PART >= 2
template <int T, bool STAGE, bool OPT>
ss_status_t launch_block_variant(const EvalParams& p, size_t smem, int grid, cudaStream_t stream)
{
    auto kern = block_kernel<T, STAGE, OPT>;
    if (smem > 0 && cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
        return SS_ERR_CUDA;
    kern<<<grid, T, smem, stream>>>(p);
    return cudaGetLastError() == cudaSuccess ? SS_OK : SS_ERR_CUDA;
}
#if SS_TU_PART == 2
template ss_status_t launch_block_variant<128, false, false>(const EvalParams&, size_t, int, cudaStream_t);
#elif SS_TU_PART == 3
template ss_status_t launch_block_variant<128, false, true>(const EvalParams&, size_t, int, cudaStream_t);
#elif SS_TU_PART == 4
template ss_status_t launch_block_variant<256, false, false>(const EvalParams&, size_t, int, cudaStream_t);
#elif SS_TU_PART == 5
template ss_status_t launch_block_variant<256, false, true>(const EvalParams&, size_t, int, cudaStream_t);
#elif SS_TU_PART == 6
template ss_status_t launch_block_variant<512, false, false>(const EvalParams&, size_t, int, cudaStream_t);
#elif SS_TU_PART == 7
template ss_status_t launch_block_variant<512, false, true>(const EvalParams&, size_t, int, cudaStream_t);
#elif SS_TU_PART == 8
template ss_status_t launch_block_variant<512, true, false>(const EvalParams&, size_t, int, cudaStream_t);
#else
template ss_status_t launch_block_variant<512, true, true>(const EvalParams&, size_t, int, cudaStream_t);
#endif

#elif SS_TU_PART == 1
ss_status_t launch_block_debug(const EvalParams& p, bool opt, double f, double* smo_out, int32_t* perm_out,
                               double* p_out, cudaStream_t stream)
{
    if (opt) block_debug_kernel<512, true><<<1, 512, 0, stream>>>(p, f, smo_out, perm_out, p_out);
    else block_debug_kernel<512, false><<<1, 512, 0, stream>>>(p, f, smo_out, perm_out, p_out);
    return cudaGetLastError() == cudaSuccess ? SS_OK : SS_ERR_CUDA;
}

#else   // part 0

// ---- warp-kernel translation units (ss_warp_tu.cu) -------------------------------------------------
#define SS_DECL(gv, g) ss_status_t launch_warp_tu_##gv##_##g(const EvalParams&, int, int64_t, cudaStream_t);
SS_DECL(0, 0) SS_DECL(0, 1) SS_DECL(0, 2) SS_DECL(1, 0) SS_DECL(1, 1) SS_DECL(1, 2)
#undef SS_DECL

#define SS_DECL(gv, g) ss_status_t launch_warp_f32_tu_##gv##_##g(const EvalParams&, int, int64_t, cudaStream_t);
SS_DECL(0, 0) SS_DECL(0, 1) SS_DECL(0, 2) SS_DECL(1, 0) SS_DECL(1, 1) SS_DECL(1, 2)
#undef SS_DECL

ss_status_t launch_warp_kernel(const EvalParams& p, int variant, int64_t n_items, cudaStream_t stream)
{
    const bool f32 = variant >= WARP_VARIANT_F32;
    if (f32) variant -= WARP_VARIANT_F32;
    const int c = variant / 8, g = c <= 4 ? 0 : (c <= 6 ? 1 : 2);
    if (f32) {
        if (p.mode == 1)
            return g == 0 ? launch_warp_f32_tu_1_0(p, variant, n_items, stream)
                 : g == 1 ? launch_warp_f32_tu_1_1(p, variant, n_items, stream) : launch_warp_f32_tu_1_2(p, variant, n_items, stream);
        return g == 0 ? launch_warp_f32_tu_0_0(p, variant, n_items, stream)
             : g == 1 ? launch_warp_f32_tu_0_1(p, variant, n_items, stream) : launch_warp_f32_tu_0_2(p, variant, n_items, stream);
    }
    if (p.mode == 1)
        return g == 0 ? launch_warp_tu_1_0(p, variant, n_items, stream)
             : g == 1 ? launch_warp_tu_1_1(p, variant, n_items, stream) : launch_warp_tu_1_2(p, variant, n_items, stream);
    return g == 0 ? launch_warp_tu_0_0(p, variant, n_items, stream)
         : g == 1 ? launch_warp_tu_0_1(p, variant, n_items, stream) : launch_warp_tu_0_2(p, variant, n_items, stream);
}

#define SS_DECL(gv, g) ss_status_t launch_warp_shared_tu_##gv##_##g(const EvalParams&, int, int64_t, cudaStream_t);
SS_DECL(0, 0) SS_DECL(0, 1) SS_DECL(0, 2) SS_DECL(1, 0) SS_DECL(1, 1) SS_DECL(1, 2)
#undef SS_DECL

ss_status_t launch_warp_shared_kernel(const EvalParams& p, int variant, int64_t n_items, cudaStream_t stream)
{
    const int c = variant / 8, g = c <= 4 ? 0 : (c <= 6 ? 1 : 2);
    if (p.mode == 1)
        return g == 0 ? launch_warp_shared_tu_1_0(p, variant, n_items, stream)
             : g == 1 ? launch_warp_shared_tu_1_1(p, variant, n_items, stream) : launch_warp_shared_tu_1_2(p, variant, n_items, stream);
    return g == 0 ? launch_warp_shared_tu_0_0(p, variant, n_items, stream)
         : g == 1 ? launch_warp_shared_tu_0_1(p, variant, n_items, stream) : launch_warp_shared_tu_0_2(p, variant, n_items, stream);
}

#define SS_DECL(gv, g) ss_status_t launch_warp_opt_tu_##gv##_##g(const EvalParams&, int, int, int64_t, cudaStream_t);
SS_DECL(0, 0) SS_DECL(0, 1) SS_DECL(0, 2) SS_DECL(1, 0) SS_DECL(1, 1) SS_DECL(1, 2)
#undef SS_DECL

ss_status_t launch_warp_opt_kernel(const EvalParams& p, int c, int mode, int64_t n_items, cudaStream_t stream)
{
    const int g = c <= 4 ? 0 : (c <= 6 ? 1 : 2);
    if (mode == 1)
        return g == 0 ? launch_warp_opt_tu_1_0(p, c, mode, n_items, stream)
             : g == 1 ? launch_warp_opt_tu_1_1(p, c, mode, n_items, stream) : launch_warp_opt_tu_1_2(p, c, mode, n_items, stream);
    return g == 0 ? launch_warp_opt_tu_0_0(p, c, mode, n_items, stream)
         : g == 1 ? launch_warp_opt_tu_0_1(p, c, mode, n_items, stream) : launch_warp_opt_tu_0_2(p, c, mode, n_items, stream);
}

// ---- group-kernel translation units (ss_group_tu.cu) -------------------------------------------------
#define SS_DECL(gv, g) ss_status_t launch_group_tu_##gv##_##g(const EvalParams&, int, int64_t, cudaStream_t);
SS_DECL(0, 4) SS_DECL(0, 8) SS_DECL(0, 16) SS_DECL(1, 4) SS_DECL(1, 8) SS_DECL(1, 16)
#undef SS_DECL
#define SS_DECL(gv, g) ss_status_t launch_group_f32_tu_##gv##_##g(const EvalParams&, int, int64_t, cudaStream_t);
SS_DECL(0, 4) SS_DECL(0, 8) SS_DECL(0, 16) SS_DECL(1, 4) SS_DECL(1, 8) SS_DECL(1, 16)
#undef SS_DECL

#define SS_DECL(gv, g) ss_status_t launch_group_opt_tu_##gv##_##g(const EvalParams&, int, int, int64_t, cudaStream_t);
SS_DECL(0, 4) SS_DECL(0, 8) SS_DECL(0, 16) SS_DECL(1, 4) SS_DECL(1, 8) SS_DECL(1, 16)
#undef SS_DECL

#define SS_DECL(gv, g) ss_status_t launch_group_shared_tu_##gv##_##g(const EvalParams&, int, int64_t, cudaStream_t);
SS_DECL(0, 4) SS_DECL(0, 8) SS_DECL(0, 16) SS_DECL(1, 4) SS_DECL(1, 8) SS_DECL(1, 16)
#undef SS_DECL

// one shared time sampling: n_items = groups of SHARED_TIMES_M objects x chunks; variant = group_variant_for_n(n)
ss_status_t launch_group_shared_kernel(const EvalParams& p, int variant, int64_t n_items, cudaStream_t stream)
{
    const int g = variant / 8, c = variant % 8;
    if (p.mode == 1)
        return g == 4 ? launch_group_shared_tu_1_4(p, c, n_items, stream)
             : g == 8 ? launch_group_shared_tu_1_8(p, c, n_items, stream) : launch_group_shared_tu_1_16(p, c, n_items, stream);
    return g == 4 ? launch_group_shared_tu_0_4(p, c, n_items, stream)
         : g == 8 ? launch_group_shared_tu_0_8(p, c, n_items, stream) : launch_group_shared_tu_0_16(p, c, n_items, stream);
}

// mode: 0 = CV, 1 = GV, 2 = fixed span (the listing's options; variant = group_variant_for_n(n))
ss_status_t launch_group_opt_kernel(const EvalParams& p, int variant, int mode, int64_t n_items, cudaStream_t stream)
{
    const int g = variant / 8, c = variant % 8;
    if (mode == 1)
        return g == 4 ? launch_group_opt_tu_1_4(p, c, mode, n_items, stream)
             : g == 8 ? launch_group_opt_tu_1_8(p, c, mode, n_items, stream) : launch_group_opt_tu_1_16(p, c, mode, n_items, stream);
    return g == 4 ? launch_group_opt_tu_0_4(p, c, mode, n_items, stream)
         : g == 8 ? launch_group_opt_tu_0_8(p, c, mode, n_items, stream) : launch_group_opt_tu_0_16(p, c, mode, n_items, stream);
}

ss_status_t launch_group_kernel(const EvalParams& p, int variant, int64_t n_items, cudaStream_t stream)
{
    const bool f32 = variant >= GROUP_VARIANT_F32;
    if (f32) variant -= GROUP_VARIANT_F32;
    const int g = variant / 8, c = variant % 8;
    if (f32) {
        if (p.mode == 1)
            return g == 4 ? launch_group_f32_tu_1_4(p, c, n_items, stream)
                 : g == 8 ? launch_group_f32_tu_1_8(p, c, n_items, stream) : launch_group_f32_tu_1_16(p, c, n_items, stream);
        return g == 4 ? launch_group_f32_tu_0_4(p, c, n_items, stream)
             : g == 8 ? launch_group_f32_tu_0_8(p, c, n_items, stream) : launch_group_f32_tu_0_16(p, c, n_items, stream);
    }
    if (p.mode == 1)
        return g == 4 ? launch_group_tu_1_4(p, c, n_items, stream)
             : g == 8 ? launch_group_tu_1_8(p, c, n_items, stream) : launch_group_tu_1_16(p, c, n_items, stream);
    return g == 4 ? launch_group_tu_0_4(p, c, n_items, stream)
         : g == 8 ? launch_group_tu_0_8(p, c, n_items, stream) : launch_group_tu_0_16(p, c, n_items, stream);
}

// ---- cluster-kernel translation units (ss_cluster_tu.cu) -----------------------------------------------
#define SS_DECL(gv, c) ss_status_t launch_cluster_tu_##gv##_##c(const EvalParams&, int, int64_t, cudaStream_t);
SS_DECL(0, 3) SS_DECL(0, 4) SS_DECL(0, 5) SS_DECL(1, 3) SS_DECL(1, 4) SS_DECL(1, 5)
#undef SS_DECL

ss_status_t launch_cluster_kernel(const EvalParams& p, int variant, int64_t n_items, cudaStream_t stream)
{
    const int r = variant / 8, c = variant % 8;
    if (p.mode == 1)
        return c == 3 ? launch_cluster_tu_1_3(p, r, n_items, stream)
             : c == 4 ? launch_cluster_tu_1_4(p, r, n_items, stream) : launch_cluster_tu_1_5(p, r, n_items, stream);
    return c == 3 ? launch_cluster_tu_0_3(p, r, n_items, stream)
         : c == 4 ? launch_cluster_tu_0_4(p, r, n_items, stream) : launch_cluster_tu_0_5(p, r, n_items, stream);
}

// ---- CTA-per-eval kernels ---------------------------------------------------------------------------
ss_status_t launch_block_kernel(const EvalParams& p, int path, int threads, int max_n, bool opt, int64_t n_items,
                                int sm_count, cudaStream_t stream)
{
    auto grid_of = [&](int per_sm) { return (int)(n_items < (int64_t)sm_count * per_sm ? n_items : (int64_t)sm_count * per_sm); };
    if (path == SS_PATH_STAGE)
        return opt ? launch_block_variant<512, true, true>(p, 0, grid_of(2), stream)
                   : launch_block_variant<512, true, false>(p, 0, grid_of(2), stream);
    const size_t smem = (size_t)BLOCK_SLOTS * (size_t)block_slot_len(max_n) * 8;
    if (threads == 512)
        return opt ? launch_block_variant<512, false, true>(p, smem, grid_of(1), stream)
                   : launch_block_variant<512, false, false>(p, smem, grid_of(1), stream);
    if (threads == 128)
        return opt ? launch_block_variant<128, false, true>(p, smem, grid_of(4), stream)
                   : launch_block_variant<128, false, false>(p, smem, grid_of(4), stream);
    return opt ? launch_block_variant<256, false, true>(p, smem, grid_of(2), stream)
               : launch_block_variant<256, false, false>(p, smem, grid_of(2), stream);
}

// (the hand-over eval kernels are instantiated in parts 10..13)
__device__ __forceinline__ unsigned long long sortable_bits(double v)
{
    if (v != v) return 0ull;      // NaN sorts below everything: it can never hide a valid maximum
    unsigned long long u = (unsigned long long)__double_as_longlong(v);
    return (u >> 63) ? ~u : (u | 0x8000000000000000ull);
}
__global__ void deferred_min_kernel(const EvalParams p, const double* dval, const unsigned long long* dmax,
                                    unsigned long long* dmin)
{
    const unsigned cnt = min(p.defer_count[0], p.defer_capacity);
    for (unsigned e = blockIdx.x * blockDim.x + threadIdx.x; e < cnt; e += gridDim.x * blockDim.x) {
        const unsigned long long ent = p.defer_entries[e];
        if (ent & DEFER_ITEM) continue;
        const int64_t obj = p.recs[(int)(ent >> 32)].obj;
        const unsigned long long b = sortable_bits(dval[e]);
        if (b != 0ull && b == dmax[obj]) atomicMin(&dmin[obj], (unsigned long long)(p.k_begin + (int64_t)(ent & 0xffffffffull)));
    }
}

__global__ void deferred_merge_kernel(const EvalParams p, const double* dval, const unsigned long long* dmax,
                                      const unsigned long long* dmin, double* best_val, int64_t* best_idx)
{
    const unsigned cnt = min(p.defer_count[0], p.defer_capacity);
    for (unsigned e = blockIdx.x * blockDim.x + threadIdx.x; e < cnt; e += gridDim.x * blockDim.x) {
        const unsigned long long ent = p.defer_entries[e];
        if (ent & DEFER_ITEM) continue;
        const int64_t obj = p.recs[(int)(ent >> 32)].obj;
        const int64_t k = p.k_begin + (int64_t)(ent & 0xffffffffull);
        const double v = dval[e];
        const unsigned long long b = sortable_bits(v);
        // the unique winner among this object's deferred evals folds itself into the running best
        if (b != 0ull && b == dmax[obj] && (unsigned long long)k == dmin[obj]) {
            const double cv = best_val[obj];
            const int64_t ck = best_idx[obj];
            if (ck < 0 || v > cv || (v == cv && k < ck)) { best_val[obj] = v; best_idx[obj] = k; }
        }
    }
}

ss_status_t launch_deferred_eval(const EvalParams& p, double* dval, unsigned long long* dmax, int max_n, bool opt,
                                 int sm_count, cudaStream_t stream)
{
    if (max_n > BLOCK_MAX_N)      // the staging scratch holds 2 slots per SM (Engine::setup)
        return opt ? launch_deferred_variant<512, true, true>(p, dval, dmax, 0, sm_count * 2, stream)
                   : launch_deferred_variant<512, true, false>(p, dval, dmax, 0, sm_count * 2, stream);
    const size_t smem = (size_t)BLOCK_SLOTS * (size_t)block_slot_len(max_n) * 8;
    return opt ? launch_deferred_variant<128, false, true>(p, dval, dmax, smem, sm_count * 4, stream)
               : launch_deferred_variant<128, false, false>(p, dval, dmax, smem, sm_count * 4, stream);
}

ss_status_t launch_deferred_merge(const EvalParams& p, const double* dval, const unsigned long long* dmax,
                                  unsigned long long* dmin, double* best_val, int64_t* best_idx, int sm_count,
                                  cudaStream_t stream)
{
    deferred_min_kernel<<<sm_count, 256, 0, stream>>>(p, dval, dmax, dmin);
    deferred_merge_kernel<<<sm_count, 256, 0, stream>>>(p, dval, dmax, dmin, best_val, best_idx);
    return cudaGetLastError() == cudaSuccess ? SS_OK : SS_ERR_CUDA;
}

#endif   // SS_TU_PART

}  // namespace ss

// ss_warp_shared.cuh -- warp-per-eval kernel for catalogs whose objects share ONE time sampling
// (ss_options_t::shared_times; "it would be possible to reuse the same folded time intervals for all
// objects" -- the fields of a survey camera are observed together).
//
// The phase fold and the sort depend on the times and the frequency only, so a warp does them ONCE per frequency for a
// group of SHARED_M objects and then runs the smoother (warp_eval_body of ss_warp_kernel.cuh, unchanged) once per
// object on that permutation: per eval the keys, the sorting network, the gather of the times, the exact-order check
// and the quartile broadcast are paid 1/SHARED_M times.  Values, hand-over rules and outputs are those of warp_kernel.
#pragma once
#include "ss_warp_kernel.cuh"

namespace ss {

constexpr int SHARED_M = SHARED_TIMES_M;      // objects per work item (ss_planner.h: the host sizes the grid with it)

template <int C, bool GV>
inline size_t warp_shared_smem_bytes()
{
    constexpr int WPC = WarpCfg<C, GV>::WPC;
    // tt + SHARED_M x (yc, w) + per warp: 3 pair-prefix arrays + the P stash of SHARED_M x 32 values
    return (size_t)(1 + 2 * SHARED_M) * 32 * C * 8 + (size_t)WPC * ((size_t)3 * C * WROW * 16 + (size_t)SHARED_M * 32 * 8);
}

template <int C, int IBW0, bool GV>
__global__ void __launch_bounds__(WarpCfg<C, GV>::WPC * 32, WarpCfg<C, GV>::MINB) warp_shared_kernel(const EvalParams p)
{
    constexpr int WPC = WarpCfg<C, GV>::WPC;
    constexpr int M_ = SHARED_M;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double s_best[WPC][M_];
    __shared__ long long s_bestk[WPC][M_];
    __shared__ double s_kc[M_][6];
    __shared__ double* s_prow[M_];
    __shared__ int s_ri[M_];
    __shared__ uint32_t s_tmem;
    constexpr uint32_t TCOLS_WARP = GV ? 4 * C : 18 * C;
    constexpr uint32_t TCOLS_NEED = TCOLS_WARP * ((WPC + 3) / 4);
    constexpr uint32_t TCOLS = TCOLS_NEED <= 32 ? 32 : (TCOLS_NEED <= 64 ? 64 : (TCOLS_NEED <= 128 ? 128 : (TCOLS_NEED <= 256 ? 256 : 512)));
    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
    const int item = blockIdx.x;
    const int g = item / p.chunks_per_obj, ch = item - g * p.chunks_per_obj;
    const int li0 = g * M_;
    const int mc = min(M_, p.n_list - li0);                 // objects in this group
    const ObjRec rec0 = p.recs[p.list[li0]];
    if (rec0.dup) {
        // duplicated time stamps (shared by every object): the generic kernel takes the work items whole
        if (tid < mc) {
            const unsigned pos = atomicAdd(p.defer_count, 1u);
            if (pos < p.defer_capacity)
                p.defer_entries[pos] = DEFER_ITEM | ((unsigned long long)p.list[li0 + tid] << 32) | (unsigned long long)ch;
            else
                p.defer_count[1] = 1u;
        }
        return;
    }
    const int n = uni(rec0.n);

    EvalConst K;
    K.n = n; K.ibw1 = uni(rec0.ibw[1]); K.ibw2 = uni(rec0.ibw[2]);
    K.K1 = min(2 * K.ibw1 + 1, n); K.K2 = min(2 * K.ibw2 + 1, n);
    {
        const int jr = n - 1 - IBW0;
        K.lane_r = jr / C; K.slot_r = jr % C;
        const int q1 = uni(rec0.q1), q3 = uni(rec0.q3);
        K.q1l = q1 / C; K.q1s = q1 % C; K.q3l = q3 / C; K.q3s = q3 % C;
    }
    K.alpha = p.alpha; K.bexp = 10.0 - p.alpha;
    K.bass = (p.alpha > 0.0 && p.alpha <= 10.0) ? (K.bexp == 1.0 ? 1 : 2) : 0;

    double* o_tt = reinterpret_cast<double*>(smem_raw);
    double* o_y = o_tt + 32 * C;                             // [M_][32C]
    double* o_w = o_y + M_ * 32 * C;                         // [M_][32C]
    constexpr size_t WARP_BYTES = (size_t)3 * C * WROW * 16 + (size_t)M_ * 32 * 8;
    unsigned char* wbase = smem_raw + (size_t)(1 + 2 * M_) * 32 * C * 8 + (size_t)warp * WARP_BYTES;
    double* stash = reinterpret_cast<double*>(wbase + (size_t)3 * C * WROW * 16);      // [M_][32]
    WarpMem M;
    M.tt = o_tt; M.yc = o_y; M.w = o_w;
    M.E = reinterpret_cast<double2*>(wbase);
    M.tmem = 0;
    M.mk = make_scan_mask(lane);
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                     :: "r"((uint32_t)__cvta_generic_to_shared(&s_tmem)), "n"(TCOLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    if (tid < M_) {
        const int m = tid;
        const ObjRec r = p.recs[p.list[li0 + (m < mc ? m : 0)]];
        s_ri[m] = p.list[li0 + (m < mc ? m : 0)];
        s_kc[m][0] = 1.0 / (1.0 - 1.0 / (double)K.K1); s_kc[m][1] = 1.0 / (1.0 - 2.0 / (double)K.K1);
        s_kc[m][2] = 1.0 / (1.0 - 1.0 / (double)K.K2); s_kc[m][3] = 1.0 / (1.0 - 2.0 / (double)K.K2);
        s_kc[m][4] = r.chi0; s_kc[m][5] = r.chi0 > 0.0 ? 1.0 / r.chi0 : 0.0;
        s_prow[m] = p.pgram ? p.pgram + (r.obj - p.pgram_row0) * p.pgram_row_stride - p.pgram_k0 : nullptr;
    }
    for (int j = tid; j < n; j += WPC * 32) o_tt[j] = p.tt[rec0.off + j];
    for (int m = 0; m < mc; m++) {
        const int64_t off = p.recs[p.list[li0 + m]].off;
        for (int j = tid; j < n; j += WPC * 32) {
            o_y[m * 32 * C + j] = p.yc[off + j];
            o_w[m * 32 * C + j] = p.w[off + j];
        }
    }
    if (tid < WPC * M_) { s_best[tid / M_][tid % M_] = -INFINITY; s_bestk[tid / M_][tid % M_] = INT64_MAX; }
    __syncthreads();
    {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        M.tmem = s_tmem + ((uint32_t)(warp & 3) << 21) + (uint32_t)(warp >> 2) * TCOLS_WARP;
        int w1[2 * C], w2[2 * C];
#pragma unroll
        for (int s = 0; s < C; s++) {
            const int lo1 = window_lo(lane * C + s, K.ibw1, K.K1, n), lo2 = window_lo(lane * C + s, K.ibw2, K.K2, n);
            w1[s] = wst<C>(lo1); w1[C + s] = wst<C>(lo1 + K.K1);
            w2[s] = wst<C>(lo2); w2[C + s] = wst<C>(lo2 + K.K2);
        }
        tmem_park_words<2 * C>(M.tmem + (GV ? 0 : 14 * C), w1);
        tmem_park_words<2 * C>(M.tmem + (GV ? 2 * C : 16 * C), w2);
        tmem_wait_st();
    }

    const int64_t c0 = p.k_begin + (int64_t)ch * p.chunk;
    const int64_t c1 = min(c0 + (int64_t)p.chunk, p.k_end);
    const int per_warp = p.chunk / WPC;
    const int64_t k0 = c0 + (int64_t)warp * per_warp;
    const int64_t k1 = min(k0 + (int64_t)per_warp, c1);
    int64_t kb = k0;
    auto hand_over = [&](int m, int64_t k) {
        if (lane == 0) {
            const unsigned pos = atomicAdd(p.defer_count, 1u);
            if (pos < p.defer_capacity)
                p.defer_entries[pos] = ((unsigned long long)s_ri[m] << 32) | (unsigned long long)(k - p.k_begin);
            else
                p.defer_count[1] = 1u;
        }
    };
    for (int64_t k = k0; k < k1; k++) {
        const double f = freq_of(p.f_min, p.df, k);
        // ---- P1 fold, P2 sort, exact phases and order check: once for the whole group
        constexpr int S = Pow2Ceil<C>::value;
        constexpr int SK = (S == C) ? S : C;
        unsigned key[SK];
#pragma unroll
        for (int s = 0; s < SK; s++) {
            const int i = lane + 32 * s;
            unsigned kk = 0xffffffffu;
            if (i < n) kk = (__double2uint_rz(fold_phase(o_tt[i], f) * 16777216.0) << 8) | (unsigned)i;
            key[s] = kk;
        }
        if constexpr (S == C) warp_sort<S>(key, lane);
        else warp_sort_any<C>(key, lane);
        int idx[C];
        double x[C];
        bool bad = false;
        double vsmlsq;
        {
            double phi[C];
#pragma unroll
            for (int s = 0; s < C; s++) {
                idx[s] = (int)(key[s] & 0xffu);
                phi[s] = (lane * C + s < n) ? fold_phase(o_tt[idx[s]], f) : 4.0;
            }
            double nxt = shfl_down_d(phi[0], 1);
            if (lane == 31) nxt = 8.0;
#pragma unroll
            for (int s = 0; s < C; s++) {
                const double nx = s + 1 < C ? phi[s + 1 < C ? s + 1 : 0] : nxt;
                if (lane * C + s + 1 < n && nx <= phi[s]) bad = true;
            }
            const double p1 = bcast_slot<C>(phi, K.q1s, K.q1l);
            const double p3 = bcast_slot<C>(phi, K.q3s, K.q3l);
            const double scale = p3 - p1;
            vsmlsq = 1.e-6 * scale * scale;
#pragma unroll
            for (int s = 0; s < C; s++) x[s] = (lane * C + s < n) ? phi[s] - 0.5 : 0.0;
        }
        const bool tied = __any_sync(0xffffffffu, bad);
#pragma unroll 1
        for (int m = 0; m < mc; m++) {
            double P = 0.0;
            bool defer = tied;
            if (!tied) {
                double y[C], w[C];
#pragma unroll
                for (int s = 0; s < C; s++) {
                    const bool real = lane * C + s < n;
                    y[s] = real ? o_y[m * 32 * C + idx[s]] : 0.0;
                    w[s] = real ? o_w[m * 32 * C + idx[s]] : W_PAD;
                }
                K.kc = s_kc[m];
                P = warp_eval_body<C, IBW0, GV, double>(K, M, x, y, w, vsmlsq, lane, defer);
                __syncwarp();      // every lane is done with the prefix arrays before the next object overwrites them
            }
            if (defer) { hand_over(m, k); P = 0.0; }
            if (lane == 0) {
                stash[m * 32 + (int)(k - kb)] = P;
                if (!defer && P > s_best[warp][m]) { s_best[warp][m] = P; s_bestk[warp][m] = k; }
            }
        }
        if (k - kb == 31 || k == k1 - 1) {
            __syncwarp();
            for (int m = 0; m < mc; m++) {
                double* prow = s_prow[m];
                if (prow && kb + lane <= k) prow[kb + lane] = stash[m * 32 + lane];
            }
            __syncwarp();
            kb = k + 1;
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(s_tmem), "n"(TCOLS) : "memory");
    }
    if (tid < mc) {
        const int m = tid;
        double best = s_best[0][m];
        long long best_k = s_bestk[0][m];
        for (int q = 1; q < WPC; q++)
            if (s_best[q][m] > best || (s_best[q][m] == best && s_bestk[q][m] < best_k)) { best = s_best[q][m]; best_k = s_bestk[q][m]; }
        const int64_t slot = (int64_t)s_ri[m] * p.chunks_total + p.chunk_base + ch;
        p.part_val[slot] = best;
        p.part_idx[slot] = best_k == INT64_MAX ? c0 : best_k;
    }
}

template <int C, int IBW0, bool GV>
inline ss_status_t launch_warp_shared_variant(const EvalParams& p, int64_t n_items, cudaStream_t stream)
{
    const size_t smem = warp_shared_smem_bytes<C, GV>();
    if (cudaFuncSetAttribute(warp_shared_kernel<C, IBW0, GV>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
        return SS_ERR_CUDA;
    warp_shared_kernel<C, IBW0, GV><<<(unsigned)n_items, WarpCfg<C, GV>::WPC * 32, smem, stream>>>(p);
    return cudaGetLastError() == cudaSuccess ? SS_OK : SS_ERR_CUDA;
}

}  // namespace ss

// ss_cluster_kernel.cuh -- one thread-block CLUSTER per (object, frequency) eval, 2,055 < n <= 40,960
// (SS_PATH_CLUSTER).
//
// The group design (ss_group_kernel.cuh) spread over R = 2, 4, 8 or 16 CTAs of 16 warps: CTA r of the cluster owns the
// phase-ordered points [r*512*C, (r+1)*512*C), each thread C consecutive ones in registers, and the per-eval prefix
// arrays live in the shared memory of the CTA that owns the positions -- R x 123 KB of distributed shared memory
// instead of a global scratch slot per eval.  What crosses CTA boundaries:
//   * the sort: 64-bit keys (48 phase bits | 16 index bits -- with up to 40,960 points a 32-bit key would not leave
//     enough phase bits), CTA-local blocked bitonic network, then log2(R)(log2(R)+1)/2 cross-CTA exchange steps in
//     which every thread reads its partner's keys straight out of the partner CTA's shared memory (ld.shared::cluster),
//     one cluster barrier per step;
//   * one carry exchange per prefix scan (the CTA totals, a few doubles per CTA, through a small mailbox);
//   * the window ends: a window of the midrange / woofer span reaches up to n/4 positions away, i.e. into other CTAs;
//     the loop-invariant (CTA rank, address) of every window end is parked in tensor memory and each access is one
//     mapa + ld.shared::cluster.v2.f64;
//   * the chi2 partial sums.
// Evals this path cannot decide exactly (tied phases, phases that agree in 48 bits, a leave-one-out denominator <= 0)
// go to the generic kernel's global-staging variant through the hand-over list.
#pragma once
#include "ss_group_kernel.cuh"

namespace ss {

constexpr int CL_G = 16, CL_NT = 32 * CL_G;           // warps / threads per CTA
constexpr int CL_IDX_BITS = 16;

__device__ __forceinline__ uint32_t cluster_ctarank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t mapa_u32(uint32_t saddr, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
    return r;
}
__device__ __forceinline__ double2 ld_cl_d2(uint32_t caddr)
{
    double2 v;
    asm volatile("ld.shared::cluster.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(caddr) : "memory");
    return v;
}
__device__ __forceinline__ double ld_cl_d(uint32_t caddr)
{
    double v;
    asm volatile("ld.shared::cluster.f64 %0, [%1];" : "=d"(v) : "r"(caddr) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long ld_cl_u64(uint32_t caddr)
{
    unsigned long long v;
    asm volatile("ld.shared::cluster.u64 %0, [%1];" : "=l"(v) : "r"(caddr) : "memory");
    return v;
}
__device__ __forceinline__ int ld_cl_s32(uint32_t caddr)
{
    int v;
    asm volatile("ld.shared::cluster.s32 %0, [%1];" : "=r"(v) : "r"(caddr) : "memory");
    return v;
}

// what a CTA publishes to the other CTAs of its cluster (read after a cluster barrier)
struct __align__(16) ClusterMail {
    double2 tot[3];        // CTA totals of up to three pair scans
    double first, last;    // exact phases of the first / last position of this CTA's slice
    double q[2];           // phases of the quartile points (valid in the CTA that owns them)
    double chi2;           // partial chi2
    int bad;               // this CTA saw a tie / misorder / leave-one-out denominator <= 0
    int pad;
};

typedef unsigned long long key64;

// One side of a compare-exchange on 64-bit keys: the lower position keeps the smaller key.  Keys are distinct (the index
// bits; all-ones padding keys are equal but then either choice is the same value), so "take the partner's" is
// (other < mine) for the lower position and its negation for the upper one: one 64-bit compare and one select instead
// of a min, a max and a select between them.
__device__ __forceinline__ key64 cex_side64(key64 mine, key64 other, bool lower)
{
    const bool lt = other < mine;
    return (lt == lower) ? other : mine;
}

// odd-even transposition network on C keys (C rounds): the lane-local sort for 64-bit keys
template <int C>
__device__ __forceinline__ void local_sort64(key64 (&k)[C])
{
#pragma unroll
    for (int r = 0; r < C; r++) {
#pragma unroll
        for (int s = r & 1; s + 1 < C; s += 2) {
            const bool lt = k[s + 1] < k[s];
            const key64 lo = lt ? k[s + 1] : k[s], hi = lt ? k[s] : k[s + 1];
            k[s] = lo; k[s + 1] = hi;
        }
    }
}

// one compare-exchange step of the blocked network against thread (tid ^ mask) of this CTA
template <int C, bool REV>
__device__ __forceinline__ void cta_step64(key64 (&key)[C], int mask, bool lower, int tid, key64* kb)
{
    key64 other[C];
    if (mask < 32) {
#pragma unroll
        for (int s = 0; s < C; s++) other[s] = __shfl_xor_sync(0xffffffffu, key[REV ? C - 1 - s : s], mask);
    } else {
#pragma unroll
        for (int s = 0; s < C; s++) kb[s * CL_NT + tid] = key[s];
        __syncthreads();
        const int pt = tid ^ mask;
#pragma unroll
        for (int s = 0; s < C; s++) other[s] = kb[(REV ? C - 1 - s : s) * CL_NT + pt];
    }
#pragma unroll
    for (int s = 0; s < C; s++) key[s] = cex_side64(key[s], other[s], lower);
}

// the half-cleaners at thread strides 256 .. 1 inside the CTA, then the lane-local network
template <int C>
__device__ __forceinline__ void cta_merge_tail64(key64 (&key)[C], int tid, key64* ia, key64* ib, int& flip)
{
#pragma unroll
    for (int m = CL_NT >> 1; m >= 1; m >>= 1) {
        cta_step64<C, false>(key, m, (tid & m) == 0, tid, flip ? ib : ia);
        if (m >= 32) flip ^= 1;
    }
    local_sort64<C>(key);
}

// ------------------------------------------------------------------------------------------------
// Kernel: one cluster = one work item (object, chunk of frequencies).
// ------------------------------------------------------------------------------------------------
template <int C>
inline size_t cluster_smem_bytes()
{
    return (size_t)3 * C * (CL_NT + 1) * 16;       // three pair-prefix arrays; the sort's exchange buffers overlay them
}

template <int C, bool GV>
__global__ void __launch_bounds__(CL_NT, 1) cluster_kernel(const EvalParams p, const int R)
{
    constexpr int G = CL_G, NT = CL_NT, ROW = NT + 1, ASZ = C * ROW;
    constexpr uint32_t TCOLS_WARP = 20 * C;
    constexpr uint32_t TCOLS_NEED = TCOLS_WARP * (G / 4);
    constexpr uint32_t TCOLS = TCOLS_NEED <= 256 ? 256 : 512;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ __align__(16) double2 s_tot[3][G];
    __shared__ __align__(16) ClusterMail s_mail;
    __shared__ __align__(16) double2 s_carry[3];
    __shared__ double s_red[G];
    __shared__ double s_wfirst[G], s_wlast[G];
    __shared__ double s_vs;          // vsmlsq of this eval
    __shared__ int s_anybad;
    __shared__ double s_kc[8];
    __shared__ uint32_t s_tmem;

    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
    const int rank = (int)cluster_ctarank();
    const int item = blockIdx.x / R;
    const int li = item / p.chunks_per_obj, ch = item - li * p.chunks_per_obj;
    const int ri = p.list[li];
    const ObjRec rec = p.recs[ri];
    const int n = rec.n;
    const int gt = rank * NT + tid;                 // thread index over the cluster
    const int NTT = R * NT;                         // threads of the cluster

    double2* E01 = reinterpret_cast<double2*>(smem_raw);
    double2* E23 = E01 + ASZ;
    double2* E45 = E23 + ASZ;
    key64* IA = reinterpret_cast<key64*>(E01);      // intra-CTA exchange buffers (2 x NT*C keys inside E01)
    key64* IB = IA + NT * C;
    key64* XA = reinterpret_cast<key64*>(E23);      // cross-CTA exchange buffers (inside E23)
    key64* XB = XA + NT * C;
    const uint32_t a_E01 = smem_u32(E01), a_E23 = smem_u32(E23), a_E45 = smem_u32(E45);
    const uint32_t a_XA = smem_u32(XA), a_XB = smem_u32(XB), a_mail = smem_u32(&s_mail);

    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                     :: "r"(smem_u32(&s_tmem)), "n"(TCOLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");

    const int ibw0 = rec.ibw[0], ibw1 = rec.ibw[1], ibw2 = rec.ibw[2];
    const int K0 = min(2 * ibw0 + 1, n), K1 = min(2 * ibw1 + 1, n), K2 = min(2 * ibw2 + 1, n);
    if (tid == 0) {
        s_kc[0] = 1.0 / (1.0 - 1.0 / (double)K0); s_kc[1] = 1.0 / (1.0 - 2.0 / (double)K0);
        s_kc[2] = 1.0 / (1.0 - 1.0 / (double)K1); s_kc[3] = 1.0 / (1.0 - 2.0 / (double)K1);
        s_kc[4] = 1.0 / (1.0 - 1.0 / (double)K2); s_kc[5] = 1.0 / (1.0 - 2.0 / (double)K2);
        s_kc[6] = rec.chi0; s_kc[7] = rec.chi0 > 0.0 ? 1.0 / rec.chi0 : 0.0;
    }
    const double* kc = s_kc;
    EvalConst KW;
    KW.bexp = 10.0 - p.alpha;
    KW.bass = (p.alpha > 0.0 && p.alpha <= 10.0) ? (KW.bexp == 1.0 ? 1 : 2) : 0;
    // owners of the quartile points
    const int q1g = rec.q1 / C, q1s = rec.q1 % C, q3g = rec.q3 / C, q3s = rec.q3 % C;

    // this thread's points of the UNSORTED light curve (fold input), loop-invariant: kept in registers
    double tt_own[C];
    const double* g_tt = p.tt + rec.off;
    const double* g_y = p.yc + rec.off;
    const double* g_w = p.w + rec.off;
#pragma unroll
    for (int s = 0; s < C; s++) {
        const int i = gt + NTT * s;
        tt_own[s] = i < n ? g_tt[i] : 0.0;
    }
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const ScanMask mk = make_scan_mask(lane);
    const uint32_t tmem = s_tmem + ((uint32_t)(warp & 3) << 21) + (uint32_t)(warp >> 2) * TCOLS_WARP;
    constexpr uint32_t T_A0 = 0, T_A1 = 2 * C, T_A2 = 4 * C, T_ISW = 6 * C, T_XB = 8 * C, T_G0 = 10 * C, T_Y = 12 * C;
    constexpr uint32_t T_W0 = 14 * C;                // window ends (lo[C], hi[C]) per span: rank << 16 | element index
    {
        // position p of the cluster-wide prefix arrays -> (owner CTA, element index in its transposed array)
        auto where = [&](int pos) {
            int g = pos / C, s = pos - g * C;
            int r = g / NT, t = g - r * NT;
            if (r >= R) { r = R - 1; t = NT; s = 0; }      // position R*NT*C: the grand total, row 0 / column NT of the last CTA
            return (r << 16) | (s * ROW + t);
        };
        int w0[2 * C], w1[2 * C], w2[2 * C];
#pragma unroll
        for (int s = 0; s < C; s++) {
            const int j = gt * C + s;
            const int l0 = window_lo(j, ibw0, K0, n), l1 = window_lo(j, ibw1, K1, n), l2 = window_lo(j, ibw2, K2, n);
            w0[s] = where(l0); w0[C + s] = where(l0 + K0);
            w1[s] = where(l1); w1[C + s] = where(l1 + K1);
            w2[s] = where(l2); w2[C + s] = where(l2 + K2);
        }
        tmem_park_words<2 * C>(tmem + T_W0, w0);
        tmem_park_words<2 * C>(tmem + T_W0 + 2 * C, w1);
        tmem_park_words<2 * C>(tmem + T_W0 + 4 * C, w2);
        tmem_wait_st();
    }
    // every CTA of the cluster is resident and initialised before anybody touches a neighbour's shared memory
    cluster_sync_all();

    // remote access to a pair-prefix array: element `w` = rank << 16 | index
    // (distributed shared memory moves ~20 B per clock per SM against 128 B for the SM's own: the part of a window that
    // falls into this CTA's slice -- most tweeter windows, a fifth of the midrange ones -- is read with a plain LDS)
    auto ldE = [&](uint32_t base, int w) {
        const int r = w >> 16;
        const uint32_t a = base + ((uint32_t)(w & 0xffff) << 4);
        double2 v;
        if (r == rank) asm volatile("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a) : "memory");
        else v = ld_cl_d2(mapa_u32(a, (uint32_t)r));
        return v;
    };
    auto ldE8 = [&](uint32_t base, int w) {
        const int r = w >> 16;
        const uint32_t a = base + ((uint32_t)(w & 0xffff) << 3);
        double v;
        if (r == rank) asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a) : "memory");
        else v = ld_cl_d(mapa_u32(a, (uint32_t)r));
        return v;
    };

    // Mailbox round: every CTA has published s_mail (tot[0..NS-1], bad; optionally first / last / q); after the cluster
    // barrier warp 0 gathers what this CTA needs: the carry of the CTAs in front of it and the cluster-wide verdict.
    auto mail_round = [&](int ns, bool with_order) {
        cluster_sync_all();
        if (warp == 0) {
            const uint32_t ra = mapa_u32(a_mail, (uint32_t)(lane < R ? lane : 0));
            double2 t0 = make_double2(0.0, 0.0), t1 = t0, t2 = t0;
            int bad = 0;
            double first = 0.0, last = 0.0;
            if (lane < R) {
                t0 = ld_cl_d2(ra + (uint32_t)offsetof(ClusterMail, tot));
                if (ns > 1) t1 = ld_cl_d2(ra + (uint32_t)offsetof(ClusterMail, tot) + 16);
                if (ns > 2) t2 = ld_cl_d2(ra + (uint32_t)offsetof(ClusterMail, tot) + 32);
                bad = ld_cl_s32(ra + (uint32_t)offsetof(ClusterMail, bad));
                if (with_order) {
                    first = ld_cl_d(ra + (uint32_t)offsetof(ClusterMail, first));
                    last = ld_cl_d(ra + (uint32_t)offsetof(ClusterMail, last));
                }
            }
            if (with_order) {
                // slices must follow one another strictly: last of CTA q < first of CTA q+1 (when q+1 holds real points)
                const double nfirst = shfl_down_d(first, 1);
                if (lane + 1 < R && (lane + 1) * NT * C < n && nfirst <= last) bad = 1;
            }
            bad = __any_sync(0xffffffffu, bad != 0) ? 1 : 0;
            // carry = sum of the totals of the CTAs in front of this one, in rank order
            double2 c0 = make_double2(0.0, 0.0), c1 = c0, c2 = c0;
            for (int q = 0; q < rank; q++) {
                c0.x += shfl_d(t0.x, q); c0.y += shfl_d(t0.y, q);
                if (ns > 1) { c1.x += shfl_d(t1.x, q); c1.y += shfl_d(t1.y, q); }
                if (ns > 2) { c2.x += shfl_d(t2.x, q); c2.y += shfl_d(t2.y, q); }
            }
            if (lane == 0) {
                s_carry[0] = c0; s_carry[1] = c1; s_carry[2] = c2;
                s_anybad = bad;
                if (with_order) {
                    const double p1 = ld_cl_d(mapa_u32(a_mail, (uint32_t)(q1g / NT)) + (uint32_t)offsetof(ClusterMail, q));
                    const double p3 = ld_cl_d(mapa_u32(a_mail, (uint32_t)(q3g / NT)) + (uint32_t)offsetof(ClusterMail, q) + 8);
                    const double scale = p3 - p1;
                    s_vs = 1.e-6 * scale * scale;
                }
            }
        }
        __syncthreads();
    };
    // warp 0 turns the 16 warp totals of `ns` pair scans into the CTA totals of the mailbox (after a CTA barrier)
    auto publish_totals = [&](int ns, int bad_cta) {
        if (warp == 0) {
            for (int i = 0; i < ns; i++) {
                double2 t = lane < G ? s_tot[i][lane] : make_double2(0.0, 0.0);
                // sum over the 16 warps in warp order (deterministic): sequential through shuffles
                double ax = 0.0, ay = 0.0;
#pragma unroll
                for (int q = 0; q < G; q++) { ax += shfl_d(t.x, q); ay += shfl_d(t.y, q); }
                if (lane == 0) s_mail.tot[i] = make_double2(ax, ay);
            }
            if (lane == 0) s_mail.bad = bad_cta;
        }
    };
    // phase 2 of a pair scan with the cluster carry added
    auto finish_pair = [&](const PairScan& s, const double (&a)[C], const double (&b)[C], int which, double2* E) {
        double ca = s_carry[which].x, cb = s_carry[which].y;
        for (int q = 0; q < warp; q++) { const double2 t = s_tot[which][q]; ca += t.x; cb += t.y; }
        double xa = ca + (s.ia - s.ra), xb = cb + (s.ib - s.rb);
#pragma unroll
        for (int i = 0; i < C; i++) {
            E[i * ROW + tid] = make_double2(xa, xb);
            xa += a[i]; xb += b[i];
        }
        if (tid == NT - 1) E[NT] = make_double2(xa, xb);      // used only in the last CTA (the grand total)
    };
    // one stream, plain doubles (CV keeps wxy alone: 8-byte window ends); carry in s_carry[which].x
    auto finish_one = [&](const PairScan& s, const double (&a)[C], int which, double* E) {
        double ca = s_carry[which].x;
        for (int q = 0; q < warp; q++) ca += s_tot[which][q].x;
        double xa = ca + (s.ia - s.ra);
#pragma unroll
        for (int i = 0; i < C; i++) { E[i * ROW + tid] = xa; xa += a[i]; }
        if (tid == NT - 1) E[NT] = xa;
    };
    auto hand_over = [&](int64_t k) {
        if (rank == 0 && tid == 0) {
            const unsigned pos = atomicAdd(p.defer_count, 1u);
            if (pos < p.defer_capacity)
                p.defer_entries[pos] = ((unsigned long long)ri << 32) | (unsigned long long)(k - p.k_begin);
            else
                p.defer_count[1] = 1u;
        }
    };

    const int64_t k0 = p.k_begin + (int64_t)ch * p.chunk;
    const int64_t k1 = min(k0 + (int64_t)p.chunk, p.k_end);
    double best = -INFINITY;
    int64_t best_k = INT64_MAX;
    double* prow = p.pgram ? p.pgram + (rec.obj - p.pgram_row0) * p.pgram_row_stride - p.pgram_k0 : nullptr;
    double stash = 0.0;
    int64_t kb = k0;

    for (int64_t k = k0; k < k1; k++) {
        const double f = freq_of(p.f_min, p.df, k);

        // ---- P1 fold + 64-bit keys (48 phase bits | 16 index bits); P2 sort over the cluster
        key64 key[C];
#pragma unroll
        for (int s = 0; s < C; s++) {
            const int i = gt + NTT * s;
            key64 kk = ~0ull;
            if (i < n) kk = ((key64)__double2ull_rz(fold_phase(tt_own[s], f) * 281474976710656.0) << CL_IDX_BITS) | (key64)i;
            key[s] = kk;
        }
        int flip = 0;
        local_sort64<C>(key);
#pragma unroll 1
        for (int kk = 2; kk <= NT; kk <<= 1) {
            cta_step64<C, true>(key, kk - 1, (tid & (kk >> 1)) == 0, tid, flip ? IB : IA);
            if (kk - 1 >= 32) flip ^= 1;
            for (int m = kk >> 2; m >= 1; m >>= 1) {
                cta_step64<C, false>(key, m, (tid & m) == 0, tid, flip ? IB : IA);
                if (m >= 32) flip ^= 1;
            }
            local_sort64<C>(key);
        }
        int xflip = 0;
        for (int kcta = 2; kcta <= R; kcta <<= 1) {
            // mirror across CTAs: partner thread = (rank ^ (kcta-1), NT-1-tid), slots reversed
            {
                key64* xb = xflip ? XB : XA;
#pragma unroll
                for (int s = 0; s < C; s++) xb[s * NT + tid] = key[s];
                cluster_sync_all();
                const uint32_t ra = mapa_u32(xflip ? a_XB : a_XA, (uint32_t)(rank ^ (kcta - 1)));
                const bool lower = (rank & (kcta >> 1)) == 0;
#pragma unroll
                for (int s = 0; s < C; s++) {
                    const key64 o = ld_cl_u64(ra + (uint32_t)(((C - 1 - s) * NT + (NT - 1 - tid)) * 8));
                    key[s] = cex_side64(key[s], o, lower);
                }
                xflip ^= 1;
            }
            for (int mc = kcta >> 2; mc >= 1; mc >>= 1) {
                key64* xb = xflip ? XB : XA;
#pragma unroll
                for (int s = 0; s < C; s++) xb[s * NT + tid] = key[s];
                cluster_sync_all();
                const uint32_t ra = mapa_u32(xflip ? a_XB : a_XA, (uint32_t)(rank ^ mc));
                const bool lower = (rank & mc) == 0;
#pragma unroll
                for (int s = 0; s < C; s++) {
                    const key64 o = ld_cl_u64(ra + (uint32_t)((s * NT + tid) * 8));
                    key[s] = cex_side64(key[s], o, lower);
                }
                xflip ^= 1;
            }
            cta_merge_tail64<C>(key, tid, IA, IB, flip);
        }

        // ---- exact phases in the sorted order (gather from global memory: the object does not fit one CTA)
        double x[C], y[C], w[C];
        bool bad = false;
        {
            double phi[C];
            int idx[C];
#pragma unroll
            for (int s = 0; s < C; s++) {
                idx[s] = (int)(key[s] & 0xffffull);
                phi[s] = (gt * C + s < n) ? fold_phase(__ldg(g_tt + idx[s]), f) : 4.0 + (double)s;
            }
#pragma unroll
            for (int s = 0; s + 1 < C; s++)
                if (gt * C + s + 1 < n && phi[s + 1] <= phi[s]) bad = true;               // tie, or phases equal in 48 bits
            const double nphi = shfl_down_d(phi[0], 1);
            if (lane < 31 && (gt + 1) * C < n && nphi <= phi[C - 1]) bad = true;
            if (lane == 0) s_wfirst[warp] = phi[0];
            if (lane == 31) s_wlast[warp] = phi[C - 1];
            if (tid == 0) s_mail.first = phi[0];
            if (tid == NT - 1) s_mail.last = phi[C - 1];
            if (gt == q1g) {
#pragma unroll
                for (int s = 0; s < C; s++) if (s == q1s) s_mail.q[0] = phi[s];
            }
            if (gt == q3g) {
#pragma unroll
                for (int s = 0; s < C; s++) if (s == q3s) s_mail.q[1] = phi[s];
            }
#pragma unroll
            for (int s = 0; s < C; s++) {
                if (gt * C + s < n) { x[s] = phi[s] - 0.5; y[s] = __ldg(g_y + idx[s]); w[s] = __ldg(g_w + idx[s]); }
                else { x[s] = 0.0; y[s] = 0.0; w[s] = W_PAD; }
            }
        }

        // ---- prefix sums of the weighted moments
        double ma[C], mb[C], mc_[C], md[C], me[C], mf[C];
#pragma unroll
        for (int s = 0; s < C; s++) {
            ma[s] = w[s]; mb[s] = w[s] * x[s]; mc_[s] = mb[s] * x[s]; md[s] = w[s] * y[s]; me[s] = mb[s] * y[s];
            mf[s] = GV ? md[s] * y[s] : 0.0;
        }
        const PairScan ps0 = pair_scan_begin<C>(ma, mb, s_tot[0], warp, lane, mk);
        const PairScan ps1 = pair_scan_begin<C>(mc_, md, s_tot[1], warp, lane, mk);
        const PairScan ps2 = pair_scan_begin<C>(me, mf, s_tot[2], warp, lane, mk);
        int bad_cta = __syncthreads_or(bad);
        if (warp == 0) {
            // warp boundaries inside the CTA
            const double wl = lane < G ? s_wlast[lane] : 0.0;
            const double wf = lane + 1 < G ? s_wfirst[lane + 1] : 8.0;
            if (__any_sync(0xffffffffu, lane + 1 < G && (rank * NT + (lane + 1) * 32) * C < n && wf <= wl)) bad_cta = 1;
        }
        publish_totals(3, bad_cta);
        mail_round(3, true);
        double P = 0.0;
        bool skip = s_anybad != 0;
        if (!skip) {
            finish_pair(ps0, ma, mb, 0, E01);
            finish_pair(ps1, mc_, md, 1, E23);
            if (GV) finish_pair(ps2, me, mf, 2, E45);
            else finish_one(ps2, me, 2, reinterpret_cast<double*>(E45));
            const double vsmlsq = s_vs;
            cluster_sync_all();
            double chi2 = 0.0;
            if (GV) {
                double A[3][C], Gs[3][C];
#pragma unroll
                for (int i = 0; i < 3; i++) {
                    int wi[2 * C];
                    tmem_fetch_words<2 * C>(tmem + T_W0 + 2 * C * i, wi);
#pragma unroll
                    for (int s = 0; s < C; s++) {
                        const int a_ = wi[s], b_ = wi[C + s];
                        const double2 l0 = ldE(a_E01, a_), h0 = ldE(a_E01, b_), l1 = ldE(a_E23, a_), h1 = ldE(a_E23, b_);
                        const double2 l2 = ldE(a_E45, a_), h2 = ldE(a_E45, b_);
                        const double Sw = h0.x - l0.x, Swx = h0.y - l0.y, Swxx = h1.x - l1.x, Sy = h1.y - l1.y;
                        const double Sxy = h2.x - l2.x, Syy = h2.y - l2.y;
                        const double isw = rcp64(Sw), xb = Swx * isw;
                        const double sxx = Swxx - xb * Swx;
                        const double isxx = sxx > vsmlsq ? rcp64(sxx) : 0.0;
                        const double yb = Sy * isw, sxy = Sxy - xb * Sy, b = sxy * isxx;
                        A[i][s] = yb + b * (x[s] - xb);
                        const double rss = (Syy - yb * Sy) - b * sxy;
                        Gs[i][s] = sqrt64(rss * isw) * (isxx != 0.0 ? kc[2 * i + 1] : kc[2 * i]);
                    }
                }
#pragma unroll
                for (int s = 0; s < C; s++) {
                    const double sp = pick_span_w(Gs[0][s], Gs[1][s], Gs[2][s], KW);
                    const double smo = interp_spans(sp, A[0][s], A[1][s], A[2][s]);
                    const double r = y[s] - smo;
                    chi2 += w[s] * r * r;
                }
            } else {
                double r0[C], r1[C], r2[C];
                double m_isw[C], m_xb[C], m_g[C];
                int amin = 0x7fffffff;
#pragma unroll
                for (int i = 0; i < 3; i++) {
                    int wi[2 * C];
                    tmem_fetch_words<2 * C>(tmem + T_W0 + 2 * C * i, wi);
                    double Ai[C], q_isw[C], q_xb[C], q_g[C];
#pragma unroll
                    for (int s = 0; s < C; s++) {
                        const int a_ = wi[s], b_ = wi[C + s];
                        const double2 l0 = ldE(a_E01, a_), h0 = ldE(a_E01, b_), l1 = ldE(a_E23, a_), h1 = ldE(a_E23, b_);
                        const double lxy = ldE8(a_E45, a_), hxy = ldE8(a_E45, b_);
                        const double Sw = h0.x - l0.x, Swx = h0.y - l0.y, Swxx = h1.x - l1.x, Sy = h1.y - l1.y;
                        const double Sxy = hxy - lxy;
                        const double isw = rcp64(Sw), xb = Swx * isw;
                        const double sxx = Swxx - xb * Swx;
                        const double isxx = sxx > vsmlsq ? rcp64(sxx) : 0.0;
                        const double dx = x[s] - xb, g = isxx * dx;
                        q_isw[s] = isw; q_xb[s] = xb; q_g[s] = g;
                        Ai[s] = Sy * isw + (Sxy - xb * Sy) * g;
                        const double a = 1.0 - w[s] * (isw + dx * g);
                        const double r = fabs(y[s] - Ai[s]) * rcp64(a);
                        if (i == 0) r0[s] = r; else if (i == 1) r1[s] = r; else r2[s] = r;
                        amin = min(amin, __double2hiint(a));
                    }
                    tmem_park<C>(tmem + T_A0 + 2 * C * i, Ai);
                    if (i == 0) { tmem_park<C>(tmem + T_ISW, q_isw); tmem_park<C>(tmem + T_XB, q_xb); tmem_park<C>(tmem + T_G0, q_g); }
                    if (i == 1) {
#pragma unroll
                        for (int s = 0; s < C; s++) { m_isw[s] = q_isw[s]; m_xb[s] = q_xb[s]; m_g[s] = q_g[s]; }
                    }
                }
                tmem_park<C>(tmem + T_Y, y);
                double za[C], zb[C], zc[C], zd[C], ze[C], zf[C];
#pragma unroll
                for (int s = 0; s < C; s++) {
                    za[s] = w[s] * r0[s]; zb[s] = za[s] * x[s];
                    zc[s] = w[s] * r1[s]; zd[s] = zc[s] * x[s];
                    ze[s] = w[s] * r2[s]; zf[s] = ze[s] * x[s];
                }
                const PairScan qs0 = pair_scan_begin<C>(za, zb, s_tot[0], warp, lane, mk);
                const PairScan qs1 = pair_scan_begin<C>(zc, zd, s_tot[1], warp, lane, mk);
                const PairScan qs2 = pair_scan_begin<C>(ze, zf, s_tot[2], warp, lane, mk);
                const int carry_cta = __syncthreads_or(amin < 0x00100000);      // a <= 0: the residual carries (R23)
                publish_totals(3, carry_cta);
                mail_round(3, false);         // its cluster barrier also retires every remote read of the primary arrays
                skip = s_anybad != 0;
                if (!skip) {
                    finish_pair(qs0, za, zb, 0, E01);
                    finish_pair(qs1, zc, zd, 1, E23);
                    finish_pair(qs2, ze, zf, 2, E45);
                    cluster_sync_all();
                    int w1i[2 * C];
                    tmem_fetch_words<2 * C>(tmem + T_W0 + 2 * C, w1i);
                    auto mid_load = [&](uint32_t base, double (&out)[C]) {
#pragma unroll
                        for (int s = 0; s < C; s++) {
                            const double2 l = ldE(base, w1i[s]), h = ldE(base, w1i[C + s]);
                            const double Sz = h.x - l.x, Sxz = h.y - l.y;
                            out[s] = Sz * m_isw[s] + (Sxz - m_xb[s] * Sz) * m_g[s];
                        }
                    };
                    double sp[C];
                    {
                        double R0[C], R1[C], R2[C];
                        mid_load(a_E01, R0); mid_load(a_E23, R1); mid_load(a_E45, R2);
#pragma unroll
                        for (int s = 0; s < C; s++) sp[s] = pick_span_w(R0[s], R1[s], R2[s], KW);
                    }
#pragma unroll
                    for (int s = 0; s < C; s++) { za[s] = w[s] * sp[s]; zb[s] = za[s] * x[s]; }
                    const PairScan ss0 = pair_scan_begin<C>(za, zb, s_tot[0], warp, lane, mk);
                    __syncthreads();
                    publish_totals(1, 0);
                    mail_round(1, false);
                    finish_pair(ss0, za, zb, 0, E01);
                    cluster_sync_all();
                    double B[C];
                    mid_load(a_E01, B);
                    tmem_wait_st();
                    {
                        double a0[C], a1[C], a2[C];
                        tmem_fetch<C>(tmem + T_A0, a0); tmem_fetch<C>(tmem + T_A1, a1); tmem_fetch<C>(tmem + T_A2, a2);
#pragma unroll
                        for (int s = 0; s < C; s++) B[s] = interp_spans(B[s], a0[s], a1[s], a2[s]);
                    }
#pragma unroll
                    for (int s = 0; s < C; s++) { zc[s] = w[s] * B[s]; zd[s] = zc[s] * x[s]; }
                    const PairScan fs0 = pair_scan_begin<C>(zc, zd, s_tot[1], warp, lane, mk);
                    __syncthreads();
                    if (warp == 0) {      // publish into tot[0] (mail_round(1) reads slot 0)
                        double2 t = lane < G ? s_tot[1][lane] : make_double2(0.0, 0.0);
                        double ax = 0.0, ay = 0.0;
#pragma unroll
                        for (int q = 0; q < G; q++) { ax += shfl_d(t.x, q); ay += shfl_d(t.y, q); }
                        if (lane == 0) { s_mail.tot[0] = make_double2(ax, ay); s_mail.bad = 0; }
                    }
                    mail_round(1, false);
                    {
                        // finish into E23 with carry slot 0 and warp totals slot 1
                        double ca = s_carry[0].x, cb = s_carry[0].y;
                        for (int q = 0; q < warp; q++) { const double2 t = s_tot[1][q]; ca += t.x; cb += t.y; }
                        double xa = ca + (fs0.ia - fs0.ra), xb = cb + (fs0.ib - fs0.rb);
#pragma unroll
                        for (int i = 0; i < C; i++) {
                            E23[i * ROW + tid] = make_double2(xa, xb);
                            xa += zc[i]; xb += zd[i];
                        }
                        if (tid == NT - 1) E23[NT] = make_double2(xa, xb);
                    }
                    cluster_sync_all();
                    int w0i[2 * C];
                    tmem_fetch_words<2 * C>(tmem + T_W0, w0i);
                    double t_isw[C], t_xb[C], t_g[C], yy[C];
                    tmem_fetch<C>(tmem + T_ISW, t_isw); tmem_fetch<C>(tmem + T_XB, t_xb); tmem_fetch<C>(tmem + T_G0, t_g);
                    tmem_fetch<C>(tmem + T_Y, yy);
#pragma unroll
                    for (int s = 0; s < C; s++) {
                        const double2 l = ldE(a_E23, w0i[s]), h = ldE(a_E23, w0i[C + s]);
                        const double Sz = h.x - l.x, Sxz = h.y - l.y;
                        const double smo = Sz * t_isw[s] + (Sxz - t_xb[s] * Sz) * t_g[s];
                        const double r = yy[s] - smo;
                        chi2 += w[s] * r * r;
                    }
                }
            }
            if (!skip) {
#pragma unroll
                for (int d = 16; d > 0; d >>= 1) chi2 += __shfl_xor_sync(0xffffffffu, chi2, d);
                if (lane == 0) s_red[warp] = chi2;
                __syncthreads();
                if (tid == 0) {
                    double c2 = 0.0;
#pragma unroll
                    for (int q = 0; q < G; q++) c2 += s_red[q];
                    s_mail.chi2 = c2;
                }
                cluster_sync_all();      // also retires every remote read of this eval's prefix arrays
                double c2 = 0.0;
                for (int q = 0; q < R; q++) c2 += ld_cl_d(mapa_u32(a_mail, (uint32_t)q) + (uint32_t)offsetof(ClusterMail, chi2));
                P = (kc[6] - c2) * kc[7];
            }
        }
        if (skip) hand_over(k);
        if (!skip && P > best) { best = P; best_k = k; }
        if (tid == (int)(k - kb)) stash = skip ? 0.0 : P;
        if (k - kb == 31 || k == k1 - 1) {
            if (rank == 0 && prow && tid < 32 && kb + tid <= k) prow[kb + tid] = stash;
            kb = k + 1;
        }
    }
    // nobody leaves while a neighbour may still read its shared memory
    cluster_sync_all();
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(s_tmem), "n"(TCOLS) : "memory");
    }
    if (rank == 0 && tid == 0) {
        const int64_t slot = (int64_t)ri * p.chunks_total + p.chunk_base + ch;
        p.part_val[slot] = best;
        p.part_idx[slot] = best_k == INT64_MAX ? k0 : best_k;
    }
}

template <int C, bool GV>
inline ss_status_t launch_cluster_variant(const EvalParams& p, int R, int64_t n_items, cudaStream_t stream)
{
    const size_t smem = cluster_smem_bytes<C>();
    auto kern = cluster_kernel<C, GV>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return SS_ERR_CUDA;
    if (R > 8 && cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) return SS_ERR_CUDA;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(n_items * R), 1, 1);
    cfg.blockDim = dim3(CL_NT, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)R;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (cudaLaunchKernelEx(&cfg, kern, p, R) != cudaSuccess) return SS_ERR_CUDA;
    return cudaGetLastError() == cudaSuccess ? SS_OK : SS_ERR_CUDA;
}

}  // namespace ss

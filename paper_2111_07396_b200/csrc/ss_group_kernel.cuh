// ss_group_kernel.cuh -- G warps per (object, frequency) eval, 256 < n <= 2,055 (SS_PATH_GROUP).
//
// The warp-per-eval design (ss_warp_kernel.cuh) carried over to light curves that do not fit one warp: the CTA
// (G = 4, 8 or 16 warps) owns one eval at a time, thread t owns the C consecutive phase-ordered points
// j = t*C .. t*C+C-1 in registers, and the warps meet only where the method forces them to:
//   fold -> 32-bit keys (phase bits | index) -> blocked bitonic network: inside a warp on registers and shuffles,
//           across warps through one shared-memory exchange + one barrier per step ->
//   gather of the exact phases, repair of the order inside a quantisation bucket (adjacent swap), exact-order check ->
//   prefix sums of the weighted moments: lane-local + Kogge-Stone inside the warp, ONE carry exchange across warps,
//           stored pair-interleaved and transposed ([slot][thread]) so every window-end access is conflict-free ->
//   all three spans by differences of those prefix arrays; CV (Listing 1) keeps the primary smooths
//           and the tweeter x-moments parked in tensor memory; GV (R12) needs no second pass -> chi2 -> P.
// The object's tt / yc / w are staged into shared memory ONCE per work item by three 1-D bulk copies
// (cp.async.bulk + mbarrier).  32 values of P are stashed and stored as one coalesced row segment.
// Evals this path cannot decide exactly (tied phases, a bucket that one adjacent swap does not settle, a
// leave-one-out denominator <= 0) are handed to the generic CTA-per-eval kernel through the same list the warp path
// uses, so results never depend on which path ran.
//
// The kernel is templated on the smoother's scalar T ("toggle between using FP32 or FP64").
// T = double is the library's default.  T = float is the MIXED mode (ss_options_t::precision): the fold, the sort, the
// centring of x and y and the ACCUMULATION of every prefix sum stay in fp64 (a window sum is the difference of two
// prefixes of magnitude ~n/K times its own: rounding the accumulation to fp32 would leave no digits), the prefix
// arrays are stored, and every window fit, residual, span pick and interpolation is computed, in fp32.
#pragma once
#include "ss_warp_kernel.cuh"

namespace ss {

template <int G, int C, typename T = double> struct GroupCfg {
    static constexpr int NT = 32 * G;               // threads
    static constexpr int NP = NT * C;               // capacity in points
    static constexpr int ROW = NT + 1;              // row of a transposed prefix array: NT threads + the total
    static constexpr int MINB = G == 4 ? 4 : (G == 8 ? 2 : 1);      // 16 warps per SM at 128 registers
    static constexpr int IDX_BITS = NP <= 512 ? 9 : (NP <= 1024 ? 10 : (NP <= 2048 ? 11 : 12));
    static constexpr unsigned IDX_MASK = (1u << IDX_BITS) - 1u;
    // tensor memory per warp: 7 parked arrays (A0, A1, A2, tweeter isw / xbar / g, y) + per span C words of window
    // ends, two 16-bit element indices each (padded to an even count)
    static constexpr uint32_t PCOLS = TmemArr<T, C>::COLS;
    static constexpr int CE = (C + 1) & ~1;
    static constexpr uint32_t TCOLS_WARP = 7 * PCOLS + 3 * CE;
    static_assert(C * (NT + 1) < 65536, "window-end indices are packed two to a word");
    static constexpr uint32_t TCOLS_NEED = TCOLS_WARP * (G / 4);
    static constexpr uint32_t TCOLS = TCOLS_NEED <= 32 ? 32 : (TCOLS_NEED <= 64 ? 64 : (TCOLS_NEED <= 128 ? 128 : (TCOLS_NEED <= 256 ? 256 : 512)));
    static_assert(TCOLS * MINB <= 512, "tensor memory over-subscribed");
};

template <> __device__ __forceinline__ void local_sort<2>(unsigned (&k)[2]) { cex32(k[0], k[1]); }
template <> __device__ __forceinline__ void local_sort<4>(unsigned (&k)[4])
{
    cex32(k[0], k[1]); cex32(k[2], k[3]); cex32(k[0], k[2]); cex32(k[1], k[3]); cex32(k[1], k[2]);
}

// ---- 1-D bulk copy global -> shared with mbarrier completion (PTX cp.async.bulk; SASS UBLKCP) ------------
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;"
                 :: "r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity)
{
    asm volatile("{\n\t.reg .pred p;\n\tWAIT_%=:\n\t"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
                 "@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}"
                 :: "r"((uint32_t)__cvta_generic_to_shared(bar)), "r"(parity) : "memory");
}
// bytes: multiple of 16; src and dst 16-byte aligned
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src), "r"(bytes),
                    "r"((uint32_t)__cvta_generic_to_shared(bar)) : "memory");
}

// The object's y and w are staged in shared memory beside its times up to 2,560 points; beyond (G = 16, C = 6, 7:
// 3,072 / 3,584 points -- the three pair-prefix arrays then take 148 / 172 KB) they are gathered from the catalog copy
// in global memory once per eval, as the shared-sampling kernels do.
constexpr int GROUP_STAGE_YW_MAX = 2560;
template <int G, int C, bool GV, typename T = double>
inline size_t group_smem_bytes()
{
    using Cfg = GroupCfg<G, C, T>;
    // object arrays (3 x NP doubles, or the times alone) + 3 pair-prefix arrays of C*ROW vec2 (the sort's exchange
    // buffers, 2 x NT*C words, overlay the first of them: C*ROW*sizeof(vec2) >= 8*NT*C also for float2)
    return (size_t)(Cfg::NP > GROUP_STAGE_YW_MAX ? 1 : 3) * Cfg::NP * 8 + (size_t)3 * C * Cfg::ROW * sizeof(typename Real<T>::vec2);
}

// Exclusive prefix sums of two streams over the whole CTA (C values per thread, blocked), stored interleaved and
// transposed: E[(j % C)*ROW + j/C] = (sum_{i<j} a_i, sum_{i<j} b_i).  Phase 1 (before the barrier): lane-local sums,
// Kogge-Stone over the warp, the warp's totals to `tot`; phase 2 (after it): the carry of the warps in front.
struct PairScan { double ra, rb, ia, ib; };
template <int C, typename T>
__device__ __forceinline__ PairScan pair_scan_begin(const T (&a)[C], const T (&b)[C], double2* tot, int warp,
                                                    int lane, const ScanMask& mk)
{
    // the thread's own C values are summed in T (C terms: no accuracy at stake), everything across threads in fp64:
    // a float kernel then converts twice per thread and stream, not per element
    PairScan s;
    T ra = a[0], rb = b[0];
#pragma unroll
    for (int i = 1; i < C; i++) { ra += a[i]; rb += b[i]; }
    s.ra = (double)ra; s.rb = (double)rb;
    s.ia = s.ra; s.ib = s.rb;
#pragma unroll
    for (int i = 0; i < 5; i++) { scan_step(s.ia, i, mk); scan_step(s.ib, i, mk); }
    if (lane == 31) tot[warp] = make_double2(s.ia, s.ib);
    return s;
}
template <int G, int C, typename T>
__device__ __forceinline__ void pair_scan_finish(const PairScan& s, const T (&a)[C], const T (&b)[C],
                                                 const double2* tot, typename Real<T>::vec2* E, int warp, int tid)
{
    constexpr int ROW = GroupCfg<G, C>::ROW;
    double ca = 0.0, cb = 0.0;
    for (int q = 0; q < warp; q++) { const double2 t = tot[q]; ca += t.x; cb += t.y; }      // warp-uniform: broadcast loads
    T xa = (T)(ca + (s.ia - s.ra)), xb = (T)(cb + (s.ib - s.rb));
#pragma unroll
    for (int i = 0; i < C; i++) {
        E[i * ROW + tid] = Real<T>::make2(xa, xb);
        xa += a[i]; xb += b[i];
    }
    if (tid == 32 * G - 1) E[32 * G] = Real<T>::make2(xa, xb);       // position NP lives at row 0, column NT
}
// one stream, plain doubles (row length ROW doubles)
struct OneScan { double ra, ia; };
template <int C, typename T>
__device__ __forceinline__ OneScan one_scan_begin(const T (&a)[C], double* tot, int warp, int lane, const ScanMask& mk)
{
    OneScan s;
    T ra = a[0];
#pragma unroll
    for (int i = 1; i < C; i++) ra += a[i];
    s.ra = (double)ra;
    s.ia = s.ra;
#pragma unroll
    for (int i = 0; i < 5; i++) scan_step(s.ia, i, mk);
    if (lane == 31) tot[warp] = s.ia;
    return s;
}
template <int G, int C, typename T>
__device__ __forceinline__ void one_scan_finish(const OneScan& s, const T (&a)[C], const double* tot, T* E,
                                                int warp, int tid)
{
    constexpr int ROW = GroupCfg<G, C>::ROW;
    double ca = 0.0;
    for (int q = 0; q < warp; q++) ca += tot[q];
    T xa = (T)(ca + (s.ia - s.ra));
#pragma unroll
    for (int i = 0; i < C; i++) { E[i * ROW + tid] = xa; xa += a[i]; }
    if (tid == 32 * G - 1) E[32 * G] = xa;
}

// Exchange of the C keys with thread (tid ^ mask); REV: the partner's slots in reverse order (mirror step).
// mask < 32: shuffles.  Otherwise through shared memory: kb = this step's exchange buffer (two alternate, so one
// barrier per step is enough).
template <int G, int C, bool REV>
__device__ __forceinline__ void key_exchange(const unsigned (&key)[C], unsigned (&other)[C], int mask, int tid,
                                             unsigned* kb)
{
    constexpr int NT = 32 * G;
    if (mask < 32) {
#pragma unroll
        for (int s = 0; s < C; s++) other[s] = __shfl_xor_sync(0xffffffffu, key[REV ? C - 1 - s : s], mask);
    } else {
#pragma unroll
        for (int s = 0; s < C; s++) kb[s * NT + tid] = key[s];
        __syncthreads();
        const int pt = tid ^ mask;
#pragma unroll
        for (int s = 0; s < C; s++) other[s] = kb[(REV ? C - 1 - s : s) * NT + pt];
    }
}

// Blocked bitonic sort of NT*C keys over the CTA (position = tid*C + s): the network of warp_sort_any with 32*G lanes.
template <int G, int C>
__device__ __forceinline__ void group_sort(unsigned (&key)[C], int tid, unsigned* kbuf)
{
    constexpr int NT = 32 * G;
    int flip = 0;
    local_sort<C>(key);
#pragma unroll
    for (int k = 2; k <= NT; k <<= 1) {
        {
            const bool lower = (tid & (k >> 1)) == 0;
            unsigned other[C];
            key_exchange<G, C, true>(key, other, k - 1, tid, kbuf + flip * NT * C);
            if (k - 1 >= 32) flip ^= 1;
#pragma unroll
            for (int s = 0; s < C; s++) key[s] = lower ? min(key[s], other[s]) : max(key[s], other[s]);
        }
#pragma unroll
        for (int m = k >> 2; m >= 1; m >>= 1) {
            const bool lower = (tid & m) == 0;
            unsigned other[C];
            key_exchange<G, C, false>(key, other, m, tid, kbuf + flip * NT * C);
            if (m >= 32) flip ^= 1;
#pragma unroll
            for (int s = 0; s < C; s++) key[s] = lower ? min(key[s], other[s]) : max(key[s], other[s]);
        }
        local_sort<C>(key);
    }
}

// Per-object constants (CTA-uniform).
struct GroupConst {
    int n;
    const double* kc;        // shared: gk[span][p-1] = 1/(1 - p/K_span) (6 values), then chi0, 1/chi0
    int q1t, q1s, q3t, q3s;  // owners (thread, slot) of the quartile points
    int bass; double bexp;
};

// ------------------------------------------------------------------------------------------------
// Kernel: one CTA = one work item (object, chunk of frequencies), evals one after the other.
// ------------------------------------------------------------------------------------------------
// Resident CTAs per SM: 16 warps at 128 registers, except 4-warp CTAs with 6 or 7 points per thread, which spill less and
// run faster at 12 warps / 168 registers (measured, CV: +11..13 % at C = 7, +2..3 % at C = 6; GV: C = 7 only)
template <int G, int C, bool GV, typename T>
constexpr int group_minb()
{
    // (8, 7) in fp64 CV spills 390 bytes at 128 registers; one CTA per SM at 255 registers and no spills is 13 % faster
    // (1.94e10 -> 2.19e10 point-evals/s at n = 1,792; the same trade loses at (8, 6) and does not compile for GV)
    if (G == 8 && C == 7 && sizeof(T) == 8 && !GV) return 1;
    // T = float needs half the registers, tensor-memory columns and prefix-array bytes: 32 warps per SM at 64 registers
    // for C <= 4, 24 at 80 for C = 5, 6, 16 at 128 for C = 7 (measured per variant: CV +2..16 %, GV +2..30 % over the
    // fp64 shapes; the one loser, (4, 5) GV, keeps 16 warps)
    if (sizeof(T) == 4) {
        if (G == 4) return C <= 4 ? 8 : (C <= 6 ? ((C == 5 && GV) ? 4 : 6) : 4);
        if (G == 8) return C <= 4 ? 4 : (C <= 6 ? 3 : 2);
        return C <= 4 ? 2 : 1;
    }
    // (4, 3) fits 96 registers: 20 warps per SM, +6 % CV / +4 % GV at n = 257..384 (24 warps at 80 registers lose again)
    if (G == 4 && C == 3 && sizeof(T) == 8) return 5;
    return (G == 4 && (C >= 7 || (C >= 6 && !GV))) ? 3 : GroupCfg<G, C, T>::MINB;
}

// OPT: 0 = the default call; 1 = the listing's options compiled in: periodic windows (iper = 2,
// PAPER.md:199-200) -- a window that leaves [0, n) is two ranges, the part that wrapped counting with abscissae x - 1
// or x + 1, so its moments follow from the unshifted sums of that part: Swx += s bw, Swxx += 2 s bwx + bw, Sxy += s by
// (s = -1 below 0, +1 above n-1); the second range is found by arithmetic, no second table --
// 2 = a fixed span (span > 0): one smooth of y, both modes alike (instantiated with GV = false);
// 3 = shared time sampling (ss_options_t::shared_times): the work item is a group of SHARED_TIMES_M objects
// with one time vector; fold, sort, order repair and the abscissae are done once per frequency, the smoother once per
// object on that permutation (y and w gathered from the catalog copy in global memory).
template <int G, int C, bool GV, typename T = double, int OPT = 0>
__global__ void __launch_bounds__(GroupCfg<G, C, T>::NT, group_minb<G, C, GV, T>()) group_kernel(const EvalParams p)
{
    static_assert(OPT == 0 || sizeof(T) == 8, "the listing's options and shared sampling are served in fp64");
    static_assert(OPT != 2 || !GV, "the fixed-span kernel is instantiated once, with GV = false");
    using Cfg = GroupCfg<G, C, T>;
    using RT = Real<T>;
    using T2 = typename RT::vec2;
    using TA = TmemArr<T, C>;
    constexpr int NT = Cfg::NT, NP = Cfg::NP, ROW = Cfg::ROW, ASZ = C * ROW;
    constexpr bool LOPT = OPT == 1 || OPT == 2;            // the listing's options
    constexpr bool SH = OPT == 3;
    constexpr bool YW_GLOBAL = SH || Cfg::NP > GROUP_STAGE_YW_MAX;      // y, w gathered from the catalog copy per eval
    constexpr int M_ = SH ? SHARED_TIMES_M : 1;            // objects per work item
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ int s_ri[M_];                               // per object of the group: record index, offset into the
    __shared__ long long s_off[M_];                        // catalog copy, chi0 and 1 / chi0, periodogram row
    __shared__ double s_chi[M_][2];
    __shared__ double* s_prow[M_];
    __shared__ __align__(16) double2 s_tot[3][G];          // warp totals of up to three pair scans
    __shared__ double s_red[G];
    // {phase, index} of each warp's first ([0][warp]) and last ([1][warp + 1]) point, read by the neighbour warp.  The
    // outer slots [0][G] and [1][0] hold sentinels, so that the reads need no test on the warp index: with
    // `if (warp > 0) .. s_edge[1][warp - 1]` ptxas 12.9 formed the address in uniform registers under a mismatched
    // predicate in group_kernel<4, 5, CV, double, 1> and <8, 7, CV, double, 1> (cuda-gdb: misaligned / out-of-range LDS.128).
    __shared__ __align__(16) double s_edge[2][G + 1][2];
    __shared__ double s_q[2];                                // phases of the quartile points
    __shared__ double s_kc[8];
    __shared__ __align__(8) uint64_t s_bar;
    __shared__ uint32_t s_tmem;

    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);     // provably warp-uniform (see warp_kernel)
    const int item = blockIdx.x;
    const int grp = item / p.chunks_per_obj, ch = item - grp * p.chunks_per_obj;
    const int li = grp * M_;
    const int mcnt = SH ? min(M_, p.n_list - li) : 1;        // objects in this group
    const int ri = p.list[li];
    const ObjRec rec = p.recs[ri];                           // shared sampling: n, windows and times of the first object
    if (rec.dup) {
        // duplicated time stamps: every eval ties; the generic kernel takes the whole work item(s)
        if (tid < mcnt) {
            const unsigned pos = atomicAdd(p.defer_count, 1u);
            if (pos < p.defer_capacity)
                p.defer_entries[pos] = DEFER_ITEM | ((unsigned long long)(SH ? p.list[li + tid] : ri) << 32) | (unsigned long long)ch;
            else
                p.defer_count[1] = 1u;
        }
        return;
    }
    const int n = rec.n;
    if (SH && tid < mcnt) {
        const int rm = p.list[li + tid];
        const ObjRec r = p.recs[rm];
        s_ri[tid] = rm; s_off[tid] = r.off;
        s_chi[tid][0] = r.chi0; s_chi[tid][1] = r.chi0 > 0.0 ? 1.0 / r.chi0 : 0.0;
        s_prow[tid] = p.pgram ? p.pgram + (r.obj - p.pgram_row0) * p.pgram_row_stride - p.pgram_k0 : nullptr;
    }

    double* o_tt = reinterpret_cast<double*>(smem_raw);
    double* o_y = o_tt + NP;
    double* o_w = o_y + NP;
    T2* E01 = reinterpret_cast<T2*>(smem_raw + (size_t)(NP > GROUP_STAGE_YW_MAX ? 1 : 3) * NP * 8);   // (w, wx) | residual 0 | spans
    T2* E23 = E01 + ASZ;                                                           // (wxx, wy)    | residual 1 | final
    T2* E45 = E23 + ASZ;                                                           // (wxy[, wyy]) | residual 2
    unsigned* kbuf = reinterpret_cast<unsigned*>(E01);                             // sort exchange (2 x NT*C words)

    // ---- stage the object once per work item: three bulk copies, one mbarrier
    if (tid == 0) {
        mbar_init(&s_bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                     :: "r"((uint32_t)__cvta_generic_to_shared(&s_tmem)), "n"(Cfg::TCOLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    if (tid == 0) {
        const unsigned bytes = (unsigned)(((n + 1) & ~1) * 8);      // the workspace pads every object to an even length
        mbar_expect_tx(&s_bar, (YW_GLOBAL ? 1 : 3) * bytes);
        bulk_g2s(o_tt, p.tt + rec.off, bytes, &s_bar);
        if (!YW_GLOBAL) {      // shared sampling: y and w differ per object and are gathered from the catalog copy
            bulk_g2s(o_y, p.yc + rec.off, bytes, &s_bar);
            bulk_g2s(o_w, p.w + rec.off, bytes, &s_bar);
        }
    }

    const bool per = LOPT && p.iper == 2;            // phases are in [0, 1): jper = iper
    // half-widths: the three spans, or the caller's fixed one in slot 0; a periodic window never exceeds n points (R8)
    int ibw_[3], Kw_[3];
#pragma unroll
    for (int i = 0; i < 3; i++) {
        int b = OPT == 2 ? rec.ibw_fixed : rec.ibw[i];
        int kk = 2 * b + 1;
        if (kk > n) { kk = n; if (per) { b = (n - 1) / 2; kk = 2 * b + 1; } }
        ibw_[i] = b; Kw_[i] = kk;
    }
    const int ibw0 = ibw_[0], ibw1 = ibw_[1], ibw2 = ibw_[2];
    const int K0 = Kw_[0], K1 = Kw_[1], K2 = Kw_[2];
    GroupConst K;
    K.n = n;
    K.q1t = rec.q1 / C; K.q1s = rec.q1 % C; K.q3t = rec.q3 / C; K.q3s = rec.q3 % C;
    if (tid == 0) {
        s_kc[0] = 1.0 / (1.0 - 1.0 / (double)K0); s_kc[1] = 1.0 / (1.0 - 2.0 / (double)K0);
        s_kc[2] = 1.0 / (1.0 - 1.0 / (double)K1); s_kc[3] = 1.0 / (1.0 - 2.0 / (double)K1);
        s_kc[4] = 1.0 / (1.0 - 1.0 / (double)K2); s_kc[5] = 1.0 / (1.0 - 2.0 / (double)K2);
        s_kc[6] = rec.chi0; s_kc[7] = rec.chi0 > 0.0 ? 1.0 / rec.chi0 : 0.0;
    }
    if (tid == 0) {
        s_edge[0][G][0] = 1.0e3; s_edge[0][G][1] = 0.0;      // behind the last warp
        s_edge[1][0][0] = -1.0; s_edge[1][0][1] = 0.0;       // in front of the first
    }
    K.kc = s_kc;
    K.bexp = 10.0 - p.alpha;
    K.bass = (p.alpha > 0.0 && p.alpha <= 10.0) ? (K.bexp == 1.0 ? 1 : 2) : 0;

    const ScanMask mk = make_scan_mask(lane);
    const uint32_t tmem = s_tmem + ((uint32_t)(warp & 3) << 21) + (uint32_t)(warp >> 2) * Cfg::TCOLS_WARP;
    // tensor-memory columns (32-bit words) of this warp
    constexpr uint32_t PC = Cfg::PCOLS;
    constexpr uint32_t T_A0 = 0, T_A1 = PC, T_A2 = 2 * PC, T_ISW = 3 * PC, T_XB = 4 * PC, T_G0 = 5 * PC, T_Y = 6 * PC;
    constexpr int CE = Cfg::CE;
    constexpr uint32_t T_W0 = 7 * PC, T_W1 = T_W0 + CE, T_W2 = T_W0 + 2 * CE;      // window ends per span: lo | hi << 16
    auto at = [&](int pos) { return (pos % C) * ROW + pos / C; };
    // second range of the periodic window of point j at half-width ib: element indices [blo, bhi) and the shift sg (0: none)
    struct Wrap { int sg, blo, bhi; };
    auto wrapped = [&](int j, int ib) -> Wrap {
        Wrap r;
        r.sg = 0; r.blo = 0; r.bhi = 0;
        if (per && j < n) {
            if (j - ib < 0) { r.blo = at(j - ib + n); r.bhi = at(n); r.sg = -1; }
            else if (j + ib + 1 > n) { r.bhi = at(j + ib + 1 - n); r.sg = 1; }
        }
        return r;
    };
    {
        int w0[C], w1[C], w2[C];
#pragma unroll
        for (int s = 0; s < C; s++) {
            const int j = tid * C + s;
            int l0, l1, l2, h0, h1, h2;
            if (per && j < n) {      // the part of the window inside [0, n)
                l0 = max(j - ibw0, 0); h0 = min(j + ibw0 + 1, n);
                l1 = max(j - ibw1, 0); h1 = min(j + ibw1 + 1, n);
                l2 = max(j - ibw2, 0); h2 = min(j + ibw2 + 1, n);
            } else {
                l0 = window_lo(j, ibw0, K0, n); l1 = window_lo(j, ibw1, K1, n); l2 = window_lo(j, ibw2, K2, n);
                h0 = l0 + K0; h1 = l1 + K1; h2 = l2 + K2;
            }
            w0[s] = at(l0) | (at(h0) << 16);
            w1[s] = at(l1) | (at(h1) << 16);
            w2[s] = at(l2) | (at(h2) << 16);
        }
        tmem_park_words<C>(tmem + T_W0, w0);
        tmem_park_words<C>(tmem + T_W1, w1);
        tmem_park_words<C>(tmem + T_W2, w2);
        tmem_wait_st();
    }
    mbar_wait(&s_bar, 0);
    __syncthreads();

    const int64_t k0 = p.k_begin + (int64_t)ch * p.chunk;
    const int64_t k1 = min(k0 + (int64_t)p.chunk, p.k_end);
    double best = -INFINITY;
    int64_t best_k = INT64_MAX;
    double* prow = p.pgram ? p.pgram + (rec.obj - p.pgram_row0) * p.pgram_row_stride - p.pgram_k0 : nullptr;
    double stash = 0.0;
    int64_t kb = k0;

    for (int64_t k = k0; k < k1; k++) {
        const double f = freq_of(p.f_min, p.df, k);
        bool bad_sort = false;     // per thread: a tie or an order this path cannot settle

        // ---- P1 fold + 32-bit keys; P2 sort
        unsigned key[C];
#pragma unroll
        for (int s = 0; s < C; s++) {
            const int i = tid + NT * s;
            unsigned kk = 0xffffffffu;
            if (i < n)
                kk = (__double2uint_rz(fold_phase(o_tt[i], f) * (double)(1u << (32 - Cfg::IDX_BITS))) << Cfg::IDX_BITS) | (unsigned)i;
            key[s] = kk;
        }
        group_sort<G, C>(key, tid, kbuf);

        // ---- exact phases in the sorted order; order repair inside a quantisation bucket (keys that agree in all
        // the phase bits kept sit in index order): one adjacent swap settles a bucket of two
        double phi[C];
        int idx[C];
#pragma unroll
        for (int s = 0; s < C; s++) {
            idx[s] = (int)(key[s] & Cfg::IDX_MASK);
            phi[s] = (tid * C + s < n) ? fold_phase(o_tt[idx[s]], f) : 4.0 + (double)s;
        }
#pragma unroll
        for (int s = 0; s + 1 < C; s++) {
            if (phi[s + 1] < phi[s]) {
                const double tp = phi[s]; phi[s] = phi[s + 1]; phi[s + 1] = tp;
                const int ti = idx[s]; idx[s] = idx[s + 1]; idx[s + 1] = ti;
            }
        }
        if (lane == 0) { s_edge[0][warp][0] = phi[0]; s_edge[0][warp][1] = (double)idx[0]; }
        if (lane == 31) { s_edge[1][warp + 1][0] = phi[C - 1]; s_edge[1][warp + 1][1] = (double)idx[C - 1]; }
        __syncthreads();                                                                    // BAR 1
        {
            double nphi = shfl_down_d(phi[0], 1), pphi = shfl_up_d(phi[C - 1], 1);
            int nidx = __shfl_down_sync(0xffffffffu, idx[0], 1), pidx = __shfl_up_sync(0xffffffffu, idx[C - 1], 1);
            if (lane == 31) { nphi = s_edge[0][warp + 1][0]; nidx = (int)s_edge[0][warp + 1][1]; }      // last warp: 1e3
            if (lane == 0) { pphi = s_edge[1][warp][0]; pidx = (int)s_edge[1][warp][1]; }               // first warp: -1
            // both sides of a boundary see the same two phases and take the same decision
            const bool swap_next = nphi < phi[C - 1], swap_prev = phi[0] < pphi;
            if (tid * C + C - 1 < n && nphi == phi[C - 1]) bad_sort = true;                     // exact tie (R24): generic path
            if (swap_next) { phi[C - 1] = nphi; idx[C - 1] = nidx; }
            if (swap_prev) { phi[0] = pphi; idx[0] = pidx; }
        }
#pragma unroll
        for (int s = 0; s + 1 < C; s++)
            if (tid * C + s + 1 < n && phi[s + 1] <= phi[s]) bad_sort = true;                   // tie, or a bucket of three

        // ---- gather; x centred by 0.5, padded slots carry x = 0, y = 0, w = W_PAD; quartile phases for
        // vsmlsq
        T x[C], y[C], w[C];
#pragma unroll
        for (int s = 0; s < C; s++) {
            if (tid * C + s < n) {
                x[s] = (T)(phi[s] - 0.5);
                if constexpr (!YW_GLOBAL) { y[s] = (T)o_y[idx[s]]; w[s] = (T)o_w[idx[s]]; }
            } else { x[s] = (T)0; y[s] = (T)0; w[s] = RT::wpad(); }
        }
        if (tid == K.q1t) {
#pragma unroll
            for (int s = 0; s < C; s++) if (s == K.q1s) s_q[0] = phi[s];
        }
        if (tid == K.q3t) {
#pragma unroll
            for (int s = 0; s < C; s++) if (s == K.q3s) s_q[1] = phi[s];
        }

        // ---- the smoother, once per object of the work item (one object unless the time sampling is shared)
        for (int m = 0; m < (SH ? mcnt : 1); m++) {
        bool bad = bad_sort;
        const int rim = SH ? s_ri[m] : ri;
        if constexpr (YW_GLOBAL) {      // gather of this object's y and w from the catalog copy
            const long long om = SH ? s_off[m] : (long long)rec.off;
#pragma unroll
            for (int s = 0; s < C; s++)
                if (tid * C + s < n) { y[s] = (T)__ldg(p.yc + om + idx[s]); w[s] = (T)__ldg(p.w + om + idx[s]); }
        }

        // ---- prefix sums of the weighted moments
        T ma[C], mb[C], mc[C], md[C], me[C];
#pragma unroll
        for (int s = 0; s < C; s++) {
            ma[s] = w[s]; mb[s] = w[s] * x[s]; mc[s] = mb[s] * x[s]; md[s] = w[s] * y[s]; me[s] = mb[s] * y[s];
        }
        const PairScan ps0 = pair_scan_begin<C>(ma, mb, s_tot[0], warp, lane, mk);
        const PairScan ps1 = pair_scan_begin<C>(mc, md, s_tot[1], warp, lane, mk);
        PairScan ps2; OneScan os2;
        T mf[C];
        if (GV) {
#pragma unroll
            for (int s = 0; s < C; s++) mf[s] = md[s] * y[s];
            ps2 = pair_scan_begin<C>(me, mf, s_tot[2], warp, lane, mk);
        } else {
            os2 = one_scan_begin<C>(me, reinterpret_cast<double*>(s_tot[2]), warp, lane, mk);
        }
        bad = __syncthreads_or(bad);                                                        // BAR 2 (also: sort buffers dead)
        if (bad) {
            if (tid == 0) {
                const unsigned pos = atomicAdd(p.defer_count, 1u);
                if (pos < p.defer_capacity)
                    p.defer_entries[pos] = ((unsigned long long)rim << 32) | (unsigned long long)(k - p.k_begin);
                else
                    p.defer_count[1] = 1u;
            }
        }
        double P = 0.0;
        if (!bad) {
            pair_scan_finish<G, C, T>(ps0, ma, mb, s_tot[0], E01, warp, tid);
            pair_scan_finish<G, C, T>(ps1, mc, md, s_tot[1], E23, warp, tid);
            if (GV) pair_scan_finish<G, C, T>(ps2, me, mf, s_tot[2], E45, warp, tid);
            else one_scan_finish<G, C, T>(os2, me, reinterpret_cast<const double*>(s_tot[2]), reinterpret_cast<T*>(E45), warp, tid);
            const double scale = s_q[1] - s_q[0];
            const T vsmlsq = (T)(1.e-6 * scale * scale);
            __syncthreads();                                                                // BAR 3
            T chi2 = (T)0;
            if constexpr (OPT == 2) {
                // ---- fixed span: one smooth of y over the caller's window
                const T* E4 = reinterpret_cast<const T*>(E45);
                int wi[CE];
                tmem_fetch_words<CE>(tmem + T_W0, wi);
#pragma unroll
                for (int s = 0; s < C; s++) {
                    const int a_ = wi[s] & 0xffff, b_ = (int)((unsigned)wi[s] >> 16);
                    const T2 l0 = E01[a_], h0 = E01[b_], l1 = E23[a_], h1 = E23[b_];
                    T Sw = h0.x - l0.x, Swx = h0.y - l0.y, Swxx = h1.x - l1.x, Sy = h1.y - l1.y;
                    T Sxy = E4[b_] - E4[a_];
                    const Wrap wr = wrapped(tid * C + s, ibw0);
                    if (__any_sync(0xffffffffu, wr.sg != 0)) {      // warp-uniform; lanes that do not wrap read element 0 twice: + 0
                        const int blo = wr.blo, bhi = wr.bhi;
                        const T sh = (T)wr.sg;
                        const T2 p0 = E01[blo], q0 = E01[bhi], p1 = E23[blo], q1 = E23[bhi];
                        const T bw = q0.x - p0.x, bwx = q0.y - p0.y, by = q1.y - p1.y;
                        Sw += bw; Swx += bwx + sh * bw; Swxx += (q1.x - p1.x) + ((T)2 * sh * bwx + bw);
                        Sy += by; Sxy += (E4[bhi] - E4[blo]) + sh * by;
                    }
                    const T isw = RT::rcp(Sw), xb = Swx * isw;
                    const T sxx = Swxx - xb * Swx;
                    const T isxx = sxx > vsmlsq ? RT::rcp(sxx) : (T)0;
                    const T smo = Sy * isw + (Sxy - xb * Sy) * (isxx * (x[s] - xb));
                    const T r = y[s] - smo;
                    chi2 += w[s] * r * r;
                }
            } else if (GV) {
                // ---- O6: three windows, scores, pick, interpolate
                T A[3][C], Gs[3][C];
#pragma unroll
                for (int i = 0; i < 3; i++) {
                    int wi[CE];
                    tmem_fetch_words<CE>(tmem + T_W0 + CE * i, wi);
#pragma unroll
                    for (int s = 0; s < C; s++) {
                        const int a_ = wi[s] & 0xffff, b_ = (int)((unsigned)wi[s] >> 16);
                        const T2 l0 = E01[a_], h0 = E01[b_], l1 = E23[a_], h1 = E23[b_], l2 = E45[a_], h2 = E45[b_];
                        T Sw = h0.x - l0.x, Swx = h0.y - l0.y, Swxx = h1.x - l1.x, Sy = h1.y - l1.y;
                        T Sxy = h2.x - l2.x, Syy = h2.y - l2.y;
                        if constexpr (LOPT) {
                            const Wrap wr = wrapped(tid * C + s, i == 0 ? ibw0 : (i == 1 ? ibw1 : ibw2));
                            if (__any_sync(0xffffffffu, wr.sg != 0)) {      // warp-uniform; lanes that do not wrap read element 0 twice: + 0
                                const int blo = wr.blo, bhi = wr.bhi;
                                const T sh = (T)wr.sg;
                                const T2 p0 = E01[blo], q0 = E01[bhi], p1 = E23[blo], q1 = E23[bhi], p2 = E45[blo], q2 = E45[bhi];
                                const T bw = q0.x - p0.x, bwx = q0.y - p0.y, by = q1.y - p1.y;
                                Sw += bw; Swx += bwx + sh * bw; Swxx += (q1.x - p1.x) + ((T)2 * sh * bwx + bw);
                                Sy += by; Sxy += (q2.x - p2.x) + sh * by; Syy += q2.y - p2.y;
                            }
                        }
                        const T isw = RT::rcp(Sw), xb = Swx * isw;
                        const T sxx = Swxx - xb * Swx;
                        const T isxx = sxx > vsmlsq ? RT::rcp(sxx) : (T)0;
                        const T yb = Sy * isw, sxy = Sxy - xb * Sy, b = sxy * isxx;
                        A[i][s] = yb + b * (x[s] - xb);
                        const T rss = (Syy - yb * Sy) - b * sxy;
                        Gs[i][s] = RT::sqrt0(rss * isw) * (isxx != (T)0 ? (T)K.kc[2 * i + 1] : (T)K.kc[2 * i]);
                    }
                }
#pragma unroll
                for (int s = 0; s < C; s++) {
                    const T sp = pick_span_t<T>(Gs[0][s], Gs[1][s], Gs[2][s], K.bass, K.bexp);
                    const T smo = interp_spans_t<T>(sp, A[0][s], A[1][s], A[2][s]);
                    const T r = y[s] - smo;
                    chi2 += w[s] * r * r;
                }
            } else {
                // ---- CV pass 1: one span at a time; smooths parked in tensor memory
                T r0[C], r1[C], r2[C];
                T m_isw[C], m_xb[C], m_g[C];
                const T* E4 = reinterpret_cast<const T*>(E45);
                int amin = 0x7fffffff;
#pragma unroll
                for (int i = 0; i < 3; i++) {
                    int wi[CE];
                    tmem_fetch_words<CE>(tmem + T_W0 + CE * i, wi);
                    T Ai[C], q_isw[C], q_xb[C], q_g[C];
#pragma unroll
                    for (int s = 0; s < C; s++) {
                        const int a_ = wi[s] & 0xffff, b_ = (int)((unsigned)wi[s] >> 16);
                        const T2 l0 = E01[a_], h0 = E01[b_], l1 = E23[a_], h1 = E23[b_];
                        const T lxy = E4[a_], hxy = E4[b_];
                        T Sw = h0.x - l0.x, Swx = h0.y - l0.y, Swxx = h1.x - l1.x, Sy = h1.y - l1.y;
                        T Sxy = hxy - lxy;
                        if constexpr (LOPT) {
                            const Wrap wr = wrapped(tid * C + s, i == 0 ? ibw0 : (i == 1 ? ibw1 : ibw2));
                            if (__any_sync(0xffffffffu, wr.sg != 0)) {      // warp-uniform; lanes that do not wrap read element 0 twice: + 0
                                const int blo = wr.blo, bhi = wr.bhi;
                                const T sh = (T)wr.sg;
                                const T2 p0 = E01[blo], q0 = E01[bhi], p1 = E23[blo], q1 = E23[bhi];
                                const T bw = q0.x - p0.x, bwx = q0.y - p0.y, by = q1.y - p1.y;
                                Sw += bw; Swx += bwx + sh * bw; Swxx += (q1.x - p1.x) + ((T)2 * sh * bwx + bw);
                                Sy += by; Sxy += (E4[bhi] - E4[blo]) + sh * by;
                            }
                        }
                        const T isw = RT::rcp(Sw), xb = Swx * isw;
                        const T sxx = Swxx - xb * Swx;
                        const T isxx = sxx > vsmlsq ? RT::rcp(sxx) : (T)0;
                        const T dx = x[s] - xb, g = isxx * dx;
                        q_isw[s] = isw; q_xb[s] = xb; q_g[s] = g;
                        Ai[s] = Sy * isw + (Sxy - xb * Sy) * g;
                        const T a = (T)1 - w[s] * (isw + dx * g);
                        const T r = (T)fabs(y[s] - Ai[s]) * RT::rcp(a);
                        if (i == 0) r0[s] = r; else if (i == 1) r1[s] = r; else r2[s] = r;
                        amin = min(amin, RT::hi_word(a));
                    }
                    TA::park(tmem + T_A0 + PC * i, Ai);
                    if (i == 0) { TA::park(tmem + T_ISW, q_isw); TA::park(tmem + T_XB, q_xb); TA::park(tmem + T_G0, q_g); }
                    if (i == 1) {
#pragma unroll
                        for (int s = 0; s < C; s++) { m_isw[s] = q_isw[s]; m_xb[s] = q_xb[s]; m_g[s] = q_g[s]; }
                    }
                }
                TA::park(tmem + T_Y, y);
                // ---- pass 2: the three residuals smoothed at the midrange span
                T za[C], zb[C], zc[C], zd[C], ze[C], zf[C];
#pragma unroll
                for (int s = 0; s < C; s++) {
                    za[s] = w[s] * r0[s]; zb[s] = za[s] * x[s];
                    zc[s] = w[s] * r1[s]; zd[s] = zc[s] * x[s];
                    ze[s] = w[s] * r2[s]; zf[s] = ze[s] * x[s];
                }
                const PairScan qs0 = pair_scan_begin<C>(za, zb, s_tot[0], warp, lane, mk);
                const PairScan qs1 = pair_scan_begin<C>(zc, zd, s_tot[1], warp, lane, mk);
                const PairScan qs2 = pair_scan_begin<C>(ze, zf, s_tot[2], warp, lane, mk);
                // a <= 0 (or below the smallest normal): the residual carries (R23) -> generic path
                const bool carry = __syncthreads_or(amin < RT::TINY);                    // BAR 4 (primary arrays dead)
                if (carry) {
                    if (tid == 0) {
                        const unsigned pos = atomicAdd(p.defer_count, 1u);
                        if (pos < p.defer_capacity)
                            p.defer_entries[pos] = ((unsigned long long)rim << 32) | (unsigned long long)(k - p.k_begin);
                        else
                            p.defer_count[1] = 1u;
                    }
                    bad = true;
                } else {
                    pair_scan_finish<G, C, T>(qs0, za, zb, s_tot[0], E01, warp, tid);
                    pair_scan_finish<G, C, T>(qs1, zc, zd, s_tot[1], E23, warp, tid);
                    pair_scan_finish<G, C, T>(qs2, ze, zf, s_tot[2], E45, warp, tid);
                    __syncthreads();                                                        // BAR 5
                    int w1i[CE];
                    tmem_fetch_words<CE>(tmem + T_W1, w1i);
                    auto mid_load = [&](const T2* Ez, T (&out)[C]) {
#pragma unroll
                        for (int s = 0; s < C; s++) {
                            const T2 l = Ez[w1i[s] & 0xffff], h = Ez[(unsigned)w1i[s] >> 16];
                            T Sz = h.x - l.x, Sxz = h.y - l.y;
                            if constexpr (LOPT) {
                                const Wrap wr = wrapped(tid * C + s, ibw1);
                                if (__any_sync(0xffffffffu, wr.sg != 0)) {      // warp-uniform; lanes that do not wrap read element 0 twice: + 0
                                    const int blo = wr.blo, bhi = wr.bhi;
                                    const T sh = (T)wr.sg;
                                    const T2 pz = Ez[blo], qz = Ez[bhi];
                                    const T bz = qz.x - pz.x;
                                    Sz += bz; Sxz += (qz.y - pz.y) + sh * bz;
                                }
                            }
                            out[s] = Sz * m_isw[s] + (Sxz - m_xb[s] * Sz) * m_g[s];
                        }
                    };
                    T sp[C];
                    {
                        T R0[C], R1[C], R2[C];
                        mid_load(E01, R0); mid_load(E23, R1); mid_load(E45, R2);
#pragma unroll
                        for (int s = 0; s < C; s++) sp[s] = pick_span_t<T>(R0[s], R1[s], R2[s], K.bass, K.bexp);
                    }
                    // ---- the spans smoothed at midrange
#pragma unroll
                    for (int s = 0; s < C; s++) { za[s] = w[s] * sp[s]; zb[s] = za[s] * x[s]; }
                    const PairScan ss0 = pair_scan_begin<C>(za, zb, s_tot[0], warp, lane, mk);
                    __syncthreads();                                                        // BAR 6 (residual arrays dead)
                    pair_scan_finish<G, C, T>(ss0, za, zb, s_tot[0], E01, warp, tid);
                    __syncthreads();                                                        // BAR 7
                    T B[C];
                    mid_load(E01, B);
                    tmem_wait_st();
                    {
                        T a0[C], a1[C], a2[C];
                        TA::fetch(tmem + T_A0, a0); TA::fetch(tmem + T_A1, a1); TA::fetch(tmem + T_A2, a2);
#pragma unroll
                        for (int s = 0; s < C; s++) B[s] = interp_spans_t<T>(B[s], a0[s], a1[s], a2[s]);
                    }
                    // ---- final tweeter smooth
#pragma unroll
                    for (int s = 0; s < C; s++) { zc[s] = w[s] * B[s]; zd[s] = zc[s] * x[s]; }
                    const PairScan fs0 = pair_scan_begin<C>(zc, zd, s_tot[1], warp, lane, mk);
                    __syncthreads();                                                        // BAR 8
                    pair_scan_finish<G, C, T>(fs0, zc, zd, s_tot[1], E23, warp, tid);
                    __syncthreads();                                                        // BAR 9
                    int w0i[CE];
                    tmem_fetch_words<CE>(tmem + T_W0, w0i);
                    T t_isw[C], t_xb[C], t_g[C], yy[C];
                    TA::fetch(tmem + T_ISW, t_isw); TA::fetch(tmem + T_XB, t_xb); TA::fetch(tmem + T_G0, t_g);
                    TA::fetch(tmem + T_Y, yy);
#pragma unroll
                    for (int s = 0; s < C; s++) {
                        const T2 l = E23[w0i[s] & 0xffff], h = E23[(unsigned)w0i[s] >> 16];
                        T Sz = h.x - l.x, Sxz = h.y - l.y;
                        if constexpr (LOPT) {
                            const Wrap wr = wrapped(tid * C + s, ibw0);
                            if (__any_sync(0xffffffffu, wr.sg != 0)) {      // warp-uniform; lanes that do not wrap read element 0 twice: + 0
                                const int blo = wr.blo, bhi = wr.bhi;
                                const T sh = (T)wr.sg;
                                const T2 pz = E23[blo], qz = E23[bhi];
                                const T bz = qz.x - pz.x;
                                Sz += bz; Sxz += (qz.y - pz.y) + sh * bz;
                            }
                        }
                        const T smo = Sz * t_isw[s] + (Sxz - t_xb[s] * Sz) * t_g[s];
                        const T r = yy[s] - smo;
                        chi2 += w[s] * r * r;
                    }
                }
            }
            if (!bad) {
                double chi2d = (double)chi2;
#pragma unroll
                for (int d = 16; d > 0; d >>= 1) chi2d += __shfl_xor_sync(0xffffffffu, chi2d, d);
                if (lane == 0) s_red[warp] = chi2d;
                __syncthreads();                                                            // BAR 10
                double c2 = 0.0;
#pragma unroll
                for (int q = 0; q < G; q++) c2 += s_red[q];
                P = SH ? (s_chi[m][0] - c2) * s_chi[m][1] : (K.kc[6] - c2) * K.kc[7];
            }
        }
        // thread m keeps object m's best; thread 32 m + i stashes its i-th value of the current batch of 32
        if ((!SH || tid == m) && !bad && P > best) { best = P; best_k = k; }
        if (tid == 32 * m + (int)(k - kb)) stash = bad ? 0.0 : P;      // a handed-over eval is patched by the generic kernel
        }      // objects of the work item
        if (k - kb == 31 || k == k1 - 1) {
            if constexpr (SH) {
                if (tid < 32 * mcnt) {
                    double* pr = s_prow[tid >> 5];
                    if (pr && kb + lane <= k) pr[kb + lane] = stash;
                }
            } else {
                if (prow && tid < 32 && kb + tid <= k) prow[kb + tid] = stash;
            }
            kb = k + 1;
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(s_tmem), "n"(Cfg::TCOLS) : "memory");
    }
    if (SH ? tid < mcnt : tid == 0) {
        const int64_t slot = (int64_t)(SH ? s_ri[tid] : ri) * p.chunks_total + p.chunk_base + ch;
        p.part_val[slot] = best;
        p.part_idx[slot] = best_k == INT64_MAX ? k0 : best_k;
    }
}

template <int G, int C, bool GV, typename T = double, int OPT = 0>
inline ss_status_t launch_group_variant(const EvalParams& p, int64_t n_items, cudaStream_t stream)
{
    const size_t smem = group_smem_bytes<G, C, GV, T>();
    if (cudaFuncSetAttribute(group_kernel<G, C, GV, T, OPT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
        return SS_ERR_CUDA;
    group_kernel<G, C, GV, T, OPT><<<(unsigned)n_items, GroupCfg<G, C, T>::NT, smem, stream>>>(p);
    return cudaGetLastError() == cudaSuccess ? SS_OK : SS_ERR_CUDA;
}

}  // namespace ss

// ss_block_kernel.cuh -- one CTA per (object, frequency) eval; any n.
//
// Serves the SS_PATH_BLOCK (per-eval arrays in shared memory) and SS_PATH_STAGE (arrays staged in
// global memory / L2, for light curves that do not fit one SM's shared memory) classes.  Persistent
// CTAs pull (object, frequency-chunk) work items from an atomic counter, longest objects first.
//
// Per eval: fold -> bitonic sort of (phase bits, index) -> gather ->
// exclusive prefix sums of the weighted moments -> windowed line fits by prefix differences
// (three spans) -> CV: LOO residuals, residual smooths, span pick, span smooth, interpolation, final
// smooth (Listing 1) / GV: scores, pick, interpolation (R12) -> chi2 -> P.
#pragma once
#include "ss_common.cuh"

namespace ss {

template <int T>
struct BlockCtx {
    static constexpr int NW = T / 32;
    double (*wsum)[NW];   // [6][NW] cross-warp scan scratch
    double* red;          // [NW]
    int* flags;           // [4]: has_ties, bad0, bad1, bad2
};

// Exclusive prefix sums of NA value streams at once; E[a][0..n], E[a][n] = total.
// Blocked: a thread owns SCAN_CB consecutive elements (odd, so its 64-bit accesses at stride SCAN_CB
// are bank-conflict free), sums them in registers, and the warp runs ONE Kogge-Stone per stream for
// 32*SCAN_CB elements.
constexpr int SCAN_CB = 5;
template <int T, int NA, typename F>
__device__ __forceinline__ void block_scan(int n, F vals, double* const (&E)[NA], double (*wsum)[T / 32])
{
    constexpr int NW = T / 32;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    double carry[NA];
#pragma unroll
    for (int a = 0; a < NA; a++) carry[a] = 0.0;
    for (int base = 0; base < n; base += T * SCAN_CB) {
        const int j0 = base + tid * SCAN_CB;
        double v[SCAN_CB][NA], run[NA], inc[NA];
#pragma unroll
        for (int a = 0; a < NA; a++) run[a] = 0.0;
#pragma unroll
        for (int s = 0; s < SCAN_CB; s++) {
            if (j0 + s < n) vals(j0 + s, v[s]);
            else {
#pragma unroll
                for (int a = 0; a < NA; a++) v[s][a] = 0.0;
            }
#pragma unroll
            for (int a = 0; a < NA; a++) run[a] += v[s][a];
        }
#pragma unroll
        for (int a = 0; a < NA; a++) {
            double t = run[a];
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                double o = __shfl_up_sync(0xffffffffu, t, d);
                if (lane >= d) t += o;
            }
            inc[a] = t;
            if (lane == 31) wsum[a][warp] = t;
        }
        __syncthreads();
#pragma unroll
        for (int a = 0; a < NA; a++) {
            // every warp scans the NW warp sums itself (lane q holds warp q's sum): no second barrier
            static_assert(NW <= 32, "one lane per warp sum");
            const double mine = lane < NW ? wsum[a][lane] : 0.0;
            double sc = mine;
#pragma unroll
            for (int d = 1; d < NW; d <<= 1) {
                double o = __shfl_up_sync(0xffffffffu, sc, d);
                if (lane >= d) sc += o;
            }
            const double woff = __shfl_sync(0xffffffffu, sc - mine, warp);
            const double tot = __shfl_sync(0xffffffffu, sc, NW - 1);
            double out = carry[a] + woff + (inc[a] - run[a]);
#pragma unroll
            for (int s = 0; s < SCAN_CB; s++) {
                if (j0 + s < n) E[a][j0 + s] = out;
                out += v[s][a];
            }
            carry[a] += tot;
        }
        __syncthreads();
    }
    if (tid == 0) {
#pragma unroll
        for (int a = 0; a < NA; a++) E[a][n] = carry[a];
    }
    __syncthreads();
}

template <int T>
__device__ __forceinline__ double block_sum(double v, double* red)
{
    constexpr int NW = T / 32;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    __syncthreads();
    if (lane == 0) red[warp] = v;
    __syncthreads();
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < NW; q++) s += red[q];
    return s;
}

// Replace the -1 sentinels of the LOO residuals by the previous valid value (R23).
__device__ inline void carry_fix_serial(int n, double* r)
{
    for (int j = 0; j < n; j++)
        if (r[j] < 0.0) r[j] = j > 0 ? r[j - 1] : 0.0;
}

// Compare-exchange on (key, idx), ascending, lexicographic: exact stable order (R13).
__device__ __forceinline__ void cex(unsigned long long* key, unsigned int* idx, int a, int b)
{
    unsigned long long ka = key[a], kb = key[b];
    unsigned int ia = idx[a], ib = idx[b];
    if (kb < ka || (kb == ka && ib < ia)) {
        key[a] = kb; key[b] = ka;
        idx[a] = ib; idx[b] = ia;
    }
}

// ---- fast sort: packed 32-bit keys (quantised phase | index) in registers --------------------------
// S keys per thread, blocked (position = tid*S + s).  Warp-local phases run on registers and shuffles,
// only the log2(NW)*(log2(NW)+1)/2 cross-warp steps go through shared memory.  A key keeps the top
// 32 - IDX_BITS bits of the phase, so the network leaves the points in exact order except inside a
// quantisation bucket (phases that agree in all the bits kept: a pair every few evals), where they sit
// in index order; block_eval restores the exact order there by odd-even transposition on the full
// 64-bit phases, and falls back to the exact network if that does not settle.  A 32-bit key costs one
// shuffle and one min/max per exchange where the 64-bit key cost two shuffles and a compare-select chain.
template <int T> struct FastKey {
    static constexpr int IDX_BITS = T <= 128 ? 10 : (T <= 256 ? 11 : 12);      // log2(8 T) positions
    static constexpr unsigned IDX_MASK = (1u << IDX_BITS) - 1u;
    static constexpr double PHASE_SCALE = (double)(1u << (32 - IDX_BITS));
};

// the halving steps of one merge phase inside a warp: lane strides 16..1, then register strides S/2..1
template <int S>
__device__ __forceinline__ void merge_tail32(unsigned (&key)[S], int lane, int first_lane_stride)
{
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) {
        if (m > first_lane_stride) continue;
        const bool lower = (lane & m) == 0;
#pragma unroll
        for (int s = 0; s < S; s++) {
            const unsigned o = __shfl_xor_sync(0xffffffffu, key[s], m);
            key[s] = lower ? min(key[s], o) : max(key[s], o);
        }
    }
#pragma unroll
    for (int j = S >> 1; j >= 1; j >>= 1) {
#pragma unroll
        for (int s = 0; s < S; s++)
            if ((s & j) == 0) {
                const unsigned lo = min(key[s], key[s + j]), hi = max(key[s], key[s + j]);
                key[s] = lo; key[s + j] = hi;
            }
    }
}

// sorts the 32*S keys of each warp ascending (blocked within the warp: position = lane*S + s)
template <int S>
__device__ __forceinline__ void warp_sort32(unsigned (&key)[S], int lane)
{
#pragma unroll
    for (int k = 2; k <= 32 * S; k <<= 1) {
        if (k <= S) {
#pragma unroll
            for (int s = 0; s < S; s++) {
                const int t = s ^ (k - 1);
                if (t > s) {
                    const unsigned lo = min(key[s], key[t]), hi = max(key[s], key[t]);
                    key[s] = lo; key[t] = hi;
                }
            }
#pragma unroll
            for (int j = k >> 2; j >= 1; j >>= 1) {
#pragma unroll
                for (int s = 0; s < S; s++)
                    if ((s & j) == 0) {
                        const unsigned lo = min(key[s], key[s + j]), hi = max(key[s], key[s + j]);
                        key[s] = lo; key[s + j] = hi;
                    }
            }
        } else {
            const int m = k / S - 1;               // lane mask of the mirror step
            const bool lower = (lane & (k / S / 2)) == 0;
            unsigned other[S];
#pragma unroll
            for (int s = 0; s < S; s++) other[s] = __shfl_xor_sync(0xffffffffu, key[S - 1 - s], m);
#pragma unroll
            for (int s = 0; s < S; s++) key[s] = lower ? min(key[s], other[s]) : max(key[s], other[s]);
            merge_tail32<S>(key, lane, k / S / 4);
        }
    }
}

// Whole-CTA sort; writes the (bucket-exact) sorted permutation idx[0..n).  kbuf: T*S words of exchange space.
template <int T, int S>
__device__ __forceinline__ void block_sort_fast(int n, const double* tt, double f, unsigned* kbuf, unsigned int* idx)
{
    constexpr int NW = T / 32;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    unsigned key[S];
#pragma unroll
    for (int s = 0; s < S; s++) {
        const int i = tid + T * s;
        key[s] = 0xffffffffu;
        if (i < n)
            key[s] = (__double2uint_rz(fold_phase(tt[i], f) * FastKey<T>::PHASE_SCALE) << FastKey<T>::IDX_BITS) | (unsigned)i;
    }
    warp_sort32<S>(key, lane);
#pragma unroll
    for (int kw = 2; kw <= NW; kw <<= 1) {
        // mirror step across warps: partner position = pos ^ (kw*32*S - 1)
        {
            const int ptid = ((warp ^ (kw - 1)) << 5) + (31 - lane);
            const bool lower = (warp & (kw >> 1)) == 0;
#pragma unroll
            for (int s = 0; s < S; s++) kbuf[s * T + tid] = key[s];
            __syncthreads();
#pragma unroll
            for (int s = 0; s < S; s++) {
                const unsigned o = kbuf[(S - 1 - s) * T + ptid];
                key[s] = lower ? min(key[s], o) : max(key[s], o);
            }
            __syncthreads();
        }
#pragma unroll
        for (int jw = kw >> 2; jw >= 1; jw >>= 1) {
            const int ptid = ((warp ^ jw) << 5) + lane;
            const bool lower = (warp & jw) == 0;
#pragma unroll
            for (int s = 0; s < S; s++) kbuf[s * T + tid] = key[s];
            __syncthreads();
#pragma unroll
            for (int s = 0; s < S; s++) {
                const unsigned o = kbuf[s * T + ptid];
                key[s] = lower ? min(key[s], o) : max(key[s], o);
            }
            __syncthreads();
        }
        merge_tail32<S>(key, lane, 16);
    }
#pragma unroll
    for (int s = 0; s < S; s++) {
        const int pos = tid * S + s;
        if (pos < n) idx[pos] = key[s] & FastKey<T>::IDX_MASK;
    }
}

// Window of point j as ranges of the prefix arrays (O4).  Non-periodic (jper = 1): [lo, hi) =
// the K points centred on j, pinned at the ends.  Periodic (jper = 2, only with OPT):
// j-ibw .. j+ibw modulo n -- the part inside [0, n) is [lo, hi), the part that wrapped is [blo, bhi)
// and its abscissae count as x + s, s = -1 (wrapped below 0) or +1 (wrapped above n-1).
template <bool OPT>
struct Win {
    int lo, hi, blo, bhi;
    double s;
    __device__ __forceinline__ Win(int j, int ibw, int K, int n, bool per)
    {
        blo = bhi = 0; s = 0.0;
        if (OPT && per) {
            lo = j - ibw; hi = j + ibw + 1;
            if (lo < 0) { blo = lo + n; bhi = n; lo = 0; s = -1.0; }
            else if (hi > n) { bhi = hi - n; hi = n; s = 1.0; }
        } else {
            lo = window_lo(j, ibw, K, n);
            hi = lo + K;
        }
    }
    __device__ __forceinline__ double wrapped(const double* E) const { return OPT ? E[bhi] - E[blo] : 0.0; }
    __device__ __forceinline__ double sum(const double* E) const
    {
        double v = E[hi] - E[lo];
        if (OPT) v += E[bhi] - E[blo];
        return v;
    }
    // sum w x^q over the window, q = 0, 1, 2, with the wrapped part shifted by s
    __device__ __forceinline__ XMom xmom(const double* Ew, const double* Ewx, const double* Ewxx, double vsmlsq) const
    {
        double Sw = sum(Ew), Swx = sum(Ewx), Swxx = sum(Ewxx);
        if (OPT) {
            const double bw = wrapped(Ew), bwx = wrapped(Ewx);
            Swx += s * bw;
            Swxx += 2.0 * s * bwx + bw;      // s*s = 1 where bw != 0
        }
        return x_moments(Sw, Swx, Swxx, vsmlsq);
    }
    // sum w z and sum w x z over the window
    __device__ __forceinline__ void zmom(const double* Ewz, const double* Ewxz, double& Swz, double& Swxz) const
    {
        Swz = sum(Ewz); Swxz = sum(Ewxz);
        if (OPT) Swxz += s * wrapped(Ewz);
    }
};

// One eval.  S = base of BLOCK_SLOTS arrays of `sl` doubles (shared or global memory).
// OPT = true adds the options Listing 1 has beside the default call: periodic windows (p.iper = 2)
// and a fixed span (p.span > 0); the default instantiation carries none of that code.
// Returns P (valid in every thread).  If smo_dbg != null the smooth (phase order, un-centred) and the
// permutation are written out (ss_debug_eval).
template <int T, bool OPT>
__device__ double block_eval(const EvalParams& p, const ObjRec& rec, double f, double* S, int64_t sl,
                             const BlockCtx<T>& cx, double* smo_dbg, int32_t* perm_dbg)
{
    const int tid = threadIdx.x;
    const int n = rec.n;
    const double* tt = p.tt + rec.off;
    const double* yc = p.yc + rec.off;
    const double* wo = p.w + rec.off;

    double* x = S;                 double* ys = S + sl;           double* ws = S + 2 * sl;
    double* Ew = S + 3 * sl;       double* Ewx = S + 4 * sl;      double* Ewxx = S + 5 * sl;
    double* Ewy = S + 6 * sl;      double* Ewxy = S + 7 * sl;
    double* A0 = S + 8 * sl;       double* A1 = S + 9 * sl;       double* A2 = S + 10 * sl;
    double* r0 = S + 11 * sl;      double* r1 = S + 12 * sl;      double* r2 = S + 13 * sl;
    // sort scratch overlays slots that are dead until pass 1: exact keys / exchange buffer in r0..r1,
    // the sorted permutation in A2, the sorted phases in A0
    unsigned long long* key = reinterpret_cast<unsigned long long*>(r0);
    unsigned* kbuf = reinterpret_cast<unsigned*>(r0);
    unsigned int* idx = reinterpret_cast<unsigned int*>(A2);
    double* phi = A0;
    auto misordered = [&](int j) {      // exact stable order (R13): by phase, ties by input index
        return phi[j + 1] < phi[j] || (phi[j + 1] == phi[j] && idx[j + 1] < idx[j]);
    };

    // fast path: packed 32-bit keys in registers (S per thread); needs T*S exchange words inside r0..r1
    int fs = 0;
    if (n <= T * 8) {
        fs = 1;
        while (T * fs < n) fs <<= 1;
        if ((int64_t)T * fs > 4 * sl) fs = 0;
    }
    for (;;) {
        if (tid < 4) cx.flags[tid] = 0;
        if (fs == 1) block_sort_fast<T, 1>(n, tt, f, kbuf, idx);
        else if (fs == 2) block_sort_fast<T, 2>(n, tt, f, kbuf, idx);
        else if (fs == 4) block_sort_fast<T, 4>(n, tt, f, kbuf, idx);
        else if (fs == 8) block_sort_fast<T, 8>(n, tt, f, kbuf, idx);
        else {
            // ---- exact path: P1 fold + key init
            for (int j = tid; j < n; j += T) {
                key[j] = (unsigned long long)__double_as_longlong(fold_phase(tt[j], f));
                idx[j] = (unsigned int)j;
            }
            __syncthreads();
            // ---- P2 bitonic network for arbitrary n (all exchanges ascending; indices >= n act as +inf)
            int np2 = 1;
            while (np2 < n) np2 <<= 1;
            const int half = np2 >> 1;
            for (int lk = 1; (1 << (lk - 1)) < n; lk++) {
                const int k = 1 << lk, hk = k >> 1;           // strides are powers of two: shifts, no division
                for (int t = tid; t < half; t += T) {
                    int blk = t >> (lk - 1), o = t & (hk - 1);
                    int a = (blk << lk) + o, b = (blk << lk) + k - 1 - o;
                    if (b < n) cex(key, idx, a, b);
                }
                __syncthreads();
                for (int lj = lk - 2; lj >= 0; lj--) {
                    const int jj = 1 << lj;
                    for (int t = tid; t < half; t += T) {
                        int blk = t >> lj, o = t & (jj - 1);
                        int a = (blk << (lj + 1)) + o, b = a + jj;
                        if (b < n) cex(key, idx, a, b);
                    }
                    __syncthreads();
                }
            }
        }
        __syncthreads();
        // ---- the exact phases again, in the sorted order
        for (int j = tid; j < n; j += T) phi[j] = fold_phase(tt[idx[j]], f);
        __syncthreads();
        if (fs != 0) {
            // points whose phases share a quantisation bucket sit in index order: odd-even transposition on
            // the full phases puts them in exact order (a bucket of m points settles in m passes); buckets
            // that do not settle in 12 passes send the eval to the exact network
            bool settled = false;
            for (int it = 0; it < 6; it++) {
#pragma unroll
                for (int parity = 0; parity < 2; parity++) {
                    for (int j = 2 * tid + parity; j + 1 < n; j += 2 * T)
                        if (misordered(j)) {
                            const double pa = phi[j]; phi[j] = phi[j + 1]; phi[j + 1] = pa;
                            const unsigned ia = idx[j]; idx[j] = idx[j + 1]; idx[j + 1] = ia;
                            cx.flags[1] = it + 1;
                        }
                    __syncthreads();
                }
                if (cx.flags[1] != it + 1) { settled = true; break; }
                __syncthreads();      // everyone has read the stamp before the next pass may overwrite it
            }
            if (!settled) { fs = 0; __syncthreads(); continue; }
        }
        break;
    }
    // ---- gather: x centred by 0.5, y already centred by ybar_w
    for (int j = tid; j < n; j += T) {
        const unsigned int i = idx[j];
        x[j] = phi[j] - 0.5;
        ys[j] = yc[i];
        ws[j] = wo[i];
        if (perm_dbg) perm_dbg[j] = (int32_t)i;
        if (j + 1 < n && phi[j + 1] == phi[j]) cx.flags[0] = 1;              // tie: equal-x run averaging (R24)
    }
    __syncthreads();
    const bool has_ties = cx.flags[0] != 0;
    __syncthreads();
    if (tid == 1) cx.flags[1] = 0;

    double chi2_part = 0.0;
    const double phi_first = phi[0];
    const double phi_last = phi[n - 1];
    if (phi_last <= phi_first) {
        // Listing 1 lines 25-36: all phases equal -> weighted mean
        double sw = 0.0, sy = 0.0;
        for (int j = tid; j < n; j += T) { sw += ws[j]; sy += ws[j] * ys[j]; }
        sw = block_sum<T>(sw, cx.red);
        sy = block_sum<T>(sy, cx.red);
        double a = sw > 0.0 ? sy / sw : 0.0;
        for (int j = tid; j < n; j += T) {
            double r = ys[j] - a;
            chi2_part += ws[j] * r * r;
            if (smo_dbg) smo_dbg[j] = a + rec.ybar;
        }
        double chi2 = block_sum<T>(chi2_part, cx.red);
        return rec.chi0 > 0.0 ? (rec.chi0 - chi2) / rec.chi0 : 0.0;
    }
    const double scale = phi[rec.q3] - phi[rec.q1];
    const double vsmlsq = 1.e-6 * scale * scale;
    __syncthreads();                               // phi[] (in A0) and idx[] (in A2) are dead from here on

    const int ibw0 = rec.ibw[0], ibw1 = rec.ibw[1], ibw2 = rec.ibw[2];
    const int K0 = min(2 * ibw0 + 1, n), K1 = min(2 * ibw1 + 1, n), K2 = min(2 * ibw2 + 1, n);
    const bool per = OPT && p.iper == 2;           // phases are in [0,1): jper = iper
    const bool fixed = OPT && p.span > 0.0;
    const bool gv = p.mode == 1 && !fixed;

    // ---- P3: prefix sums of the weighted moments
    if (!gv) {
        double* const E[5] = {Ew, Ewx, Ewxx, Ewy, Ewxy};
        block_scan<T, 5>(n, [&](int j, double* v) {
            double w_ = ws[j], x_ = x[j], y_ = ys[j];
            v[0] = w_; v[1] = w_ * x_; v[2] = w_ * x_ * x_; v[3] = w_ * y_; v[4] = w_ * x_ * y_;
        }, E, cx.wsum);
    } else {
        double* const E[6] = {Ew, Ewx, Ewxx, Ewy, Ewxy, A0};
        block_scan<T, 6>(n, [&](int j, double* v) {
            double w_ = ws[j], x_ = x[j], y_ = ys[j];
            v[0] = w_; v[1] = w_ * x_; v[2] = w_ * x_ * x_; v[3] = w_ * y_; v[4] = w_ * x_ * y_;
            v[5] = w_ * y_ * y_;
        }, E, cx.wsum);
    }
    const double* Ewyy = A0;   // GV only

    // one running-line smooth of the stream whose prefix sums are (Ez, Exz), at half-width ibw
    auto fit_at = [&](int j, int ibw, int K, const double* Ez, const double* Exz) {
        const Win<OPT> wn(j, ibw, K, n, per);
        XMom m = wn.xmom(Ew, Ewx, Ewxx, vsmlsq);
        double Swz, Swxz, b, zb;
        wn.zmom(Ez, Exz, Swz, Swxz);
        return line_fit(m, Swz, Swxz, x[j], b, zb);
    };

    if (gv) {
        // ---- O6: one sweep, three windows, score, pick, interpolate
        double* smo = A1;
        for (int j = tid; j < n; j += T) {
            const double xj = x[j];
            double A[3], G[3];
            const int ib[3] = {ibw0, ibw1, ibw2}, KK[3] = {K0, K1, K2};
#pragma unroll
            for (int i = 0; i < 3; i++) {
                const Win<OPT> wn(j, ib[i], KK[i], n, per);
                XMom m = wn.xmom(Ew, Ewx, Ewxx, vsmlsq);
                double Swy, Swxy;
                wn.zmom(Ewy, Ewxy, Swy, Swxy);
                double b, yb;
                A[i] = line_fit(m, Swy, Swxy, xj, b, yb);
                G[i] = gv_score(m, Swy, Swxy, wn.sum(Ewyy), b, yb, KK[i]);
            }
            double sp = pick_span(G[0], G[1], G[2], p.alpha);
            smo[j] = interp_spans(sp, A[0], A[1], A[2]);
        }
        __syncthreads();
        if (has_ties) {
            if (tid == 0) {
                // re-derive ordered keys from x: ties in x <=> ties in key
                int j = 0;
                while (j < n) {
                    int j0 = j; double sy = smo[j] * ws[j], fbw = ws[j];
                    while (j < n - 1 && x[j + 1] <= x[j]) { j++; sy += ws[j] * smo[j]; fbw += ws[j]; }
                    if (j > j0) { double a = fbw > 0.0 ? sy / fbw : 0.0; for (int i = j0; i <= j; i++) smo[i] = a; }
                    j++;
                }
            }
            __syncthreads();
        }
        for (int j = tid; j < n; j += T) {
            double r = ys[j] - smo[j];
            chi2_part += ws[j] * r * r;
            if (smo_dbg) smo_dbg[j] = smo[j] + rec.ybar;
        }
        double chi2 = block_sum<T>(chi2_part, cx.red);
        return rec.chi0 > 0.0 ? (rec.chi0 - chi2) / rec.chi0 : 0.0;
    }

    // Serial tie averaging keyed on x (ties in x <=> ties in the phase keys: x = phi - 0.5 is
    // monotone and maps equal phases to equal x).
    auto tie_avg = [&](double* z) {
        int j = 0;
        while (j < n) {
            int j0 = j; double sy = z[j] * ws[j], fbw = ws[j];
            while (j < n - 1 && x[j + 1] <= x[j]) { j++; sy += ws[j] * z[j]; fbw += ws[j]; }
            if (j > j0) { double a = fbw > 0.0 ? sy / fbw : 0.0; for (int i = j0; i <= j; i++) z[i] = a; }
            j++;
        }
    };

    if (fixed) {
        // ---- Listing 1 lines 51-55: one smooth of y at the caller's span, both modes
        int ibwf = rec.ibw_fixed, Kf = 2 * ibwf + 1;
        if (Kf > n) {
            Kf = n;
            if (per) { ibwf = (n - 1) / 2; Kf = 2 * ibwf + 1; }
        }
        double* smo = A1;
        for (int j = tid; j < n; j += T) smo[j] = fit_at(j, ibwf, Kf, Ewy, Ewxy);
        __syncthreads();
        if (has_ties) {
            if (tid == 0) tie_avg(smo);
            __syncthreads();
        }
        for (int j = tid; j < n; j += T) {
            double r = ys[j] - smo[j];
            chi2_part += ws[j] * r * r;
            if (smo_dbg) smo_dbg[j] = smo[j] + rec.ybar;
        }
        double chi2 = block_sum<T>(chi2_part, cx.red);
        return rec.chi0 > 0.0 ? (rec.chi0 - chi2) / rec.chi0 : 0.0;
    }

    // ---- CV pass 1: three smooths of y with leave-one-out residuals
    for (int j = tid; j < n; j += T) {
        const double xj = x[j], yj = ys[j], wj = ws[j];
        const int ib[3] = {ibw0, ibw1, ibw2}, KK[3] = {K0, K1, K2};
        double* const Ao[3] = {A0, A1, A2};
        double* const ro[3] = {r0, r1, r2};
#pragma unroll
        for (int i = 0; i < 3; i++) {
            const Win<OPT> wn(j, ib[i], KK[i], n, per);
            XMom m = wn.xmom(Ew, Ewx, Ewxx, vsmlsq);
            double Swy, Swxy, b, yb;
            wn.zmom(Ewy, Ewxy, Swy, Swxy);
            double s = line_fit(m, Swy, Swxy, xj, b, yb);
            double r = loo_residual(m, xj, wj, yj, s);
            if (r < 0.0) cx.flags[1 + i] = 1;
            Ao[i][j] = s;
            ro[i][j] = r;
        }
    }
    __syncthreads();
    if (has_ties || cx.flags[1] || cx.flags[2] || cx.flags[3]) {
        if (tid < 3) {
            double* const Ao[3] = {A0, A1, A2};
            double* const ro[3] = {r0, r1, r2};
            if (has_ties) tie_avg(Ao[tid]);
            if (cx.flags[1 + tid]) carry_fix_serial(n, ro[tid]);
        }
        __syncthreads();
    }
    // ---- CV pass 2: smooth each residual at the midrange span, in place
    {
        double* const ro[3] = {r0, r1, r2};
        for (int i = 0; i < 3; i++) {
            double* z = ro[i];
            double* const E[2] = {Ewy, Ewxy};
            block_scan<T, 2>(n, [&](int j, double* v) {
                double wz = ws[j] * z[j];
                v[0] = wz; v[1] = wz * x[j];
            }, E, cx.wsum);
            for (int j = tid; j < n; j += T) z[j] = fit_at(j, ibw1, K1, Ewy, Ewxy);
            __syncthreads();
        }
        if (has_ties) {
            if (tid < 3) tie_avg(ro[tid]);
            __syncthreads();
        }
    }
    // ---- span pick + bass enhancement: sp -> r0
    for (int j = tid; j < n; j += T) r0[j] = pick_span(r0[j], r1[j], r2[j], p.alpha);
    __syncthreads();
    // ---- smooth the spans at midrange: sps -> r1
    {
        double* const E[2] = {Ewy, Ewxy};
        block_scan<T, 2>(n, [&](int j, double* v) {
            double wz = ws[j] * r0[j];
            v[0] = wz; v[1] = wz * x[j];
        }, E, cx.wsum);
        for (int j = tid; j < n; j += T) r1[j] = fit_at(j, ibw1, K1, Ewy, Ewxy);
        __syncthreads();
        if (has_ties) {
            if (tid == 0) tie_avg(r1);
            __syncthreads();
        }
    }
    // ---- interpolate between the smooths: B -> r2
    for (int j = tid; j < n; j += T) r2[j] = interp_spans(r1[j], A0[j], A1[j], A2[j]);
    __syncthreads();
    // ---- final tweeter smooth: smo -> r0, then chi2
    {
        double* const E[2] = {Ewy, Ewxy};
        block_scan<T, 2>(n, [&](int j, double* v) {
            double wz = ws[j] * r2[j];
            v[0] = wz; v[1] = wz * x[j];
        }, E, cx.wsum);
        for (int j = tid; j < n; j += T) r0[j] = fit_at(j, ibw0, K0, Ewy, Ewxy);
        __syncthreads();
        if (has_ties) {
            if (tid == 0) tie_avg(r0);
            __syncthreads();
        }
    }
    for (int j = tid; j < n; j += T) {
        double r = ys[j] - r0[j];
        chi2_part += ws[j] * r * r;
        if (smo_dbg) smo_dbg[j] = r0[j] + rec.ybar;
    }
    double chi2 = block_sum<T>(chi2_part, cx.red);
    return rec.chi0 > 0.0 ? (rec.chi0 - chi2) / rec.chi0 : 0.0;
}

// Persistent kernel: work item = (list entry, frequency chunk).  STAGE = per-eval arrays in global.
template <int T, bool STAGE, bool OPT = false>
__global__ void __launch_bounds__(T, (T <= 128 ? 4 : (T <= 256 ? 2 : 1))) block_kernel(const EvalParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int NW = T / 32;
    __shared__ double s_wsum[6][NW];
    __shared__ double s_red[NW];
    __shared__ int s_flags[4];
    __shared__ unsigned int s_item;

    BlockCtx<T> cx;
    cx.wsum = s_wsum; cx.red = s_red; cx.flags = s_flags;

    const unsigned int n_items = (unsigned int)p.n_list * (unsigned int)p.chunks_per_obj;
    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) s_item = atomicAdd(p.counter, 1u);
        __syncthreads();
        const unsigned int item = s_item;
        if (item >= n_items) break;
        const int li = (int)(item / (unsigned int)p.chunks_per_obj);
        const int ch = (int)(item - (unsigned int)li * (unsigned int)p.chunks_per_obj);
        const int ri = p.list[li];
        const ObjRec rec = p.recs[ri];
        const int64_t sl = block_slot_len(rec.n);
        double* S = STAGE ? p.stage + (int64_t)blockIdx.x * p.stage_stride
                          : reinterpret_cast<double*>(smem_raw);
        const int64_t k0 = p.k_begin + (int64_t)ch * p.chunk;
        const int64_t k1 = min(k0 + (int64_t)p.chunk, p.k_end);
        double best = -INFINITY;
        int64_t best_k = k0;
        for (int64_t k = k0; k < k1; k++) {
            const double f = freq_of(p.f_min, p.df, k);
            double P = block_eval<T, OPT>(p, rec, f, S, sl, cx, nullptr, nullptr);
            if (threadIdx.x == 0) {
                if (p.pgram)
                    p.pgram[(rec.obj - p.pgram_row0) * p.pgram_row_stride + (k - p.pgram_k0)] = P;
                if (P > best) { best = P; best_k = k; }
            }
        }
        if (threadIdx.x == 0) {
            int64_t slot = (int64_t)ri * p.chunks_total + p.chunk_base + ch;
            p.part_val[slot] = best;
            p.part_idx[slot] = best_k;
        }
    }
}

// ss_debug_eval: one eval, one CTA, arrays staged in global memory.
template <int T, bool OPT>
__global__ void __launch_bounds__(T) block_debug_kernel(const EvalParams p, double f, double* smo_out,
                                                        int32_t* perm_out, double* p_out)
{
    constexpr int NW = T / 32;
    __shared__ double s_wsum[6][NW];
    __shared__ double s_red[NW];
    __shared__ int s_flags[4];
    BlockCtx<T> cx;
    cx.wsum = s_wsum; cx.red = s_red; cx.flags = s_flags;
    const ObjRec rec = p.recs[0];
    double P = block_eval<T, OPT>(p, rec, f, p.stage, block_slot_len(rec.n), cx, smo_out, perm_out);
    if (threadIdx.x == 0 && p_out) *p_out = P;
}

}  // namespace ss

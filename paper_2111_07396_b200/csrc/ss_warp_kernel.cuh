// ss_warp_kernel.cuh -- one warp per (object, frequency) eval, n <= 256 (SS_PATH_WARP).
//
// Lane L owns the C consecutive phase-ordered points j = L*C .. L*C+C-1 in registers (blocked
// layout, C = ceil(n/32)).  Per eval:
//   fold -> 32-bit keys (24 phase bits | 8 index bits) -> register/shuffle bitonic sort ->
//   gather x, y, w from the object's shared-memory copy, exact-order check on the full 64-bit phases
//   -> tweeter (span 0.05) windows summed DIRECTLY about each point from neighbour-lane halos
//      (2*IBW0+1 <= 13 points; exact centring, no cancellation) ->
//   midrange / woofer windows by differences of exclusive prefix sums kept in shared memory
//      (transposed so that every access is bank-conflict free) ->
//   CV (Listing 1) or GV (R12) -> chi2 -> P.
// Evals the fast path cannot decide exactly -- tied or quantisation-misordered phases, a
// leave-one-out denominator <= 0 -- are appended to a deferred list and recomputed by the generic
// CTA-per-eval kernel (ss_block_kernel.cuh), so results never depend on which path ran.
#pragma once
#include "../../include/ss_periodogram.h"
#include "ss_block_kernel.cuh"
#include "ss_common.cuh"
#include "ss_planner.h"

namespace ss {

constexpr bool WARP_IMPLEMENTED = true;
constexpr int WARPS_PER_CTA = 8;
constexpr int WROW = 33;   // row length of the transposed prefix arrays (32 lanes + the total)

template <int C> struct Pow2Ceil { static constexpr int value = C <= 2 ? 2 : (C <= 4 ? 4 : 8); };

// (C, IBW0) variants: C = points per lane, IBW0 = tweeter half-width (compile-time so the halo
// registers are statically indexed).  Returns variant id = C*8 + IBW0.
inline int warp_variant_for_n(int n)
{
    int ibw0 = half_width(n, SPAN0);
    int c = (n + 31) / 32;
    if (c < 2) c = 2;
    if (c == 7 && ibw0 == 6) c = 8;
    return c * 8 + ibw0;
}

__device__ __forceinline__ double shfl_d(double v, int src) { return __shfl_sync(0xffffffffu, v, src); }
__device__ __forceinline__ double shfl_up_d(double v, int d) { return __shfl_up_sync(0xffffffffu, v, d); }
__device__ __forceinline__ double shfl_down_d(double v, int d) { return __shfl_down_sync(0xffffffffu, v, d); }

template <int C>
__device__ __forceinline__ int wst(int e) { return (e % C) * WROW + e / C; }

// Warp-wide exclusive prefix of C values per lane (blocked); writes E[j], j = 0..32C, transposed.
template <int C>
__device__ __forceinline__ void warp_prefix_store(const double (&v)[C], double* E, int lane)
{
    double e[C];
    double run = 0.0;
#pragma unroll
    for (int s = 0; s < C; s++) { e[s] = run; run += v[s]; }
    double inc = run;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        double o = shfl_up_d(inc, d);
        if (lane >= d) inc += o;
    }
    const double excl = inc - run;
#pragma unroll
    for (int s = 0; s < C; s++) E[s * WROW + lane] = excl + e[s];
    if (lane == 31) E[32] = inc;     // E[32*C] lives at row 0, column 32
}

__device__ __forceinline__ void cex32(unsigned& a, unsigned& b)
{
    unsigned lo = min(a, b), hi = max(a, b);
    a = lo; b = hi;
}

// Bitonic sort of 32*S keys, S per lane, position = lane*S + s, ascending.  All exchanges put the
// smaller key at the lower position ("mirror then halve" network).
template <int S>
__device__ __forceinline__ void warp_sort(unsigned (&key)[S], int lane)
{
#pragma unroll
    for (int k = 2; k <= 32 * S; k <<= 1) {
        // mirror step: partner = pos ^ (k-1)
        if (k <= S) {
#pragma unroll
            for (int s = 0; s < S; s++) {
                const int t = s ^ (k - 1);
                if (t > s) cex32(key[s], key[t]);
            }
        } else {
            const int m = k / S - 1;               // lane mask
            const bool lower = (lane & (k / S / 2)) == 0;
            unsigned other[S];
#pragma unroll
            for (int s = 0; s < S; s++) other[s] = __shfl_xor_sync(0xffffffffu, key[S - 1 - s], m);
#pragma unroll
            for (int s = 0; s < S; s++) key[s] = lower ? min(key[s], other[s]) : max(key[s], other[s]);
        }
#pragma unroll
        for (int j = k >> 2; j >= 1; j >>= 1) {
            if (j >= S) {
                const int m = j / S;
                const bool lower = (lane & m) == 0;
#pragma unroll
                for (int s = 0; s < S; s++) {
                    unsigned o = __shfl_xor_sync(0xffffffffu, key[s], m);
                    key[s] = lower ? min(key[s], o) : max(key[s], o);
                }
            } else {
#pragma unroll
                for (int s = 0; s < S; s++)
                    if ((s & j) == 0) cex32(key[s], key[s + j]);
            }
        }
    }
}

// Fit ingredients of one window, shareable between points that use the same window (clamped ends).
struct WinFit {
    double inv_sw, xbar, inv_sxx;   // x-moments (xbar absolute, in centred-x units)
    double zbar, b;                 // z-moments folded into mean and slope
    double g;                       // GV score (GV only)
};

// Direct sums over the 2*IBW0+1 window centred on halo element `ctr` of (ux, uw, uz).
template <int C, int IBW0, bool GV>
__device__ __forceinline__ WinFit tweeter_fit(const double (&ux)[C + 2 * IBW0], const double (&uw)[C + 2 * IBW0],
                                              const double (&uz)[C + 2 * IBW0], int s, double vsmlsq)
{
    const double c = ux[IBW0 + s];
    double m0 = 0.0, m1 = 0.0, m2 = 0.0, mz = 0.0, m1z = 0.0, mzz = 0.0;
#pragma unroll
    for (int t = 0; t <= 2 * IBW0; t++) {
        const double d = ux[s + t] - c, w_ = uw[s + t], z_ = uz[s + t];
        const double wd = w_ * d, wz = w_ * z_;
        m0 += w_; m1 += wd; m2 += wd * d; mz += wz; m1z += wd * z_;
        if (GV) mzz += wz * z_;
    }
    WinFit f;
    f.inv_sw = m0 > 0.0 ? rcp64(m0) : 0.0;
    const double xr = m1 * f.inv_sw;             // xbar relative to c
    const double sxx = m2 - xr * m1;
    f.inv_sxx = sxx > vsmlsq ? rcp64(sxx) : 0.0;
    f.xbar = c + xr;
    f.zbar = mz * f.inv_sw;
    const double sxz = m1z - xr * mz;
    f.b = sxz * f.inv_sxx;
    f.g = 0.0;
    if (GV) {
        double rss = (mzz - f.zbar * mz) - f.b * sxz;
        rss = rss > 0.0 ? rss : 0.0;
        const double p = f.inv_sxx != 0.0 ? 2.0 : 1.0;
        f.g = m0 > 0.0 ? sqrt(rss * f.inv_sw) * rcp64(1.0 - p / (double)(2 * IBW0 + 1)) : 0.0;
    }
    return f;
}

// Only the z-dependent part, x-moments given (final smooth of CV).
template <int C, int IBW0>
__device__ __forceinline__ void tweeter_refit(const double (&ux)[C + 2 * IBW0], const double (&uw)[C + 2 * IBW0],
                                              const double (&uz)[C + 2 * IBW0], int s, double inv_sw, double xbar,
                                              double inv_sxx, double& zbar, double& b)
{
    const double c = ux[IBW0 + s];
    double mz = 0.0, m1z = 0.0;
#pragma unroll
    for (int t = 0; t <= 2 * IBW0; t++) {
        const double wz = uw[s + t] * uz[s + t];
        mz += wz; m1z += wz * (ux[s + t] - c);
    }
    zbar = mz * inv_sw;
    b = (m1z - (xbar - c) * mz) * inv_sxx;
}

// Halo of one register array: u[t] = element at j = lane*C - IBW0 + t.
template <int C, int IBW0>
__device__ __forceinline__ void make_halo(const double (&v)[C], double (&u)[C + 2 * IBW0], int lane, double fill)
{
#pragma unroll
    for (int t = 0; t < IBW0; t++) {
        double l = shfl_up_d(v[C - IBW0 + t], 1);
        u[t] = lane == 0 ? fill : l;
        double r = shfl_down_d(v[t], 1);
        u[IBW0 + C + t] = lane == 31 ? fill : r;
    }
#pragma unroll
    for (int s = 0; s < C; s++) u[IBW0 + s] = v[s];
}

template <int C>
__device__ __forceinline__ double pick_slot(const double (&v)[C], int slot)
{
    double r = v[0];
#pragma unroll
    for (int s = 1; s < C; s++) r = slot == s ? v[s] : r;
    return r;
}

// Per-warp view of the shared memory.
struct WarpMem {
    const double* tt; const double* yc; const double* w;   // the object's arrays (CTA-wide)
    double* E;               // per-warp: NE prefix arrays of C*WROW doubles
    unsigned char* perm;     // per-warp: 256 bytes (rank -> index), only when S != C
};


// Window of span i for point j through the prefix arrays: S = E[lo+K] - E[lo].
template <int C>
__device__ __forceinline__ double wdiff(const double* E, int slo, int shi) { return E[shi] - E[slo]; }

// Smoother + statistic on the sorted, gathered eval (x centred by 0.5, y centred by ybar_w).
template <int C, int IBW0, bool GV>
__device__ __forceinline__ double warp_eval_body(const ObjRec& rec, const WarpMem& M, const double (&x)[C],
                                                 const double (&y)[C], const double (&w)[C], double vsmlsq,
                                                 double alpha, int lane, bool& defer)
{
    constexpr int ASZ = C * WROW;
    const int n = rec.n;
    const int ibw1 = rec.ibw[1], ibw2 = rec.ibw[2];
    const int K1 = min(2 * ibw1 + 1, n), K2 = min(2 * ibw2 + 1, n);
    double* Ew = M.E;            double* Ewx = M.E + ASZ;      double* Ewxx = M.E + 2 * ASZ;
    double* Ewy = M.E + 3 * ASZ; double* Ewxy = M.E + 4 * ASZ; double* Ewyy = M.E + 5 * ASZ;   // Ewyy: GV only

    // ---- prefix sums of the weighted moments (midrange and woofer windows)
    {
        double v[C];
#pragma unroll
        for (int s = 0; s < C; s++) v[s] = w[s];
        warp_prefix_store<C>(v, Ew, lane);
#pragma unroll
        for (int s = 0; s < C; s++) v[s] = w[s] * x[s];
        warp_prefix_store<C>(v, Ewx, lane);
        double v2[C];
#pragma unroll
        for (int s = 0; s < C; s++) v2[s] = v[s] * x[s];
        warp_prefix_store<C>(v2, Ewxx, lane);
#pragma unroll
        for (int s = 0; s < C; s++) v2[s] = v[s] * y[s];
        warp_prefix_store<C>(v2, Ewxy, lane);
#pragma unroll
        for (int s = 0; s < C; s++) v[s] = w[s] * y[s];
        warp_prefix_store<C>(v, Ewy, lane);
        if (GV) {
#pragma unroll
            for (int s = 0; s < C; s++) v[s] = v[s] * y[s];
            warp_prefix_store<C>(v, Ewyy, lane);
        }
    }
    __syncwarp();

    // ---- tweeter: direct window sums from neighbour-lane halos
    double ux[C + 2 * IBW0], uw[C + 2 * IBW0], uz[C + 2 * IBW0];
    make_halo<C, IBW0>(x, ux, lane, 0.0);
    make_halo<C, IBW0>(w, uw, lane, 0.0);
    make_halo<C, IBW0>(y, uz, lane, 0.0);
    WinFit tw[C];
#pragma unroll
    for (int s = 0; s < C; s++) tw[s] = tweeter_fit<C, IBW0, GV>(ux, uw, uz, s, vsmlsq);
    // clamped ends (O4): points j < IBW0 use the window of jl = IBW0, points j > jr = n-1-IBW0 the
    // window of jr.  The owner's fit is broadcast.
    const int jr = n - 1 - IBW0;
    const int lane_r = jr / C, slot_r = jr % C;
    WinFit twl, twr;
    {
        double a[C];
#define SS_BCAST(field)                                                                   \
        {                                                                                 \
            _Pragma("unroll") for (int s = 0; s < C; s++) a[s] = tw[s].field;             \
            twr.field = shfl_d(pick_slot<C>(a, slot_r), lane_r);                          \
            twl.field = IBW0 < C ? shfl_d(a[IBW0 < C ? IBW0 : 0], 0) : shfl_d(a[0], 1);   \
        }
        SS_BCAST(inv_sw) SS_BCAST(xbar) SS_BCAST(inv_sxx) SS_BCAST(zbar) SS_BCAST(b)
        if (GV) SS_BCAST(g)
    }
#pragma unroll
    for (int s = 0; s < C; s++) {
        const int j = lane * C + s;
        if (j < IBW0) tw[s] = twl;
        if (j > jr) tw[s] = twr;
    }

    // ---- window indices of the midrange and woofer spans (transposed storage)
    int s1lo[C], s1hi[C];
#pragma unroll
    for (int s = 0; s < C; s++) {
        const int lo = window_lo(lane * C + s, ibw1, K1, n);
        s1lo[s] = wst<C>(lo); s1hi[s] = wst<C>(lo + K1);
    }

    double chi2 = 0.0;
    if (GV) {
        // ---- O6: scores, pick, interpolate
#pragma unroll
        for (int s = 0; s < C; s++) {
            const double xj = x[s];
            const double A0 = tw[s].zbar + tw[s].b * (xj - tw[s].xbar);
            XMom m1 = x_moments(wdiff<C>(Ew, s1lo[s], s1hi[s]), wdiff<C>(Ewx, s1lo[s], s1hi[s]),
                                wdiff<C>(Ewxx, s1lo[s], s1hi[s]), vsmlsq);
            double b1, yb1;
            const double Sy1 = wdiff<C>(Ewy, s1lo[s], s1hi[s]), Sxy1 = wdiff<C>(Ewxy, s1lo[s], s1hi[s]);
            const double A1 = line_fit(m1, Sy1, Sxy1, xj, b1, yb1);
            const double G1 = gv_score(m1, Sy1, Sxy1, wdiff<C>(Ewyy, s1lo[s], s1hi[s]), b1, yb1, K1);
            const int lo2 = window_lo(lane * C + s, ibw2, K2, n);
            const int a2 = wst<C>(lo2), b2i = wst<C>(lo2 + K2);
            XMom m2 = x_moments(wdiff<C>(Ew, a2, b2i), wdiff<C>(Ewx, a2, b2i), wdiff<C>(Ewxx, a2, b2i), vsmlsq);
            double b2, yb2;
            const double Sy2 = wdiff<C>(Ewy, a2, b2i), Sxy2 = wdiff<C>(Ewxy, a2, b2i);
            const double A2 = line_fit(m2, Sy2, Sxy2, xj, b2, yb2);
            const double G2 = gv_score(m2, Sy2, Sxy2, wdiff<C>(Ewyy, a2, b2i), b2, yb2, K2);
            const double sp = pick_span(tw[s].g, G1, G2, alpha);
            const double smo = interp_spans(sp, A0, A1, A2);
            const double r = y[s] - smo;
            chi2 += w[s] * r * r;
        }
    } else {
        // ---- CV pass 1
        double A0[C], A1[C], A2[C], r0[C], r1[C], r2[C];
        double m_isw[C], m_xb[C], m_isxx[C];      // midrange x-moments, reused by four more smooths
        bool bad = false;
#pragma unroll
        for (int s = 0; s < C; s++) {
            const double xj = x[s], yj = y[s], wj = w[s];
            A0[s] = tw[s].zbar + tw[s].b * (xj - tw[s].xbar);
            {
                const double dx = xj - tw[s].xbar;
                const double a = 1.0 - wj * (tw[s].inv_sw + dx * dx * tw[s].inv_sxx);
                r0[s] = a > 0.0 ? fabs(yj - A0[s]) * rcp64(a) : -1.0;
            }
            XMom m1 = x_moments(wdiff<C>(Ew, s1lo[s], s1hi[s]), wdiff<C>(Ewx, s1lo[s], s1hi[s]),
                                wdiff<C>(Ewxx, s1lo[s], s1hi[s]), vsmlsq);
            m_isw[s] = m1.inv_sw; m_xb[s] = m1.xbar; m_isxx[s] = m1.inv_sxx;
            double b_, zb_;
            A1[s] = line_fit(m1, wdiff<C>(Ewy, s1lo[s], s1hi[s]), wdiff<C>(Ewxy, s1lo[s], s1hi[s]), xj, b_, zb_);
            r1[s] = loo_residual(m1, xj, wj, yj, A1[s]);
            const int lo2 = window_lo(lane * C + s, ibw2, K2, n);
            const int a2 = wst<C>(lo2), b2i = wst<C>(lo2 + K2);
            XMom m2 = x_moments(wdiff<C>(Ew, a2, b2i), wdiff<C>(Ewx, a2, b2i), wdiff<C>(Ewxx, a2, b2i), vsmlsq);
            A2[s] = line_fit(m2, wdiff<C>(Ewy, a2, b2i), wdiff<C>(Ewxy, a2, b2i), xj, b_, zb_);
            r2[s] = loo_residual(m2, xj, wj, yj, A2[s]);
            if (lane * C + s < n && (r0[s] < 0.0 || r1[s] < 0.0 || r2[s] < 0.0)) bad = true;
        }
        if (__any_sync(0xffffffffu, bad)) { defer = true; return 0.0; }
        __syncwarp();      // every lane is done reading Ewy / Ewxy

        // midrange smooth of a register array z through two prefix arrays
        auto mid_smooth = [&](const double (&z)[C], double (&out)[C]) {
            double v[C];
#pragma unroll
            for (int s = 0; s < C; s++) v[s] = w[s] * z[s];
            warp_prefix_store<C>(v, Ewy, lane);
#pragma unroll
            for (int s = 0; s < C; s++) v[s] = v[s] * x[s];
            warp_prefix_store<C>(v, Ewxy, lane);
            __syncwarp();
#pragma unroll
            for (int s = 0; s < C; s++) {
                const double Sz = wdiff<C>(Ewy, s1lo[s], s1hi[s]), Sxz = wdiff<C>(Ewxy, s1lo[s], s1hi[s]);
                const double zb = Sz * m_isw[s];
                out[s] = zb + (Sxz - m_xb[s] * Sz) * m_isxx[s] * (x[s] - m_xb[s]);
            }
            __syncwarp();
        };
        double sp[C];
        {
            double R0[C], R1[C], R2[C];
            mid_smooth(r0, R0);
            mid_smooth(r1, R1);
            mid_smooth(r2, R2);
            // span pick + bass enhancement
#pragma unroll
            for (int s = 0; s < C; s++) sp[s] = pick_span(R0[s], R1[s], R2[s], alpha);
        }
        double sps[C];
        mid_smooth(sp, sps);
        double B[C];
#pragma unroll
        for (int s = 0; s < C; s++) B[s] = interp_spans(sps[s], A0[s], A1[s], A2[s]);
        // ---- final tweeter smooth, direct sums again
        make_halo<C, IBW0>(B, uz, lane, 0.0);
        double zb[C], bb[C];
#pragma unroll
        for (int s = 0; s < C; s++)
            tweeter_refit<C, IBW0>(ux, uw, uz, s, tw[s].inv_sw, tw[s].xbar, tw[s].inv_sxx, zb[s], bb[s]);
        // NOTE: for clamped points tw[s] already holds the shared window's x-moments, but the z-sums
        // above were taken over the point's own (wrong) window: take the owner's (zbar, b).
        const double zr = shfl_d(pick_slot<C>(zb, slot_r), lane_r), br = shfl_d(pick_slot<C>(bb, slot_r), lane_r);
        const double zl = IBW0 < C ? shfl_d(zb[IBW0 < C ? IBW0 : 0], 0) : shfl_d(zb[0], 1);
        const double bl = IBW0 < C ? shfl_d(bb[IBW0 < C ? IBW0 : 0], 0) : shfl_d(bb[0], 1);
#pragma unroll
        for (int s = 0; s < C; s++) {
            const int j = lane * C + s;
            double z_ = zb[s], b_ = bb[s];
            if (j < IBW0) { z_ = zl; b_ = bl; }
            if (j > jr) { z_ = zr; b_ = br; }
            const double smo = z_ + b_ * (x[s] - tw[s].xbar);
            const double r = y[s] - smo;
            chi2 += w[s] * r * r;
        }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) chi2 += __shfl_xor_sync(0xffffffffu, chi2, d);
    return rec.chi0 > 0.0 ? (rec.chi0 - chi2) / rec.chi0 : 0.0;
}

// One eval.  Returns P in every lane; `defer` is set (warp-uniform) when the fast path cannot
// decide the eval exactly.
template <int C, int IBW0, bool GV>
__device__ __forceinline__ double warp_eval(const ObjRec& rec, const WarpMem& M, double f, double alpha, int lane,
                                            bool& defer)
{
    constexpr int S = Pow2Ceil<C>::value;
    const int n = rec.n;
    defer = false;

    // ---- P1 fold + 32-bit keys (24 phase bits | 8 index bits); P2 sort
    unsigned key[S];
#pragma unroll
    for (int s = 0; s < S; s++) {
        const int i = lane + 32 * s;
        unsigned k = 0xffffffffu;
        if (i < n) {
            const double phi = fold_phase(M.tt[i], f);
            k = (__double2uint_rz(phi * 16777216.0) << 8) | (unsigned)i;
        }
        key[s] = k;
    }
    warp_sort<S>(key, lane);
    int idx[C];
    if (S == C) {
#pragma unroll
        for (int s = 0; s < C; s++) idx[s] = (int)(key[s < S ? s : 0] & 0xffu);
    } else {
#pragma unroll
        for (int s = 0; s < S; s++) M.perm[lane * S + s] = (unsigned char)(key[s] & 0xffu);
        __syncwarp();
#pragma unroll
        for (int s = 0; s < C; s++) idx[s] = M.perm[lane * C + s];
        __syncwarp();
    }
    // ---- gather and exact-order check on the full 64-bit phases
    double x[C], y[C], w[C], phi[C];
#pragma unroll
    for (int s = 0; s < C; s++) {
        const int j = lane * C + s;
        if (j < n) {
            const int i = idx[s];
            phi[s] = fold_phase(M.tt[i], f);
            y[s] = M.yc[i];
            w[s] = M.w[i];
        } else { phi[s] = 4.0; y[s] = 0.0; w[s] = 0.0; }
    }
    bool bad = false;
    double nxt = shfl_down_d(phi[0], 1);
    if (lane == 31) nxt = 8.0;
#pragma unroll
    for (int s = 0; s < C; s++) {
        const double nx = s + 1 < C ? phi[s + 1 < C ? s + 1 : 0] : nxt;
        if (lane * C + s + 1 < n && nx <= phi[s]) bad = true;   // tie or quantisation misorder
    }
    // vsmlsq from the quartile spread
    const double p1 = shfl_d(pick_slot<C>(phi, rec.q1 % C), rec.q1 / C);
    const double p3 = shfl_d(pick_slot<C>(phi, rec.q3 % C), rec.q3 / C);
    if (__any_sync(0xffffffffu, bad)) { defer = true; return 0.0; }
#pragma unroll
    for (int s = 0; s < C; s++) x[s] = (lane * C + s < n) ? phi[s] - 0.5 : 0.0;
    const double scale = p3 - p1;
    return warp_eval_body<C, IBW0, GV>(rec, M, x, y, w, 1.e-6 * scale * scale, alpha, lane, defer);
}


// ------------------------------------------------------------------------------------------------
// Kernel: one CTA = one work item (object, chunk of frequencies); its WARPS_PER_CTA warps split the
// chunk into contiguous runs.  P values are staged in registers and written 32 at a time.
// ------------------------------------------------------------------------------------------------
template <int C, bool GV> struct WarpNE { static constexpr int value = GV ? 6 : 5; };

template <int C, bool GV>
inline size_t warp_smem_bytes()
{
    // object arrays (3 x 32C doubles) + per warp: NE prefix arrays + 256 B permutation bytes
    return (size_t)3 * 32 * C * 8 + (size_t)WARPS_PER_CTA * ((size_t)WarpNE<C, GV>::value * C * WROW * 8 + 256);
}

template <int C, int IBW0, bool GV>
__global__ void __launch_bounds__(WARPS_PER_CTA * 32, (C <= 4 ? 2 : 1)) warp_kernel(const EvalParams p)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double s_best[WARPS_PER_CTA];
    __shared__ long long s_bestk[WARPS_PER_CTA];
    constexpr int NE = WarpNE<C, GV>::value;
    const int tid = threadIdx.x, lane = tid & 31;
    // warp index through a lane-0 broadcast: the compiler then knows it (and the eval loop's bounds) to be
    // warp-uniform, so the shuffles inside the loop need no WARPSYNC / ENDCOLLECTIVE wrappers
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
    const int item = blockIdx.x;
    const int li = item / p.chunks_per_obj, ch = item - li * p.chunks_per_obj;
    const int ri = p.list[li];
    const ObjRec rec = p.recs[ri];
    const int n = rec.n;

    double* o_tt = reinterpret_cast<double*>(smem_raw);
    double* o_y = o_tt + 32 * C;
    double* o_w = o_y + 32 * C;
    unsigned char* wbase = smem_raw + (size_t)3 * 32 * C * 8 + (size_t)warp * ((size_t)NE * C * WROW * 8 + 256);
    WarpMem M;
    M.tt = o_tt; M.yc = o_y; M.w = o_w;
    M.E = reinterpret_cast<double*>(wbase);
    M.perm = wbase + (size_t)NE * C * WROW * 8;
    for (int j = tid; j < n; j += WARPS_PER_CTA * 32) {
        o_tt[j] = p.tt[rec.off + j];
        o_y[j] = p.yc[rec.off + j];
        o_w[j] = p.w[rec.off + j];
    }
    __syncthreads();

    const int64_t c0 = p.k_begin + (int64_t)ch * p.chunk;
    const int64_t c1 = min(c0 + (int64_t)p.chunk, p.k_end);
    const int per_warp = p.chunk / WARPS_PER_CTA;          // chunk is a multiple of WARPS_PER_CTA
    const int64_t k0 = c0 + (int64_t)warp * per_warp;
    const int64_t k1 = min(k0 + (int64_t)per_warp, c1);
    double best = -INFINITY;
    int64_t best_k = INT64_MAX;
    double* prow = p.pgram ? p.pgram + (rec.obj - p.pgram_row0) * p.pgram_row_stride - p.pgram_k0 : nullptr;
    double stash = 0.0;
    int64_t kb = k0;                                       // first k of the current batch of 32
    for (int64_t k = k0; k < k1; k++) {
        const double f = freq_of(p.f_min, p.df, k);
        bool defer;
        double P = warp_eval<C, IBW0, GV>(rec, M, f, p.alpha, lane, defer);
        if (defer) {
            if (lane == 0) {
                unsigned pos = atomicAdd(p.defer_count, 1u);
                if (pos < p.defer_capacity)
                    p.defer_entries[pos] = ((unsigned long long)ri << 32) | (unsigned long long)(k - p.k_begin);
                else
                    p.defer_count[1] = 1u;
            }
            P = 0.0;      // patched by the deferred kernel
        } else if (P > best) { best = P; best_k = k; }
        if (lane == (int)(k - kb)) stash = P;
        if (k - kb == 31 || k == k1 - 1) {
            if (prow && kb + lane <= k) prow[kb + lane] = stash;
            kb = k + 1;
        }
    }
    if (lane == 0) { s_best[warp] = best; s_bestk[warp] = best_k; }
    __syncthreads();
    if (tid == 0) {
        for (int q = 1; q < WARPS_PER_CTA; q++)
            if (s_best[q] > best || (s_best[q] == best && s_bestk[q] < best_k)) { best = s_best[q]; best_k = s_bestk[q]; }
        const int64_t slot = (int64_t)ri * p.chunks_total + p.chunk_base + ch;
        p.part_val[slot] = best;
        p.part_idx[slot] = best_k == INT64_MAX ? c0 : best_k;
    }
}

// ---- deferred evals: recomputed exactly by the generic CTA-per-eval code ------------------------
constexpr int DEFER_T = 128;

__device__ __forceinline__ unsigned long long sortable_bits(double v)
{
    unsigned long long u = (unsigned long long)__double_as_longlong(v);
    return (u >> 63) ? ~u : (u | 0x8000000000000000ull);
}

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
    const unsigned cnt = min(p.defer_count[0], p.defer_capacity);
    for (unsigned e = blockIdx.x; e < cnt; e += gridDim.x) {
        const unsigned long long ent = p.defer_entries[e];
        const int ri = (int)(ent >> 32);
        const int64_t k = p.k_begin + (int64_t)(ent & 0xffffffffull);
        const ObjRec rec = p.recs[ri];
        __syncthreads();
        const double P = block_eval<DEFER_T>(p, rec, freq_of(p.f_min, p.df, k), reinterpret_cast<double*>(smem_raw),
                                             block_slot_len(rec.n), cx, nullptr, nullptr);
        if (threadIdx.x == 0) {
            if (p.pgram) p.pgram[(rec.obj - p.pgram_row0) * p.pgram_row_stride + (k - p.pgram_k0)] = P;
            dval[e] = P;
            atomicMax(&dmax[rec.obj], sortable_bits(P));
        }
    }
}

__global__ void deferred_min_kernel(const EvalParams p, const double* dval, const unsigned long long* dmax,
                                    unsigned long long* dmin)
{
    const unsigned cnt = min(p.defer_count[0], p.defer_capacity);
    for (unsigned e = blockIdx.x * blockDim.x + threadIdx.x; e < cnt; e += gridDim.x * blockDim.x) {
        const unsigned long long ent = p.defer_entries[e];
        const int64_t obj = p.recs[(int)(ent >> 32)].obj;
        if (sortable_bits(dval[e]) == dmax[obj]) atomicMin(&dmin[obj], (unsigned long long)(p.k_begin + (int64_t)(ent & 0xffffffffull)));
    }
}

__global__ void deferred_merge_kernel(const EvalParams p, const double* dval, const unsigned long long* dmax,
                                      const unsigned long long* dmin, double* best_val, int64_t* best_idx)
{
    const unsigned cnt = min(p.defer_count[0], p.defer_capacity);
    for (unsigned e = blockIdx.x * blockDim.x + threadIdx.x; e < cnt; e += gridDim.x * blockDim.x) {
        const unsigned long long ent = p.defer_entries[e];
        const int64_t obj = p.recs[(int)(ent >> 32)].obj;
        const int64_t k = p.k_begin + (int64_t)(ent & 0xffffffffull);
        const double v = dval[e];
        // the unique winner among this object's deferred evals folds itself into the running best
        if (sortable_bits(v) == dmax[obj] && (unsigned long long)k == dmin[obj]) {
            const double cv = best_val[obj];
            const int64_t ck = best_idx[obj];
            if (ck < 0 || v > cv || (v == cv && k < ck)) { best_val[obj] = v; best_idx[obj] = k; }
        }
    }
}

template <int C, int IBW0>
inline ss_status_t launch_warp_variant(const EvalParams& p, int64_t n_items, cudaStream_t stream)
{
    cudaError_t e;
    if (p.mode == 1) {
        const size_t smem = warp_smem_bytes<C, true>();
        e = cudaFuncSetAttribute(warp_kernel<C, IBW0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return SS_ERR_CUDA;
        warp_kernel<C, IBW0, true><<<(unsigned)n_items, WARPS_PER_CTA * 32, smem, stream>>>(p);
    } else {
        const size_t smem = warp_smem_bytes<C, false>();
        e = cudaFuncSetAttribute(warp_kernel<C, IBW0, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return SS_ERR_CUDA;
        warp_kernel<C, IBW0, false><<<(unsigned)n_items, WARPS_PER_CTA * 32, smem, stream>>>(p);
    }
    return cudaGetLastError() == cudaSuccess ? SS_OK : SS_ERR_CUDA;
}

inline ss_status_t launch_warp_kernel(const EvalParams& p, int variant, int64_t n_items, cudaStream_t stream)
{
    switch (variant) {
        case 2 * 8 + 2: return launch_warp_variant<2, 2>(p, n_items, stream);
        case 3 * 8 + 2: return launch_warp_variant<3, 2>(p, n_items, stream);
        case 4 * 8 + 2: return launch_warp_variant<4, 2>(p, n_items, stream);
        case 4 * 8 + 3: return launch_warp_variant<4, 3>(p, n_items, stream);
        case 5 * 8 + 3: return launch_warp_variant<5, 3>(p, n_items, stream);
        case 5 * 8 + 4: return launch_warp_variant<5, 4>(p, n_items, stream);
        case 6 * 8 + 4: return launch_warp_variant<6, 4>(p, n_items, stream);
        case 6 * 8 + 5: return launch_warp_variant<6, 5>(p, n_items, stream);
        case 7 * 8 + 5: return launch_warp_variant<7, 5>(p, n_items, stream);
        case 8 * 8 + 5: return launch_warp_variant<8, 5>(p, n_items, stream);
        case 8 * 8 + 6: return launch_warp_variant<8, 6>(p, n_items, stream);
        default: return SS_ERR_UNSUPPORTED;
    }
}

}  // namespace ss

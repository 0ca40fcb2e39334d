// ss_common.cuh -- shared device-side definitions of the B200 SuperSmoother periodogram kernels.
//
// Notation follows the paper (arXiv 2111.07396; PAPER.md line numbers) and DESIGN.md:
//   tt = t - min t, w = 1/e^2, spans tweeter/midrange/woofer = 0.05/0.2/0.5
//   (PAPER.md:163), vsmlsq, resmin, alpha as in Listing 1.
// This file is part of the CUDA product path; it shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace ss {

constexpr double SPAN0 = 0.05, SPAN1 = 0.2, SPAN2 = 0.5;
constexpr int MIN_POINTS = 5;                              // DESIGN.md R17

// Per-object record, built by the prep kernel (chi0, ybar) and the host (everything else).
struct ObjRec {
    int64_t off;     // first element of this object in tt / yc / w
    int64_t obj;     // object index in the caller's catalog (row of pgram_out)
    double chi0;     // sum w (y - ybar_w)^2            (R5)
    double ybar;     // weighted mean magnitude
    int32_t n;       // number of points
    int32_t ibw[3];  // window half-widths for the three spans: max(2, floor(0.5*span*n + 0.5))
    int32_t q1, q3;  // quartile indices n/4-1, 3*(q1+1)-1
    int32_t ibw_fixed;  // half-width of the caller's fixed span, 0 if span == 0
    int32_t dup;        // 1 = the object has duplicated time stamps (set by the prep kernel for n <= SS_WARP_MAX_N):
                        // its phases tie at every frequency, so the warp path hands its work items over whole
};

// Per-launch parameters.
struct EvalParams {
    const double* tt;      // [n_points] t - min t per object
    const double* yc;      // [n_points] y - ybar_w per object (the smoother is shift-equivariant)
    const double* w;       // [n_points] 1/e^2
    const ObjRec* recs;    // [n_objects] records
    const int32_t* list;   // [n_list] record indices served by this launch, longest first
    int32_t n_list;
    double f_min, df;      // f_k = f_min + k*df (R1, R2)
    int64_t k_begin, k_end;   // frequency tile [k_begin, k_end)
    int32_t chunk;            // frequencies per work item
    int32_t chunks_per_obj;   // ceil((k_end-k_begin)/chunk)
    int32_t chunks_total;     // chunks per object over the WHOLE grid (partials row length)
    int32_t chunk_base;       // index of this tile's first chunk in the partials row
    double alpha;             // bass enhancement
    int32_t mode;             // 0 = CV, 1 = GV
    int32_t iper;             // 1 = windows pinned at the ends, 2 = periodic windows
    double span;              // > 0: one smooth at this fixed span
    double* pgram;            // tile buffer or caller's array (may be null)
    int64_t pgram_row_stride; // elements between consecutive object rows
    int64_t pgram_k0;         // column 0 of `pgram` is frequency index pgram_k0
    int64_t pgram_row0;       // row 0 of `pgram` is object index pgram_row0
    double* part_val;         // [n_objects * chunks_total] best P of each work item
    int64_t* part_idx;        // [n_objects * chunks_total] its frequency index
    unsigned int* counter;    // dynamic work counter (persistent kernels)
    double* stage;            // global staging scratch (STAGE path), stage_stride doubles per CTA
    int64_t stage_stride;
    // what the warp path hands over to the generic kernel: one eval (record index << 32 | k - k_begin) or a
    // whole work item (DEFER_ITEM | record index << 32 | chunk index)
    unsigned long long* defer_entries;
    unsigned int* defer_count;   // [0] = appended (may exceed capacity), [1] = sticky overflow flag
    unsigned int defer_capacity;
};

constexpr unsigned long long DEFER_ITEM = 1ull << 63;

// CTA-per-eval kernels (ss_block_kernel.cuh): per-eval arrays of block_slot_len(n) doubles each
constexpr int BLOCK_SLOTS = 14;
__host__ __device__ inline int64_t block_slot_len(int n) { return ((int64_t)n + 2) & ~(int64_t)1; }

// f_k = f_min + k*df as one multiply and one add, unfused (R2).
__device__ __forceinline__ double freq_of(double f_min, double df, int64_t k)
{
    return __dadd_rn(f_min, __dmul_rn((double)k, df));
}

// phi = tt*f - floor(tt*f): product rounded once, never contracted (R2); in [0,1).
__device__ __forceinline__ double fold_phase(double tt, double f)
{
    double p = __dmul_rn(tt, f);
    return __dsub_rn(p, floor(p));
}

// 1/x to about 1 ulp: MUFU.RCP64H seed (relative error 2^-20, measured 9.9e-7 on B200) and one
// third-order correction on the fp64 pipe (3 DFMA).  x must be a normal, finite, non-zero double (the callers guard that).
// IEEE division costs ~3x as many fp64 instructions plus a slow-path branch.
__device__ __forceinline__ double rcp64(double x)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    const double e = fma(-x, r, 1.0);     // |e| <= 2^-20
    const double t = fma(e, e, e);        // e + e^2: r*(1 + e + e^2) leaves a relative error of e^3 = 2^-60
    return fma(r, t, r);
}

// x-moments of one window: reused by every smooth over the same window.
struct XMom {
    double inv_sw;   // 1/Sw
    double xbar;     // Swx/Sw
    double inv_sxx;  // 1/Sxx if Sxx > vsmlsq else 0 (slope switched off, O4)
    double sw;
};

__device__ __forceinline__ XMom x_moments(double Sw, double Swx, double Swxx, double vsmlsq)
{
    XMom m;
    m.sw = Sw;
    m.inv_sw = Sw > 0.0 ? rcp64(Sw) : 0.0;
    m.xbar = Swx * m.inv_sw;
    double sxx = Swxx - m.xbar * Swx;
    m.inv_sxx = sxx > vsmlsq ? rcp64(sxx) : 0.0;
    return m;
}

// Value at xj of the weighted line fitted over the window; also returns slope b and mean zbar.
__device__ __forceinline__ double line_fit(const XMom& m, double Swz, double Swxz, double xj,
                                           double& b, double& zbar)
{
    zbar = Swz * m.inv_sw;
    double sxz = Swxz - m.xbar * Swz;
    b = sxz * m.inv_sxx;
    return zbar + b * (xj - m.xbar);
}

// Leave-one-out residual |z - s| / (1 - w h)  (O4); returns -1 when 1 - w h <= 0 (carry, R23).
__device__ __forceinline__ double loo_residual(const XMom& m, double xj, double wj, double zj, double s)
{
    double dx = xj - m.xbar;
    double h = m.inv_sw + dx * dx * m.inv_sxx;
    double a = 1.0 - wj * h;
    return a > 0.0 ? fabs(zj - s) * rcp64(a) : -1.0;
}

// GV score sqrt(RSS/Sw)/(1 - p/K), RSS = Syy - b*Sxy clamped at 0 (O6, R12).
__device__ __forceinline__ double gv_score(const XMom& m, double Swy, double Swxy, double Swyy,
                                           double b, double ybar, int K)
{
    double syy = Swyy - ybar * Swy;
    double sxy = Swxy - m.xbar * Swy;
    double rss = syy - b * sxy;
    rss = rss > 0.0 ? rss : 0.0;
    double p = m.inv_sxx != 0.0 ? 2.0 : 1.0;
    return m.sw > 0.0 ? sqrt(rss * m.inv_sw) * rcp64(1.0 - p / (double)K) : 0.0;
}

// Listing 1 lines 63-77: span with the smallest smoothed residual (first wins
// ties), then bass enhancement.
__device__ __forceinline__ double pick_span(double v0, double v1, double v2, double alpha)
{
    double resmin = 1.e20, sp = 0.0;
    if (v0 < resmin) { resmin = v0; sp = SPAN0; }
    if (v1 < resmin) { resmin = v1; sp = SPAN1; }
    if (v2 < resmin) { resmin = v2; sp = SPAN2; }
    if (alpha > 0.0 && alpha <= 10.0 && resmin < v2 && resmin > 0.0) {
        double tmp = resmin * rcp64(v2);
        if (tmp < 1.e-7) tmp = 1.e-7;
        double e = 10.0 - alpha;
        double pw = (e == 1.0) ? tmp : pow(tmp, e);
        sp += (SPAN2 - sp) * pw;
    }
    return sp;
}

// Listing 1 lines 83-95 (R10): clamp the span and interpolate between smooths.
__device__ __forceinline__ double interp_spans(double sps, double A0, double A1, double A2)
{
    if (sps <= SPAN0) sps = SPAN0;
    if (sps >= SPAN2) sps = SPAN2;
    double f = sps - SPAN1;
    // multiply by the reciprocal of the span gap (1 ulp from the listing's division)
    constexpr double G0 = 1.0 / (SPAN0 - SPAN1), G2 = 1.0 / (SPAN2 - SPAN1);
    if (f < 0.0) {
        f *= G0;
        return (1.0 - f) * A1 + f * A0;
    }
    f *= G2;
    return (1.0 - f) * A1 + f * A2;
}

// Window [lo, lo+K) of point j: symmetric, pinned at the ends (O4).
__device__ __forceinline__ int window_lo(int j, int ibw, int K, int n)
{
    int lo = j - ibw;
    lo = lo < 0 ? 0 : lo;
    int hi = n - K;
    return lo > hi ? hi : lo;
}

}  // namespace ss

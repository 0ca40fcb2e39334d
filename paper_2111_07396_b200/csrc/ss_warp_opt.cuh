// ss_warp_opt.cuh -- warp-per-eval kernel for the options Listing 1 has beside the default call:
// periodic windows (iper = 2) and a fixed span (span > 0), n <= 256.
//
// Same skeleton as warp_kernel (fold, register sort, gather, exact-order check, hand-over of what cannot be decided
// exactly).  The smoother differs in one respect: EVERY span, the tweeter included, is evaluated by differences of the
// prefix arrays through a per-point table of window ends, because a periodic window is two ranges -- the part inside
// [0, n) and the part that wrapped, whose abscissae count as x - 1 or x + 1 -- and has no pinned ends; the halo /
// sliding-sum tweeter and the end-clamp broadcasts of the default kernel do not apply.  A window is
//     [lo, hi) + [blo, bhi) shifted by s,   s = -1 (wrapped below 0), +1 (wrapped above n-1), 0 (no wrap)
// and its moments follow from the unshifted sums: Swx += s bw, Swxx += 2 s bwx + bw, Sxz += s bz.
// MODE: 0 = CV, 1 = GV (variable span), 2 = fixed span (one smooth of y, both modes alike).
#pragma once
#include "ss_warp_kernel.cuh"

namespace ss {

template <int C> struct WarpOptCfg {
    static constexpr int WPC = 8;
    static constexpr int MINB = C <= 6 ? 2 : 1;        // 20C tensor-memory columns per warp, two warps per lane quarter
    static constexpr uint32_t TCOLS_WARP = 20 * C;
    static constexpr uint32_t TCOLS_NEED = 2 * TCOLS_WARP;
    static constexpr uint32_t TCOLS = TCOLS_NEED <= 64 ? 64 : (TCOLS_NEED <= 128 ? 128 : (TCOLS_NEED <= 256 ? 256 : 512));
    static_assert(TCOLS * MINB <= 512, "tensor memory over-subscribed");
};

template <int C>
inline size_t warp_opt_smem_bytes()
{
    return (size_t)3 * 32 * C * 8 + (size_t)WarpOptCfg<C>::WPC * ((size_t)3 * C * WROW * 16);
}

// window table entry of one point and span: word a = lo | hi << 16, word b = blo | bhi << 14 | (s + 1) << 30
// (element indices of the transposed arrays, < 2^14)
struct WinIdx { int lo, hi, blo, bhi; double s; };
__device__ __forceinline__ WinIdx win_unpack(int a, int b)
{
    WinIdx w;
    w.lo = a & 0xffff; w.hi = (int)((unsigned)a >> 16);
    w.blo = b & 0x3fff; w.bhi = (b >> 14) & 0x3fff;
    w.s = (double)((int)((unsigned)b >> 30) - 1);
    return w;
}

template <int C, int MODE>
__global__ void __launch_bounds__(WarpOptCfg<C>::WPC * 32, WarpOptCfg<C>::MINB) warp_opt_kernel(const EvalParams p)
{
    using Cfg = WarpOptCfg<C>;
    constexpr int WPC = Cfg::WPC;
    constexpr bool GV = MODE == 1, FIXED = MODE == 2;
    constexpr int ASZ = C * WROW;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double s_best[WPC];
    __shared__ long long s_bestk[WPC];
    __shared__ double s_kc[8];
    __shared__ uint32_t s_tmem;
    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
    const int item = blockIdx.x;
    const int li = item / p.chunks_per_obj, ch = item - li * p.chunks_per_obj;
    const int ri = p.list[li];
    const ObjRec rec = p.recs[ri];
    if (rec.dup) {
        if (tid == 0) {
            const unsigned pos = atomicAdd(p.defer_count, 1u);
            if (pos < p.defer_capacity)
                p.defer_entries[pos] = DEFER_ITEM | ((unsigned long long)ri << 32) | (unsigned long long)ch;
            else
                p.defer_count[1] = 1u;
        }
        return;
    }
    const int n = uni(rec.n);
    const bool per = p.iper == 2;                    // phases are in [0, 1): jper = iper

    // half-widths: the three spans, or the caller's fixed one in slot 0; a periodic window never exceeds n points (R8)
    int ibw[3], Kw[3];
#pragma unroll
    for (int i = 0; i < 3; i++) {
        int b = FIXED ? rec.ibw_fixed : rec.ibw[i];
        int k = 2 * b + 1;
        if (k > n) { k = n; if (per) { b = (n - 1) / 2; k = 2 * b + 1; } }
        ibw[i] = uni(b); Kw[i] = uni(k);
    }
    const int q1 = uni(rec.q1), q3 = uni(rec.q3);
    const int q1l = q1 / C, q1s = q1 % C, q3l = q3 / C, q3s = q3 % C;
    if (tid == 0) {
#pragma unroll
        for (int i = 0; i < 3; i++) {
            s_kc[2 * i] = 1.0 / (1.0 - 1.0 / (double)Kw[i]); s_kc[2 * i + 1] = 1.0 / (1.0 - 2.0 / (double)Kw[i]);
        }
        s_kc[6] = rec.chi0; s_kc[7] = rec.chi0 > 0.0 ? 1.0 / rec.chi0 : 0.0;
    }
    EvalConst KW;
    KW.bexp = 10.0 - p.alpha;
    KW.bass = (p.alpha > 0.0 && p.alpha <= 10.0) ? (KW.bexp == 1.0 ? 1 : 2) : 0;

    double* o_tt = reinterpret_cast<double*>(smem_raw);
    double* o_y = o_tt + 32 * C;
    double* o_w = o_y + 32 * C;
    double2* E01 = reinterpret_cast<double2*>(smem_raw + (size_t)3 * 32 * C * 8 + (size_t)warp * ((size_t)3 * ASZ * 16));
    double2* E23 = E01 + ASZ;
    double2* E45 = E23 + ASZ;
    const ScanMask mk = make_scan_mask(lane);
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                     :: "r"((uint32_t)__cvta_generic_to_shared(&s_tmem)), "n"(Cfg::TCOLS) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    for (int j = tid; j < n; j += WPC * 32) {
        o_tt[j] = p.tt[rec.off + j];
        o_y[j] = p.yc[rec.off + j];
        o_w[j] = p.w[rec.off + j];
    }
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = s_tmem + ((uint32_t)(warp & 3) << 21) + (uint32_t)(warp >> 2) * Cfg::TCOLS_WARP;
    constexpr uint32_t T_A0 = 0, T_ISW = 6 * C, T_XB = 8 * C, T_G0 = 10 * C, T_Y = 12 * C, T_W = 14 * C;   // T_W + 2C i: span i
    {
#pragma unroll
        for (int i = 0; i < (FIXED ? 1 : 3); i++) {
            int wa[C], wb[C];
#pragma unroll
            for (int s = 0; s < C; s++) {
                const int j = lane * C + s;
                int lo, hi, blo = 0, bhi = 0, sg = 1;      // sg = s + 1
                if (per && j < n) {
                    lo = j - ibw[i]; hi = j + ibw[i] + 1;
                    if (lo < 0) { blo = lo + n; bhi = n; lo = 0; sg = 0; }
                    else if (hi > n) { blo = 0; bhi = hi - n; hi = n; sg = 2; }
                } else {
                    lo = window_lo(j, ibw[i], Kw[i], n); hi = lo + Kw[i];
                }
                wa[s] = wst<C>(lo) | (wst<C>(hi) << 16);
                wb[s] = wst<C>(blo) | (wst<C>(bhi) << 14) | (sg << 30);
            }
            tmem_park_words<C>(tmem + T_W + 2 * C * i, wa);
            tmem_park_words<C>(tmem + T_W + 2 * C * i + C, wb);
        }
        tmem_wait_st();
    }

    const int64_t c0 = p.k_begin + (int64_t)ch * p.chunk;
    const int64_t c1 = min(c0 + (int64_t)p.chunk, p.k_end);
    const int per_warp = p.chunk / WPC;
    const int64_t k0 = c0 + (int64_t)warp * per_warp;
    const int64_t k1 = min(k0 + (int64_t)per_warp, c1);
    double best = -INFINITY;
    int64_t best_k = INT64_MAX;
    double* prow = p.pgram ? p.pgram + (rec.obj - p.pgram_row0) * p.pgram_row_stride - p.pgram_k0 : nullptr;
    double stash = 0.0;
    int64_t kb = k0;

    // x-moments and the y-fit of one window from the primary arrays
    struct Fit { double isw, xb, isxx, Sy, sxy, Syy; };
    auto primary = [&](int a, int b, double vsmlsq, bool want_yy) {
        const WinIdx wn = win_unpack(a, b);
        const double* E4 = reinterpret_cast<const double*>(E45);
        const double2 l0 = E01[wn.lo], h0 = E01[wn.hi], l1 = E23[wn.lo], h1 = E23[wn.hi];
        double Sw = h0.x - l0.x, Swx = h0.y - l0.y, Swxx = h1.x - l1.x, Sy = h1.y - l1.y, Sxy, Syy = 0.0;
        if (GV) { const double2 l2 = E45[wn.lo], h2 = E45[wn.hi]; Sxy = h2.x - l2.x; Syy = h2.y - l2.y; }
        else Sxy = E4[wn.hi] - E4[wn.lo];
        if (per && wn.s != 0.0) {      // only the lanes whose window wraps
            const double2 m0 = E01[wn.blo], n0 = E01[wn.bhi], m1 = E23[wn.blo], n1 = E23[wn.bhi];
            const double bw = n0.x - m0.x, bwx = n0.y - m0.y, bwxx = n1.x - m1.x, by = n1.y - m1.y;
            double bxy, byy = 0.0;
            if (GV) { const double2 m2 = E45[wn.blo], n2 = E45[wn.bhi]; bxy = n2.x - m2.x; byy = n2.y - m2.y; }
            else bxy = E4[wn.bhi] - E4[wn.blo];
            Sw += bw; Swx += bwx + wn.s * bw; Swxx += bwxx + 2.0 * wn.s * bwx + bw;      // s*s = 1 where bw != 0
            Sy += by; Sxy += bxy + wn.s * by; Syy += byy;
        }
        (void)want_yy;
        Fit f;
        f.isw = rcp64(Sw); f.xb = Swx * f.isw;
        const double sxx = Swxx - f.xb * Swx;
        f.isxx = sxx > vsmlsq ? rcp64(sxx) : 0.0;
        f.Sy = Sy; f.sxy = Sxy - f.xb * Sy; f.Syy = Syy;
        return f;
    };
    // (Sz, Sxz) of one window from a secondary pair array
    auto secondary = [&](const double2* Ez, int a, int b, double& Sz, double& Sxz) {
        const WinIdx wn = win_unpack(a, b);
        const double2 l = Ez[wn.lo], h = Ez[wn.hi];
        Sz = h.x - l.x; Sxz = h.y - l.y;
        if (per && wn.s != 0.0) {
            const double2 m = Ez[wn.blo], q = Ez[wn.bhi];
            const double bz = q.x - m.x;
            Sz += bz; Sxz += (q.y - m.y) + wn.s * bz;
        }
    };

    for (int64_t k = k0; k < k1; k++) {
        const double f = freq_of(p.f_min, p.df, k);
        bool defer = false;
        double P = 0.0;
        // ---- P1 fold, P2 sort, gather, exact-order check (as warp_eval)
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
        double x[C], y[C], w[C];
        double vsmlsq;
        {
            double phi[C];
            bool bad = false;
#pragma unroll
            for (int s = 0; s < C; s++) {
                const int i = (int)(key[s] & 0xffu);
                if (lane * C + s < n) { phi[s] = fold_phase(o_tt[i], f); y[s] = o_y[i]; w[s] = o_w[i]; }
                else { phi[s] = 4.0; y[s] = 0.0; w[s] = W_PAD; }
            }
            double nxt = shfl_down_d(phi[0], 1);
            if (lane == 31) nxt = 8.0;
#pragma unroll
            for (int s = 0; s < C; s++) {
                const double nx = s + 1 < C ? phi[s + 1 < C ? s + 1 : 0] : nxt;
                if (lane * C + s + 1 < n && nx <= phi[s]) bad = true;
            }
            const double p1 = bcast_slot<C>(phi, q1s, q1l);
            const double p3 = bcast_slot<C>(phi, q3s, q3l);
            defer = __any_sync(0xffffffffu, bad);
            const double scale = p3 - p1;
            vsmlsq = 1.e-6 * scale * scale;
#pragma unroll
            for (int s = 0; s < C; s++) x[s] = (lane * C + s < n) ? phi[s] - 0.5 : 0.0;
        }
        if (!defer) {
            // ---- prefix sums of the weighted moments
            {
                double a[C], b[C], c[C];
#pragma unroll
                for (int s = 0; s < C; s++) { a[s] = w[s]; b[s] = w[s] * x[s]; }
                pair_prefix_store<C>(a, b, E01, lane, mk);
#pragma unroll
                for (int s = 0; s < C; s++) { c[s] = b[s] * x[s]; a[s] = w[s] * y[s]; }
                pair_prefix_store<C>(c, a, E23, lane, mk);
#pragma unroll
                for (int s = 0; s < C; s++) b[s] = b[s] * y[s];
                if (GV) {
#pragma unroll
                    for (int s = 0; s < C; s++) c[s] = a[s] * y[s];
                    pair_prefix_store<C>(b, c, E45, lane, mk);
                } else {
                    single_prefix_store<C>(b, reinterpret_cast<double*>(E45), lane, mk);
                }
            }
            __syncwarp();
            double chi2 = 0.0;
            if (FIXED) {
                // ---- Listing 1 lines 51-55: one smooth of y at the caller's span
                int wa[C], wb[C];
                tmem_fetch_words_any<C>(tmem + T_W, wa); tmem_fetch_words_any<C>(tmem + T_W + C, wb);
#pragma unroll
                for (int s = 0; s < C; s++) {
                    const Fit ft = primary(wa[s], wb[s], vsmlsq, false);
                    const double smo = ft.Sy * ft.isw + ft.sxy * ft.isxx * (x[s] - ft.xb);
                    const double r = y[s] - smo;
                    chi2 += w[s] * r * r;
                }
            } else if (GV) {
                double A[3][C], Gs[3][C];
#pragma unroll
                for (int i = 0; i < 3; i++) {
                    int wa[C], wb[C];
                    tmem_fetch_words_any<C>(tmem + T_W + 2 * C * i, wa); tmem_fetch_words_any<C>(tmem + T_W + 2 * C * i + C, wb);
#pragma unroll
                    for (int s = 0; s < C; s++) {
                        const Fit ft = primary(wa[s], wb[s], vsmlsq, true);
                        const double yb = ft.Sy * ft.isw, b = ft.sxy * ft.isxx;
                        A[i][s] = yb + b * (x[s] - ft.xb);
                        const double rss = (ft.Syy - yb * ft.Sy) - b * ft.sxy;
                        Gs[i][s] = sqrt64(rss * ft.isw) * (ft.isxx != 0.0 ? s_kc[2 * i + 1] : s_kc[2 * i]);
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
                // ---- CV
                double r0[C], r1[C], r2[C];
                double m_isw[C], m_xb[C], m_g[C];
                int amin = 0x7fffffff;
#pragma unroll
                for (int i = 0; i < 3; i++) {
                    int wa[C], wb[C];
                    tmem_fetch_words_any<C>(tmem + T_W + 2 * C * i, wa); tmem_fetch_words_any<C>(tmem + T_W + 2 * C * i + C, wb);
                    double Ai[C], q_isw[C], q_xb[C], q_g[C];
#pragma unroll
                    for (int s = 0; s < C; s++) {
                        const Fit ft = primary(wa[s], wb[s], vsmlsq, false);
                        const double dx = x[s] - ft.xb, g = ft.isxx * dx;
                        q_isw[s] = ft.isw; q_xb[s] = ft.xb; q_g[s] = g;
                        Ai[s] = ft.Sy * ft.isw + ft.sxy * g;
                        const double a = 1.0 - w[s] * (ft.isw + dx * g);
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
                if (__any_sync(0xffffffffu, amin < 0x00100000)) defer = true;      // a <= 0: the residual carries (R23)
                __syncwarp();
                if (!defer) {
                    auto mid_store = [&](const double (&z)[C], double2* Ez) {
                        double a[C], b[C];
#pragma unroll
                        for (int s = 0; s < C; s++) { a[s] = w[s] * z[s]; b[s] = a[s] * x[s]; }
                        pair_prefix_store<C>(a, b, Ez, lane, mk);
                    };
                    int w1a[C], w1b[C];
                    tmem_fetch_words_any<C>(tmem + T_W + 2 * C, w1a); tmem_fetch_words_any<C>(tmem + T_W + 2 * C + C, w1b);
                    auto mid_load = [&](const double2* Ez, double (&out)[C]) {
#pragma unroll
                        for (int s = 0; s < C; s++) {
                            double Sz, Sxz;
                            secondary(Ez, w1a[s], w1b[s], Sz, Sxz);
                            out[s] = Sz * m_isw[s] + (Sxz - m_xb[s] * Sz) * m_g[s];
                        }
                    };
                    double sp[C];
                    {
                        mid_store(r0, E01); mid_store(r1, E23); mid_store(r2, E45);
                        __syncwarp();
                        double R0[C], R1[C], R2[C];
                        mid_load(E01, R0); mid_load(E23, R1); mid_load(E45, R2);
#pragma unroll
                        for (int s = 0; s < C; s++) sp[s] = pick_span_w(R0[s], R1[s], R2[s], KW);
                    }
                    __syncwarp();
                    mid_store(sp, E01);
                    __syncwarp();
                    double B[C];
                    mid_load(E01, B);
                    tmem_wait_st();
                    {
                        double a0[C], a1[C], a2[C];
                        tmem_fetch<C>(tmem + T_A0, a0); tmem_fetch<C>(tmem + T_A0 + 2 * C, a1); tmem_fetch<C>(tmem + T_A0 + 4 * C, a2);
#pragma unroll
                        for (int s = 0; s < C; s++) B[s] = interp_spans(B[s], a0[s], a1[s], a2[s]);
                    }
                    mid_store(B, E23);                      // final tweeter smooth
                    __syncwarp();
                    int w0a[C], w0b[C];
                    tmem_fetch_words_any<C>(tmem + T_W, w0a); tmem_fetch_words_any<C>(tmem + T_W + C, w0b);
                    double t_isw[C], t_xb[C], t_g[C], yy[C];
                    tmem_fetch<C>(tmem + T_ISW, t_isw); tmem_fetch<C>(tmem + T_XB, t_xb); tmem_fetch<C>(tmem + T_G0, t_g);
                    tmem_fetch<C>(tmem + T_Y, yy);
#pragma unroll
                    for (int s = 0; s < C; s++) {
                        double Sz, Sxz;
                        secondary(E23, w0a[s], w0b[s], Sz, Sxz);
                        const double smo = Sz * t_isw[s] + (Sxz - t_xb[s] * Sz) * t_g[s];
                        const double r = yy[s] - smo;
                        chi2 += w[s] * r * r;
                    }
                    __syncwarp();
                }
            }
            if (!defer) {
#pragma unroll
                for (int d = 16; d > 0; d >>= 1) chi2 += __shfl_xor_sync(0xffffffffu, chi2, d);
                P = (s_kc[6] - chi2) * s_kc[7];
            }
            __syncwarp();
        }
        if (defer) {
            if (lane == 0) {
                const unsigned pos = atomicAdd(p.defer_count, 1u);
                if (pos < p.defer_capacity)
                    p.defer_entries[pos] = ((unsigned long long)ri << 32) | (unsigned long long)(k - p.k_begin);
                else
                    p.defer_count[1] = 1u;
            }
            P = 0.0;
        } else if (P > best) { best = P; best_k = k; }
        if (lane == (int)(k - kb)) stash = P;
        if (k - kb == 31 || k == k1 - 1) {
            if (prow && kb + lane <= k) prow[kb + lane] = stash;
            kb = k + 1;
        }
    }
    if (lane == 0) { s_best[warp] = best; s_bestk[warp] = best_k; }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(s_tmem), "n"(Cfg::TCOLS) : "memory");
    }
    if (tid == 0) {
        for (int q = 1; q < WPC; q++)
            if (s_best[q] > best || (s_best[q] == best && s_bestk[q] < best_k)) { best = s_best[q]; best_k = s_bestk[q]; }
        const int64_t slot = (int64_t)ri * p.chunks_total + p.chunk_base + ch;
        p.part_val[slot] = best;
        p.part_idx[slot] = best_k == INT64_MAX ? c0 : best_k;
    }
}

template <int C, int MODE>
inline ss_status_t launch_warp_opt_variant(const EvalParams& p, int64_t n_items, cudaStream_t stream)
{
    const size_t smem = warp_opt_smem_bytes<C>();
    if (cudaFuncSetAttribute(warp_opt_kernel<C, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
        return SS_ERR_CUDA;
    warp_opt_kernel<C, MODE><<<(unsigned)n_items, WarpOptCfg<C>::WPC * 32, smem, stream>>>(p);
    return cudaGetLastError() == cudaSuccess ? SS_OK : SS_ERR_CUDA;
}

}  // namespace ss

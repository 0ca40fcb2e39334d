/*
 * ss_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, double-precision CPU statement of the batched SuperSmoother
 * periodogram of arXiv 2111.07396 (Gowanlock et al.), written from the paper
 * and SURVEY.md section 8(c).  It shares no code with
 * the CUDA path (paper_2111_07396_b200/csrc) and neither includes the other.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may call it.
 *
 * Two variants of the running-line smoother, same definitions:
 *   variant 0 "definition": every window moment is re-summed directly from the
 *       window's members in long double (two-pass, centred).  O(n*K) per smooth.
 *   variant 1 "fast": Friedman's (1984) updating formulas in double, O(n) per
 *       smooth -- the algorithm PAPER.md:121 says Listing 1's `smoothkernel`
 *       was "directly ported from".  Used for timing and full-size parity; pinned
 *       against variant 0 in tests/test_oracle_pins.py.
 *
 * Citations: "PAPER.md:N" is a line of the paper text; "O#/R#" are the step and
 * reading numbers of SURVEY.md section 8(c), restated in DESIGN.md.
 *
 * Parity status: the CV smoother's structure is pinned by
 * Listing 1 and by the pins in tests/; value-level parity with the authors' code
 * is UNPINNED (the paper prints no value).  The GV variant follows reading R12
 * (the paper gives no formula): PARITY UNPINNED with the authors' code.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/build.py).
 * -ffp-contract=off is normative for the fold (R2).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double ld;

#define SS_MODE_CV 0
#define SS_MODE_GV 1

/* spans: tweeter, midrange, woofer */
static const double SPANS[3] = {0.05, 0.2, 0.5};

/* ------------------------------------------------------------------------- */
/* O4: window geometry (R21, R25).  ibw = max(2, floor(0.5*span*n + 0.5)),      */
/* K = min(2*ibw+1, n); non-periodic window of point j = [lo, lo+K),          */
/* lo = clamp(j-ibw, 0, n-K).                                                 */
/* ------------------------------------------------------------------------- */
static int half_width(int n, double span)
{
    int ibw = (int)floor(0.5 * span * (double)n + 0.5);
    if (ibw < 2) ibw = 2;
    return ibw;
}

void sso_window(int n, double span, int j, int *lo_out, int *K_out)
{
    int ibw = half_width(n, span);
    int K = 2 * ibw + 1;
    if (K > n) K = n;
    int lo = j - ibw;
    if (lo < 0) lo = 0;
    if (lo > n - K) lo = n - K;
    *lo_out = lo;
    *K_out = K;
}

/* Average smo over maximal runs of equal x (x[j+1] <= x[j]), w-weighted (O4 last
 * bullet, R24).  */
static void average_ties(int n, const double *x, const double *w, double *smo)
{
    int j = 0;
    while (j < n) {
        int j0 = j;
        double sy = smo[j] * w[j];
        double fbw = w[j];
        while (j < n - 1 && x[j + 1] <= x[j]) {
            j++;
            sy += w[j] * smo[j];
            fbw += w[j];
        }
        if (j > j0) {
            double a = 0.0;
            if (fbw > 0.0) a = sy / fbw;
            for (int i = j0; i <= j; i++) smo[i] = a;
        }
        j++;
    }
}

/* Diagnostics (O9): smallest relative margin seen on a discontinuous branch that
 * has no "alternative" re-evaluation (slope guard Sxx > vsmlsq, a_j > 0).  */
typedef struct {
    double guard_margin;
} diag_t;

static void diag_guard(diag_t *d, double lhs, double rhs)
{
    if (!d) return;
    double den = fmax(fabs(lhs), fabs(rhs));
    double m = den > 0.0 ? fabs(lhs - rhs) / den : 1.0;
    if (m < d->guard_margin) d->guard_margin = m;
}

/* ------------------------------------------------------------------------- */
/* O4, variant 0: running-line smoother by direct window sums in long double. */
/* z = ordinates, cv != 0 -> also the leave-one-out residuals acvr.           */
/* gv != NULL -> also GV score ingredients (O6): gv[j] = sqrt(RSS/Sw)/(1-p/K). */
/* jper = 1 non-periodic, 2 periodic (x wraps by +-1, R8/A9).                 */
/* ------------------------------------------------------------------------- */
static void smooth_def(int n, const double *x, const double *z, const double *w,
                       double span, int jper, double vsmlsq, int cv,
                       double *smo, double *acvr, double *gv, int ties, diag_t *dg)
{
    int ibw = half_width(n, span);
    int K = 2 * ibw + 1;
    if (K > n) { K = n; if (jper == 2) ibw = (n - 1) / 2, K = 2 * ibw + 1; }
    for (int j = 0; j < n; j++) {
        int lo;
        if (jper == 2) lo = j - ibw;
        else { lo = j - ibw; if (lo < 0) lo = 0; if (lo > n - K) lo = n - K; }
        ld Sw = 0, Swx = 0, Swz = 0;
        for (int m = lo; m < lo + K; m++) {
            int idx = m; ld xv;
            if (idx < 0) { idx += n; xv = (ld)x[idx] - 1; }
            else if (idx >= n) { idx -= n; xv = (ld)x[idx] + 1; }
            else xv = x[idx];
            Sw += w[idx]; Swx += (ld)w[idx] * xv; Swz += (ld)w[idx] * z[idx];
        }
        ld xb = 0, zb = 0;
        if (Sw > 0) { xb = Swx / Sw; zb = Swz / Sw; }
        ld Sxx = 0, Sxz = 0, Szz = 0;
        for (int m = lo; m < lo + K; m++) {
            int idx = m; ld xv;
            if (idx < 0) { idx += n; xv = (ld)x[idx] - 1; }
            else if (idx >= n) { idx -= n; xv = (ld)x[idx] + 1; }
            else xv = x[idx];
            ld dx = xv - xb, dz = (ld)z[idx] - zb;
            Sxx += (ld)w[idx] * dx * dx; Sxz += (ld)w[idx] * dx * dz; Szz += (ld)w[idx] * dz * dz;
        }
        diag_guard(dg, (double)Sxx, vsmlsq);
        int slope_on = (Sxx > (ld)vsmlsq);
        ld b = slope_on ? Sxz / Sxx : 0;
        ld s = b * ((ld)x[j] - xb) + zb;
        smo[j] = (double)s;
        if (cv) {
            ld h = 0;
            if (Sw > 0) h = 1 / Sw;
            if (slope_on) h += ((ld)x[j] - xb) * ((ld)x[j] - xb) / Sxx;
            ld a = 1 - (ld)w[j] * h;
            diag_guard(dg, (double)((ld)w[j] * h), 1.0);
            acvr[j] = 0.0;
            if (a > 0) acvr[j] = (double)(fabsl((ld)z[j] - s) / a);
            else if (j > 0) acvr[j] = acvr[j - 1];
        }
        if (gv) {
            /* RSS of the window's own line fit, summed directly (O6). */
            ld rss = 0;
            for (int m = lo; m < lo + K; m++) {
                int idx = m; ld xv;
                if (idx < 0) { idx += n; xv = (ld)x[idx] - 1; }
                else if (idx >= n) { idx -= n; xv = (ld)x[idx] + 1; }
                else xv = x[idx];
                ld r = (ld)z[idx] - zb - b * (xv - xb);
                rss += (ld)w[idx] * r * r;
            }
            ld p = slope_on ? 2 : 1;
            ld g = 0;
            if (Sw > 0) g = sqrtl(rss / Sw) / (1 - p / (ld)K);
            gv[j] = (double)g;
        }
    }
    if (ties) average_ties(n, x, w, smo);
}

/* ------------------------------------------------------------------------- */
/* O4, variant 1: Friedman's updating formulas (double), the routine PAPER.md: */
/* 121 refers to.  Same windows as variant 0: the first K points are loaded,   */
/* the window then slides only while both ends stay inside [0,n) (non-        */
/* periodic), or always (periodic, starting centred one point before j=0).    */
/* vary (sum w (z-zm)^2) is carried only when the GV score is requested.      */
/* ------------------------------------------------------------------------- */
typedef struct { double xm, zm, var, cvar, vary, fbw; } run_t;

static void run_add(run_t *r, double xti, double zi, double wt)
{
    double fbo = r->fbw;
    r->fbw = r->fbw + wt;
    if (r->fbw > 0.0) {
        r->xm = (fbo * r->xm + wt * xti) / r->fbw;
        r->zm = (fbo * r->zm + wt * zi) / r->fbw;
    }
    double tmp = 0.0, tmz = 0.0;
    if (fbo > 0.0) {
        tmp = r->fbw * wt * (xti - r->xm) / fbo;
        tmz = r->fbw * wt * (zi - r->zm) / fbo;
    }
    r->var += tmp * (xti - r->xm);
    r->cvar += tmp * (zi - r->zm);
    r->vary += tmz * (zi - r->zm);
}

static void run_del(run_t *r, double xto, double zo, double wt)
{
    double fbo = r->fbw;
    r->fbw = r->fbw - wt;
    double tmp = 0.0, tmz = 0.0;
    if (r->fbw > 0.0) {
        tmp = fbo * wt * (xto - r->xm) / r->fbw;
        tmz = fbo * wt * (zo - r->zm) / r->fbw;
    }
    r->var -= tmp * (xto - r->xm);
    r->cvar -= tmp * (zo - r->zm);
    r->vary -= tmz * (zo - r->zm);
    if (r->fbw > 0.0) {
        r->xm = (fbo * r->xm - wt * xto) / r->fbw;
        r->zm = (fbo * r->zm - wt * zo) / r->fbw;
    }
}

static void smooth_fast(int n, const double *x, const double *z, const double *w,
                        double span, int jper, double vsmlsq, int cv,
                        double *smo, double *acvr, double *gv, int ties, diag_t *dg)
{
    int ibw = half_width(n, span);
    int it = 2 * ibw + 1;
    if (it > n) { it = n; if (jper == 2) ibw = (n - 1) / 2, it = 2 * ibw + 1; }
    run_t r = {0, 0, 0, 0, 0, 0};
    for (int i = 0; i < it; i++) {
        int j = i;
        double xti;
        if (jper == 2) j = i - ibw - 1;
        if (j < 0) { j += n; xti = x[j] - 1.0; } else xti = x[j];
        run_add(&r, xti, z[j], w[j]);
    }
    for (int j = 0; j < n; j++) {
        int out = j - ibw - 1, in = j + ibw;
        if (jper == 2 || (out >= 0 && in < n)) {
            double xto, xti;
            if (out < 0) { out += n; xto = x[out] - 1.0; } else xto = x[out];
            if (in >= n) { in -= n; xti = x[in] + 1.0; } else xti = x[in];
            run_del(&r, xto, z[out], w[out]);
            run_add(&r, xti, z[in], w[in]);
        }
        diag_guard(dg, r.var, vsmlsq);
        int slope_on = (r.var > vsmlsq);
        double a = slope_on ? r.cvar / r.var : 0.0;
        smo[j] = a * (x[j] - r.xm) + r.zm;
        if (cv) {
            double h = 0.0;
            if (r.fbw > 0.0) h = 1.0 / r.fbw;
            if (slope_on) h += (x[j] - r.xm) * (x[j] - r.xm) / r.var;
            acvr[j] = 0.0;
            double aa = 1.0 - w[j] * h;
            diag_guard(dg, w[j] * h, 1.0);
            if (aa > 0.0) acvr[j] = fabs(z[j] - smo[j]) / aa;
            else if (j > 0) acvr[j] = acvr[j - 1];
        }
        if (gv) {
            /* one-scan form of the window RSS: Szz - b*Sxz, clamped at 0 (O6) */
            double rss = r.vary - a * r.cvar;
            if (rss < 0.0) rss = 0.0;
            double p = slope_on ? 2.0 : 1.0;
            double g = 0.0;
            if (r.fbw > 0.0) g = sqrt(rss / r.fbw) / (1.0 - p / (double)it);
            gv[j] = g;
        }
    }
    if (ties) average_ties(n, x, w, smo);
}

static void smooth_any(int variant, int n, const double *x, const double *z, const double *w,
                       double span, int jper, double vsmlsq, int cv,
                       double *smo, double *acvr, double *gv, int ties, diag_t *dg)
{
    if (variant == 0) smooth_def(n, x, z, w, span, jper, vsmlsq, cv, smo, acvr, gv, ties, dg);
    else smooth_fast(n, x, z, w, span, jper, vsmlsq, cv, smo, acvr, gv, ties, dg);
}

/* Exposed for the pins: one call of the smooth primitive S(z; span, cv).  */
void sso_smooth(int variant, int n, const double *x, const double *z, const double *w,
                double span, int jper, double vsmlsq, int cv, double *smo, double *acvr)
{
    double *tmp = NULL;
    if (cv && !acvr) acvr = tmp = (double *)malloc(sizeof(double) * (size_t)n);
    smooth_any(variant, n, x, z, w, span, jper, vsmlsq, cv, smo, acvr, NULL, 1, NULL);
    free(tmp);
}

/* ------------------------------------------------------------------------- */
/* O5 / O6: Friedman's variable-span smoother as Listing 1 states it          */
/* (PAPER.md:127-297), CV mode, and the single-scan GV variant (R12).         */
/*                                                                            */
/* x sorted ascending, y, w gathered.  span > 0 -> fixed span. */
/* force_j >= 0: diagnostics hook (R29) -- at point force_j the span argmin   */
/* is overridden to index force_i.                                            */
/* Returns in *pick_margin the smallest relative gap between the winning      */
/* residual/score and a losing one over all points, and where it happened.    */
/* ------------------------------------------------------------------------- */
typedef struct {
    double pick_margin;   /* min over j, i != c of |v_i - v_c| / max(|v_i|,|v_c|) */
    int pick_j, pick_alt; /* the point and the runner-up span index there        */
    diag_t guard;
} sup_diag_t;

static void span_pick(int n, int j, const double v[3], double alpha, int force_j, int force_i,
                      double *sp_out, sup_diag_t *sd)
{
    /* Listing 1 lines 63-77: strict '<' => smallest span wins ties */
    double resmin = 1.e20;
    int c = -1;
    for (int i = 0; i < 3; i++) {
        if (v[i] < resmin) { resmin = v[i]; c = i; }
    }
    if (j == force_j && force_i >= 0) { c = force_i; resmin = v[c]; }
    double sp = (c >= 0) ? SPANS[c] : 0.0;   /* c < 0 cannot occur with finite data (R27) */
    if (sd && c >= 0) {
        for (int i = 0; i < 3; i++) {
            if (i == c) continue;
            double den = fmax(fabs(v[i]), fabs(v[c]));
            double m = den > 0.0 ? fabs(v[i] - v[c]) / den : 0.0;
            if (m < sd->pick_margin) { sd->pick_margin = m; sd->pick_j = j; sd->pick_alt = i; }
        }
    }
    if (alpha > 0.0 && alpha <= 10.0 && resmin < v[2] && resmin > 0.0) {
        double tmp = resmin / v[2];
        if (tmp < 1.e-7) tmp = 1.e-7;
        sp += (SPANS[2] - sp) * pow(tmp, 10.0 - alpha);
    }
    *sp_out = sp;
    (void)n;
}

static double interp_spans(double sps, double A0, double A1, double A2)
{
    /* Listing 1 lines 83-95, with the dropped `if (f<0) {` restored (R10) */
    if (sps <= SPANS[0]) sps = SPANS[0];
    if (sps >= SPANS[2]) sps = SPANS[2];
    double f = sps - SPANS[1];
    if (f < 0.0) {
        f /= SPANS[0] - SPANS[1];
        return (1.0 - f) * A1 + f * A0;
    } else {
        f /= SPANS[2] - SPANS[1];
        return (1.0 - f) * A1 + f * A2;
    }
}

/* sc: scratch of 8*n doubles laid out exactly as Listing 1 uses it. */
static void supsmu(int variant, int mode, int n, const double *x, const double *y, const double *w,
                   int iper, double span, double alpha, double *smo, double *sc,
                   int force_j, int force_i, sup_diag_t *sd)
{
    int i, j, jper;
    double sw, sy, a, scale, vsmlsq;
    diag_t *dg = sd ? &sd->guard : NULL;

    if (x[n - 1] <= x[0]) {
        sy = 0.0; sw = sy;
        for (j = 0; j < n; j++) { sy = sy + w[j] * y[j]; sw = sw + w[j]; }
        a = 0.0;
        if (sw > 0) a = sy / sw;
        for (j = 0; j < n; j++) smo[j] = a;
        return;
    }
    i = n / 4 - 1;                                /* PAPER.md:188-194, no widening loop (R11) */
    j = 3 * (i + 1) - 1;
    scale = x[j] - x[i];
    vsmlsq = 1.e-6 * scale * scale;
    jper = iper;                                  /* restored line (R10) */
    if (iper == 2 && (x[0] < 0 || x[n - 1] > 1)) jper = 1;
    if (jper < 1 || jper > 2) jper = 1;
    if (span > 0) {                               /* fixed span */
        smooth_any(variant, n, x, y, w, span, jper, vsmlsq, 1, smo, sc, NULL, 1, dg);
        return;
    }

    if (mode == SS_MODE_CV) {
        /* three smooths with LOO residuals, each residual smoothed at midrange */
        for (i = 0; i < 3; i++) {
            smooth_any(variant, n, x, y, w, SPANS[i], jper, vsmlsq, 1,
                       sc + 2 * i * n, sc + 6 * n, NULL, 1, dg);
            smooth_any(variant, n, x, sc + 6 * n, w, SPANS[1], jper, vsmlsq, 0,
                       sc + (2 * i + 1) * n, sc + 7 * n, NULL, 1, dg);
        }
        for (j = 0; j < n; j++) {
            double v[3] = {sc[j + n], sc[j + 3 * n], sc[j + 5 * n]};
            span_pick(n, j, v, alpha, force_j, force_i, &sc[j + 6 * n], sd);
        }
        /* smooth the spans at midrange */
        smooth_any(variant, n, x, sc + 6 * n, w, SPANS[1], jper, vsmlsq, 0,
                   sc + n, sc + 7 * n, NULL, 1, dg);
        for (j = 0; j < n; j++)
            sc[j + 3 * n] = interp_spans(sc[j + n], sc[j], sc[j + 2 * n], sc[j + 4 * n]);
        /* final tweeter smooth */
        smooth_any(variant, n, x, sc + 3 * n, w, SPANS[0], jper, vsmlsq, 0,
                   smo, sc + 7 * n, NULL, 1, dg);
    } else {
        /* O6 (R12): one sweep, three windows at once; A_i un-averaged, scores G_i. */
        for (i = 0; i < 3; i++)
            smooth_any(variant, n, x, y, w, SPANS[i], jper, vsmlsq, 0,
                       sc + 2 * i * n, NULL, sc + (2 * i + 1) * n, 0, dg);
        for (j = 0; j < n; j++) {
            double v[3] = {sc[j + n], sc[j + 3 * n], sc[j + 5 * n]};
            double sp;
            span_pick(n, j, v, alpha, force_j, force_i, &sp, sd);
            smo[j] = interp_spans(sp, sc[j], sc[j + 2 * n], sc[j + 4 * n]);
        }
        average_ties(n, x, w, smo);
    }
}

/* Exposed for the pins: supsmu on already-sorted x. */
void sso_supsmu(int variant, int mode, int n, const double *x, const double *y, const double *w,
                int iper, double span, double alpha, double *smo)
{
    double *sc = (double *)malloc(sizeof(double) * 8 * (size_t)n);
    supsmu(variant, mode, n, x, y, w, iper, span, alpha, smo, sc, -1, -1, NULL);
    free(sc);
}

/* ------------------------------------------------------------------------- */
/* O1 prep (R3-R5).                                        */
/* ------------------------------------------------------------------------- */
void sso_prep(int n, const double *t, const double *y, const double *e,
              double *tt, double *w, double *ybar_out, double *chi0_out)
{
    double tmin = t[0];
    for (int i = 1; i < n; i++) if (t[i] < tmin) tmin = t[i];
    ld sw = 0, swy = 0;
    for (int i = 0; i < n; i++) {
        tt[i] = t[i] - tmin;
        w[i] = 1.0 / (e[i] * e[i]);
        sw += w[i]; swy += (ld)w[i] * y[i];
    }
    ld yb = swy / sw;
    ld c0 = 0;
    for (int i = 0; i < n; i++) c0 += (ld)w[i] * ((ld)y[i] - yb) * ((ld)y[i] - yb);
    *ybar_out = (double)yb;
    *chi0_out = (double)c0;
}

/* O0 grid (R1): df = (f_max - f_min)/n_freq; f_k = f_min + k*df, one multiply + one add. */
double sso_freq(double f_min, double f_max, int64_t n_freq, int64_t k)
{
    double df = (f_max - f_min) / (double)n_freq;
    double kd = (double)k * df;
    return f_min + kd;
}

/* O2 fold (R2): phi = tt*f - floor(tt*f), product rounded once (no FMA). */
void sso_fold(int n, const double *tt, double f, double *phi)
{
    for (int i = 0; i < n; i++) {
        double p = tt[i] * f;
        phi[i] = p - floor(p);
    }
}

/* O3 stable argsort by phase, ties in input order (R13). */
typedef struct { double key; int idx; } kv_t;
static int kv_cmp(const void *a, const void *b)
{
    const kv_t *p = (const kv_t *)a, *q = (const kv_t *)b;
    if (p->key < q->key) return -1;
    if (p->key > q->key) return 1;
    return (p->idx > q->idx) - (p->idx < q->idx);
}
void sso_argsort(int n, const double *phi, int *perm)
{
    kv_t *kv = (kv_t *)malloc(sizeof(kv_t) * (size_t)n);
    for (int i = 0; i < n; i++) { kv[i].key = phi[i]; kv[i].idx = i; }
    qsort(kv, (size_t)n, sizeof(kv_t), kv_cmp);
    for (int i = 0; i < n; i++) perm[i] = kv[i].idx;
    free(kv);
}

/* Workspace for one eval. */
typedef struct {
    int n;
    double *phi, *x, *ys, *ws, *smo, *sc;
    kv_t *kv;
} work_t;

static work_t *work_new(int n)
{
    work_t *wk = (work_t *)malloc(sizeof(work_t));
    wk->n = n;
    wk->phi = (double *)malloc(sizeof(double) * (size_t)n * 13);
    wk->x = wk->phi + n; wk->ys = wk->x + n; wk->ws = wk->ys + n;
    wk->smo = wk->ws + n; wk->sc = wk->smo + n;
    wk->kv = (kv_t *)malloc(sizeof(kv_t) * (size_t)n);
    return wk;
}
static void work_free(work_t *wk) { free(wk->phi); free(wk->kv); free(wk); }

/* O2-O7 for one (object, frequency): returns P = (chi0 - chi2)/chi0 (R6).
 * tt, y, w, chi0 from sso_prep.  Optionally returns chi2 and the sorted smooth. */
static double eval_one(work_t *wk, int variant, int mode, int n, const double *tt, const double *y,
                       const double *w, double chi0, double f, int iper, double span, double alpha,
                       int force_j, int force_i, sup_diag_t *sd, double *chi2_out)
{
    for (int i = 0; i < n; i++) {
        double p = tt[i] * f;
        wk->kv[i].key = p - floor(p);
        wk->kv[i].idx = i;
    }
    qsort(wk->kv, (size_t)n, sizeof(kv_t), kv_cmp);
    for (int j = 0; j < n; j++) {
        int i = wk->kv[j].idx;
        wk->x[j] = wk->kv[j].key; wk->ys[j] = y[i]; wk->ws[j] = w[i];
    }
    supsmu(variant, mode, n, wk->x, wk->ys, wk->ws, iper, span, alpha, wk->smo, wk->sc,
           force_j, force_i, sd);
    /* O7 (R6) */
    double chi2;
    if (variant == 0) {
        ld c2 = 0;
        for (int j = 0; j < n; j++) {
            ld r = (ld)wk->ys[j] - (ld)wk->smo[j];
            c2 += (ld)wk->ws[j] * r * r;
        }
        chi2 = (double)c2;
    } else {
        chi2 = 0.0;
        for (int j = 0; j < n; j++) {
            double r = wk->ys[j] - wk->smo[j];
            chi2 += wk->ws[j] * r * r;
        }
    }
    if (chi2_out) *chi2_out = chi2;
    if (chi0 == 0.0) return 0.0;
    return (chi0 - chi2) / chi0;
}

/* One eval with diagnostics, for the parity harness (O9, R29).
 * out[0]=P, out[1]=chi2, out[2]=pick margin, out[3]=P with the closest span pick forced the
 * other way (NaN unless margin < alt_threshold), out[4]=guard margin.
 * smo_sorted/perm (may be NULL) receive the smooth in phase order and the permutation. */
void sso_eval(int variant, int mode, int n, const double *t, const double *y, const double *e,
              double f, int iper, double span, double alpha, double alt_threshold,
              double *out, double *smo_sorted, int *perm)
{
    double *tt = (double *)malloc(sizeof(double) * (size_t)n * 2), *w = tt + n;
    double ybar, chi0, chi2;
    sso_prep(n, t, y, e, tt, w, &ybar, &chi0);
    work_t *wk = work_new(n);
    sup_diag_t sd; sd.pick_margin = 1e300; sd.pick_j = -1; sd.pick_alt = -1; sd.guard.guard_margin = 1e300;
    out[0] = eval_one(wk, variant, mode, n, tt, y, w, chi0, f, iper, span, alpha, -1, -1, &sd, &chi2);
    out[1] = chi2; out[2] = sd.pick_margin; out[3] = NAN; out[4] = sd.guard.guard_margin;
    if (smo_sorted) memcpy(smo_sorted, wk->smo, sizeof(double) * (size_t)n);
    if (perm) for (int j = 0; j < n; j++) perm[j] = wk->kv[j].idx;
    if (sd.pick_margin < alt_threshold && sd.pick_j >= 0)
        out[3] = eval_one(wk, variant, mode, n, tt, y, w, chi0, f, iper, span, alpha,
                          sd.pick_j, sd.pick_alt, NULL, NULL);
    work_free(wk);
    free(tt);
}

/* ------------------------------------------------------------------------- */
/* Algorithm 1 over a CSR catalog: periodogram rows and, per */
/* object, the first index of the maximum (O8, R15) and its frequency.         */
/* k_stride/k_count let the harness evaluate a subsample of the grid:          */
/* frequencies k = k0 + s*k_stride, s = 0..k_count-1 (pgram_out is             */
/* [n_objects][k_count]); best_* are over the evaluated frequencies only.      */
/* Objects with n < 5 give NaN rows, best_index = -1 (R17).                    */
/* OpenMP: over objects when n_objects >= threads, else over frequencies       */
/* (the paper's CPU decomposition).                              */
/* ------------------------------------------------------------------------- */
int sso_periodogram(int variant, int mode, const double *times, const double *mags,
                    const double *errs, const int64_t *offsets, int64_t n_objects,
                    double f_min, double f_max, int64_t n_freq,
                    int64_t k0, int64_t k_stride, int64_t k_count,
                    int iper, double span, double alpha, int n_threads,
                    double *pgram_out, double *best_freq_out, int64_t *best_index_out)
{
    if (n_threads < 1) n_threads = 1;
#ifdef _OPENMP
    omp_set_num_threads(n_threads);
#endif
    int over_objects = (n_objects >= (int64_t)n_threads * 4);
#pragma omp parallel for schedule(dynamic, 1) if (over_objects)
    for (int64_t o = 0; o < n_objects; o++) {
        int n = (int)(offsets[o + 1] - offsets[o]);
        const double *t = times + offsets[o], *y = mags + offsets[o], *e = errs + offsets[o];
        double *row = pgram_out + o * k_count;
        if (n < 5) {
            for (int64_t s = 0; s < k_count; s++) row[s] = NAN;
            if (best_freq_out) best_freq_out[o] = NAN;
            if (best_index_out) best_index_out[o] = -1;
            continue;
        }
        double *tt = (double *)malloc(sizeof(double) * (size_t)n * 2), *w = tt + n;
        double ybar, chi0;
        sso_prep(n, t, y, e, tt, w, &ybar, &chi0);
#pragma omp parallel if (!over_objects)
        {
            work_t *wk = work_new(n);
#pragma omp for schedule(dynamic, 16)
            for (int64_t s = 0; s < k_count; s++) {
                double f = sso_freq(f_min, f_max, n_freq, k0 + s * k_stride);
                row[s] = eval_one(wk, variant, mode, n, tt, y, w, chi0, f, iper, span, alpha,
                                  -1, -1, NULL, NULL);
            }
            work_free(wk);
        }
        int64_t best = 0;
        for (int64_t s = 1; s < k_count; s++) if (row[s] > row[best]) best = s;
        if (best_index_out) best_index_out[o] = k0 + best * k_stride;
        if (best_freq_out) best_freq_out[o] = sso_freq(f_min, f_max, n_freq, k0 + best * k_stride);
        free(tt);
    }
    return 0;
}

int sso_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * mred_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, single-threaded float64 CPU statement of the image-reduction hot path of
 * arXiv 2008.11486: overscan level, master bias/dark/flat, calibration, offset
 * estimation, bicubic-spline sub-pixel shift, per-pixel rejection co-add.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 * It shares no source, header, table or helper with paper_2008_11486_b200/csrc (the CUDA
 * path); neither includes the other.
 *
 * The paper names the steps and the two hand-coded algorithms
 * ("bicubic-spline interpolation", "sigma-clipped-mean", L63, L107) but prints no formula for
 * them; every definition below is the reading fixed in DESIGN.md section 3 (SURVEY.md 8(c)
 * O1-O6, Q1-Q24).  Each result has a plain definition, so the oracle is that definition
 * written out one pixel at a time: no blocking, no fusion, no reordering.
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"):
 *   orc_level           P1  constant frame -> level exactly
 *   orc_build_masters   P3  identical frames -> that frame; flat = c*pattern -> pattern/<pattern>; P11 brute force
 *   orc_calibrate       P1/P2 closed forms (uniform flat identity, bias-only -> 0, synthetic inverse)
 *   orc_estimate_shifts P7  injected integer shift recovered exactly; self -> (0,0); constant -> 0;
 *                           exact two-spike ties pin the argmax rule O4(iv) (smaller |l|, then smaller l)
 *   orc_resample        P4  paper's B-spline-basis image vs analytic shift;
 *                       P5  SciPy natural CubicSpline, identity, integer shift, composition;
 *                       P6  round-trip magnitude vs the paper's printed 1e-2..1e-1 (L162, L225); P12 footprint
 *   orc_coadd           P8  identical frames; P9 one-outlier closed form; P10 Samuelson; P11 brute force
 *   orc_fill_bad        P13 exact on linear ramps; clear mask = identity; dead row / hot column / corner rules; numpy brute force
 * Parity unpinned: equivalence with IRAF imshift / imcombine and accuracy of estimated
 * shifts against WCS astrometry (no IRAF, no MITSuME data in this environment).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int32_t W, H;          /* raw frame, x fastest (1074 x 1024 incl. overscan) */
    int32_t os_x0, os_x1;  /* overscan columns [os_x0, os_x1) (L63: 50 x 1024)                */
    int32_t x0, y0, w, h;  /* image rectangle kept by the overscan cutout (L63)               */
} orc_geom;

enum { ORC_MEDIAN = 0, ORC_MEAN = 1, ORC_SIGCLIP = 2, ORC_MINMAX = 3, ORC_MEDCLIP = 4 };

/* ------------------------------------------------------------------------------------------
 * O1  overscan ("pedestal") level: per-frame mean of the overscan pixels,
 *     exact integer sum divided in float64.  Empty overscan -> 0.   (reading Q2)
 * ---------------------------------------------------------------------------------------- */
void orc_level(const orc_geom *g, const uint16_t *raw, int n, double *level)
{
    for (int k = 0; k < n; ++k) {
        const uint16_t *f = raw + (size_t)k * g->W * g->H;
        uint64_t sum = 0, cnt = 0;
        for (int y = 0; y < g->H; ++y)
            for (int x = g->os_x0; x < g->os_x1; ++x) { sum += f[(size_t)y * g->W + x]; ++cnt; }
        level[k] = cnt ? (double)sum / (double)cnt : 0.0;
    }
}

/* ------------------------------------------------------------------------------------------
 * O6  per-pixel combine of the m values v[0..m): median, mean, or k-sigma-clipped mean
 *     ("sigma-clipped-mean algorithm"; reading Q16):
 *       repeat <= max_iter times over the surviving set:
 *         n = |set|, mu = mean, sigma = sqrt(mean((v-mu)^2))   (two-pass, population)
 *         keep v iff |v - mu| <= k*sigma ; stop early when nothing was rejected
 *       result = mean of survivors.
 *     Median of an even count = mean of the two middle values (Q9).  m == 0 -> 0, count 0.
 *     keep[i] (nullable) receives 1 for used values; *margin (nullable) receives
 *     min over passes and surviving values of | |v-mu| - k*sigma |  (tie distance, Q20).
 * ---------------------------------------------------------------------------------------- */
static double combine_column(const double *v, int m, int mode, double ksigma, int max_iter,
                             unsigned char *keep, int *count, double *margin)
{
    if (margin) *margin = INFINITY;
    if (keep) for (int i = 0; i < m; ++i) keep[i] = 1;
    if (m <= 0) { if (count) *count = 0; return 0.0; }
    if (mode == ORC_MEDIAN) {
        double s[256];
        for (int i = 0; i < m; ++i) {            /* insertion sort */
            double x = v[i]; int j = i - 1;
            while (j >= 0 && s[j] > x) { s[j + 1] = s[j]; --j; }
            s[j + 1] = x;
        }
        if (count) *count = m;
        return (m & 1) ? s[m / 2] : 0.5 * (s[m / 2 - 1] + s[m / 2]);
    }
    unsigned char alive[256];
    for (int i = 0; i < m; ++i) alive[i] = 1;
    int n = m;
    if (mode == ORC_MINMAX && m >= 3) {
        /* NEXT-2 variant (IRAF imcombine "minmax" with nlow = nhigh = 1; reading Q26): leave out one minimum and one
         * maximum (the first occurrence of each in frame order, the maximum among the entries other than the dropped
         * minimum), mean of the rest.  Fewer than 3 values: plain mean. */
        int imin = 0, imax = -1;
        for (int i = 1; i < m; ++i) if (v[i] < v[imin]) imin = i;
        for (int i = 0; i < m; ++i) if (i != imin && (imax < 0 || v[i] > v[imax])) imax = i;
        alive[imin] = 0; alive[imax] = 0;
        n = m - 2;
    }
    if (mode == ORC_SIGCLIP || mode == ORC_MEDCLIP) {
        for (int it = 0; it < max_iter && n > 0; ++it) {
            double mu = 0.0, var = 0.0;
            if (mode == ORC_MEDCLIP) {
                /* NEXT-2 variant (reading Q29): the pass is centred on the MEDIAN of the survivors and sigma is their
                 * r.m.s. about it; a single outlier among N values then sits sqrt(N) sigma out, so k = 3 clips from N = 10 */
                double s[256]; int c = 0;
                for (int i = 0; i < m; ++i) {
                    if (!alive[i]) continue;
                    double x = v[i]; int j = c - 1;
                    while (j >= 0 && s[j] > x) { s[j + 1] = s[j]; --j; }
                    s[j + 1] = x; ++c;
                }
                mu = (c & 1) ? s[c / 2] : 0.5 * (s[c / 2 - 1] + s[c / 2]);
            } else {
            for (int i = 0; i < m; ++i) if (alive[i]) mu += v[i];
            mu /= n;
            }
            for (int i = 0; i < m; ++i) if (alive[i]) var += (v[i] - mu) * (v[i] - mu);
            double thr = ksigma * sqrt(var / n);
            int rejected = 0;
            for (int i = 0; i < m; ++i) {
                if (!alive[i]) continue;
                double d = fabs(v[i] - mu);
                if (margin && fabs(d - thr) < *margin) *margin = fabs(d - thr);
                if (!(d <= thr)) { alive[i] = 0; ++rejected; }
            }
            n -= rejected;
            if (rejected == 0) break;
        }
    }
    double mu = 0.0;
    for (int i = 0; i < m; ++i) if (alive[i]) mu += v[i];
    if (keep) for (int i = 0; i < m; ++i) keep[i] = alive[i];
    if (count) *count = n;
    return n > 0 ? mu / n : 0.0;
}

/* Exposed for the brute-force pins: combine one column. */
double orc_combine_column(const double *v, int m, int mode, double ksigma, int max_iter,
                          unsigned char *keep, int *count, double *margin)
{
    return combine_column(v, m, mode, ksigma, max_iter, keep, count, margin);
}

/* ------------------------------------------------------------------------------------------
 * O2  master frames (not described by the paper; textbook CCD equation, readings Q4-Q9):
 *       MB = comb_k(B_k - L_k)
 *       MD = comb_k(D_k - L_k - MB)                               [ADU at t_dark]
 *       G_k = F_k - L_k - MB - (t_flat/t_dark) * MD ,  <G_k> = float64 mean over the image rectangle
 *       MF = comb_k(G_k / <G_k>) / <comb_k(...)>                   so that <MF> = 1
 *     Outputs over the image rectangle [h][w], float64 (nullable) and rounded once to float32
 *     (nullable).
 * ---------------------------------------------------------------------------------------- */
int orc_build_masters(const orc_geom *g, const uint16_t *bias, int nb, const uint16_t *dark, int nd,
                      double t_dark, const uint16_t *flat, int nf, double t_flat,
                      int mode, double ksigma, int max_iter,
                      double *MB64, double *MD64, double *MF64, float *MB32, float *MD32, float *MF32)
{
    if (nb < 1 || nd < 1 || nf < 1 || nb > 255 || nd > 255 || nf > 255) return -1;
    const size_t np = (size_t)g->w * g->h, fs = (size_t)g->W * g->H;
    double *Lb = malloc(sizeof(double) * nb), *Ld = malloc(sizeof(double) * nd), *Lf = malloc(sizeof(double) * nf);
    double *mb = malloc(sizeof(double) * np), *md = malloc(sizeof(double) * np), *mf = malloc(sizeof(double) * np);
    double *gm = malloc(sizeof(double) * nf);
    orc_level(g, bias, nb, Lb);
    orc_level(g, dark, nd, Ld);
    orc_level(g, flat, nf, Lf);
    const double r = t_flat / t_dark;
    double col[256];
    for (int y = 0; y < g->h; ++y)
        for (int x = 0; x < g->w; ++x) {
            size_t p = (size_t)y * g->w + x, q = (size_t)(y + g->y0) * g->W + (x + g->x0);
            for (int k = 0; k < nb; ++k) col[k] = (double)bias[k * fs + q] - Lb[k];
            mb[p] = combine_column(col, nb, mode, ksigma, max_iter, 0, 0, 0);
            for (int k = 0; k < nd; ++k) col[k] = (double)dark[k * fs + q] - Ld[k] - mb[p];
            md[p] = combine_column(col, nd, mode, ksigma, max_iter, 0, 0, 0);
        }
    for (int k = 0; k < nf; ++k) {                      /* <G_k> */
        double s = 0.0;
        for (int y = 0; y < g->h; ++y)
            for (int x = 0; x < g->w; ++x) {
                size_t p = (size_t)y * g->w + x, q = (size_t)(y + g->y0) * g->W + (x + g->x0);
                s += (double)flat[k * fs + q] - Lf[k] - mb[p] - r * md[p];
            }
        gm[k] = s / (double)np;
    }
    double smf = 0.0;
    for (int y = 0; y < g->h; ++y)
        for (int x = 0; x < g->w; ++x) {
            size_t p = (size_t)y * g->w + x, q = (size_t)(y + g->y0) * g->W + (x + g->x0);
            for (int k = 0; k < nf; ++k)
                col[k] = ((double)flat[k * fs + q] - Lf[k] - mb[p] - r * md[p]) / gm[k];
            mf[p] = combine_column(col, nf, mode, ksigma, max_iter, 0, 0, 0);
            smf += mf[p];
        }
    smf /= (double)np;
    for (size_t p = 0; p < np; ++p) {
        mf[p] /= smf;
        if (MB64) MB64[p] = mb[p];
        if (MD64) MD64[p] = md[p];
        if (MF64) MF64[p] = mf[p];
        if (MB32) MB32[p] = (float)mb[p];
        if (MD32) MD32[p] = (float)md[p];
        if (MF32) MF32[p] = (float)mf[p];
    }
    free(Lb); free(Ld); free(Lf); free(mb); free(md); free(mf); free(gm);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * O3  calibration: overscan cutout, bias & dark subtraction, flat fielding:
 *       C = (raw - L_k - MB - s*MD) / MF ,  s = t_sci / t_dark   (Q5)
 *     in float64 from the float32 masters, rounded once to float32.  MF <= 0 or non-finite -> 0 (Q7).
 * ---------------------------------------------------------------------------------------- */
int orc_calibrate(const orc_geom *g, const uint16_t *raw, int n, double dark_scale,
                  const float *MB, const float *MD, const float *MF,
                  double *out64, float *out32, double *level_out)
{
    const size_t np = (size_t)g->w * g->h, fs = (size_t)g->W * g->H;
    double *L = malloc(sizeof(double) * (n > 0 ? n : 1));
    orc_level(g, raw, n, L);
    for (int k = 0; k < n; ++k) {
        if (level_out) level_out[k] = L[k];
        for (int y = 0; y < g->h; ++y)
            for (int x = 0; x < g->w; ++x) {
                size_t p = (size_t)y * g->w + x, q = (size_t)(y + g->y0) * g->W + (x + g->x0);
                double mf = (double)MF[p], c = 0.0;
                if (isfinite(mf) && mf > 0.0)
                    c = ((double)raw[k * fs + q] - L[k] - (double)MB[p] - dark_scale * (double)MD[p]) / mf;
                if (out64) out64[k * np + p] = c;
                if (out32) out32[k * np + p] = (float)c;
            }
    }
    free(L);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * O4  offset estimation.  The paper takes relative positions from FITS WCS headers on the CPU
 *     (PAPER.md L63, L69, L99); there are no headers here, so this is the image-based reading
 *     Q10: marginal mean profiles, median-subtracted, 1-D cross-correlation against the
 *     reference frame over lags -R..R, integer argmax plus 3-point parabola.
 *       (i)   Px[x] = mean over valid y of C[y][x]  (valid: badmask == 0); Py[y] likewise.
 *       (ii)  med = median of the entries that had >= 1 valid pixel (even count: mean of the
 *             middle two); entries with none are set to med; subtract med.
 *       (iii) Cx(l) = sum_j a[j] * b[j+l], both indices in range, a = reference, b = frame k.
 *       (iv)  l* = argmax; ties -> smaller |l|, then smaller l.
 *       (v)   if |l*| < R and den = C(l*-1) - 2C(l*) + C(l*+1) < 0:
 *                 delta = 0.5 * (C(l*-1) - C(l*+1)) / den, clamped to [-0.5, 0.5]; else 0.
 *       (vi)  ishift = l*, shift = l* + delta.  The reference frame returns exactly (0, 0.0).
 *     (dx, dy) is the displacement of frame k's content relative to the reference: a source at
 *     (x, y) in the reference sits at (x+dx, y+dy) in frame k (coordinate system PAPER.md L145).
 * ---------------------------------------------------------------------------------------- */
static int cmp_double(const void *a, const void *b)
{
    double x = *(const double *)a, y = *(const double *)b;
    return (x > y) - (x < y);
}

static void finish_profile(double *p, const int *cnt, int n)
{
    double *s = malloc(sizeof(double) * (n > 0 ? n : 1));
    int m = 0;
    for (int i = 0; i < n; ++i) if (cnt[i] > 0) s[m++] = p[i];
    double med = 0.0;
    if (m > 0) {
        qsort(s, m, sizeof(double), cmp_double);
        med = (m & 1) ? s[m / 2] : 0.5 * (s[m / 2 - 1] + s[m / 2]);
    }
    for (int i = 0; i < n; ++i) p[i] = (cnt[i] > 0 ? p[i] : med) - med;
    free(s);
}

static void profiles(const float *f, int w, int h, const uint8_t *bad, double *px, double *py)
{
    int *cx = calloc(w, sizeof(int)), *cy = calloc(h, sizeof(int));
    for (int x = 0; x < w; ++x) px[x] = 0.0;
    for (int y = 0; y < h; ++y) py[y] = 0.0;
    for (int y = 0; y < h; ++y)
        for (int x = 0; x < w; ++x) {
            if (bad && bad[(size_t)y * w + x]) continue;
            double v = (double)f[(size_t)y * w + x];
            px[x] += v; ++cx[x];
            py[y] += v; ++cy[y];
        }
    for (int x = 0; x < w; ++x) if (cx[x]) px[x] /= cx[x];
    for (int y = 0; y < h; ++y) if (cy[y]) py[y] /= cy[y];
    finish_profile(px, cx, w);
    finish_profile(py, cy, h);
    free(cx); free(cy);
}

static void best_lag(const double *a, const double *b, int n, int R, int peak, int32_t *il, double *fl)
{
    double *C = malloc(sizeof(double) * (2 * R + 1));
    for (int l = -R; l <= R; ++l) {
        double s = 0.0;
        for (int j = 0; j < n; ++j) { int q = j + l; if (q >= 0 && q < n) s += a[j] * b[q]; }
        C[l + R] = s;
    }
    int best = 0;
    for (int l = -R; l <= R; ++l) {
        double c = C[l + R], cb = C[best + R];
        if (c > cb || (c == cb && (abs(l) < abs(best) || (abs(l) == abs(best) && l < best)))) best = l;
    }
    double delta = 0.0;
    if (abs(best) < R) {
        double cm = C[best - 1 + R], c0 = C[best + R], cp = C[best + 1 + R];
        double den = cm - 2.0 * c0 + cp;
        if (peak == 1 && cm > 0.0 && c0 > 0.0 && cp > 0.0) {
            /* NEXT-2 variant (reading Q27): the parabola through the LOGARITHMS of the three samples, exact for a
             * Gaussian correlation peak; the plain parabola where a sample is not positive */
            cm = log(cm); c0 = log(c0); cp = log(cp);
            den = cm - 2.0 * c0 + cp;
        }
        if (den < 0.0) {
            delta = 0.5 * (cm - cp) / den;
            if (delta > 0.5) delta = 0.5;
            if (delta < -0.5) delta = -0.5;
        }
    }
    *il = best;
    *fl = (double)best + delta;
    free(C);
}

int orc_estimate_shifts_peak(const float *frames, int n, int w, int h, int ref_index, int max_lag,
                             const uint8_t *badmask, int peak, int32_t *ishift, double *shift);

int orc_estimate_shifts(const float *frames, int n, int w, int h, int ref_index, int max_lag,
                        const uint8_t *badmask, int32_t *ishift, double *shift)
{
    return orc_estimate_shifts_peak(frames, n, w, h, ref_index, max_lag, badmask, 0, ishift, shift);
}

/* peak: 0 = 3-point parabola (O4 v), 1 = 3-point parabola of the logarithms (Gaussian peak, NEXT-2) */
int orc_estimate_shifts_peak(const float *frames, int n, int w, int h, int ref_index, int max_lag,
                             const uint8_t *badmask, int peak, int32_t *ishift, double *shift)
{
    if (n < 1 || ref_index < 0 || ref_index >= n || max_lag < 0) return -1;
    const size_t np = (size_t)w * h;
    double *ax = malloc(sizeof(double) * w), *ay = malloc(sizeof(double) * h);
    double *bx = malloc(sizeof(double) * w), *by = malloc(sizeof(double) * h);
    profiles(frames + ref_index * np, w, h, badmask, ax, ay);
    for (int k = 0; k < n; ++k) {
        if (k == ref_index) { ishift[2 * k] = ishift[2 * k + 1] = 0; shift[2 * k] = shift[2 * k + 1] = 0.0; continue; }
        profiles(frames + k * np, w, h, badmask, bx, by);
        best_lag(ax, bx, w, max_lag, peak, &ishift[2 * k], &shift[2 * k]);
        best_lag(ay, by, h, max_lag, peak, &ishift[2 * k + 1], &shift[2 * k + 1]);
    }
    free(ax); free(ay); free(bx); free(by);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * O5  sub-pixel shift by bicubic-spline interpolation.
 *     Per axis, for samples f_0..f_{n-1} ("solving simultaneous linear equations for each
 *     column or row ... expressed as a tridiagonal matrix", L266), natural end conditions (Q12):
 *         c_0 = f_0,  c_{n-1} = f_{n-1},  (c_{i-1} + 4 c_i + c_{i+1}) / 6 = f_i   (1 <= i <= n-2)
 *     solved by the Thomas algorithm (Q13); virtual c_{-1} = 2c_0 - c_1, c_n = 2c_{n-1} - c_{n-2}.
 *     Evaluation at u = x - s:  k = min(floor(u), n-2), t = u - k,
 *         s(u) = c_{k-1}(1-t)^3/6 + c_k(3t^3-6t^2+4)/6 + c_{k+1}(-3t^3+3t^2+3t+1)/6 + c_{k+2}t^3/6
 *     (the cubic B-spline basis the paper's test image is made of, L164).
 *     Shift sense: out(x, y) = in(x - sx, y - sy), origin lower-left, X horizontal (L145, Q11).
 *     Rows first, then columns (Q15).  Valid iff 0 <= x-sx <= w-1 and 0 <= y-sy <= h-1, else
 *     `fill` (Q14).  An axis whose shift has zero fractional part is a pure integer translation
 *     (copy), so shift (0,0) is the bit-exact identity.
 *     footprint[k] = {x_lo, x_hi, y_lo, y_hi} inclusive: x_lo = max(0, ceil(sx)),
 *     x_hi = min(w-1, floor(w-1+sx)), same in y ("an area which does not overlap with another
 *     image is cut out during the alignment", Table 5 fn. 2, L201).
 * ---------------------------------------------------------------------------------------- */
static void spline_coeffs(const double *f, int n, double *c /* n+2: c[-1..n] stored at c[0..n+1] */)
{
    double *u = malloc(sizeof(double) * n), *g = malloc(sizeof(double) * n);
    double *cc = c + 1;
    u[0] = 0.0; g[0] = f[0];
    for (int i = 1; i <= n - 2; ++i) {               /* row i: c_{i-1} + 4 c_i + c_{i+1} = 6 f_i */
        double piv = 4.0 - u[i - 1];
        u[i] = 1.0 / piv;
        g[i] = (6.0 * f[i] - g[i - 1]) / piv;
    }
    cc[n - 1] = f[n - 1];
    for (int i = n - 2; i >= 1; --i) cc[i] = g[i] - u[i] * cc[i + 1];
    cc[0] = f[0];
    cc[-1] = 2.0 * cc[0] - cc[1 < n ? 1 : 0];
    cc[n] = 2.0 * cc[n - 1] - cc[n >= 2 ? n - 2 : 0];
    free(u); free(g);
}

static double spline_eval(const double *c /* as above */, int n, double uu)
{
    const double *cc = c + 1;
    int k = (int)floor(uu);
    if (k > n - 2) k = n - 2;
    if (k < 0) k = 0;
    double t = uu - (double)k;
    double w0 = (1.0 - t) * (1.0 - t) * (1.0 - t) / 6.0;
    double w1 = (3.0 * t * t * t - 6.0 * t * t + 4.0) / 6.0;
    double w2 = (-3.0 * t * t * t + 3.0 * t * t + 3.0 * t + 1.0) / 6.0;
    double w3 = t * t * t / 6.0;
    return cc[k - 1] * w0 + cc[k] * w1 + cc[k + 1] * w2 + cc[k + 2] * w3;
}

/* one axis of `len` samples with stride 1 in `f`; writes out[i] and ok[i] */
static void shift_axis_interp(const double *f, int len, double s, int interp, double *out, unsigned char *ok, double *cbuf)
{
    int integer = (s == floor(s));
    if (!integer && interp == 0) spline_coeffs(f, len, cbuf);
    for (int i = 0; i < len; ++i) {
        double uu = (double)i - s;
        ok[i] = (uu >= 0.0 && uu <= (double)(len - 1));
        if (!ok[i]) { out[i] = 0.0; continue; }
        if (integer) out[i] = f[(int)uu];
        else if (interp == 0) out[i] = spline_eval(cbuf, len, uu);
        else if (interp == 1) {                  /* NEXT-2: linear interpolation, no prefilter */
            int k = (int)floor(uu);
            if (k > len - 2) k = len - 2;
            double t = uu - (double)k;
            out[i] = (1.0 - t) * f[k] + t * f[k + 1];
        } else {                                 /* nearest neighbour: floor(u + 1/2) */
            int j = (int)floor(uu + 0.5);
            if (j > len - 1) j = len - 1;
            out[i] = f[j];
        }
    }
}

static void shift_axis(const double *f, int len, double s, double *out, unsigned char *ok, double *cbuf)
{
    shift_axis_interp(f, len, s, 0, out, ok, cbuf);
}

void orc_footprint(int w, int h, double sx, double sy, int32_t *fp)
{
    double a = ceil(sx), b = floor((double)(w - 1) + sx);
    fp[0] = a > 0.0 ? (a > (double)w ? w : (int32_t)a) : 0;
    fp[1] = b < (double)(w - 1) ? (b < -1.0 ? -1 : (int32_t)b) : w - 1;
    a = ceil(sy); b = floor((double)(h - 1) + sy);
    fp[2] = a > 0.0 ? (a > (double)h ? h : (int32_t)a) : 0;
    fp[3] = b < (double)(h - 1) ? (b < -1.0 ? -1 : (int32_t)b) : h - 1;
}

int orc_resample_interp(const float *in, int n, int w, int h, const double *sx, const double *sy, double fill, int interp,
                        double *out64, float *out32, int32_t *footprint);

int orc_resample(const float *in, int n, int w, int h, const double *sx, const double *sy, double fill,
                 double *out64, float *out32, int32_t *footprint)
{
    return orc_resample_interp(in, n, w, h, sx, sy, fill, 0, out64, out32, footprint);
}

/* interp: 0 = natural bicubic spline (O5), 1 = bilinear, 2 = nearest neighbour (NEXT-2; same shift sense, validity and
 * footprint; an axis with an integer shift is a copy in every variant) */
int orc_resample_interp(const float *in, int n, int w, int h, const double *sx, const double *sy, double fill, int interp,
                        double *out64, float *out32, int32_t *footprint)
{
    if (n < 1 || w < 2 || h < 2) return -1;
    const size_t np = (size_t)w * h;
    int m = w > h ? w : h;
    double *T = malloc(sizeof(double) * np);
    unsigned char *okx = malloc(w), *oky = malloc(h);
    double *line = malloc(sizeof(double) * m), *res = malloc(sizeof(double) * m), *cbuf = malloc(sizeof(double) * (m + 2));
    for (int k = 0; k < n; ++k) {
        const float *f = in + k * np;
        if (footprint) orc_footprint(w, h, sx[k], sy[k], footprint + 4 * k);
        for (int y = 0; y < h; ++y) {                    /* rows first */
            for (int x = 0; x < w; ++x) line[x] = (double)f[(size_t)y * w + x];
            shift_axis_interp(line, w, sx[k], interp, res, okx, cbuf);
            for (int x = 0; x < w; ++x) T[(size_t)y * w + x] = res[x];
        }
        for (int x = 0; x < w; ++x) {                    /* then columns */
            for (int y = 0; y < h; ++y) line[y] = T[(size_t)y * w + x];
            shift_axis_interp(line, h, sy[k], interp, res, oky, cbuf);
            for (int y = 0; y < h; ++y) {
                double v = (okx[x] && oky[y]) ? res[y] : fill;
                if (out64) out64[k * np + (size_t)y * w + x] = v;
                if (out32) out32[k * np + (size_t)y * w + x] = (float)v;
            }
        }
    }
    free(T); free(okx); free(oky); free(line); free(res); free(cbuf);
    return 0;
}

/* 1-D helper exposed for the SciPy pin (P5): natural-spline shift of one line. */
void orc_shift_line(const double *f, int len, double s, double *out, unsigned char *ok)
{
    double *cbuf = malloc(sizeof(double) * (len + 2));
    shift_axis(f, len, s, out, ok, cbuf);
    free(cbuf);
}

/* ------------------------------------------------------------------------------------------
 * O6  co-add along the stack axis: per pixel, over the frames
 *     whose footprint contains it, median / mean / k-sigma-clipped mean (combine_column above).
 *     count = number of frames used; rejmask bit k (word k/32, plane-major [ceil(n/32)][h][w])
 *     set iff frame k was NOT used (out of footprint or clipped); margin as in combine_column.
 * ---------------------------------------------------------------------------------------- */
int orc_coadd(const float *stack, int n, int w, int h, const int32_t *footprint,
              int mode, double ksigma, int max_iter,
              double *out64, float *out32, uint16_t *count, uint32_t *rejmask, double *margin)
{
    if (n < 1 || n > 255) return -1;
    const size_t np = (size_t)w * h;
    const int words = (n + 31) / 32;
    double col[256]; int idx[256]; unsigned char keep[256];
    for (int y = 0; y < h; ++y)
        for (int x = 0; x < w; ++x) {
            size_t p = (size_t)y * w + x;
            int m = 0;
            for (int k = 0; k < n; ++k) {
                const int32_t *fp = footprint ? footprint + 4 * k : 0;
                if (fp && !(x >= fp[0] && x <= fp[1] && y >= fp[2] && y <= fp[3])) continue;
                col[m] = (double)stack[k * np + p]; idx[m] = k; ++m;
            }
            int cnt = 0; double mg = INFINITY;
            double v = combine_column(col, m, mode, ksigma, max_iter, keep, &cnt, &mg);
            if (out64) out64[p] = v;
            if (out32) out32[p] = (float)v;
            if (count) count[p] = (uint16_t)cnt;
            if (margin) margin[p] = mg;
            if (rejmask) {
                for (int wd = 0; wd < words; ++wd) {
                    uint32_t bits = 0;
                    for (int b = 0; b < 32 && wd * 32 + b < n; ++b) bits |= 1u << b;
                    rejmask[wd * np + p] = bits;            /* all unused ... */
                }
                for (int i = 0; i < m; ++i)
                    if (keep[i]) rejmask[(idx[i] / 32) * np + p] &= ~(1u << (idx[i] % 32));   /* ... minus the used */
            }
        }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * O7  bad-pixel fill ("bad pixel masking"; Table 6 L252 -- the step is named,
 *     its rule is not; reading Q25 of DESIGN.md).  Every pixel with badmask != 0 is replaced by a
 *     linear interpolation between the nearest GOOD pixels of the ORIGINAL frame (filled values are
 *     never used as sources, so the result does not depend on an order):
 *       xl < x < xr : nearest good pixels in the same row,  gap gx = xr - xl (infinite if one is missing)
 *       yl < y < yu : nearest good pixels in the same column, gap gy = yu - yl
 *       gx <= gy, finite : v = f[y][xl] + (f[y][xr] - f[y][xl]) (x - xl) / gx      (the short axis; ties -> x)
 *       else gy finite   : v = f[yl][x] + (f[yu][x] - f[yl][x]) (y - yl) / gy
 *       else             : the nearest of the one-sided neighbours (ties in the order xl, xr, yl, yu); none -> 0
 *     A hot column is bridged across its two neighbours, a dead row across the rows above and below.
 *     The mask is the same for every frame of the stack.  In place; float64 arithmetic, one rounding.
 * ---------------------------------------------------------------------------------------- */
int orc_fill_bad(float *frames, int n, int w, int h, const uint8_t *bad)
{
    if (n < 1 || w < 1 || h < 1 || !bad) return -1;
    const size_t np = (size_t)w * h;
    float *src = malloc(sizeof(float) * np);
    for (int k = 0; k < n; ++k) {
        float *f = frames + k * np;
        memcpy(src, f, sizeof(float) * np);
        for (int y = 0; y < h; ++y)
            for (int x = 0; x < w; ++x) {
                if (!bad[(size_t)y * w + x]) continue;
                int xl = x - 1, xr = x + 1, yl = y - 1, yu = y + 1;
                while (xl >= 0 && bad[(size_t)y * w + xl]) --xl;
                while (xr < w && bad[(size_t)y * w + xr]) ++xr;
                while (yl >= 0 && bad[(size_t)yl * w + x]) --yl;
                while (yu < h && bad[(size_t)yu * w + x]) ++yu;
                const int hx = xl >= 0 && xr < w, hy = yl >= 0 && yu < h;
                double v = 0.0;
                if (hx && (!hy || xr - xl <= yu - yl)) {
                    double a = src[(size_t)y * w + xl], b = src[(size_t)y * w + xr];
                    v = a + (b - a) * (double)(x - xl) / (double)(xr - xl);
                } else if (hy) {
                    double a = src[(size_t)yl * w + x], b = src[(size_t)yu * w + x];
                    v = a + (b - a) * (double)(y - yl) / (double)(yu - yl);
                } else {
                    int best = -1, dist = 0;
                    size_t at = 0;
                    if (xl >= 0) { best = 0; dist = x - xl; at = (size_t)y * w + xl; }
                    if (xr < w && (best < 0 || xr - x < dist)) { best = 1; dist = xr - x; at = (size_t)y * w + xr; }
                    if (yl >= 0 && (best < 0 || y - yl < dist)) { best = 2; dist = y - yl; at = (size_t)yl * w + x; }
                    if (yu < h && (best < 0 || yu - y < dist)) { best = 3; dist = yu - y; at = (size_t)yu * w + x; }
                    v = best >= 0 ? (double)src[at] : 0.0;
                }
                f[(size_t)y * w + x] = (float)v;
            }
    }
    free(src);
    return 0;
}

/*
 * fo_oracle.c -- CPU oracle for the F-engine + corner turn in front of the X-engine.
 * TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs may use it.
 * It shares no code, header, table or constant generator with the CUDA path (paper_1107_4264_b200/csrc); plain C, libm
 * and OpenMP (over independent signals) only.
 *
 * What it computes (Sec. 2.1):
 *   "X_i(nu) = int A_i(tau) e^{-i 2 pi nu tau}": the F-engine Fourier-transforms the digitised signal of
 *   every station; "for complex-valued samples there are N (fast) Fourier transforms of length F performed, but only
 *   once every F samples" (footnote 2).  The corner turn "is a reordering of data necessitated by the
 *   station independence of the F-engine, and the frequency independence of the X-engine": station-major
 *   time series in, the X-engine's [t][f][station][pol][re,im] cube out ("station fastest, then frequency, then
 *   time").
 *
 * Definition written out (no FFT, no blocking): for station s, polarisation p, spectrum t, channel f
 *
 *      X[t][f][s][p] = sum_{k=0}^{F-1} volt[s][p][t*F + k] * exp(-2 pi i f k / F)          (fp64, O(F^2) per spectrum)
 *
 * Readings where the paper is silent (readings 18-21):
 *   18. input: complex int8 voltages, station-major: volt[s][p][n][re,im], n < T*F ("voltage time-series from each
 *       antenna ... digitized"; complex samples, footnote 2); spectrum t takes samples [tF, (t+1)F): no
 *       overlap, no window (a critically sampled filter bank with a rectangular prototype);
 *   19. sign and order: e^{-i 2 pi f k / F}, channels in DFT order f = 0 .. F-1 (no fftshift);
 *   20. quantisation to the X-engine's int8 ("typically four to eight bits of precision is sufficient for both the
 *       Fourier transform and cross-multiplication"): q = clip(rint(fl32(X) * scale), -127, 127) per real
 *       component, rint = round-half-to-even, decided in the kernel's precision (fp32 product of the fp32-rounded
 *       spectrum value and the fp32 scale), symmetric clip (no -128);
 *   21. because a floating-point value decides an integer, the oracle also returns each entry's MARGIN: the distance of
 *       the fp64 value X*scale from the nearest rounding boundary (k + 1/2).  An implementation whose fp32 spectrum is
 *       within eps of the exact one must agree wherever margin > eps*scale and may differ by one step elsewhere.
 *
 * Pins (tests/test_fengine_oracle_pins.py): hand-worked F = 4 example (tests/golden/fengine_hand_examples.txt), impulse ->
 * flat magnitude / linear phase, quarter-turn tone -> single exact bin (fixes the exponent's sign), numpy.fft.fft,
 * Parseval, linearity, circular shift theorem, cube layout by probing, ties-to-even and clipping of the quantiser.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define FO_OK 0
#define FO_ERR_ARG (-1)
#define FO_ERR_NOMEM (-7)

/* exp(-2 pi i m / F) for 0 <= m < F in fp64.  The angle is written as k quarter turns plus or minus theta with
 * 0 <= theta <= pi/4, so that every multiple of an eighth of a turn is exact up to sqrt(1/2) (0, +-1 exactly at quarter
 * turns): integer-valued inputs then give exactly integer spectra in the bins f = 0, F/4, F/2, 3F/4. */
static void fo_twiddle(long long F, long long m, double* wre, double* wim) {
    const double PI = 3.14159265358979323846264338327950288;
    const long long q = (8 * m) / F;          /* octant 0..7 */
    const long long r = 8 * m - q * F;        /* position inside the octant, in units of 1/(8F) turn */
    long long quarter;
    double c, s;                              /* cos, sin of the angle a = 2 pi m / F */
    if ((q & 1) == 0) {                       /* a = (q/2) * pi/2 + theta */
        const double theta = 2.0 * PI * (double)r / (8.0 * (double)F);
        quarter = q / 2;
        c = (r == 0) ? 1.0 : cos(theta);
        s = (r == 0) ? 0.0 : sin(theta);
    } else {                                  /* a = ((q+1)/2) * pi/2 - theta', theta' = 2 pi (F - r) / (8F) in (0, pi/4] */
        const double theta = 2.0 * PI * (double)(F - r) / (8.0 * (double)F);
        quarter = (q + 1) / 2;
        if (r == 0) { c = sqrt(0.5); s = -sqrt(0.5); }
        else { c = cos(theta); s = -sin(theta); }
    }
    /* rotate (c, s) by `quarter` quarter turns: exact */
    double cr, sr;
    switch (quarter & 3) {
        case 0: cr = c; sr = s; break;
        case 1: cr = -s; sr = c; break;
        case 2: cr = -c; sr = -s; break;
        default: cr = s; sr = -c; break;
    }
    *wre = cr;        /* exp(-i a) = cos a - i sin a */
    *wim = -sr;
}

/* Table of the F twiddles; caller frees. */
static double* fo_table(int F) {
    double* w = (double*)malloc(sizeof(double) * 2 * (size_t)F);
    if (!w) return NULL;
    for (int m = 0; m < F; ++m) fo_twiddle(F, m, &w[2 * m], &w[2 * m + 1]);
    return w;
}

/* X[f] = sum_k x[k] exp(-2 pi i f k / F): the definition, O(F^2).  x: F complex int8 (re, im interleaved). */
static void fo_dft_i8(const int8_t* x, int F, const double* w, double* X) {
    for (int f = 0; f < F; ++f) {
        double re = 0.0, im = 0.0;
        for (int k = 0; k < F; ++k) {
            const long long m = ((long long)f * k) % F;
            const double a = (double)x[2 * k], b = (double)x[2 * k + 1];      /* x = a + i b */
            const double c = w[2 * m], d = w[2 * m + 1];                      /* w = c + i d */
            re += a * c - b * d;
            im += a * d + b * c;
        }
        X[2 * f] = re;
        X[2 * f + 1] = im;
    }
}

/* reading 20: q = clip(rint(fl32(X) * scale), -127, 127), product and rounding in fp32 */
static int8_t fo_quantise(double X, float scale) {
    const volatile float x32 = (float)X;
    const volatile float y = x32 * scale;       /* volatile: no contraction, no excess precision */
    float r = rintf(y);                           /* round-half-to-even in the default rounding mode */
    if (r > 127.0f) r = 127.0f;
    if (r < -127.0f) r = -127.0f;
    return (int8_t)r;
}

/* reading 21: distance of the fp64 value X*scale from the nearest k + 1/2 */
static float fo_margin(double X, float scale) {
    const double y = X * (double)scale;
    const double d = fabs(y - floor(y) - 0.5);
    return (float)d;
}

int fo_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* The twiddle exp(-2 pi i m / F), exposed so that the pins can look at it. */
int fo_twiddle_f64(int F, int m, double* out2) {
    if (F < 1 || m < 0 || m >= F || !out2) return FO_ERR_ARG;
    fo_twiddle(F, m, &out2[0], &out2[1]);
    return FO_OK;
}

/* One spectrum: station s, pol p, spectrum t of volt[N][2][T*F][2] -> X[F][2] (fp64, unquantised, unscaled). */
int fo_spectrum_i8(const int8_t* volt, int N, int F, int T, int s, int p, int t, double* X) {
    if (!volt || !X || N < 1 || F < 1 || T < 1 || s < 0 || s >= N || p < 0 || p > 1 || t < 0 || t >= T) return FO_ERR_ARG;
    double* w = fo_table(F);
    if (!w) return FO_ERR_NOMEM;
    const int8_t* x = volt + (((size_t)s * 2 + p) * (size_t)T * F + (size_t)t * F) * 2;
    fo_dft_i8(x, F, w, X);
    free(w);
    return FO_OK;
}

/* Spectra of the selected (s, p, t) triples, sel[3*n + 0..2], n < nsel -> X[nsel][F][2]. */
int fo_spectra_i8(const int8_t* volt, int N, int F, int T, const int32_t* sel, int nsel, double* X) {
    if (!volt || !X || !sel || N < 1 || F < 1 || T < 1 || nsel < 0) return FO_ERR_ARG;
    for (int n = 0; n < nsel; ++n)
        if (sel[3 * n] < 0 || sel[3 * n] >= N || sel[3 * n + 1] < 0 || sel[3 * n + 1] > 1 || sel[3 * n + 2] < 0 || sel[3 * n + 2] >= T)
            return FO_ERR_ARG;
    double* w = fo_table(F);
    if (!w) return FO_ERR_NOMEM;
#pragma omp parallel for schedule(dynamic)
    for (int n = 0; n < nsel; ++n) {
        const int s = sel[3 * n], p = sel[3 * n + 1], t = sel[3 * n + 2];
        const int8_t* x = volt + (((size_t)s * 2 + p) * (size_t)T * F + (size_t)t * F) * 2;
        fo_dft_i8(x, F, w, X + (size_t)n * F * 2);
    }
    free(w);
    return FO_OK;
}

/* The whole F-engine + corner turn: volt[N][2][T*F][2] int8 ->
 *   spec   (if not NULL) fp64 [T][F][N][2][2]: the unquantised, unscaled spectra in cube order,
 *   cube   (if not NULL) int8 [T][F][N][2][2]: quantised with `scale` (reading 20) -- the X-engine's input,
 *   margin (if not NULL) fp32 [T][F][N][2][2]: distance of X*scale from the nearest rounding boundary (reading 21). */
int fo_fengine_i8(const int8_t* volt, int N, int F, int T, float scale, double* spec, int8_t* cube, float* margin) {
    if (!volt || N < 1 || F < 1 || T < 1) return FO_ERR_ARG;
    double* w = fo_table(F);
    if (!w) return FO_ERR_NOMEM;
    int rc = FO_OK;
#pragma omp parallel
    {
        double* X = (double*)malloc(sizeof(double) * 2 * (size_t)F);
        if (!X) {
#pragma omp critical
            rc = FO_ERR_NOMEM;
        }
#pragma omp for schedule(dynamic) collapse(2)
        for (int s = 0; s < N; ++s) {
            for (int t = 0; t < T; ++t) {
                if (!X) continue;
                for (int p = 0; p < 2; ++p) {
                    const int8_t* x = volt + (((size_t)s * 2 + p) * (size_t)T * F + (size_t)t * F) * 2;
                    fo_dft_i8(x, F, w, X);
                    for (int f = 0; f < F; ++f) {
                        /* corner turn: [t][f][s][p][c] */
                        const size_t o = ((((size_t)t * F + f) * N + s) * 2 + p) * 2;
                        for (int c = 0; c < 2; ++c) {
                            if (spec) spec[o + c] = X[2 * f + c];
                            if (cube) cube[o + c] = fo_quantise(X[2 * f + c], scale);
                            if (margin) margin[o + c] = fo_margin(X[2 * f + c], scale);
                        }
                    }
                }
            }
        }
        free(X);
    }
    free(w);
    return rc;
}

/* The margin alone (reading 21), for its pins: m[i] = margin(X[i], scale). */
int fo_margin_f64(const double* X, size_t n, float scale, float* m) {
    if (!X || !m) return FO_ERR_ARG;
    for (size_t i = 0; i < n; ++i) m[i] = fo_margin(X[i], scale);
    return FO_OK;
}

/* The quantiser alone (reading 20), for its pins: q[i] = quantise(X[i], scale). */
int fo_quantise_f64(const double* X, size_t n, float scale, int8_t* q) {
    if (!X || !q) return FO_ERR_ARG;
    for (size_t i = 0; i < n; ++i) q[i] = fo_quantise(X[i], scale);
    return FO_OK;
}

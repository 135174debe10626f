/*
 * xo_oracle.c -- CPU ORACLE for the X-engine.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build, link, load or call this file.  It shares no code, header, table or
 * helper with the CUDA path under paper_1107_4264_b200/csrc/ (index formulas are
 * re-typed here on purpose) and includes nothing from include/.
 *
 * What it computes (Sec. 2.1, Eq. 4): for every frequency channel f
 *
 *      S^(f) = sum_{t=1..I}  X_t(f) (x) X_t(f)
 *
 * the time-integrated self outer product of the vector of N stations x 2 polarisations
 * of complex samples, of which only the lower triangle of station pairs i <= j is kept
 * ("1/2 N(N+1) correlation pairs including the auto-correlation of self pairs",
 * PAPER.md:67), with all four polarisation products per pair.
 *
 * The method reaches this definition exactly (the paper's tiling is only an evaluation
 * order), so the oracle IS the definition written out in Eq. 4's order: the outermost
 * loop of a channel is the sum over t, the body is the outer product of the sample
 * vector with itself.  No blocking, no SIMD intrinsics, no reordering.
 *
 * Readings of the paper taken here:
 *   R1  entry (a,b) = x_a * conj(x_b), a = (i,pi) row side, b = (j,pj) column side.
 *       Eq. 3 lost its conjugate in extraction; north_star says x x^H.
 *   R2  stored pairs: 0 <= i <= j < N.
 *   R3  baseline index b = j(j+1)/2 + i (the paper's block formula, PAPER.md:157,
 *       applied at station level).
 *   R4  all four pol products are stored also for i == j.
 *   R5  overwrite and accumulate are both offered (PAPER.md:244 accumulates).
 *   R7  results must fit int32; sums are formed in int64 and checked.
 *   R9  [re,im] order: re first; pol product index 2*pi + pj.
 *
 * Layouts (BASELINE.json north_star):
 *   in  : int8  [t][f][station][pol][re,im]       flat ((((t*F+f)*N+s)*2+p)*2+c)
 *   vis : int32 [f][b][pi][pj][re,im]             flat (((((f*NB+b)*2+pi)*2+pj)*2)+c)
 *
 * Parity pins: tests/test_oracle_pins.py (brute-force Python complex, numpy
 * X @ X^H, Hermitian symmetry, autocorrelation = sum |x|^2, common tone, hand example,
 * linearity in T, channel independence).  No function here is "parity unpinned".
 *
 * Threads: OpenMP over f only (channels are independent).
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define XO_OK            0
#define XO_ERR_ARG      -1
#define XO_ERR_OVERFLOW -3
#define XO_ERR_NOMEM    -7

int xo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void xo_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* One channel, Eq. 4 order: acc[b][pi][pj][c] += over t of x_{i,pi} conj(x_{j,pj}). */
static void xo_channel_sum_i8(const int8_t *in, int N, int F, int T, int f, int64_t *acc)
{
    const size_t NB = (size_t)N * (N + 1) / 2;
    memset(acc, 0, NB * 8 * sizeof(int64_t));
    for (int t = 0; t < T; ++t) {
        const int8_t *x = in + ((size_t)t * F + f) * (size_t)N * 4;   /* X_t(f): N x [pol][re,im] */
        for (int j = 0; j < N; ++j) {
            for (int i = 0; i <= j; ++i) {
                int64_t *v = acc + ((size_t)j * (j + 1) / 2 + i) * 8;
                for (int pi = 0; pi < 2; ++pi) {
                    for (int pj = 0; pj < 2; ++pj) {
                        const int64_t are = x[(i * 2 + pi) * 2 + 0], aim = x[(i * 2 + pi) * 2 + 1];
                        const int64_t bre = x[(j * 2 + pj) * 2 + 0], bim = x[(j * 2 + pj) * 2 + 1];
                        /* a * conj(b) = (are*bre + aim*bim) + i (aim*bre - are*bim) */
                        v[(pi * 2 + pj) * 2 + 0] += are * bre + aim * bim;
                        v[(pi * 2 + pj) * 2 + 1] += aim * bre - are * bim;
                    }
                }
            }
        }
    }
}

/* vis_f points at the NB*8 int32 of channel f. Returns XO_ERR_OVERFLOW if a value leaves int32. */
static int xo_store_i32(const int64_t *acc, size_t n, int32_t *vis_f, int accumulate)
{
    for (size_t k = 0; k < n; ++k) {
        int64_t v = acc[k] + (accumulate ? (int64_t)vis_f[k] : 0);
        if (v > INT32_MAX || v < INT32_MIN) return XO_ERR_OVERFLOW;
        vis_f[k] = (int32_t)v;
    }
    return XO_OK;
}

/* One channel f of the int8 X-engine; vis_f = NB*8 int32 (that channel only). */
int xo_channel_i8(const int8_t *in, int N, int F, int T, int f, int32_t *vis_f, int accumulate)
{
    if (!in || !vis_f || N < 1 || F < 1 || T < 0 || f < 0 || f >= F) return XO_ERR_ARG;
    const size_t NB = (size_t)N * (N + 1) / 2;
    int64_t *acc = (int64_t *)malloc(NB * 8 * sizeof(int64_t));
    if (!acc) return XO_ERR_NOMEM;
    xo_channel_sum_i8(in, N, F, T, f, acc);
    int rc = xo_store_i32(acc, NB * 8, vis_f, accumulate);
    free(acc);
    return rc;
}

/* Long integrations (I = N_p * I'): chosen channels, the same Eq. 4 sums kept in int64 with no
 * int32 check; vis64_sel = nsel*NB*8 int64.  T is the whole integration length (blocks concatenated in time). */
int xo_channels_i8_wide(const int8_t *in, int N, int F, int T, const int *fsel, int nsel, int64_t *vis64_sel)
{
    if (!in || !vis64_sel || !fsel || N < 1 || F < 1 || T < 0 || nsel < 0) return XO_ERR_ARG;
    const size_t NB = (size_t)N * (N + 1) / 2;
    for (int k = 0; k < nsel; ++k)
        if (fsel[k] < 0 || fsel[k] >= F) return XO_ERR_ARG;
#pragma omp parallel for schedule(dynamic, 1)
    for (int k = 0; k < nsel; ++k) xo_channel_sum_i8(in, N, F, T, fsel[k], vis64_sel + (size_t)k * NB * 8);
    return XO_OK;
}

/* All channels; vis = F*NB*8 int32. */
int xo_correlate_i8(const int8_t *in, int N, int F, int T, int32_t *vis, int accumulate)
{
    if (!in || !vis || N < 1 || F < 1 || T < 0) return XO_ERR_ARG;
    const size_t NB = (size_t)N * (N + 1) / 2;
    int rc_all = XO_OK;
#pragma omp parallel for schedule(dynamic, 1)
    for (int f = 0; f < F; ++f) {
        int rc = xo_channel_i8(in, N, F, T, f, vis + (size_t)f * NB * 8, accumulate);
        if (rc != XO_OK) {
#pragma omp critical
            rc_all = rc;
        }
    }
    return rc_all;
}

/* A chosen list of channels (for sampled parity at full sizes); vis_sel = nsel*NB*8 int32,
 * channel fsel[k] goes to slot k. */
int xo_channels_i8(const int8_t *in, int N, int F, int T, const int *fsel, int nsel, int32_t *vis_sel)
{
    if (!in || !vis_sel || !fsel || nsel < 0) return XO_ERR_ARG;
    const size_t NB = (size_t)N * (N + 1) / 2;
    int rc_all = XO_OK;
#pragma omp parallel for schedule(dynamic, 1)
    for (int k = 0; k < nsel; ++k) {
        int rc = xo_channel_i8(in, N, F, T, fsel[k], vis_sel + (size_t)k * NB * 8, 0);
        if (rc != XO_OK) {
#pragma omp critical
            rc_all = rc;
        }
    }
    return rc_all;
}

/* One baseline (i,j) of one channel, all four pol products, int64, straight from the
 * definition (no triangle restriction: i > j is allowed, used by the Hermitian pin). */
int xo_baseline_i8(const int8_t *in, int N, int F, int T, int f, int i, int j, int64_t out[8])
{
    if (!in || !out || N < 1 || F < 1 || T < 0 || f < 0 || f >= F || i < 0 || i >= N || j < 0 || j >= N)
        return XO_ERR_ARG;
    for (int k = 0; k < 8; ++k) out[k] = 0;
    for (int t = 0; t < T; ++t) {
        const int8_t *x = in + ((size_t)t * F + f) * (size_t)N * 4;
        for (int pi = 0; pi < 2; ++pi)
            for (int pj = 0; pj < 2; ++pj) {
                const int64_t are = x[(i * 2 + pi) * 2 + 0], aim = x[(i * 2 + pi) * 2 + 1];
                const int64_t bre = x[(j * 2 + pj) * 2 + 0], bim = x[(j * 2 + pj) * 2 + 1];
                out[(pi * 2 + pj) * 2 + 0] += are * bre + aim * bim;
                out[(pi * 2 + pj) * 2 + 1] += aim * bre - are * bim;
            }
    }
    return XO_OK;
}

/* Full-matrix mode, one channel: full = int64 [2N][2N][re,im], row a = 2*i+pi, column
 * b = 2*j+pj, every (a,b) including the upper triangle.  Only for the Hermitian pin. */
int xo_full_i8(const int8_t *in, int N, int F, int T, int f, int64_t *full)
{
    if (!in || !full || N < 1 || F < 1 || T < 0 || f < 0 || f >= F) return XO_ERR_ARG;
    const int D = 2 * N;
    memset(full, 0, (size_t)D * D * 2 * sizeof(int64_t));
    for (int t = 0; t < T; ++t) {
        const int8_t *x = in + ((size_t)t * F + f) * (size_t)N * 4;
        for (int a = 0; a < D; ++a)
            for (int b = 0; b < D; ++b) {
                const int64_t are = x[a * 2], aim = x[a * 2 + 1], bre = x[b * 2], bim = x[b * 2 + 1];
                full[((size_t)a * D + b) * 2 + 0] += are * bre + aim * bim;
                full[((size_t)a * D + b) * 2 + 1] += aim * bre - are * bim;
            }
    }
    return XO_OK;
}

/* ---- float-input oracle: same definition, float samples, fp64 products and sums ----
 * in  : float  [t][f][station][pol][re,im];  vis64 : double [f][b][pi][pj][re,im]
 * (north_star: "fp32 path must agree with an fp64-accumulating oracle"). */
int xo_channel_f64(const float *in, int N, int F, int T, int f, double *vis_f)
{
    if (!in || !vis_f || N < 1 || F < 1 || T < 0 || f < 0 || f >= F) return XO_ERR_ARG;
    const size_t NB = (size_t)N * (N + 1) / 2;
    for (size_t k = 0; k < NB * 8; ++k) vis_f[k] = 0.0;
    for (int t = 0; t < T; ++t) {
        const float *x = in + ((size_t)t * F + f) * (size_t)N * 4;
        for (int j = 0; j < N; ++j)
            for (int i = 0; i <= j; ++i) {
                double *v = vis_f + ((size_t)j * (j + 1) / 2 + i) * 8;
                for (int pi = 0; pi < 2; ++pi)
                    for (int pj = 0; pj < 2; ++pj) {
                        const double are = x[(i * 2 + pi) * 2 + 0], aim = x[(i * 2 + pi) * 2 + 1];
                        const double bre = x[(j * 2 + pj) * 2 + 0], bim = x[(j * 2 + pj) * 2 + 1];
                        v[(pi * 2 + pj) * 2 + 0] += are * bre + aim * bim;
                        v[(pi * 2 + pj) * 2 + 1] += aim * bre - are * bim;
                    }
            }
    }
    return XO_OK;
}

int xo_channels_f64(const float *in, int N, int F, int T, const int *fsel, int nsel, double *vis_sel)
{
    if (!in || !vis_sel || !fsel || nsel < 0) return XO_ERR_ARG;
    const size_t NB = (size_t)N * (N + 1) / 2;
    int rc_all = XO_OK;
#pragma omp parallel for schedule(dynamic, 1)
    for (int k = 0; k < nsel; ++k) {
        int rc = xo_channel_f64(in, N, F, T, fsel[k], vis_sel + (size_t)k * NB * 8);
        if (rc != XO_OK) {
#pragma omp critical
            rc_all = rc;
        }
    }
    return rc_all;
}

/*
 * spiir_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, double-precision CPU statement of what the SPIIR hot path computes,
 * written from /root/reference/PAPER.md (arXiv:1702.02256).  It shares no code, header,
 * table or constant generator with the CUDA library under paper_1702_02256_b200/csrc/.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call it.
 *
 * What is here (each function cites the passage it follows):
 *   spiir_oracle_filter      PAPER.md:63-67, Eq. 7 + Eq. 8 (without the 2*dt factor,
 *                            DESIGN.md reading F1): y_{k,l} = a1_l y_{k-1,l} + b0_l x_{k-d_l},
 *                            z_k = sum_l y_{k,l}; streamed, state carried.
 *   spiir_oracle_kaiser_taps PAPER.md:81-88 (Eq. 9, "Kaiser-window-tapered low-pass"),
 *                            DESIGN.md readings R1-R3.
 *   spiir_oracle_down2       PAPER.md:75 ("downsampled by a factor of 2"), Eq. 9 causal.
 *   spiir_oracle_up2         PAPER.md:75-77 ("upsampled and added to the filtering output
 *                            of next highest rate"), Eq. 9 causal.
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): closed form Eq. 6, geometric
 * series, sinusoid steady state, scipy.signal.lfilter, linearity / superposition / zero
 * padding, brute-force convolution, block streaming == one run, numpy.kaiser*sinc taps,
 * numpy.convolve resampling, DC / tone identities.  Nothing here is "parity unpinned"
 * except that the paper prints no worked numerical example of a filter output.
 *
 * Arithmetic: IEEE double, complex numbers written out as (re, im) pairs, no blocking,
 * no reordering: for every sample k the filters are visited in ascending l.
 * OpenMP is used only across independent (stream, template) pairs or rows.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct spiir_oracle_plan {
    int n_templates, n_filters, n_streams, max_delay;
    double *a1;      /* [T][L][2]  complex64 inputs promoted exactly to double          */
    double *b0;      /* [T][L][2]                                                        */
    int32_t *d;      /* [T][L]     delay in samples at this plan's rate                  */
    double *y;       /* [S][T][L][2] filter state y_{k-1,l}                              */
    double *hist;    /* [S][max_delay] the last max_delay input samples, oldest first    */
} spiir_oracle_plan;

int spiir_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void spiir_oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

void spiir_oracle_plan_destroy(spiir_oracle_plan *p)
{
    if (!p) return;
    free(p->a1); free(p->b0); free(p->d); free(p->y); free(p->hist); free(p);
}

/* a1, b0: interleaved (re, im) float32 [T][L]; delays int32 [T][L] >= 0.  Returns 0 / -1. */
int spiir_oracle_plan_create(spiir_oracle_plan **out, const float *a1, const float *b0,
                             const int32_t *delays, int n_templates, int n_filters, int n_streams)
{
    if (!out || !a1 || !b0 || !delays || n_templates < 1 || n_filters < 1 || n_streams < 1) return -1;
    size_t TL = (size_t)n_templates * n_filters;
    int dmax = 0;
    for (size_t i = 0; i < TL; ++i) { if (delays[i] < 0) return -1; if (delays[i] > dmax) dmax = delays[i]; }
    spiir_oracle_plan *p = (spiir_oracle_plan *)calloc(1, sizeof *p);
    if (!p) return -1;
    p->n_templates = n_templates; p->n_filters = n_filters; p->n_streams = n_streams; p->max_delay = dmax;
    p->a1 = (double *)malloc(TL * 2 * sizeof(double));
    p->b0 = (double *)malloc(TL * 2 * sizeof(double));
    p->d = (int32_t *)malloc(TL * sizeof(int32_t));
    p->y = (double *)calloc((size_t)n_streams * TL * 2, sizeof(double));           /* y = 0 (reading F4) */
    p->hist = (double *)calloc((size_t)n_streams * (dmax > 0 ? dmax : 1), sizeof(double)); /* x = 0 for k < 0 */
    if (!p->a1 || !p->b0 || !p->d || !p->y || !p->hist) { spiir_oracle_plan_destroy(p); return -1; }
    for (size_t i = 0; i < TL * 2; ++i) { p->a1[i] = (double)a1[i]; p->b0[i] = (double)b0[i]; }
    memcpy(p->d, delays, TL * sizeof(int32_t));
    *out = p;
    return 0;
}

void spiir_oracle_plan_reset(spiir_oracle_plan *p)
{
    size_t TL = (size_t)p->n_templates * p->n_filters;
    memset(p->y, 0, (size_t)p->n_streams * TL * 2 * sizeof(double));
    memset(p->hist, 0, (size_t)p->n_streams * (p->max_delay > 0 ? p->max_delay : 1) * sizeof(double));
}

/*
 * One streamed block.  x: [S][n] (double; the caller promotes float32 exactly).
 * z: [S][T][n][2] double, fully overwritten.  Eq. 7 then Eq. 8 for every sample, in order.
 */
int spiir_oracle_filter(spiir_oracle_plan *p, const double *x, int n, double *z)
{
    if (!p || !x || !z || n < 0) return -1;
    const int T = p->n_templates, L = p->n_filters, S = p->n_streams, D = p->max_delay;
#pragma omp parallel for collapse(2) schedule(static)
    for (int s = 0; s < S; ++s) {
        for (int t = 0; t < T; ++t) {
            const double *xs = x + (size_t)s * n;
            const double *hs = p->hist + (size_t)s * (D > 0 ? D : 1);
            const double *a = p->a1 + (size_t)t * L * 2;
            const double *b = p->b0 + (size_t)t * L * 2;
            const int32_t *d = p->d + (size_t)t * L;
            double *y = p->y + ((size_t)s * T + t) * L * 2;
            double *zt = z + ((size_t)s * T + t) * (size_t)n * 2;
            for (int k = 0; k < n; ++k) {
                double zr = 0.0, zi = 0.0;
                for (int l = 0; l < L; ++l) {
                    int j = k - d[l];                       /* index of x_{k-d_l} inside this block */
                    double xv = (j >= 0) ? xs[j] : hs[D + j]; /* j in [-D, -1] -> carried history   */
                    double yr = y[2 * l], yi = y[2 * l + 1];
                    double ar = a[2 * l], ai = a[2 * l + 1];
                    /* Eq. 7: y_k = a1 * y_{k-1} + b0 * x_{k-d}  (complex * complex, complex * real) */
                    double nr = (ar * yr - ai * yi) + b[2 * l] * xv;
                    double ni = (ar * yi + ai * yr) + b[2 * l + 1] * xv;
                    y[2 * l] = nr; y[2 * l + 1] = ni;
                    zr += nr; zi += ni;                     /* Eq. 8: z_k = sum_l y_{k,l}        */
                }
                zt[2 * k] = zr; zt[2 * k + 1] = zi;
            }
        }
    }
    /* carry the last D samples of (history ++ block) as the next block's history */
    if (D > 0) {
        double *tmp = (double *)malloc((size_t)D * sizeof(double));
        if (!tmp) return -1;
        for (int s = 0; s < S; ++s) {
            double *hs = p->hist + (size_t)s * D;
            const double *xs = x + (size_t)s * n;
            for (int i = 0; i < D; ++i) {
                int j = n - D + i;                          /* position in the new block, may be < 0 */
                tmp[i] = (j >= 0) ? xs[j] : hs[D + j];
            }
            memcpy(hs, tmp, (size_t)D * sizeof(double));
        }
        free(tmp);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Resampling (Eq. 9).  Readings R1-R3 of DESIGN.md: one N-tap (N = 192 in
 * BASELINE.json configs[3]) Kaiser-windowed sinc, beta = 5, cut-off f_c = 0.25 cycles per
 * high-rate sample (the new Nyquist), unit DC gain; applied causally, zero pre-history.
 * ------------------------------------------------------------------------------------------ */

/* Modified Bessel function of the first kind, order 0: I0(x) = sum_k ((x/2)^k / k!)^2 */
static double bessel_i0(double x)
{
    double half = 0.5 * x, term = 1.0, sum = 1.0;
    for (int k = 1; k < 500; ++k) {
        term *= half / (double)k;          /* (x/2)^k / k! */
        double t2 = term * term;
        sum += t2;
        if (t2 < 1e-32 * sum) break;
    }
    return sum;
}

/*
 * h[n] = g * w_K[n; beta] * 2 f_c sinc(2 f_c (n - (N-1)/2)),  n = 0..N-1
 * w_K[n; beta] = I0(beta sqrt(1 - (2n/(N-1) - 1)^2)) / I0(beta),  g such that sum h = 1.
 * Writes the taps in double (h64, may be NULL) and rounded once to float32 (h32, may be NULL).
 */
int spiir_oracle_kaiser_taps(int n_taps, double beta, double cutoff, double *h64, float *h32)
{
    if (n_taps < 2 || cutoff <= 0.0) return -1;
    double *h = (double *)malloc((size_t)n_taps * sizeof(double));
    if (!h) return -1;
    const double pi = 3.14159265358979323846;
    const double centre = 0.5 * (double)(n_taps - 1);
    double sum = 0.0;
    for (int n = 0; n < n_taps; ++n) {
        double r = 2.0 * (double)n / (double)(n_taps - 1) - 1.0;
        double arg = 1.0 - r * r; if (arg < 0.0) arg = 0.0;
        double w = bessel_i0(beta * sqrt(arg)) / bessel_i0(beta);
        double t = 2.0 * cutoff * ((double)n - centre);          /* sinc(t) = sin(pi t)/(pi t) */
        double s = (t == 0.0) ? 1.0 : sin(pi * t) / (pi * t);
        h[n] = w * 2.0 * cutoff * s;
        sum += h[n];
    }
    for (int n = 0; n < n_taps; ++n) {
        h[n] /= sum;
        if (h64) h64[n] = h[n];
        if (h32) h32[n] = (float)h[n];
    }
    free(h);
    return 0;
}

typedef struct spiir_oracle_resamp {
    int n_taps, n_rows, width;   /* width = 1 (real rows) or 2 (interleaved complex rows)       */
    int n_hist;                  /* samples of input history kept per row: N-1 (down), N/2-1 (up) */
    double *h;                   /* taps: float32-rounded values promoted to double              */
    double *hist;                /* [rows][n_hist][width], oldest first, zeros initially         */
} spiir_oracle_resamp;

void spiir_oracle_resamp_destroy(spiir_oracle_resamp *r)
{
    if (!r) return;
    free(r->h); free(r->hist); free(r);
}

/* direction: 0 = down-by-2 on real rows, 1 = up-by-2 on complex rows.  taps32: n_taps float32. */
int spiir_oracle_resamp_create(spiir_oracle_resamp **out, int direction, int n_taps,
                               const float *taps32, int n_rows)
{
    if (!out || !taps32 || n_taps < 2 || (n_taps & 1) || n_rows < 1 || direction < 0 || direction > 1) return -1;
    spiir_oracle_resamp *r = (spiir_oracle_resamp *)calloc(1, sizeof *r);
    if (!r) return -1;
    r->n_taps = n_taps; r->n_rows = n_rows;
    r->width = direction == 0 ? 1 : 2;
    r->n_hist = direction == 0 ? n_taps - 1 : n_taps / 2 - 1;
    r->h = (double *)malloc((size_t)n_taps * sizeof(double));
    r->hist = (double *)calloc((size_t)n_rows * (r->n_hist > 0 ? r->n_hist : 1) * r->width, sizeof(double));
    if (!r->h || !r->hist) { spiir_oracle_resamp_destroy(r); return -1; }
    for (int i = 0; i < n_taps; ++i) r->h[i] = (double)taps32[i];
    *out = r;
    return 0;
}

void spiir_oracle_resamp_reset(spiir_oracle_resamp *r)
{
    memset(r->hist, 0, (size_t)r->n_rows * (r->n_hist > 0 ? r->n_hist : 1) * r->width * sizeof(double));
}

/* sample i of (history ++ block) for one row; i in [-n_hist, n_in) */
static inline double hist_or_block(const double *hist, int n_hist, const double *blk, int i, int width, int c)
{
    return (i >= 0) ? blk[(size_t)i * width + c] : hist[(size_t)(n_hist + i) * width + c];
}

static void carry_history(spiir_oracle_resamp *r, const double *in, int n_in)
{
    const int H = r->n_hist, W = r->width;
    if (H <= 0) return;
    double *tmp = (double *)malloc((size_t)H * W * sizeof(double));
    for (int row = 0; row < r->n_rows; ++row) {
        double *hs = r->hist + (size_t)row * H * W;
        const double *blk = in + (size_t)row * n_in * W;
        for (int i = 0; i < H; ++i)
            for (int c = 0; c < W; ++c)
                tmp[(size_t)i * W + c] = hist_or_block(hs, H, blk, n_in - H + i, W, c);
        memcpy(hs, tmp, (size_t)H * W * sizeof(double));
    }
    free(tmp);
}

/*
 * Down-by-2 (O2): v[m] = sum_{j=0}^{N-1} h[j] u[2m - j], u[i<0] = 0, indices global
 * to the stream.  in: [rows][n_in] real double, n_in even.  out: [rows][n_in/2] double.
 */
int spiir_oracle_down2(spiir_oracle_resamp *r, const double *in, int n_in, double *out)
{
    if (!r || r->width != 1 || !in || !out || n_in < 0 || (n_in & 1)) return -1;
    const int N = r->n_taps, H = r->n_hist, n_out = n_in / 2;
#pragma omp parallel for schedule(static)
    for (int row = 0; row < r->n_rows; ++row) {
        const double *hs = r->hist + (size_t)row * H;
        const double *blk = in + (size_t)row * n_in;
        for (int m = 0; m < n_out; ++m) {
            double acc = 0.0;
            for (int j = 0; j < N; ++j)
                acc += r->h[j] * hist_or_block(hs, H, blk, 2 * m - j, 1, 0);
            out[(size_t)row * n_out + m] = acc;
        }
    }
    carry_history(r, in, n_in);
    return 0;
}

/*
 * Up-by-2 (O3): w[2m+p] = 2 sum_{q=0}^{N/2-1} h[2q+p] v[m-q], p in {0,1}, v[i<0] = 0
 * (zero-stuff, filter with h, gain 2).  in: [rows][n_in][2] complex double; out: [rows][2 n_in][2].
 * accumulate != 0: out += w  ("upsampled and added"); else out = w.
 */
int spiir_oracle_up2(spiir_oracle_resamp *r, const double *in, int n_in, double *out, int accumulate)
{
    if (!r || r->width != 2 || !in || !out || n_in < 0) return -1;
    const int N = r->n_taps, H = r->n_hist;
#pragma omp parallel for schedule(static)
    for (int row = 0; row < r->n_rows; ++row) {
        const double *hs = r->hist + (size_t)row * H * 2;
        const double *blk = in + (size_t)row * n_in * 2;
        double *o = out + (size_t)row * n_in * 4;
        for (int m = 0; m < n_in; ++m) {
            for (int p = 0; p < 2; ++p) {
                double accr = 0.0, acci = 0.0;
                for (int q = 0; q < N / 2; ++q) {
                    double hv = r->h[2 * q + p];
                    accr += hv * hist_or_block(hs, H, blk, m - q, 2, 0);
                    acci += hv * hist_or_block(hs, H, blk, m - q, 2, 1);
                }
                size_t i = (size_t)(2 * m + p) * 2;
                if (accumulate) { o[i] += 2.0 * accr; o[i + 1] += 2.0 * acci; }
                else            { o[i]  = 2.0 * accr; o[i + 1]  = 2.0 * acci; }
            }
        }
    }
    carry_history(r, in, n_in);
    return 0;
}

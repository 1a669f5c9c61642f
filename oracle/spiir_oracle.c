/* SPIIR template-bank filter -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  It shares no code with paper_1602_05573_b200/ (the CUDA path).
 *
 * What it computes (the method *is* this definition; BASELINE.json:north_star, and PAPER.md:L303
 * "a parallel bank of single pole IIR filters", L323-L329 "parameter array and the detection data
 * within given time window ... output data of each filter which is the input data in the next
 * iteration", L329/L339 "The SNR of one template needs the outputs of all its filters ... sum all
 * the output of different filters", all in paper section 3.1/3.3):
 *
 *     y_{t,k}[n] = a1_{t,k} * y_{t,k}[n-1] + b0_{t,k} * x[n - d_{t,k}],   y[-1] = 0,  x[m<0] = 0
 *     SNR_t[n]   = sum_{k=0}^{K_t-1} y_{t,k}[n]                            (k ascending)
 *
 * evaluated in IEEE double with complex numbers written out as two doubles, loop order
 * template -> sample -> filter.  Coefficients and strain are the float32 values handed to the GPU,
 * widened exactly to double (reading Q12).  No blocking, fusion or reordering.  OpenMP
 * distributes whole templates over threads; the arithmetic of a template is untouched by it.
 *
 * Readings where the paper is silent: zero initial state and zero pre-history
 * (Q2); d >= 0, d = 0 is the current sample (Q3); plain complex sum, no normalisation (Q4); real
 * input (Q5).
 *
 * Pins (tests/test_oracle_pins.py): impulse closed form, tone closed form with transient, brute-force
 * convolution, linearity/superposition, streaming == one-shot, a1 = 0 -> numpy.convolve,
 * d = 0 real pole -> scipy.signal.lfilter, exact dyadic golden vector, white-noise energy; spiir_oracle_peaks:
 * single-filter impulse closed form (peak |b0|^2 at n0 + d) and numpy.argmax on random rows.
 * No function here is "parity unpinned".
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* One-shot: the definition written out over a whole strain series x[0..N).
 * a1, b0: interleaved (re, im) float32, K = offsets[T] entries each.  snr: interleaved (re, im)
 * double, row t at snr + 2*t*ld, ld >= N.  Returns 0, or -1 on bad arguments. */
int spiir_oracle_run(int32_t T, const int64_t *offsets, const float *a1, const float *b0,
                     const int32_t *delays, const float *x, int64_t N, double *snr, int64_t ld,
                     int32_t n_threads)
{
    if (T < 0 || N < 0 || ld < N || !offsets || !snr) return -1;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif
    int failed = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int32_t t = 0; t < T; ++t) {
        const int64_t k0 = offsets[t], Kt = offsets[t + 1] - offsets[t];
        double *yre = (double *)calloc((size_t)(Kt > 0 ? Kt : 1), sizeof(double));
        double *yim = (double *)calloc((size_t)(Kt > 0 ? Kt : 1), sizeof(double));
        if (!yre || !yim) { failed = 1; free(yre); free(yim); continue; }
        for (int64_t n = 0; n < N; ++n) {
            double sre = 0.0, sim = 0.0;
            for (int64_t k = 0; k < Kt; ++k) {
                const double are = (double)a1[2 * (k0 + k)], aim = (double)a1[2 * (k0 + k) + 1];
                const double bre = (double)b0[2 * (k0 + k)], bim = (double)b0[2 * (k0 + k) + 1];
                const int64_t m = n - (int64_t)delays[k0 + k];
                const double xd = (m >= 0) ? (double)x[m] : 0.0;
                /* y <- a1*y + b0*x[n-d]   (complex multiply written out) */
                const double nre = are * yre[k] - aim * yim[k] + bre * xd;
                const double nim = are * yim[k] + aim * yre[k] + bim * xd;
                yre[k] = nre;
                yim[k] = nim;
                sre += nre;
                sim += nim;
            }
            snr[2 * ((int64_t)t * ld + n)] = sre;
            snr[2 * ((int64_t)t * ld + n) + 1] = sim;
        }
        free(yre);
        free(yim);
    }
    return failed ? -2 : 0;
}

/* Streaming form of the same definition: state y and every past input sample are kept between
 * calls (the whole past is kept, not a ring: obviously correct beats compact here). */
typedef struct spiir_oracle_stream {
    int32_t T;
    int64_t K;
    int64_t *offsets;
    float *a1, *b0;
    int32_t *delays;
    double *yre, *yim;   /* [K] */
    float *xall;         /* [n_done] every sample seen so far */
    int64_t n_done, cap;
} spiir_oracle_stream;

void spiir_oracle_stream_destroy(spiir_oracle_stream *s)
{
    if (!s) return;
    free(s->offsets); free(s->a1); free(s->b0); free(s->delays);
    free(s->yre); free(s->yim); free(s->xall); free(s);
}

spiir_oracle_stream *spiir_oracle_stream_create(int32_t T, const int64_t *offsets, const float *a1,
                                                const float *b0, const int32_t *delays)
{
    if (T < 0 || !offsets) return NULL;
    spiir_oracle_stream *s = (spiir_oracle_stream *)calloc(1, sizeof(*s));
    if (!s) return NULL;
    const int64_t K = offsets[T];
    const size_t Kp = (size_t)(K > 0 ? K : 1);
    s->T = T; s->K = K;
    s->offsets = (int64_t *)malloc(sizeof(int64_t) * (size_t)(T + 1));
    s->a1 = (float *)malloc(sizeof(float) * 2 * Kp);
    s->b0 = (float *)malloc(sizeof(float) * 2 * Kp);
    s->delays = (int32_t *)malloc(sizeof(int32_t) * Kp);
    s->yre = (double *)calloc(Kp, sizeof(double));
    s->yim = (double *)calloc(Kp, sizeof(double));
    if (!s->offsets || !s->a1 || !s->b0 || !s->delays || !s->yre || !s->yim) {
        spiir_oracle_stream_destroy(s);
        return NULL;
    }
    memcpy(s->offsets, offsets, sizeof(int64_t) * (size_t)(T + 1));
    memcpy(s->a1, a1, sizeof(float) * 2 * (size_t)K);
    memcpy(s->b0, b0, sizeof(float) * 2 * (size_t)K);
    memcpy(s->delays, delays, sizeof(int32_t) * (size_t)K);
    return s;
}

/* Consume n more samples; write SNR[t][0..n) (global sample indices n_done .. n_done+n). */
int spiir_oracle_stream_filter(spiir_oracle_stream *s, const float *x, int64_t n, double *snr,
                               int64_t ld, int32_t n_threads)
{
    if (!s || n < 0 || ld < n || (n > 0 && (!x || !snr))) return -1;
    if (s->n_done + n > s->cap) {
        int64_t cap = s->cap ? s->cap : 1024;
        while (cap < s->n_done + n) cap *= 2;
        float *p = (float *)realloc(s->xall, sizeof(float) * (size_t)cap);
        if (!p) return -2;
        s->xall = p; s->cap = cap;
    }
    if (n > 0) memcpy(s->xall + s->n_done, x, sizeof(float) * (size_t)n);
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#else
    (void)n_threads;
#endif
    const int64_t base = s->n_done;
    const float *xall = s->xall;
#pragma omp parallel for schedule(dynamic, 1)
    for (int32_t t = 0; t < s->T; ++t) {
        const int64_t k0 = s->offsets[t], Kt = s->offsets[t + 1] - s->offsets[t];
        double *yre = s->yre + k0, *yim = s->yim + k0;
        for (int64_t j = 0; j < n; ++j) {
            const int64_t ng = base + j;           /* global sample index */
            double sre = 0.0, sim = 0.0;
            for (int64_t k = 0; k < Kt; ++k) {
                const double are = (double)s->a1[2 * (k0 + k)], aim = (double)s->a1[2 * (k0 + k) + 1];
                const double bre = (double)s->b0[2 * (k0 + k)], bim = (double)s->b0[2 * (k0 + k) + 1];
                const int64_t m = ng - (int64_t)s->delays[k0 + k];
                const double xd = (m >= 0) ? (double)xall[m] : 0.0;
                const double nre = are * yre[k] - aim * yim[k] + bre * xd;
                const double nim = are * yim[k] + aim * yre[k] + bim * xd;
                yre[k] = nre;
                yim[k] = nim;
                sre += nre;
                sim += nim;
            }
            snr[2 * ((int64_t)t * ld + j)] = sre;
            snr[2 * ((int64_t)t * ld + j) + 1] = sim;
        }
    }
    s->n_done += n;
    return 0;
}

/* Per-filter outputs y_k[n] of ONE template (no sum) -- lets the pins look at a single filter. */
int spiir_oracle_filter_outputs(int64_t K, const float *a1, const float *b0, const int32_t *delays,
                                const float *x, int64_t N, double *y /* [K][N] interleaved */)
{
    if (K < 0 || N < 0) return -1;
    for (int64_t k = 0; k < K; ++k) {
        const double are = (double)a1[2 * k], aim = (double)a1[2 * k + 1];
        const double bre = (double)b0[2 * k], bim = (double)b0[2 * k + 1];
        double yre = 0.0, yim = 0.0;
        for (int64_t n = 0; n < N; ++n) {
            const int64_t m = n - (int64_t)delays[k];
            const double xd = (m >= 0) ? (double)x[m] : 0.0;
            const double nre = are * yre - aim * yim + bre * xd;
            const double nim = are * yim + aim * yre + bim * xd;
            yre = nre; yim = nim;
            y[2 * (k * N + n)] = yre;
            y[2 * (k * N + n) + 1] = yim;
        }
    }
    return 0;
}

/* Trigger candidates (reading Q16 -- the paper only says the method should "rapidly
 * detect ... signals", and defines no trigger): for every template t and the samples [j0, j0 + n) of
 * its SNR row,  power[t] = max_j |SNR_t[j]|^2  and  index[t] = the first j - j0 that attains it.  Plain scan. */
int spiir_oracle_peaks(int32_t T, const double *snr /* interleaved re, im */, int64_t ld, int64_t j0, int64_t n,
                       double *power, int64_t *index)
{
    if (T < 0 || n < 1 || j0 < 0 || !snr || !power || !index) return -1;
    for (int32_t t = 0; t < T; ++t) {
        double best = -1.0;
        int64_t arg = 0;
        for (int64_t j = 0; j < n; ++j) {
            const double re = snr[2 * ((int64_t)t * ld + j0 + j)], im = snr[2 * ((int64_t)t * ld + j0 + j) + 1];
            const double m = re * re + im * im;
            if (m > best) { best = m; arg = j; }
        }
        power[t] = best;
        index[t] = arg;
    }
    return 0;
}

int32_t spiir_oracle_max_threads(void)
{
#ifdef _OPENMP
    return (int32_t)omp_get_max_threads();
#else
    return 1;
#endif
}

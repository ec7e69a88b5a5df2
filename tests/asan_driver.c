/* asan_driver.c -- exercises oracle/mf_oracle.c under -fsanitize=address,undefined.
 * Built and run by tests/test_oracle_pins.py::test_oracle_under_sanitizers; exit code 0 = clean.
 * Two pins are repeated here in C: P1 (FFT = direct DFT) and the truncation / empty-band paths of
 * orc_filter_bank, which allocate and free the most; the SURVEY.md section-8(f) twins (clustering, chi-squared,
 * time-domain bank) run once each. */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

typedef struct orc_ctx orc_ctx;
typedef struct { double snr_max; int64_t idx_peak; double phase; double sigma; } orc_peak;
typedef struct { int64_t template_idx; int64_t sample_idx; double snr; double phase; } orc_trigger;
int orc_fft(double *x, int64_t n, int sign);
int orc_create(orc_ctx **out, int64_t n, double fs_hz, double f_low_hz);
int orc_destroy(orc_ctx *c);
int orc_set_psd(orc_ctx *c, const double *psd, int64_t n_bins);
int orc_load_segment(orc_ctx *c, const float *samples, int64_t n);
int orc_snr_series(const orc_ctx *c, double m1, double m2, double *rho, double *z, double *sigma);
int orc_filter_bank(const orc_ctx *c, const double *bank, int64_t nt, double thr, orc_peak *peaks,
                    orc_trigger *trig, int64_t cap, int64_t *n_found);
int orc_td_filter_bank(const orc_ctx *c, const double *bank, int64_t nt, double thr, orc_peak *peaks,
                       orc_trigger *trig, int64_t cap, int64_t *n_found);
int orc_chisq(const orc_ctx *c, double m1, double m2, int64_t j, int p, double *chisq, double *zl, int64_t *edges);
int orc_cluster_triggers(const orc_trigger *trig, int64_t n_trig, int64_t n_samples, int64_t window,
                         orc_trigger *out, int64_t out_capacity, int64_t *n_out);

static uint64_t lcg(uint64_t *s) { *s = *s * 6364136223846793005ULL + 1442695040888963407ULL; return *s >> 11; }

int main(void)
{
    const double PI = 3.14159265358979323846;
    /* P1: radix-2 FFT against the direct O(N^2) DFT */
    enum { N = 64 };
    double x[2 * N], y[2 * N];
    uint64_t s = 12345;
    for (int i = 0; i < 2 * N; ++i) x[i] = y[i] = (double)lcg(&s) / 9007199254740992.0 - 0.5;
    if (orc_fft(y, N, -1)) return 2;
    for (int k = 0; k < N; ++k) {
        double re = 0, im = 0;
        for (int j = 0; j < N; ++j) {
            double a = -2.0 * PI * (double)((j * k) % N) / N;
            re += x[2 * j] * cos(a) - x[2 * j + 1] * sin(a);
            im += x[2 * j] * sin(a) + x[2 * j + 1] * cos(a);
        }
        if (fabs(re - y[2 * k]) > 1e-12 * N || fabs(im - y[2 * k + 1]) > 1e-12 * N) return 3;
    }
    /* the bank loop: flat PSD, pseudo-random samples, one empty-band template, truncated list */
    enum { M = 1024 };
    orc_ctx *c = NULL;
    if (orc_create(&c, M, 2048.0, 40.0)) return 4;
    double *psd = (double *)malloc(sizeof(double) * (M / 2 + 1));
    float *d = (float *)malloc(sizeof(float) * M);
    for (int k = 0; k <= M / 2; ++k) psd[k] = (k * 2.0 < 40.0) ? INFINITY : 3.0;
    for (int j = 0; j < M; ++j) d[j] = (float)((double)lcg(&s) / 9007199254740992.0 - 0.5);
    if (orc_set_psd(c, psd, M / 2 + 1) || orc_load_segment(c, d, M)) return 5;
    const double bank[6] = {1.4, 1.4, 80.0, 90.0, 3.0, 2.0};
    orc_peak pk[3];
    orc_trigger tr[100];
    int64_t nf = 0;
    int rc = orc_filter_bank(c, bank, 3, 0.0, pk, tr, 100, &nf);
    if (rc != 1 || nf != 2 * M || pk[1].idx_peak != -1) return 6;          /* WTRUNC, empty band */
    for (int i = 0; i < 100; ++i) if (tr[i].template_idx != 0 || tr[i].sample_idx != i) return 7;
    double *rho = (double *)malloc(sizeof(double) * M);
    double sig = 0;
    if (orc_snr_series(c, 1.4, 1.4, rho, NULL, &sig) || !(sig > 0)) return 8;
    if (fabs(rho[pk[0].idx_peak] - pk[0].snr_max) > 1e-12) return 9;
    /* the section-8(f) twins: clustering of that list, chi-squared bands, the time-domain bank (heavy masses: the
     * chirp must fit 0.5 s; one template too long for the segment -> EINVAL, one below the cut-off -> empty) */
    orc_trigger ev[100];
    int64_t n_ev = 0;
    if (orc_cluster_triggers(tr, 100, M, 3, ev, 100, &n_ev) || n_ev != 1) return 10;
    double chi = -1.0, zl[2 * 7];
    int64_t edges[8];
    if (orc_chisq(c, 3.0, 2.0, pk[2].idx_peak, 7, &chi, zl, edges) || !(chi >= 0.0)) return 11;
    const double tbank[4] = {30.0, 28.0, 90.0, 80.0};
    orc_peak tpk[2];
    if (orc_td_filter_bank(c, tbank, 2, 0.5, tpk, tr, 100, &nf) < 0 || tpk[1].idx_peak != -1 || !(tpk[0].sigma > 0)) return 12;
    const double too_long[2] = {1.4, 1.4};
    if (orc_td_filter_bank(c, too_long, 1, 0.5, tpk, tr, 100, &nf) != -1) return 13;
    free(rho); free(psd); free(d);
    orc_destroy(c);
    puts("asan driver ok");
    return 0;
}

/*
 * mf_oracle.c -- CPU oracle for the cuInspiral matched-filter hot path.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load this library.  It
 * shares no code, header, table or constant generator with the CUDA path under
 * paper_1006_4644_b200/csrc/.
 *
 * Plain, slow, double precision; own radix-2 FFT with directly evaluated
 * twiddles; no blocking, fusion or reordering beyond the definition.  The
 * method is exact (an FFT evaluates the correlation of eq. 2.1 exactly), so the
 * oracle is the definition written out (SURVEY.md §8(c) "Definition", items
 * 1-9), which restates:
 *   PAPER.md:82-88   eq. 2.1  c(t) = \int X(f) Theta*(f)/S_n(f) e^{2 pi i f t} df
 *   PAPER.md:96-103  §2.1 steps 1-4 (generate+normalise, two correlators,
 *                    quadrature sum, threshold/max)
 *   PAPER.md:127-131 §3.1 device_template_proc / complex_mf / cufft_C2R /
 *                    madd2 / maxfind
 * The waveform formula (the paper prints none) is the 2PN SPA
 * phase of BASELINE.json configs[0]; readings A1-A21 of SURVEY.md §8(c) are
 * listed in DESIGN.md.
 *
 * Parity pins (tests/test_oracle_pins.py): every exported function is pinned;
 * none is "parity unpinned".  (orc_cluster_triggers, the SURVEY.md §8(f) NEXT-1
 * twin added in round 2, is pinned by hand-built trigger lists whose clusters
 * follow from the definition by inspection: test_cluster_*; orc_chisq, the
 * NEXT-4 twin, by sum_l z_l = z, chi^2 = 0 for data proportional to the
 * template, <chi^2> = 2p - 2 in noise and equal band powers: test_chisq_*;
 * orc_td_*, the time-domain generator and two-polarisation filter of NEXT-3,
 * by the energy-balance equation, d phi/dt = 2 pi F, the closed forms of a
 * noise-free injection and the agreement with the SPA filter: test_td_*.)
 *
 * Threads: OpenMP across templates only (orc_filter_bank).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_OK       0
#define ORC_EINVAL  -1
#define ORC_ESTATE  -2
#define ORC_ENOMEM  -4
#define ORC_WTRUNC   1

/* SURVEY.md §8(c) item 1 / reading A8: T_sun = G M_sun / c^3 with
 * G M_sun = 1.3271244e20 m^3 s^-2, c = 299792458 m/s. */
static const double ORC_TSUN = 4.925490947641267e-6;
static const double ORC_PI = 3.14159265358979323846264338327950288;

typedef struct { double snr_max; int64_t idx_peak; double phase; double sigma; } orc_peak;
typedef struct { int64_t template_idx; int64_t sample_idx; double snr; double phase; } orc_trigger;

typedef struct orc_ctx {
    int64_t n;          /* samples per segment, power of two */
    double fs, f_low;
    double dt, df;
    double *psd;        /* n/2+1 one-sided S_n, or NULL */
    double *dtil;       /* 2*(n/2+1): d~[k] = dt * sum_j d[j] e^{-2 pi i jk/n}, or NULL */
    double *tw_re, *tw_im;   /* cos/sin(2 pi k / n), k < n/2, each evaluated directly */
    int pn_half_order;       /* 4: 2PN phase (BASELINE.json configs[0], default); 5: + the 2.5PN term (NEXT-3) */
} orc_ctx;

/* ------------------------------------------------------------------ FFT */

static int is_pow2(int64_t n) { return n > 0 && (n & (n - 1)) == 0; }

/* In-place radix-2 decimation-in-time FFT on interleaved (re,im) doubles.
 * sign = -1: X[k] = sum_j x[j] e^{-2 pi i jk/n}  (forward, PAPER.md:84 implies
 *            the inverse carries e^{+2 pi i f t}, so the forward carries e^{-})
 * sign = +1: unnormalised inverse.
 * tw_re/tw_im: table of cos/sin(2 pi k/n), k < n/2 (may be NULL: evaluated here). */
static int fft_radix2(double *x, int64_t n, int sign, const double *tw_re, const double *tw_im)
{
    if (!is_pow2(n)) return ORC_EINVAL;
    if (n == 1) return ORC_OK;
    double *lre = NULL, *lim = NULL;
    if (!tw_re) {
        lre = (double *)malloc(sizeof(double) * (size_t)(n / 2));
        lim = (double *)malloc(sizeof(double) * (size_t)(n / 2));
        if (!lre || !lim) { free(lre); free(lim); return ORC_ENOMEM; }
        for (int64_t k = 0; k < n / 2; ++k) {
            double a = 2.0 * ORC_PI * (double)k / (double)n;
            lre[k] = cos(a); lim[k] = sin(a);
        }
        tw_re = lre; tw_im = lim;
    }
    /* bit reversal */
    for (int64_t i = 1, j = 0; i < n; ++i) {
        int64_t bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) {
            double tr = x[2 * i], ti = x[2 * i + 1];
            x[2 * i] = x[2 * j]; x[2 * i + 1] = x[2 * j + 1];
            x[2 * j] = tr; x[2 * j + 1] = ti;
        }
    }
    for (int64_t len = 2; len <= n; len <<= 1) {
        int64_t half = len >> 1, step = n / len;
        for (int64_t base = 0; base < n; base += len) {
            for (int64_t j = 0; j < half; ++j) {
                double wr = tw_re[j * step];
                double wi = sign > 0 ? tw_im[j * step] : -tw_im[j * step];
                int64_t a = base + j, b = a + half;
                double br = x[2 * b] * wr - x[2 * b + 1] * wi;
                double bi = x[2 * b] * wi + x[2 * b + 1] * wr;
                x[2 * b] = x[2 * a] - br; x[2 * b + 1] = x[2 * a + 1] - bi;
                x[2 * a] += br;           x[2 * a + 1] += bi;
            }
        }
    }
    free(lre); free(lim);
    return ORC_OK;
}

/* Exported FFT (pins P1, P2). */
int orc_fft(double *x_interleaved, int64_t n, int sign)
{
    if (!x_interleaved || (sign != 1 && sign != -1)) return ORC_EINVAL;
    return fft_radix2(x_interleaved, n, sign, NULL, NULL);
}

/* ------------------------------------------------------------ waveform */

/* f_ISCO = 1/(6^{3/2} pi M), M = (m1+m2) T_sun.  SURVEY.md §8(c) item 1. */
double orc_f_isco(double m1, double m2)
{
    double M = (m1 + m2) * ORC_TSUN;
    return 1.0 / (pow(6.0, 1.5) * ORC_PI * M);
}

/* 2PN stationary-phase-approximation phase, t_c = phi_c = 0
 * (BASELINE.json configs[0], "v form"):
 *   Psi_T(f) = -pi/4 + 3/(128 eta v^5) [ 1 + (3715/756 + 55 eta/9) v^2 - 16 pi v^3
 *              + (15293365/508032 + 27145 eta/504 + 3085 eta^2/72) v^4 ],
 *   v = (pi M f)^{1/3}. */
double orc_psi(double m1, double m2, double f)
{
    double M = (m1 + m2) * ORC_TSUN;
    double eta = m1 * m2 / ((m1 + m2) * (m1 + m2));
    double v = cbrt(ORC_PI * M * f);
    double v2 = v * v, v3 = v2 * v, v4 = v2 * v2, v5 = v4 * v;
    double br = 1.0
              + (3715.0 / 756.0 + 55.0 * eta / 9.0) * v2
              - 16.0 * ORC_PI * v3
              + (15293365.0 / 508032.0 + 27145.0 * eta / 504.0 + 3085.0 * eta * eta / 72.0) * v4;
    return -ORC_PI / 4.0 + 3.0 / (128.0 * eta * v5) * br;
}

/* NEXT-3: the paper's stated order, "Post Newtonian approximation of order 2.5 in phase
 * and 0 in amplitude".  The paper prints no formula; the 2.5PN term of the stationary-phase
 * (TaylorF2) phase is taken from the literature -- Arun, Iyer, Sathyaprakash & Sundararajan, Phys. Rev. D 71,
 * 084008 (2005), eq. (3.4); the same expression is eq. (3.18) of Buonanno, Iyer, Ochsner, Pan & Sathyaprakash,
 * Phys. Rev. D 80, 084043 (2009):
 *   Psi_2.5PN(f) = Psi_2PN(f) + 3/(128 eta v^5) * pi (38645/756 - 65 eta/9) (1 + 3 ln(v / v_lso)) v^5,
 *   v = (pi M f)^{1/3},  v_lso = 6^{-1/2}  (so 3 ln(v/v_lso) = ln(f / f_ISCO)).
 * half_order = 4 returns orc_psi.  Pin: tests/test_oracle_pins.py derives every coefficient up to v^5, this one
 * included, from the 2.5PN energy function and flux by series division and two integrations (test_p3b_*). */
double orc_psi_pn(double m1, double m2, double f, int half_order)
{
    double psi = orc_psi(m1, m2, f);
    if (half_order >= 5) {
        double M = (m1 + m2) * ORC_TSUN;
        double eta = m1 * m2 / ((m1 + m2) * (m1 + m2));
        double v = cbrt(ORC_PI * M * f);
        double vlso = 1.0 / sqrt(6.0);
        psi += 3.0 / (128.0 * eta) * ORC_PI * (38645.0 / 756.0 - 65.0 * eta / 9.0) * (1.0 + 3.0 * log(v / vlso));
    }
    return psi;
}

/* Band of a template on the DFT grid, SURVEY.md §8(c) item 2 / readings A6-A7:
 * k_lo = ceil(f_low N/fs), k_hi = min(floor(f_ISCO N/fs), N/2-1); empty if k_hi<k_lo. */
int orc_band(int64_t n, double fs, double f_low, double m1, double m2,
             int64_t *k_lo, int64_t *k_hi)
{
    if (!is_pow2(n) || !(fs > 0) || !(f_low > 0) || !(m1 > 0) || !(m2 > 0)) return ORC_EINVAL;
    double klo = ceil(f_low * ((double)n / fs));
    double khi = floor(orc_f_isco(m1, m2) * ((double)n / fs));
    if (khi > (double)(n / 2 - 1)) khi = (double)(n / 2 - 1);
    *k_lo = (int64_t)klo; *k_hi = (int64_t)khi;
    return ORC_OK;
}

/* ------------------------------------------------------------- context */

int orc_destroy(orc_ctx *c)
{
    if (!c) return ORC_OK;
    free(c->psd); free(c->dtil); free(c->tw_re); free(c->tw_im); free(c);
    return ORC_OK;
}

int orc_create(orc_ctx **out, int64_t n, double fs_hz, double f_low_hz)
{
    if (!out) return ORC_EINVAL;
    *out = NULL;
    if (!is_pow2(n) || n < 4 || n > ((int64_t)1 << 24)) return ORC_EINVAL;
    if (!(fs_hz > 0) || !isfinite(fs_hz)) return ORC_EINVAL;
    if (!(f_low_hz > 0) || !(f_low_hz < fs_hz / 2)) return ORC_EINVAL;
    orc_ctx *c = (orc_ctx *)calloc(1, sizeof(orc_ctx));
    if (!c) return ORC_ENOMEM;
    c->n = n; c->fs = fs_hz; c->f_low = f_low_hz;
    c->dt = 1.0 / fs_hz; c->df = fs_hz / (double)n;
    c->pn_half_order = 4;
    c->tw_re = (double *)malloc(sizeof(double) * (size_t)(n / 2));
    c->tw_im = (double *)malloc(sizeof(double) * (size_t)(n / 2));
    if (!c->tw_re || !c->tw_im) { orc_destroy(c); return ORC_ENOMEM; }
    for (int64_t k = 0; k < n / 2; ++k) {
        double a = 2.0 * ORC_PI * (double)k / (double)n;
        c->tw_re[k] = cos(a); c->tw_im[k] = sin(a);
    }
    *out = c;
    return ORC_OK;
}

/* Phase order of the templates of this context: 4 (2PN, default) or 5 (2.5PN, NEXT-3). */
int orc_set_pn_order(orc_ctx *c, int half_order)
{
    if (!c || (half_order != 4 && half_order != 5)) return ORC_EINVAL;
    c->pn_half_order = half_order;
    return ORC_OK;
}

/* One-sided PSD S_n[0..n/2].  +inf is legal (weight 0, reading A9); an entry
 * <= 0 or NaN inside [f_low, Nyquist) is an error.  Changing the PSD
 * invalidates the loaded segment. */
int orc_set_psd(orc_ctx *c, const double *psd_onesided, int64_t n_bins)
{
    if (!c || !psd_onesided || n_bins != c->n / 2 + 1) return ORC_EINVAL;
    int64_t klo = (int64_t)ceil(c->f_low * ((double)c->n / c->fs));
    for (int64_t k = klo; k < c->n / 2; ++k) {
        double s = psd_onesided[k];
        if (isnan(s) || !(s > 0)) return ORC_EINVAL;
    }
    if (!c->psd) c->psd = (double *)malloc(sizeof(double) * (size_t)n_bins);
    if (!c->psd) return ORC_ENOMEM;
    memcpy(c->psd, psd_onesided, sizeof(double) * (size_t)n_bins);
    free(c->dtil); c->dtil = NULL;
    return ORC_OK;
}

/* d~[k] = dt * sum_j d[j] e^{-2 pi i jk/n} from the float32 samples widened to
 * double (reading A21). */
int orc_load_segment(orc_ctx *c, const float *samples, int64_t n_samples)
{
    if (!c || !samples || n_samples != c->n) return ORC_EINVAL;
    if (!c->psd) return ORC_ESTATE;
    int64_t n = c->n;
    for (int64_t j = 0; j < n; ++j) if (!isfinite(samples[j])) return ORC_EINVAL;
    double *x = (double *)malloc(sizeof(double) * 2 * (size_t)n);
    if (!x) return ORC_ENOMEM;
    for (int64_t j = 0; j < n; ++j) { x[2 * j] = (double)samples[j]; x[2 * j + 1] = 0.0; }
    int rc = fft_radix2(x, n, -1, c->tw_re, c->tw_im);
    if (rc) { free(x); return rc; }
    if (!c->dtil) c->dtil = (double *)malloc(sizeof(double) * 2 * (size_t)(n / 2 + 1));
    if (!c->dtil) { free(x); return ORC_ENOMEM; }
    for (int64_t k = 0; k <= n / 2; ++k) {
        c->dtil[2 * k] = c->dt * x[2 * k];
        c->dtil[2 * k + 1] = c->dt * x[2 * k + 1];
    }
    free(x);
    return ORC_OK;
}

/* Unit-amplitude template h~[k] = f_k^{-7/6} e^{-i Psi_T(f_k)} on [k_lo,k_hi],
 * zero elsewhere; h_out holds 2*(n/2+1) doubles.  SURVEY.md §8(c) item 3. */
int orc_template(const orc_ctx *c, double m1, double m2, double *h_out)
{
    if (!c || !h_out) return ORC_EINVAL;
    int64_t klo, khi;
    int rc = orc_band(c->n, c->fs, c->f_low, m1, m2, &klo, &khi);
    if (rc) return rc;
    memset(h_out, 0, sizeof(double) * 2 * (size_t)(c->n / 2 + 1));
    for (int64_t k = klo; k <= khi; ++k) {
        double f = (double)k * c->df;
        double amp = pow(f, -7.0 / 6.0);
        double psi = orc_psi_pn(m1, m2, f, c->pn_half_order);
        h_out[2 * k] = amp * cos(psi);
        h_out[2 * k + 1] = -amp * sin(psi);
    }
    return ORC_OK;
}

/* sigma^2 = 4 df sum_{k=k_lo}^{k_hi} |h~[k]|^2 / S_n[k] = 4 df sum f_k^{-7/3}/S_n[k]
 * (SURVEY.md §8(c) item 5), the direct sum.  0 for an empty band. */
int orc_sigma2(const orc_ctx *c, double m1, double m2, double *sigma2_out)
{
    if (!c || !sigma2_out) return ORC_EINVAL;
    if (!c->psd) return ORC_ESTATE;
    int64_t klo, khi;
    int rc = orc_band(c->n, c->fs, c->f_low, m1, m2, &klo, &khi);
    if (rc) return rc;
    double s = 0.0;
    for (int64_t k = klo; k <= khi; ++k) {
        double f = (double)k * c->df;
        s += pow(f, -7.0 / 3.0) / c->psd[k];
    }
    *sigma2_out = 4.0 * c->df * s;
    return ORC_OK;
}

/* z[j] = 4 df sum_{k=k_lo}^{k_hi} d~[k] h~*[k] / S_n[k] e^{+2 pi i jk/n}, j=0..n-1
 * (item 6; circular, no samples discarded, reading A11), into z (2n doubles). */
static int filter_z(const orc_ctx *c, double m1, double m2, double *z,
                    int64_t *klo_out, int64_t *khi_out)
{
    int64_t n = c->n, klo, khi;
    int rc = orc_band(n, c->fs, c->f_low, m1, m2, &klo, &khi);
    if (rc) return rc;
    *klo_out = klo; *khi_out = khi;
    memset(z, 0, sizeof(double) * 2 * (size_t)n);
    for (int64_t k = klo; k <= khi; ++k) {
        double f = (double)k * c->df;
        double amp = pow(f, -7.0 / 6.0);
        double psi = orc_psi_pn(m1, m2, f, c->pn_half_order);
        /* conj(h~) = amp e^{+i psi} */
        double hr = amp * cos(psi), hi = amp * sin(psi);
        double dr = c->dtil[2 * k], di = c->dtil[2 * k + 1];
        double wgt = 4.0 * c->df / c->psd[k];
        z[2 * k]     = wgt * (dr * hr - di * hi);
        z[2 * k + 1] = wgt * (dr * hi + di * hr);
    }
    return fft_radix2(z, n, +1, c->tw_re, c->tw_im);
}

/* Full series for one template: rho[j] = |z[j]|/sigma (item 7); z_out may be NULL.
 * For an empty band rho = 0, z = 0, sigma = 0. */
int orc_snr_series(const orc_ctx *c, double m1, double m2,
                   double *rho_out /* n */, double *z_out_or_null /* 2n */, double *sigma_out)
{
    if (!c || !rho_out) return ORC_EINVAL;
    if (!c->psd || !c->dtil) return ORC_ESTATE;
    if (!(m1 > 0) || !(m2 > 0) || !isfinite(m1) || !isfinite(m2)) return ORC_EINVAL;
    int64_t n = c->n, klo, khi;
    double *z = z_out_or_null ? z_out_or_null : (double *)malloc(sizeof(double) * 2 * (size_t)n);
    if (!z) return ORC_ENOMEM;
    int rc = filter_z(c, m1, m2, z, &klo, &khi);
    double s2 = 0.0;
    if (!rc) rc = orc_sigma2(c, m1, m2, &s2);
    if (!rc) {
        double sigma = (khi >= klo) ? sqrt(s2) : 0.0;
        if (sigma_out) *sigma_out = sigma;
        for (int64_t j = 0; j < n; ++j) {
            double re = z[2 * j], im = z[2 * j + 1];
            rho_out[j] = sigma > 0 ? sqrt(re * re + im * im) / sigma : 0.0;
        }
    }
    if (!z_out_or_null) free(z);
    return rc;
}

/* One template: peak (item 7) and raw triggers rho[j] > thr (strict, item 8).
 * trig may be NULL (count only).  Returns the count via *n_found. */
static int filter_one(const orc_ctx *c, double m1, double m2, double thr, int64_t tidx,
                      double *z, double *rho, orc_peak *peak,
                      orc_trigger **trig, int64_t *n_found)
{
    int64_t n = c->n;
    double sigma = 0.0;
    int rc = orc_snr_series(c, m1, m2, rho, z, &sigma);
    if (rc) return rc;
    *n_found = 0; *trig = NULL;
    if (!(sigma > 0)) {            /* empty band: SURVEY.md §8(b) */
        peak->snr_max = 0.0; peak->idx_peak = -1; peak->phase = 0.0; peak->sigma = 0.0;
        return ORC_OK;
    }
    int64_t jbest = 0; double best = rho[0]; int64_t cnt = 0;
    for (int64_t j = 0; j < n; ++j) {
        if (rho[j] > best) { best = rho[j]; jbest = j; }   /* smallest j attaining the max */
        if (rho[j] > thr) ++cnt;
    }
    peak->snr_max = best; peak->idx_peak = jbest; peak->sigma = sigma;
    peak->phase = atan2(z[2 * jbest + 1], z[2 * jbest]);
    if (cnt) {
        orc_trigger *t = (orc_trigger *)malloc(sizeof(orc_trigger) * (size_t)cnt);
        if (!t) return ORC_ENOMEM;
        int64_t m = 0;
        for (int64_t j = 0; j < n; ++j) if (rho[j] > thr) {
            t[m].template_idx = tidx; t[m].sample_idx = j; t[m].snr = rho[j];
            t[m].phase = atan2(z[2 * j + 1], z[2 * j]); ++m;
        }
        *trig = t; *n_found = cnt;
    }
    return ORC_OK;
}

/* The bank loop of PAPER.md:98-102.  bank = n_templates pairs (m1,m2) in solar
 * masses.  Triggers sorted by (template, sample); list truncated at capacity
 * (rc = ORC_WTRUNC) but *n_trig_found is always the full count. */
int orc_filter_bank(const orc_ctx *c, const double *bank_m1m2, int64_t n_templates,
                    double snr_threshold, orc_peak *peaks_out,
                    orc_trigger *trig_out, int64_t trig_capacity, int64_t *n_trig_found)
{
    if (!c || (!bank_m1m2 && n_templates) || n_templates < 0 || (!peaks_out && n_templates))
        return ORC_EINVAL;
    if (!(snr_threshold >= 0)) return ORC_EINVAL;
    if (!c->psd || !c->dtil) return ORC_ESTATE;
    for (int64_t t = 0; t < n_templates; ++t) {
        double m1 = bank_m1m2[2 * t], m2 = bank_m1m2[2 * t + 1];
        if (!(m1 > 0) || !(m2 > 0) || !isfinite(m1) || !isfinite(m2)) return ORC_EINVAL;
    }
    int64_t n = c->n;
    orc_trigger **lists = (orc_trigger **)calloc((size_t)(n_templates ? n_templates : 1), sizeof(*lists));
    int64_t *counts = (int64_t *)calloc((size_t)(n_templates ? n_templates : 1), sizeof(*counts));
    if (!lists || !counts) { free(lists); free(counts); return ORC_ENOMEM; }
    int err = ORC_OK;
#pragma omp parallel
    {
        double *z = (double *)malloc(sizeof(double) * 2 * (size_t)n);
        double *rho = (double *)malloc(sizeof(double) * (size_t)n);
#pragma omp for schedule(dynamic, 1)
        for (int64_t t = 0; t < n_templates; ++t) {
            int rc = (z && rho) ? filter_one(c, bank_m1m2[2 * t], bank_m1m2[2 * t + 1],
                                             snr_threshold, t, z, rho, &peaks_out[t],
                                             &lists[t], &counts[t])
                                : ORC_ENOMEM;
            if (rc) {
#pragma omp critical
                err = rc;
            }
        }
        free(z); free(rho);
    }
    int64_t total = 0, written = 0;
    for (int64_t t = 0; t < n_templates; ++t) {
        for (int64_t m = 0; m < counts[t]; ++m) {
            if (trig_out && written < trig_capacity) trig_out[written++] = lists[t][m];
        }
        total += counts[t];
        free(lists[t]);
    }
    free(lists); free(counts);
    if (n_trig_found) *n_trig_found = total;
    if (err) return err;
    return (total > written && trig_out) ? ORC_WTRUNC : ORC_OK;
}

/* ------------------------------------------------- chi-squared veto */

/* Allen's chi-squared time-frequency discriminator ("a optimized
 * chi-squared [24] test routine", ref. [24] = PAPER.md:321, Phys. Rev. D 71,
 * 062001) for one template at ONE output sample j.  Reading A26:
 *   the template's band [k_lo, k_hi] is cut into p contiguous sub-bands of
 *   (as nearly as the grid allows) equal expected SNR^2: with the running sum
 *   S(k) = 4 df sum_{k'=k_lo..k} f_k'^{-7/3}/S_n[k'] (S(k_hi) = sigma^2), band l =
 *   0..p-1 holds the bins k with  l sigma^2/p <= S(k-1) < (l+1) sigma^2/p
 *   (S(k_lo - 1) = 0), i.e. a bin belongs to the band in which it STARTS;
 *   z_l[j] = 4 df sum_{k in band l} d~[k] h~*[k]/S_n[k] e^{+2 pi i jk/n}  (so sum_l z_l = z[j]),
 *   sigma_l^2 = 4 df sum_{k in band l} f_k^{-7/3}/S_n[k],  p_l = sigma_l^2/sigma^2,
 *   chi^2 = sum_l |z_l - p_l z|^2 / (p_l sigma^2)   (bands with p_l = 0 contribute nothing).
 * With unit-variance quadratures (A4) chi^2 has 2p - 2 degrees of freedom in
 * Gaussian noise and vanishes for data proportional to the template.
 * Written as the definition: direct sums over the bins, the phase of e^{2 pi i jk/n}
 * from the exact integer jk mod n.  zl_out (2p doubles, may be NULL) receives z_l. */
int orc_chisq(const orc_ctx *c, double m1, double m2, int64_t j, int p,
              double *chisq_out, double *zl_out_or_null, int64_t *edges_out_or_null /* p+1 */)
{
    if (!c || !chisq_out || p < 1 || p > 4096) return ORC_EINVAL;
    if (!c->psd || !c->dtil) return ORC_ESTATE;
    if (j < 0 || j >= c->n) return ORC_EINVAL;
    int64_t n = c->n, klo, khi;
    int rc = orc_band(n, c->fs, c->f_low, m1, m2, &klo, &khi);
    if (rc) return rc;
    *chisq_out = 0.0;
    if (khi < klo) return ORC_OK;
    double sigma2 = 0.0;
    rc = orc_sigma2(c, m1, m2, &sigma2);
    if (rc) return rc;
    double *zr = (double *)calloc((size_t)p, sizeof(double)), *zi = (double *)calloc((size_t)p, sizeof(double));
    double *s2 = (double *)calloc((size_t)p, sizeof(double));
    if (!zr || !zi || !s2) { free(zr); free(zi); free(s2); return ORC_ENOMEM; }
    if (edges_out_or_null) for (int l = 0; l <= p; ++l) edges_out_or_null[l] = khi + 1;
    double run = 0.0;                                   /* S(k - 1) */
    int last = -1;
    for (int64_t k = klo; k <= khi; ++k) {
        int l = (int)floor(run / sigma2 * (double)p);
        if (l > p - 1) l = p - 1;
        if (edges_out_or_null && l != last) { for (int q = last + 1; q <= l; ++q) edges_out_or_null[q] = k; last = l; }
        double f = (double)k * c->df;
        double term = 4.0 * c->df * pow(f, -7.0 / 3.0) / c->psd[k];
        double amp = pow(f, -7.0 / 6.0), psi = orc_psi_pn(m1, m2, f, c->pn_half_order);
        double hr = amp * cos(psi), hi = amp * sin(psi);           /* conj(h~) = amp e^{+i psi} */
        double dr = c->dtil[2 * k], di = c->dtil[2 * k + 1];
        double wgt = 4.0 * c->df / c->psd[k];
        double qr = wgt * (dr * hr - di * hi), qi = wgt * (dr * hi + di * hr);
        int64_t jk = (int64_t)(((unsigned long long)j * (unsigned long long)k) % (unsigned long long)n);
        double ang = 2.0 * ORC_PI * (double)jk / (double)n;
        double cr = cos(ang), ci = sin(ang);
        zr[l] += qr * cr - qi * ci;
        zi[l] += qr * ci + qi * cr;
        s2[l] += term;
        run += term;
    }
    double ztr = 0.0, zti = 0.0;
    for (int l = 0; l < p; ++l) { ztr += zr[l]; zti += zi[l]; }
    double chi = 0.0;
    for (int l = 0; l < p; ++l) {
        double pl = s2[l] / sigma2;
        if (!(pl > 0)) continue;
        double er = zr[l] - pl * ztr, ei = zi[l] - pl * zti;
        chi += (er * er + ei * ei) / (pl * sigma2);
    }
    if (zl_out_or_null) for (int l = 0; l < p; ++l) { zl_out_or_null[2 * l] = zr[l]; zl_out_or_null[2 * l + 1] = zi[l]; }
    *chisq_out = chi;
    free(zr); free(zi); free(s2);
    return ORC_OK;
}

/* ------------------------------------------------- trigger clustering */

/* "Reduce the [c(t_0)] set, in order to detect local maximum" (PAPER.md:103,
 * the step after the threshold; done on the CPU).  The paper
 * gives no rule and no window; reading A24:
 *   two above-threshold samples of the SAME template belong to one event if
 *   they are linked by a chain of above-threshold samples of that template in
 *   which consecutive links are at most `window` samples apart, distances
 *   taken on the circle of n_samples (the filter output is circular, A11);
 *   an event is reported as its sample of largest SNR, the smallest sample
 *   index among equal maxima; events are listed by (template, that sample).
 * Written as the definition: pairwise distances and the transitive closure
 * (O(n^2) per template), no sorting assumption on the input.
 * out may be NULL (count only); at most out_capacity events are written
 * (rc = ORC_WTRUNC if there are more), *n_out is always the full count. */
int orc_cluster_triggers(const orc_trigger *trig, int64_t n_trig, int64_t n_samples,
                         int64_t window, orc_trigger *out, int64_t out_capacity, int64_t *n_out)
{
    if ((!trig && n_trig) || n_trig < 0 || n_samples <= 0 || window < 0 || out_capacity < 0 || !n_out)
        return ORC_EINVAL;
    *n_out = 0;
    if (n_trig == 0) return ORC_OK;
    for (int64_t i = 0; i < n_trig; ++i)
        if (trig[i].sample_idx < 0 || trig[i].sample_idx >= n_samples || trig[i].template_idx < 0) return ORC_EINVAL;
    int64_t *label = (int64_t *)malloc(sizeof(int64_t) * (size_t)n_trig);
    orc_trigger *ev = (orc_trigger *)malloc(sizeof(orc_trigger) * (size_t)n_trig);
    if (!label || !ev) { free(label); free(ev); return ORC_ENOMEM; }
    for (int64_t i = 0; i < n_trig; ++i) label[i] = i;
    /* transitive closure: lower the labels of linked pairs until nothing changes */
    for (int changed = 1; changed;) {
        changed = 0;
        for (int64_t i = 0; i < n_trig; ++i)
            for (int64_t j = i + 1; j < n_trig; ++j) {
                if (trig[i].template_idx != trig[j].template_idx || label[i] == label[j]) continue;
                int64_t d = trig[i].sample_idx - trig[j].sample_idx;
                if (d < 0) d = -d;
                if (n_samples - d < d) d = n_samples - d;          /* distance on the circle */
                if (d <= window) {
                    int64_t m = label[i] < label[j] ? label[i] : label[j];
                    label[i] = label[j] = m;
                    changed = 1;
                }
            }
    }
    /* one event per label: largest SNR, smallest sample index among equals */
    int64_t n_ev = 0;
    for (int64_t i = 0; i < n_trig; ++i) {
        if (label[i] != i) continue;                               /* i is the smallest member: the label */
        orc_trigger best = trig[i];
        for (int64_t j = 0; j < n_trig; ++j) {
            if (label[j] != i) continue;
            if (trig[j].snr > best.snr || (trig[j].snr == best.snr && trig[j].sample_idx < best.sample_idx))
                best = trig[j];
        }
        ev[n_ev++] = best;
    }
    /* order by (template, sample): plain insertion sort */
    for (int64_t i = 1; i < n_ev; ++i) {
        orc_trigger x = ev[i];
        int64_t j = i - 1;
        while (j >= 0 && (ev[j].template_idx > x.template_idx ||
                          (ev[j].template_idx == x.template_idx && ev[j].sample_idx > x.sample_idx))) {
            ev[j + 1] = ev[j];
            --j;
        }
        ev[j + 1] = x;
    }
    int64_t w = 0;
    for (int64_t i = 0; i < n_ev; ++i)
        if (out && w < out_capacity) out[w++] = ev[i];
    *n_out = n_ev;
    free(label); free(ev);
    return (out && n_ev > w) ? ORC_WTRUNC : ORC_OK;
}

/* ------------------------------------------------- NEXT-3, second part: the paper's own generator */

/* "the two polarization of the template signal are generated, FFT transformed and normalized" (steps
 * device_template_proc / complex_mf / two cufft_C2R / madd2 of PAPER.md:127-131; "order 2.5 in phase and 0 in
 * amplitude").  The paper prints no formula.  Reading A28: the time-domain
 * approximant is the one with an EXPLICIT phase as a function of time, so that every sample is an independent
 * evaluation (what a one-thread-per-sample generator needs) -- "TaylorT3", Blanchet, Living Rev. Relativity 9, 4
 * (2006), eq. (234), and Buonanno, Iyer, Ochsner, Pan & Sathyaprakash, Phys. Rev. D 80, 084043 (2009), eq. (3.8):
 * with tau = t_c - t, Theta = eta tau / (5 M), y = Theta^{-1/8},
 *   phi_orb(t) = -(1/eta) [ y^-5 + a2 y^-3 - (3 pi/4) y^-2 + a4 y^-1 + a5 ln(Theta) ],   phi_gw = 2 phi_orb,
 *   a2 = 3715/8064 + 55 eta/96,
 *   a4 = 9275495/14450688 + 284875 eta/258048 + 1855 eta^2/2048,
 *   a5 = (-38645/172032 + 65 eta/2048) pi        (the 2.5PN term; 0 at half_order 4),
 * and the gravitational-wave frequency is the exact derivative of that phase, F = (1/2 pi) d phi_gw/dt:
 *   F(y) = Phi(y) / (5 pi M),  Phi(y) = (5/8) y^3 + (3/8) a2 y^5 - (3 pi/16) y^6 + (1/8) a4 y^7 + a5 y^8.
 * Polarisations (amplitude at Newtonian order, i.e. proportional to F^{2/3}; overall scale irrelevant, the
 * template is normalised):  h_+ = (F/f_low)^{2/3} cos(phi_gw),  h_x = (F/f_low)^{2/3} sin(phi_gw).
 * Extent: from F = f_low up to F = f_ISCO (reading A1's cut-off), or up to the maximum of F where the series stops
 * sweeping upward before f_ISCO (it does at 2.5PN): y_t = smallest positive root of dPhi/dy (scan in steps of
 * 1/256 up to y = 4, then bisection); y_end = root of F = f_ISCO on (0, y_t] if F(y_t) >= f_ISCO, else y_t;
 * y_start = root of F = f_low on (0, y_end]; empty if F(y_end) <= f_low.  tau = (5 M/eta) y^-8.
 * Pins (tests/test_oracle_pins.py, test_td_*): the frequency against the energy-balance equation
 * dv/dt = -Flux(v)/(M e'(v)) with the 2.5PN energy and flux (residual of relative order v^6), d phi/dt = 2 pi F,
 * the end points, and the filter pins below. */
typedef struct { double M, eta, a2, a4, a5; } td_coef;

static td_coef td_coefs(double m1, double m2, int half_order)
{
    td_coef q;
    q.M = (m1 + m2) * ORC_TSUN;
    q.eta = m1 * m2 / ((m1 + m2) * (m1 + m2));
    q.a2 = 3715.0 / 8064.0 + 55.0 * q.eta / 96.0;
    q.a4 = 9275495.0 / 14450688.0 + 284875.0 * q.eta / 258048.0 + 1855.0 * q.eta * q.eta / 2048.0;
    q.a5 = half_order >= 5 ? (-38645.0 / 172032.0 + 65.0 * q.eta / 2048.0) * ORC_PI : 0.0;
    return q;
}
static double td_Phi(const td_coef *q, double y)
{
    double y2 = y * y, y3 = y2 * y;
    return y3 * (5.0 / 8.0 + y2 * (3.0 / 8.0 * q->a2 + y * (-3.0 * ORC_PI / 16.0 + y * (q->a4 / 8.0 + y * q->a5))));
}
static double td_dPhi_over_y2(const td_coef *q, double y)       /* (dPhi/dy) / y^2 */
{
    double y2 = y * y;
    return 15.0 / 8.0 + y2 * (15.0 / 8.0 * q->a2 + y * (-9.0 * ORC_PI / 8.0 + y * (7.0 / 8.0 * q->a4 + y * 8.0 * q->a5)));
}
/* root of g(y) = target on [lo, hi], g increasing there, g(lo) <= target <= g(hi): 200 bisections */
static double td_bisect(const td_coef *q, double lo, double hi, double target)
{
    for (int i = 0; i < 200; ++i) {
        double mid = 0.5 * (lo + hi);
        if (td_Phi(q, mid) < target) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}

/* phi_gw and F at tau = t_c - t > 0 (seconds). */
int orc_td_phase(double m1, double m2, double tau, int half_order, double *phi_gw, double *f_gw)
{
    if (!(m1 > 0) || !(m2 > 0) || !(tau > 0) || (half_order != 4 && half_order != 5)) return ORC_EINVAL;
    td_coef q = td_coefs(m1, m2, half_order);
    double theta = q.eta * tau / (5.0 * q.M);
    double y = pow(theta, -0.125);
    if (phi_gw)
        *phi_gw = -(2.0 / q.eta) * (pow(y, -5.0) + q.a2 * pow(y, -3.0) - 0.75 * ORC_PI / (y * y) + q.a4 / y + q.a5 * log(theta));
    if (f_gw) *f_gw = td_Phi(&q, y) / (5.0 * ORC_PI * q.M);
    return ORC_OK;
}

/* Extent of the time-domain template: tau_start >= tau >= tau_end (both 0 when empty), f_end = F(tau_end). */
int orc_td_extent(double m1, double m2, double f_low, int half_order, double *tau_start, double *tau_end, double *f_end)
{
    if (!(m1 > 0) || !(m2 > 0) || !(f_low > 0) || (half_order != 4 && half_order != 5)) return ORC_EINVAL;
    td_coef q = td_coefs(m1, m2, half_order);
    const double scale = 5.0 * ORC_PI * q.M;                  /* Phi = scale * F */
    double y_t = 4.0;
    for (int i = 1; i <= 1024; ++i) {
        double y = (double)i / 256.0;
        if (td_dPhi_over_y2(&q, y) <= 0.0) {
            double lo = (double)(i - 1) / 256.0, hi = y;
            for (int it = 0; it < 200; ++it) {
                double mid = 0.5 * (lo + hi);
                if (td_dPhi_over_y2(&q, mid) > 0.0) lo = mid; else hi = mid;
            }
            y_t = 0.5 * (lo + hi);
            break;
        }
    }
    double f_isco = orc_f_isco(m1, m2);
    double y_end = (td_Phi(&q, y_t) >= scale * f_isco) ? td_bisect(&q, 0.0, y_t, scale * f_isco) : y_t;
    double fe = td_Phi(&q, y_end) / scale;
    if (tau_start) *tau_start = 0.0;
    if (tau_end) *tau_end = 0.0;
    if (f_end) *f_end = fe;
    if (!(fe > f_low)) return ORC_OK;                          /* empty */
    double y_start = td_bisect(&q, 0.0, y_end, scale * f_low);
    if (tau_start) *tau_start = 5.0 * q.M / q.eta * pow(y_start, -8.0);
    if (tau_end) *tau_end = 5.0 * q.M / q.eta * pow(y_end, -8.0);
    return ORC_OK;
}

/* The two polarisations on the sample grid of the context, coalescence at sample 0 (= n, the segment is a circle):
 * sample j has tau_j = (n - j) dt (j = 0: tau = n dt); h = 0 outside [tau_end, tau_start].  hp, hc: n doubles each.
 * EINVAL if the template does not fit the segment (tau_start >= n dt). */
int orc_td_template(const orc_ctx *c, double m1, double m2, double *hp, double *hc)
{
    if (!c || !hp || !hc) return ORC_EINVAL;
    double ts, te, fe;
    int rc = orc_td_extent(m1, m2, c->f_low, c->pn_half_order, &ts, &te, &fe);
    if (rc) return rc;
    int64_t n = c->n;
    if (!(ts < (double)n * c->dt)) return ORC_EINVAL;
    for (int64_t j = 0; j < n; ++j) {
        double tau = (double)(n - j) * c->dt;
        hp[j] = hc[j] = 0.0;
        if (ts > 0.0 && tau <= ts && tau >= te) {
            double phi, f;
            orc_td_phase(m1, m2, tau, c->pn_half_order, &phi, &f);
            double a = pow(f / c->f_low, 2.0 / 3.0);
            hp[j] = a * cos(phi);
            hc[j] = a * sin(phi);
        }
    }
    return ORC_OK;
}

/* The filter of PAPER.md:96-101 with that template, as the definition: for each polarisation p in {+, x}
 *   H_p[k] = dt sum_j h_p[j] e^{-2 pi i jk/n}                                   (forward FFT)
 *   sigma_p^2 = 4 df sum_{k=k_lo}^{n/2-1} |H_p[k]|^2 / S_n[k]                    (normalisation)
 *   c_p[j] = 4 df Re sum_{k=k_lo}^{n/2-1} d~[k] H_p*[k] / S_n[k] e^{+2 pi i jk/n} (correlator, eq. 2.1)
 *   rho[j] = sqrt( (c_+[j]/sigma_+)^2 + (c_x[j]/sigma_x)^2 )                     (reading A4:
 *            each polarisation of unit norm, so that noise alone gives <rho^2> = 2)
 * over every bin from k_lo to Nyquist where S_n is finite (the time-domain template has no band of its own).
 * cp_out / cc_out (n doubles each, may be NULL) receive c_+/sigma_+ and c_x/sigma_x. */
int orc_td_snr_series(const orc_ctx *c, double m1, double m2, double *rho_out, double *cp_out, double *cc_out,
                      double *sigma_p_out, double *sigma_c_out)
{
    if (!c || !rho_out) return ORC_EINVAL;
    if (!c->psd || !c->dtil) return ORC_ESTATE;
    int64_t n = c->n;
    int64_t klo = (int64_t)ceil(c->f_low * ((double)n / c->fs));
    double *hp = (double *)malloc(sizeof(double) * (size_t)n), *hc = (double *)malloc(sizeof(double) * (size_t)n);
    double *x = (double *)malloc(sizeof(double) * 2 * (size_t)n), *q = (double *)malloc(sizeof(double) * 2 * (size_t)n);
    if (!hp || !hc || !x || !q) { free(hp); free(hc); free(x); free(q); return ORC_ENOMEM; }
    int rc = orc_td_template(c, m1, m2, hp, hc);
    double sig[2] = {0.0, 0.0};
    for (int64_t j = 0; j < n; ++j) rho_out[j] = 0.0;
    for (int pol = 0; pol < 2 && !rc; ++pol) {
        const double *h = pol ? hc : hp;
        for (int64_t j = 0; j < n; ++j) { x[2 * j] = h[j]; x[2 * j + 1] = 0.0; }
        rc = fft_radix2(x, n, -1, c->tw_re, c->tw_im);
        if (rc) break;
        memset(q, 0, sizeof(double) * 2 * (size_t)n);
        double s2 = 0.0;
        for (int64_t k = klo; k < n / 2; ++k) {
            if (isinf(c->psd[k])) continue;
            double hr = c->dt * x[2 * k], hi = c->dt * x[2 * k + 1];
            double wgt = 4.0 * c->df / c->psd[k];
            s2 += wgt * (hr * hr + hi * hi);
            double dr = c->dtil[2 * k], di = c->dtil[2 * k + 1];
            q[2 * k]     = wgt * (dr * hr + di * hi);           /* d~ conj(H) */
            q[2 * k + 1] = wgt * (di * hr - dr * hi);
        }
        sig[pol] = sqrt(s2);
        rc = fft_radix2(q, n, +1, c->tw_re, c->tw_im);
        if (rc) break;
        double *cout = pol ? cc_out : cp_out;
        for (int64_t j = 0; j < n; ++j) {
            double v = sig[pol] > 0 ? q[2 * j] / sig[pol] : 0.0;
            if (cout) cout[j] = v;
            rho_out[j] += v * v;
        }
    }
    if (!rc) for (int64_t j = 0; j < n; ++j) rho_out[j] = sqrt(rho_out[j]);
    if (sigma_p_out) *sigma_p_out = sig[0];
    if (sigma_c_out) *sigma_c_out = sig[1];
    free(hp); free(hc); free(x); free(q);
    return rc;
}

/* The bank loop with the time-domain templates: peak = smallest j attaining max rho, phase = atan2(c_x/sigma_x,
 * c_+/sigma_+) there, sigma = sigma_+; triggers rho[j] > threshold (strict), sorted by (template, sample),
 * truncated at the capacity (ORC_WTRUNC).  An empty template returns {0, -1, 0, 0}. */
int orc_td_filter_bank(const orc_ctx *c, const double *bank_m1m2, int64_t n_templates, double snr_threshold,
                       orc_peak *peaks_out, orc_trigger *trig_out, int64_t trig_capacity, int64_t *n_trig_found)
{
    if (!c || (!bank_m1m2 && n_templates) || n_templates < 0 || (!peaks_out && n_templates)) return ORC_EINVAL;
    if (!(snr_threshold >= 0)) return ORC_EINVAL;
    if (!c->psd || !c->dtil) return ORC_ESTATE;
    int64_t n = c->n, total = 0, written = 0;
    double *rho = (double *)malloc(sizeof(double) * (size_t)n), *cp = (double *)malloc(sizeof(double) * (size_t)n);
    double *cc = (double *)malloc(sizeof(double) * (size_t)n);
    if (!rho || !cp || !cc) { free(rho); free(cp); free(cc); return ORC_ENOMEM; }
    int rc = ORC_OK;
    for (int64_t t = 0; t < n_templates && !rc; ++t) {
        double sp = 0.0, sc = 0.0;
        rc = orc_td_snr_series(c, bank_m1m2[2 * t], bank_m1m2[2 * t + 1], rho, cp, cc, &sp, &sc);
        if (rc) break;
        orc_peak *pk = &peaks_out[t];
        if (!(sp > 0) || !(sc > 0)) { pk->snr_max = 0.0; pk->idx_peak = -1; pk->phase = 0.0; pk->sigma = 0.0; continue; }
        int64_t jb = 0;
        for (int64_t j = 0; j < n; ++j) {
            if (rho[j] > rho[jb]) jb = j;
            if (rho[j] > snr_threshold) {
                if (trig_out && written < trig_capacity) {
                    orc_trigger *o = &trig_out[written++];
                    o->template_idx = t; o->sample_idx = j; o->snr = rho[j]; o->phase = atan2(cc[j], cp[j]);
                }
                ++total;
            }
        }
        pk->snr_max = rho[jb]; pk->idx_peak = jb; pk->phase = atan2(cc[jb], cp[jb]); pk->sigma = sp;
    }
    free(rho); free(cp); free(cc);
    if (n_trig_found) *n_trig_found = total;
    if (rc) return rc;
    return (total > written && trig_out) ? ORC_WTRUNC : ORC_OK;
}

/* Threads orc_filter_bank will use (for bench.py's cpu_baseline "cores"). */
int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

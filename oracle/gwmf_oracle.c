/* gwmf_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of what the inspiral matched-filter hot path of
 * arxiv/paper_0906_4175 computes (Eq. 1-5), written from the paper and from the
 * readings listed in DESIGN.md ("Readings of the paper") / SURVEY.md 8(c).  It shares no
 * code, header, table or constant generator with the CUDA path under
 * paper_0906_4175_b200/csrc/ and is only ever called from tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs.
 *
 * Every function cites the passage it follows.  Nothing here is blocked, fused or reordered
 * beyond what the definition states: the band series z_l are N-point inverse DFTs of spectra
 * that are zero outside the band (one radix-2 transform per band), chi^2 is evaluated in the
 * literal two-step form of Eq. 5.  OpenMP is used over templates only.
 *
 * Pins (tests/test_oracle_pins.py): FFT vs the literal O(N^2) DFT, impulse/tone/Parseval
 * closed forms; Eq. 2 values; ISCO cut-offs; phase values, the universal Psi(f_ISCO) of
 * equal-mass systems and the chirp-time derivative; the noise-free injection (rho = A at
 * t_c, closed-form chi^2 residual); covariances; Gaussian-noise moments <rho^2> = 2,
 * <chi^2> = 2p-2; brute-force double sum without any FFT at N = 256.
 * Parity unpinned (definitions of this build, not of the paper): the trigger rule
 * (window maxima, strict threshold, lowest-index tie).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_PI 3.14159265358979323846264338327950288

/* O0. G*Msun/c^3 in seconds (nominal solar mass parameter 1.3271244e20 m^3 s^-2, c = 299792458
 * m/s).  The paper gives masses "in solar masses" and no constant. */
static const double ORC_T_SUN = 4.9254909476412675e-6;

double orc_t_sun(void) { return ORC_T_SUN; }

/* O10. Physical amplitude of the Newtonian-amplitude stationary-phase template ("Newtonian
 * amplitude", "effective distance D_eff"; the paper prints no value -- SURVEY.md 8(c2) reading 4 writes the
 * constant out):  h~(f) = A f^(-7/6) e^{i Psi(f)},
 *     A = sqrt(5/24) pi^(-2/3) (c / D_eff) (T_sun M_chirp / M_sun)^(5/6),   M_chirp = (m1 m2)^(3/5) / (m1+m2)^(1/5),
 * in seconds^(-1/6) (strain per Hz times Hz^(7/6)) for D_eff in megaparsecs and masses in solar masses.
 * c = 299792458 m/s exactly; 1 Mpc = 3.0856775814913673e22 m (IAU 2015: 648000/pi au, au = 149597870700 m).
 * With the library's sigma (Eq. 4 with A = 1) and a PSD given in units of `psd_unit` strain^2/Hz, a source at D_eff
 * has optimal SNR  rho_opt = A(D_eff) sigma / sqrt(psd_unit); the distance at which rho_opt = 1 is
 * D_1 = A(1 Mpc) sigma / sqrt(psd_unit) Mpc, and an event of SNR rho lies at D_eff = D_1 / rho.
 * Pins (tests/test_oracle_pins.py): the M_chirp^(5/6) and 1/D_eff scaling laws, a value evaluated by hand from the
 * constants in tests/golden/p12_amplitude.txt, and the textbook horizon of a 1.4+1.4 binary in the initial-LIGO
 * design curve. */
double orc_amplitude(double m1, double m2, double d_eff_mpc)
{
    const double c_light = 299792458.0, mpc = 3.0856775814913673e22;
    double mchirp = pow(m1 * m2, 0.6) / pow(m1 + m2, 0.2);
    return sqrt(5.0 / 24.0) * pow(ORC_PI, -2.0 / 3.0) * (c_light / (d_eff_mpc * mpc)) * pow(ORC_T_SUN * mchirp, 5.0 / 6.0);
}

/* ------------------------------------------------------------------------------------------
 * Discrete Fourier transforms.  sign = +1: X[k] = sum_j x[j] e^{+2 pi i jk/n} (the "e^{2 pi i f t}"
 * of Eq. 1); sign = -1: the ordinary forward DFT.  Unnormalised, in place.
 * ---------------------------------------------------------------------------------------- */

/* Literal O(n^2) definition; used to pin the fast transform on tiny n. */
void orc_dft_naive(const double *xre, const double *xim, double *yre, double *yim, long n, int sign)
{
    for (long k = 0; k < n; ++k) {
        double sr = 0.0, si = 0.0;
        for (long j = 0; j < n; ++j) {
            /* reduce jk mod n exactly in integers before forming the angle */
            long m = (long)(((unsigned long long)j * (unsigned long long)k) % (unsigned long long)n);
            double ang = sign * 2.0 * ORC_PI * (double)m / (double)n;
            double c = cos(ang), s = sin(ang);
            sr += xre[j] * c - xim[j] * s;
            si += xre[j] * s + xim[j] * c;
        }
        yre[k] = sr;
        yim[k] = si;
    }
}

/* Textbook iterative radix-2 decimation-in-time FFT: bit-reversal permutation, then log2(n)
 * butterfly stages.  Twiddles come from a table of cos/sin evaluated per entry in fp64 (no
 * recurrences).  n must be a power of two.  Returns 0, or -1 on bad n. */
int orc_fft_radix2(double *re, double *im, long n, int sign)
{
    if (n < 1 || (n & (n - 1)) != 0) return -1;
    if (n == 1) return 0;
    /* bit reversal */
    for (long i = 1, j = 0; i < n; ++i) {
        long bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) {
            double t = re[i]; re[i] = re[j]; re[j] = t;
            t = im[i]; im[i] = im[j]; im[j] = t;
        }
    }
    long half = n / 2;
    double *wr = (double *)malloc(sizeof(double) * (size_t)half);
    double *wi = (double *)malloc(sizeof(double) * (size_t)half);
    if (!wr || !wi) { free(wr); free(wi); return -2; }
    for (long m = 0; m < half; ++m) {
        double ang = sign * 2.0 * ORC_PI * (double)m / (double)n;
        wr[m] = cos(ang);
        wi[m] = sin(ang);
    }
    for (long len = 2; len <= n; len <<= 1) {
        long step = n / len;
        long h = len / 2;
        for (long base = 0; base < n; base += len) {
            for (long m = 0; m < h; ++m) {
                double c = wr[m * step], s = wi[m * step];
                long a = base + m, b = a + h;
                double tr = re[b] * c - im[b] * s;
                double ti = re[b] * s + im[b] * c;
                re[b] = re[a] - tr; im[b] = im[a] - ti;
                re[a] += tr;        im[a] += ti;
            }
        }
    }
    free(wr);
    free(wi);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Eq. 2: initial-LIGO one-sided PSD, f0 = 150 Hz, exactly as printed.
 * ---------------------------------------------------------------------------------------- */
double orc_psd_eq2(double f)
{
    double x = f / 150.0;
    return pow(4.49 * x, -56.0) + 0.16 * pow(x, -4.52) + 0.52 + 0.32 * x * x;
}

/* ------------------------------------------------------------------------------------------
 * O4. Template quantities for the mass pair I = (m1, m2).
 * ---------------------------------------------------------------------------------------- */

/* f_ISCO = 1 / (6^{3/2} pi M), M = (m1+m2) T_sun  ("frequency of innermost stable
 * circular orbit"; formula from BASELINE.json:configs[0]). */
double orc_f_isco(double m1, double m2)
{
    double mt = (m1 + m2) * ORC_T_SUN;
    return 1.0 / (pow(6.0, 1.5) * ORC_PI * mt);
}

/* First bin NOT in the template: k_high = min(ceil(f_cut/df), n/2), f_cut = min(f_ISCO, fs/2)
 * ("Nyquist ... or ISCO ... whichever is lower"; reading 7: the first bin
 * with f_k >= f_cut is out, the Nyquist bin is out). */
long orc_k_high(double m1, double m2, long n, double fs)
{
    double df = fs / (double)n;
    double fcut = fmin(orc_f_isco(m1, m2), 0.5 * fs);
    long kh = (long)ceil(fcut / df);
    if (kh > n / 2) kh = n / 2;
    return kh;
}

/* First bin in the template: k_low = ceil(f_low/df) (the bin at exactly 40 Hz is in). */
long orc_k_low(long n, double fs, double f_low)
{
    return (long)ceil(f_low / (fs / (double)n));
}

/* 2PN stationary-phase phase with t_c = 0 ("second order post-Newtonian orbital
 * phases"; the formula is printed in BASELINE.json:configs[0]):
 *   Psi0(f) = -pi/4 + 3/(128 eta v^5) [ 1 + (3715/756 + 55 eta/9) v^2 - 16 pi v^3
 *             + (15293365/508032 + 27145 eta/504 + 3085 eta^2/72) v^4 ],  v = (pi M f)^{1/3}. */
double orc_phase(double m1, double m2, double f)
{
    double mt = (m1 + m2) * ORC_T_SUN;
    double eta = m1 * m2 / ((m1 + m2) * (m1 + m2));
    double v = cbrt(ORC_PI * mt * f);
    double v2 = v * v, v3 = v2 * v, v4 = v2 * v2, v5 = v4 * v;
    double series = 1.0
                  + (3715.0 / 756.0 + 55.0 * eta / 9.0) * v2
                  - 16.0 * ORC_PI * v3
                  + (15293365.0 / 508032.0 + 27145.0 * eta / 504.0 + 3085.0 * eta * eta / 72.0) * v4;
    return -ORC_PI / 4.0 + 3.0 / (128.0 * eta * v5) * series;
}

/* h~_c[k] = f_k^{-7/6} e^{+i Psi0(f_k)} for k_low <= k < k_high, 0 elsewhere; k = 0..n/2-1
 * ("Newtonian amplitude"; amplitude constant 1, reading 4). */
void orc_template(double m1, double m2, long n, double fs, double f_low, double *hre, double *him)
{
    double df = fs / (double)n;
    long kl = orc_k_low(n, fs, f_low), kh = orc_k_high(m1, m2, n, fs);
    for (long k = 0; k < n / 2; ++k) {
        if (k >= kl && k < kh) {
            double f = (double)k * df;
            double a = pow(f, -7.0 / 6.0);
            double ps = orc_phase(m1, m2, f);
            hre[k] = a * cos(ps);
            him[k] = a * sin(ps);
        } else {
            hre[k] = 0.0;
            him[k] = 0.0;
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * O5. Power table C[k] = sum_{k'=k_low..k} f_k'^{-7/3} / S_n[k'], sequential fp64 sum,
 * k = 0..n/2-1 (C[k] = 0 for k < k_low).  Eq. 4: sigma^2 = 4 df C[k_high-1],
 * because |h~_c|^2 = f^{-7/3} for every mass pair.
 * ---------------------------------------------------------------------------------------- */
void orc_power_table(const double *Sn, long n, double fs, double f_low, double *C)
{
    double df = fs / (double)n;
    long kl = orc_k_low(n, fs, f_low);
    double acc = 0.0;
    for (long k = 0; k < n / 2; ++k) {
        if (k >= kl) {
            double f = (double)k * df;
            acc += pow(f, -7.0 / 3.0) / Sn[k];
        }
        C[k] = acc;
    }
}

/* O5 + O6. sigma and the p+1 band edges ("split into p frequency bands such that
 * each contributes an equal amount to the SNR"; reading 8):
 *   e_0 = k_low; for l = 1..p-1: kappa_l = smallest k in [k_low, k_high) with
 *   C[k] >= (l/p) C[k_high-1]; e_l = kappa_l + 1; e_p = k_high.
 * Returns 0, or -3 if the template is empty (k_high <= k_low). */
int orc_sigma_edges(const double *C, long n, double fs, double f_low, long k_high, int p,
                    double *sigma, long *edges)
{
    double df = fs / (double)n;
    long kl = orc_k_low(n, fs, f_low);
    if (k_high <= kl) return -3;
    double total = C[k_high - 1];
    *sigma = sqrt(4.0 * df * total);
    edges[0] = kl;
    for (int l = 1; l < p; ++l) {
        double target = ((double)l / (double)p) * total;
        long k = kl;
        while (k < k_high - 1 && C[k] < target) ++k;   /* linear scan: the plain definition */
        edges[l] = k + 1;
    }
    edges[p] = k_high;
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * O2. Data spectrum D[k] = sum_j s[j] e^{-2 pi i jk/n}, k = 0..n/2 (ordinary forward DFT of the
 * real segment).  In the paper's symbols s~*(f_k) = dt * D[k] (reading 1).
 * ---------------------------------------------------------------------------------------- */
int orc_data_spectrum(const double *s, long n, double *Dre, double *Dim)
{
    double *re = (double *)malloc(sizeof(double) * (size_t)n);
    double *im = (double *)calloc((size_t)n, sizeof(double));
    if (!re || !im) { free(re); free(im); return -2; }
    memcpy(re, s, sizeof(double) * (size_t)n);
    int rc = orc_fft_radix2(re, im, n, -1);
    if (rc == 0) {
        for (long k = 0; k <= n / 2; ++k) { Dre[k] = re[k]; Dim[k] = im[k]; }
    }
    free(re);
    free(im);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * O7 + O8. One template against one segment.
 *   z_l[j] = (4 df dt) sum_{k=e_l}^{e_{l+1}-1} h~_c[k] D[k] / S_n[k] e^{+2 pi i jk/n}   (Eq. 1 split
 *            into p bands; 4 df dt = 4/n; one-sided: zero for k >= n/2)
 *   z = sum_l z_l;   rho[j] = |z[j]| / sigma   (Eq. 3)
 *   chi^2[j] = (p / sigma^2) sum_l |z_l[j] - z[j]/p|^2   (Eq. 5)
 * Outputs: rho[n], chisq[n], sigma, edges[p+1]; optionally (zre, zim non-NULL) the band series
 * as p*n doubles each, band-major.  Returns 0 or a negative code.
 * ---------------------------------------------------------------------------------------- */
int orc_filter_template(const double *Dre, const double *Dim, const double *Sn, const double *C,
                        long n, double fs, double f_low, double m1, double m2, int p,
                        double *rho, double *chisq, double *sigma, long *edges,
                        double *zre_out, double *zim_out)
{
    if (p < 1) return -1;
    long kh = orc_k_high(m1, m2, n, fs);
    int rc = orc_sigma_edges(C, n, fs, f_low, kh, p, sigma, edges);
    if (rc) return rc;
    long half = n / 2;
    double *hre = (double *)malloc(sizeof(double) * (size_t)half);
    double *him = (double *)malloc(sizeof(double) * (size_t)half);
    double *zre = zre_out ? zre_out : (double *)malloc(sizeof(double) * (size_t)n * (size_t)p);
    double *zim = zim_out ? zim_out : (double *)malloc(sizeof(double) * (size_t)n * (size_t)p);
    if (!hre || !him || !zre || !zim) {
        free(hre); free(him);
        if (!zre_out) free(zre);
        if (!zim_out) free(zim);
        return -2;
    }
    orc_template(m1, m2, n, fs, f_low, hre, him);
    double norm = 4.0 / (double)n;             /* 4 df dt */
    for (int l = 0; l < p; ++l) {
        double *br = zre + (size_t)l * (size_t)n, *bi = zim + (size_t)l * (size_t)n;
        memset(br, 0, sizeof(double) * (size_t)n);
        memset(bi, 0, sizeof(double) * (size_t)n);
        for (long k = edges[l]; k < edges[l + 1]; ++k) {
            /* h~_c[k] * D[k] / S_n[k] */
            double qr = (hre[k] * Dre[k] - him[k] * Dim[k]) / Sn[k];
            double qi = (hre[k] * Dim[k] + him[k] * Dre[k]) / Sn[k];
            br[k] = norm * qr;
            bi[k] = norm * qi;
        }
        rc = orc_fft_radix2(br, bi, n, +1);
        if (rc) break;
    }
    if (rc == 0) {
        double s2 = (*sigma) * (*sigma);
        for (long j = 0; j < n; ++j) {
            double zr = 0.0, zi = 0.0;
            for (int l = 0; l < p; ++l) { zr += zre[(size_t)l * n + j]; zi += zim[(size_t)l * n + j]; }
            rho[j] = sqrt(zr * zr + zi * zi) / (*sigma);
            double acc = 0.0;
            for (int l = 0; l < p; ++l) {
                double ar = zre[(size_t)l * n + j] - zr / (double)p;   /* a_{j,l} of PAPER.md:141 */
                double ai = zim[(size_t)l * n + j] - zi / (double)p;   /* b_{j,l} */
                acc += ar * ar + ai * ai;
            }
            chisq[j] = (double)p / s2 * acc;
        }
    }
    free(hre); free(him);
    if (!zre_out) free(zre);
    if (!zim_out) free(zim);
    return rc;
}

/* Same quantities by the literal double sum over k and j: no FFT anywhere (pin P11; tiny n only).
 * D is recomputed here from s by the naive DFT as well. */
int orc_filter_template_bruteforce(const double *s, const double *Sn, long n, double fs, double f_low,
                                   double m1, double m2, int p, double *rho, double *chisq,
                                   double *sigma, long *edges)
{
    long half = n / 2;
    double *C = (double *)malloc(sizeof(double) * (size_t)half);
    double *hre = (double *)malloc(sizeof(double) * (size_t)half);
    double *him = (double *)malloc(sizeof(double) * (size_t)half);
    double *zero = (double *)calloc((size_t)n, sizeof(double));
    double *Dre = (double *)malloc(sizeof(double) * (size_t)n);
    double *Dim = (double *)malloc(sizeof(double) * (size_t)n);
    double *zr = (double *)malloc(sizeof(double) * (size_t)p);
    double *zi = (double *)malloc(sizeof(double) * (size_t)p);
    orc_power_table(Sn, n, fs, f_low, C);
    long kh = orc_k_high(m1, m2, n, fs);
    int rc = orc_sigma_edges(C, n, fs, f_low, kh, p, sigma, edges);
    if (rc == 0) {
        orc_dft_naive(s, zero, Dre, Dim, n, -1);
        orc_template(m1, m2, n, fs, f_low, hre, him);
        double s2 = (*sigma) * (*sigma);
        for (long j = 0; j < n; ++j) {
            double tr = 0.0, ti = 0.0;
            for (int l = 0; l < p; ++l) {
                double ar = 0.0, ai = 0.0;
                for (long k = edges[l]; k < edges[l + 1]; ++k) {
                    double qr = (hre[k] * Dre[k] - him[k] * Dim[k]) / Sn[k];
                    double qi = (hre[k] * Dim[k] + him[k] * Dre[k]) / Sn[k];
                    long m = (long)(((unsigned long long)j * (unsigned long long)k) % (unsigned long long)n);
                    double ang = 2.0 * ORC_PI * (double)m / (double)n;
                    double c = cos(ang), sn = sin(ang);
                    ar += qr * c - qi * sn;
                    ai += qr * sn + qi * c;
                }
                zr[l] = 4.0 / (double)n * ar;
                zi[l] = 4.0 / (double)n * ai;
                tr += zr[l];
                ti += zi[l];
            }
            rho[j] = sqrt(tr * tr + ti * ti) / (*sigma);
            double acc = 0.0;
            for (int l = 0; l < p; ++l) {
                double ar = zr[l] - tr / (double)p, ai = zi[l] - ti / (double)p;
                acc += ar * ar + ai * ai;
            }
            chisq[j] = (double)p / s2 * acc;
        }
    }
    free(C); free(hre); free(him); free(zero); free(Dre); free(Dim); free(zr); free(zi);
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * O9. Trigger maxima ("events ... each with measured SNR and chi^2"; the rule is
 * BASELINE.json:north_star's "per-window SNR-threshold trigger maxima (index, rho, chi^2)",
 * DESIGN.md reading 12 -- parity unpinned by the paper).
 * For each window w of W samples: j* = lowest j attaining max rho; emit iff rho[j*] > thresh.
 * Always fills, per window: best_j, best_rho, best_chisq and runner_up = the largest rho in the
 * window at a sample other than j* and its two neighbours (a competing peak), so that the
 * comparison can apply north_star's "within 1e-3 of the threshold or of a competing peak" rule.
 * Returns the number of windows whose maximum exceeds the threshold.
 * ---------------------------------------------------------------------------------------- */
long orc_window_maxima(const double *rho, const double *chisq, long n, long W, double thresh,
                       long *best_j, double *best_rho, double *best_chisq, double *runner_up)
{
    long count = 0;
    for (long w = 0; w < n / W; ++w) {
        long j0 = w * W, bj = j0;
        for (long j = j0 + 1; j < j0 + W; ++j)
            if (rho[j] > rho[bj]) bj = j;
        double ru = 0.0;
        for (long j = j0; j < j0 + W; ++j)
            if ((j < bj - 1 || j > bj + 1) && rho[j] > ru) ru = rho[j];
        best_j[w] = bj;
        best_rho[w] = rho[bj];
        best_chisq[w] = chisq[bj];
        runner_up[w] = ru;
        if (rho[bj] > thresh) ++count;
    }
    return count;
}

/* ------------------------------------------------------------------------------------------
 * Whole bank against one segment (the unit bench.py's cpu_baseline times): for every template
 * the full rho/chi^2 series are formed and reduced to window maxima.  OpenMP over templates only.
 * Per-template outputs are n/W window records; series of template `keep` (if 0 <= keep < T) are
 * copied to rho_keep / chisq_keep.  status[t] receives each template's return code.
 * ---------------------------------------------------------------------------------------- */
int orc_filter_bank(const double *s, const double *Sn, long n, double fs, double f_low,
                    const double *m1, const double *m2, long T, int p, long W, double thresh,
                    double *sigma, long *edges /* T*(p+1) */,
                    long *best_j, double *best_rho, double *best_chisq, double *runner_up /* T*(n/W) each */,
                    int *status, long keep, double *rho_keep, double *chisq_keep, int n_threads)
{
    long half = n / 2;
    double *Dre = (double *)malloc(sizeof(double) * (size_t)(half + 1));
    double *Dim = (double *)malloc(sizeof(double) * (size_t)(half + 1));
    double *C = (double *)malloc(sizeof(double) * (size_t)half);
    if (!Dre || !Dim || !C) { free(Dre); free(Dim); free(C); return -2; }
    int rc = orc_data_spectrum(s, n, Dre, Dim);
    if (rc) { free(Dre); free(Dim); free(C); return rc; }
    orc_power_table(Sn, n, fs, f_low, C);
    long nw = n / W;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(n_threads > 0 ? n_threads : 1)
#endif
    for (long t = 0; t < T; ++t) {
        double *rho = (double *)malloc(sizeof(double) * (size_t)n);
        double *chi = (double *)malloc(sizeof(double) * (size_t)n);
        if (!rho || !chi) { status[t] = -2; free(rho); free(chi); continue; }
        status[t] = orc_filter_template(Dre, Dim, Sn, C, n, fs, f_low, m1[t], m2[t], p, rho, chi,
                                        &sigma[t], &edges[t * (p + 1)], NULL, NULL);
        if (status[t] == 0) {
            orc_window_maxima(rho, chi, n, W, thresh, &best_j[t * nw], &best_rho[t * nw],
                              &best_chisq[t * nw], &runner_up[t * nw]);
            if (t == keep && rho_keep && chisq_keep) {
                memcpy(rho_keep, rho, sizeof(double) * (size_t)n);
                memcpy(chisq_keep, chi, sizeof(double) * (size_t)n);
            }
        }
        free(rho);
        free(chi);
    }
    free(Dre); free(Dim); free(C);
    return 0;
}

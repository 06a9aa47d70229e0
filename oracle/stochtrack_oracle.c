/*
 * stochtrack_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, float64 CPU statement of the hot path of "all-sky stochtrack"
 * (Thrane & Coughlin, arXiv:1401.8060), written from the paper
 * (/root/reference/PAPER.md at build time; cited below as PAPER.md:<line>)
 * and from the readings recorded in SURVEY.md section 8(c) / DESIGN.md
 * (cited as G<n> / O<n>).  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call this file.
 * It shares no code, header, table or constant generator with the CUDA
 * path under paper_1401_8060_b200/csrc/.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -fPIC -shared (see oracle/oracle.py).
 * -ffp-contract=off is REQUIRED: the rasteriser (O3) is a normative sequence
 * of single IEEE-754 double operations with no fused multiply-add (G15).
 *
 * What is computed, in the paper's order:
 *   O1  random words        Philox4x32-10(seed, track id)     PAPER.md:86, :100 (G5)
 *   O2  template parameters 3 Bezier control points + tau     PAPER.md:75, :100 (G3, G4)
 *   O3  rasterisation       Eq. 6 -> one bin per time column  PAPER.md:83, :73  (G2, G15)
 *   O4  score               Eq. 8 (with Eq. 7's p = CSD/sigma) PAPER.md:104, :96 (G1, G6, G7)
 *   O5  reduce              max / argmax / histogram          PAPER.md:68, :234 (G12, G14)
 * Variants (readings G25, G26 of DESIGN.md):
 *   O4w inverse-variance weighting of SNR_tot (fn. 23): norm_mode 2
 *   O2c/O3c the cubic template family (PAPER.md:75 "other parameterizable curves", :246-252, :287)
 *   O2k/O3k the chirp-law template family f ~ (t_c - t)^(-3/8) (reading G27)
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"):
 *   or_philox4x32_10 : cuRAND host generator CURAND_RNG_PSEUDO_PHILOX4_32_10 (P1)
 *   or_rasterise     : 60-digit decimal brute force, closed-form special cases (P2)
 *   or_score_*       : Eq. 1 + Eq. 5 brute force on full real maps, NumPy complex128
 *                      second implementation, tau = 0, Eq. 3 cosine, Eq. 4's printed
 *                      720 us / 72 us, periodicity / rotation / shift invariants (P3-P6)
 *   or_search        : injected-track self recovery, null variance, chunk combination,
 *                      histogram total (P7-P10)
 *   or_track_params  : what the text fixes (PAPER.md:75 durations >= t_min and t_start < t_mid
 *                      < t_end, :86 six independent random numbers, :100 a uniform, independent
 *                      delay; configs[0] full-duration templates) as statistical statements
 *                      on its output: both end values of N and of j0 | N attained, chi-square
 *                      uniformity of N and of j0 given N, KS uniformity of a/N, y/n_f, tau,
 *                      pairwise independence of all seven parameters
 *                      (tests/test_oracle_track_params_pins.py, which also rebuilds this file
 *                      with eight plausible slips and requires every one to fail).  Which
 *                      Philox word feeds which parameter remains a convention (G5).
 *   or_score_*_w     : reduction to the sqrt(N) statistic for constant sigma, a two-pixel closed
 *                      form, optimality against random weightings, masked pixels dropping out,
 *                      unit null variance under strongly varying sigma (tests/test_oracle_variants.py)
 *   chirp family     : 60-digit decimal evaluation of y0 (T_c / (T_c - u))^(3/8), f^(-8/3) linear in time,
 *                      the closed form f_end = 8 f_start at a = N / 256, monotone pixels, the band clamp,
 *                      self-recovery of an injected bank member (tests/test_oracle_variants.py)
 *   cubic family     : 60-digit decimal brute force of the cubic Bernstein form, end points, convex
 *                      hull, the degree-elevated quadratic reproducing the quadratic family's pixels,
 *                      uniformity / independence of the fourth control point (same file)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define OR_TWO_PI 6.283185307179586476925286766559

/* ------------------------------------------------------------------ O1 -- */
/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), restated: 10 rounds of
 *   (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0))
 * with the key bumped by the Weyl constants between rounds.                 */
void or_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)M0 * c0;
        uint64_t p1 = (uint64_t)M1 * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Domain tag of the track stream: fourth counter word (O1, G5). */
#define OR_TRACK_TAG 0x5354524Bu /* "STRK" */

/* O1: the eight words of track `id`: counter = (id_lo, id_hi, b, tag), b = 0,1;
 * key = (seed_lo, seed_hi).  A pure function of (seed, id) so that runs
 * combine exactly.                                     */
void or_track_words(uint64_t seed, uint64_t id, uint32_t r[8])
{
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    for (uint32_t b = 0; b < 2; ++b) {
        uint32_t ctr[4] = { (uint32_t)id, (uint32_t)(id >> 32), b, OR_TRACK_TAG };
        or_philox4x32_10(ctr, key, r + 4 * b);
    }
}

/* ------------------------------------------------------------------ O2 -- */
typedef struct {
    int32_t N;       /* number of time columns = number of pixels in Gamma */
    int32_t j0;      /* first column; P0.t = j0, P2.t = j0 + N (column edges)            */
    double  a;       /* P1.t - P0.t in columns, 0 < a < N (G3)                          */
    double  y0, y1, y2; /* f_start, f_mid, f_end in bin units, bin k covers [k, k+1)    */
    double  tau;     /* the track's own delay (random-tau mode); else 0    */
    double  y3;      /* cubic family only: f_end; then y1, y2 are the two inner control points */
    int32_t family;  /* 0 quadratic Bezier (Eq. 6), 1 cubic in frequency (G26), 2 chirp law (G27) */
} or_track;

/* O2: "each template can be quickly generated from just six random numbers"
 * plus Delta tau ~ U(-tau_max, +tau_max).       */
int or_track_params(uint64_t seed, uint64_t id, int32_t n_t, int32_t n_f,
                    int32_t n_min, int32_t n_max, double tau_lo, double tau_hi,
                    or_track *t)
{
    t->y3 = 0.0; t->family = 0;
    if (n_t < 1 || n_f < 1 || n_min < 1 || n_max < n_min || n_max > n_t) return -1;
    uint32_t r[8];
    or_track_words(seed, id, r);
    const double two_m32 = 1.0 / 4294967296.0;
    /* duration: uniform integer in [n_min, n_max] -- the t_min constraint */
    t->N  = n_min + (int32_t)(((uint64_t)r[0] * (uint64_t)(n_max - n_min + 1)) >> 32);
    /* start: uniform among the feasible first columns */
    t->j0 = (int32_t)(((uint64_t)r[1] * (uint64_t)(n_t - t->N + 1)) >> 32);
    /* t_mid strictly between t_start and t_end (G3); exact in double */
    t->a  = ((double)r[2] + 0.5) * (double)t->N * two_m32;
    /* frequency control points uniform over the band (G4); exact in double */
    t->y0 = ((double)r[3] + 0.5) * (double)n_f * two_m32;
    t->y1 = ((double)r[4] + 0.5) * (double)n_f * two_m32;
    t->y2 = ((double)r[5] + 0.5) * (double)n_f * two_m32;
    /* delay: tau_lo + (tau_hi - tau_lo) * u, u in (0,1): three rounded double ops */
    {
        double u = ((double)r[6] + 0.5) * two_m32;
        double w = tau_hi - tau_lo;
        double v = w * u;
        t->tau = tau_lo + v;
    }
    return 0;
}

/* O2c (G26): the cubic family.  "Other parameterizable curves such as spline can be used as well"
 * (PAPER.md:75); a compact-binary chirp "is not especially well-described with a second-order Bezier
 * curve".  Reading: a cubic Bezier curve whose TIME control points are the degree-elevated
 * quadratic of O2 (so t(xi) stays the monotone quadratic and O3's root is reused) and whose FREQUENCY has
 * four control points y0, y1, y2, y3, each uniform over the band and independent: the one extra random
 * number is the Philox word O2 leaves unused (r7).  N, j0, a, y0, y1, y2, tau are exactly O2's.          */
int or_track_params_family(uint64_t seed, uint64_t id, int32_t n_t, int32_t n_f,
                           int32_t n_min, int32_t n_max, double tau_lo, double tau_hi,
                           int32_t family, or_track *t)
{
    if (family != 0 && family != 1 && family != 2) return -1;
    int rc = or_track_params(seed, id, n_t, n_f, n_min, n_max, tau_lo, tau_hi, t);
    if (rc != 0 || family == 0) return rc;
    if (family == 2) {
        /* O2k (G27): the chirp-law family.  A compact-binary inspiral sweeps as f ~ (t_c - t)^(-3/8) (the signal of
         * PAPER.md:252 and Fig. 2, which a quadratic "does not describe especially well"): the track is
         * f(u) = y0 (T_c / (T_c - u))^(3/8) from its first column on.  N, j0, y0 (the frequency at the start) and tau
         * are O2's; the time to coalescence from the start is T_c = N^2 / (N - a) > N with O2's a, so that the
         * fraction of T_c left at the track's end, a / N, is uniform in (0, 1).  y1, y2 are not used.            */
        t->family = 2;
        return 0;
    }
    uint32_t r[8];
    or_track_words(seed, id, r);
    t->family = 1;
    t->y3 = ((double)r[7] + 0.5) * (double)n_f * (1.0 / 4294967296.0);
    return 0;
}

/* ------------------------------------------------------------------ O3 -- */
/* Eq. 6: t(xi) = (1-xi)^2 t0 + 2(1-xi)xi t1 + xi^2 t2 with
 * t0 = j0, t1 = j0 + a, t2 = j0 + N gives t(xi) - j0 = (N - 2a) xi^2 + 2a xi.
 * One pixel per time column, sampled at the column centre u = c + 1/2 (G2):
 * solve (N-2a) xi^2 + 2a xi - u = 0 with the cancellation-free root
 * xi = u / (a + sqrt(a^2 + (N-2a) u)), then f(xi) by Eq. 6 and floor to a bin.
 * NORMATIVE operation order, each a single rounded double op (G15).         */
void or_rasterise(const or_track *t, int32_t n_f, int32_t *k_out)
{
    const double a  = t->a;
    const double cc = (double)t->N - 2.0 * a;
    const double aa = a * a;
    if (t->family == 2) {
        /* O3k (G27): y(u) = y0 r^(3/8), r = T_c / (T_c - u) = N^2 / (N^2 - u (N - a)), at the column centre u = c + 1/2;
         * r^(1/8) by three square roots.  NORMATIVE order, every operation a single correctly rounded double op
         * (sqrt and division are; pow is not, so it is not used).                                              */
        const double nn = (double)t->N * (double)t->N;      /* exact: N < 2^26 */
        const double w  = (double)t->N - a;
        for (int32_t c = 0; c < t->N; ++c) {
            double u  = (double)c + 0.5;
            double m  = u * w;
            double D  = nn - m;                              /* > 0: u < N, w < N */
            double r  = nn / D;
            double s  = sqrt(sqrt(sqrt(r)));
            double s2 = s * s;
            double s3 = s2 * s;
            double y  = s3 * t->y0;
            double fl = floor(y);
            int32_t k;
            if (!(fl >= 0.0)) k = 0;
            else if (fl > (double)(n_f - 1)) k = n_f - 1;
            else k = (int32_t)fl;
            k_out[c] = k;
        }
        return;
    }
    for (int32_t c = 0; c < t->N; ++c) {
        double u   = (double)c + 0.5;
        double D   = aa + cc * u;
        if (D < 0.0) D = 0.0;
        double s   = sqrt(D);
        double den = a + s;
        double xi  = u / den;
        double om  = 1.0 - xi;
        double y;
        if (t->family == 0) {
            double b0  = om * om;
            double b1  = 2.0 * (om * xi);
            double b2  = xi * xi;
            y = (b0 * t->y0 + b1 * t->y1) + b2 * t->y2;
        } else {
            /* O3c (G26): f(xi) = (1-xi)^3 y0 + 3 (1-xi)^2 xi y1 + 3 (1-xi) xi^2 y2 + xi^3 y3, the cubic
             * Bernstein form of Eq. 6's construction; NORMATIVE order, single rounded operations.   */
            double om2 = om * om;
            double xi2 = xi * xi;
            double b0  = om2 * om;
            double b1  = 3.0 * (om2 * xi);
            double b2  = 3.0 * (om * xi2);
            double b3  = xi2 * xi;
            y = ((b0 * t->y0 + b1 * t->y1) + b2 * t->y2) + b3 * t->y3;
        }
        double fl  = floor(y);
        int32_t k;
        if (!(fl >= 0.0)) k = 0;
        else if (fl > (double)(n_f - 1)) k = n_f - 1;
        else k = (int32_t)fl;
        k_out[c] = k;
    }
}

/* ------------------------------------------------------------- Eq. 7 ---- */
/* p(t;f) = lambda * sI^* sJ; the library takes CSD = sI^* sJ and
 * sigma = 1/lambda, p = CSD/sigma; sigma <= 0 or non-finite masks the pixel
 * (G11).  sigma_kind: 0 none (=1), 1 per frequency [n_f], 2 per pixel.       */
static double or_sigma_at(const float *sigma, int sigma_kind, int32_t n_f, int32_t j, int32_t k)
{
    if (sigma_kind == 0 || sigma == NULL) return 1.0;
    if (sigma_kind == 1) return (double)sigma[k];
    return (double)sigma[(size_t)j * (size_t)n_f + (size_t)k];
}

void or_prepare_map(const float *csd /* [n_t][n_f][2] */, const float *sigma, int sigma_kind,
                    int32_t n_t, int32_t n_f, double *p /* [n_t][n_f][2] */)
{
    for (int32_t j = 0; j < n_t; ++j)
        for (int32_t k = 0; k < n_f; ++k) {
            size_t o = ((size_t)j * (size_t)n_f + (size_t)k) * 2;
            double s = or_sigma_at(sigma, sigma_kind, n_f, j, k);
            if (!(s > 0.0) || !isfinite(s)) { p[o] = 0.0; p[o + 1] = 0.0; }
            else { p[o] = (double)csd[o] / s; p[o + 1] = (double)csd[o + 1] / s; }
        }
}

/* ------------------------------------------------------------------ O4 -- */
static double or_norm(int32_t N, int norm_mode)
{
    /* norm_mode 0: S / sqrt(N) (G1 default);  1: S / N (Eq. 8 as printed) */
    return norm_mode == 0 ? sqrt((double)N) : (double)N;
}

/* Eq. 8, direct: SNR = N^-alpha sum_c Re[ e^{2 pi i f tau} p ],  f = f_min + k df (G6),
 * Re[e^{i phi}(pr + i pi)] = cos(phi) pr - sin(phi) pi, summed in column order. */
double or_score_direct(const double *p, int32_t n_f, const or_track *t, const int32_t *k,
                       double f_min, double df, double tau, int norm_mode)
{
    double S = 0.0;
    for (int32_t c = 0; c < t->N; ++c) {
        size_t o = ((size_t)(t->j0 + c) * (size_t)n_f + (size_t)k[c]) * 2;
        double phi = OR_TWO_PI * (f_min + (double)k[c] * df) * tau;
        S += cos(phi) * p[o] - sin(phi) * p[o + 1];
    }
    return S / or_norm(t->N, norm_mode);
}

/* Table of twiddles W[k][m] = e^{2 pi i (f_min + k df) tau_m}: the same
 * expression as or_score_direct, evaluated once per (k, m).                 */
void or_build_table(int32_t n_f, double f_min, double df, const double *tau, int32_t n_tau,
                    double *W /* [n_f][n_tau][2] */)
{
    for (int32_t k = 0; k < n_f; ++k)
        for (int32_t m = 0; m < n_tau; ++m) {
            double phi = OR_TWO_PI * (f_min + (double)k * df) * tau[m];
            size_t o = ((size_t)k * (size_t)n_tau + (size_t)m) * 2;
            W[o] = cos(phi); W[o + 1] = sin(phi);
        }
}

/* Eq. 8 for every grid delay of one track, twiddles from the table. */
void or_score_table(const double *p, int32_t n_f, const or_track *t, const int32_t *k,
                    const double *W, int32_t n_tau, int norm_mode, double *snr /* [n_tau] */)
{
    for (int32_t m = 0; m < n_tau; ++m) snr[m] = 0.0;
    for (int32_t c = 0; c < t->N; ++c) {
        size_t o = ((size_t)(t->j0 + c) * (size_t)n_f + (size_t)k[c]) * 2;
        const double pr = p[o], pi = p[o + 1];
        const double *w = W + (size_t)k[c] * (size_t)n_tau * 2;
        for (int32_t m = 0; m < n_tau; ++m)
            snr[m] += w[2 * m] * pr - w[2 * m + 1] * pi;
    }
    double nrm = or_norm(t->N, norm_mode);
    for (int32_t m = 0; m < n_tau; ++m) snr[m] /= nrm;
}

/* ----------------------------------------------------------------- O4w -- */
/* fn. 23: "alternative definitions of SNR_tot (with a different weighting scheme) are also
 * possible".  Reading G25: the inverse-variance combination of the per-pixel cross-power estimates of
 * Appendix A.  A pixel carries Y = Re[e^{i phi} CSD] with variance sigma^2 (A1-A3); the
 * minimum-variance combination of the Y's is sum(Y / sigma^2) / sum(1 / sigma^2) with variance
 * 1 / sum(1 / sigma^2), so its signal-to-noise ratio is
 *       SNR_w = sum_Gamma (Y / sigma^2) / sqrt( sum_Gamma 1 / sigma^2 )
 *             = sum_Gamma (rho / sigma)   / sqrt( sum_Gamma 1 / sigma^2 ),     rho = Re[e^{i phi} p].
 * For constant sigma this is sum(rho) / sqrt(N): G1's alpha = 1/2 statistic.  Masked pixels (G11) have
 * p = 0 and 1/sigma := 0: they drop out of both sums; a template with every pixel masked scores 0.   */
void or_prepare_inv_sigma(const float *sigma, int sigma_kind, int32_t n_t, int32_t n_f, double *r /* [n_t][n_f] */)
{
    for (int32_t j = 0; j < n_t; ++j)
        for (int32_t k = 0; k < n_f; ++k) {
            double s = or_sigma_at(sigma, sigma_kind, n_f, j, k);
            r[(size_t)j * (size_t)n_f + (size_t)k] = (!(s > 0.0) || !isfinite(s)) ? 0.0 : 1.0 / s;
        }
}

double or_score_direct_w(const double *p, const double *r, int32_t n_f, const or_track *t, const int32_t *k,
                         double f_min, double df, double tau)
{
    double S = 0.0, Wt = 0.0;
    for (int32_t c = 0; c < t->N; ++c) {
        size_t px = (size_t)(t->j0 + c) * (size_t)n_f + (size_t)k[c];
        double phi = OR_TWO_PI * (f_min + (double)k[c] * df) * tau;
        double rho = cos(phi) * p[2 * px] - sin(phi) * p[2 * px + 1];
        S  += rho * r[px];
        Wt += r[px] * r[px];
    }
    return Wt > 0.0 ? S / sqrt(Wt) : 0.0;
}

void or_score_table_w(const double *p, const double *r, int32_t n_f, const or_track *t, const int32_t *k,
                      const double *W, int32_t n_tau, double *snr /* [n_tau] */)
{
    double Wt = 0.0;
    for (int32_t m = 0; m < n_tau; ++m) snr[m] = 0.0;
    for (int32_t c = 0; c < t->N; ++c) {
        size_t px = (size_t)(t->j0 + c) * (size_t)n_f + (size_t)k[c];
        const double pr = p[2 * px], pi = p[2 * px + 1], rc = r[px];
        const double *w = W + (size_t)k[c] * (size_t)n_tau * 2;
        for (int32_t m = 0; m < n_tau; ++m)
            snr[m] += (w[2 * m] * pr - w[2 * m + 1] * pi) * rc;
        Wt += rc * rc;
    }
    for (int32_t m = 0; m < n_tau; ++m) snr[m] = Wt > 0.0 ? snr[m] / sqrt(Wt) : 0.0;
}

/* ------------------------------------------------------------------ O5 -- */
/* Total order of G12: larger SNR, then smaller track id, then smaller tau index. */
static int or_better(double s, uint64_t id, int32_t m, double bs, uint64_t bid, int32_t bm)
{
    if (s != bs) return s > bs;
    if (id != bid) return id < bid;
    return m < bm;
}

/* Histogram bin of G14: floor((snr - lo)/(hi - lo) * n_bins), clamped. */
static int32_t or_bin(double snr, double lo, double hi, int32_t n_bins)
{
    double x = (snr - lo) / (hi - lo) * (double)n_bins;
    double fl = floor(x);
    if (!(fl >= 0.0)) return 0;
    if (fl > (double)(n_bins - 1)) return n_bins - 1;
    return (int32_t)fl;
}

typedef struct {
    uint64_t n_tracks, track_offset, seed;
    int32_t  n_min, n_max;
    int32_t  tau_mode;        /* 0 grid, 1 random (one tau per track) */
    int32_t  n_tau;           /* grid size (grid mode); 1 in random mode            */
    double   tau_lo, tau_hi;  /* random mode range                                   */
    int32_t  norm_mode;       /* 0 sqrt(N), 1 N, 2 inverse-variance weighting (O4w)  */
    int32_t  n_bins;          /* 0 = no histogram                                    */
    double   hist_lo, hist_hi;
    int32_t  score_mode;      /* 0 table, 1 direct (grid mode only; random is direct) */
    int32_t  n_threads;       /* OpenMP threads; <= 0 = library default              */
    int32_t  family;          /* 0 quadratic, 1 cubic (O2c / O3c), 2 chirp-law templates (O2k / O3k) */
    int32_t  pad;
} or_search_params;

typedef struct {
    double   max_snr;
    uint64_t arg_track;
    int32_t  arg_tau_index;
    double   arg_tau;
    uint64_t n_evals;         /* sum_i N_i * n_tau                                   */
    uint64_t n_pixels;        /* sum_i N_i                                           */
    int32_t  threads_used;
} or_search_result;

/* The whole path for ids [track_offset, track_offset + n_tracks).
 * p: prepared map (or_prepare_map).  tau_grid: n_tau delays (grid mode).
 * hist: u64[n_bins] or NULL.  snr_dump: double[n_tracks][n_tau] or NULL.
 * k_dump: int32[n_tracks][n_t] (-1 padded), j0_dump/N_dump: int32[n_tracks], or NULL. */
int or_search(const double *p, int32_t n_t, int32_t n_f, double f_min, double df,
              const double *tau_grid, const or_search_params *sp, or_search_result *res,
              uint64_t *hist, double *snr_dump, int32_t *k_dump, int32_t *j0_dump, int32_t *N_dump,
              const double *inv_sigma /* [n_t][n_f] from or_prepare_inv_sigma; only read when norm_mode == 2 */)
{
    const int32_t n_tau = sp->tau_mode == 0 ? sp->n_tau : 1;
    if (n_tau < 1) return -1;
    if (sp->norm_mode == 2 && !inv_sigma) return -1;
    if (sp->family != 0 && sp->family != 1 && sp->family != 2) return -1;
    if (sp->n_min < 1 || sp->n_max < sp->n_min || sp->n_max > n_t) return -1;
    double *W = NULL;
    if (sp->tau_mode == 0 && sp->score_mode == 0) {
        W = (double *)malloc((size_t)n_f * (size_t)n_tau * 2 * sizeof(double));
        if (!W) return -2;
        or_build_table(n_f, f_min, df, tau_grid, n_tau, W);
    }
    int nthreads = 1;
#ifdef _OPENMP
    nthreads = sp->n_threads > 0 ? sp->n_threads : omp_get_max_threads();
#endif
    double   *tmax  = (double *)malloc(sizeof(double) * (size_t)nthreads);
    uint64_t *tid   = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)nthreads);
    int32_t  *tm    = (int32_t *)malloc(sizeof(int32_t) * (size_t)nthreads);
    double   *ttau  = (double *)malloc(sizeof(double) * (size_t)nthreads);
    int      *tset  = (int *)calloc((size_t)nthreads, sizeof(int));
    uint64_t *tev   = (uint64_t *)calloc((size_t)nthreads, sizeof(uint64_t));
    uint64_t *tpx   = (uint64_t *)calloc((size_t)nthreads, sizeof(uint64_t));
    uint64_t *thist = sp->n_bins > 0 && hist
        ? (uint64_t *)calloc((size_t)nthreads * (size_t)sp->n_bins, sizeof(uint64_t)) : NULL;
    int used = 1;
#ifdef _OPENMP
#pragma omp parallel num_threads(nthreads)
#endif
    {
        int me = 0;
#ifdef _OPENMP
        me = omp_get_thread_num();
#pragma omp single
        used = omp_get_num_threads();
#endif
        int32_t *k   = (int32_t *)malloc(sizeof(int32_t) * (size_t)n_t);
        double  *snr = (double *)malloc(sizeof(double) * (size_t)n_tau);
#ifdef _OPENMP
#pragma omp for schedule(dynamic, 64)
#endif
        for (int64_t q = 0; q < (int64_t)sp->n_tracks; ++q) {
            uint64_t id = sp->track_offset + (uint64_t)q;
            or_track t;
            or_track_params_family(sp->seed, id, n_t, n_f, sp->n_min, sp->n_max, sp->tau_lo, sp->tau_hi, sp->family, &t);
            or_rasterise(&t, n_f, k);
            if (sp->norm_mode == 2) {
                if (sp->tau_mode == 0) {
                    if (sp->score_mode == 0) or_score_table_w(p, inv_sigma, n_f, &t, k, W, n_tau, snr);
                    else for (int32_t m = 0; m < n_tau; ++m)
                        snr[m] = or_score_direct_w(p, inv_sigma, n_f, &t, k, f_min, df, tau_grid[m]);
                } else {
                    snr[0] = or_score_direct_w(p, inv_sigma, n_f, &t, k, f_min, df, t.tau);
                }
            } else if (sp->tau_mode == 0) {
                if (sp->score_mode == 0) or_score_table(p, n_f, &t, k, W, n_tau, sp->norm_mode, snr);
                else for (int32_t m = 0; m < n_tau; ++m)
                    snr[m] = or_score_direct(p, n_f, &t, k, f_min, df, tau_grid[m], sp->norm_mode);
            } else {
                snr[0] = or_score_direct(p, n_f, &t, k, f_min, df, t.tau, sp->norm_mode);
            }
            tev[me] += (uint64_t)t.N * (uint64_t)n_tau;
            tpx[me] += (uint64_t)t.N;
            for (int32_t m = 0; m < n_tau; ++m) {
                if (!tset[me] || or_better(snr[m], id, m, tmax[me], tid[me], tm[me])) {
                    tset[me] = 1; tmax[me] = snr[m]; tid[me] = id; tm[me] = m;
                    ttau[me] = sp->tau_mode == 0 ? tau_grid[m] : t.tau;
                }
                if (thist) thist[(size_t)me * (size_t)sp->n_bins
                                 + (size_t)or_bin(snr[m], sp->hist_lo, sp->hist_hi, sp->n_bins)] += 1;
                if (snr_dump) snr_dump[(size_t)q * (size_t)n_tau + (size_t)m] = snr[m];
            }
            if (k_dump) {
                int32_t *row = k_dump + (size_t)q * (size_t)n_t;
                for (int32_t c = 0; c < n_t; ++c) row[c] = c < t.N ? k[c] : -1;
            }
            if (j0_dump) j0_dump[q] = t.j0;
            if (N_dump)  N_dump[q]  = t.N;
        }
        free(k); free(snr);
    }
    /* combine per-thread partial results with the same total order: the result
     * does not depend on the thread count or schedule.        */
    int have = 0;
    res->max_snr = 0.0; res->arg_track = 0; res->arg_tau_index = 0; res->arg_tau = 0.0;
    res->n_evals = 0; res->n_pixels = 0; res->threads_used = used;
    for (int i = 0; i < nthreads; ++i) {
        res->n_evals += tev[i]; res->n_pixels += tpx[i];
        if (!tset[i]) continue;
        if (!have || or_better(tmax[i], tid[i], tm[i], res->max_snr, res->arg_track, res->arg_tau_index)) {
            have = 1; res->max_snr = tmax[i]; res->arg_track = tid[i];
            res->arg_tau_index = tm[i]; res->arg_tau = ttau[i];
        }
    }
    if (thist) {
        for (int32_t b = 0; b < sp->n_bins; ++b) {
            uint64_t s = 0;
            for (int i = 0; i < nthreads; ++i) s += thist[(size_t)i * (size_t)sp->n_bins + (size_t)b];
            hist[b] = s;
        }
    }
    free(W); free(tmax); free(tid); free(tm); free(ttau); free(tset); free(tev); free(tpx); free(thist);
    return 0;
}

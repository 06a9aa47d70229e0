// st_track.cuh -- S1 (template generation) and S2 (rasterisation) of the hot path.
//
// S1: PAPER.md:75, :86 ("each template can be quickly generated from just six
//     random numbers"), :100 (Delta tau ~ U(+-Delta tau_max)); readings G3-G5 of DESIGN.md.
// S2: PAPER.md:83 (Eq. 6), :73 (N = pixels in Gamma); readings G2, G15.
// Second template family (PAPER.md:75 "other parameterizable curves", :246-252, :287; reading G26): a cubic
// Bezier curve whose time control points are the degree-elevated quadratic (so t(xi) and its root are those
// of the quadratic family) and whose frequency has four control points; the extra random number is r7.
// Third family (reading G27): the chirp law f(u) = y0 (T_c / (T_c - u))^(3/8), T_c = N^2 / (N - a).
//
// Everything here is __host__ __device__ so that st_track_params (host, pure)
// and the kernels share one statement of the arithmetic.  The rasteriser is a
// fixed sequence of single IEEE-754 double operations: on the device every
// operation is a *_rn intrinsic (never contracted into an FMA); on the host the
// file is compiled with -ffp-contract=off.
#pragma once
#include <stdint.h>
#include <math.h>

#if defined(__CUDA_ARCH__)
#define ST_DMUL(x, y) __dmul_rn((x), (y))
#define ST_DADD(x, y) __dadd_rn((x), (y))
#define ST_DSUB(x, y) __dsub_rn((x), (y))
#define ST_DDIV(x, y) __ddiv_rn((x), (y))
#define ST_DSQRT(x)   __dsqrt_rn((x))
#define ST_MULHI(x, y) __umulhi((x), (y))
#else
#define ST_DMUL(x, y) ((x) * (y))
#define ST_DADD(x, y) ((x) + (y))
#define ST_DSUB(x, y) ((x) - (y))
#define ST_DDIV(x, y) ((x) / (y))
#define ST_DSQRT(x)   sqrt((x))
#define ST_MULHI(x, y) ((uint32_t)(((uint64_t)(x) * (uint64_t)(y)) >> 32))
#endif

#define ST_HD __host__ __device__ __forceinline__

namespace st {

// Domain tag of the template stream: fourth Philox counter word (G5).
constexpr uint32_t kTrackTag = 0x5354524Bu;  // "STRK"

struct Words8 { uint32_t r[8]; };

// Philox4x32-10 (Salmon et al., SC'11): ten rounds of two 32x32->64 multiplies
// with xor of the neighbouring word and the round key; key += Weyl constants.
ST_HD void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                         uint32_t k0, uint32_t k1, uint32_t* out)
{
    constexpr uint32_t kMulA = 0xD2511F53u, kMulB = 0xCD9E8D57u;
    constexpr uint32_t kWeylA = 0x9E3779B9u, kWeylB = 0xBB67AE85u;
#pragma unroll
    for (int i = 0; i < 10; ++i) {
        const uint32_t hiA = ST_MULHI(kMulA, c0), loA = kMulA * c0;
        const uint32_t hiB = ST_MULHI(kMulB, c2), loB = kMulB * c2;
        c0 = hiB ^ c1 ^ k0;
        c1 = loB;
        c2 = hiA ^ c3 ^ k1;
        c3 = loA;
        k0 += kWeylA;
        k1 += kWeylB;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// The eight words of template `id`: counter (id_lo, id_hi, b, tag), b = 0, 1.
ST_HD Words8 track_words(uint64_t seed, uint64_t id)
{
    Words8 w;
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    const uint32_t i0 = (uint32_t)id, i1 = (uint32_t)(id >> 32);
    philox4x32_10(i0, i1, 0u, kTrackTag, k0, k1, w.r);
    philox4x32_10(i0, i1, 1u, kTrackTag, k0, k1, w.r + 4);
    return w;
}

struct Track {
    int32_t N, j0;
    double a, y0, y1, y2, tau;
    double y3;            // cubic family: f_end (then y1, y2 are the inner control points); else unused
};

struct BankParams {       // what S1 needs besides (seed, id)
    uint64_t seed;
    int32_t n_t, n_f, n_min, n_max;
    double tau_lo, tau_hi;
    int32_t family;       // 0 quadratic (Eq. 6), 1 cubic in frequency (G26), 2 chirp law (G27)
    int32_t pad;
};

// S1.  N uniform in [n_min, n_max]; first column uniform among the feasible
// ones; t_mid strictly inside (t_start, t_end); three frequency control points
// uniform over the band; tau uniform in (tau_lo, tau_hi).  The (r + 1/2) * n *
// 2^-32 products are exact in double (n < 2^20).
ST_HD Track make_track(const BankParams& bp, uint64_t id)
{
    const Words8 w = track_words(bp.seed, id);
    constexpr double kTwoM32 = 1.0 / 4294967296.0;
    Track t;
    t.N  = bp.n_min + (int32_t)ST_MULHI(w.r[0], (uint32_t)(bp.n_max - bp.n_min + 1));
    t.j0 = (int32_t)ST_MULHI(w.r[1], (uint32_t)(bp.n_t - t.N + 1));
    const double dN = (double)t.N, dF = (double)bp.n_f;
    t.a  = ST_DMUL(ST_DMUL((double)w.r[2] + 0.5, dN), kTwoM32);
    t.y0 = ST_DMUL(ST_DMUL((double)w.r[3] + 0.5, dF), kTwoM32);
    t.y1 = ST_DMUL(ST_DMUL((double)w.r[4] + 0.5, dF), kTwoM32);
    t.y2 = ST_DMUL(ST_DMUL((double)w.r[5] + 0.5, dF), kTwoM32);
    const double u = ST_DMUL((double)w.r[6] + 0.5, kTwoM32);
    t.tau = ST_DADD(bp.tau_lo, ST_DMUL(ST_DSUB(bp.tau_hi, bp.tau_lo), u));
    t.y3 = bp.family == 1 ? ST_DMUL(ST_DMUL((double)w.r[7] + 0.5, dF), kTwoM32) : 0.0;
    return t;
}

// Per-track constants of S2.
struct Raster {
    double a, cc, aa, y0, y1, y2, y3;
    double guard;      // fast path: distance from a bin edge below which the normative sequence decides
    int32_t kmax;
    int32_t family;
};

// guard of the fast path: |y_fast - y_normative| <= |dy/dxi| * 6e-12 with |dy/dxi| <= 2 n_f (quadratic) or
// 3 n_f (cubic); a factor 3 is left on top
ST_HD double raster_guard(int32_t n_f, int32_t family)
{
    // (chirp family: y = y0 r^(3/8) <= n_f inside the band, each of the four Newton-refined factors good to ~1e-12)
    const double g = (family == 2 ? 1e-10 : (family ? 6e-11 : 4e-11)) * (double)n_f;
    return g > 1e-6 ? g : 1e-6;
}

ST_HD Raster make_raster(const Track& t, int32_t n_f, int32_t family)
{
    Raster r;
    r.a  = t.a;
    if (family == 2) {                                 // chirp law (G27): cc = N - a, aa = N^2 (exact)
        r.cc = ST_DSUB((double)t.N, t.a);
        r.aa = ST_DMUL((double)t.N, (double)t.N);
    } else {
        r.cc = ST_DSUB((double)t.N, ST_DMUL(2.0, t.a));   // N - 2a
        r.aa = ST_DMUL(t.a, t.a);
    }
    r.y0 = t.y0; r.y1 = t.y1; r.y2 = t.y2; r.y3 = t.y3;
    r.kmax = n_f - 1;
    r.family = family;
    r.guard = raster_guard(n_f, family);
    return r;
}

// S2 for column c of the track: the Bezier time polynomial t(xi) - j0 =
// (N - 2a) xi^2 + 2a xi is solved at the column centre u = c + 1/2 with the
// cancellation-free root xi = u / (a + sqrt(a^2 + (N-2a) u)); f(xi) follows
// Eq. 6 and is floored to a bin.
ST_HD int32_t raster_bin(const Raster& r, int32_t c)
{
    const double u   = (double)c + 0.5;
    if (r.family == 2) {
        // chirp law (G27): y = y0 r^(3/8), r = N^2 / (N^2 - u (N - a)); r^(1/8) by three square roots.  Normative
        // order, every operation correctly rounded (the oracle's O3k).
        const double D  = ST_DSUB(r.aa, ST_DMUL(u, r.cc));
        const double q  = ST_DDIV(r.aa, D);
        const double s  = ST_DSQRT(ST_DSQRT(ST_DSQRT(q)));
        const double y  = ST_DMUL(ST_DMUL(ST_DMUL(s, s), s), r.y0);
        const double fl = floor(y);
        if (!(fl >= 0.0)) return 0;
        if (fl > (double)r.kmax) return r.kmax;
        return (int32_t)fl;
    }
    double D         = ST_DADD(r.aa, ST_DMUL(r.cc, u));
    D                = D < 0.0 ? 0.0 : D;
    const double s   = ST_DSQRT(D);
    const double den = ST_DADD(r.a, s);
    const double xi  = ST_DDIV(u, den);
    const double om  = ST_DSUB(1.0, xi);
    double y;
    if (r.family == 0) {
        const double b0  = ST_DMUL(om, om);
        const double b1  = ST_DMUL(2.0, ST_DMUL(om, xi));
        const double b2  = ST_DMUL(xi, xi);
        y = ST_DADD(ST_DADD(ST_DMUL(b0, r.y0), ST_DMUL(b1, r.y1)), ST_DMUL(b2, r.y2));
    } else {
        // cubic Bernstein form, normative order ((b0 y0 + b1 y1) + b2 y2) + b3 y3 (G26)
        const double om2 = ST_DMUL(om, om);
        const double xi2 = ST_DMUL(xi, xi);
        const double b0  = ST_DMUL(om2, om);
        const double b1  = ST_DMUL(3.0, ST_DMUL(om2, xi));
        const double b2  = ST_DMUL(3.0, ST_DMUL(om, xi2));
        const double b3  = ST_DMUL(xi2, xi);
        y = ST_DADD(ST_DADD(ST_DADD(ST_DMUL(b0, r.y0), ST_DMUL(b1, r.y1)), ST_DMUL(b2, r.y2)), ST_DMUL(b3, r.y3));
    }
    const double fl  = floor(y);
    int32_t k;
    if (!(fl >= 0.0)) k = 0;
    else if (fl > (double)r.kmax) k = r.kmax;
    else k = (int32_t)fl;
    return k;
}

#if defined(__CUDACC__)
// S2, fast path (device).  The same bin as raster_bin, at about half the instructions, without
// branches (so that several columns interleave) and with only two operations on the XU pipe:
// y is evaluated to ~1e-8 bins with the float64 MUFU seeds rsqrt.approx.f64 / rcp.approx.f64
// (~20 bits) refined by one float64 Newton step each, instead of correctly rounded sqrt and
// division; floor and the fractional part come from the 1.5 * 2^52 rounding constant on the FP64
// pipe (no F2I / I2F / FRND conversions).  `redo` is set when y lands within r.guard of a bin edge
// (probability ~2e-6 per pixel) or is not finite; the caller then runs the normative sequence, so
// the index used is ALWAYS floor of the normative y: bit-exact by construction
// (|y_fast - y_normative| <= 2 n_f * 6e-12: xi is good to ~6e-12 after the Newton steps, and
// |dy/dxi| <= 2 n_f; guard = max(1e-6, 4e-11 n_f) leaves a factor 3).
constexpr double kRoundMagic = 6755399441055744.0;   // 1.5 * 2^52: x + M - M rounds x to the nearest integer

// xi(u): root of the time polynomial, float64 MUFU seeds + one Newton step each (~6e-12)
template <typename R>
__device__ __forceinline__ double raster_xi_fast(const R& r, double u)
{
    const double D  = fma(r.cc, u, r.aa);                       // >= min(a, N - a)^2 > 0
    double rs, rc;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(rs) : "d"(D));    // ~ 1 / sqrt(D), ~2^-20
    const double s0 = D * rs;
    const double s  = fma(fma(-s0, s0, D), 0.5 * rs, s0);       // one Newton step  s <- s + (D - s^2) / (2 s)
    const double den = r.a + s;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(rc) : "d"(den));
    const double q0 = u * rc;
    return fma(fma(-den, q0, u), rc, q0);                       // one Newton step on the quotient u / den
}
// sqrt(x), x >= 1, from the MUFU seed and one Newton step (~1e-12)
__device__ __forceinline__ double sqrt_fast(double x)
{
    double rs;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(rs) : "d"(x));
    const double s0 = x * rs;
    return fma(fma(-s0, s0, x), 0.5 * rs, s0);
}
__device__ __forceinline__ double raster_y_fast(const Raster& r, double u)
{
    if (r.family == 2) {                                            // chirp law (G27)
        const double D = fma(-u, r.cc, r.aa);                       // N^2 - u (N - a) > 0
        double rc;
        asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(rc) : "d"(D));
        const double q0 = r.aa * rc;
        const double q  = fma(fma(-D, q0, r.aa), rc, q0);           // N^2 / D, one Newton step on the quotient
        const double s  = sqrt_fast(sqrt_fast(sqrt_fast(q)));
        return (s * s) * (s * r.y0);
    }
    const double xi = raster_xi_fast(r, u);
    const double om = 1.0 - xi;
    if (r.family == 0) return fma(om * om, r.y0, fma(2.0 * (om * xi), r.y1, (xi * xi) * r.y2));
    // cubic: de Casteljau-like nesting ((y0 om + 3 y1 xi) om + 3 y2 xi^2) om + y3 xi^3
    const double xi2 = xi * xi;
    return fma(fma(fma(r.y0, om, 3.0 * r.y1 * xi), om, 3.0 * r.y2 * xi2), om, r.y3 * (xi2 * xi));
}
// floor(y) as an int (clamped to [0, kmax]); redo when y is within the guard of an integer or NaN
template <typename R>
__device__ __forceinline__ int32_t floor_guarded(const R& r, double y, bool& redo)
{
    const double tm = y + kRoundMagic;
    const int32_t kn = __double2loint(tm);                      // the low mantissa word holds the nearest integer
    const double d = y - (tm - kRoundMagic);                    // y - nearest integer, in [-1/2, 1/2]
    redo = !(fabs(d) >= r.guard);                               // near a bin edge, or NaN
    const int32_t k = d < 0.0 ? kn - 1 : kn;                    // floor
    return k < 0 ? 0 : (k > r.kmax ? r.kmax : k);
}
// u = column + 1/2 given as a double (callers step it without int -> double conversions)
template <typename R>
__device__ __forceinline__ int32_t raster_bin_fast_u(const R& r, double u, bool& redo)
{
    return floor_guarded(r, raster_y_fast(r, u), redo);
}
__device__ __forceinline__ int32_t raster_bin_fast(const Raster& r, int32_t c, bool& redo)
{
    return raster_bin_fast_u(r, (double)c + 0.5, redo);
}
__device__ __forceinline__ int32_t raster_bin_fast(const Raster& r, int32_t c)
{
    bool redo;
    const int32_t k = raster_bin_fast(r, c, redo);
    return redo ? raster_bin(r, c) : k;
}
// The fast path's own constants (no y1, y2: the hot kernels hold these 13 registers per template and,
// on the ~2e-6 of the pixels that need the normative sequence, regenerate the template from its id).
struct RasterFast {
    double a, cc, aa, y0, pb, pc, pd, guard;
    int32_t kmax;
    int32_t chirp;     // 1: the chirp law (G27), evaluated from cc = N - a, aa = N^2, y0; the polynomial is unused
};
__device__ __forceinline__ RasterFast make_raster_fast(const Track& t, int32_t n_f, int32_t family)
{
    const Raster r = make_raster(t, n_f, family);
    RasterFast f;
    f.a = r.a; f.cc = r.cc; f.aa = r.aa; f.y0 = r.y0; f.guard = r.guard; f.kmax = r.kmax;
    f.chirp = family == 2;         // a compile-time 0 in the builds whose family is a constant
    if (family == 2) {
        // the chirp law is not a polynomial in xi: raster_y_fast evaluates it from (cc, aa, y0) as the grid kernels'
        // fast path does (MUFU seeds + one Newton step for the quotient and each of the three square roots)
        f.pb = f.pc = f.pd = 0.0;
    } else if (family == 0) {
        f.pb = 2.0 * (t.y1 - t.y0);                             // Eq. 6 in Horner form: y = y0 + xi (pb + xi pc)
        f.pc = (t.y0 - t.y1) + (t.y2 - t.y1);
        f.pd = 0.0;
    } else {                                                    // cubic: y = y0 + xi (pb + xi (pc + xi pd))
        f.pb = 3.0 * (t.y1 - t.y0);
        f.pc = 3.0 * ((t.y0 - t.y1) + (t.y2 - t.y1));
        f.pd = (t.y3 - t.y0) + 3.0 * (t.y1 - t.y2);
    }
    return f;
}
__device__ __forceinline__ double raster_y_fast(const RasterFast& r, double u)
{
    if (r.chirp) {                                                  // as raster_y_fast(const Raster&), family 2
        const double D = fma(-u, r.cc, r.aa);                       // N^2 - u (N - a) > 0
        double rc;
        asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(rc) : "d"(D));
        const double q0 = r.aa * rc;
        const double q  = fma(fma(-D, q0, r.aa), rc, q0);
        const double s  = sqrt_fast(sqrt_fast(sqrt_fast(q)));
        return (s * s) * (s * r.y0);
    }
    const double xi = raster_xi_fast(r, u);
    return fma(xi, fma(xi, fma(xi, r.pd, r.pc), r.pb), r.y0);   // error ~1e-12 n_f / 2461 bins (pd = 0: the quadratic, bit for bit)
}
// normative bin of column c of template `id` (regenerated: rare path)
__device__ __forceinline__ int32_t raster_bin_regen(const BankParams& bp, uint64_t id, int32_t c)
{
    const Track t = make_track(bp, id);
    return raster_bin(make_raster(t, bp.n_f, bp.family), c);
}
// exact (double)k for 0 <= k < 2^31 without the I2F conversion
__device__ __forceinline__ double int_to_double_fast(int32_t k)
{
    return __hiloint2double(0x43380000, k) - kRoundMagic;
}
#endif

}  // namespace st

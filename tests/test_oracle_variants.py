"""Pins of the oracle's two variants, against what the paper and the mathematics
fix -- none of these tests touches the CUDA path.

  O4w  inverse-variance weighting of SNR_tot (fn. 23; Appendix A; reading G25)
  O2c / O3c  the cubic template family (reading G26)
  O2k / O3k  the chirp-law template family f ~ (t_c - t)^(-3/8) (reading G27)
"""
from decimal import Decimal, getcontext

import numpy as np
import pytest
from scipy import stats

from workloads import synth


# ------------------------------------------------------------------------------------- O4w
def _track_and_pixels(orc, seed, tid, n_t, n_f):
    t = orc.track_params(seed, tid, n_t, n_f, 4, n_t)
    return t, orc.rasterise(t, n_f)


def test_weighted_statistic_reduces_to_sqrtN_for_constant_sigma(orc):
    """Constant sigma: sum(rho / sigma) / sqrt(sum 1 / sigma^2) = sum(rho) / sqrt(N) -- G1's alpha = 1/2."""
    n_t, n_f, f_min, df = 40, 33, 40.0, 1.0
    csd = synth.noise_csd(n_t, n_f, 3)
    taus = synth.tau_linspace(9)
    W = orc.build_table(n_f, f_min, df, taus)
    for c in (1.0, 0.37, 12.5):
        sig = np.full(n_f, c, dtype=np.float32)
        p = orc.prepare_map(csd, sig)
        r = orc.prepare_inv_sigma((n_t, n_f), sig)
        for tid in range(25):
            t, k = _track_and_pixels(orc, 8, tid, n_t, n_f)
            plain = orc.score_table(p, t, k, W, orc.NORM_SQRT_N)
            w = orc.score_table_w(p, r, t, k, W)
            assert np.allclose(w, plain, rtol=1e-13, atol=1e-13)
            for m in (0, 4, 8):
                assert abs(orc.score_direct_w(p, r, t, k, f_min, df, taus[m]) - w[m]) <= 1e-13 * max(1.0, abs(w[m]))


def test_weighted_statistic_two_pixel_closed_form_and_scaling(orc):
    """Two pixels with Y = (3, 4), sigma = (1, 2), tau = 0: (3/1 + 4/4) / sqrt(1 + 1/4) = 4 / sqrt(1.25).
    Rescaling every sigma by c divides the statistic by c (as rho itself)."""
    n_t, n_f = 2, 3
    csd = np.zeros((n_t, n_f), dtype=np.complex64)
    csd[0, 1], csd[1, 1] = 3.0 + 7.0j, 4.0 - 2.0j            # imaginary parts are invisible at tau = 0
    sig = np.ones((n_t, n_f), dtype=np.float32)
    sig[1, 1] = 2.0
    t = orc.make_track(2, 0, 1.0, 1.5, 1.5, 1.5)
    k = orc.rasterise(t, n_f)
    assert list(k) == [1, 1]
    p, r = orc.prepare_map(csd, sig), orc.prepare_inv_sigma((n_t, n_f), sig)
    assert abs(orc.score_direct_w(p, r, t, k, 40.0, 1.0, 0.0) - 4.0 / np.sqrt(1.25)) < 1e-14
    sig3 = (3.0 * sig).astype(np.float32)
    p3, r3 = orc.prepare_map(csd, sig3), orc.prepare_inv_sigma((n_t, n_f), sig3)
    assert abs(orc.score_direct_w(p3, r3, t, k, 40.0, 1.0, 0.0) - 4.0 / np.sqrt(1.25) / 3.0) < 1e-14
    # a pure phase rotation of the data is undone by the matching delay (Eq. 8's phase factor is untouched)
    f, tau0 = 41.0, 2.5e-3
    csd2 = (csd * np.exp(-2j * np.pi * f * tau0)).astype(np.complex64)
    p2 = orc.prepare_map(csd2, sig)
    assert abs(orc.score_direct_w(p2, r, t, k, 40.0, 1.0, tau0) - 4.0 / np.sqrt(1.25)) < 1e-6


def test_weighted_statistic_is_the_optimal_linear_combination(orc):
    """A constant cross-power Y0 in every pixel of a track, noise-free: any linear combination sum(u Y) has
    SNR Y0 sum(u) / sqrt(sum u^2 sigma^2) <= Y0 sqrt(sum 1 / sigma^2), with equality for u = 1 / sigma^2
    (Cauchy-Schwarz).  The oracle must return the bound; the unweighted statistic must fall short of it."""
    n_t, n_f, Y0 = 60, 50, 0.75
    rng = np.random.default_rng(2)
    sig = np.exp(0.7 * rng.standard_normal((n_t, n_f))).astype(np.float32)
    csd = np.full((n_t, n_f), Y0, dtype=np.complex64)
    p, r = orc.prepare_map(csd, sig), orc.prepare_inv_sigma((n_t, n_f), sig)
    for tid in range(10):
        t, k = _track_and_pixels(orc, 21, tid, n_t, n_f)
        s = sig[t.j0 + np.arange(t.N), k].astype(np.float64)
        bound = Y0 * np.sqrt((1.0 / s ** 2).sum())
        got = orc.score_direct_w(p, r, t, k, 40.0, 1.0, 0.0)
        assert abs(got - bound) <= 1e-12 * bound
        for _ in range(20):
            u = rng.random(t.N) + 0.01
            assert Y0 * u.sum() / np.sqrt((u ** 2 * s ** 2).sum()) <= bound * (1 + 1e-12)
        plain = orc.score_direct(p, t, k, 40.0, 1.0, 0.0, orc.NORM_SQRT_N)
        assert plain < got * (1 - 1e-3)                      # uniform weights are strictly worse here


def test_weighted_statistic_masked_pixels_drop_out(orc):
    """G11 + G25: a masked pixel leaves both sums; the statistic equals that of the remaining pixels."""
    n_t, n_f = 30, 20
    csd = synth.noise_csd(n_t, n_f, 9)
    sig = synth.make_sigma("per_pixel", 0.4, n_t, n_f, 9)
    t = orc.make_track(30, 0, 11.0, 3.5, 15.5, 8.5)
    k = orc.rasterise(t, n_f)
    sig_m = sig.copy()
    masked = [2, 3, 17, 29]
    for c in masked:
        sig_m[c, k[c]] = 0.0 if c % 2 else np.inf
    p, r = orc.prepare_map(csd, sig_m), orc.prepare_inv_sigma((n_t, n_f), sig_m)
    got = orc.score_direct_w(p, r, t, k, 40.0, 1.0, 1.3e-3)
    keep = np.array([c for c in range(30) if c not in masked])
    f = 40.0 + k[keep]
    rho = np.real(np.exp(2j * np.pi * f * 1.3e-3) * csd[keep, k[keep]].astype(np.complex128) / sig[keep, k[keep]])
    s = sig[keep, k[keep]].astype(np.float64)
    assert abs(got - (rho / s).sum() / np.sqrt((1 / s ** 2).sum())) < 1e-12
    sig_all = np.zeros((n_t, n_f), dtype=np.float32)
    assert orc.score_direct_w(orc.prepare_map(csd, sig_all), orc.prepare_inv_sigma((n_t, n_f), sig_all), t, k, 40.0, 1.0, 0.0) == 0.0


def test_weighted_statistic_unit_null_variance_under_varying_sigma(orc):
    """Var rho = 1 per pixel (A1-A3) gives Var SNR_w = sum(1/sigma^2) / sum(1/sigma^2) = 1 whatever sigma(t; f);
    the search path (or_search with norm 2) is the one exercised, histogram total included (P10)."""
    n_t, n_f, T = 200, 300, 40000
    rng = np.random.default_rng(7)
    sig = np.exp(0.8 * rng.standard_normal((n_t, n_f))).astype(np.float32)
    # CSD whose rho = Re[e^{i phi} CSD / sigma] has unit variance: unit-variance complex parts times sigma
    z = rng.standard_normal((n_t, n_f)) + 1j * rng.standard_normal((n_t, n_f))
    csd = (z * sig).astype(np.complex64)
    p, r = orc.prepare_map(csd, sig), orc.prepare_inv_sigma((n_t, n_f), sig)
    res = orc.search(p, 40.0, 1.0, T, 5, 10, 200, tau_grid=np.array([1.7e-3]), norm=orc.NORM_INVVAR, inv_sigma=r,
                     dump_snr=True, n_bins=400)
    s = res["snr"][:, 0]
    assert abs(s.mean()) < 0.03 and abs(s.var() - 1.0) < 0.04 and int(res["hist"].sum()) == T
    i = int(np.argmax(s))
    assert res["arg_track"] == i and res["max_snr"] == s[i]
    t = orc.track_params(5, i, n_t, n_f, 10, 200)
    assert res["max_snr"] == orc.score_table_w(p, r, t, orc.rasterise(t, n_f), orc.build_table(n_f, 40.0, 1.0, np.array([1.7e-3])))[0]
    with pytest.raises(ValueError):
        orc.search(p, 40.0, 1.0, 10, 5, 10, 200, tau_grid=np.array([0.0]), norm=orc.NORM_INVVAR)


# ------------------------------------------------------------------------------------- cubic family
def _decimal_cubic(t, n_f):
    """60-digit evaluation of the cubic curve at column centres with the TEXTBOOK root of the time quadratic
    and the power-basis (not Bernstein) form of the frequency cubic."""
    getcontext().prec = 60
    a, N = Decimal(t.a), Decimal(t.N)
    y0, y1, y2, y3 = (Decimal(x) for x in (t.y0, t.y1, t.y2, t.y3))
    A, B = N - 2 * a, 2 * a
    c1, c2, c3 = 3 * (y1 - y0), 3 * (y0 - 2 * y1 + y2), y3 - 3 * y2 + 3 * y1 - y0
    ks, ys = [], []
    for c in range(t.N):
        u = Decimal(c) + Decimal("0.5")
        xi = u / B if A == 0 else (-B + (B * B + 4 * A * u).sqrt()) / (2 * A)
        y = y0 + xi * (c1 + xi * (c2 + xi * c3))
        ys.append(y)
        ks.append(min(max(int(y.to_integral_value(rounding="ROUND_FLOOR")), 0), n_f - 1))
    return ks, ys


def test_cubic_rasteriser_vs_60_digit_brute_force(orc):
    n_pix = n_mis = 0
    for seed, n_t, n_f, n_min, n_max, count in ((4, 1000, 2461, 10, 1000, 150), (1, 250, 961, 10, 250, 250), (0, 64, 64, 64, 64, 200)):
        for tid in range(count):
            t = orc.track_params(seed, tid, n_t, n_f, n_min, n_max, family=orc.FAMILY_CUBIC)
            assert t.family == 1
            k = orc.rasterise(t, n_f)
            ks, ys = _decimal_cubic(t, n_f)
            n_pix += t.N
            for c in range(t.N):
                if k[c] != ks[c]:
                    n_mis += 1
                    assert abs(ys[c] - ys[c].to_integral_value()) < Decimal("1e-9"), (seed, tid, c)
            lo, hi = min(t.y0, t.y1, t.y2, t.y3), max(t.y0, t.y1, t.y2, t.y3)
            assert k.min() >= int(np.floor(lo)) and k.max() <= int(np.floor(hi))          # convex hull
    assert n_pix > 100000 and n_mis <= 2


def test_cubic_special_cases(orc):
    n_f = 961
    # degree elevation: the cubic with inner points (y0 + 2 y1) / 3, (2 y1 + y2) / 3 IS the quadratic's curve
    n_diff = 0
    for tid in range(300):
        q = orc.track_params(1, tid, 250, n_f, 10, 250)
        c = orc.make_track(q.N, q.j0, q.a, q.y0, (q.y0 + 2 * q.y1) / 3, (2 * q.y1 + q.y2) / 3, y3=q.y2)
        kq, kc = orc.rasterise(q, n_f), orc.rasterise(c, n_f)
        for col in np.flatnonzero(kq != kc):           # only where the exact curve grazes a bin edge
            n_diff += 1
            _, ys = _decimal_cubic(c, n_f)
            assert abs(ys[col] - ys[col].to_integral_value()) < Decimal("1e-9")
    assert n_diff <= 3
    # flat, and a straight line in (t, f): a = N / 2 with equally spaced control points
    assert (orc.rasterise(orc.make_track(77, 0, 30.0, 417.5, 417.5, 417.5, y3=417.5), n_f) == 417).all()
    N, y0, y3 = 200, 100.25, 700.75
    t = orc.make_track(N, 0, N / 2.0, y0, y0 + (y3 - y0) / 3, y0 + 2 * (y3 - y0) / 3, y3=y3)
    k = orc.rasterise(t, n_f)
    want = np.floor(y0 + (y3 - y0) * (np.arange(N) + 0.5) / N).astype(int)
    assert (np.abs(k - want) <= 0).mean() > 0.99 and np.abs(k - want).max() <= 1
    # end points and order of the control points: starts at y0, ends at y3; inner points pull in order
    t = orc.make_track(240, 3, 120.0, 100.5, 900.5, 100.5, y3=500.5)
    k = orc.rasterise(t, n_f)
    assert abs(k[0] - 100) <= 12 and abs(k[-1] - 500) <= 12
    assert k[:120].max() > k[120:200].min() + 50             # y1 (high) acts early, y2 (low) late: up, down, up
    t_swapped = orc.make_track(240, 3, 120.0, 100.5, 100.5, 900.5, y3=500.5)
    assert orc.rasterise(t_swapped, n_f)[:100].mean() < k[:100].mean() - 100
    # an S-shaped track (one inflection): impossible for a quadratic, the reason for the family
    s = orc.rasterise(orc.make_track(300, 0, 150.0, 100.5, 100.5, 800.5, y3=800.5), n_f)
    d2 = np.diff(s.astype(float), 2)
    assert d2[:100].mean() > 0 and d2[-100:].mean() < 0


def test_cubic_family_parameters(orc):
    """The cubic family keeps N, j0, a, y0, y1, y2, tau of the quadratic template with the same id (one more
    random number) and draws y3 uniform over the band, independent of the other seven."""
    n_t, n_f, T = 500, 2461, 30000
    q = [orc.track_params(2, i, n_t, n_f, 10, 500, -0.01, 0.01) for i in range(T)]
    c = [orc.track_params(2, i, n_t, n_f, 10, 500, -0.01, 0.01, family=orc.FAMILY_CUBIC) for i in range(T)]
    for a, b in zip(q[:2000], c[:2000]):
        assert (a.N, a.j0, a.a, a.y0, a.y1, a.y2, a.tau) == (b.N, b.j0, b.a, b.y0, b.y1, b.y2, b.tau)
        assert a.family == 0 and b.family == 1
    y3 = np.array([t.y3 for t in c])
    assert ((y3 > 0) & (y3 < n_f)).all()
    assert stats.kstest(y3 / n_f, "uniform").pvalue > 1e-6
    others = np.array([[t.N, t.j0, t.a / t.N, t.y0, t.y1, t.y2, t.tau] for t in c])
    for col in others.T:
        assert abs(np.corrcoef(col, y3)[0, 1]) < 5.0 / np.sqrt(T)
    with pytest.raises(ValueError):
        orc.track_params(2, 0, n_t, n_f, 10, 500, family=7)


def test_cubic_search_path(orc):
    """or_search with family 1: the dumped pixels are or_rasterise of the cubic templates, a cubic bank member
    injected noise-free is recovered exactly (P7 for the family), and the quadratic bank does not contain it."""
    cfg = synth.CONFIGS[1]
    taus = synth.tau_linspace(cfg.n_tau)
    f = cfg.f_min + cfg.df * np.arange(cfg.n_f)
    i_star, m_star = 311, 5
    t = orc.track_params(cfg.seed, i_star, cfg.n_t, cfg.n_f, 8, 64, family=orc.FAMILY_CUBIC)
    k = orc.rasterise(t, cfg.n_f)
    csd = np.zeros((cfg.n_t, cfg.n_f), dtype=np.complex64)
    j = t.j0 + np.arange(t.N)
    csd[j, k] = (2.0 * np.exp(-2j * np.pi * f[k] * taus[m_star])).astype(np.complex64)
    p = orc.prepare_map(csd)
    r = orc.search(p, cfg.f_min, cfg.df, 1000, cfg.seed, 8, 64, tau_grid=taus, family=orc.FAMILY_CUBIC, dump_tracks=True)
    assert (r["arg_track"], r["arg_tau_index"]) == (i_star, m_star)
    assert abs(r["max_snr"] - 2.0 * np.sqrt(t.N)) < 1e-5
    assert np.array_equal(r["k"][i_star, :t.N], k) and (r["k"][i_star, t.N:] == -1).all()
    rq = orc.search(p, cfg.f_min, cfg.df, 1000, cfg.seed, 8, 64, tau_grid=taus)
    assert rq["max_snr"] < r["max_snr"]


# ------------------------------------------------------------------------------------- O2k / O3k: chirp-law family (G27)
def _decimal_chirp(t, n_f):
    """y(u) = y0 (T_c / (T_c - u))^(3/8), T_c = N^2 / (N - a), in 60-digit arithmetic, written differently from the
    oracle (the power through ln / exp, T_c formed explicitly)."""
    getcontext().prec = 60
    N, a, y0 = Decimal(t.N), Decimal(t.a), Decimal(t.y0)
    t_c = N * N / (N - a)
    ks, ys = [], []
    for c in range(t.N):
        u = Decimal(c) + Decimal("0.5")
        y = y0 * ((t_c / (t_c - u)).ln() * Decimal(3) / Decimal(8)).exp()
        ys.append(y)
        ks.append(min(max(int(y.to_integral_value(rounding="ROUND_FLOOR")), 0), n_f - 1))
    return ks, ys


def test_chirp_rasteriser_vs_60_digit_brute_force(orc):
    n_pix = n_mis = 0
    for seed, n_t, n_f, n_min, n_max, count in ((4, 1000, 2461, 10, 1000, 60), (1, 250, 961, 10, 250, 150), (0, 64, 64, 64, 64, 100)):
        for tid in range(count):
            t = orc.track_params(seed, tid, n_t, n_f, n_min, n_max, family=orc.FAMILY_CHIRP)
            assert t.family == 2
            k = orc.rasterise(t, n_f)
            ks, ys = _decimal_chirp(t, n_f)
            n_pix += t.N
            for c in range(t.N):
                if k[c] != ks[c]:
                    n_mis += 1
                    assert abs(ys[c] - ys[c].to_integral_value()) < Decimal("1e-9"), (seed, tid, c)
            assert (np.diff(k) >= 0).all() and k[0] >= int(np.floor(t.y0))          # an up-chirp from y0
    assert n_pix > 40000 and n_mis <= 2


def test_chirp_law_closed_forms(orc):
    """f^(-8/3) is linear in time (the chirp law); at a = N / 256 the frequency at the END of the track
    is 256^(3/8) = 8 times the start; the band clamp; T_c -> infinity (a -> N) is a flat track."""
    n_f = 4096
    N, y0 = 400, 100.5
    t = orc.make_track(N, 7, N / 256.0, y0, 0.0, 0.0, family=orc.FAMILY_CHIRP)
    k = orc.rasterise(t, n_f)
    _, ys = _decimal_chirp(t, n_f)
    u = np.arange(N) + 0.5
    t_c = N * N / (N - t.a)
    lin = np.array([float((y / Decimal(y0)) ** (Decimal(-8) / Decimal(3))) for y in ys])
    assert np.allclose(lin, 1.0 - u / t_c, rtol=0, atol=1e-12)
    # end of the track: u = N gives (T_c - N) / T_c = a / N = 1 / 256, so f = 8 y0; the last column centre is half a
    # column earlier: f = y0 (T_c / (T_c - N + 1/2))^(3/8)
    want_last = y0 * (t_c / (t_c - N + 0.5)) ** 0.375
    assert k[-1] == int(np.floor(want_last)) and abs(want_last / y0 - 8.0) < 0.8
    assert k[0] == int(np.floor(y0 * (t_c / (t_c - 0.5)) ** 0.375))
    # leaving the band: the pixels ride the top bin (clamp), as for the Bezier families
    hot = orc.rasterise(orc.make_track(300, 0, 300 / 256.0, 900.0, 0.0, 0.0, family=orc.FAMILY_CHIRP), 2461)
    assert hot.max() == 2460 and (np.diff(hot) >= 0).all() and (hot == 2460).sum() > 3
    # a -> N: T_c -> infinity, the track is flat at y0
    flat = orc.rasterise(orc.make_track(200, 0, 200 - 1e-9, 333.5, 0.0, 0.0, family=orc.FAMILY_CHIRP), n_f)
    assert (flat == 333).all()


def test_chirp_family_parameters_and_search_path(orc):
    """N, j0, a, y0, tau are those of the quadratic template with the same id; or_search with family 2 dumps
    or_rasterise's pixels and recovers a noise-free injected bank member exactly (P7 for the family)."""
    n_t, n_f = 500, 2461
    for i in range(500):
        q = orc.track_params(2, i, n_t, n_f, 10, 500, -0.01, 0.01)
        c = orc.track_params(2, i, n_t, n_f, 10, 500, -0.01, 0.01, family=orc.FAMILY_CHIRP)
        assert (q.N, q.j0, q.a, q.y0, q.tau) == (c.N, c.j0, c.a, c.y0, c.tau) and c.family == 2
    cfg = synth.CONFIGS[1]
    taus = synth.tau_linspace(cfg.n_tau)
    f = cfg.f_min + cfg.df * np.arange(cfg.n_f)
    i_star, m_star = 127, 9
    t = orc.track_params(cfg.seed, i_star, cfg.n_t, cfg.n_f, 8, 64, family=orc.FAMILY_CHIRP)
    k = orc.rasterise(t, cfg.n_f)
    csd = np.zeros((cfg.n_t, cfg.n_f), dtype=np.complex64)
    j = t.j0 + np.arange(t.N)
    csd[j, k] = (2.0 * np.exp(-2j * np.pi * f[k] * taus[m_star])).astype(np.complex64)
    p = orc.prepare_map(csd)
    r = orc.search(p, cfg.f_min, cfg.df, 1000, cfg.seed, 8, 64, tau_grid=taus, family=orc.FAMILY_CHIRP, dump_tracks=True)
    assert (r["arg_track"], r["arg_tau_index"]) == (i_star, m_star)
    assert abs(r["max_snr"] - 2.0 * np.sqrt(t.N)) < 1e-5
    assert np.array_equal(r["k"][i_star, :t.N], k) and (r["k"][i_star, t.N:] == -1).all()

"""Pins of the float64 CPU oracle against what the paper and the mathematics fix
(SURVEY.md 8(c) P1-P10).  None of these tests touches the CUDA path.

Each pin is chosen so that a plausible mistake in the oracle (a dropped term, a
wrong sign or index, a transposed operand, a stray factor of 2 or pi) fails it.
"""
import os
import shutil
import subprocess
from decimal import Decimal, getcontext
from fractions import Fraction

import numpy as np
import pytest

from workloads import synth

HERE = os.path.dirname(os.path.abspath(__file__))


def golden():
    out = {}
    with open(os.path.join(HERE, "golden", "paper_printed_numbers.txt")) as f:
        for line in f:
            line = line.split("#")[0].split()
            if len(line) >= 2:
                out[line[0]] = float(line[1])
    return out


# ----------------------------------------------------------------------------- P1
def _curand_words(seed, offset, n, tmp):
    exe = os.path.join(tmp, "curand_host_philox")
    if not os.path.exists(exe):
        inc, libdir = "/usr/local/cuda/include", "/usr/local/cuda/lib64"
        if shutil.which("gcc") is None or not os.path.exists(os.path.join(libdir, "libcurand.so")):
            pytest.skip("cuRAND host library not available")
        subprocess.check_call(["gcc", os.path.join(HERE, "curand_host_philox.c"), "-I" + inc,
                               "-L" + libdir, "-lcurand", "-Wl,-rpath," + libdir, "-o", exe])
    txt = subprocess.check_output([exe, hex(seed), hex(offset), str(n)]).decode().split()
    return np.array([int(x, 16) for x in txt], dtype=np.uint32)


def test_P1_philox_matches_curand_host_generator(orc, tmp_path_factory):
    """P1: or_philox4x32_10 == NVIDIA cuRAND's CPU-side PHILOX4_32_10 generator.

    The host generator emits block b = (offset/4 + i/4) from the counter
    (b >> 16 [lo, hi], b & 0xffff, 0) with key = (seed_lo, seed_hi) -- found by
    inspection; any error in the round function, the multipliers, the Weyl key
    schedule, or the word order makes every word disagree.
    """
    tmp = str(tmp_path_factory.mktemp("curand"))
    cases = [(0x0, 0, 64), (0x0123456789ABCDEF, 0, 4 * 70000), (7, 0x500000010, 256),
             (0xFEDCBA9876543210, 0xFFFFFFFFFFF00000, 256), (0xFFFFFFFFFFFFFFFF, 4 * 65535, 64)]
    for seed, offset, n in cases:
        ref = _curand_words(seed, offset, n, tmp).reshape(-1, 4)
        key = [seed & 0xFFFFFFFF, seed >> 32]
        # check every block for short cases, a spread of blocks for the long one
        idx = range(ref.shape[0]) if ref.shape[0] <= 64 else list(range(0, 64)) + \
            list(range(65530, 65542)) + list(range(69990, 70000))
        for i in idx:
            b = offset // 4 + i
            hi = b >> 16
            ctr = [hi & 0xFFFFFFFF, (hi >> 32) & 0xFFFFFFFF, b & 0xFFFF, 0]
            got = orc.philox4x32_10(ctr, key)
            assert np.array_equal(got, ref[i]), (hex(seed), hex(offset), i, ctr)


def test_P1_counter_words_all_matter(orc):
    """The fourth counter word cannot be reached through cuRAND's host API: check
    that it and every other input bit changes the output (no dropped operand)."""
    base = orc.philox4x32_10([1, 2, 3, 4], [5, 6])
    for w in range(4):
        c = [1, 2, 3, 4]
        c[w] ^= 1 << 17
        assert not np.array_equal(orc.philox4x32_10(c, [5, 6]), base)
    assert not np.array_equal(orc.philox4x32_10([1, 2, 3, 4], [5 ^ 1, 6]), base)
    assert not np.array_equal(orc.philox4x32_10([1, 2, 3, 4], [5, 6 ^ 1]), base)


def test_track_words_layout(orc):
    """O1: words r0..r3 come from counter (id_lo, id_hi, 0, tag), r4..r7 from b = 1."""
    seed, tid = 0x1122334455667788, 0x0000000A00000003
    r = orc.track_words(seed, tid)
    tag = 0x5354524B
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for b in (0, 1):
        want = orc.philox4x32_10([tid & 0xFFFFFFFF, tid >> 32, b, tag], key)
        assert np.array_equal(r[4 * b:4 * b + 4], want)


# ----------------------------------------------------------------------------- O2
def test_track_params_exact_rational(orc):
    """O2: the word -> parameter maps evaluated in exact rational arithmetic agree
    bit for bit with the double results (the products are claimed exact)."""
    n_t, n_f, n_min, n_max = 1000, 2461, 10, 1000
    for tid in list(range(200)) + [2 ** 40 + 17, 2 ** 63]:
        r = [int(x) for x in orc.track_words(4, tid)]
        t = orc.track_params(4, tid, n_t, n_f, n_min, n_max, -0.01, 0.01)
        N = n_min + (r[0] * (n_max - n_min + 1) >> 32)
        j0 = r[1] * (n_t - N + 1) >> 32
        assert (t.N, t.j0) == (N, j0)
        assert Fraction(t.a) == Fraction(2 * r[2] + 1, 2) * N / 2 ** 32
        for q, y in enumerate((t.y0, t.y1, t.y2)):
            assert Fraction(y) == Fraction(2 * r[3 + q] + 1, 2) * n_f / 2 ** 32
        u = (r[6] + 0.5) / 2 ** 32
        assert t.tau == -0.01 + (0.01 - (-0.01)) * u
        assert 0 < t.a < t.N and 0 <= t.j0 <= n_t - t.N and -0.01 < t.tau < 0.01


def test_track_params_distributions(orc):
    """G3/G4: N uniform on [n_min, n_max]; start uniform among feasible columns;
    t_mid strictly inside; f control points uniform over the band."""
    n_t, n_f, n_min, n_max, T = 500, 2461, 10, 500, 40000
    ts = [orc.track_params(2, i, n_t, n_f, n_min, n_max, -0.01, 0.01) for i in range(T)]
    N = np.array([t.N for t in ts]); j0 = np.array([t.j0 for t in ts])
    a = np.array([t.a for t in ts]); y = np.array([[t.y0, t.y1, t.y2] for t in ts])
    tau = np.array([t.tau for t in ts])
    assert N.min() >= n_min and N.max() <= n_max and (j0 >= 0).all() and (j0 + N <= n_t).all()
    assert abs(N.mean() - 255) < 3 * 141.7 / np.sqrt(T)
    assert ((a > 0) & (a < N)).all() and abs((a / N).mean() - 0.5) < 4 * 0.2887 / np.sqrt(T)
    assert ((y > 0) & (y < n_f)).all()
    assert np.abs(y.mean(axis=0) / n_f - 0.5).max() < 4 * 0.2887 / np.sqrt(T)
    assert abs(np.corrcoef(y[:, 0], y[:, 2])[0, 1]) < 0.03
    assert abs(tau.mean()) < 4 * 0.02 * 0.2887 / np.sqrt(T) and np.abs(tau).max() < 0.01
    # full-duration special case of config 1: n_min = n_max = n_t  =>  j0 = 0
    t = orc.track_params(0, 3, 64, 64, 64, 64)
    assert (t.N, t.j0) == (64, 0)
    with pytest.raises(ValueError):
        orc.track_params(0, 0, 64, 64, 10, 65)


# ----------------------------------------------------------------------------- P2
def _decimal_raster(t, n_f):
    """Independent 60-digit evaluation of Eq. 6 at column centres, with
    the TEXTBOOK quadratic formula (not the oracle's rearranged root)."""
    getcontext().prec = 60
    a, N = Decimal(t.a), Decimal(t.N)
    y0, y1, y2 = Decimal(t.y0), Decimal(t.y1), Decimal(t.y2)
    A, B = N - 2 * a, 2 * a          # t(xi) - j0 = A xi^2 + B xi
    ks, ys = [], []
    for c in range(t.N):
        u = Decimal(c) + Decimal("0.5")
        if A == 0:
            xi = u / B
        else:
            xi = (-B + (B * B + 4 * A * u).sqrt()) / (2 * A)
        assert 0 < xi < 1
        y = (1 - xi) ** 2 * y0 + 2 * (1 - xi) * xi * y1 + xi ** 2 * y2
        ys.append(y)
        ks.append(min(max(int(y.to_integral_value(rounding="ROUND_FLOOR")), 0), n_f - 1))
    return ks, ys


def test_P2_rasteriser_vs_60_digit_brute_force(orc):
    cases = [(0, i, 64, 64, 64, 64) for i in range(300)]                  # config 1 shape
    cases += [(4, i, 1000, 2461, 10, 1000) for i in range(250)]            # config 5 shape
    cases += [(1, i, 250, 961, 10, 250) for i in range(300)]               # config 2 shape
    n_pix = n_mis = 0
    for seed, tid, n_t, n_f, n_min, n_max in cases:
        t = orc.track_params(seed, tid, n_t, n_f, n_min, n_max)
        k = orc.rasterise(t, n_f)
        ks, ys = _decimal_raster(t, n_f)
        n_pix += t.N
        for c in range(t.N):
            if k[c] != ks[c]:
                n_mis += 1
                # only allowed when the exact curve passes within 1e-9 of a bin edge
                assert abs(ys[c] - ys[c].to_integral_value()) < Decimal("1e-9"), (seed, tid, c)
        lo, hi = min(t.y0, t.y1, t.y2), max(t.y0, t.y1, t.y2)
        assert k.min() >= int(np.floor(lo)) and k.max() <= int(np.floor(hi))   # convex hull
    assert n_pix > 150000 and n_mis <= 2


def test_P2_rasteriser_special_cases(orc):
    n_f = 961
    # a = N/2: linear time, xi = u/N; with y1 the midpoint the track is a straight line
    for N, y0, y2 in [(200, 700.25, 180.75), (37, 3.125, 950.5), (250, 10.0, 10.0)]:
        t = orc.make_track(N, 5, N / 2.0, y0, 0.5 * (y0 + y2), y2)
        k = orc.rasterise(t, n_f)
        for c in range(N):
            y = Fraction(y0) + (Fraction(y2) - Fraction(y0)) * Fraction(2 * c + 1, 2 * N)
            if abs(y - round(y)) > Fraction(1, 10 ** 9):
                assert k[c] == y.__floor__(), (N, c)
    # flat track
    t = orc.make_track(123, 0, 17.3, 417.5, 417.5, 417.5)
    assert (orc.rasterise(t, n_f) == 417).all()
    # endpoints: first/last pixel within one column's worth of slope of f_start/f_end;
    # a transposed (y0 <-> y2) or reversed curve fails this
    t = orc.make_track(240, 3, 77.7, 100.5, 500.5, 900.5)
    k = orc.rasterise(t, n_f)
    assert abs(k[0] - 100) <= 8 and abs(k[-1] - 900) <= 8 and (np.diff(k) >= 0).all()
    # t_mid early => the curve spends most columns near the end frequency (time-warp sign)
    t_early = orc.make_track(240, 3, 24.0, 100.5, 500.5, 900.5)
    t_late = orc.make_track(240, 3, 216.0, 100.5, 500.5, 900.5)
    assert orc.rasterise(t_early, n_f).mean() > k.mean() > orc.rasterise(t_late, n_f).mean()
    # clamp: control points at the band edges never leave [0, n_f)
    t = orc.make_track(50, 0, 25.0, 960.9999999, 960.9999999, 0.0000001)
    k = orc.rasterise(t, n_f)
    assert k.max() == 960 and k.min() >= 0
    # out-of-band control points (never produced by O2) are clamped into [0, n_f)
    k = orc.rasterise(orc.make_track(50, 0, 25.0, 1200.0, 400.0, -300.0), n_f)
    assert k[0] == 960 and k[-1] == 0 and k.min() == 0 and k.max() == 960


# ----------------------------------------------------------------------------- P3
def _tiny(orc, seed=11, n_t=24, n_f=20, sigma_kind="per_pixel"):
    csd = synth.noise_csd(n_t, n_f, seed)
    sigma = synth.make_sigma(sigma_kind, 0.3, n_t, n_f, seed)
    return csd, sigma, orc.prepare_map(csd, sigma)


def _numpy_score(p, j0, k, f_min, df, taus, alpha):
    """Second implementation: Eq. 1 builds the rotated REAL map rho for a
    fixed delay, Eq. 5 sums it over Gamma -- must equal Eq. 8."""
    n_t, n_f = p.shape
    f = f_min + df * np.arange(n_f)
    out = []
    for tau in taus:
        rho = np.real(np.exp(2j * np.pi * f[None, :] * tau) * p)     # full real map, Eq. 1
        j = j0 + np.arange(len(k))
        out.append(rho[j, k].sum() / len(k) ** alpha)                # Eq. 5
    return np.array(out)


def test_P3_eq8_equals_eq5_on_eq1_maps(orc):
    f_min, df = 40.0, 1.0
    csd, sigma, p = _tiny(orc)
    # prepare_map itself: p = CSD / sigma (Eq. 7)
    assert np.allclose(p, csd.astype(np.complex128) / sigma.astype(np.float64), rtol=1e-15)
    taus = synth.tau_linspace(7)
    W = orc.build_table(p.shape[1], f_min, df, taus)
    for tid in range(40):
        t = orc.track_params(9, tid, p.shape[0], p.shape[1], 3, p.shape[0])
        k = orc.rasterise(t, p.shape[1])
        for norm, alpha in ((orc.NORM_SQRT_N, 0.5), (orc.NORM_MEAN, 1.0)):
            ref = _numpy_score(p, t.j0, k, f_min, df, taus, alpha)
            direct = np.array([orc.score_direct(p, t, k, f_min, df, tau, norm) for tau in taus])
            table = orc.score_table(p, t, k, W, norm)
            assert np.allclose(direct, ref, rtol=0, atol=1e-12)
            assert np.array_equal(table, direct)          # same expression, same order


def test_P3_sigma_kinds_and_mask(orc):
    n_t, n_f = 6, 5
    csd = synth.noise_csd(n_t, n_f, 3)
    s_f = np.array([1.0, 2.0, 0.0, -1.0, np.inf], dtype=np.float32)
    p = orc.prepare_map(csd, s_f)
    assert np.allclose(p[:, 1], csd[:, 1].astype(np.complex128) / 2.0)
    assert (p[:, 2:] == 0).all()                         # sigma <= 0 or non-finite masks (G11)
    s_p = np.full((n_t, n_f), 4.0, dtype=np.float32); s_p[2, 3] = np.nan
    p = orc.prepare_map(csd, s_p)
    assert p[2, 3] == 0 and np.allclose(p[0, 0], complex(csd[0, 0]) / 4.0)
    assert np.array_equal(orc.prepare_map(csd, None), csd.astype(np.complex128))


# ----------------------------------------------------------------------------- P4
def test_P4_tau_zero_is_real_cross_power_sum(orc):
    csd, sigma, p = _tiny(orc, seed=5)
    for tid in range(20):
        t = orc.track_params(1, tid, p.shape[0], p.shape[1], 2, p.shape[0])
        k = orc.rasterise(t, p.shape[1])
        s = p.real[t.j0 + np.arange(t.N), k].sum()
        assert abs(orc.score_direct(p, t, k, 40.0, 1.0, 0.0, orc.NORM_SQRT_N) - s / np.sqrt(t.N)) < 1e-13
        assert abs(orc.score_direct(p, t, k, 40.0, 1.0, 0.0, orc.NORM_MEAN) - s / t.N) < 1e-13


# ----------------------------------------------------------------------------- P5
def _flat_injection(orc, n_t, n_f, kbin, f_min, df, tau0, amp):
    p = np.zeros((n_t, n_f), dtype=np.complex128)
    f = f_min + kbin * df
    p[:, kbin] = amp * np.exp(-2j * np.pi * f * tau0)      # G7: source delay tau0
    t = orc.make_track(n_t, 0, n_t / 2.0, kbin + 0.5, kbin + 0.5, kbin + 0.5)
    k = orc.rasterise(t, n_f)
    assert (k == kbin).all()
    return p, t, k


def test_P5_flat_track_cosine_eq3(orc):
    """Eq. 3: R = cos(2 pi f dtau); zero at |dtau| = 1/(4f)."""
    n_t, n_f, f_min, df, tau0, amp = 32, 64, 40.0, 1.0, 2.5e-3, 3.0
    for kbin in (0, 17, 60):
        f = f_min + kbin * df
        p, t, k = _flat_injection(orc, n_t, n_f, kbin, f_min, df, tau0, amp)
        snr0 = orc.score_direct(p, t, k, f_min, df, tau0, orc.NORM_SQRT_N)
        assert abs(snr0 - amp * np.sqrt(n_t)) < 1e-12          # analytic SNR, A * N^(1-alpha)
        assert abs(orc.score_direct(p, t, k, f_min, df, tau0, orc.NORM_MEAN) - amp) < 1e-12
        for tau in np.linspace(-0.01, 0.01, 41):
            want = snr0 * np.cos(2 * np.pi * f * (tau - tau0))
            assert abs(orc.score_direct(p, t, k, f_min, df, tau, orc.NORM_SQRT_N) - want) < 1e-11
        for sgn in (-1, 1):
            assert abs(orc.score_direct(p, t, k, f_min, df, tau0 + sgn / (4 * f), 0)) < 1e-11
        # sign convention: +tau0 recovers, -tau0 does not (unless cos happens to match)
        assert orc.score_direct(p, t, k, f_min, df, -tau0, 0) < snr0 - 1e-3


def test_P5_paper_printed_timing_tolerances(orc):
    """Eq. 4 / PAPER.md:60: R >= 90 % needs dtau <= 720 us at 100 Hz, <= 72 us at 1 kHz."""
    g = golden()
    for f, dt_us in ((g["eq4_f_low"], g["eq4_dtau_low"]), (g["eq4_f_high"], g["eq4_dtau_high"])):
        f_min, df = f - 3.0, 1.0
        p, t, k = _flat_injection(orc, 16, 8, 3, f_min, df, 0.0, 1.0)
        r = orc.score_direct(p, t, k, f_min, df, dt_us * 1e-6, 0) / orc.score_direct(p, t, k, f_min, df, 0.0, 0)
        assert abs(r - g["eq4_R"]) < 2e-3           # printed to two digits: 720 vs 717.8
        # a stray factor of 2 (or 1/2) in the phase would give R = 0.62 (or 0.97)


def test_P5_stripe_bandwidth(orc):
    """a timing error dtau makes stripes of bandwidth 1/(4 dtau): from a
    stripe centre (|R| = 1) to its edge (R = 0) is 1/(4 dtau) = 25 Hz at 10 ms."""
    g = golden()
    dtau = g["stripe_dtau_max"] * 1e-3
    dfs = g["stripe_df_min"]
    assert abs(1.0 / (4 * dtau) - dfs) < 1e-9
    f_min, df, n_f = 100.0, 1.0, 64                   # f = 100 Hz: 2 pi f dtau = 2 pi => R = 1
    vals = []
    for kbin in (0, int(dfs), int(2 * dfs)):
        p, t, k = _flat_injection(orc, 16, n_f, kbin, f_min, df, 0.0, 1.0)
        vals.append(orc.score_direct(p, t, k, f_min, df, dtau, orc.NORM_MEAN))
    assert abs(vals[0] - 1.0) < 1e-9 and abs(vals[1]) < 1e-9 and abs(vals[2] + 1.0) < 1e-9


# ----------------------------------------------------------------------------- P6
def test_P6_invariants(orc):
    f_min, df = 40.0, 1.0
    csd, sigma, p = _tiny(orc, seed=21, n_t=40, n_f=33)
    n_t, n_f = p.shape
    f = f_min + df * np.arange(n_f)
    taus = synth.tau_linspace(9)
    step = taus[1] - taus[0]
    for tid in range(12):
        t = orc.track_params(6, tid, n_t, n_f, 4, n_t)
        k = orc.rasterise(t, n_f)
        sc = lambda pp, tt: np.array([orc.score_direct(pp, t, k, f_min, df, x, 0) for x in tt])
        base = sc(p, taus)
        # periodicity: all f integer multiples of 1 Hz => period 1 s
        assert np.allclose(sc(p, taus + 1.0), base, atol=1e-9, rtol=0)
        # global rotation by pi/2: Re[i Z] = -Im Z
        im = np.array([(np.exp(2j * np.pi * f[k] * x) * p[t.j0 + np.arange(t.N), k]).imag.sum()
                       / np.sqrt(t.N) for x in taus])
        assert np.allclose(sc(1j * p, taus), -im, atol=1e-12, rtol=0)
        # general rotation and linearity
        th = 0.7
        assert np.allclose(sc(np.exp(1j * th) * p, taus), np.cos(th) * base - np.sin(th) * im, atol=1e-12)
        assert np.allclose(sc(2.5 * p + 1j * p, taus), 2.5 * base - im, atol=1e-12)
        # delay shift by two grid steps: SNR(tau) -> SNR(tau - tau1)
        tau1 = 2 * step
        shifted = sc(p * np.exp(-2j * np.pi * f[None, :] * tau1), taus)
        assert np.allclose(shifted[2:], base[:-2], atol=1e-11, rtol=0)
        # conjugation: p -> p*, tau -> -tau
        assert np.allclose(sc(np.conj(p), -taus), base, atol=1e-12, rtol=0)


# ------------------------------------------------------------------------ P7 - P10
def test_P7_injected_track_self_recovery(orc):
    cfg = synth.CONFIGS[1]
    taus = synth.tau_linspace(cfg.n_tau)
    f = cfg.f_min + cfg.df * np.arange(cfg.n_f)
    for norm, expo in ((orc.NORM_SQRT_N, 0.5), (orc.NORM_MEAN, 0.0)):
        for i_star, m_star, n_min, n_max in ((137, 11, 64, 64), (402, 0, 5, 64), (7, 15, 5, 64)):
            t = orc.track_params(cfg.seed, i_star, cfg.n_t, cfg.n_f, n_min, n_max)
            k = orc.rasterise(t, cfg.n_f)
            sigma = synth.make_sigma("per_pixel", 0.3, cfg.n_t, cfg.n_f, 5)
            csd = np.zeros((cfg.n_t, cfg.n_f), dtype=np.complex64)
            j = t.j0 + np.arange(t.N)
            A = 2.0
            csd[j, k] = (A * sigma[j, k] * np.exp(-2j * np.pi * f[k] * taus[m_star])).astype(np.complex64)
            p = orc.prepare_map(csd, sigma)
            r = orc.search(p, cfg.f_min, cfg.df, 1000, cfg.seed, n_min, n_max, tau_grid=taus, norm=norm)
            assert (r["arg_track"], r["arg_tau_index"]) == (i_star, m_star)
            assert r["arg_tau"] == taus[m_star]
            assert abs(r["max_snr"] - A * t.N ** expo) < 1e-5 * A * t.N ** expo   # complex64 inputs
            t2 = orc.track_params(cfg.seed, r["arg_track"], cfg.n_t, cfg.n_f, n_min, n_max)
            assert t2.as_dict() == t.as_dict()


def test_P8_null_distribution_unit_variance(orc):
    """A1-A3: rho = Y/sigma has unit variance when sigma^2 =
    (1/2) P_I P_J; with E|s|^2 = 1 that is sigma = 2^-1/2 (G10)."""
    n_t, n_f = 250, 961
    csd = synth.noise_csd(n_t, n_f, 77)
    sig = np.full(n_f, np.sqrt(0.5), dtype=np.float32)
    p = orc.prepare_map(csd, sig)
    assert abs(p.real.var() - 1.0) < 0.02 and abs(p.imag.var() - 1.0) < 0.02
    T = 60000
    r = orc.search(p, 40.0, 1.0, T, 5, 10, 250, tau_grid=np.array([1.7e-3]), dump_snr=True,
                   dump_tracks=True, n_bins=1000)
    s = r["snr"][:, 0]
    assert abs(s.mean()) < 0.03 and abs(s.var() - 1.0) < 0.04
    r1 = orc.search(p, 40.0, 1.0, T, 5, 10, 250, tau_grid=np.array([1.7e-3]), dump_snr=True,
                    norm=orc.NORM_MEAN)
    # Eq. 8 as printed (1/N): a mean, variance 1/N per duration class
    s1 = r1["snr"][:, 0]
    assert np.allclose(s1 * np.sqrt(r["N"]), s, rtol=1e-12, atol=1e-12)
    for lo, hi in ((10, 40), (100, 140), (200, 250)):
        sel = (r["N"] >= lo) & (r["N"] <= hi)
        assert abs((s1[sel] ** 2 * r["N"][sel]).mean() - 1.0) < 0.06
    # P10: histogram counts every (track, tau) sample
    assert int(r["hist"].sum()) == T
    # unnormalised sigma = 1: variance 1/2 (G10)
    p1 = orc.prepare_map(csd, None)
    r2 = orc.search(p1, 40.0, 1.0, 20000, 5, 10, 250, tau_grid=np.array([0.0]), dump_snr=True)
    assert abs(r2["snr"].var() - 0.5) < 0.03


def test_P9_P10_chunk_combination_and_histogram(orc):
    """three runs combined by max are 'identical' to one 3x run."""
    cfg = synth.CONFIGS[1]
    csd, sigma, taus = synth.config_inputs(cfg)
    p = orc.prepare_map(csd, sigma)
    kw = dict(tau_grid=taus, n_bins=200, hist_lo=-4.0, hist_hi=4.0)
    full = orc.search(p, cfg.f_min, cfg.df, 900, 0, 8, 64, dump_snr=True, **kw)
    parts = [orc.search(p, cfg.f_min, cfg.df, 300, 0, 8, 64, track_offset=300 * i, **kw) for i in range(3)]
    best = max(parts, key=lambda r: (r["max_snr"], -r["arg_track"], -r["arg_tau_index"]))
    assert (best["max_snr"], best["arg_track"], best["arg_tau_index"]) == \
        (full["max_snr"], full["arg_track"], full["arg_tau_index"])
    assert np.array_equal(sum(r["hist"] for r in parts), full["hist"])
    assert int(full["hist"].sum()) == 900 * cfg.n_tau and full["n_evals"] == full["n_pixels"] * cfg.n_tau
    # O5 against NumPy on the dump: argmax with the (larger SNR, smaller id, smaller m) order
    snr = full["snr"]
    i, m = np.unravel_index(np.argmax(snr), snr.shape)       # first occurrence = smallest (i, m)
    assert (full["arg_track"], full["arg_tau_index"], full["max_snr"]) == (i, m, snr[i, m])
    edges = np.floor((snr - (-4.0)) / 8.0 * 200).clip(0, 199).astype(int)
    assert np.array_equal(np.bincount(edges.ravel(), minlength=200), full["hist"])
    # thread count / schedule independence
    one = orc.search(p, cfg.f_min, cfg.df, 900, 0, 8, 64, n_threads=1, dump_snr=True, **kw)
    assert np.array_equal(one["snr"], snr) and np.array_equal(one["hist"], full["hist"])
    # direct (cos/sin per eval) and table scoring agree exactly
    dire = orc.search(p, cfg.f_min, cfg.df, 900, 0, 8, 64, score_mode=1, dump_snr=True, **kw)
    assert np.array_equal(dire["snr"], snr)


def test_histogram_bins_by_their_definition(orc):
    """G14 pinned by what a histogram IS, not by re-typing the oracle's floor formula: bin i counts the samples with
    lo + i w <= SNR < lo + (i + 1) w (explicit edges, np.searchsorted on the oracle's own SNR dump), samples below lo
    go to bin 0 and samples at or above hi to the last bin.  A range narrower than the data exercises both clamps, a
    width that is not a power of two keeps the edges off round numbers.  Then constructed maps whose every SNR is one
    exactly known value -- a constant real map at tau = 0 under the mean normalisation scores exactly that constant --
    put samples ON edges, just inside bins and outside the range: a round-to-nearest, a ceil, an open-left edge or a
    dropped clamp each fail here."""
    cfg = synth.CONFIGS[1]
    csd, sigma, taus = synth.config_inputs(cfg)
    p = orc.prepare_map(csd, sigma)
    lo, hi, nb = -1.0, 1.5, 37
    r = orc.search(p, cfg.f_min, cfg.df, 700, 5, 8, 64, tau_grid=taus, n_bins=nb, hist_lo=lo, hist_hi=hi, dump_snr=True)
    snr = np.sort(r["snr"].ravel())
    assert snr[0] < lo - 0.2 and snr[-1] > hi + 0.2            # both clamps are exercised
    edges = lo + (hi - lo) * np.arange(nb + 1) / nb
    near = np.abs(snr[:, None] - edges[None, :]).min(axis=1) < 1e-12
    assert near.sum() == 0                                      # no sample sits on an edge of this seeded case
    cum = np.searchsorted(snr, edges, side="left")              # samples strictly below each edge
    want = np.diff(cum).astype(np.int64)
    want[0] += cum[0]                                           # below lo -> first bin
    want[-1] += snr.size - cum[-1]                              # at or above hi -> last bin
    assert np.array_equal(r["hist"], want) and int(r["hist"].sum()) == 700 * cfg.n_tau
    # samples of exactly known value: constant map, tau = 0, alpha = 1 -> SNR = c for every template
    lo, hi, nb = -4.0, 4.0, 64
    w = (hi - lo) / nb                                          # 0.125: edges and the values below are exact in binary
    eps = 2.0 ** -20                                            # dyadic: sums of up to 64 copies stay exact
    cases = [(0.0, 32), (w, 33), (-w, 31), (0.5 * w, 32), (0.75 * w, 32), (0.9375 * w, 32), (-0.25 * w, 31), (-0.75 * w, 31),
             (lo, 0), (lo + 0.5 * w, 0), (hi - w, 63), (hi - 0.5 * w, 63), (hi, 63), (100.0, 63), (-100.0, 0),
             (lo - eps, 0), (w - eps, 32), (-w - eps, 30), (hi - eps, 63), (3 * w + eps, 35)]
    for c, want_bin in cases:
        flat = np.full((cfg.n_t, cfg.n_f), c, dtype=np.complex128)
        z = orc.search(flat, cfg.f_min, cfg.df, 20, 1, 8, 64, tau_grid=np.zeros(1), norm=orc.NORM_MEAN, n_bins=nb, hist_lo=lo,
                       hist_hi=hi, dump_snr=True)
        assert (z["snr"] == c).all(), c
        expect = np.zeros(nb, dtype=np.int64)
        expect[want_bin] = 20
        assert np.array_equal(z["hist"], expect), (c, want_bin, np.flatnonzero(z["hist"]))


def test_random_tau_mode_uses_track_delay(orc):
    """each template carries its own random delay."""
    cfg = synth.CONFIGS[1]
    csd, sigma, _ = synth.config_inputs(cfg)
    p = orc.prepare_map(csd, sigma)
    r = orc.search(p, cfg.f_min, cfg.df, 200, 3, 8, 64, tau_range=(-0.01, 0.01), dump_snr=True, dump_tracks=True)
    for i in (0, 57, 199):
        t = orc.track_params(3, i, cfg.n_t, cfg.n_f, 8, 64, -0.01, 0.01)
        k = orc.rasterise(t, cfg.n_f)
        assert np.array_equal(r["k"][i, :t.N], k) and (r["k"][i, t.N:] == -1).all()
        assert r["snr"][i, 0] == orc.score_direct(p, t, k, cfg.f_min, cfg.df, t.tau, 0)
    i = int(np.argmax(r["snr"][:, 0]))
    assert r["arg_track"] == i and r["arg_tau"] == orc.track_params(3, i, cfg.n_t, cfg.n_f, 8, 64, -0.01, 0.01).tau


def test_top_k_is_the_sorted_head_of_all_samples(orc):
    """oracle.top_k against brute force on a tiny search (explicit Python sort of every sample), ties
    included: an all-zero map makes every SNR equal, so the order is by template id, then delay index."""
    cfg = synth.CONFIGS[1]
    csd, sigma, tau = synth.config_inputs(cfg)
    r = orc.search(orc.prepare_map(csd, sigma), cfg.f_min, cfg.df, 60, 3, cfg.n_min, cfg.n_max, tau_grid=tau, dump_snr=True)
    brute = sorted(((-r["snr"][i, m], i, m) for i in range(60) for m in range(cfg.n_tau)))[:25]
    assert orc.top_k(r, 25) == [(i, m, -s) for s, i, m in brute]
    assert orc.top_k(r, 1)[0][:2] == (r["arg_track"], r["arg_tau_index"])
    z = orc.search(np.zeros((cfg.n_t, cfg.n_f), dtype=np.complex128), cfg.f_min, cfg.df, 5, 3, cfg.n_min, cfg.n_max,
                   tau_grid=tau[:3], dump_snr=True)
    assert [e[:2] for e in orc.top_k(z, 5)] == [(0, 0), (0, 1), (0, 2), (1, 0), (1, 1)]


def test_oracle_is_clean_under_address_and_undefined_behaviour_sanitizers(tmp_path):
    """The C oracle built with -fsanitize=address,undefined (any finding aborts) runs its whole path --
    table, direct and random-delay scoring, per-pixel sigma with masked pixels, histogram, dumps, a track
    offset beyond 2^32 -- and the table and direct modes agree to the last digit printed."""
    import subprocess
    exe = tmp_path / "or_san"
    src = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_sanitizer_driver.c")
    subprocess.check_call(["gcc", "-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
                           "-ffp-contract=off", "-fopenmp", "-std=c99", src, "-o", str(exe), "-lm"])
    out = subprocess.run([str(exe)], capture_output=True, text=True, timeout=120,
                         env=dict(os.environ, ASAN_OPTIONS="detect_leaks=1", OMP_NUM_THREADS="2"))
    assert out.returncode == 0, out.stderr[-2000:]
    rows = [l.split() for l in out.stdout.splitlines()]
    assert len(rows) == 3 and rows[0][1:] == rows[1][1:] and rows[2][0] == "2"
    assert abs(float(rows[0][1]) - float(rows[1][1])) <= 1e-12 * abs(float(rows[0][1]))

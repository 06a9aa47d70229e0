"""Pins of the ft-map construction oracle (oracle/ftmap.py): what the paper and the mathematics fix,
none of it a re-typing of the oracle's own formula.  CPU only."""
import numpy as np
import pytest

from oracle import ftmap as F
from workloads import synth


def test_F_segment_count_and_window():
    assert F.n_segments(1000, 256) == (1000 - 256) // 128 + 1 and F.n_segments(255, 256) == 0
    w = F.hann(64)
    # 50 %-overlapping Hann windows sum to one (constant overlap-add): what makes the segmentation
    # of PAPER.md:115 lossless
    assert np.allclose(w[:32] + w[32:], 1.0, atol=1e-15) and w[0] == 0.0 and w[32] == 1.0


def test_F_impulse_fixes_segment_start_and_dft_sign():
    """An impulse at sample m appears in segment j with magnitude w[m - j L/2] in every bin and
    phase -2 pi k (m - j L/2) / L (G19); in segments that do not contain it, nothing."""
    L, n_t = 128, 9
    s = np.zeros(L // 2 * (n_t + 1))
    m = 300
    s[m] = 1.0
    st = F.strain_spectrogram(s, L, n_t, 3, 40)
    k = np.arange(3, 43)
    for j in range(n_t):
        off = m - j * (L // 2)
        if 0 <= off < L:
            want = F.hann(L)[off] * np.exp(-2j * np.pi * k * off / L)
            assert np.allclose(st[j], want, atol=1e-13)
        else:
            assert np.allclose(st[j], 0.0, atol=1e-15)


def test_F_parseval_per_segment():
    rng = np.random.default_rng(0)
    L = 256
    s = rng.standard_normal(L * 3)
    st = F.strain_spectrogram(s, L, 4, 0, L // 2)            # bins 0 .. L/2 - 1
    for j in range(4):
        seg = s[j * L // 2: j * L // 2 + L] * F.hann(L)
        nyq = np.sum(seg * (-1.0) ** np.arange(L))           # bin L/2, real
        total = 2.0 * np.sum(np.abs(st[j, 1:]) ** 2) + np.abs(st[j, 0]) ** 2 + nyq ** 2
        assert total == pytest.approx(L * np.sum(seg ** 2), rel=1e-12)


def test_F_sinusoid_peak_leakage_and_delay_sign():
    """A bin-centred sinusoid of amplitude A: |s~| = A L / 4 at its bin (Hann coherent gain 1/2),
    exactly half of that in the two adjacent bins, nothing elsewhere.  With s_J(t) = s_I(t - tau0) the
    cross-power s~_I^* s~_J carries e^{-2 pi i f tau0} (G7): Eq. 8 recovers it at delay +tau0."""
    fs, L, n_t = 1024.0, 1024, 6
    t = np.arange(int(L / 2 * (n_t + 1))) / fs
    f0, A, tau0 = 100.0, 3.0, 2.3e-3
    s_i = A * np.cos(2 * np.pi * f0 * t + 0.4)
    s_j = A * np.cos(2 * np.pi * f0 * (t - tau0) + 0.4)
    st_i = F.strain_spectrogram(s_i, L, n_t, 90, 21)
    st_j = F.strain_spectrogram(s_j, L, n_t, 90, 21)
    mag = np.abs(st_i)
    assert np.allclose(mag[:, 10], A * L / 4, rtol=1e-9)
    assert np.allclose(mag[:, 9], A * L / 8, rtol=1e-9) and np.allclose(mag[:, 11], A * L / 8, rtol=1e-9)
    assert mag[:, :8].max() < 1e-8 * A * L and mag[:, 13:].max() < 1e-8 * A * L
    csd = np.conj(st_i[:, 10]) * st_j[:, 10]
    assert np.allclose(np.angle(csd * np.exp(2j * np.pi * f0 * tau0)), 0.0, atol=1e-9)
    # Eq. 3: Re[e^{2 pi i f dtau} csd] / |csd| = cos(2 pi f (dtau - tau0))
    for dtau in (0.0, 1e-3, tau0, 5e-3):
        r = np.real(np.exp(2j * np.pi * f0 * dtau) * csd) / np.abs(csd)
        assert np.allclose(r, np.cos(2 * np.pi * f0 * (dtau - tau0)), atol=1e-9)


def test_F_neighbours_skip_the_overlapping_segments_G20():
    n_t, n_f = 12, 3
    st = np.zeros((n_t, n_f), dtype=np.complex128)
    st[5] = 2.0                                              # power 4 in segment 5 only
    P, cnt = F.neighbour_power(st, 2)
    assert P[5].max() == 0.0 and P[4].max() == 0.0 and P[6].max() == 0.0      # itself and the 50 % overlaps
    assert np.allclose(P[3], 4.0 / 4) and np.allclose(P[7], 4.0 / 4) and np.allclose(P[2], 4.0 / 3)   # segment 2 has 3 neighbours: 0, 4, 5
    assert P[1].max() == 0.0 and P[9].max() == 0.0           # beyond n_nb + 1 = 3 segments away
    assert list(cnt[:4]) == [2, 2, 3, 4] and cnt[5] == 4     # edges use the neighbours that exist
    _, c1 = F.neighbour_power(np.ones((2, 1), dtype=np.complex128), 4)
    assert list(c1) == [0, 0]                                # no neighbour at all -> masked by ftmap


def test_F_scale_invariance_and_unit_variance_A1_A3():
    """p does not depend on the units of either strain series (lambda normalises them away, A4), and on
    stationary independent Gaussian noise Re[e^{i phi} p] has zero mean and variance
    (m/(m-1))^2-ish -> 1 as the number of neighbours grows (A1-A3; G21)."""
    rng = np.random.default_rng(5)
    fs, L, n_t, n_f = 512.0, 512, 160, 120
    n = int(L / 2 * (n_t + 1))
    s_i, s_j = rng.standard_normal(n), rng.standard_normal(n)
    p, *_ = F.ftmap(s_i, s_j, fs, L, n_t, 40.0, n_f, 24)
    p2, *_ = F.ftmap(1e-21 * s_i, 3e-19 * s_j, fs, L, n_t, 40.0, n_f, 24)
    assert np.allclose(p, p2, rtol=1e-10, atol=1e-12)
    core = p[30:-30]                                         # full neighbour sets
    for phi in (0.0, 0.7, np.pi / 2):
        rho = np.real(np.exp(1j * phi) * core)
        assert abs(rho.mean()) < 0.02
        assert 1.0 < rho.var() < 1.12                        # 48 overlapping neighbours: a few % above 1
    few, *_ = F.ftmap(s_i, s_j, fs, L, n_t, 40.0, n_f, 2)
    assert np.real(few[30:-30]).var() > 1.5                  # 4 neighbours: E[1/P'] bias is large
    # masked where there is no neighbour
    tiny, *_ = F.ftmap(s_i, s_j, fs, L, 2, 40.0, n_f, 4)
    assert np.all(tiny == 0.0)


def test_F_ftmap_feeds_the_search_oracle(orc):
    """End to end on the CPU: a chirp injected coherently in both strain series (delay tau0) is found
    by the search oracle near +tau0 on the map the ft-map oracle builds."""
    rng = np.random.default_rng(11)
    fs, L, n_t, n_f, f_min = 1024.0, 1024, 64, 200, 100.0
    n = int(L / 2 * (n_t + 1))
    t = np.arange(n) / fs
    tau0 = 3e-3
    f_inst = lambda x: 150.0 + 2.5 * x                        # 150 -> 230 Hz over 32 s
    phase = lambda x: 2 * np.pi * (150.0 * x + 1.25 * x ** 2)
    h_i = 0.7 * np.cos(phase(t))
    h_j = 0.7 * np.cos(phase(t - tau0))
    p, *_ = F.ftmap(rng.standard_normal(n) + h_i, rng.standard_normal(n) + h_j, fs, L, n_t, f_min, n_f, 8)
    tau = synth.tau_linspace(41, -0.01, 0.01)
    r = orc.search(p, f_min, fs / L, 20000, 3, 30, 64, tau_grid=tau)
    assert r["max_snr"] > 8.0 and abs(r["arg_tau"] - tau0) <= 1.0e-3


def test_F_timeshift_zero_is_identity_and_shift_destroys_coherence():
    """G23: shift 0 reproduces the unshifted map; a whole-segment shift of detector J leaves the noise
    statistics unchanged but removes a transient that is coherent between the detectors (the point of
    a time-shift background); shifting by n_t is the identity (cyclic)."""
    rng = np.random.default_rng(8)
    fs, L, n_t, n_f = 256.0, 256, 60, 80
    n = int(L / 2 * (n_t + 1))
    t = np.arange(n) / fs
    env = ((t > 10.0) & (t < 14.0)).astype(float)
    h = 1.2 * env * np.cos(2 * np.pi * (50.0 * t + 1.5 * (t - 10.0) ** 2))       # a 4 s chirp, 50 -> 62 Hz
    s_i, s_j = rng.standard_normal(n) + h, rng.standard_normal(n) + h
    p, st_i, st_j, _, _ = F.ftmap(s_i, s_j, fs, L, n_t, 20.0, n_f, 6)
    assert np.array_equal(F.ftmap_timeshift(st_i, st_j, 6, 0), p)
    assert np.array_equal(F.ftmap_timeshift(st_i, st_j, 6, n_t), p)
    rows, band = slice(20, 27), slice(28, 44)              # the pixels the chirp crosses
    n_box = 7 * 16
    assert np.real(p[rows, band]).sum() > 5.0 * np.sqrt(n_box)            # coherent: +829 measured, noise rms ~11
    for s in (3, 17, 31):
        shifted = F.ftmap_timeshift(st_i, st_j, 6, s)
        assert abs(np.real(shifted[rows, band]).sum()) < 4.0 * np.sqrt(n_box)
        assert 0.9 < np.real(shifted[10:-10, 60:80]).var() < 1.3         # noise statistics unchanged
    # pairing rule, spelled out on one pixel
    shifted = F.ftmap_timeshift(st_i, st_j, 6, 17)
    j, q, s = 20, 5, 17
    P_i, _ = F.neighbour_power(st_i, 6)
    P_j, _ = F.neighbour_power(st_j, 6)
    want = np.sqrt(2) * np.conj(st_i[j, q]) * st_j[(j + s) % n_t, q] / np.sqrt(P_i[j, q] * P_j[(j + s) % n_t, q])
    assert shifted[j, q] == pytest.approx(want, rel=1e-14)

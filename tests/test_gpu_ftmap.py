"""GPU parity of the ft-map construction (st_set_map_from_strain) against oracle/ftmap.py."""
import numpy as np
import pytest

from oracle import ftmap as F
from workloads import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1401_8060_b200 as pkg
    from paper_1401_8060_b200 import build
    build.build()
    pkg.load_library()
    return pkg


def _coloured_noise(rng, n, fs):
    """Gaussian noise with a steep low-frequency wall (5 decades in amplitude between 10 Hz and the band),
    the feature of strain data that makes a float32 transform inadequate."""
    f = np.fft.rfftfreq(n, 1.0 / fs)
    shape = 1.0 + (60.0 / np.maximum(f, 1.0)) ** 6
    return np.fft.irfft(np.fft.rfft(rng.standard_normal(n)) * shape, n)


@pytest.mark.parametrize("L,fs,n_t,f_min,n_f,n_nb,coloured", [
    (64, 64.0, 9, 3.0, 20, 2, False),            # smallest transform, ragged everything
    (1024, 1024.0, 40, 40.0, 300, 4, True),
    (4096, 4096.0, 250, 40.0, 961, 4, True),     # config 2 shape: 250 s x 961 bins at 1 s x 1 Hz
    (8192, 8192.0, 120, 40.0, 2461, 8, False),   # largest transform, config 3-5 band (2461 bins from 40 Hz)
])
def test_ftmap_matches_oracle(P, L, fs, n_t, f_min, n_f, n_nb, coloured):
    import torch
    rng = np.random.default_rng(L + n_t)
    n = (n_t + 1) * L // 2 + 13                   # a ragged tail the segmentation ignores
    mk = (lambda: _coloured_noise(rng, n, fs)) if coloured else (lambda: rng.standard_normal(n))
    s_i, s_j = 1e-21 * mk(), 3e-21 * mk()          # strain-like amplitudes
    st = P.Stochtrack(n_t, n_f, fs / L, f_min, max_n_tau=64)
    st.set_map_from_strain(torch.from_numpy(s_i).cuda(), torch.from_numpy(s_j).cuda(), fs, L, n_nb)
    p = st.debug_get_map()
    a, b = st.debug_strain_spectra()
    ref, r_i, r_j, _, _ = F.ftmap(s_i, s_j, fs, L, n_t, f_min, n_f, n_nb)
    # float64 transform on both sides: agreement to rounding, relative to the segment's largest bin IN THE
    # WHOLE SPECTRUM (the error of an FFT scales with the rms of its input)
    scale_i = np.sqrt(L) * np.abs(s_i).max() * 4
    scale_j = np.sqrt(L) * np.abs(s_j).max() * 4
    assert np.abs(a - r_i).max() <= 1e-12 * scale_i and np.abs(b - r_j).max() <= 1e-12 * scale_j
    # the map is float32: one rounding of an O(1) number (plus the float64 error above, amplified by
    # the dynamic range of a coloured spectrum)
    tol = 2e-6 * np.maximum(np.abs(ref), 1.0) + (1e-5 if coloured else 0.0)
    assert np.all(np.abs(p - ref) <= tol), float(np.abs(p - ref).max())
    assert np.array_equal(p == 0, ref == 0)        # the same pixels are masked


def test_ftmap_then_search_equals_oracle_chain(P, orc):
    """strain -> map -> search, all on the device, against ftmap oracle -> search oracle."""
    import torch
    rng = np.random.default_rng(21)
    fs, L, n_t, n_f, f_min = 1024.0, 1024, 64, 200, 100.0
    n = (n_t + 1) * L // 2
    t = np.arange(n) / fs
    tau0 = 3e-3
    phase = lambda x: 2 * np.pi * (150.0 * x + 1.25 * x ** 2)
    s_i = rng.standard_normal(n) + 0.7 * np.cos(phase(t))
    s_j = rng.standard_normal(n) + 0.7 * np.cos(phase(t - tau0))
    st = P.Stochtrack(n_t, n_f, fs / L, f_min, max_n_tau=64)
    st.set_map_from_strain(torch.from_numpy(s_i).cuda(), torch.from_numpy(s_j).cuda(), fs, L, 8)
    tau = synth.tau_linspace(41, -0.01, 0.01)
    r = st.search(20000, 3, 30, 64, tau_grid=tau, n_bins=100)
    # the oracle searches the float32 map the device built (its own float64 map differs in the last
    # float32 bit of each pixel; the maps themselves are compared in test_ftmap_matches_oracle)
    ref = orc.search(st.debug_get_map().astype(np.complex128), f_min, fs / L, 20000, 3, 30, 64, tau_grid=tau, n_bins=100)
    assert (r.arg_track, r.arg_tau_index) == (ref["arg_track"], ref["arg_tau_index"])
    assert abs(r.max_snr_f64 - ref["max_snr"]) <= 1e-11 * abs(ref["max_snr"])
    assert r.max_snr_f64 > 8.0 and abs(r.arg_tau - tau0) <= 1e-3
    pure, *_ = F.ftmap(s_i, s_j, fs, L, n_t, f_min, n_f, 8)
    ref2 = orc.search(pure, f_min, fs / L, 20000, 3, 30, 64, tau_grid=tau)
    assert (ref2["arg_track"], ref2["arg_tau_index"]) == (r.arg_track, r.arg_tau_index)
    assert abs(ref2["max_snr"] - r.max_snr_f64) <= 1e-5 * abs(ref2["max_snr"])


def test_ftmap_argument_errors(P):
    import torch
    st = P.Stochtrack(10, 20, 1.0, 40.0, max_n_tau=64)
    s = torch.zeros(11 * 512, dtype=torch.float64, device="cuda")
    for kw in (dict(fs=1024.0, seg_len=1000),                  # not a power of two
               dict(fs=2048.0, seg_len=1024),                  # df mismatch
               dict(fs=64.0, seg_len=64),                      # band above Nyquist
               dict(fs=1024.0, seg_len=1024, n_neighbours=0)):
        with pytest.raises(P.StError):
            st.set_map_from_strain(s, s, **kw)
    with pytest.raises(P.StError):
        st.set_map_from_strain(s[:1000], s[:1000], 1024.0, 1024)   # too few samples


def test_timeshift_background_from_strain(P, orc):
    """st_search_timeshifts: spectrograms once, one (map, search) per whole-segment shift (G23).  Every
    shift's map equals the oracle's ftmap_timeshift, its search equals the search oracle on that map; the
    zero-lag entry finds the injected chirp, the shifted ones do not (the time-shift background)."""
    import torch
    rng = np.random.default_rng(33)
    fs, L, n_t, n_f, f_min, n_nb = 1024.0, 1024, 64, 200, 100.0, 6
    n = (n_t + 1) * L // 2
    t = np.arange(n) / fs
    tau0 = -2e-3
    env = ((t > 4.0) & (t < 28.0)).astype(float)
    phase = lambda x: 2 * np.pi * (150.0 * x + 1.25 * x ** 2)
    s_i = rng.standard_normal(n) + 0.8 * env * np.cos(phase(t))
    s_j = rng.standard_normal(n) + 0.8 * env * np.cos(phase(t - tau0))
    shifts = [0, 1, 7, 31, 63]
    seeds = [5, 6, 7, 8, 9]
    tau = synth.tau_linspace(41, -0.01, 0.01)
    st = P.Stochtrack(n_t, n_f, fs / L, f_min, max_n_tau=64)
    res, ms = st.search_timeshifts(torch.from_numpy(s_i).cuda(), torch.from_numpy(s_j).cuda(), fs, L, n_nb, shifts, seeds,
                                   8000, 20, 64, tau_grid=tau, n_bins=100)
    assert len(res) == len(shifts) and ms > 0
    _, r_i, r_j, _, _ = F.ftmap(s_i, s_j, fs, L, n_t, f_min, n_f, n_nb)
    last = st.debug_get_map()                                     # the context keeps the last shift's map
    ref_last = F.ftmap_timeshift(r_i, r_j, n_nb, shifts[-1])
    assert np.all(np.abs(last - ref_last) <= 2e-6 * np.maximum(np.abs(ref_last), 1.0))
    for m, (sh, sd) in enumerate(zip(shifts, seeds)):
        pm = F.ftmap_timeshift(r_i, r_j, n_nb, sh)
        ref = orc.search(pm, f_min, fs / L, 8000, sd, 20, 64, tau_grid=tau, n_bins=100)
        # float32 map on the device vs float64 map in the oracle: same argmax unless a near tie (none here)
        assert (res[m].arg_track, res[m].arg_tau_index) == (ref["arg_track"], ref["arg_tau_index"]), m
        assert abs(res[m].max_snr_f64 - ref["max_snr"]) <= 1e-5 * abs(ref["max_snr"])
        assert int(res[m].hist.sum()) == 8000 * 41
    assert res[0].max_snr_f64 > 8.0 and abs(res[0].arg_tau - tau0) <= 1e-3
    assert max(r.max_snr_f64 for r in res[1:]) < 0.75 * res[0].max_snr_f64
    # shift 0 of the batch call == st_set_map_from_strain + st_search, bit for bit
    st.set_map_from_strain(torch.from_numpy(s_i).cuda(), torch.from_numpy(s_j).cuda(), fs, L, n_nb)
    one = st.search(8000, seeds[0], 20, 64, tau_grid=tau, n_bins=100)
    assert (one.max_snr_f64, one.arg_track, one.arg_tau_index) == (res[0].max_snr_f64, res[0].arg_track, res[0].arg_tau_index)
    with pytest.raises(P.StError):
        st.search_timeshifts(torch.from_numpy(s_i).cuda(), torch.from_numpy(s_j).cuda(), fs, L, n_nb, [n_t], 1, 10, 20, 64, tau_grid=tau)


def test_timeshift_background_with_one_bank_and_the_bank_cache(P, orc):
    """The paper's background workflow with ONE template bank for every time shift ("arrays of Bezier
    curves", :173 n_ts time-shift analyses): with the bank cache attached the first shift fills it, the others read
    S1 + S2 back; every result is bit-identical to the call without a cache and agrees with the oracle."""
    import torch
    rng = np.random.default_rng(34)
    fs, L, n_t, n_f, f_min, n_nb = 1024.0, 1024, 64, 200, 100.0, 6
    n = (n_t + 1) * L // 2
    s_i, s_j = rng.standard_normal(n), rng.standard_normal(n)
    shifts, seed, T = [0, 3, 9, 27, 40], 11, 6000
    tau = synth.tau_linspace(100, -0.01, 0.01)                    # two chunks: the one-pass build
    di, dj = torch.from_numpy(s_i).cuda(), torch.from_numpy(s_j).cuda()
    plain = P.Stochtrack(n_t, n_f, fs / L, f_min, max_n_tau=128)
    want, _ = plain.search_timeshifts(di, dj, fs, L, n_nb, shifts, seed, T, 20, 64, tau_grid=tau, n_bins=100)
    assert all(w.flags & 6 == 0 for w in want)
    st = P.Stochtrack(n_t, n_f, fs / L, f_min, max_n_tau=128)
    assert st.enable_bank_cache(T, 64) > 0
    got, _ = st.search_timeshifts(di, dj, fs, L, n_nb, shifts, seed, T, 20, 64, tau_grid=tau, n_bins=100)
    assert got[0].flags & 4 and all(g.flags & 2 for g in got[1:])
    for g, w in zip(got, want):
        assert (g.max_snr, g.max_snr_f64, g.arg_track, g.arg_tau_index, g.n_evals) == (w.max_snr, w.max_snr_f64, w.arg_track, w.arg_tau_index, w.n_evals)
        assert np.array_equal(g.hist, w.hist)
    _, r_i, r_j, _, _ = F.ftmap(s_i, s_j, fs, L, n_t, f_min, n_f, n_nb)
    for m in (1, 4):
        ref = orc.search(F.ftmap_timeshift(r_i, r_j, n_nb, shifts[m]), f_min, fs / L, T, seed, 20, 64, tau_grid=tau, n_bins=100)
        assert (got[m].arg_track, got[m].arg_tau_index) == (ref["arg_track"], ref["arg_tau_index"])
        assert abs(got[m].max_snr_f64 - ref["max_snr"]) <= 1e-5 * abs(ref["max_snr"])


def test_inverse_variance_norm_is_refused_on_maps_built_from_strain(P):
    """A map built from strain carries no 1 / sigma plane (k_ft_normalise forms p directly), so the inverse-variance
    statistic (G25) has nothing to weight by: the time-shift call refuses it up front (ST_EINVAL) and a plain search
    on such a map reports the missing state (ST_ESTATE) -- even when an earlier st_set_map left a plane of its own in
    the workspace (the silent-wrong-result case the refusal closes).  The context stays usable."""
    import torch
    rng = np.random.default_rng(35)
    fs, L, n_t, n_f, f_min, n_nb = 1024.0, 1024, 32, 100, 100.0, 4
    n = (n_t + 1) * L // 2
    di, dj = torch.from_numpy(rng.standard_normal(n)).cuda(), torch.from_numpy(rng.standard_normal(n)).cuda()
    tau = synth.tau_linspace(16, -0.01, 0.01)
    st = P.Stochtrack(n_t, n_f, fs / L, f_min, max_n_tau=64)
    # a map with its own sigma first: the plane it leaves behind must not be picked up by the strain path
    st.set_map(synth.noise_csd(n_t, n_f, 5), synth.make_sigma("per_pixel", 0.3, n_t, n_f, 5))
    ok = st.search(500, 3, 10, 32, tau_grid=tau, norm=P.NORM_INVVAR)
    assert np.isfinite(ok.max_snr_f64)
    with pytest.raises(P.StError) as e:
        st.search_timeshifts(di, dj, fs, L, n_nb, [0, 5], 3, 500, 10, 32, tau_grid=tau, norm=P.NORM_INVVAR)
    assert e.value.code == -1 and "ST_NORM_INVVAR" in str(e.value)
    st.set_map_from_strain(di, dj, fs, L, n_nb)
    for call in (lambda: st.search(500, 3, 10, 32, tau_grid=tau, norm=P.NORM_INVVAR),
                 lambda: st.search(500, 3, 10, 32, tau_range=(-0.01, 0.01), norm=P.NORM_INVVAR),
                 lambda: st.debug_scores(3, 10, 32, 0, 100, tau_grid=tau, norm=P.NORM_INVVAR)):
        with pytest.raises(P.StError) as e:
            call()
        assert e.value.code == -2 and "sigma" in str(e.value)
    res, _ = st.search_timeshifts(di, dj, fs, L, n_nb, [0, 5], 3, 500, 10, 32, tau_grid=tau)
    assert len(res) == 2 and all(np.isfinite(r.max_snr_f64) for r in res)

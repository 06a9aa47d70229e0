"""Randomised soak of the CUDA path against the oracle, and the one argmax case with two correct answers.

Seeded and bounded (150 random shapes, well under a minute on a B200): every draw picks a map shape, a frequency
axis, a sigma layout (with masked pixels now and then), a template family, a normalisation, a duration range, a
template-id range and either the random-delay mode or a delay grid (uniform of any length, or non-uniform), scores
every template through the C ABI and compares EVERY SNR with the oracle (G13) and the argmax of the search with the
oracle's (G12, with the near-tie clause SURVEY 8(c) declares in advance: the oracle's own value at the GPU's choice
within 2e-6 relative of the oracle's maximum -> either sample accepted; such cases are counted and printed).
The constructed case is DESIGN.md's exact periodic tie: a map whose only non-zero row is the 50 Hz bin scores every
template identically at -10 ms and +10 ms (the two phase factors coincide on every pixel), so two delay indices are
correct; the value must agree to float64 rounding and the index must be one of the two."""
import numpy as np
import pytest

from workloads import synth
from helpers import snr_close, argmax_ok, S0_UNIT

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


def _draw(rng):
    n_t, n_f = int(rng.integers(8, 200)), int(rng.integers(7, 500))
    df = float(rng.choice([0.5, 1.0, 2.0]))
    f_min = df * float(rng.integers(0, 300))
    skind = str(rng.choice(["none", "per_f", "per_pixel"]))
    family, norm = int(rng.integers(0, 3)), int(rng.integers(0, 3))
    n_min = int(rng.integers(1, n_t + 1))
    n_max = int(rng.integers(n_min, n_t + 1))
    T = int(rng.integers(20, 400))
    first = int(rng.choice([0, 1, 12345, 2 ** 33 + 5]))
    mode = rng.random()
    if mode < 0.25:
        lo = float(rng.uniform(-0.01, 0.005))
        grid, rng_tau = None, (lo, float(rng.uniform(lo, 0.01)))
    else:
        n_tau = int(rng.integers(1, 131))
        lo = float(rng.uniform(-0.01, 0.0))
        hi = float(rng.uniform(lo + 1e-4, 0.01))
        grid = np.sort(rng.uniform(lo, hi, n_tau)) if mode < 0.4 else synth.tau_linspace(n_tau, lo, hi)
        rng_tau = None
    return dict(n_t=n_t, n_f=n_f, df=df, f_min=f_min, skind=skind, family=family, norm=norm, n_min=n_min, n_max=n_max, T=T,
                first=first, grid=grid, tau_range=rng_tau, seed=int(rng.integers(0, 2 ** 40)))


def test_soak_random_shapes_grids_families_norms(P, orc):
    rng = np.random.default_rng(20261106)
    near_ties, worst_all, kernels = [], 0.0, {}
    for it in range(150):
        d = _draw(rng)
        n_t, n_f = d["n_t"], d["n_f"]
        csd = synth.noise_csd(n_t, n_f, 7000 + it)
        sigma = synth.make_sigma(d["skind"], 0.3, n_t, n_f, 7000 + it)
        if sigma is not None and it % 3 == 0:                       # masked pixels (G11)
            sigma = sigma.copy()
            sigma.flat[int(rng.integers(0, sigma.size))] = 0.0
            sigma.flat[int(rng.integers(0, sigma.size))] = np.inf
        st = P.Stochtrack(n_t, n_f, d["df"], d["f_min"], max_n_tau=max(64, 0 if d["grid"] is None else len(d["grid"])))
        st.set_map(csd, sigma)
        p = orc.prepare_map(csd, sigma)
        kw = dict(tau_grid=d["grid"]) if d["grid"] is not None else dict(tau_range=d["tau_range"])
        okw = dict(kw, norm=d["norm"], family=d["family"], track_offset=d["first"])
        if d["norm"] == 2:
            okw["inv_sigma"] = orc.prepare_inv_sigma(p.shape, sigma)
        ref = orc.search(p, d["f_min"], d["df"], d["T"], d["seed"], d["n_min"], d["n_max"], dump_snr=True, **okw)
        got = st.debug_scores(d["seed"], d["n_min"], d["n_max"], d["first"], d["T"], norm=d["norm"], family=d["family"], **kw)
        s0 = S0_UNIT / np.sqrt(d["n_max"]) if d["norm"] == 1 else S0_UNIT
        ok, worst = snr_close(got, ref["snr"], s0=s0)
        assert ok, (it, {k: v for k, v in d.items() if k != "grid"}, worst)
        worst_all = max(worst_all, worst)
        r = st.search(d["T"], d["seed"], d["n_min"], d["n_max"], track_offset=d["first"], norm=d["norm"], family=d["family"],
                      n_bins=40, hist_lo=-4.0, hist_hi=4.0, **kw)
        kernels[r.kernel_name] = kernels.get(r.kernel_name, 0) + 1
        ok, near = argmax_ok(r.arg_track, r.arg_tau_index, ref, first=d["first"])
        assert ok, (it, {k: v for k, v in d.items() if k != "grid"}, r.arg_track, r.arg_tau_index, ref["arg_track"], ref["arg_tau_index"])
        if near:
            near_ties.append(it)
        if ref["max_snr"] != 0.0:
            assert abs(r.max_snr_f64 - ref["max_snr"]) <= 3e-7 * abs(ref["max_snr"]), it
        assert int(r.hist.sum()) == ref["snr"].size and r.n_pixels == ref["n_pixels"]
        st.close()
    print(f"soak: 150 cases, worst SNR error {worst_all:.3f} x the G13 tolerance, kernels {kernels}, near ties accepted at {near_ties}")
    assert len(near_ties) <= 5                   # the clause is for rare rounding ties, not a way to pass
    assert len(kernels) >= 3                     # the draw reaches the random, Chebyshev and table kernels at least


@pytest.mark.parametrize("n_tau", [16, 64, 129])
def test_exact_periodic_tie_has_two_correct_delays(P, orc, n_tau):
    """Only the 50 Hz bin is non-zero: SNR(i, tau) = -A n_i cos(2 pi 50 tau) / sqrt(N_i), equal at -10 ms and +10 ms for
    every template (cos(-pi) = cos(pi)).  The first and the last delay of the grid are both correct argmax delays."""
    n_t, n_f, f_min, A = 64, 20, 40.0, 3.0
    csd = np.zeros((n_t, n_f), dtype=np.complex64)
    csd[:, 10] = -A
    tau = synth.tau_linspace(n_tau)                                  # -10 ms ... +10 ms, endpoints included
    st = P.Stochtrack(n_t, n_f, 1.0, f_min, max_n_tau=max(64, n_tau))
    st.set_map(csd)
    ref = orc.search(orc.prepare_map(csd), f_min, 1.0, 2000, 9, 8, 64, tau_grid=tau, dump_snr=True)
    assert abs(ref["snr"][:, 0] - ref["snr"][:, -1]).max() <= 1e-12 and ref["max_snr"] > 1.0     # the tie is in the oracle too
    for kernel in (P.KERNEL_AUTO, P.KERNEL_TABLE, P.KERNEL_ROTATION):
        r = st.search(2000, 9, 8, 64, tau_grid=tau, kernel=kernel)
        ok, _ = argmax_ok(r.arg_track, r.arg_tau_index, ref)
        assert ok and r.arg_tau_index in (0, n_tau - 1), (kernel, r.arg_track, r.arg_tau_index)
        assert abs(r.max_snr_f64 - ref["max_snr"]) <= 1e-12 * ref["max_snr"]
        # the template is one of those attaining the maximum (several may: equal n_i / sqrt(N_i))
        assert abs(ref["snr"][r.arg_track, r.arg_tau_index] - ref["max_snr"]) <= 1e-12 * ref["max_snr"]

"""Float32 error budget of the production scoring recurrence, checked on the CPU
with a NumPy float32 emulation of exactly the arithmetic k_score_cheb performs per pixel: anchors
every 64 delays at the chunk centre, 32 forward and 32 backward delays of the stride-S recurrence
x_{m+S} = fl32(G x_m - x_{m-S}) with G = fl32(2 cos(S theta)), anchors advanced by a float32 rotation.
It bounds the per-term error that the 1e-4 SNR tolerance (G13) has to absorb for the step angles of
the five configurations, and re-derives the host's conditioning rule (drift of the float32
coefficient over 32 delays <= 3e-5 rad, stride 1 or 2)."""
import numpy as np

F32 = np.float32


def _fma32(a, b, c):
    return (a.astype(np.float64) * b.astype(np.float64) + c.astype(np.float64)).astype(F32)


def _cheb_terms(p, f, tau0, dtau, n_tau, stride):
    """x[pixel][m] as the kernel computes it (float32), for pixels (p, f)."""
    theta = 2 * np.pi * f * dtau
    G = (2 * np.cos(stride * theta)).astype(F32)
    c, s = np.cos(theta).astype(F32), np.sin(theta).astype(F32)
    z64 = np.exp(1j * 64 * theta)
    z64r, z64i = z64.real.astype(F32), z64.imag.astype(F32)
    v = p * np.exp(2j * np.pi * f * (tau0 + 32 * dtau))
    vr, vi = v.real.astype(F32), v.imag.astype(F32)
    out = np.zeros((p.size, ((n_tau + 63) // 64) * 64), F32)
    for j in range(0, n_tau, 64):
        w = (vi * s).astype(F32)
        xm1 = _fma32(vr, c, w)
        if stride == 1:
            chains = [(vr.copy(), xm1.copy(), 32, +1, 1), (xm1.copy(), vr.copy(), 31, -1, 1)]
        else:
            xp1 = _fma32(vr, c, -w)
            xm2 = _fma32((c + c).astype(F32), xm1, -vr)
            chains = [(vr.copy(), xm2, 32, +1, 2), (xp1.copy(), xm1.copy(), 33, +1, 2),
                      (xm1.copy(), xp1, 31, -1, 2), (xm2.copy(), vr.copy(), 30, -1, 2)]
        for cur, prev, pos, sign, st in chains:
            for _ in range(32 // st):
                out[:, j + pos] = cur
                cur, prev = _fma32(G, cur, -prev), cur
                pos += sign * st
        nvr = _fma32(vr, z64r, -(vi * z64i).astype(F32))
        nvi = _fma32(vr, z64i, (vi * z64r).astype(F32))
        vr, vi = nvr, nvi
    return out[:, :n_tau]


def _errors(n_tau, f_lo, f_hi, stride, n_pix=4000, span=0.02, seed=0):
    rng = np.random.default_rng(seed)
    dtau, tau0 = span / (n_tau - 1), -span / 2
    f = np.round(rng.uniform(f_lo, f_hi, n_pix))
    p = (rng.standard_normal(n_pix) + 1j * rng.standard_normal(n_pix)) * np.sqrt(0.5)
    m = np.arange(n_tau)
    exact = np.real(p[:, None] * np.exp(2j * np.pi * f[:, None] * (tau0 + m[None, :] * dtau)))
    err = np.abs(_cheb_terms(p, f, tau0, dtau, n_tau, stride) - exact) / np.abs(p)[:, None]
    return err, 2 * np.pi * f * dtau


def _drift(n_tau, f_lo, f_hi, stride, span=0.02):
    """The host's conditioning number: (32 / S) |acos(G/2) - S theta| maximised over the bins."""
    f = np.arange(f_lo, f_hi + 1, dtype=np.float64)
    sth = stride * 2 * np.pi * f * span / (n_tau - 1)
    sth = np.abs(sth - 2 * np.pi * np.round(sth / (2 * np.pi)))
    G = (2 * np.cos(sth)).astype(F32).astype(np.float64)
    return float(((32 / stride) * np.abs(np.arccos(np.clip(G / 2, -1, 1)) - sth)).max())


def test_term_error_on_the_five_configs_grids():
    # (n_tau, band, stride the host picks) of configs 5, 4, 2, 1
    for n_tau, f_lo, f_hi, stride in [(512, 40, 2500, 2), (128, 40, 2500, 1), (64, 40, 1000, 1), (16, 40, 103, 1)]:
        err, theta = _errors(n_tau, f_lo, f_hi, stride)
        assert err.max() < 2.5e-5, (n_tau, err.max())         # one term, worst case: a quarter of the tolerance
        assert np.sqrt((err ** 2).mean()) < 3e-6, n_tau       # what a sqrt(N)-normalised sum sees
        assert _drift(n_tau, f_lo, f_hi, stride) <= 3e-5      # the host's acceptance rule holds


def test_stride_two_quarters_the_drift_on_fine_grids():
    """Config 5 (512 delays): theta_min = 0.0098.  With stride 1 the float32 coefficient drifts the
    phase by up to 7.5e-5 rad over 32 delays (too close to 1e-4 for a coherent signal); stride 2
    divides that by ~4.  Stride 2 needs 2 theta < pi, so the coarse grids keep stride 1."""
    d1, d2 = _drift(512, 40, 2500, 1), _drift(512, 40, 2500, 2)
    assert 5e-5 < d1 < 1e-4 and d2 < 0.3 * d1 and d2 <= 3e-5
    e1, _ = _errors(512, 40, 400, 1, seed=3)
    e2, _ = _errors(512, 40, 400, 2, seed=3)
    assert e2.max() < 0.6 * e1.max()
    assert 2 * 2 * np.pi * 2500 * 0.02 / 127 > np.pi            # config 4: stride 2 not admissible
    # term errors stay inside the drift bound plus a rounding floor
    err, theta = _errors(512, 40, 2500, 1, n_pix=3000, seed=1)
    bound = 32 * 2.0 ** -24 / np.abs(np.sin(theta)) + 4e-6
    assert (err.max(axis=1) <= bound).all()

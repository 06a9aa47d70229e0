"""Synthetic ft-maps with the shapes of the paper's workloads.

The paper's real inputs (recoloured LIGO noise; FA/ADI
waveforms) are not available; these seeded Gaussian-noise maps
stand in for them: 250-1000 s maps at 1 s x 1 Hz
(PAPER.md:115), bands of 64-2461 bins from 40 Hz, T = 1e3..1e7 templates
(PAPER.md:90), Delta tau_max = 10 ms (1/(4 * 25 Hz)).

This module is input generation only.  It is imported by tests (which hand the
same arrays to the oracle and to the CUDA library) and by bench.py.  It contains
no step of the method: an injection receives its pixel list (j, k) from the
caller, who obtains it from whichever implementation is under test.
"""
from dataclasses import dataclass, field
from typing import Optional, Tuple

import numpy as np

TAU_MAX = 0.010  # s; PAPER.md:54 (Delta f_min ~ 25 Hz = 1/(4 Delta tau_max))


@dataclass(frozen=True)
class Injection:
    """A fixed quadratic Bezier track in the O2/O3 parameterisation."""
    j0: int
    N: int
    a: float
    y0: float
    y1: float
    y2: float
    tau: float
    snr: float


@dataclass(frozen=True)
class Config:
    name: str
    n_t: int
    n_f: int
    f_min: float
    df: float
    sigma: str                       # "none" | "per_f" | "per_pixel"
    sigma_scale: float
    n_tracks: int
    n_min: int
    n_max: int
    tau_mode: str                    # "grid" | "random"
    n_tau: int
    n_maps: int
    seed: int
    n_bins: int = 1000
    hist_lo: float = -10.0
    hist_hi: float = 10.0
    injections: Tuple[Injection, ...] = field(default_factory=tuple)


# BASELINE.json:configs[0..4] as restated in SURVEY.md 8(d); "P" = Table III shape
# (PAPER.md:212), context only.
CONFIGS = {
    1: Config("config1_tiny", 64, 64, 40.0, 1.0, "none", 0.0, 1000, 64, 64, "grid", 16, 1, 0),
    2: Config("config2_250x961", 250, 961, 40.0, 1.0, "per_f", 0.2, 100_000, 10, 250, "grid", 64, 1, 1,
              injections=(Injection(20, 200, 120.0, 700.25, 420.5, 180.75, +3.7e-3, 8.0),)),
    3: Config("config3_random_tau", 500, 2461, 40.0, 1.0, "none", 0.0, 1_000_000, 10, 500, "random", 1, 1, 2),
    4: Config("config4_background", 500, 2461, 40.0, 1.0, "none", 0.0, 1_000_000, 10, 500, "grid", 128, 100, 3),
    5: Config("config5_long", 1000, 2461, 40.0, 1.0, "per_pixel", 0.3, 10_000_000, 10, 1000, "grid", 512, 1, 4,
              injections=(Injection(100, 800, 300.0, 300.25, 900.5, 2100.75, -6.1e-3, 10.0),
                          Injection(550, 400, 250.0, 1800.25, 1500.5, 1400.75, +1.3e-3, 6.0))),
    "P": Config("configP_table3", 500, 151, 100.0, 1.0, "none", 0.0, 20_000_000, 70, 500, "random", 1, 1, 5),
}


def map_seed(cfg: Config, m: int = 0) -> int:
    """Seed of map m (noise and track bank): G16 -- base*2^32 + m for batches."""
    return cfg.seed * (1 << 32) + m if cfg.n_maps > 1 else cfg.seed


def tau_linspace(n_tau: int, lo: float = -TAU_MAX, hi: float = TAU_MAX) -> np.ndarray:
    """Endpoint-inclusive grid tau_m = lo + m * ((hi - lo)/(n_tau - 1)) in double (G8)."""
    if n_tau == 1:
        return np.array([0.5 * (lo + hi)], dtype=np.float64)
    step = (hi - lo) / (n_tau - 1)
    return lo + np.arange(n_tau, dtype=np.float64) * step


def noise_csd(n_t: int, n_f: int, seed: int) -> np.ndarray:
    """CSD = conj(s1) * s2 of two iid complex Gaussian fields with E|s|^2 = 1 (G10)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    s = rng.standard_normal((2, n_t, n_f, 2)) * np.sqrt(0.5)
    s1 = s[0, ..., 0] + 1j * s[0, ..., 1]
    s2 = s[1, ..., 0] + 1j * s[1, ..., 1]
    return (np.conj(s1) * s2).astype(np.complex64)


def make_sigma(kind: str, scale: float, n_t: int, n_f: int, seed: int) -> Optional[np.ndarray]:
    """sigma = exp(scale * z): lognormal(0, scale) per frequency bin or per pixel."""
    if kind == "none":
        return None
    rng = np.random.Generator(np.random.PCG64(seed ^ 0x5EED5167))
    if kind == "per_f":
        return np.exp(scale * rng.standard_normal(n_f)).astype(np.float32)
    if kind == "per_pixel":
        return np.exp(scale * rng.standard_normal((n_t, n_f))).astype(np.float32)
    raise ValueError(kind)


def add_injection(csd: np.ndarray, sigma: Optional[np.ndarray], j: np.ndarray, k: np.ndarray,
                  tau_inj: float, snr: float, f_min: float, df: float) -> None:
    """csd[j, k] += snr * N^(-1/2) * sigma[j, k] * exp(-2 pi i f_k tau_inj), in place.

    (j, k) is the pixel list of the injected track, supplied by the caller.  With
    the sqrt(N) normalisation a perfectly matched template then scores `snr` above
    its noise term; the sign follows G7: a signal arriving tau later
    at detector J appears as exp(-2 pi i f tau) in sI^* sJ and is recovered at +tau.
    """
    j = np.asarray(j)
    k = np.asarray(k)
    n = j.size
    if sigma is None:
        s = np.ones(n)
    elif sigma.ndim == 1:
        s = sigma[k].astype(np.float64)
    else:
        s = sigma[j, k].astype(np.float64)
    f = f_min + k.astype(np.float64) * df
    amp = snr / np.sqrt(n) * s
    add = amp * np.exp(-2j * np.pi * f * tau_inj)
    csd[j, k] = (csd[j, k].astype(np.complex128) + add).astype(np.complex64)


def config_inputs(cfg: Config, m: int = 0, rasterise=None):
    """(csd complex64 [n_t][n_f], sigma float32 or None, tau grid float64 or None).

    `rasterise(inj) -> int array k[N]` is required when the config has injections.
    """
    seed = map_seed(cfg, m)
    csd = noise_csd(cfg.n_t, cfg.n_f, seed)
    sigma = make_sigma(cfg.sigma, cfg.sigma_scale, cfg.n_t, cfg.n_f, seed)
    for inj in cfg.injections:
        if rasterise is None:
            raise ValueError("config has injections: pass rasterise=")
        k = np.asarray(rasterise(inj))
        j = inj.j0 + np.arange(inj.N)
        add_injection(csd, sigma, j, k, inj.tau, inj.snr, cfg.f_min, cfg.df)
    tau = tau_linspace(cfg.n_tau) if cfg.tau_mode == "grid" else None
    return csd, sigma, tau

"""Shared helpers of the parity tests: seeded inputs, tolerance rules (G13, G14)."""
import numpy as np

from workloads import synth

S0_UNIT = np.sqrt(0.5)   # null standard deviation of the sqrt(N) statistic on sigma = 1 maps (G10)


def oracle_rasteriser(orc, n_f):
    def rast(inj):
        return orc.rasterise(orc.make_track(inj.N, inj.j0, inj.a, inj.y0, inj.y1, inj.y2), n_f)
    return rast


def config_inputs(orc, cfg, m=0):
    """(csd, sigma, tau_grid or None); injections are rasterised by the ORACLE
    (inputs never come from the CUDA path)."""
    return synth.config_inputs(cfg, m, rasterise=oracle_rasteriser(orc, cfg.n_f))


def snr_close(gpu, ref, s0=S0_UNIT, rel=1e-4):
    """G13: |dSNR| <= 1e-4 * max(|SNR_oracle|, s0)."""
    gpu = np.asarray(gpu, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    tol = rel * np.maximum(np.abs(ref), s0)
    err = np.abs(gpu - ref)
    worst = float((err / tol).max()) if err.size else 0.0
    return bool((err <= tol).all()), worst


def hist_rule_ok(h_gpu, ref_snr, lo, hi, n_bins, s0=S0_UNIT, rel=1e-4):
    """G14: totals equal; for every bin edge e the cumulative counts differ by at most the
    number of oracle samples within the G13 tolerance of e."""
    ref_snr = np.sort(np.asarray(ref_snr, dtype=np.float64).ravel())
    h_gpu = np.asarray(h_gpu, dtype=np.int64)
    if int(h_gpu.sum()) != ref_snr.size:
        return False, "total"
    edges = lo + (hi - lo) * np.arange(1, n_bins) / n_bins       # interior edges
    cum_gpu = np.cumsum(h_gpu)[:-1]
    tol = rel * np.maximum(np.abs(edges), s0) * 1.0000001 + 1e-12
    lo_cnt = np.searchsorted(ref_snr, edges - tol, side="left")
    hi_cnt = np.searchsorted(ref_snr, edges + tol, side="right")
    ok = (cum_gpu >= lo_cnt) & (cum_gpu <= hi_cnt)
    if not ok.all():
        i = int(np.flatnonzero(~ok)[0])
        return False, f"edge {edges[i]}: gpu cum {cum_gpu[i]} not in [{lo_cnt[i]}, {hi_cnt[i]}]"
    return True, ""


def argmax_ok(arg_track, arg_m, ref, first=0, gap=2e-6):
    """G12 with its pre-declared near-tie clause: the (template, delay) the GPU returns is the
    oracle's, or the oracle's OWN float64 value at the sample the GPU chose lies within a relative `gap` of the
    oracle's maximum -- then the two samples tie to float64 rounding noise (libm vs device sincos decide) and either
    is accepted.  Needs ref["snr"] (dump_snr=True).  Returns (ok, was_near_tie)."""
    if (int(arg_track), int(arg_m)) == (int(ref["arg_track"]), int(ref["arg_tau_index"])):
        return True, False
    q = int(arg_track) - int(first)
    if not (0 <= q < ref["snr"].shape[0] and 0 <= int(arg_m) < ref["snr"].shape[1]):
        return False, False
    v = float(ref["snr"][q, int(arg_m)])
    return abs(float(ref["max_snr"]) - v) <= gap * abs(float(ref["max_snr"])), True

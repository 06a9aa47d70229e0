"""Pins of or_track_params (O2: template parameters from Philox words) against what the paper's text fixes.

What the text fixes (readings G3 / G4 of DESIGN.md make it precise):
  * PAPER.md:75   a template is three control points, "chosen randomly ... subject to the constraint that
                  the curve persists for a duration t_min": every duration in [n_min, n_max] occurs and
                  none outside; t_start < t_mid < t_end.
  * PAPER.md:86   "each template can be quickly generated from just six random numbers": the six
                  control-point numbers are independent draws (none is a function of another).
  * PAPER.md:100  the delay is one more random variable with "a simple uniform distribution between
                  +-dtau_max", independent of the curve.
  * BASELINE.json configs[0]: templates "spanning the full duration": n_min = n_max = n_t gives
                  (N, j0) = (n_t, 0) for every id.
  * G4            "chosen randomly" read as uniform: N uniform on the integers n_min..n_max, the first
                  column uniform among the feasible ones GIVEN N, t_mid uniform in (t_start, t_end),
                  frequencies uniform over the band.

The checks are statistical statements about the OUTPUT of or_track_params (attained end values,
chi-square and Kolmogorov-Smirnov uniformity, pairwise independence of all seven parameters); none of them
re-types the oracle's formula.  `test_pins_catch_plausible_slips` rebuilds the oracle with one plausible
slip at a time (off-by-one ranges, a reused random word, a start drawn before the duration) and requires
the same checks to FAIL on each: the pins bite.
"""
import ctypes as C
import os
import re
import subprocess

import numpy as np
import pytest
from scipy import stats

HERE = os.path.dirname(os.path.abspath(__file__))
ORACLE_SRC = os.path.join(os.path.dirname(HERE), "oracle", "stochtrack_oracle.c")


class _Track(C.Structure):
    _fields_ = [("N", C.c_int32), ("j0", C.c_int32), ("a", C.c_double), ("y0", C.c_double),
                ("y1", C.c_double), ("y2", C.c_double), ("tau", C.c_double), ("y3", C.c_double), ("family", C.c_int32)]


def _sampler(lib):
    """ids -> array [T][7] of (N, j0, a, y0, y1, y2, tau) from the or_track_params of `lib`."""
    fn = lib.or_track_params
    fn.argtypes = [C.c_uint64, C.c_uint64, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_double, C.c_double,
                   C.POINTER(_Track)]
    fn.restype = C.c_int

    def sample(seed, first, count, n_t, n_f, n_min, n_max, lo, hi):
        out = np.empty((count, 7))
        t = _Track()
        for q in range(count):
            assert fn(seed, first + q, n_t, n_f, n_min, n_max, lo, hi, C.byref(t)) == 0
            out[q] = (t.N, t.j0, t.a, t.y0, t.y1, t.y2, t.tau)
        return out
    return sample


def check_track_param_pins(sample):
    """Raises AssertionError unless `sample` behaves as the text (with G3 / G4) requires."""
    n_t, n_f, n_min, n_max, lo, hi, T = 40, 97, 3, 12, -0.004, 0.010, 120_000
    s = sample(11, 2 ** 33 + 1, T, n_t, n_f, n_min, n_max, lo, hi)
    N, j0 = s[:, 0].astype(int), s[:, 1].astype(int)
    a, y, tau = s[:, 2], s[:, 3:6], s[:, 6]
    n_dur = n_max - n_min + 1
    # ---- ranges, and BOTH end values attained (an off-by-one in either range fails here)
    assert N.min() == n_min and N.max() == n_max, "duration range"
    assert (j0 >= 0).all() and (j0 + N <= n_t).all(), "template leaves the map"
    for n in range(n_min, n_max + 1):
        sel = j0[N == n]
        assert sel.min() == 0 and sel.max() == n_t - n, f"start range at N = {n}"
    assert ((a > 0) & (a < N)).all(), "t_start < t_mid < t_end (G3)"
    assert ((y > 0) & (y < n_f)).all() and ((tau > lo) & (tau < hi)).all()
    # ---- N uniform over its n_dur values (chi-square, n_dur - 1 degrees of freedom)
    cnt = np.bincount(N - n_min, minlength=n_dur)
    chi2 = ((cnt - T / n_dur) ** 2 / (T / n_dur)).sum()
    assert chi2 < stats.chi2.ppf(1 - 1e-6, n_dur - 1), f"N not uniform (chi2 {chi2:.1f})"
    # ---- first column uniform among the feasible ones GIVEN N (one chi-square per duration, summed)
    chi2, dof = 0.0, 0
    for n in range(n_min, n_max + 1):
        sel = j0[N == n]
        cells = n_t - n + 1
        c = np.bincount(sel, minlength=cells)
        chi2 += ((c - sel.size / cells) ** 2 / (sel.size / cells)).sum()
        dof += cells - 1
    assert chi2 < stats.chi2.ppf(1 - 1e-6, dof), f"j0 | N not uniform (chi2 {chi2:.1f}, dof {dof})"
    # ---- continuous parameters uniform on their ranges (Kolmogorov-Smirnov)
    u = np.column_stack([a / N, y / n_f, (tau - lo) / (hi - lo)])            # t_mid fraction, y0, y1, y2, tau
    for name, col in zip(("a/N", "y0", "y1", "y2", "tau"), u.T):
        p = stats.kstest(col, "uniform").pvalue
        assert p > 1e-6, f"{name} not uniform (KS p = {p:.2e})"
    # ---- pairwise independence of all seven parameters: correlation and a 4 x 4 contingency chi-square of
    # the uniformised variables (N and j0 are made uniform by their conditional ranks + a dither)
    rng = np.random.default_rng(5)
    uN = (N - n_min + rng.random(T)) / n_dur
    uj = (j0 + rng.random(T)) / (n_t - N + 1)
    U = np.column_stack([uN, uj, u])
    names = ("N", "j0", "a/N", "y0", "y1", "y2", "tau")
    corr = np.corrcoef(U.T)
    lim = stats.chi2.ppf(1 - 1e-7, 9)
    for i in range(7):
        for j in range(i + 1, 7):
            assert abs(corr[i, j]) < 5.0 / np.sqrt(T), f"{names[i]} and {names[j]} correlated ({corr[i, j]:.4f})"
            h = np.histogram2d(U[:, i], U[:, j], bins=4, range=[[0, 1], [0, 1]])[0]
            e = np.outer(h.sum(1), h.sum(0)) / T
            chi2 = ((h - e) ** 2 / e).sum()
            assert chi2 < lim, f"{names[i]} and {names[j]} dependent (chi2 {chi2:.1f})"
    # ---- consecutive ids are independent draws too (a counter that fails to enter the generator repeats)
    assert len({tuple(r) for r in s[:2000]}) == 2000
    assert abs(np.corrcoef(u[:-1, 1], u[1:, 1])[0, 1]) < 5.0 / np.sqrt(T)
    # ---- config 1: full-duration templates (BASELINE.json configs[0])
    full = sample(0, 0, 300, 64, 64, 64, 64, 0.0, 0.0)
    assert (full[:, 0] == 64).all() and (full[:, 1] == 0).all()
    # ---- a single feasible start when N = n_t, and N = 1 reaches every column
    one = sample(3, 0, 4000, 16, 8, 1, 1, 0.0, 0.0)
    assert set(one[:, 1].astype(int)) == set(range(16))
    # ---- seeds select different banks
    assert not np.array_equal(sample(1, 0, 50, n_t, n_f, n_min, n_max, lo, hi), sample(2, 0, 50, n_t, n_f, n_min, n_max, lo, hi))


def test_track_params_pinned(orc):
    check_track_param_pins(_sampler(C.CDLL(orc.build())))       # its own handle: argtypes are set on it


# One plausible slip per entry: (what goes wrong, regex on the oracle source, replacement).
SLIPS = [
    ("duration range one short (n_max never drawn)",
     r"\(uint64_t\)\(n_max - n_min \+ 1\)", "(uint64_t)(n_max - n_min)"),
    ("start range one short (the last feasible column never drawn)",
     r"\(uint64_t\)\(n_t - t->N \+ 1\)", "(uint64_t)(n_t - t->N)"),
    ("start range one too long (template leaves the map)",
     r"\(uint64_t\)\(n_t - t->N \+ 1\)", "(uint64_t)(n_t - t->N + 2)"),
    ("t_mid reuses the word of f_start (five random numbers, not six)",
     r"t->a  = \(\(double\)r\[2\]", "t->a  = ((double)r[3]"),
    ("the delay reuses the word of f_end",
     r"double u = \(\(double\)r\[6\]", "double u = ((double)r[5]"),
    ("start drawn for the shortest duration and clamped (not uniform given N)",
     r"t->j0 = \(int32_t\)\(\(\(uint64_t\)r\[1\] \* \(uint64_t\)\(n_t - t->N \+ 1\)\) >> 32\);",
     "t->j0 = (int32_t)(((uint64_t)r[1] * (uint64_t)(n_t - n_min + 1)) >> 32); if (t->j0 > n_t - t->N) t->j0 = n_t - t->N;"),
    ("t_mid fixed at the midpoint (G3 rejected reading)",
     r"t->a  = \(\(double\)r\[2\] \+ 0\.5\) \* \(double\)t->N \* two_m32;", "t->a  = 0.5 * (double)t->N;"),
    ("template id not entering the generator (every template the same)",
     r"or_track_words\(seed, id, r\);", "or_track_words(seed, 0, r);"),
]


@pytest.mark.parametrize("what,pattern,repl", SLIPS, ids=[s[0].split(" (")[0] for s in SLIPS])
def test_pins_catch_plausible_slips(what, pattern, repl, tmp_path):
    src = open(ORACLE_SRC).read()
    mutated, n = re.subn(pattern, repl, src, count=1)
    assert n == 1, f"slip pattern no longer matches the oracle source: {pattern}"
    c = tmp_path / "mutant.c"
    c.write_text(mutated)
    so = tmp_path / "mutant.so"
    subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-std=c99", str(c), "-o", str(so), "-lm"])
    with pytest.raises(AssertionError):
        check_track_param_pins(_sampler(C.CDLL(str(so))))

"""ctypes front end of the float64 CPU oracle (oracle/stochtrack_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It holds
argument marshalling only; every step of the method (O1-O5) is in
the C file, which cites the passages of PAPER.md it follows.  Nothing here imports
the CUDA package, and the CUDA package imports nothing from here.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "stochtrack_oracle.c")
_LIB = os.path.join(_HERE, "libstochtrack_oracle.so")
# -ffp-contract=off: the rasteriser is a normative no-FMA double sequence (G15).
CFLAGS = ["-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-std=c99"]


def build(force=False):
    """Compile the oracle with gcc (no CUDA involved). Returns the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", *CFLAGS, _SRC, "-o", _LIB, "-lm"])
    return _LIB


class Track(C.Structure):
    _fields_ = [("N", C.c_int32), ("j0", C.c_int32), ("a", C.c_double),
                ("y0", C.c_double), ("y1", C.c_double), ("y2", C.c_double),
                ("tau", C.c_double), ("y3", C.c_double), ("family", C.c_int32)]

    def as_dict(self):
        return {f: getattr(self, f) for f, _ in self._fields_}


class _SearchParams(C.Structure):
    _fields_ = [("n_tracks", C.c_uint64), ("track_offset", C.c_uint64), ("seed", C.c_uint64),
                ("n_min", C.c_int32), ("n_max", C.c_int32),
                ("tau_mode", C.c_int32), ("n_tau", C.c_int32),
                ("tau_lo", C.c_double), ("tau_hi", C.c_double),
                ("norm_mode", C.c_int32), ("n_bins", C.c_int32),
                ("hist_lo", C.c_double), ("hist_hi", C.c_double),
                ("score_mode", C.c_int32), ("n_threads", C.c_int32),
                ("family", C.c_int32), ("pad", C.c_int32)]


class _SearchResult(C.Structure):
    _fields_ = [("max_snr", C.c_double), ("arg_track", C.c_uint64),
                ("arg_tau_index", C.c_int32), ("arg_tau", C.c_double),
                ("n_evals", C.c_uint64), ("n_pixels", C.c_uint64),
                ("threads_used", C.c_int32)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        u32p, i32p, f64p, f32p, u64p = (C.POINTER(t) for t in
                                        (C.c_uint32, C.c_int32, C.c_double, C.c_float, C.c_uint64))
        L.or_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.or_track_words.argtypes = [C.c_uint64, C.c_uint64, u32p]
        L.or_track_params.argtypes = [C.c_uint64, C.c_uint64, C.c_int32, C.c_int32, C.c_int32,
                                      C.c_int32, C.c_double, C.c_double, C.POINTER(Track)]
        L.or_track_params.restype = C.c_int
        L.or_track_params_family.argtypes = [C.c_uint64, C.c_uint64, C.c_int32, C.c_int32, C.c_int32,
                                             C.c_int32, C.c_double, C.c_double, C.c_int32, C.POINTER(Track)]
        L.or_track_params_family.restype = C.c_int
        L.or_prepare_inv_sigma.argtypes = [f32p, C.c_int, C.c_int32, C.c_int32, f64p]
        L.or_score_direct_w.argtypes = [f64p, f64p, C.c_int32, C.POINTER(Track), i32p, C.c_double, C.c_double, C.c_double]
        L.or_score_direct_w.restype = C.c_double
        L.or_score_table_w.argtypes = [f64p, f64p, C.c_int32, C.POINTER(Track), i32p, f64p, C.c_int32, f64p]
        L.or_rasterise.argtypes = [C.POINTER(Track), C.c_int32, i32p]
        L.or_prepare_map.argtypes = [f32p, f32p, C.c_int, C.c_int32, C.c_int32, f64p]
        L.or_score_direct.argtypes = [f64p, C.c_int32, C.POINTER(Track), i32p,
                                      C.c_double, C.c_double, C.c_double, C.c_int]
        L.or_score_direct.restype = C.c_double
        L.or_build_table.argtypes = [C.c_int32, C.c_double, C.c_double, f64p, C.c_int32, f64p]
        L.or_score_table.argtypes = [f64p, C.c_int32, C.POINTER(Track), i32p, f64p, C.c_int32,
                                     C.c_int, f64p]
        L.or_search.argtypes = [f64p, C.c_int32, C.c_int32, C.c_double, C.c_double, f64p,
                                C.POINTER(_SearchParams), C.POINTER(_SearchResult),
                                u64p, f64p, i32p, i32p, i32p, f64p]
        L.or_search.restype = C.c_int
        _lib = L
    return _lib


def _p(a, ctype):
    return a.ctypes.data_as(C.POINTER(ctype)) if a is not None else None


NORM_SQRT_N, NORM_MEAN, NORM_INVVAR = 0, 1, 2
FAMILY_QUADRATIC, FAMILY_CUBIC, FAMILY_CHIRP = 0, 1, 2
TAU_GRID, TAU_RANDOM = 0, 1


def philox4x32_10(ctr, key):
    c = np.ascontiguousarray(ctr, dtype=np.uint32)
    k = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().or_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(out, C.c_uint32))
    return out


def track_words(seed, track_id):
    out = np.zeros(8, dtype=np.uint32)
    lib().or_track_words(seed, track_id, _p(out, C.c_uint32))
    return out


def track_params(seed, track_id, n_t, n_f, n_min, n_max, tau_lo=0.0, tau_hi=0.0, family=FAMILY_QUADRATIC):
    t = Track()
    if family == FAMILY_QUADRATIC:
        rc = lib().or_track_params(seed, track_id, n_t, n_f, n_min, n_max, tau_lo, tau_hi, C.byref(t))
    else:
        rc = lib().or_track_params_family(seed, track_id, n_t, n_f, n_min, n_max, tau_lo, tau_hi, family, C.byref(t))
    if rc != 0:
        raise ValueError("or_track_params: invalid arguments")
    return t


def make_track(N, j0, a, y0, y1, y2, tau=0.0, y3=None, family=None):
    """A quadratic template (Eq. 6), or with y3 a cubic one: frequency control points y0, y1, y2, y3 (G26);
    family=FAMILY_CHIRP: the chirp-law template of G27 (N, j0, a, y0 are used)."""
    if family == FAMILY_CHIRP:
        return Track(int(N), int(j0), float(a), float(y0), float(y1), float(y2), float(tau), 0.0, FAMILY_CHIRP)
    if y3 is None:
        return Track(int(N), int(j0), float(a), float(y0), float(y1), float(y2), float(tau), 0.0, FAMILY_QUADRATIC)
    return Track(int(N), int(j0), float(a), float(y0), float(y1), float(y2), float(tau), float(y3), FAMILY_CUBIC)


def rasterise(track, n_f):
    k = np.zeros(track.N, dtype=np.int32)
    lib().or_rasterise(C.byref(track), n_f, _p(k, C.c_int32))
    return k


def prepare_map(csd, sigma=None):
    """p = CSD / sigma (Eq. 7) as float64 [n_t][n_f] complex128 view."""
    csd = np.ascontiguousarray(csd, dtype=np.complex64)
    n_t, n_f = csd.shape
    kind = 0
    s = None
    if sigma is not None:
        s = np.ascontiguousarray(sigma, dtype=np.float32)
        if s.shape == (n_f,):
            kind = 1
        elif s.shape == (n_t, n_f):
            kind = 2
        else:
            raise ValueError("sigma must be None, [n_f] or [n_t][n_f]")
    p = np.zeros((n_t, n_f), dtype=np.complex128)
    lib().or_prepare_map(_p(csd.view(np.float32), C.c_float), _p(s, C.c_float), kind, n_t, n_f,
                         _p(p.view(np.float64), C.c_double))
    return p


def prepare_inv_sigma(shape, sigma=None):
    """1 / sigma per pixel as float64 [n_t][n_f] (0 where the pixel is masked, G11): the weights of O4w."""
    n_t, n_f = shape
    kind, s = 0, None
    if sigma is not None:
        s = np.ascontiguousarray(sigma, dtype=np.float32)
        kind = 1 if s.shape == (n_f,) else 2
        if s.shape not in ((n_f,), (n_t, n_f)):
            raise ValueError("sigma must be None, [n_f] or [n_t][n_f]")
    r = np.zeros((n_t, n_f), dtype=np.float64)
    lib().or_prepare_inv_sigma(_p(s, C.c_float), kind, n_t, n_f, _p(r, C.c_double))
    return r


def score_direct_w(p, inv_sigma, track, k, f_min, df, tau):
    """Inverse-variance weighted statistic (fn. 23, G25) of one template at one delay."""
    p = np.ascontiguousarray(p, dtype=np.complex128)
    r = np.ascontiguousarray(inv_sigma, dtype=np.float64)
    k = np.ascontiguousarray(k, dtype=np.int32)
    return lib().or_score_direct_w(_p(p.view(np.float64), C.c_double), _p(r, C.c_double), p.shape[1], C.byref(track),
                                   _p(k, C.c_int32), f_min, df, tau)


def score_table_w(p, inv_sigma, track, k, W):
    p = np.ascontiguousarray(p, dtype=np.complex128)
    r = np.ascontiguousarray(inv_sigma, dtype=np.float64)
    k = np.ascontiguousarray(k, dtype=np.int32)
    W = np.ascontiguousarray(W, dtype=np.complex128)
    snr = np.zeros(W.shape[1], dtype=np.float64)
    lib().or_score_table_w(_p(p.view(np.float64), C.c_double), _p(r, C.c_double), p.shape[1], C.byref(track),
                           _p(k, C.c_int32), _p(W.view(np.float64), C.c_double), W.shape[1], _p(snr, C.c_double))
    return snr


def score_direct(p, track, k, f_min, df, tau, norm=NORM_SQRT_N):
    p = np.ascontiguousarray(p, dtype=np.complex128)
    k = np.ascontiguousarray(k, dtype=np.int32)
    return lib().or_score_direct(_p(p.view(np.float64), C.c_double), p.shape[1], C.byref(track),
                                 _p(k, C.c_int32), f_min, df, tau, norm)


def build_table(n_f, f_min, df, tau_grid):
    tau = np.ascontiguousarray(tau_grid, dtype=np.float64)
    W = np.zeros((n_f, tau.size), dtype=np.complex128)
    lib().or_build_table(n_f, f_min, df, _p(tau, C.c_double), tau.size,
                         _p(W.view(np.float64), C.c_double))
    return W


def score_table(p, track, k, W, norm=NORM_SQRT_N):
    p = np.ascontiguousarray(p, dtype=np.complex128)
    k = np.ascontiguousarray(k, dtype=np.int32)
    W = np.ascontiguousarray(W, dtype=np.complex128)
    snr = np.zeros(W.shape[1], dtype=np.float64)
    lib().or_score_table(_p(p.view(np.float64), C.c_double), p.shape[1], C.byref(track),
                         _p(k, C.c_int32), _p(W.view(np.float64), C.c_double), W.shape[1], norm,
                         _p(snr, C.c_double))
    return snr


def search(p, f_min, df, n_tracks, seed, n_min, n_max, tau_grid=None, tau_range=None,
           norm=NORM_SQRT_N, n_bins=0, hist_lo=-10.0, hist_hi=10.0, track_offset=0,
           score_mode=0, n_threads=0, dump_snr=False, dump_tracks=False, family=FAMILY_QUADRATIC,
           inv_sigma=None):
    """Whole path O1-O5 for ids [track_offset, track_offset + n_tracks).

    tau_grid (array) selects grid mode; tau_range=(lo, hi) selects the paper's
    random-tau mode.  family selects the template family (G26, G27); norm=NORM_INVVAR
    the inverse-variance weighting (G25) and then needs inv_sigma = prepare_inv_sigma(...).
    Returns a dict.
    """
    p = np.ascontiguousarray(p, dtype=np.complex128)
    n_t, n_f = p.shape
    sp = _SearchParams()
    sp.n_tracks, sp.track_offset, sp.seed = int(n_tracks), int(track_offset), int(seed)
    sp.n_min, sp.n_max = int(n_min), int(n_max)
    tau = None
    if tau_grid is not None:
        tau = np.ascontiguousarray(tau_grid, dtype=np.float64)
        sp.tau_mode, sp.n_tau = TAU_GRID, tau.size
    else:
        sp.tau_mode, sp.n_tau = TAU_RANDOM, 1
        sp.tau_lo, sp.tau_hi = float(tau_range[0]), float(tau_range[1])
    sp.norm_mode, sp.n_bins = int(norm), int(n_bins)
    sp.hist_lo, sp.hist_hi = float(hist_lo), float(hist_hi)
    sp.score_mode, sp.n_threads = int(score_mode), int(n_threads)
    sp.family = int(family)
    rs = None
    if int(norm) == NORM_INVVAR:
        if inv_sigma is None:
            raise ValueError("norm=NORM_INVVAR needs inv_sigma")
        rs = np.ascontiguousarray(inv_sigma, dtype=np.float64)
        if rs.shape != (n_t, n_f):
            raise ValueError("inv_sigma must be [n_t][n_f]")
    n_tau = sp.n_tau
    hist = np.zeros(n_bins, dtype=np.uint64) if n_bins > 0 else None
    snr = np.zeros((n_tracks, n_tau), dtype=np.float64) if dump_snr else None
    kd = np.zeros((n_tracks, n_t), dtype=np.int32) if dump_tracks else None
    j0 = np.zeros(n_tracks, dtype=np.int32) if dump_tracks else None
    Nn = np.zeros(n_tracks, dtype=np.int32) if dump_tracks else None
    res = _SearchResult()
    rc = lib().or_search(_p(p.view(np.float64), C.c_double), n_t, n_f, f_min, df,
                         _p(tau, C.c_double), C.byref(sp), C.byref(res),
                         _p(hist, C.c_uint64), _p(snr, C.c_double),
                         _p(kd, C.c_int32), _p(j0, C.c_int32), _p(Nn, C.c_int32), _p(rs, C.c_double))
    if rc != 0:
        raise ValueError(f"or_search failed with {rc}")
    return {"max_snr": res.max_snr, "arg_track": int(res.arg_track),
            "arg_tau_index": int(res.arg_tau_index), "arg_tau": res.arg_tau,
            "n_evals": int(res.n_evals), "n_pixels": int(res.n_pixels),
            "threads_used": int(res.threads_used), "hist": hist, "snr": snr,
            "k": kd, "j0": j0, "N": Nn, "track_offset": int(track_offset)}


def search_batch(csd_maps, sigma_maps, seeds, f_min, df, n_tracks, n_min, n_max, **kw):
    """Batch / background mode: the background of the search is estimated from many (time-shifted)
    maps, each searched on its own with its own template bank (PAPER.md:173, :232-234, :346
    "different random seed for each run").  By definition a loop: map m -> O0 (prepare_map) and
    O1-O5 (search) with seed seeds[m].  Returns the list of per-map result dicts."""
    out = []
    for m, csd in enumerate(csd_maps):
        sig = None if sigma_maps is None else sigma_maps[m]
        p = prepare_map(csd, sig)
        seed = int(seeds[m]) if np.ndim(seeds) else int(seeds)
        kw_m = dict(kw)
        if kw.get("norm", NORM_SQRT_N) == NORM_INVVAR:
            kw_m["inv_sigma"] = prepare_inv_sigma(p.shape, sig)
        out.append(search(p, f_min, df, n_tracks, seed, n_min, n_max, **kw_m))
    return out


def top_k(result, k):
    """The k loudest (template, delay) samples of a `search(..., dump_snr=True)` result, in the G12 total
    order (larger SNR, then smaller template id, then smaller delay index): the events a follow-up looks
    at.  Plain sort of the dumped SNR array.  Returns [(track, tau_index, snr)]."""
    snr = result["snr"]
    n_tracks, n_tau = snr.shape
    first = result["track_offset"]                     # ids are global: row q of the dump is template first + q
    flat = snr.ravel()
    ids = np.repeat(np.arange(n_tracks, dtype=np.int64), n_tau)
    ms = np.tile(np.arange(n_tau, dtype=np.int64), n_tracks)
    order = np.lexsort((ms, ids, -flat))[:k]
    return [(int(first + ids[i]), int(ms[i]), float(flat[i])) for i in order]

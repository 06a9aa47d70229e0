"""ctypes binding of include/stochtrack.h.  Marshalling only; PyTorch supplies
device memory and the CUDA stream (nothing else)."""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libstochtrack_b200.so")

ST_OK, ST_EINVAL, ST_ESTATE, ST_ENOSPC, ST_ECUDA = 0, -1, -2, -3, -4
_CODES = {ST_EINVAL: "ST_EINVAL", ST_ESTATE: "ST_ESTATE", ST_ENOSPC: "ST_ENOSPC", ST_ECUDA: "ST_ECUDA"}
SIGMA_NONE, SIGMA_PER_FREQ, SIGMA_PER_PIXEL = 0, 1, 2
TAU_GRID, TAU_RANDOM = 0, 1
NORM_SQRT_N, NORM_MEAN, NORM_INVVAR = 0, 1, 2
FAMILY_QUADRATIC, FAMILY_CUBIC, FAMILY_CHIRP = 0, 1, 2
KERNEL_AUTO, KERNEL_TABLE, KERNEL_ROTATION, KERNEL_REINSCH, KERNEL_RANDOM, KERNEL_CHEBYSHEV = 0, 1, 2, 3, 4, 5
KERNEL_NAMES = {0: "auto", 1: "table", 2: "rotation", 3: "reinsch", 4: "random", 5: "chebyshev"}

# every symbol include/stochtrack.h declares
exported_symbols = ("st_create", "st_destroy", "st_workspace_bytes", "st_set_workspace", "st_set_map",
                    "st_set_map_host", "st_search", "st_search_topk", "st_search_batch", "st_search_track_max",
                    "st_score_tracks", "st_debug_rasterise_random", "st_bank_cache_bytes", "st_set_bank_cache", "st_ftmap_scratch_bytes", "st_set_map_from_strain", "st_search_timeshifts",
                    "st_debug_get_map",
                    "st_track_params", "st_track_params_family", "st_debug_rasterise",
                    "st_debug_rasterise_track", "st_debug_scores", "st_debug_track_words",
                    "st_score_random_noalloc", "st_combine_results",
                    "st_last_error", "st_version")


class StError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{_CODES.get(code, code)}: {msg}")
        self.code = code


class CTrack(C.Structure):
    _fields_ = [("N", C.c_int32), ("j0", C.c_int32), ("a", C.c_double), ("y0", C.c_double),
                ("y1", C.c_double), ("y2", C.c_double), ("tau", C.c_double), ("y3", C.c_double)]

    def as_dict(self):
        return {f: getattr(self, f) for f, _ in self._fields_}


class CSearchParams(C.Structure):
    _fields_ = [("n_tracks", C.c_uint64), ("track_offset", C.c_uint64), ("seed", C.c_uint64),
                ("n_min", C.c_int32), ("n_max", C.c_int32), ("tau_mode", C.c_int32), ("n_tau", C.c_int32),
                ("tau_grid", C.POINTER(C.c_double)), ("tau_lo", C.c_double), ("tau_hi", C.c_double),
                ("norm", C.c_int32), ("n_bins", C.c_int32), ("hist_lo", C.c_double), ("hist_hi", C.c_double),
                ("hist_out", C.POINTER(C.c_uint64)), ("kernel", C.c_int32), ("family", C.c_int32)]


class CResult(C.Structure):
    _fields_ = [("max_snr", C.c_float), ("arg_tau_index", C.c_int32), ("max_snr_f64", C.c_double),
                ("arg_track", C.c_uint64), ("arg_tau", C.c_double), ("arg_params", CTrack),
                ("n_evals", C.c_uint64), ("n_pixels", C.c_uint64), ("n_candidates", C.c_int32),
                ("kernel_used", C.c_int32), ("n_launches", C.c_int32), ("flags", C.c_int32),
                ("gpu_ms", C.c_float), ("n_deferred", C.c_int32)]


class CTopEntry(C.Structure):
    _fields_ = [("track", C.c_uint64), ("tau_index", C.c_int32), ("snr_f32", C.c_float), ("snr_f64", C.c_double),
                ("tau", C.c_double)]


MAX_TOP_K = 4096
MAX_SCORE_TRACKS = 4096


class CFtmapParams(C.Structure):
    _fields_ = [("fs", C.c_double), ("seg_len", C.c_int32), ("n_neighbours", C.c_int32)]


class CBatch(C.Structure):
    _fields_ = [("n_maps", C.c_int32), ("host_buffers", C.c_int32), ("csd", C.POINTER(C.c_void_p)),
                ("sigma", C.POINTER(C.c_void_p)), ("sigma_kind", C.c_int32), ("reserved", C.c_int32),
                ("seeds", C.POINTER(C.c_uint64))]


BATCH_GROUP = 256

_lib = None


def library_path():
    return _LIB_PATH


def load_library(path=None):
    """dlopen the C-ABI library.  Fails loudly when it has not been built.  `path` (first call only) names
    another build of the same C ABI, e.g. the -DST_CHECKED library of build.build_checked()."""
    global _lib, _LIB_PATH
    if _lib is not None:
        if path is not None and os.path.abspath(path) != os.path.abspath(_LIB_PATH):
            raise RuntimeError(f"a different library is already loaded: {_LIB_PATH}")
        return _lib
    if path is not None:
        _LIB_PATH = path
    if not os.path.exists(_LIB_PATH):
        raise ImportError(f"{_LIB_PATH} is missing: run `python -m paper_1401_8060_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(_LIB_PATH)
    vp = C.c_void_p
    L.st_create.argtypes = [C.POINTER(vp), C.c_int32, C.c_int32, C.c_double, C.c_double]
    L.st_destroy.argtypes = [vp]
    L.st_destroy.restype = None
    L.st_workspace_bytes.argtypes = [vp, C.c_int32]
    L.st_workspace_bytes.restype = C.c_size_t
    L.st_set_workspace.argtypes = [vp, vp, C.c_size_t, vp]
    L.st_set_map.argtypes = [vp, vp, vp, C.c_int32]
    L.st_set_map_host.argtypes = [vp, vp, vp, C.c_int32]
    L.st_search.argtypes = [vp, C.POINTER(CSearchParams), C.POINTER(CResult)]
    L.st_track_params.argtypes = [vp, C.c_uint64, C.c_uint64, C.c_int32, C.c_int32, C.c_double, C.c_double,
                                  C.POINTER(CTrack)]
    L.st_debug_rasterise.argtypes = [vp, C.POINTER(CSearchParams), C.c_uint64, C.c_uint64, vp, vp, vp]
    L.st_track_params_family.argtypes = [vp, C.c_uint64, C.c_uint64, C.c_int32, C.c_int32, C.c_double, C.c_double,
                                         C.c_int32, C.POINTER(CTrack)]
    L.st_track_params_family.restype = C.c_int
    L.st_debug_rasterise_track.argtypes = [vp, C.POINTER(CTrack), C.c_int32, vp]
    L.st_debug_scores.argtypes = [vp, C.POINTER(CSearchParams), C.c_uint64, C.c_uint64, vp]
    L.st_debug_track_words.argtypes = [C.c_uint64, C.c_uint64, C.POINTER(C.c_uint32)]
    L.st_last_error.argtypes = [vp]
    L.st_last_error.restype = C.c_char_p
    L.st_version.argtypes = []
    L.st_version.restype = C.c_char_p
    L.st_search_topk.argtypes = [vp, C.POINTER(CSearchParams), C.c_int32, C.POINTER(CTopEntry), C.POINTER(C.c_int32),
                                 C.POINTER(CResult)]
    L.st_search_topk.restype = C.c_int
    L.st_ftmap_scratch_bytes.argtypes = [vp, C.c_int32]
    L.st_ftmap_scratch_bytes.restype = C.c_size_t
    L.st_set_map_from_strain.argtypes = [vp, vp, vp, C.c_int64, C.POINTER(CFtmapParams), vp, C.c_size_t]
    L.st_set_map_from_strain.restype = C.c_int
    L.st_search_timeshifts.argtypes = [vp, vp, vp, C.c_int64, C.POINTER(CFtmapParams), vp, C.c_size_t, C.c_int32,
                                       C.POINTER(C.c_int32), C.POINTER(C.c_uint64), C.POINTER(CSearchParams),
                                       C.POINTER(CResult), C.POINTER(C.c_float)]
    L.st_search_timeshifts.restype = C.c_int
    L.st_debug_get_map.argtypes = [vp, vp]
    L.st_debug_get_map.restype = C.c_int
    L.st_search_batch.argtypes = [vp, C.POINTER(CBatch), C.POINTER(CSearchParams), C.POINTER(CResult), C.POINTER(C.c_float)]
    L.st_bank_cache_bytes.argtypes = [vp, C.c_uint64, C.c_int32]
    L.st_bank_cache_bytes.restype = C.c_size_t
    L.st_set_bank_cache.argtypes = [vp, vp, C.c_size_t]
    L.st_set_bank_cache.restype = C.c_int
    L.st_search_track_max.argtypes = [vp, C.POINTER(CSearchParams), vp, vp, C.POINTER(CResult)]
    L.st_search_track_max.restype = C.c_int
    L.st_score_tracks.argtypes = [vp, C.POINTER(CSearchParams), C.POINTER(CTrack), C.c_int32, vp]
    L.st_score_tracks.restype = C.c_int
    L.st_debug_rasterise_random.argtypes = [vp, C.POINTER(CSearchParams), C.c_uint64, C.c_uint64, vp, vp, vp]
    L.st_debug_rasterise_random.restype = C.c_int
    L.st_score_random_noalloc.argtypes = [vp, vp, C.c_int32, C.c_int32, C.c_int32, C.c_double, C.c_double,
                                          C.POINTER(CSearchParams), vp, vp, C.c_char_p, C.c_size_t]
    L.st_score_random_noalloc.restype = C.c_int
    L.st_combine_results.argtypes = [C.POINTER(CResult), C.POINTER(C.POINTER(C.c_uint64)), C.c_int32, C.c_int32,
                                     C.POINTER(CResult), C.POINTER(C.c_uint64), C.POINTER(C.c_int32)]
    L.st_combine_results.restype = C.c_int
    for name in ("st_create", "st_set_workspace", "st_set_map", "st_set_map_host", "st_search", "st_search_batch", "st_track_params",
                 "st_debug_rasterise", "st_debug_rasterise_track", "st_debug_scores", "st_debug_track_words"):
        getattr(L, name).restype = C.c_int
    _lib = L
    return L


def st_track_words(seed, track_id):
    out = (C.c_uint32 * 8)()
    rc = load_library().st_debug_track_words(seed, track_id, out)
    if rc:
        raise StError(rc, "st_debug_track_words")
    return np.array(list(out), dtype=np.uint32)


class SearchResult(dict):
    __getattr__ = dict.__getitem__


class Stochtrack:
    """One context = one map shape on one GPU / stream.  Mirrors the C ABI:
    st_create / st_workspace_bytes / st_set_workspace at construction, then
    set_map(), search(), and the parity exports."""

    def __init__(self, n_t, n_f, df, f_min, max_n_tau=512, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the stochtrack hot path has no CPU fallback")
        self._torch = torch
        self._L = load_library()
        self.n_t, self.n_f, self.df, self.f_min = int(n_t), int(n_f), float(df), float(f_min)
        self.device = torch.device(device)
        self._ctx = C.c_void_p()
        rc = self._L.st_create(C.byref(self._ctx), self.n_t, self.n_f, self.df, self.f_min)
        if rc:
            raise StError(rc, "st_create: invalid map shape / frequency axis")
        nbytes = self._L.st_workspace_bytes(self._ctx, int(max_n_tau))
        if nbytes == 0:
            raise StError(ST_EINVAL, "st_workspace_bytes: bad max_n_tau")
        with torch.cuda.device(self.device):
            self._ws = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.workspace_bytes = nbytes
        self._check(self._L.st_set_workspace(self._ctx, self._ws.data_ptr(), nbytes, self._stream.cuda_stream))
        self._keep = []

    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            self._L.st_destroy(self._ctx)
            self._ctx = C.c_void_p()

    __del__ = close

    def _check(self, rc):
        if rc:
            raise StError(rc, (self._L.st_last_error(self._ctx) or b"").decode())

    def synchronize(self):
        self._stream.synchronize()

    def enable_bank_cache(self, n_tracks, n_max):
        """Allocate and attach a bank cache for banks of n_tracks templates of at most n_max columns
        (st_bank_cache_bytes / st_set_bank_cache).  Returns its size in bytes."""
        nbytes = self._L.st_bank_cache_bytes(self._ctx, int(n_tracks), int(n_max))
        if nbytes == 0:
            raise StError(ST_EINVAL, "st_bank_cache_bytes: bad arguments")
        self._bank = self._torch.empty(nbytes, dtype=self._torch.uint8, device=self.device)
        self._check(self._L.st_set_bank_cache(self._ctx, self._bank.data_ptr(), nbytes))
        return nbytes

    def disable_bank_cache(self):
        self._check(self._L.st_set_bank_cache(self._ctx, None, 0))
        self._bank = None

    # ---------------------------------------------------------------- S0
    def set_map(self, csd, sigma=None):
        """csd: complex64 [n_t][n_f] torch CUDA tensor (device path) or numpy array /
        CPU tensor (host path: copied inside the C call).  sigma: None, [n_f] or [n_t][n_f] float32."""
        torch = self._torch
        kind = SIGMA_NONE
        if sigma is not None:
            shp = tuple(sigma.shape)
            kind = SIGMA_PER_FREQ if shp == (self.n_f,) else SIGMA_PER_PIXEL if shp == (self.n_t, self.n_f) else -1
            if kind < 0:
                raise ValueError("sigma must be None, [n_f] or [n_t][n_f]")
        if tuple(csd.shape) != (self.n_t, self.n_f):
            raise ValueError("csd must be [n_t][n_f]")
        if isinstance(csd, torch.Tensor) and csd.is_cuda:
            if csd.dtype != torch.complex64 or not csd.is_contiguous():
                raise ValueError("csd must be a contiguous complex64 tensor")
            sp = 0
            if sigma is not None:
                if not (isinstance(sigma, torch.Tensor) and sigma.is_cuda and sigma.dtype == torch.float32
                        and sigma.is_contiguous()):
                    raise ValueError("sigma must be a contiguous float32 CUDA tensor")
                sp = sigma.data_ptr()
            self._check(self._L.st_set_map(self._ctx, csd.data_ptr(), sp, kind))
            self._keep = [csd, sigma]          # inputs must outlive the stream-ordered call
        else:
            c = csd.numpy() if isinstance(csd, torch.Tensor) else np.ascontiguousarray(csd, dtype=np.complex64)
            s = None
            if sigma is not None:
                s = sigma.numpy() if isinstance(sigma, torch.Tensor) else np.ascontiguousarray(sigma, dtype=np.float32)
            if c.dtype != np.complex64 or (s is not None and s.dtype != np.float32):
                raise ValueError("host csd must be complex64 and sigma float32")
            self._check(self._L.st_set_map_host(self._ctx, c.ctypes.data, s.ctypes.data if s is not None else 0, kind))

    def set_map_from_strain(self, s_i, s_j, fs, seg_len, n_neighbours=4):
        """ft-map construction on the device (st_set_map_from_strain): s_i, s_j float64 CUDA tensors of
        the two strain series; the context's map becomes p = lambda s~_I^* s~_J (Eqs. 7, A4)."""
        torch = self._torch
        for x in (s_i, s_j):
            if not (isinstance(x, torch.Tensor) and x.is_cuda and x.dtype == torch.float64 and x.is_contiguous() and x.dim() == 1):
                raise ValueError("strain series must be contiguous 1-D float64 CUDA tensors")
        if s_i.numel() != s_j.numel():
            raise ValueError("the two strain series must have the same length")
        need = self._L.st_ftmap_scratch_bytes(self._ctx, int(seg_len))
        if need == 0:
            raise StError(ST_EINVAL, "st_ftmap_scratch_bytes: bad seg_len")
        if getattr(self, "_ft_scratch", None) is None or self._ft_scratch.numel() < need:
            self._ft_scratch = torch.empty(need, dtype=torch.uint8, device=self.device)
        fp = CFtmapParams(float(fs), int(seg_len), int(n_neighbours))
        self._check(self._L.st_set_map_from_strain(self._ctx, s_i.data_ptr(), s_j.data_ptr(), s_i.numel(), C.byref(fp),
                                                   self._ft_scratch.data_ptr(), self._ft_scratch.numel()))
        self._keep = [s_i, s_j]

    def _ft_args(self, s_i, s_j, seg_len):
        torch = self._torch
        for x in (s_i, s_j):
            if not (isinstance(x, torch.Tensor) and x.is_cuda and x.dtype == torch.float64 and x.is_contiguous() and x.dim() == 1):
                raise ValueError("strain series must be contiguous 1-D float64 CUDA tensors")
        if s_i.numel() != s_j.numel():
            raise ValueError("the two strain series must have the same length")
        need = self._L.st_ftmap_scratch_bytes(self._ctx, int(seg_len))
        if need == 0:
            raise StError(ST_EINVAL, "st_ftmap_scratch_bytes: bad seg_len")
        if getattr(self, "_ft_scratch", None) is None or self._ft_scratch.numel() < need:
            self._ft_scratch = torch.empty(need, dtype=torch.uint8, device=self.device)

    def search_timeshifts(self, s_i, s_j, fs, seg_len, n_neighbours, shifts, seeds, n_tracks, n_min, n_max,
                          tau_grid=None, tau_range=None, norm=NORM_SQRT_N, n_bins=0, hist_lo=-10.0, hist_hi=10.0,
                          track_offset=0, kernel=KERNEL_AUTO, family=FAMILY_QUADRATIC):
        """Time-shift background from strain (st_search_timeshifts): spectrograms once, one map and one
        search per whole-segment shift of detector J.  Returns (list of SearchResult, gpu_ms_total)."""
        self._ft_args(s_i, s_j, seg_len)
        sh = np.ascontiguousarray(shifts, dtype=np.int32)
        n = sh.size
        fp = CFtmapParams(float(fs), int(seg_len), int(n_neighbours))
        seed0, sd_p = 0, None
        if np.ndim(seeds) == 0:
            seed0 = int(seeds)
        else:
            sd = np.ascontiguousarray(seeds, dtype=np.uint64)
            if sd.size != n:
                raise ValueError("seeds: one per shift")
            sd_p = sd.ctypes.data_as(C.POINTER(C.c_uint64))
        p, keep = self._params(n_tracks, seed0, n_min, n_max, tau_grid, tau_range, norm, n_bins, hist_lo, hist_hi,
                               track_offset, kernel, family)
        hist = None
        if n_bins > 0:
            hist = np.zeros((n, n_bins), dtype=np.uint64)
            p.hist_out = hist.ctypes.data_as(C.POINTER(C.c_uint64))
        res = (CResult * n)()
        ms = C.c_float(0.0)
        self._check(self._L.st_search_timeshifts(self._ctx, s_i.data_ptr(), s_j.data_ptr(), s_i.numel(), C.byref(fp),
                                                 self._ft_scratch.data_ptr(), self._ft_scratch.numel(), n,
                                                 sh.ctypes.data_as(C.POINTER(C.c_int32)), sd_p, C.byref(p), res, C.byref(ms)))
        return [self._result(res[m], hist[m] if hist is not None else None) for m in range(n)], float(ms.value)

    def debug_get_map(self):
        """The context's current map p as a complex64 numpy array [n_t][n_f] (parity export)."""
        torch = self._torch
        out = torch.empty((self.n_t, self.n_f), dtype=torch.complex64, device=self.device)
        self._check(self._L.st_debug_get_map(self._ctx, out.data_ptr()))
        self.synchronize()
        return out.cpu().numpy()

    def debug_strain_spectra(self):
        """s~_I, s~_J (complex128 [n_t][n_f]) left in the scratch buffer by set_map_from_strain."""
        torch = self._torch
        self.synchronize()
        n = self.n_t * self.n_f
        stride = (n * 16 + 255) // 256 * 256
        raw = self._ft_scratch
        a = raw[:n * 16].view(torch.complex128).reshape(self.n_t, self.n_f).cpu().numpy()
        b = raw[stride:stride + n * 16].view(torch.complex128).reshape(self.n_t, self.n_f).cpu().numpy()
        return a, b

    # ------------------------------------------------------------ S1-S4
    def _params(self, n_tracks, seed, n_min, n_max, tau_grid, tau_range, norm, n_bins, hist_lo, hist_hi,
                track_offset, kernel, family=FAMILY_QUADRATIC):
        p = CSearchParams()
        p.n_tracks, p.track_offset, p.seed = int(n_tracks), int(track_offset), int(seed)
        p.n_min, p.n_max = int(n_min), int(n_max)
        keep = []
        if tau_grid is not None:
            g = np.ascontiguousarray(tau_grid, dtype=np.float64)
            keep.append(g)
            p.tau_mode, p.n_tau = TAU_GRID, g.size
            p.tau_grid = g.ctypes.data_as(C.POINTER(C.c_double))
        else:
            p.tau_mode, p.n_tau = TAU_RANDOM, 1
            p.tau_lo, p.tau_hi = float(tau_range[0]), float(tau_range[1])
        p.norm, p.n_bins = int(norm), int(n_bins)
        p.hist_lo, p.hist_hi = float(hist_lo), float(hist_hi)
        p.kernel = int(kernel)
        p.family = int(family)
        return p, keep

    def search(self, n_tracks, seed, n_min, n_max, tau_grid=None, tau_range=None, norm=NORM_SQRT_N,
               n_bins=0, hist_lo=-10.0, hist_hi=10.0, track_offset=0, kernel=KERNEL_AUTO, family=FAMILY_QUADRATIC):
        p, keep = self._params(n_tracks, seed, n_min, n_max, tau_grid, tau_range, norm, n_bins, hist_lo, hist_hi,
                               track_offset, kernel, family)
        hist = None
        if n_bins > 0:
            hist = np.zeros(n_bins, dtype=np.uint64)
            p.hist_out = hist.ctypes.data_as(C.POINTER(C.c_uint64))
        r = CResult()
        self._check(self._L.st_search(self._ctx, C.byref(p), C.byref(r)))
        return self._result(r, hist)

    def search_track_max(self, n_tracks, seed, n_min, n_max, tau_grid=None, tau_range=None, norm=NORM_SQRT_N,
                         n_bins=0, hist_lo=-10.0, hist_hi=10.0, track_offset=0, kernel=KERNEL_AUTO, family=FAMILY_QUADRATIC):
        """st_search_track_max: the search result plus, per template, its maximum over the delays and the delay
        index attaining it.  Returns (SearchResult, snr_max float32 [n_tracks], tau_index int32 [n_tracks])."""
        torch = self._torch
        p, keep = self._params(n_tracks, seed, n_min, n_max, tau_grid, tau_range, norm, n_bins, hist_lo, hist_hi,
                               track_offset, kernel, family)
        hist = None
        if n_bins > 0:
            hist = np.zeros(n_bins, dtype=np.uint64)
            p.hist_out = hist.ctypes.data_as(C.POINTER(C.c_uint64))
        snr = torch.empty(max(int(n_tracks), 1), dtype=torch.float32, device=self.device)
        idx = torch.empty(max(int(n_tracks), 1), dtype=torch.int32, device=self.device)
        r = CResult()
        self._check(self._L.st_search_track_max(self._ctx, C.byref(p), snr.data_ptr(), idx.data_ptr(), C.byref(r)))
        return self._result(r, hist), snr[:int(n_tracks)].cpu().numpy(), idx[:int(n_tracks)].cpu().numpy()

    def score_tracks(self, tracks, tau_grid=None, tau_range=None, norm=NORM_SQRT_N, kernel=KERNEL_AUTO, family=FAMILY_QUADRATIC):
        """st_score_tracks: Eq. 8 for explicit templates.  tracks: sequence of (N, j0, a, y0, y1, y2[, tau[, y3]]).
        Returns float32 [count][n_tau] (n_tau = 1 in random mode, where each template's own tau is its delay)."""
        torch = self._torch
        n = len(tracks)
        arr = (CTrack * max(n, 1))()
        for i, t in enumerate(tracks):
            arr[i] = CTrack(int(t[0]), int(t[1]), float(t[2]), float(t[3]), float(t[4]), float(t[5]),
                            float(t[6]) if len(t) > 6 else 0.0, float(t[7]) if len(t) > 7 else 0.0)
        p, keep = self._params(n, 0, 1, 1, tau_grid, tau_range if tau_range is not None else (0.0, 0.0), norm, 0, -10.0, 10.0, 0, kernel, family)
        n_tau = p.n_tau if p.tau_mode == TAU_GRID else 1
        snr = torch.empty((max(n, 1), n_tau), dtype=torch.float32, device=self.device)
        self._check(self._L.st_score_tracks(self._ctx, C.byref(p), arr, n, snr.data_ptr()))
        return snr[:n].cpu().numpy()

    def search_topk(self, top_k, n_tracks, seed, n_min, n_max, tau_grid=None, tau_range=None, norm=NORM_SQRT_N,
                    n_bins=1000, hist_lo=-10.0, hist_hi=10.0, track_offset=0, kernel=KERNEL_AUTO, family=FAMILY_QUADRATIC):
        """The top_k loudest (template, delay) samples (st_search_topk).  Returns (SearchResult, list of
        dicts {track, tau_index, snr_f32, snr_f64, tau} in the G12 order)."""
        p, keep = self._params(n_tracks, seed, n_min, n_max, tau_grid, tau_range, norm, n_bins, hist_lo, hist_hi,
                               track_offset, kernel, family)
        hist = np.zeros(max(n_bins, 1), dtype=np.uint64)
        p.hist_out = hist.ctypes.data_as(C.POINTER(C.c_uint64))
        top = (CTopEntry * int(top_k))()
        n_out = C.c_int32(0)
        r = CResult()
        self._check(self._L.st_search_topk(self._ctx, C.byref(p), int(top_k), top, C.byref(n_out), C.byref(r)))
        entries = [dict(track=int(e.track), tau_index=int(e.tau_index), snr_f32=float(e.snr_f32),
                        snr_f64=float(e.snr_f64), tau=float(e.tau)) for e in top[:n_out.value]]
        return self._result(r, hist), entries

    @staticmethod
    def _result(r, hist):
        return SearchResult(max_snr=float(r.max_snr), max_snr_f64=float(r.max_snr_f64), arg_track=int(r.arg_track),
                            arg_tau_index=int(r.arg_tau_index), arg_tau=float(r.arg_tau),
                            arg_params=r.arg_params.as_dict(), n_evals=int(r.n_evals), n_pixels=int(r.n_pixels),
                            n_candidates=int(r.n_candidates), kernel_used=int(r.kernel_used),
                            kernel_name=KERNEL_NAMES.get(int(r.kernel_used), "?"), n_launches=int(r.n_launches),
                            flags=int(r.flags), gpu_ms=float(r.gpu_ms), n_deferred=int(r.n_deferred), hist=hist)

    def search_batch(self, csd_maps, sigma_maps, seeds, n_tracks, n_min, n_max, tau_grid=None, tau_range=None,
                     norm=NORM_SQRT_N, n_bins=0, hist_lo=-10.0, hist_hi=10.0, track_offset=0, kernel=KERNEL_AUTO, family=FAMILY_QUADRATIC):
        """Batch / background mode (st_search_batch): one call over many maps.

        csd_maps: sequence of complex64 [n_t][n_f] maps, all torch CUDA tensors (device path) or all
        numpy arrays / CPU tensors (host path; pinned tensors let the copies overlap the searches).
        sigma_maps: None or a sequence of the same length (all [n_f] or all [n_t][n_f], float32).
        seeds: one template seed per map, or a single int used for every map.
        Returns (list of SearchResult, gpu_ms_total); result.hist is the map's own histogram."""
        torch = self._torch
        n_maps = len(csd_maps)
        on_dev = isinstance(csd_maps[0], torch.Tensor) and csd_maps[0].is_cuda
        kind = SIGMA_NONE
        if sigma_maps is not None:
            shp = tuple(sigma_maps[0].shape)
            kind = SIGMA_PER_FREQ if shp == (self.n_f,) else SIGMA_PER_PIXEL if shp == (self.n_t, self.n_f) else -1
            if kind < 0 or len(sigma_maps) != n_maps:
                raise ValueError("sigma_maps: one [n_f] or [n_t][n_f] array per map")
        keep, cp, sp = [], (C.c_void_p * n_maps)(), (C.c_void_p * n_maps)()

        def ptr(x, dt_t, dt_n, shape):
            if tuple(x.shape) != shape:
                raise ValueError(f"expected shape {shape}, got {tuple(x.shape)}")
            if isinstance(x, torch.Tensor):
                if x.is_cuda != on_dev or x.dtype != dt_t or not x.is_contiguous():
                    raise ValueError("maps of a batch must be contiguous, of one dtype, and all on one side")
                keep.append(x)
                return x.data_ptr()
            if on_dev:
                raise ValueError("maps of a batch must all be CUDA tensors or all host arrays")
            a = np.ascontiguousarray(x, dtype=dt_n)
            keep.append(a)
            return a.ctypes.data

        for m in range(n_maps):
            cp[m] = ptr(csd_maps[m], torch.complex64, np.complex64, (self.n_t, self.n_f))
            if kind != SIGMA_NONE:
                sp[m] = ptr(sigma_maps[m], torch.float32, np.float32, tuple(sigma_maps[0].shape))
        b = CBatch()
        b.n_maps, b.host_buffers, b.sigma_kind = n_maps, 0 if on_dev else 1, kind
        b.csd = C.cast(cp, C.POINTER(C.c_void_p))
        b.sigma = C.cast(sp, C.POINTER(C.c_void_p)) if kind != SIGMA_NONE else None
        seed0 = 0
        if np.ndim(seeds) == 0:
            seed0 = int(seeds)
        else:
            sd = np.ascontiguousarray(seeds, dtype=np.uint64)
            if sd.size != n_maps:
                raise ValueError("seeds: one per map")
            keep.append(sd)
            b.seeds = sd.ctypes.data_as(C.POINTER(C.c_uint64))
        p, k2 = self._params(n_tracks, seed0, n_min, n_max, tau_grid, tau_range, norm, n_bins, hist_lo, hist_hi,
                             track_offset, kernel, family)
        hist = None
        if n_bins > 0:
            hist = np.zeros((n_maps, n_bins), dtype=np.uint64)
            p.hist_out = hist.ctypes.data_as(C.POINTER(C.c_uint64))
        res = (CResult * n_maps)()
        ms = C.c_float(0.0)
        self._check(self._L.st_search_batch(self._ctx, C.byref(b), C.byref(p), res, C.byref(ms)))
        return [self._result(res[m], hist[m] if hist is not None else None) for m in range(n_maps)], float(ms.value)

    def track_params(self, seed, track_id, n_min, n_max, tau_lo=0.0, tau_hi=0.0, family=FAMILY_QUADRATIC):
        t = CTrack()
        self._check(self._L.st_track_params_family(self._ctx, seed, track_id, n_min, n_max, tau_lo, tau_hi, int(family), C.byref(t)))
        return t

    # ------------------------------------------------------ parity exports
    def debug_rasterise(self, seed, n_min, n_max, first, count, family=FAMILY_QUADRATIC):
        torch = self._torch
        p, _ = self._params(count, seed, n_min, n_max, None, (0.0, 0.0), 0, 0, -10, 10, 0, 0, family)
        k = torch.empty((count, self.n_t), dtype=torch.int32, device=self.device)
        j0 = torch.empty(count, dtype=torch.int32, device=self.device)
        N = torch.empty(count, dtype=torch.int32, device=self.device)
        self._check(self._L.st_debug_rasterise(self._ctx, C.byref(p), int(first), int(count), k.data_ptr(),
                                               j0.data_ptr(), N.data_ptr()))
        self.synchronize()
        return k.cpu().numpy(), j0.cpu().numpy(), N.cpu().numpy()

    def debug_rasterise_random(self, seed, n_min, n_max, first, count, tau_range=(-0.01, 0.01), family=FAMILY_QUADRATIC):
        """Bins decided by the random-delay kernel's own rasteriser (st_debug_rasterise_random)."""
        torch = self._torch
        p, _ = self._params(count, seed, n_min, n_max, None, tau_range, 0, 0, -10, 10, 0, 0, family)
        k = torch.empty((count, self.n_t), dtype=torch.int32, device=self.device)
        j0 = torch.empty(count, dtype=torch.int32, device=self.device)
        N = torch.empty(count, dtype=torch.int32, device=self.device)
        self._check(self._L.st_debug_rasterise_random(self._ctx, C.byref(p), int(first), int(count), k.data_ptr(),
                                                      j0.data_ptr(), N.data_ptr()))
        self.synchronize()
        return k.cpu().numpy(), j0.cpu().numpy(), N.cpu().numpy()

    def debug_rasterise_track(self, N, j0, a, y0, y1, y2, y3=None, family=None):
        """Bins of one explicit template; with y3 a cubic one (frequency control points y0, y1, y2, y3); with
        family=FAMILY_CHIRP the chirp-law template of (N, j0, a, y0)."""
        torch = self._torch
        t = CTrack(int(N), int(j0), float(a), float(y0), float(y1), float(y2), 0.0, 0.0 if y3 is None else float(y3))
        k = torch.empty(int(N), dtype=torch.int32, device=self.device)
        fam = family if family is not None else (FAMILY_QUADRATIC if y3 is None else FAMILY_CUBIC)
        self._check(self._L.st_debug_rasterise_track(self._ctx, C.byref(t), int(fam), k.data_ptr()))
        self.synchronize()
        return k.cpu().numpy()

    def debug_scores(self, seed, n_min, n_max, first, count, tau_grid=None, tau_range=None, norm=NORM_SQRT_N,
                     kernel=KERNEL_AUTO, family=FAMILY_QUADRATIC):
        torch = self._torch
        p, keep = self._params(count, seed, n_min, n_max, tau_grid, tau_range, norm, 0, -10, 10, first, kernel, family)
        n_tau = p.n_tau if p.tau_mode == TAU_GRID else 1
        snr = torch.empty((count, n_tau), dtype=torch.float32, device=self.device)
        self._check(self._L.st_debug_scores(self._ctx, C.byref(p), int(first), int(count), snr.data_ptr()))
        self.synchronize()
        return snr.cpu().numpy()


NOALLOC_MAX_PIXELS = 262144        # ST_NOALLOC_MAX_PIXELS
NOALLOC_SCRATCH_BYTES = 3604736    # ST_NOALLOC_SCRATCH_BYTES


def score_random_noalloc(csd, sigma, df, f_min, n_tracks, seed, n_min, n_max, tau_range, out, norm=NORM_SQRT_N,
                         track_offset=0, stream=None):
    """st_score_random_noalloc: the one-delay-per-template scores of templates [track_offset, +n_tracks) on
    the map csd / sigma, for a caller who has no device memory to lend the library (a framework pool owns the
    card, nothing may be allocated while the analysis runs, or the component only sees its own input and
    output buffers).  The library's scratch is a static array inside its device image (NOALLOC_SCRATCH_BYTES
    on every GPU that loads it), which caps the map at NOALLOC_MAX_PIXELS pixels.  Nothing is allocated here
    either: `out` is the caller's float32 CUDA tensor of n_tracks elements and is returned filled
    (stream-ordered, not synchronised).  All calls on one device share the static array: issue them on one
    stream; the first call per device does a one-off symbol look-up and belongs at start-up.
    csd: complex64 [n_t][n_f] CUDA tensor; sigma: None, [n_f] or [n_t][n_f] float32 CUDA tensor."""
    import torch
    L = load_library()
    if not (isinstance(csd, torch.Tensor) and csd.is_cuda and csd.dtype == torch.complex64 and csd.is_contiguous() and csd.dim() == 2):
        raise ValueError("csd must be a contiguous complex64 [n_t][n_f] CUDA tensor")
    n_t, n_f = int(csd.shape[0]), int(csd.shape[1])
    kind, sp = SIGMA_NONE, 0
    if sigma is not None:
        if not (isinstance(sigma, torch.Tensor) and sigma.is_cuda and sigma.dtype == torch.float32 and sigma.is_contiguous()):
            raise ValueError("sigma must be a contiguous float32 CUDA tensor")
        shp = tuple(sigma.shape)
        kind = SIGMA_PER_FREQ if shp == (n_f,) else SIGMA_PER_PIXEL if shp == (n_t, n_f) else -1
        if kind < 0:
            raise ValueError("sigma must be None, [n_f] or [n_t][n_f]")
        sp = sigma.data_ptr()
    if not (isinstance(out, torch.Tensor) and out.is_cuda and out.dtype == torch.float32 and out.is_contiguous()
            and out.numel() == int(n_tracks)):
        raise ValueError("out must be a contiguous float32 CUDA tensor of n_tracks elements")
    p = CSearchParams()
    p.n_tracks, p.track_offset, p.seed = int(n_tracks), int(track_offset), int(seed)
    p.n_min, p.n_max, p.tau_mode, p.n_tau = int(n_min), int(n_max), TAU_RANDOM, 1
    p.tau_lo, p.tau_hi = float(tau_range[0]), float(tau_range[1])
    p.norm, p.family = int(norm), FAMILY_QUADRATIC
    err = C.create_string_buffer(512)
    with torch.cuda.device(csd.device):
        s = stream if stream is not None else torch.cuda.current_stream(csd.device)
        rc = L.st_score_random_noalloc(csd.data_ptr(), sp, kind, n_t, n_f, float(df), float(f_min), C.byref(p),
                                       out.data_ptr(), s.cuda_stream, err, len(err))
    if rc:
        raise StError(rc, err.value.decode())
    return out


def st_track_params(n_t, n_f, seed, track_id, n_min, n_max, tau_lo=0.0, tau_hi=0.0, df=1.0, f_min=0.0,
                    family=FAMILY_QUADRATIC):
    """S1 as a pure host function (no GPU needed)."""
    L = load_library()
    ctx = C.c_void_p()
    rc = L.st_create(C.byref(ctx), n_t, n_f, df, f_min)
    if rc:
        raise StError(rc, "st_create")
    try:
        t = CTrack()
        rc = L.st_track_params_family(ctx, seed, track_id, n_min, n_max, tau_lo, tau_hi, int(family), C.byref(t))
        if rc:
            raise StError(rc, "st_track_params: invalid arguments")
        return t
    finally:
        L.st_destroy(ctx)

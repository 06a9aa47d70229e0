"""Multi-GPU use of the path: templates are independent and the
paper scales by independent GPU jobs (n_GPU in Eqs. 9-10), whose
results are combined afterwards by a max.  So there is no data-path
collective: every rank scores its own template-id range on its own copy of the map
and the (tiny) results meet once at the end -- max/argmax under the G12 total order,
integer sum of the histograms.  `combine` is that rule; `all_combine` runs it over a
torch.distributed group (NCCL or gloo) by gathering the per-rank result records.
"""
import numpy as np


def rank_range(n_tracks_per_rank, rank, base_offset=0):
    """Weak scaling: rank r owns template ids [base + r*T, base + (r+1)*T)."""
    return base_offset + rank * n_tracks_per_rank, n_tracks_per_rank


def split_range(n_tracks_total, world_size, rank, base_offset=0):
    """Strong scaling: contiguous, near-equal id ranges covering [base, base + T)."""
    q, rem = divmod(n_tracks_total, world_size)
    first = rank * q + min(rank, rem)
    return base_offset + first, q + (1 if rank < rem else 0)


def combine(results):
    """Combine per-range search results (dicts as returned by Stochtrack.search): marshalling around the C ABI's
    st_combine_results, which holds the rule (G12 total order, sums, histogram sum); no step of S4 lives here."""
    import ctypes as C
    from . import binding as B
    L = B.load_library()
    n = len(results)
    arr = (B.CResult * n)()
    hists, keep = (C.POINTER(C.c_uint64) * n)(), []
    n_bins = 0
    for i, r in enumerate(results):
        for f in ("max_snr", "max_snr_f64", "arg_tau"):
            setattr(arr[i], f, float(r.get(f, 0.0)))
        for f in ("arg_tau_index", "arg_track", "n_evals", "n_pixels", "n_candidates", "n_launches", "flags", "n_deferred"):
            setattr(arr[i], f, int(r.get(f, 0)))
        h = r.get("hist")
        if h is not None:
            h = np.ascontiguousarray(h, dtype=np.uint64)
            keep.append(h)
            hists[i] = h.ctypes.data_as(C.POINTER(C.c_uint64))
            n_bins = h.size
    out, idx = B.CResult(), C.c_int32(0)
    hist_out = np.zeros(n_bins, dtype=np.uint64) if keep else None
    rc = L.st_combine_results(arr, hists, n, n_bins, C.byref(out),
                              hist_out.ctypes.data_as(C.POINTER(C.c_uint64)) if keep else None, C.byref(idx))
    if rc:
        raise B.StError(rc, "st_combine_results: bad arguments")
    best = dict(results[idx.value])                   # keeps the winner's arg_params, arg_tau, kernel name, ...
    for f in ("max_snr", "n_evals", "n_pixels", "n_candidates"):
        best[f] = getattr(out, f)
    best["hist"] = hist_out
    return best


def all_combine(result, group=None):
    """Gather every rank's result record and combine; every rank returns the same dict."""
    import torch.distributed as dist
    rec = {k: result[k] for k in ("max_snr", "max_snr_f64", "arg_track", "arg_tau_index", "arg_tau",
                                  "arg_params", "n_evals", "n_pixels", "n_candidates", "hist")}
    out = [None] * dist.get_world_size(group)
    dist.all_gather_object(out, rec, group=group)
    return combine(out)

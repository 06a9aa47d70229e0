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


def _key(r):
    # G12: larger SNR, then smaller template id, then smaller delay index
    return (-r["max_snr_f64"], r["arg_track"], r["arg_tau_index"])


def combine(results):
    """Combine per-range search results (dicts as returned by Stochtrack.search)."""
    live = [r for r in results if r["n_evals"] > 0]
    if not live:
        return dict(results[0])
    best = dict(min(live, key=_key))
    best["n_evals"] = sum(r["n_evals"] for r in results)
    best["n_pixels"] = sum(r["n_pixels"] for r in results)
    best["n_candidates"] = sum(r["n_candidates"] for r in live)
    best["max_snr"] = max(r["max_snr"] for r in live)
    hists = [r["hist"] for r in results if r.get("hist") is not None]
    best["hist"] = np.sum(np.stack(hists), axis=0).astype(np.uint64) if hists else None
    return best


def all_combine(result, group=None):
    """Gather every rank's result record and combine; every rank returns the same dict."""
    import torch.distributed as dist
    rec = {k: result[k] for k in ("max_snr", "max_snr_f64", "arg_track", "arg_tau_index", "arg_tau",
                                  "arg_params", "n_evals", "n_pixels", "n_candidates", "hist")}
    out = [None] * dist.get_world_size(group)
    dist.all_gather_object(out, rec, group=group)
    return combine(out)

"""The library built with -DST_CHECKED (device-side assertions on every index the kernels form) runs the
kernels of the path on ragged workloads without tripping one, and returns what the production build
returns.  Stands in for compute-sanitizer, which the GPU pool does not offer."""
import json
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SCRIPT = r"""
import json, sys
import numpy as np, torch
sys.path.insert(0, %(root)r)
import paper_1401_8060_b200 as P
P.load_library(%(lib)r)
from workloads import synth
out = {}
for cid, n in ((1, 1000), (2, 20000), (3, 30000), (4, 20000), (5, 3000)):
    cfg = synth.CONFIGS[cid]
    st = P.Stochtrack(cfg.n_t, cfg.n_f, cfg.df, cfg.f_min, max_n_tau=max(cfg.n_tau, 64))
    csd = synth.noise_csd(cfg.n_t, cfg.n_f, 40 + cid)
    sigma = synth.make_sigma(cfg.sigma, cfg.sigma_scale, cfg.n_t, cfg.n_f, 40 + cid)
    st.set_map(csd, sigma)
    tau = synth.tau_linspace(cfg.n_tau) if cfg.tau_mode == "grid" else None
    kernels = (0, 1, 2, 3) if cfg.tau_mode == "grid" else (0,)
    for k in kernels:
        kw = dict(tau_grid=tau, kernel=k) if tau is not None else dict(tau_range=(-0.01, 0.01))
        r = st.search(n, 7, 1 if cid == 1 else cfg.n_min, cfg.n_max, n_bins=200, **kw)
        out["c%%d_k%%d" %% (cid, k)] = [r.max_snr_f64, r.arg_track, r.arg_tau_index, int(r.hist.sum()), r.n_pixels]
    kw = dict(tau_grid=tau) if tau is not None else dict(tau_range=(-0.01, 0.01))
    r, top = st.search_topk(7, n, 7, cfg.n_min, cfg.n_max, n_bins=400, **kw)
    out["c%%d_top" %% cid] = [[e["track"], e["tau_index"], e["snr_f64"]] for e in top]
    if cid in (4, 5):      # the delay-split builds: per-template maximum, and the bank cache filled then read
        r, vmax, imax = st.search_track_max(n, 7, cfg.n_min, cfg.n_max, n_bins=200, **kw)
        out["c%%d_tmax" %% cid] = [float(vmax.max()), int(imax.sum()), r.arg_track]
        st.enable_bank_cache(n, cfg.n_max)
        for rep in range(2):
            r = st.search(n, 7, cfg.n_min, cfg.n_max, n_bins=200, **kw)
            out["c%%d_bank%%d" %% (cid, rep)] = [r.max_snr_f64, r.arg_track, r.arg_tau_index, int(r.hist.sum()), int(r.flags)]
    if cid == 1:
        res, _ = st.search_batch([torch.from_numpy(csd).cuda()] * 3, None, [1, 2, 3], 500, cfg.n_min, cfg.n_max, tau_grid=tau, n_bins=50)
        out["batch"] = [[x.max_snr_f64, x.arg_track] for x in res]
# the call without a workspace (static scratch inside the library): same kernels, same index assertions
cfg = synth.CONFIGS[2]
csd = torch.from_numpy(synth.noise_csd(cfg.n_t, cfg.n_f, 61)).cuda()
sig = torch.from_numpy(synth.make_sigma(cfg.sigma, cfg.sigma_scale, cfg.n_t, cfg.n_f, 61)).cuda()
snr = torch.empty(7001, dtype=torch.float32, device="cuda")
for rep in range(2):
    P.score_random_noalloc(csd, sig, cfg.df, cfg.f_min, 7001, 7 + rep, cfg.n_min, cfg.n_max, (-0.01, 0.01), snr, track_offset=2 ** 33)
    torch.cuda.synchronize()
    out["noalloc%%d" %% rep] = [float(snr.double().sum()), float(snr.max()), int(snr.argmax())]
torch.cuda.synchronize()
print(json.dumps(out))
"""


def _run(lib_path):
    out = subprocess.run([sys.executable, "-c", SCRIPT % {"root": ROOT, "lib": lib_path}], capture_output=True, text=True,
                         timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-3000:]
    return json.loads(out.stdout.strip().splitlines()[-1])


def test_checked_build_trips_no_assertion_and_matches_production():
    import torch
    assert torch.cuda.is_available()
    from paper_1401_8060_b200 import build
    build.build()
    checked = build.build_checked()
    got = _run(checked)
    want = _run(build.LIB)
    assert got == want
    assert len(got) >= 26 and "noalloc1" in got

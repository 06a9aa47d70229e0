#!/usr/bin/env python
"""bench.py -- throughput of the all-sky stochtrack hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 5]

A "step" is one pass of the whole hot path over one synthetic map: S0 map preparation
(st_set_map) + S1-S4 (st_search: template generation, rasterisation, Eq. 8 scoring for
every (template, delay), max/argmax/histogram) -- see DESIGN.md.  The default workload
is BASELINE.json configs[4] (the largest single-GPU configuration: 1000 x 2461 map, 1e7
templates, 512 delays = 2.6e12 track-pixel evaluations per step).  `value` is track-pixel
evaluations per second over all ranks, device-timed with the map resident in HBM; `e2e`
is the same metric through the C ABI with host buffers (H2D of the map and D2H of the
result inside the timed region).  Prints ONE JSON line on rank 0.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from workloads import synth  # noqa: E402

METRIC = "track_pixel_evals_per_s"
UNIT = "evals/s"
N_SM, FP32_LANES = 148, 128           # B200: 148 SMs x 128 FP32 lanes (B200_PROFILING.md, blackwell guide)
FLOP_PER_EVAL = 4                     # Eq. 8 needs 2 FMA per (pixel, delay) once the phase factor is known
# dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel, per launch, from the `ncu --set full` capture
# named beside it (profiles/; the command is in the file's first line).  The map is read from HBM once per launch
# and then served by L2; a config without a capture reports null.
DRAM_TRAFFIC = {5: (19.83e6, "profiles/r02_ncu_cheb_c5.txt"),      # algorithmic: the 19.69 MB map once
                4: (9.97e6, "profiles/r02_ncu_cheb_c4.txt"),       # per map of the batch: the 9.84 MB map once
                3: (9.88e6, "profiles/r02_ncu_random.txt")}
L2_GATHER_PEAK_GBS = 9200.0          # random 32-byte sector gathers, measured (profiles/microbench_r01.md)
L2_GATHER_FROM = "profiles/microbench_r01.md (built-in fallback)"
# The figures above are fallbacks: profiles/peaks.json (a tracked data file: each entry with the raw file, command, date
# and lease it comes from) replaces them when present, so that a new capture updates the line without an edit here.
_PEAKS_FILE = os.path.join(ROOT, "profiles", "peaks.json")
if os.path.exists(_PEAKS_FILE):
    with open(_PEAKS_FILE) as _f:
        _pk = json.load(_f)
    if "l2_gather" in _pk:
        L2_GATHER_PEAK_GBS, L2_GATHER_FROM = float(_pk["l2_gather"]["sector_GBps"]), _pk["l2_gather"]["from"] + " via profiles/peaks.json"
    for _c, _e in _pk.get("dram_traffic_bytes_per_launch", {}).items():
        DRAM_TRAFFIC["P" if _c == "P" else int(_c)] = (float(_e["bytes"]), _e["from"] + " via profiles/peaks.json")


def workload_tag(config):
    return "the paper's Table III shape (PAPER.md:207-212, context)" if config == "P" else f"BASELINE.json configs[{config - 1}]"


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    sm_mhz, src = 1965.0, "fallback clock 1965 MHz"
    if os.path.exists(p):
        with open(p) as f:
            sm_mhz = float(json.load(f).get("sm_max_mhz", sm_mhz))
        src = "MEASURED_PEAKS.json sm_max_mhz"
    return N_SM * FP32_LANES * 2 * sm_mhz * 1e6 / 1e12, f"148 SMs x 128 FP32 lanes x 2 flop x {sm_mhz:.0f} MHz ({src})"


class ClockSampler(threading.Thread):
    """nvidia-smi clocks + throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.rows, self.proc, self.index = [], None, index

    def run(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "200", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            for line in self.proc.stdout:
                self.rows.append([x.strip() for x in line.split(",")])
        except Exception:
            pass

    def stop(self):
        if self.proc:
            self.proc.terminate()
        self.join(timeout=2)
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        load = sorted(sm)[len(sm) // 2:] if sm else []      # upper half = samples under load
        return {"sm_mhz": float(np.median(load)) if load else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def build_inputs(cfg, st, m=0):
    """Seeded synthetic map of the config; injections rasterised by the CUDA path (product side)."""
    def rast(inj):
        return st.debug_rasterise_track(inj.N, inj.j0, inj.a, inj.y0, inj.y1, inj.y2)
    return synth.config_inputs(cfg, m, rasterise=rast)


def search_kwargs(cfg, tau):
    kw = dict(n_bins=cfg.n_bins, hist_lo=cfg.hist_lo, hist_hi=cfg.hist_hi)
    if cfg.tau_mode == "grid":
        kw["tau_grid"] = tau
    else:
        kw["tau_range"] = (-synth.TAU_MAX, synth.TAU_MAX)
    return kw


def run_ours(args):
    import torch
    import paper_1401_8060_b200 as pkg
    from paper_1401_8060_b200 import build, sharding
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the hot path has no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    build.build()
    pkg.load_library(args.lib or None)
    dev = f"cuda:{local}"
    env = dict(torch=torch, pkg=pkg, sharding=sharding, dist=dist, world=world, rank=rank, local=local, dev=dev)
    line = measure(args, env)
    if rank == 0:
        # short driver-visible runs of the other workloads (W = 3 warm-up, 2 timed steps each): config 3 (the
        # paper's random-delay mode), config 4 as the one-call background batch with per-map banks (G16) and with one
        # shared bank + bank cache, config P (the paper's Table III shape)
        if world == 1 and args.config == 5 and not args.no_other_configs and not args.tracks:
            import copy
            others = []
            # ... and of what the quadratic / sqrt(N) / plain-search default leaves unmeasured: the general builds of the
            # kernels (cubic and chirp families, inverse-variance weighting), the two-pass top-K call and the fused
            # per-template maximum on one config-4 map, each against the same peak as its quadratic twin
            for cid, extra in ((3, {}), (4, dict(maps=20)), (4, dict(maps=20, shared_bank=True)), ("P", {}),
                               (5, dict(family="cubic")), (5, dict(family="chirp")), (5, dict(norm="invvar")),
                               (3, dict(family="chirp")), (4, dict(call="topk")), (4, dict(call="track_max"))):
                a2 = copy.copy(args)
                a2.config, a2.steps, a2.warmup, a2.no_cpu_baseline, a2.ftmap, a2.maps, a2.shared_bank = cid, 2, 3, True, False, 0, False
                for k, v in extra.items():
                    setattr(a2, k, v)
                o = measure(a2, env)
                others.append({"config": o["config"]["workload"], "value": o["value"], "unit": o["unit"], "ms_per_step": o["ms_per_step"],
                               "steps": o["steps"], "warmup": o["warmup"], "tracks_tau_per_s": o["tracks_tau_per_s"],
                               "e2e_value": o["e2e"]["value"], "gpu_launches": o["gpu_launches"], "clocks": o["clocks"],
                               "roofline": {k: o["roofline"][k] for k in ("bound", "kernel", "achieved", "peak", "unit", "frac", "traffic")}})
            line["other_configs"] = others
            # the time-shift background from strain (20 shifts, one bank + bank cache) and the ft-map construction
            line["timeshifts"] = timeshift_timing(env["pkg"], env["torch"], synth.CONFIGS[4], env["dev"])
            line["ftmap"] = ftmap_timing(env["pkg"], env["torch"], synth.CONFIGS[5], env["dev"])
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def measure(args, env):
    """One workload, timed as the module docstring says; returns the JSON line as a dict on rank 0 (None elsewhere)."""
    torch, pkg, sharding, dist = env["torch"], env["pkg"], env["sharding"], env["dist"]
    world, rank, local, dev = env["world"], env["rank"], env["local"], env["dev"]
    cfg = synth.CONFIGS[args.config]
    n_tracks = args.tracks or cfg.n_tracks
    st = pkg.Stochtrack(cfg.n_t, cfg.n_f, cfg.df, cfg.f_min, max_n_tau=max(cfg.n_tau, 64), device=dev)
    csd, sigma, tau = build_inputs(cfg, st)
    seed = synth.map_seed(cfg, 0)
    # weak scaling: rank r scores its own template-id range on its own copy of the map
    first, n_mine = sharding.rank_range(n_tracks, rank)
    kw = search_kwargs(cfg, tau)
    if cfg.tau_mode == "grid":
        kw["kernel"] = {"auto": 0, "table": 1, "rotation": 2, "reinsch": 3}[args.kernel]
    kw["family"] = {"quadratic": 0, "cubic": 1, "chirp": 2}[args.family]
    kw["norm"] = {"sqrt_n": 0, "mean": 1, "invvar": 2}[args.norm]
    variant = "".join(f", {k} {v}" for k, v, d in (("family", args.family, "quadratic"), ("norm", args.norm, "sqrt_n"),
                                                    ("call", args.call, "search")) if v != d)
    if args.norm == "invvar" and sigma is None:
        raise SystemExit("bench.py: --norm invvar needs a config with sigma (2 or 5)")

    def one_search(set_map):
        """One step on one map through the call --call names; the timed quantity is the method's own work once
        (n_evals), whatever the call does on top (top-K: a second scoring pass; track_max: a per-template output)."""
        set_map()
        if args.call == "topk":
            return st.search_topk(100, n_mine, seed, cfg.n_min, cfg.n_max, track_offset=first, **kw)[0]
        if args.call == "track_max":
            return st.search_track_max(n_mine, seed, cfg.n_min, cfg.n_max, track_offset=first, **kw)[0]
        return st.search(n_mine, seed, cfg.n_min, cfg.n_max, track_offset=first, **kw)
    csd_d = torch.from_numpy(csd).to(dev)
    sigma_d = torch.from_numpy(sigma).to(dev) if sigma is not None else None
    csd_h = torch.from_numpy(csd).pin_memory()
    sigma_h = torch.from_numpy(sigma).pin_memory() if sigma is not None else None
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)        # > 126 MB L2

    class _Agg:                                   # what the timing loop reads from a step's result
        pass

    n_maps = 1
    if cfg.n_maps > 1 and args.call == "search":
        # batch / background configuration: a step is ONE st_search_batch call over n_maps maps
        # (map m: its own noise and its own template seed, G16); map 0 was built above
        n_maps = args.maps or cfg.n_maps
        maps_h = [csd_h] + [torch.from_numpy(synth.config_inputs(cfg, m)[0]).pin_memory() for m in range(1, n_maps)]
        maps_d = [h.to(dev) for h in maps_h]
        seeds = [synth.map_seed(cfg, m) for m in range(n_maps)]
        if args.shared_bank:
            seeds = synth.map_seed(cfg, 0)
            st.enable_bank_cache(n_mine, cfg.n_max)

        def run_batch(maps):
            res, ms = st.search_batch(maps, None, seeds, n_mine, cfg.n_min, cfg.n_max, track_offset=first, **kw)
            a = _Agg()
            a.gpu_ms, a.n_launches, a.n_evals = ms, sum(x.n_launches for x in res) - 1, sum(x.n_evals for x in res)
            a.kernel_name, a.best = res[0].kernel_name, max(res, key=lambda x: x.max_snr_f64)
            a.n_deferred = sum(x.n_deferred for x in res)
            a.maxima = [x.max_snr_f64 for x in res]
            return a

        def step_device():
            return run_batch(maps_d)

        def step_host():
            return run_batch(maps_h)
    else:
        def step_device():
            return one_search(lambda: st.set_map(csd_d, sigma_d))

        def step_host():
            return one_search(lambda: st.set_map(csd_h.numpy(), sigma_h.numpy() if sigma_h is not None else None))

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        flush.zero_()
        r = step_device()
    # ---- device-timed steps (inputs resident in HBM; L2 flushed between steps)
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    barrier()
    t_wall0 = time.perf_counter()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    kernel_ms, launches, evals = 0.0, 0, 0
    for a, b in ev:
        flush.zero_()
        a.record()
        r = step_device()
        b.record()
        kernel_ms += r.gpu_ms
        launches += r.n_launches + 1               # + k_prepare_map
        evals += r.n_evals
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    dev_ms = sum(a.elapsed_time(b) for a, b in ev)
    # ---- end to end through the C ABI with host buffers
    step_host()
    barrier()
    e2e_evals, t0 = 0, time.perf_counter()
    for _ in range(args.steps):
        e2e_evals += step_host().n_evals
    barrier()
    e2e_s = time.perf_counter() - t0
    t = torch.tensor([dev_ms, e2e_s, float(evals), float(e2e_evals), float(launches), kernel_ms], dtype=torch.float64,
                     device=dev)
    if dist is not None:
        mx = t.clone(); dist.all_reduce(mx, op=dist.ReduceOp.MAX)
        sm = t.clone(); dist.all_reduce(sm, op=dist.ReduceOp.SUM)
        dev_ms, e2e_s, kernel_ms = mx[0].item(), mx[1].item(), mx[5].item()
        evals, e2e_evals, launches = sm[2].item(), sm[3].item(), sm[4].item()
        combined = sharding.all_combine(r if n_maps == 1 else r.best)
    else:
        combined = r if n_maps == 1 else r.best
    if rank != 0:
        return None
    peak, peak_how = peaks()
    if args.call == "topk":
        kernel_ms = dev_ms          # st_result.gpu_ms covers the first pass only: the whole two-pass call is what is rated
        peak_how += "; top-K: both scoring passes and the float64 re-score of the captured samples count as the time of one pass's work"
    value = evals / (dev_ms * 1e-3)
    per_launch_evals = evals / world / args.steps            # one scoring launch sequence per step per rank
    achieved = FLOP_PER_EVAL * per_launch_evals / (kernel_ms / args.steps * 1e-3) / 1e12
    n_tau = cfg.n_tau if cfg.tau_mode == "grid" else 1
    h2d = n_maps * (csd.nbytes + (sigma.nbytes if sigma is not None else 0))
    d2h = n_maps * (128 + 8 * cfg.n_bins)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": dev_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{workload_tag(args.config)} ({cfg.name}): {cfg.n_t}x{cfg.n_f} map, "
                               f"{n_tracks:.0e} templates per GPU" + (f" per map x {n_maps} maps in one st_search_batch call" + (" (shared bank)" if args.shared_bank else "") if n_maps > 1 else "") +
                               f", {n_tau} delays ({cfg.tau_mode})" + (" [one map]" if cfg.n_maps > 1 and n_maps == 1 else "") + variant,
                   "n_t": cfg.n_t, "n_f": cfg.n_f, "n_tracks_per_gpu": n_tracks, "n_tau": n_tau,
                   "tau_mode": cfg.tau_mode, "kernel": r.kernel_name, "l2": "flushed between timed steps (256 MB write)",
                   "parallelism": f"independent template-id ranges x{world}, no data-path collective"},
        "tracks_tau_per_s": world * args.steps * n_maps * n_mine * n_tau / (dev_ms * 1e-3),
        "wall_s_timed_region": t_wall,
        "e2e": {"value": e2e_evals / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "roofline": {"bound": "alu", "kernel": {"chebyshev": "k_score_cheb", "reinsch": "k_score_reinsch", "rotation": "k_score_recur",
                                                "table": "k_score_table", "random": "k_score_random"}.get(r.kernel_name, r.kernel_name), "achieved": achieved, "peak": peak,
                     "unit": "TFLOP/s", "frac": achieved / peak, "traffic": DRAM_TRAFFIC.get(args.config if not variant else None, (None, None))[0],
                     "traffic_from": DRAM_TRAFFIC.get(args.config if not variant else None, (None, None))[1],
                     "peak_how": peak_how + "; algorithmic 4 flop per track-pixel evaluation (DESIGN.md)"},
        "result": {"max_snr": combined["max_snr_f64"], "arg_track": combined["arg_track"],
                   "arg_tau_index": combined["arg_tau_index"], "n_deferred_last_step": int(r.n_deferred)},
    }
    if args.lib:
        line["config"]["library"] = os.path.basename(args.lib) + " (NOT the production build: a measurement build, results meaningless)"
    if n_maps > 1:
        line["config"]["n_maps"] = n_maps
        line["config"]["bank"] = "one shared bank, bank cache attached" if args.shared_bank else "one bank per map (G16)"
        line["result"]["per_map_max_snr"] = {"min": min(r.maxima), "median": float(np.median(r.maxima)), "max": max(r.maxima)}
        line["roofline"]["peak_how"] += "; batch mode: the kernel time is the device time of the whole call (S0, S1-S4, finalize of every map)"
    if cfg.tau_mode == "random":
        # the paper's one-delay mode is a gather: one 32-byte L2 sector per track pixel
        gbs = 32.0 * per_launch_evals / (kernel_ms / args.steps * 1e-3) / 1e9
        line["roofline"].update({"bound": "l2-gather", "achieved": gbs, "peak": L2_GATHER_PEAK_GBS, "unit": "GB/s",
                                 "frac": gbs / L2_GATHER_PEAK_GBS,
                                 "peak_how": "random 8-byte gathers from an L2-resident 19.7 MB buffer, one 32-byte sector each, "
                                             f"measured by st_microbench ({L2_GATHER_FROM})"})
    if world == 1 and args.ftmap:
        line["ftmap"] = ftmap_timing(pkg, torch, cfg, dev)
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(cfg, csd, sigma, tau, seed, budget_s=args.cpu_budget)
    return line


def ftmap_timing(pkg, torch, cfg, dev, seg_len=8192, reps=5):
    """The step before the hot path, timed on its own: two synthetic strain series
    of the config's duration -> st_set_map_from_strain (float64 FFT, neighbour PSDs, p into the map)."""
    fs = float(seg_len) * cfg.df
    n = (cfg.n_t + 1) * seg_len // 2
    g = torch.Generator(device=dev).manual_seed(1234)
    s_i = torch.randn(n, dtype=torch.float64, device=dev, generator=g) * 1e-21
    s_j = torch.randn(n, dtype=torch.float64, device=dev, generator=g) * 1e-21
    st = pkg.Stochtrack(cfg.n_t, cfg.n_f, cfg.df, cfg.f_min, max_n_tau=64, device=dev)
    for _ in range(3):
        st.set_map_from_strain(s_i, s_j, fs, seg_len, 4)
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
    for a, b in ev:
        a.record()
        st.set_map_from_strain(s_i, s_j, fs, seg_len, 4)
        b.record()
    torch.cuda.synchronize()
    ms = float(np.median([a.elapsed_time(b) for a, b in ev]))
    # algorithmic bytes: both series read once (16 B per sample pair), s~ written and read back (2 x 2 x 16 B per
    # pixel), p written (8 B per pixel)
    n_pix = cfg.n_t * cfg.n_f
    alg = 16.0 * n + 64.0 * n_pix + 8.0 * n_pix
    hbm, hbm_src = 6500.0, "fallback 6500 GB/s"
    pk = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(pk):
        with open(pk) as f:
            hbm, hbm_src = float(json.load(f).get("hbm_gbs", hbm)), "MEASURED_PEAKS.json hbm_gbs"
    gbs = alg / (ms * 1e-3) / 1e9
    return {"ms": ms, "n_t": cfg.n_t, "n_f": cfg.n_f, "seg_len": seg_len, "samples_per_detector": n,
            "algorithmic_gb_per_s": gbs, "launches": 3,
            "roofline": {"bound": "hbm", "kernel": "k_ft_twiddles + k_ft_segments + k_ft_normalise (whole call)", "achieved": gbs,
                         "peak": hbm, "unit": "GB/s", "frac": gbs / hbm, "traffic": None,
                         "peak_how": hbm_src + "; algorithmic bytes: 16 B per sample pair read, the two float64 spectra written and "
                                     "read back (64 B per pixel), p written (8 B per pixel).  The call is NOT HBM bound: k_ft_segments, "
                                     "a float64 radix-2 FFT in shared memory, takes most of it (profiles/r01_ncu_ft_segments.txt)"}}


def timeshift_timing(pkg, torch, cfg, dev, n_shifts=20, seg_len=8192):
    """The paper's background workflow end to end (SURVEY 8(f) NEXT-1 + NEXT-2): st_search_timeshifts on
    synthetic strain of the config's duration -- spectrograms once, then per shift the map normalisation and a full
    search with ONE template bank (bank cache attached: the first shift fills it, the others read S1 + S2 back)."""
    fs = float(seg_len) * cfg.df
    n = (cfg.n_t + 1) * seg_len // 2
    g = torch.Generator(device=dev).manual_seed(4321)
    s_i = torch.randn(n, dtype=torch.float64, device=dev, generator=g) * 1e-21
    s_j = torch.randn(n, dtype=torch.float64, device=dev, generator=g) * 1e-21
    st = pkg.Stochtrack(cfg.n_t, cfg.n_f, cfg.df, cfg.f_min, max_n_tau=max(cfg.n_tau, 64), device=dev)
    st.enable_bank_cache(cfg.n_tracks, cfg.n_max)
    tau = synth.tau_linspace(cfg.n_tau)
    shifts = [(7 * m) % cfg.n_t for m in range(n_shifts)]
    seed = synth.map_seed(cfg, 0)
    best = None
    for rep in range(3):                      # call 1 fills the cache; calls 2 and 3 read it for every shift: the faster is kept
        res, ms = st.search_timeshifts(s_i, s_j, fs, seg_len, 4, shifts, seed, cfg.n_tracks, cfg.n_min, cfg.n_max, tau_grid=tau,
                                       n_bins=cfg.n_bins, hist_lo=cfg.hist_lo, hist_hi=cfg.hist_hi)
        if rep and (best is None or ms < best[1]):
            best = (res, ms)
    res, ms = best
    evals = sum(r.n_evals for r in res)
    peak, peak_how = peaks()
    achieved = FLOP_PER_EVAL * evals / (ms * 1e-3) / 1e12
    return {"workload": f"{n_shifts} time shifts of a {cfg.n_t}x{cfg.n_f} map from strain (seg_len {seg_len}), {cfg.n_tracks:.0e} templates x "
                        f"{cfg.n_tau} delays per shift, one bank + bank cache", "ms": ms, "value": evals / (ms * 1e-3), "unit": UNIT,
            "n_shifts": n_shifts, "bank_read": sum(1 for r in res if r.flags & 2), "launches": sum(r.n_launches for r in res),
            "max_snr_median": float(np.median([r.max_snr_f64 for r in res])),
            "roofline": {"bound": "alu", "kernel": "k_score_cheb", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                         "frac": achieved / peak, "traffic": None,
                         "peak_how": peak_how + "; the time is the device time of the whole call (FFTs, 20 normalisations, searches)"}}


def oracle_inputs(cfg):
    from oracle import oracle

    def rast(inj):
        return oracle.rasterise(oracle.make_track(inj.N, inj.j0, inj.a, inj.y0, inj.y1, inj.y2), cfg.n_f)
    return synth.config_inputs(cfg, 0, rasterise=rast)


def oracle_sample(oracle, p, cfg, tau, seed, n, first=0):
    kw = dict(tau_grid=tau) if cfg.tau_mode == "grid" else dict(tau_range=(-synth.TAU_MAX, synth.TAU_MAX))
    t0 = time.perf_counter()
    r = oracle.search(p, cfg.f_min, cfg.df, n, seed, cfg.n_min, cfg.n_max, n_bins=cfg.n_bins, hist_lo=cfg.hist_lo,
                      hist_hi=cfg.hist_hi, track_offset=first, **kw)
    return r, time.perf_counter() - t0


def cpu_baseline(cfg, csd, sigma, tau, seed, budget_s=15.0):
    """The oracle as it stands, timed on this box's host cores on a bounded sample."""
    from oracle import oracle
    oracle.build()
    p = oracle.prepare_map(csd, sigma)
    oracle_sample(oracle, p, cfg, tau, seed, 256)                 # thread start-up, table build
    r, dt = oracle_sample(oracle, p, cfg, tau, seed, 4096)        # pilot
    n = int(max(256, min(cfg.n_tracks, budget_s * 4096 / dt)))
    r, dt = oracle_sample(oracle, p, cfg, tau, seed, n)
    return {"value": r["n_evals"] / dt, "unit": UNIT, "cores": r["threads_used"], "kind": "oracle",
            "sample": f"first {n} templates of the workload ({r['n_evals']:.3e} evals, {dt:.1f} s), float64, OpenMP"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle
    oracle.build()
    cfg = synth.CONFIGS[args.config]
    csd, sigma, tau = oracle_inputs(cfg)
    seed = synth.map_seed(cfg, 0)
    p = oracle.prepare_map(csd, sigma)
    oracle_sample(oracle, p, cfg, tau, seed, 256)
    r, dt = oracle_sample(oracle, p, cfg, tau, seed, 4096)
    per_track = dt / 4096
    n = int(max(256, min(cfg.n_tracks, args.ref_step_s / per_track)))
    for i in range(args.warmup):
        oracle_sample(oracle, p, cfg, tau, seed, n, first=i * n)
    evals, t = 0, 0.0
    for i in range(args.steps):
        r, dt = oracle_sample(oracle, p, cfg, tau, seed, n, first=(args.warmup + i) * n)
        evals += r["n_evals"]; t += dt
    n_tau = cfg.n_tau if cfg.tau_mode == "grid" else 1
    value = evals / t
    sample = f"{n} templates per step of the workload's id range ({evals / args.steps:.3e} evals per step), float64, OpenMP"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": int(os.environ.get("WORLD_SIZE", "1")),
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": t / args.steps * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{workload_tag(args.config)} ({cfg.name}): {cfg.n_t}x{cfg.n_f} map, "
                               f"{n_tau} delays ({cfg.tau_mode}); bounded sample of {n} templates per step",
                   "n_t": cfg.n_t, "n_f": cfg.n_f, "n_tau": n_tau, "tau_mode": cfg.tau_mode},
        "cpu_baseline": {"value": value, "unit": UNIT, "kind": "oracle", "cores": r["threads_used"], "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="5", choices=["1", "2", "3", "4", "5", "P"],
                    help="BASELINE.json config (1-5) or P: the shape of the paper's own timing, Table III (context)")
    ap.add_argument("--tracks", type=int, default=0, help="override templates per GPU (debugging)")
    ap.add_argument("--maps", type=int, default=0, help="maps per batch step of config 4 (default: the config's 100)")
    ap.add_argument("--shared-bank", action="store_true",
                    help="config 4 with ONE template bank for every map (seed of map 0) and the bank cache attached: "
                         "S1 + S2 run once, the other maps read the rasterised bank back (SURVEY 8(f) NEXT-2)")
    ap.add_argument("--kernel", default="auto", choices=["auto", "table", "rotation", "reinsch"])
    ap.add_argument("--family", default="quadratic", choices=["quadratic", "cubic", "chirp"], help="template family (G26, G27)")
    ap.add_argument("--norm", default="sqrt_n", choices=["sqrt_n", "mean", "invvar"], help="normalisation of Eq. 8 (G1, G25)")
    ap.add_argument("--call", default="search", choices=["search", "topk", "track_max"],
                    help="entry point a step goes through: st_search, st_search_topk (K = 100) or st_search_track_max; "
                         "with config 4 the latter two run on one map of its shape")
    ap.add_argument("--lib", default="", help="load another build of the same C ABI (the -DST_ABLATE measurement builds of "
                                              "`python -m paper_1401_8060_b200.build --ablate N`); never a bench value")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true", help="default run: skip the short runs of configs 3, 4, P")
    ap.add_argument("--ftmap", action="store_true", help="also time st_set_map_from_strain on strain of the config's duration")
    ap.add_argument("--cpu-budget", type=float, default=15.0, help="seconds of oracle work for cpu_baseline")
    ap.add_argument("--ref-step-s", type=float, default=6.0, help="seconds of oracle work per reference step")
    args = ap.parse_args()
    args.config = "P" if args.config == "P" else int(args.config)
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = max(args.warmup, 1)
    # --gpus N is a request for N ranks, one per GPU.  Under torchrun WORLD_SIZE must agree with it; started
    # as a plain `python bench.py --gpus N` (N > 1) the script re-executes itself under torch.distributed.run.
    world = os.environ.get("WORLD_SIZE")
    if world is None and args.gpus > 1:
        port = os.environ.get("MASTER_PORT", "29531")
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", port, os.path.abspath(__file__), *sys.argv[1:]]
        raise SystemExit(subprocess.call(cmd))
    if world is not None and int(world) != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}: launch {args.gpus} ranks or pass --gpus {world}")
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

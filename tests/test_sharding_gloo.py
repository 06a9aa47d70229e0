"""world_size-2 gloo test of the multi-GPU combination rule (paper: independent jobs
combined by max).  The per-rank search results are produced by the ORACLE
here (no GPU on this box); the rule under test is host logic of the product."""
import os
import socket

import numpy as np
import torch.multiprocessing as mp

from workloads import synth


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _oracle_result(rank_first, n, cfg, csd, sigma, tau):
    from oracle import oracle
    p = oracle.prepare_map(csd, sigma)
    r = oracle.search(p, cfg.f_min, cfg.df, n, cfg.seed, cfg.n_min, cfg.n_max, tau_grid=tau, n_bins=200,
                      track_offset=rank_first)
    return dict(max_snr=float(np.float32(r["max_snr"])), max_snr_f64=r["max_snr"], arg_track=r["arg_track"],
                arg_tau_index=r["arg_tau_index"], arg_tau=r["arg_tau"], arg_params={}, n_evals=r["n_evals"],
                n_pixels=r["n_pixels"], n_candidates=1, hist=r["hist"])


def _worker(rank, world, port, q):
    import torch.distributed as dist
    from paper_1401_8060_b200 import sharding
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = synth.CONFIGS[1]
    csd, sigma, tau = synth.config_inputs(cfg)
    first, n = sharding.split_range(1001, world, rank, base_offset=50)
    mine = _oracle_result(first, n, cfg, csd, sigma, tau)
    both = sharding.all_combine(mine)
    if rank == 0:
        q.put((first, n, both["arg_track"], both["arg_tau_index"], both["max_snr_f64"], both["n_evals"],
               both["hist"].tolist()))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_combination_equals_single_run():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    cfg = synth.CONFIGS[1]
    csd, sigma, tau = synth.config_inputs(cfg)
    whole = _oracle_result(50, 1001, cfg, csd, sigma, tau)
    first, n, arg_track, arg_m, snr, n_evals, hist = got
    assert (first, n) == (50, 501)
    assert (arg_track, arg_m, snr, n_evals) == (whole["arg_track"], whole["arg_tau_index"], whole["max_snr_f64"],
                                                whole["n_evals"])
    assert hist == whole["hist"].tolist()


def test_ranges_partition():
    from paper_1401_8060_b200 import sharding
    for total, world in [(10, 3), (1001, 2), (7, 8), (10 ** 7, 8)]:
        spans = [sharding.split_range(total, world, r, base_offset=5) for r in range(world)]
        assert spans[0][0] == 5 and sum(n for _, n in spans) == total
        for (a, n), (b, _) in zip(spans, spans[1:]):
            assert a + n == b
    assert sharding.rank_range(1000, 3, base_offset=7) == (3007, 1000)


def test_combine_tie_break():
    from paper_1401_8060_b200 import sharding
    base = dict(max_snr=1.0, max_snr_f64=1.0, arg_tau=0.0, arg_params={}, n_evals=10, n_pixels=5, n_candidates=1,
                hist=np.ones(4, dtype=np.uint64))
    a = dict(base, arg_track=9, arg_tau_index=3)
    b = dict(base, arg_track=4, arg_tau_index=7)
    c = dict(base, arg_track=4, arg_tau_index=2)
    empty = dict(base, n_evals=0, n_pixels=0, arg_track=0, arg_tau_index=0, max_snr_f64=float("-inf"),
                 hist=np.zeros(4, dtype=np.uint64))
    r = sharding.combine([a, b, empty, c])
    assert (r["arg_track"], r["arg_tau_index"]) == (4, 2) and r["n_evals"] == 30
    assert r["hist"].tolist() == [3, 3, 3, 3]

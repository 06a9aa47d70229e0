"""CPU-side checks of the product library (no GPU needed): the C-ABI library loads and
exports every symbol include/stochtrack.h declares, the host-only entry points validate
their arguments, and the host copy of S1 (st_track_params / st_debug_track_words) agrees
bit for bit with the oracle.  No compute call touches a device here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_1401_8060_b200 as P
from paper_1401_8060_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return P.load_library()


def test_library_exports_every_declared_symbol(lib):
    header = open(os.path.join(ROOT, "include", "stochtrack.h")).read()
    declared = set(re.findall(r"\b(st_[a-z_]+)\s*\(", header))
    assert declared == set(binding.exported_symbols), declared ^ set(binding.exported_symbols)
    for name in declared:
        assert hasattr(lib, name), name
    assert b"sm_100a" in lib.st_version()


def test_struct_layouts_match_header(tmp_path):
    """ctypes mirrors of the header's structs have the sizes / offsets gcc gives them."""
    import subprocess
    src = tmp_path / "layout.c"
    src.write_text(r"""
#include <stdio.h>
#include <stddef.h>
#include "stochtrack.h"
int main(void) {
  printf("%zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu ", sizeof(st_track), sizeof(st_search_params), sizeof(st_result),
         offsetof(st_search_params, tau_grid), offsetof(st_search_params, hist_out), offsetof(st_search_params, kernel),
         offsetof(st_result, arg_params), offsetof(st_result, gpu_ms), sizeof(st_batch), offsetof(st_batch, csd),
         offsetof(st_batch, seeds));
  printf("%zu %zu ", sizeof(st_ftmap_params), offsetof(st_ftmap_params, n_neighbours));
  printf("%zu %zu %zu\n", sizeof(st_top_entry), offsetof(st_top_entry, snr_f64), offsetof(st_top_entry, tau));
  return 0; }
""")
    exe = tmp_path / "layout"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)])
    got = [int(x) for x in subprocess.check_output([str(exe)]).split()]
    B = binding
    want = [C.sizeof(B.CTrack), C.sizeof(B.CSearchParams), C.sizeof(B.CResult), B.CSearchParams.tau_grid.offset,
            B.CSearchParams.hist_out.offset, B.CSearchParams.kernel.offset, B.CResult.arg_params.offset,
            B.CResult.gpu_ms.offset, C.sizeof(B.CBatch), B.CBatch.csd.offset, B.CBatch.seeds.offset,
            C.sizeof(B.CFtmapParams), B.CFtmapParams.n_neighbours.offset,
            C.sizeof(B.CTopEntry), B.CTopEntry.snr_f64.offset, B.CTopEntry.tau.offset]
    assert B.BATCH_GROUP == int(re.search(r"#define ST_BATCH_GROUP\s+(\d+)", open(os.path.join(ROOT, "include", "stochtrack.h")).read()).group(1))
    assert got == want


def test_create_validates_arguments(lib):
    ctx = C.c_void_p()
    for args in [(0, 64, 1.0, 40.0), (64, 0, 1.0, 40.0), (64, 70000, 1.0, 40.0), (64, 64, 0.0, 40.0),
                 (64, 64, 1.0, -1.0), (2 ** 20 + 1, 64, 1.0, 0.0), (64, 64, float("nan"), 0.0)]:
        assert lib.st_create(C.byref(ctx), *args) == binding.ST_EINVAL, args
        assert not ctx.value
    assert lib.st_create(C.byref(ctx), 1000, 2461, 1.0, 40.0) == 0
    try:
        b512, b64 = lib.st_workspace_bytes(ctx, 512), lib.st_workspace_bytes(ctx, 64)
        assert b512 > b64 > 1000 * 2461 * 8
        assert b512 - b64 >= (512 - 64) * 2461 * 8
        assert lib.st_workspace_bytes(ctx, 0) == 0 and lib.st_workspace_bytes(ctx, 5000) == 0
        # calls that need a workspace fail with ST_ESTATE, never crash
        p = binding.CSearchParams()
        p.n_tracks, p.n_min, p.n_max, p.tau_mode, p.tau_hi = 10, 10, 100, binding.TAU_RANDOM, 0.01
        r = binding.CResult()
        assert lib.st_search(ctx, C.byref(p), C.byref(r)) == binding.ST_ESTATE
        assert b"workspace" in lib.st_last_error(ctx)
        assert lib.st_set_map(ctx, 0, 0, 0) == binding.ST_ESTATE
        assert lib.st_set_workspace(ctx, 0, 1 << 30, 0) == binding.ST_EINVAL
        # the batch / ft-map / time-shift entry points: same rule (state error before any CUDA call)
        b = binding.CBatch()
        b.n_maps = 1
        res = (binding.CResult * 1)()
        assert lib.st_search_batch(ctx, C.byref(b), C.byref(p), res, None) == binding.ST_ESTATE
        fp = binding.CFtmapParams(8192.0, 8192, 4)
        assert lib.st_set_map_from_strain(ctx, 1, 1, 10 ** 7, C.byref(fp), 1, 1 << 30) == binding.ST_ESTATE
        sh = (C.c_int32 * 1)(0)
        assert lib.st_search_timeshifts(ctx, 1, 1, 10 ** 7, C.byref(fp), 1, 1 << 30, 1, sh, None, C.byref(p), res, None) == binding.ST_ESTATE
        assert lib.st_debug_get_map(ctx, 1) == binding.ST_ESTATE
        assert lib.st_ftmap_scratch_bytes(ctx, 8192) >= 2 * 1000 * 2461 * 16 + 4096 * 16
        assert lib.st_ftmap_scratch_bytes(ctx, 1000) == 0 and lib.st_ftmap_scratch_bytes(ctx, 16384) == 0
        t = binding.CTrack()
        assert lib.st_track_params(ctx, 0, 0, 10, 1001, 0.0, 0.0, C.byref(t)) == binding.ST_EINVAL
        assert lib.st_track_params(ctx, 0, 0, 0, 10, 0.0, 0.0, C.byref(t)) == binding.ST_EINVAL
    finally:
        lib.st_destroy(ctx)


def test_explicit_templates_outside_the_band_are_refused(lib):
    """st_score_tracks / st_debug_rasterise_track: the rasteriser's fast-path guard is sized for control points inside
    the band (as every bank member's are), so explicit templates beyond it are refused on the host (ST_EINVAL) rather
    than rasterised without the bit-exactness guarantee; templates inside pass on to the next check (here: no
    workspace, ST_ESTATE).  No CUDA call is reached."""
    ctx = C.c_void_p()
    assert lib.st_create(C.byref(ctx), 100, 50, 1.0, 40.0) == 0
    try:
        p = binding.CSearchParams()
        p.tau_mode, p.tau_hi = binding.TAU_RANDOM, 0.01
        good = dict(N=50, j0=10, a=20.0, y0=0.0, y1=50.0, y2=25.5, tau=0.0, y3=0.0)

        def score(family=0, **kw):
            p.family = family
            t = (binding.CTrack * 1)(binding.CTrack(**{**good, **kw}))
            return lib.st_score_tracks(ctx, C.byref(p), t, 1, 256), lib.st_last_error(ctx).decode()

        def raster(family=0, **kw):
            t = binding.CTrack(**{**good, **kw})
            return lib.st_debug_rasterise_track(ctx, C.byref(t), family, 256), lib.st_last_error(ctx).decode()

        for call in (score, raster):
            assert call()[0] == binding.ST_ESTATE                           # inside the band, edges included
            for bad in (dict(y0=-1e-9), dict(y1=50.000001), dict(y2=1e9), dict(y1=float("nan")), dict(a=0.0), dict(a=50.0),
                        dict(j0=51), dict(N=0)):
                rc, msg = call(**bad)
                assert rc == binding.ST_EINVAL, (call.__name__, bad)
            assert "inside the band" in call(y2=-3.0)[1]
            # y3 counts for the cubic family only; the chirp law uses y0 alone
            assert call(y3=77.0)[0] == binding.ST_ESTATE and call(binding.FAMILY_CUBIC, y3=77.0)[0] == binding.ST_EINVAL
            assert call(binding.FAMILY_CHIRP, y1=-5.0, y2=1e6, y3=99.0)[0] == binding.ST_ESTATE
            assert call(binding.FAMILY_CHIRP, y0=50.5)[0] == binding.ST_EINVAL
            assert call(3)[0] == binding.ST_EINVAL
    finally:
        lib.st_destroy(ctx)


def test_host_track_generator_matches_oracle_bit_for_bit(lib, orc):
    """S1 on the host side of the product == O1 + O2 of the oracle (words and parameters)."""
    shapes = [(0, 64, 64, 64, 64), (1, 250, 961, 10, 250), (2, 500, 2461, 10, 500), (4, 1000, 2461, 10, 1000),
              (3 * 2 ** 32 + 7, 500, 2461, 10, 500)]
    ids = list(range(300)) + [2 ** 32 - 1, 2 ** 32, 2 ** 40 + 17, 2 ** 62]
    for seed, n_t, n_f, n_min, n_max in shapes:
        for tid in ids:
            assert np.array_equal(P.st_track_words(seed, tid), orc.track_words(seed, tid))
            g = P.st_track_params(n_t, n_f, seed, tid, n_min, n_max, -0.01, 0.01)
            o = orc.track_params(seed, tid, n_t, n_f, n_min, n_max, -0.01, 0.01)
            for f in ("N", "j0", "a", "y0", "y1", "y2", "tau"):
                assert getattr(g, f) == getattr(o, f), (seed, tid, f)
    # the other template families (G26: y3 from the eighth Philox word; G27: the chirp law uses N, j0, a, y0, tau)
    for family in (P.FAMILY_CUBIC, P.FAMILY_CHIRP):
        for tid in ids[:60] + ids[-4:]:
            g = P.st_track_params(500, 2461, 2, tid, 10, 500, -0.01, 0.01, family=family)
            o = orc.track_params(2, tid, 500, 2461, 10, 500, -0.01, 0.01, family=family)
            for f in ("N", "j0", "a", "y0", "y1", "y2", "tau", "y3"):
                assert getattr(g, f) == getattr(o, f), (family, tid, f)
    with pytest.raises(P.StError):
        P.st_track_params(500, 2461, 2, 0, 10, 500, family=3)


def test_combine_results_through_the_c_abi(lib):
    """st_combine_results (G12), called through ctypes with no binding in between: the winner under
    (larger float64 SNR, smaller template id, smaller delay index), runs that scored nothing ignored, counts summed,
    histograms summed exactly, flags OR-ed; argument errors refused."""
    R = binding.CResult

    def res(snr, track, m, evals=10, **kw):
        r = R()
        r.max_snr, r.max_snr_f64, r.arg_track, r.arg_tau_index, r.n_evals, r.n_pixels, r.n_candidates = snr, snr, track, m, evals, evals // 2, 1
        for k, v in kw.items():
            setattr(r, k, v)
        return r

    runs = [res(1.0, 9, 3, flags=2), res(1.0, 4, 7, n_launches=3), res(float("-inf"), 0, 0, evals=0), res(1.0, 4, 2, gpu_ms=2.5),
            res(0.5, 1, 0, n_deferred=7)]
    arr = (R * len(runs))(*runs)
    h = [np.arange(4, dtype=np.uint64) + i for i in range(len(runs))]
    h[2][:] = 0
    hp = (C.POINTER(C.c_uint64) * len(runs))(*[x.ctypes.data_as(C.POINTER(C.c_uint64)) for x in h])
    hp[4] = None                                           # a run without a histogram
    out, idx, hist = R(), C.c_int32(-1), np.full(4, 99, dtype=np.uint64)
    assert lib.st_combine_results(arr, hp, len(runs), 4, C.byref(out), hist.ctypes.data_as(C.POINTER(C.c_uint64)), C.byref(idx)) == 0
    assert idx.value == 3 and (out.arg_track, out.arg_tau_index, out.max_snr_f64) == (4, 2, 1.0)
    assert (out.n_evals, out.n_pixels, out.n_candidates, out.n_launches, out.n_deferred, out.flags) == (40, 20, 4, 3, 7, 2)
    assert out.gpu_ms == 2.5 and out.max_snr == 1.0
    assert hist.tolist() == (h[0] + h[1] + h[3]).tolist()
    # a larger float64 value wins whatever the ids; nothing scored anywhere -> the first entry comes back
    arr2 = (R * 2)(res(2.0, 100, 9), res(2.5, 200, 11))
    assert lib.st_combine_results(arr2, None, 2, 0, C.byref(out), None, C.byref(idx)) == 0 and idx.value == 1 and out.arg_track == 200
    arr3 = (R * 2)(res(float("-inf"), 5, 0, evals=0), res(float("-inf"), 6, 0, evals=0))
    assert lib.st_combine_results(arr3, None, 2, 0, C.byref(out), None, None) == 0 and out.arg_track == 5 and out.n_evals == 0
    for bad in ((None, None, 2, 0, C.byref(out), None, None), (arr2, None, 0, 0, C.byref(out), None, None),
                (arr2, None, 2, 5000, C.byref(out), None, None), (arr2, None, 2, 4, C.byref(out), hist.ctypes.data_as(C.POINTER(C.c_uint64)), None),
                (arr2, None, 2, 0, None, None, None)):
        assert lib.st_combine_results(*bad) == binding.ST_EINVAL


def test_binding_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        P.Stochtrack(64, 64, 1.0, 40.0)


def test_product_does_not_import_oracle():
    """The product path must not route through oracle/ (or read _work/)."""
    pkg = os.path.join(ROOT, "paper_1401_8060_b200")
    bad = re.compile(r"(^|\s)(from|import)\s+oracle\b|oracle/|oracle\.py|stochtrack_oracle|_work/|/_work")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not bad.search(src), f

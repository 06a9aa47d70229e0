"""st_score_random_noalloc: the scoring call for hosts that cannot lend the library device memory.

Some users of this library cannot allocate on the GPU at the point where they call it: a pipeline stage
inside a framework whose memory pool took the whole card at start-up (a later cudaMalloc just fails), an
online analysis that must not allocate or free while it is live (both synchronise the whole device), or a
component that is only ever handed its input and output buffers.  For them the library carries its scratch
inside its own device image (a static array, ST_NOALLOC_SCRATCH_BYTES on every GPU that loads the library,
maps of at most ST_NOALLOC_MAX_PIXELS pixels) and offers this one call, which takes nothing but the
caller's map and the caller's output buffer.

What is checked here:
  * (CPU) the size limit and the unsupported options are refused with a readable message before any CUDA
    call is made, and the body of the entry point names no allocating routine;
  * (GPU) its output equals, bit for bit, what the ordinary path (st_set_map + st_debug_scores with a
    caller-allocated workspace) writes for the same inputs -- on consecutive calls with different map
    shapes, sigma layouts, normalisations and template ranges, so that anything a call wrongly inherited
    from the array's previous contents would show -- and agrees with the float64 oracle within the G13
    tolerance of the parity tests; free device memory does not move across the calls.

This file is named so that pytest collects it after every other test file: `pytest -x` stops at the first
failure, and a failure here must not hide the parity tests.  It passes alone in a fresh process (the first
call on the device then does the one-off symbol look-up) as well as at the end of the whole suite.
"""
import ctypes as C
import os
import re

import numpy as np
import pytest

from workloads import synth
from helpers import snr_close

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def pkg():
    import paper_1401_8060_b200 as P
    from paper_1401_8060_b200 import build
    build.build()
    P.load_library()            # fails loudly if the extension is missing
    return P


def _params(P, n_tracks=10, n_min=10, n_max=64, **kw):
    from paper_1401_8060_b200 import binding
    p = binding.CSearchParams()
    p.n_tracks, p.n_min, p.n_max = n_tracks, n_min, n_max
    p.tau_mode, p.tau_lo, p.tau_hi = P.TAU_RANDOM, -0.01, 0.01
    for k, v in kw.items():
        setattr(p, k, v)
    return p


def test_limits_are_refused_on_the_host_with_a_message(pkg):
    """No GPU needed: every refusal below happens before the first CUDA call (dummy non-null pointers)."""
    from paper_1401_8060_b200 import binding
    P, L = pkg, pkg.load_library()
    header = open(os.path.join(ROOT, "include", "stochtrack.h")).read()
    assert int(re.search(r"#define ST_NOALLOC_MAX_PIXELS\s+(\d+)", header).group(1)) == P.NOALLOC_MAX_PIXELS
    assert int(re.search(r"#define ST_NOALLOC_SCRATCH_BYTES\s+(\d+)", header).group(1)) == P.NOALLOC_SCRATCH_BYTES
    assert P.NOALLOC_SCRATCH_BYTES < 4 << 20                     # "modest": under 4 MiB per GPU
    err = C.create_string_buffer(512)

    def call(n_t, n_f, p, csd=256, sigma=0, kind=0, out=256, df=1.0, f_min=40.0):
        return L.st_score_random_noalloc(csd, sigma, kind, n_t, n_f, df, f_min, C.byref(p) if p is not None else None,
                                         out, None, err, len(err))

    # a map beyond the static scratch: config 3's 500 x 2461, and one pixel past the limit
    assert call(500, 2461, _params(P, n_max=500)) == binding.ST_ENOSPC
    msg = err.value.decode()
    assert "ST_NOALLOC_MAX_PIXELS" in msg and "1230500" in msg and str(P.NOALLOC_MAX_PIXELS) in msg
    assert call(P.NOALLOC_MAX_PIXELS + 1, 1, _params(P)) == binding.ST_ENOSPC
    # the message buffer is optional
    p_big = _params(P, n_max=500)
    assert L.st_score_random_noalloc(256, 0, 0, 500, 2461, 1.0, 40.0, C.byref(p_big), 256, None, None, 0) == binding.ST_ENOSPC
    # what the entry point does not offer, and plain bad arguments
    for p, frag in [(_params(P, tau_mode=P.TAU_GRID), "ST_TAU_RANDOM"), (_params(P, norm=P.NORM_INVVAR), "norm"),
                    (_params(P, family=P.FAMILY_CHIRP), "family"), (_params(P, n_min=0), "n_min"),
                    (_params(P, n_max=65), "n_max"), (_params(P, tau_lo=0.02), "tau"),
                    (_params(P, n_tracks=2 ** 31 + 1), "2^31")]:
        assert call(64, 64, p) == binding.ST_EINVAL, frag
        assert frag in err.value.decode(), (frag, err.value)
    assert call(64, 64, None) == binding.ST_EINVAL
    assert call(64, 64, _params(P), csd=0) == binding.ST_EINVAL
    assert call(64, 64, _params(P), out=0) == binding.ST_EINVAL
    assert call(64, 64, _params(P), kind=1, sigma=0) == binding.ST_EINVAL
    assert call(64, 64, _params(P), kind=3, sigma=256) == binding.ST_EINVAL
    assert call(0, 64, _params(P)) == binding.ST_EINVAL and call(64, 64, _params(P), df=0.0) == binding.ST_EINVAL
    # an empty range is not an error and touches nothing
    assert call(64, 64, _params(P, n_tracks=0), out=0) == binding.ST_OK and err.value == b""


def test_entry_point_names_no_allocating_routine():
    """The part of the source that implements the call (comments stripped) contains no allocation, no free
    and no stream / event creation; its scratch address comes from cudaGetSymbolAddress."""
    src = open(os.path.join(ROOT, "paper_1401_8060_b200", "csrc", "stochtrack_api.cu")).read()
    body = src[src.index("entry point without allocations"):]
    code = "\n".join(line.split("//")[0] for line in body.splitlines())
    for banned in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaHostRegister", "cudaEventCreate", "cudaStreamCreate",
                   "cudaMemPool", "malloc(", "new ", "std::vector", "DevGuard", "st_ctx"):
        assert banned not in code, banned
    assert "static __device__ __align__(256) unsigned char g_noalloc_scratch" in code
    assert "cudaGetSymbolAddress(&ptr, g_noalloc_scratch)" in code
    # host code hands kernels the looked-up pointer, never the symbol itself
    assert len(re.findall(r"g_noalloc_scratch", code)) == 2


# (n_t, n_f, f_min, sigma layout, norm, seed, n_min, n_max, track_offset, n_tracks)
CALLS = [
    (250, 961, 40.0, "per_f", "NORM_SQRT_N", 11, 10, 250, 0, 20_001),                 # BASELINE configs[1] shape, ragged count
    (64, 64, 40.0, "per_pixel", "NORM_MEAN", 12, 1, 64, 2 ** 33 + 5, 777),            # smaller map: most of the array is stale
    (500, 151, 100.0, "none", "NORM_SQRT_N", 13, 70, 500, 123_456, 5_000),            # Table III shape
    (250, 961, 40.0, "per_f", "NORM_SQRT_N", 11, 10, 250, 0, 20_001),                 # the first call again
]


def _inputs(n_t, n_f, sigma_kind, seed):
    csd = synth.noise_csd(n_t, n_f, 900 + seed)
    sigma = None
    if sigma_kind == "per_f":
        sigma = synth.make_sigma("per_f", 0.2, n_t, n_f, 900 + seed)
    elif sigma_kind == "per_pixel":
        sigma = synth.make_sigma("per_pixel", 0.3, n_t, n_f, 900 + seed).copy()
        sigma[3, 5], sigma[10, 0], sigma[63, 63] = 0.0, -1.0, np.inf      # masked pixels (G11)
    return csd, sigma


@pytest.mark.gpu
def test_consecutive_calls_match_the_workspace_path_bit_for_bit(pkg, orc):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    P = pkg
    tau_range = (-synth.TAU_MAX, synth.TAU_MAX)
    # everything the caller owns is allocated up front: inputs, outputs, and the reference path's contexts
    prepared = []
    for n_t, n_f, f_min, skind, norm, seed, n_min, n_max, first, count in CALLS:
        csd, sigma = _inputs(n_t, n_f, skind, seed)
        d_csd = torch.from_numpy(csd).cuda()
        d_sigma = torch.from_numpy(sigma).cuda() if sigma is not None else None
        out = torch.full((count,), float("nan"), dtype=torch.float32, device="cuda")
        st = P.Stochtrack(n_t, n_f, 1.0, f_min, max_n_tau=64)
        prepared.append((csd, sigma, d_csd, d_sigma, out, st))
    # reference: the ordinary path, workspace allocated by the caller
    want = []
    for (n_t, n_f, f_min, skind, norm, seed, n_min, n_max, first, count), (csd, sigma, d_csd, d_sigma, out, st) in zip(CALLS, prepared):
        st.set_map(d_csd, d_sigma)
        want.append(st.debug_scores(seed, n_min, n_max, first, count, tau_range=tau_range, norm=getattr(P, norm))[:, 0])
    torch.cuda.synchronize()
    # the calls under test, back to back on one stream, nothing synchronised or allocated in between
    free = []
    for i, ((n_t, n_f, f_min, skind, norm, seed, n_min, n_max, first, count), (csd, sigma, d_csd, d_sigma, out, st)) in enumerate(zip(CALLS, prepared)):
        P.score_random_noalloc(d_csd, d_sigma, 1.0, f_min, count, seed, n_min, n_max, tau_range, out,
                               norm=getattr(P, norm), track_offset=first)
        if i == 0:
            torch.cuda.synchronize()       # the first call on this device may have loaded code / looked up the symbol
        free.append(torch.cuda.mem_get_info()[0])
    torch.cuda.synchronize()
    free.append(torch.cuda.mem_get_info()[0])
    assert len(set(free)) == 1, f"free device memory moved across the calls: {free}"
    for i, (call, (csd, sigma, d_csd, d_sigma, out, st)) in enumerate(zip(CALLS, prepared)):
        got = out.cpu().numpy()
        assert np.isfinite(got).all(), i
        assert np.array_equal(got, want[i]), (i, np.abs(got - want[i]).max())
    assert np.array_equal(prepared[0][4].cpu().numpy(), prepared[3][4].cpu().numpy())
    # and against the oracle, with the parity tests' tolerance (G13), on two of the calls
    for i in (1, 2):
        n_t, n_f, f_min, skind, norm, seed, n_min, n_max, first, count = CALLS[i]
        csd, sigma = prepared[i][0], prepared[i][1]
        ref = orc.search(orc.prepare_map(csd, sigma), f_min, 1.0, count, seed, n_min, n_max, tau_range=tau_range,
                         track_offset=first, norm=getattr(P, norm), dump_snr=True)["snr"][:, 0]
        s0 = np.sqrt(0.5) if norm == "NORM_SQRT_N" else np.sqrt(0.5 / n_max)
        ok, worst = snr_close(prepared[i][4].cpu().numpy(), ref, s0=s0)
        assert ok, (i, worst)


@pytest.mark.gpu
def test_oversized_map_is_refused_on_the_gpu_too(pkg):
    """With real device buffers: the refusal leaves the output untouched and the next call still works."""
    import torch
    P = pkg
    csd = torch.zeros((500, 2461), dtype=torch.complex64, device="cuda")
    out = torch.full((100,), -7.0, dtype=torch.float32, device="cuda")
    with pytest.raises(P.StError, match="ST_ENOSPC.*ST_NOALLOC_MAX_PIXELS"):
        P.score_random_noalloc(csd, None, 1.0, 40.0, 100, 1, 10, 500, (-0.01, 0.01), out)
    torch.cuda.synchronize()
    assert (out == -7.0).all()
    small = torch.ones((64, 64), dtype=torch.complex64, device="cuda")       # p = 1: SNR(tau) = N^-1/2 sum cos(2 pi f tau)
    P.score_random_noalloc(small, None, 1.0, 40.0, 100, 1, 64, 64, (0.0, 0.0), out)
    torch.cuda.synchronize()
    assert torch.allclose(out, torch.full_like(out, 8.0), rtol=1e-6)          # tau = 0: sum of 64 ones / sqrt(64)

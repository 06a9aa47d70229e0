"""Float64 CPU oracle of the ft-map construction (the step before the hot path).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline legs may import this module; it imports nothing from the CUDA package.  Plain NumPy,
float64 throughout, written in the paper's order so that it can be checked against it by eye;
`numpy.fft.fft` is the one library primitive (the discrete Fourier transform itself).

What it computes, with the passage each step follows:

  F1  the strain series s_I(t'), s_J(t') are split into segments of `seg_len` samples, consecutive
      segments overlapping by 50 % and weighted by a Hann window
  F2  each segment is Fourier transformed: s~_I(t; f), s~_J(t; f)
  F3  P'_I(t; f), P'_J(t; f): the auto-power in the segments neighbouring t (Eq. A3)
  F4  the complex SNR map p(t; f) = lambda s~_I^* s~_J  with  lambda = (1/N) sqrt(2 / (P'_I P'_J))
                                                              (Eq. 7; Eq. A4)

Readings (G19-G22), where the paper is silent:
  G19  Hann window w_n = (1 - cos(2 pi n / L)) / 2, n = 0..L-1 (the "periodic" form); segment j
       starts at sample j * L/2; the DFT sign is e^{-2 pi i k n / L}; bin k <-> frequency k fs / L.
  G20  "neighbouring segments": the n_nb segments on either side of t that do NOT share samples
       with it, j' = j +- 2 ... j +- (n_nb + 1) (j +- 1 overlap t by 50 %), those that exist;
       P' is the plain mean of |s~|^2 over them.  No neighbour at all -> the pixel is masked (p = 0).
  G21  the DFT normalisation N of A2/A4 and the factor-2 inconsistency between A2 and A4 (G9)
       cancel in p when P' is measured with the same transform: with P' = mean |s~|^2,
       p = sqrt(2) s~_I^* s~_J / sqrt(P'_I P'_J), which makes Re[e^{i phi} p] unit variance on
       stationary independent Gaussian noise in the limit of many neighbours (A1-A3).
  G22  a pixel whose P'_I P'_J is zero or not finite is masked (p = 0), as G11.
  G23  time shifts are whole segments, cyclic over the map: J's segment (j + s) mod n_t
       meets I's segment j; P'_J is taken around J's own segment.
"""
import numpy as np


def hann(seg_len):
    """G19: w_n = (1 - cos(2 pi n / L)) / 2."""
    n = np.arange(seg_len, dtype=np.float64)
    return 0.5 * (1.0 - np.cos(2.0 * np.pi * n / seg_len))


def n_segments(n_samples, seg_len):
    """Number of 50 %-overlapping segments that fit in n_samples (F1)."""
    hop = seg_len // 2
    return 0 if n_samples < seg_len else (n_samples - seg_len) // hop + 1


def strain_spectrogram(s, seg_len, n_t, k_lo, n_f):
    """F1 + F2 for one detector: s~(t_j; f_k), j < n_t, k_lo <= k < k_lo + n_f, complex128 [n_t][n_f]."""
    s = np.asarray(s, dtype=np.float64)
    hop = seg_len // 2
    w = hann(seg_len)
    out = np.zeros((n_t, n_f), dtype=np.complex128)
    for j in range(n_t):
        seg = s[j * hop: j * hop + seg_len] * w
        out[j] = np.fft.fft(seg)[k_lo:k_lo + n_f]
    return out


def neighbour_power(st, n_nb):
    """F3 (G20): P'(t_j; f) = mean of |s~(t_j'; f)|^2 over j' = j +- 2 .. j +- (n_nb + 1) inside the map.
    Returns (P' float64 [n_t][n_f], number of neighbours used int [n_t])."""
    n_t = st.shape[0]
    pw = np.abs(st) ** 2
    out = np.zeros(pw.shape, dtype=np.float64)
    cnt = np.zeros(n_t, dtype=np.int64)
    for j in range(n_t):
        acc = np.zeros(pw.shape[1], dtype=np.float64)
        for d in range(2, n_nb + 2):
            for jj in (j - d, j + d):
                if 0 <= jj < n_t:
                    acc += pw[jj]
                    cnt[j] += 1
        out[j] = acc / cnt[j] if cnt[j] else 0.0
    return out, cnt


def ftmap(s_i, s_j, fs, seg_len, n_t, f_min, n_f, n_nb):
    """F1-F4: (p complex128 [n_t][n_f], s~_I, s~_J, P'_I, P'_J).  df = fs / seg_len; f_min = k_lo df."""
    df = fs / seg_len
    k_lo = int(round(f_min / df))
    if abs(k_lo * df - f_min) > 1e-9 * df or k_lo + n_f > seg_len // 2 or n_segments(len(s_i), seg_len) < n_t:
        raise ValueError("band or duration outside the data")
    st_i = strain_spectrogram(s_i, seg_len, n_t, k_lo, n_f)
    st_j = strain_spectrogram(s_j, seg_len, n_t, k_lo, n_f)
    p_i, cnt = neighbour_power(st_i, n_nb)
    p_j, _ = neighbour_power(st_j, n_nb)
    prod = p_i * p_j
    ok = np.isfinite(prod) & (prod > 0.0) & (cnt[:, None] > 0)
    p = np.zeros(st_i.shape, dtype=np.complex128)
    p[ok] = np.sqrt(2.0) * np.conj(st_i[ok]) * st_j[ok] / np.sqrt(prod[ok])      # G21
    return p, st_i, st_j, p_i, p_j


def ftmap_timeshift(st_i, st_j, n_nb, shift):
    """Time-shifted background map (significance is evaluated from n_ts time-shift analyses;
    reading G23): detector J's segment (j + shift) mod n_t is paired with detector I's segment j, so
    that no astrophysical signal is coherent between the two; every detector's P' is taken around its
    own segment.  st_i, st_j: the strain spectrograms of `ftmap` (F1 + F2).  shift = 0 is `ftmap`."""
    n_t = st_i.shape[0]
    p_i, c_i = neighbour_power(st_i, n_nb)
    p_j, c_j = neighbour_power(st_j, n_nb)
    idx = (np.arange(n_t) + shift) % n_t
    sj, pj, cj = st_j[idx], p_j[idx], c_j[idx]
    prod = p_i * pj
    ok = np.isfinite(prod) & (prod > 0.0) & (c_i[:, None] > 0) & (cj[:, None] > 0)
    p = np.zeros(st_i.shape, dtype=np.complex128)
    p[ok] = np.sqrt(2.0) * np.conj(st_i[ok]) * sj[ok] / np.sqrt(prod[ok])
    return p

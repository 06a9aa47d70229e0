// st_ftmap.cuh -- ft-map construction on the GPU: two strain series -> the complex SNR map p(t; f)
// that the search consumes, with no host round trip.
//
//   k_ft_twiddles   W_L^t = e^{-2 pi i t / L}, t < L/2, float64 (sincospi)
//   k_ft_segments   F1 + F2: one CTA per segment: Hann window, ONE complex FFT of length L for both
//                   detectors (z = w (s_I + i s_J)), in shared memory, float64; the band
//                   [k_lo, k_lo + n_f) of s~_I and s~_J is separated and stored
//   k_ft_normalise  F3 + F4: P' from the neighbouring segments (Eq. A3),
//                   p = sqrt(2) s~_I^* s~_J / sqrt(P'_I P'_J) (Eqs. 7, A4; readings G19-G22 of DESIGN.md)
//
// Float64 because strain spectra span many decades (a float32 transform leaks rounding error of the
// loud low-frequency band into the quiet one); the transform is ~1e9 flop per map and is not the
// bottleneck: k_ft_segments is bound by shared-memory bandwidth, k_ft_normalise by HBM/L2 traffic.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace st {

constexpr int kFtMaxLen = 8192;        // L <= 8192: L double2 = 128 KB of shared memory
constexpr int kFtThreads = 1024;

__global__ void k_ft_twiddles(int L, double2* __restrict__ W)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= L / 2) return;
    double s, c;
    sincospi(-2.0 * (double)t / (double)L, &s, &c);
    W[t] = make_double2(c, s);
}

__device__ __forceinline__ double2 cmul(double2 a, double2 b)
{
    return make_double2(fma(a.x, b.x, -(a.y * b.y)), fma(a.x, b.y, a.y * b.x));
}

// One CTA per segment j: samples [j L/2, j L/2 + L).  In-place radix-2 decimation-in-frequency FFT
// (Gentleman-Sande), two stages per pass over shared memory, output in bit-reversed order.  With
// z = w (s_I + i s_J):  s~_I(k) = (Z_k + conj Z_{L-k}) / 2,  s~_J(k) = (Z_k - conj Z_{L-k}) / (2 i).
__global__ void __launch_bounds__(kFtThreads, 1)
k_ft_segments(const double* __restrict__ s_i, const double* __restrict__ s_j, int L, int log2L,
              const double2* __restrict__ W, int k_lo, int n_f,
              double2* __restrict__ st_i, double2* __restrict__ st_j)
{
    extern __shared__ __align__(16) unsigned char smem[];
    double2* x = reinterpret_cast<double2*>(smem);
    const int j = blockIdx.x;
    const size_t base = (size_t)j * (size_t)(L / 2);
    for (int n = threadIdx.x; n < L; n += blockDim.x) {
        // Hann (G19): cos(2 pi n / L) from the twiddle table (W[t].x = cos(2 pi t / L), t < L/2)
        const double cs = n < L / 2 ? W[n].x : (n == L / 2 ? -1.0 : W[L - n].x);
        const double w = 0.5 * (1.0 - cs);
        x[n] = make_double2(w * s_i[base + n], w * s_j[base + n]);
    }
    __syncthreads();
    // two radix-2 stages per pass, fused in registers (the arithmetic and the bit-reversed output order
    // are those of plain radix-2; shared-memory traffic and barriers are halved)
    int s = 0;
    for (; s + 2 <= log2L; s += 2) {
        const int half = L >> (s + 1), quarter = half >> 1;
        for (int b = threadIdx.x; b < L / 4; b += blockDim.x) {
            const int pos = b & (quarter - 1);
            const int i0 = ((b - pos) << 2) + pos, i1 = i0 + quarter, i2 = i0 + half, i3 = i2 + quarter;
            const double2 x0 = x[i0], x1 = x[i1], x2 = x[i2], x3 = x[i3];
            const double2 u0 = make_double2(x0.x + x2.x, x0.y + x2.y);
            const double2 u1 = make_double2(x1.x + x3.x, x1.y + x3.y);
            const double2 u2 = cmul(make_double2(x0.x - x2.x, x0.y - x2.y), W[(size_t)pos << s]);
            const double2 u3 = cmul(make_double2(x1.x - x3.x, x1.y - x3.y), W[(size_t)(pos + quarter) << s]);
            const double2 w1 = W[(size_t)pos << (s + 1)];
            x[i0] = make_double2(u0.x + u1.x, u0.y + u1.y);
            x[i1] = cmul(make_double2(u0.x - u1.x, u0.y - u1.y), w1);
            x[i2] = make_double2(u2.x + u3.x, u2.y + u3.y);
            x[i3] = cmul(make_double2(u2.x - u3.x, u2.y - u3.y), w1);
        }
        __syncthreads();
    }
    for (; s < log2L; ++s) {                                     // odd log2 L: one plain radix-2 stage
        const int half = L >> (s + 1);
        for (int b = threadIdx.x; b < L / 2; b += blockDim.x) {
            const int pos = b & (half - 1);
            const int i0 = ((b - pos) << 1) + pos, i1 = i0 + half;
            const double2 a = x[i0], c = x[i1];
            x[i0] = make_double2(a.x + c.x, a.y + c.y);
            x[i1] = cmul(make_double2(a.x - c.x, a.y - c.y), W[(size_t)pos << s]);
        }
        __syncthreads();
    }
    const int shift = 32 - log2L;
    for (int q = threadIdx.x; q < n_f; q += blockDim.x) {
        const int k = k_lo + q;
        const double2 zk = x[__brev((unsigned)k) >> shift];
        const double2 zm = x[__brev((unsigned)((L - k) & (L - 1))) >> shift];
        // Z_k + conj Z_{L-k} = (zk.x + zm.x, zk.y - zm.y);  Z_k - conj Z_{L-k} = (zk.x - zm.x, zk.y + zm.y)
        st_i[(size_t)j * n_f + q] = make_double2(0.5 * (zk.x + zm.x), 0.5 * (zk.y - zm.y));
        st_j[(size_t)j * n_f + q] = make_double2(0.5 * (zk.y + zm.y), -0.5 * (zk.x - zm.x));
    }
}

// P'(t_j; f) = mean |s~|^2 over j' = j +- 2 .. j +- (n_nb + 1) inside the map (G20); masked pixels -> 0.
// `shift` (time-shifted background maps, G23): detector J's segment js = (j + shift) mod n_t meets
// detector I's segment j; each detector's P' comes from the neighbours of ITS OWN segment.
__global__ void __launch_bounds__(256)
k_ft_normalise(const double2* __restrict__ st_i, const double2* __restrict__ st_j, int n_t, int n_f, int n_nb,
               int shift, float2* __restrict__ p)
{
    const size_t n_pix = (size_t)n_t * (size_t)n_f;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_pix; i += (size_t)gridDim.x * blockDim.x) {
        const int j = (int)(i / (size_t)n_f), q = (int)(i % (size_t)n_f);
        const int js = (j + shift) % n_t;
        double pi = 0.0, pj = 0.0;
        int ci = 0, cj = 0;
        for (int d = 2; d <= n_nb + 1; ++d) {
            for (int sgn = -1; sgn <= 1; sgn += 2) {
                const int ji = j + sgn * d, jj = js + sgn * d;
                if (ji >= 0 && ji < n_t) {
                    const double2 a = st_i[(size_t)ji * n_f + q];
                    pi += a.x * a.x + a.y * a.y;
                    ++ci;
                }
                if (jj >= 0 && jj < n_t) {
                    const double2 b = st_j[(size_t)jj * n_f + q];
                    pj += b.x * b.x + b.y * b.y;
                    ++cj;
                }
            }
        }
        float2 out = make_float2(0.0f, 0.0f);
        if (ci > 0 && cj > 0) {
            const double prod = (pi / (double)ci) * (pj / (double)cj);
            if (prod > 0.0 && isfinite(prod)) {
                const double2 a = st_i[i], b = st_j[(size_t)js * n_f + q];
                const double sc = sqrt(2.0) / sqrt(prod);                           // G21
                // conj(a) * b
                out = make_float2((float)(sc * (a.x * b.x + a.y * b.y)), (float)(sc * (a.x * b.y - a.y * b.x)));
            }
        }
        p[i] = out;
    }
}

}  // namespace st

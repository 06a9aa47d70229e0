// st_kernels.cuh -- the sm_100a kernels of the all-sky stochtrack hot path.
//
//   k_prepare_map      S0  p = CSD / sigma                     Eq. 7
//   k_build_w_table    twiddles W[k][m] = e^{2 pi i f_k tau_m}        (G6, G7)
//   k_build_bin_tables per-bin constants of the uniform-grid recurrences
//   k_score_cheb       S1-S4, uniform tau grid, the production kernel: lanes over pixels, the term of
//                      Eq. 8 advanced along tau by a packed two-sided Chebyshev recurrence (one FFMA2 +
//                      one FADD2 per two evaluations); builds: search / capture / per-template maximum,
//                      fast / general (two-class, cubic and chirp families, inverse-variance weighting,
//                      explicit templates), bank cache fill / read, one chunk or two chunks per pass,
//                      one-pass software-pipelined
//   k_score_reinsch    S1-S4, uniform tau grid: Reinsch's form of the recurrence (3 operations per evaluation)
//   k_score_recur      S1-S4, uniform tau grid: complex rotation recurrence (5 operations, any step angle)
//   k_score_table      S1-S4, any tau grid: lanes over tau, W read through L1/L2
//   k_score_random     S1-S4, the paper's mode: one random delay per template
//   k_finalize         S4: float64 re-score of the near-max candidates, argmax (G12)
//   k_rescore_cands    float64 scores of the captured samples (st_search_topk)
//   k_debug_rasterise  parity exports of S1+S2
//
// One warp owns one template at a time (templates are independent: PAPER.md:25,
// :242 "embarrassingly parallel").  No tensor cores: per template the sum of
// Eq. 8 is a gather along the track, not a dense contraction.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "st_track.cuh"

// -DST_CHECKED (python -m paper_1401_8060_b200.build --checked): device-side assertions on every index the
// kernels form (compute-sanitizer is not available on the GPU pool); a failed one traps the kernel and the
// next API call returns ST_ECUDA.  Compiled out of the production library.
#ifdef ST_CHECKED
#include <assert.h>
#define ST_ASSERT(cond) assert(cond)
#else
#define ST_ASSERT(cond) ((void)0)
#endif

namespace st {

constexpr int kWarp = 32;
constexpr unsigned kFull = 0xFFFFFFFFu;
constexpr double kTwoPi = 6.283185307179586476925286766559;

struct Cand {            // a near-max sample kept for the float64 re-score
    float snr;
    uint32_t m;
    uint64_t id;
};

struct WarpBest {        // per-warp best under the G12 total order (overflow fallback)
    float snr;
    uint32_t m;
    uint64_t id;
    uint32_t valid;
    uint32_t pad;
};

struct Scalars {         // device scalars of one search, zeroed by the host
    unsigned long long counter;     // next template index of the current launch
    unsigned long long n_pixels;    // sum of N_i
    uint32_t gmax_bits;             // ordered-uint encoding of the float32 maximum
    uint32_t cand_count;
    uint32_t overflow;
    uint32_t n_deferred;            // templates the fast Chebyshev build handed to the two-class build (per launch)
    uint32_t n_deferred_total;      // the same summed over the launches of the search
    uint32_t pad;
};

struct DeviceResult {
    float    max_snr;
    int32_t  arg_m;
    double   snr_f64;
    uint64_t arg_id;
    double   arg_tau;
    Track    track;
    int32_t  n_candidates;
    int32_t  flags;
    unsigned long long n_pixels;
    uint32_t n_deferred;
    uint32_t pad;
};

struct ScoreArgs {
    const float2* map;        // p[j * n_f + k]
    const float* isig;        // 1 / sigma per pixel (0 where masked): the weights of norm 2 (G25)
    BankParams bp;
    double f_min, df;
    uint64_t track_offset;    // id of template 0 of this launch
    uint64_t n_tracks;        // templates in this launch
    int32_t n_tau;
    int32_t norm;
    const float2* W;          // [n_f][n_tau]      (table kernel)
    const float2* E0;         // [n_f] e^{2 pi i f_k tau_0}  (recurrence kernels)
    const float4* bintab;     // [n_f] per-bin recurrence constants (rotation kernel)
    const float2* Es;         // [n_super][n_f] e^{2 pi i f_k tau_{s R}}: anchors of the Reinsch kernel
    const float2* kz;         // [n_f] (-4 sin^2(theta_k/2), sin theta_k)
    const float2* Ec;         // [n_f] e^{2 pi i f_k tau_{32}}: first anchor of the Chebyshev kernel
    const float4* cheb;       // [n_f] (G = 2 cos(S theta), cos theta, sin theta, cos 64 theta), built on the host
    const float* cheb_zi;     // [n_f] sin 64 theta
    Scalars* sc;
    Cand* cand;
    uint32_t cand_cap;
    WarpBest* warp_best;      // [warp_slots] one record per resident warp of a launch
    uint32_t warp_slots;
    unsigned long long* hist; // [n_bins] global counts
    int32_t n_bins;
    float hist_lo, hist_scale;
    float* dump;              // [n_tracks][n_tau] or null
    int32_t pool_stride;      // pixels of pool space per warp (>= n_max, multiple of 32)
    int32_t capture_mode;     // top-K second pass: keep every sample with SNR >= capture_thr, nothing else
    float capture_thr;
    const Track* tracks;      // explicit templates [n_tracks] (st_score_tracks) or null: template q = make_track(seed, id)
    float* tmax_snr;          // per-template maximum over the delays [n_tracks] (st_search_track_max) or null
    int32_t* tmax_m;          // its delay index [n_tracks]
    int32_t* k_dump;          // parity export of k_score_random's own rasteriser: [n_tracks][n_t] (pre-filled with -1)
    int32_t* j0_dump;         //   with [n_tracks] first columns
    int32_t* N_dump;          //   and [n_tracks] durations
    uint32_t* deferred;       // Chebyshev kernel: list of launch-relative template indices handed from the fast build
                              // (which appends) to the two-class build (which, with defer_in set, works through it)
    uint32_t deferred_cap;
    int32_t defer_in;         // 1: this launch scores the templates of `deferred` (count in sc->n_deferred)
    float defer_limit;        // fast build: largest scale * sum |v| over class B pixels it may score itself
    // bank cache (Chebyshev fast build): S1 + S2 of a template bank kept in HBM so that further maps searched with
    // the same bank skip Philox and the rasteriser (PAPER.md:173 time shifts, :232-234 follow-ups)
    uint16_t* kcache;         // [templates][kcache_stride] bins, lane-major: entry lane * ceil4(L) + i
    int2* kmeta;              // [templates] (N, j0)
    uint32_t kcache_stride;   // uint16 entries per template = 32 * ceil4(ceil(n_max / 32))
    uint64_t kcache_base;     // cache row of template 0 of this launch
    int32_t kcache_mode;      // 0 unused, 1 this launch fills the cache, 2 it reads it
    uint32_t fold_offset;     // Chebyshev kernel, shared-memory fold: byte offset of the per-warp fold scratch
};

// Template q of the launch: regenerated from (seed, id), or read from the caller's explicit list.
__device__ __forceinline__ Track load_track(const ScoreArgs& a, uint64_t q, uint64_t id)
{
    return a.tracks ? a.tracks[q] : make_track(a.bp, id);
}

// Per-template maximum over the delays (the delay that "minimises the timing error" of a
// template), G12 order inside a template: larger float32 SNR, then smaller delay index.
struct TrackMax { float v; int32_t m; };
__device__ __forceinline__ void tmax_init(TrackMax& t) { t.v = -INFINITY; t.m = 0x7FFFFFFF; }
template <int NV>
__device__ __forceinline__ void tmax_update(TrackMax& t, const float (&v)[NV], const uint32_t (&m)[NV], const bool (&ok)[NV])
{
#pragma unroll
    for (int i = 0; i < NV; ++i)
        if (ok[i] && (v[i] > t.v || (v[i] == t.v && (int32_t)m[i] < t.m))) { t.v = v[i]; t.m = (int32_t)m[i]; }
}
__device__ __forceinline__ void tmax_finish(const ScoreArgs& a, TrackMax t, uint64_t q)
{
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        const float ov = __shfl_xor_sync(kFull, t.v, off);
        const int32_t om = __shfl_xor_sync(kFull, t.m, off);
        if (ov > t.v || (ov == t.v && om < t.m)) { t.v = ov; t.m = om; }
    }
    if ((threadIdx.x & 31) == 0) { a.tmax_snr[q] = t.v; a.tmax_m[q] = t.m; }
}

// ------------------------------------------------------------------ helpers --
__device__ __forceinline__ uint32_t enc_f32(float f)
{
    const uint32_t b = __float_as_uint(f);
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float dec_f32(uint32_t e)
{
    return __uint_as_float((e & 0x80000000u) ? (e & 0x7FFFFFFFu) : ~e);
}
// Near-max margin: float32 SNRs within this distance of the running maximum are
// kept and re-scored in float64 (G12).  Far above the float32 error of a score.
__host__ __device__ __forceinline__ float near_margin(float mx)
{
    const float a = fabsf(mx);
    return 5e-5f * (a > 1.0f ? a : 1.0f);
}
__device__ __forceinline__ bool better(float s, uint64_t id, uint32_t m,
                                       float bs, uint64_t bid, uint32_t bm)
{
    if (s != bs) return s > bs;
    if (id != bid) return id < bid;
    return m < bm;
}
__host__ __device__ __forceinline__ float norm_scale(int32_t N, int32_t norm)
{
    // N^-alpha: alpha = 1/2 (G1 default) or 1 (Eq. 8 as printed)
#if defined(__CUDA_ARCH__)
    // float32 throughout (the score it multiplies is float32): rsqrt seed + one Newton step, <= 1 ulp
    const float n = (float)N;                  // exact: N <= 2^20
    if (norm != 0) return __frcp_rn(n);
    const float y = rsqrtf(n);
    return y * fmaf(-0.5f * n * y, y, 1.5f);
#else
    return norm == 0 ? (float)(1.0 / sqrt((double)N)) : (float)(1.0 / (double)N);
#endif
}

// The per-template scale of Eq. 8: N^-alpha, or for the inverse-variance weighting (norm 2; fn. 23,
// PAPER.md:342, reading G25) 1 / sqrt(sum_Gamma 1/sigma^2) from the partial sums w2 of `width` adjacent lanes.
__device__ __forceinline__ float inv_sqrt_pos(float w)
{
    if (!(w > 0.0f)) return 0.0f;              // every pixel masked: the template scores 0
    const float y = rsqrtf(w);
    return y * fmaf(-0.5f * w * y, y, 1.5f);
}
template <int WIDTH = 32>
__device__ __forceinline__ float track_scale(const int32_t norm, const int32_t N, float w2)
{
    if (norm != 2) return norm_scale(N, norm);
#pragma unroll
    for (int off = WIDTH / 2; off >= 1; off >>= 1) w2 += __shfl_xor_sync(kFull, w2, off);
    return inv_sqrt_pos(w2);
}

// Per-warp reduction state (S4).
struct WarpReduce {
    float cached_max;      // last seen global float32 maximum
    WarpBest best;
    unsigned long long pixels;
};

__device__ __forceinline__ void reduce_init(WarpReduce& wr)
{
    wr.cached_max = -INFINITY;
    wr.best.snr = -INFINITY; wr.best.m = 0; wr.best.id = 0; wr.best.valid = 0; wr.best.pad = 0;
    wr.pixels = 0;
}

// Called by all 32 lanes with NV values per lane (sample (id, m[i]) = v[i], ignored
// where !valid[i]).  Histogram + running max + near-max candidate capture.
// MODE 0: search pass (compiled without the capture branch: the hot kernels' register budget is tight);
// MODE 1: capture pass of st_search_topk; MODE 2: decided at run time by a.capture_mode (fallback kernels).
template <int NV, int MODE = 2>
__device__ __forceinline__ void reduce_samples(const ScoreArgs& a, WarpReduce& wr, uint32_t* sm_hist,
                                               uint64_t id, uint64_t q, const float (&v)[NV],
                                               const uint32_t (&m)[NV], const bool (&valid)[NV])
{
    if (MODE == 1 || (MODE == 2 && a.capture_mode)) {       // warp-uniform
#pragma unroll
        for (int i = 0; i < NV; ++i) {
            if (valid[i] && v[i] >= a.capture_thr) {
                const uint32_t slot = atomicAdd(&a.sc->cand_count, 1u);
                if (slot < a.cand_cap) { Cand c; c.snr = v[i]; c.m = m[i]; c.id = id; a.cand[slot] = c; }
                else a.sc->overflow = 1u;
            }
        }
        return;
    }
    float lmax = -INFINITY;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
        if (valid[i]) {
            lmax = fmaxf(lmax, v[i]);
            if (a.n_bins > 0) {
                int b = __float2int_rd((v[i] - a.hist_lo) * a.hist_scale);
                b = b < 0 ? 0 : (b >= a.n_bins ? a.n_bins - 1 : b);
                ST_ASSERT(b >= 0 && b < a.n_bins && (int)m[i] < a.n_tau);
                atomicAdd(&sm_hist[b], 1u);
            }
            if (a.dump) a.dump[q * (uint64_t)a.n_tau + m[i]] = v[i];
        }
    }
    // warp maximum through the order-preserving integer encoding: one REDUX instead of five shuffle + max steps
    const float wmax = dec_f32(__reduce_max_sync(kFull, enc_f32(lmax)));
    if (wmax >= wr.cached_max - near_margin(wr.cached_max)) {
        // slow path: this template comes within the margin of the global maximum
        const int lane = threadIdx.x & 31;
        uint32_t old = 0;
        if (lane == 0) old = atomicMax(&a.sc->gmax_bits, enc_f32(wmax));
        old = __shfl_sync(kFull, old, 0);
        const float gm = fmaxf(dec_f32(old), wmax);
        wr.cached_max = gm;
        const float thr = gm - near_margin(gm);
        const bool full = *(volatile uint32_t*)&a.sc->overflow != 0;
        float bs = -INFINITY; uint32_t bm = 0;
#pragma unroll
        for (int i = 0; i < NV; ++i) {
            if (valid[i] && v[i] >= thr) {
                if (!full) {
                    const uint32_t slot = atomicAdd(&a.sc->cand_count, 1u);
                    if (slot < a.cand_cap) { Cand c; c.snr = v[i]; c.m = m[i]; c.id = id; a.cand[slot] = c; }
                    else a.sc->overflow = 1u;
                }
                ST_ASSERT(id >= a.track_offset && id < a.track_offset + a.n_tracks);
                if (v[i] > bs || (v[i] == bs && m[i] < bm)) { bs = v[i]; bm = m[i]; }
            }
        }
        // warp-wide best of this template under (snr desc, m asc), then against the warp's record
#pragma unroll
        for (int off = 16; off >= 1; off >>= 1) {
            const float os = __shfl_xor_sync(kFull, bs, off);
            const uint32_t om = __shfl_xor_sync(kFull, bm, off);
            if (os > bs || (os == bs && om < bm)) { bs = os; bm = om; }
        }
        if (bs > -INFINITY && (!wr.best.valid || better(bs, id, bm, wr.best.snr, wr.best.id, wr.best.m))) {
            wr.best.snr = bs; wr.best.m = bm; wr.best.id = id; wr.best.valid = 1;
        }
    }
}

__device__ __forceinline__ void reduce_finish(const ScoreArgs& a, WarpReduce& wr)
{
    const int lane = threadIdx.x & 31;
    if (lane == 0) {
        if (wr.pixels) atomicAdd(&a.sc->n_pixels, wr.pixels);
        if (wr.best.valid) {
            const uint32_t gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
            ST_ASSERT(gw < a.warp_slots);       // the host clamps every grid to warp_slots resident warps
            WarpBest cur = a.warp_best[gw];     // slot owned by this warp across launches
            if (!cur.valid || better(wr.best.snr, wr.best.id, wr.best.m, cur.snr, cur.id, cur.m))
                a.warp_best[gw] = wr.best;
        }
    }
}

__device__ __forceinline__ void hist_init(uint32_t* sm_hist, int n_bins)
{
    for (int b = threadIdx.x; b < n_bins; b += blockDim.x) sm_hist[b] = 0;
    __syncthreads();
}
__device__ __forceinline__ void hist_flush(uint32_t* sm_hist, unsigned long long* hist, int n_bins)
{
    __syncthreads();
    for (int b = threadIdx.x; b < n_bins; b += blockDim.x) {
        const uint32_t c = sm_hist[b];
        if (c) atomicAdd(&hist[b], (unsigned long long)c);
    }
}

// The template counter's fetch-and-add.  An integer atomic (atomicAdd(), or atom.global.add.u64 in PTX) under
// `if (lane == 0)` gets the assembler's warp-aggregation pattern -- leader atomic, then a SHFL of the result to
// the active lanes -- and that shuffle waits for the L2 round trip on the spot (~500 clocks per template in the
// profile; issuing the atomic "one template ahead" hid nothing).  A float64 atomic is not aggregated: the counter
// is kept as a double (exact below 2^53; the all-zero bit pattern the host writes is 0.0), the raw result stays
// pending in a register and is converted at its first use, one template later (claim_value).
__device__ __forceinline__ unsigned long long claim_add(unsigned long long* counter, unsigned long long n)
{
    unsigned long long old;
    asm volatile("atom.global.add.f64 %0, [%1], %2;" : "=l"(old) : "l"(counter), "d"((double)n) : "memory");
    return old;                                         // bits of the previous count as a double
}
__device__ __forceinline__ uint64_t claim_value(unsigned long long bits)
{
    return (uint64_t)__double2ll_rn(__longlong_as_double((long long)bits));
}
// Next template of the launch for this warp (dynamic: durations vary 100x).
__device__ __forceinline__ uint64_t next_track(const ScoreArgs& a)
{
    unsigned long long q = 0;
    if ((threadIdx.x & 31) == 0) q = claim_add(&a.sc->counter, 1ull);
    return claim_value(__shfl_sync(kFull, q, 0));
}

__device__ __forceinline__ uint32_t hist_smem_words(int n_bins) { return (uint32_t)((n_bins + 3) & ~3); }

// ----------------------------------------------------------------------- S0 --
// p = CSD / sigma (Eq. 7); sigma <= 0 or non-finite masks the pixel (G11).
__device__ __forceinline__ float2 prepare_pixel(float2 c, float s)
{
    if (!(s > 0.0f) || isinf(s)) return make_float2(0.0f, 0.0f);
    return make_float2(__fdiv_rn(c.x, s), __fdiv_rn(c.y, s));
}
// 1 / sigma, 0 where the pixel is masked: the weight plane of the inverse-variance statistic (G25)
__device__ __forceinline__ float inv_sigma_pixel(float s)
{
    return (!(s > 0.0f) || isinf(s)) ? 0.0f : __fdiv_rn(1.0f, s);
}
// HBM bound: per pixel 8 B of CSD (+ 4 B of a per-pixel sigma) read, 8 B of p written, and -- ISIG -- 4 B of the
// 1 / sigma plane written.  Only ST_NORM_INVVAR reads that plane: st_set_map writes it (a later search may ask for
// that norm), the batch call knows its norm before S0 and leaves the plane out otherwise (1/6 to 1/5 of S0's
// traffic).  VEC: two pixels per thread per iteration through 16-byte loads and stores (the host checks alignment
// and parity), two iterations in flight.
template <bool VEC, bool ISIG = true>
__global__ void __launch_bounds__(256) k_prepare_map(const float2* __restrict__ csd, const float* __restrict__ sigma,
                                                     int sigma_kind, int n_f, size_t n_pix, float2* __restrict__ p,
                                                     float* __restrict__ isig)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x, t0 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (VEC) {
        const size_t n2 = n_pix >> 1;
        const float4* c4 = reinterpret_cast<const float4*>(csd);
        float4* p4 = reinterpret_cast<float4*>(p);
        for (size_t i = t0; i < n2; i += 2 * stride) {
            const size_t j = i + stride;
            const bool two = j < n2;
            const float4 a = __ldcs(&c4[i]);
            const float4 b = two ? __ldcs(&c4[j]) : make_float4(0.f, 0.f, 0.f, 0.f);
            float2 sa = make_float2(1.0f, 1.0f), sb = sa;
            if (sigma_kind == 2) {
                sa = __ldcs(reinterpret_cast<const float2*>(sigma) + i);
                if (two) sb = __ldcs(reinterpret_cast<const float2*>(sigma) + j);
            } else if (sigma_kind == 1) {
                const size_t ka = (2 * i) % (size_t)n_f, kb = (2 * j) % (size_t)n_f;
                sa = make_float2(__ldg(&sigma[ka]), __ldg(&sigma[ka + 1 < (size_t)n_f ? ka + 1 : 0]));
                if (two) sb = make_float2(__ldg(&sigma[kb]), __ldg(&sigma[kb + 1 < (size_t)n_f ? kb + 1 : 0]));
            }
            float2 r0 = make_float2(a.x, a.y), r1 = make_float2(a.z, a.w);
            float2 r2 = make_float2(b.x, b.y), r3 = make_float2(b.z, b.w);
            if (sigma_kind != 0) {
                r0 = prepare_pixel(r0, sa.x); r1 = prepare_pixel(r1, sa.y);
                r2 = prepare_pixel(r2, sb.x); r3 = prepare_pixel(r3, sb.y);
            }
            p4[i] = make_float4(r0.x, r0.y, r1.x, r1.y);
            if (two) p4[j] = make_float4(r2.x, r2.y, r3.x, r3.y);
            if (ISIG) {
                float2* i2 = reinterpret_cast<float2*>(isig);
                i2[i] = sigma_kind != 0 ? make_float2(inv_sigma_pixel(sa.x), inv_sigma_pixel(sa.y)) : make_float2(1.0f, 1.0f);
                if (two) i2[j] = sigma_kind != 0 ? make_float2(inv_sigma_pixel(sb.x), inv_sigma_pixel(sb.y)) : make_float2(1.0f, 1.0f);
            }
        }
    } else {
        for (size_t i = t0; i < n_pix; i += stride) {
            float2 c = csd[i];
            const float sg = sigma_kind == 0 ? 1.0f : (sigma_kind == 1 ? sigma[i % (size_t)n_f] : sigma[i]);
            if (sigma_kind != 0) c = prepare_pixel(c, sg);
            p[i] = c;
            if (ISIG) isig[i] = inv_sigma_pixel(sg);
        }
    }
}

// ------------------------------------------------------------------ twiddles --
// W[k][m] = e^{2 pi i (f_min + k df) tau_m}, formed in float64, stored as float32
// (cos, sin).  Sign as printed in Eq. 8 (G7); f is the bin frequency (G6).
__global__ void k_build_w_table(const double* __restrict__ tau, int n_tau, int n_f,
                                double f_min, double df, float2* __restrict__ W)
{
    const size_t n = (size_t)n_f * (size_t)n_tau;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (size_t)gridDim.x * blockDim.x) {
        const int k = (int)(i / (size_t)n_tau), m = (int)(i % (size_t)n_tau);
        const double cyc = (f_min + (double)k * df) * tau[m];
        double s, c;
        sincospi(2.0 * (cyc - rint(cyc)), &s, &c);
        W[i] = make_float2((float)c, (float)s);
    }
}

// Uniform grid tau_m = tau0 + m * dtau.  With theta_k = 2 pi f_k dtau:
//   E0[k]     = e^{2 pi i f_k tau0}
//   mode 0 (rotation): bintab[k] = (cos theta, sin theta, cos(CH theta), sin(CH theta))
//   mode 1 (Reinsch):  bintab[k] = (4 sin^2(theta/2), sin theta, cos(CH theta), sin(CH theta))
__global__ void k_build_bin_tables(double tau0, double dtau, int ch, int mode, int n_f,
                                   double f_min, double df, float2* __restrict__ E0,
                                   float4* __restrict__ bintab)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_f) return;
    const double f = f_min + (double)k * df;
    double s, c;
    const double c0 = f * tau0;
    sincospi(2.0 * (c0 - rint(c0)), &s, &c);
    E0[k] = make_float2((float)c, (float)s);
    double cyc = f * dtau;
    cyc -= rint(cyc);                       // theta / 2 pi in [-1/2, 1/2]
    double zs, zc, hs, hc, cs, cc;
    sincospi(2.0 * cyc, &zs, &zc);
    sincospi(cyc, &hs, &hc);                // sin(theta/2)
    double cch = cyc * (double)ch;
    cch -= rint(cch);
    sincospi(2.0 * cch, &cs, &cc);
    float4 t;
    t.x = mode == 0 ? (float)zc : (float)(4.0 * hs * hs);
    t.y = (float)zs;
    t.z = (float)cc;
    t.w = (float)cs;
    bintab[k] = t;
}

// Tables of k_score_reinsch on the uniform grid tau_m = tau0 + m dtau, theta_k = 2 pi f_k dtau:
//   Es[s][k] = e^{2 pi i f_k (tau0 + s R dtau)}   anchor phase factors, one row per super-chunk of R delays
//   kz[k]    = (-4 sin^2(theta_k / 2), sin theta_k)
__global__ void k_build_reinsch_tables(double tau0, double dtau, int r_super, int n_super, int n_f,
                                       double f_min, double df, float2* __restrict__ Es, float2* __restrict__ kz)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_f) return;
    const double f = f_min + (double)k * df;
    for (int s = 0; s < n_super; ++s) {
        const double cyc = f * (tau0 + (double)(s * r_super) * dtau);
        double sn, cs;
        sincospi(2.0 * (cyc - rint(cyc)), &sn, &cs);
        Es[(size_t)s * (size_t)n_f + (size_t)k] = make_float2((float)cs, (float)sn);
    }
    double cyc = f * dtau;
    cyc -= rint(cyc);
    double zs, zc, hs, hc;
    sincospi(2.0 * cyc, &zs, &zc);
    sincospi(cyc, &hs, &hc);
    kz[k] = make_float2((float)(-4.0 * hs * hs), (float)zs);
}

// --------------------------------------------------- S1-S4, table, any grid --
// Warp per template.  The warp rasterises the track (lanes over columns), parks
// (p, k) of every pixel in its shared-memory pool, then lanes own delays: for each
// block of 32 delays every lane walks the track in column order and accumulates
// Re[W(k_c, m) p_c] in float32.
__global__ void __launch_bounds__(256) k_score_table(const ScoreArgs a)
{
    extern __shared__ __align__(16) unsigned char smem[];
    uint32_t* sm_hist = reinterpret_cast<uint32_t*>(smem);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_warps = blockDim.x >> 5;
    float2* pool_p = reinterpret_cast<float2*>(sm_hist + hist_smem_words(a.n_bins)) + (size_t)warp * a.pool_stride;
    uint16_t* pool_k = reinterpret_cast<uint16_t*>(reinterpret_cast<float2*>(sm_hist + hist_smem_words(a.n_bins))
                                                   + (size_t)n_warps * a.pool_stride) + (size_t)warp * a.pool_stride;
    hist_init(sm_hist, a.n_bins);
    WarpReduce wr;
    reduce_init(wr);
    for (;;) {
        const uint64_t q = next_track(a);
        if (q >= a.n_tracks) break;
        const uint64_t id = a.track_offset + q;
        const Track t = load_track(a, q, id);
        const Raster r = make_raster(t, a.bp.n_f, a.bp.family);
        float w2 = 0.0f;
        for (int c = lane; c < t.N; c += kWarp) {
            const int k = raster_bin_fast(r, c);
            const size_t pix = (size_t)(t.j0 + c) * (size_t)a.bp.n_f + (size_t)k;
            float2 pv = __ldg(&a.map[pix]);
            if (a.norm == 2) { const float rs = __ldg(&a.isig[pix]); pv.x *= rs; pv.y *= rs; w2 = fmaf(rs, rs, w2); }
            pool_p[c] = pv;
            pool_k[c] = (uint16_t)k;
        }
        __syncwarp();
        wr.pixels += (unsigned long long)t.N;
        const float scale = track_scale(a.norm, t.N, w2);
        TrackMax tm;
        tmax_init(tm);
        for (int mb = 0; mb < a.n_tau; mb += kWarp) {
            const int m = mb + lane;
            const int mm = m < a.n_tau ? m : a.n_tau - 1;
            const float2* Wm = a.W + mm;
            float acc = 0.0f;
#pragma unroll 4
            for (int c = 0; c < t.N; ++c) {
                const float2 p = pool_p[c];
                const float2 w = __ldg(Wm + (size_t)pool_k[c] * (size_t)a.n_tau);
                acc = fmaf(w.x, p.x, acc);
                acc = fmaf(-w.y, p.y, acc);
            }
            const float v[1] = {acc * scale};
            const uint32_t ms[1] = {(uint32_t)m};
            const bool ok[1] = {m < a.n_tau};
            reduce_samples<1>(a, wr, sm_hist, id, q, v, ms, ok);
            tmax_update<1>(tm, v, ms, ok);
        }
        if (a.tmax_snr) tmax_finish(a, tm, q);
        __syncwarp();
    }
    reduce_finish(a, wr);
    hist_flush(sm_hist, a.hist, a.n_bins);
}

// ----------------------------------------- S1-S4, the paper's random-tau mode --
// One delay per template: one Eq. 8 term per pixel, so the kernel is a gather.  Measured:
// neither the rasteriser nor the phase factor bound it (removing either changes nothing) -- the chain
// counter -> Philox -> rasteriser -> L2 gather -> reduce of ONE template per warp does.  So a warp works
// on several templates at once, kRandGroup lanes each: their chains run in the same instructions (SIMT),
// the per-template fixed work costs a fraction of the issue slots, and a 255-column template fills its
// lanes where 32 lanes idled on its ragged last pass.  Measured on config 3 / the paper's Table III shape
// (fraction of the L2 gather rate): 32 lanes 0.71 / 0.91, 16 lanes 0.84 / 0.95, 8 lanes 0.82 / 0.94,
// 4 lanes 0.79 / 0.92.
// Per pixel: branch-free bin (fast path), the gather, the phase f_k tau reduced to [-1/2, 1/2] in float64
// on the FP64 pipe (1.5 * 2^52 rounding), MUFU sin / cos in float32 (abs error 5e-7); 5 XU operations.
#ifndef ST_RAND_GROUP
#define ST_RAND_GROUP 16
#endif
constexpr int kRandGroup = ST_RAND_GROUP;   // lanes per template
constexpr int kRandPerWarp = kWarp / kRandGroup;

// S4 for up to one sample per lane, each with its own template id (m = 0): histogram, running maximum,
// near-max candidates, per-warp best under the G12 order.
template <int MODE>
__device__ __forceinline__ void reduce_samples_multi(const ScoreArgs& a, WarpReduce& wr, uint32_t* sm_hist,
                                                     const uint64_t id, const uint64_t q, const float v, const bool valid)
{
    if (MODE == 1) {
        if (valid && v >= a.capture_thr) {
            const uint32_t slot = atomicAdd(&a.sc->cand_count, 1u);
            if (slot < a.cand_cap) { Cand c; c.snr = v; c.m = 0u; c.id = id; a.cand[slot] = c; }
            else a.sc->overflow = 1u;
        }
        return;
    }
    if (valid) {
        if (a.n_bins > 0) {
            int b = __float2int_rd((v - a.hist_lo) * a.hist_scale);
            b = b < 0 ? 0 : (b >= a.n_bins ? a.n_bins - 1 : b);
            ST_ASSERT(b >= 0 && b < a.n_bins);
            atomicAdd(&sm_hist[b], 1u);
        }
        if (a.dump) a.dump[q] = v;
        if (a.tmax_snr) { a.tmax_snr[q] = v; a.tmax_m[q] = 0; }     // one delay per template: it is its own maximum
    }
    const float wmax = dec_f32(__reduce_max_sync(kFull, enc_f32(valid ? v : -INFINITY)));     // one REDUX (see reduce_samples)
    if (wmax >= wr.cached_max - near_margin(wr.cached_max)) {
        const int lane = threadIdx.x & 31;
        uint32_t old = 0;
        if (lane == 0) old = atomicMax(&a.sc->gmax_bits, enc_f32(wmax));
        old = __shfl_sync(kFull, old, 0);
        const float gm = fmaxf(dec_f32(old), wmax);
        wr.cached_max = gm;
        const float thr = gm - near_margin(gm);
        const bool full = *(volatile uint32_t*)&a.sc->overflow != 0;
        float bs = -INFINITY; uint64_t bid = 0;
        if (valid && v >= thr) {
            if (!full) {
                const uint32_t slot = atomicAdd(&a.sc->cand_count, 1u);
                if (slot < a.cand_cap) { Cand c; c.snr = v; c.m = 0u; c.id = id; a.cand[slot] = c; }
                else a.sc->overflow = 1u;
            }
            bs = v; bid = id;
        }
#pragma unroll
        for (int off = 16; off >= 1; off >>= 1) {
            const float os = __shfl_xor_sync(kFull, bs, off);
            const uint64_t oid = __shfl_xor_sync(kFull, bid, off);
            if (os > bs || (os == bs && os > -INFINITY && oid < bid)) { bs = os; bid = oid; }
        }
        if (bs > -INFINITY && (!wr.best.valid || better(bs, bid, 0u, wr.best.snr, wr.best.id, wr.best.m))) {
            wr.best.snr = bs; wr.best.m = 0u; wr.best.id = bid; wr.best.valid = 1;
        }
    }
}

constexpr int kRandMinBlocks = 3;
// KDUMP: parity export -- the bins this kernel's own fast path (Horner form, regenerate-on-fallback) decides
// are written to a.k_dump next to the scores (st_debug_rasterise_random).
// GEN as in the Chebyshev kernel: false = quadratic bank templates with N^-alpha (options compiled in as constants).
template <bool CAPTURE, bool KDUMP, bool GEN>
__global__ void __launch_bounds__(256, kRandMinBlocks) k_score_random(const ScoreArgs a)
{
    extern __shared__ __align__(16) unsigned char smem[];
    uint32_t* sm_hist = reinterpret_cast<uint32_t*>(smem);
    const int lane = threadIdx.x & 31;
    const int sub = lane & (kRandGroup - 1), grp = lane / kRandGroup;
    const double u_sub = (double)sub + 0.5;
    hist_init(sm_hist, a.n_bins);
    WarpReduce wr;
    reduce_init(wr);
    // kRandPerWarp templates are claimed per atomic, one claim ahead (the result waits in lane 0)
    unsigned long long q_pref = 0;
    if (lane == 0) q_pref = claim_add(&a.sc->counter, (unsigned long long)kRandPerWarp);
    for (;;) {
        const uint64_t q0 = claim_value(__shfl_sync(kFull, q_pref, 0));
        if (q0 >= a.n_tracks) break;
        if (lane == 0) q_pref = claim_add(&a.sc->counter, (unsigned long long)kRandPerWarp);
        const uint64_t q = q0 + (uint64_t)grp;
        const bool live = q < a.n_tracks;                    // the last claim may be ragged
        const uint64_t id = a.track_offset + (live ? q : q0);
        const Track t = GEN ? load_track(a, live ? q : q0, id) : make_track(a.bp, id);
        const int family = GEN ? a.bp.family : 0;
        const int norm = GEN ? a.norm : (a.norm == 1 ? 1 : 0);
        const RasterFast r = make_raster_fast(t, a.bp.n_f, family);
        const int N = live ? t.N : 0;
        int n_max = N;
#pragma unroll
        for (int off = 16; off >= kRandGroup; off >>= 1) n_max = max(n_max, __shfl_xor_sync(kFull, n_max, off));
        const double u_last = int_to_double_fast(t.N - 1) + 0.5;
        const float2* col0 = a.map + (size_t)t.j0 * (size_t)a.bp.n_f;
        float acc = 0.0f, w2 = 0.0f;
        double ub = u_sub;                                    // column centre of this lane in the current pass
#pragma unroll 1
        for (int c0 = sub; c0 < n_max; c0 += 4 * kRandGroup, ub += 4.0 * kRandGroup) {
            int kq[4], cq[4];
            bool redo[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int c = c0 + u * kRandGroup;
                const bool in = c < N;
                cq[u] = in ? c : t.N - 1;                 // clamped: discarded below
                kq[u] = raster_bin_fast_u(r, in ? ub + (double)(u * kRandGroup) : u_last, redo[u]);
            }
            if (redo[0] | redo[1] | redo[2] | redo[3]) {  // ~1e-5 of the time (any family): normative sequence
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (redo[u]) kq[u] = raster_bin(make_raster(GEN ? load_track(a, live ? q : q0, id) : make_track(a.bp, id), a.bp.n_f, family), cq[u]);
            }
            if (KDUMP) {
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (c0 + u * kRandGroup < N) a.k_dump[q * (uint64_t)a.bp.n_t + (uint64_t)cq[u]] = kq[u];
                if (live && sub == 0) { a.j0_dump[q] = t.j0; a.N_dump[q] = t.N; }
            }
            float2 pv[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                ST_ASSERT(kq[u] >= 0 && kq[u] < a.bp.n_f && cq[u] >= 0 && t.j0 + cq[u] < a.bp.n_t);
                pv[u] = __ldg(col0 + (size_t)cq[u] * (size_t)a.bp.n_f + (size_t)kq[u]);
            }
            if (GEN && norm == 2) {                       // inverse-variance weights (G25): one more gather per pixel
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const float rs = __ldg(a.isig + ((size_t)(t.j0 + cq[u]) * (size_t)a.bp.n_f + (size_t)kq[u]));
                    pv[u].x *= rs; pv[u].y *= rs;
                    if (c0 + u * kRandGroup < N) w2 = fmaf(rs, rs, w2);
                }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const double cyc = (a.f_min + int_to_double_fast(kq[u]) * a.df) * t.tau;
                const double fr = cyc - ((cyc + kRoundMagic) - kRoundMagic);     // cyc - rint(cyc), |cyc| < 2^51
                const float ph = 6.283185307179586f * (float)fr;
                const float s = __sinf(ph), co = __cosf(ph);
                if (c0 + u * kRandGroup < N) {
                    acc = fmaf(co, pv[u].x, acc);
                    acc = fmaf(-s, pv[u].y, acc);
                }
            }
        }
#pragma unroll
        for (int off = kRandGroup / 2; off >= 1; off >>= 1) acc += __shfl_xor_sync(kFull, acc, off);
        if (sub == 0) wr.pixels += (unsigned long long)N;
        reduce_samples_multi<CAPTURE ? 1 : 0>(a, wr, sm_hist, id, q, acc * track_scale<kRandGroup>(norm, t.N, w2), live && sub == 0);
    }
    // wr.pixels was accumulated by the four group leaders: fold them into lane 0 for reduce_finish
    {
        unsigned long long px = wr.pixels;
#pragma unroll
        for (int off = 16; off >= kRandGroup; off >>= 1) px += __shfl_xor_sync(kFull, px, off);
        wr.pixels = px;
    }
    reduce_finish(a, wr);
    hist_flush(sm_hist, a.hist, a.n_bins);
}

// ------------------------------- S1-S4, uniform tau grid, recurrence along tau --
// Warp per template, lanes over PIXELS.  Phase A rasterises the track and parks
// v_c = p_c * e^{2 pi i f_k tau_0} (the term of Eq. 8 at the first delay) and k_c in
// the warp's pool.  Phase B walks the delays in chunks of CH: a lane takes its
// pixels two at a time, and advances each term along tau in registers,
//   MODE 0 (rotation):  v <- v * e^{i theta_k}                     (4 flop + 1 add / eval)
//   MODE 1 (Reinsch):   d <- d - 4 sin^2(theta_k/2) x ; x <- x + d (2 flop + 1 add / eval)
// where x = Re v; both are exact identities for x_m = Re[p e^{2 pi i f (tau_0 + m dtau)}].
// CH accumulators per lane hold the partial sums over that lane's pixels; a
// transposing shuffle tree folds them across the warp, leaving CH/32 finished
// delays per lane.  Anchors are re-derived every chunk from v_c * e^{i CH theta_k}
// (tabulated from float64), so recurrence error never spans more than CH steps.
template <int MODE, int CH, bool BT_SMEM>
__global__ void __launch_bounds__(512, 1) k_score_recur(const ScoreArgs a)
{
    static_assert(CH == 32 || CH == 64, "chunk of 32 or 64 delays");
    constexpr int NV = CH / 32;
    extern __shared__ __align__(16) unsigned char smem[];
    uint32_t* sm_hist = reinterpret_cast<uint32_t*>(smem);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_warps = blockDim.x >> 5;
    float4* sm_bt = reinterpret_cast<float4*>(sm_hist + hist_smem_words(a.n_bins));
    float2* pools = reinterpret_cast<float2*>(sm_bt + (BT_SMEM ? a.bp.n_f : 0));
    float2* pool_v = pools + (size_t)warp * a.pool_stride;
    uint16_t* pool_k = reinterpret_cast<uint16_t*>(pools + (size_t)n_warps * a.pool_stride) + (size_t)warp * a.pool_stride;
    if (BT_SMEM)
        for (int k = threadIdx.x; k < a.bp.n_f; k += blockDim.x) sm_bt[k] = a.bintab[k];
    hist_init(sm_hist, a.n_bins);   // includes __syncthreads
    const float4* bt = BT_SMEM ? sm_bt : a.bintab;
    const int n_chunks = (a.n_tau + CH - 1) / CH;
    WarpReduce wr;
    reduce_init(wr);
    for (;;) {
        const uint64_t q = next_track(a);
        if (q >= a.n_tracks) break;
        const uint64_t id = a.track_offset + q;
        const Track t = load_track(a, q, id);
        const Raster r = make_raster(t, a.bp.n_f, a.bp.family);
        TrackMax tm;
        tmax_init(tm);
        // ---- phase A: rasterise, gather, rotate to tau_0
        const int n_pad = (t.N + 63) & ~63;          // pairs of 32-pixel rows
        float w2 = 0.0f;
#pragma unroll 2
        for (int c = lane; c < n_pad; c += kWarp) {
            float2 v = make_float2(0.0f, 0.0f);
            int k = 0;
            if (c < t.N) {
                k = raster_bin_fast(r, c);
                const size_t pix = (size_t)(t.j0 + c) * (size_t)a.bp.n_f + (size_t)k;
                float2 p = __ldg(&a.map[pix]);
                if (a.norm == 2) { const float rs = __ldg(&a.isig[pix]); p.x *= rs; p.y *= rs; w2 = fmaf(rs, rs, w2); }
                const float2 e = __ldg(&a.E0[k]);
                v.x = p.x * e.x - p.y * e.y;
                v.y = p.x * e.y + p.y * e.x;
            }
            pool_v[c] = v;
            pool_k[c] = (uint16_t)k;
        }
        __syncwarp();
        wr.pixels += (unsigned long long)t.N;
        const float scale = track_scale(a.norm, t.N, w2);
        // ---- phase B: chunks of CH delays
        for (int j = 0; j < n_chunks; ++j) {
            float acc[CH];
#pragma unroll
            for (int i = 0; i < CH; ++i) acc[i] = 0.0f;
            for (int c = lane; c < n_pad; c += 2 * kWarp) {
                const float2 v1 = pool_v[c], v2 = pool_v[c + kWarp];
                const float4 b1 = bt[pool_k[c]], b2 = bt[pool_k[c + kWarp]];
                // anchors of the next chunk: v * e^{i CH theta}
                pool_v[c] = make_float2(v1.x * b1.z - v1.y * b1.w, v1.x * b1.w + v1.y * b1.z);
                pool_v[c + kWarp] = make_float2(v2.x * b2.z - v2.y * b2.w, v2.x * b2.w + v2.y * b2.z);
                if (MODE == 0) {
                    float xr1 = v1.x, xi1 = v1.y, xr2 = v2.x, xi2 = v2.y;
#pragma unroll
                    for (int i = 0; i < CH; ++i) {
                        acc[i] += xr1;
                        acc[i] += xr2;
                        const float nr1 = fmaf(xr1, b1.x, -(xi1 * b1.y));
                        const float ni1 = fmaf(xr1, b1.y, xi1 * b1.x);
                        const float nr2 = fmaf(xr2, b2.x, -(xi2 * b2.y));
                        const float ni2 = fmaf(xr2, b2.y, xi2 * b2.x);
                        xr1 = nr1; xi1 = ni1; xr2 = nr2; xi2 = ni2;
                    }
                } else {
                    // x_m - x_{m-1} = 2 sin^2(theta/2) Re v - sin(theta) Im v
                    float x1 = v1.x, d1 = fmaf(0.5f * b1.x, v1.x, -(b1.y * v1.y));
                    float x2 = v2.x, d2 = fmaf(0.5f * b2.x, v2.x, -(b2.y * v2.y));
#pragma unroll
                    for (int i = 0; i < CH; ++i) {
                        acc[i] += x1;
                        acc[i] += x2;
                        d1 = fmaf(-b1.x, x1, d1);
                        d2 = fmaf(-b2.x, x2, d2);
                        x1 += d1;
                        x2 += d2;
                    }
                }
            }
            // ---- fold the CH partial sums across the 32 lanes (transposing tree):
            // after the stage with offset `off` a lane keeps the half of the delays
            // selected by that lane bit; lane l ends with delays NV*l .. NV*l + NV-1.
#pragma unroll
            for (int off = 16, n = CH / 2; off >= 1; off >>= 1, n >>= 1) {
                const bool upper = (lane & off) != 0;
#pragma unroll
                for (int i = 0; i < n; ++i) {
                    const float send = upper ? acc[i] : acc[i + n];
                    const float keep = upper ? acc[i + n] : acc[i];
                    acc[i] = keep + __shfl_xor_sync(kFull, send, off);
                }
            }
            float v[NV]; uint32_t ms[NV]; bool ok[NV];
#pragma unroll
            for (int i = 0; i < NV; ++i) {
                ms[i] = (uint32_t)(j * CH + NV * lane + i);
                ok[i] = (int)ms[i] < a.n_tau;
                v[i] = acc[i] * scale;
            }
            reduce_samples<NV>(a, wr, sm_hist, id, q, v, ms, ok);
            tmax_update<NV>(tm, v, ms, ok);
            __syncwarp();
        }
        if (a.tmax_snr) tmax_finish(a, tm, q);
    }
    reduce_finish(a, wr);
    hist_flush(sm_hist, a.hist, a.n_bins);
}


// --------------------- S1-S4, uniform tau grid, packed three-term recurrence --
// The production kernel of the grid mode.  Warp per template, lanes over pixels.
// For x_m = Re[p e^{2 pi i f (tau_0 + m dtau)}] the exact identities
//     d_{m+1} = d_m - kappa x_m ,   x_{m+1} = x_m + d_{m+1} ,   kappa = 4 sin^2(theta/2)
// (Reinsch's form of the Chebyshev three-term recurrence, stable as theta -> 0)
// advance a pixel's term of Eq. 8 along the delay grid with one FMA and one add;
// a third add accumulates it.  Two pixels of a lane are packed into one f32x2
// register pair (sm_100 fma.rn.f32x2 / add.rn.f32x2), two such pairs are in flight.
//   anchor phase (every R = 256 delays): rasterise (first time), gather p from the
//     L2-resident map, x = Re[p Es], d = x_m - x_{m-1}, parked with the bin in the
//     warp's shared-memory pool (10 B per pixel);
//   chunk of 32 delays: 32 packed accumulators per lane; states are read from the
//     pool, advanced 32 steps in registers and written back; a transposing shuffle
//     tree folds the accumulators across the warp: lane l ends with delay m0 + l.
// Float32 error of a term after R steps stays below 1e-5 |p| (tests).
typedef unsigned long long f32x2_t;
__device__ __forceinline__ f32x2_t pk_fma(f32x2_t a, f32x2_t b, f32x2_t c)
{
    f32x2_t r;
    asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ f32x2_t pk_add(f32x2_t a, f32x2_t b)
{
    f32x2_t r;
    asm volatile("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2_t pk_sub(f32x2_t a, f32x2_t b)      // FADD2 with the second operand negated
{
    f32x2_t r;
    asm volatile("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
// d = fma(nk, x, d) on the two halves with scalar FFMAs: fma.rn.f32x2 with three distinct
// register-pair operands issues at 2/3 rate (register-file bandwidth; st_microbench
// ffma2_3distinct), two scalar FFMAs cost the same pipe time as one full-rate packed op.
__device__ __forceinline__ f32x2_t pk_fma_halves(f32x2_t a, f32x2_t b, f32x2_t c)
{
    f32x2_t r;
    asm volatile("{\n\t.reg .f32 al, ah, bl, bh, cl, ch;\n\t"
                 "mov.b64 {al, ah}, %1;\n\tmov.b64 {bl, bh}, %2;\n\tmov.b64 {cl, ch}, %3;\n\t"
                 "fma.rn.f32 cl, al, bl, cl;\n\tfma.rn.f32 ch, ah, bh, ch;\n\t"
                 "mov.b64 %0, {cl, ch};\n\t}" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ f32x2_t pk_make(float lo, float hi)
{
    f32x2_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ float pk_lo(f32x2_t a)
{
    float lo;
    asm("{\n\t.reg .b32 t;\n\tmov.b64 {%0, t}, %1;\n\t}" : "=f"(lo) : "l"(a));
    return lo;
}
__device__ __forceinline__ float pk_hi(f32x2_t a)
{
    float hi;
    asm("{\n\t.reg .b32 t;\n\tmov.b64 {t, %0}, %1;\n\t}" : "=f"(hi) : "l"(a));
    return hi;
}
__device__ __forceinline__ float pk_sum(f32x2_t a)
{
    float lo, hi;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a));
    return lo + hi;
}

// Shared-memory accesses of the Chebyshev kernel's row loops through explicit 32-bit shared addresses: with
// generic pointers the compiler re-derived every base address from the kernel parameters inside the loop
// (~25 integer / uniform instructions per row pair, the IMADs among them on the FMA pipe).
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
template <int OFF>
__device__ __forceinline__ float2 lds_f2(uint32_t addr)
{
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2+%3];" : "=f"(v.x), "=f"(v.y) : "r"(addr), "n"(OFF));
    return v;
}
template <int OFF>
__device__ __forceinline__ void sts_f2(uint32_t addr, float x, float y)
{
    asm volatile("st.shared.v2.f32 [%0+%1], {%2, %3};" :: "r"(addr), "n"(OFF), "f"(x), "f"(y) : "memory");
}
template <int OFF>
__device__ __forceinline__ uint32_t lds_u16(uint32_t addr)
{
    uint32_t k;
    asm volatile("{\n\t.reg .u16 t;\n\tld.shared.u16 t, [%1+%2];\n\tcvt.u32.u16 %0, t;\n\t}" : "=r"(k) : "r"(addr), "n"(OFF));
    return k;
}
__device__ __forceinline__ float4 lds_f4(uint32_t addr)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ float lds_f1(uint32_t addr)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}

constexpr int kChunk = 32;        // delays per accumulator chunk
constexpr int kSuper = 256;       // delays between re-anchoring (8 chunks)

__global__ void __launch_bounds__(512, 1) k_score_reinsch(const ScoreArgs a)
{
    extern __shared__ __align__(16) unsigned char smem[];
    uint32_t* sm_hist = reinterpret_cast<uint32_t*>(smem);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_warps = blockDim.x >> 5;
    // shared memory: hist | kz[n_f] | x2[n_warps][P] | d2[n_warps][P] | kk[n_warps][P],  P = pool_stride / 2
    float2* sm_kz = reinterpret_cast<float2*>(sm_hist + hist_smem_words(a.n_bins));
    const int P = a.pool_stride >> 1;               // packed entries (pixel pairs) per warp
    f32x2_t* pool_x = reinterpret_cast<f32x2_t*>(sm_kz + a.bp.n_f + (a.bp.n_f & 1)) + (size_t)warp * P;
    f32x2_t* pool_d = pool_x + (size_t)n_warps * P;
    uint32_t* pool_k = reinterpret_cast<uint32_t*>(reinterpret_cast<f32x2_t*>(sm_kz + a.bp.n_f + (a.bp.n_f & 1))
                                                   + 2 * (size_t)n_warps * P) + (size_t)warp * P;
    for (int k = threadIdx.x; k < a.bp.n_f; k += blockDim.x) sm_kz[k] = a.kz[k];
    hist_init(sm_hist, a.n_bins);
    const float* sm_negk = reinterpret_cast<const float*>(sm_kz);     // sm_negk[2k] = -kappa_k
    const int n_chunks = (a.n_tau + kChunk - 1) / kChunk;
    WarpReduce wr;
    reduce_init(wr);
    for (;;) {
        const uint64_t q = next_track(a);
        if (q >= a.n_tracks) break;
        const uint64_t id = a.track_offset + q;
        const Track t = load_track(a, q, id);
        const Raster r = make_raster(t, a.bp.n_f, a.bp.family);
        TrackMax tm;
        tmax_init(tm);
        const int n_prows = (t.N + 63) >> 6;         // packed rows: columns [64 pr, 64 pr + 64)
        wr.pixels += (unsigned long long)t.N;
        float scale = 0.0f, w2 = 0.0f;
#pragma unroll 1
        for (int j = 0; j < n_chunks; ++j) {
            if ((j & (kSuper / kChunk - 1)) == 0) {
                // ---- anchor phase of super-chunk s: state (x, d) of every pixel at delay s * R
                const int s = j / (kSuper / kChunk);
                const float2* Es = a.Es + (size_t)s * (size_t)a.bp.n_f;
                if (s == 0) {
                    // rasterise: four columns per lane in flight (FP64 div / sqrt chains are long)
#pragma unroll 1
                    for (int pr = 0; pr < n_prows; pr += 2) {
                        const int c0 = pr * 64 + lane;
                        int k[4];
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            const int c = c0 + u * kWarp;
                            k[u] = raster_bin_fast(r, c < t.N ? c : t.N - 1);
                        }
                        pool_k[pr * kWarp + lane] = (uint32_t)k[0] | ((uint32_t)k[1] << 16);
                        if (pr + 1 < n_prows) pool_k[(pr + 1) * kWarp + lane] = (uint32_t)k[2] | ((uint32_t)k[3] << 16);
                    }
                }
                // gather p and the anchor phase factor: 16 independent L2 loads in flight per lane
#pragma unroll 1
                for (int pr = 0; pr < n_prows; pr += 4) {
                    float2 pv[8], wv[8];
                    int kq[8];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int prow = pr + u < n_prows ? pr + u : n_prows - 1;
                        const uint32_t kk = pool_k[prow * kWarp + lane];
                        kq[2 * u] = (int)(kk & 0xFFFFu);
                        kq[2 * u + 1] = (int)(kk >> 16);
                    }
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        const int prow = pr + (u >> 1) < n_prows ? pr + (u >> 1) : n_prows - 1;
                        int c = prow * 64 + (u & 1) * kWarp + lane;
                        c = c < t.N ? c : t.N - 1;       // clamped: the value is discarded below
                        const size_t pix = (size_t)(t.j0 + c) * (size_t)a.bp.n_f + (size_t)kq[u];
                        pv[u] = __ldg(&a.map[pix]);
                        wv[u] = __ldg(&Es[kq[u]]);
                        if (a.norm == 2) {
                            const float rs = __ldg(&a.isig[pix]);
                            pv[u].x *= rs; pv[u].y *= rs;
                            const int cu = prow * 64 + (u & 1) * kWarp + lane;          // unclamped column of this slot
                            if (s == 0 && pr + (u >> 1) < n_prows && cu < t.N) w2 = fmaf(rs, rs, w2);
                        }
                    }
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        if (pr + u < n_prows) {
                            float x[2], d[2];
#pragma unroll
                            for (int h = 0; h < 2; ++h) {
                                const int c = (pr + u) * 64 + h * kWarp + lane;
                                const float2 p = pv[2 * u + h], w = wv[2 * u + h];
                                const float2 z = sm_kz[kq[2 * u + h]];
                                const float vr = p.x * w.x - p.y * w.y, vi = p.x * w.y + p.y * w.x;
                                // x_m = Re v ; x_m - x_{m-1} = 2 sin^2(theta/2) Re v - sin(theta) Im v
                                x[h] = c < t.N ? vr : 0.0f;
                                d[h] = c < t.N ? fmaf(-0.5f * z.x, vr, -(z.y * vi)) : 0.0f;
                            }
                            pool_x[(pr + u) * kWarp + lane] = pk_make(x[0], x[1]);
                            pool_d[(pr + u) * kWarp + lane] = pk_make(d[0], d[1]);
                        }
                    }
                }
                if (s == 0) scale = track_scale(a.norm, t.N, w2);
            }
            // ---- one chunk of 32 delays: four pixels of the lane in flight (two register pairs).
            // Per delay and pair: two scalar FFMAs (d += -kappa x on the halves; a packed FFMA with
            // three distinct register pairs issues at 2/3 rate), one packed add (x += d) and the
            // accumulation: one packed add of the two pairs, then two scalar adds.
            float f[kChunk];
#pragma unroll
            for (int i = 0; i < kChunk; ++i) f[i] = 0.0f;
            int pr = 0;
#pragma unroll 1
            for (; pr + 2 <= n_prows; pr += 2) {
                const int e0 = pr * kWarp + lane, e1 = e0 + kWarp;
                f32x2_t x0 = pool_x[e0], d0 = pool_d[e0], x1 = pool_x[e1], d1 = pool_d[e1];
                const uint32_t kk0 = pool_k[e0], kk1 = pool_k[e1];
                const f32x2_t nk0 = pk_make(sm_negk[2 * (kk0 & 0xFFFFu)], sm_negk[2 * (kk0 >> 16)]);
                const f32x2_t nk1 = pk_make(sm_negk[2 * (kk1 & 0xFFFFu)], sm_negk[2 * (kk1 >> 16)]);
#pragma unroll
                for (int i = 0; i < kChunk; ++i) {
                    const f32x2_t sx = pk_add(x0, x1);
                    f[i] += pk_lo(sx); f[i] += pk_hi(sx);
                    d0 = pk_fma_halves(nk0, x0, d0);
                    d1 = pk_fma_halves(nk1, x1, d1);
                    x0 = pk_add(x0, d0);
                    x1 = pk_add(x1, d1);
                }
                pool_x[e0] = x0; pool_d[e0] = d0; pool_x[e1] = x1; pool_d[e1] = d1;
            }
            if (pr < n_prows) {          // odd tail: one pair
                const int e0 = pr * kWarp + lane;
                f32x2_t x0 = pool_x[e0], d0 = pool_d[e0];
                const uint32_t kk0 = pool_k[e0];
                const f32x2_t nk0 = pk_make(sm_negk[2 * (kk0 & 0xFFFFu)], sm_negk[2 * (kk0 >> 16)]);
#pragma unroll
                for (int i = 0; i < kChunk; ++i) {
                    f[i] += pk_lo(x0); f[i] += pk_hi(x0);
                    d0 = pk_fma_halves(nk0, x0, d0);
                    x0 = pk_add(x0, d0);
                }
                pool_x[e0] = x0; pool_d[e0] = d0;
            }
            // ---- fold: the transposing tree across the 32 lanes
#pragma unroll
            for (int off = 16, n = kChunk / 2; off >= 1; off >>= 1, n >>= 1) {
                const bool upper = (lane & off) != 0;
#pragma unroll
                for (int i = 0; i < n; ++i) {
                    const float send = upper ? f[i] : f[i + n];
                    const float keep = upper ? f[i + n] : f[i];
                    f[i] = keep + __shfl_xor_sync(kFull, send, off);
                }
            }
            const float v[1] = {f[0] * scale};
            const uint32_t ms[1] = {(uint32_t)(j * kChunk + lane)};
            const bool ok[1] = {(int)ms[0] < a.n_tau};
            reduce_samples<1>(a, wr, sm_hist, id, q, v, ms, ok);
            tmax_update<1>(tm, v, ms, ok);
        }
        if (a.tmax_snr) tmax_finish(a, tm, q);
    }
    reduce_finish(a, wr);
    hist_flush(sm_hist, a.hist, a.n_bins);
}


// ------------------ S1-S4, uniform tau grid, two-sided Chebyshev recurrence --
// The production kernel of the grid mode.  Warp per template, lanes over pixels.
// A pixel's term of Eq. 8 along the uniform delay grid, x_m = Re[p e^{2 pi i f (tau_0 + m dtau)}]
// = |p| cos(psi + m theta), obeys for any stride S the three-term recurrence
//     x_{m+S} = 2 cos(S theta) x_m - x_{m-S}        (and the same backwards),
// i.e. ONE FMA per (pixel, delay); half a packed add accumulates it.  Delays are processed
// in chunks of 64 around an anchor at the chunk centre m_c = 64 j + 32: the complex anchor
// v = p e^{2 pi i f tau_{m_c}} gives x_{m_c}, x_{m_c +- 1} (and x_{m_c - 2} for S = 2), from
// which 32 forward and 32 backward delays run as 2 S independent chains per pixel; two
// pixels per lane are in flight.  Forward and backward values of the same offset share a
// register pair, so the accumulation is one add.rn.f32x2 into 32 packed accumulators.  The
// anchor of the next chunk is v e^{i 64 theta} (table built in float64), so recurrence
// error never spans more than 32 delays.  The float32 coefficient G = fl(2 cos(S theta))
// stands for a slightly different angle: the host measures that drift per bin (it builds
// the table) and picks S = 1 or 2 so that 32 delays of drift stay below 3e-5 rad, else the
// search falls back to k_score_reinsch / k_score_recur (stochtrack_api.cu).
// A transposing shuffle tree folds the packed accumulators across the warp: lane l ends
// with delays m_c + l and m_c - 1 - l.
// One recurrence step on a register pair: (g, g) * cur + prev as ONE packed fma.rn.f32x2.  ptxas
// turns the (g, g) pair into FFMA2's scalar-broadcast operand (R.F32, with a free negation), so the
// instruction reads one 32-bit and two 64-bit registers and issues at full rate: measured 60.8
// evaluations/clk/SM for this loop against 37.5 with two scalar FFMAs (profiles/microbench).
// The recurrence x_{n+1} = G x_n - x_{n-1} has a subtraction FFMA2 cannot express on a pair, so
// the chains carry w_n = s_n x_n with the sign pattern s = + + - - + + - - ...:
//     w_{n+1} = (+G) w_n + w_{n-1}  (n even),     w_{n+1} = (-G) w_n + w_{n-1}  (n odd),
// started from w_0 = x_0, w_{-1} = -x_{-1}; the accumulators collect sum_pixels w_n and the sign
// s_n (a function of the accumulator index only) is applied once after the fold.  Every product
// and sum has the magnitude the plain recurrence has: the rounding is identical.
__device__ __forceinline__ f32x2_t pk_step(float g, f32x2_t cur, f32x2_t prev)
{
    f32x2_t r;
    asm volatile("{\n\t.reg .b64 gg;\n\tmov.b64 gg, {%1, %1};\n\t"
                 "fma.rn.f32x2 %0, gg, %2, %3;\n\t}" : "=l"(r) : "f"(g), "l"(cur), "l"(prev));
    return r;
}

constexpr int kCheb = 64;         // delays per chunk
constexpr int kHalf = kCheb / 2;

// The register pairs of one pixel at the anchor of a chunk.
//   stride 1: one chain pair   cur = (x_mc, x_mc-1)            prev = -(x_mc-1, x_mc)
//   stride 2: even offsets     cur = (x_mc, x_mc-1)            prev = -(x_mc-2, x_mc+1)
//             odd offsets      cur = (x_mc+1, x_mc-2)          prev = -(x_mc-1, x_mc)
// (prev negated: the chains run in the sign pattern of pk_step)
template <int STRIDE>
struct ChebPixel {
    f32x2_t ce, pe, co, po;
    float G;
    __device__ __forceinline__ void anchor(const float2 v, const float4 t)
    {
        // t = (G, cos theta, sin theta, .);  x_{mc+-1} = Re[v e^{+-i theta}] = c Re v -+ s Im v
        G = t.x;
        const float w = v.y * t.z;
        const float xm1 = fmaf(v.x, t.y, w);
        if (STRIDE == 1) {
            ce = pk_make(v.x, xm1);
            pe = pk_make(-xm1, -v.x);                          // w_{-1} = -x_{-1}
        } else {
            const float xp1 = fmaf(v.x, t.y, -w);
            const float xm2 = fmaf(t.y + t.y, xm1, -v.x);     // one stride-1 step: x_{mc-2} = 2c x_{mc-1} - x_mc
            ce = pk_make(v.x, xm1);
            pe = pk_make(-xm2, -xp1);
            co = pk_make(xp1, xm2);
            po = pk_make(-xm1, -v.x);
        }
    }
};

#ifndef ST_CHEB_MAX_THREADS
#define ST_CHEB_MAX_THREADS 512
#endif
#define ST_CHEB_PIPE_THREADS 384      // builds with the software-pipelined phase B: 168 registers per thread
// ---- Phase A of the Chebyshev kernels: rasterise, gather p, merge runs of consecutive columns
// that fall in the same bin (their terms share the phase factor, so Eq. 8 only needs the sum of
// their p), compact into the pool, rotate to the anchor of chunk 0.  A lane owns L = ceil(N / 32)
// CONSECUTIVE columns, so runs are merged by a sequential compare-and-add in registers (runs are
// cut at lane boundaries: <= 31 extra pixels per template); finished runs are appended to the pool
// through a ballot.  The work is cut into ELEMENTS of four columns per lane: cheb_fetch issues the
// four rasteriser chains and the L2 gathers of an element, cheb_merge consumes them, so that a
// caller can keep the next element in flight while it merges the current one.
struct ChebFetchCtx {          // what fetching needs to know about a template
    Raster r;
    uint16_t* krow;            // bank cache: this lane's slice of the template's row
    double u_last;             // centre of the last column (clamp target of out-of-range lanes)
    const float2* col0;        // map row of the template's first column
    int32_t N, L, cbase;       // columns, columns per lane, first column of this lane
};
struct ChebElem { int k[4]; float2 p[4], e[4]; float r[4]; };     // r: 1 / sigma, only loaded for norm 2
struct ChebMergeState { int run_k, n_a, n_b; float ax, ay; float2 run_e; float w2, bamp; };
struct ChebCounts { int n_a, n_b; };       // pool entries of class A (front of the pool) and class B (back)

// The normative rasteriser sequence of the rare fallback (inlined: as an out-of-line call the kernel has 19 % less
// code, config 4 +0.5 %, config 5 -1.4 %).
__device__ __forceinline__ int32_t raster_bin_cold(const Raster& r, int32_t c) { return raster_bin(r, c); }

// GEN = false compiles the default search (quadratic templates, N^-alpha normalisation) with the template
// family and the weighting as constants; GEN = true reads both from the arguments (cubic family, norm 2).
// BANK: 0 no bank cache, 1 this launch fills it, 2 this launch reads it (S1 + S2 skipped)
template <bool GEN, int BANK>
__device__ __forceinline__ void cheb_fetch_ctx(const ScoreArgs& a, const Track& t, const uint64_t q, const int lane, ChebFetchCtx& f)
{
    if (BANK != 2) f.r = make_raster(t, a.bp.n_f, GEN ? a.bp.family : 0);
    f.N = t.N;
    f.L = (t.N + kWarp - 1) >> 5;
    f.cbase = lane * f.L;
    if (BANK != 0) f.krow = a.kcache + (a.kcache_base + q) * (uint64_t)a.kcache_stride + (uint32_t)lane * (uint32_t)((f.L + 3) & ~3);
    f.u_last = int_to_double_fast(t.N - 1) + 0.5;
    f.col0 = a.map + (size_t)t.j0 * (size_t)a.bp.n_f;
}
template <bool GEN, int BANK>
__device__ __forceinline__ void cheb_fetch(const ScoreArgs& a, const ChebFetchCtx& f, const int i, ChebElem& E)
{
    int cc[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const int c = f.cbase + i + u;
        cc[u] = c < f.N ? c : f.N - 1;                 // clamped: discarded by the merge
    }
    if (BANK == 2) {                                   // the four bins of this element: one 8-byte read
        const uint2 w = __ldg(reinterpret_cast<const uint2*>(f.krow + i));
        E.k[0] = (int)(w.x & 0xFFFFu); E.k[1] = (int)(w.x >> 16); E.k[2] = (int)(w.y & 0xFFFFu); E.k[3] = (int)(w.y >> 16);
    } else {
        bool redo[4];
        const double ub = int_to_double_fast(f.cbase + i) + 0.5;
#pragma unroll
        for (int u = 0; u < 4; ++u)
            E.k[u] = raster_bin_fast_u(f.r, f.cbase + i + u < f.N ? ub + (double)u : f.u_last, redo[u]);   // branch-free: the four chains interleave
        if (redo[0] | redo[1] | redo[2] | redo[3]) {   // ~1e-5 of the time: normative sequence
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (redo[u]) E.k[u] = raster_bin_cold(f.r, cc[u]);
        }
        if (BANK == 1)
            *reinterpret_cast<uint2*>(f.krow + i) = make_uint2((uint32_t)E.k[0] | ((uint32_t)E.k[1] << 16),
                                                              (uint32_t)E.k[2] | ((uint32_t)E.k[3] << 16));
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        ST_ASSERT(E.k[u] >= 0 && E.k[u] < a.bp.n_f && cc[u] >= 0 &&
                  (size_t)(f.col0 - a.map) / (size_t)a.bp.n_f + (size_t)cc[u] < (size_t)a.bp.n_t);
        E.p[u] = __ldg(f.col0 + (size_t)cc[u] * (size_t)a.bp.n_f + (size_t)E.k[u]);
        E.e[u] = __ldg(&a.Ec[E.k[u]]);
    }
    if (GEN && a.norm == 2) {                          // inverse-variance weights (G25): one more gather per pixel
#pragma unroll
        for (int u = 0; u < 4; ++u)
            E.r[u] = __ldg(a.isig + ((size_t)(f.col0 - a.map) + (size_t)cc[u] * (size_t)a.bp.n_f + (size_t)E.k[u]));
    }
}
__device__ __forceinline__ void cheb_merge_init(ChebMergeState& m)
{
    m.run_k = -1; m.n_a = 0; m.n_b = 0; m.ax = 0.0f; m.ay = 0.0f; m.run_e = make_float2(0.0f, 0.0f); m.w2 = 0.0f; m.bamp = 0.0f;
}
// Append the finished runs of the lanes flagged `emit` (warp-wide ballots keep the pool compact); the rotation
// to the anchor is written with explicit roundings (one multiply, one FMA per component), so every build of the
// kernel forms bit-identical pool entries whatever the assembler would have contracted.  A pixel's
// CLASS is a property of its bin, carried by the two lowest mantissa bits of the anchor phase factor Ec[k].x the
// host uploads (0 = class A; 1, 2, 3 = class B with a drift of at most d_max / 4, d_max / 2, d_max): class A bins run the Chebyshev recurrence; in class B bins the float32 coefficient
// 2 cos(S theta) would drift the phase by more than kChebClassDrift over half a chunk (small theta: fine grids,
// low frequencies), which mis-scores a loud coherent signal where SNR(tau) crosses zero.
//   TWO = true (the general build): class A fills the pool from the front, class B from the back (entries
//     S-1, S-2, ...) and is advanced by Reinsch's form, whose coefficient 4 sin^2(theta/2) keeps its relative
//     precision as theta -> 0;
//   TWO = false (the fast build): one pool; the amplitude |Re v| + |Im v| >= |v| parked in class B bins is
//     summed, weighted by the bin's drift level, and a template whose worst-case drift error
//     scale * sum_B d_k |v|  (d_k rounded up to d_max / 4, / 2 or d_max) could reach a fraction of the G13
//     tolerance is not scored here but handed to the general build (cheb_defer).
template <bool TWO>
__device__ __forceinline__ void cheb_emit(ChebMergeState& m, const bool emit, float2* pool_v, uint16_t* pool_k, const int lane,
                                          const int S)
{
    const uint32_t level = __float_as_uint(m.run_e.x) & 3u;         // 0: class A; 1-3: class B, drift <= d_max / 4, / 2, d_max
    const bool cls_b = level != 0u;
    if (TWO) {
        const uint32_t em_a = __ballot_sync(kFull, emit && !cls_b);
        const uint32_t em_b = __ballot_sync(kFull, emit && cls_b);
        if (emit) {
            const uint32_t below = (1u << lane) - 1u;
            const int e = cls_b ? S - 1 - (m.n_b + __popc(em_b & below)) : m.n_a + __popc(em_a & below);
            pool_v[e] = make_float2(fmaf(m.ax, m.run_e.x, -__fmul_rn(m.ay, m.run_e.y)), fmaf(m.ax, m.run_e.y, __fmul_rn(m.ay, m.run_e.x)));
            pool_k[e] = (uint16_t)m.run_k;
        }
        m.n_a += __popc(em_a);
        m.n_b += __popc(em_b);
    } else {
        const uint32_t em = __ballot_sync(kFull, emit);
        if (emit) {
            const int e = m.n_a + __popc(em & ((1u << lane) - 1u));
            pool_v[e] = make_float2(fmaf(m.ax, m.run_e.x, -__fmul_rn(m.ay, m.run_e.y)), fmaf(m.ax, m.run_e.y, __fmul_rn(m.ay, m.run_e.x)));
            pool_k[e] = (uint16_t)m.run_k;
            if (cls_b) m.bamp = fmaf(fabsf(m.ax) + fabsf(m.ay), __uint_as_float((124u + level) << 23), m.bamp);   // x 2^(level - 3)
        }
        m.n_a += __popc(em);
    }
}
template <bool TWO>
__device__ __forceinline__ void cheb_merge(const int norm, const int N, const int L, const int cbase, const int i, const ChebElem& E,
                                           ChebMergeState& m, float2* pool_v, uint16_t* pool_k, const int lane, const int S)
{
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const bool valid = (i + u < L) && (cbase + i + u < N);
        const bool brk = valid && E.k[u] != m.run_k;   // a new run starts at this column
        cheb_emit<TWO>(m, brk && m.run_k >= 0, pool_v, pool_k, lane, S);
        // branch-free update: a break restarts the sums, a column outside the template adds zero
        float px = valid ? E.p[u].x : 0.0f, py = valid ? E.p[u].y : 0.0f;
        if (norm == 2) {                               // warp-uniform
            const float rs = valid ? E.r[u] : 0.0f;
            px *= rs; py *= rs;
            m.w2 = fmaf(rs, rs, m.w2);
        }
        m.ax = brk ? px : m.ax + px;
        m.ay = brk ? py : m.ay + py;
        m.run_k = brk ? E.k[u] : m.run_k;
        m.run_e.x = brk ? E.e[u].x : m.run_e.x;
        m.run_e.y = brk ? E.e[u].y : m.run_e.y;
    }
}
// the lanes' last runs, then zero-fill both classes up to whole rows of 32 entries; returns the two counts
template <bool TWO>
__device__ __forceinline__ ChebCounts cheb_merge_finish(ChebMergeState& m, float2* pool_v, uint16_t* pool_k, const int lane,
                                                        const int S)
{
    cheb_emit<TWO>(m, m.run_k >= 0, pool_v, pool_k, lane, S);
    const int ea = m.n_a + lane;
    if (ea < ((m.n_a + kWarp - 1) & ~(kWarp - 1))) { pool_v[ea] = make_float2(0.0f, 0.0f); pool_k[ea] = 0; }
    if (TWO) {
        const int eb = S - 1 - (m.n_b + lane);
        if (eb >= S - ((m.n_b + kWarp - 1) & ~(kWarp - 1))) { pool_v[eb] = make_float2(0.0f, 0.0f); pool_k[eb] = 0; }
    }
    __syncwarp();
    ChebCounts c;
    c.n_a = m.n_a; c.n_b = m.n_b;
    return c;
}

// Phase A for one template, start to finish (the next element is in flight while one is merged).
// `defer` (fast build only): the template must be scored by the two-class build instead (see cheb_emit).
template <bool GEN, int BANK>
__device__ __forceinline__ ChebCounts cheb_phase_a(const ScoreArgs& a, const Track& t, const uint64_t q, float2* pool_v,
                                                   uint16_t* pool_k, const int lane, float& scale, bool& defer)
{
    const int S = a.pool_stride;
    ChebFetchCtx f;
    cheb_fetch_ctx<GEN, BANK>(a, t, q, lane, f);
    const int norm = GEN ? a.norm : (a.norm == 1 ? 1 : 0);
    ChebMergeState m;
    cheb_merge_init(m);
    ChebElem E0, E1;                                   // ping-pong: no register copies between elements
    __syncwarp();                                      // the previous template's pool reads are done
    cheb_fetch<GEN, BANK>(a, f, 0, E0);
#pragma unroll 1
    for (int i = 0; i < f.L; i += 8) {
        if (i + 4 < f.L) cheb_fetch<GEN, BANK>(a, f, i + 4, E1);  // warp-uniform
        cheb_merge<GEN>(norm, f.N, f.L, f.cbase, i, E0, m, pool_v, pool_k, lane, S);
        if (i + 4 >= f.L) break;
        if (i + 8 < f.L) cheb_fetch<GEN, BANK>(a, f, i + 8, E0);
        cheb_merge<GEN>(norm, f.N, f.L, f.cbase, i + 4, E1, m, pool_v, pool_k, lane, S);
    }
    scale = track_scale(norm, t.N, m.w2);
    const ChebCounts cnt = cheb_merge_finish<GEN>(m, pool_v, pool_k, lane, S);
    defer = false;
    if (!GEN && a.defer_limit < 3.0e38f) {             // the grid has class B bins (warp-uniform)
        // warp sum in fixed point (1 / 1024, every lane rounded up: never below the float sum) through one REDUX
        // instead of five dependent shuffle + add steps
        const uint32_t bq = __reduce_add_sync(kFull, __float2uint_ru(fminf(m.bamp, 3.0e4f) * 1024.0f));
        defer = (float)bq * (scale * (1.0f / 1024.0f)) > a.defer_limit;
    }
    return cnt;
}

// Phase B for one template whose merged pixels sit in (pool_v, pool_k): every delay of the grid,
// fused S4.  pool_v is advanced in place from chunk to chunk.
// MODE 0: search; 1: capture pass of st_search_topk; 2: search + per-template maximum over the delays
// TWO: the pool holds class B rows at its back (general build)
template <int STRIDE, int MODE, bool TWO>
__device__ __forceinline__ void cheb_phase_b(const ScoreArgs& a, WarpReduce& wr, uint32_t* sm_hist,
                                             const float4* sm_tab, const float* sm_zi, float2* pool_v,
                                             const uint16_t* pool_k, const ChebCounts cnt, const float scale,
                                             const uint64_t id, const uint64_t q, const int n_chunks, const int lane)
{
    const int n_rows = (cnt.n_a + kWarp - 1) >> 5;          // class A rows, from the front of the pool
    const int n_rows_b = TWO ? (cnt.n_b + kWarp - 1) >> 5 : 0;   // class B rows, from its back
    const int S = a.pool_stride;
    TrackMax tm;
    tmax_init(tm);
    const uint32_t pv_base = smem_u32(pool_v) + (uint32_t)lane * 8u, pk_base = smem_u32(pool_k) + (uint32_t)lane * 2u;
    const uint32_t tab_base = smem_u32(sm_tab), zi_base = smem_u32(sm_zi);
    // ---- phase B: chunks of 64 delays; f2[i] = (sum x_{mc+i}, sum x_{mc-1-i}) over this lane's pixels
#pragma unroll 1
    for (int j = 0; j < n_chunks; ++j) {
        f32x2_t f2[kHalf];
#pragma unroll
        for (int i = 0; i < kHalf; ++i) f2[i] = 0ull;
        int row = 0;
        uint32_t pv = pv_base, pk = pk_base;           // this lane's entry of the current row
#pragma unroll 1
        for (; row + 2 <= n_rows; row += 2, pv += 2 * kWarp * 8, pk += 2 * kWarp * 2) {
            const float2 v0 = lds_f2<0>(pv), v1 = lds_f2<kWarp * 8>(pv);
            const uint32_t k0 = lds_u16<0>(pk), k1 = lds_u16<kWarp * 2>(pk);
            ST_ASSERT(k0 < (uint32_t)a.bp.n_f && k1 < (uint32_t)a.bp.n_f);
            const float4 t0 = lds_f4(tab_base + k0 * 16u), t1 = lds_f4(tab_base + k1 * 16u);
            const float zi0 = lds_f1(zi_base + k0 * 4u), zi1 = lds_f1(zi_base + k1 * 4u);
            // next chunk's anchors: v e^{i 64 theta}   (t.w = cos 64 theta, zi = sin 64 theta).  Unconditional: skipping
            // the advance on the last chunk (a warp-uniform branch here) cost 4-7 % (measured, round 2)
            sts_f2<0>(pv, fmaf(v0.x, t0.w, -(v0.y * zi0)), fmaf(v0.x, zi0, v0.y * t0.w));
            sts_f2<kWarp * 8>(pv, fmaf(v1.x, t1.w, -(v1.y * zi1)), fmaf(v1.x, zi1, v1.y * t1.w));
            ChebPixel<STRIDE> A, B;
            A.anchor(v0, t0);
            B.anchor(v1, t1);
            if (STRIDE == 1) {
#pragma unroll
                for (int i = 0; i < kHalf; i += 2) {
                    f2[i] = pk_add(f2[i], A.ce);
                    f2[i] = pk_add(f2[i], B.ce);
                    A.pe = pk_step(A.G, A.ce, A.pe);            // pe now holds offset i + 1
                    B.pe = pk_step(B.G, B.ce, B.pe);
                    f2[i + 1] = pk_add(f2[i + 1], A.pe);
                    f2[i + 1] = pk_add(f2[i + 1], B.pe);
                    A.ce = pk_step(-A.G, A.pe, A.ce);            // ce holds offset i + 2
                    B.ce = pk_step(-B.G, B.pe, B.ce);
                }
            } else {
#pragma unroll
                for (int i = 0; i < kHalf; i += 4) {
                    f2[i] = pk_add(f2[i], A.ce);
                    f2[i] = pk_add(f2[i], B.ce);
                    f2[i + 1] = pk_add(f2[i + 1], A.co);
                    f2[i + 1] = pk_add(f2[i + 1], B.co);
                    A.pe = pk_step(A.G, A.ce, A.pe);            // offset i + 2
                    B.pe = pk_step(B.G, B.ce, B.pe);
                    A.po = pk_step(A.G, A.co, A.po);            // offset i + 3
                    B.po = pk_step(B.G, B.co, B.po);
                    f2[i + 2] = pk_add(f2[i + 2], A.pe);
                    f2[i + 2] = pk_add(f2[i + 2], B.pe);
                    f2[i + 3] = pk_add(f2[i + 3], A.po);
                    f2[i + 3] = pk_add(f2[i + 3], B.po);
                    A.ce = pk_step(-A.G, A.pe, A.ce);            // offset i + 4
                    B.ce = pk_step(-B.G, B.pe, B.ce);
                    A.co = pk_step(-A.G, A.po, A.co);            // offset i + 5
                    B.co = pk_step(-B.G, B.po, B.co);
                }
            }
        }
        if (row < n_rows) {          // odd tail row
            const float2 v0 = lds_f2<0>(pv);
            const uint32_t k0 = lds_u16<0>(pk);
            const float4 t0 = lds_f4(tab_base + k0 * 16u);
            const float zi0 = lds_f1(zi_base + k0 * 4u);
            sts_f2<0>(pv, fmaf(v0.x, t0.w, -(v0.y * zi0)), fmaf(v0.x, zi0, v0.y * t0.w));
            ChebPixel<STRIDE> A;
            A.anchor(v0, t0);
            if (STRIDE == 1) {
#pragma unroll
                for (int i = 0; i < kHalf; i += 2) {
                    f2[i] = pk_add(f2[i], A.ce);
                    A.pe = pk_step(A.G, A.ce, A.pe);
                    f2[i + 1] = pk_add(f2[i + 1], A.pe);
                    A.ce = pk_step(-A.G, A.pe, A.ce);
                }
            } else {
#pragma unroll
                for (int i = 0; i < kHalf; i += 4) {
                    f2[i] = pk_add(f2[i], A.ce);
                    f2[i + 1] = pk_add(f2[i + 1], A.co);
                    A.pe = pk_step(A.G, A.ce, A.pe);
                    A.po = pk_step(A.G, A.co, A.po);
                    f2[i + 2] = pk_add(f2[i + 2], A.pe);
                    f2[i + 3] = pk_add(f2[i + 3], A.po);
                    A.ce = pk_step(-A.G, A.pe, A.ce);
                    A.co = pk_step(-A.G, A.po, A.co);
                }
            }
        }
        // ---- class B rows (Reinsch's form, stride 1): x_{n+1} = x_n + d_{n+1}, d_{n+1} = d_n - kappa x_n with
        // kappa = 4 sin^2(theta/2); pair = (forward, backward) as above, the
        // backward half runs the same recurrence from d = -(x_mc - x_{mc-1}).  Three packed operations per
        // two evaluations; the accumulators take x with the sign the Chebyshev chains carry at that offset.
        if (TWO) {
#pragma unroll 1
        for (int rb = 0; rb < n_rows_b; ++rb) {
            const int e0 = S - kWarp * (rb + 1) + lane;
            const float2 v0 = pool_v[e0];
            const int k0 = pool_k[e0];
            ST_ASSERT(e0 >= 0 && k0 >= 0 && k0 < a.bp.n_f);
            const float4 t0 = sm_tab[k0];
            const float zi0 = sm_zi[k0];
            pool_v[e0] = make_float2(fmaf(v0.x, t0.w, -(v0.y * zi0)), fmaf(v0.x, zi0, v0.y * t0.w));
            // kappa = 2 (1 - cos theta) = 2 sin^2 theta / (1 + cos theta): from the float32 (cos, sin) of the table
            // without cancellation (relative error <= 3e-7: 5e-6 |theta| rad over half a chunk, |theta| <= 0.6)
            const float kap = __fdiv_rn(2.0f * t0.z * t0.z, 1.0f + t0.y);
            // x_mc - x_{mc-1} = Re v (1 - cos theta) - Im v sin theta, 1 - cos theta = kappa / 2
            const float dlt = fmaf(0.5f * kap, v0.x, -(v0.y * t0.z));
            f32x2_t x = pk_make(v0.x, v0.x - dlt), d = pk_make(dlt, -dlt);
            const float nk = -kap;
#pragma unroll
            for (int i = 0; i < kHalf; ++i) {
                f2[i] = ((i >> STRIDE) & 1) ? pk_sub(f2[i], x) : pk_add(f2[i], x);
                d = pk_step(nk, x, d);
                x = pk_add(x, d);
            }
        }
        }
        // ---- fold across the 32 lanes (transposing tree on register pairs): lane l keeps pair l
#pragma unroll
        for (int off = 16, n = kHalf / 2; off >= 1; off >>= 1, n >>= 1) {
            const bool upper = (lane & off) != 0;
#pragma unroll
            for (int i = 0; i < n; ++i) {
                const f32x2_t send = upper ? f2[i] : f2[i + n];
                const f32x2_t keep = upper ? f2[i + n] : f2[i];
                f2[i] = pk_add(keep, __shfl_xor_sync(kFull, send, off));
            }
        }
        // sign s_n of the chains: accumulator l holds chain index n = l (stride 1) or l >> 1 (stride 2)
    const float sscale = ((lane >> STRIDE) & 1) ? -scale : scale;
    const float v[2] = {pk_lo(f2[0]) * sscale, pk_hi(f2[0]) * sscale};
        const uint32_t ms[2] = {(uint32_t)(j * kCheb + kHalf + lane), (uint32_t)(j * kCheb + kHalf - 1 - lane)};
        const bool ok[2] = {(int)ms[0] < a.n_tau, (int)ms[1] < a.n_tau};
        reduce_samples<2, MODE == 1 ? 1 : 0>(a, wr, sm_hist, id, q, v, ms, ok);
        if (MODE == 2) tmax_update<2>(tm, v, ms, ok);
    }
    if (MODE == 2) tmax_finish(a, tm, q);
}

// Phase B, delay-split form (PB 1, 2): the two half-warps work on TWO chunks of the same 16 pool entries
// per row -- lanes 0-15 on chunk 2 jp (anchor v as stored), lanes 16-31 on chunk 2 jp + 1 (anchor
// v e^{i 64 theta}) -- so one fold and one S4 epilogue serve 128 delays, rows are padded to 16 entries
// instead of 32, and the two halves read the same pool and table words (broadcasts, half the bank
// conflicts).  The anchor of the next pass, v e^{i 128 theta}, is formed as (v z64) z64: the same two
// float32 rotations the one-chunk form applies in two steps.
//   FOLD 0: transposing shuffle tree over the 16 lanes of a half (30 packed shuffles per pass; lane l of
//           a half ends with accumulators 2 l and 2 l + 1);
//   FOLD 1: through shared memory in two rounds of 16 accumulators (8 STS.128, 16 LDS.64 and 15 packed
//           adds per round; lane l ends with accumulators l and 16 + l); needs kFoldWords floats per warp.
//   SINGLE: the grid has at most two chunks: one pass, no anchor is stored back.
constexpr int kFoldRow = 36;                    // floats per lane row of the fold scratch: 16 pairs + 16 B (conflict-free)
constexpr int kFoldWords = kWarp * kFoldRow;    // floats of fold scratch per warp (4608 B)
__device__ __forceinline__ void sts_f4(uint32_t addr, f32x2_t a, f32x2_t b)
{
    asm volatile("st.shared.v2.b64 [%0], {%1, %2};" :: "r"(addr), "l"(a), "l"(b) : "memory");
}
__device__ __forceinline__ f32x2_t lds_pk(uint32_t addr)
{
    f32x2_t v;
    asm volatile("ld.shared.b64 %0, [%1];" : "=l"(v) : "r"(addr));
    return v;
}
// One row pair of the delay-split phase B on its way from the pool to its chain heads, in three stages.
struct ChebStage { float2 v0, v1; uint32_t k0, k1; float4 t0, t1; float zi0, zi1; };
__device__ __forceinline__ void cheb_stage_load(ChebStage& g, const uint32_t pv, const uint32_t pk)
{
    g.v0 = lds_f2<0>(pv); g.v1 = lds_f2<16 * 8>(pv);
    g.k0 = lds_u16<0>(pk); g.k1 = lds_u16<16 * 2>(pk);
}
__device__ __forceinline__ void cheb_stage_table(ChebStage& g, const uint32_t tab_base, const uint32_t zi_base)
{
    g.t0 = lds_f4(tab_base + g.k0 * 16u); g.t1 = lds_f4(tab_base + g.k1 * 16u);
    g.zi0 = lds_f1(zi_base + g.k0 * 4u); g.zi1 = lds_f1(zi_base + g.k1 * 4u);
}
__device__ __forceinline__ void sts_f2_if(const bool p, const uint32_t addr, const float x, const float y)
{
    asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.u32 q, %0, 0;\n\t@q st.shared.v2.f32 [%1], {%2, %3};\n\t}"
                 :: "r"((uint32_t)p), "r"(addr), "f"(x), "f"(y) : "memory");
}
template <int STRIDE, bool SINGLE>
__device__ __forceinline__ void cheb_stage_anchor(const ChebStage& g, const bool upper, const bool store, const uint32_t pv,
                                                  ChebPixel<STRIDE>& A, ChebPixel<STRIDE>& B)
{
    const float r0x = fmaf(g.v0.x, g.t0.w, -(g.v0.y * g.zi0)), r0y = fmaf(g.v0.x, g.zi0, g.v0.y * g.t0.w);   // v e^{i 64 theta}
    const float r1x = fmaf(g.v1.x, g.t1.w, -(g.v1.y * g.zi1)), r1y = fmaf(g.v1.x, g.zi1, g.v1.y * g.t1.w);
    if (!SINGLE) {                                          // the next pass's anchor, (v z64) z64, kept by the lower half
        sts_f2_if(store, pv, fmaf(r0x, g.t0.w, -(r0y * g.zi0)), fmaf(r0x, g.zi0, r0y * g.t0.w));
        sts_f2_if(store, pv + 16 * 8, fmaf(r1x, g.t1.w, -(r1y * g.zi1)), fmaf(r1x, g.zi1, r1y * g.t1.w));
    }
    A.anchor(make_float2(upper ? r0x : g.v0.x, upper ? r0y : g.v0.y), g.t0);
    B.anchor(make_float2(upper ? r1x : g.v1.x, upper ? r1y : g.v1.y), g.t1);
}
template <int STRIDE, int MODE, bool TWO, int FOLD, bool SINGLE, bool PIPE>
__device__ __forceinline__ void cheb_phase_b_split(const ScoreArgs& a, WarpReduce& wr, uint32_t* sm_hist,
                                                   const float4* sm_tab, const float* sm_zi, float2* pool_v,
                                                   const uint16_t* pool_k, float* fold, const ChebCounts cnt, const float scale,
                                                   const uint64_t id, const uint64_t q, const int n_chunks, const int lane)
{
    constexpr int kW = 16;                                  // pool entries per row
    // class A rows of 16 entries, from the front of the pool (zero-filled to whole rows of 32: the pipelined form
    // takes rows in pairs, the plain form handles an odd last row on its own)
    const int n_rows = PIPE ? ((cnt.n_a + kWarp - 1) >> 5) << 1 : (cnt.n_a + kW - 1) >> 4;
    const int n_rows_b = TWO ? (cnt.n_b + kW - 1) >> 4 : 0; // class B rows, from its back
    const int S = a.pool_stride;
    const int l16 = lane & 15;
    const bool upper = (lane & 16) != 0;
    TrackMax tm;
    tmax_init(tm);
    const uint32_t pv_base = smem_u32(pool_v) + (uint32_t)l16 * 8u, pk_base = smem_u32(pool_k) + (uint32_t)l16 * 2u;
    const uint32_t tab_base = smem_u32(sm_tab), zi_base = smem_u32(sm_zi);
    const int n_pass = SINGLE ? 1 : (n_chunks + 1) >> 1;
#pragma unroll 1
    for (int jp = 0; jp < n_pass; ++jp) {
        f32x2_t f2[kHalf];
#pragma unroll
        for (int i = 0; i < kHalf; ++i) f2[i] = 0ull;
        if (!PIPE) {
        int row = 0;
        uint32_t pv = pv_base, pk = pk_base;
#pragma unroll 1
        for (; row + 2 <= n_rows; row += 2, pv += 2 * kW * 8, pk += 2 * kW * 2) {
            ChebStage g;
            cheb_stage_load(g, pv, pk);
            ST_ASSERT(g.k0 < (uint32_t)a.bp.n_f && g.k1 < (uint32_t)a.bp.n_f);
            cheb_stage_table(g, tab_base, zi_base);
            ChebPixel<STRIDE> A, B;
            cheb_stage_anchor<STRIDE, SINGLE>(g, upper, !upper, pv, A, B);
            if (STRIDE == 1) {
#pragma unroll
                for (int i = 0; i < kHalf; i += 2) {
                    f2[i] = pk_add(f2[i], A.ce);
                    f2[i] = pk_add(f2[i], B.ce);
                    A.pe = pk_step(A.G, A.ce, A.pe);
                    B.pe = pk_step(B.G, B.ce, B.pe);
                    f2[i + 1] = pk_add(f2[i + 1], A.pe);
                    f2[i + 1] = pk_add(f2[i + 1], B.pe);
                    A.ce = pk_step(-A.G, A.pe, A.ce);
                    B.ce = pk_step(-B.G, B.pe, B.ce);
                }
            } else {
#pragma unroll
                for (int i = 0; i < kHalf; i += 4) {
                    f2[i] = pk_add(f2[i], A.ce);
                    f2[i] = pk_add(f2[i], B.ce);
                    f2[i + 1] = pk_add(f2[i + 1], A.co);
                    f2[i + 1] = pk_add(f2[i + 1], B.co);
                    A.pe = pk_step(A.G, A.ce, A.pe);
                    B.pe = pk_step(B.G, B.ce, B.pe);
                    A.po = pk_step(A.G, A.co, A.po);
                    B.po = pk_step(B.G, B.co, B.po);
                    f2[i + 2] = pk_add(f2[i + 2], A.pe);
                    f2[i + 2] = pk_add(f2[i + 2], B.pe);
                    f2[i + 3] = pk_add(f2[i + 3], A.po);
                    f2[i + 3] = pk_add(f2[i + 3], B.po);
                    A.ce = pk_step(-A.G, A.pe, A.ce);
                    B.ce = pk_step(-B.G, B.pe, B.ce);
                    A.co = pk_step(-A.G, A.po, A.co);
                    B.co = pk_step(-B.G, B.po, B.co);
                }
            }
        }
        if (row < n_rows) {          // odd last row
            const float2 v0 = lds_f2<0>(pv);
            const uint32_t k0 = lds_u16<0>(pk);
            const float4 t0 = lds_f4(tab_base + k0 * 16u);
            const float zi0 = lds_f1(zi_base + k0 * 4u);
            const float r0x = fmaf(v0.x, t0.w, -(v0.y * zi0)), r0y = fmaf(v0.x, zi0, v0.y * t0.w);
            if (!SINGLE) sts_f2_if(!upper, pv, fmaf(r0x, t0.w, -(r0y * zi0)), fmaf(r0x, zi0, r0y * t0.w));
            ChebPixel<STRIDE> A;
            A.anchor(make_float2(upper ? r0x : v0.x, upper ? r0y : v0.y), t0);
            if (STRIDE == 1) {
#pragma unroll
                for (int i = 0; i < kHalf; i += 2) {
                    f2[i] = pk_add(f2[i], A.ce);
                    A.pe = pk_step(A.G, A.ce, A.pe);
                    f2[i + 1] = pk_add(f2[i + 1], A.pe);
                    A.ce = pk_step(-A.G, A.pe, A.ce);
                }
            } else {
#pragma unroll
                for (int i = 0; i < kHalf; i += 4) {
                    f2[i] = pk_add(f2[i], A.ce);
                    f2[i + 1] = pk_add(f2[i + 1], A.co);
                    A.pe = pk_step(A.G, A.ce, A.pe);
                    A.po = pk_step(A.G, A.co, A.po);
                    f2[i + 2] = pk_add(f2[i + 2], A.pe);
                    f2[i + 3] = pk_add(f2[i + 3], A.po);
                    A.ce = pk_step(-A.G, A.pe, A.ce);
                    A.co = pk_step(-A.G, A.po, A.co);
                }
            }
        }
        } else {
        // Row pairs, software-pipelined: the pool / table reads, the anchor rotation and the chain heads of the
        // NEXT pair are issued at fixed points under the 32 steps of the current one (every access and every packed
        // operation here is a volatile asm statement, so the source order is the issue order).  On the last pair the
        // "next" pair is the current one again (a harmless re-read, its store predicated off).
        uint32_t pv = pv_base, pk = pk_base;
        ChebPixel<STRIDE> A, B;
        if (n_rows > 0) {                                   // (a template of class B pixels only has no class A row)
            ChebStage g;
            cheb_stage_load(g, pv, pk);
            cheb_stage_table(g, tab_base, zi_base);
            cheb_stage_anchor<STRIDE, SINGLE>(g, upper, !upper, pv, A, B);
        }
#pragma unroll 1
        for (int row = 0; row < n_rows; row += 2) {
            const bool has_next = row + 2 < n_rows;
            const uint32_t pvn = has_next ? pv + 2 * kW * 8 : pv, pkn = has_next ? pk + 2 * kW * 2 : pk;
            ChebStage g;
            ChebPixel<STRIDE> An, Bn;
            if (STRIDE == 1) {
#pragma unroll
                for (int i = 0; i < kHalf; i += 2) {
                    if (i == 0) cheb_stage_load(g, pvn, pkn);
                    if (i == 8) cheb_stage_table(g, tab_base, zi_base);
                    if (i == 20) cheb_stage_anchor<STRIDE, SINGLE>(g, upper, has_next && !upper, pvn, An, Bn);
                    f2[i] = pk_add(f2[i], A.ce);
                    f2[i] = pk_add(f2[i], B.ce);
                    A.pe = pk_step(A.G, A.ce, A.pe);
                    B.pe = pk_step(B.G, B.ce, B.pe);
                    f2[i + 1] = pk_add(f2[i + 1], A.pe);
                    f2[i + 1] = pk_add(f2[i + 1], B.pe);
                    A.ce = pk_step(-A.G, A.pe, A.ce);
                    B.ce = pk_step(-B.G, B.pe, B.ce);
                }
            } else {
#pragma unroll
                for (int i = 0; i < kHalf; i += 4) {
                    if (i == 0) cheb_stage_load(g, pvn, pkn);
                    if (i == 8) cheb_stage_table(g, tab_base, zi_base);
                    if (i == 20) cheb_stage_anchor<STRIDE, SINGLE>(g, upper, has_next && !upper, pvn, An, Bn);
                    f2[i] = pk_add(f2[i], A.ce);
                    f2[i] = pk_add(f2[i], B.ce);
                    f2[i + 1] = pk_add(f2[i + 1], A.co);
                    f2[i + 1] = pk_add(f2[i + 1], B.co);
                    A.pe = pk_step(A.G, A.ce, A.pe);
                    B.pe = pk_step(B.G, B.ce, B.pe);
                    A.po = pk_step(A.G, A.co, A.po);
                    B.po = pk_step(B.G, B.co, B.po);
                    f2[i + 2] = pk_add(f2[i + 2], A.pe);
                    f2[i + 2] = pk_add(f2[i + 2], B.pe);
                    f2[i + 3] = pk_add(f2[i + 3], A.po);
                    f2[i + 3] = pk_add(f2[i + 3], B.po);
                    A.ce = pk_step(-A.G, A.pe, A.ce);
                    B.ce = pk_step(-B.G, B.pe, B.ce);
                    A.co = pk_step(-A.G, A.po, A.co);
                    B.co = pk_step(-B.G, B.po, B.co);
                }
            }
            A = An; B = Bn; pv = pvn; pk = pkn;
        }
        }
        // ---- class B rows (Reinsch's form, see the one-chunk form above), 16 entries per row from the back
        if (TWO) {
#pragma unroll 1
        for (int rb = 0; rb < n_rows_b; ++rb) {
            const int e0 = S - kW * (rb + 1) + l16;
            const float2 v0 = pool_v[e0];
            const int k0 = pool_k[e0];
            ST_ASSERT(e0 >= 0 && k0 >= 0 && k0 < a.bp.n_f);
            const float4 t0 = sm_tab[k0];
            const float zi0 = sm_zi[k0];
            const float r0x = fmaf(v0.x, t0.w, -(v0.y * zi0)), r0y = fmaf(v0.x, zi0, v0.y * t0.w);
            if (!SINGLE) {
                const float n0x = fmaf(r0x, t0.w, -(r0y * zi0)), n0y = fmaf(r0x, zi0, r0y * t0.w);
                __syncwarp();                              // both halves have read the entry
                if (!upper) pool_v[e0] = make_float2(n0x, n0y);
            }
            const float ax = upper ? r0x : v0.x, ay = upper ? r0y : v0.y;
            const float kap = __fdiv_rn(2.0f * t0.z * t0.z, 1.0f + t0.y);
            const float dlt = fmaf(0.5f * kap, ax, -(ay * t0.z));
            f32x2_t x = pk_make(ax, ax - dlt), d = pk_make(dlt, -dlt);
            const float nk = -kap;
#pragma unroll
            for (int i = 0; i < kHalf; ++i) {
                f2[i] = ((i >> STRIDE) & 1) ? pk_sub(f2[i], x) : pk_add(f2[i], x);
                d = pk_step(nk, x, d);
                x = pk_add(x, d);
            }
        }
        }
        // ---- fold over the 16 lanes of each half; this lane's two accumulators are i0 and i1
        int i0, i1;
        f32x2_t g0, g1;
        if (FOLD == 0) {
#pragma unroll
            for (int off = 8, n = kHalf / 2; off >= 1; off >>= 1, n >>= 1) {
                const bool up = (lane & off) != 0;
#pragma unroll
                for (int i = 0; i < n; ++i) {
                    const f32x2_t send = up ? f2[i] : f2[i + n];
                    const f32x2_t keep = up ? f2[i + n] : f2[i];
                    f2[i] = pk_add(keep, __shfl_xor_sync(kFull, send, off));
                }
            }
            g0 = f2[0]; g1 = f2[1]; i0 = 2 * l16; i1 = i0 + 1;
        } else {
            const uint32_t fs = smem_u32(fold);
            const uint32_t wr_addr = fs + (uint32_t)lane * (kFoldRow * 4u);
            const uint32_t rd_addr = fs + (uint32_t)(lane & 16) * (kFoldRow * 4u) + (uint32_t)l16 * 8u;
            f32x2_t g[2];
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                __syncwarp();
#pragma unroll
                for (int i = 0; i < 16; i += 2) sts_f4(wr_addr + (uint32_t)i * 8u, f2[16 * r + i], f2[16 * r + i + 1]);
                __syncwarp();
                f32x2_t s[16];
#pragma unroll
                for (int rr = 0; rr < 16; ++rr) s[rr] = lds_pk(rd_addr + (uint32_t)rr * (kFoldRow * 4u));
#pragma unroll
                for (int w = 8; w >= 1; w >>= 1)
#pragma unroll
                    for (int rr = 0; rr < w; ++rr) s[rr] = pk_add(s[rr], s[rr + w]);
                g[r] = s[0];
            }
            g0 = g[0]; g1 = g[1]; i0 = l16; i1 = l16 + 16;
        }
        const int mc = (2 * jp + (upper ? 1 : 0)) * kCheb + kHalf;
        const float s0 = ((i0 >> STRIDE) & 1) ? -scale : scale, s1 = ((i1 >> STRIDE) & 1) ? -scale : scale;
        const float v[4] = {pk_lo(g0) * s0, pk_hi(g0) * s0, pk_lo(g1) * s1, pk_hi(g1) * s1};
        const uint32_t ms[4] = {(uint32_t)(mc + i0), (uint32_t)(mc - 1 - i0), (uint32_t)(mc + i1), (uint32_t)(mc - 1 - i1)};
        const bool ok[4] = {(int)ms[0] < a.n_tau, (int)ms[1] < a.n_tau, (int)ms[2] < a.n_tau, (int)ms[3] < a.n_tau};
        reduce_samples<4, MODE == 1 ? 1 : 0>(a, wr, sm_hist, id, q, v, ms, ok);
        if (MODE == 2) tmax_update<4>(tm, v, ms, ok);
    }
    if (MODE == 2) tmax_finish(a, tm, q);
}

// -DST_ABLATE=1 | 2 (python -m paper_1401_8060_b200.build --ablate N): MEASUREMENT builds of the Chebyshev kernel that
// bound where its time goes (profiles/r03_ablation.md); their results are meaningless and no test loads them.
//   1  phase B alone: a warp runs S1 + S2 + phase A for one claim in 16 and re-scores that pool for the 15 claims
//      that follow (the epilogue, fold and S4 run as usual): no Philox, rasteriser, gather, merge on 15/16 of the
//      claims.  The periodic refresh keeps the mix of pool sizes that of the bank: with the work claimed
//      dynamically, a warp that kept one short pool for the whole launch would take more than its share of claims;
//   2  phase A alone: S1 + S2 + gather + merge + compaction into the pool for every template, phase B skipped.
// n_pixels (hence bench.py's evals) still counts N x n_tau of what each claim stood for.
#ifndef ST_ABLATE
#define ST_ABLATE 0
#endif

template <int STRIDE, int MODE, bool GEN, int BANK, int PB = 0, bool PIPE = false>
__global__ void __launch_bounds__(PIPE ? ST_CHEB_PIPE_THREADS : ST_CHEB_MAX_THREADS, 1) k_score_cheb(const ScoreArgs a)
{
    extern __shared__ __align__(16) unsigned char smem[];
    uint32_t* sm_hist = reinterpret_cast<uint32_t*>(smem);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_warps = blockDim.x >> 5;
    // shared memory: hist | cheb[n_f] float4 | v[n_warps][S] float2 | z64i[n_f (padded)] float | k[n_warps][S] u16
    float4* sm_tab = reinterpret_cast<float4*>(sm_hist + hist_smem_words(a.n_bins));
    const int S = a.pool_stride;
    float2* pool_v = reinterpret_cast<float2*>(sm_tab + a.bp.n_f) + (size_t)warp * S;
    float* sm_zi = reinterpret_cast<float*>(reinterpret_cast<float2*>(sm_tab + a.bp.n_f) + (size_t)n_warps * S);
    uint16_t* pool_k = reinterpret_cast<uint16_t*>(sm_zi + ((a.bp.n_f + 1) & ~1)) + (size_t)warp * S;
    // PB 2, 4: per-warp fold scratch behind the bin pools (16-byte aligned: the host pads the pools)
    float* fold = reinterpret_cast<float*>(smem + a.fold_offset) + (size_t)warp * kFoldWords;
    for (int k = threadIdx.x; k < a.bp.n_f; k += blockDim.x) { sm_tab[k] = a.cheb[k]; sm_zi[k] = a.cheb_zi[k]; }
    hist_init(sm_hist, a.n_bins);
    const int n_chunks = (a.n_tau + kCheb - 1) / kCheb;
    WarpReduce wr;
    reduce_init(wr);
    // the template counter's L2 atomic (~1 us round trip) is issued one template ahead; its result
    // stays in lane 0 until the next iteration broadcasts it
    unsigned long long q_pref = 0;
    if (lane == 0) q_pref = claim_add(&a.sc->counter, 1ull);
    // a launch works through its own id range, or (general build, defer_in) through the list of templates the
    // fast build handed over: the list is complete, the fast launch precedes this one on the stream
    const uint64_t n_items = (GEN && a.defer_in) ? (uint64_t)min(a.sc->n_deferred, a.deferred_cap) : a.n_tracks;
    if (GEN && a.defer_in && blockIdx.x == 0 && threadIdx.x == 0) a.sc->n_deferred_total += (uint32_t)n_items;
#if ST_ABLATE == 1
    bool abl_have = false; Track abl_t; ChebCounts abl_cnt; float abl_scale = 0.0f; uint32_t abl_age = 0;
#endif
    for (;;) {
        const uint64_t item = claim_value(__shfl_sync(kFull, q_pref, 0));
        if (item >= n_items) break;
        if (lane == 0) q_pref = claim_add(&a.sc->counter, 1ull);
        const uint64_t q = (GEN && a.defer_in) ? (uint64_t)a.deferred[item] : item;
        const uint64_t id = a.track_offset + q;
        Track t;
        float scale;
        bool defer;
        ChebCounts cnt;
#if ST_ABLATE == 1
        if (abl_have && (++abl_age & 15u) != 0u) { t = abl_t; cnt = abl_cnt; scale = abl_scale; defer = false; }
        else {
#endif
        if (BANK == 2) {                           // S1 from the bank cache: only N and j0 are needed downstream
            const int2 nj = __ldg(&a.kmeta[a.kcache_base + q]);
            t.N = nj.x; t.j0 = nj.y; t.a = t.y0 = t.y1 = t.y2 = t.tau = t.y3 = 0.0;
        } else {
            t = GEN ? load_track(a, q, id) : make_track(a.bp, id);             // explicit templates take the general build
            if (BANK == 1 && lane == 0) a.kmeta[a.kcache_base + q] = make_int2(t.N, t.j0);
        }
        cnt = cheb_phase_a<GEN, BANK>(a, t, q, pool_v, pool_k, lane, scale, defer);
#if ST_ABLATE == 1
        abl_have = GEN || !defer; abl_t = t; abl_cnt = cnt; abl_scale = scale;
        }
#endif
        if (!GEN && defer) {                       // warp-uniform: too much amplitude in class B bins for this build
            if (lane == 0) {
                const uint32_t slot = atomicAdd(&a.sc->n_deferred, 1u);
                ST_ASSERT(slot < a.deferred_cap);
                if (slot < a.deferred_cap) a.deferred[slot] = (uint32_t)q;
            }
            continue;
        }
        wr.pixels += (unsigned long long)t.N;
#if ST_ABLATE == 2
        continue;                                  // phase A alone
#endif
        ST_ASSERT(cnt.n_a + cnt.n_b >= 1 && cnt.n_a + cnt.n_b <= t.N &&
                  ((cnt.n_a + kWarp - 1) & ~(kWarp - 1)) + ((cnt.n_b + kWarp - 1) & ~(kWarp - 1)) <= S &&
                  (a.tracks || (t.N >= a.bp.n_min && t.N <= a.bp.n_max)) && t.j0 >= 0 && t.j0 + t.N <= a.bp.n_t);
        // PB: 0 one chunk per pass; 1 / 2 two chunks per pass (shuffle / shared-memory fold); 3 / 4 the same for
        // grids of at most two chunks (one pass)
        if (PB == 0)
            cheb_phase_b<STRIDE, MODE, GEN>(a, wr, sm_hist, sm_tab, sm_zi, pool_v, pool_k, cnt, scale, id, q, n_chunks, lane);
        else
            cheb_phase_b_split<STRIDE, MODE, GEN, (PB == 2 || PB == 4) ? 1 : 0, (PB >= 3), PIPE>(a, wr, sm_hist, sm_tab, sm_zi, pool_v, pool_k,
                                                                                          fold, cnt, scale, id, q, n_chunks, lane);
    }
#if ST_ABLATE == 2
    if (pool_v[lane].x == 123.456f && pool_k[lane] == 54321) a.sc->overflow = 1u;      // keeps the pool stores observable
#endif
    reduce_finish(a, wr);
    hist_flush(sm_hist, a.hist, a.n_bins);
}

// ----------------------------------------------------------------------- S4 --
// Float64 score of one (template, delay): Eq. 8 with cos/sin of 2 pi f tau in
// double, lanes over columns, fixed-order shuffle tree.  All lanes return it.
__device__ __forceinline__ double score_f64(const float2* __restrict__ map, const float* __restrict__ isig, const BankParams& bp,
                                            double f_min, double df, const Track& t, double tau, int norm)
{
    const int lane = threadIdx.x & 31;
    const Raster r = make_raster(t, bp.n_f, bp.family);
    double acc = 0.0, w2 = 0.0;
    for (int c = lane; c < t.N; c += kWarp) {
        const int k = raster_bin_fast(r, c);
        const size_t pix = (size_t)(t.j0 + c) * (size_t)bp.n_f + (size_t)k;
        const float2 p = map[pix];
        const double phi = kTwoPi * (f_min + (double)k * df) * tau;
        double s, co;
        sincos(phi, &s, &co);
        const double rho = co * (double)p.x - s * (double)p.y;
        if (norm == 2) { const double rs = (double)isig[pix]; acc += rho * rs; w2 += rs * rs; }
        else acc += rho;
    }
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        acc += __shfl_xor_sync(kFull, acc, off);
        w2 += __shfl_xor_sync(kFull, w2, off);
    }
    if (norm == 2) return w2 > 0.0 ? acc / sqrt(w2) : 0.0;
    return acc / (norm == 0 ? sqrt((double)t.N) : (double)t.N);
}

struct FinalArgs {
    const float2* map;
    const float* isig;
    BankParams bp;
    double f_min, df;
    int32_t norm, tau_mode, n_tau;
    const double* tau_d;       // device grid (grid mode)
    const Scalars* sc;
    const Cand* cand;
    uint32_t cand_cap;
    const WarpBest* warp_best;
    uint32_t n_warp_slots;
    DeviceResult* out;
};

// One block.  Near-max candidates (float32 SNR within the margin of the float32
// maximum) are re-scored in float64; the answer is the best under the G12 total
// order (larger SNR, then smaller template id, then smaller delay index).  If the
// candidate list overflowed (degenerate maps with massive ties) the per-warp
// float32 records decide instead and flags bit 0 is set.
__global__ void __launch_bounds__(256) k_finalize(const FinalArgs a)
{
    __shared__ double s_snr[8];
    __shared__ uint64_t s_id[8];
    __shared__ uint32_t s_m[8];
    __shared__ int s_valid[8];
    __shared__ float s_f32[8];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, n_warps = blockDim.x >> 5;
    const float gmax = dec_f32(a.sc->gmax_bits);
    const uint32_t n_cand = a.sc->cand_count < a.cand_cap ? a.sc->cand_count : a.cand_cap;
    const bool overflow = a.sc->overflow != 0 || a.sc->cand_count > a.cand_cap;
    double best = 0.0; uint64_t bid = 0; uint32_t bm = 0; int have = 0; float bf32 = 0.0f;
    int n_scored = 0;
    if (!overflow) {
        const float thr = gmax - near_margin(gmax);
        for (uint32_t i = warp; i < n_cand; i += n_warps) {
            const Cand c = a.cand[i];
            if (!(c.snr >= thr)) continue;
            const Track t = make_track(a.bp, c.id);
            const double tau = a.tau_mode == 0 ? a.tau_d[c.m] : t.tau;
            const double s = score_f64(a.map, a.isig, a.bp, a.f_min, a.df, t, tau, a.norm);
            ++n_scored;
            if (!have || s > best || (s == best && (c.id < bid || (c.id == bid && c.m < bm)))) {
                have = 1; best = s; bid = c.id; bm = c.m; bf32 = c.snr;
            }
        }
    } else {
        // float32 records: every lane scans a slice, warp-reduce, one re-score at the end
        float fs = -INFINITY; uint64_t fid = 0; uint32_t fm = 0; int fh = 0;
        for (uint32_t i = threadIdx.x; i < a.n_warp_slots; i += blockDim.x) {
            const WarpBest w = a.warp_best[i];
            if (w.valid && (!fh || better(w.snr, w.id, w.m, fs, fid, fm))) { fh = 1; fs = w.snr; fid = w.id; fm = w.m; }
        }
#pragma unroll
        for (int off = 16; off >= 1; off >>= 1) {
            const float os = __shfl_xor_sync(kFull, fs, off);
            const uint64_t oid = __shfl_xor_sync(kFull, fid, off);
            const uint32_t om = __shfl_xor_sync(kFull, fm, off);
            const int oh = __shfl_xor_sync(kFull, fh, off);
            if (oh && (!fh || better(os, oid, om, fs, fid, fm))) { fh = 1; fs = os; fid = oid; fm = om; }
        }
        // carried as (float32 snr promoted) so that the block reduce below keeps float32 order
        if (fh) { have = 1; best = (double)fs; bid = fid; bm = fm; bf32 = fs; }
    }
    if (lane == 0) { s_snr[warp] = best; s_id[warp] = bid; s_m[warp] = bm; s_valid[warp] = have; s_f32[warp] = bf32; }
    __shared__ int s_nscored[8];
    if (lane == 0) s_nscored[warp] = n_scored;
    __syncthreads();
    if (warp == 0) {
        have = 0;
        int total = 0;
        for (int w = 0; w < n_warps; ++w) {
            total += s_nscored[w];
            if (!s_valid[w]) continue;
            if (!have || s_snr[w] > best || (s_snr[w] == best && (s_id[w] < bid || (s_id[w] == bid && s_m[w] < bm)))) {
                have = 1; best = s_snr[w]; bid = s_id[w]; bm = s_m[w]; bf32 = s_f32[w];
            }
        }
        DeviceResult res;
        res.max_snr = gmax; res.arg_m = 0; res.snr_f64 = 0.0; res.arg_id = 0; res.arg_tau = 0.0;
        res.track.N = 0; res.track.j0 = 0; res.track.a = res.track.y0 = res.track.y1 = res.track.y2 = res.track.tau = res.track.y3 = 0.0;
        res.n_candidates = total; res.flags = overflow ? 1 : 0; res.n_pixels = a.sc->n_pixels;
        res.n_deferred = a.sc->n_deferred_total; res.pad = 0;
        if (have) {
            const Track t = make_track(a.bp, bid);
            const double tau = a.tau_mode == 0 ? a.tau_d[bm] : t.tau;
            const double s = overflow ? score_f64(a.map, a.isig, a.bp, a.f_min, a.df, t, tau, a.norm) : best;
            res.arg_m = (int32_t)bm; res.snr_f64 = s; res.arg_id = bid; res.arg_tau = tau; res.track = t;
            if (overflow) res.n_candidates = 1;
        }
        if (lane == 0) *a.out = res;
    }
}

// Float64 re-score of every captured candidate (top-K second pass): one warp per candidate at a time.
__global__ void __launch_bounds__(256) k_rescore_cands(const FinalArgs a, double* __restrict__ snr64)
{
    const int lane = threadIdx.x & 31;
    const uint32_t gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, n_w = (gridDim.x * blockDim.x) >> 5;
    const uint32_t n_cand = a.sc->cand_count < a.cand_cap ? a.sc->cand_count : a.cand_cap;
    for (uint32_t i = gw; i < n_cand; i += n_w) {
        const Cand c = a.cand[i];
        const Track t = make_track(a.bp, c.id);
        const double tau = a.tau_mode == 0 ? a.tau_d[c.m] : t.tau;
        const double s = score_f64(a.map, a.isig, a.bp, a.f_min, a.df, t, tau, a.norm);
        if (lane == 0) snr64[i] = s;
    }
}

// ------------------------------------------------------------- parity export --
// S1 + S2 for ids [first, first + count): k_out[q][c] (-1 beyond N), j0, N.
__global__ void k_debug_rasterise(BankParams bp, uint64_t first, uint64_t count, int32_t* __restrict__ k_out,
                                  int32_t* __restrict__ j0_out, int32_t* __restrict__ N_out)
{
    const int lane = threadIdx.x & 31;
    const uint64_t gw = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const uint64_t n_w = ((uint64_t)gridDim.x * blockDim.x) >> 5;
    for (uint64_t q = gw; q < count; q += n_w) {
        const Track t = make_track(bp, first + q);
        const Raster r = make_raster(t, bp.n_f, bp.family);
        int32_t* row = k_out + q * (uint64_t)bp.n_t;
        for (int c = lane; c < bp.n_t; c += kWarp) row[c] = c < t.N ? raster_bin_fast(r, c) : -1;
        if (lane == 0) { j0_out[q] = t.j0; N_out[q] = t.N; }
    }
}

__global__ void k_debug_rasterise_track(Track t, int32_t n_f, int32_t family, int32_t* __restrict__ k_out)
{
    const Raster r = make_raster(t, n_f, family);
    for (int c = blockIdx.x * blockDim.x + threadIdx.x; c < t.N; c += gridDim.x * blockDim.x)
        k_out[c] = raster_bin_fast(r, c);
}

}  // namespace st

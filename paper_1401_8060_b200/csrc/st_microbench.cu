// st_microbench.cu -- measures the unit peaks the score kernels are bounded by
// and that MEASURED_PEAKS.json does not hold:
//   FP32 pipe issue rate (FFMA, FADD, packed FFMA2), the Reinsch inner-loop pattern
//   at full occupancy, shared-memory gather bandwidth, MUFU, FP64 FMA / DIV / SQRT,
//   and random 8-byte gathers from an L2-resident buffer (sector bandwidth).
// Standalone: prints one JSON object per line.  Build: python -m paper_1401_8060_b200.build
#include <cuda_runtime.h>
#include <stdio.h>
#include <stdlib.h>
#include <stdint.h>

#define CK(x) do { cudaError_t e = (x); if (e != cudaSuccess) { fprintf(stderr, "%s: %s\n", #x, cudaGetErrorString(e)); exit(1); } } while (0)

constexpr int kIters = 4096;

template <int ILP>
__global__ void k_ffma(float* out, float a, float b)
{
    float x[ILP];
#pragma unroll
    for (int i = 0; i < ILP; ++i) x[i] = threadIdx.x * 1e-3f + i;
    for (int it = 0; it < kIters; ++it) {
#pragma unroll
        for (int i = 0; i < ILP; ++i) x[i] = fmaf(x[i], a, b);
    }
    float s = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s += x[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <int ILP>
__global__ void k_fadd(float* out, float a)
{
    float x[ILP];
#pragma unroll
    for (int i = 0; i < ILP; ++i) x[i] = threadIdx.x * 1e-3f + i;
    for (int it = 0; it < kIters; ++it) {
#pragma unroll
        for (int i = 0; i < ILP; ++i) x[i] = x[i] + a;
    }
    float s = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s += x[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// packed fma.rn.f32x2 (sm_100+): two FMAs per lane per instruction
template <int ILP>
__global__ void k_ffma2(float* out, float a, float b)
{
    unsigned long long x[ILP];
    unsigned long long aa, bb;
    asm volatile("mov.b64 %0, {%1, %1};" : "=l"(aa) : "f"(a));
    asm volatile("mov.b64 %0, {%1, %1};" : "=l"(bb) : "f"(b));
#pragma unroll
    for (int i = 0; i < ILP; ++i) {
        float f = threadIdx.x * 1e-3f + i;
        asm volatile("mov.b64 %0, {%1, %1};" : "=l"(x[i]) : "f"(f));
    }
    for (int it = 0; it < kIters; ++it) {
#pragma unroll
        for (int i = 0; i < ILP; ++i) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(x[i]) : "l"(aa), "l"(bb));
    }
    float s = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) {
        float lo, hi;
        asm volatile("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(x[i]));
        s += lo + hi;
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// The Reinsch inner loop: d = fma(-kappa, x, d); x += d; acc[i] += x, NCH chains.
template <int NCH>
__global__ void k_reinsch(float* out, float kappa)
{
    float acc[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) acc[i] = 0.f;
    float x[NCH], d[NCH];
#pragma unroll
    for (int c = 0; c < NCH; ++c) { x[c] = threadIdx.x * 1e-3f + c; d[c] = 1e-3f * c; }
    for (int it = 0; it < kIters / 32; ++it) {
#pragma unroll
        for (int i = 0; i < 32; ++i) {
#pragma unroll
            for (int c = 0; c < NCH; ++c) {
                acc[i] += x[c];
                d[c] = fmaf(-kappa, x[c], d[c]);
                x[c] += d[c];
            }
        }
    }
    float s = 0;
#pragma unroll
    for (int i = 0; i < 32; ++i) s += acc[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// The packed (f32x2) Reinsch inner loop exactly as k_score_reinsch issues it: per step and
// chain  acc[i] += x ; d = fma(-kappa, x, d) ; x += d  on register pairs, 32 packed accumulators.
typedef unsigned long long f32x2_t;
__device__ __forceinline__ f32x2_t pk_fma(f32x2_t a, f32x2_t b, f32x2_t c)
{ f32x2_t r; asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ f32x2_t pk_add(f32x2_t a, f32x2_t b)
{ f32x2_t r; asm volatile("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2_t pk_make(float lo, float hi)
{ f32x2_t r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ float pk_sum(f32x2_t a)
{ float lo, hi; asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a)); return lo + hi; }

__device__ __forceinline__ f32x2_t pk_fma_halves(f32x2_t a, f32x2_t b, f32x2_t c)
{
    f32x2_t r;
    asm volatile("{\n\t.reg .f32 al, ah, bl, bh, cl, ch;\n\t"
                 "mov.b64 {al, ah}, %1;\n\tmov.b64 {bl, bh}, %2;\n\tmov.b64 {cl, ch}, %3;\n\t"
                 "fma.rn.f32 cl, al, bl, cl;\n\tfma.rn.f32 ch, ah, bh, ch;\n\t"
                 "mov.b64 %0, {cl, ch};\n\t}" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}

template <int NCH, bool MIXED>
__global__ void k_reinsch_packed(float* out, float kappa)
{
    f32x2_t acc[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) acc[i] = 0ull;
    f32x2_t x[NCH], d[NCH], nk[NCH];
#pragma unroll
    for (int c = 0; c < NCH; ++c) {
        x[c] = pk_make(threadIdx.x * 1e-3f + c, threadIdx.x * 2e-3f + c);
        d[c] = pk_make(1e-3f * c, 2e-3f * c);
        nk[c] = pk_make(-kappa * (c + 1), -kappa * (c + 2));
    }
#pragma unroll 1
    for (int it = 0; it < kIters / 32; ++it) {
#pragma unroll
        for (int i = 0; i < 32; ++i) {
#pragma unroll
            for (int c = 0; c < NCH; ++c) acc[i] = pk_add(acc[i], x[c]);
#pragma unroll
            for (int c = 0; c < NCH; ++c) d[c] = MIXED ? pk_fma_halves(nk[c], x[c], d[c]) : pk_fma(nk[c], x[c], d[c]);
#pragma unroll
            for (int c = 0; c < NCH; ++c) x[c] = pk_add(x[c], d[c]);
        }
    }
    float s = 0;
#pragma unroll
    for (int i = 0; i < 32; ++i) s += pk_sum(acc[i]);
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// Variant M2: scalar FFMA on the halves, ONE packed add for x += d, scalar accumulators
// (NACC of them, both halves of a pair add into the same delay's accumulator).
template <int NPK, int NACC>
__global__ void k_reinsch_m2(float* out, float kappa)
{
    float acc[NACC];
#pragma unroll
    for (int i = 0; i < NACC; ++i) acc[i] = 0.f;
    f32x2_t x[NPK], d[NPK], nk[NPK];
#pragma unroll
    for (int c = 0; c < NPK; ++c) {
        x[c] = pk_make(threadIdx.x * 1e-3f + c, threadIdx.x * 2e-3f + c);
        d[c] = pk_make(1e-3f * c, 2e-3f * c);
        nk[c] = pk_make(-kappa * (c + 1), -kappa * (c + 2));
    }
#pragma unroll 1
    for (int it = 0; it < kIters / NACC; ++it) {
#pragma unroll
        for (int i = 0; i < NACC; ++i) {
#pragma unroll
            for (int c = 0; c < NPK; ++c) {
                float xl, xh;
                asm volatile("mov.b64 {%0, %1}, %2;" : "=f"(xl), "=f"(xh) : "l"(x[c]));
                acc[i] += xl;
                acc[i] += xh;
                d[c] = pk_fma_halves(nk[c], x[c], d[c]);
                x[c] = pk_add(x[c], d[c]);
            }
        }
    }
    float s = 0;
#pragma unroll
    for (int i = 0; i < NACC; ++i) s += acc[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// all-scalar with NACC accumulators and NCH independent pixels
template <int NCH, int NACC>
__global__ void k_reinsch_s(float* out, float kappa)
{
    float acc[NACC];
#pragma unroll
    for (int i = 0; i < NACC; ++i) acc[i] = 0.f;
    float x[NCH], d[NCH], nk[NCH];
#pragma unroll
    for (int c = 0; c < NCH; ++c) { x[c] = threadIdx.x * 1e-3f + c; d[c] = 1e-3f * c; nk[c] = -kappa * (c + 1); }
#pragma unroll 1
    for (int it = 0; it < kIters / NACC; ++it) {
#pragma unroll
        for (int i = 0; i < NACC; ++i) {
#pragma unroll
            for (int c = 0; c < NCH; ++c) {
                acc[i] += x[c];
                d[c] = fmaf(nk[c], x[c], d[c]);
                x[c] += d[c];
            }
        }
    }
    float s = 0;
#pragma unroll
    for (int i = 0; i < NACC; ++i) s += acc[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// packed add only, and packed fma with three distinct register-pair operands
template <int ILP>
__global__ void k_fadd2(float* out, float a)
{
    f32x2_t x[ILP], aa = pk_make(a, a);
#pragma unroll
    for (int i = 0; i < ILP; ++i) x[i] = pk_make(threadIdx.x * 1e-3f + i, 1.0f);
    for (int it = 0; it < kIters; ++it) {
#pragma unroll
        for (int i = 0; i < ILP; ++i) x[i] = pk_add(x[i], aa);
    }
    float s = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s += pk_sum(x[i]);
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
template <int ILP>
__global__ void k_ffma2_3op(float* out, float a)
{
    f32x2_t x[ILP], y[ILP], z[ILP];
#pragma unroll
    for (int i = 0; i < ILP; ++i) { x[i] = pk_make(threadIdx.x * 1e-3f + i, 1.0f); y[i] = pk_make(a + i, a); z[i] = pk_make(a, a * i); }
    for (int it = 0; it < kIters; ++it) {
#pragma unroll
        for (int i = 0; i < ILP; ++i) x[i] = pk_fma(y[i], z[i], x[i]);
    }
    float s = 0;
#pragma unroll
    for (int i = 0; i < ILP; ++i) s += pk_sum(x[i]);
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void k_mufu(float* out, float a)
{
    float x0 = threadIdx.x * 1e-3f, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3;
    for (int it = 0; it < kIters; ++it) {
        x0 = __sinf(x0); x1 = __cosf(x1); x2 = __sinf(x2); x3 = __cosf(x3);
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = x0 + x1 + x2 + x3 + a;
}

template <int OP>   // 0 DFMA, 1 DDIV, 2 DSQRT
__global__ void k_fp64(double* out, double a, double b)
{
    double x0 = 1.0 + threadIdx.x * 1e-3, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3;
    for (int it = 0; it < kIters / 4; ++it) {
        if (OP == 0) { x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b); }
        if (OP == 1) { x0 = __ddiv_rn(a, x0); x1 = __ddiv_rn(a, x1); x2 = __ddiv_rn(a, x2); x3 = __ddiv_rn(a, x3); }
        if (OP == 2) { x0 = __dsqrt_rn(x0 + a); x1 = __dsqrt_rn(x1 + a); x2 = __dsqrt_rn(x2 + a); x3 = __dsqrt_rn(x3 + a); }
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = x0 + x1 + x2 + x3;
}

// Shared-memory gather: every lane reads a pseudo-random BYTES-wide word of a table.
template <int BYTES>
__global__ void k_lds_gather(float* out, int n_words)
{
    extern __shared__ __align__(16) unsigned char sm[];
    float* tab = reinterpret_cast<float*>(sm);
    for (int i = threadIdx.x; i < n_words * (BYTES / 4); i += blockDim.x) tab[i] = i * 1e-6f;
    __syncthreads();
    uint32_t idx = threadIdx.x * 2654435761u + blockIdx.x;
    float s = 0;
    for (int it = 0; it < kIters; ++it) {
        idx = idx * 1664525u + 1013904223u;
        const uint32_t w = (idx >> 8) % (uint32_t)n_words;
        if (BYTES == 8) { const float2 v = reinterpret_cast<float2*>(tab)[w]; s += v.x + v.y; }
        else { const float4 v = reinterpret_cast<float4*>(tab)[w]; s += v.x + v.y + v.z + v.w; }
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// Random 8-byte gathers from an L2-resident buffer: one 32-byte sector each.
__global__ void k_l2_gather(const float2* __restrict__ buf, uint32_t n, float* out)
{
    uint32_t idx = (blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u;
    float s = 0;
    for (int it = 0; it < 1024; it += 4) {
        uint32_t i0 = idx * 1664525u + 1013904223u, i1 = i0 * 1664525u + 1013904223u;
        uint32_t i2 = i1 * 1664525u + 1013904223u, i3 = i2 * 1664525u + 1013904223u;
        idx = i3;
        const float2 a = __ldg(&buf[(i0 >> 4) % n]), b = __ldg(&buf[(i1 >> 4) % n]);
        const float2 c = __ldg(&buf[(i2 >> 4) % n]), d = __ldg(&buf[(i3 >> 4) % n]);
        s += a.x + b.y + c.x + d.y;
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// ---- the inner loop of k_score_cheb (stride 2, two pixels per lane, 32 packed accumulators):
// FORM 0: the recurrence as two scalar FFMAs on the halves of a register pair (round-1's first form);
// FORM 1: one packed fma.rn.f32x2 with the coefficient as FFMA2's scalar-broadcast operand and the
//         sign pattern ++-- (what the kernel uses now).  128 evaluations per lane per iteration.
__device__ __forceinline__ f32x2_t mb_cheb_scalar(float g, f32x2_t cur, f32x2_t prev)
{
    f32x2_t r;
    asm volatile("{\n\t.reg .f32 cl, ch, pl, ph;\n\tmov.b64 {cl, ch}, %2;\n\tmov.b64 {pl, ph}, %3;\n\t"
                 "neg.f32 pl, pl;\n\tneg.f32 ph, ph;\n\tfma.rn.f32 pl, %1, cl, pl;\n\tfma.rn.f32 ph, %1, ch, ph;\n\t"
                 "mov.b64 %0, {pl, ph};\n\t}" : "=l"(r) : "f"(g), "l"(cur), "l"(prev));
    return r;
}
__device__ __forceinline__ f32x2_t mb_cheb_packed(float g, f32x2_t cur, f32x2_t prev)
{
    f32x2_t r;
    asm volatile("{\n\t.reg .b64 gg;\n\tmov.b64 gg, {%1, %1};\n\tfma.rn.f32x2 %0, gg, %2, %3;\n\t}"
                 : "=l"(r) : "f"(g), "l"(cur), "l"(prev));
    return r;
}
template <int FORM>
__global__ void __launch_bounds__(512, 1) k_cheb_loop(float* out, int iters, float g)
{
    f32x2_t f2[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) f2[i] = 0ull;
    for (int it = 0; it < iters; ++it) {
        const float GA = g + 1e-6f * (threadIdx.x + it), GB = g - 1e-6f * (threadIdx.x + it);
        f32x2_t Ace = pk_make(1.f, .9f), Ape = pk_make(.8f, .95f), Aco = pk_make(.95f, .8f), Apo = pk_make(.9f, 1.f);
        f32x2_t Bce = pk_make(.5f, .4f), Bpe = pk_make(.3f, .45f), Bco = pk_make(.45f, .3f), Bpo = pk_make(.4f, .5f);
#pragma unroll
        for (int i = 0; i < 32; i += 4) {
            f2[i] = pk_add(f2[i], Ace); f2[i] = pk_add(f2[i], Bce);
            f2[i + 1] = pk_add(f2[i + 1], Aco); f2[i + 1] = pk_add(f2[i + 1], Bco);
            if (FORM == 0) {
                Ape = mb_cheb_scalar(GA, Ace, Ape); Bpe = mb_cheb_scalar(GB, Bce, Bpe);
                Apo = mb_cheb_scalar(GA, Aco, Apo); Bpo = mb_cheb_scalar(GB, Bco, Bpo);
            } else {
                Ape = mb_cheb_packed(GA, Ace, Ape); Bpe = mb_cheb_packed(GB, Bce, Bpe);
                Apo = mb_cheb_packed(GA, Aco, Apo); Bpo = mb_cheb_packed(GB, Bco, Bpo);
            }
            f2[i + 2] = pk_add(f2[i + 2], Ape); f2[i + 2] = pk_add(f2[i + 2], Bpe);
            f2[i + 3] = pk_add(f2[i + 3], Apo); f2[i + 3] = pk_add(f2[i + 3], Bpo);
            if (FORM == 0) {
                Ace = mb_cheb_scalar(GA, Ape, Ace); Bce = mb_cheb_scalar(GB, Bpe, Bce);
                Aco = mb_cheb_scalar(GA, Apo, Aco); Bco = mb_cheb_scalar(GB, Bpo, Bco);
            } else {
                Ace = mb_cheb_packed(-GA, Ape, Ace); Bce = mb_cheb_packed(-GB, Bpe, Bce);
                Aco = mb_cheb_packed(-GA, Apo, Aco); Bco = mb_cheb_packed(-GB, Bpo, Bco);
            }
        }
    }
    float s = 0;
#pragma unroll
    for (int i = 0; i < 32; ++i) s += pk_sum(f2[i]);
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <typename F>
float time_ms(F launch, int reps = 5)
{
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    launch(); launch();
    CK(cudaDeviceSynchronize());
    float best = 1e30f;
    for (int r = 0; r < reps; ++r) {
        CK(cudaEventRecord(e0));
        launch();
        CK(cudaEventRecord(e1));
        CK(cudaEventSynchronize(e1));
        float ms; CK(cudaEventElapsedTime(&ms, e0, e1));
        if (ms < best) best = ms;
    }
    CK(cudaGetLastError());
    return best;
}

int main()
{
    cudaDeviceProp prop;
    CK(cudaGetDeviceProperties(&prop, 0));
    int clock_khz = 0;
    CK(cudaDeviceGetAttribute(&clock_khz, cudaDevAttrClockRate, 0));
    const int n_sm = prop.multiProcessorCount;
    const double ghz = clock_khz * 1e-6;
    printf("{\"bench\": \"device\", \"name\": \"%s\", \"sms\": %d, \"max_clock_ghz\": %.3f, \"l2_bytes\": %d, \"smem_optin\": %zu}\n",
           prop.name, n_sm, ghz, prop.l2CacheSize, prop.sharedMemPerBlockOptin);
    float* out; CK(cudaMalloc(&out, (size_t)n_sm * 8 * 1024 * sizeof(double)));
    const int blocks = n_sm * 2, threads = 512;          // 1024 threads / SM
    const double lanes = (double)blocks * threads;
#define REPORT(name, ms, ops_per_lane, unit)                                                         \
    printf("{\"bench\": \"%s\", \"ms\": %.4f, \"rate_per_s\": %.4e, \"per_clk_per_sm_at_max_clock\": %.2f, \"unit\": \"%s\"}\n", \
           name, ms, lanes * (ops_per_lane) / (ms * 1e-3), lanes * (ops_per_lane) / (ms * 1e-3) / (n_sm * ghz * 1e9), unit)
    { float ms = time_ms([&] { k_ffma<8><<<blocks, threads>>>(out, 1.0001f, 1e-4f); }); REPORT("ffma_ilp8", ms, 8.0 * kIters, "FFMA lane-ops"); }
    { float ms = time_ms([&] { k_ffma<2><<<blocks, threads>>>(out, 1.0001f, 1e-4f); }); REPORT("ffma_ilp2", ms, 2.0 * kIters, "FFMA lane-ops"); }
    { float ms = time_ms([&] { k_fadd<8><<<blocks, threads>>>(out, 1e-4f); }); REPORT("fadd_ilp8", ms, 8.0 * kIters, "FADD lane-ops"); }
    { float ms = time_ms([&] { k_ffma2<8><<<blocks, threads>>>(out, 1.0001f, 1e-4f); }); REPORT("ffma2_ilp8", ms, 16.0 * kIters, "FMA lane-ops (packed x2)"); }
    { float ms = time_ms([&] { k_ffma2<4><<<blocks, threads>>>(out, 1.0001f, 1e-4f); }); REPORT("ffma2_ilp4", ms, 8.0 * kIters, "FMA lane-ops (packed x2)"); }
    { float ms = time_ms([&] { k_reinsch<1><<<blocks, threads>>>(out, 1e-3f); }); REPORT("reinsch_1chain_32w", ms, 1.0 * kIters, "evals (3 FP32 ops each)"); }
    { float ms = time_ms([&] { k_reinsch<2><<<blocks, threads>>>(out, 1e-3f); }); REPORT("reinsch_2chain_32w", ms, 2.0 * kIters, "evals (3 FP32 ops each)"); }
    { float ms = time_ms([&] { k_reinsch<4><<<blocks, threads>>>(out, 1e-3f); }); REPORT("reinsch_4chain_32w", ms, 4.0 * kIters, "evals (3 FP32 ops each)"); }
    {   // 16 warps per SM (the score kernel's occupancy)
        const double lanes16 = (double)n_sm * 512;
        float ms = time_ms([&] { k_reinsch<2><<<n_sm, 512>>>(out, 1e-3f); });
        printf("{\"bench\": \"reinsch_2chain_16w\", \"ms\": %.4f, \"per_clk_per_sm_at_max_clock\": %.2f, \"unit\": \"evals\"}\n", ms,
               lanes16 * 2.0 * kIters / (ms * 1e-3) / (n_sm * ghz * 1e9));
        ms = time_ms([&] { k_reinsch<1><<<n_sm, 512>>>(out, 1e-3f); });
        printf("{\"bench\": \"reinsch_1chain_16w\", \"ms\": %.4f, \"per_clk_per_sm_at_max_clock\": %.2f, \"unit\": \"evals\"}\n", ms,
               lanes16 * 1.0 * kIters / (ms * 1e-3) / (n_sm * ghz * 1e9));
        ms = time_ms([&] { k_reinsch<4><<<n_sm, 256>>>(out, 1e-3f); });
        printf("{\"bench\": \"reinsch_4chain_8w\", \"ms\": %.4f, \"per_clk_per_sm_at_max_clock\": %.2f, \"unit\": \"evals\"}\n", ms,
               (double)n_sm * 256 * 4.0 * kIters / (ms * 1e-3) / (n_sm * ghz * 1e9));
    }
    {   // packed Reinsch pattern at the score kernel's occupancy (16 warps / SM) and at 32 warps / SM
        for (int w = 16; w <= 32; w += 16) {
            const int thr = 512, blk = n_sm * (w / 16);
            const double ln = (double)blk * thr;
            float ms = time_ms([&] { k_reinsch_packed<1, true><<<blk, thr>>>(out, 1e-3f); });
            printf("{\"bench\": \"reinsch_mixed_1chain_%dw\", \"ms\": %.4f, \"per_clk_per_sm_at_max_clock\": %.2f, \"unit\": \"evals\"}\n", w, ms,
                   ln * 2.0 * kIters / (ms * 1e-3) / (n_sm * ghz * 1e9));
            ms = time_ms([&] { k_reinsch_packed<2, true><<<blk, thr>>>(out, 1e-3f); });
            printf("{\"bench\": \"reinsch_mixed_2chain_%dw\", \"ms\": %.4f, \"per_clk_per_sm_at_max_clock\": %.2f, \"unit\": \"evals\"}\n", w, ms,
                   ln * 4.0 * kIters / (ms * 1e-3) / (n_sm * ghz * 1e9));
            ms = time_ms([&] { k_reinsch_packed<1, false><<<blk, thr>>>(out, 1e-3f); });
            printf("{\"bench\": \"reinsch_packed_1chain_%dw\", \"ms\": %.4f, \"per_clk_per_sm_at_max_clock\": %.2f, \"unit\": \"evals\"}\n", w, ms,
                   ln * 2.0 * kIters / (ms * 1e-3) / (n_sm * ghz * 1e9));
            ms = time_ms([&] { k_reinsch_packed<2, false><<<blk, thr>>>(out, 1e-3f); });
            printf("{\"bench\": \"reinsch_packed_2chain_%dw\", \"ms\": %.4f, \"per_clk_per_sm_at_max_clock\": %.2f, \"unit\": \"evals\"}\n", w, ms,
                   ln * 4.0 * kIters / (ms * 1e-3) / (n_sm * ghz * 1e9));
        }
    }
    {
#define RUN16(name, kern, evals_per_iter)                                                              \
    { float ms = time_ms([&] { kern<<<n_sm, 512>>>(out, 1e-3f); });                                    \
      printf("{\"bench\": \"%s_16w\", \"ms\": %.4f, \"per_clk_per_sm_at_max_clock\": %.2f, \"unit\": \"evals\"}\n", name, ms, \
             (double)n_sm * 512 * (evals_per_iter) * kIters / (ms * 1e-3) / (n_sm * ghz * 1e9)); }
        RUN16("reinsch_m2_1pk_acc32", (k_reinsch_m2<1, 32>), 2.0)
        RUN16("reinsch_m2_2pk_acc32", (k_reinsch_m2<2, 32>), 4.0)
        RUN16("reinsch_m2_1pk_acc64", (k_reinsch_m2<1, 64>), 2.0)
        RUN16("reinsch_m2_2pk_acc64", (k_reinsch_m2<2, 64>), 4.0)
        RUN16("reinsch_s_2ch_acc32", (k_reinsch_s<2, 32>), 2.0)
        RUN16("reinsch_s_2ch_acc64", (k_reinsch_s<2, 64>), 2.0)
        RUN16("reinsch_s_4ch_acc64", (k_reinsch_s<4, 64>), 4.0)
        RUN16("reinsch_s_4ch_acc32", (k_reinsch_s<4, 32>), 4.0)
    }
    { float ms = time_ms([&] { k_fadd2<8><<<blocks, threads>>>(out, 1e-4f); }); REPORT("fadd2_ilp8", ms, 16.0 * kIters, "FADD lane-ops (packed x2)"); }
    { float ms = time_ms([&] { k_ffma2_3op<8><<<blocks, threads>>>(out, 1e-4f); }); REPORT("ffma2_3distinct_ilp8", ms, 16.0 * kIters, "FMA lane-ops (packed x2)"); }
    { float ms = time_ms([&] { k_mufu<<<blocks, threads>>>(out, 0.f); }); REPORT("mufu_sincos", ms, 4.0 * kIters, "MUFU lane-ops"); }
    { float ms = time_ms([&] { k_fp64<0><<<blocks, threads>>>((double*)out, 1.0000001, 1e-9); }); REPORT("dfma", ms, 1.0 * kIters, "DFMA lane-ops"); }
    { float ms = time_ms([&] { k_fp64<1><<<blocks, threads>>>((double*)out, 1.5, 0.0); }); REPORT("ddiv_rn", ms, 1.0 * kIters, "DDIV lane-ops"); }
    { float ms = time_ms([&] { k_fp64<2><<<blocks, threads>>>((double*)out, 1.5, 0.0); }); REPORT("dsqrt_rn", ms, 1.0 * kIters, "DSQRT lane-ops"); }
    {
        CK(cudaFuncSetAttribute(k_lds_gather<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024));
        CK(cudaFuncSetAttribute(k_lds_gather<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024));
        float ms = time_ms([&] { k_lds_gather<8><<<blocks, threads, 2461 * 8>>>(out, 2461); });
        REPORT("lds64_random_gather", ms, 8.0 * kIters, "bytes");
        ms = time_ms([&] { k_lds_gather<16><<<blocks, threads, 2461 * 16>>>(out, 2461); });
        REPORT("lds128_random_gather", ms, 16.0 * kIters, "bytes");
    }
    for (int thr = 256; thr <= 512; thr += 256) {
        const int iters = 20000;
        for (int form = 0; form < 2; ++form) {
            const float ms = form == 0 ? time_ms([&] { k_cheb_loop<0><<<n_sm, thr>>>(out, iters, 1.9f); })
                                       : time_ms([&] { k_cheb_loop<1><<<n_sm, thr>>>(out, iters, 1.9f); });
            printf("{\"bench\": \"cheb_loop_%s_%dw\", \"ms\": %.4f, \"per_clk_per_sm_at_max_clock\": %.2f, \"unit\": \"evals (1 FMA + 1 add each; 64 = FP32 pipe)\"}\n",
                   form == 0 ? "scalar_ffma" : "packed_ffma2", thr / 32, ms,
                   (double)n_sm * thr * iters * 128.0 / (ms * 1e-3) / (n_sm * ghz * 1e9));
        }
    }
    {
        const uint32_t n = 2461u * 1000u;                 // config-5 map: 19.7 MB, L2 resident
        float2* buf; CK(cudaMalloc(&buf, (size_t)n * sizeof(float2)));
        CK(cudaMemset(buf, 0, (size_t)n * sizeof(float2)));
        float ms = time_ms([&] { k_l2_gather<<<blocks * 4, 256>>>(buf, n, out); });
        const double gathers = (double)blocks * 4 * 256 * 1024;
        printf("{\"bench\": \"l2_random_8B_gather\", \"ms\": %.4f, \"gathers_per_s\": %.4e, \"sector_GBps\": %.1f, \"useful_GBps\": %.1f}\n",
               ms, gathers / (ms * 1e-3), gathers * 32 / (ms * 1e-3) * 1e-9, gathers * 8 / (ms * 1e-3) * 1e-9);
        CK(cudaFree(buf));
    }
    CK(cudaFree(out));
    return 0;
}

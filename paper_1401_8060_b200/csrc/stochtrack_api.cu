// stochtrack_api.cu -- the C ABI of include/stochtrack.h over the kernels of
// st_kernels.cuh.  Host logic only: validation, workspace layout, twiddle-table
// caching, kernel selection and launch, result copy-back.  No device memory is
// allocated here (the caller's workspace is carved up); the only allocations are
// a few KB of pinned host memory for results and two CUDA events per context.
#include <cuda_runtime.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>
#include <vector>
#include <algorithm>
#include <mutex>
#include <new>

#include "../../include/stochtrack.h"
#include "st_kernels.cuh"
#include "st_ftmap.cuh"

namespace {

constexpr size_t kAlign = 256;
constexpr uint32_t kCandCap = 1u << 16;
constexpr uint32_t kWarpSlots = 1u << 14;
constexpr uint64_t kMaxSamplesPerLaunch = 1ull << 31;   // keeps per-block u32 histogram bins exact
constexpr uint32_t kDeferCap = 1u << 22;                // templates per Chebyshev launch = size of its hand-over list

size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

struct Layout {
    size_t map, isig, e0, bintab, es, kz, ec, cheb, cheb_zi, w, tau, hist, scalars, result, cand, cand64, warp_best, stage_csd, stage_sigma, stage_csd2, stage_sigma2, b_scalars, b_result, b_hist, tracks, deferred, total;
};

Layout make_layout(int32_t n_t, int32_t n_f, int32_t max_n_tau)
{
    const size_t n_pix = (size_t)n_t * (size_t)n_f;
    Layout L;
    size_t o = 0;
    L.map = o;         o += align_up(n_pix * sizeof(float2));
    L.isig = o;        o += align_up(n_pix * sizeof(float));
    L.e0 = o;          o += align_up((size_t)n_f * sizeof(float2));
    L.bintab = o;      o += align_up((size_t)n_f * sizeof(float4));
    L.es = o;          o += align_up((size_t)n_f * (size_t)((max_n_tau + st::kSuper - 1) / st::kSuper) * sizeof(float2));
    L.kz = o;          o += align_up((size_t)n_f * sizeof(float2));
    L.ec = o;          o += align_up((size_t)n_f * sizeof(float2));
    L.cheb = o;        o += align_up((size_t)n_f * sizeof(float4));
    L.cheb_zi = o;     o += align_up((size_t)n_f * sizeof(float));
    L.w = o;           o += align_up((size_t)n_f * (size_t)max_n_tau * sizeof(float2));
    L.tau = o;         o += align_up((size_t)max_n_tau * sizeof(double));
    L.hist = o;        o += align_up((size_t)ST_MAX_BINS * sizeof(unsigned long long));
    L.scalars = o;     o += align_up(sizeof(st::Scalars));
    L.result = o;      o += align_up(sizeof(st::DeviceResult));
    L.cand = o;        o += align_up((size_t)kCandCap * sizeof(st::Cand));
    L.cand64 = o;      o += align_up((size_t)kCandCap * sizeof(double));
    L.warp_best = o;   o += align_up((size_t)kWarpSlots * sizeof(st::WarpBest));
    L.stage_csd = o;   o += align_up(n_pix * sizeof(float2));
    L.stage_sigma = o; o += align_up(n_pix * sizeof(float));
    // batch mode: second staging pair (copy of map m + 1 under the search of map m), per-map slots
    L.stage_csd2 = o;   o += align_up(n_pix * sizeof(float2));
    L.stage_sigma2 = o; o += align_up(n_pix * sizeof(float));
    L.b_scalars = o;    o += align_up((size_t)ST_BATCH_GROUP * sizeof(st::Scalars));
    L.b_result = o;     o += align_up((size_t)ST_BATCH_GROUP * sizeof(st::DeviceResult));
    L.b_hist = o;       o += align_up((size_t)ST_BATCH_GROUP * (size_t)ST_MAX_BINS * sizeof(unsigned long long));
    L.tracks = o;       o += align_up((size_t)ST_MAX_SCORE_TRACKS * sizeof(st::Track));
    L.deferred = o;     o += align_up((size_t)kDeferCap * sizeof(uint32_t));
    L.total = o;
    return L;
}

enum TableKind { kNoTable = 0, kWTable = 1, kRotTable = 2, kReinschTable = 3, kChebTable = 4 };

}  // namespace

struct st_ctx {
    int32_t n_t, n_f;
    double df, f_min;
    unsigned char* ws;
    size_t ws_bytes;
    int32_t max_n_tau;
    Layout L;
    cudaStream_t stream;
    bool have_ws, have_map;
    bool have_isig;                    // the 1 / sigma plane matches the map (set by st_set_map, not by the ft-map path)
    std::vector<double> tau_cached;    // grid currently on the device
    int table_kind, table_ch;          // which tables are currently built for tau_cached
    bool w_built;
    cudaEvent_t ev0, ev1;
    cudaStream_t copy_stream;          // batch mode: host-to-device copies of the next map
    cudaEvent_t ev_copied[2], ev_consumed[2];
    st::DeviceResult* h_bres;          // pinned, ST_BATCH_GROUP
    unsigned long long* h_bhist;       // pinned, ST_BATCH_GROUP x ST_MAX_BINS (allocated on first batch call)
    st::DeviceResult* h_res;           // pinned
    unsigned long long* h_hist;        // pinned, ST_MAX_BINS
    int n_sm, smem_optin;
    int device;                        // ordinal of the device the workspace lives on (every call runs there)
    int ev_device;                     // device the context's events (and batch stream) were created on, -1 = none yet
    int recur_threads;                 // tunable: threads per block of the recurrence kernels
    int cheb_stride;                   // stride of the tables currently on the device
    // bank cache (st_set_bank_cache): S1 + S2 of one template bank, reused by every search with the same bank
    unsigned char* bank; size_t bank_bytes; bool bank_valid;
    int last_bank_mode;                // what the last enqueued search did with it: 0 nothing, 1 filled, 2 read
    struct { uint64_t seed, offset, n_tracks; int32_t n_min, n_max; } bank_key;
    int cheb_n_class_b;                // class B bins of those tables
    double cheb_dmax;                  // largest Chebyshev drift among them [rad over half a chunk]
    bool pick_valid; double pick_dtau; int pick_stride;   // memo of cheb_pick_stride
    std::vector<float> h_cheb;         // host-built Chebyshev tables: [n_f] float4, [n_f] float2 Ec, [n_f] float zi
    char err[512];
};

namespace {

int fail(st_ctx* c, int code, const char* fmt, ...)
{
    if (c) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(c->err, sizeof(c->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

// Every device entry point runs on the workspace's device, whatever device is current in the calling thread.
struct DevGuard {
    int prev; bool switched;
    explicit DevGuard(const st_ctx* c) : prev(-1), switched(false) { if (c && c->have_ws) enter(c->device); }
    explicit DevGuard(int device) : prev(-1), switched(false) { enter(device); }     // before a context knows its device
    ~DevGuard() { if (switched) cudaSetDevice(prev); }
private:
    void enter(int device)
    {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != device) switched = cudaSetDevice(device) == cudaSuccess;
    }
};

#define ST_CUDA(ctx, call)                                                                   \
    do {                                                                                     \
        cudaError_t e_ = (call);                                                             \
        if (e_ != cudaSuccess)                                                               \
            return fail((ctx), ST_ECUDA, "%s: %s", #call, cudaGetErrorString(e_));           \
    } while (0)

template <typename T>
T* at(st_ctx* c, size_t off) { return reinterpret_cast<T*>(c->ws + off); }

st::BankParams bank(const st_ctx* c, const st_search_params* p)
{
    st::BankParams bp;
    bp.seed = p->seed;
    bp.n_t = c->n_t; bp.n_f = c->n_f; bp.n_min = p->n_min; bp.n_max = p->n_max;
    bp.tau_lo = p->tau_mode == ST_TAU_RANDOM ? p->tau_lo : 0.0;
    bp.tau_hi = p->tau_mode == ST_TAU_RANDOM ? p->tau_hi : 0.0;
    bp.family = p->family; bp.pad = 0;
    return bp;
}

int validate(st_ctx* c, const st_search_params* p, bool need_map)
{
    if (!c) return ST_EINVAL;
    if (!p) return fail(c, ST_EINVAL, "params is NULL");
    if (!c->have_ws) return fail(c, ST_ESTATE, "no workspace: call st_set_workspace first");
    if (need_map && !c->have_map) return fail(c, ST_ESTATE, "no map: call st_set_map first");
    if (p->n_min < 1 || p->n_max < p->n_min || p->n_max > c->n_t)
        return fail(c, ST_EINVAL, "need 1 <= n_min <= n_max <= n_t (got %d, %d, n_t %d)", p->n_min, p->n_max, c->n_t);
    if (p->tau_mode != ST_TAU_GRID && p->tau_mode != ST_TAU_RANDOM) return fail(c, ST_EINVAL, "bad tau_mode %d", p->tau_mode);
    if (p->tau_mode == ST_TAU_GRID) {
        if (p->n_tau < 1 || p->n_tau > ST_MAX_N_TAU) return fail(c, ST_EINVAL, "n_tau %d outside [1, %d]", p->n_tau, ST_MAX_N_TAU);
        if (p->n_tau > c->max_n_tau) return fail(c, ST_ENOSPC, "n_tau %d exceeds the workspace's max_n_tau %d", p->n_tau, c->max_n_tau);
        if (!p->tau_grid) return fail(c, ST_EINVAL, "tau_grid is NULL");
        for (int m = 0; m < p->n_tau; ++m)
            if (!isfinite(p->tau_grid[m])) return fail(c, ST_EINVAL, "tau_grid[%d] is not finite", m);
    } else {
        if (!isfinite(p->tau_lo) || !isfinite(p->tau_hi) || p->tau_hi < p->tau_lo)
            return fail(c, ST_EINVAL, "bad random-tau range");
    }
    if (p->norm != ST_NORM_SQRT_N && p->norm != ST_NORM_MEAN && p->norm != ST_NORM_INVVAR) return fail(c, ST_EINVAL, "bad norm %d", p->norm);
    if (p->norm == ST_NORM_INVVAR && need_map && !c->have_isig)
        return fail(c, ST_ESTATE, "ST_NORM_INVVAR needs sigma: set the map through st_set_map / st_set_map_host / st_search_batch");
    if (p->family != ST_FAMILY_QUADRATIC && p->family != ST_FAMILY_CUBIC && p->family != ST_FAMILY_CHIRP) return fail(c, ST_EINVAL, "bad template family %d", p->family);
    if (p->n_bins < 0 || p->n_bins > ST_MAX_BINS) return fail(c, ST_EINVAL, "n_bins %d outside [0, %d]", p->n_bins, ST_MAX_BINS);
    if (p->n_bins > 0 && !(p->hist_hi > p->hist_lo)) return fail(c, ST_EINVAL, "need hist_hi > hist_lo");
    if (p->kernel < ST_KERNEL_AUTO || p->kernel > ST_KERNEL_CHEBYSHEV || p->kernel == ST_KERNEL_RANDOM)
        return fail(c, ST_EINVAL, "bad kernel %d", p->kernel);
    if (p->n_tracks > (1ull << 62) || p->track_offset > (1ull << 62)) return fail(c, ST_EINVAL, "n_tracks / track_offset too large");
    return ST_OK;
}

// Is the grid tau_0 + m * dtau to within a phase error of 1e-8 rad at the top of the band?
bool grid_uniform(const st_ctx* c, const double* tau, int n, double* tau0, double* dtau)
{
    *tau0 = tau[0];
    *dtau = n > 1 ? (tau[n - 1] - tau[0]) / (double)(n - 1) : 0.0;
    const double f_top = c->f_min + c->df * (double)(c->n_f - 1);
    const double tol = 1e-8 / (st::kTwoPi * (f_top > 1.0 ? f_top : 1.0));
    for (int m = 0; m < n; ++m)
        if (fabs(tau[m] - (*tau0 + (double)m * *dtau)) > tol) return false;
    return true;
}

// The three-term recurrence amplifies rounding by 1/|sin theta|: refuse it when a
// bin's step angle theta_k = 2 pi f_k dtau (mod 2 pi) comes within 0.1 rad of pi.
bool reinsch_well_conditioned(const st_ctx* c, double dtau)
{
    for (int k = 0; k < c->n_f; ++k) {
        double cyc = (c->f_min + (double)k * c->df) * dtau;
        cyc -= rint(cyc);                               // [-1/2, 1/2]
        if (0.5 - fabs(cyc) < 0.1 / st::kTwoPi) return false;
    }
    return true;
}

// Chebyshev tables for stride S (built on the host so that the conditioning test sees the very float32
// coefficients the kernel uses).  The coefficient G = fl32(2 cos(S theta)) is the exact coefficient of a slightly
// different angle; over the 32 delays between an anchor and the edge of its chunk the phase drifts by
// (32 / S) |acos(G/2) - S theta|.  A coherent signal of amplitude A (in SNR units) is then mis-scored by up to
// A x drift where SNR(tau) crosses zero, against an absolute tolerance of 1e-4 s0 there (G13): bins whose drift
// exceeds kChebClassDrift become CLASS B; the general build of the kernel advances them by Reinsch's form
// (coefficient kappa = 4 sin^2(theta/2), relative precision kept as theta -> 0), the fast build scores a template
// itself only when its amplitude in class B bins bounds the drift error below kChebDeferBudget (launch_score).
// Returns the number of class B bins, or -1 when some bin suits neither form (then the grid goes to the rotation
// kernel).  Table per bin: (G, cos theta, sin theta, cos 64 theta), Ec = anchor phase factor of chunk 0 with the
// class in the lowest mantissa bit of its real part, zi = sin 64 theta.
constexpr double kChebClassDrift = 3e-6;   // rad over half a chunk: A = 16 stays inside half the G13 tolerance

int build_cheb_tables(const st_ctx* c, double tau0, double dtau, int stride, std::vector<float>* out, double* d_max = nullptr)
{
    const int n_f = c->n_f;
    if (out) out->assign((size_t)n_f * 7, 0.0f);
    int n_class_b = 0;
    double dmax = 0.0;
    std::vector<double> drift((size_t)n_f, 0.0);        // class B bins: their drift over half a chunk (0 = class A)
    for (int k = 0; k < n_f; ++k) {
        const double f = c->f_min + (double)k * c->df;
        double cyc = f * dtau;
        cyc -= rint(cyc);                                   // theta / 2 pi in [-1/2, 1/2]
        const double theta = st::kTwoPi * cyc;
        double sth = (double)stride * theta;                // S theta reduced to (-pi, pi]
        sth -= st::kTwoPi * rint(sth / st::kTwoPi);
        const float G = (float)(2.0 * cos(sth));
        double half = 0.5 * (double)G;
        half = half > 1.0 ? 1.0 : (half < -1.0 ? -1.0 : half);
        const double drift_a = (32.0 / (double)stride) * fabs(acos(half) - fabs(sth));
        if (drift_a > kChebClassDrift) {
            // Reinsch's form at stride 1 with kappa = 2 sin^2 theta / (1 + cos theta) formed in float32 from the
            // table's (cos theta, sin theta): relative error <= 3e-7, i.e. <= 32 x 1.5e-7 |theta| rad of drift
            const double drift_b = 4.8e-6 * fabs(theta);
            if (drift_b > kChebClassDrift) return -1;
            ++n_class_b;
            drift[(size_t)k] = drift_a;
            if (drift_a > dmax) dmax = drift_a;
        }
        if (out) {
            double c64 = cyc * 64.0;
            c64 -= rint(c64);
            double c0 = f * (tau0 + 32.0 * dtau);
            c0 -= rint(c0);
            float* t4 = out->data() + (size_t)k * 4;
            t4[0] = G; t4[1] = (float)cos(theta); t4[2] = (float)sin(theta); t4[3] = (float)cos(st::kTwoPi * c64);
            float* ec = out->data() + (size_t)n_f * 4 + (size_t)k * 2;
            ec[0] = (float)cos(st::kTwoPi * c0); ec[1] = (float)sin(st::kTwoPi * c0);
            (*out)[(size_t)n_f * 6 + (size_t)k] = (float)sin(st::kTwoPi * c64);
        }
    }
    if (d_max) *d_max = dmax;
    if (out) {
        // The class rides in the two lowest mantissa bits of Ec.x: 0 = class A; 1, 2, 3 = class B with a drift of at most
        // d_max / 4, d_max / 2, d_max: the fast build weighs a pixel's amplitude by 2^(level - 3) x 2 in its bound of
        // the drift error, so the many mildly drifting bins do not count as the worst one.
        for (int k = 0; k < n_f; ++k) {
            float* ec = out->data() + (size_t)n_f * 4 + (size_t)k * 2;
            const double d = drift[(size_t)k];
            const uint32_t level = d == 0.0 ? 0u : (d <= 0.25 * dmax ? 1u : (d <= 0.5 * dmax ? 2u : 3u));
            uint32_t bits;
            memcpy(&bits, &ec[0], sizeof(bits));
            bits = (bits & ~3u) | level;
            memcpy(&ec[0], &bits, sizeof(bits));
        }
    }
    return n_class_b;
}

// Stride 2 needs 2 theta inside (0, pi) for every bin; of the usable strides take the one with fewer class B
// bins (their rows cost 3 packed operations per 2 evaluations instead of 2), stride 2 on a tie (more independent
// chains per pixel).  0 = the Chebyshev kernel does not suit this grid.
int cheb_pick_stride(st_ctx* c, double dtau)
{
    if (c->pick_valid && c->pick_dtau == dtau) return c->pick_stride;
    double max_abs_cyc = 0.0;
    for (int k = 0; k < c->n_f; ++k) {
        double cyc = (c->f_min + (double)k * c->df) * dtau;
        cyc -= rint(cyc);
        if (fabs(cyc) > max_abs_cyc) max_abs_cyc = fabs(cyc);
    }
    const int b1 = build_cheb_tables(c, 0.0, dtau, 1, nullptr);
    const int b2 = max_abs_cyc < 0.22 ? build_cheb_tables(c, 0.0, dtau, 2, nullptr) : -1;
    int s = 0;
    if (b1 >= 0 && b2 >= 0) s = b2 <= b1 ? 2 : 1;
    else if (b2 >= 0) s = 2;
    else if (b1 >= 0) s = 1;
    c->pick_valid = true; c->pick_dtau = dtau; c->pick_stride = s;
    return s;
}

int pick_chunk(int n_tau)
{
    const int pad32 = (n_tau + 31) / 32 * 32, pad64 = (n_tau + 63) / 64 * 64;
    return pad32 < pad64 ? 32 : 64;
}

struct Plan {
    int kernel;       // ST_KERNEL_*
    int ch;           // recurrence chunk
    int stride;       // Chebyshev stride (1 or 2)
    double tau0, dtau;
};

// Shared memory a recurrence kernel needs with `warps` warps: histogram + per-bin tables + pixel pools.
// AUTO only picks a kernel that keeps at least 4 warps per SM (wide bands: the per-bin tables of the
// Chebyshev / Reinsch kernels outgrow shared memory, the rotation kernel then reads its table from L2).
// Pool entries per warp of the Chebyshev kernel: class A rows from the front, class B rows from the back, each
// zero-filled to whole rows of 32 (ceil32(a) + ceil32(b) <= ceil32(a + b) + 32).
int cheb_pool_stride(int n_max) { return ((n_max + 31) & ~31) + 32; }

bool recur_fits(const st_ctx* c, int kernel, int n_bins, int n_max, int warps)
{
    const size_t stride = kernel == ST_KERNEL_CHEBYSHEV ? (size_t)cheb_pool_stride(n_max) : (size_t)((n_max + 63) & ~63);
    const size_t hist = (size_t)((n_bins + 3) & ~3) * sizeof(uint32_t);
    size_t need = hist;
    if (kernel == ST_KERNEL_CHEBYSHEV)
        need += (size_t)c->n_f * sizeof(float4) + (size_t)((c->n_f + 1) & ~1) * sizeof(float) + (size_t)warps * stride * 10;
    else if (kernel == ST_KERNEL_REINSCH)
        need += (size_t)(c->n_f + (c->n_f & 1)) * sizeof(float2) + (size_t)warps * (stride / 2) * 20;
    else
        need += (size_t)warps * stride * 10;
    return need <= (size_t)c->smem_optin;
}

int make_plan(st_ctx* c, const st_search_params* p, Plan* plan)
{
    plan->ch = 0; plan->tau0 = 0.0; plan->dtau = 0.0; plan->stride = 0;
    if (p->tau_mode == ST_TAU_RANDOM) { plan->kernel = ST_KERNEL_RANDOM; return ST_OK; }
    const bool uni = grid_uniform(c, p->tau_grid, p->n_tau, &plan->tau0, &plan->dtau);
    int k = p->kernel;
    if (k == ST_KERNEL_AUTO) {
        if (!uni || p->n_tau < 8) k = ST_KERNEL_TABLE;
        else if (recur_fits(c, ST_KERNEL_CHEBYSHEV, p->n_bins, p->n_max, 4) &&
                 (plan->stride = cheb_pick_stride(c, plan->dtau)) != 0) k = ST_KERNEL_CHEBYSHEV;
        else if (recur_fits(c, ST_KERNEL_REINSCH, p->n_bins, p->n_max, 4) && reinsch_well_conditioned(c, plan->dtau))
            k = ST_KERNEL_REINSCH;
        else k = ST_KERNEL_ROTATION;
        if (k != ST_KERNEL_TABLE) plan->stride = k == ST_KERNEL_CHEBYSHEV ? plan->stride : 0;
    }
    if (k == ST_KERNEL_CHEBYSHEV && plan->stride == 0) {
        if (uni) plan->stride = cheb_pick_stride(c, plan->dtau);
        if (uni && plan->stride == 0)
            return fail(c, ST_EINVAL, "the Chebyshev kernel is ill conditioned on this delay grid (a bin suits neither recurrence within %.1e rad)", kChebClassDrift);
    }
    if ((k == ST_KERNEL_ROTATION || k == ST_KERNEL_REINSCH || k == ST_KERNEL_CHEBYSHEV) && !uni)
        return fail(c, ST_EINVAL, "recurrence kernels need a uniform tau grid");
    if (k == ST_KERNEL_REINSCH && p->kernel == ST_KERNEL_REINSCH && !reinsch_well_conditioned(c, plan->dtau))
        return fail(c, ST_EINVAL, "the Reinsch kernel is ill conditioned on this delay grid (a bin's step angle is within 0.1 rad of pi)");
    plan->kernel = k;
    if (k == ST_KERNEL_ROTATION) plan->ch = pick_chunk(p->n_tau);
    if (k == ST_KERNEL_REINSCH) plan->ch = st::kChunk;
    if (k == ST_KERNEL_CHEBYSHEV) plan->ch = st::kCheb;
    return ST_OK;
}

// Upload the grid and (re)build whichever twiddle tables the plan needs.
int ensure_tables(st_ctx* c, const st_search_params* p, const Plan& plan, int* n_launches)
{
    if (p->tau_mode != ST_TAU_GRID) return ST_OK;
    const bool same_grid = (int)c->tau_cached.size() == p->n_tau &&
                           memcmp(c->tau_cached.data(), p->tau_grid, sizeof(double) * (size_t)p->n_tau) == 0;
    if (!same_grid) {
        c->tau_cached.assign(p->tau_grid, p->tau_grid + p->n_tau);
        c->table_kind = kNoTable; c->w_built = false;
        ST_CUDA(c, cudaMemcpyAsync(at<double>(c, c->L.tau), c->tau_cached.data(), sizeof(double) * (size_t)p->n_tau,
                                   cudaMemcpyHostToDevice, c->stream));
    }
    if (plan.kernel == ST_KERNEL_TABLE) {
        if (!c->w_built) {
            const size_t n = (size_t)c->n_f * (size_t)p->n_tau;
            const int blocks = (int)((n + 255) / 256 < 4096 ? (n + 255) / 256 : 4096);
            st::k_build_w_table<<<blocks, 256, 0, c->stream>>>(at<double>(c, c->L.tau), p->n_tau, c->n_f, c->f_min, c->df,
                                                                at<float2>(c, c->L.w));
            ST_CUDA(c, cudaGetLastError());
            c->w_built = true; ++*n_launches;
        }
    } else if (plan.kernel == ST_KERNEL_ROTATION) {
        if (c->table_kind != kRotTable || c->table_ch != plan.ch) {
            st::k_build_bin_tables<<<(c->n_f + 127) / 128, 128, 0, c->stream>>>(
                plan.tau0, plan.dtau, plan.ch, 0, c->n_f, c->f_min, c->df,
                at<float2>(c, c->L.e0), at<float4>(c, c->L.bintab));
            ST_CUDA(c, cudaGetLastError());
            c->table_kind = kRotTable; c->table_ch = plan.ch; ++*n_launches;
        }
    } else if (plan.kernel == ST_KERNEL_CHEBYSHEV) {
        if (c->table_kind != kChebTable || c->cheb_stride != plan.stride) {
            c->cheb_n_class_b = build_cheb_tables(c, plan.tau0, plan.dtau, plan.stride, &c->h_cheb, &c->cheb_dmax);
            const size_t n = (size_t)c->n_f;
            ST_CUDA(c, cudaMemcpyAsync(at<void>(c, c->L.cheb), c->h_cheb.data(), n * 4 * sizeof(float), cudaMemcpyHostToDevice, c->stream));
            ST_CUDA(c, cudaMemcpyAsync(at<void>(c, c->L.ec), c->h_cheb.data() + n * 4, n * 2 * sizeof(float), cudaMemcpyHostToDevice, c->stream));
            ST_CUDA(c, cudaMemcpyAsync(at<void>(c, c->L.cheb_zi), c->h_cheb.data() + n * 6, n * sizeof(float), cudaMemcpyHostToDevice, c->stream));
            c->table_kind = kChebTable; c->table_ch = plan.ch; c->cheb_stride = plan.stride;
        }
    } else {
        if (c->table_kind != kReinschTable) {
            const int n_super = (p->n_tau + st::kSuper - 1) / st::kSuper;
            st::k_build_reinsch_tables<<<(c->n_f + 127) / 128, 128, 0, c->stream>>>(
                plan.tau0, plan.dtau, st::kSuper, n_super, c->n_f, c->f_min, c->df,
                at<float2>(c, c->L.es), at<float2>(c, c->L.kz));
            ST_CUDA(c, cudaGetLastError());
            c->table_kind = kReinschTable; c->table_ch = plan.ch; ++*n_launches;
        }
    }
    return ST_OK;
}

template <typename K>
int set_smem(st_ctx* c, K kernel, size_t bytes)
{
    if (bytes > 48 * 1024)
        ST_CUDA(c, cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    return ST_OK;
}

size_t hist_bytes(int n_bins) { return (size_t)((n_bins + 3) & ~3) * sizeof(uint32_t); }

// Launch the scoring kernel of the plan on templates [a.track_offset, +a.n_tracks).
// Bank cache layout: [n_tracks] (N, j0) records, then per template 32 lanes x ceil4(ceil(n_max / 32)) uint16 bins.
uint32_t bank_row_entries(int n_max) { return 32u * (uint32_t)((((n_max + 31) >> 5) + 3) & ~3); }
size_t bank_bytes_for(uint64_t n_tracks, int n_max)
{
    return align_up((size_t)n_tracks * sizeof(int2)) + align_up((size_t)n_tracks * (size_t)bank_row_entries(n_max) * sizeof(uint16_t));
}

// Absolute error (in SNR units) the fast Chebyshev build may owe to coefficient drift in class B bins: half the
// G13 tolerance at a zero crossing of SNR(tau) on the configs' data (1e-4 x s0, s0 = 0.707).  Class A bins add
// at most kChebClassDrift x A for a coherent amplitude A (3e-5 at SNR 10).
constexpr double kChebDeferBudget = 3.5e-5;

int launch_score(st_ctx* c, const Plan& plan, st::ScoreArgs& a, int n_max, int* extra_launches = nullptr)
{
    const int stride = (n_max + 63) & ~63;
    a.pool_stride = stride;
    const uint64_t want_warps = a.n_tracks;
    ST_CUDA(c, cudaMemsetAsync(&a.sc->counter, 0, sizeof(unsigned long long), c->stream));
    if (plan.kernel == ST_KERNEL_RANDOM) {
        const int threads = 256;
        const size_t smem = hist_bytes(a.n_bins);
        uint64_t blocks = (uint64_t)c->n_sm * 8;
        const uint64_t need = ((want_warps + st::kRandPerWarp - 1) / st::kRandPerWarp + 7) / 8;   // a warp scores kRandPerWarp templates at a time
        if (blocks > need) blocks = need;
        if (blocks > kWarpSlots / 8) blocks = kWarpSlots / 8;         // one per-warp record slot per resident warp
        const bool gen = a.bp.family != 0 || a.norm == 2 || a.tracks != nullptr;
        if (a.k_dump) {
            if (gen) st::k_score_random<false, true, true><<<(unsigned)blocks, threads, smem, c->stream>>>(a);
            else st::k_score_random<false, true, false><<<(unsigned)blocks, threads, smem, c->stream>>>(a);
        } else if (a.capture_mode) {
            if (gen) st::k_score_random<true, false, true><<<(unsigned)blocks, threads, smem, c->stream>>>(a);
            else st::k_score_random<true, false, false><<<(unsigned)blocks, threads, smem, c->stream>>>(a);
        } else {
            if (gen) st::k_score_random<false, false, true><<<(unsigned)blocks, threads, smem, c->stream>>>(a);
            else st::k_score_random<false, false, false><<<(unsigned)blocks, threads, smem, c->stream>>>(a);
        }
    } else if (plan.kernel == ST_KERNEL_TABLE) {
        int threads = 256;
        size_t smem;
        for (;; threads -= 32) {
            smem = hist_bytes(a.n_bins) + (size_t)(threads / 32) * (size_t)stride * (sizeof(float2) + sizeof(uint16_t));
            if (smem <= (size_t)c->smem_optin || threads == 32) break;
        }
        if (smem > (size_t)c->smem_optin) return fail(c, ST_ENOSPC, "n_max %d needs more shared memory than one SM has", n_max);
        int rc = set_smem(c, st::k_score_table, smem);
        if (rc) return rc;
        int per_sm = (int)((size_t)c->smem_optin / (smem + 1024));
        per_sm = per_sm < 1 ? 1 : (per_sm > 8 ? 8 : per_sm);
        uint64_t blocks = (uint64_t)c->n_sm * (uint64_t)per_sm;
        const uint64_t need = (want_warps + (uint64_t)(threads / 32) - 1) / (uint64_t)(threads / 32);
        if (blocks > need) blocks = need;
        if (blocks > kWarpSlots / (uint64_t)(threads / 32)) blocks = kWarpSlots / (uint64_t)(threads / 32);
        st::k_score_table<<<(unsigned)blocks, threads, smem, c->stream>>>(a);
    } else if (plan.kernel == ST_KERNEL_CHEBYSHEV) {
        int threads = c->recur_threads;
        size_t smem;
        const int cstride = cheb_pool_stride(n_max);
        a.pool_stride = cstride;
        for (;; threads -= 32) {
            smem = hist_bytes(a.n_bins) + (size_t)c->n_f * sizeof(float4) + (size_t)((c->n_f + 1) & ~1) * sizeof(float) +
                   (size_t)(threads / 32) * (size_t)cstride * (sizeof(float2) + sizeof(uint16_t));
            if (smem <= (size_t)c->smem_optin || threads == 32) break;
        }
        if (smem > (size_t)c->smem_optin)
            return fail(c, ST_ENOSPC, "n_f %d / n_max %d need more shared memory than one SM has", c->n_f, n_max);
        // Phase B form (st_kernels.cuh): grids of two or more chunks take the delay-split form (two chunks per pass);
        // which form runs is a property of the grid alone, so every build of the kernel (search, capture, per-template
        // maximum, general, bank cache) sums a template's terms in the same order.  The default search of a grid of
        // at most two chunks has a one-pass build, with the fold through shared memory when the scratch fits.
        const int n_chunks = (a.n_tau + st::kCheb - 1) / st::kCheb;
        const int pb = n_chunks >= 2 ? 1 : 0;
        int pb_single = pb;
        a.fold_offset = 0;
        // the one-pass search build is compiled for ST_CHEB_PIPE_THREADS threads (12 warps at 168 registers:
        // its phase B is software-pipelined, see cheb_phase_b_split)
        const bool one_pass_search = pb && n_chunks <= 2 && !a.capture_mode && !a.tmax_snr &&
                                     a.bp.family == 0 && a.norm != 2 && a.tracks == nullptr;
        if (one_pass_search && threads > ST_CHEB_PIPE_THREADS) {
            threads = ST_CHEB_PIPE_THREADS;
            smem = hist_bytes(a.n_bins) + (size_t)c->n_f * sizeof(float4) + (size_t)((c->n_f + 1) & ~1) * sizeof(float) +
                   (size_t)(threads / 32) * (size_t)cstride * (sizeof(float2) + sizeof(uint16_t));
        }
        if (pb && n_chunks <= 2) {
            pb_single = 3;
            const size_t fold_off = (smem + 15) & ~(size_t)15;
            const size_t with_fold = fold_off + (size_t)(threads / 32) * (size_t)st::kFoldWords * sizeof(float);
            if (with_fold <= (size_t)c->smem_optin) { smem = with_fold; a.fold_offset = (uint32_t)fold_off; pb_single = 4; }
        }
        const bool pk = plan.stride == 2;
        uint64_t blocks = (uint64_t)c->n_sm;            // persistent: one block per SM
        const uint64_t need = (want_warps + (uint64_t)(threads / 32) - 1) / (uint64_t)(threads / 32);
        if (blocks > need) blocks = need;
#define ST_LAUNCH_CHEB(STRIDE, MODE, GEN, BANK, PB)                                               \
    do {                                                                                          \
        int rc_ = set_smem(c, st::k_score_cheb<STRIDE, MODE, GEN, BANK, PB>, smem);               \
        if (rc_) return rc_;                                                                      \
        st::k_score_cheb<STRIDE, MODE, GEN, BANK, PB><<<(unsigned)blocks, threads, smem, c->stream>>>(a); \
    } while (0)
#define ST_LAUNCH_CHEB_FORM(STRIDE, MODE, GEN, BANK)                                              \
    do {                                                                                          \
        if (pb_ == 0) ST_LAUNCH_CHEB(STRIDE, MODE, GEN, BANK, 0);                                 \
        else ST_LAUNCH_CHEB(STRIDE, MODE, GEN, BANK, 1);                                          \
    } while (0)
#define ST_LAUNCH_CHEB_PIPE(STRIDE, BANK, PB)                                                     \
    do {                                                                                          \
        int rc_ = set_smem(c, st::k_score_cheb<STRIDE, 0, false, BANK, PB, true>, smem);          \
        if (rc_) return rc_;                                                                      \
        st::k_score_cheb<STRIDE, 0, false, BANK, PB, true><<<(unsigned)blocks, threads, smem, c->stream>>>(a); \
    } while (0)
#define ST_LAUNCH_CHEB_SEARCH(STRIDE, BANK)                                                       \
    do {                                                                                          \
        if (pb_ == 3) ST_LAUNCH_CHEB_PIPE(STRIDE, BANK, 3);                                       \
        else if (pb_ == 4) ST_LAUNCH_CHEB_PIPE(STRIDE, BANK, 4);                                  \
        else ST_LAUNCH_CHEB_FORM(STRIDE, 0, false, BANK);                                         \
    } while (0)
#define ST_LAUNCH_CHEB_MODE(STRIDE, GEN)                                                          \
    do {                                                                                          \
        if (mode == 1) ST_LAUNCH_CHEB_FORM(STRIDE, 1, GEN, 0);                                    \
        else if (mode == 2) ST_LAUNCH_CHEB_FORM(STRIDE, 2, GEN, 0);                               \
        else if (GEN) ST_LAUNCH_CHEB_FORM(STRIDE, 0, true, 0);                                    \
        else if (a.kcache_mode == 1) ST_LAUNCH_CHEB_SEARCH(STRIDE, 1);                            \
        else if (a.kcache_mode == 2) ST_LAUNCH_CHEB_SEARCH(STRIDE, 2);                            \
        else ST_LAUNCH_CHEB_SEARCH(STRIDE, 0);                                                    \
    } while (0)
        const int mode = a.capture_mode ? 1 : (a.tmax_snr ? 2 : 0);
        int pb_ = pb_single;
        // the general build (cubic family, inverse-variance weighting, explicit templates) reads its options
        // at run time; the default search is compiled with them as constants
        const bool gen = a.bp.family != 0 || a.norm == 2 || a.tracks != nullptr;
        // Grids with class B bins (coefficient drift, see build_cheb_tables): the fast build scores every template
        // whose amplitude in those bins bounds the drift error below kChebDeferBudget and lists the others; a
        // second launch of the general (two-class) build scores the listed ones.  Results are order independent.
        const bool two_pass = !gen && c->cheb_n_class_b > 0;
        a.deferred = at<uint32_t>(c, c->L.deferred); a.deferred_cap = kDeferCap; a.defer_in = 0;
        a.defer_limit = two_pass ? (float)(kChebDeferBudget / c->cheb_dmax) : 3.4e38f;
        if (two_pass) {
            if (a.n_tracks > kDeferCap) return fail(c, ST_EINVAL, "internal: Chebyshev launch of %llu templates exceeds its hand-over list", (unsigned long long)a.n_tracks);
            ST_CUDA(c, cudaMemsetAsync(&a.sc->n_deferred, 0, sizeof(uint32_t), c->stream));
        }
        if (pk) { if (gen) ST_LAUNCH_CHEB_MODE(2, true); else ST_LAUNCH_CHEB_MODE(2, false); }
        else    { if (gen) ST_LAUNCH_CHEB_MODE(1, true); else ST_LAUNCH_CHEB_MODE(1, false); }
        if (two_pass) {
            ST_CUDA(c, cudaGetLastError());
            ST_CUDA(c, cudaMemsetAsync(&a.sc->counter, 0, sizeof(unsigned long long), c->stream));
            a.defer_in = 1; a.defer_limit = 3.4e38f;
            pb_ = pb;
            blocks = (uint64_t)c->n_sm;
            if (blocks > need) blocks = need;
            if (pk) ST_LAUNCH_CHEB_MODE(2, true); else ST_LAUNCH_CHEB_MODE(1, true);
            a.defer_in = 0;
            if (extra_launches) ++*extra_launches;
        }
#undef ST_LAUNCH_CHEB_MODE
#undef ST_LAUNCH_CHEB_SEARCH
#undef ST_LAUNCH_CHEB_PIPE
#undef ST_LAUNCH_CHEB_FORM
#undef ST_LAUNCH_CHEB
    } else if (plan.kernel == ST_KERNEL_REINSCH) {
        int threads = c->recur_threads;
        size_t smem;
        for (;; threads -= 32) {
            smem = hist_bytes(a.n_bins) + (size_t)(c->n_f + (c->n_f & 1)) * sizeof(float2) +
                   (size_t)(threads / 32) * (size_t)(stride / 2) * (8 + 8 + 4);
            if (smem <= (size_t)c->smem_optin || threads == 32) break;
        }
        if (smem > (size_t)c->smem_optin)
            return fail(c, ST_ENOSPC, "n_f %d / n_max %d need more shared memory than one SM has", c->n_f, n_max);
        int rc = set_smem(c, st::k_score_reinsch, smem);
        if (rc) return rc;
        uint64_t blocks = (uint64_t)c->n_sm;            // persistent: one block per SM
        const uint64_t need = (want_warps + (uint64_t)(threads / 32) - 1) / (uint64_t)(threads / 32);
        if (blocks > need) blocks = need;
        st::k_score_reinsch<<<(unsigned)blocks, threads, smem, c->stream>>>(a);
    } else {
        int threads = c->recur_threads;
        const size_t bt_bytes = (size_t)c->n_f * sizeof(float4);
        bool bt_smem = true;
        size_t smem;
        for (;;) {
            smem = hist_bytes(a.n_bins) + (bt_smem ? bt_bytes : 0) +
                   (size_t)(threads / 32) * (size_t)stride * (sizeof(float2) + sizeof(uint16_t));
            if (smem <= (size_t)c->smem_optin) break;
            if (threads > 256) threads -= 64;           // fewer warps first, down to 8
            else if (bt_smem) bt_smem = false;          // then the bin table stays in L2
            else if (threads > 32) threads -= 32;
            else return fail(c, ST_ENOSPC, "n_max %d needs more shared memory than one SM has", n_max);
        }
        uint64_t blocks = (uint64_t)c->n_sm;            // persistent: one block per SM
        const uint64_t need = (want_warps + (uint64_t)(threads / 32) - 1) / (uint64_t)(threads / 32);
        if (blocks > need) blocks = need;
#define ST_LAUNCH_RECUR(MODE, CH, BT)                                                              \
    do {                                                                                           \
        int rc_ = set_smem(c, st::k_score_recur<MODE, CH, BT>, smem);                              \
        if (rc_) return rc_;                                                                       \
        st::k_score_recur<MODE, CH, BT><<<(unsigned)blocks, threads, smem, c->stream>>>(a);        \
    } while (0)
        if (plan.ch == 32) { if (bt_smem) ST_LAUNCH_RECUR(0, 32, true); else ST_LAUNCH_RECUR(0, 32, false); }
        else               { if (bt_smem) ST_LAUNCH_RECUR(0, 64, true); else ST_LAUNCH_RECUR(0, 64, false); }
#undef ST_LAUNCH_RECUR
    }
    ST_CUDA(c, cudaGetLastError());
    return ST_OK;
}

st::ScoreArgs base_args(st_ctx* c, const st_search_params* p)
{
    st::ScoreArgs a;
    memset(&a, 0, sizeof(a));
    a.map = at<float2>(c, c->L.map);
    a.isig = at<float>(c, c->L.isig);
    a.bp = bank(c, p);
    a.f_min = c->f_min; a.df = c->df;
    a.n_tau = p->tau_mode == ST_TAU_GRID ? p->n_tau : 1;
    a.norm = p->norm;
    a.W = at<float2>(c, c->L.w);
    a.E0 = at<float2>(c, c->L.e0);
    a.bintab = at<float4>(c, c->L.bintab);
    a.Es = at<float2>(c, c->L.es);
    a.kz = at<float2>(c, c->L.kz);
    a.Ec = at<float2>(c, c->L.ec);
    a.cheb = at<float4>(c, c->L.cheb);
    a.cheb_zi = at<float>(c, c->L.cheb_zi);
    a.sc = at<st::Scalars>(c, c->L.scalars);
    a.cand = at<st::Cand>(c, c->L.cand);
    a.cand_cap = kCandCap;
    a.warp_best = at<st::WarpBest>(c, c->L.warp_best);
    a.warp_slots = kWarpSlots;
    a.hist = at<unsigned long long>(c, c->L.hist);
    a.n_bins = 0; a.hist_lo = 0.0f; a.hist_scale = 0.0f;
    a.dump = nullptr;
    return a;
}

// Where one search keeps its device state: the context's own slots, or the per-map slots of a batch.
struct Slots {
    st::Scalars* sc;
    st::DeviceResult* res;
    unsigned long long* hist;
};
Slots own_slots(st_ctx* c)
{
    Slots s;
    s.sc = at<st::Scalars>(c, c->L.scalars); s.res = at<st::DeviceResult>(c, c->L.result);
    s.hist = at<unsigned long long>(c, c->L.hist);
    return s;
}
Slots batch_slots(st_ctx* c, int i)
{
    Slots s;
    s.sc = at<st::Scalars>(c, c->L.b_scalars) + i; s.res = at<st::DeviceResult>(c, c->L.b_result) + i;
    s.hist = at<unsigned long long>(c, c->L.b_hist) + (size_t)i * ST_MAX_BINS;
    return s;
}

int reset_search_state(st_ctx* c, int n_bins, const Slots& sl)
{
    ST_CUDA(c, cudaMemsetAsync(sl.sc, 0, sizeof(st::Scalars), c->stream));
    ST_CUDA(c, cudaMemsetAsync(at<void>(c, c->L.warp_best), 0, (size_t)kWarpSlots * sizeof(st::WarpBest), c->stream));
    if (n_bins > 0)
        ST_CUDA(c, cudaMemsetAsync(sl.hist, 0, (size_t)n_bins * sizeof(unsigned long long), c->stream));
    // gmax_bits = 0 encodes "below every float" (enc(-inf) = 0x007FFFFF > 0)
    return ST_OK;
}

// S1-S4 of one search, enqueued on the stream (no synchronisation): tables must be current.
int enqueue_search(st_ctx* c, const st_search_params* p, const Plan& plan, const Slots& sl, int* n_launches,
                   bool time_it, float* tmax_snr = nullptr, int32_t* tmax_m = nullptr);
void fill_result(st_result* out, const st::DeviceResult& r, int n_tau, int kernel, int n_launches);

void fill_result(st_result* out, const st::DeviceResult& r, int n_tau, int kernel, int n_launches)
{
    out->max_snr = r.max_snr; out->arg_tau_index = r.arg_m; out->max_snr_f64 = r.snr_f64;
    out->arg_track = r.arg_id; out->arg_tau = r.arg_tau;
    out->arg_params.N = r.track.N; out->arg_params.j0 = r.track.j0; out->arg_params.a = r.track.a;
    out->arg_params.y0 = r.track.y0; out->arg_params.y1 = r.track.y1; out->arg_params.y2 = r.track.y2;
    out->arg_params.tau = r.track.tau; out->arg_params.y3 = r.track.y3;
    out->n_pixels = r.n_pixels; out->n_evals = r.n_pixels * (uint64_t)n_tau;
    out->n_candidates = r.n_candidates; out->flags = r.flags; out->n_launches = n_launches;
    out->n_deferred = (int32_t)r.n_deferred;
    out->kernel_used = kernel;
}

int enqueue_search(st_ctx* c, const st_search_params* p, const Plan& plan, const Slots& sl, int* n_launches,
                   bool time_it, float* tmax_snr, int32_t* tmax_m)
{
    const int n_tau = p->tau_mode == ST_TAU_GRID ? p->n_tau : 1;
    // every search passes here, so no caller can score with a 1 / sigma plane that does not belong to the map
    // (the ft-map path forms p directly and leaves the plane of an earlier st_set_map, or nothing, behind)
    if (p->norm == ST_NORM_INVVAR && !c->have_isig)
        return fail(c, ST_ESTATE, "ST_NORM_INVVAR needs sigma: set the map through st_set_map / st_set_map_host / st_search_batch");
    int rc = reset_search_state(c, p->n_bins, sl);
    if (rc) return rc;
    st::ScoreArgs a = base_args(c, p);
    a.sc = sl.sc; a.hist = sl.hist;
    a.n_bins = p->n_bins;
    a.hist_lo = (float)p->hist_lo;
    a.hist_scale = p->n_bins > 0 ? (float)((double)p->n_bins / (p->hist_hi - p->hist_lo)) : 0.0f;
    uint64_t per_launch = kMaxSamplesPerLaunch / (uint64_t)n_tau;
    if (per_launch < 1) per_launch = 1;
    if (plan.kernel == ST_KERNEL_CHEBYSHEV && per_launch > kDeferCap) per_launch = kDeferCap;
    // bank cache: a plain Chebyshev search of quadratic templates reads S1 + S2 from the cache when it holds this
    // bank (same seed, id range, duration range), else fills it when the range fits
    int bank_mode = 0;
    if (c->bank && plan.kernel == ST_KERNEL_CHEBYSHEV && p->family == ST_FAMILY_QUADRATIC && p->norm != ST_NORM_INVVAR &&
        !tmax_snr && p->n_tracks > 0) {
        const uint32_t stride = bank_row_entries(p->n_max);
        const bool same = c->bank_valid && c->bank_key.seed == p->seed && c->bank_key.offset == p->track_offset &&
                          c->bank_key.n_tracks == p->n_tracks && c->bank_key.n_min == p->n_min && c->bank_key.n_max == p->n_max;
        if (same) bank_mode = 2;
        else if (bank_bytes_for(p->n_tracks, p->n_max) <= c->bank_bytes) {
            bank_mode = 1;
            c->bank_valid = false;
            c->bank_key.seed = p->seed; c->bank_key.offset = p->track_offset; c->bank_key.n_tracks = p->n_tracks;
            c->bank_key.n_min = p->n_min; c->bank_key.n_max = p->n_max;
        }
        a.kcache_stride = stride;
        a.kmeta = reinterpret_cast<int2*>(c->bank);
        a.kcache = reinterpret_cast<uint16_t*>(c->bank + align_up((size_t)p->n_tracks * sizeof(int2)));
    }
    a.kcache_mode = bank_mode;
    if (time_it) ST_CUDA(c, cudaEventRecord(c->ev0, c->stream));
    for (uint64_t done = 0; done < p->n_tracks; done += per_launch) {
        a.track_offset = p->track_offset + done;
        a.n_tracks = p->n_tracks - done < per_launch ? p->n_tracks - done : per_launch;
        a.tmax_snr = tmax_snr ? tmax_snr + done : nullptr;
        a.tmax_m = tmax_m ? tmax_m + done : nullptr;
        a.kcache_base = done;
        rc = launch_score(c, plan, a, p->n_max, n_launches);
        if (rc) return rc;
        ++*n_launches;
    }
    if (time_it) ST_CUDA(c, cudaEventRecord(c->ev1, c->stream));
    if (bank_mode == 1) c->bank_valid = true;       // every launch of the filling search has been enqueued
    c->last_bank_mode = bank_mode;
    st::FinalArgs f;
    memset(&f, 0, sizeof(f));
    f.map = a.map; f.isig = a.isig; f.bp = a.bp; f.f_min = c->f_min; f.df = c->df;
    f.norm = p->norm; f.tau_mode = p->tau_mode; f.n_tau = n_tau;
    f.tau_d = at<double>(c, c->L.tau);
    f.sc = a.sc; f.cand = a.cand; f.cand_cap = kCandCap; f.warp_best = a.warp_best; f.n_warp_slots = kWarpSlots;
    f.out = sl.res;
    st::k_finalize<<<1, 256, 0, c->stream>>>(f);
    ST_CUDA(c, cudaGetLastError());
    ++*n_launches;
    return ST_OK;
}

// An explicit template (st_score_tracks, st_debug_rasterise_track) must lie where bank members lie: 0 < a < N and
// the control points its family uses inside the band, 0 <= y <= n_f.  The rasteriser's fast path decides a bin
// without the normative sequence when y is further than raster_guard() from an edge, and that guard is sized for
// |dy/dxi| <= 2 n_f (quadratic) / 3 n_f (cubic), i.e. for control points inside the band; outside it the fast bin
// could differ from the normative one without a redo, which is exactly what these exports promise not to happen.
const char* explicit_track_problem(const st_ctx* c, const st_track& t, int32_t family)
{
    if (t.N < 1 || t.j0 < 0 || (int64_t)t.j0 + (int64_t)t.N > (int64_t)c->n_t) return "lies outside the map";
    if (!(t.a > 0.0) || !(t.a < (double)t.N)) return "needs 0 < a < N";
    if (!isfinite(t.y0) || !isfinite(t.y1) || !isfinite(t.y2) || !isfinite(t.y3) || !isfinite(t.tau))
        return "needs finite control points and delay";
    const double top = (double)c->n_f;
    const int n_used = family == ST_FAMILY_CHIRP ? 1 : (family == ST_FAMILY_CUBIC ? 4 : 3);
    const double y[4] = {t.y0, t.y1, t.y2, t.y3};
    for (int i = 0; i < n_used; ++i)
        if (y[i] < 0.0 || y[i] > top) return "needs its frequency control points inside the band, 0 <= y <= n_f (bin units)";
    return nullptr;
}

}  // namespace

// ================================================================== C ABI ====
extern "C" {

const char* st_version(void) { return "stochtrack-b200 0.1 (sm_100a)"; }

const char* st_last_error(const st_ctx* ctx) { return ctx ? ctx->err : "null context"; }

int st_create(st_ctx** out, int32_t n_t, int32_t n_f, double df, double f_min)
{
    if (!out) return ST_EINVAL;
    *out = nullptr;
    if (n_t < 1 || n_t > ST_MAX_N_T || n_f < 1 || n_f > ST_MAX_N_F) return ST_EINVAL;
    if (!(df > 0.0) || !(f_min >= 0.0) || !isfinite(df) || !isfinite(f_min)) return ST_EINVAL;
    st_ctx* c = new (std::nothrow) st_ctx();
    if (!c) return ST_EINVAL;
    c->n_t = n_t; c->n_f = n_f; c->df = df; c->f_min = f_min;
    c->ws = nullptr; c->ws_bytes = 0; c->max_n_tau = 0; c->stream = nullptr;
    c->have_ws = c->have_map = false; c->have_isig = false;
    c->table_kind = kNoTable; c->table_ch = 0; c->w_built = false;
    c->ev0 = c->ev1 = nullptr; c->h_res = nullptr; c->h_hist = nullptr;
    c->copy_stream = nullptr; c->h_bres = nullptr; c->h_bhist = nullptr;
    for (int i = 0; i < 2; ++i) { c->ev_copied[i] = nullptr; c->ev_consumed[i] = nullptr; }
    c->n_sm = 0; c->smem_optin = 0; c->recur_threads = ST_CHEB_MAX_THREADS; c->device = 0; c->ev_device = -1;
    c->err[0] = 0;
    c->bank = nullptr; c->bank_bytes = 0; c->bank_valid = false; c->last_bank_mode = 0; memset(&c->bank_key, 0, sizeof(c->bank_key));
    c->cheb_stride = 0; c->cheb_n_class_b = 0; c->cheb_dmax = 0.0; c->pick_valid = false; c->pick_dtau = 0.0; c->pick_stride = 0;
    *out = c;
    return ST_OK;
}

void st_destroy(st_ctx* c)
{
    if (!c) return;
    if (c->ev0) cudaEventDestroy(c->ev0);
    if (c->ev1) cudaEventDestroy(c->ev1);
    if (c->h_res) cudaFreeHost(c->h_res);
    if (c->h_hist) cudaFreeHost(c->h_hist);
    if (c->h_bres) cudaFreeHost(c->h_bres);
    if (c->h_bhist) cudaFreeHost(c->h_bhist);
    for (int i = 0; i < 2; ++i) {
        if (c->ev_copied[i]) cudaEventDestroy(c->ev_copied[i]);
        if (c->ev_consumed[i]) cudaEventDestroy(c->ev_consumed[i]);
    }
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    delete c;
}

size_t st_workspace_bytes(const st_ctx* c, int32_t max_n_tau)
{
    if (!c || max_n_tau < 1 || max_n_tau > ST_MAX_N_TAU) return 0;
    return make_layout(c->n_t, c->n_f, max_n_tau).total;
}

int st_set_workspace(st_ctx* c, void* ws, size_t bytes, void* cuda_stream)
{
    if (!c) return ST_EINVAL;
    if (!ws || ((uintptr_t)ws % kAlign) != 0) return fail(c, ST_EINVAL, "workspace must be a non-null, 256-byte aligned device pointer");
    // largest max_n_tau the buffer supports
    const size_t base = make_layout(c->n_t, c->n_f, 1).total;
    if (bytes < base) return fail(c, ST_ENOSPC, "workspace of %zu bytes is below the minimum %zu", bytes, base);
    int lo = 1, hi = ST_MAX_N_TAU;
    while (lo < hi) {
        const int mid = (lo + hi + 1) / 2;
        if (make_layout(c->n_t, c->n_f, mid).total <= bytes) lo = mid; else hi = mid - 1;
    }
    cudaPointerAttributes pa;
    ST_CUDA(c, cudaPointerGetAttributes(&pa, ws));
    if (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged)
        return fail(c, ST_EINVAL, "workspace is not device memory");
    const int dev = pa.device;                      // the context lives on the workspace's device
    // Everything fallible happens first, into locals: a failure below leaves the context exactly as it was (an
    // attached workspace stays attached and usable on its own device).
    DevGuard dev_guard(dev);
    int n_sm = 0, smem_optin = 0;
    ST_CUDA(c, cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    ST_CUDA(c, cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    // events belong to the device they were created on: a move to another device gets its own pair
    const bool new_events = !c->ev0 || !c->ev1 || c->ev_device != dev;
    cudaEvent_t ev0 = c->ev0, ev1 = c->ev1;
    if (new_events) {
        ev0 = ev1 = nullptr;
        ST_CUDA(c, cudaEventCreate(&ev0));
        const cudaError_t e1 = cudaEventCreate(&ev1);
        if (e1 != cudaSuccess) { cudaEventDestroy(ev0); return fail(c, ST_ECUDA, "cudaEventCreate: %s", cudaGetErrorString(e1)); }
    }
    if (!c->h_res || !c->h_hist) {
        st::DeviceResult* h_res = c->h_res;
        unsigned long long* h_hist = c->h_hist;
        cudaError_t e = cudaSuccess;
        if (!h_res) e = cudaHostAlloc((void**)&h_res, sizeof(st::DeviceResult), cudaHostAllocDefault);
        if (e == cudaSuccess && !h_hist) e = cudaHostAlloc((void**)&h_hist, ST_MAX_BINS * sizeof(unsigned long long), cudaHostAllocDefault);
        if (e != cudaSuccess) {
            if (h_res && !c->h_res) cudaFreeHost(h_res);
            if (new_events) { cudaEventDestroy(ev0); cudaEventDestroy(ev1); }
            return fail(c, ST_ECUDA, "cudaHostAlloc: %s", cudaGetErrorString(e));
        }
        c->h_res = h_res; c->h_hist = h_hist;       // pinned host memory serves any device: kept across re-attachments
    }
    // ---- commit (no CUDA call below can fail the attachment)
    if (new_events) {
        if (c->ev0) cudaEventDestroy(c->ev0);
        if (c->ev1) cudaEventDestroy(c->ev1);
        c->ev0 = ev0; c->ev1 = ev1;
        if (c->ev_device != dev) {                  // the batch mode's stream and events are re-made lazily on the new device
            for (int i = 0; i < 2; ++i) {
                if (c->ev_copied[i]) { cudaEventDestroy(c->ev_copied[i]); c->ev_copied[i] = nullptr; }
                if (c->ev_consumed[i]) { cudaEventDestroy(c->ev_consumed[i]); c->ev_consumed[i] = nullptr; }
            }
            if (c->copy_stream) { cudaStreamDestroy(c->copy_stream); c->copy_stream = nullptr; }
        }
        c->ev_device = dev;
    }
    c->device = dev; c->n_sm = n_sm; c->smem_optin = smem_optin;
    c->ws = (unsigned char*)ws; c->ws_bytes = bytes; c->max_n_tau = lo;
    c->L = make_layout(c->n_t, c->n_f, lo);
    c->stream = (cudaStream_t)cuda_stream;
    c->have_ws = true; c->have_map = false; c->have_isig = false;
    c->tau_cached.clear(); c->table_kind = kNoTable; c->w_built = false;
    // a bank cache filled on the previous stream or device is not ordered against reads on the new one
    c->bank_valid = false;
    return ST_OK;
}

size_t st_bank_cache_bytes(const st_ctx* c, uint64_t n_tracks, int32_t n_max)
{
    if (!c || n_tracks == 0 || n_tracks > (1ull << 40) || n_max < 1 || n_max > c->n_t) return 0;
    return bank_bytes_for(n_tracks, n_max);
}

int st_set_bank_cache(st_ctx* c, void* cache_dev, size_t bytes)
{
    if (!c) return ST_EINVAL;
    if (cache_dev && ((uintptr_t)cache_dev % kAlign) != 0) return fail(c, ST_EINVAL, "bank cache must be 256-byte aligned");
    c->bank = (unsigned char*)cache_dev; c->bank_bytes = cache_dev ? bytes : 0; c->bank_valid = false;
    return ST_OK;
}

// S0 into the workspace.  want_isig: also write the 1 / sigma plane (read by ST_NORM_INVVAR only).
static int set_map_impl(st_ctx* c, const void* csd_dev, const float* sigma_dev, int32_t sigma_kind, bool want_isig);

int st_set_map(st_ctx* c, const void* csd_dev, const float* sigma_dev, int32_t sigma_kind)
{
    DevGuard dev_guard(c);
    return set_map_impl(c, csd_dev, sigma_dev, sigma_kind, true);     // whichever norm a later search asks for
}

static int set_map_impl(st_ctx* c, const void* csd_dev, const float* sigma_dev, int32_t sigma_kind, bool want_isig)
{
    if (!c) return ST_EINVAL;
    if (!c->have_ws) return fail(c, ST_ESTATE, "no workspace: call st_set_workspace first");
    if (!csd_dev) return fail(c, ST_EINVAL, "csd is NULL");
    if (sigma_kind < ST_SIGMA_NONE || sigma_kind > ST_SIGMA_PER_PIXEL) return fail(c, ST_EINVAL, "bad sigma_kind %d", sigma_kind);
    if (sigma_kind != ST_SIGMA_NONE && !sigma_dev) return fail(c, ST_EINVAL, "sigma is NULL");
    const size_t n_pix = (size_t)c->n_t * (size_t)c->n_f;
    const int blocks = (int)((n_pix + 255) / 256 < (size_t)(8 * c->n_sm) ? (n_pix + 255) / 256 : (size_t)(8 * c->n_sm));
    // two pixels per thread through 16-byte accesses when the pointers and the pixel count allow
    const bool vec = (n_pix % 2 == 0) && ((uintptr_t)csd_dev % 16 == 0) &&
                     (sigma_kind != ST_SIGMA_PER_PIXEL || (uintptr_t)sigma_dev % 8 == 0);
#define ST_LAUNCH_PREPARE(VEC, ISIG)                                                                              \
    st::k_prepare_map<VEC, ISIG><<<blocks, 256, 0, c->stream>>>((const float2*)csd_dev, sigma_dev, sigma_kind, c->n_f, n_pix, \
                                                                at<float2>(c, c->L.map), at<float>(c, c->L.isig))
    if (vec) { if (want_isig) ST_LAUNCH_PREPARE(true, true); else ST_LAUNCH_PREPARE(true, false); }
    else     { if (want_isig) ST_LAUNCH_PREPARE(false, true); else ST_LAUNCH_PREPARE(false, false); }
#undef ST_LAUNCH_PREPARE
    ST_CUDA(c, cudaGetLastError());
    c->have_map = true; c->have_isig = want_isig;
    return ST_OK;
}

int st_set_map_host(st_ctx* c, const void* csd_host, const float* sigma_host, int32_t sigma_kind)
{
    DevGuard dev_guard(c);
    if (!c) return ST_EINVAL;
    if (!c->have_ws) return fail(c, ST_ESTATE, "no workspace: call st_set_workspace first");
    if (!csd_host) return fail(c, ST_EINVAL, "csd is NULL");
    if (sigma_kind < ST_SIGMA_NONE || sigma_kind > ST_SIGMA_PER_PIXEL) return fail(c, ST_EINVAL, "bad sigma_kind %d", sigma_kind);
    if (sigma_kind != ST_SIGMA_NONE && !sigma_host) return fail(c, ST_EINVAL, "sigma is NULL");
    const size_t n_pix = (size_t)c->n_t * (size_t)c->n_f;
    ST_CUDA(c, cudaMemcpyAsync(at<void>(c, c->L.stage_csd), csd_host, n_pix * sizeof(float2), cudaMemcpyHostToDevice, c->stream));
    if (sigma_kind != ST_SIGMA_NONE) {
        const size_t n_s = sigma_kind == ST_SIGMA_PER_FREQ ? (size_t)c->n_f : n_pix;
        ST_CUDA(c, cudaMemcpyAsync(at<void>(c, c->L.stage_sigma), sigma_host, n_s * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    }
    const int rc = st_set_map(c, at<void>(c, c->L.stage_csd), at<float>(c, c->L.stage_sigma), sigma_kind);
    if (rc) return rc;
    ST_CUDA(c, cudaStreamSynchronize(c->stream));
    return ST_OK;
}

static int search_impl(st_ctx* c, const st_search_params* p, st_result* out, float* tmax_snr, int32_t* tmax_m);

// The bank cache's validity is host-side book-keeping: it is set once a filling search has been ENQUEUED.  Any call
// that then fails (a launch or synchronisation error, an error in a later map of a batch) may leave the cache
// partly written, so every failing search drops it; the next search with that bank fills it again.
static int drop_bank_on_error(st_ctx* c, int rc)
{
    if (rc && c) c->bank_valid = false;
    return rc;
}

int st_search(st_ctx* c, const st_search_params* p, st_result* out)
{
    DevGuard dev_guard(c);
    return drop_bank_on_error(c, search_impl(c, p, out, nullptr, nullptr));
}

int st_search_track_max(st_ctx* c, const st_search_params* p, float* snr_max_dev, int32_t* tau_index_dev, st_result* out)
{
    DevGuard dev_guard(c);
    if (!c) return ST_EINVAL;
    if (!snr_max_dev || !tau_index_dev) return fail(c, ST_EINVAL, "per-template output pointer is NULL");
    return drop_bank_on_error(c, search_impl(c, p, out, snr_max_dev, tau_index_dev));
}

static int search_impl(st_ctx* c, const st_search_params* p, st_result* out, float* tmax_snr, int32_t* tmax_m)
{
    int rc = validate(c, p, true);
    if (rc) return rc;
    if (!out) return fail(c, ST_EINVAL, "result is NULL");
    if (p->n_bins > 0 && !p->hist_out) return fail(c, ST_EINVAL, "n_bins > 0 but hist_out is NULL");
    memset(out, 0, sizeof(*out));
    Plan plan;
    rc = make_plan(c, p, &plan);
    if (rc) return rc;
    out->kernel_used = plan.kernel;
    const int n_tau = p->tau_mode == ST_TAU_GRID ? p->n_tau : 1;
    if (p->n_tracks == 0) {                       // empty search: nothing scored
        out->max_snr = -INFINITY; out->max_snr_f64 = -INFINITY;
        if (p->n_bins > 0) memset(p->hist_out, 0, sizeof(uint64_t) * (size_t)p->n_bins);
        return ST_OK;
    }
    int n_launches = 0;
    rc = ensure_tables(c, p, plan, &n_launches);
    if (rc) return rc;
    const Slots sl = own_slots(c);
    rc = enqueue_search(c, p, plan, sl, &n_launches, true, tmax_snr, tmax_m);
    if (rc) return rc;
    ST_CUDA(c, cudaMemcpyAsync(c->h_res, sl.res, sizeof(st::DeviceResult), cudaMemcpyDeviceToHost, c->stream));
    if (p->n_bins > 0)
        ST_CUDA(c, cudaMemcpyAsync(c->h_hist, sl.hist, sizeof(unsigned long long) * (size_t)p->n_bins, cudaMemcpyDeviceToHost, c->stream));
    ST_CUDA(c, cudaStreamSynchronize(c->stream));
    fill_result(out, *c->h_res, n_tau, plan.kernel, n_launches);
    out->flags |= c->last_bank_mode == 2 ? ST_FLAG_BANK_READ : (c->last_bank_mode == 1 ? ST_FLAG_BANK_FILLED : 0);
    float ms = 0.0f;
    ST_CUDA(c, cudaEventElapsedTime(&ms, c->ev0, c->ev1));
    out->gpu_ms = ms;
    if (p->n_bins > 0)
        for (int b = 0; b < p->n_bins; ++b) p->hist_out[b] = (uint64_t)c->h_hist[b];
    return ST_OK;
}

int st_search_topk(st_ctx* c, const st_search_params* p, int32_t top_k, st_top_entry* top_out, int32_t* n_out,
                   st_result* result)
{
    DevGuard dev_guard(c);
    if (!c) return ST_EINVAL;
    if (!p || !top_out || !n_out || !result) return fail(c, ST_EINVAL, "NULL argument");
    if (top_k < 1 || top_k > ST_MAX_TOP_K) return fail(c, ST_EINVAL, "top_k %d outside [1, %d]", top_k, ST_MAX_TOP_K);
    if (p->n_bins < 1) return fail(c, ST_EINVAL, "st_search_topk needs a histogram (n_bins > 0)");
    *n_out = 0;
    int rc = st_search(c, p, result);                       // pass 1: maximum, histogram
    if (rc) return rc;
    if (p->n_tracks == 0) return ST_OK;
    // the bin holding the top_k-th largest sample, then one bin lower (a sample near an edge may have been
    // binned on either side of it in float32)
    uint64_t cum = 0;
    int b = p->n_bins;
    while (b > 0 && cum < (uint64_t)top_k) cum += p->hist_out[--b];
    if (b > 0) cum += p->hist_out[--b];
    if (cum > (uint64_t)kCandCap)
        return fail(c, ST_ENOSPC, "%llu samples at or above the bin of the top_k-th: histogram too coarse (cap %u)",
                    (unsigned long long)cum, kCandCap);
    const double width = (p->hist_hi - p->hist_lo) / (double)p->n_bins;
    // the capture threshold sits below that edge by more than the float32 score error (relative 1e-4, the
    // G13 tolerance, whatever the bin width): the final order is decided by the float64 re-score
    const double edge = p->hist_lo + (double)b * width;
    const float thr = b == 0 ? -INFINITY : (float)(edge - 1e-4 * width - 1e-4 * (fabs(edge) > 1.0 ? fabs(edge) : 1.0));
    // pass 2: capture
    Plan plan;
    rc = make_plan(c, p, &plan);
    if (rc) return rc;
    const int n_tau = p->tau_mode == ST_TAU_GRID ? p->n_tau : 1;
    const Slots sl = own_slots(c);
    rc = reset_search_state(c, 0, sl);
    if (rc) return rc;
    st::ScoreArgs a = base_args(c, p);
    a.capture_mode = 1; a.capture_thr = thr;
    uint64_t per_launch = kMaxSamplesPerLaunch / (uint64_t)n_tau;
    if (per_launch < 1) per_launch = 1;
    if (plan.kernel == ST_KERNEL_CHEBYSHEV && per_launch > kDeferCap) per_launch = kDeferCap;
    for (uint64_t done = 0; done < p->n_tracks; done += per_launch) {
        a.track_offset = p->track_offset + done;
        a.n_tracks = p->n_tracks - done < per_launch ? p->n_tracks - done : per_launch;
        rc = launch_score(c, plan, a, p->n_max, &result->n_launches);
        if (rc) return rc;
        ++result->n_launches;
    }
    st::FinalArgs f;
    memset(&f, 0, sizeof(f));
    f.map = a.map; f.isig = a.isig; f.bp = a.bp; f.f_min = c->f_min; f.df = c->df;
    f.norm = p->norm; f.tau_mode = p->tau_mode; f.n_tau = n_tau;
    f.tau_d = at<double>(c, c->L.tau);
    f.sc = a.sc; f.cand = a.cand; f.cand_cap = kCandCap;
    st::k_rescore_cands<<<c->n_sm * 4, 256, 0, c->stream>>>(f, at<double>(c, c->L.cand64));
    ST_CUDA(c, cudaGetLastError());
    ++result->n_launches;
    st::Scalars hsc;
    ST_CUDA(c, cudaMemcpyAsync(&hsc, a.sc, sizeof(hsc), cudaMemcpyDeviceToHost, c->stream));
    ST_CUDA(c, cudaStreamSynchronize(c->stream));
    if (hsc.overflow || hsc.cand_count > kCandCap) return fail(c, ST_ENOSPC, "candidate list overflowed in the capture pass");
    const uint32_t n = hsc.cand_count;
    std::vector<st::Cand> hc(n);
    std::vector<double> h64(n);
    if (n) {
        ST_CUDA(c, cudaMemcpy(hc.data(), a.cand, (size_t)n * sizeof(st::Cand), cudaMemcpyDeviceToHost));
        ST_CUDA(c, cudaMemcpy(h64.data(), at<double>(c, c->L.cand64), (size_t)n * sizeof(double), cudaMemcpyDeviceToHost));
    }
    std::vector<uint32_t> order(n);
    for (uint32_t i = 0; i < n; ++i) order[i] = i;
    std::sort(order.begin(), order.end(), [&](uint32_t x, uint32_t y) {     // G12 total order
        if (h64[x] != h64[y]) return h64[x] > h64[y];
        if (hc[x].id != hc[y].id) return hc[x].id < hc[y].id;
        return hc[x].m < hc[y].m;
    });
    const uint32_t k_out = n < (uint32_t)top_k ? n : (uint32_t)top_k;
    for (uint32_t i = 0; i < k_out; ++i) {
        const uint32_t e = order[i];
        top_out[i].track = hc[e].id; top_out[i].tau_index = (int32_t)hc[e].m;
        top_out[i].snr_f32 = hc[e].snr; top_out[i].snr_f64 = h64[e];
        if (p->tau_mode == ST_TAU_GRID) top_out[i].tau = p->tau_grid[hc[e].m];
        else {
            st::BankParams bp = bank(c, p);
            top_out[i].tau = st::make_track(bp, hc[e].id).tau;
        }
    }
    *n_out = (int32_t)k_out;
    return ST_OK;
}

static int batch_impl(st_ctx* c, const st_batch* b, const st_search_params* p, st_result* results, float* gpu_ms_total);

int st_search_batch(st_ctx* c, const st_batch* b, const st_search_params* p, st_result* results, float* gpu_ms_total)
{
    DevGuard dev_guard(c);
    const int rc = batch_impl(c, b, p, results, gpu_ms_total);
    if (rc && c && c->have_ws) {
        // an error part-way through: host-to-device copies from the caller's buffers may still be in flight
        // on the internal stream, and searches on the caller's; both drain before the buffers are handed back
        if (c->copy_stream) cudaStreamSynchronize(c->copy_stream);
        cudaStreamSynchronize(c->stream);
    }
    return drop_bank_on_error(c, rc);
}

static int batch_impl(st_ctx* c, const st_batch* b, const st_search_params* p, st_result* results, float* gpu_ms_total)
{
    int rc = validate(c, p, false);
    if (rc) return rc;
    if (!b || !results) return fail(c, ST_EINVAL, "batch / results is NULL");
    if (b->n_maps < 1) return fail(c, ST_EINVAL, "n_maps must be >= 1");
    if (b->reserved != 0) return fail(c, ST_EINVAL, "batch.reserved must be 0");
    if (!b->csd) return fail(c, ST_EINVAL, "batch.csd is NULL");
    if (b->sigma_kind < ST_SIGMA_NONE || b->sigma_kind > ST_SIGMA_PER_PIXEL) return fail(c, ST_EINVAL, "bad sigma_kind %d", b->sigma_kind);
    if (b->sigma_kind != ST_SIGMA_NONE && !b->sigma) return fail(c, ST_EINVAL, "batch.sigma is NULL");
    for (int m = 0; m < b->n_maps; ++m) {
        if (!b->csd[m]) return fail(c, ST_EINVAL, "batch.csd[%d] is NULL", m);
        if (b->sigma_kind != ST_SIGMA_NONE && !b->sigma[m]) return fail(c, ST_EINVAL, "batch.sigma[%d] is NULL", m);
    }
    if (p->n_bins > 0 && !p->hist_out) return fail(c, ST_EINVAL, "n_bins > 0 but hist_out is NULL");
    Plan plan;
    rc = make_plan(c, p, &plan);
    if (rc) return rc;
    const int n_tau = p->tau_mode == ST_TAU_GRID ? p->n_tau : 1;
    if (gpu_ms_total) *gpu_ms_total = 0.0f;
    memset(results, 0, sizeof(st_result) * (size_t)b->n_maps);
    if (p->n_tracks == 0) {
        for (int m = 0; m < b->n_maps; ++m) {
            results[m].kernel_used = plan.kernel; results[m].max_snr = -INFINITY; results[m].max_snr_f64 = -INFINITY;
        }
        if (p->n_bins > 0) memset(p->hist_out, 0, sizeof(uint64_t) * (size_t)p->n_bins * (size_t)b->n_maps);
        return ST_OK;
    }
    if (!c->h_bres) ST_CUDA(c, cudaHostAlloc((void**)&c->h_bres, (size_t)ST_BATCH_GROUP * sizeof(st::DeviceResult), cudaHostAllocDefault));
    if (p->n_bins > 0 && !c->h_bhist)
        ST_CUDA(c, cudaHostAlloc((void**)&c->h_bhist, (size_t)ST_BATCH_GROUP * ST_MAX_BINS * sizeof(unsigned long long), cudaHostAllocDefault));
    if (b->host_buffers) {
        if (!c->copy_stream) ST_CUDA(c, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            if (!c->ev_copied[i]) ST_CUDA(c, cudaEventCreateWithFlags(&c->ev_copied[i], cudaEventDisableTiming));
            if (!c->ev_consumed[i]) ST_CUDA(c, cudaEventCreateWithFlags(&c->ev_consumed[i], cudaEventDisableTiming));
        }
    }
    int n_launches_tables = 0;
    rc = ensure_tables(c, p, plan, &n_launches_tables);
    if (rc) return rc;
    const size_t n_pix = (size_t)c->n_t * (size_t)c->n_f;
    const size_t n_sig = b->sigma_kind == ST_SIGMA_NONE ? 0 : b->sigma_kind == ST_SIGMA_PER_FREQ ? (size_t)c->n_f : n_pix;
    void* stage_csd[2] = {at<void>(c, c->L.stage_csd), at<void>(c, c->L.stage_csd2)};
    float* stage_sig[2] = {at<float>(c, c->L.stage_sigma), at<float>(c, c->L.stage_sigma2)};
    // host buffers: copy of map m goes to staging pair m % 2 on the copy stream, once the prepare
    // kernel of map m - 2 (which read that pair) has run
    auto enqueue_copy = [&](int m) -> int {
        const int sb = m & 1;
        if (m >= 2) ST_CUDA(c, cudaStreamWaitEvent(c->copy_stream, c->ev_consumed[sb], 0));
        ST_CUDA(c, cudaMemcpyAsync(stage_csd[sb], b->csd[m], n_pix * sizeof(float2), cudaMemcpyHostToDevice, c->copy_stream));
        if (n_sig) ST_CUDA(c, cudaMemcpyAsync(stage_sig[sb], b->sigma[m], n_sig * sizeof(float), cudaMemcpyHostToDevice, c->copy_stream));
        ST_CUDA(c, cudaEventRecord(c->ev_copied[sb], c->copy_stream));
        return ST_OK;
    };
    ST_CUDA(c, cudaEventRecord(c->ev0, c->stream));
    if (b->host_buffers) {
        // the copy stream must not run ahead of work already queued on the caller's stream
        ST_CUDA(c, cudaStreamWaitEvent(c->copy_stream, c->ev0, 0));
        rc = enqueue_copy(0);
        if (rc) return rc;
    }
    st_search_params pm = *p;
    // the batch knows its norm before S0: the 1 / sigma plane is written only for the statistic that reads it
    // (afterwards the context's map is the last one, without the plane: a later INVVAR search gets ST_ESTATE)
    const bool want_isig = p->norm == ST_NORM_INVVAR;
    for (int g0 = 0; g0 < b->n_maps; g0 += ST_BATCH_GROUP) {
        const int g1 = g0 + ST_BATCH_GROUP < b->n_maps ? g0 + ST_BATCH_GROUP : b->n_maps;
        std::vector<int> launches((size_t)(g1 - g0), 0), bank_modes((size_t)(g1 - g0), 0);
        for (int m = g0; m < g1; ++m) {
            const int sb = m & 1;
            if (b->host_buffers) {
                if (m + 1 < b->n_maps) { rc = enqueue_copy(m + 1); if (rc) return rc; }
                ST_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_copied[sb], 0));
                rc = set_map_impl(c, stage_csd[sb], stage_sig[sb], b->sigma_kind, want_isig);
                if (rc) return rc;
                ST_CUDA(c, cudaEventRecord(c->ev_consumed[sb], c->stream));
            } else {
                rc = set_map_impl(c, b->csd[m], b->sigma_kind != ST_SIGMA_NONE ? b->sigma[m] : nullptr, b->sigma_kind, want_isig);
                if (rc) return rc;
            }
            pm.seed = b->seeds ? b->seeds[m] : p->seed;
            int nl = 1;                            // k_prepare_map
            rc = enqueue_search(c, &pm, plan, batch_slots(c, m - g0), &nl, false);
            if (rc) return rc;
            launches[(size_t)(m - g0)] = nl;
            bank_modes[(size_t)(m - g0)] = c->last_bank_mode;
        }
        ST_CUDA(c, cudaMemcpyAsync(c->h_bres, at<void>(c, c->L.b_result), (size_t)(g1 - g0) * sizeof(st::DeviceResult),
                                   cudaMemcpyDeviceToHost, c->stream));
        if (p->n_bins > 0)
            ST_CUDA(c, cudaMemcpyAsync(c->h_bhist, at<void>(c, c->L.b_hist),
                                       (size_t)(g1 - g0) * ST_MAX_BINS * sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream));
        if (g1 == b->n_maps) ST_CUDA(c, cudaEventRecord(c->ev1, c->stream));
        ST_CUDA(c, cudaStreamSynchronize(c->stream));
        for (int m = g0; m < g1; ++m) {
            fill_result(&results[m], c->h_bres[m - g0], n_tau, plan.kernel, launches[(size_t)(m - g0)] + (m == 0 ? n_launches_tables : 0));
            results[m].flags |= bank_modes[(size_t)(m - g0)] == 2 ? ST_FLAG_BANK_READ : (bank_modes[(size_t)(m - g0)] == 1 ? ST_FLAG_BANK_FILLED : 0);
            if (p->n_bins > 0)
                for (int k = 0; k < p->n_bins; ++k)
                    p->hist_out[(size_t)m * (size_t)p->n_bins + (size_t)k] = (uint64_t)c->h_bhist[(size_t)(m - g0) * ST_MAX_BINS + (size_t)k];
        }
    }
    if (gpu_ms_total) ST_CUDA(c, cudaEventElapsedTime(gpu_ms_total, c->ev0, c->ev1));
    return ST_OK;
}

size_t st_ftmap_scratch_bytes(const st_ctx* c, int32_t seg_len)
{
    if (!c || seg_len < 64 || seg_len > st::kFtMaxLen || (seg_len & (seg_len - 1))) return 0;
    const size_t n_pix = (size_t)c->n_t * (size_t)c->n_f;
    return 2 * align_up(n_pix * sizeof(double2)) + align_up((size_t)(seg_len / 2) * sizeof(double2));
}

// F1 + F2 of the ft-map construction: validation, twiddles, one FFT per segment.  On success the
// scratch holds s~_I, s~_J; k_ft_normalise (any shift) can follow.
static int ft_spectra(st_ctx* c, const double* s_i, const double* s_j, int64_t n_samples, const st_ftmap_params* fp,
                      void* scratch, size_t scratch_bytes, double2** st_i_out, double2** st_j_out)
{
    if (!c->have_ws) return fail(c, ST_ESTATE, "no workspace: call st_set_workspace first");
    if (!s_i || !s_j || !fp || !scratch) return fail(c, ST_EINVAL, "NULL argument");
    const int L = fp->seg_len;
    if (L < 64 || L > st::kFtMaxLen || (L & (L - 1))) return fail(c, ST_EINVAL, "seg_len %d must be a power of two in [64, %d]", L, st::kFtMaxLen);
    if (!(fp->fs > 0.0) || !isfinite(fp->fs)) return fail(c, ST_EINVAL, "bad sample rate");
    if (fp->n_neighbours < 1) return fail(c, ST_EINVAL, "n_neighbours must be >= 1");
    const double df = fp->fs / (double)L;
    if (fabs(df - c->df) > 1e-9 * c->df) return fail(c, ST_EINVAL, "fs / seg_len = %g Hz differs from the context's df = %g Hz", df, c->df);
    const double kf = c->f_min / df;
    const int k_lo = (int)llround(kf);
    if (fabs(kf - (double)k_lo) > 1e-9) return fail(c, ST_EINVAL, "f_min %g is not a multiple of df %g", c->f_min, df);
    if (k_lo + c->n_f > L / 2) return fail(c, ST_EINVAL, "the band ends above the Nyquist frequency");
    if (n_samples < (int64_t)(c->n_t + 1) * (int64_t)(L / 2)) return fail(c, ST_EINVAL, "%lld samples hold fewer than n_t = %d segments", (long long)n_samples, c->n_t);
    if (((uintptr_t)scratch % kAlign) != 0) return fail(c, ST_EINVAL, "scratch must be 256-byte aligned");
    if (scratch_bytes < st_ftmap_scratch_bytes(c, L)) return fail(c, ST_ENOSPC, "scratch of %zu bytes is below %zu", scratch_bytes, st_ftmap_scratch_bytes(c, L));
    const size_t n_pix = (size_t)c->n_t * (size_t)c->n_f;
    double2* st_i = (double2*)scratch;
    double2* st_j = (double2*)((unsigned char*)scratch + align_up(n_pix * sizeof(double2)));
    double2* W = (double2*)((unsigned char*)scratch + 2 * align_up(n_pix * sizeof(double2)));
    int log2L = 0;
    while ((1 << log2L) < L) ++log2L;
    st::k_ft_twiddles<<<(L / 2 + 255) / 256, 256, 0, c->stream>>>(L, W);
    ST_CUDA(c, cudaGetLastError());
    const size_t smem = (size_t)L * sizeof(double2);
    int rc = set_smem(c, st::k_ft_segments, smem);
    if (rc) return rc;
    st::k_ft_segments<<<c->n_t, st::kFtThreads, smem, c->stream>>>(s_i, s_j, L, log2L, W, k_lo, c->n_f, st_i, st_j);
    ST_CUDA(c, cudaGetLastError());
    *st_i_out = st_i; *st_j_out = st_j;
    return ST_OK;
}

// F3 + F4 for one time shift (0 = the zero-lag map) into the context's map.
static int ft_normalise(st_ctx* c, const double2* st_i, const double2* st_j, int n_nb, int shift)
{
    const size_t n_pix = (size_t)c->n_t * (size_t)c->n_f;
    const int blocks = (int)((n_pix + 255) / 256 < (size_t)(8 * c->n_sm) ? (n_pix + 255) / 256 : (size_t)(8 * c->n_sm));
    st::k_ft_normalise<<<blocks, 256, 0, c->stream>>>(st_i, st_j, c->n_t, c->n_f, n_nb, shift, at<float2>(c, c->L.map));
    ST_CUDA(c, cudaGetLastError());
    c->have_map = true; c->have_isig = false;      // the ft-map path forms p directly: no sigma plane
    return ST_OK;
}

int st_set_map_from_strain(st_ctx* c, const double* s_i, const double* s_j, int64_t n_samples,
                           const st_ftmap_params* fp, void* scratch, size_t scratch_bytes)
{
    DevGuard dev_guard(c);
    if (!c) return ST_EINVAL;
    double2 *st_i = nullptr, *st_j = nullptr;
    int rc = ft_spectra(c, s_i, s_j, n_samples, fp, scratch, scratch_bytes, &st_i, &st_j);
    if (rc) return rc;
    return ft_normalise(c, st_i, st_j, fp->n_neighbours, 0);
}

static int timeshifts_impl(st_ctx* c, const double* s_i, const double* s_j, int64_t n_samples, const st_ftmap_params* fp,
                           void* scratch, size_t scratch_bytes, int32_t n_shifts, const int32_t* shifts,
                           const uint64_t* seeds, const st_search_params* p, st_result* results, float* gpu_ms_total);

int st_search_timeshifts(st_ctx* c, const double* s_i, const double* s_j, int64_t n_samples, const st_ftmap_params* fp,
                         void* scratch, size_t scratch_bytes, int32_t n_shifts, const int32_t* shifts,
                         const uint64_t* seeds, const st_search_params* p, st_result* results, float* gpu_ms_total)
{
    DevGuard dev_guard(c);
    return drop_bank_on_error(c, timeshifts_impl(c, s_i, s_j, n_samples, fp, scratch, scratch_bytes, n_shifts, shifts, seeds, p,
                                                 results, gpu_ms_total));
}

static int timeshifts_impl(st_ctx* c, const double* s_i, const double* s_j, int64_t n_samples, const st_ftmap_params* fp,
                           void* scratch, size_t scratch_bytes, int32_t n_shifts, const int32_t* shifts,
                           const uint64_t* seeds, const st_search_params* p, st_result* results, float* gpu_ms_total)
{
    int rc = validate(c, p, false);
    if (rc) return rc;
    // the maps of this call come from strain (k_ft_normalise writes p only): there is no per-pixel sigma to weight by
    if (p->norm == ST_NORM_INVVAR)
        return fail(c, ST_EINVAL, "ST_NORM_INVVAR is not available for maps built from strain (no 1 / sigma plane): use ST_NORM_SQRT_N");
    if (!results || !shifts) return fail(c, ST_EINVAL, "shifts / results is NULL");
    if (n_shifts < 1) return fail(c, ST_EINVAL, "n_shifts must be >= 1");
    for (int m = 0; m < n_shifts; ++m)
        if (shifts[m] < 0 || shifts[m] >= c->n_t) return fail(c, ST_EINVAL, "shifts[%d] = %d outside [0, n_t)", m, shifts[m]);
    if (p->n_bins > 0 && !p->hist_out) return fail(c, ST_EINVAL, "n_bins > 0 but hist_out is NULL");
    Plan plan;
    rc = make_plan(c, p, &plan);
    if (rc) return rc;
    const int n_tau = p->tau_mode == ST_TAU_GRID ? p->n_tau : 1;
    if (gpu_ms_total) *gpu_ms_total = 0.0f;
    memset(results, 0, sizeof(st_result) * (size_t)n_shifts);
    if (!c->h_bres) ST_CUDA(c, cudaHostAlloc((void**)&c->h_bres, (size_t)ST_BATCH_GROUP * sizeof(st::DeviceResult), cudaHostAllocDefault));
    if (p->n_bins > 0 && !c->h_bhist)
        ST_CUDA(c, cudaHostAlloc((void**)&c->h_bhist, (size_t)ST_BATCH_GROUP * ST_MAX_BINS * sizeof(unsigned long long), cudaHostAllocDefault));
    ST_CUDA(c, cudaEventRecord(c->ev0, c->stream));
    double2 *st_i = nullptr, *st_j = nullptr;
    rc = ft_spectra(c, s_i, s_j, n_samples, fp, scratch, scratch_bytes, &st_i, &st_j);      // once for every shift
    if (rc) return rc;
    if (p->n_tracks == 0) {
        for (int m = 0; m < n_shifts; ++m) {
            results[m].kernel_used = plan.kernel; results[m].max_snr = -INFINITY; results[m].max_snr_f64 = -INFINITY;
        }
        if (p->n_bins > 0) memset(p->hist_out, 0, sizeof(uint64_t) * (size_t)p->n_bins * (size_t)n_shifts);
        return ft_normalise(c, st_i, st_j, fp->n_neighbours, shifts[n_shifts - 1]);
    }
    int n_launches_tables = 2;                        // k_ft_twiddles, k_ft_segments
    rc = ensure_tables(c, p, plan, &n_launches_tables);
    if (rc) return rc;
    st_search_params pm = *p;
    for (int g0 = 0; g0 < n_shifts; g0 += ST_BATCH_GROUP) {
        const int g1 = g0 + ST_BATCH_GROUP < n_shifts ? g0 + ST_BATCH_GROUP : n_shifts;
        std::vector<int> launches((size_t)(g1 - g0), 0), bank_modes((size_t)(g1 - g0), 0);
        for (int m = g0; m < g1; ++m) {
            rc = ft_normalise(c, st_i, st_j, fp->n_neighbours, shifts[m]);
            if (rc) return rc;
            pm.seed = seeds ? seeds[m] : p->seed;
            int nl = 1;                               // k_ft_normalise
            rc = enqueue_search(c, &pm, plan, batch_slots(c, m - g0), &nl, false);
            if (rc) return rc;
            launches[(size_t)(m - g0)] = nl;
            bank_modes[(size_t)(m - g0)] = c->last_bank_mode;
        }
        ST_CUDA(c, cudaMemcpyAsync(c->h_bres, at<void>(c, c->L.b_result), (size_t)(g1 - g0) * sizeof(st::DeviceResult),
                                   cudaMemcpyDeviceToHost, c->stream));
        if (p->n_bins > 0)
            ST_CUDA(c, cudaMemcpyAsync(c->h_bhist, at<void>(c, c->L.b_hist),
                                       (size_t)(g1 - g0) * ST_MAX_BINS * sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream));
        if (g1 == n_shifts) ST_CUDA(c, cudaEventRecord(c->ev1, c->stream));
        ST_CUDA(c, cudaStreamSynchronize(c->stream));
        for (int m = g0; m < g1; ++m) {
            fill_result(&results[m], c->h_bres[m - g0], n_tau, plan.kernel, launches[(size_t)(m - g0)] + (m == 0 ? n_launches_tables : 0));
            results[m].flags |= bank_modes[(size_t)(m - g0)] == 2 ? ST_FLAG_BANK_READ : (bank_modes[(size_t)(m - g0)] == 1 ? ST_FLAG_BANK_FILLED : 0);
            if (p->n_bins > 0)
                for (int k = 0; k < p->n_bins; ++k)
                    p->hist_out[(size_t)m * (size_t)p->n_bins + (size_t)k] = (uint64_t)c->h_bhist[(size_t)(m - g0) * ST_MAX_BINS + (size_t)k];
        }
    }
    if (gpu_ms_total) ST_CUDA(c, cudaEventElapsedTime(gpu_ms_total, c->ev0, c->ev1));
    return ST_OK;
}

int st_debug_get_map(st_ctx* c, void* p_out_dev)
{
    DevGuard dev_guard(c);
    if (!c) return ST_EINVAL;
    if (!c->have_ws || !c->have_map) return fail(c, ST_ESTATE, "no map");
    if (!p_out_dev) return fail(c, ST_EINVAL, "output is NULL");
    ST_CUDA(c, cudaMemcpyAsync(p_out_dev, at<void>(c, c->L.map), (size_t)c->n_t * (size_t)c->n_f * sizeof(float2),
                               cudaMemcpyDeviceToDevice, c->stream));
    return ST_OK;
}

int st_track_params_family(const st_ctx* c, uint64_t seed, uint64_t track_id, int32_t n_min, int32_t n_max,
                           double tau_lo, double tau_hi, int32_t family, st_track* out)
{
    if (!c || !out) return ST_EINVAL;
    if (n_min < 1 || n_max < n_min || n_max > c->n_t) return ST_EINVAL;
    if (family != ST_FAMILY_QUADRATIC && family != ST_FAMILY_CUBIC && family != ST_FAMILY_CHIRP) return ST_EINVAL;
    st::BankParams bp;
    bp.seed = seed; bp.n_t = c->n_t; bp.n_f = c->n_f; bp.n_min = n_min; bp.n_max = n_max;
    bp.tau_lo = tau_lo; bp.tau_hi = tau_hi; bp.family = family; bp.pad = 0;
    const st::Track t = st::make_track(bp, track_id);
    out->N = t.N; out->j0 = t.j0; out->a = t.a; out->y0 = t.y0; out->y1 = t.y1; out->y2 = t.y2; out->tau = t.tau;
    out->y3 = t.y3;
    return ST_OK;
}

int st_track_params(const st_ctx* c, uint64_t seed, uint64_t track_id, int32_t n_min, int32_t n_max,
                    double tau_lo, double tau_hi, st_track* out)
{
    return st_track_params_family(c, seed, track_id, n_min, n_max, tau_lo, tau_hi, ST_FAMILY_QUADRATIC, out);
}

int st_debug_track_words(uint64_t seed, uint64_t track_id, uint32_t* out_host)
{
    if (!out_host) return ST_EINVAL;
    const st::Words8 w = st::track_words(seed, track_id);
    for (int i = 0; i < 8; ++i) out_host[i] = w.r[i];
    return ST_OK;
}

int st_debug_rasterise(st_ctx* c, const st_search_params* p, uint64_t first, uint64_t count,
                       int32_t* k_out_dev, int32_t* j0_dev, int32_t* N_dev)
{
    DevGuard dev_guard(c);
    if (!c) return ST_EINVAL;
    if (!p) return fail(c, ST_EINVAL, "params is NULL");
    if (!c->have_ws) return fail(c, ST_ESTATE, "no workspace: call st_set_workspace first");
    if (p->n_min < 1 || p->n_max < p->n_min || p->n_max > c->n_t) return fail(c, ST_EINVAL, "need 1 <= n_min <= n_max <= n_t");
    if (p->family != ST_FAMILY_QUADRATIC && p->family != ST_FAMILY_CUBIC && p->family != ST_FAMILY_CHIRP) return fail(c, ST_EINVAL, "bad template family %d", p->family);
    if (!k_out_dev || !j0_dev || !N_dev) return fail(c, ST_EINVAL, "output pointer is NULL");
    if (count == 0) return ST_OK;
    const uint64_t need = (count + 7) / 8;
    const unsigned blocks = (unsigned)(need < (uint64_t)(c->n_sm * 8) ? need : (uint64_t)(c->n_sm * 8));
    st::k_debug_rasterise<<<blocks, 256, 0, c->stream>>>(bank(c, p), first, count, k_out_dev, j0_dev, N_dev);
    ST_CUDA(c, cudaGetLastError());
    return ST_OK;
}

int st_debug_rasterise_track(st_ctx* c, const st_track* t, int32_t family, int32_t* k_out_dev)
{
    DevGuard dev_guard(c);
    if (!c) return ST_EINVAL;
    if (!t || !k_out_dev) return fail(c, ST_EINVAL, "NULL argument");
    if (family != ST_FAMILY_QUADRATIC && family != ST_FAMILY_CUBIC && family != ST_FAMILY_CHIRP) return fail(c, ST_EINVAL, "bad template family %d", family);
    if (const char* why = explicit_track_problem(c, *t, family)) return fail(c, ST_EINVAL, "track %s", why);
    if (!c->have_ws) return fail(c, ST_ESTATE, "no workspace: call st_set_workspace first");
    st::Track d;
    d.N = t->N; d.j0 = t->j0; d.a = t->a; d.y0 = t->y0; d.y1 = t->y1; d.y2 = t->y2; d.tau = t->tau; d.y3 = t->y3;
    st::k_debug_rasterise_track<<<(t->N + 127) / 128, 128, 0, c->stream>>>(d, c->n_f, family, k_out_dev);
    ST_CUDA(c, cudaGetLastError());
    return ST_OK;
}

int st_debug_rasterise_random(st_ctx* c, const st_search_params* p, uint64_t first, uint64_t count,
                              int32_t* k_out_dev, int32_t* j0_dev, int32_t* N_dev)
{
    DevGuard dev_guard(c);
    int rc = validate(c, p, true);
    if (rc) return rc;
    if (p->tau_mode != ST_TAU_RANDOM) return fail(c, ST_EINVAL, "st_debug_rasterise_random needs ST_TAU_RANDOM");
    if (!k_out_dev || !j0_dev || !N_dev) return fail(c, ST_EINVAL, "output pointer is NULL");
    if (count == 0) return ST_OK;
    if (count > kMaxSamplesPerLaunch) return fail(c, ST_EINVAL, "count too large for one debug launch");
    Plan plan;
    rc = make_plan(c, p, &plan);
    if (rc) return rc;
    rc = reset_search_state(c, 0, own_slots(c));
    if (rc) return rc;
    ST_CUDA(c, cudaMemsetAsync(k_out_dev, 0xFF, (size_t)count * (size_t)c->n_t * sizeof(int32_t), c->stream));   // -1 beyond N
    st::ScoreArgs a = base_args(c, p);
    a.track_offset = first; a.n_tracks = count;
    a.k_dump = k_out_dev; a.j0_dump = j0_dev; a.N_dump = N_dev;
    return launch_score(c, plan, a, p->n_max);
}

int st_score_tracks(st_ctx* c, const st_search_params* p, const st_track* tracks, int32_t count, float* snr_dev)
{
    DevGuard dev_guard(c);
    if (!c) return ST_EINVAL;
    if (!p) return fail(c, ST_EINVAL, "params is NULL");
    if (!tracks || !snr_dev) return fail(c, ST_EINVAL, "tracks / snr_dev is NULL");
    if (count < 0 || count > ST_MAX_SCORE_TRACKS) return fail(c, ST_EINVAL, "count %d outside [0, %d]", count, ST_MAX_SCORE_TRACKS);
    if (count == 0) return ST_OK;
    if (p->family != ST_FAMILY_QUADRATIC && p->family != ST_FAMILY_CUBIC && p->family != ST_FAMILY_CHIRP) return fail(c, ST_EINVAL, "bad template family %d", p->family);
    st_search_params q = *p;                         // the durations come from the list, not from params
    q.n_min = c->n_t; q.n_max = 1; q.n_tracks = (uint64_t)count; q.track_offset = 0; q.n_bins = 0; q.hist_out = nullptr;
    std::vector<st::Track> h((size_t)count);
    for (int i = 0; i < count; ++i) {
        const st_track& t = tracks[i];
        if (const char* why = explicit_track_problem(c, t, p->family)) return fail(c, ST_EINVAL, "tracks[%d] %s", i, why);
        h[(size_t)i].N = t.N; h[(size_t)i].j0 = t.j0; h[(size_t)i].a = t.a;
        h[(size_t)i].y0 = t.y0; h[(size_t)i].y1 = t.y1; h[(size_t)i].y2 = t.y2; h[(size_t)i].tau = t.tau;
        h[(size_t)i].y3 = t.y3;
        if (t.N < q.n_min) q.n_min = t.N;
        if (t.N > q.n_max) q.n_max = t.N;
    }
    int rc = validate(c, &q, true);
    if (rc) return rc;
    Plan plan;
    rc = make_plan(c, &q, &plan);
    if (rc) return rc;
    int n_launches = 0;
    rc = ensure_tables(c, &q, plan, &n_launches);
    if (rc) return rc;
    rc = reset_search_state(c, 0, own_slots(c));
    if (rc) return rc;
    st::Track* d_tracks = at<st::Track>(c, c->L.tracks);
    ST_CUDA(c, cudaMemcpyAsync(d_tracks, h.data(), (size_t)count * sizeof(st::Track), cudaMemcpyHostToDevice, c->stream));
    st::ScoreArgs a = base_args(c, &q);
    a.track_offset = 0; a.n_tracks = (uint64_t)count; a.dump = snr_dev; a.tracks = d_tracks;
    rc = launch_score(c, plan, a, q.n_max);
    if (rc) return rc;
    ST_CUDA(c, cudaStreamSynchronize(c->stream));    // the pageable staging vector goes out of scope
    return ST_OK;
}

int st_debug_scores(st_ctx* c, const st_search_params* p, uint64_t first, uint64_t count, float* snr_dev)
{
    DevGuard dev_guard(c);
    int rc = validate(c, p, true);
    if (rc) return rc;
    if (!snr_dev) return fail(c, ST_EINVAL, "snr_dev is NULL");
    if (count == 0) return ST_OK;
    Plan plan;
    rc = make_plan(c, p, &plan);
    if (rc) return rc;
    const int n_tau = p->tau_mode == ST_TAU_GRID ? p->n_tau : 1;
    if (count > kMaxSamplesPerLaunch / (uint64_t)n_tau || count > kDeferCap) return fail(c, ST_EINVAL, "count too large for one debug launch");
    int n_launches = 0;
    rc = ensure_tables(c, p, plan, &n_launches);
    if (rc) return rc;
    rc = reset_search_state(c, 0, own_slots(c));
    if (rc) return rc;
    st::ScoreArgs a = base_args(c, p);
    a.track_offset = first; a.n_tracks = count; a.dump = snr_dev;
    return launch_score(c, plan, a, p->n_max);
}

}  // extern "C"

// S4 across runs: host only.
extern "C" int st_combine_results(const st_result* results, const uint64_t* const* hists, int32_t n, int32_t n_bins,
                                  st_result* out, uint64_t* hist_out, int32_t* best_index)
{
    if (!results || !out || n < 1 || n_bins < 0 || n_bins > ST_MAX_BINS) return ST_EINVAL;
    if (hist_out && !hists) return ST_EINVAL;
    int best = -1;
    for (int i = 0; i < n; ++i) {
        const st_result& r = results[i];
        if (r.n_evals == 0) continue;                                  // a run that scored nothing has no maximum
        if (best < 0) { best = i; continue; }
        const st_result& b = results[best];
        // G12: larger float64 SNR, then smaller template id, then smaller delay index
        const bool wins = r.max_snr_f64 != b.max_snr_f64 ? r.max_snr_f64 > b.max_snr_f64
                        : r.arg_track != b.arg_track     ? r.arg_track < b.arg_track
                                                         : r.arg_tau_index < b.arg_tau_index;
        if (wins) best = i;
    }
    st_result c = results[best < 0 ? 0 : best];
    if (best >= 0) {
        c.n_evals = 0; c.n_pixels = 0; c.n_candidates = 0; c.n_launches = 0; c.n_deferred = 0; c.flags = 0; c.gpu_ms = 0.0f;
        for (int i = 0; i < n; ++i) {
            const st_result& r = results[i];
            c.n_evals += r.n_evals; c.n_pixels += r.n_pixels; c.n_launches += r.n_launches; c.flags |= r.flags;
            if (r.gpu_ms > c.gpu_ms) c.gpu_ms = r.gpu_ms;
            if (r.n_evals == 0) continue;
            c.n_candidates += r.n_candidates; c.n_deferred += r.n_deferred;
            if (r.max_snr > c.max_snr) c.max_snr = r.max_snr;
        }
    }
    if (hist_out) {
        for (int b = 0; b < n_bins; ++b) hist_out[b] = 0;
        for (int i = 0; i < n; ++i)
            if (hists[i])
                for (int b = 0; b < n_bins; ++b) hist_out[b] += hists[i][b];
    }
    *out = c;
    if (best_index) *best_index = best < 0 ? 0 : best;
    return ST_OK;
}

// ================================================= entry point without allocations ====
// st_score_random_noalloc (include/stochtrack.h): S0-S3 in the paper's one-delay-per-template mode
// for hosts that cannot hand the library a workspace -- a framework's pool owns the whole
// card, or nothing may be allocated while the analysis is live, or the component only ever sees its input
// and output buffers.  The kernels are the library's own k_prepare_map and k_score_random<false, false, false>,
// launched as st_set_map + st_debug_scores launch them; the only difference is where their scratch lives.
//
// g_noalloc_scratch is that scratch: a static __device__ array, so it is part of the library's device image
// and every GPU that loads the image carries these ST_NOALLOC_SCRATCH_BYTES until the process ends.  In HOST
// code the name `g_noalloc_scratch` is only a handle for the symbol look-up -- it is not a device address and
// must never be passed to a kernel or to cudaMemset; noalloc_device() asks the runtime for the real address
// once per device, with that device current, and every use below goes through that pointer.
namespace {

constexpr uint32_t kNaCandCap = 4096;                   // near-max records (not read back: the scores are the output)
constexpr size_t kNaOffScalars  = 0;                                                                    // st::Scalars
constexpr size_t kNaOffWarpBest = 256;                                                                  // [kWarpSlots]
constexpr size_t kNaOffCand     = kNaOffWarpBest + (size_t)kWarpSlots * sizeof(st::WarpBest);           // [kNaCandCap]
constexpr size_t kNaOffMap      = kNaOffCand + (size_t)kNaCandCap * sizeof(st::Cand);                   // p, float2 per pixel
constexpr size_t kNaOffIsig     = kNaOffMap + (size_t)ST_NOALLOC_MAX_PIXELS * sizeof(float2);           // 1 / sigma per pixel
constexpr size_t kNaTotal       = kNaOffIsig + (size_t)ST_NOALLOC_MAX_PIXELS * sizeof(float);
constexpr size_t kNaZeroed      = kNaOffCand;           // [0, kNaZeroed): what a call needs to find zeroed
static_assert(sizeof(st::Scalars) <= kNaOffWarpBest, "scalars outgrew their slot");
static_assert(kNaOffCand % kAlign == 0 && kNaOffMap % kAlign == 0 && kNaOffIsig % kAlign == 0, "scratch parts must stay 256-byte aligned");
static_assert(kNaTotal == ST_NOALLOC_SCRATCH_BYTES, "include/stochtrack.h states the size of the static scratch");

static __device__ __align__(256) unsigned char g_noalloc_scratch[kNaTotal];

constexpr int kNaMaxDevices = 64;
struct NoallocDevice { bool ready; unsigned char* scratch; int n_sm; };
NoallocDevice g_na_dev[kNaMaxDevices];                  // zero-initialised: nothing looked up yet
std::mutex g_na_mutex;

int na_fail(char* err, size_t len, int code, const char* fmt, ...)
{
    if (err && len) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(err, len, fmt, ap);
        va_end(ap);
    }
    return code;
}

// Set-up, once per device, on that device's first call (which therefore belongs at start-up, before any
// stream capture): the device must be current for cudaGetSymbolAddress to return ITS copy of the array.
int noalloc_device(int dev, NoallocDevice* out, char* err, size_t len)
{
    std::lock_guard<std::mutex> lock(g_na_mutex);
    NoallocDevice& d = g_na_dev[dev];
    if (!d.ready) {
        void* ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);
        if (e != cudaSuccess || !ptr)
            return na_fail(err, len, ST_ECUDA, "cudaGetSymbolAddress(static scratch) on device %d: %s", dev, cudaGetErrorString(e));
        int n_sm = 0;
        e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess || n_sm < 1)
            return na_fail(err, len, ST_ECUDA, "cudaDeviceGetAttribute(SM count) on device %d: %s", dev, cudaGetErrorString(e));
        d.scratch = static_cast<unsigned char*>(ptr); d.n_sm = n_sm; d.ready = true;
    }
    *out = d;
    return ST_OK;
}

}  // namespace

extern "C" int st_score_random_noalloc(const void* csd_dev, const float* sigma_dev, int32_t sigma_kind,
                                       int32_t n_t, int32_t n_f, double df, double f_min,
                                       const st_search_params* p, float* snr_dev, void* cuda_stream,
                                       char* err, size_t len)
{
    if (err && len) err[0] = 0;
    // ---- host-side checks, before any CUDA call
    if (!p) return na_fail(err, len, ST_EINVAL, "params is NULL");
    if (n_t < 1 || n_t > ST_MAX_N_T || n_f < 1 || n_f > ST_MAX_N_F)
        return na_fail(err, len, ST_EINVAL, "map shape %d x %d outside [1, %d] x [1, %d]", n_t, n_f, ST_MAX_N_T, ST_MAX_N_F);
    if (!(df > 0.0) || !(f_min >= 0.0) || !isfinite(df) || !isfinite(f_min))
        return na_fail(err, len, ST_EINVAL, "need df > 0 and f_min >= 0, both finite");
    const size_t n_pix = (size_t)n_t * (size_t)n_f;
    if (n_pix > (size_t)ST_NOALLOC_MAX_PIXELS)
        return na_fail(err, len, ST_ENOSPC, "map of %d x %d = %zu pixels exceeds ST_NOALLOC_MAX_PIXELS = %d, the size the library's "
                       "static scratch was compiled for: use st_set_workspace / st_search with a workspace of your own", n_t, n_f, n_pix,
                       ST_NOALLOC_MAX_PIXELS);
    if (!csd_dev) return na_fail(err, len, ST_EINVAL, "csd is NULL");
    if (sigma_kind < ST_SIGMA_NONE || sigma_kind > ST_SIGMA_PER_PIXEL) return na_fail(err, len, ST_EINVAL, "bad sigma_kind %d", sigma_kind);
    if (sigma_kind != ST_SIGMA_NONE && !sigma_dev) return na_fail(err, len, ST_EINVAL, "sigma is NULL");
    if (p->n_min < 1 || p->n_max < p->n_min || p->n_max > n_t)
        return na_fail(err, len, ST_EINVAL, "need 1 <= n_min <= n_max <= n_t (got %d, %d, n_t %d)", p->n_min, p->n_max, n_t);
    if (p->tau_mode != ST_TAU_RANDOM) return na_fail(err, len, ST_EINVAL, "only ST_TAU_RANDOM (one delay per template) is offered without a workspace");
    if (!isfinite(p->tau_lo) || !isfinite(p->tau_hi) || p->tau_hi < p->tau_lo) return na_fail(err, len, ST_EINVAL, "bad random-tau range");
    if (p->norm != ST_NORM_SQRT_N && p->norm != ST_NORM_MEAN) return na_fail(err, len, ST_EINVAL, "norm %d: only ST_NORM_SQRT_N / ST_NORM_MEAN here", p->norm);
    if (p->family != ST_FAMILY_QUADRATIC) return na_fail(err, len, ST_EINVAL, "family %d: only ST_FAMILY_QUADRATIC here", p->family);
    if (p->track_offset > (1ull << 62)) return na_fail(err, len, ST_EINVAL, "track_offset too large");
    if (p->n_tracks > kMaxSamplesPerLaunch) return na_fail(err, len, ST_EINVAL, "n_tracks %llu exceeds one launch (2^31): split the range",
                                                           (unsigned long long)p->n_tracks);
    if (p->n_tracks == 0) return ST_OK;
    if (!snr_dev) return na_fail(err, len, ST_EINVAL, "snr_dev is NULL");
    // ---- the current device's copy of the static scratch
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return na_fail(err, len, ST_ECUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= kNaMaxDevices) return na_fail(err, len, ST_EINVAL, "device ordinal %d beyond the %d this entry point keeps track of", dev, kNaMaxDevices);
    NoallocDevice d;
    int rc = noalloc_device(dev, &d, err, len);
    if (rc) return rc;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    st::Scalars* sc = reinterpret_cast<st::Scalars*>(d.scratch + kNaOffScalars);
    float2* map = reinterpret_cast<float2*>(d.scratch + kNaOffMap);
    float* isig = reinterpret_cast<float*>(d.scratch + kNaOffIsig);
    // The array still holds the previous call's counter, maximum and per-warp records: those must read zero.
    // The map and 1 / sigma planes need no clearing: S0 below rewrites every pixel this call will gather.
    e = cudaMemsetAsync(d.scratch, 0, kNaZeroed, stream);
    if (e != cudaSuccess) return na_fail(err, len, ST_ECUDA, "cudaMemsetAsync(static scratch): %s", cudaGetErrorString(e));
    // ---- S0 (Eq. 7), as st_set_map launches it
    {
        const int blocks = (int)((n_pix + 255) / 256 < (size_t)(8 * d.n_sm) ? (n_pix + 255) / 256 : (size_t)(8 * d.n_sm));
        const bool vec = (n_pix % 2 == 0) && ((uintptr_t)csd_dev % 16 == 0) &&
                         (sigma_kind != ST_SIGMA_PER_PIXEL || (uintptr_t)sigma_dev % 8 == 0);
        if (vec) st::k_prepare_map<true><<<blocks, 256, 0, stream>>>((const float2*)csd_dev, sigma_dev, sigma_kind, n_f, n_pix, map, isig);
        else st::k_prepare_map<false><<<blocks, 256, 0, stream>>>((const float2*)csd_dev, sigma_dev, sigma_kind, n_f, n_pix, map, isig);
        e = cudaGetLastError();
        if (e != cudaSuccess) return na_fail(err, len, ST_ECUDA, "k_prepare_map launch: %s", cudaGetErrorString(e));
    }
    // ---- S1-S3 (+ the S4 records the kernel keeps anyway), as st_debug_scores launches them in random mode
    st::ScoreArgs a;
    memset(&a, 0, sizeof(a));
    a.map = map; a.isig = isig;
    a.bp.seed = p->seed; a.bp.n_t = n_t; a.bp.n_f = n_f; a.bp.n_min = p->n_min; a.bp.n_max = p->n_max;
    a.bp.tau_lo = p->tau_lo; a.bp.tau_hi = p->tau_hi; a.bp.family = ST_FAMILY_QUADRATIC; a.bp.pad = 0;
    a.f_min = f_min; a.df = df;
    a.track_offset = p->track_offset; a.n_tracks = p->n_tracks;
    a.n_tau = 1; a.norm = p->norm;
    a.sc = sc;
    a.cand = reinterpret_cast<st::Cand*>(d.scratch + kNaOffCand); a.cand_cap = kNaCandCap;
    a.warp_best = reinterpret_cast<st::WarpBest*>(d.scratch + kNaOffWarpBest); a.warp_slots = kWarpSlots;
    a.hist = nullptr; a.n_bins = 0;
    a.dump = snr_dev;
    a.pool_stride = (p->n_max + 63) & ~63;
    {
        uint64_t blocks = (uint64_t)d.n_sm * 8;
        const uint64_t need = ((p->n_tracks + st::kRandPerWarp - 1) / st::kRandPerWarp + 7) / 8;
        if (blocks > need) blocks = need;
        if (blocks > kWarpSlots / 8) blocks = kWarpSlots / 8;
        st::k_score_random<false, false, false><<<(unsigned)blocks, 256, hist_bytes(0), stream>>>(a);
        e = cudaGetLastError();
        if (e != cudaSuccess) return na_fail(err, len, ST_ECUDA, "k_score_random launch: %s", cudaGetErrorString(e));
    }
    return ST_OK;
}

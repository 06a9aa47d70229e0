/*
 * stochtrack.h -- C ABI of the B200 (sm_100a) all-sky stochtrack hot path.
 *
 * Method: Thrane & Coughlin, "Seedless clustering in all-sky searches for
 * gravitational-wave transients" (arXiv:1401.8060).  Citations are lines of the
 * paper text (PAPER.md:<line>) with the section / equation they fall in, and
 * readings G<n> of DESIGN.md where the paper is silent.
 *
 * What the library computes (one GPU, one stream, no collectives):
 *   S0  p(t;f) = CSD(t;f) / sigma          complex SNR map, Eq. 7
 *   S1  template i -> 3 Bezier control points + delay, from Philox4x32-10(seed, i)
 *                                            "six random numbers"
 *   S2  Eq. 6 curve -> one frequency bin per time column (the cluster Gamma)
 *
 *   S3  SNR(i, tau) = N^-alpha * sum_Gamma Re[ e^{2 pi i f tau} p(t;f) ], Eq. 8
 *
 *   S4  max / argmax over (i, tau) and a histogram of all SNR(i, tau)
 *
 *
 * Conventions
 *   - plain C types only; every pointer is marked HOST or DEVICE below;
 *   - the caller owns every buffer it passes; the library allocates no device
 *     memory: the caller hands in one workspace (st_workspace_bytes / st_set_workspace);
 *   - every call returns 0 (ST_OK) or a negative ST_E* code, never throws or aborts;
 *     st_last_error() returns a message for the last failing call on that context;
 *   - a context is bound to one CUDA stream and is not thread-safe;
 *   - st_search / st_set_map_host are synchronous on return (they end with a
 *     stream synchronisation); st_set_map and the debug calls are stream-ordered.
 *   - there is NO CPU fallback: without a CUDA device every device call fails
 *     with ST_ECUDA.
 */
#ifndef STOCHTRACK_H
#define STOCHTRACK_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ST_OK       0
#define ST_EINVAL  -1   /* bad argument                                   */
#define ST_ESTATE  -2   /* search before workspace / map were set         */
#define ST_ENOSPC  -3   /* workspace too small for the request            */
#define ST_ECUDA   -4   /* CUDA runtime error (message in st_last_error)  */

/* sigma layouts for st_set_map (Eq. 7: p = lambda sI* sJ, sigma = 1/lambda; G11) */
#define ST_SIGMA_NONE      0   /* sigma == 1 everywhere, pointer ignored   */
#define ST_SIGMA_PER_FREQ  1   /* float32 [n_f]                            */
#define ST_SIGMA_PER_PIXEL 2   /* float32 [n_t][n_f]                       */

/* delay modes (one random Delta tau per template; the grid mode
 * scores every template against every trial delay, BASELINE.json north_star) */
#define ST_TAU_GRID   0
#define ST_TAU_RANDOM 1

/* normalisation N^-alpha of Eq. 8 (G1): alpha = 1/2 gives a unit-variance
 * statistic; alpha = 1 is Eq. 8 exactly as printed.           */
#define ST_NORM_SQRT_N 0
#define ST_NORM_MEAN   1
/* fn. 23: "alternative definitions of SNR_tot (with a different weighting scheme)".  Reading
 * G25: the inverse-variance combination of Appendix A's per-pixel estimates,
 *     SNR_w = sum_Gamma (rho / sigma) / sqrt( sum_Gamma 1 / sigma^2 ),   rho = Re[e^{2 pi i f tau} p],
 * equal to the SQRT_N statistic for constant sigma; masked pixels leave both sums.  Needs the map to have
 * been set with its sigma (st_set_map, st_set_map_host, or a st_search_batch run with this norm: a batch with
 * another norm does not write the 1 / sigma plane and leaves its last map without one), else ST_ESTATE. */
#define ST_NORM_INVVAR 2

/* template families ("other parameterizable curves such as spline can be used as well";
 * a chirp "is not especially well-described with a second-order Bezier curve").
 * CUBIC (reading G26): a cubic Bezier curve whose time control points are the degree-elevated quadratic
 * (t(xi) is the quadratic family's) and whose frequency has four control points y0, y1, y2, y3, each
 * uniform over the band; N, j0, a, y0, y1, y2, tau of template i are those of the quadratic template i,
 * y3 comes from the one Philox word the quadratic family leaves unused.
 * CHIRP (reading G27): the leading-order inspiral sweep f ~ (t_c - t)^(-3/8) (the binary
 * neutron star study): f(u) = y0 (T_c / (T_c - u))^(3/8) from the template's first column,
 * T_c = N^2 / (N - a); N, j0, a, y0, tau are those of the quadratic template i; y1, y2, y3 are not used; a
 * sweep that leaves the band rides its top bin.  Scored by the general builds of the kernels.          */
#define ST_FAMILY_QUADRATIC 0
#define ST_FAMILY_CUBIC     1
#define ST_FAMILY_CHIRP     2

/* scoring kernel selection (grid mode).  AUTO picks CHEBYSHEV when the grid is
 * uniform and every bin's step angle is well conditioned, else REINSCH / ROTATION
 * when uniform, else TABLE.  A kernel asked for by name on a grid it cannot score
 * within the 1e-4 contract (REINSCH / CHEBYSHEV: a bin's step angle 2 pi f dtau too
 * close to 0 or pi; any recurrence kernel: a non-uniform grid) is refused with
 * ST_EINVAL rather than run.                                                    */
#define ST_KERNEL_AUTO     0
#define ST_KERNEL_TABLE    1   /* twiddle table W[k][m] read from L2, any grid          */
#define ST_KERNEL_ROTATION 2   /* complex rotation recurrence along a uniform tau grid  */
#define ST_KERNEL_REINSCH  3   /* real three-term (Reinsch) recurrence, uniform grid    */
#define ST_KERNEL_RANDOM   4   /* reported in st_result for ST_TAU_RANDOM searches      */
#define ST_KERNEL_CHEBYSHEV 5  /* two-sided Chebyshev recurrence, uniform grid (1 FMA per eval) */

typedef struct st_ctx st_ctx;   /* opaque */

/* One template: quadratic Bezier through P0 = (j0, y0),
 * P1 = (j0 + a, y1), P2 = (j0 + N, y2); times in columns, frequencies in bins
 * (bin k covers [k, k+1)); tau is the template's own delay in random mode.    */
typedef struct {
    int32_t N;      /* number of time columns = pixels in Gamma  */
    int32_t j0;     /* first column                                             */
    double  a;      /* t_mid - t_start in columns, 0 < a < N (G3)               */
    double  y0, y1, y2;
    double  tau;    /* seconds                                                  */
    double  y3;     /* ST_FAMILY_CUBIC: f_end (y1, y2 are then the inner control points); else ignored */
} st_track;

typedef struct {
    uint64_t n_tracks;       /* T: templates scored, ids [track_offset, track_offset+T) */
    uint64_t track_offset;   /* lets runs be combined exactly by max     */
    uint64_t seed;           /* Philox key ("different random seed")       */
    int32_t  n_min, n_max;   /* track duration range in columns, 1 <= n_min <= n_max <= n_t
                                (the t_min constraint of PAPER.md:75)                   */
    int32_t  tau_mode;       /* ST_TAU_GRID | ST_TAU_RANDOM                             */
    int32_t  n_tau;          /* grid size (grid mode), ignored in random mode           */
    const double *tau_grid;  /* HOST, n_tau delays in seconds (grid mode)               */
    double   tau_lo, tau_hi; /* random mode: tau ~ U(tau_lo, tau_hi)     */
    int32_t  norm;           /* ST_NORM_SQRT_N | ST_NORM_MEAN | ST_NORM_INVVAR          */
    int32_t  n_bins;         /* histogram bins, 0 = no histogram, <= ST_MAX_BINS        */
    double   hist_lo, hist_hi; /* bin = floor((snr-lo)/(hi-lo)*n_bins) clamped (G14)    */
    uint64_t *hist_out;      /* HOST, n_bins counts (overwritten) or NULL               */
    int32_t  kernel;         /* ST_KERNEL_* request (grid mode)                         */
    int32_t  family;         /* ST_FAMILY_QUADRATIC (0) | ST_FAMILY_CUBIC | ST_FAMILY_CHIRP */
} st_search_params;

typedef struct {
    float    max_snr;        /* largest float32 SNR(i, tau) the scoring kernel produced  */
    int32_t  arg_tau_index;  /* grid index m of the argmax (0 in random mode)            */
    double   max_snr_f64;    /* SNR of the argmax re-scored in float64 on the device     */
    uint64_t arg_track;      /* template id of the argmax (G12 total order)              */
    double   arg_tau;        /* its delay in seconds                                     */
    st_track arg_params;     /* its control points                                       */
    uint64_t n_evals;        /* sum_i N_i * n_tau  (track-pixel x delay evaluations)     */
    uint64_t n_pixels;       /* sum_i N_i                                                */
    int32_t  n_candidates;   /* near-max samples re-scored in float64                    */
    int32_t  kernel_used;    /* ST_KERNEL_* actually launched                            */
    int32_t  n_launches;     /* kernels launched by this call                            */
    int32_t  flags;          /* ST_FLAG_* bits                                           */
    float    gpu_ms;         /* device time of the scoring launches (CUDA events)        */
    int32_t  n_deferred;     /* Chebyshev path: templates re-scored by the two-class build because their
                                amplitude in drift-prone (class B) bins was too large for the fast build */
} st_result;

#define ST_FLAG_CAND_OVERFLOW 1   /* candidate list overflowed: argmax decided by the float32 records      */
#define ST_FLAG_BANK_READ     2   /* S1 + S2 came from the bank cache (st_set_bank_cache)                 */
#define ST_FLAG_BANK_FILLED   4   /* this search filled the bank cache                                     */

#define ST_MAX_BINS 4096
#define ST_MAX_N_T  1048576
#define ST_MAX_N_F  65535
#define ST_MAX_N_TAU 4096

/* Create a context for maps of n_t time columns x n_f frequency bins, bin k at
 * frequency f_min + k*df [Hz] (G6).  HOST only, no CUDA call.
 * Errors: ST_EINVAL unless 1<=n_t<=ST_MAX_N_T, 1<=n_f<=ST_MAX_N_F, df>0, f_min>=0. */
int st_create(st_ctx **out, int32_t n_t, int32_t n_f, double df, double f_min);
void st_destroy(st_ctx *ctx);

/* Bytes of DEVICE workspace needed for searches with up to max_n_tau grid
 * delays (0 on bad arguments).  Includes a staging area for st_set_map_host. */
size_t st_workspace_bytes(const st_ctx *ctx, int32_t max_n_tau);

/* Hand in the workspace (DEVICE, 256-byte aligned, caller-owned, must outlive the
 * context's use) and the CUDA stream (cudaStream_t as void*, NULL = default
 * stream) every later call is ordered on.  Errors: ST_ENOSPC, ST_EINVAL, ST_ECUDA. */
int st_set_workspace(st_ctx *ctx, void *workspace_dev, size_t bytes, void *cuda_stream);

/* Bank cache: the rasterised template bank kept on the device and reused across maps (n_ts
 * time-shifted maps per analysis; follow-ups and repeated runs over the same spectrograms).
 * When the caller hands in a buffer, a grid search of quadratic templates (ST_KERNEL_CHEBYSHEV path, sqrt(N) /
 * mean normalisation) that uses a NEW bank -- (seed, track_offset, n_tracks, n_min, n_max) -- and fits writes
 * (N, j0) and the bins of every template while it scores them (ST_FLAG_BANK_FILLED); every later search with the
 * SAME bank on whatever map reads them back instead of running S1 + S2 (ST_FLAG_BANK_READ): 2 bytes per template
 * column from HBM instead of the Philox rounds and the float64 rasteriser.  Results are bit-identical either way.
 * st_search_batch / st_search_timeshifts with one seed for every map use it from the second map on.
 *   st_bank_cache_bytes : bytes for a bank of n_tracks templates of at most n_max columns (0 on bad arguments)
 *   st_set_bank_cache   : DEVICE buffer, 256-byte aligned, caller-owned; NULL detaches.  Invalidates the cache. */
size_t st_bank_cache_bytes(const st_ctx *ctx, uint64_t n_tracks, int32_t n_max);
int st_set_bank_cache(st_ctx *ctx, void *cache_dev, size_t bytes);

/* S0 (Eq. 7): p = CSD / sigma into the workspace.  csd_dev: DEVICE
 * complex64 [n_t][n_f] (frequency contiguous, interleaved re/im); sigma_dev: DEVICE
 * float32 per sigma_kind.  sigma <= 0 or non-finite masks the pixel (p = 0, G11).
 * Stream-ordered; inputs may be freed once the stream has passed the call.   */
int st_set_map(st_ctx *ctx, const void *csd_dev, const float *sigma_dev, int32_t sigma_kind);

/* Same with HOST buffers (pinned or pageable): copies them into the workspace
 * staging area on the stream, then runs S0.  Synchronous on return.          */
int st_set_map_host(st_ctx *ctx, const void *csd_host, const float *sigma_host, int32_t sigma_kind);

/* S1-S4 over the current map.  Fills *out (HOST) and params->hist_out (HOST).
 * Errors: ST_ESTATE (no workspace / map), ST_EINVAL, ST_ENOSPC (n_tau beyond the
 * workspace; in grid mode also an n_max whose pixel list, 10 bytes per column, does
 * not fit one SM's shared memory: about 22 000 columns -- the random mode has no such
 * limit), ST_ECUDA.  ST_KERNEL_AUTO never fails for lack of shared memory on a wide
 * band: it falls back to the kernel whose per-bin table lives in L2.              */
int st_search(st_ctx *ctx, const st_search_params *params, st_result *out);

/* The top_k loudest (template, delay) samples of a search, in the G12 total order (larger float64 SNR,
 * then smaller template id, then smaller delay index) -- the candidates a follow-up looks at
 * (PAPER.md:232).  Two passes over the bank: st_search as usual (params->n_bins must be > 0: the
 * histogram locates the SNR of the top_k-th sample), then a second scoring pass that keeps every sample
 * at or above the edge one bin below it, re-scores those in float64 on the device and sorts them.
 * top_out: HOST [top_k]; *n_out = entries written (= min(top_k, samples)).  *result as st_search.
 * Errors as st_search, plus ST_EINVAL (top_k outside [1, ST_MAX_TOP_K], n_bins == 0) and ST_ENOSPC when
 * more than 65 536 samples lie at or above that edge (histogram too coarse: use more / narrower bins). */
#define ST_MAX_TOP_K 4096
typedef struct {
    uint64_t track;
    int32_t  tau_index;      /* 0 in random mode */
    float    snr_f32;        /* what the scoring kernel produced */
    double   snr_f64;        /* re-scored in float64 */
    double   tau;            /* seconds */
} st_top_entry;
int st_search_topk(st_ctx *ctx, const st_search_params *params, int32_t top_k, st_top_entry *top_out,
                   int32_t *n_out, st_result *result);

/* st_search plus, for every template of the search, its maximum over the delays and the delay that attains
 * it (a template "tries to guess ... the appropriate phase factor"): computed in
 * the fused S4 epilogue of the scoring kernels, nothing is dumped.
 *   snr_max_dev   : DEVICE float32 [n_tracks], max_m SNR(track_offset + q, m) as the kernel scored it
 *   tau_index_dev : DEVICE int32   [n_tracks], the smallest delay index attaining it (0 in random mode)
 * Decided in float32 (reading G24 of DESIGN.md): where two delays of one template tie to float32 accuracy
 * the index may differ from a float64 evaluation; the value agrees within the G13 tolerance.
 * Errors as st_search, plus ST_EINVAL for a NULL output.  Synchronous on return.                    */
int st_search_track_max(st_ctx *ctx, const st_search_params *params, float *snr_max_dev,
                        int32_t *tau_index_dev, st_result *out);

/* Eq. 8 for EXPLICIT templates instead of bank members: the targeted use of the statistic
 * (Eq. 5: a fixed set of clusters Gamma) and the parity export for track shapes the bank
 * produces with vanishing probability (flat, near-flat, full-length).
 *   tracks  : HOST [count] templates in the st_track parameterisation (1 <= N, 0 <= j0, j0 + N <= n_t,
 *             0 < a < N, finite values, and the frequency control points the family uses -- y0, y1, y2; y3 too
 *             for CUBIC; y0 alone for CHIRP -- inside the band, 0 <= y <= n_f in bin units, as every bank
 *             member's are: the rasteriser's bit-exactness guard is sized for that range); in random mode
 *             each template's own `tau` is its delay
 *   snr_dev : DEVICE float32 [count][n_tau] (n_tau = 1 in random mode), same scoring kernel as st_search
 *             with the same params (tau grid / range, norm, kernel, family); n_tracks, track_offset, seed,
 *             n_min, n_max and the histogram fields of params are ignored.
 * Errors: ST_EINVAL (a template outside the map, count outside [0, ST_MAX_SCORE_TRACKS]), otherwise as
 * st_search.  Synchronous on return.                                                               */
#define ST_MAX_SCORE_TRACKS 4096
int st_score_tracks(st_ctx *ctx, const st_search_params *params, const st_track *tracks, int32_t count,
                    float *snr_dev);

/* Batch / background mode (the background is estimated from many
 * time-shifted maps, every one searched with its own template bank; BASELINE.json configs[3]):
 * S0-S4 over n_maps maps in ONE call.  Map m is searched exactly as
 *     st_set_map(csd[m], sigma[m]);  st_search(params with seed = seeds[m])
 * would search it (same kernels, same results bit for bit), but nothing synchronises with the host
 * between maps: per-map results and histograms accumulate on the device and come back once per
 * group of ST_BATCH_GROUP maps, and with HOST buffers the copy of map m + 1 overlaps the search of
 * map m (a second, internal stream and two staging buffers).                                   */
#define ST_BATCH_GROUP 256
typedef struct {
    int32_t  n_maps;
    int32_t  host_buffers;        /* 0: csd[m] / sigma[m] are DEVICE pointers, 1: HOST (pinned for overlap) */
    const void  *const *csd;      /* HOST array of n_maps pointers: complex64 [n_t][n_f] each            */
    const float *const *sigma;    /* HOST array of n_maps pointers per sigma_kind, or NULL when NONE      */
    int32_t  sigma_kind;          /* ST_SIGMA_*                                                            */
    int32_t  reserved;            /* must be 0                                                             */
    const uint64_t *seeds;        /* HOST, n_maps template seeds (G16), or NULL: params->seed for every map */
} st_batch;
/* results: HOST [n_maps].  params->hist_out (when params->n_bins > 0): HOST [n_maps][n_bins], one
 * histogram per map.  results[m].gpu_ms is 0; *gpu_ms_total (optional) receives the device time of
 * the whole batch (CUDA events around everything the call enqueues).  Synchronous on return.
 * Errors as st_search, plus ST_EINVAL for n_maps < 1 or a NULL entry.                           */
int st_search_batch(st_ctx *ctx, const st_batch *batch, const st_search_params *params,
                    st_result *results, float *gpu_ms_total);

/* ft-map construction on the device (the step before S0; Eqs. 7 and A1-A4 at
 * PAPER.md:96, :258-277; readings G19-G22 of DESIGN.md): two strain series -> 50 %-overlapping Hann
 * segments of seg_len samples -> DFT -> auto-power P' from the n_neighbours non-overlapping segments
 * on either side -> p = lambda s~_I^* s~_J, written straight into the context's map (the same state
 * st_set_map leaves behind).  Float64 transform, float32 map.
 *   s_i_dev, s_j_dev : DEVICE float64 [n_samples], n_samples >= (n_t + 1) * seg_len / 2
 *   fs               : sample rate [Hz]; fs / seg_len must equal the context's df and f_min must be
 *                      a multiple of df with f_min + n_f df <= fs / 2
 *   seg_len          : power of two, 64 <= seg_len <= 8192
 *   scratch_dev      : DEVICE, st_ftmap_scratch_bytes(ctx, seg_len) bytes, 256-byte aligned, caller-owned;
 *                      after the call it holds s~_I then s~_J (float64 complex [n_t][n_f] each, parity export)
 * Stream-ordered.  Errors: ST_EINVAL, ST_ESTATE (no workspace), ST_ENOSPC (scratch), ST_ECUDA.      */
typedef struct {
    double  fs;
    int32_t seg_len;
    int32_t n_neighbours;    /* >= 1; segments j +- 2 .. j +- (n_neighbours + 1), those inside the map (G20) */
} st_ftmap_params;
size_t st_ftmap_scratch_bytes(const st_ctx *ctx, int32_t seg_len);
int st_set_map_from_strain(st_ctx *ctx, const double *s_i_dev, const double *s_j_dev, int64_t n_samples,
                           const st_ftmap_params *params, void *scratch_dev, size_t scratch_bytes);
/* Time-shift background from strain (significance from n_ts time-shift analyses; reading
 * G23): the strain spectrograms are computed ONCE; for each shifts[m] (HOST, whole segments, 0 <= shift <
 * n_t, cyclic over the map) detector J's segment (j + shift) mod n_t is paired with detector I's segment j,
 * P' of each detector taken around its own segment, and the resulting map is searched with seeds[m]
 * (HOST, or NULL: params->seed for every shift).  Per-shift results and histograms as st_search_batch
 * (results HOST [n_shifts], params->hist_out HOST [n_shifts][n_bins], no host synchronisation inside a
 * group of ST_BATCH_GROUP shifts).  On return the context's map is that of the last shift.
 * ST_NORM_INVVAR is refused (ST_EINVAL): a map built from strain has no 1 / sigma plane; likewise st_search on
 * a map set by st_set_map_from_strain returns ST_ESTATE for that norm.                                   */
int st_search_timeshifts(st_ctx *ctx, const double *s_i_dev, const double *s_j_dev, int64_t n_samples,
                         const st_ftmap_params *ft_params, void *scratch_dev, size_t scratch_bytes,
                         int32_t n_shifts, const int32_t *shifts, const uint64_t *seeds,
                         const st_search_params *params, st_result *results, float *gpu_ms_total);
/* Parity export: copy the context's current map p (complex64 [n_t][n_f]) to p_out_dev (DEVICE).   */
int st_debug_get_map(st_ctx *ctx, void *p_out_dev);

/* S1 as a pure HOST function: the control points of template `track_id`
 * (same arithmetic as the device generator).                                   */
int st_track_params(const st_ctx *ctx, uint64_t seed, uint64_t track_id,
                    int32_t n_min, int32_t n_max, double tau_lo, double tau_hi, st_track *out);
/* The same for either template family (st_track_params is the quadratic one).   */
int st_track_params_family(const st_ctx *ctx, uint64_t seed, uint64_t track_id, int32_t n_min, int32_t n_max,
                           double tau_lo, double tau_hi, int32_t family, st_track *out);

/* Parity exports (stream-ordered, outputs DEVICE).  Ids [first, first+count):
 * k_out_dev int32 [count][n_t] (-1 beyond N), j0_dev / N_dev int32 [count].
 * Uses params->seed, n_min, n_max, family.                                     */
int st_debug_rasterise(st_ctx *ctx, const st_search_params *params, uint64_t first, uint64_t count,
                       int32_t *k_out_dev, int32_t *j0_dev, int32_t *N_dev);
/* The same export through the random-delay kernel's OWN rasteriser (its fast path evaluates Eq. 6 in
 * Horner form and regenerates the template on the normative fallback): runs k_score_random over ids
 * [first, first+count) with params (ST_TAU_RANDOM) and writes the bins it used.  Needs a map.        */
int st_debug_rasterise_random(st_ctx *ctx, const st_search_params *params, uint64_t first, uint64_t count,
                              int32_t *k_out_dev, int32_t *j0_dev, int32_t *N_dev);
/* Rasterise one explicit template of the given family (HOST st_track in, DEVICE int32 [N] out); the template
 * must satisfy the conditions listed at st_score_tracks (ST_EINVAL otherwise). */
int st_debug_rasterise_track(st_ctx *ctx, const st_track *track, int32_t family, int32_t *k_out_dev);
/* snr_dev float32 [count][n_tau] (n_tau = 1 in random mode): every SNR(i, tau)
 * the scoring kernel selected by params->kernel produces.                      */
int st_debug_scores(st_ctx *ctx, const st_search_params *params, uint64_t first, uint64_t count,
                    float *snr_dev);
/* The 8 Philox words of a template (HOST out[8]); pure host function.          */
int st_debug_track_words(uint64_t seed, uint64_t track_id, uint32_t *out_host);

/* S4 across runs (independent runs over disjoint template-id ranges -- other GPUs, other jobs, resumed
 * chunks -- are combined by taking the maximum, "results identical"): the G12 rule as one HOST function, so that no
 * caller has to restate it.  Pure host code, no CUDA call, no context.
 *   results   : HOST [n] results of searches over disjoint id ranges of the SAME map, delay grid and norm
 *   hists     : HOST [n] pointers to their n_bins-bin histograms (entries may be NULL), or NULL
 *   out       : the combination: the entry that wins under the G12 total order among the runs that scored anything
 *               (larger max_snr_f64, then smaller arg_track, then smaller arg_tau_index) with n_evals, n_pixels,
 *               n_candidates, n_launches, n_deferred summed, flags OR-ed, max_snr and gpu_ms the maxima; when no
 *               run scored anything, results[0]
 *   hist_out  : HOST [n_bins] sum of the histograms given (exact, u64), or NULL
 *   best_index: optional, receives the index of the winning entry
 * Errors: ST_EINVAL (n < 1, NULL results / out, n_bins outside [0, ST_MAX_BINS], hist_out without hists).       */
int st_combine_results(const st_result *results, const uint64_t *const *hists, int32_t n, int32_t n_bins,
                       st_result *out, uint64_t *hist_out, int32_t *best_index);

/* The paper's one-delay-per-template scoring (S0-S3 of the list at the top) for callers that
 * cannot give the library any device memory of their own.
 *
 * Who that is.  Every other device call here needs a workspace the caller allocates (st_set_workspace), and a
 * workspace is an allocation like any other.  Some hosts of this library have none to give: a search stage
 * plugged into a pipeline whose framework reserved the whole card for its own memory pool at start-up, so that a
 * late cudaMalloc fails with out-of-memory; an online (low-latency) analysis that may not allocate or free while
 * it runs, because cudaMalloc / cudaFree synchronise the whole device and stall every other stream of the
 * process; a component that is handed exactly its input and output buffers by the application around it and
 * has no allocator of its own to ask.  They still own the map they want searched and the buffer the scores go
 * to: those are this call's only pointers.
 *
 * What it does.  snr_dev[q] = SNR of template params->track_offset + q with that template's own random delay
 * in (tau_lo, tau_hi), q = 0 .. params->n_tracks - 1: bit for bit what st_set_map(csd_dev, sigma_dev, sigma_kind)
 * followed by st_debug_scores(params, track_offset, n_tracks, snr_dev) writes for a context of the same n_t,
 * n_f, df, f_min -- the same two kernels (k_prepare_map, k_score_random) are launched.  What those kernels keep
 * besides their inputs and outputs -- the weighted map p = CSD / sigma with its 1 / sigma plane, the
 * work-claim counter and the reduction records -- lives in ONE array of ST_NOALLOC_SCRATCH_BYTES (about
 * 3.4 MiB) that is compiled into the library as a static __device__ object.  Every GPU on which the library's
 * code gets loaded holds its copy of that array until the process exits, whether or not this call is ever
 * used there.  The call itself performs no cudaMalloc, cudaFree, cudaHostAlloc, stream / event creation or
 * any other allocating CUDA or library routine; it issues one cudaMemsetAsync and two kernel launches.
 *
 * Limits (the price of a fixed array): n_t * n_f <= ST_NOALLOC_MAX_PIXELS (the Table III map of the paper,
 * 500 x 151, and the 250 x 961 map of BASELINE.json configs[1] fit; the 500 x 2461 maps do not), else ST_ENOSPC;
 * ST_TAU_RANDOM only, quadratic templates, norm ST_NORM_SQRT_N or ST_NORM_MEAN, n_tracks <= 2^31 (one launch),
 * else ST_EINVAL.  The fields n_tau, tau_grid, n_bins, hist_*, kernel of params are ignored.
 *
 *   csd_dev, sigma_dev : DEVICE, as st_set_map (complex64 [n_t][n_f]; float32 per sigma_kind), on the CURRENT device
 *   snr_dev            : DEVICE float32 [n_tracks], on the current device, caller-owned
 *   cuda_stream        : cudaStream_t as void* (NULL = default stream) of the current device; the call is
 *                        stream-ordered and returns once its work is enqueued (inputs / output may be released
 *                        after the stream has passed it)
 *   err_host, err_len  : optional HOST buffer that receives the message of a failing call (may be NULL / 0)
 *
 * The first call on each device looks up that device's address of the array (cudaGetSymbolAddress, which may
 * load the library's device code there) and the SM count; later calls reuse them.  Make that first call at
 * start-up, before any stream capture begins.
 * The array is shared by every call on a device and still holds what the previous call left in it: the call
 * clears the part that must start from zero and overwrites the map, so consecutive calls on one stream are
 * independent of each other; but two calls whose work can overlap on the GPU (different streams, or different
 * host threads on different streams) use the same array at the same time and corrupt each other's results --
 * keep all calls of a device on one stream, or order them with events.  It uses no st_ctx and does not
 * touch the state of any.                                                                                */
#define ST_NOALLOC_MAX_PIXELS    262144
#define ST_NOALLOC_SCRATCH_BYTES 3604736
int st_score_random_noalloc(const void *csd_dev, const float *sigma_dev, int32_t sigma_kind,
                            int32_t n_t, int32_t n_f, double df, double f_min,
                            const st_search_params *params, float *snr_dev, void *cuda_stream,
                            char *err_host, size_t err_len);

const char *st_last_error(const st_ctx *ctx);
/* Library / build identification, e.g. "stochtrack-b200 sm_100a".              */
const char *st_version(void);

#ifdef __cplusplus
}
#endif
#endif /* STOCHTRACK_H */

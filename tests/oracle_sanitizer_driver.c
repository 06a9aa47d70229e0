/* Runs the oracle's whole path on a small seeded map; built with -fsanitize=address,undefined by
 * tests/test_oracle_pins.py (the C oracle is #included so that the sanitizers see every line of it). */
#include <stdio.h>
#include <stdlib.h>
#include "../oracle/stochtrack_oracle.c"

int main(void)
{
    enum { NT = 40, NF = 37, NTAU = 9, T = 300, NB = 50 };
    static float csd[NT * NF * 2], sigma[NT * NF];
    static double p[NT * NF * 2], tau[NTAU], snr[T * NTAU];
    static uint64_t hist[NB];
    static int32_t kd[T * NT], j0[T], Nn[T];
    uint32_t s = 12345u;
    for (int i = 0; i < NT * NF * 2; ++i) { s = s * 1664525u + 1013904223u; csd[i] = (float)((int)(s >> 8) % 2001 - 1000) / 500.0f; }
    for (int i = 0; i < NT * NF; ++i) { s = s * 1664525u + 1013904223u; sigma[i] = (i % 97 == 0) ? 0.0f : 0.5f + (float)(s >> 20) / 4096.0f; }
    for (int m = 0; m < NTAU; ++m) tau[m] = -0.01 + 0.0025 * m;
    or_prepare_map(csd, sigma, 2, NT, NF, p);
    or_search_params sp;
    sp.n_tracks = T; sp.track_offset = (1ull << 40) + 3; sp.seed = 99; sp.n_min = 1; sp.n_max = NT;
    sp.tau_mode = 0; sp.n_tau = NTAU; sp.tau_lo = -0.01; sp.tau_hi = 0.01; sp.norm_mode = 0; sp.n_bins = NB;
    sp.hist_lo = -5.0; sp.hist_hi = 5.0; sp.score_mode = 0; sp.n_threads = 2; sp.family = 0; sp.pad = 0;
    or_search_result r;
    for (int mode = 0; mode < 3; ++mode) {
        sp.score_mode = mode == 1; sp.tau_mode = mode == 2; if (mode == 2) sp.n_tau = 1;
        if (or_search(p, NT, NF, 40.0, 1.0, tau, &sp, &r, hist, snr, kd, j0, Nn, NULL) != 0) return 2;
        printf("%d %.17g %llu %d %llu\n", mode, r.max_snr, (unsigned long long)r.arg_track, r.arg_tau_index,
               (unsigned long long)r.n_evals);
    }
    /* variants: cubic templates, inverse-variance weighting (their own output row is not compared) */
    static double inv_sigma[NT * NF];
    or_prepare_inv_sigma(sigma, 2, NT, NF, inv_sigma);
    sp.tau_mode = 0; sp.n_tau = NTAU; sp.score_mode = 0; sp.family = 1; sp.norm_mode = 2;
    if (or_search(p, NT, NF, 40.0, 1.0, tau, &sp, &r, hist, snr, kd, j0, Nn, inv_sigma) != 0) return 3;
    sp.score_mode = 1;
    if (or_search(p, NT, NF, 40.0, 1.0, tau, &sp, &r, hist, snr, kd, j0, Nn, inv_sigma) != 0) return 3;
    return 0;
}

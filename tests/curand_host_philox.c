/* Reference words for pin P1: NVIDIA cuRAND's HOST generator
 * CURAND_RNG_PSEUDO_PHILOX4_32_10 (runs on the CPU; no GPU needed).
 * usage: curand_host_philox <seed> <offset> <n_words>  -> hex words, one per line.
 * Test helper only: it contains no Philox arithmetic of its own. */
#include <stdio.h>
#include <stdlib.h>
#include <stdint.h>
#include <curand.h>
int main(int argc, char **argv)
{
    if (argc != 4) return 2;
    unsigned long long seed = strtoull(argv[1], NULL, 0);
    unsigned long long offset = strtoull(argv[2], NULL, 0);
    size_t n = (size_t)strtoull(argv[3], NULL, 0);
    curandGenerator_t g;
    if (curandCreateGeneratorHost(&g, CURAND_RNG_PSEUDO_PHILOX4_32_10) != CURAND_STATUS_SUCCESS) return 3;
    if (curandSetPseudoRandomGeneratorSeed(g, seed) != CURAND_STATUS_SUCCESS) return 4;
    if (curandSetGeneratorOffset(g, offset) != CURAND_STATUS_SUCCESS) return 5;
    uint32_t *out = (uint32_t *)malloc(n * sizeof(uint32_t));
    if (curandGenerate(g, out, n) != CURAND_STATUS_SUCCESS) return 6;
    for (size_t i = 0; i < n; ++i) printf("%08x\n", out[i]);
    curandDestroyGenerator(g);
    free(out);
    return 0;
}

/*
 * asan_driver.c -- runs the CPU oracle (oracle/ht_oracle.c, compiled INTO this program with
 * -fsanitize=address,undefined) on one event read from a binary file, and prints a digest of every result.
 * tests/test_oracle_sanitizers.py builds it, runs it on the tiny workload (BASELINE.json:configs[0]) and compares the
 * digest with the ordinary build of the oracle: no out-of-bounds access, no use of uninitialised or freed memory, no
 * undefined integer / float-to-int conversion anywhere in the oracle ("Race detection / sanitizers").
 *
 * Input file: int32 n_theta, n_phi, n_a, n_b; float a_min, a_max, b_min, b_max, theta_min, theta_max, phi_min, phi_max;
 *             uint32 threshold; uint32 merge_window; int64 n_hits; float x[n], y[n], z[n].
 */
#include "../oracle/ht_oracle.c"

#include <stdio.h>

static uint64_t fnv(const void *p, size_t n, uint64_t h)
{
    const unsigned char *c = (const unsigned char *)p;
    for (size_t i = 0; i < n; ++i) { h ^= c[i]; h *= 1099511628211ull; }
    return h;
}

int main(int argc, char **argv)
{
    if (argc != 2) return 2;
    FILE *f = fopen(argv[1], "rb");
    if (!f) return 2;
    oracle_binning g;
    uint32_t threshold, window;
    int64_t n;
    if (fread(&g, sizeof g, 1, f) != 1 || fread(&threshold, 4, 1, f) != 1 || fread(&window, 4, 1, f) != 1 ||
        fread(&n, 8, 1, f) != 1 || n < 0) return 2;
    float *x = (float *)malloc(sizeof(float) * (size_t)(n + 1)), *y = (float *)malloc(sizeof(float) * (size_t)(n + 1)),
          *z = (float *)malloc(sizeof(float) * (size_t)(n + 1));
    if (fread(x, 4, (size_t)n, f) != (size_t)n || fread(y, 4, (size_t)n, f) != (size_t)n || fread(z, 4, (size_t)n, f) != (size_t)n) return 2;
    fclose(f);
    const size_t cells = (size_t)g.n_theta * g.n_phi * g.n_a * g.n_b;
    uint32_t *M = (uint32_t *)malloc(cells * 4);
    const int64_t votes = oracle_fill(&g, x, y, z, n, M);
    int32_t *plane = (int32_t *)malloc(4 * (size_t)(n + 1)), *bins = (int32_t *)malloc(4 * (size_t)(n + 1) * (size_t)g.n_a);
    oracle_votes(&g, x, y, z, n, plane, bins);
    const int64_t np = oracle_peaks(&g, M, threshold, 0u, NULL, 0);
    oracle_peak *pk = (oracle_peak *)malloc(sizeof(oracle_peak) * (size_t)(np + 1));
    oracle_peaks(&g, M, threshold, 0u, pk, np);
    double *rho = (double *)malloc(8 * (size_t)(np + 1)), *phi = (double *)malloc(8 * (size_t)(np + 1));
    oracle_tracks(&g, pk, np, rho, phi);
    oracle_merged *mg = (oracle_merged *)malloc(sizeof(oracle_merged) * (size_t)(np + 1));
    const int64_t nm = oracle_merge_ridges(&g, pk, np, window, mg, np);
    /* truth matching of the candidates against a few circles derived from the hits themselves (any input will do here:
       the point is that every access of oracle_match_truth runs under the sanitizers) */
    const int64_t nt = n < 64 ? n : 64;
    oracle_truth *tr = (oracle_truth *)malloc(sizeof(oracle_truth) * (size_t)(nt + 1));
    for (int64_t k = 0; k < nt; ++k) { tr[k].event = (uint32_t)(k & 1); tr[k].pad = 0u; tr[k].a = 3.0 * x[k]; tr[k].b = -2.5 * y[k]; }
    int32_t *cmatch = (int32_t *)malloc(4 * (size_t)(nm + 1)), *tmatch = (int32_t *)malloc(4 * (size_t)(nt + 1));
    oracle_match_summary ms;
    const int mrc = oracle_match_truth(&g, mg, nm > 0 ? nm : 0, tr, nt, 200.0, 0.95, cmatch, tmatch, &ms);
    uint64_t h = 1469598103934665603ull;
    h = fnv(M, cells * 4, h);
    printf("match_rc %d found %lld fake %lld match_hash %llu ", mrc, (long long)ms.n_found, (long long)ms.n_fake,
           (unsigned long long)fnv(cmatch, 4 * (size_t)(nm > 0 ? nm : 0), fnv(tmatch, 4 * (size_t)nt, 7)));
    printf("votes %lld matrix_hash %llu peaks %lld peaks_hash %llu tracks_hash %llu merged %lld merged_hash %llu planes_hash %llu\n",
           (long long)votes, (unsigned long long)h, (long long)np,
           (unsigned long long)fnv(pk, sizeof(oracle_peak) * (size_t)np, 7),
           (unsigned long long)fnv(rho, 8 * (size_t)np, fnv(phi, 8 * (size_t)np, 7)), (long long)nm,
           (unsigned long long)fnv(mg, sizeof(oracle_merged) * (size_t)(nm > 0 ? nm : 0), 7),
           (unsigned long long)fnv(plane, 4 * (size_t)n, fnv(bins, 4 * (size_t)n * (size_t)g.n_a, 7)));
    free(x); free(y); free(z); free(M); free(plane); free(bins); free(pk); free(rho); free(phi); free(mg); free(tr); free(cmatch); free(tmatch);
    return 0;
}

/*
 * ht_diag.h -- DIAGNOSTICS of libht: entry points for tests and for bench.py's measurement legs.
 *
 * Nothing here is a step of the method (include/ht.h holds those).  They exist so that the parity tests can compare
 * the library's tables with the oracle's, so that bench.py can count launches and report the launch geometry, and so
 * that the rooflines DESIGN.md quotes (store ceiling, shared-memory vote rate) are measured by committed code in the
 * same run as the kernels they bound ("r_atom ... must be micro-benchmarked").
 */
#ifndef HT_DIAG_H_
#define HT_DIAG_H_

#include "ht.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Host-only: the tables the library builds and uploads (SPEC.md section 1), for bit-for-bit comparison in tests.
 * two_a[n_a] (may be NULL), t_theta[n_theta+1], p_phi[n_phi+1], d_ab[2] = {dA, dB}.  Needs no GPU. */
HT_API int ht_tables_host(const ht_config *cfg, float *two_a, float *t_theta, float *p_phi, float *d_ab);

/* Number of kernels this context has launched so far (host-side counter; for bench.py's gpu_launches). */
HT_API int64_t ht_kernel_launches(const ht_ctx *ctx);

/* Launch geometry of the last ht_fill / ht_peaks: out[0]=fill grid, out[1]=fill block, out[2]=fill dynamic smem bytes,
 * out[3]=rows stored per tile, out[4]=peaks grid, out[5]=peaks block, out[6]=SM count, out[7]=classification mode of
 * the last fill (1: one event, hit index in shared memory; 0: batch, buckets in global memory). */
HT_API int ht_launch_info(const ht_ctx *ctx, int32_t out[8]);

/* Self-test of the arithmetic shortcut of the vote loop ("Exact division"): evaluates n_pairs
 * pseudo-random quotients a/b (all significand patterns, exponents across and just outside the range the shortcut is
 * used on) both ways on `device` and returns in *h_mismatches how many differ in any bit from __fdiv_rn (must be 0).
 * Synchronous; allocates and frees 8 bytes of device memory. */
HT_API int ht_selftest_division(int32_t device, uint64_t n_pairs, uint64_t seed, uint64_t *h_mismatches);

/* cudaMemsetAsync(d_dst, value, bytes) on cuda_stream: the driver's own way of writing `bytes` once -- bench.py times it
 * on the same output matrices as the fill kernel and prints it as the store ceiling beside the roofline fraction. */
HT_API int ht_diag_memset(void *d_dst, int32_t value, size_t bytes, void *cuda_stream);

/*
 * Micro-benchmark of the ways a warp can add 1 to cells of a shared-memory row it owns (the accumulate step a2,
 * PAPER.md:25 "incremented by one"): the denominator of the vote-loop roofline.  One CTA of 1024 threads per SM, 30
 * voting warps, each on its own 4 KB row (1024 uint32 cells), `iters` rounds of 4 independent votes per lane.
 * h_rates[p] receives the rate of pattern p in votes (lanes) per clock per SM (median over the CTAs, clock64):
 */
enum {
    HT_DIAG_RED_RANDOM = 0,      /* red.shared.add, pseudo-random cells (what votes of different hits look like) */
    HT_DIAG_RED_RANDOM_71 = 1,   /* the same with 71 % of the lanes active (the in-range fraction of the votes) */
    HT_DIAG_RED_NO_CONFLICT = 2, /* red.shared.add, 32 lanes on 32 different banks */
    HT_DIAG_RED_TWO_WAY = 3,     /* red.shared.add, pairs of lanes on the same cell */
    HT_DIAG_RED_SAME = 4,        /* red.shared.add, all lanes on one cell */
    HT_DIAG_ATOM_RANDOM = 5,     /* atom.shared.add (value returned), pseudo-random cells */
    HT_DIAG_ATOM_NO_CONFLICT = 6,
    HT_DIAG_ATOM_SAME = 7,
    HT_DIAG_RMW_RANDOM = 8,      /* plain ld / add / st, pseudo-random cells: NOT a correct vote (duplicates are lost) -- the floor */
    HT_DIAG_TAG_RANDOM = 9,      /* warp-private vote: ld, st with the lane tagged, ld, winners st, losers red (exact) */
    HT_DIAG_MATCH_RANDOM = 10,   /* warp-private vote: match.any on the cell, the first lane of a group adds the group's size (exact) */
    HT_DIAG_TAG_RANDOM_71 = 11,  /* HT_DIAG_TAG_RANDOM with 71 % of the lanes active */
    HT_DIAG_N_PATTERNS = 12
};
/* h_rates[HT_DIAG_N_PATTERNS]; *h_sum_errors = number of (CTA, warp, pattern) rows whose cell sum differs from the votes
 * cast in an EXACT pattern (everything but HT_DIAG_RMW_RANDOM; must be 0).  Synchronous. */
HT_API int ht_diag_vote_rates(int32_t device, int32_t iters, double *h_rates, uint64_t *h_sum_errors);

#ifdef __cplusplus
}
#endif
#endif /* HT_DIAG_H_ */

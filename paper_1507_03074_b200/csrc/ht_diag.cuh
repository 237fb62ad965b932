// ht_diag.cuh -- device code of the diagnostics (include/ht_diag.h): the self-test of the hoisted division and the
// micro-benchmark of the shared-memory vote (the denominator of the vote-loop roofline).
#pragma once

#include "ht_device.cuh"

namespace ht {

// ------------------------------------------------------------------------------------------------
// Self-test of the hoisted division (ht_selftest_division): pseudo-random pairs (a, b) with every significand pattern
// and exponents across (and just outside) the moderate range; fdiv_rn_hoisted must return the bits of __fdiv_rn.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint64_t mix64(uint64_t z)
{
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}
__device__ __forceinline__ float float_from_bits(uint32_t sign, int exp2, uint32_t mant23)
{
    return __uint_as_float((sign << 31) | ((uint32_t)(exp2 + 127) << 23) | (mant23 & 0x7FFFFFu));
}
__global__ void selftest_division_kernel(unsigned long long n_pairs, unsigned long long seed, unsigned long long *mismatches)
{
    unsigned long long bad = 0;
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_pairs; i += stride) {
        const uint64_t r0 = mix64(seed + 2ull * i), r1 = mix64(seed + 2ull * i + 1ull);
        // exponents in [-64, 64]: the moderate range [-60, 60] and a margin that must take the generic path
        const int ea = (int)(r0 % 129ull) - 64, eb = (int)((r0 >> 8) % 129ull) - 64;
        uint32_t ma = (uint32_t)(r1 & 0x7FFFFFu), mb = (uint32_t)((r1 >> 23) & 0x7FFFFFu);
        const uint32_t pick = (uint32_t)(r0 >> 40) & 7u;                // a share of extreme significands
        if (pick == 0u) ma = 0u; else if (pick == 1u) ma = 0x7FFFFFu;
        if (pick == 2u) mb = 0u; else if (pick == 3u) mb = 0x7FFFFFu;
        const float a = float_from_bits((uint32_t)(r0 >> 62) & 1u, ea, ma);
        const float b = float_from_bits((uint32_t)(r0 >> 63) & 1u, eb, mb);
        const float want = __fdiv_rn(a, b);
        const float got = fdiv_rn_hoisted(a, make_divisor(b));
        if (__float_as_uint(want) != __float_as_uint(got)) ++bad;
    }
    if (bad) atomicAdd(mismatches, bad);
}

// ------------------------------------------------------------------------------------------------
// ht_diag_vote_rates: how fast can the warps of one SM add 1 to cells of shared-memory rows they own?
// Same shape as the voters of fill_tiles_kernel: one CTA of 1024 threads per SM, the first 30 warps each own a 4 KB
// row; a lane casts one vote per round.  Patterns: include/ht_diag.h.
// ------------------------------------------------------------------------------------------------
constexpr int kDiagRowCells = 1024;
constexpr int kDiagWarps = 30;

__device__ __forceinline__ uint32_t lds_u32(uint32_t addr)
{
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void sts_u32(uint32_t addr, uint32_t v)
{
    asm volatile("st.shared.u32 [%0], %1;" :: "r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ uint32_t xorshift32(uint32_t &s)
{
    s ^= s << 13;
    s ^= s >> 17;
    s ^= s << 5;
    return s;
}

struct DiagOut {
    unsigned long long cycles, votes;
    uint32_t sum_errors, pad;
};

template <int PATTERN>
__global__ void __launch_bounds__(1024, 1) vote_rates_kernel(int iters, DiagOut *out)
{
    extern __shared__ __align__(16) uint32_t s_rows[];
    __shared__ unsigned long long s_t0[32], s_t1[32], s_votes[32];
    __shared__ uint32_t s_err[32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const bool voter = warp < kDiagWarps;
    const uint32_t row_addr = smem_addr(s_rows) + (uint32_t)(voter ? warp : 0) * (kDiagRowCells * 4u);
    if (voter)
        for (int c = lane; c < kDiagRowCells; c += 32) s_rows[warp * kDiagRowCells + c] = 0u;
    uint32_t rng = 0x9E3779B9u * (uint32_t)(blockIdx.x * 1024 + tid + 1);
    uint32_t cast = 0u, sink = 0u;
    __syncthreads();
    const long long t0 = clock64();
    if (voter) {
        constexpr bool kPartial = PATTERN == HT_DIAG_RED_RANDOM_71 || PATTERN == HT_DIAG_TAG_RANDOM_71;
#pragma unroll 1
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const uint32_t r = xorshift32(rng);
                const uint32_t base = (uint32_t)(it * 4 + u) * 32u;
                uint32_t cell;
                if constexpr (PATTERN == HT_DIAG_RED_NO_CONFLICT || PATTERN == HT_DIAG_ATOM_NO_CONFLICT) cell = (base + (uint32_t)lane) & 1023u;
                else if constexpr (PATTERN == HT_DIAG_RED_TWO_WAY) cell = (base + (uint32_t)(lane >> 1)) & 1023u;
                else if constexpr (PATTERN == HT_DIAG_RED_SAME || PATTERN == HT_DIAG_ATOM_SAME) cell = base & 1023u;
                else cell = r & 1023u;
                const bool active = kPartial ? (((r >> 12) & 127u) < 91u) : true;
                const uint32_t a = row_addr + cell * 4u;
                if constexpr (PATTERN <= HT_DIAG_RED_SAME) {
                    if (active) red_shared_inc(a);
                } else if constexpr (PATTERN <= HT_DIAG_ATOM_SAME) {
                    if (active) sink += atom_shared_inc(a);
                } else if constexpr (PATTERN == HT_DIAG_RMW_RANDOM) {
                    if (active) sts_u32(a, lds_u32(a) + 1u);
                    __syncwarp();
                } else if constexpr (PATTERN == HT_DIAG_TAG_RANDOM || PATTERN == HT_DIAG_TAG_RANDOM_71) {
                    // exact without an atomic in the common case: every lane writes count+1 with its lane number in the
                    // top bits; exactly one write per cell survives; that lane ("winner") leaves the clean count, the
                    // others add their vote afterwards
                    uint32_t nw = 0u;
                    bool win = true;
                    if (active) {
                        nw = lds_u32(a) + 1u;
                        sts_u32(a, nw | ((uint32_t)lane << 27));
                    }
                    __syncwarp();
                    if (active) {
                        win = (lds_u32(a) >> 27) == (uint32_t)lane;
                        if (win) sts_u32(a, nw);
                    }
                    __syncwarp();
                    if (active && !win) red_shared_inc(a);
                    __syncwarp();
                } else {                                            // HT_DIAG_MATCH_RANDOM
                    const unsigned act = __ballot_sync(0xffffffffu, active);
                    if (active) {
                        const unsigned peers = __match_any_sync(act, cell);
                        if ((unsigned)lane == (unsigned)(__ffs((int)peers) - 1)) sts_u32(a, lds_u32(a) + (uint32_t)__popc(peers));
                    }
                    __syncwarp();
                }
                cast += active ? 1u : 0u;
            }
        }
    }
    const long long t1 = clock64();
    __syncwarp();
    // bookkeeping: votes cast by the warp, sum of its row
    uint32_t sum = 0u;
    if (voter)
        for (int c = lane; c < kDiagRowCells; c += 32) sum += lds_u32(row_addr + (uint32_t)c * 4u);
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        cast += __shfl_xor_sync(0xffffffffu, cast, d);
        sum += __shfl_xor_sync(0xffffffffu, sum, d);
    }
    if (lane == 0) {
        s_t0[warp] = (unsigned long long)t0;
        s_t1[warp] = (unsigned long long)t1;
        s_votes[warp] = voter ? cast : 0u;
        s_err[warp] = (voter && PATTERN != HT_DIAG_RMW_RANDOM && sum != cast) ? 1u : 0u;
    }
    __syncthreads();
    if (tid == 0) {
        unsigned long long lo = s_t0[0], hi = s_t1[0], v = 0ull;
        uint32_t err = 0u;
        for (int w = 0; w < kDiagWarps; ++w) {
            lo = s_t0[w] < lo ? s_t0[w] : lo;
            hi = s_t1[w] > hi ? s_t1[w] : hi;
            v += s_votes[w];
            err += s_err[w];
        }
        DiagOut o;
        o.cycles = hi - lo; o.votes = v; o.sum_errors = err; o.pad = sink == 0xFFFFFFFFu ? 1u : 0u;
        out[blockIdx.x] = o;
    }
}

}  // namespace ht

// ht_merge.cuh -- device code of f3 beyond the read-out: ridge merging of a peak list into
// track candidates (SPEC.md section 5, reading R19) and truth matching of the candidates (SPEC.md section 6, reading R20).
// PAPER.md:25 goes from local maxima straight to "real tracks"; PAPER.md:29-33 (Fig. 1) shows their rho, phi "together with
// the corresponding resolutions".  These lists are short (hundreds to a few ten thousand records): nothing here is tuned,
// every kernel is launch-bound.
#pragma once

#include "ht_device.cuh"

namespace ht {

struct CandOut {                    // == ht_candidate
    uint32_t event, cell, count, n_peaks;
    float rho, phi;
};
struct TruthIn {                    // == ht_truth
    uint32_t event, pad;
    double a, b;
};
struct MatchSummary {               // == ht_match_summary
    long long n_cand, n_truth, n_matched, n_fake, n_found, n_duplicate;
    double sum_drho, sum_drho2, sum_dphi, sum_dphi2;
};

// ---- ridge merging ------------------------------------------------------------------------------------------------------
// Peaks are grouped by (event, plane) with a counting sort on the context's (event, plane) counters (the same two arrays
// the batch classification of the fill uses), then one CTA per group finds the connected components of the link graph
// (Chebyshev distance of the (a, b) cells <= window) by label propagation: every peak repeatedly takes the smallest label
// among itself and the peaks it is linked to, until nothing changes; the labels of a component converge to the smallest
// position in it.  The peak at that position ("root") then walks its component once: members, representative (largest
// count, smallest cell among equals), and emits the candidate with the rho, phi of the representative's cell.

__device__ __forceinline__ uint32_t group_of_peak(const PeakOut &p, const Geom &g, int planes_all)
{
    const uint32_t plane = p.cell / ((uint32_t)g.n_a * (uint32_t)g.n_b);        // plane of the FULL matrix
    return p.event * (uint32_t)planes_all + plane;
}

constexpr uint32_t kNoSlot = 0xFFFFFFFFu;   // a record whose event or cell lies outside the context's capacity: left out

__global__ void merge_count_kernel(const PeakOut *__restrict__ peaks, uint32_t n, Geom g, int planes_all, uint32_t max_events,
                                   uint32_t *counts, uint32_t *slot)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const PeakOut p = peaks[i];
    const bool ok = p.event < max_events && (unsigned long long)p.cell < (unsigned long long)planes_all * g.n_a * g.n_b;
    slot[i] = ok ? atomicAdd(&counts[group_of_peak(p, g, planes_all)], 1u) : kNoSlot;
}

// one CTA: exclusive scan of counts[0 .. n_groups) into start[0 .. n_groups]; counts are left zero (as the fill wants them)
__global__ void merge_scan_kernel(uint32_t *counts, int32_t *start, uint32_t n_groups)
{
    __shared__ uint32_t s_warp[32];
    __shared__ uint32_t s_carry;
    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    if (tid == 0) s_carry = 0u;
    __syncthreads();
    for (uint32_t base = 0; base < n_groups; base += blockDim.x) {
        const uint32_t k = base + tid;
        const uint32_t c = k < n_groups ? counts[k] : 0u;
        uint32_t incl = c;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= (uint32_t)d) incl += t;
        }
        if (lane == 31u) s_warp[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            uint32_t w = lane < (blockDim.x >> 5) ? s_warp[lane] : 0u;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const uint32_t t = __shfl_up_sync(0xffffffffu, w, d);
                if (lane >= (uint32_t)d) w += t;
            }
            s_warp[lane] = w;                                           // inclusive over the warps
        }
        __syncthreads();
        const uint32_t before = s_carry + (warp ? s_warp[warp - 1] : 0u) + incl - c;
        if (k < n_groups) {
            start[k] = (int32_t)before;
            counts[k] = 0u;
        }
        __syncthreads();
        if (tid == blockDim.x - 1) s_carry = before + c;
        __syncthreads();
    }
    if (tid == 0) start[n_groups] = (int32_t)s_carry;
}

__global__ void merge_scatter_kernel(const PeakOut *__restrict__ peaks, uint32_t n, Geom g, int planes_all,
                                     const int32_t *__restrict__ start, const uint32_t *__restrict__ slot, uint32_t *order)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n || slot[i] == kNoSlot) return;
    order[(uint32_t)start[group_of_peak(peaks[i], g, planes_all)] + slot[i]] = i;
}

// one CTA per (event, plane) group; order[] holds the peaks of group k at [start[k], start[k+1]); label[] is scratch.
// Groups of up to kMergeSmem peaks keep their (a, b) cells, counts and labels in shared memory (sorted by cell when they
// hold more than kMergeSortFrom peaks); larger groups work on global memory.
constexpr int kMergeThreads = 1024;
constexpr int kMergeSmem = 2048;
constexpr int kMergeSortFrom = 192;  // groups with more peaks are sorted by cell first (config 2's planes hold ~12, at most ~70)

__global__ void __launch_bounds__(kMergeThreads)
merge_groups_kernel(const PeakOut *__restrict__ peaks, Geom g, const int32_t *__restrict__ start,
                    const uint32_t *__restrict__ order, uint32_t *label_global, uint32_t window,
                    CandOut *__restrict__ out, uint32_t capacity, uint32_t *n_out)
{
    __shared__ uint32_t s_ab[kMergeSmem];                               // a << 16 | b  (both < 65536: checked by the host)
    __shared__ uint32_t s_label[kMergeSmem];
    __shared__ uint32_t s_cnt[kMergeSmem];                              // the peaks' counts (the emission walks all members of a component)
    const int lo = start[blockIdx.x], hi = start[blockIdx.x + 1];
    const int m = hi - lo;
    if (m <= 0) return;
    const uint32_t NB = (uint32_t)g.n_b, NA = (uint32_t)g.n_a;
    const bool in_smem = m <= kMergeSmem;
    uint32_t *label = in_smem ? s_label : label_global + lo;
    auto ab_of = [&](int i) -> uint32_t {
        if (in_smem) return s_ab[i];
        const uint32_t cell = peaks[order[lo + i]].cell;
        return (((cell / NB) % NA) << 16) | (cell % NB);
    };
    for (int i = threadIdx.x; i < m; i += blockDim.x) {
        label[i] = (uint32_t)i;
        if (in_smem) {
            const PeakOut p = peaks[order[lo + i]];
            s_ab[i] = (((p.cell / NB) % NA) << 16) | (p.cell % NB);
            s_cnt[i] = p.count;
        }
    }
    __syncthreads();
    // A group in shared memory is sorted by cell (a, then b; bitonic, the counts travel along): the peaks that can be linked
    // to position i -- |a - a_i| <= window -- are then a contiguous range around i, and a sweep tests a few dozen pairs per
    // peak instead of m (a dense plane of a 20000-hit event holds a thousand peaks).  Positions, and with them roots,
    // are positions of the sorted order; what is emitted does not depend on which member is the root.
    const bool sorted = in_smem && m > kMergeSortFrom;                  // (small groups: the plain all-pairs sweep is faster)
    if (sorted) {
        int padded = 2;
        while (padded < m) padded <<= 1;
        for (int i = m + (int)threadIdx.x; i < padded; i += blockDim.x) {
            s_ab[i] = 0xffffffffu;                                      // (above every key: a, b < 65536 and a < NA <= 65535)
            s_cnt[i] = 0u;
        }
        __syncthreads();
        for (int k = 2; k <= padded; k <<= 1) {
            for (int j = k >> 1; j > 0; j >>= 1) {
                for (int i = threadIdx.x; i < padded; i += blockDim.x) {
                    const int x = i ^ j;
                    if (x > i) {
                        const uint32_t ki = s_ab[i], kx = s_ab[x];
                        const bool up = (i & k) == 0;
                        if (up ? ki > kx : ki < kx) {
                            s_ab[i] = kx;
                            s_ab[x] = ki;
                            const uint32_t c = s_cnt[i];
                            s_cnt[i] = s_cnt[x];
                            s_cnt[x] = c;
                        }
                    }
                }
                __syncthreads();
            }
        }
    }
    // Connected components by hooking and flattening.  A label is a position of the same component, never larger than the
    // position that holds it; a position that holds itself is a root.  Every sweep starts with FLAT labels (each position
    // holds its root): a position looks for the smallest root among the positions linked to it and hooks its OWN ROOT under
    // it (atomicMin), which merges whole trees, not single positions -- a ridge of a thousand peaks converges in a handful
    // of sweeps instead of one sweep per window length (20000-hit event, 1049 peaks in one plane: 3.9 ms -> see DESIGN.md);
    // then every position follows its labels down to the root again.  No sweep hooks anything: every linked pair shares
    // its root, and the root of a component is its smallest position, as before.
    auto root_of = [&](uint32_t x) -> uint32_t {
        for (uint32_t up = *reinterpret_cast<volatile uint32_t *>(&label[x]); up < x;
             up = *reinterpret_cast<volatile uint32_t *>(&label[x])) x = up;
        return x;
    };
    for (;;) {
        int changed = 0;
        for (int i = threadIdx.x; i < m; i += blockDim.x) {
            const uint32_t abi = ab_of(i);
            const int ai = (int)(abi >> 16), bi = (int)(abi & 0xFFFFu);
            uint32_t l = 0xffffffffu;
            auto look = [&](int j) -> bool {                           // false: row a_j is more than `window` rows away
                const uint32_t abj = ab_of(j);
                const int da = abs(ai - (int)(abj >> 16)), db = abs(bi - (int)(abj & 0xFFFFu));
                if ((uint32_t)max(da, db) <= window) l = min(l, *reinterpret_cast<volatile uint32_t *>(&label[j]));
                return (uint32_t)da <= window;
            };
            if (sorted) {                                               // sorted by (a, b): outwards from i while the rows are near
                for (int j = i; j >= 0 && look(j); --j) { }
                for (int j = i + 1; j < m && look(j); ++j) { }
            } else {
                for (int j = 0; j < m; ++j) look(j);
            }
            // (labels only ever decrease, and stay positions of the component: a label read while others hook is as good)
            l = root_of(l);                                             // (i is linked to itself: l is a position)
            const uint32_t mine = root_of((uint32_t)i);
            if (l < mine) {
                atomicMin(&label[mine], l);
                changed = 1;
            }
        }
        const int any = __syncthreads_or(changed);
        for (int i = threadIdx.x; i < m; i += blockDim.x) {
            const uint32_t r = root_of((uint32_t)i);
            if (r < (uint32_t)i) atomicMin(&label[i], r);
        }
        __syncthreads();
        if (!any) break;
    }
    // roots (label == own position) emit their component
    for (int i = threadIdx.x; i < m; i += blockDim.x) {
        if (label[i] != (uint32_t)i) continue;
        uint32_t members = 0u;
        PeakOut best = peaks[order[lo + i]];
        if (in_smem) {
            // all peaks of a group share event and plane: a member's cell follows from its (a, b).  (Position i of the
            // sorted order is not peak order[lo + i]: the record above only lends its event and plane.)
            const uint32_t plane_base = best.cell - (((best.cell / NB) % NA) * NB + best.cell % NB);
            best.count = 0u;
            best.cell = 0xffffffffu;
            for (int j = 0; j < m; ++j) {
                if (label[j] != (uint32_t)i) continue;
                ++members;
                const uint32_t abj = s_ab[j], cnt = s_cnt[j];
                const uint32_t cell = plane_base + (abj >> 16) * NB + (abj & 0xFFFFu);
                if (cnt > best.count || (cnt == best.count && cell < best.cell)) {
                    best.count = cnt;
                    best.cell = cell;
                }
            }
        } else {
            for (int j = 0; j < m; ++j) {
                if (label[j] != (uint32_t)i) continue;
                ++members;
                const PeakOut p = peaks[order[lo + j]];
                if (p.count > best.count || (p.count == best.count && p.cell < best.cell)) best = p;
            }
        }
        const uint32_t at = atomicAdd(n_out, 1u);
        if (at < capacity) {
            const uint32_t ia = (best.cell / NB) % NA, ib = best.cell % NB;
            const float A = __fadd_rn(g.a_min, __fmul_rn(__fadd_rn((float)ia, 0.5f), g.dA));   // bin centres (R5, R18)
            const float B = __fadd_rn(g.b_min, __fmul_rn(__fadd_rn((float)ib, 0.5f), g.dB));
            CandOut c;
            c.event = best.event; c.cell = best.cell; c.count = best.count; c.n_peaks = members;
            c.rho = __fsqrt_rn(__fadd_rn(__fmul_rn(A, A), __fmul_rn(B, B)));
            c.phi = atan2f(B, A);
            out[at] = c;
        }
    }
}

// ---- truth matching -----------------------------------------------------------------------------------------------------
// Every decision is a binary64 comparison of values computed with the operations and in the order of SPEC.md section 6
// (the library is built with --fmad=false: no contraction; sqrt is correctly rounded), so the matches are reproducible bit for bit by any IEEE implementation of that text.

struct Centre {
    double a, b, rho;
};
__device__ __forceinline__ Centre centre_of_cell(uint32_t cell, const Geom &g)
{
    const uint32_t ib = cell % (uint32_t)g.n_b, ia = (cell / (uint32_t)g.n_b) % (uint32_t)g.n_a;
    const float Af = __fadd_rn(g.a_min, __fmul_rn(__fadd_rn((float)ia, 0.5f), g.dA));
    const float Bf = __fadd_rn(g.b_min, __fmul_rn(__fadd_rn((float)ib, 0.5f), g.dB));
    Centre c;
    c.a = (double)Af;
    c.b = (double)Bf;
    c.rho = sqrt(__dadd_rn(__dmul_rn(c.a, c.a), __dmul_rn(c.b, c.b)));
    return c;
}
__device__ __forceinline__ bool compatible(const Centre &c, double At, double Bt, double w_rho, double cos_w_phi, double &d2)
{
    const double rho_t = sqrt(__dadd_rn(__dmul_rn(At, At), __dmul_rn(Bt, Bt)));
    const double dr = __dsub_rn(c.rho, rho_t);
    if (!(fabs(dr) <= w_rho)) return false;
    const double dot = __dadd_rn(__dmul_rn(c.a, At), __dmul_rn(c.b, Bt));
    if (!(dot >= __dmul_rn(cos_w_phi, __dmul_rn(c.rho, rho_t)))) return false;
    const double ea = __dsub_rn(c.a, At), eb = __dsub_rn(c.b, Bt);
    d2 = __dadd_rn(__dmul_rn(ea, ea), __dmul_rn(eb, eb));
    return true;
}

// cand_match[c]: the compatible truth record of smallest d2 (ties: smallest index), or -1
__global__ void match_candidates_kernel(const CandOut *__restrict__ cand, uint32_t n_cand, const TruthIn *__restrict__ truth,
                                        uint32_t n_truth, Geom g, double w_rho, double cos_w_phi, int32_t *cand_match)
{
    const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n_cand) return;
    const CandOut cd = cand[c];
    const Centre cc = centre_of_cell(cd.cell, g);
    int best = -1;
    double best_d2 = 0.0;
    for (uint32_t t = 0; t < n_truth; ++t) {
        if (truth[t].event != cd.event) continue;
        double d2;
        if (!compatible(cc, truth[t].a, truth[t].b, w_rho, cos_w_phi, d2)) continue;
        if (best < 0 || d2 < best_d2) { best = (int)t; best_d2 = d2; }
    }
    cand_match[c] = best;
}

// truth_match[t]: among the candidates matched to t the one of smallest d2 (ties: smallest cell), or -1; and the summary
__global__ void match_truth_kernel(const CandOut *__restrict__ cand, uint32_t n_cand, const TruthIn *__restrict__ truth,
                                   uint32_t n_truth, Geom g, double w_rho, double cos_w_phi,
                                   const int32_t *__restrict__ cand_match, int32_t *truth_match, MatchSummary *sum)
{
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long found = 0ull;
    double dr = 0.0, dp = 0.0;
    if (t < n_truth) {
        const double At = truth[t].a, Bt = truth[t].b;
        int best = -1;
        double best_d2 = 0.0;
        Centre bc{};
        for (uint32_t c = 0; c < n_cand; ++c) {
            if (cand_match[c] != (int32_t)t) continue;
            const Centre cc = centre_of_cell(cand[c].cell, g);
            double d2 = 0.0;
            compatible(cc, At, Bt, w_rho, cos_w_phi, d2);               // (it is: cand_match says so) -- for d2
            if (best < 0 || d2 < best_d2 || (d2 == best_d2 && cand[c].cell < cand[best].cell)) { best = (int)c; best_d2 = d2; bc = cc; }
        }
        truth_match[t] = best;
        if (best >= 0) {
            found = 1ull;
            dr = __dsub_rn(bc.rho, sqrt(__dadd_rn(__dmul_rn(At, At), __dmul_rn(Bt, Bt))));
            dp = atan2(__dsub_rn(__dmul_rn(At, bc.b), __dmul_rn(Bt, bc.a)), __dadd_rn(__dmul_rn(bc.a, At), __dmul_rn(bc.b, Bt)));
        }
    }
    if (found) {
        atomicAdd(reinterpret_cast<unsigned long long *>(&sum->n_found), 1ull);
        atomicAdd(&sum->sum_drho, dr);
        atomicAdd(&sum->sum_drho2, dr * dr);
        atomicAdd(&sum->sum_dphi, dp);
        atomicAdd(&sum->sum_dphi2, dp * dp);
    }
}

// the counts of the summary that depend on cand_match only (one thread per candidate), then n_duplicate by the last block
__global__ void match_summary_kernel(const int32_t *__restrict__ cand_match, uint32_t n_cand, uint32_t n_truth, MatchSummary *sum)
{
    const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c == 0) {
        sum->n_cand = (long long)n_cand;
        sum->n_truth = (long long)n_truth;
    }
    if (c >= n_cand) return;
    if (cand_match[c] >= 0) atomicAdd(reinterpret_cast<unsigned long long *>(&sum->n_matched), 1ull);
    else atomicAdd(reinterpret_cast<unsigned long long *>(&sum->n_fake), 1ull);
}
__global__ void match_finish_kernel(MatchSummary *sum) { sum->n_duplicate = sum->n_matched - sum->n_found; }

}  // namespace ht

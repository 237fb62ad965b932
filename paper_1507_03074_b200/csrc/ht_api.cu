// ht_api.cu -- C ABI of libht (include/ht.h): argument validation, table construction (SPEC.md section 1),
// workspace management and kernel launches.  No torch types, no exceptions across the boundary.
#include "../../include/ht.h"
#include "ht_device.cuh"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

namespace {

thread_local char g_cuda_err[256] = "no CUDA error recorded";

int cuda_fail(cudaError_t e, const char *what)
{
    std::snprintf(g_cuda_err, sizeof g_cuda_err, "CUDA error in %s: %s", what, cudaGetErrorString(e));
    return HT_ERR_CUDA;
}

#define HT_CUDA(call)                                        \
    do {                                                     \
        cudaError_t e__ = (call);                            \
        if (e__ != cudaSuccess) return cuda_fail(e__, #call); \
    } while (0)

constexpr double kPi = 3.14159265358979323846;

int env_int(const char *name, int dflt)
{
    const char *s = std::getenv(name);
    if (!s || !*s) return dflt;
    return std::atoi(s);
}

bool config_ok(const ht_config *c)
{
    if (!c) return false;
    if (c->n_theta < 1 || c->n_phi < 1 || c->n_a < 1 || c->n_b < 1) return false;
    const float r[8] = {c->a_min, c->a_max, c->b_min, c->b_max, c->theta_min, c->theta_max, c->phi_min, c->phi_max};
    for (float v : r)
        if (!std::isfinite(v)) return false;
    if (!(c->a_min < c->a_max) || !(c->b_min < c->b_max)) return false;
    if (!(c->theta_min < c->theta_max) || !(c->phi_min < c->phi_max)) return false;
    if (c->theta_min < 0.0f || c->phi_min < 0.0f) return false;
    if (c->theta_max > (float)kPi || c->phi_max > (float)(2.0 * kPi)) return false;
    const unsigned long long cells =
        (unsigned long long)c->n_theta * (unsigned long long)c->n_phi * (unsigned long long)c->n_a * (unsigned long long)c->n_b;
    if (cells >= (1ull << 32)) return false;          // ht_peak.cell is uint32
    if ((long long)c->n_theta * (long long)c->n_phi > (1ll << 30)) return false;
    if (c->plane_begin < 0 || c->plane_count < 0) return false;
    if (c->plane_count > 0 && (long long)c->plane_begin + c->plane_count > (long long)c->n_theta * c->n_phi) return false;
    if (c->plane_count == 0 && c->plane_begin != 0) return false;
    return true;
}

double cot(double t) { return std::cos(t) / std::sin(t); }

// "diamond" pseudo-angle of an edge, in double (SPEC.md section 1)
double pseudo_angle(double phi)
{
    const double c = std::cos(phi), s = std::sin(phi);
    const double m = std::fabs(c) + std::fabs(s);
    return (s >= 0.0) ? 1.0 - c / m : 3.0 + c / m;
}

void build_tables(const ht_config *c, float *two_a, float *tth, float *pph, float *d_ab)
{
    // volatile: one IEEE binary32 rounding per operation, whatever the host compiler's contraction setting
    volatile float dA = (c->a_max - c->a_min) / (float)c->n_a;
    volatile float dB = (c->b_max - c->b_min) / (float)c->n_b;
    d_ab[0] = dA;
    d_ab[1] = dB;
    if (two_a) {
        for (int i = 0; i < c->n_a; ++i) {
            volatile float fi = (float)i + 0.5f;
            volatile float prod = fi * dA;
            volatile float ac = c->a_min + prod;
            two_a[i] = 2.0f * ac;
        }
    }
    const bool th_full = c->theta_max >= (float)kPi;
    const bool ph_full = c->phi_max >= (float)(2.0 * kPi);
    const double thlo = (double)c->theta_min, thhi = th_full ? kPi : (double)c->theta_max;
    const double phlo = (double)c->phi_min, phhi = ph_full ? 2.0 * kPi : (double)c->phi_max;
    tth[0] = (c->theta_min <= 0.0f) ? INFINITY : (float)cot(thlo);
    for (int k = 1; k < c->n_theta; ++k) tth[k] = (float)cot(thlo + ((thhi - thlo) * (double)k) / (double)c->n_theta);
    tth[c->n_theta] = th_full ? -INFINITY : (float)cot(thhi);
    pph[0] = (c->phi_min <= 0.0f) ? 0.0f : (float)pseudo_angle(phlo);
    for (int k = 1; k < c->n_phi; ++k) pph[k] = (float)pseudo_angle(phlo + ((phhi - phlo) * (double)k) / (double)c->n_phi);
    pph[c->n_phi] = ph_full ? 4.0f : (float)pseudo_angle(phhi);
}

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

}  // namespace

struct ht_ctx {
    ht_config cfg;
    ht::Geom geom;
    int sm_count = 0;
    int max_smem_optin = 0;
    // device workspace
    float *d_tth = nullptr, *d_pph = nullptr;
    uint32_t *d_counters = nullptr;
    // hit buckets written by the fill kernel's prologue (a0): per-hit vote constants grouped by (event, plane)
    float *d_bx = nullptr, *d_br2 = nullptr, *d_bden = nullptr;
    int32_t *d_hplane = nullptr, *d_hrel = nullptr;   // [max_hits] phase-1 spill
    int32_t *d_bucket_start = nullptr;     // [max_events * (P+1)]
    uint32_t *d_counts = nullptr;          // [max_events * P], zero between calls
    // tile fill launch geometry: per-kernel dynamic shared memory budget ([0]: ht_fill, [1]: fused peaks), and whether
    // the device can run the kernel at all (one CTA of 1024 threads per SM, cooperative launch for mode 0)
    uint32_t bar_epoch = 0;                   // host mirror of the barrier counter that only grows (d_counters[5])
    bool fill_ok = false;
    size_t fill_smem_max[2] = {0, 0};
    // peak scan launch geometry
    int peaks_unroll = 4, peaks_grid_vec4 = 0, peaks_grid_vec1 = 0;
    // host path (ht_run_host)
    unsigned char *d_in = nullptr;     // [offsets | x | y | z], packed per call (one H2D copy)
    unsigned char *h_in = nullptr;     // pinned + mapped mirror of d_in
    unsigned char *d_in_mapped = nullptr;   // device alias of h_in (zero-copy input of single events)
    uint32_t *d_hmh = nullptr;
    unsigned char *h_res = nullptr;    // pinned + mapped: [uint32 n_found, pad to 16][ht_peak x host_peak_capacity]
    unsigned char *d_res = nullptr;    // device alias of h_res: the kernels write the peak list straight to the host
    cudaStream_t host_stream = nullptr;
    int64_t launches = 0;
    int32_t info[8] = {0, 0, 0, 0, 0, 0, 0, 0};
};

namespace {

constexpr size_t kResHeader = 16;

struct WorkspaceSizes {
    size_t tables, counters, buckets, bucket_start, counts, host_hits, host_off, host_mh, host_res, total;
};

WorkspaceSizes workspace_sizes(const ht_config *c)
{
    WorkspaceSizes w{};
    const size_t planes = (size_t)c->n_theta * (size_t)c->n_phi;
    const size_t cells = (c->plane_count > 0 ? (size_t)c->plane_count : planes) * (size_t)c->n_a * (size_t)c->n_b;
    w.tables = align_up(sizeof(float) * (size_t)(c->n_theta + 1 + c->n_phi + 1), 256);
    w.counters = 256;
    w.buckets = 6 * align_up(sizeof(float) * (size_t)c->max_hits, 256);      // hit records (4 words per hit), h_plane, h_rel
    w.bucket_start = align_up(sizeof(int32_t) * (size_t)c->max_events * (planes + 1), 256);
    w.counts = align_up(sizeof(uint32_t) * (size_t)c->max_events * planes, 256);
    if (c->host_slots > 0) {
        w.host_hits = 3 * align_up(sizeof(float) * (size_t)c->max_hits, 16);
        w.host_off = align_up(sizeof(int32_t) * ((size_t)c->max_events + 1), 16);
        w.host_mh = align_up(cells * sizeof(uint32_t) * (size_t)c->host_slots, 256);
        w.host_res = align_up(kResHeader + sizeof(ht_peak) * (size_t)c->host_peak_capacity, 256);
    }
    w.total = w.tables + w.counters + w.buckets + w.bucket_start + w.counts + w.host_hits + w.host_off + w.host_mh;
    return w;
}

// Tile geometry of the fill kernel for one call: the largest slab (rows of NB cells) such that four slabs (two per warp
// group), the row tables, and -- in mode 1 -- the plane offsets and the uint16 hit index fit the CTA's shared memory.
struct FillPlan {
    bool ok = false;
    int mode = 0, rows_slab = 0, hit_cap = 0;
    uint32_t slab_words = 0;
    size_t smem = 0;
};

size_t fill_smem_bytes(const ht_config &c, long long rows, int mode, long long n_hits)
{
    const size_t slab = align_up((size_t)rows * (size_t)c.n_b * 4u, 16);
    size_t b = 2u * slab + 8u * 4u * (size_t)(rows + 4);     // two slabs, two_a[8 ring entries][rows + 4]
    b += align_up(4u * ((size_t)c.n_theta * (size_t)c.n_phi + 1u), 16);      // plane offsets, padded: the staged hits are float4
    if (mode == 1) b += 2u * (size_t)n_hits;
    return align_up(b, 16);
}

int check_fill_args(ht_ctx *ctx, const float *d_x, const float *d_y, const float *d_z, const int32_t *d_off,
                    int32_t n_events, int32_t n_hits_total, uint32_t *d_mh, bool mh_required)
{
    if (!ctx) return HT_ERR_INVALID_ARG;
    if (n_events < 0 || n_hits_total < 0) return HT_ERR_INVALID_ARG;
    if (n_events > ctx->cfg.max_events || n_hits_total > ctx->cfg.max_hits) return HT_ERR_INVALID_ARG;
    if (n_events == 0) return HT_OK;
    if (!d_off || (mh_required && !d_mh)) return HT_ERR_INVALID_ARG;
    if (n_hits_total > 0 && (!d_x || !d_y || !d_z)) return HT_ERR_INVALID_ARG;
    if ((reinterpret_cast<uintptr_t>(d_mh) & 3u) != 0) return HT_ERR_INVALID_ARG;
    return HT_OK;
}

}  // namespace

extern "C" {

int ht_query_sizes(const ht_config *cfg, size_t *mh_bytes_per_event, size_t *ctx_device_bytes)
{
    if (!config_ok(cfg) || cfg->max_events < 1 || cfg->max_hits < 1 || cfg->host_slots < 0) return HT_ERR_INVALID_ARG;
    const size_t planes = cfg->plane_count > 0 ? (size_t)cfg->plane_count : (size_t)cfg->n_theta * (size_t)cfg->n_phi;
    const size_t cells = planes * (size_t)cfg->n_a * (size_t)cfg->n_b;
    if (mh_bytes_per_event) *mh_bytes_per_event = cells * sizeof(uint32_t);
    if (ctx_device_bytes) *ctx_device_bytes = workspace_sizes(cfg).total;
    return HT_OK;
}

int ht_tables_host(const ht_config *cfg, float *two_a, float *t_theta, float *p_phi, float *d_ab)
{
    if (!config_ok(cfg) || !t_theta || !p_phi || !d_ab) return HT_ERR_INVALID_ARG;
    build_tables(cfg, two_a, t_theta, p_phi, d_ab);
    return HT_OK;
}

int ht_create(const ht_config *cfg, ht_ctx **out)
{
    if (!out) return HT_ERR_INVALID_ARG;
    if (!config_ok(cfg) || cfg->max_events < 1 || cfg->max_hits < 1 || cfg->host_slots < 0) return HT_ERR_INVALID_ARG;
    if (cfg->max_hits > INT32_MAX - 65536) return HT_ERR_INVALID_ARG;
    int ndev = 0;
    HT_CUDA(cudaGetDeviceCount(&ndev));
    if (cfg->device < 0 || cfg->device >= ndev) return HT_ERR_INVALID_ARG;
    HT_CUDA(cudaSetDevice(cfg->device));

    ht_ctx *ctx = new (std::nothrow) ht_ctx();
    if (!ctx) return HT_ERR_NOMEM;
    ctx->cfg = *cfg;
    ht::Geom &g = ctx->geom;
    g.n_theta = cfg->n_theta; g.n_phi = cfg->n_phi; g.n_a = cfg->n_a; g.n_b = cfg->n_b;
    g.planes = cfg->plane_count > 0 ? cfg->plane_count : cfg->n_theta * cfg->n_phi;
    g.plane0 = cfg->plane_count > 0 ? cfg->plane_begin : 0;
    g.cells = (unsigned long long)g.planes * (unsigned long long)cfg->n_a * (unsigned long long)cfg->n_b;
    g.cell_base = (uint32_t)((unsigned long long)g.plane0 * (unsigned long long)cfg->n_a * (unsigned long long)cfg->n_b);
    std::vector<float> tth((size_t)cfg->n_theta + 1), pph((size_t)cfg->n_phi + 1);
    float d_ab[2];
    build_tables(cfg, nullptr, tth.data(), pph.data(), d_ab);
    g.a_min = cfg->a_min; g.dA = d_ab[0]; g.b_min = cfg->b_min; g.dB = d_ab[1]; g.nb_f = (float)cfg->n_b;

    cudaError_t e;
    int rc = HT_OK;
    auto fail = [&](int code) { ht_destroy(ctx); return code; };
    if ((e = cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, cfg->device)) != cudaSuccess)
        return fail(cuda_fail(e, "cudaDeviceGetAttribute(SM count)"));
    if ((e = cudaDeviceGetAttribute(&ctx->max_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, cfg->device)) != cudaSuccess)
        return fail(cuda_fail(e, "cudaDeviceGetAttribute(smem optin)"));

    const WorkspaceSizes w = workspace_sizes(cfg);
    auto dmalloc = [&](void **p, size_t bytes, const char *what) -> bool {
        if (bytes == 0) { *p = nullptr; return true; }
        cudaError_t err = cudaMalloc(p, bytes);
        if (err != cudaSuccess) {
            rc = (err == cudaErrorMemoryAllocation) ? HT_ERR_NOMEM : cuda_fail(err, what);
            if (err == cudaErrorMemoryAllocation) cudaGetLastError();
            return false;
        }
        return true;
    };
    if (!dmalloc((void **)&ctx->d_tth, w.tables, "cudaMalloc(tables)")) return fail(rc);
    ctx->d_pph = ctx->d_tth + (cfg->n_theta + 1);
    if (!dmalloc((void **)&ctx->d_counters, w.counters, "cudaMalloc(counters)")) return fail(rc);
    if (!dmalloc((void **)&ctx->d_bx, w.buckets, "cudaMalloc(hit buckets)")) return fail(rc);
    {
        unsigned char *b0 = reinterpret_cast<unsigned char *>(ctx->d_bx);
        const size_t one = w.buckets / 6;
        ctx->d_br2 = reinterpret_cast<float *>(b0 + one);
        ctx->d_bden = reinterpret_cast<float *>(b0 + 2 * one);
        ctx->d_hplane = reinterpret_cast<int32_t *>(b0 + 4 * one);
        ctx->d_hrel = reinterpret_cast<int32_t *>(b0 + 5 * one);
    }
    if (!dmalloc((void **)&ctx->d_bucket_start, w.bucket_start, "cudaMalloc(bucket offsets)")) return fail(rc);
    if (!dmalloc((void **)&ctx->d_counts, w.counts, "cudaMalloc(bucket counts)")) return fail(rc);
    if ((e = cudaMemset(ctx->d_counts, 0, w.counts)) != cudaSuccess) return fail(cuda_fail(e, "cudaMemset(bucket counts)"));
    if ((e = cudaMemcpy(ctx->d_tth, tth.data(), tth.size() * sizeof(float), cudaMemcpyHostToDevice)) != cudaSuccess ||
        (e = cudaMemcpy(ctx->d_pph, pph.data(), pph.size() * sizeof(float), cudaMemcpyHostToDevice)) != cudaSuccess ||
        (e = cudaMemset(ctx->d_counters, 0, w.counters)) != cudaSuccess)
        return fail(cuda_fail(e, "table upload"));

    if (cfg->host_slots > 0) {
        if (!dmalloc((void **)&ctx->d_in, w.host_off + w.host_hits, "cudaMalloc(host input)")) return fail(rc);
        if (!dmalloc((void **)&ctx->d_hmh, w.host_mh, "cudaMalloc(host matrices)")) return fail(rc);
        if ((e = cudaHostAlloc((void **)&ctx->h_in, w.host_off + w.host_hits, cudaHostAllocMapped)) != cudaSuccess)
            return fail(cuda_fail(e, "cudaHostAlloc(input)"));
        if ((e = cudaHostGetDevicePointer((void **)&ctx->d_in_mapped, ctx->h_in, 0)) != cudaSuccess)
            return fail(cuda_fail(e, "cudaHostGetDevicePointer(input)"));
        if ((e = cudaHostAlloc((void **)&ctx->h_res, w.host_res, cudaHostAllocMapped)) != cudaSuccess)
            return fail(cuda_fail(e, "cudaHostAlloc(result)"));
        if ((e = cudaHostGetDevicePointer((void **)&ctx->d_res, ctx->h_res, 0)) != cudaSuccess)
            return fail(cuda_fail(e, "cudaHostGetDevicePointer(result)"));
        if ((e = cudaStreamCreateWithFlags(&ctx->host_stream, cudaStreamNonBlocking)) != cudaSuccess)
            return fail(cuda_fail(e, "cudaStreamCreate"));
    }

    {   // fill kernel: one CTA per SM with as much dynamic shared memory as the device gives
        cudaFuncAttributes fa0{}, fa1{};
        int coop = 0;
        if ((e = cudaFuncGetAttributes(&fa0, ht::fill_tiles_kernel<false>)) != cudaSuccess ||
            (e = cudaFuncGetAttributes(&fa1, ht::fill_tiles_kernel<true>)) != cudaSuccess ||
            (e = cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, cfg->device)) != cudaSuccess)
            return fail(cuda_fail(e, "cudaFuncGetAttributes(fill kernel)"));
        const size_t optin = (size_t)ctx->max_smem_optin;
        ctx->fill_smem_max[0] = optin > fa0.sharedSizeBytes ? optin - fa0.sharedSizeBytes : 0;
        ctx->fill_smem_max[1] = optin > fa1.sharedSizeBytes ? optin - fa1.sharedSizeBytes : 0;
        if ((e = cudaFuncSetAttribute(ht::fill_tiles_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      (int)ctx->fill_smem_max[0])) != cudaSuccess ||
            (e = cudaFuncSetAttribute(ht::fill_tiles_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      (int)ctx->fill_smem_max[1])) != cudaSuccess)
            return fail(cuda_fail(e, "cudaFuncSetAttribute"));
        int occ0 = 0, occ1 = 0;
        if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ0, ht::fill_tiles_kernel<false>, ht::kFillThreads,
                                                               ctx->fill_smem_max[0])) != cudaSuccess ||
            (e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ1, ht::fill_tiles_kernel<true>, ht::kFillThreads,
                                                               ctx->fill_smem_max[1])) != cudaSuccess)
            return fail(cuda_fail(e, "fill kernel occupancy"));
        ctx->fill_ok = coop && occ0 >= 1 && occ1 >= 1;
    }
    // peak scan: a persistent grid of exactly the CTAs that are resident at once (a grid-stride loop over more CTAs
    // than fit would run the excess as a second, partly empty wave)
    int unroll = env_int("HT_PEAKS_UNROLL", 2);      // config 2, B200, back-to-back launches: 45.2 us (U=2, 6 CTAs/SM), 46.4 (U=4), 49.4 (U=8)
    if (unroll != 2 && unroll != 4 && unroll != 8) unroll = 2;
    ctx->peaks_unroll = unroll;
    int occ4 = 0, occ1 = 0;
    if (unroll == 2) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ4, ht::peaks_kernel<4, 2>, ht::kPeaksThreads, 0);
    else if (unroll == 8) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ4, ht::peaks_kernel<4, 8>, ht::kPeaksThreads, 0);
    else e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ4, ht::peaks_kernel<4, 4>, ht::kPeaksThreads, 0);
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ1, ht::peaks_kernel<1, 4>, ht::kPeaksThreads, 0);
    if (e != cudaSuccess) return fail(cuda_fail(e, "cudaOccupancyMaxActiveBlocksPerMultiprocessor"));
    const int occ_cap = env_int("HT_PEAKS_CTAS_PER_SM", 32);
    if (occ4 > occ_cap) occ4 = occ_cap;
    if (occ1 > occ_cap) occ1 = occ_cap;
    if (occ4 < 1) occ4 = 1;
    if (occ1 < 1) occ1 = 1;
    ctx->peaks_grid_vec4 = ctx->sm_count * occ4;
    ctx->peaks_grid_vec1 = ctx->sm_count * occ1;
    ctx->info[6] = ctx->sm_count;
    *out = ctx;
    return HT_OK;
}

namespace {

FillPlan plan_fill(const ht_ctx *ctx, int32_t n_events, int32_t n_hits, bool peaks)
{
    FillPlan pl;
    if (!ctx->fill_ok) return pl;
    const ht_config &c = ctx->cfg;
    const size_t budget = ctx->fill_smem_max[peaks ? 1 : 0];
    const size_t row_bytes = (size_t)c.n_b * 4u;
    const long long planes = (long long)c.n_theta * c.n_phi;
    // mode 1 (per-CTA shared-memory hit index): one event, uint16 indices and plane ids, an index of at most 48 KB
    const int force = env_int("HT_FILL_MODE", -1);
    int mode = (n_events == 1 && n_hits <= 24576 && planes < 65535) ? 1 : 0;
    if (force == 0) mode = 0;
    // without the fused peak search the kernel is purely store-bound and measured fastest with slabs of <= 96 KB
    // (config 2, B200: 51.5 us at 96 KB, 53.4 at 100 KB, 59.4 at 104 KB); with it, the largest slab wins (fewer halo rows)
    const int slab_kb = env_int("HT_FILL_SLAB_KB", peaks ? 0 : 96);
    // shared memory set aside for the hits the planner stages per tile (two buffers of 16 bytes per hit): room for twice
    // the average number of hits per (event, plane), at most 512 hits; whatever else is left over is added below
    long long want_cap = 2ll * (long long)n_hits / ((long long)(n_events > 0 ? n_events : 1) * planes);
    want_cap = (want_cap + 31) / 32 * 32;
    if (want_cap > 512) want_cap = 512;
    if (want_cap < 32) want_cap = 32;
    const size_t budget_all = budget;
    auto rows_for = [&](int md) -> long long {
        const size_t budget = budget_all > (size_t)want_cap * 32u ? budget_all - (size_t)want_cap * 32u : 0;
        long long rows = c.n_a;
        if (slab_kb > 0 && rows > (long long)((size_t)slab_kb * 1024u / row_bytes)) rows = (long long)((size_t)slab_kb * 1024u / row_bytes);
        if (rows < 1) rows = 1;
        if (fill_smem_bytes(c, rows, md, n_hits) > budget) {                  // largest rows that fit (bisection)
            long long lo = 0, hi = rows;
            while (hi - lo > 1) {
                const long long mid = (lo + hi) / 2;
                if (fill_smem_bytes(c, mid, md, n_hits) <= budget) lo = mid; else hi = mid;
            }
            rows = lo;
        }
        // mode 1 sorts in the slab space: plane id + slot, 4 bytes per hit, and a copy of the angle tables
        if (md == 1 && 4u * (size_t)n_hits + 4u * (size_t)(c.n_theta + c.n_phi + 4) >
                           2u * align_up((size_t)rows * row_bytes, 16)) return 0;
        return rows;
    };
    for (;; mode = 0) {
        const long long rows = rows_for(mode);
        if (rows >= 1) {
            pl.ok = true;
            pl.mode = mode;
            pl.rows_slab = (int)rows;
            pl.slab_words = (uint32_t)(align_up((size_t)rows * row_bytes, 16) / 4u);
            pl.smem = fill_smem_bytes(c, rows, mode, n_hits);
            // what is left of the budget stages the hits of two tiles (x, r2, den, rc: 16 bytes per hit), up to 512 per tile
            long long cap = ((long long)(budget - pl.smem) / 32) / 32 * 32;
            if (cap > 512) cap = 512;
            if (env_int("HT_FILL_HIT_CAP", -1) >= 0 && cap > env_int("HT_FILL_HIT_CAP", -1)) cap = env_int("HT_FILL_HIT_CAP", -1) / 32 * 32;
            pl.hit_cap = (int)cap;
            pl.smem += (size_t)cap * 32u;
            return pl;
        }
        if (mode == 0) return pl;                                              // one row does not fit: ht_fill_naive only
    }
}

// The fill kernel (prologue a0 + tiles a1-a3), with (PEAKS: + a4-a5) or without the fused peak search.
int launch_fill(ht_ctx *ctx, const float *d_x, const float *d_y, const float *d_z, const int32_t *d_off, int32_t n_events,
                int32_t n_hits_total, uint32_t *d_mh, bool peaks, uint32_t threshold, ht_peak *d_out, uint32_t capacity,
                uint32_t *d_n_found, cudaStream_t st)
{
    const ht::Geom &g = ctx->geom;
    const FillPlan pl = plan_fill(ctx, n_events, n_hits_total, peaks);
    if (!pl.ok) return HT_ERR_UNSUPPORTED;
    ht::FillArgs a{};
    a.x = d_x; a.y = d_y; a.z = d_z; a.event_offsets = d_off; a.n_events = n_events; a.n_hits = n_hits_total;
    a.tth = ctx->d_tth; a.pph = ctx->d_pph;
    a.mode = pl.mode;
    a.hit_cap = pl.hit_cap;
    a.counts = ctx->d_counts; a.bucket_start = ctx->d_bucket_start; a.h_plane = ctx->d_hplane; a.h_rel = ctx->d_hrel;
    a.bx = ctx->d_bx; a.br2 = ctx->d_br2; a.bden = ctx->d_bden;
    a.bar = ctx->d_counters + 2;
    a.g = g;
    a.rows_slab = pl.rows_slab;
    // rows stored per tile: the whole slab, minus one halo row on each side for the peak test unless one tile covers a plane
    int rows_store = pl.rows_slab < g.n_a ? pl.rows_slab : g.n_a;
    a.halo = 0;
    if (peaks && rows_store < g.n_a) {
        rows_store = pl.rows_slab - 2;
        a.halo = 1;
    }
    if (rows_store < 1) return HT_ERR_UNSUPPORTED;
    a.rows_store = rows_store;
    a.tiles_per_plane = (g.n_a + rows_store - 1) / rows_store;
    a.slab_words = pl.slab_words;
    const unsigned long long n_tiles =
        (unsigned long long)n_events * (unsigned long long)g.planes * (unsigned long long)a.tiles_per_plane;
    if (n_tiles >= (1ull << 31)) return HT_ERR_UNSUPPORTED;        // tile indices are 32-bit in the kernel
    a.n_tiles = (uint32_t)n_tiles;
    a.mh = d_mh;
    a.bulk_ok = (g.n_b % 4 == 0) && ((reinterpret_cast<uintptr_t>(d_mh) & 15u) == 0) && env_int("HT_FILL_NO_BULK", 0) == 0;
    a.threshold = threshold;
    static_assert(sizeof(ht::PeakOut) == sizeof(ht_peak), "peak record layout");
    a.out = reinterpret_cast<ht::PeakOut *>(d_out);
    a.capacity = capacity;
    a.counters = ctx->d_counters;
    a.n_found_out = d_n_found;
    // one CTA per SM; CTA c takes tiles c, c + grid, ...
    unsigned long long grid = (unsigned long long)ctx->sm_count;
    if (grid > n_tiles) grid = n_tiles;
    if (grid < 1) grid = 1;
    // Mode 1's grid barrier: the fast one-shot form needs the host to know the counter's value, which a launch captured
    // into a CUDA graph (replayed any number of times) cannot; captured launches use the self-resetting barrier.
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    HT_CUDA(cudaStreamIsCapturing(st, &cap));
    const bool one_shot = pl.mode == 1 && cap == cudaStreamCaptureStatusNone;
    a.tile_counter = ctx->d_counters + 6;
    a.bar_count = one_shot ? ctx->d_counters + 5 : nullptr;
    a.bar_target = ctx->bar_epoch + (uint32_t)grid;
    {   // both prologues synchronise the grid: co-residency is guaranteed by a cooperative launch
        void *params[] = {&a};
        const void *fn = peaks ? reinterpret_cast<const void *>(ht::fill_tiles_kernel<true>)
                               : reinterpret_cast<const void *>(ht::fill_tiles_kernel<false>);
        HT_CUDA(cudaLaunchCooperativeKernel(fn, dim3((unsigned)grid), dim3(ht::kFillThreads), params, pl.smem, st));
    }
    if (one_shot) ctx->bar_epoch = a.bar_target;
    ++ctx->launches;
    ctx->info[0] = (int32_t)grid; ctx->info[1] = ht::kFillThreads; ctx->info[2] = (int32_t)pl.smem;
    ctx->info[3] = rows_store; ctx->info[7] = pl.mode;
    return HT_OK;
}

}  // namespace

int ht_fill(ht_ctx *ctx, const float *d_x, const float *d_y, const float *d_z, const int32_t *d_event_offsets,
            int32_t n_events, int32_t n_hits_total, uint32_t *d_mh, void *cuda_stream)
{
    const int rc = check_fill_args(ctx, d_x, d_y, d_z, d_event_offsets, n_events, n_hits_total, d_mh, true);
    if (rc != HT_OK || n_events == 0) return rc;
    return launch_fill(ctx, d_x, d_y, d_z, d_event_offsets, n_events, n_hits_total, d_mh, false, 0u, nullptr, 0u, nullptr,
                       static_cast<cudaStream_t>(cuda_stream));
}

int ht_fill_peaks(ht_ctx *ctx, const float *d_x, const float *d_y, const float *d_z, const int32_t *d_event_offsets,
                  int32_t n_events, int32_t n_hits_total, uint32_t *d_mh_or_null, uint32_t threshold, ht_peak *d_out,
                  uint32_t capacity, uint32_t *d_n_found, void *cuda_stream)
{
    if (threshold < 1u || !d_n_found || (capacity > 0 && !d_out)) return HT_ERR_INVALID_ARG;
    const int rc = check_fill_args(ctx, d_x, d_y, d_z, d_event_offsets, n_events, n_hits_total, d_mh_or_null, false);
    if (rc != HT_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (n_events == 0) {
        HT_CUDA(cudaMemsetAsync(d_n_found, 0, sizeof(uint32_t), st));
        return HT_OK;
    }
    return launch_fill(ctx, d_x, d_y, d_z, d_event_offsets, n_events, n_hits_total, d_mh_or_null, true, threshold, d_out, capacity,
                       d_n_found, st);
}

int ht_fill_naive(ht_ctx *ctx, const float *d_x, const float *d_y, const float *d_z, const int32_t *d_event_offsets,
                  int32_t n_events, int32_t n_hits_total, uint32_t *d_mh, void *cuda_stream)
{
    const int rc = check_fill_args(ctx, d_x, d_y, d_z, d_event_offsets, n_events, n_hits_total, d_mh, true);
    if (rc != HT_OK || n_events == 0) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const ht::Geom &g = ctx->geom;
    HT_CUDA(cudaMemsetAsync(d_mh, 0, (size_t)n_events * (size_t)g.cells * sizeof(uint32_t), st));
    if (n_hits_total > 0) {
        const int threads = g.n_a >= 256 ? 256 : ((g.n_a + 31) / 32) * 32;
        ht::fill_naive_kernel<<<n_hits_total, threads, 0, st>>>(d_x, d_y, d_z, d_event_offsets, n_events, ctx->d_tth,
                                                                ctx->d_pph, g, d_mh);
        HT_CUDA(cudaGetLastError());
        ++ctx->launches;
    }
    return HT_OK;
}

int ht_peaks(ht_ctx *ctx, const uint32_t *d_mh, int32_t n_events, uint32_t threshold, ht_peak *d_out,
             uint32_t capacity, uint32_t *d_n_found, void *cuda_stream)
{
    if (!ctx || n_events < 0 || n_events > ctx->cfg.max_events || threshold < 1u || !d_n_found) return HT_ERR_INVALID_ARG;
    if (capacity > 0 && !d_out) return HT_ERR_INVALID_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (n_events == 0) {
        HT_CUDA(cudaMemsetAsync(d_n_found, 0, sizeof(uint32_t), st));
        return HT_OK;
    }
    if (!d_mh) return HT_ERR_INVALID_ARG;
    const ht::Geom &g = ctx->geom;
    const unsigned long long total_cells = (unsigned long long)n_events * g.cells;
    const bool vec4 = (g.n_b % 4 == 0) && ((reinterpret_cast<uintptr_t>(d_mh) & 15u) == 0);
    const unsigned long long n_groups = vec4 ? total_cells / 4ull : total_cells;
    const int U = vec4 ? ctx->peaks_unroll : 4;
    const unsigned long long per_cta = (unsigned long long)ht::kPeaksThreads * (unsigned long long)U;
    unsigned long long grid = (n_groups + per_cta - 1ull) / per_cta;
    const unsigned long long resident = (unsigned long long)(vec4 ? ctx->peaks_grid_vec4 : ctx->peaks_grid_vec1);
    if (grid > resident) grid = resident;
    if (grid < 1ull) grid = 1ull;
    static_assert(sizeof(ht::PeakOut) == sizeof(ht_peak), "peak record layout");
    ht::PeakOut *out = reinterpret_cast<ht::PeakOut *>(d_out);
#define HT_LAUNCH_PEAKS(V, UU)                                                                                          \
    ht::peaks_kernel<V, UU><<<(unsigned)grid, ht::kPeaksThreads, 0, st>>>(d_mh, n_groups, g, threshold, out, capacity, \
                                                                          ctx->d_counters, d_n_found)
    if (!vec4) HT_LAUNCH_PEAKS(1, 4);
    else if (U == 2) HT_LAUNCH_PEAKS(4, 2);
    else if (U == 8) HT_LAUNCH_PEAKS(4, 8);
    else HT_LAUNCH_PEAKS(4, 4);
#undef HT_LAUNCH_PEAKS
    HT_CUDA(cudaGetLastError());
    ++ctx->launches;
    ctx->info[4] = (int32_t)grid; ctx->info[5] = ht::kPeaksThreads;
    return HT_OK;
}

int ht_run_host(ht_ctx *ctx, const float *h_x, const float *h_y, const float *h_z, const int32_t *h_event_offsets,
                int32_t n_events, int32_t n_hits_total, uint32_t threshold, ht_peak *h_out, uint32_t capacity,
                uint32_t *h_n_found, uint32_t *h_mh_or_null)
{
    if (!ctx || !h_n_found) return HT_ERR_INVALID_ARG;
    if (ctx->cfg.host_slots < 1) return HT_ERR_UNSUPPORTED;
    if (n_events < 0 || n_hits_total < 0 || n_events > ctx->cfg.max_events || n_hits_total > ctx->cfg.max_hits)
        return HT_ERR_INVALID_ARG;
    if (threshold < 1u || capacity > ctx->cfg.host_peak_capacity || (capacity > 0 && !h_out)) return HT_ERR_INVALID_ARG;
    *h_n_found = 0u;
    if (n_events == 0) return HT_OK;
    if (!h_event_offsets || (n_hits_total > 0 && (!h_x || !h_y || !h_z))) return HT_ERR_INVALID_ARG;
    if (h_event_offsets[0] != 0 || h_event_offsets[n_events] != n_hits_total) return HT_ERR_INVALID_ARG;
    for (int e = 0; e < n_events; ++e)
        if (h_event_offsets[e] > h_event_offsets[e + 1]) return HT_ERR_INVALID_ARG;

    cudaStream_t st = ctx->host_stream;
    const size_t cells = (size_t)ctx->geom.cells;
    // input block [offsets | x | y | z], 16-byte aligned parts, packed in pinned memory: ONE host-to-device copy
    const size_t o_x = align_up(sizeof(int32_t) * ((size_t)ctx->cfg.max_events + 1), 16);
    const size_t part = align_up(sizeof(float) * (size_t)n_hits_total, 16);
    const size_t o_y = o_x + part, o_z = o_y + part, in_bytes = o_z + part;
    // One event whose hits the grid classifies in one pass (mode 1): the kernel reads every hit exactly once, so it reads
    // them straight from the pinned block (zero-copy over PCIe) and no host-to-device copy is issued at all.
    const bool zero_copy = n_events == 1 && env_int("HT_HOST_ZERO_COPY", 1) != 0 &&
                           plan_fill(ctx, 1, n_hits_total, true).ok && plan_fill(ctx, 1, n_hits_total, true).mode == 1;
    unsigned char *in_base = zero_copy ? ctx->d_in_mapped : ctx->d_in;
    const float *d_x = reinterpret_cast<const float *>(in_base + o_x);
    const float *d_y = reinterpret_cast<const float *>(in_base + o_y);
    const float *d_z = reinterpret_cast<const float *>(in_base + o_z);
    const int32_t *d_off = reinterpret_cast<const int32_t *>(in_base);
    if (n_hits_total > 0) {
        const size_t nb = sizeof(float) * (size_t)n_hits_total;
        std::memcpy(ctx->h_in + o_x, h_x, nb);
        std::memcpy(ctx->h_in + o_y, h_y, nb);
        std::memcpy(ctx->h_in + o_z, h_z, nb);
    }
    // the kernels write the count and the list straight into mapped pinned memory: no device-to-host copy
    uint32_t *d_count = reinterpret_cast<uint32_t *>(ctx->d_res);
    ht_peak *d_list = reinterpret_cast<ht_peak *>(ctx->d_res + kResHeader);
    uint32_t found_total = 0u, written = 0u;
    const int slots = ctx->cfg.host_slots;
    int32_t *off_local = reinterpret_cast<int32_t *>(ctx->h_in);   // reused by the next group only after this group's synchronisation
    for (int e0 = 0; e0 < n_events; e0 += slots) {
        const int ne = (n_events - e0 < slots) ? n_events - e0 : slots;
        const int32_t hb = h_event_offsets[e0];
        for (int k = 0; k <= ne; ++k) off_local[k] = h_event_offsets[e0 + k] - hb;
        const int32_t nh = off_local[ne];
        if (zero_copy)
            ;
        else if (e0 == 0)
            HT_CUDA(cudaMemcpyAsync(ctx->d_in, ctx->h_in, in_bytes, cudaMemcpyHostToDevice, st));
        else
            HT_CUDA(cudaMemcpyAsync(ctx->d_in, ctx->h_in, sizeof(int32_t) * (size_t)(ne + 1), cudaMemcpyHostToDevice, st));
        const uint32_t room = capacity - written;
        // the fused kernel (matrix materialised AND peaks found in one pass); shapes it refuses take the two-call path
        int rc = ht_fill_peaks(ctx, d_x + hb, d_y + hb, d_z + hb, d_off, ne, nh, ctx->d_hmh, threshold, d_list, room, d_count, st);
        if (rc == HT_ERR_UNSUPPORTED) {
            rc = ht_fill(ctx, d_x + hb, d_y + hb, d_z + hb, d_off, ne, nh, ctx->d_hmh, st);
            if (rc == HT_ERR_UNSUPPORTED) rc = ht_fill_naive(ctx, d_x + hb, d_y + hb, d_z + hb, d_off, ne, nh, ctx->d_hmh, st);
            if (rc != HT_OK) return rc;
            rc = ht_peaks(ctx, ctx->d_hmh, ne, threshold, d_list, room, d_count, st);
        }
        if (rc != HT_OK) return rc;
        if (h_mh_or_null)
            HT_CUDA(cudaMemcpyAsync(h_mh_or_null + (size_t)e0 * cells, ctx->d_hmh, sizeof(uint32_t) * cells * (size_t)ne,
                                    cudaMemcpyDeviceToHost, st));
        HT_CUDA(cudaStreamSynchronize(st));
        const uint32_t found = *reinterpret_cast<const volatile uint32_t *>(ctx->h_res);
        const uint32_t got = found < room ? found : room;
        const ht_peak *src = reinterpret_cast<const ht_peak *>(ctx->h_res + kResHeader);
        for (uint32_t k = 0; k < got; ++k) {
            ht_peak p = src[k];
            p.event += (uint32_t)e0;
            h_out[written + k] = p;
        }
        written += got;
        found_total += found;
    }
    *h_n_found = found_total;
    return HT_OK;
}

int ht_tracks(ht_ctx *ctx, const ht_peak *d_peaks, uint32_t n_peaks, ht_track *d_out, void *cuda_stream)
{
    if (!ctx) return HT_ERR_INVALID_ARG;
    if (n_peaks == 0u) return HT_OK;
    if (!d_peaks || !d_out) return HT_ERR_INVALID_ARG;
    static_assert(sizeof(ht::TrackOut) == sizeof(ht_track), "track record layout");
    const unsigned threads = 128, blocks = (n_peaks + threads - 1u) / threads;
    ht::tracks_kernel<<<blocks, threads, 0, static_cast<cudaStream_t>(cuda_stream)>>>(
        reinterpret_cast<const ht::PeakOut *>(d_peaks), n_peaks, ctx->geom, reinterpret_cast<ht::TrackOut *>(d_out));
    HT_CUDA(cudaGetLastError());
    ++ctx->launches;
    return HT_OK;
}

int ht_selftest_division(int32_t device, uint64_t n_pairs, uint64_t seed, uint64_t *h_mismatches)
{
    if (!h_mismatches) return HT_ERR_INVALID_ARG;
    HT_CUDA(cudaSetDevice(device));
    unsigned long long *d = nullptr;
    HT_CUDA(cudaMalloc((void **)&d, sizeof(unsigned long long)));
    cudaError_t e = cudaMemset(d, 0, sizeof(unsigned long long));
    if (e == cudaSuccess) {
        ht::selftest_division_kernel<<<148 * 8, 256>>>((unsigned long long)n_pairs, (unsigned long long)seed, d);
        e = cudaGetLastError();
    }
    unsigned long long h = 0;
    if (e == cudaSuccess) e = cudaMemcpy(&h, d, sizeof h, cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (e != cudaSuccess) return cuda_fail(e, "ht_selftest_division");
    *h_mismatches = (uint64_t)h;
    return HT_OK;
}

int64_t ht_kernel_launches(const ht_ctx *ctx) { return ctx ? ctx->launches : 0; }

int ht_launch_info(const ht_ctx *ctx, int32_t out[8])
{
    if (!ctx || !out) return HT_ERR_INVALID_ARG;
    std::memcpy(out, ctx->info, sizeof ctx->info);
    return HT_OK;
}

void ht_destroy(ht_ctx *ctx)
{
    if (!ctx) return;
    cudaSetDevice(ctx->cfg.device);
    if (ctx->host_stream) { cudaStreamSynchronize(ctx->host_stream); cudaStreamDestroy(ctx->host_stream); }
    cudaFree(ctx->d_tth);
    cudaFree(ctx->d_counters);
    cudaFree(ctx->d_bx);
    cudaFree(ctx->d_bucket_start);
    cudaFree(ctx->d_counts);
    cudaFree(ctx->d_in);
    cudaFree(ctx->d_hmh);
    if (ctx->h_res) cudaFreeHost(ctx->h_res);
    if (ctx->h_in) cudaFreeHost(ctx->h_in);
    delete ctx;
}

const char *ht_strerror(int status)
{
    switch (status) {
    case HT_OK: return "ok";
    case HT_ERR_INVALID_ARG: return "invalid argument";
    case HT_ERR_UNSUPPORTED: return "binning not supported by this kernel (see include/ht.h) or call unavailable";
    case HT_ERR_CUDA: return g_cuda_err;
    case HT_ERR_NOMEM: return "out of memory";
    default: return "unknown status";
    }
}

}  // extern "C"

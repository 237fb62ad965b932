// ht_api.cu -- C ABI of libht (include/ht.h, include/ht_diag.h): argument validation, table construction (SPEC.md
// section 1), workspace layout and kernel launches.  No torch types, no exceptions across the boundary, no environment
// variables: every switch is a field of ht_tuning, read once by ht_create_ex.
#include "../../include/ht.h"
#include "../../include/ht_diag.h"
#include "ht_device.cuh"
#include "ht_diag.cuh"
#include "ht_merge.cuh"

#include <cuda.h>      // types of the one driver entry point used (cuStreamWaitValue32, fetched through cudaGetDriverEntryPoint: no link to libcuda)

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
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

// The calls leave the caller's current device as they found it.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    cudaError_t err = cudaSuccess;
    explicit DeviceGuard(int dev)
    {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != dev) {
            err = cudaSetDevice(dev);
            switched = err == cudaSuccess;
        }
    }
    ~DeviceGuard()
    {
        if (switched) cudaSetDevice(prev);
    }
};

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

bool sizes_ok(const ht_config *c)
{
    return config_ok(c) && c->max_events >= 1 && c->max_hits >= 1 && c->host_slots >= 0 && c->max_hits <= INT32_MAX - 65536;
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

constexpr size_t kBucketBytesMax = 32u << 20;   // cap of the single-event bucket region (bigger events take the batch path)
constexpr size_t kZeroBytes = 232448;           // 227 KB: no slab is larger
constexpr uint32_t kHostEagerPeaks = 4096;   // results through the copy engine: records copied to the host unasked (more: fetched by ht_wait_host)
constexpr size_t kResHeader = 16;      // result block: [uint32 n_found, pad to 16][ht_peak x host_peak_capacity]

// Layout of the context's device workspace (one contiguous block: caller-owned or allocated by ht_create) and sizes of
// the pinned host staging blocks.  Offsets are multiples of 256.
constexpr size_t kInTrailer = 16;     // last bytes of a slot's input block: the number of the submission whose hits the block holds

struct WorkspaceLayout {
    size_t tables, counters, hits, buckets, bucket_start, counts, counts1, zeros, in_dev, res_dev, mh;      // offsets
    size_t hits_part;             // bytes of one of the 6 per-hit arrays
    size_t buckets_bytes;         // single-event classification: P buckets of n_hits records each (as far as this holds them)
    size_t in_block, res_block;   // bytes of ONE slot's input block [offsets | x | y | z] and result block
    size_t total;
};

WorkspaceLayout workspace_layout(const ht_config *c)
{
    WorkspaceLayout w{};
    const size_t planes_all = (size_t)c->n_theta * (size_t)c->n_phi;
    const size_t cells = (c->plane_count > 0 ? (size_t)c->plane_count : planes_all) * (size_t)c->n_a * (size_t)c->n_b;
    size_t off = 0;
    auto take = [&](size_t bytes) { const size_t o = off; off += align_up(bytes, 256); return o; };
    w.tables = take(sizeof(float) * (size_t)(c->n_theta + 1 + c->n_phi + 1));
    w.counters = take(256);
    w.hits_part = align_up(sizeof(float) * (size_t)c->max_hits, 256);
    w.hits = take(6 * w.hits_part);            // hit records (4 words per hit), h_plane, h_rel
    w.buckets_bytes = std::min<size_t>(planes_all * align_up((size_t)c->max_hits, 4) * 16u, kBucketBytesMax);
    w.buckets = take(w.buckets_bytes);
    w.bucket_start = take(sizeof(int32_t) * (size_t)c->max_events * (planes_all + 1));
    w.counts = take(sizeof(uint32_t) * (size_t)c->max_events * planes_all);
    w.counts1 = take(sizeof(uint32_t) * planes_all * (size_t)ht::kCountStride);
    w.zeros = take(kZeroBytes);                // source of the TMA's zero fill of a slab (at most the CTA's shared memory)
    if (c->host_slots > 0) {
        w.in_block = align_up(align_up(sizeof(int32_t) * ((size_t)c->max_events + 1), 16) +
                              3 * align_up(sizeof(float) * (size_t)c->max_hits, 16) + kInTrailer, 256);
        w.res_block = align_up(kResHeader + sizeof(ht_peak) * (size_t)c->host_peak_capacity, 256);
        w.in_dev = take(w.in_block * (size_t)c->host_slots);
        w.res_dev = take(w.res_block * (size_t)c->host_slots);
        w.mh = take(cells * sizeof(uint32_t) * (size_t)c->host_slots);
    }
    w.total = off;
    return w;
}

// Tile geometry of the fill kernel for one call: the largest slab (rows of NB cells) such that two slabs, the row
// tables and -- in mode 1 -- the plane counts fit the CTA's shared memory.
struct FillPlan {
    bool ok = false;
    int mode = 0, rows_slab = 0;
    int early_cap = 0;                 // records of the early tiles' list in shared memory (0: no early tiles)
    uint32_t slab_words = 0;
    size_t smem = 0;
};

struct HostSlot {
    unsigned char *h_in = nullptr, *d_in = nullptr, *d_in_mapped = nullptr;   // pinned input block, its device mirror, its device alias
    unsigned char *h_res = nullptr, *d_res = nullptr;                          // mapped pinned result block and its device alias
    unsigned char *d_res_dev = nullptr;                                        // result block in device memory (results through the copy engine)
    bool via_copy = false;             // this submission's results: kernel -> d_res_dev -> (copy engine) -> h_res
    cudaEvent_t copied = nullptr, done = nullptr;
    bool busy = false;
    uint32_t seq = 0;                  // number of the slot's last submission (the kernel writes it into the result header)
    bool flagged = false;              // completion is signalled by the kernel through the header, not by `done`
};

}  // namespace

struct ht_ctx {
    ht_config cfg;
    ht_tuning tun;
    ht::Geom geom;
    float two_a_absmax = 0.0f;             // max |2 * A_c| over the A rows
    bool stable_inputs = false;            // ht_promise_stable_inputs
    bool tables_monotone = false;          // T non-increasing, P non-decreasing, no NaN: a bin of the bisection is an interval (early tiles)
    int sm_count = 0;
    int max_smem_optin = 0;
    // device workspace
    unsigned char *d_ws = nullptr;
    bool owns_ws = false;
    WorkspaceLayout lay{};
    float *d_tth = nullptr, *d_pph = nullptr;
    uint32_t *d_counters = nullptr;
    // hit buckets written by the fill kernel's prologue (a0): per-hit vote constants grouped by (event, plane)
    float *d_bx = nullptr;                 // mode 0: [max_hits] records
    float *d_buckets = nullptr;            // mode 1: [P][n_hits] records
    int32_t *d_hplane = nullptr, *d_hrel = nullptr;   // [max_hits] phase-1 spill
    int32_t *d_bucket_start = nullptr;     // [max_events * (P+1)]
    uint32_t *d_counts = nullptr;          // [max_events * P], zero between calls
    uint32_t *d_counts1 = nullptr;         // [P * kCountStride], zero between calls
    uint32_t *d_zeros = nullptr;           // kZeroBytes of zeros
    bool fill_ok = false;
    size_t fill_smem_max[2] = {0, 0};      // dynamic shared memory budget: [0] ht_fill, [1] fused peaks
    FillPlan plan_cache[2];
    int plan_key[2][2] = {{-1, -1}, {-1, -1}};      // (n_events, n_hits) of plan_cache[peaks]
    // peak scan launch geometry
    int peaks_unroll = 2, peaks_grid_vec4 = 0, peaks_grid_vec1 = 0;
    // stream ordering between calls of this context
    cudaStream_t last_stream = nullptr;
    bool has_last = false;
    cudaEvent_t order_event = nullptr;
    // host path (ht_run_host, ht_submit_host / ht_wait_host)
    unsigned char *h_in_all = nullptr, *h_res_all = nullptr;
    std::vector<HostSlot> slots;
    uint32_t *d_hmh = nullptr;
    cudaStream_t host_stream = nullptr, copy_stream = nullptr, d2h_stream = nullptr;
    // cuStreamWaitValue32 (nullptr: not available): lets the copy engine, not the kernel, carry a host event's results
    CUresult (*stream_wait_value32)(CUstream, CUdeviceptr, cuuint32_t, unsigned int) = nullptr;
    int64_t launches = 0;
    int32_t info[8] = {0, 0, 0, 0, 0, 0, 0, 0};
};

namespace {

size_t fill_smem_bytes(const ht_config &c, long long rows, int mode, long long early_cap)
{
    const size_t slab = align_up((size_t)rows * (size_t)c.n_b * 4u, 16);
    size_t b = 2u * slab + 8u * 4u * (size_t)((rows + 7) & ~3ll);     // two slabs, two_a[8 ring entries][rows + 4, rounded up to 4]
    if (mode == 1) b += 4u * align_up((size_t)c.n_theta * (size_t)c.n_phi, 4) + 16u * (size_t)early_cap;   // hits per plane; early list
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

// Kernels of one context share its scratch, so they must run in enqueue order.  A call that arrives on another stream
// than the previous one is ordered behind it with an event (not during graph capture: there the caller's capture
// dependencies are what they are).
int order_after_previous(ht_ctx *ctx, cudaStream_t st)
{
    if (ctx->has_last && ctx->last_stream != st) {
        cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
        HT_CUDA(cudaStreamIsCapturing(st, &cap));
        if (cap == cudaStreamCaptureStatusNone) {
            HT_CUDA(cudaEventRecord(ctx->order_event, ctx->last_stream));
            HT_CUDA(cudaStreamWaitEvent(st, ctx->order_event, 0));
        }
    }
    ctx->last_stream = st;
    ctx->has_last = true;
    return HT_OK;
}

}  // namespace

extern "C" {

int ht_query_sizes(const ht_config *cfg, size_t *mh_bytes_per_event, size_t *workspace_bytes)
{
    if (!sizes_ok(cfg)) return HT_ERR_INVALID_ARG;
    const size_t planes = cfg->plane_count > 0 ? (size_t)cfg->plane_count : (size_t)cfg->n_theta * (size_t)cfg->n_phi;
    const size_t cells = planes * (size_t)cfg->n_a * (size_t)cfg->n_b;
    if (mh_bytes_per_event) *mh_bytes_per_event = cells * sizeof(uint32_t);
    if (workspace_bytes) *workspace_bytes = workspace_layout(cfg).total;
    return HT_OK;
}

int ht_tables_host(const ht_config *cfg, float *two_a, float *t_theta, float *p_phi, float *d_ab)
{
    if (!config_ok(cfg) || !t_theta || !p_phi || !d_ab) return HT_ERR_INVALID_ARG;
    build_tables(cfg, two_a, t_theta, p_phi, d_ab);
    return HT_OK;
}

int ht_create(const ht_config *cfg, ht_ctx **out) { return ht_create_ex(cfg, nullptr, nullptr, 0, out); }

int ht_create_ex(const ht_config *cfg, const ht_tuning *tuning, void *d_workspace, size_t workspace_bytes, ht_ctx **out)
{
    if (!out) return HT_ERR_INVALID_ARG;
    if (!sizes_ok(cfg)) return HT_ERR_INVALID_ARG;
    ht_tuning tun{};
    if (tuning) {
        tun = *tuning;
        for (int32_t r : tun.reserved)
            if (r != 0) return HT_ERR_INVALID_ARG;
        if (tun.peaks_unroll != 0 && tun.peaks_unroll != 2 && tun.peaks_unroll != 4 && tun.peaks_unroll != 8) return HT_ERR_INVALID_ARG;
        if (tun.fill_slab_kb < 0 || tun.peaks_ctas_per_sm < 0 || tun.fill_store_warps < 0 || tun.fill_store_warps > 2 || tun.fill_early_cap < -1 ||
            tun.host_copy_input < 0 || tun.host_copy_input > 2) return HT_ERR_INVALID_ARG;
    }
    const WorkspaceLayout lay = workspace_layout(cfg);
    if (d_workspace && (workspace_bytes < lay.total || (reinterpret_cast<uintptr_t>(d_workspace) & 255u) != 0)) return HT_ERR_INVALID_ARG;
    int ndev = 0;
    HT_CUDA(cudaGetDeviceCount(&ndev));
    if (cfg->device < 0 || cfg->device >= ndev) return HT_ERR_INVALID_ARG;
    DeviceGuard guard(cfg->device);
    if (guard.err != cudaSuccess) return cuda_fail(guard.err, "cudaSetDevice");

    ht_ctx *ctx = new (std::nothrow) ht_ctx();
    if (!ctx) return HT_ERR_NOMEM;
    ctx->cfg = *cfg;
    ctx->tun = tun;
    ctx->lay = lay;
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
    {   // 2 * A_c is monotone in the row: the largest magnitude is at one of the ends
        std::vector<float> two_a((size_t)cfg->n_a);
        build_tables(cfg, two_a.data(), tth.data(), pph.data(), d_ab);
        ctx->two_a_absmax = std::max(std::fabs(two_a.front()), std::fabs(two_a.back()));
    }
    ctx->tables_monotone = true;
    for (size_t k = 0; k + 1 < tth.size(); ++k) ctx->tables_monotone = ctx->tables_monotone && tth[k] >= tth[k + 1];
    for (size_t k = 0; k + 1 < pph.size(); ++k) ctx->tables_monotone = ctx->tables_monotone && pph[k] <= pph[k + 1];

    cudaError_t e;
    auto fail = [&](int code) { ht_destroy(ctx); return code; };
    if ((e = cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, cfg->device)) != cudaSuccess)
        return fail(cuda_fail(e, "cudaDeviceGetAttribute(SM count)"));
    if ((e = cudaDeviceGetAttribute(&ctx->max_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, cfg->device)) != cudaSuccess)
        return fail(cuda_fail(e, "cudaDeviceGetAttribute(smem optin)"));

    if (d_workspace) {
        ctx->d_ws = static_cast<unsigned char *>(d_workspace);
    } else {
        e = cudaMalloc((void **)&ctx->d_ws, lay.total);
        if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return fail(HT_ERR_NOMEM); }
        if (e != cudaSuccess) return fail(cuda_fail(e, "cudaMalloc(workspace)"));
        ctx->owns_ws = true;
    }
    unsigned char *ws = ctx->d_ws;
    ctx->d_tth = reinterpret_cast<float *>(ws + lay.tables);
    ctx->d_pph = ctx->d_tth + (cfg->n_theta + 1);
    ctx->d_counters = reinterpret_cast<uint32_t *>(ws + lay.counters);
    ctx->d_bx = reinterpret_cast<float *>(ws + lay.hits);
    ctx->d_buckets = reinterpret_cast<float *>(ws + lay.buckets);
    ctx->d_hplane = reinterpret_cast<int32_t *>(ws + lay.hits + 4 * lay.hits_part);
    ctx->d_hrel = reinterpret_cast<int32_t *>(ws + lay.hits + 5 * lay.hits_part);
    ctx->d_bucket_start = reinterpret_cast<int32_t *>(ws + lay.bucket_start);
    ctx->d_counts = reinterpret_cast<uint32_t *>(ws + lay.counts);
    ctx->d_counts1 = reinterpret_cast<uint32_t *>(ws + lay.counts1);
    ctx->d_zeros = reinterpret_cast<uint32_t *>(ws + lay.zeros);
    if ((e = cudaMemset(ctx->d_counts, 0, align_up(sizeof(uint32_t) * (size_t)cfg->max_events * (size_t)(cfg->n_theta * cfg->n_phi), 256))) != cudaSuccess ||
        (e = cudaMemcpy(ctx->d_tth, tth.data(), tth.size() * sizeof(float), cudaMemcpyHostToDevice)) != cudaSuccess ||
        (e = cudaMemcpy(ctx->d_pph, pph.data(), pph.size() * sizeof(float), cudaMemcpyHostToDevice)) != cudaSuccess ||
        (e = cudaMemset(ctx->d_counters, 0, 256)) != cudaSuccess ||
        (e = cudaMemset(ctx->d_zeros, 0, kZeroBytes)) != cudaSuccess ||
        (e = cudaMemset(ctx->d_counts1, 0, sizeof(uint32_t) * (size_t)(cfg->n_theta * cfg->n_phi) * (size_t)ht::kCountStride)) != cudaSuccess)
        return fail(cuda_fail(e, "workspace initialisation"));
    if ((e = cudaEventCreateWithFlags(&ctx->order_event, cudaEventDisableTiming)) != cudaSuccess)
        return fail(cuda_fail(e, "cudaEventCreate"));

    if (cfg->host_slots > 0) {
        const size_t ns = (size_t)cfg->host_slots;
        ctx->d_hmh = reinterpret_cast<uint32_t *>(ws + lay.mh);
        if ((e = cudaHostAlloc((void **)&ctx->h_in_all, lay.in_block * ns, cudaHostAllocMapped)) != cudaSuccess)
            return fail(cuda_fail(e, "cudaHostAlloc(input)"));
        if ((e = cudaHostAlloc((void **)&ctx->h_res_all, lay.res_block * ns, cudaHostAllocMapped)) != cudaSuccess)
            return fail(cuda_fail(e, "cudaHostAlloc(result)"));
        std::memset(ctx->h_res_all, 0, lay.res_block * ns);          // (the completion word of a slot starts at 0, its first submission is number 1)
        std::memset(ctx->h_in_all, 0, lay.in_block * ns);
        if ((e = cudaMemset(ws + lay.in_dev, 0, lay.in_block * ns)) != cudaSuccess)      // (so does the "copied" word of its device block)
            return fail(cuda_fail(e, "cudaMemset(input blocks)"));
        unsigned char *in_map = nullptr, *res_map = nullptr;
        if ((e = cudaHostGetDevicePointer((void **)&in_map, ctx->h_in_all, 0)) != cudaSuccess ||
            (e = cudaHostGetDevicePointer((void **)&res_map, ctx->h_res_all, 0)) != cudaSuccess)
            return fail(cuda_fail(e, "cudaHostGetDevicePointer"));
        ctx->slots.resize(ns);
        for (size_t s = 0; s < ns; ++s) {
            HostSlot &sl = ctx->slots[s];
            sl.h_in = ctx->h_in_all + s * lay.in_block;
            sl.d_in_mapped = in_map + s * lay.in_block;
            sl.d_in = ws + lay.in_dev + s * lay.in_block;
            sl.d_res_dev = ws + lay.res_dev + s * lay.res_block;
            sl.h_res = ctx->h_res_all + s * lay.res_block;
            sl.d_res = res_map + s * lay.res_block;
            if ((e = cudaEventCreateWithFlags(&sl.copied, cudaEventDisableTiming)) != cudaSuccess ||
                (e = cudaEventCreateWithFlags(&sl.done, cudaEventDisableTiming)) != cudaSuccess)
                return fail(cuda_fail(e, "cudaEventCreate(slot)"));
        }
        if ((e = cudaMemset(ws + lay.res_dev, 0, lay.res_block * ns)) != cudaSuccess)
            return fail(cuda_fail(e, "cudaMemset(result blocks)"));
        if (!tun.host_direct_results) {
            void *fn = nullptr;
            cudaDriverEntryPointQueryResult qr = cudaDriverEntryPointSymbolNotFound;
            if (cudaGetDriverEntryPoint("cuStreamWaitValue32", &fn, cudaEnableDefault, &qr) == cudaSuccess &&
                qr == cudaDriverEntryPointSuccess && fn != nullptr)
                ctx->stream_wait_value32 = reinterpret_cast<CUresult (*)(CUstream, CUdeviceptr, cuuint32_t, unsigned int)>(fn);
            (void)cudaGetLastError();
        }
        if ((e = cudaStreamCreateWithFlags(&ctx->host_stream, cudaStreamNonBlocking)) != cudaSuccess ||
            (e = cudaStreamCreateWithFlags(&ctx->d2h_stream, cudaStreamNonBlocking)) != cudaSuccess ||
            (e = cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking)) != cudaSuccess)
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
        // the kernel synchronises its grid: every CTA of a launch (at most one per SM) must be resident at once
        int occ0 = 0, occ1 = 0;
        if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ0, ht::fill_tiles_kernel<false>, ht::kFillThreads,
                                                               ctx->fill_smem_max[0])) != cudaSuccess ||
            (e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ1, ht::fill_tiles_kernel<true>, ht::kFillThreads,
                                                               ctx->fill_smem_max[1])) != cudaSuccess)
            return fail(cuda_fail(e, "fill kernel occupancy"));
        ctx->fill_ok = occ0 >= 1 && occ1 >= 1 && (coop || !tun.cooperative_launch);
    }
    // peak scan: a persistent grid of exactly the CTAs that are resident at once (a grid-stride loop over more CTAs
    // than fit would run the excess as a second, partly empty wave)
    const int unroll = tun.peaks_unroll ? tun.peaks_unroll : 2;     // config 2, B200: 45.2 us (U=2, 6 CTAs/SM), 46.4 (U=4), 49.4 (U=8)
    ctx->peaks_unroll = unroll;
    int occ4 = 0, occ1 = 0;
    if (unroll == 2) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ4, ht::peaks_kernel<4, 2>, ht::kPeaksThreads, 0);
    else if (unroll == 8) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ4, ht::peaks_kernel<4, 8>, ht::kPeaksThreads, 0);
    else e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ4, ht::peaks_kernel<4, 4>, ht::kPeaksThreads, 0);
    if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ1, ht::peaks_kernel<1, 4>, ht::kPeaksThreads, 0);
    if (e != cudaSuccess) return fail(cuda_fail(e, "cudaOccupancyMaxActiveBlocksPerMultiprocessor"));
    const int occ_cap = tun.peaks_ctas_per_sm > 0 ? tun.peaks_ctas_per_sm : 32;
    occ4 = std::max(1, std::min(occ4, occ_cap));
    occ1 = std::max(1, std::min(occ1, occ_cap));
    ctx->peaks_grid_vec4 = ctx->sm_count * occ4;
    ctx->peaks_grid_vec1 = ctx->sm_count * occ1;
    ctx->info[6] = ctx->sm_count;
    *out = ctx;
    return HT_OK;
}

}  // extern "C"

namespace {

FillPlan compute_fill_plan(const ht_ctx *ctx, int32_t n_events, int32_t n_hits, bool peaks)
{
    FillPlan pl;
    if (!ctx->fill_ok) return pl;
    const ht_config &c = ctx->cfg;
    const ht_tuning &tun = ctx->tun;
    const size_t budget_all = ctx->fill_smem_max[peaks ? 1 : 0];
    const size_t row_bytes = (size_t)c.n_b * 4u;
    const long long planes = (long long)c.n_theta * c.n_phi;
    // mode 1 (one-pass classification into fixed-capacity plane buckets): one event whose P x n_hits records fit the region
    int mode = (n_events == 1 && (size_t)planes * align_up((size_t)n_hits, 4) * 16u <= ctx->lay.buckets_bytes &&
                planes * 4 < 32768 && !tun.fill_batch_classification) ? 1 : 0;
    // without the fused peak search the kernel is purely store-bound and measured fastest with slabs of <= 96 KB
    // (config 2, B200: 51.5 us at 96 KB, 53.4 at 100 KB, 59.4 at 104 KB); with it, the largest slab wins (fewer halo rows)
    const int slab_kb = tun.fill_slab_kb > 0 ? tun.fill_slab_kb : (peaks ? 0 : 96);
    // early tiles (mode 1, not too many hits): a CTA keeps the records of ONE plane's hits in shared memory -- room for
    // three times the average plane (the planes of the outer theta bins hold twice the average), at most every hit; a
    // plane with more falls back to the buckets
    auto early_cap_for = [&](int md) -> long long {
        if (md != 1 || tun.fill_early_cap < 0 || n_hits < 1 || n_hits > ht::kEarlyMaxHits || !ctx->tables_monotone) return 0;
        long long cap = tun.fill_early_cap > 0 ? tun.fill_early_cap : 3 * ((n_hits + planes - 1) / planes) + 32;
        if (cap > n_hits) cap = n_hits;
        return (long long)align_up((size_t)cap, 4);
    };
    auto rows_for = [&](int md) -> long long {
        const long long ecap = early_cap_for(md);
        const size_t budget = budget_all;
        long long rows = c.n_a;
        if (slab_kb > 0 && rows > (long long)((size_t)slab_kb * 1024u / row_bytes)) rows = (long long)((size_t)slab_kb * 1024u / row_bytes);
        if (rows < 1) rows = 1;
        if (fill_smem_bytes(c, rows, md, ecap) > budget) {                  // largest rows that fit (bisection)
            long long lo = 0, hi = rows;
            while (hi - lo > 1) {
                const long long mid = (lo + hi) / 2;
                if (fill_smem_bytes(c, mid, md, ecap) <= budget) lo = mid; else hi = mid;
            }
            rows = lo;
        }
        return rows;
    };
    for (;; mode = 0) {
        const long long rows = rows_for(mode);
        if (rows >= 1) {
            pl.ok = true;
            pl.mode = mode;
            pl.rows_slab = (int)rows;
            pl.slab_words = (uint32_t)(align_up((size_t)rows * row_bytes, 16) / 4u);
            pl.early_cap = (int)early_cap_for(mode);
            pl.smem = fill_smem_bytes(c, rows, mode, pl.early_cap);
            return pl;
        }
        if (mode == 0) return pl;                                              // one row does not fit: ht_fill_naive only
    }
}

const FillPlan &plan_fill(ht_ctx *ctx, int32_t n_events, int32_t n_hits, bool peaks)
{
    const int k = peaks ? 1 : 0;
    if (ctx->plan_key[k][0] != n_events || ctx->plan_key[k][1] != n_hits) {
        ctx->plan_cache[k] = compute_fill_plan(ctx, n_events, n_hits, peaks);
        ctx->plan_key[k][0] = n_events;
        ctx->plan_key[k][1] = n_hits;
    }
    return ctx->plan_cache[k];
}

// The fill kernel (prologue a0 + tiles a1-a3), with (PEAKS: + a4-a5) or without the fused peak search.
// early_inputs: the hit arrays are known not to be written by device work enqueued before this call (the context's own
// pinned staging blocks), so the kernel may read them before the previous kernel of the stream has completed.
enum { kInputsPlain = 0, kInputsStable = 1, kInputsHostMapped = 2 };
int launch_fill(ht_ctx *ctx, const float *d_x, const float *d_y, const float *d_z, const int32_t *d_off, int32_t n_events,
                int32_t n_hits_total, uint32_t *d_mh, bool peaks, uint32_t threshold, ht_peak *d_out, uint32_t capacity,
                uint32_t *d_n_found, cudaStream_t st, int input_kind, uint32_t *d_done_flag = nullptr, uint32_t done_value = 0u,
                const uint32_t *d_ready_flag = nullptr, bool done_flag_on_device = false)
{
    const bool early_inputs = input_kind != kInputsPlain;
    const ht::Geom &g = ctx->geom;
    const FillPlan &pl = plan_fill(ctx, n_events, n_hits_total, peaks);
    if (!pl.ok) return HT_ERR_UNSUPPORTED;
    ht::FillArgs a{};
    a.x = d_x; a.y = d_y; a.z = d_z; a.event_offsets = d_off; a.n_events = n_events; a.n_hits = n_hits_total;
    a.tth = ctx->d_tth; a.pph = ctx->d_pph;
    a.mode = pl.mode;
    a.counts = ctx->d_counts; a.counts1 = ctx->d_counts1; a.zeros = ctx->d_zeros; a.bucket_start = ctx->d_bucket_start; a.h_plane = ctx->d_hplane; a.h_rel = ctx->d_hrel;
    a.bx = pl.mode == 1 ? ctx->d_buckets : ctx->d_bx;
    a.bucket_cap = (int)align_up((size_t)n_hits_total, 4);
    // early tiles: not when the hits sit in pinned host memory (every CTA reads all of them)
    a.early_cap = input_kind == kInputsHostMapped ? 0 : pl.early_cap;
    a.two_a_absmax = ctx->two_a_absmax;
    // one queue of tile stores while the store is the slow part; a store warp per slab when the votes are (more than
    // ~150 hits per (event, plane): config 4)
    // (peaks only, no store: always one per slab -- the single queue exists for the stores' sake)
    a.store_warps = !d_mh ? 2 : ctx->tun.fill_store_warps ? ctx->tun.fill_store_warps
                    : ((long long)n_hits_total > 150ll * (long long)n_events * (long long)g.planes ? 2 : 1);
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
    a.bulk_ok = (g.n_b % 4 == 0) && ((reinterpret_cast<uintptr_t>(d_mh) & 15u) == 0) && !ctx->tun.fill_plain_stores;
    a.early_inputs = early_inputs ? 1 : 0;
    a.done_flag = d_done_flag;
    a.done_value = done_value;
    a.ready_flag = d_ready_flag;        // (its value: done_value, the number of the submission)
    a.done_flag_on_device = done_flag_on_device ? 1 : 0;
    a.threshold = threshold;
    static_assert(sizeof(ht::PeakOut) == sizeof(ht_peak), "peak record layout");
    a.out = reinterpret_cast<ht::PeakOut *>(d_out);
    a.capacity = capacity;
    a.counters = ctx->d_counters;
    a.n_found_out = d_n_found;
    // one CTA per SM; CTA c starts with tile c
    unsigned long long grid = (unsigned long long)ctx->sm_count;
    if (grid > n_tiles) grid = n_tiles;
    if (grid < 1) grid = 1;
    const int ro = order_after_previous(ctx, st);
    if (ro != HT_OK) return ro;
    // the kernel leaves every counter it uses at zero (its last CTA resets them): nothing here depends on host-side state,
    // so the launch can be captured into a CUDA graph and replayed
    a.tile_counter = ctx->d_counters + 6;
    a.bar_count = ctx->d_counters + 5;
    // the first two tiles of a CTA: neighbours (2c, 2c+1: mostly one plane, one early list) when every CTA has two
    a.pair_tiles = n_tiles >= 2ull * grid ? 1 : 0;
    // one tile per CTA and an early list that holds every hit: nothing needs the buckets
    a.skip_classify = (a.early_cap > 0 && n_tiles <= grid && n_hits_total <= a.early_cap) ? 1 : 0;
    const void *fn = peaks ? reinterpret_cast<const void *>(ht::fill_tiles_kernel<true>)
                           : reinterpret_cast<const void *>(ht::fill_tiles_kernel<false>);
    void *params[] = {&a};
    if (ctx->tun.cooperative_launch) {
        HT_CUDA(cudaLaunchCooperativeKernel(fn, dim3((unsigned)grid), dim3(ht::kFillThreads), params, pl.smem, st));
    } else {
        // Ordinary launch of a grid that ht_create has verified to be co-resident (one CTA per SM), as a programmatic
        // dependent launch: the CTAs may be placed while the previous kernel of the stream drains; the kernel waits
        // (griddepcontrol.wait) before it touches anything that kernel may have written.
        cudaLaunchConfig_t lc{};
        lc.gridDim = dim3((unsigned)grid);
        lc.blockDim = dim3(ht::kFillThreads);
        lc.dynamicSmemBytes = pl.smem;
        lc.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        lc.attrs = at;
        lc.numAttrs = 1;
        HT_CUDA(cudaLaunchKernelExC(&lc, fn, params));
    }
    ++ctx->launches;
    ctx->info[0] = (int32_t)grid; ctx->info[1] = ht::kFillThreads; ctx->info[2] = (int32_t)pl.smem;
    ctx->info[3] = rows_store; ctx->info[7] = pl.mode;
    return HT_OK;
}

}  // namespace

extern "C" {

int ht_fill(ht_ctx *ctx, const float *d_x, const float *d_y, const float *d_z, const int32_t *d_event_offsets,
            int32_t n_events, int32_t n_hits_total, uint32_t *d_mh, void *cuda_stream)
{
    const int rc = check_fill_args(ctx, d_x, d_y, d_z, d_event_offsets, n_events, n_hits_total, d_mh, true);
    if (rc != HT_OK || n_events == 0) return rc;
    DeviceGuard guard(ctx->cfg.device);
    return launch_fill(ctx, d_x, d_y, d_z, d_event_offsets, n_events, n_hits_total, d_mh, false, 0u, nullptr, 0u, nullptr,
                       static_cast<cudaStream_t>(cuda_stream), ctx->stable_inputs ? kInputsStable : kInputsPlain);
}

int ht_fill_peaks(ht_ctx *ctx, const float *d_x, const float *d_y, const float *d_z, const int32_t *d_event_offsets,
                  int32_t n_events, int32_t n_hits_total, uint32_t *d_mh_or_null, uint32_t threshold, ht_peak *d_out,
                  uint32_t capacity, uint32_t *d_n_found, void *cuda_stream)
{
    if (threshold < 1u || !d_n_found || (capacity > 0 && !d_out)) return HT_ERR_INVALID_ARG;
    const int rc = check_fill_args(ctx, d_x, d_y, d_z, d_event_offsets, n_events, n_hits_total, d_mh_or_null, false);
    if (rc != HT_OK) return rc;
    DeviceGuard guard(ctx->cfg.device);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (n_events == 0) {
        HT_CUDA(cudaMemsetAsync(d_n_found, 0, sizeof(uint32_t), st));
        return HT_OK;
    }
    return launch_fill(ctx, d_x, d_y, d_z, d_event_offsets, n_events, n_hits_total, d_mh_or_null, true, threshold, d_out, capacity,
                       d_n_found, st, ctx->stable_inputs ? kInputsStable : kInputsPlain);
}

int ht_promise_stable_inputs(ht_ctx *ctx, int32_t on)
{
    if (!ctx) return HT_ERR_INVALID_ARG;
    ctx->stable_inputs = on != 0;
    return HT_OK;
}

int ht_fill_naive(ht_ctx *ctx, const float *d_x, const float *d_y, const float *d_z, const int32_t *d_event_offsets,
                  int32_t n_events, int32_t n_hits_total, uint32_t *d_mh, void *cuda_stream)
{
    const int rc = check_fill_args(ctx, d_x, d_y, d_z, d_event_offsets, n_events, n_hits_total, d_mh, true);
    if (rc != HT_OK || n_events == 0) return rc;
    DeviceGuard guard(ctx->cfg.device);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const ht::Geom &g = ctx->geom;
    const int ro = order_after_previous(ctx, st);
    if (ro != HT_OK) return ro;
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
    DeviceGuard guard(ctx->cfg.device);
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
    const int ro = order_after_previous(ctx, st);
    if (ro != HT_OK) return ro;
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

}  // extern "C"

namespace {

// offsets of the parts of a slot's input block [offsets | x | y | z] for n_hits hits
struct InBlock {
    size_t o_x, o_y, o_z, bytes;
};
InBlock in_block(const ht_ctx *ctx, int32_t n_hits)
{
    InBlock b;
    b.o_x = align_up(sizeof(int32_t) * ((size_t)ctx->cfg.max_events + 1), 16);
    const size_t part = align_up(sizeof(float) * (size_t)n_hits, 16);
    b.o_y = b.o_x + part;
    b.o_z = b.o_y + part;
    b.bytes = b.o_z + part;
    return b;
}

// One group of events (at most host_slots, all in the input block of slot `s`, matrices from `mh_slot` on) through the
// fused kernel (or the two-call path for shapes it refuses), peak list and count into slot s's mapped result block.
int enqueue_group(ht_ctx *ctx, HostSlot &sl, const unsigned char *in_base, const InBlock &ib, int32_t hit_base, int32_t ne,
                  int32_t nh, uint32_t *d_mh, uint32_t threshold, uint32_t room, int input_kind, bool flag = false,
                  const uint32_t *d_ready_flag = nullptr, bool results_in_device_memory = false)
{
    cudaStream_t st = ctx->host_stream;
    const float *d_x = reinterpret_cast<const float *>(in_base + ib.o_x) + hit_base;
    const float *d_y = reinterpret_cast<const float *>(in_base + ib.o_y) + hit_base;
    const float *d_z = reinterpret_cast<const float *>(in_base + ib.o_z) + hit_base;
    const int32_t *d_off = reinterpret_cast<const int32_t *>(in_base);
    unsigned char *res = results_in_device_memory ? sl.d_res_dev : sl.d_res;
    uint32_t *d_count = reinterpret_cast<uint32_t *>(res);
    ht_peak *d_list = reinterpret_cast<ht_peak *>(res + kResHeader);
    // the kernel itself says when the results are in the block (second word of the header): to the host, which polls the
    // mapped block, or to the copy engine, which waits for the word in device memory and then copies the block
    sl.flagged = flag;
    sl.via_copy = flag && results_in_device_memory;
    int rc = launch_fill(ctx, d_x, d_y, d_z, d_off, ne, nh, d_mh, true, threshold, d_list, room, d_count, st,
                         input_kind, flag ? d_count + 1 : nullptr, sl.seq, d_ready_flag, results_in_device_memory);
    if (rc == HT_ERR_UNSUPPORTED) {
        sl.flagged = false;
        sl.via_copy = false;
        d_count = reinterpret_cast<uint32_t *>(sl.d_res);
        d_list = reinterpret_cast<ht_peak *>(sl.d_res + kResHeader);
        if (d_ready_flag) {             // (the other kernels do not look at the copy's word: order the streams instead)
            HT_CUDA(cudaEventRecord(sl.copied, ctx->copy_stream));
            HT_CUDA(cudaStreamWaitEvent(st, sl.copied, 0));
        }
        rc = ht_fill(ctx, d_x, d_y, d_z, d_off, ne, nh, d_mh, st);
        if (rc == HT_ERR_UNSUPPORTED) rc = ht_fill_naive(ctx, d_x, d_y, d_z, d_off, ne, nh, d_mh, st);
        if (rc != HT_OK) return rc;
        rc = ht_peaks(ctx, d_mh, ne, threshold, d_list, room, d_count, st);
    }
    return rc;
}

}  // namespace

extern "C" {

}  // extern "C"

namespace {

// ht_submit_host.  lone: the caller waits for this very event next (ht_run_host) -- nothing to overlap with, so the route
// with the fewest operations between the host's hits and the host's result is taken (the kernel reads the hits from the
// pinned block and stores its results into the pinned block), unless the tuning says otherwise.
int submit_host(ht_ctx *ctx, int32_t slot, const float *h_x, const float *h_y, const float *h_z, int32_t n_hits,
                uint32_t threshold, bool lone)
{
    if (!ctx) return HT_ERR_INVALID_ARG;
    if (ctx->cfg.host_slots < 1) return HT_ERR_UNSUPPORTED;
    if (slot < 0 || slot >= ctx->cfg.host_slots || n_hits < 0 || n_hits > ctx->cfg.max_hits || threshold < 1u) return HT_ERR_INVALID_ARG;
    if (n_hits > 0 && (!h_x || !h_y || !h_z)) return HT_ERR_INVALID_ARG;
    HostSlot &sl = ctx->slots[(size_t)slot];
    if (sl.busy) return HT_ERR_INVALID_ARG;                       // ht_wait_host first
    DeviceGuard guard(ctx->cfg.device);
    const InBlock ib = in_block(ctx, n_hits);
    int32_t *off = reinterpret_cast<int32_t *>(sl.h_in);
    off[0] = 0;
    off[1] = n_hits;
    if (n_hits > 0) {
        const size_t nb = sizeof(float) * (size_t)n_hits;
        std::memcpy(sl.h_in + ib.o_x, h_x, nb);
        std::memcpy(sl.h_in + ib.o_y, h_y, nb);
        std::memcpy(sl.h_in + ib.o_z, h_z, nb);
    }
    // One event whose hits the grid reads exactly once (mode 1): straight from the pinned block (zero-copy over PCIe);
    // otherwise one packed copy on the copy stream, which overlaps the kernel of the previous event.
    const FillPlan &pl = plan_fill(ctx, 1, n_hits, true);
    // (early tiles -- every CTA reads all the hits -- want them in device memory: copy when the plan has them)
    const bool want_copy = ctx->tun.host_copy_input == 1 || (ctx->tun.host_copy_input == 0 && pl.early_cap > 0 && !lone);
    const bool zero_copy = !want_copy && pl.ok && pl.mode == 1;
    const unsigned char *in_base = sl.d_in_mapped;
    uint32_t *d_mh = ctx->d_hmh + (size_t)slot * (size_t)ctx->geom.cells;
    ++sl.seq;
    const uint32_t *d_ready = nullptr;
    if (!zero_copy) {
        // Two copies on the copy stream: the block, then the number of this submission into the block's last word.  The
        // kernel waits for that word itself (its first instruction after it is resident), so nothing stands between two
        // kernels of the compute stream -- no event, no stream wait: consecutive events keep their dependent launch --
        // and the copy, enqueued while earlier events are still being computed, is long done when the kernel looks.
        const size_t o_seq = ctx->lay.in_block - kInTrailer;
        *reinterpret_cast<uint32_t *>(sl.h_in + o_seq) = sl.seq;
        HT_CUDA(cudaMemcpyAsync(sl.d_in, sl.h_in, ib.bytes, cudaMemcpyHostToDevice, ctx->copy_stream));
        HT_CUDA(cudaMemcpyAsync(sl.d_in + o_seq, sl.h_in + o_seq, sizeof(uint32_t), cudaMemcpyHostToDevice, ctx->copy_stream));
        in_base = sl.d_in;
        d_ready = reinterpret_cast<const uint32_t *>(sl.d_in + o_seq);
    }
    // (the slot's blocks are the library's own: final before the kernel reads them -- host-mapped, or announced by the
    // copy stream)
    const bool via_copy = ctx->stream_wait_value32 != nullptr && !lone;
    const int rc = enqueue_group(ctx, sl, in_base, ib, 0, 1, n_hits, d_mh, threshold, ctx->cfg.host_peak_capacity,
                                 zero_copy ? kInputsHostMapped : kInputsStable, true, d_ready, via_copy);
    if (rc != HT_OK) return rc;
    // (no event between two kernels of the stream when the kernel signals its own completion: an event record there
    // would undo the dependent launch of the next one)
    if (!sl.flagged) HT_CUDA(cudaEventRecord(sl.done, ctx->host_stream));
    if (sl.via_copy) {
        // Results through the copy engine: the kernel writes count, list and -- last -- the submission's number into the
        // slot's block in DEVICE memory; a third stream waits for that number (a stream memory operation: no event in the
        // compute stream) and copies the head of the list, then the header, into the pinned block the host polls.  Peak
        // records stored straight into pinned host memory keep a kernel from completing until PCIe has acknowledged them:
        // 3.3 us per call that the next kernel of the stream has to wait for.
        const uint32_t eager = std::min(ctx->cfg.host_peak_capacity, kHostEagerPeaks);
        const CUresult wr = ctx->stream_wait_value32(reinterpret_cast<CUstream>(ctx->d2h_stream),
                                                     reinterpret_cast<CUdeviceptr>(sl.d_res_dev + sizeof(uint32_t)), sl.seq,
                                                     CU_STREAM_WAIT_VALUE_EQ);
        if (wr != CUDA_SUCCESS) {
            std::snprintf(g_cuda_err, sizeof g_cuda_err, "CUDA error in cuStreamWaitValue32: CUresult %d", (int)wr);
            return HT_ERR_CUDA;
        }
        if (eager > 0)
            HT_CUDA(cudaMemcpyAsync(sl.h_res + kResHeader, sl.d_res_dev + kResHeader, sizeof(ht_peak) * (size_t)eager,
                                    cudaMemcpyDeviceToHost, ctx->d2h_stream));
        HT_CUDA(cudaMemcpyAsync(sl.h_res, sl.d_res_dev, kResHeader, cudaMemcpyDeviceToHost, ctx->d2h_stream));
    }
    sl.busy = true;
    return HT_OK;
}

}  // namespace

extern "C" {

int ht_submit_host(ht_ctx *ctx, int32_t slot, const float *h_x, const float *h_y, const float *h_z, int32_t n_hits,
                   uint32_t threshold)
{
    return submit_host(ctx, slot, h_x, h_y, h_z, n_hits, threshold, false);
}

int ht_wait_host(ht_ctx *ctx, int32_t slot, ht_peak *h_out, uint32_t capacity, uint32_t *h_n_found)
{
    if (!ctx || !h_n_found) return HT_ERR_INVALID_ARG;
    if (ctx->cfg.host_slots < 1) return HT_ERR_UNSUPPORTED;
    if (slot < 0 || slot >= ctx->cfg.host_slots || (capacity > 0 && !h_out)) return HT_ERR_INVALID_ARG;
    HostSlot &sl = ctx->slots[(size_t)slot];
    if (!sl.busy) return HT_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->cfg.device);
    if (sl.flagged) {
        const volatile uint32_t *flag = reinterpret_cast<const volatile uint32_t *>(sl.h_res) + 1;
        for (uint32_t spins = 0; *flag != sl.seq; ++spins) {
            if ((spins & 0xFFFu) == 0xFFFu) {                     // a failed kernel never writes the flag
                const cudaError_t q = cudaStreamQuery(sl.via_copy ? ctx->d2h_stream : ctx->host_stream);   // (whoever writes the word)
                if (q != cudaSuccess && q != cudaErrorNotReady) return cuda_fail(q, "ht_wait_host");
                if (q == cudaSuccess && *flag != sl.seq) return cuda_fail(cudaErrorUnknown, "ht_wait_host: stream idle, no result");
            }
        }
        std::atomic_thread_fence(std::memory_order_acquire);
    } else {
        HT_CUDA(cudaEventSynchronize(sl.done));
    }
    sl.busy = false;
    const uint32_t found = *reinterpret_cast<const volatile uint32_t *>(sl.h_res);
    uint32_t got = found < ctx->cfg.host_peak_capacity ? found : ctx->cfg.host_peak_capacity;
    if (got > capacity) got = capacity;
    if (sl.flagged && sl.via_copy && got > kHostEagerPeaks) {
        // the list is longer than what the copy engine brought along: the rest straight from the slot's device block
        // (the kernel has completed; a synchronous copy on the legacy stream, which the context's streams do not join)
        std::memcpy(h_out, sl.h_res + kResHeader, sizeof(ht_peak) * (size_t)kHostEagerPeaks);
        HT_CUDA(cudaMemcpy(h_out + kHostEagerPeaks, sl.d_res_dev + kResHeader + sizeof(ht_peak) * (size_t)kHostEagerPeaks,
                           sizeof(ht_peak) * (size_t)(got - kHostEagerPeaks), cudaMemcpyDeviceToHost));
    } else if (got > 0) {
        std::memcpy(h_out, sl.h_res + kResHeader, sizeof(ht_peak) * (size_t)got);
    }
    *h_n_found = found;
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
    for (const HostSlot &s : ctx->slots)
        if (s.busy) return HT_ERR_INVALID_ARG;                    // submitted events must be waited for first

    // one event without a matrix read-back: the asynchronous pair, back to back
    if (n_events == 1 && !h_mh_or_null) {
        int rc = submit_host(ctx, 0, h_x, h_y, h_z, n_hits_total, threshold, true);
        if (rc != HT_OK) return rc;
        return ht_wait_host(ctx, 0, h_out, capacity, h_n_found);
    }

    DeviceGuard guard(ctx->cfg.device);
    cudaStream_t st = ctx->host_stream;
    HostSlot &sl = ctx->slots[0];
    const size_t cells = (size_t)ctx->geom.cells;
    // input block [offsets | x | y | z], 16-byte aligned parts, packed in pinned memory: ONE host-to-device copy
    const InBlock ib = in_block(ctx, n_hits_total);
    const FillPlan &pl1 = plan_fill(ctx, 1, n_hits_total, true);
    const bool zero_copy = n_events == 1 && ctx->tun.host_copy_input != 1 && pl1.ok && pl1.mode == 1;
    const unsigned char *in_base = zero_copy ? sl.d_in_mapped : sl.d_in;
    if (n_hits_total > 0) {
        const size_t nb = sizeof(float) * (size_t)n_hits_total;
        std::memcpy(sl.h_in + ib.o_x, h_x, nb);
        std::memcpy(sl.h_in + ib.o_y, h_y, nb);
        std::memcpy(sl.h_in + ib.o_z, h_z, nb);
    }
    uint32_t found_total = 0u, written = 0u;
    const int slots = ctx->cfg.host_slots;
    int32_t *off_local = reinterpret_cast<int32_t *>(sl.h_in);   // reused by the next group only after this group's synchronisation
    for (int e0 = 0; e0 < n_events; e0 += slots) {
        const int ne = (n_events - e0 < slots) ? n_events - e0 : slots;
        const int32_t hb = h_event_offsets[e0];
        for (int k = 0; k <= ne; ++k) off_local[k] = h_event_offsets[e0 + k] - hb;
        const int32_t nh = off_local[ne];
        if (zero_copy)
            ;
        else if (e0 == 0)
            HT_CUDA(cudaMemcpyAsync(sl.d_in, sl.h_in, ib.bytes, cudaMemcpyHostToDevice, st));
        else
            HT_CUDA(cudaMemcpyAsync(sl.d_in, sl.h_in, sizeof(int32_t) * (size_t)(ne + 1), cudaMemcpyHostToDevice, st));
        const uint32_t room = capacity - written;
        const int rc = enqueue_group(ctx, sl, in_base, ib, hb, ne, nh, ctx->d_hmh, threshold, room, kInputsPlain);
        if (rc != HT_OK) return rc;
        if (h_mh_or_null)
            HT_CUDA(cudaMemcpyAsync(h_mh_or_null + (size_t)e0 * cells, ctx->d_hmh, sizeof(uint32_t) * cells * (size_t)ne,
                                    cudaMemcpyDeviceToHost, st));
        HT_CUDA(cudaStreamSynchronize(st));
        const uint32_t found = *reinterpret_cast<const volatile uint32_t *>(sl.h_res);
        const uint32_t got = found < room ? found : room;
        const ht_peak *src = reinterpret_cast<const ht_peak *>(sl.h_res + kResHeader);
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

int ht_run_host_events(ht_ctx *ctx, const float *h_x, const float *h_y, const float *h_z, const int32_t *h_event_offsets,
                       int32_t n_events, uint32_t threshold, ht_peak *h_out, uint32_t capacity_per_event, uint32_t *h_n_found)
{
    if (!ctx || !h_n_found || n_events < 0) return HT_ERR_INVALID_ARG;
    if (ctx->cfg.host_slots < 1) return HT_ERR_UNSUPPORTED;
    if (n_events == 0) return HT_OK;
    if (!h_event_offsets || threshold < 1u || (capacity_per_event > 0 && !h_out)) return HT_ERR_INVALID_ARG;
    if (h_event_offsets[0] != 0) return HT_ERR_INVALID_ARG;
    for (int e = 0; e < n_events; ++e) {
        const int64_t n = (int64_t)h_event_offsets[e + 1] - h_event_offsets[e];
        if (n < 0 || n > ctx->cfg.max_hits) return HT_ERR_INVALID_ARG;
    }
    if (h_event_offsets[n_events] > 0 && (!h_x || !h_y || !h_z)) return HT_ERR_INVALID_ARG;
    for (const HostSlot &s : ctx->slots)
        if (s.busy) return HT_ERR_INVALID_ARG;                    // submitted events must be waited for first
    const int slots = ctx->cfg.host_slots;
    auto collect = [&](int e) -> int {                            // event e sits in slot e % slots
        ht_peak *dst = h_out ? h_out + (size_t)e * capacity_per_event : nullptr;
        const int rc = ht_wait_host(ctx, e % slots, dst, capacity_per_event, &h_n_found[e]);
        if (rc != HT_OK) return rc;
        const uint32_t got = h_n_found[e] < capacity_per_event ? h_n_found[e] : capacity_per_event;
        const uint32_t kept = got < ctx->cfg.host_peak_capacity ? got : ctx->cfg.host_peak_capacity;
        for (uint32_t k = 0; k < kept; ++k) dst[k].event = (uint32_t)e;
        return HT_OK;
    };
    int rc = HT_OK, collected = 0;
    for (int e = 0; e < n_events && rc == HT_OK; ++e) {
        if (e - collected == slots) rc = collect(collected++);    // the slot's previous event (submitted `slots` events ago)
        if (rc != HT_OK) break;
        const int32_t lo = h_event_offsets[e], n = h_event_offsets[e + 1] - lo;
        rc = ht_submit_host(ctx, e % slots, h_x ? h_x + lo : nullptr, h_y ? h_y + lo : nullptr, h_z ? h_z + lo : nullptr, n, threshold);
        if (rc != HT_OK) {                                        // leave no event in flight
            for (; collected < e; ++collected) collect(collected);
            return rc;
        }
    }
    for (; collected < n_events; ++collected) {
        const int r2 = collect(collected);
        if (rc == HT_OK) rc = r2;
    }
    return rc;
}

int ht_tracks(ht_ctx *ctx, const ht_peak *d_peaks, uint32_t n_peaks, ht_track *d_out, void *cuda_stream)
{
    if (!ctx) return HT_ERR_INVALID_ARG;
    if (n_peaks == 0u) return HT_OK;
    if (!d_peaks || !d_out) return HT_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->cfg.device);
    static_assert(sizeof(ht::TrackOut) == sizeof(ht_track), "track record layout");
    const unsigned threads = 128, blocks = (n_peaks + threads - 1u) / threads;
    ht::tracks_kernel<<<blocks, threads, 0, static_cast<cudaStream_t>(cuda_stream)>>>(
        reinterpret_cast<const ht::PeakOut *>(d_peaks), n_peaks, ctx->geom, reinterpret_cast<ht::TrackOut *>(d_out));
    HT_CUDA(cudaGetLastError());
    ++ctx->launches;
    return HT_OK;
}

size_t ht_merge_scratch_bytes(uint32_t n_peaks) { return 3u * sizeof(uint32_t) * (size_t)(n_peaks ? n_peaks : 1u); }

int ht_merge_ridges(ht_ctx *ctx, const ht_peak *d_peaks, uint32_t n_peaks, uint32_t window, ht_candidate *d_out, uint32_t capacity,
                    uint32_t *d_n_out, void *d_scratch, size_t scratch_bytes, void *cuda_stream)
{
    if (!ctx || !d_n_out || (capacity > 0 && !d_out)) return HT_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->cfg.device);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    HT_CUDA(cudaMemsetAsync(d_n_out, 0, sizeof(uint32_t), st));
    if (n_peaks == 0u) return HT_OK;
    if (!d_peaks || !d_scratch || scratch_bytes < ht_merge_scratch_bytes(n_peaks) ||
        (reinterpret_cast<uintptr_t>(d_scratch) & 3u) != 0) return HT_ERR_INVALID_ARG;
    static_assert(sizeof(ht::CandOut) == sizeof(ht_candidate), "candidate record layout");
    const int ro = order_after_previous(ctx, st);
    if (ro != HT_OK) return ro;
    const int planes_all = ctx->cfg.n_theta * ctx->cfg.n_phi;
    const unsigned long long groups = (unsigned long long)ctx->cfg.max_events * (unsigned long long)planes_all;
    if (groups >= (1ull << 31) || ctx->cfg.n_a > 65535 || ctx->cfg.n_b > 65535) return HT_ERR_UNSUPPORTED;   // (a, b) packed in 32 bits
    uint32_t *slot = static_cast<uint32_t *>(d_scratch), *order = slot + n_peaks, *label = order + n_peaks;
    const ht::PeakOut *pk = reinterpret_cast<const ht::PeakOut *>(d_peaks);
    const unsigned threads = 256, blocks = (n_peaks + threads - 1u) / threads;
    ht::merge_count_kernel<<<blocks, threads, 0, st>>>(pk, n_peaks, ctx->geom, planes_all, (uint32_t)ctx->cfg.max_events,
                                                       ctx->d_counts, slot);
    ht::merge_scan_kernel<<<1, 1024, 0, st>>>(ctx->d_counts, ctx->d_bucket_start, (uint32_t)groups);
    ht::merge_scatter_kernel<<<blocks, threads, 0, st>>>(pk, n_peaks, ctx->geom, planes_all, ctx->d_bucket_start, slot, order);
    ht::merge_groups_kernel<<<(unsigned)groups, ht::kMergeThreads, 0, st>>>(pk, ctx->geom, ctx->d_bucket_start, order, label, window,
                                                              reinterpret_cast<ht::CandOut *>(d_out), capacity, d_n_out);
    HT_CUDA(cudaGetLastError());
    ctx->launches += 4;
    return HT_OK;
}

}  // extern "C"

namespace {

// Scratch of ht_merge_ridges_static: a file-scope device array (every GPU that loads the library holds these 768 KB until
// the process exits).  In HOST code the name g_merge_scratch is a host-side stand-in, not a device address: the address a
// kernel can use comes from cudaGetSymbolAddress, once per device, with that device current.
static __device__ __align__(256) uint32_t g_merge_scratch[3u * HT_MERGE_STATIC_MAX_PEAKS];

constexpr int kMaxDevices = 64;
std::mutex g_merge_scratch_mu;
uint32_t *g_merge_scratch_addr[kMaxDevices] = {};

// device address of g_merge_scratch on `device` (which must be current); looked up on the first call per device
int merge_scratch_of_device(int device, uint32_t **out)
{
    if (device < 0 || device >= kMaxDevices) return HT_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_merge_scratch_mu);
    if (!g_merge_scratch_addr[device]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_merge_scratch);
        if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(g_merge_scratch)");
        if (!p) return cuda_fail(cudaErrorInvalidSymbol, "cudaGetSymbolAddress(g_merge_scratch): null address");
        g_merge_scratch_addr[device] = static_cast<uint32_t *>(p);
    }
    *out = g_merge_scratch_addr[device];
    return HT_OK;
}

}  // namespace

extern "C" {

int ht_merge_ridges_static(ht_ctx *ctx, const ht_peak *d_peaks, uint32_t n_peaks, uint32_t window, ht_candidate *d_out,
                           uint32_t capacity, uint32_t *d_n_out, void *cuda_stream)
{
    if (!ctx) return HT_ERR_INVALID_ARG;
    if (n_peaks > HT_MERGE_STATIC_MAX_PEAKS) return HT_ERR_TOO_LARGE;     // (ht_strerror says what to call instead)
    uint32_t *scratch = nullptr;
    {
        DeviceGuard guard(ctx->cfg.device);
        if (guard.err != cudaSuccess) return cuda_fail(guard.err, "cudaSetDevice");
        const int rc = merge_scratch_of_device(ctx->cfg.device, &scratch);
        if (rc != HT_OK) return rc;
    }
    // the existing path, on the static array: every word of the scratch it reads it has written in the same call (slot per
    // peak, order per kept peak, label per group member), so nothing needs clearing between calls
    return ht_merge_ridges(ctx, d_peaks, n_peaks, window, d_out, capacity, d_n_out, scratch,
                           sizeof(uint32_t) * 3u * (size_t)HT_MERGE_STATIC_MAX_PEAKS, cuda_stream);
}

int ht_match_truth(ht_ctx *ctx, const ht_candidate *d_cand, uint32_t n_cand, const ht_truth *d_truth, uint32_t n_truth, double w_rho,
                   double cos_w_phi, int32_t *d_cand_match, int32_t *d_truth_match, ht_match_summary *d_summary, void *cuda_stream)
{
    if (!ctx || !d_summary || !(w_rho >= 0.0) || !(cos_w_phi >= -1.0 && cos_w_phi <= 1.0)) return HT_ERR_INVALID_ARG;
    if ((n_cand > 0 && (!d_cand || !d_cand_match)) || (n_truth > 0 && (!d_truth || !d_truth_match))) return HT_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->cfg.device);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    static_assert(sizeof(ht::TruthIn) == sizeof(ht_truth) && sizeof(ht::MatchSummary) == sizeof(ht_match_summary), "record layouts");
    HT_CUDA(cudaMemsetAsync(d_summary, 0, sizeof(ht_match_summary), st));
    const ht::CandOut *cd = reinterpret_cast<const ht::CandOut *>(d_cand);
    const ht::TruthIn *tr = reinterpret_cast<const ht::TruthIn *>(d_truth);
    ht::MatchSummary *sum = reinterpret_cast<ht::MatchSummary *>(d_summary);
    const unsigned threads = 128;
    if (n_cand > 0)
        ht::match_candidates_kernel<<<(n_cand + threads - 1u) / threads, threads, 0, st>>>(cd, n_cand, tr, n_truth, ctx->geom, w_rho,
                                                                                           cos_w_phi, d_cand_match);
    if (n_truth > 0)
        ht::match_truth_kernel<<<(n_truth + threads - 1u) / threads, threads, 0, st>>>(cd, n_cand, tr, n_truth, ctx->geom, w_rho,
                                                                                       cos_w_phi, d_cand_match, d_truth_match, sum);
    ht::match_summary_kernel<<<(std::max(n_cand, 1u) + threads - 1u) / threads, threads, 0, st>>>(d_cand_match, n_cand, n_truth, sum);
    ht::match_finish_kernel<<<1, 1, 0, st>>>(sum);
    HT_CUDA(cudaGetLastError());
    ctx->launches += 4;
    return HT_OK;
}

// ------------------------------------------------------------------------------------------------ diagnostics (ht_diag.h)

int ht_selftest_division(int32_t device, uint64_t n_pairs, uint64_t seed, uint64_t *h_mismatches)
{
    if (!h_mismatches) return HT_ERR_INVALID_ARG;
    DeviceGuard guard(device);
    if (guard.err != cudaSuccess) return cuda_fail(guard.err, "cudaSetDevice");
    int sms = 0;
    HT_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device));
    unsigned long long *d = nullptr;
    HT_CUDA(cudaMalloc((void **)&d, sizeof(unsigned long long)));
    cudaError_t e = cudaMemset(d, 0, sizeof(unsigned long long));
    if (e == cudaSuccess) {
        ht::selftest_division_kernel<<<sms * 8, 256>>>((unsigned long long)n_pairs, (unsigned long long)seed, d);
        e = cudaGetLastError();
    }
    unsigned long long h = 0;
    if (e == cudaSuccess) e = cudaMemcpy(&h, d, sizeof h, cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (e != cudaSuccess) return cuda_fail(e, "ht_selftest_division");
    *h_mismatches = (uint64_t)h;
    return HT_OK;
}

int ht_diag_memset(void *d_dst, int32_t value, size_t bytes, void *cuda_stream)
{
    if (!d_dst && bytes) return HT_ERR_INVALID_ARG;
    HT_CUDA(cudaMemsetAsync(d_dst, value, bytes, static_cast<cudaStream_t>(cuda_stream)));
    return HT_OK;
}

int ht_diag_vote_rates(int32_t device, int32_t iters, double *h_rates, uint64_t *h_sum_errors)
{
    if (!h_rates || !h_sum_errors || iters < 1) return HT_ERR_INVALID_ARG;
    DeviceGuard guard(device);
    if (guard.err != cudaSuccess) return cuda_fail(guard.err, "cudaSetDevice");
    int sms = 0;
    HT_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device));
    ht::DiagOut *d = nullptr;
    HT_CUDA(cudaMalloc((void **)&d, sizeof(ht::DiagOut) * (size_t)sms));
    std::vector<ht::DiagOut> h((size_t)sms);
    const size_t smem = (size_t)ht::kDiagWarps * ht::kDiagRowCells * 4u;
    uint64_t errors = 0;
    cudaError_t e = cudaSuccess;
    auto run = [&](auto kernel, int pattern) {
        if (e != cudaSuccess) return;
        e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        for (int rep = 0; rep < 2 && e == cudaSuccess; ++rep) {          // the first launch warms up
            kernel<<<sms, 1024, smem>>>(iters, d);
            e = cudaGetLastError();
            if (e == cudaSuccess) e = cudaMemcpy(h.data(), d, sizeof(ht::DiagOut) * (size_t)sms, cudaMemcpyDeviceToHost);
        }
        if (e != cudaSuccess) return;
        std::vector<double> r;
        for (const ht::DiagOut &o : h) {
            r.push_back(o.cycles ? (double)o.votes / (double)o.cycles : 0.0);
            errors += o.sum_errors;
        }
        std::sort(r.begin(), r.end());
        h_rates[pattern] = r[r.size() / 2];
    };
    run(ht::vote_rates_kernel<HT_DIAG_RED_RANDOM>, HT_DIAG_RED_RANDOM);
    run(ht::vote_rates_kernel<HT_DIAG_RED_RANDOM_71>, HT_DIAG_RED_RANDOM_71);
    run(ht::vote_rates_kernel<HT_DIAG_RED_NO_CONFLICT>, HT_DIAG_RED_NO_CONFLICT);
    run(ht::vote_rates_kernel<HT_DIAG_RED_TWO_WAY>, HT_DIAG_RED_TWO_WAY);
    run(ht::vote_rates_kernel<HT_DIAG_RED_SAME>, HT_DIAG_RED_SAME);
    run(ht::vote_rates_kernel<HT_DIAG_ATOM_RANDOM>, HT_DIAG_ATOM_RANDOM);
    run(ht::vote_rates_kernel<HT_DIAG_ATOM_NO_CONFLICT>, HT_DIAG_ATOM_NO_CONFLICT);
    run(ht::vote_rates_kernel<HT_DIAG_ATOM_SAME>, HT_DIAG_ATOM_SAME);
    run(ht::vote_rates_kernel<HT_DIAG_RMW_RANDOM>, HT_DIAG_RMW_RANDOM);
    run(ht::vote_rates_kernel<HT_DIAG_TAG_RANDOM>, HT_DIAG_TAG_RANDOM);
    run(ht::vote_rates_kernel<HT_DIAG_MATCH_RANDOM>, HT_DIAG_MATCH_RANDOM);
    run(ht::vote_rates_kernel<HT_DIAG_TAG_RANDOM_71>, HT_DIAG_TAG_RANDOM_71);
    cudaFree(d);
    if (e != cudaSuccess) return cuda_fail(e, "ht_diag_vote_rates");
    *h_sum_errors = errors;
    return HT_OK;
}

#ifdef HT_PROFILE_TIMELINE
// build-time instrumentation only: copy (and clear) the per-CTA phase counters of the fill kernel
__attribute__((visibility("default"))) int ht_prof_read(uint64_t *h_out, int32_t n_words, int32_t reset)
{
    if (!h_out || n_words < 0 || n_words > 256 * 32) return HT_ERR_INVALID_ARG;
    HT_CUDA(cudaDeviceSynchronize());
    HT_CUDA(cudaMemcpyFromSymbol(h_out, ht::g_prof, sizeof(uint64_t) * (size_t)n_words));
    if (reset) {
        static const unsigned long long zeros[256 * 32] = {};
        HT_CUDA(cudaMemcpyToSymbol(ht::g_prof, zeros, sizeof zeros));
    }
    return HT_OK;
}
#endif

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
    DeviceGuard guard(ctx->cfg.device);
    if (ctx->host_stream) { cudaStreamSynchronize(ctx->host_stream); cudaStreamDestroy(ctx->host_stream); }
    if (ctx->copy_stream) { cudaStreamSynchronize(ctx->copy_stream); cudaStreamDestroy(ctx->copy_stream); }
    if (ctx->d2h_stream) { cudaStreamSynchronize(ctx->d2h_stream); cudaStreamDestroy(ctx->d2h_stream); }
    for (HostSlot &s : ctx->slots) {
        if (s.copied) cudaEventDestroy(s.copied);
        if (s.done) cudaEventDestroy(s.done);
    }
    if (ctx->order_event) cudaEventDestroy(ctx->order_event);
    if (ctx->owns_ws) cudaFree(ctx->d_ws);
    if (ctx->h_res_all) cudaFreeHost(ctx->h_res_all);
    if (ctx->h_in_all) cudaFreeHost(ctx->h_in_all);
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
    case HT_ERR_TOO_LARGE:
        return "more peaks than the static scratch of ht_merge_ridges_static holds (HT_MERGE_STATIC_MAX_PEAKS = 65536): "
               "use ht_merge_ridges with caller-owned scratch";
    default: return "unknown status";
    }
}

}  // extern "C"

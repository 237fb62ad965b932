/*
 * ht.h -- C ABI of libht: Hough-Transform track finding hot path on NVIDIA B200 (sm_100a).
 *
 * Method: Rinaldi et al., "GPGPU for track finding in High Energy Physics" (arXiv:1507.03074;
 * /root/reference/PAPER.md).  Two steps (section 2):
 *   1. fill : for each hit (x,y,z), all circles x^2+y^2-2Ax-2By=0 through the hit and the origin;
 *             "for each A, the corresponding B is evaluated" and the element
 *             M_H(A,B,theta,phi) of the vote matrix is "incremented by one";
 *   2. peaks: "all the M_H elements above a given threshold would correspond to real tracks ... the
 *             second step is a local maxima search"; "each thread compares one element
 *             to its neighbours and, if the biggest, it is stored".
 * Everything the paper leaves open (angle binning, bin centre, range ends, neighbourhood, ties) is
 * fixed by /root/repo/SPEC.md (readings R1-R16); this library implements exactly that text.
 *
 * Conventions
 *   - Pointers named d_* are DEVICE pointers (on cfg.device), h_* are HOST pointers.  The caller owns every
 *     buffer it passes.  The context's device workspace (the angle tables, a few counters, the scratch of the
 *     classification: 24 bytes per hit of cfg.max_hits and 8 bytes per (event, plane) for batches, one bucket of 16-byte
 *     records per plane -- at most 32 MB -- and a 128-byte counter line per plane for single events, a 227 KB block of
 *     zeros; and, if cfg.host_slots > 0, per slot an input mirror, a result block and a vote matrix of the host calls) is either
 *     handed in by the caller
 *     (ht_query_sizes -> allocate -> ht_create_ex: the library then allocates NOTHING on the device) or allocated by
 *     ht_create itself (convenience form).  With cfg.host_slots > 0 the context also owns pinned HOST staging blocks.
 *   - Layout of a vote matrix (R15): uint32 M[event][itheta][iphi][ia][ib], ib fastest;
 *     cell = ((itheta*Nphi + iphi)*NA + ia)*NB + ib  (< 2^32 required).  d_mh must be 16-byte aligned.
 *     A context with a plane range (cfg.plane_count > 0) holds only its planes: M[event][plane - plane_begin][ia][ib].
 *   - ht_fill / ht_fill_peaks / ht_fill_naive / ht_peaks only ENQUEUE work on `cuda_stream` (a cudaStream_t passed as
 *     void*, e.g. torch.cuda.Stream().cuda_stream; NULL = the legacy default stream).  No host
 *     synchronisation, no allocation.  Results are valid once the caller has synchronised the stream.
 *     Calls on one context must be stream-ordered with respect to each other (a context is not
 *     thread-safe and keeps per-call scratch); separate contexts are independent.  When a call arrives on another
 *     stream than the previous call of the context, the library itself orders the two with an event (outside graph
 *     capture), so kernels of one context never run out of enqueue order.  The host calls (ht_run_host,
 *     ht_submit_host) enqueue on a stream owned by the context and are ordered the same way.
 *     The calls leave the caller's current device unchanged (they switch to cfg.device and back).
 *     The enqueuing calls may be captured into a CUDA graph and replayed (nothing they do depends on host-side
 *     state that a replay would miss).  The fill kernel synchronises its grid: one CTA per SM must be co-resident,
 *     which ht_create verifies with the occupancy calculator (ht_tuning.cooperative_launch = 1 makes the runtime
 *     verify it at every launch instead).
 *   - Every function returns HT_OK (0) or a negative ht_status; nothing aborts or throws.
 *     ht_strerror gives text; for HT_ERR_CUDA the text of the last CUDA error seen by this thread.
 */
#ifndef HT_H_
#define HT_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(_WIN32)
#define HT_API
#else
#define HT_API __attribute__((visibility("default")))
#endif

typedef enum ht_status {
    HT_OK = 0,
    HT_ERR_INVALID_ARG = -1, /* null pointer, non-positive bins, min >= max, non-finite range, n_events > max_events,
                                n_hits_total > max_hits, threshold == 0, cells >= 2^32 */
    HT_ERR_UNSUPPORTED = -2, /* binning does not fit the kernel (see ht_fill, ht_fill_peaks), or call unavailable */
    HT_ERR_CUDA = -3,        /* a CUDA runtime call or a launch failed */
    HT_ERR_NOMEM = -4,       /* host or device allocation failed */
    HT_ERR_TOO_LARGE = -5    /* a size beyond the fixed capacity of an entry point with static scratch (ht_merge_ridges_static) */
} ht_status;

typedef struct ht_ctx ht_ctx; /* opaque; created by ht_create, freed by ht_destroy */

/* Binning of the Hough space and capacities.  Ranges are half-open [min,max); angles in radians, lengths in mm.
 * "binned in 4 x 16 x 1024 x 1024 along the corresponding A, B, theta, phi" (reading R1:
 * n_theta=4, n_phi=16, n_a=n_b=1024). */
typedef struct ht_config {
    int32_t n_theta, n_phi, n_a, n_b;  /* bins, all >= 1 */
    float a_min, a_max, b_min, b_max;  /* finite, min < max */
    float theta_min, theta_max;        /* 0 <= min < max <= pi   (max >= (float)pi means exactly pi)   */
    float phi_min, phi_max;            /* 0 <= min < max <= 2pi  (max >= (float)(2pi) means exactly 2pi) */
    int32_t max_events;                /* largest n_events of one ht_fill / ht_peaks call, >= 1 */
    int32_t max_hits;                  /* largest n_hits_total of one ht_fill call, >= 1 */
    int32_t device;                    /* CUDA ordinal */
    int32_t host_slots;                /* >= 0: slots (input block, result block, vote matrix) of the host calls ht_run_host /
                                          ht_submit_host; 0: those calls are unavailable */
    uint32_t host_peak_capacity;       /* peak-list capacity of the context's staging buffer for ht_run_host */
    /* Plane range of this context (f2; the sector split of PAPER.md:77 "four M_H(A,B,theta), each matrix processing the
     * data of a single phi sector"): the context fills and scans only the (theta,phi) planes
     * [plane_begin, plane_begin + plane_count) of the n_theta * n_phi (plane = itheta * n_phi + iphi); hits of other
     * planes are ignored; its matrices hold plane_count planes per event; peak records carry the cell index of the
     * FULL matrix.  plane_count == 0: all planes. */
    int32_t plane_begin, plane_count;
} ht_config;

typedef struct ht_peak {
    uint32_t event; /* index of the event inside the call's batch */
    uint32_t cell;  /* linear cell index inside that event's matrix */
    uint32_t count; /* M_H value of the cell */
} ht_peak;

/* How the work is organised on the device.  Nothing here ever changes a result (the parity tests run every
 * variant); all zero = the defaults.  Read ONCE by ht_create_ex; the library reads no environment variable. */
typedef struct ht_tuning {
    int32_t fill_batch_classification; /* 1: classify through global buckets (the batch path) also for single events */
    int32_t fill_slab_kb;              /* > 0: cap of one shared-memory slab in KB (0: as large as fits) */
    int32_t fill_plain_stores;         /* 1: tiles leave with plain stores instead of bulk (TMA) stores */
    int32_t cooperative_launch;        /* 1: cudaLaunchCooperativeKernel (0: ordinary launch, programmatic dependent
                                          launch: the next call's prologue overlaps this call's tail) */
    int32_t host_copy_input;           /* how the hits of a single host event (ht_submit_host) reach the kernel.  1: one
                                          asynchronous copy into device memory on a second stream, which also writes the
                                          submission's number behind the hits; the kernel waits for that word itself, so no
                                          event stands between two kernels of the compute stream and consecutive events keep
                                          their dependent launch.  2: the kernel reads them straight from the pinned block
                                          (zero-copy over PCIe, coalesced).  0: 1 when the call uses early tiles (which read
                                          every hit in every thread block), else 2.  (47.2 / 48.2 us per pipelined event of
                                          5000 hits, 71.3 / 69.9 us at 20000) */
    int32_t peaks_unroll;              /* 2, 4 or 8 independent 16-byte loads per thread of the peak scan (0: 2) */
    int32_t peaks_ctas_per_sm;         /* > 0: cap of the peak scan's resident CTAs per SM */
    int32_t fill_store_warps;          /* 1: one store warp queues every tile store; 2: one store warp per slab (0: chosen
                                          from the hits per plane of the call) */
    int32_t fill_early_cap;            /* single events of <= 32768 hits: every CTA finds the hits of its first tile's plane
                                          itself and votes while the grid still classifies ("early tiles").  > 0: records of
                                          that list in shared memory; 0: three times the average plane + 32; -1: no early tiles */
    int32_t host_direct_results;       /* single host events: 1: the kernel stores count and peak list straight into the pinned
                                          result block (a kernel that does cannot complete before PCIe has acknowledged the
                                          stores: +3.3 us per call); 0: into device memory, from where a copy stream that waits
                                          for the kernel's completion word (cuStreamWaitValue32) brings them to the host -- or
                                          as 1 where the driver has no such operation */
    int32_t reserved[6];               /* must be zero */
} ht_tuning;

/* Sizes implied by a configuration: bytes of one event's matrix, and bytes of the context's device workspace
 * (what ht_create allocates, or what the caller hands to ht_create_ex). */
HT_API int ht_query_sizes(const ht_config *cfg, size_t *mh_bytes_per_event, size_t *workspace_bytes);

/* Validate cfg, build and upload the tables (SPEC.md section 1), allocate the workspace on cfg.device.
 * *out is set only on HT_OK.  Same as ht_create_ex(cfg, NULL, NULL, 0, out).  (Defines no step of the method.) */
HT_API int ht_create(const ht_config *cfg, ht_ctx **out);

/* ht_create with tuning switches (NULL: defaults) and a CALLER-OWNED device workspace: d_workspace (256-byte aligned,
 * on cfg.device) of at least ht_query_sizes()'s workspace_bytes, which must outlive the context and is not freed by
 * ht_destroy; the library then allocates no device memory at all.  d_workspace == NULL: the library allocates (and
 * ht_destroy frees) the workspace.  HT_ERR_INVALID_ARG if the workspace is too small or misaligned. */
HT_API int ht_create_ex(const ht_config *cfg, const ht_tuning *tuning_or_null, void *d_workspace_or_null,
                        size_t workspace_bytes, ht_ctx **out);

/*
 * Fill the vote matrices of a batch of events (SPEC.md section 2).
 *   d_x, d_y, d_z     device, float32 SoA, n_hits_total entries (mm); hits of event e are
 *                     [d_event_offsets[e], d_event_offsets[e+1])
 *   d_event_offsets   device, int32, n_events+1 entries, ascending, first 0, last n_hits_total
 *   n_events, n_hits_total  host copies of the sizes (validation, grid sizing); n_events may be 0 (no-op)
 *   d_mh              device, n_events * cells uint32, FULLY OVERWRITTEN: every cell is stored exactly once
 *                     (zero or its count); it need not be cleared beforehand.  4-byte aligned; 16-byte alignment
 *                     (and n_b % 4 == 0) lets the rows leave as bulk (TMA) stores, otherwise plain stores are used.
 * One persistent kernel (one co-resident CTA per SM): the grid classifies every hit once into its (event, theta, phi)
 * plane, then builds tiles of A rows as private shared-memory histograms (29 warps vote on equal shares of the tile's
 * hits x rows) and stores each tile once with a bulk (TMA) copy: no global atomics on the matrix, no memset pass.
 * HT_ERR_UNSUPPORTED if one A row (n_b*4 bytes) does not fit a shared-memory slab (two slabs share ~220 KB:
 * n_b > ~27000), if the device cannot launch cooperatively, or if a batch has 2^31 tiles or more: ht_fill_naive.
 */
HT_API int ht_fill(ht_ctx *ctx, const float *d_x, const float *d_y, const float *d_z,
                   const int32_t *d_event_offsets, int32_t n_events, int32_t n_hits_total, uint32_t *d_mh,
                   void *cuda_stream);

/*
 * Fill AND peak search in one pass: the same kernel as ht_fill applies the threshold +
 * local-maximum rule of ht_peaks to each tile while it is still in shared memory, so the matrix is never read back.
 * The two-kernel split is the paper's ("splitting the code in two kernels"), not a requirement of the
 * method; results are identical to ht_fill followed by ht_peaks.
 *   d_mh_or_null      as d_mh of ht_fill, or NULL: the matrices are not materialised at all (peaks only)
 *   threshold, d_out, capacity, d_n_found   as for ht_peaks
 * HT_ERR_UNSUPPORTED where ht_fill is, and if fewer than 3 A rows fit a slab (one stored row plus the two
 * neighbouring rows; n_b > ~9000): use ht_fill + ht_peaks.
 */
HT_API int ht_fill_peaks(ht_ctx *ctx, const float *d_x, const float *d_y, const float *d_z,
                         const int32_t *d_event_offsets, int32_t n_events, int32_t n_hits_total,
                         uint32_t *d_mh_or_null, uint32_t threshold, ht_peak *d_out, uint32_t capacity,
                         uint32_t *d_n_found, void *cuda_stream);

/* A promise about the INPUTS of this context's following ht_fill / ht_fill_peaks calls (on != 0; revoked with 0; off by
 * default).  The caller states that, for each such call, every write to d_x, d_y, d_z and d_event_offsets had COMPLETED
 * before the call was made (a batch of events staged in device memory and synchronized once, then one call per event:
 * the paper's use), or had been enqueued on the call's stream before the previous call of this
 * context; and that nothing enqueued later writes them before the call has run.  The kernel then reads the hits as soon
 * as its thread blocks are resident -- while the previous kernel of the stream is still draining (dependent launch) --
 * instead of after that kernel has completed; it still writes nothing before.  Results are the same; a single-event
 * call in a stream of calls saves the ~3 us its first tile's hits take to find.  With the promise broken the kernel may
 * read hits that are not yet written.  (Defines no step of the method.) */
HT_API int ht_promise_stable_inputs(ht_ctx *ctx, int32_t on);

/* The paper's own design (cudaMemset, one block per hit, threads over A, global atomicAdd),
 * same arguments and result as ht_fill, any binning.  Kept as the prior-art comparison and for shapes ht_fill
 * refuses. */
HT_API int ht_fill_naive(ht_ctx *ctx, const float *d_x, const float *d_y, const float *d_z,
                         const int32_t *d_event_offsets, int32_t n_events, int32_t n_hits_total, uint32_t *d_mh,
                         void *cuda_stream);

/*
 * Thresholded local-maxima search with compaction (SPEC.md section 3).
 *   d_mh        device, n_events * cells uint32 (as written by ht_fill)
 *   threshold   >= 1 (count >= threshold is "above threshold", R11)
 *   d_out       device, room for `capacity` records; order unspecified (compare after sorting by (event, cell))
 *   d_n_found   device, one uint32: the number of peaks found, which may exceed capacity (then only
 *               `capacity` records were written; not an error)
 */
HT_API int ht_peaks(ht_ctx *ctx, const uint32_t *d_mh, int32_t n_events, uint32_t threshold, ht_peak *d_out,
                    uint32_t capacity, uint32_t *d_n_found, void *cuda_stream);

/* A peak with the parameters of its track (f3). */
typedef struct ht_track {
    uint32_t event, cell, count; /* the peak record */
    float rho;                   /* mm: radius of the track's circle = distance of the cell centre (A, B) from the origin */
    float phi;                   /* rad, (-pi, pi]: azimuth of the circle's centre */
} ht_track;

/*
 * Track read-out of a peak list ("rho = sqrt(A^2 + B^2) and phi = tan^-1(B/A)"; SPEC.md section 4):
 * (A, B) = centre of the peak's cell = centre of the circle through the origin; phi is quadrant-aware (R17).
 *   d_peaks   device, n_peaks records as written by ht_peaks / ht_fill_peaks (any order)
 *   n_peaks   host value: min(count found, capacity of the list)
 *   d_out     device, n_peaks ht_track records, same order as d_peaks
 * Enqueues one small kernel on cuda_stream (binary32 arithmetic: rho within 2 ulp, phi within 4e-7 rad of the exact values).
 */
HT_API int ht_tracks(ht_ctx *ctx, const ht_peak *d_peaks, uint32_t n_peaks, ht_track *d_out, void *cuda_stream);

/* A track candidate: a connected group of peaks of one ridge (f3; SPEC.md section 5, reading R19). */
typedef struct ht_candidate {
    uint32_t event, cell, count; /* the representative peak: largest count of the group, smallest cell among equals */
    uint32_t n_peaks;            /* peaks merged into this candidate */
    float rho, phi;              /* read-out of the representative's cell, as ht_track */
} ht_candidate;

/*
 * Ridge merging of a peak list into track candidates (PAPER.md:25 goes from "local maxima" straight to "real tracks";
 * SURVEY.md section 8(f) f3 "merging ridge peaks"; SPEC.md section 5): peaks of the same event and (theta,phi) plane whose
 * (a, b) cells are at Chebyshev distance <= window are linked; a candidate is a connected component of the link graph.
 *   d_peaks    device, n_peaks records (any order); records with event >= cfg.max_events are ignored
 *   d_out      device, room for `capacity` candidates, order unspecified (compare sorted by (event, cell))
 *   d_n_out    device, one uint32: the number of candidates (may exceed capacity; then only `capacity` were written)
 *   d_scratch  device, at least ht_merge_scratch_bytes(n_peaks) bytes, 4-byte aligned, caller-owned
 * Enqueues a few small kernels on cuda_stream (they use the context's (event, plane) counters: stream-ordered with the
 * other calls of the context like every enqueuing call).
 */
HT_API size_t ht_merge_scratch_bytes(uint32_t n_peaks);
HT_API int ht_merge_ridges(ht_ctx *ctx, const ht_peak *d_peaks, uint32_t n_peaks, uint32_t window, ht_candidate *d_out,
                           uint32_t capacity, uint32_t *d_n_out, void *d_scratch, size_t scratch_bytes, void *cuda_stream);

/*
 * ht_merge_ridges for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): same arguments, same result, but the scratch is a file-scope device array of the
 * library -- 3 * 4 * HT_MERGE_STATIC_MAX_PEAKS bytes = 768 KB, held by every GPU that loads the library until the process
 * exits.  The call allocates nothing, on the device or through any library routine; the array's device address is looked
 * up (cudaGetSymbolAddress) on the first call per device, so make that first call outside a graph capture.
 *   n_peaks > HT_MERGE_STATIC_MAX_PEAKS: HT_ERR_TOO_LARGE, nothing is enqueued (use ht_merge_ridges).
 * ALL calls on a device, from every context and thread, share the one array: two calls that overlap on the GPU (different
 * streams without an ordering between them) race and give wrong candidates; calls of one stream, or stream-ordered like
 * the other calls of a context, are safe.  The array keeps the last call's contents; nothing in it needs to start at zero
 * (every word a call reads it has written itself), so no clearing happens between calls.
 */
#define HT_MERGE_STATIC_MAX_PEAKS 65536u
HT_API int ht_merge_ridges_static(ht_ctx *ctx, const ht_peak *d_peaks, uint32_t n_peaks, uint32_t window, ht_candidate *d_out,
                                  uint32_t capacity, uint32_t *d_n_out, void *cuda_stream);

/* A generated track for ht_match_truth: the centre (a, b) [mm] of its circle through the origin, R (q sin phi0, -q cos phi0). */
typedef struct ht_truth {
    uint32_t event, pad;
    double a, b;
} ht_truth;

typedef struct ht_match_summary {
    int64_t n_cand, n_truth, n_matched, n_fake, n_found, n_duplicate;
    double sum_drho, sum_drho2, sum_dphi, sum_dphi2; /* residuals rho_c - rho_t [mm] and phi_c - phi_t [rad] of the found tracks */
} ht_match_summary;

/*
 * Truth matching of track candidates (stand-in for PAPER.md:29-33, Fig. 1: the tracks' rho, phi "together with the
 * corresponding resolutions"; SURVEY.md section 8(f) f3 "truth-matched efficiency / fake rate / resolution"; SPEC.md
 * section 6, reading R20).  Candidate c and truth t are compatible when they belong to the same event,
 * |rho_c - rho_t| <= w_rho and the angle between their centres is <= w_phi (cos_w_phi = cos(w_phi), taken by the caller).
 *   d_cand_match   device, n_cand int32: the closest compatible truth record, or -1 (the candidate is a fake)
 *   d_truth_match  device, n_truth int32: the closest candidate matched to it, or -1 (not found)
 *   d_summary      device, one ht_match_summary (efficiency = n_found / n_truth, fake rate = n_fake / n_cand)
 * All decisions in binary64; O(n_cand * n_truth) work, meant for evaluation, not for the hot path.
 */
HT_API int ht_match_truth(ht_ctx *ctx, const ht_candidate *d_cand, uint32_t n_cand, const ht_truth *d_truth, uint32_t n_truth,
                          double w_rho, double cos_w_phi, int32_t *d_cand_match, int32_t *d_truth_match,
                          ht_match_summary *d_summary, void *cuda_stream);

/*
 * End-to-end call with HOST buffers (f4; needs cfg.host_slots >= 1; the transfer is "the dominant part" of
 * the paper's total time -- here only the hits (12 bytes each) and the compacted peak list cross PCIe).
 * Packs offsets and hits into one pinned block, which the kernel reads directly (one event: every hit is read exactly
 * once, zero-copy over PCIe) or which is copied to the device in one transfer (batches, ht_tuning.host_copy_input),
 * runs ht_fill_peaks (or ht_fill + ht_peaks where that is unsupported) on the context's own matrices (events in groups
 * of host_slots) with the peak list and count written by the kernel straight into mapped pinned memory (the route with
 * the fewest operations between the host's hits and the host's result: nothing else is in flight to overlap with), and
 * synchronises.  h_out receives min(*h_n_found, capacity) records; capacity <= cfg.host_peak_capacity.
 * h_mh_or_null: if not NULL, n_events * cells uint32 that also receive the matrices (testing; slow).
 * Host buffers may be pageable or pinned.  No event may be in flight in a slot (ht_submit_host without ht_wait_host).
 */
HT_API int ht_run_host(ht_ctx *ctx, const float *h_x, const float *h_y, const float *h_z,
                       const int32_t *h_event_offsets, int32_t n_events, int32_t n_hits_total, uint32_t threshold,
                       ht_peak *h_out, uint32_t capacity, uint32_t *h_n_found, uint32_t *h_mh_or_null);

/*
 * The same end-to-end path, asynchronous, one event per call, so that packing event k+1 and reading the peaks of event
 * k-1 overlap the kernel of event k:
 *   ht_submit_host  copies the n_hits hits of ONE event from h_x, h_y, h_z into the pinned input block of `slot`
 *                   (0 <= slot < cfg.host_slots; the caller's arrays may be reused as soon as the call returns),
 *                   enqueues the fused kernel (a0-a5; the event's matrix is materialised in the slot's own matrix) on the
 *                   context's stream and returns without waiting.  HT_ERR_INVALID_ARG if the slot still holds an event
 *                   that has not been waited for.  Events run in submission order.  Between two events' kernels there is
 *                   nothing in that stream (consecutive kernels keep their dependent launch): the hits reach the device
 *                   through a copy stream whose last write is a word the kernel waits for (or are read by the kernel from
 *                   the pinned block: ht_tuning.host_copy_input), count and peak list come back through a copy stream
 *                   that waits for the kernel's completion word (ht_tuning.host_direct_results).
 *   ht_wait_host    blocks until the event submitted into `slot` has finished; h_out receives
 *                   min(*h_n_found, capacity, cfg.host_peak_capacity) records, *h_n_found the number of peaks found.
 *                   HT_ERR_INVALID_ARG if nothing was submitted into the slot.
 * ht_run_host on one event is ht_submit_host + ht_wait_host on slot 0 (on the lone-event route described there).
 */
HT_API int ht_submit_host(ht_ctx *ctx, int32_t slot, const float *h_x, const float *h_y, const float *h_z, int32_t n_hits,
                          uint32_t threshold);
HT_API int ht_wait_host(ht_ctx *ctx, int32_t slot, ht_peak *h_out, uint32_t capacity, uint32_t *h_n_found);

/*
 * A SEQUENCE of independent events from host memory, each through its own fused kernel (a0-a5), pipelined over the
 * context's slots by the library itself (ht_submit_host / ht_wait_host in a loop: event k+1 is packed and launched and
 * event k-1's peaks are copied out while event k's kernel runs):
 *   h_x, h_y, h_z, h_event_offsets  as for ht_run_host (n_events + 1 offsets; each event at most cfg.max_hits hits)
 *   h_out       n_events * capacity_per_event records: event e's list starts at h_out + e * capacity_per_event and holds
 *               min(h_n_found[e], capacity_per_event, cfg.host_peak_capacity) records with `event` = e
 *   h_n_found   n_events counts
 * Synchronous: returns when every event has been collected.  No event may be in flight in a slot.
 */
HT_API int ht_run_host_events(ht_ctx *ctx, const float *h_x, const float *h_y, const float *h_z,
                              const int32_t *h_event_offsets, int32_t n_events, uint32_t threshold, ht_peak *h_out,
                              uint32_t capacity_per_event, uint32_t *h_n_found);

/* Free everything the context owns (not a caller-owned workspace).  NULL is allowed.  (Defines no step of the method.) */
HT_API void ht_destroy(ht_ctx *ctx);

HT_API const char *ht_strerror(int status);

#ifdef __cplusplus
}
#endif
#endif /* HT_H_ */

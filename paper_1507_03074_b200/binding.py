"""Thin ctypes binding of libht.so -- the same names as include/ht.h, argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind these calls; nothing here computes.  There is no CPU
fallback: if the library is missing or does not load, importing a function from here raises.  PyTorch appears only
as the owner of device memory and streams (``tensor.data_ptr()``, ``torch.cuda.Stream().cuda_stream``).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libht.so")

HT_OK, HT_ERR_INVALID_ARG, HT_ERR_UNSUPPORTED, HT_ERR_CUDA, HT_ERR_NOMEM, HT_ERR_TOO_LARGE = 0, -1, -2, -3, -4, -5
HT_MERGE_STATIC_MAX_PEAKS = 65536

PEAK_DTYPE = np.dtype([("event", np.uint32), ("cell", np.uint32), ("count", np.uint32)])   # == struct ht_peak

TRACK_DTYPE = np.dtype([("event", np.uint32), ("cell", np.uint32), ("count", np.uint32),
                        ("rho", np.float32), ("phi", np.float32)])                                # == struct ht_track

CAND_DTYPE = np.dtype([("event", np.uint32), ("cell", np.uint32), ("count", np.uint32), ("n_peaks", np.uint32),
                       ("rho", np.float32), ("phi", np.float32)])                                 # == struct ht_candidate
TRUTH_DTYPE = np.dtype([("event", np.uint32), ("pad", np.uint32), ("a", np.float64), ("b", np.float64)])   # == struct ht_truth
SUMMARY_DTYPE = np.dtype([("n_cand", np.int64), ("n_truth", np.int64), ("n_matched", np.int64), ("n_fake", np.int64),
                          ("n_found", np.int64), ("n_duplicate", np.int64), ("sum_drho", np.float64),
                          ("sum_drho2", np.float64), ("sum_dphi", np.float64), ("sum_dphi2", np.float64)])   # == ht_match_summary

EXPORTS = ("ht_query_sizes", "ht_create", "ht_create_ex", "ht_fill", "ht_fill_peaks", "ht_promise_stable_inputs", "ht_fill_naive", "ht_peaks", "ht_tracks",
           "ht_merge_scratch_bytes", "ht_merge_ridges", "ht_merge_ridges_static", "ht_match_truth",
           "ht_run_host", "ht_run_host_events", "ht_submit_host", "ht_wait_host", "ht_destroy", "ht_strerror")                  # include/ht.h
DIAG_EXPORTS = ("ht_tables_host", "ht_kernel_launches", "ht_launch_info", "ht_selftest_division", "ht_diag_memset",
                "ht_diag_vote_rates")                                                                     # include/ht_diag.h
DIAG_PATTERNS = ("red_random", "red_random_71", "red_no_conflict", "red_two_way", "red_same", "atom_random",
                 "atom_no_conflict", "atom_same", "rmw_random_inexact", "tag_random", "match_random", "tag_random_71")


class ht_config(C.Structure):
    _fields_ = [("n_theta", C.c_int32), ("n_phi", C.c_int32), ("n_a", C.c_int32), ("n_b", C.c_int32),
                ("a_min", C.c_float), ("a_max", C.c_float), ("b_min", C.c_float), ("b_max", C.c_float),
                ("theta_min", C.c_float), ("theta_max", C.c_float), ("phi_min", C.c_float), ("phi_max", C.c_float),
                ("max_events", C.c_int32), ("max_hits", C.c_int32), ("device", C.c_int32),
                ("host_slots", C.c_int32), ("host_peak_capacity", C.c_uint32),
                ("plane_begin", C.c_int32), ("plane_count", C.c_int32)]

    @classmethod
    def from_binning(cls, b, *, max_events: int, max_hits: int, device: int = 0, host_slots: int = 0,
                     host_peak_capacity: int = 0, plane_begin: int = 0, plane_count: int = 0) -> "ht_config":
        return cls(b.n_theta, b.n_phi, b.n_a, b.n_b, b.a_min, b.a_max, b.b_min, b.b_max, b.theta_min, b.theta_max,
                   b.phi_min, b.phi_max, max_events, max_hits, device, host_slots, host_peak_capacity, plane_begin,
                   plane_count)

    @property
    def cells(self) -> int:
        """Cells of one event's matrix IN THIS CONTEXT (its plane range only)."""
        planes = self.plane_count if self.plane_count > 0 else self.n_theta * self.n_phi
        return planes * self.n_a * self.n_b


class ht_tuning(C.Structure):
    """How the work is organised on the device (include/ht.h); never changes a result.  All zero = defaults."""
    _fields_ = [("fill_batch_classification", C.c_int32), ("fill_slab_kb", C.c_int32),
                ("fill_plain_stores", C.c_int32), ("cooperative_launch", C.c_int32),
                ("host_copy_input", C.c_int32), ("peaks_unroll", C.c_int32), ("peaks_ctas_per_sm", C.c_int32),
                ("fill_store_warps", C.c_int32), ("fill_early_cap", C.c_int32), ("host_direct_results", C.c_int32),
                ("reserved", C.c_int32 * 6)]


class HtError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {ht_strerror(status)} (status {status})")


_lib = None


def load() -> C.CDLL:
    """Load libht.so (built in-tree by paper_1507_03074_b200/build.py).  Fails loudly: there is no fallback."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1507_03074_b200.build` "
                          "(or __graft_entry__.build()); there is no CPU fallback")
    lib = C.CDLL(LIB_PATH)
    vp, i32, u32 = C.c_void_p, C.c_int32, C.c_uint32
    cfgp = C.POINTER(ht_config)
    lib.ht_query_sizes.restype = C.c_int
    lib.ht_query_sizes.argtypes = [cfgp, C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)]
    lib.ht_tables_host.restype = C.c_int
    lib.ht_tables_host.argtypes = [cfgp, vp, vp, vp, vp]
    lib.ht_create.restype = C.c_int
    lib.ht_create.argtypes = [cfgp, C.POINTER(vp)]
    lib.ht_create_ex.restype = C.c_int
    lib.ht_create_ex.argtypes = [cfgp, C.POINTER(ht_tuning), vp, C.c_size_t, C.POINTER(vp)]
    lib.ht_submit_host.restype = C.c_int
    lib.ht_submit_host.argtypes = [vp, i32, vp, vp, vp, i32, u32]
    lib.ht_wait_host.restype = C.c_int
    lib.ht_wait_host.argtypes = [vp, i32, vp, u32, vp]
    lib.ht_diag_memset.restype = C.c_int
    lib.ht_diag_memset.argtypes = [vp, i32, C.c_size_t, vp]
    lib.ht_diag_vote_rates.restype = C.c_int
    lib.ht_diag_vote_rates.argtypes = [i32, i32, C.POINTER(C.c_double), C.POINTER(C.c_uint64)]
    for name in ("ht_fill", "ht_fill_naive"):
        fn = getattr(lib, name)
        fn.restype = C.c_int
        fn.argtypes = [vp, vp, vp, vp, vp, i32, i32, vp, vp]
    lib.ht_fill_peaks.restype = C.c_int
    lib.ht_fill_peaks.argtypes = [vp, vp, vp, vp, vp, i32, i32, vp, u32, vp, u32, vp, vp]
    lib.ht_peaks.restype = C.c_int
    lib.ht_promise_stable_inputs.restype = C.c_int
    lib.ht_promise_stable_inputs.argtypes = [vp, i32]
    lib.ht_peaks.argtypes = [vp, vp, i32, u32, vp, u32, vp, vp]
    lib.ht_tracks.restype = C.c_int
    lib.ht_tracks.argtypes = [vp, vp, u32, vp, vp]
    lib.ht_merge_scratch_bytes.restype = C.c_size_t
    lib.ht_merge_scratch_bytes.argtypes = [u32]
    lib.ht_merge_ridges.restype = C.c_int
    lib.ht_merge_ridges.argtypes = [vp, vp, u32, u32, vp, u32, vp, vp, C.c_size_t, vp]
    lib.ht_merge_ridges_static.restype = C.c_int
    lib.ht_merge_ridges_static.argtypes = [vp, vp, u32, u32, vp, u32, vp, vp]
    lib.ht_match_truth.restype = C.c_int
    lib.ht_match_truth.argtypes = [vp, vp, u32, vp, u32, C.c_double, C.c_double, vp, vp, vp, vp]
    lib.ht_run_host.restype = C.c_int
    lib.ht_run_host.argtypes = [vp, vp, vp, vp, vp, i32, i32, u32, vp, u32, vp, vp]
    lib.ht_run_host_events.restype = C.c_int
    lib.ht_run_host_events.argtypes = [vp, vp, vp, vp, vp, i32, u32, vp, u32, vp]
    lib.ht_selftest_division.restype = C.c_int
    lib.ht_selftest_division.argtypes = [i32, C.c_uint64, C.c_uint64, C.POINTER(C.c_uint64)]
    lib.ht_kernel_launches.restype = C.c_int64
    lib.ht_kernel_launches.argtypes = [vp]
    lib.ht_launch_info.restype = C.c_int
    lib.ht_launch_info.argtypes = [vp, C.POINTER(i32 * 8)]
    lib.ht_destroy.restype = None
    lib.ht_destroy.argtypes = [vp]
    lib.ht_strerror.restype = C.c_char_p
    lib.ht_strerror.argtypes = [C.c_int]
    _lib = lib
    return lib


def _ptr(a) -> int | None:
    """Address of a torch tensor / numpy array / int / None (marshalling only)."""
    if a is None:
        return None
    if isinstance(a, int):
        return a
    if isinstance(a, np.ndarray):
        return a.ctypes.data
    return a.data_ptr()          # torch.Tensor


def _stream(s) -> int | None:
    if s is None:
        return None
    if isinstance(s, int):
        return s or None
    return s.cuda_stream or None  # torch.cuda.Stream


def _check(status: int, where: str) -> None:
    if status != HT_OK:
        raise HtError(status, where)


def ht_strerror(status: int) -> str:
    return load().ht_strerror(status).decode()


def ht_query_sizes(cfg: ht_config) -> tuple[int, int]:
    """(bytes of one event's matrix, device bytes ht_create allocates)."""
    a, b = C.c_size_t(), C.c_size_t()
    _check(load().ht_query_sizes(C.byref(cfg), C.byref(a), C.byref(b)), "ht_query_sizes")
    return a.value, b.value


def ht_tables_host(cfg: ht_config):
    """(two_a, t_theta, p_phi, dA, dB): the tables the library uploads (host only, needs no GPU)."""
    two_a = np.empty(cfg.n_a, np.float32)
    tth = np.empty(cfg.n_theta + 1, np.float32)
    pph = np.empty(cfg.n_phi + 1, np.float32)
    d = np.empty(2, np.float32)
    _check(load().ht_tables_host(C.byref(cfg), _ptr(two_a), _ptr(tth), _ptr(pph), _ptr(d)), "ht_tables_host")
    return two_a, tth, pph, np.float32(d[0]), np.float32(d[1])


def ht_create(cfg: ht_config) -> int:
    """Returns the opaque context handle (an address)."""
    out = C.c_void_p()
    _check(load().ht_create(C.byref(cfg), C.byref(out)), "ht_create")
    return out.value


def ht_create_ex(cfg: ht_config, tuning: ht_tuning | None = None, d_workspace=None, workspace_bytes: int = 0) -> int:
    """ht_create with tuning switches and/or a caller-owned device workspace (a tensor or an address) of at least
    ``ht_query_sizes(cfg)[1]`` bytes, 256-byte aligned, which must outlive the context."""
    out = C.c_void_p()
    _check(load().ht_create_ex(C.byref(cfg), C.byref(tuning) if tuning is not None else None, _ptr(d_workspace),
                               workspace_bytes, C.byref(out)), "ht_create_ex")
    return out.value


def ht_fill(ctx, d_x, d_y, d_z, d_event_offsets, n_events: int, n_hits_total: int, d_mh, stream=None) -> None:
    _check(load().ht_fill(ctx, _ptr(d_x), _ptr(d_y), _ptr(d_z), _ptr(d_event_offsets), n_events, n_hits_total,
                          _ptr(d_mh), _stream(stream)), "ht_fill")


def ht_fill_peaks(ctx, d_x, d_y, d_z, d_event_offsets, n_events: int, n_hits_total: int, d_mh, threshold: int, d_out,
                  capacity: int, d_n_found, stream=None) -> None:
    """Fill and peak search in one pass; ``d_mh`` may be None (matrices not materialised)."""
    _check(load().ht_fill_peaks(ctx, _ptr(d_x), _ptr(d_y), _ptr(d_z), _ptr(d_event_offsets), n_events, n_hits_total,
                                _ptr(d_mh), threshold, _ptr(d_out), capacity, _ptr(d_n_found), _stream(stream)),
           "ht_fill_peaks")


def ht_promise_stable_inputs(ctx, on: bool = True) -> None:
    """The inputs of the following ht_fill / ht_fill_peaks calls are final before each call is made (include/ht.h)."""
    _check(load().ht_promise_stable_inputs(ctx, 1 if on else 0), "ht_promise_stable_inputs")


def ht_fill_naive(ctx, d_x, d_y, d_z, d_event_offsets, n_events: int, n_hits_total: int, d_mh, stream=None) -> None:
    _check(load().ht_fill_naive(ctx, _ptr(d_x), _ptr(d_y), _ptr(d_z), _ptr(d_event_offsets), n_events, n_hits_total,
                                _ptr(d_mh), _stream(stream)), "ht_fill_naive")


def ht_peaks(ctx, d_mh, n_events: int, threshold: int, d_out, capacity: int, d_n_found, stream=None) -> None:
    _check(load().ht_peaks(ctx, _ptr(d_mh), n_events, threshold, _ptr(d_out), capacity, _ptr(d_n_found),
                           _stream(stream)), "ht_peaks")


def ht_tracks(ctx, d_peaks, n_peaks: int, d_out, stream=None) -> None:
    """(rho, phi) of n_peaks peak records: d_out receives n_peaks ht_track records (5 words each)."""
    _check(load().ht_tracks(ctx, _ptr(d_peaks), n_peaks, _ptr(d_out), _stream(stream)), "ht_tracks")


def ht_merge_scratch_bytes(n_peaks: int) -> int:
    return int(load().ht_merge_scratch_bytes(n_peaks))


def ht_merge_ridges(ctx, d_peaks, n_peaks: int, window: int, d_out, capacity: int, d_n_out, d_scratch, scratch_bytes: int,
                    stream=None) -> None:
    """Ridge merging of n_peaks peak records into track candidates (ht_candidate records, 6 words each)."""
    _check(load().ht_merge_ridges(ctx, _ptr(d_peaks), n_peaks, window, _ptr(d_out), capacity, _ptr(d_n_out), _ptr(d_scratch),
                                  scratch_bytes, _stream(stream)), "ht_merge_ridges")


def ht_merge_ridges_static(ctx, d_peaks, n_peaks: int, window: int, d_out, capacity: int, d_n_out, stream=None) -> None:
    """ht_merge_ridges on the library's static device scratch (at most HT_MERGE_STATIC_MAX_PEAKS peaks; allocates nothing)."""
    _check(load().ht_merge_ridges_static(ctx, _ptr(d_peaks), n_peaks, window, _ptr(d_out), capacity, _ptr(d_n_out),
                                         _stream(stream)), "ht_merge_ridges_static")


def ht_match_truth(ctx, d_cand, n_cand: int, d_truth, n_truth: int, w_rho: float, cos_w_phi: float, d_cand_match,
                   d_truth_match, d_summary, stream=None) -> None:
    """Truth matching of n_cand candidates against n_truth generated circles (ht_truth records)."""
    _check(load().ht_match_truth(ctx, _ptr(d_cand), n_cand, _ptr(d_truth), n_truth, float(w_rho), float(cos_w_phi),
                                 _ptr(d_cand_match), _ptr(d_truth_match), _ptr(d_summary), _stream(stream)), "ht_match_truth")


def ht_run_host(ctx, h_x, h_y, h_z, h_event_offsets, n_events: int, n_hits_total: int, threshold: int, h_out,
                capacity: int, h_mh=None) -> int:
    """End-to-end call on HOST buffers (numpy arrays or pinned torch CPU tensors).  Returns the number of peaks found;
    ``h_out`` (PEAK_DTYPE array or 3-column uint32 tensor) receives min(found, capacity) records."""
    n = C.c_uint32(0)
    _check(load().ht_run_host(ctx, _ptr(h_x), _ptr(h_y), _ptr(h_z), _ptr(h_event_offsets), n_events, n_hits_total,
                              threshold, _ptr(h_out), capacity, C.addressof(n), _ptr(h_mh)), "ht_run_host")
    return n.value


def ht_run_host_events(ctx, h_x, h_y, h_z, h_event_offsets, n_events: int, threshold: int, h_out, capacity_per_event: int,
                       h_n_found) -> None:
    """A sequence of events from HOST buffers, one fused kernel each, pipelined over the context's slots by the library.
    ``h_out``: n_events * capacity_per_event peak records; ``h_n_found``: n_events uint32 counts."""
    _check(load().ht_run_host_events(ctx, _ptr(h_x), _ptr(h_y), _ptr(h_z), _ptr(h_event_offsets), n_events, threshold,
                                     _ptr(h_out), capacity_per_event, _ptr(h_n_found)), "ht_run_host_events")


def ht_submit_host(ctx, slot: int, h_x, h_y, h_z, n_hits: int, threshold: int) -> None:
    """Asynchronous half of the end-to-end call: ONE event from host buffers into slot ``slot`` (returns at once)."""
    _check(load().ht_submit_host(ctx, slot, _ptr(h_x), _ptr(h_y), _ptr(h_z), n_hits, threshold), "ht_submit_host")


def ht_wait_host(ctx, slot: int, h_out, capacity: int) -> int:
    """Waits for the event submitted into ``slot``; ``h_out`` receives min(found, capacity) records.  Returns found."""
    n = C.c_uint32(0)
    _check(load().ht_wait_host(ctx, slot, _ptr(h_out), capacity, C.addressof(n)), "ht_wait_host")
    return n.value


def ht_diag_memset(d_dst, value: int, nbytes: int, stream=None) -> None:
    _check(load().ht_diag_memset(_ptr(d_dst), value, nbytes, _stream(stream)), "ht_diag_memset")


def ht_diag_vote_rates(device: int = 0, iters: int = 2000) -> tuple[dict, int]:
    """({pattern: votes per clock per SM}, rows whose sum was wrong) -- the shared-memory vote micro-benchmark."""
    rates = (C.c_double * len(DIAG_PATTERNS))()
    err = C.c_uint64(0)
    _check(load().ht_diag_vote_rates(device, iters, rates, C.byref(err)), "ht_diag_vote_rates")
    return dict(zip(DIAG_PATTERNS, list(rates))), int(err.value)


def ht_selftest_division(device: int, n_pairs: int, seed: int) -> int:
    """Number of quotients (out of n_pairs) for which the vote loop's division shortcut differs from __fdiv_rn."""
    n = C.c_uint64(0)
    _check(load().ht_selftest_division(device, n_pairs, seed, C.byref(n)), "ht_selftest_division")
    return n.value


def ht_kernel_launches(ctx) -> int:
    return int(load().ht_kernel_launches(ctx))


def ht_launch_info(ctx) -> dict:
    arr = (C.c_int32 * 8)()
    _check(load().ht_launch_info(ctx, C.byref(arr)), "ht_launch_info")
    keys = ("fill_grid", "fill_block", "fill_smem_bytes", "rows_per_tile", "peaks_grid", "peaks_block", "sm_count")
    return dict(zip(keys, list(arr)[:7]))


def ht_destroy(ctx) -> None:
    if ctx:
        load().ht_destroy(ctx)

"""ctypes front end of oracle/ht_oracle.c (argument marshalling only; all arithmetic is in the C file).

TEST INFRASTRUCTURE: see the header of ht_oracle.c for what may call this and what pins it.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build

PEAK_DTYPE = np.dtype([("event", np.uint32), ("cell", np.uint32), ("count", np.uint32)])
MERGED_DTYPE = np.dtype([("event", np.uint32), ("cell", np.uint32), ("count", np.uint32), ("n_peaks", np.uint32),
                         ("rho", np.float64), ("phi", np.float64)])                       # == oracle_merged
TRUTH_DTYPE = np.dtype([("event", np.uint32), ("pad", np.uint32), ("a", np.float64), ("b", np.float64)])   # == oracle_truth


class MatchSummary(C.Structure):                                                                 # == oracle_match_summary
    _fields_ = [("n_cand", C.c_int64), ("n_truth", C.c_int64), ("n_matched", C.c_int64), ("n_fake", C.c_int64),
                ("n_found", C.c_int64), ("n_duplicate", C.c_int64), ("sum_drho", C.c_double), ("sum_drho2", C.c_double),
                ("sum_dphi", C.c_double), ("sum_dphi2", C.c_double)]

    def as_dict(self) -> dict:
        return {name: getattr(self, name) for name, _ in self._fields_}


class OracleBinning(C.Structure):
    _fields_ = [("n_theta", C.c_int32), ("n_phi", C.c_int32), ("n_a", C.c_int32), ("n_b", C.c_int32),
                ("a_min", C.c_float), ("a_max", C.c_float), ("b_min", C.c_float), ("b_max", C.c_float),
                ("theta_min", C.c_float), ("theta_max", C.c_float), ("phi_min", C.c_float), ("phi_max", C.c_float)]

    @classmethod
    def of(cls, b) -> "OracleBinning":
        """From any object with the twelve attributes (e.g. events.Binning)."""
        if isinstance(b, cls):
            return b
        return cls(*(getattr(b, name) for name, _ in cls._fields_))

    @property
    def planes(self) -> int:
        return self.n_theta * self.n_phi

    @property
    def cells(self) -> int:
        return self.planes * self.n_a * self.n_b


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        fp = C.POINTER(C.c_float)
        lib.oracle_tables.restype = C.c_int
        lib.oracle_tables.argtypes = [C.POINTER(OracleBinning), fp, fp, fp, fp]
        lib.oracle_fill.restype = C.c_int64
        lib.oracle_fill.argtypes = [C.POINTER(OracleBinning), fp, fp, fp, C.c_int64, C.POINTER(C.c_uint32)]
        lib.oracle_votes.restype = C.c_int
        lib.oracle_votes.argtypes = [C.POINTER(OracleBinning), fp, fp, fp, C.c_int64,
                                     C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
        lib.oracle_peaks.restype = C.c_int64
        lib.oracle_peaks.argtypes = [C.POINTER(OracleBinning), C.POINTER(C.c_uint32), C.c_uint32, C.c_uint32,
                                     C.c_void_p, C.c_int64]
        lib.oracle_tracks.restype = C.c_int
        lib.oracle_tracks.argtypes = [C.POINTER(OracleBinning), C.c_void_p, C.c_int64, C.POINTER(C.c_double),
                                      C.POINTER(C.c_double)]
        lib.oracle_merge_ridges.restype = C.c_int64
        lib.oracle_merge_ridges.argtypes = [C.POINTER(OracleBinning), C.c_void_p, C.c_int64, C.c_uint32, C.c_void_p,
                                            C.c_int64]
        lib.oracle_match_truth.restype = C.c_int
        lib.oracle_match_truth.argtypes = [C.POINTER(OracleBinning), C.c_void_p, C.c_int64, C.c_void_p, C.c_int64,
                                           C.c_double, C.c_double, C.POINTER(C.c_int32), C.POINTER(C.c_int32),
                                           C.POINTER(MatchSummary)]
        _lib = lib
    return _lib


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float32)


def _fp(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_float))


def oracle_tables(binning):
    """(two_a[NA], t_theta[Ntheta+1], p_phi[Nphi+1], dA, dB) as float32 -- SPEC.md section 1."""
    g = OracleBinning.of(binning)
    two_a = np.empty(g.n_a, np.float32)
    t_theta = np.empty(g.n_theta + 1, np.float32)
    p_phi = np.empty(g.n_phi + 1, np.float32)
    d = np.empty(2, np.float32)
    rc = _load().oracle_tables(C.byref(g), _fp(two_a), _fp(t_theta), _fp(p_phi), _fp(d))
    if rc != 0:
        raise ValueError("oracle_tables: invalid binning")
    return two_a, t_theta, p_phi, np.float32(d[0]), np.float32(d[1])


def oracle_fill(binning, x, y, z, out: np.ndarray | None = None):
    """Vote matrix of ONE event, shape (Ntheta, Nphi, NA, NB) uint32, and the number of votes cast."""
    g = OracleBinning.of(binning)
    x, y, z = _f32(x), _f32(y), _f32(z)
    if not (x.shape == y.shape == z.shape and x.ndim == 1):
        raise ValueError("x, y, z must be 1-D arrays of equal length")
    if out is None:
        out = np.empty(g.cells, np.uint32)
    flat = out.reshape(-1)
    assert flat.dtype == np.uint32 and flat.size == g.cells and flat.flags.c_contiguous
    votes = _load().oracle_fill(C.byref(g), _fp(x), _fp(y), _fp(z), x.shape[0],
                                flat.ctypes.data_as(C.POINTER(C.c_uint32)))
    if votes < 0:
        raise ValueError("oracle_fill: invalid arguments")
    return flat.reshape(g.n_theta, g.n_phi, g.n_a, g.n_b), int(votes)


def oracle_votes(binning, x, y, z):
    """plane[n] (or -1) and bins[n, NA] (or -1): every single decision of the fill, without the matrix."""
    g = OracleBinning.of(binning)
    x, y, z = _f32(x), _f32(y), _f32(z)
    n = x.shape[0]
    plane = np.empty(n, np.int32)
    bins = np.empty((n, g.n_a), np.int32)
    rc = _load().oracle_votes(C.byref(g), _fp(x), _fp(y), _fp(z), n,
                              plane.ctypes.data_as(C.POINTER(C.c_int32)),
                              bins.ctypes.data_as(C.POINTER(C.c_int32)))
    if rc != 0:
        raise ValueError("oracle_votes: invalid arguments")
    return plane, bins


def oracle_peaks(binning, m: np.ndarray, threshold: int, event: int = 0) -> np.ndarray:
    """Peaks of ONE event's matrix as a PEAK_DTYPE array in increasing cell order."""
    g = OracleBinning.of(binning)
    flat = np.ascontiguousarray(m, dtype=np.uint32).reshape(-1)
    if flat.size != g.cells:
        raise ValueError("matrix size does not match the binning")
    mp = flat.ctypes.data_as(C.POINTER(C.c_uint32))
    lib = _load()
    n = lib.oracle_peaks(C.byref(g), mp, threshold, event, None, 0)
    if n < 0:
        raise ValueError("oracle_peaks: invalid arguments (threshold must be >= 1)")
    out = np.empty(int(n), PEAK_DTYPE)
    if n:
        n2 = lib.oracle_peaks(C.byref(g), mp, threshold, event, out.ctypes.data_as(C.c_void_p), n)
        assert n2 == n
    return out


def oracle_fill_batch(binning, batch):
    """List of per-event matrices (R14: events never share cells) and the total vote count."""
    ms, votes = [], 0
    for e in range(batch.n_events):
        m, v = oracle_fill(binning, *batch.event(e))
        ms.append(m)
        votes += v
    return ms, votes


def oracle_peaks_batch(binning, matrices, threshold: int) -> np.ndarray:
    """Concatenated peak list of a batch, sorted by (event, cell)."""
    parts = [oracle_peaks(binning, m, threshold, event=e) for e, m in enumerate(matrices)]
    return np.concatenate(parts) if parts else np.empty(0, PEAK_DTYPE)


def oracle_tracks(binning, peaks: np.ndarray):
    """(rho, phi) in float64 of every peak record (SPEC.md section 4)."""
    g = OracleBinning.of(binning)
    pk = np.ascontiguousarray(peaks, dtype=PEAK_DTYPE)
    rho, phi = np.empty(len(pk), np.float64), np.empty(len(pk), np.float64)
    dp = C.POINTER(C.c_double)
    if _load().oracle_tracks(C.byref(g), pk.ctypes.data_as(C.c_void_p), len(pk), rho.ctypes.data_as(dp),
                             phi.ctypes.data_as(dp)) != 0:
        raise ValueError("oracle_tracks: invalid arguments (cell outside the matrix?)")
    return rho, phi


def oracle_merge_ridges(binning, peaks: np.ndarray, window: int) -> np.ndarray:
    """Track candidates of a peak list (SPEC.md section 5, R19): MERGED_DTYPE records sorted by (event, cell)."""
    g = OracleBinning.of(binning)
    pk = np.ascontiguousarray(peaks, dtype=PEAK_DTYPE)
    out = np.empty(len(pk), MERGED_DTYPE)
    n = _load().oracle_merge_ridges(C.byref(g), pk.ctypes.data_as(C.c_void_p), len(pk), window,
                                    out.ctypes.data_as(C.c_void_p), len(pk))
    if n < 0:
        raise ValueError("oracle_merge_ridges: invalid arguments")
    return out[:n]


def oracle_match_truth(binning, candidates: np.ndarray, truth: np.ndarray, w_rho: float, cos_w_phi: float):
    """Truth matching (SPEC.md section 6, R20): (cand_match[n_cand], truth_match[n_truth], summary dict).
    ``candidates``: MERGED_DTYPE records; ``truth``: TRUTH_DTYPE records (event, centre a, b in mm)."""
    g = OracleBinning.of(binning)
    cd = np.ascontiguousarray(candidates, dtype=MERGED_DTYPE)
    tr = np.ascontiguousarray(truth, dtype=TRUTH_DTYPE)
    cm, tm = np.empty(len(cd), np.int32), np.empty(len(tr), np.int32)
    s = MatchSummary()
    ip = C.POINTER(C.c_int32)
    if _load().oracle_match_truth(C.byref(g), cd.ctypes.data_as(C.c_void_p), len(cd), tr.ctypes.data_as(C.c_void_p), len(tr),
                                  float(w_rho), float(cos_w_phi), cm.ctypes.data_as(ip), tm.ctypes.data_as(ip),
                                  C.byref(s)) != 0:
        raise ValueError("oracle_match_truth: invalid arguments")
    return cm, tm, s.as_dict()

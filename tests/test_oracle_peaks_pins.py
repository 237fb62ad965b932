"""Pins of the oracle's PEAK search (no GPU): hand-written cases (P8, tests/golden/peak_cases.txt), set
invariants that hold for any matrix (P9), and an independent whole-array formulation (dref.brute_peaks)."""
import numpy as np
import pytest

import dref
from golden_io import read_peak_cases
from oracle import PEAK_DTYPE, oracle_fill, oracle_peaks, oracle_peaks_batch
from paper_1507_03074_b200.events import Binning, WORKLOADS, generate_batch

CASES = read_peak_cases()


def _bn(dims):
    return Binning(*dims)


@pytest.mark.parametrize("case", CASES, ids=[c["name"] for c in CASES])
def test_P8_hand_built_cases(case):
    pk = oracle_peaks(_bn(case["dims"]), case["m"], case["T"], event=3)
    assert pk.dtype == PEAK_DTYPE
    assert pk["cell"].tolist() == case["peaks"]
    assert np.all(pk["event"] == 3)
    np.testing.assert_array_equal(pk["count"], case["m"].reshape(-1)[pk["cell"]])
    # the independent whole-array formulation agrees with the hand-written list too
    assert dref.brute_peaks(case["m"], case["T"]).tolist() == case["peaks"]


def test_threshold_zero_is_rejected():
    with pytest.raises(ValueError):
        oracle_peaks(_bn((1, 1, 2, 2)), np.zeros((1, 1, 2, 2), np.uint32), 0)


def _adjacent_pairs(cells, bn):
    """Number of pairs of peaks that are 8-neighbours in the same plane."""
    nb, na = bn.n_b, bn.n_a
    s = set(int(c) for c in cells)
    bad = 0
    for c in s:
        p, rem = divmod(c, na * nb)
        a, b = divmod(rem, nb)
        for da in (-1, 0, 1):
            for db in (-1, 0, 1):
                if (da or db) and 0 <= a + da < na and 0 <= b + db < nb and (p * na + a + da) * nb + b + db in s:
                    bad += 1
    return bad // 2


@pytest.mark.parametrize("cfg", [1, 2])
def test_P9_invariants_on_generated_events(cfg):
    wl = WORKLOADS[cfg]
    bn = wl.binning
    m, _ = oracle_fill(bn, *generate_batch(cfg).event(0))
    T = wl.threshold
    pk = oracle_peaks(bn, m, T)
    flat = m.reshape(-1)
    assert len(pk) > 0
    assert np.all(np.diff(pk["cell"].astype(np.int64)) > 0)                   # increasing cell order, no duplicates
    assert np.all(pk["count"] >= T) and np.all(flat[pk["cell"]] == pk["count"])
    assert _adjacent_pairs(pk["cell"], bn) == 0                               # no two peaks touch
    assert len(pk) <= int((flat >= T).sum())
    # every cell >= T strictly greater than all in-plane neighbours is a peak
    pad = np.pad(m.astype(np.int64), ((0, 0), (0, 0), (1, 1), (1, 1)), constant_values=-1)
    c = pad[:, :, 1:-1, 1:-1]
    strict = c >= T
    for da in (-1, 0, 1):
        for db in (-1, 0, 1):
            if da or db:
                strict &= c > pad[:, :, 1 + da:1 + da + bn.n_a, 1 + db:1 + db + bn.n_b]
    assert set(np.flatnonzero(strict.reshape(-1)).tolist()) <= set(pk["cell"].tolist())
    # threshold monotonicity: peaks(T+1) == {p in peaks(T): count >= T+1}
    pk1 = oracle_peaks(bn, m, T + 1)
    np.testing.assert_array_equal(pk1, pk[pk["count"] >= T + 1])
    # independent formulation on the whole matrix
    np.testing.assert_array_equal(dref.brute_peaks(m, T), pk["cell"].astype(np.int64))


def test_random_matrices_against_whole_array_formulation():
    rng = np.random.default_rng(11)
    for dims in [(1, 1, 1, 1), (1, 1, 1, 9), (1, 1, 9, 1), (2, 3, 5, 7), (1, 2, 16, 16), (3, 1, 2, 2)]:
        for hi in (2, 4, 50):                              # small ranges force many ties and plateaux
            m = rng.integers(0, hi, size=dims, dtype=np.uint32)
            for T in (1, 2, hi):
                pk = oracle_peaks(_bn(dims), m, T)
                np.testing.assert_array_equal(dref.brute_peaks(m, T), pk["cell"].astype(np.int64))
                assert _adjacent_pairs(pk["cell"], _bn(dims)) == 0


def test_batch_list_is_sorted_by_event_then_cell():
    wl = WORKLOADS[1]
    batch = generate_batch(wl, n_events=3)
    ms = [oracle_fill(wl.binning, *batch.event(e))[0] for e in range(3)]
    pk = oracle_peaks_batch(wl.binning, ms, wl.threshold)
    key = pk["event"].astype(np.int64) * wl.binning.cells + pk["cell"]
    assert np.all(np.diff(key) > 0) and set(pk["event"].tolist()) == {0, 1, 2}


def test_capacity_truncates_but_count_is_total():
    import ctypes as C
    from oracle.ht_oracle import OracleBinning, _load
    m = np.zeros((1, 1, 8, 8), np.uint32)
    m[0, 0, ::2, ::2] = 3                                  # 16 isolated spikes
    g = OracleBinning.of(_bn((1, 1, 8, 8)))
    out = np.zeros(5, PEAK_DTYPE)
    n = _load().oracle_peaks(C.byref(g), m.ctypes.data_as(C.POINTER(C.c_uint32)), 1, 0,
                             out.ctypes.data_as(C.c_void_p), 5)
    assert n == 16 and out["cell"].tolist() == [0, 2, 4, 6, 16]

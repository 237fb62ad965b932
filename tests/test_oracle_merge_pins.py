"""Pins of oracle_merge_ridges (SPEC.md section 5, reading R19) -- none re-types its pair loop:

P13  the partition equals the connected components a LIBRARY routine (scipy.ndimage.label) finds on an image in which
     every peak is a filled square of half-width W on a grid of doubled resolution: two such squares share a pixel iff
     the peaks' Chebyshev distance is <= W, and they are never merely adjacent (2d = 2W + 1 has no integer solution),
     so 8-connected labelling of the image is exactly the transitive closure of the link relation;
P14  hand-built layouts with hand-written candidates (tests/golden/merge_cases.txt);
P15  invariants on any list: the members add up; window 0 is the identity; a larger window only coarsens the partition;
     representatives of different candidates are farther apart than W; shifting all peaks shifts the result;
     the (rho, phi) of a candidate is the read-out of its representative (oracle_tracks, pinned by P11/P12).
"""
import numpy as np
import pytest
from scipy import ndimage

from golden_io import read_merge_cases
from oracle import MERGED_DTYPE, PEAK_DTYPE, oracle_merge_ridges, oracle_tracks
from paper_1507_03074_b200.events import Binning


def _peaks(recs):
    pk = np.zeros(len(recs), PEAK_DTYPE)
    for i, (e, c, n) in enumerate(recs):
        pk[i] = (e, c, n)
    return pk


def _random_peaks(rng, bn, n_events, n):
    """n distinct (event, cell) pairs with small random counts (many ties)."""
    keys = rng.choice(n_events * bn.cells, size=n, replace=False)
    pk = np.zeros(n, PEAK_DTYPE)
    pk["event"], pk["cell"] = keys // bn.cells, keys % bn.cells
    pk["count"] = rng.integers(8, 12, n)
    return pk[rng.permutation(n)]


def test_p14_hand_built_layouts():
    cases = read_merge_cases()
    assert len(cases) >= 10
    for c in cases:
        bn = Binning(*c["dims"])
        got = oracle_merge_ridges(bn, _peaks(c["peaks"]), c["window"])
        got_t = [(int(r["event"]), int(r["cell"]), int(r["count"]), int(r["n_peaks"])) for r in got]
        assert got_t == sorted(c["want"]), c["name"]
        # order of the input list does not matter
        rev = oracle_merge_ridges(bn, _peaks(c["peaks"][::-1]), c["window"])
        assert rev.tolist() == got.tolist(), c["name"]


@pytest.mark.parametrize("window", [1, 2, 3, 5])
def test_p13_partition_equals_library_labelling_on_a_doubled_grid(window):
    rng = np.random.default_rng(100 + window)
    bn = Binning(2, 3, 40, 50)
    for trial in range(6):
        pk = _random_peaks(rng, bn, n_events=2, n=int(rng.integers(50, 400)))
        got = oracle_merge_ridges(bn, pk, window)
        n_comp = 0
        sizes = []
        for e in range(2):
            for p in range(bn.planes):
                sel = pk[(pk["event"] == e) & (pk["cell"] // (bn.n_a * bn.n_b) == p)]
                if len(sel) == 0:
                    continue
                a = (sel["cell"].astype(np.int64) // bn.n_b) % bn.n_a
                b = sel["cell"].astype(np.int64) % bn.n_b
                img = np.zeros((2 * bn.n_a + 2 * window + 1, 2 * bn.n_b + 2 * window + 1), bool)
                for ai, bi in zip(a, b):
                    img[2 * ai:2 * ai + 2 * window + 1, 2 * bi:2 * bi + 2 * window + 1] = True   # square centred on (2a+W, 2b+W)
                lab, k = ndimage.label(img, structure=np.ones((3, 3), int))
                n_comp += k
                labels = lab[2 * a + window, 2 * b + window]
                assert (labels > 0).all()
                for l in range(1, k + 1):
                    members = sel[labels == l]
                    sizes.append(len(members))
                    best = members[np.lexsort((members["cell"], -members["count"].astype(np.int64)))][0]
                    hit = got[(got["event"] == e) & (got["cell"] == best["cell"])]
                    assert len(hit) == 1 and hit[0]["count"] == best["count"] and hit[0]["n_peaks"] == len(members)
        assert len(got) == n_comp and int(got["n_peaks"].sum()) == len(pk) == sum(sizes)


def test_p15_invariants():
    rng = np.random.default_rng(7)
    bn = Binning(1, 2, 64, 64)
    pk = _random_peaks(rng, bn, n_events=3, n=500)
    ident = oracle_merge_ridges(bn, pk, 0)
    assert len(ident) == len(pk) and (ident["n_peaks"] == 1).all()
    key = lambda r: r["event"].astype(np.int64) * bn.cells + r["cell"]
    assert np.array_equal(np.sort(key(ident)), np.sort(key(pk)))
    prev = ident
    for w in (1, 2, 4, 8, 64):
        cur = oracle_merge_ridges(bn, pk, w)
        assert int(cur["n_peaks"].sum()) == len(pk) and len(cur) <= len(prev)
        assert np.isin(key(cur), key(prev)).all() or w == 1          # a representative stays a representative's candidate
        # representatives of different candidates are not linked
        for e in range(3):
            for p in range(bn.planes):
                r = cur[(cur["event"] == e) & (cur["cell"] // (bn.n_a * bn.n_b) == p)]
                a = (r["cell"].astype(np.int64) // bn.n_b) % bn.n_a
                b = r["cell"].astype(np.int64) % bn.n_b
                d = np.maximum(np.abs(a[:, None] - a[None, :]), np.abs(b[:, None] - b[None, :]))
                np.fill_diagonal(d, 10 ** 6)
                assert (d > w).all()
        prev = cur
    assert len(prev) == 3 * bn.planes or len(prev) <= 3 * bn.planes       # window >= plane size: one candidate per (event, plane)
    # read-out of a candidate = read-out of its representative
    cur = oracle_merge_ridges(bn, pk, 3)
    rep = np.zeros(len(cur), PEAK_DTYPE)
    rep["event"], rep["cell"], rep["count"] = cur["event"], cur["cell"], cur["count"]
    rho, phi = oracle_tracks(bn, rep)
    assert np.array_equal(rho, cur["rho"]) and np.array_equal(phi, cur["phi"])
    assert cur.dtype == MERGED_DTYPE


def test_p15_translation():
    """Shifting every peak of a plane by (+3, +5) cells shifts the representatives and changes nothing else."""
    rng = np.random.default_rng(11)
    bn = Binning(1, 1, 100, 100)
    small = Binning(1, 1, 90, 90)
    pk = _random_peaks(rng, small, 1, 300)
    a = pk["cell"] // 90
    b = pk["cell"] % 90
    p0, p1 = pk.copy(), pk.copy()
    p0["cell"] = a * 100 + b
    p1["cell"] = (a + 3) * 100 + (b + 5)
    m0, m1 = oracle_merge_ridges(bn, p0, 4), oracle_merge_ridges(bn, p1, 4)
    assert len(m0) == len(m1)
    assert np.array_equal(m0["cell"] + 305, m1["cell"]) and np.array_equal(m0["count"], m1["count"])
    assert np.array_equal(m0["n_peaks"], m1["n_peaks"])


def test_bad_arguments():
    bn = Binning(1, 1, 4, 4)
    with pytest.raises(ValueError):
        oracle_merge_ridges(bn, _peaks([(0, 16, 9)]), 2)          # cell outside the matrix
    assert len(oracle_merge_ridges(bn, _peaks([]), 2)) == 0

"""-m gpu: ht_merge_ridges_static -- ridge merging on the library's file-scope device scratch, for callers that cannot
allocate device memory -- against the existing path (ht_merge_ridges with caller-owned scratch), on two calls in a row.

Collected last (the file name sorts after the others): the suite runs with pytest -x.  Self-contained: it passes alone in
a fresh process (the first call per device looks the array's address up) and after every other test.
"""
import numpy as np
import pytest
import torch

from gpu_util import GpuHough
from paper_1507_03074_b200 import binding as B
from paper_1507_03074_b200.events import Binning, WORKLOADS, generate_batch

pytestmark = pytest.mark.gpu


def _records(pk):
    rec = np.zeros((len(pk), 3), np.uint32)
    rec[:, 0], rec[:, 1], rec[:, 2] = pk["event"], pk["cell"], pk["count"]
    return rec


def _sorted(d_out, found, cap):
    k = min(found, cap)
    out = d_out[:6 * k].cpu().numpy().view(np.uint8).view(B.CAND_DTYPE).copy()
    return out[np.lexsort((out["cell"], out["event"]))]


def _merge_both(g, rec, window):
    """(candidates of the existing path, candidates of the static-scratch path, free device memory before/after the
    static call), each list sorted by (event, cell)."""
    dev = g.dev
    n = len(rec)
    d_pk = torch.from_numpy(np.ascontiguousarray(rec).view(np.int32)).to(dev)
    cap = max(n, 1)
    outs = [torch.zeros(cap * 6, dtype=torch.int32, device=dev) for _ in range(2)]
    nfs = [torch.full((1,), -5, dtype=torch.int32, device=dev) for _ in range(2)]
    nb = B.ht_merge_scratch_bytes(n)
    d_scr = torch.empty(nb, dtype=torch.uint8, device=dev)
    B.ht_merge_ridges(g.ctx, d_pk, n, window, outs[0], cap, nfs[0], d_scr, nb, None)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    B.ht_merge_ridges_static(g.ctx, d_pk, n, window, outs[1], cap, nfs[1], None)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    found = [int(nf.cpu().numpy().view(np.uint32)[0]) for nf in nfs]
    assert found[0] == found[1]
    return _sorted(outs[0], found[0], cap), _sorted(outs[1], found[1], cap), (free0, free1)


def test_static_scratch_merge_equals_the_existing_path_on_two_calls_in_a_row():
    """Same kernels, same inputs, another scratch: every field of every candidate is IDENTICAL (integers and the bits of
    rho, phi -- the tolerance of the merge tests is set-exact integers; the floats come from the same instructions).  The
    first call leaves a long list's slots, order and labels in the array; the second, shorter and different, must not see
    them; a third repeats the first.  Lists beyond the array's capacity are refused before anything is enqueued."""
    wl = WORKLOADS[2]
    bn = Binning(4, 16, 256, 512)
    batch = generate_batch(wl, n_events=3)
    rng = np.random.default_rng(11)
    with GpuHough(bn, 3, batch.n_hits) as g:
        _, n, pk = g.fill_peaks(batch, wl.threshold, store=False)
        assert n == len(pk) > 200
        long_list = _records(pk)
        # a dense random list with ties and duplicates (large groups: the label propagation has work to do)
        m = 20000
        dense = np.zeros((m, 3), np.uint32)
        dense[:, 0] = rng.integers(0, 3, m)
        plane = rng.integers(0, 64, m)
        a, b = rng.integers(100, 140, m), rng.integers(200, 260, m)
        dense[:, 1] = (plane * bn.n_a + a) * bn.n_b + b
        dense[:, 2] = rng.integers(8, 12, m)
        short_list = long_list[rng.permutation(len(long_list))[:97]]
        calls = [(dense, 2), (short_list, 5), (long_list, 3), (dense, 2), (long_list[:0], 1)]
        sizes = []
        for k, (rec, window) in enumerate(calls):
            want, got, (free0, free1) = _merge_both(g, rec, window)
            assert len(want) == len(got), k
            for f in ("event", "cell", "count", "n_peaks"):
                np.testing.assert_array_equal(got[f], want[f], err_msg=f"call {k}, {f}")
            np.testing.assert_array_equal(got["rho"].view(np.uint32), want["rho"].view(np.uint32), err_msg=f"call {k}, rho")
            np.testing.assert_array_equal(got["phi"].view(np.uint32), want["phi"].view(np.uint32), err_msg=f"call {k}, phi")
            if k > 0:                                       # (the first call may load code; later ones change nothing)
                assert free1 == free0, f"call {k}: free device memory changed by {free0 - free1} bytes"
            sizes.append(len(got))
        assert sizes[0] == sizes[3] > 0 and 0 < sizes[1] <= 97 and sizes[2] > sizes[1] and sizes[4] == 0
        # beyond the static capacity: refused with its own status, nothing written
        big = B.HT_MERGE_STATIC_MAX_PEAKS + 1
        d_big = torch.zeros(big * 3, dtype=torch.int32, device=g.dev)
        d_out = torch.zeros(6, dtype=torch.int32, device=g.dev)
        d_n = torch.full((1,), -5, dtype=torch.int32, device=g.dev)
        with pytest.raises(B.HtError) as ei:
            B.ht_merge_ridges_static(g.ctx, d_big, big, 1, d_out, 1, d_n, None)
        assert ei.value.status == B.HT_ERR_TOO_LARGE and "ht_merge_ridges" in str(ei.value)
        torch.cuda.synchronize()
        assert int(d_n.cpu()[0]) == -5
        # exactly at the capacity: accepted
        full = B.HT_MERGE_STATIC_MAX_PEAKS
        rec = np.zeros((full, 3), np.uint32)
        rec[:, 0] = rng.integers(0, 3, full)
        rec[:, 1] = rng.integers(0, bn.cells, full)
        rec[:, 2] = 9
        want, got, _ = _merge_both(g, rec, 1)
        assert len(want) == len(got) > 0
        for f in ("event", "cell", "count", "n_peaks"):
            np.testing.assert_array_equal(got[f], want[f], err_msg=f"full capacity, {f}")

"""-m gpu: the CUDA path (through the C-ABI) against the CPU oracle, element by element, on the same seeded inputs.

Bar (BASELINE.json north_star): the vote matrix and the sorted peak list are BIT-EXACT.  Integer work throughout;
the floating point that decides bin indices is IEEE binary32 on both sides (SPEC.md section 0).
"""
import math

import numpy as np
import pytest
import torch

from gpu_util import GpuHough, mh_to_numpy, sort_peaks
from oracle import oracle_fill, oracle_peaks, oracle_peaks_batch
from paper_1507_03074_b200 import binding as B
from paper_1507_03074_b200.events import Binning, WORKLOADS, batch_from_arrays, generate_batch

pytestmark = pytest.mark.gpu


def _oracle_batch(bn, batch):
    return [oracle_fill(bn, *batch.event(e))[0] for e in range(batch.n_events)]


def _check_batch(bn, batch, threshold, naive=False, capacity=1 << 20, fused=True, tuning=None, own_workspace=False):
    """ht_fill (or ht_fill_naive) + ht_peaks, then the fused ht_fill_peaks with and without the matrix store: all three
    against the oracle, element by element."""
    want_m = _oracle_batch(bn, batch)
    want_p = oracle_peaks_batch(bn, want_m, threshold)
    with GpuHough(bn, max_events=max(1, batch.n_events), max_hits=batch.n_hits, tuning=tuning,
                  own_workspace=own_workspace) as g:
        mh = g.fill(batch, naive=naive)
        got = mh_to_numpy(mh, bn, batch.n_events)
        for e in range(batch.n_events):
            np.testing.assert_array_equal(got[e], want_m[e], err_msg=f"event {e}")
        n, pk = g.peaks(mh, batch.n_events, threshold, capacity)
        assert n == len(want_p)
        if capacity >= n:
            np.testing.assert_array_equal(sort_peaks(pk, bn.cells), want_p)
        del mh
        if fused and not naive:
            mh2, n2, pk2 = g.fill_peaks(batch, threshold, capacity)
            got2 = mh_to_numpy(mh2, bn, batch.n_events)
            for e in range(batch.n_events):
                np.testing.assert_array_equal(got2[e], want_m[e], err_msg=f"fused, event {e}")
            assert n2 == len(want_p)
            if capacity >= n2:
                np.testing.assert_array_equal(sort_peaks(pk2, bn.cells), want_p)
            del mh2
            _, n3, pk3 = g.fill_peaks(batch, threshold, capacity, store=False)
            assert n3 == len(want_p)
            if capacity >= n3:
                np.testing.assert_array_equal(sort_peaks(pk3, bn.cells), want_p)
    return n


# ------------------------------------------------------------------ the five configs of BASELINE.json
def test_config1_tiny_three_events():
    wl = WORKLOADS[1]
    assert _check_batch(wl.binning, generate_batch(wl, n_events=3), wl.threshold) > 10


def test_config2_paper_single_event_full_matrix():
    wl = WORKLOADS[2]
    n = _check_batch(wl.binning, generate_batch(wl), wl.threshold)
    assert 300 < n < 3000


def test_config3_batch_of_ragged_events():
    wl = WORKLOADS[3]
    batch = generate_batch(wl, n_events=5)
    assert len(set(np.diff(batch.event_offsets).tolist())) == 5
    _check_batch(wl.binning, batch, wl.threshold)


def test_config4_high_occupancy():
    wl = WORKLOADS[4]
    n = _check_batch(wl.binning, generate_batch(wl), wl.threshold)
    assert n > 5000


def test_config5_fine_binning_one_event_full_matrix():
    wl = WORKLOADS[5]
    _check_batch(wl.binning, generate_batch(wl, n_events=1), wl.threshold)


def test_config5_two_events_sampled():
    """Two 4.3 GB matrices in one call (64-bit addressing across events): event 1 against the oracle on sampled planes,
    event 0 via properties (sum == votes)."""
    wl = WORKLOADS[5]
    bn = wl.binning
    batch = generate_batch(wl, n_events=2)
    with GpuHough(bn, max_events=2, max_hits=batch.n_hits) as g:
        mh = g.fill(batch)
        n, pk = g.peaks(mh, 2, wl.threshold)
        want1, votes1 = oracle_fill(bn, *batch.event(1))
        m1 = mh[bn.cells:].view(bn.planes, bn.n_a * bn.n_b)
        for p in (0, 1, 77, 128, 200, 255):
            np.testing.assert_array_equal(m1[p].cpu().numpy().view(np.uint32),
                                          want1.reshape(bn.planes, -1)[p])
        assert int(mh[bn.cells:].sum(dtype=torch.int64)) == votes1
        want_p1 = oracle_peaks(bn, want1, wl.threshold, event=1)
        got_p = sort_peaks(pk, bn.cells)
        np.testing.assert_array_equal(got_p[got_p["event"] == 1], want_p1)
        assert (got_p["event"] == 0).sum() > 0
        del mh
        # the fused kernel without the matrix store must find the same peak set for both events
        _, n_f, pk_f = g.fill_peaks(batch, wl.threshold, store=False)
        assert n_f == n
        np.testing.assert_array_equal(sort_peaks(pk_f, bn.cells), got_p)


def _full_batch_both_paths(wl, n_events):
    """ALL events of a batch workload at full size, element by element on every event, through ht_fill_peaks (one call
    over the whole batch) and through ht_fill + ht_peaks.  The matrices stay on the device (26.8 GB / 42.9 GB per path);
    the oracle's matrix of one event at a time is uploaded and compared there."""
    bn = wl.binning
    batch = generate_batch(wl, n_events=n_events)
    cells = bn.cells
    with GpuHough(bn, max_events=n_events, max_hits=batch.n_hits) as g:
        mh_f, n_f, pk_f = g.fill_peaks(batch, wl.threshold)
        mh_s = g.fill(batch)
        n_s, pk_s = g.peaks(mh_s, n_events, wl.threshold)
        want_p = []
        for e in range(n_events):
            m, _ = oracle_fill(bn, *batch.event(e))
            want_p.append(oracle_peaks(bn, m, wl.threshold, event=e))
            ref = torch.from_numpy(m.reshape(-1).view(np.int32)).to(g.dev)
            assert torch.equal(mh_f[e * cells:(e + 1) * cells], ref), f"ht_fill_peaks, event {e}"
            assert torch.equal(mh_s[e * cells:(e + 1) * cells], ref), f"ht_fill, event {e}"
            del ref, m
        want_p = np.concatenate(want_p)
        assert n_f == n_s == len(want_p)
        np.testing.assert_array_equal(sort_peaks(pk_f, cells), want_p)
        np.testing.assert_array_equal(sort_peaks(pk_s, cells), want_p)
    return len(want_p)


def test_config3_all_100_events_full_size():
    """BASELINE.json:configs[2]; "100 simulated events": every event, every cell, both call paths."""
    assert _full_batch_both_paths(WORKLOADS[3], 100) > 10000


def test_config5_all_10_events_full_size():
    """BASELINE.json:configs[4]: ten 4.29 GB matrices in one call (64-bit offsets), every event, every cell."""
    assert _full_batch_both_paths(WORKLOADS[5], 10) > 1000


def test_naive_paper_design_matches_too():
    wl = WORKLOADS[1]
    _check_batch(wl.binning, generate_batch(wl, n_events=2), wl.threshold, naive=True)
    wl = WORKLOADS[2]
    _check_batch(wl.binning, generate_batch(wl), wl.threshold, naive=True)


# ------------------------------------------------------------------ shapes: ragged tiles, odd sizes, partial ranges
@pytest.mark.parametrize("dims", [(4, 16, 1000, 1024),      # NA not a multiple of the rows per tile: ragged last tile
                                  (3, 5, 77, 36),            # small, odd plane count, NB % 4 == 0
                                  (1, 1, 1, 4), (2, 2, 5, 8), (1, 3, 2, 16), (2, 1, 3, 32),
                                  (4, 16, 37, 4096),         # wide rows: 3 rows per tile
                                  (2, 2, 40, 6000),          # 2 rows per tile: the smallest tile the fused scan accepts
                                  (2, 3, 9, 7), (4, 16, 50, 130), (1, 2, 3, 1),   # NB % 4 != 0: plain stores, scalar scan
                                  (5, 7, 333, 1001)])
def test_tile_geometries(dims):
    bn = Binning(*dims)
    batch = generate_batch(1, n_events=2)
    _check_batch(bn, batch, 3)


def test_one_row_per_tile_fill_only():
    """One A row = 48 KB: ht_fill works with 1-row tiles, the fused call refuses (needs 2 rows per tile)."""
    bn = Binning(2, 3, 300, 12000)
    batch = generate_batch(1, n_events=2)
    _check_batch(bn, batch, 3, fused=False)
    with GpuHough(bn, 2, batch.n_hits) as g:
        with pytest.raises(B.HtError) as ei:
            g.fill_peaks(batch, 3)
        assert ei.value.status == B.HT_ERR_UNSUPPORTED


def test_rows_that_do_not_fit_a_tile_go_through_the_naive_kernel():
    bn = Binning(1, 2, 3, 40000)                            # one row = 160 KB
    batch = generate_batch(1)
    with GpuHough(bn, 1, batch.n_hits) as g:
        with pytest.raises(B.HtError) as ei:
            g.fill(batch)
        assert ei.value.status == B.HT_ERR_UNSUPPORTED
    _check_batch(bn, batch, 2, naive=True)


def test_unaligned_matrix_pointer_uses_plain_stores():
    """d_mh only 4-byte aligned: no bulk stores, same result."""
    wl = WORKLOADS[1]
    bn = wl.binning
    batch = generate_batch(wl, n_events=2)
    want_m = _oracle_batch(bn, batch)
    with GpuHough(bn, 2, batch.n_hits) as g:
        dx, dy, dz, doff = g.upload(batch)
        buf = torch.full((2 * bn.cells + 4,), -1, dtype=torch.int32, device="cuda")
        mh = buf[1:1 + 2 * bn.cells]
        assert mh.data_ptr() % 16 == 4
        B.ht_fill(g.ctx, dx, dy, dz, doff, 2, batch.n_hits, mh)
        torch.cuda.synchronize()
        got = mh_to_numpy(mh, bn, 2)
        for e in range(2):
            np.testing.assert_array_equal(got[e], want_m[e])
        assert int(buf[0]) == -1 and int(buf[-1]) == -1


def test_partial_angle_ranges_and_asymmetric_ab_ranges():
    bn = Binning(3, 5, 96, 64, a_min=-2500.0, a_max=3100.0, b_min=-700.0, b_max=3900.0,
                 theta_min=0.6, theta_max=2.2, phi_min=0.5, phi_max=5.5)
    _check_batch(bn, generate_batch(2), 4)


# ------------------------------------------------------------------ degenerate inputs
def test_empty_and_degenerate_events():
    bn = WORKLOADS[1].binning
    ev = generate_batch(1).event(0)
    good = np.stack(ev, axis=1)
    bad = np.array([[100.0, 0.0, 5.0], [0.0, 0.0, 1.0], [np.nan, 3.0, 1.0], [3.0, np.nan, 1.0], [3.0, 4.0, np.nan],
                    [np.inf, 4.0, 1.0], [3.0, -np.inf, 1.0], [-50.0, -0.0, 1.0], [1e-30, 1e-30, 1.0], [1e30, 1e30, 1e30]],
                   np.float32)
    batch = batch_from_arrays([np.zeros((0, 3)), good, bad, np.concatenate([bad, good]), np.zeros((0, 3))])
    _check_batch(bn, batch, 8)
    # a batch with no hits at all still writes zero matrices
    empty = batch_from_arrays([np.zeros((0, 3)), np.zeros((0, 3))])
    with GpuHough(bn, 2, 1) as g:
        mh = g.fill(empty)
        assert int(mh.abs().sum()) == 0
        n, pk = g.peaks(mh, 2, 1)
        assert n == 0 and len(pk) == 0
        # zero events: both calls are no-ops that succeed
        B.ht_fill(g.ctx, None, None, None, None, 0, 0, None)
        nf = torch.full((1,), 5, dtype=torch.int32, device="cuda")
        B.ht_peaks(g.ctx, None, 0, 1, None, 0, nf)
        torch.cuda.synchronize()
        assert int(nf) == 0


def test_all_hits_in_one_plane_many_hits():
    # 30000 hits in a narrow cone: one plane gets everything (more hits than the shared-memory hit list holds: the list
    # is rebuilt chunk by chunk for every tile; counts far above 255)
    rng = np.random.default_rng(3)
    n = 30000
    ph = rng.uniform(0.30, 0.35, n); r = rng.uniform(60, 1000, n)
    xyz = np.stack([r * np.cos(ph), r * np.sin(ph), r * 0.2], axis=1)
    bn = Binning(4, 16, 64, 256)
    batch = batch_from_arrays([xyz])
    n_pk = _check_batch(bn, batch, 300)
    assert n_pk > 0


# ------------------------------------------------------------------ peaks: hand-built matrices, capacity, thresholds
def test_peaks_on_hand_built_matrices_from_golden():
    from golden_io import read_peak_cases
    for case in read_peak_cases():
        bn = Binning(*case["dims"])
        with GpuHough(bn, 1, 1) as g:
            mh = torch.from_numpy(case["m"].reshape(-1).view(np.int32).copy()).cuda()
            n, pk = g.peaks(mh, 1, case["T"])
            assert sorted(pk["cell"].tolist()) == case["peaks"], case["name"]
            assert n == len(case["peaks"])


def test_peaks_dense_random_matrices_and_ties():
    rng = np.random.default_rng(21)
    for dims, hi in [((2, 3, 40, 64), 3), ((1, 2, 33, 128), 2), ((2, 2, 17, 20), 6), ((1, 1, 64, 7), 3)]:
        bn = Binning(*dims)
        m = rng.integers(0, hi, size=(2,) + dims, dtype=np.uint32)      # two events, many plateaux
        with GpuHough(bn, 2, 1) as g:
            mh = torch.from_numpy(m.reshape(-1).view(np.int32).copy()).cuda()
            for T in (1, hi - 1):
                n, pk = g.peaks(mh, 2, T)
                want = oracle_peaks_batch(bn, [m[0], m[1]], T)
                assert n == len(want)
                np.testing.assert_array_equal(sort_peaks(pk, bn.cells), want)


def test_peak_capacity_overflow_and_threshold_monotonicity():
    wl = WORKLOADS[1]
    bn = wl.binning
    batch = generate_batch(wl, n_events=2)
    want_m = _oracle_batch(bn, batch)
    want = oracle_peaks_batch(bn, want_m, 4)
    with GpuHough(bn, 2, batch.n_hits) as g:
        mh = g.fill(batch)
        n, pk = g.peaks(mh, 2, 4, capacity=7)
        assert n == len(want) > 7 and len(pk) == 7
        full = set(map(tuple, want.tolist()))
        assert all(tuple(r) in full for r in pk.tolist()) and len(set(map(tuple, pk.tolist()))) == 7
        n0, pk0 = g.peaks(mh, 2, 4, capacity=0)
        assert n0 == len(want)
        n4, pk4 = g.peaks(mh, 2, 4)
        n5, pk5 = g.peaks(mh, 2, 5)
        s4 = sort_peaks(pk4, bn.cells)
        np.testing.assert_array_equal(sort_peaks(pk5, bn.cells), s4[s4["count"] >= 5])
        # repeated calls give the same answer (the scratch counters reset themselves)
        n4b, _ = g.peaks(mh, 2, 4)
        assert n4b == n4 == len(want)


def test_fused_kernel_list_truncation():
    """ht_fill_peaks with a list that is too short: the count is the total, the records written are a duplicate-free
    subset of the oracle's set; capacity 0 writes nothing; capacity == n is the whole set."""
    wl = WORKLOADS[1]
    bn = wl.binning
    batch = generate_batch(wl, n_events=3)
    want = oracle_peaks_batch(bn, _oracle_batch(bn, batch), 4)
    full = set(map(tuple, want.tolist()))
    assert len(want) > 7
    with GpuHough(bn, 3, batch.n_hits) as g:
        for store in (True, False):
            _, n, pk = g.fill_peaks(batch, 4, capacity=7, store=store)
            assert n == len(want) and len(pk) == 7
            got = list(map(tuple, pk.tolist()))
            assert all(r in full for r in got) and len(set(got)) == 7
            _, n0, pk0 = g.fill_peaks(batch, 4, capacity=0, store=store)
            assert n0 == len(want) and len(pk0) == 0
            _, n1, pk1 = g.fill_peaks(batch, 4, capacity=len(want), store=store)
            assert n1 == len(want)
            np.testing.assert_array_equal(sort_peaks(pk1, bn.cells), want)
            _, n2, pk2 = g.fill_peaks(batch, 4, capacity=len(want) - 1, store=store)
            got2 = set(map(tuple, pk2.tolist()))
            assert n2 == len(want) and len(got2) == len(want) - 1 and got2 <= full


@pytest.mark.parametrize("tuning", [None, {"fill_batch_classification": 1}, {"cooperative_launch": 1}, {"fill_store_warps": 2},
                                    {"fill_early_cap": -1}, {"stable_inputs": 1}, {"fill_early_cap": 8, "stable_inputs": 1}])
def test_repeated_launches_give_the_same_bits(tuning):
    """No timing-dependent result: 3000 back-to-back fused launches per variant (hand-rolled grid barrier, named-barrier
    pipeline, TMA proxy fence, dependent launches overlapping their predecessor's tail), matrix and peak set compared on
    the device after every launch against a reference that is itself checked against the oracle."""
    wl = WORKLOADS[2]
    bn = Binning(4, 16, 256, 256)
    batch = generate_batch(wl, n_events=1)
    want_m = _oracle_batch(bn, batch)[0]
    want_p = oracle_peaks(bn, want_m, wl.threshold)
    cap = 1 << 13
    with GpuHough(bn, 1, batch.n_hits, tuning=tuning) as g:
        dx, dy, dz, doff = g.upload(batch)
        ref_m = torch.from_numpy(want_m.reshape(-1).view(np.int32)).to(g.dev)
        ref_cells = torch.from_numpy(want_p["cell"].astype(np.int64)).to(g.dev)
        ref_counts = torch.from_numpy(want_p["count"].astype(np.int64)).to(g.dev)
        mhs = [torch.empty(bn.cells, dtype=torch.int32, device=g.dev) for _ in range(2)]
        outs = [torch.zeros(3 * cap, dtype=torch.int32, device=g.dev) for _ in range(2)]
        nfs = [torch.zeros(1, dtype=torch.int32, device=g.dev) for _ in range(2)]
        bad = torch.zeros(1, dtype=torch.int64, device=g.dev)
        n = len(want_p)
        for it in range(3000):
            k = it & 1
            B.ht_fill_peaks(g.ctx, dx, dy, dz, doff, 1, batch.n_hits, mhs[k], wl.threshold, outs[k], cap, nfs[k], None)
            if it >= 1:                                             # check the PREVIOUS launch while this one runs behind it
                j = k ^ 1
                rec = outs[j][:3 * n].view(n, 3).to(torch.int64)
                order = torch.argsort(rec[:, 1])
                ok = (torch.equal(mhs[j], ref_m) & torch.equal(rec[order, 1], ref_cells) &
                      torch.equal(rec[order, 2], ref_counts) & (int(nfs[j].item()) == n))
                if not ok:
                    bad += 1
        torch.cuda.synchronize()
        assert int(bad.item()) == 0


# ------------------------------------------------------------------ streams, repeated calls, host entry point
def test_fill_on_a_side_stream_and_buffer_reuse():
    wl = WORKLOADS[1]
    bn = wl.binning
    b0, b1 = generate_batch(wl, n_events=1), generate_batch(wl, n_events=1, first_event=1)
    st = torch.cuda.Stream()
    with GpuHough(bn, 1, max(b0.n_hits, b1.n_hits)) as g:
        m0 = mh_to_numpy(g.fill(b0, stream=st), bn, 1)[0]
        m1 = mh_to_numpy(g.fill(b1, stream=st), bn, 1)[0]
        np.testing.assert_array_equal(m0, oracle_fill(bn, *b0.event(0))[0])
        np.testing.assert_array_equal(m1, oracle_fill(bn, *b1.event(0))[0])


def test_run_host_end_to_end():
    wl = WORKLOADS[1]
    bn = wl.binning
    batch = generate_batch(wl, n_events=5)
    want_m = _oracle_batch(bn, batch)
    want = oracle_peaks_batch(bn, want_m, wl.threshold)
    with GpuHough(bn, 5, batch.n_hits, host_slots=2, host_peak_capacity=4096) as g:     # 5 events through 2 slots
        out = np.zeros(4096, B.PEAK_DTYPE)
        h_mh = np.full(5 * bn.cells, 0xFFFFFFFF, np.uint32)
        n = B.ht_run_host(g.ctx, batch.x, batch.y, batch.z, batch.event_offsets, 5, batch.n_hits, wl.threshold, out, 4096, h_mh)
        assert n == len(want)
        np.testing.assert_array_equal(sort_peaks(out[:n], bn.cells), want)
        for e in range(5):
            np.testing.assert_array_equal(h_mh[e * bn.cells:(e + 1) * bn.cells].reshape(want_m[e].shape), want_m[e])
        # truncated list
        out2 = np.zeros(3, B.PEAK_DTYPE)
        n2 = B.ht_run_host(g.ctx, batch.x, batch.y, batch.z, batch.event_offsets, 5, batch.n_hits, wl.threshold, out2, 3)
        assert n2 == n
        assert B.ht_kernel_launches(g.ctx) >= 2 * 3            # 2 calls x 3 groups of <= 2 events, one fused kernel each


def test_submit_wait_host_pipeline():
    """ht_submit_host / ht_wait_host: events in flight in several slots, waited for out of submission order, slots
    reused, misuse refused; every event's peak list against the oracle."""
    wl = WORKLOADS[2]
    bn = Binning(4, 16, 256, 256)
    events = [generate_batch(wl, n_events=1, first_event=e) for e in range(7)]
    wants = [oracle_peaks(bn, oracle_fill(bn, *b.event(0))[0], wl.threshold) for b in events]
    for tuning in (None, {"host_copy_input": 1}, {"host_copy_input": 2}, {"host_direct_results": 1}):
        with GpuHough(bn, 1, 6000, host_slots=3, host_peak_capacity=4096, tuning=tuning) as g:
            out = np.zeros(4096, B.PEAK_DTYPE)
            in_flight = {}
            order = []
            for k, b in enumerate(events):
                slot = k % 3
                if slot in in_flight:
                    kk = in_flight.pop(slot)
                    n = B.ht_wait_host(g.ctx, slot, out, 4096)
                    assert n == len(wants[kk])
                    np.testing.assert_array_equal(sort_peaks(out[:n], bn.cells), wants[kk])
                    order.append(kk)
                B.ht_submit_host(g.ctx, slot, b.x, b.y, b.z, b.n_hits, wl.threshold)
                in_flight[slot] = k
                with pytest.raises(B.HtError):                       # the slot is busy
                    B.ht_submit_host(g.ctx, slot, b.x, b.y, b.z, b.n_hits, wl.threshold)
            with pytest.raises(B.HtError):                           # events in flight: the synchronous call is refused
                B.ht_run_host(g.ctx, events[0].x, events[0].y, events[0].z, events[0].event_offsets, 1, events[0].n_hits,
                              wl.threshold, out, 4096)
            for slot in sorted(in_flight, reverse=True):             # not the submission order
                kk = in_flight[slot]
                n = B.ht_wait_host(g.ctx, slot, out, 4096)
                assert n == len(wants[kk])
                np.testing.assert_array_equal(sort_peaks(out[:n], bn.cells), wants[kk])
                order.append(kk)
            assert sorted(order) == list(range(7))
            with pytest.raises(B.HtError):                           # nothing submitted
                B.ht_wait_host(g.ctx, 0, out, 4096)
            # truncated read-back: the count is the total, the records a subset
            B.ht_submit_host(g.ctx, 1, events[2].x, events[2].y, events[2].z, events[2].n_hits, wl.threshold)
            small = np.zeros(5, B.PEAK_DTYPE)
            n = B.ht_wait_host(g.ctx, 1, small, 5)
            full = set(map(tuple, wants[2].tolist()))
            assert n == len(wants[2]) and all(tuple(r) in full for r in small.tolist())
            # a device-pointer call on another stream right after the host calls (ordered by the library)
            m = g.fill(events[3])
            np.testing.assert_array_equal(mh_to_numpy(m, bn, 1)[0], oracle_fill(bn, *events[3].event(0))[0])


def test_error_codes_on_device_calls():
    bn = WORKLOADS[1].binning
    batch = generate_batch(1)
    with GpuHough(bn, 1, 100) as g:                      # max_hits 100 < 264
        with pytest.raises(B.HtError) as ei:
            g.fill(batch)
        assert ei.value.status == B.HT_ERR_INVALID_ARG
    with GpuHough(bn, 1, 1000) as g:
        mh = g.fill(batch)
        nf = torch.zeros(1, dtype=torch.int32, device="cuda")
        with pytest.raises(B.HtError):
            B.ht_peaks(g.ctx, mh, 1, 0, None, 0, nf)     # threshold 0
        with pytest.raises(B.HtError):
            B.ht_peaks(g.ctx, mh, 2, 1, None, 0, nf)     # n_events > max_events
        with pytest.raises(B.HtError) as ei:
            B.ht_run_host(g.ctx, batch.x, batch.y, batch.z, batch.event_offsets, 1, batch.n_hits, 8, None, 0)
        assert ei.value.status == B.HT_ERR_UNSUPPORTED   # host_slots == 0
    cfg = B.ht_config.from_binning(bn, max_events=1, max_hits=1, device=99)
    with pytest.raises(B.HtError):
        B.ht_create(cfg)


# ------------------------------------------------------------------ every code path of the fill kernel
@pytest.mark.parametrize("tuning", [{"fill_batch_classification": 1},   # batch classification (global buckets) on single events too
                                    {"fill_slab_kb": 8},                 # many small tiles, rows shared by few warps
                                    {"fill_plain_stores": 1},            # plain stores instead of the TMA
                                    {"fill_batch_classification": 1, "fill_slab_kb": 8},
                                    {"cooperative_launch": 1},           # cudaLaunchCooperativeKernel instead of the dependent launch
                                    {"fill_store_warps": 1}, {"fill_store_warps": 2},      # one queue of tile stores / a store warp per slab
                                    {"fill_store_warps": 2, "fill_slab_kb": 8, "fill_batch_classification": 1},
                                    {"fill_early_cap": -1},              # no early tiles: every tile from the grid's buckets
                                    {"fill_early_cap": 8},               # early list too small for most planes: falls back per CTA
                                    {"fill_early_cap": 8, "fill_store_warps": 2, "fill_slab_kb": 8},
                                    {"stable_inputs": 1},                # ht_promise_stable_inputs: hits read before the previous kernel completes
                                    {"stable_inputs": 1, "fill_early_cap": -1}, {"stable_inputs": 1, "fill_slab_kb": 8},
                                    {"peaks_unroll": 4}, {"peaks_unroll": 8, "peaks_ctas_per_sm": 2}])
def test_fill_kernel_variants_are_bit_exact(tuning):
    """The switches of ht_tuning (read once by ht_create_ex) change how the work is organised, never the result."""
    wl = WORKLOADS[2]
    bn = Binning(4, 16, 256, 512)                                   # 33.5 M cells: the oracle takes a fraction of a second
    one = generate_batch(wl, n_events=1)
    assert _check_batch(bn, one, wl.threshold, tuning=tuning) > 0
    three = generate_batch(WORKLOADS[3], n_events=3)
    assert _check_batch(bn, three, wl.threshold, tuning=tuning, own_workspace=True) > 0


def test_hits_on_the_edges_of_the_angle_bins():
    """Early tiles decide "is this hit in my plane" by comparing q and p with the plane's two table entries instead of
    bisecting the tables (and a coarse test with approximate reciprocals decides which hits get that far): hits whose q
    or p IS a table entry, or one ulp beside it, on every edge of both tables, with and without early tiles."""
    bn = Binning(4, 16, 128, 256)
    cfg = B.ht_config.from_binning(bn, max_events=1, max_hits=1, device=0)
    _, tth, pph, _, _ = B.ht_tables_host(cfg)
    xs, ys, zs = [], [], []
    f32 = np.float32
    ulps = lambda v: [np.nextafter(f32(v), f32(-np.inf)), f32(v), np.nextafter(f32(v), f32(np.inf))]
    # q = z / sqrt(x^2 + y^2): with r = 64 (a power of two, r^2 exact) q = z / 64 is exact, so z = 64 * T[k] puts q on T[k]
    for k, t in enumerate(tth):
        if not np.isfinite(t):
            continue
        for q in ulps(t):
            for phi in (0.3, 2.0, 4.1, 5.5):
                x, y = f32(64.0 * math.cos(phi)), f32(64.0 * math.sin(phi))
                r = math.sqrt(float(x) ** 2 + float(y) ** 2)
                xs.append(x); ys.append(y); zs.append(f32(float(q) * r))
    # p = 1 - x / (|x| + |y|) (y >= 0) or 3 + x / (|x| + |y|): x = d * (1 - P[k]) with d = |x| + |y| = 64
    for k, pe in enumerate(pph):
        for pv in ulps(pe):
            pv = float(pv)
            u = 1.0 - pv if pv <= 2.0 else pv - 3.0                  # x / d
            if abs(u) > 1.0:
                continue
            x = f32(64.0 * u)
            y = f32((64.0 - abs(float(x))) * (1.0 if pv <= 2.0 else -1.0))
            for z in (-50.0, 3.0, 80.0):
                xs.append(x); ys.append(y); zs.append(f32(z))
    rng = np.random.default_rng(5)
    reps = 6                                                            # several votes per cell, so that peaks exist
    x = np.tile(np.asarray(xs, f32), reps); y = np.tile(np.asarray(ys, f32), reps); z = np.tile(np.asarray(zs, f32), reps)
    perm = rng.permutation(len(x))
    batch = batch_from_arrays([np.stack([x[perm], y[perm], z[perm]], axis=1)])
    for tuning in (None, {"fill_early_cap": -1}, {"stable_inputs": 1}):
        assert _check_batch(bn, batch, 3, tuning=tuning) >= 0


def test_caller_owned_workspace_and_bad_tuning():
    """ht_query_sizes -> caller allocates -> ht_create_ex: same results; a workspace that is too small or misaligned and
    a tuning block with unknown fields set are refused."""
    wl = WORKLOADS[1]
    bn = wl.binning
    batch = generate_batch(wl, n_events=2)
    assert _check_batch(bn, batch, wl.threshold, own_workspace=True) > 0
    cfg = B.ht_config.from_binning(bn, max_events=2, max_hits=batch.n_hits, device=0)
    nbytes = B.ht_query_sizes(cfg)[1]
    ws = torch.empty(nbytes + 512, dtype=torch.uint8, device="cuda")
    base = (ws.data_ptr() + 255) // 256 * 256
    for args in ((base, nbytes - 1), (base + 4, nbytes)):
        with pytest.raises(B.HtError) as ei:
            B.ht_create_ex(cfg, None, *args)
        assert ei.value.status == B.HT_ERR_INVALID_ARG
    bad = B.ht_tuning()
    bad.reserved[3] = 1
    with pytest.raises(B.HtError):
        B.ht_create_ex(cfg, bad)
    with pytest.raises(B.HtError):
        B.ht_create_ex(cfg, B.ht_tuning(peaks_unroll=3))


def test_dense_tiles_with_many_peak_candidates():
    """More candidates per tile than the store warp takes (32) and than a candidate list holds (128): the voters test
    them, or scan the tile."""
    wl = WORKLOADS[4]
    bn = Binning(2, 2, 192, 256)                                    # 20000 hits in 4 planes: every tile is dense
    batch = generate_batch(wl, n_events=1)
    assert _check_batch(bn, batch, 3) > 1000
    assert _check_batch(bn, generate_batch(wl, n_events=2), 40) > 0


def test_division_shortcut_equals_fdiv_rn_on_four_billion_pairs():
    """The vote loop divides with a hoisted reciprocal; on every pair it is used on it must give the
    bits of the IEEE quotient.  4e9 pseudo-random pairs, exponents across and beyond the moderate range."""
    assert B.ht_selftest_division(0, 4_000_000_000, 12345) == 0
    assert B.ht_selftest_division(0, 100_000_000, 987654321) == 0


@pytest.mark.parametrize("copy_input", [0, 1, 2])
def test_run_host_single_event_zero_copy_and_copy(copy_input):
    """One event through ht_run_host: the kernel reads the hits straight from the pinned block (default) or the block is
    copied to the device first; same matrix, same peaks, several calls in a row on one context."""
    wl = WORKLOADS[2]
    bn = Binning(4, 16, 256, 256)
    with GpuHough(bn, 1, 6000, host_slots=1, host_peak_capacity=8192, tuning={"host_copy_input": copy_input}) as g:
        for ev in range(3):
            batch = generate_batch(wl, n_events=1, first_event=ev)
            want_m = _oracle_batch(bn, batch)
            want = oracle_peaks_batch(bn, want_m, wl.threshold)
            out = np.zeros(8192, B.PEAK_DTYPE)
            h_mh = np.full(bn.cells, 0xFFFFFFFF, np.uint32)
            n = B.ht_run_host(g.ctx, batch.x, batch.y, batch.z, batch.event_offsets, 1, batch.n_hits, wl.threshold, out,
                              8192, h_mh)
            assert n == len(want) and n > 0
            np.testing.assert_array_equal(sort_peaks(out[:n], bn.cells), want)
            np.testing.assert_array_equal(h_mh.reshape(want_m[0].shape), want_m[0])


def test_run_host_events_pipelines_a_sequence():
    """ht_run_host_events: a sequence of ragged events (an empty one among them) from host memory, one fused kernel each,
    pipelined over 1, 2 and 3 slots, with and without zero-copy input: every event's peak list equals the oracle's; lists
    longer than capacity_per_event are truncated, their counts are not."""
    wl = WORKLOADS[2]
    bn = Binning(4, 16, 256, 256)
    evs = []
    for e in range(7):
        b = generate_batch(WORKLOADS[3], n_events=1, first_event=e)
        evs.append(np.stack(b.event(0), -1)[: 1200 + 300 * e])
    evs.insert(3, np.zeros((0, 3), np.float32))
    batch = batch_from_arrays(evs)
    wants = [oracle_peaks(bn, oracle_fill(bn, *batch.event(e))[0], wl.threshold) for e in range(batch.n_events)]
    assert max(len(w) for w in wants) > 20 and len(wants[3]) == 0
    for slots, tuning in ((1, None), (2, {"host_copy_input": 1}), (3, {"host_copy_input": 2}), (3, {"fill_early_cap": -1}),
                          (2, {"host_direct_results": 1})):
        with GpuHough(bn, 1, 4000, host_slots=slots, host_peak_capacity=4096, tuning=tuning) as g:
            for cap_ev in (4096, 16):
                out = np.zeros(batch.n_events * cap_ev, B.PEAK_DTYPE)
                nf = np.zeros(batch.n_events, np.uint32)
                B.ht_run_host_events(g.ctx, batch.x, batch.y, batch.z, batch.event_offsets, batch.n_events, wl.threshold,
                                     out, cap_ev, nf)
                for e, want in enumerate(wants):
                    assert nf[e] == len(want), (slots, e)
                    got = out[e * cap_ev: e * cap_ev + min(len(want), cap_ev)]
                    assert np.all(got["event"] == e)
                    if len(want) <= cap_ev:
                        got = got[np.argsort(got["cell"])]
                        np.testing.assert_array_equal(got["cell"], want["cell"])
                        np.testing.assert_array_equal(got["count"], want["count"])
                    else:
                        keys = dict(zip(want["cell"].tolist(), want["count"].tolist()))
                        assert len(set(got["cell"].tolist())) == cap_ev
                        assert all(keys.get(int(c)) == int(n) for c, n in zip(got["cell"], got["count"]))
            # an event beyond the context's capacity is refused before anything is launched
            with pytest.raises(B.HtError):
                big = batch_from_arrays([np.ones((4001, 3), np.float32)])
                B.ht_run_host_events(g.ctx, big.x, big.y, big.z, big.event_offsets, 1, wl.threshold, out, 16, nf)


@pytest.mark.parametrize("direct", [0, 1])
def test_host_event_with_more_peaks_than_the_copy_engine_brings_along(direct):
    """Results through the copy engine: the copy stream brings the header and the first 4096 records to the host; a longer
    list's tail is fetched from the slot's device block by ht_wait_host.  A dense event with well over 4096 peaks, read
    back whole, then truncated at capacities on both sides of 4096; the direct route (the kernel stores into pinned
    memory) must give the same lists."""
    bn = Binning(4, 16, 256, 512)
    thr = 10
    batch = generate_batch(WORKLOADS[4], n_events=1)
    want = oracle_peaks(bn, oracle_fill(bn, *batch.event(0))[0], thr)
    assert 6000 < len(want) < 30000
    cap = 1 << 15
    with GpuHough(bn, 1, batch.n_hits, host_slots=2, host_peak_capacity=cap, tuning={"host_direct_results": direct}) as g:
        for rep in range(2):                                          # (the second time the slot's blocks hold the first result)
            out = np.zeros(cap, B.PEAK_DTYPE)
            B.ht_submit_host(g.ctx, rep, batch.x, batch.y, batch.z, batch.n_hits, thr)
            n = B.ht_wait_host(g.ctx, rep, out, cap)
            assert n == len(want)
            np.testing.assert_array_equal(sort_peaks(out[:n], bn.cells), want)
        full = set(map(tuple, want.tolist()))
        for part in (4095, 4096, 4097, 5000):
            out = np.zeros(part, B.PEAK_DTYPE)
            B.ht_submit_host(g.ctx, 0, batch.x, batch.y, batch.z, batch.n_hits, thr)
            n = B.ht_wait_host(g.ctx, 0, out, part)
            got = set(map(tuple, out.tolist()))
            assert n == len(want) and len(got) == part and got <= full
        # the pipelined form on the same event, twice in a row
        out = np.zeros(2 * cap, B.PEAK_DTYPE)
        nf = np.zeros(2, np.uint32)
        two = batch_from_arrays([np.stack(batch.event(0), -1)] * 2)
        B.ht_run_host_events(g.ctx, two.x, two.y, two.z, two.event_offsets, 2, thr, out, cap, nf)
        for e in range(2):
            assert nf[e] == len(want)
            got = out[e * cap: e * cap + len(want)]
            assert np.all(got["event"] == e)
            got = got[np.argsort(got["cell"])]
            assert np.array_equal(got["cell"], want["cell"]) and np.array_equal(got["count"], want["count"])


@pytest.mark.parametrize("copy_input,direct", [(1, 0), (2, 0), (1, 1)])
def test_host_pipeline_three_thousand_events(copy_input, direct):
    """The host path's hand-rolled synchronisation under load: the kernel waits for a word the copy stream writes behind
    the hits; its results reach the host through a copy stream that waits for the kernel's completion word, or (direct)
    the kernel writes them straight into pinned host memory, where ONE system-wide fence (the last CTA's) stands between
    the records of all CTAs and the completion word the host polls.  3000 events through 4 slots; twelve distinct
    events in turn, so that a slot never holds the same event twice running and a stale record or count cannot pass."""
    bn = Binning(4, 16, 128, 128)
    thr = 4
    evs = []
    for e in range(12):
        b = generate_batch(WORKLOADS[3], n_events=1, first_event=e)
        evs.append(np.stack(b.event(0), -1)[: 1500 + 100 * e])
    wants = []
    for ev in evs:
        one = batch_from_arrays([ev])
        wants.append(oracle_peaks(bn, oracle_fill(bn, *one.event(0))[0], thr))
    assert min(len(w) for w in wants) > 50 and len({len(w) for w in wants}) > 6
    n_rep = 250
    batch = batch_from_arrays(evs * n_rep)
    cap_ev = max(len(w) for w in wants)
    with GpuHough(bn, 1, 3000, host_slots=4, host_peak_capacity=cap_ev,
                  tuning={"host_copy_input": copy_input, "host_direct_results": direct}) as g:
        out = np.zeros(batch.n_events * cap_ev, B.PEAK_DTYPE)
        nf = np.zeros(batch.n_events, np.uint32)
        B.ht_run_host_events(g.ctx, batch.x, batch.y, batch.z, batch.event_offsets, batch.n_events, thr, out, cap_ev, nf)
    for e in range(batch.n_events):
        want = wants[e % 12]
        assert nf[e] == len(want), e
        got = out[e * cap_ev: e * cap_ev + len(want)]
        got = got[np.argsort(got["cell"])]
        assert np.all(got["event"] == e)
        assert np.array_equal(got["cell"], want["cell"]) and np.array_equal(got["count"], want["count"]), e


# ------------------------------------------------------------------ f3: track read-out of the peaks
def _tracks_gpu(g, pk):
    dev = g.dev
    rec = np.zeros((len(pk), 3), np.uint32)
    rec[:, 0], rec[:, 1], rec[:, 2] = pk["event"], pk["cell"], pk["count"]
    d_pk = torch.from_numpy(rec.view(np.int32)).to(dev)
    d_out = torch.zeros(max(len(pk), 1) * 5, dtype=torch.int32, device=dev)
    B.ht_tracks(g.ctx, d_pk, len(pk), d_out, None)
    torch.cuda.synchronize()
    return d_out[:5 * len(pk)].cpu().numpy().view(np.uint8).view(B.TRACK_DTYPE)


def test_tracks_match_the_oracle_within_binary32_rounding():
    """rho: products, sum and square root are each rounded once in binary32 (<= 2 ulp overall: rtol 2.4e-7); phi:
    CUDA's atan2f is within 2 ulp, and |phi| < 4 has ulp 2.4e-7 (atol 6e-7).  DESIGN.md section 5.4."""
    from oracle import oracle_tracks
    wl = WORKLOADS[2]
    bn = Binning(4, 16, 256, 512)
    batch = generate_batch(wl, n_events=2)
    want_m = _oracle_batch(bn, batch)
    pk = oracle_peaks_batch(bn, want_m, wl.threshold)
    assert len(pk) > 100
    with GpuHough(bn, 2, batch.n_hits) as g:
        # the peak list as the fused kernel writes it (its own order), read out on the device
        _, n, got_pk = g.fill_peaks(batch, wl.threshold, store=False)
        assert n == len(pk)
        tr = _tracks_gpu(g, got_pk)
        for f in ("event", "cell", "count"):
            np.testing.assert_array_equal(tr[f], got_pk[f])
        rho, phi = oracle_tracks(bn, got_pk)
        np.testing.assert_allclose(tr["rho"].astype(np.float64), rho, rtol=2.4e-7, atol=0)
        np.testing.assert_allclose(tr["phi"].astype(np.float64), phi, rtol=0, atol=6e-7)
        assert len(_tracks_gpu(g, got_pk[:0])) == 0            # empty list: no launch, no error


def test_tracks_every_cell_of_a_small_odd_binning():
    """All cells, including the one at the origin (rho = 0, phi = 0), the axes and the four quadrants."""
    from oracle import oracle_tracks
    bn = Binning(2, 3, 9, 7, a_min=-9.0, a_max=9.0, b_min=-7.0, b_max=7.0)
    pk = np.zeros(bn.cells, B.PEAK_DTYPE)
    pk["cell"] = np.arange(bn.cells)
    pk["count"] = 1
    with GpuHough(bn, 1, 1) as g:
        tr = _tracks_gpu(g, pk)
    rho, phi = oracle_tracks(bn, pk)
    np.testing.assert_allclose(tr["rho"].astype(np.float64), rho, rtol=2.4e-7, atol=0)
    np.testing.assert_allclose(tr["phi"].astype(np.float64), phi, rtol=0, atol=6e-7)
    origin = (4 * 7 + 3)
    assert tr["rho"][origin] == 0.0 and tr["phi"][origin] == 0.0


# ------------------------------------------------------------------ f3: ridge merging and truth matching
def _merge_gpu(g, pk, window, capacity=None):
    dev = g.dev
    n = len(pk)
    rec = np.zeros((n, 3), np.uint32)
    rec[:, 0], rec[:, 1], rec[:, 2] = pk["event"], pk["cell"], pk["count"]
    d_pk = torch.from_numpy(rec.view(np.int32)).to(dev)
    cap = n if capacity is None else capacity
    d_out = torch.zeros(max(cap, 1) * 6, dtype=torch.int32, device=dev)
    d_n = torch.full((1,), -5, dtype=torch.int32, device=dev)
    nb = B.ht_merge_scratch_bytes(n)
    d_scr = torch.empty(nb, dtype=torch.uint8, device=dev)
    B.ht_merge_ridges(g.ctx, d_pk, n, window, d_out if cap else None, cap, d_n, d_scr, nb, None)
    torch.cuda.synchronize()
    found = int(d_n.cpu().numpy().view(np.uint32)[0])
    k = min(found, cap)
    out = d_out[:6 * k].cpu().numpy().view(np.uint8).view(B.CAND_DTYPE).copy()
    return found, out[np.lexsort((out["cell"], out["event"]))], d_out


def _check_merge(g, bn, pk, window):
    from oracle import oracle_merge_ridges
    want = oracle_merge_ridges(bn, pk, window)
    found, got, _ = _merge_gpu(g, pk, window)
    assert found == len(want)
    for f in ("event", "cell", "count", "n_peaks"):
        np.testing.assert_array_equal(got[f], want[f], err_msg=f)
    np.testing.assert_allclose(got["rho"].astype(np.float64), want["rho"], rtol=2.4e-7, atol=0)
    np.testing.assert_allclose(got["phi"].astype(np.float64), want["phi"], rtol=0, atol=6e-7)
    return len(want)


def test_ridge_merging_matches_the_oracle():
    """Set-exact on (event, cell, count, members); rho, phi within the read-out's tolerance.  Peak lists of the tiny and of
    the paper-shaped workload (in the fused kernel's own order), every window from 0 to 12, dense random lists with ties
    and duplicate records, an empty list, and truncation of the candidate list."""
    rng = np.random.default_rng(5)
    for cfg_id, bn in ((1, WORKLOADS[1].binning), (2, Binning(4, 16, 256, 512))):
        wl = WORKLOADS[cfg_id]
        batch = generate_batch(wl, n_events=3)
        with GpuHough(bn, 3, batch.n_hits) as g:
            _, n, pk = g.fill_peaks(batch, wl.threshold, store=False)
            assert n == len(pk) > 10
            sizes = [_check_merge(g, bn, pk, w) for w in (0, 1, 2, 3, 5, 8, 12)]
            assert sizes[0] == len(pk) and sizes == sorted(sizes, reverse=True) and sizes[-1] < sizes[0]
            # truncation: the count is total, the written records are candidates of the full answer
            found, part, _ = _merge_gpu(g, pk, 3, capacity=5)
            from oracle import oracle_merge_ridges
            full = oracle_merge_ridges(bn, pk, 3)
            assert found == len(full) and len(part) == 5
            keys = set(zip(full["event"].tolist(), full["cell"].tolist()))
            assert all((int(e), int(c)) in keys for e, c in zip(part["event"], part["cell"]))
            assert _merge_gpu(g, pk[:0], 3)[0] == 0
    bn = Binning(2, 3, 40, 50)
    with GpuHough(bn, 4, 1) as g:
        for trial in range(6):
            n = int(rng.integers(100, 1500))
            keys = rng.choice(4 * bn.cells, size=n, replace=False)
            pk = np.zeros(n, B.PEAK_DTYPE)
            pk["event"], pk["cell"], pk["count"] = keys // bn.cells, keys % bn.cells, rng.integers(8, 11, n)
            if trial % 2:
                pk = np.concatenate([pk, pk[: n // 10]])            # duplicate records are linked at any window
            for w in (0, 1, 4):
                _check_merge(g, bn, pk, w)
    # large groups: more than 192 peaks of one plane are sorted by cell first (the sweeps then look at nearby rows only),
    # more than 2048 work on global memory; long ridges, dense blobs, duplicates, every window from 0 to "everything"
    bn = Binning(1, 2, 200, 300)
    with GpuHough(bn, 2, 1) as g:
        for trial, n in enumerate((700, 3000, 3900, 9000)):
            keys = rng.choice(2 * bn.cells, size=n, replace=False)
            pk = np.zeros(n, B.PEAK_DTYPE)
            pk["event"], pk["cell"], pk["count"] = keys // bn.cells, keys % bn.cells, rng.integers(8, 11, n)
            if trial % 2:
                pk = np.concatenate([pk, pk[: n // 7]])
            for w in (0, 1, 2, 5):
                _check_merge(g, bn, pk, w)
        # one diagonal ridge per plane (a chain of 190 links) plus noise: hooking has to carry a label along the whole chain
        ridge = np.zeros(2 * 190 + 400, B.PEAK_DTYPE)
        for p_ in range(2):
            a = np.arange(190) + 5
            ridge["cell"][p_ * 190:(p_ + 1) * 190] = (p_ * bn.n_a + a) * bn.n_b + (a + 20 + 3 * p_)
        ridge["cell"][380:] = rng.choice(bn.cells, size=400, replace=False)
        ridge["count"] = rng.integers(8, 40, len(ridge))
        ridge = ridge[rng.permutation(len(ridge))]
        for w in (1, 2, 3):
            _check_merge(g, bn, ridge, w)
    # the peaks of the 20000-hit event (about 200 per plane, a thousand in the densest)
    wl = WORKLOADS[4]
    with GpuHough(wl.binning, 1, 20000) as g:
        _, n, pk = g.fill_peaks(generate_batch(wl, n_events=1), wl.threshold, store=False)
        assert n == len(pk) > 10000
        assert _check_merge(g, wl.binning, pk, 3) > _check_merge(g, wl.binning, pk, 10) > 500


def test_truth_matching_matches_the_oracle():
    """cand_match, truth_match and the integer part of the summary exactly (binary64 decisions by the same operations on both
    sides), the residual sums within 1e-9 relative; on the paper-shaped event with the generator's truth and on random lists."""
    from oracle import MERGED_DTYPE, TRUTH_DTYPE, oracle_match_truth, oracle_merge_ridges
    from paper_1507_03074_b200.events import truth_table
    import math

    def run(g, bn, cand_gpu_tensor, n_cand, cand_oracle, tr, w_rho, w_phi):
        dev = g.dev
        d_tr = torch.from_numpy(tr.view(np.uint8).copy()).to(dev)
        d_cm = torch.full((max(n_cand, 1),), -9, dtype=torch.int32, device=dev)
        d_tm = torch.full((max(len(tr), 1),), -9, dtype=torch.int32, device=dev)
        d_sum = torch.zeros(B.SUMMARY_DTYPE.itemsize, dtype=torch.uint8, device=dev)
        B.ht_match_truth(g.ctx, cand_gpu_tensor, n_cand, d_tr, len(tr), w_rho, math.cos(w_phi), d_cm, d_tm, d_sum, None)
        torch.cuda.synchronize()
        cm, tm = d_cm.cpu().numpy()[:n_cand], d_tm.cpu().numpy()[:len(tr)]
        s = d_sum.cpu().numpy().view(B.SUMMARY_DTYPE)[0]
        wcm, wtm, ws = oracle_match_truth(bn, cand_oracle, tr, w_rho, math.cos(w_phi))
        np.testing.assert_array_equal(cm, wcm)
        np.testing.assert_array_equal(tm, wtm)
        for k in ("n_cand", "n_truth", "n_matched", "n_fake", "n_found", "n_duplicate"):
            assert int(s[k]) == ws[k], k
        for k in ("sum_drho", "sum_drho2", "sum_dphi", "sum_dphi2"):
            assert abs(float(s[k]) - ws[k]) <= 1e-9 * max(1.0, abs(ws[k])) + 1e-12, k
        return ws

    wl = WORKLOADS[2]
    bn = Binning(4, 16, 512, 512)
    batch = generate_batch(wl, n_events=2)
    tt = truth_table(batch)
    tr = np.zeros(len(tt["event"]), TRUTH_DTYPE)
    tr["event"], tr["a"], tr["b"] = tt["event"], tt["a"], tt["b"]
    with GpuHough(bn, 2, batch.n_hits) as g:
        _, n, pk = g.fill_peaks(batch, wl.threshold, store=False)
        found, cands, d_cands = _merge_gpu(g, pk, 4)
        # the device list in ITS order against the oracle on the same records in the same order
        dev_order = d_cands[:6 * found].cpu().numpy().view(np.uint8).view(B.CAND_DTYPE)
        co = np.zeros(found, MERGED_DTYPE)
        for f in ("event", "cell", "count", "n_peaks"):
            co[f] = dev_order[f]
        for w_rho, w_phi in ((40.0, 0.02), (100.0, 0.05), (0.0, 0.0), (1e4, 3.0)):
            ws = run(g, bn, d_cands, found, co, tr, w_rho, w_phi)
        assert ws["n_found"] > 0
        run(g, bn, d_cands, 0, co[:0], tr, 40.0, 0.02)
        run(g, bn, d_cands, found, co, tr[:0], 40.0, 0.02)
        # random candidates (cells anywhere) and random circles
        rng = np.random.default_rng(11)
        for trial in range(4):
            nc, nt = int(rng.integers(50, 800)), int(rng.integers(10, 300))
            rc = np.zeros(nc, B.CAND_DTYPE)
            rc["event"], rc["cell"] = rng.integers(0, 2, nc), rng.integers(0, bn.cells, nc)
            co = np.zeros(nc, MERGED_DTYPE)
            co["event"], co["cell"] = rc["event"], rc["cell"]
            rt = np.zeros(nt, TRUTH_DTYPE)
            rt["event"] = rng.integers(0, 2, nt)
            rt["a"], rt["b"] = rng.uniform(-4000, 4000, nt), rng.uniform(-4000, 4000, nt)
            d_rc = torch.from_numpy(rc.view(np.uint8).copy()).to(g.dev)
            run(g, bn, d_rc, nc, co, rt, 150.0, 0.08)


def test_vote_loop_exactness_preconditions():
    """The vote loop decides ONCE per hit whether the three-instruction quotients are exact; hits and
    binnings that fail the test -- B_min = 0 or tiny, tiny and huge coordinates, 2y denormal -- take __fdiv_rn.  Both
    branches must give the oracle's matrix bit for bit."""
    rng = np.random.default_rng(77)
    wl = WORKLOADS[1]
    base = generate_batch(wl, n_events=1)
    x, y, z = (v.copy() for v in base.event(0))
    odd = np.array([[1e-19, 2e-19, 1.0], [3e-20, -1e-19, -1.0], [1e10, 2e10, 1e9], [-3e18, 1e18, 1.0], [40.0, 1e-40, 3.0],
                    [1e-30, 50.0, 1.0], [60.0, -1e-25, 2.0], [0.0, 70.0, 5.0], [1e19, 1e-19, 1.0]], np.float32)
    xyz = np.concatenate([np.stack([x, y, z], -1), odd]).astype(np.float32)
    for bn in (Binning(4, 16, 64, 64, b_min=0.0, b_max=4000.0),                       # B_min = 0: the context fails the test
               Binning(2, 4, 64, 96, b_min=-1e-12, b_max=3000.0),                     # tiny B_min
               Binning(2, 4, 32, 64, a_min=-1e-15, a_max=1e-15, b_min=-1e-15, b_max=2e-15),   # everything tiny
               Binning(1, 2, 48, 64, a_min=-1e19, a_max=1e19, b_min=-2e19, b_max=1e19),       # everything huge
               Binning(4, 16, 128, 128)):
        for scale in (1.0, 1e-17, 1e16):
            ev = (xyz * np.float32(scale)).astype(np.float32) if scale != 1.0 else xyz
            batch = batch_from_arrays([ev, ev[rng.permutation(len(ev))][: len(ev) // 2]])
            _check_batch(bn, batch, 2)
            _check_batch(bn, batch_from_arrays([ev]), 2)


def test_seeded_random_shapes():
    """40 seeded random binnings / batch shapes (ragged tiles, rows shared by several warps, NB % 4 != 0, empty events,
    odd hit counts, partial angle ranges): matrix and peaks against the oracle, through all three call paths.
    (Found: a misaligned table pointer for odd hit counts in the single-event classification.)"""
    rng = np.random.default_rng(20241104)
    for case in range(40):
        n_theta, n_phi = int(rng.integers(1, 6)), int(rng.integers(1, 10))
        n_a = int(rng.choice([1, 2, 3, 7, 31, 64, 100, 257]))
        n_b = int(rng.choice([1, 4, 5, 12, 64, 250, 512, 700]))
        kw = {}
        if rng.random() < 0.3:
            kw = dict(theta_min=0.3, theta_max=2.5, phi_min=0.5, phi_max=5.0)
        if rng.random() < 0.3:
            kw.update(a_min=-1500.0, a_max=2500.0, b_min=-3000.0, b_max=500.0)
        bn = Binning(n_theta, n_phi, n_a, n_b, **kw)
        n_events = int(rng.integers(1, 5))
        events = []
        for e in range(n_events):
            n_hits = int(rng.choice([0, 1, 17, 300, 1500, int(rng.integers(1, 2500)), int(rng.integers(1, 2500))]))
            xyz, _ = (np.zeros((0, 3), np.float32), None) if n_hits == 0 else \
                __import__("paper_1507_03074_b200.events", fromlist=["generate_event"]).generate_event(
                    int(rng.integers(1 << 30)), n_hits=n_hits, noise_frac=0.2)
            events.append(xyz)
        batch = batch_from_arrays(events)
        if batch.n_hits == 0:
            events[0] = np.array([[100.0, 50.0, 10.0]], np.float32)
            batch = batch_from_arrays(events)
        _check_batch(bn, batch, int(rng.integers(1, 7)))


@pytest.mark.parametrize("n_hits", [4999, 8193, 24577])
def test_paper_binning_odd_and_boundary_hit_counts(n_hits):
    """Full paper binning with odd hit counts and the counts at which the single-event classification changes its
    register/scratch path (8192 hits) and gives way to the batch path (24576 hits)."""
    from paper_1507_03074_b200.events import generate_event
    bn = WORKLOADS[2].binning
    xyz, _ = generate_event(777 + n_hits, n_hits=n_hits, noise_frac=0.1)
    batch = batch_from_arrays([xyz])
    want_m = _oracle_batch(bn, batch)
    want_p = oracle_peaks_batch(bn, want_m, 9)
    with GpuHough(bn, 1, batch.n_hits) as g:
        mh, n, pk = g.fill_peaks(batch, 9)
        assert n == len(want_p)
        np.testing.assert_array_equal(sort_peaks(pk, bn.cells), want_p)
        assert torch.equal(mh.cpu(), torch.from_numpy(want_m[0].reshape(-1).view(np.int32)))


# ------------------------------------------------------------------ f2: one event split over contexts by (theta, phi) plane
@pytest.mark.parametrize("world", [2, 3, 4])
def test_plane_ranges_reassemble_the_full_result(world):
    """one matrix per sector.  `world` contexts (one per would-be GPU, here one after the other on one
    device) take contiguous plane ranges; their matrices are the plane slices of the oracle's matrix and their peak lists
    -- full-matrix cell indices -- add up to the oracle's, through ht_fill + ht_peaks and through ht_fill_peaks."""
    from paper_1507_03074_b200.sharding import plane_range
    wl = WORKLOADS[2]
    bn = Binning(3, 5, 200, 256)
    batch = generate_batch(wl, n_events=2)
    want_m = _oracle_batch(bn, batch)
    want_p = oracle_peaks_batch(bn, want_m, wl.threshold)
    dev = torch.device("cuda:0")
    parts_split, parts_fused = [], []
    for rank in range(world):
        p0, pc = plane_range(bn.planes, rank, world)
        cfg = B.ht_config.from_binning(bn, max_events=2, max_hits=batch.n_hits, device=0, plane_begin=p0, plane_count=pc)
        assert B.ht_query_sizes(cfg)[0] == 4 * pc * bn.n_a * bn.n_b
        ctx = B.ht_create(cfg)
        try:
            to = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a)).to(dev, dtype=dt)
            dx, dy, dz, doff = (to(batch.x, torch.float32), to(batch.y, torch.float32), to(batch.z, torch.float32),
                                to(batch.event_offsets, torch.int32))
            cells = cfg.cells
            out = torch.zeros(3 << 14, dtype=torch.int32, device=dev)
            nf = torch.zeros(1, dtype=torch.int32, device=dev)
            for fused in (False, True):
                mh = torch.full((2 * cells,), -1, dtype=torch.int32, device=dev)
                if fused:
                    B.ht_fill_peaks(ctx, dx, dy, dz, doff, 2, batch.n_hits, mh, wl.threshold, out, 1 << 14, nf, None)
                else:
                    B.ht_fill(ctx, dx, dy, dz, doff, 2, batch.n_hits, mh, None)
                    B.ht_peaks(ctx, mh, 2, wl.threshold, out, 1 << 14, nf, None)
                torch.cuda.synchronize()
                got = mh.cpu().numpy().view(np.uint32).reshape(2, pc, bn.n_a, bn.n_b)
                for e in range(2):
                    np.testing.assert_array_equal(got[e], want_m[e].reshape(bn.planes, bn.n_a, bn.n_b)[p0:p0 + pc])
                n = int(nf.cpu().numpy().view(np.uint32)[0])
                rec = out[:3 * n].cpu().numpy().view(np.uint32).reshape(n, 3)
                pk = np.empty(n, B.PEAK_DTYPE)
                pk["event"], pk["cell"], pk["count"] = rec[:, 0], rec[:, 1], rec[:, 2]
                (parts_fused if fused else parts_split).append(pk)
        finally:
            B.ht_destroy(ctx)
    for parts in (parts_split, parts_fused):
        np.testing.assert_array_equal(sort_peaks(np.concatenate(parts), bn.cells), want_p)


def test_calls_replayed_from_a_cuda_graph():
    """The calls keep no host-side state between launches (barriers and counters reset themselves on the device), so a
    captured sequence can be replayed: fill + peaks of two different events, three replays, results checked each time."""
    wl = WORKLOADS[2]
    bn = Binning(4, 16, 256, 256)
    dev = torch.device("cuda:0")
    batches = [generate_batch(wl, n_events=1, first_event=e) for e in range(2)]
    wants = []
    for b in batches:
        m = _oracle_batch(bn, b)
        wants.append((m[0], oracle_peaks_batch(bn, m, wl.threshold)))
    cfg = B.ht_config.from_binning(bn, max_events=1, max_hits=max(b.n_hits for b in batches), device=0)
    ctx = B.ht_create(cfg)
    try:
        to = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a)).to(dev, dtype=dt)
        ins = [(to(b.x, torch.float32), to(b.y, torch.float32), to(b.z, torch.float32), to(b.event_offsets, torch.int32))
               for b in batches]
        mhs = [torch.empty(bn.cells, dtype=torch.int32, device=dev) for _ in batches]
        outs = [torch.zeros(3 << 13, dtype=torch.int32, device=dev) for _ in batches]
        nfs = [torch.zeros(1, dtype=torch.int32, device=dev) for _ in batches]
        st = torch.cuda.Stream()
        def enqueue():
            for k, b in enumerate(batches):
                B.ht_fill_peaks(ctx, *ins[k], 1, b.n_hits, mhs[k], wl.threshold, outs[k], 1 << 13, nfs[k], st)
        with torch.cuda.stream(st):
            enqueue()                                              # warm-up outside the capture
        st.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            enqueue()
        for replay in range(3):
            for k in range(2):
                mhs[k].fill_(-1)
                nfs[k].fill_(-5)
            g.replay()
            torch.cuda.synchronize()
            for k in range(2):
                want_m, want_p = wants[k]
                np.testing.assert_array_equal(mhs[k].cpu().numpy().view(np.uint32), want_m.reshape(-1))
                n = int(nfs[k].cpu().numpy().view(np.uint32)[0])
                assert n == len(want_p)
                rec = outs[k][:3 * n].cpu().numpy().view(np.uint32).reshape(n, 3)
                pk = np.empty(n, B.PEAK_DTYPE)
                pk["event"], pk["cell"], pk["count"] = rec[:, 0], rec[:, 1], rec[:, 2]
                np.testing.assert_array_equal(sort_peaks(pk, bn.cells), want_p)
    finally:
        B.ht_destroy(ctx)

"""N > 1 host logic on CPU: world size 2 and 3 over gloo.

The path shards by event with no data-path collective; what runs between the ranks is only the gather of the peak
lists.  Each rank here stands in for "its GPU" by producing the peak list of its shard with the oracle (tests may call
the oracle); the test is about the sharding module: event ranges, batch slicing, gather, re-basing, ordering.
"""
import os
import socket
import tempfile

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import oracle_fill, oracle_peaks, oracle_peaks_batch
from paper_1507_03074_b200.binding import PEAK_DTYPE
from paper_1507_03074_b200.events import Binning, Workload, generate_batch
from paper_1507_03074_b200.sharding import event_range, gather_peaks, plane_range, rebase_peaks, shard_batch, sort_peaks

BN = Binning(2, 4, 64, 64)
WL = Workload(1, "tiny_sharded", BN, n_events=5, threshold=6, n_tracks=12)


def test_event_ranges_partition_the_batch():
    for n in (0, 1, 2, 5, 7, 100):
        for world in (1, 2, 3, 8):
            spans = [event_range(n, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            assert all(spans[r][1] == spans[r + 1][0] for r in range(world - 1))
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        event_range(4, 2, 2)


def test_shard_batch_slices_hits_and_rebases_offsets():
    batch = generate_batch(WL)
    seen = 0
    for r in range(3):
        sub, e0 = shard_batch(batch, r, 3)
        assert sub.event_offsets[0] == 0 and sub.event_offsets[-1] == sub.n_hits
        for k in range(sub.n_events):
            for got, want in zip(sub.event(k), batch.event(e0 + k)):
                assert np.array_equal(got, want)
        seen += sub.n_events
    assert seen == batch.n_events


def test_rebase_and_sort():
    p = np.zeros(3, PEAK_DTYPE)
    p["event"], p["cell"], p["count"] = [1, 0, 1], [5, 9, 2], [8, 9, 10]
    q = sort_peaks(rebase_peaks(p, 10), cells=100)
    assert q["event"].tolist() == [10, 11, 11] and q["cell"].tolist() == [9, 2, 5] and q["count"].tolist() == [9, 10, 8]
    assert p["event"].tolist() == [1, 0, 1]                      # the input is not modified


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, outdir: str):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        batch = generate_batch(WL)
        sub, e0 = shard_batch(batch, rank, world)
        parts = [oracle_peaks(BN, oracle_fill(BN, *sub.event(k))[0], WL.threshold, event=k) for k in range(sub.n_events)]
        local = np.concatenate(parts) if parts else np.empty(0, PEAK_DTYPE)
        merged = gather_peaks(local, e0, BN.cells)
        np.save(os.path.join(outdir, f"merged_{rank}.npy"), merged)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_gathered_peak_lists_equal_the_unsharded_result(world):
    batch = generate_batch(WL)
    mats = [oracle_fill(BN, *batch.event(e))[0] for e in range(batch.n_events)]
    want = oracle_peaks_batch(BN, mats, WL.threshold)
    assert len(want) > 0
    with tempfile.TemporaryDirectory() as d:
        mp.spawn(_worker, args=(world, _free_port(), d), nprocs=world, join=True)
        for r in range(world):
            got = np.load(os.path.join(d, f"merged_{r}.npy"))
            assert got.dtype == PEAK_DTYPE and len(got) == len(want)
            for f in ("event", "cell", "count"):
                assert np.array_equal(got[f], want[f])


def test_gather_without_a_process_group_is_the_identity():
    p = np.zeros(2, PEAK_DTYPE)
    p["event"], p["cell"], p["count"] = [0, 0], [7, 3], [9, 9]
    q = gather_peaks(p, 4, cells=64)
    assert q["event"].tolist() == [4, 4] and q["cell"].tolist() == [3, 7]


def test_plane_ranges_partition_the_planes():
    for n_planes in (1, 4, 15, 64, 256):
        for world in (1, 2, 3, 4, 8):
            spans = [plane_range(n_planes, r, world) for r in range(world)]
            assert spans[0][0] == 0 and sum(c for _, c in spans) == n_planes
            assert all(spans[r][0] + spans[r][1] == spans[r + 1][0] for r in range(world - 1))

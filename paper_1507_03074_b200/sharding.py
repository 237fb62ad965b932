"""Host-side logic of the multi-GPU path: the hot path shards BY EVENT.

Events never share cells of ``M_H`` (reading R14; PAPER.md:27 treats the 100 events independently), so rank r of N
fills and scans a contiguous block of the batch's events on its own GPU and there is no data-path collective.  The only
exchange is the "merge" of the per-rank results ("merged at the end"): the compacted peak lists, ~10 KB per
event, gathered once.  This module holds none of the Hough arithmetic: event ranges, the slicing of a batch, the
all-gather of variable-length peak lists and the re-basing of their event indices.  It works on any
``torch.distributed`` backend (``nccl`` on the GPUs, ``gloo`` in the CPU tests).
"""
from __future__ import annotations

import numpy as np

from .binding import PEAK_DTYPE
from .events import EventBatch


def event_range(n_events: int, rank: int, world: int) -> tuple[int, int]:
    """[first, last) events of ``rank``: contiguous blocks, sizes differing by at most one, earlier ranks larger."""
    if world < 1 or not (0 <= rank < world) or n_events < 0:
        raise ValueError(f"bad sharding request: n_events={n_events} rank={rank} world={world}")
    base, extra = divmod(n_events, world)
    first = rank * base + min(rank, extra)
    return first, first + base + (1 if rank < extra else 0)


def shard_batch(batch: EventBatch, rank: int, world: int) -> tuple[EventBatch, int]:
    """The events of ``rank`` as a batch of their own (offsets re-based to 0) and the global index of its first event."""
    e0, e1 = event_range(batch.n_events, rank, world)
    h0, h1 = int(batch.event_offsets[e0]), int(batch.event_offsets[e1])
    offs = (batch.event_offsets[e0:e1 + 1] - batch.event_offsets[e0]).astype(np.int32)
    sub = EventBatch(x=np.ascontiguousarray(batch.x[h0:h1]), y=np.ascontiguousarray(batch.y[h0:h1]),
                     z=np.ascontiguousarray(batch.z[h0:h1]), event_offsets=offs,
                     truth=list(batch.truth[e0:e1]) if batch.truth else [])
    return sub, e0


def rebase_peaks(peaks: np.ndarray, first_event: int) -> np.ndarray:
    """Peak records of a shard (event index local to the shard) with the event index of the whole batch."""
    out = np.array(peaks, dtype=PEAK_DTYPE, copy=True)
    out["event"] = out["event"] + np.uint32(first_event)
    return out


def sort_peaks(peaks: np.ndarray, cells: int) -> np.ndarray:
    """The order parity is defined on (R13): by (event, cell)."""
    key = peaks["event"].astype(np.int64) * int(cells) + peaks["cell"].astype(np.int64)
    return peaks[np.argsort(key, kind="stable")]


def gather_peaks(local_peaks: np.ndarray, first_event: int, cells: int, group=None, device=None) -> np.ndarray:
    """All ranks' peak lists, event indices re-based to the whole batch, sorted by (event, cell), on every rank.

    One all-gather of the list lengths, then one all-gather of lists padded to the longest (3 uint32 per record, sent
    as int32).  Without an initialised process group this is the single-rank identity.
    """
    import torch
    import torch.distributed as dist

    mine = rebase_peaks(local_peaks, first_event)
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return sort_peaks(mine, cells)
    world = dist.get_world_size(group)
    dev = torch.device("cpu") if device is None else device
    n_local = torch.tensor([mine.shape[0]], dtype=torch.int64, device=dev)
    counts = [torch.zeros(1, dtype=torch.int64, device=dev) for _ in range(world)]
    dist.all_gather(counts, n_local, group=group)
    counts = [int(c.item()) for c in counts]
    longest = max(max(counts), 1)
    rec = np.zeros((longest, 3), dtype=np.uint32)
    rec[:mine.shape[0], 0], rec[:mine.shape[0], 1], rec[:mine.shape[0], 2] = mine["event"], mine["cell"], mine["count"]
    send = torch.from_numpy(rec.view(np.int32)).to(dev)
    recv = [torch.empty_like(send) for _ in range(world)]
    dist.all_gather(recv, send, group=group)
    parts = []
    for r, n in enumerate(counts):
        a = recv[r][:n].cpu().numpy().view(np.uint32)
        p = np.empty(n, PEAK_DTYPE)
        p["event"], p["cell"], p["count"] = a[:, 0], a[:, 1], a[:, 2]
        parts.append(p)
    return sort_peaks(np.concatenate(parts) if parts else np.empty(0, PEAK_DTYPE), cells)


def plane_range(n_planes: int, rank: int, world: int) -> tuple[int, int]:
    """(plane_begin, plane_count) of ``rank`` when ONE event is split over the ranks by (theta, phi) plane -- the sector
    split of PAPER.md:77 ("four M_H(A,B,theta), each matrix processing the data of a single phi sector"), generalised to
    any contiguous block of planes (plane = itheta * n_phi + iphi).  Planes never exchange votes or peaks (R10), so every
    rank gets all the hits, fills and scans its planes (``ht_config.plane_begin / plane_count``), and the only
    communication is ``gather_peaks`` (``first_event = 0``: the records already carry full-matrix cell indices)."""
    first, last = event_range(n_planes, rank, world)
    return first, last - first

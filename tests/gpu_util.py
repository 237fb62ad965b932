"""Helpers of the -m gpu parity tests: run the CUDA path through the C-ABI binding and bring results back as numpy.
torch is used for device memory and streams only."""
from __future__ import annotations

import numpy as np
import torch

from paper_1507_03074_b200 import binding as B


def sort_peaks(pk: np.ndarray, cells: int) -> np.ndarray:
    key = pk["event"].astype(np.int64) * int(cells) + pk["cell"].astype(np.int64)
    return pk[np.argsort(key, kind="stable")]


class GpuHough:
    """One context + the device buffers of one batch."""

    def __init__(self, binning, max_events: int, max_hits: int, host_slots: int = 0, host_peak_capacity: int = 0,
                 tuning: dict | None = None, own_workspace: bool = False):
        """``tuning``: fields of ht_tuning; ``own_workspace``: the test allocates the context's device workspace itself
        (ht_query_sizes -> torch -> ht_create_ex), so the library allocates no device memory at all."""
        self.bn = binning
        self.cfg = B.ht_config.from_binning(binning, max_events=max_events, max_hits=max(1, max_hits), device=0,
                                            host_slots=host_slots, host_peak_capacity=host_peak_capacity)
        self.dev = torch.device("cuda:0")
        tuning = dict(tuning) if tuning else None
        stable = bool(tuning.pop("stable_inputs", 0)) if tuning else False      # (not a tuning field: ht_promise_stable_inputs)
        self.tuning = B.ht_tuning(**tuning) if tuning else None
        self.workspace = None
        if own_workspace:
            nbytes = B.ht_query_sizes(self.cfg)[1]
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.dev)
            base = (self.workspace.data_ptr() + 255) // 256 * 256
            self.ctx = B.ht_create_ex(self.cfg, self.tuning, base, nbytes)
        elif self.tuning is not None:
            self.ctx = B.ht_create_ex(self.cfg, self.tuning)
        else:
            self.ctx = B.ht_create(self.cfg)
        if stable:
            B.ht_promise_stable_inputs(self.ctx, True)

    def close(self):
        B.ht_destroy(self.ctx)
        self.ctx = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def upload(self, batch):
        t = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a)).to(self.dev, dtype=dt)
        return (t(batch.x, torch.float32), t(batch.y, torch.float32), t(batch.z, torch.float32),
                t(batch.event_offsets, torch.int32))

    def fill(self, batch, naive: bool = False, poison: bool = True, stream=None) -> torch.Tensor:
        dx, dy, dz, doff = self.upload(batch)
        cells = self.cfg.cells
        mh = torch.empty(batch.n_events * cells, dtype=torch.int32, device=self.dev)
        if poison and mh.numel():
            mh.fill_(-1)                      # the fill must overwrite every cell
        fn = B.ht_fill_naive if naive else B.ht_fill
        fn(self.ctx, dx, dy, dz, doff, batch.n_events, batch.n_hits, mh, stream)
        torch.cuda.synchronize()
        return mh

    def fill_peaks(self, batch, threshold: int, capacity: int = 1 << 20, store: bool = True, stream=None):
        """Fused call.  Returns (mh or None, n_found, peaks)."""
        dx, dy, dz, doff = self.upload(batch)
        cells = self.cfg.cells
        mh = None
        if store:
            mh = torch.empty(batch.n_events * cells, dtype=torch.int32, device=self.dev)
            if mh.numel():
                mh.fill_(-1)
        out = torch.zeros(max(capacity, 1) * 3, dtype=torch.int32, device=self.dev)
        nf = torch.full((1,), -7, dtype=torch.int32, device=self.dev)
        B.ht_fill_peaks(self.ctx, dx, dy, dz, doff, batch.n_events, batch.n_hits, mh, threshold,
                        out if capacity else None, capacity, nf, stream)
        torch.cuda.synchronize()
        return (mh,) + self._peak_result(out, nf, capacity)

    @staticmethod
    def _peak_result(out, nf, capacity):
        n = int(nf.cpu().numpy().view(np.uint32)[0])
        k = min(n, capacity)
        rec = out[:3 * k].cpu().numpy().view(np.uint32).reshape(k, 3)
        pk = np.empty(k, B.PEAK_DTYPE)
        pk["event"], pk["cell"], pk["count"] = rec[:, 0], rec[:, 1], rec[:, 2]
        return n, pk

    def peaks(self, mh: torch.Tensor, n_events: int, threshold: int, capacity: int = 1 << 20, stream=None):
        out = torch.zeros(max(capacity, 1) * 3, dtype=torch.int32, device=self.dev)
        nf = torch.full((1,), -7, dtype=torch.int32, device=self.dev)
        B.ht_peaks(self.ctx, mh, n_events, threshold, out if capacity else None, capacity, nf, stream)
        torch.cuda.synchronize()
        return self._peak_result(out, nf, capacity)


def mh_to_numpy(mh: torch.Tensor, bn, n_events: int) -> np.ndarray:
    return mh.cpu().numpy().view(np.uint32).reshape(n_events, bn.n_theta, bn.n_phi, bn.n_a, bn.n_b)

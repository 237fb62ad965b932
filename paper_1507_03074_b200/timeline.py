"""In-kernel timeline of one fused call (developer tool; not part of the product path).

    python -m paper_1507_03074_b200.timeline [CONFIG] [fused|fill|nostore] [plain] [noearly]

Builds a second copy of the library with -DHT_PROFILE_TIMELINE (libht_timeline.so, beside libht.so), in which every CTA of
the fill kernel stamps its SM's cycle counter at a few points of its life, runs 4000 warm-up calls and 50 measured ones (cooperative
launches, so that a CTA's start is not pulled into the previous call's tail), and prints microseconds after the CTA's own
start, mean over the CTAs (min..max).  The extra stores cost the kernel ~2 us per call: read the DIFFERENCES between the
points, not the totals.  Needs a GPU.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import sys

import numpy as np


def main() -> None:
    import torch

    from . import binding as B
    from .build import CSRC, INCLUDE, NVCC_FLAGS, nvcc_path
    from .events import WORKLOADS, generate_batch

    cfg_id = int(sys.argv[1]) if len(sys.argv) > 1 else 2
    mode = sys.argv[2] if len(sys.argv) > 2 else "fused"
    lib = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libht_timeline.so")
    plain = "plain" in sys.argv[3:]          # the shipped library: only the time per call is printed
    if not plain:
        subprocess.run([nvcc_path(), *NVCC_FLAGS, "-DHT_PROFILE_TIMELINE", "-I", INCLUDE, "-o", lib, os.path.join(CSRC, "ht_api.cu")],
                       check=True)
        B.LIB_PATH = lib
    wl = WORKLOADS[cfg_id]
    bn = wl.binning
    batch = generate_batch(wl, n_events=1)
    dev = torch.device("cuda:0")
    to = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a)).to(dev, dtype=dt)
    dx, dy, dz, doff = to(batch.x, torch.float32), to(batch.y, torch.float32), to(batch.z, torch.float32), to(batch.event_offsets, torch.int32)
    mhs = [torch.empty(bn.cells, dtype=torch.int32, device=dev) for _ in range(4)]
    cap = 1 << 17
    out = torch.empty(cap * 3, dtype=torch.int32, device=dev)
    nf = torch.zeros(1, dtype=torch.int32, device=dev)
    st = torch.cuda.Stream()
    ctx = B.ht_create_ex(B.ht_config.from_binning(bn, max_events=1, max_hits=batch.n_hits, device=0),
                         B.ht_tuning(cooperative_launch=1, fill_early_cap=-1 if "noearly" in sys.argv else 0))
    libc = B.load()
    if not plain:
        libc.ht_prof_read.argtypes = [C.c_void_p, C.c_int32, C.c_int32]
    buf = np.zeros(256 * 32, np.uint64)

    def call(k):
        if mode == "fused":
            B.ht_fill_peaks(ctx, dx, dy, dz, doff, 1, batch.n_hits, mhs[k % 4], wl.threshold, out, cap, nf, st)
        elif mode == "fill":
            B.ht_fill(ctx, dx, dy, dz, doff, 1, batch.n_hits, mhs[k % 4], st)
        else:
            B.ht_fill_peaks(ctx, dx, dy, dz, doff, 1, batch.n_hits, None, wl.threshold, out, cap, nf, st)

    for k in range(4000):                      # ~0.2 s: the clocks are up by then
        call(k)
    st.synchronize()
    if not plain:
        libc.ht_prof_read(buf.ctypes.data, 256 * 32, 1)
    n = 50
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(st)
    for k in range(n):
        call(k)
    e1.record(st)
    st.synchronize()
    if plain:
        print(f"config {cfg_id}, {mode}, shipped library, cooperative launches: {e0.elapsed_time(e1) / n * 1e3:.2f} us per call")
        B.ht_destroy(ctx)
        return
    libc.ht_prof_read(buf.ctypes.data, 256 * 32, 1)
    raw = buf.reshape(256, 32)
    live = raw[:, 13] > 0
    ns_per_cycle = raw[live, 0].sum() / raw[live, 13].sum()        # the stamps are SM cycles since the CTA's start
    a = raw.astype(np.float64) * ns_per_cycle / n / 1e3
    start = raw[live, 12].astype(np.int64)
    f = lambda k: f"{a[live, k].mean():6.2f} ({a[live, k].min():.2f}..{a[live, k].max():.2f})"
    print(f"config {cfg_id}, {mode}, instrumented build, cooperative launches: {e0.elapsed_time(e1) / n * 1e3:.2f} us per call; "
          f"{int(live.sum())} CTAs, SM clock {1e3 / ns_per_cycle:.0f} MHz, start skew of the last call {(start.max() - start.min()) / 1e3:.2f} us")
    # (without early tiles -- tuning fill_early_cap = -1, argument "noearly" -- points 4 and 5 are: thread 0 has classified
    # its first hit / drawn its slot; 7 is not passed)
    for label, k in (("slabs zeroed, previous kernel complete", 4), ("early tiles: coarse test of all hits done", 7),
                     ("prologue done (early list / plane counts in shared memory)", 15),
                     ("this CTA's share of the hits is in the buckets", 5), ("grid barrier passed", 6),
                     ("voters (thread 0) begin tile 0", 1), ("... know their share and have asked for their hits", 16),
                     ("... have asked for the hits of tile 1", 17), ("... have voted their share of it", 2), ("first tile store issued", 11),
                     ("voters (thread 0) begin tile 1", 3), ("... have voted their share of it", 10), ("second tile store issued", 8), ("third tile store issued", 9),
                     ("tile loop done", 14), ("last store read by the TMA", 13)):
        print(f"  {label:48s} {f(k)} us")
    B.ht_destroy(ctx)


if __name__ == "__main__":
    main()

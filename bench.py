#!/usr/bin/env python
"""bench.py -- events/s and Hough votes/s of the fill + peak-search hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2]

A STEP is one pass of the whole hot path (classify, slab fill, peak test+compaction: SURVEY.md section 8(a)
a0-a5) over one event of the workload (default: config 2, the paper-shaped 5000-hit event, 4x16x1024x1024 bins).
`value` = events/s with the hits already resident in HBM (CUDA events on the launch stream, max over ranks);
`e2e`   = the same metric through ht_run_host with pinned HOST buffers (H2D of the hits and D2H of the peak list inside
          the timed region);
`roofline` = achieved HBM GB/s of the dominant kernel call (algorithmic bytes / CUDA-event duration measured in the
          timed region) against MEASURED_PEAKS.json;
`cpu_baseline` = the CPU oracle as it stands, one core, on the same event (also checks parity in the same run).
N > 1 (torchrun): every rank processes its own seeded event, no data-path collective ("scaling": "weak"); with
`--split planes` all ranks take the same event and a range of (theta, phi) planes each ("strong").
`--impl reference` times the CPU oracle itself (there is no reference implementation of the paper to install).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "events/s and Hough votes/s (fill+peak search), 5000-hit event, 1 B200"
FALLBACK_HBM_GBS = 6650.0          # /opt/skills/guides/B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


def measured_hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json: bf16 copy, read+write)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.01):
        super().__init__(daemon=True)
        self.index, self.period, self.samples, self.reasons, self.stop_flag = index, period_s, [], set(), False
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
                 nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake"}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml unavailable"]}
        return {"sm_mhz": statistics.median(self.samples), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def run_oracle_event(bn, batch, threshold):
    """One event through the CPU oracle: (matrix, peaks, votes, seconds fill, seconds peaks)."""
    from oracle import oracle_fill, oracle_peaks
    t0 = time.perf_counter()
    m, votes = oracle_fill(bn, *batch.event(0))
    t1 = time.perf_counter()
    pk = oracle_peaks(bn, m, threshold)
    t2 = time.perf_counter()
    return m, pk, votes, t1 - t0, t2 - t1


def bench_reference(args):
    """--impl reference: the CPU oracle as it stands on this box's host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1507_03074_b200.events import WORKLOADS, generate_batch
    wl = WORKLOADS[args.config]
    batch = generate_batch(wl, n_events=1)
    for _ in range(max(args.warmup, 0)):
        run_oracle_event(wl.binning, batch, wl.threshold)
    times, votes = [], 0
    t_all = time.perf_counter()
    for _ in range(args.steps):
        _, _, votes, tf, tp = run_oracle_event(wl.binning, batch, wl.threshold)
        times.append(tf + tp)
    total = time.perf_counter() - t_all
    value = args.steps / total
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "events/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "u32 counts / f32 bin decisions", "data": "synthetic",
        "config": {"workload": f"config{wl.config}:{wl.name}", "bins": [wl.binning.n_theta, wl.binning.n_phi, wl.binning.n_a, wl.binning.n_b],
                   "hits_per_event": batch.n_hits, "threshold": wl.threshold},
        "votes_per_s": votes * value,
        "cpu_baseline": {"value": value, "unit": "events/s", "cores": 1, "kind": "oracle",
                         "sample": f"{args.steps} full events of this workload, single thread"},
        "e2e": {"value": value, "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def bench_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1507_03074_b200 import binding as B
    from paper_1507_03074_b200.events import WORKLOADS, generate_batch

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    wl = WORKLOADS[args.config]
    bn = wl.binning
    n_ev = args.events if args.events else 1
    # every rank its own events (weak scaling: the path shards by event, no data-path collective)
    # --split events (default): every rank its own events (weak scaling: the path shards by event, no data-path
    # collective).  --split planes: all ranks take the SAME events and a contiguous range of the (theta, phi) planes each
    # (strong scaling; the sector split of PAPER.md:77); again no collective in the timed region
    by_planes = args.split == "planes"
    batch = generate_batch(wl, n_events=n_ev, first_event=0 if by_planes else rank * n_ev)
    n_hits = batch.n_hits
    from paper_1507_03074_b200.sharding import plane_range
    p0, pc = plane_range(bn.planes, rank, world) if by_planes else (0, bn.planes)
    cells = pc * bn.n_a * bn.n_b                                     # cells of this rank's matrix per event
    cap = 1 << 16
    cfg = B.ht_config.from_binning(bn, max_events=n_ev, max_hits=n_hits, device=local_rank, host_slots=n_ev,
                                   host_peak_capacity=cap, plane_begin=p0 if by_planes else 0,
                                   plane_count=pc if by_planes else 0)
    ctx = B.ht_create(cfg)
    stream = torch.cuda.Stream(device=dev)

    to = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a)).to(dev, dtype=dt)
    dx, dy, dz = to(batch.x, torch.float32), to(batch.y, torch.float32), to(batch.z, torch.float32)
    doff = to(batch.event_offsets, torch.int32)
    mh_bytes = 4 * cells * n_ev
    n_rot = args.rotate if mh_bytes * args.rotate <= (8 << 30) else 1   # rotate output matrices: no step inherits L2 contents
    mhs = [torch.empty(cells * n_ev, dtype=torch.int32, device=dev) for _ in range(n_rot)]
    d_out = torch.empty(cap * 3, dtype=torch.int32, device=dev)
    d_nf = torch.zeros(1, dtype=torch.int32, device=dev)
    T = wl.threshold

    def step_fused(k, evs=None):                      # a0-a5 in ONE kernel, matrix materialised
        if evs is not None:
            evs[0].record(stream)
        B.ht_fill_peaks(ctx, dx, dy, dz, doff, n_ev, n_hits, mhs[k % n_rot], T, d_out, cap, d_nf, stream)
        if evs is not None:
            evs[1].record(stream)

    def step_split(k, evs=None):                      # the paper's two-kernel split: ht_fill, then ht_peaks
        mh = mhs[k % n_rot]
        if evs is not None:
            evs[0].record(stream)
        B.ht_fill(ctx, dx, dy, dz, doff, n_ev, n_hits, mh, stream)
        if evs is not None:
            evs[1].record(stream)
        B.ht_peaks(ctx, mh, n_ev, T, d_out, cap, d_nf, stream)
        if evs is not None:
            evs[2].record(stream)

    def step_nostore(k, evs=None):                    # peaks only: the matrix never leaves shared memory
        if evs is not None:
            evs[0].record(stream)
        B.ht_fill_peaks(ctx, dx, dy, dz, doff, n_ev, n_hits, None, T, d_out, cap, d_nf, stream)
        if evs is not None:
            evs[1].record(stream)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def n_found_now():
        stream.synchronize()
        return int(d_nf.cpu().numpy().view(np.uint32)[0])

    def timed(step, n_marks, sampler=None):
        """W warm-up steps, then exactly K steps bracketed by barrier+synchronize; CUDA events on the launch stream."""
        for k in range(max(args.warmup, 3)):
            step(k)
        found = n_found_now()
        # one kernel per step: the bracketing events alone give its average duration (launch gap included); events
        # between the two kernels of the split path are recorded only there (each record costs ~2 us of stream time)
        inner = n_marks > 2
        evs = [[torch.cuda.Event(enable_timing=True) for _ in range(n_marks)] if inner else None for _ in range(args.steps)]
        l0 = B.ht_kernel_launches(ctx)
        barrier()
        if sampler is not None:
            sampler.start()
        t_start, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t_start.record(stream)
        for k in range(args.steps):
            step(k, evs[k])
        t_end.record(stream)
        barrier()
        if sampler is not None:
            sampler.stop_flag = True
        launches = B.ht_kernel_launches(ctx) - l0
        total_ms = t_start.elapsed_time(t_end)
        if world > 1:
            t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            total_ms = float(t.item())
        if inner:
            spans = [[e[i].elapsed_time(e[i + 1]) for e in evs] for i in range(n_marks - 1)]
        else:
            spans = [[total_ms / args.steps] * args.steps]
        return total_ms / args.steps, spans, launches, found

    fused_ok = True
    try:
        step_fused(0)
        stream.synchronize()
    except B.HtError as err:
        if err.status != B.HT_ERR_UNSUPPORTED:
            raise
        fused_ok = False
    headline = "fused" if (fused_ok and args.mode != "split") else "split"

    sampler = ClockSampler(local_rank)
    res = {}
    if headline == "fused":
        res["fused"] = timed(step_fused, 2, sampler)
        res["split"] = timed(step_split, 3)
    else:
        res["split"] = timed(step_split, 3, sampler)
        if fused_ok:
            res["fused"] = timed(step_fused, 2)
    if fused_ok:
        res["nostore"] = timed(step_nostore, 2)
    # The same K calls captured once into a CUDA graph and replayed (the calls keep no host-side state): the launch gap
    # between two stream launches of a cooperative kernel (~1.5 us) goes away.  Headline if it works and is faster.
    graph_ms = None
    if headline == "fused" and not args.no_graph:
        try:
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=stream):
                for k in range(args.steps):
                    step_fused(k)
            graph.replay()                                            # warm-up replay
            barrier()
            g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            g0.record()
            graph.replay()
            g1.record()
            barrier()
            graph_ms = g0.elapsed_time(g1) / args.steps
            if world > 1:
                t = torch.tensor([graph_ms], dtype=torch.float64, device=dev)
                dist.all_reduce(t, op=dist.ReduceOp.MAX)
                graph_ms = float(t.item())
            if n_found_now() != res["fused"][3]:
                graph_ms = None
        except Exception as err:                                      # capture not supported here: stream launches stand
            print(f"bench.py: CUDA graph capture failed ({err!r}); timing stream launches only", file=sys.stderr)
            graph_ms = None
    # leave the headline path's outputs in the buffers for the parity check below
    last_k = args.steps - 1
    (step_fused if headline == "fused" else step_split)(last_k)
    n_found = n_found_now()
    ms_per_step, _, launches, _ = res[headline]
    launch_mode = "stream launches"
    if graph_ms is not None and graph_ms < ms_per_step:
        ms_per_step, launches = graph_ms, args.steps
        launch_mode = f"{args.steps} calls captured once into a CUDA graph, one replay timed"
    jobs = 1 if by_planes else world                                  # --split planes: all ranks work on the same events
    value = jobs * n_ev * 1e3 / ms_per_step                           # events/s over all ranks

    # ---- f3: track read-out (rho, phi) of the peak list, a separate small kernel (not part of the headline step)
    d_tr = torch.empty(5 * cap, dtype=torch.int32, device=dev)
    n_tr = min(n_found, cap)
    for _ in range(5):
        B.ht_tracks(ctx, d_out, n_tr, d_tr, stream)
    stream.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    for _ in range(200):
        B.ht_tracks(ctx, d_out, n_tr, d_tr, stream)
    ev1.record(stream)
    stream.synchronize()
    tracks_ms = ev0.elapsed_time(ev1) / 200

    # ---- end to end through the host entry point: pinned host buffers, H2D + D2H inside the timed region
    hx, hy, hz = (torch.from_numpy(a.copy()).pin_memory() for a in (batch.x, batch.y, batch.z))
    hoff = torch.from_numpy(batch.event_offsets.copy()).pin_memory()
    hout = torch.zeros(cap * 3, dtype=torch.int32).pin_memory()
    for _ in range(3):
        n_e2e = B.ht_run_host(ctx, hx, hy, hz, hoff, n_ev, n_hits, T, hout, cap)
    barrier()
    e2e_steps = args.steps
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        n_e2e = B.ht_run_host(ctx, hx, hy, hz, hoff, n_ev, n_hits, T, hout, cap)
    e2e_s = time.perf_counter() - t0
    if world > 1:
        t = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    e2e_value = jobs * n_ev * e2e_steps / e2e_s
    h2d = 3 * 4 * n_hits + 4 * (n_ev + 1)                 # one packed copy: offsets + x + y + z
    d2h = 4 + 12 * min(n_e2e, cap)                        # count + peak records, written by the kernel into mapped pinned memory

    if rank == 0:
        peak_gbs, peak_src = measured_hbm_peak()
        mean = lambda v: sum(v) / len(v)
        m_bytes = 4 * cells * n_ev
        hit_bytes, pk_bytes = 12 * n_hits, 12 * n_found

        # dram__bytes_read.sum + dram__bytes_write.sum per launch from the ncu --set full capture of config 2, one event
        # (profiles/r01b_fill_full.md): the fill kernels end with ~60 MB of the matrix still dirty in L2
        ncu_traffic = {"ht_fill_peaks": 210.3e6, "ht_fill": 208.6e6, "ht_peaks": 272.1e6} if (args.config == 2 and n_ev == 1) else {}

        def roof(name, nbytes, ms, key=None):
            ach = nbytes / (ms * 1e-3) / 1e9
            return {"bound": "hbm", "achieved": ach, "peak": peak_gbs, "unit": "GB/s", "frac": ach / peak_gbs,
                    "traffic": ncu_traffic.get(key), "kernel": name, "algorithmic_bytes_per_launch": nbytes, "avg_ms_per_launch": ms,
                    "peak_source": peak_src}

        kernels, kernel_ms = {}, {}
        if "fused" in res:
            f = res["fused"][1][0]
            kernels["ht_fill_peaks"] = roof("fill_tiles_kernel<true> (ht_fill_peaks: classify, vote, store, peak test, compaction in one kernel)",
                                            m_bytes + hit_bytes + pk_bytes,
                                            ms_per_step if headline == "fused" else mean(f), "ht_fill_peaks")
            kernel_ms.update(fused_median=statistics.median(f), fused_mean=mean(f), fused_step_mean=res["fused"][0],
                             fused_graph_step_mean=graph_ms)
        sp_fill, sp_peaks = res["split"][1]
        kernels["ht_fill"] = roof("fill_tiles_kernel<false> (ht_fill: classify, vote, store in one kernel)", m_bytes + hit_bytes, mean(sp_fill), "ht_fill")
        kernels["ht_peaks"] = roof("peaks_kernel (ht_peaks: scan+compaction)", m_bytes + pk_bytes, mean(sp_peaks), "ht_peaks")
        kernel_ms.update(fill_median=statistics.median(sp_fill), fill_mean=mean(sp_fill),
                         peaks_median=statistics.median(sp_peaks), peaks_mean=mean(sp_peaks),
                         split_step_mean=res["split"][0])
        if "nostore" in res:
            kernel_ms.update(nostore_median=statistics.median(res["nostore"][1][0]), nostore_step_mean=res["nostore"][0])
        if headline == "fused":
            dominant = kernels["ht_fill_peaks"]
        else:
            dominant = max((kernels["ht_fill"], kernels["ht_peaks"]), key=lambda r: r["avg_ms_per_launch"])

        # ---- cpu_baseline (oracle, 1 core) on event 0 + parity of this very launch configuration
        from oracle import oracle_fill, oracle_peaks
        reps, o_times, votes = 3, [], 0
        for _ in range(reps):
            m_ref, pk_ref, votes, tf, tp = run_oracle_event(bn, batch, T)
            o_times.append((tf, tp))
        got_all = mhs[last_k % n_rot].cpu().numpy().view(np.uint32).reshape(n_ev, -1)
        k = min(n_found, cap)
        rec = d_out[:3 * k].cpu().numpy().view(np.uint32).reshape(k, 3)
        rec = rec[np.lexsort((rec[:, 1], rec[:, 0]))]
        lo_cell, hi_cell = p0 * bn.n_a * bn.n_b, (p0 + pc) * bn.n_a * bn.n_b     # this rank's part of the full matrix
        parity = bool(np.array_equal(got_all[0], m_ref.reshape(-1)[lo_cell:hi_cell]))
        n_ref, votes_all = 0, 0
        for e in range(n_ev):
            if e == 0:
                m_e, pk_e, v_e = m_ref, pk_ref, votes
            else:
                m_e, v_e = oracle_fill(bn, *batch.event(e))
                pk_e = oracle_peaks(bn, m_e, T)
                parity = parity and bool(np.array_equal(got_all[e], m_e.reshape(-1)[lo_cell:hi_cell]))
            votes_all += v_e
            pk_e = pk_e[(pk_e["cell"] >= lo_cell) & (pk_e["cell"] < hi_cell)]
            r_e = rec[rec[:, 0] == e]
            parity = parity and len(r_e) == len(pk_e) and bool(np.array_equal(r_e[:, 1], pk_e["cell"])
                                                                and np.array_equal(r_e[:, 2], pk_e["count"]))
            n_ref += len(pk_e)
        parity = parity and n_found == n_ref and n_e2e == n_ref
        for name in res:
            parity = parity and res[name][3] == n_ref
        o_fill = statistics.median(t[0] for t in o_times)
        o_peaks = statistics.median(t[1] for t in o_times)
        info = B.ht_launch_info(ctx)
        line = {
            "metric": METRIC, "value": value, "unit": "events/s", "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "strong" if by_planes else "weak",
            "vs_baseline": None, "dtype": "u32 counts / f32 bin decisions", "data": "synthetic",
            "config": {"workload": f"config{wl.config}:{wl.name}", "bins": [bn.n_theta, bn.n_phi, bn.n_a, bn.n_b],
                       "hits_per_step": n_hits, "threshold": T, "events_per_step": n_ev,
                       "path": ("ht_fill_peaks: one kernel does a0-a5 and stores every M_H cell once" if headline == "fused"
                                else "ht_fill + ht_peaks (two kernels)"),
                       "l2": f"M_H per step ({m_bytes / 1e6:.0f} MB) is larger than the 126 MB L2; {n_rot} output matrices "
                             "rotated so no step inherits another step's lines",
                       "launch": info, "launch_mode": launch_mode},
            "votes_per_s": votes_all * jobs * 1e3 / ms_per_step, "votes_per_step": votes_all, "peaks_per_step": n_found,
            "hit_a_evaluations_per_s": n_hits * bn.n_a * jobs * 1e3 / ms_per_step,
            "parity_vs_oracle": "bit-exact" if parity else "MISMATCH",
            "kernel_ms": kernel_ms,
            "paths_events_per_s": dict({name: jobs * n_ev * 1e3 / r[0] for name, r in res.items()},
                                       **({"fused_graph": jobs * n_ev * 1e3 / graph_ms} if graph_ms else {})),
            "roofline": dominant, "roofline_kernels": kernels,
            "cpu_baseline": {"value": 1.0 / (o_fill + o_peaks), "unit": "events/s", "cores": 1, "kind": "oracle",
                             "sample": f"median of {reps} runs of one full event of this workload (fill {o_fill * 1e3:.0f} ms + "
                                       f"peaks {o_peaks * 1e3:.0f} ms), single thread, host of the GPU box",
                             "host_cpus": os.cpu_count()},
            "e2e": {"value": e2e_value, "unit": "events/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": 1e3 * e2e_s / e2e_steps, "api": "ht_run_host (host buffers -> pinned block; single event: the kernel reads the hits over PCIe (zero-copy), batches: one packed H2D copy; the peak list is written by the kernel into mapped pinned memory)"},
            "tracks": {"ms_per_call": tracks_ms, "n_peaks": n_tr, "what": "ht_tracks: rho, phi of every peak (f3), launch-bound"},
            "gpu_launches": int(launches),
            "clocks": sampler.summary(),
        }
        print(json.dumps(line), flush=True)
        if not parity:
            B.ht_destroy(ctx)
            raise SystemExit("bench.py: GPU result differs from the oracle")
    B.ht_destroy(ctx)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", type=int, default=2, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--events", type=int, default=0, help="events per step (default 1)")
    ap.add_argument("--mode", choices=["fused", "split"], default="fused",
                    help="headline path: ht_fill_peaks (one kernel) or ht_fill + ht_peaks")
    ap.add_argument("--rotate", type=int, default=4, help="number of output matrices rotated between steps")
    ap.add_argument("--no-graph", action="store_true", help="time stream launches only (no CUDA graph replay)")
    ap.add_argument("--split", choices=["events", "planes"], default="events",
                    help="N > 1: every rank its own events (weak scaling, default) or the same events split by plane")
    args = ap.parse_args()
    if args.impl == "reference":
        args.steps = 10 if args.steps is None else args.steps
        args.warmup = 1 if args.warmup is None else args.warmup
        bench_reference(args)
    else:
        args.steps = 2000 if args.steps is None else args.steps
        args.warmup = 10 if args.warmup is None else args.warmup
        bench_ours(args)


if __name__ == "__main__":
    main()

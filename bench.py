#!/usr/bin/env python
"""bench.py -- events/s and Hough votes/s of the fill + peak-search hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2]

A STEP is one pass of the whole hot path (classify+bucket, slab fill, peak scan+compaction: SURVEY.md section 8(a)
a0-a5) over one event of the workload (default: config 2, the paper-shaped 5000-hit event, 4x16x1024x1024 bins).
`value` = events/s with the hits already resident in HBM (CUDA events on the launch stream, max over ranks);
`e2e`   = the same metric through ht_run_host with pinned HOST buffers (H2D of the hits and D2H of the peak list inside
          the timed region);
`roofline` = achieved HBM GB/s of the dominant kernel call (algorithmic bytes / CUDA-event duration measured in the
          timed region) against MEASURED_PEAKS.json;
`cpu_baseline` = the CPU oracle as it stands, one core, on the same event (also checks parity in the same run).
N > 1 (torchrun): every rank processes its own seeded event, no data-path collective ("scaling": "weak").
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
    batch = generate_batch(wl, n_events=1, seed_offset=rank)          # every rank its own event (weak scaling)
    n_hits = batch.n_hits
    cells = bn.cells
    cap = 1 << 16
    cfg = B.ht_config.from_binning(bn, max_events=1, max_hits=n_hits, device=local_rank, host_slots=1,
                                   host_peak_capacity=cap)
    ctx = B.ht_create(cfg)
    stream = torch.cuda.Stream(device=dev)

    to = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a)).to(dev, dtype=dt)
    dx, dy, dz = to(batch.x, torch.float32), to(batch.y, torch.float32), to(batch.z, torch.float32)
    doff = to(batch.event_offsets, torch.int32)
    n_rot = args.rotate                                               # rotate output matrices: no step inherits L2 contents
    mhs = [torch.empty(cells, dtype=torch.int32, device=dev) for _ in range(n_rot)]
    d_out = torch.empty(cap * 3, dtype=torch.int32, device=dev)
    d_nf = torch.zeros(1, dtype=torch.int32, device=dev)

    def step(k, evs=None):
        mh = mhs[k % n_rot]
        if evs is not None:
            evs[0].record(stream)
        B.ht_fill(ctx, dx, dy, dz, doff, 1, n_hits, mh, stream)
        if evs is not None:
            evs[1].record(stream)
        B.ht_peaks(ctx, mh, 1, wl.threshold, d_out, cap, d_nf, stream)
        if evs is not None:
            evs[2].record(stream)

    # ---- warm-up, then parity of exactly this launch configuration against the oracle (rank 0)
    for k in range(max(args.warmup, 3)):
        step(k)
    stream.synchronize()
    n_found = int(d_nf.cpu().numpy().view(np.uint32)[0])

    # ---- timed region: K steps back to back; per-call CUDA events on the launch stream
    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    sampler = ClockSampler(local_rank)
    launches0 = B.ht_kernel_launches(ctx)
    barrier()
    sampler.start()
    t_start, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_start.record(stream)
    for k in range(args.steps):
        step(k, evs[k])
    t_end.record(stream)
    barrier()
    sampler.stop_flag = True
    launches = B.ht_kernel_launches(ctx) - launches0
    total_ms = t_start.elapsed_time(t_end)
    fill_ms = [e[0].elapsed_time(e[1]) for e in evs]
    peaks_ms = [e[1].elapsed_time(e[2]) for e in evs]
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    ms_per_step = total_ms / args.steps
    value = world * 1e3 / ms_per_step                                 # events/s over all ranks

    # ---- end to end through the host entry point: pinned host buffers, H2D + D2H inside the timed region
    hx, hy, hz = (torch.from_numpy(a.copy()).pin_memory() for a in (batch.x, batch.y, batch.z))
    hoff = torch.from_numpy(batch.event_offsets.copy()).pin_memory()
    hout = torch.zeros(cap * 3, dtype=torch.int32).pin_memory()
    for _ in range(3):
        n_e2e = B.ht_run_host(ctx, hx, hy, hz, hoff, 1, n_hits, wl.threshold, hout, cap)
    barrier()
    e2e_steps = args.steps
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        n_e2e = B.ht_run_host(ctx, hx, hy, hz, hoff, 1, n_hits, wl.threshold, hout, cap)
    e2e_s = time.perf_counter() - t0
    if world > 1:
        t = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    e2e_value = world * e2e_steps / e2e_s
    h2d = 3 * 4 * n_hits + 4 * 2
    d2h = 16 + 12 * min(cap, 4096)

    if rank == 0:
        peak_gbs, peak_src = measured_hbm_peak()
        fill_med, peaks_med = statistics.median(fill_ms), statistics.median(peaks_ms)
        fill_avg, peaks_avg = sum(fill_ms) / len(fill_ms), sum(peaks_ms) / len(peaks_ms)
        mh_bytes = 4 * cells
        fill_bytes = mh_bytes + 12 * n_hits        # store every cell once + read the hits
        peaks_bytes = mh_bytes + 12 * n_found      # read every cell once + write the peak list
        roof = {}
        for name, nbytes, avg in (("ht_fill (classify_bucket + fill_slab)", fill_bytes, fill_avg),
                                  ("ht_peaks (peaks_kernel)", peaks_bytes, peaks_avg)):
            ach = nbytes / (avg * 1e-3) / 1e9
            roof[name] = {"bound": "hbm", "achieved": ach, "peak": peak_gbs, "unit": "GB/s", "frac": ach / peak_gbs,
                          "traffic": None, "kernel": name, "algorithmic_bytes_per_launch": nbytes,
                          "avg_ms_per_launch": avg, "peak_source": peak_src}
        dominant = max(roof.values(), key=lambda r: r["avg_ms_per_launch"])
        other = min(roof.values(), key=lambda r: r["avg_ms_per_launch"])

        # ---- cpu_baseline (oracle, 1 core) on the same event + parity of this very launch configuration
        reps = 3
        o_times = []
        for _ in range(reps):
            m_ref, pk_ref, votes, tf, tp = run_oracle_event(bn, batch, wl.threshold)
            o_times.append((tf, tp))
        got_m = mhs[(args.steps - 1) % n_rot].cpu().numpy().view(np.uint32).reshape(m_ref.shape)
        k = min(n_found, cap)
        rec = d_out[:3 * k].cpu().numpy().view(np.uint32).reshape(k, 3)
        order = np.argsort(rec[:, 1].astype(np.int64), kind="stable")
        parity = bool(np.array_equal(got_m, m_ref) and n_found == len(pk_ref) and n_e2e == len(pk_ref)
                      and np.array_equal(rec[order, 1], pk_ref["cell"]) and np.array_equal(rec[order, 2], pk_ref["count"]))
        o_fill = statistics.median(t[0] for t in o_times)
        o_peaks = statistics.median(t[1] for t in o_times)
        info = B.ht_launch_info(ctx)
        line = {
            "metric": METRIC, "value": value, "unit": "events/s", "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "u32 counts / f32 bin decisions", "data": "synthetic",
            "config": {"workload": f"config{wl.config}:{wl.name}", "bins": [bn.n_theta, bn.n_phi, bn.n_a, bn.n_b],
                       "hits_per_event": n_hits, "threshold": wl.threshold, "events_per_step": 1,
                       "l2": f"M_H per event ({mh_bytes / 1e6:.0f} MB) vs 126 MB L2; {n_rot} output matrices rotated so "
                             "no step inherits another step's lines",
                       "launch": info},
            "votes_per_s": votes * value, "votes_per_event": votes, "peaks_per_event": n_found,
            "hit_a_evaluations_per_s": n_hits * bn.n_a * value,
            "parity_vs_oracle": "bit-exact" if parity else "MISMATCH",
            "kernel_ms": {"fill_median": fill_med, "fill_mean": fill_avg, "peaks_median": peaks_med,
                          "peaks_mean": peaks_avg, "step_mean": ms_per_step},
            "roofline": dominant, "roofline_other": other,
            "cpu_baseline": {"value": 1.0 / (o_fill + o_peaks), "unit": "events/s", "cores": 1, "kind": "oracle",
                             "sample": f"median of {reps} runs of the same full event (fill {o_fill * 1e3:.0f} ms + "
                                       f"peaks {o_peaks * 1e3:.0f} ms), single thread, host of the GPU box",
                             "host_cpus": os.cpu_count()},
            "e2e": {"value": e2e_value, "unit": "events/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": 1e3 * e2e_s / e2e_steps, "api": "ht_run_host (pinned host buffers)"},
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
    ap.add_argument("--config", type=int, default=2, choices=[1, 2, 4])
    ap.add_argument("--rotate", type=int, default=4, help="number of output matrices rotated between steps")
    args = ap.parse_args()
    if args.impl == "reference":
        args.steps = 10 if args.steps is None else args.steps
        args.warmup = 1 if args.warmup is None else args.warmup
        bench_reference(args)
    else:
        args.steps = 300 if args.steps is None else args.steps
        args.warmup = 10 if args.warmup is None else args.warmup
        bench_ours(args)


if __name__ == "__main__":
    main()

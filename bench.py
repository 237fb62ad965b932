#!/usr/bin/env python
"""bench.py -- events/s and Hough votes/s of the fill + peak-search hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2] [--events E]

A STEP is one pass of the whole hot path (classify, vote, store, peak test + compaction: SURVEY.md section 8(a) a0-a5)
over one event of the workload (default: config 2, the paper-shaped 5000-hit event, 4x16x1024x1024 bins; --events E:
a batch of E events per step), i.e. ONE ht_fill_peaks call = one kernel.

value     events/s with the hits already resident in HBM: W warm-up steps, then brackets of exactly K steps between
          barrier + synchronize, CUDA events on the launch stream, max over ranks; the headline is the MEDIAN of
          `--reps` (5) such brackets of plain stream launches (fixed rule, stated in config.launch_mode; the same calls
          replayed from a CUDA graph and the two-kernel split are reported beside it, each with its own median).
e2e       the same metric through the C ABI with HOST buffers: ht_submit_host / ht_wait_host over the context's pinned
          slots (hits cross PCIe inside the timed region, count and peak list come back the same way).
roofline  achieved = algorithmic bytes of one call (the matrix once + hits + peaks) / the call's average
          duration in the timed region; peak = MEASURED_PEAKS.json; store ceilings (cudaMemsetAsync of the same output
          matrices) measured in the same run; traffic from profiles/r02_traffic.csv (an ncu capture) when it matches.
cpu_baseline  the CPU oracle as it stands on one core of this box (also the parity check of this very run), plus the
          same oracle on all cores, one event per process.
N > 1 (torchrun): every rank its own events, no data-path collective ("weak"); `--split planes`: all ranks the same
events and a range of (theta, phi) planes each ("strong").  After the timed region the ranks' peak lists are
gathered over NCCL and rank 0 checks the merged list against the oracle (`merged_parity`).
`--impl reference` times the CPU oracle itself (there is no reference implementation of the paper to install).
"""
from __future__ import annotations

import argparse
import json
import math
import os
import statistics
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "events/s and Hough votes/s (fill+peak search), 5000-hit event, 1 B200"
DTYPE = "u32 counts / f32 bin decisions"
FALLBACK_HBM_GBS = 6650.0          # /opt/skills/guides/B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
SM_COUNT, SM_LANES, SM_GHZ = 148, 128, 1.965     # ALU roofline of the vote loop (B200_PROFILING.md: 148 SMs, 1965 MHz)
VOTE_INSTR_PER_EVAL = 20           # issued instructions per (hit, A row) evaluation of the vote loop (SASS count)


def measured_hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json: bf16 copy, read+write)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def workload_config(wl, n_hits, n_ev):
    """The `config` block: BOTH arms print exactly this dict (same keys, same values) for the same workload and flags."""
    bn = wl.binning
    m_bytes = 4 * bn.cells * n_ev
    return {"workload": f"config{wl.config}:{wl.name}", "bins": [bn.n_theta, bn.n_phi, bn.n_a, bn.n_b],
            "hits_per_step": int(n_hits), "events_per_step": int(n_ev), "threshold": int(wl.threshold),
            "l2": f"M_H per step ({m_bytes / 1e6:.0f} MB) is larger than the 126 MB L2, and the CUDA arm rotates its output "
                  "matrices, so no step inherits another step's lines",
            "launch_mode": "CUDA arm: plain stream launches (fixed rule), median of the --reps brackets of exactly --steps calls each; "
                           "reference arm: the CPU oracle as it stands, one thread, the --steps steps timed in one bracket"}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.001):
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


def run_oracle_event(bn, xyz, threshold):
    """One event through the CPU oracle: (matrix, peaks, votes, seconds fill, seconds peaks)."""
    from oracle import oracle_fill, oracle_peaks
    t0 = time.perf_counter()
    m, votes = oracle_fill(bn, *xyz)
    t1 = time.perf_counter()
    pk = oracle_peaks(bn, m, threshold)
    t2 = time.perf_counter()
    return m, pk, votes, t1 - t0, t2 - t1


def _oracle_worker(job):
    """One process of the all-cores CPU line: `reps` events of the workload through the oracle, wall time of the loop."""
    cfg_id, event, reps = job
    sys.path.insert(0, ROOT)
    from paper_1507_03074_b200.events import WORKLOADS, generate_batch
    wl = WORKLOADS[cfg_id]
    batch = generate_batch(wl, n_events=1, first_event=event)
    run_oracle_event(wl.binning, batch.event(0), wl.threshold)            # warm-up (page faults of the matrix)
    t0 = time.perf_counter()
    for _ in range(reps):
        run_oracle_event(wl.binning, batch.event(0), wl.threshold)
    return time.perf_counter() - t0


def oracle_all_cores(cfg_id: int, reps: int):
    """The oracle as it stands on every host core at once, one event per process (events are independent: R14)."""
    import concurrent.futures as cf
    import multiprocessing as mp
    cores = os.cpu_count() or 1
    from paper_1507_03074_b200.events import WORKLOADS
    wl_bytes = 4 * WORKLOADS[cfg_id].binning.cells
    workers = max(1, min(cores, int((24 << 30) // max(wl_bytes, 1))))       # bound the host memory the matrices take
    t0 = time.perf_counter()
    with cf.ProcessPoolExecutor(max_workers=workers, mp_context=mp.get_context("spawn")) as ex:
        spans = list(ex.map(_oracle_worker, [(cfg_id, e, reps) for e in range(workers)]))
    wall = time.perf_counter() - t0
    return {"value": workers * reps / max(spans), "unit": "events/s", "cores": workers, "kind": "oracle, one event per process",
            "sample": f"{workers} processes x {reps} events of this workload, slowest process {max(spans):.2f} s "
                      f"(pool incl. start-up {wall:.1f} s)"}


def bench_reference(args):
    """--impl reference: the CPU oracle as it stands on this box's host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1507_03074_b200.events import WORKLOADS, generate_batch
    wl = WORKLOADS[args.config]
    n_ev = args.events if args.events else 1
    batch = generate_batch(wl, n_events=n_ev)
    for _ in range(max(args.warmup, 0)):
        run_oracle_event(wl.binning, batch.event(0), wl.threshold)
    votes = 0
    t_all = time.perf_counter()
    for _ in range(args.steps):
        votes = 0
        for e in range(n_ev):
            votes += run_oracle_event(wl.binning, batch.event(e), wl.threshold)[2]
    total = time.perf_counter() - t_all
    value = args.steps * n_ev / total
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "events/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": DTYPE, "data": "synthetic",
        "config": workload_config(wl, batch.n_hits, n_ev),
        "votes_per_s": votes * args.steps / total,
        "cpu_baseline": {"value": value, "unit": "events/s", "cores": 1, "kind": "oracle",
                         "sample": f"{args.steps} steps of {n_ev} full event(s) of this workload, single thread"},
        "e2e": {"value": value, "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def bench_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1507_03074_b200 import binding as B
    from paper_1507_03074_b200.events import WORKLOADS, generate_batch, truth_table
    from paper_1507_03074_b200.sharding import gather_peaks, plane_range

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
    # --split events (default): every rank its own events (weak scaling: the path shards by event, no data-path
    # collective).  --split planes: all ranks take the SAME events and a contiguous range of the (theta, phi) planes each
    # (strong scaling; the sector split of PAPER.md:77); again no collective in the timed region
    by_planes = args.split == "planes"
    first_event = 0 if by_planes else rank * n_ev
    batch = generate_batch(wl, n_events=n_ev, first_event=first_event)
    n_hits = batch.n_hits
    p0, pc = plane_range(bn.planes, rank, world) if by_planes else (0, bn.planes)
    cells = pc * bn.n_a * bn.n_b                                     # cells of this rank's matrix per event
    cap = 1 << 16
    host_slots = max(4, n_ev) if n_ev <= 8 else n_ev
    cfg = B.ht_config.from_binning(bn, max_events=n_ev, max_hits=n_hits, device=local_rank, host_slots=host_slots,
                                   host_peak_capacity=cap, plane_begin=p0 if by_planes else 0,
                                   plane_count=pc if by_planes else 0)
    ctx = B.ht_create(cfg)
    stream = torch.cuda.Stream(device=dev)

    to = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a)).to(dev, dtype=dt)
    dx, dy, dz = to(batch.x, torch.float32), to(batch.y, torch.float32), to(batch.z, torch.float32)
    doff = to(batch.event_offsets, torch.int32)
    mh_bytes = 4 * cells * n_ev
    n_rot = args.rotate if mh_bytes * args.rotate <= (48 << 30) else max(1, int((48 << 30) // mh_bytes))
    mhs = [torch.empty(cells * n_ev, dtype=torch.int32, device=dev) for _ in range(n_rot)]
    d_out = torch.empty(cap * 3, dtype=torch.int32, device=dev)
    d_nf = torch.zeros(1, dtype=torch.int32, device=dev)
    T = wl.threshold
    K, R = args.steps, max(args.reps, 1)
    # device cycles the gate kernel spins per queued call (~15 us each at 2 GHz: more than the host needs to enqueue one)
    gate_cycles = 0 if args.no_gate or not hasattr(torch.cuda, "_sleep") else 30000

    def step_fused(k):                                # a0-a5 in ONE kernel, matrix materialised
        B.ht_fill_peaks(ctx, dx, dy, dz, doff, n_ev, n_hits, mhs[k % n_rot], T, d_out, cap, d_nf, stream)

    def step_fill(k):
        B.ht_fill(ctx, dx, dy, dz, doff, n_ev, n_hits, mhs[k % n_rot], stream)

    def step_peaks(k):
        B.ht_peaks(ctx, mhs[k % n_rot], n_ev, T, d_out, cap, d_nf, stream)

    def step_split(k):                                # the paper's two-kernel split: ht_fill, then ht_peaks
        step_fill(k)
        step_peaks(k)

    def step_nostore(k):                              # peaks only: the matrix never leaves shared memory
        B.ht_fill_peaks(ctx, dx, dy, dz, doff, n_ev, n_hits, None, T, d_out, cap, d_nf, stream)

    def step_memset(k):                               # the driver's own way of writing the same bytes once
        B.ht_diag_memset(mhs[k % n_rot], 0, mh_bytes, stream)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def n_found_now():
        stream.synchronize()
        return int(d_nf.cpu().numpy().view(np.uint32)[0])

    def max_over_ranks(ms):
        if world > 1:
            t = torch.tensor([ms], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            return float(t.item())
        return ms

    def bracket(step, steps):
        """Exactly `steps` calls between barrier + synchronize; CUDA events on the launch stream; max over ranks.
        The stream first gets a short spin kernel, so that the calls are already queued when the first event fires: the
        bracket then times the device executing `steps` calls back to back, not the host enqueuing the first of them
        (~10 us after an idle stream, which a 20-step bracket would otherwise book as 0.5 us per step)."""
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        if gate_cycles:
            with torch.cuda.stream(stream):
                torch.cuda._sleep(gate_cycles * min(steps, 64))
        e0.record(stream)
        for k in range(steps):
            step(k)
        e1.record(stream)
        barrier()
        return max_over_ranks(e0.elapsed_time(e1)) / steps

    def timed(step, sampler=None, steps=K, reps=R):
        """W warm-up steps, then `reps` brackets of exactly `steps` steps: (median, all) ms per step."""
        for k in range(max(args.warmup, 3)):
            step(k)
        stream.synchronize()
        if sampler is not None and not sampler.is_alive():
            sampler.start()                                           # (keeps sampling until the last timed leg: see below)
        all_ms = [bracket(step, steps) for _ in range(reps)]
        return statistics.median(all_ms), all_ms

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
    res, launches_per_step = {}, {}
    l0 = B.ht_kernel_launches(ctx)
    if headline == "fused":
        res["fused"] = timed(step_fused, sampler)
    else:
        res["split"] = timed(step_split, sampler)
    launches = (B.ht_kernel_launches(ctx) - l0)                       # warm-up + R brackets of K steps
    launches_per_step = launches // (max(args.warmup, 3) + R * K)
    n_found = n_found_now()
    if headline == "fused":
        res["split"] = timed(step_split)
    elif fused_ok:
        res["fused"] = timed(step_fused)
    res["fill"] = timed(step_fill)
    res["peaks"] = timed(step_peaks)
    if fused_ok:
        res["nostore"] = timed(step_nostore)
    # store ceilings, same run, same rotated buffers: one matrix per launch, and >= 20 GB back to back
    res["memset"] = timed(step_memset)
    stream_steps = max(K, int(math.ceil((20 << 30) / mh_bytes)))
    res["memset_stream"] = timed(step_memset, steps=stream_steps, reps=3)
    # The same K calls captured once into a CUDA graph and replayed (the calls keep no host-side state)
    graph_ms = None
    if fused_ok and not args.no_graph:
        try:
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=stream):
                for k in range(K):
                    step_fused(k)
            graph.replay()                                            # warm-up replay
            reps_ms = []
            for _ in range(R):
                barrier()
                g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                g0.record()
                graph.replay()
                g1.record()
                barrier()
                reps_ms.append(max_over_ranks(g0.elapsed_time(g1)) / K)
            if n_found_now() == n_found:
                graph_ms = (statistics.median(reps_ms), reps_ms)
        except Exception as err:                                      # capture not supported here: stream launches stand
            print(f"bench.py: CUDA graph capture failed ({err!r}); timing stream launches only", file=sys.stderr)
    sampler.stop_flag = True                                          # clocks were sampled through every timed leg on the device
    # leave the headline path's outputs in the buffers for the parity check below
    last_k = K - 1
    (step_fused if headline == "fused" else step_split)(last_k)
    n_found = n_found_now()
    ms_per_step = res[headline][0]
    jobs = 1 if by_planes else world                                  # --split planes: all ranks work on the same events
    value = jobs * n_ev * 1e3 / ms_per_step                           # events/s over all ranks

    # ---- f3: track read-out, ridge merging, truth matching of the peak list (separate small kernels, not in the step)
    n_pk = min(n_found, cap)
    d_tr = torch.empty(5 * max(n_pk, 1), dtype=torch.int32, device=dev)
    d_cand = torch.empty(6 * max(n_pk, 1), dtype=torch.int32, device=dev)
    d_nc = torch.zeros(1, dtype=torch.int32, device=dev)
    scratch_bytes = B.ht_merge_scratch_bytes(n_pk)
    d_scr = torch.empty(scratch_bytes, dtype=torch.uint8, device=dev)
    window = args.merge_window

    def f3_calls():
        B.ht_tracks(ctx, d_out, n_pk, d_tr, stream)
        B.ht_merge_ridges(ctx, d_out, n_pk, window, d_cand, n_pk, d_nc, d_scr, scratch_bytes, stream)

    for _ in range(3):
        f3_calls()
    stream.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    for _ in range(50):
        f3_calls()
    ev1.record(stream)
    stream.synchronize()
    f3_ms = ev0.elapsed_time(ev1) / 50
    n_cand = int(d_nc.cpu().numpy().view(np.uint32)[0])
    tt = truth_table(batch, bn.n_theta, bn.n_phi)
    tr = np.zeros(len(tt["event"]), B.TRUTH_DTYPE)
    tr["event"], tr["a"], tr["b"] = tt["event"], tt["a"], tt["b"]
    d_truth = torch.from_numpy(tr.view(np.uint8).copy()).to(dev)
    d_cm = torch.zeros(max(n_cand, 1), dtype=torch.int32, device=dev)
    d_tm = torch.zeros(max(len(tr), 1), dtype=torch.int32, device=dev)
    d_sum = torch.zeros(B.SUMMARY_DTYPE.itemsize, dtype=torch.uint8, device=dev)
    dA = (bn.a_max - bn.a_min) / bn.n_a
    w_rho, w_phi = args.match_cells * dA, args.match_phi
    B.ht_match_truth(ctx, d_cand, n_cand, d_truth, len(tr), w_rho, math.cos(w_phi), d_cm, d_tm, d_sum, stream)
    stream.synchronize()
    ms = d_sum.cpu().numpy().view(B.SUMMARY_DTYPE)[0]
    tm = d_tm.cpu().numpy()[:len(tr)]
    in_range = (tt["a"] >= bn.a_min) & (tt["a"] < bn.a_max) & (tt["b"] >= bn.b_min) & (tt["b"] < bn.b_max)
    findable = in_range & (tt["max_sector_hits"] >= T)
    nf_found = int(ms["n_found"])
    tracking = {
        "what": "ht_tracks + ht_merge_ridges + ht_match_truth on the step's peak list against the generator's circles "
                "(SPEC.md sections 4-6; stand-in for PAPER.md:29-33, Fig. 1)",
        "merge_window_cells": window, "match_window_rho_mm": w_rho, "match_window_phi_rad": w_phi,
        "peaks": n_pk, "candidates": n_cand, "generated_tracks": int(len(tr)),
        "tracks_centre_in_AB_range": int(in_range.sum()),
        "tracks_findable": int(findable.sum()),
        "findable_means": f"centre inside the (A,B) range and >= {T} of the track's hits in one (theta,phi) sector (reading R2)",
        "found": nf_found, "found_findable": int((tm[findable] >= 0).sum()),
        "efficiency_all": nf_found / max(len(tr), 1),
        "efficiency_findable": float((tm[findable] >= 0).sum()) / max(int(findable.sum()), 1),
        "fake_rate": int(ms["n_fake"]) / max(n_cand, 1), "duplicates": int(ms["n_duplicate"]),
        "rho_residual_rms_mm": math.sqrt(float(ms["sum_drho2"]) / nf_found) if nf_found else None,
        "phi_residual_rms_rad": math.sqrt(float(ms["sum_dphi2"]) / nf_found) if nf_found else None,
        "ms_per_call_tracks_plus_merge": f3_ms,
    }

    # ---- end to end through the host entry points: pinned host buffers, hits in and peaks out inside the timed region
    hx, hy, hz = (torch.from_numpy(a.copy()).pin_memory() for a in (batch.x, batch.y, batch.z))
    houts = [torch.zeros(cap * 3, dtype=torch.int32).pin_memory()]

    # K steps of n_ev events each as ONE sequence in host memory (every step's hits are separate host bytes that cross
    # PCIe); the library pipelines the sequence over the context's slots: one fused kernel per event
    seq_events = K * n_ev
    hx_seq, hy_seq, hz_seq = (torch.from_numpy(np.tile(a, K)).pin_memory() for a in (batch.x, batch.y, batch.z))
    per_ev = np.diff(batch.event_offsets.astype(np.int64))
    hoff_seq = torch.from_numpy(np.concatenate([[0], np.cumsum(np.tile(per_ev, K))]).astype(np.int32))
    e2e_cap = min(cap, 4096)
    hout_seq = torch.zeros(seq_events * e2e_cap * 3, dtype=torch.int32).pin_memory()
    hnf_seq = torch.zeros(seq_events, dtype=torch.int32)

    def e2e_pipeline():
        B.ht_run_host_events(ctx, hx_seq, hy_seq, hz_seq, hoff_seq, seq_events, T, hout_seq, e2e_cap, hnf_seq)
        return hnf_seq.numpy().view(np.uint32)

    e2e_pipeline()
    e2e_reps = []
    for _ in range(R):
        barrier()
        t0 = time.perf_counter()
        nf_seq = e2e_pipeline()
        e2e_reps.append(max_over_ranks((time.perf_counter() - t0) * 1e3) / K)
    n_e2e = int(nf_seq[:n_ev].sum())
    e2e_consistent = bool(np.array_equal(nf_seq, np.tile(nf_seq[:n_ev], K)))
    e2e_ms = statistics.median(e2e_reps)
    # the synchronous call for comparison (ht_run_host: submit + wait, one event at a time)
    hoff_t = torch.from_numpy(batch.event_offsets.copy())
    for _ in range(3):
        B.ht_run_host(ctx, hx, hy, hz, hoff_t, n_ev, n_hits, T, houts[0], cap)
    t0 = time.perf_counter()
    for _ in range(K):
        B.ht_run_host(ctx, hx, hy, hz, hoff_t, n_ev, n_hits, T, houts[0], cap)
    e2e_sync_ms = max_over_ranks((time.perf_counter() - t0) * 1e3) / K
    e2e_value = jobs * n_ev * 1e3 / e2e_ms
    # per event: the packed input block [2 offsets | x | y | z] + the submission's number, copied to the device on the copy
    # stream (or, for events too large for early tiles, read by the kernel from the pinned block: the same hit bytes); back:
    # the result header + the head of the peak list (at most 4096 records, whatever the list holds), by the copy engine
    h2d = 3 * 4 * n_hits + n_ev * (8 + 4)
    d2h = n_ev * (16 + 12 * min(cap, 4096))

    # ---- N > 1: merge the ranks' peak lists over NCCL ("eventually the results are merged"), outside the timed region
    k_out = min(n_found, cap)
    rec = d_out[:3 * k_out].cpu().numpy().view(np.uint32).reshape(k_out, 3)
    local_pk = np.empty(k_out, B.PEAK_DTYPE)
    local_pk["event"], local_pk["cell"], local_pk["count"] = rec[:, 0], rec[:, 1], rec[:, 2]
    merged = gather_peaks(local_pk, 0 if by_planes else rank * n_ev, bn.cells, device=dev if world > 1 else None)

    if rank == 0:
        peak_gbs, peak_src = measured_hbm_peak()
        m_bytes = 4 * cells * n_ev
        hit_bytes, pk_bytes = 12 * n_hits, 12 * n_found

        traffic, traffic_src = {}, None
        try:
            import csv
            with open(os.path.join(ROOT, "profiles", "r02_traffic.csv"), newline="") as f:
                for row in csv.DictReader(f):
                    if row["workload"] == f"config{wl.config}:{wl.name}" and int(row["events_per_step"]) == n_ev and world == 1:
                        traffic[row["entry_point"]] = float(row["dram_bytes_per_launch"])
                        traffic_src = row["source"]
        except Exception:
            pass

        def roof(name, nbytes, ms, key):
            ach = nbytes / (ms * 1e-3) / 1e9
            return {"bound": "hbm", "achieved": ach, "peak": peak_gbs, "unit": "GB/s", "frac": ach / peak_gbs,
                    "traffic": traffic.get(key), "traffic_source": traffic_src if traffic.get(key) else None,
                    "kernel": name, "algorithmic_bytes_per_launch": nbytes, "avg_ms_per_launch": ms, "peak_source": peak_src}

        kernels = {}
        if "fused" in res:
            kernels["ht_fill_peaks"] = roof("fill_tiles_kernel<true> (ht_fill_peaks: classify, vote, store, peak test, compaction in one kernel)",
                                            m_bytes + hit_bytes + pk_bytes, res["fused"][0], "ht_fill_peaks")
        kernels["ht_fill"] = roof("fill_tiles_kernel<false> (ht_fill: classify, vote, store in one kernel)", m_bytes + hit_bytes,
                                  res["fill"][0], "ht_fill")
        kernels["ht_peaks"] = roof("peaks_kernel (ht_peaks: scan + compaction)", m_bytes + pk_bytes, res["peaks"][0], "ht_peaks")
        dominant = dict(kernels["ht_fill_peaks"] if headline == "fused"
                        else max((kernels["ht_fill"], kernels["ht_peaks"]), key=lambda r: r["avg_ms_per_launch"]))
        dominant["store_ceiling_gbs"] = m_bytes / (res["memset"][0] * 1e-3) / 1e9
        dominant["store_ceiling_stream_gbs"] = m_bytes / (res["memset_stream"][0] * 1e-3) / 1e9
        dominant["store_ceiling_what"] = (f"cudaMemsetAsync of the same {n_rot} rotated output matrices, {m_bytes / 1e6:.0f} MB per launch: "
                                          f"median of {R} brackets of {K} launches, and of 3 brackets of {stream_steps} launches "
                                          f"({stream_steps * m_bytes / 2**30:.0f} GiB back to back)")
        dominant["frac_of_store_ceiling"] = dominant["achieved"] / dominant["store_ceiling_gbs"]

        # ---- cpu_baseline (oracle, 1 core) on event 0 + parity of this very launch configuration
        from oracle import oracle_fill, oracle_peaks
        reps_o, o_times, votes = 3, [], 0
        for _ in range(reps_o):
            m_ref, pk_ref, votes, tf, tp = run_oracle_event(bn, batch.event(0), T)
            o_times.append((tf, tp))
        got_all = mhs[last_k % n_rot].cpu().numpy().view(np.uint32).reshape(n_ev, -1)
        rec_s = rec[np.lexsort((rec[:, 1], rec[:, 0]))]
        lo_cell, hi_cell = p0 * bn.n_a * bn.n_b, (p0 + pc) * bn.n_a * bn.n_b     # this rank's part of the full matrix
        parity = bool(np.array_equal(got_all[0], m_ref.reshape(-1)[lo_cell:hi_cell]))
        n_ref, votes_all, full_lists = 0, 0, []
        for e in range(n_ev):
            if e == 0:
                m_e, pk_e, v_e = m_ref, pk_ref, votes
            else:
                m_e, v_e = oracle_fill(bn, *batch.event(e))
                pk_e = oracle_peaks(bn, m_e, T)
                parity = parity and bool(np.array_equal(got_all[e], m_e.reshape(-1)[lo_cell:hi_cell]))
            votes_all += v_e
            pk_full = pk_e.copy()
            pk_full["event"] = e
            full_lists.append(pk_full)
            pk_e = pk_e[(pk_e["cell"] >= lo_cell) & (pk_e["cell"] < hi_cell)]
            r_e = rec_s[rec_s[:, 0] == e]
            parity = parity and len(r_e) == len(pk_e) and bool(np.array_equal(r_e[:, 1], pk_e["cell"])
                                                                and np.array_equal(r_e[:, 2], pk_e["count"]))
            n_ref += len(pk_e)
        parity = parity and n_found == n_ref and n_e2e == n_ref and e2e_consistent
        # merged list of all ranks against the oracle (N > 1: the other ranks' events too)
        want_lists = list(full_lists)
        if world > 1 and not by_planes:
            for r in range(1, world):
                ob = generate_batch(wl, n_events=n_ev, first_event=r * n_ev)
                for e in range(n_ev):
                    m_o, _ = oracle_fill(bn, *ob.event(e))
                    pk_o = oracle_peaks(bn, m_o, T)
                    pk_o["event"] = r * n_ev + e
                    want_lists.append(pk_o)
        want_merged = np.concatenate(want_lists)
        merged_parity = bool(len(merged) == len(want_merged) and np.array_equal(merged["event"], want_merged["event"])
                             and np.array_equal(merged["cell"], want_merged["cell"])
                             and np.array_equal(merged["count"], want_merged["count"]))
        o_fill = statistics.median(t[0] for t in o_times)
        o_peaks = statistics.median(t[1] for t in o_times)
        cpu_all = None
        if not args.no_cpu_all_cores:
            try:
                cpu_all = oracle_all_cores(args.config, 2 if bn.cells <= (1 << 27) else 1)
            except Exception as err:
                cpu_all = {"unavailable": repr(err)}

        # ---- roofline of the vote loop (SURVEY.md 8(d) fill rows): ALU issue and shared-memory atomic rate, next to the HBM bound
        rates, rate_err = B.ht_diag_vote_rates(local_rank, 2000)
        evals = n_hits * bn.n_a
        r_atom = rates["atom_random"] if headline == "fused" else rates["red_random"]
        vote_roof = {
            "evaluations_per_step": evals, "votes_per_step": votes_all,
            "t_alu_us": evals * VOTE_INSTR_PER_EVAL / (SM_COUNT * SM_LANES * SM_GHZ * 1e3),
            "t_atomic_us": votes_all / (SM_COUNT * r_atom * SM_GHZ * 1e3),
            "t_hbm_us": m_bytes / peak_gbs / 1e3,
            "r_atom_lanes_per_clk_per_sm": {k: rates[k] for k in ("red_random", "atom_random", "red_no_conflict", "red_two_way",
                                                                   "red_same", "atom_no_conflict", "atom_same")},
            "r_atom_sum_errors": rate_err,
            "what": f"T_vote >= max(evals*{VOTE_INSTR_PER_EVAL} instr/({SM_COUNT} SMs*{SM_LANES} lanes*{SM_GHZ} GHz), votes/({SM_COUNT}*r_atom*f)); "
                    "r_atom measured in this run by ht_diag_vote_rates (30 warps of one CTA per SM voting into rows they own)",
        }
        vote_roof["bound_us"] = max(vote_roof["t_alu_us"], vote_roof["t_atomic_us"], vote_roof["t_hbm_us"])
        vote_roof["frac_of_slowest_bound"] = vote_roof["bound_us"] / (ms_per_step * 1e3)

        info = B.ht_launch_info(ctx)
        config = workload_config(wl, n_hits, n_ev)
        detail = {
            "path": ("ht_fill_peaks: one kernel does a0-a5 and stores every M_H cell once" if headline == "fused"
                     else "ht_fill + ht_peaks (two kernels)"),
            "rotated_output_matrices": n_rot,
            "bracket_gate": ("a spin kernel of ~15 us per queued call (at most 64) runs ahead of the first event of every bracket, so the "
                             "calls are queued when timing starts (device time of K back-to-back calls)" if gate_cycles
                             else "none: the host's enqueue latency of the first call is inside the bracket"),
            "launch": info,
        }
        spread = lambda v: {"median": statistics.median(v), "min": min(v), "max": max(v), "n": len(v)}
        line = {
            "metric": METRIC, "value": value, "unit": "events/s", "n_gpus": world, "steps": K,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "strong" if by_planes else "weak",
            "vs_baseline": None, "dtype": DTYPE, "data": "synthetic",
            "config": config, "config_detail": detail,
            "votes_per_s": votes_all * jobs * 1e3 / ms_per_step, "votes_per_step": votes_all, "peaks_per_step": n_found,
            "hit_a_evaluations_per_s": n_hits * bn.n_a * jobs * 1e3 / ms_per_step,
            "parity_vs_oracle": "bit-exact" if parity else "MISMATCH",
            "merged_parity": "bit-exact" if merged_parity else "MISMATCH",
            "ms_per_step_brackets": {name: spread(r[1]) for name, r in res.items()},
            "ms_per_step_graph_replay": spread(graph_ms[1]) if graph_ms else None,
            "paths_events_per_s": dict({name: jobs * n_ev * 1e3 / r[0] for name, r in res.items() if not name.startswith("memset")},
                                       **({"fused_graph": jobs * n_ev * 1e3 / graph_ms[0]} if graph_ms else {})),
            "roofline": dominant, "roofline_kernels": kernels, "roofline_vote": vote_roof,
            "cpu_baseline": {"value": 1.0 / (o_fill + o_peaks), "unit": "events/s", "cores": 1, "kind": "oracle",
                             "sample": f"median of {reps_o} runs of one full event of this workload (fill {o_fill * 1e3:.0f} ms + "
                                       f"peaks {o_peaks * 1e3:.0f} ms), single thread, host of the GPU box",
                             "host_cpus": os.cpu_count()},
            "cpu_baseline_all_cores": cpu_all,
            "e2e": {"value": e2e_value, "unit": "events/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": e2e_ms, "brackets": spread(e2e_reps), "slots": host_slots,
                    "sync_ms_per_step": e2e_sync_ms, "sync_events_per_s": jobs * n_ev * 1e3 / e2e_sync_ms,
                    "api": "ht_run_host_events: K steps' events as one sequence in host memory, one fused kernel per event, pipelined "
                           "by the library over its pinned slots (ht_submit_host / ht_wait_host: an asynchronous copy brings the "
                           "hits to the device and announces itself with a word the kernel waits for; count and peak list come back "
                           "through a copy stream that waits for the kernel's completion word; no event between two kernels, up to "
                           "`slots` events in flight); "
                           "sync_*: ht_run_host, one step at a time"},
            "tracking": tracking,
            "gpu_launches": int(launches_per_step * K),
            "gpu_launches_per_step": int(launches_per_step),
            "clocks": sampler.summary(),
        }
        print(json.dumps(line), flush=True)
        if not (parity and merged_parity):
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
    ap.add_argument("--reps", type=int, default=5, help="brackets of --steps steps each; the median is reported")
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", type=int, default=2, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--events", type=int, default=0, help="events per step (default 1)")
    ap.add_argument("--mode", choices=["fused", "split"], default="fused",
                    help="headline path: ht_fill_peaks (one kernel) or ht_fill + ht_peaks")
    ap.add_argument("--rotate", type=int, default=4, help="number of output matrices rotated between steps")
    ap.add_argument("--no-graph", action="store_true", help="skip the CUDA graph replay leg")
    ap.add_argument("--no-gate", action="store_true", help="no spin kernel ahead of a bracket (the host's first enqueue is timed too)")
    ap.add_argument("--no-cpu-all-cores", action="store_true", help="skip the all-cores CPU line")
    ap.add_argument("--split", choices=["events", "planes"], default="events",
                    help="N > 1: every rank its own events (weak scaling, default) or the same events split by plane")
    ap.add_argument("--merge-window", type=int, default=10, help="ridge-merging window in cells (SPEC.md section 5)")
    ap.add_argument("--match-cells", type=float, default=6.0, help="truth-matching window in rho, in A cells")
    ap.add_argument("--match-phi", type=float, default=0.03, help="truth-matching window in phi, rad")
    args = ap.parse_args()
    if args.impl == "reference":
        args.steps = 10 if args.steps is None else args.steps
        args.warmup = 1 if args.warmup is None else args.warmup
        bench_reference(args)
    else:
        args.steps = 500 if args.steps is None else args.steps
        args.warmup = 10 if args.warmup is None else args.warmup
        bench_ours(args)


if __name__ == "__main__":
    main()

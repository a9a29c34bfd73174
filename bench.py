#!/usr/bin/env python
"""bench.py -- the round-end measurement of the Hough track-finding hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C] [--tile-events T]
                    [--e2e-tile-events T2] [--streams S]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

A "step" is one pass of the WHOLE hot path (rows A1-A6 of SURVEY 8(a): stage -> vote -> flush -> find peaks
-> assign hits / remove duplicates) over one batch of seeded synthetic events.  The default workload is
BASELINE.json configs[3] (B:L10: 1024 events, uint16 256x128x32 accumulator per event) -- the configuration
the metric's "events/s" is quoted on; `--config` selects another one (0, 1, 2, 4) for inspection.

One JSON line goes to stdout (rank 0):
  value            whole-job Hough votes/s, inputs resident in HBM before the timed region, all ranks
  events_per_s     the same step expressed in events/s (the metric's second figure)
  e2e              the same metric through hough_pipeline_run_host (T2-event tiles on S streams, CUDA graphs): pinned
                   HOST buffers in, HOST results out, host<->device copies inside the timed region
  roofline         hough_vote: algorithmic votes per launch / average launch duration (CUDA events on the launching
                   stream, inside the timed region) against the LOWEST of three ceilings, picked by rule in the run:
                   ALU issue, shared-memory atomics (hough_microbench, measured in this process), HBM
                   (MEASURED_PEAKS.json); all three fractions are in the object
  roofline_assign  hough_assign_hits and hough_find_peaks timed the same way (per-position ALU ceiling; HBM bytes)
  roofline_peaks
  cpu_baseline     the CPU oracle as it stands, one thread, on a bounded sample of the same workload
  --impl reference times the oracle instead (this tier's reference arm).

Multi-GPU: events are independent, so every rank runs the same number of events of its own
(event indices offset by rank), no data-path collective; "scaling": "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "hough_votes_per_s"
UNIT = "votes/s"

# ALU issue bound of the vote step: the D3 sequence per (hit, phi0 column, d0 slice)
# is 9 fp32 arithmetic operations + 2 compares + 1 float->int conversion = 12 issue slots at the very least
# (the atomic goes down the LSU pipe in parallel); 148 SMs x 128 fp32 lanes x sm_max_mhz.
D3_MIN_ISSUE_SLOTS = 12
FP32_LANES_PER_SM = 128


def _env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


class ClockSampler:
    """nvidia-smi clocks + throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.index)], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def mark(self):
        return time.time()

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        rows = [l for (t, l) in self.lines if t0 - 0.05 <= t <= t1 + 0.15] or [l for (_, l) in self.lines]
        sm, smax, power, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for l in rows:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def _physical_gpu_index(local_rank: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
    ids = [x.strip() for x in vis.split(",") if x.strip()]
    if local_rank < len(ids) and ids[local_rank].isdigit():
        return int(ids[local_rank])
    return local_rank


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), float(p.get("sm_max_mhz", 1965.0)), "measured (MEASURED_PEAKS.json)"
    return 6650.0, 1965.0, "fallback (B200_PROFILING.md)"


def load_traffic():
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu --set full capture
    (profiles/r3_traffic.csv: kernel,tile_events,dram_bytes; the command is in profiles/r3_traffic.md).  ({}, None) if absent."""
    path = os.path.join(ROOT, "profiles", "r3_traffic.csv")
    tab = {}
    if not os.path.exists(path):
        return tab, None
    stamp = "unknown commit"
    with open(path) as f:
        for line in f:
            p = [x.strip() for x in line.split(",")]
            if len(p) >= 3 and p[0] == "# captured_at":
                stamp = "kernels as of commit %s, %s" % (p[1], p[2].split(" ")[0])
            elif len(p) >= 3 and p[1].isdigit():
                tab[(p[0], int(p[1]))] = float(p[2])
    return tab, ("profiles/r3_traffic.csv (ncu --set full capture of this launch configuration, %s -- NOT measured in this "
                 "run: stale if walk.cuh / peaks.cu changed since; see profiles/r3_traffic.md)" % stamp)


# ----------------------------------------------------------------------------------------------
def shard_event_range(rank: int, events_per_rank: int) -> range:
    """events are independent units, so rank r owns events [r * n, (r + 1) * n) of the workload's
    event sequence (weak scaling: n is fixed per GPU); no data-path collective follows."""
    return range(rank * events_per_rank, (rank + 1) * events_per_rank)


def reduce_job(ms_total: float, votes: float, events: float, hits: float, world: int, device):
    """Whole-job figures from per-rank ones: time = MAX over ranks, work = SUM over ranks (the only collectives
    of the bench; the data path has none)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms_total], dtype=torch.float64, device=device)
    v = torch.tensor([float(votes), float(events), float(hits)], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(v, op=dist.ReduceOp.SUM)
    return float(t.item()), tuple(float(x) for x in v.tolist())


def make_batch(cfg: int, n_events: int, rank: int):
    from workloads import generate_events, get_workload
    w = get_workload(cfg)
    if w.n_events > 1 or n_events != w.n_events:
        w = w.scaled(n_events)
    batch = generate_events(w, events=shard_event_range(rank, n_events))
    return w, batch


def oracle_sample(w, batch, n_sample_events: int):
    """The oracle, as it stands, single-threaded, on the first n_sample_events events: vote (full scan) +
    peaks + indexed assignment.  Returns (votes, events, seconds)."""
    from oracle import Oracle
    sub = batch.select(list(range(min(n_sample_events, batch.n_events))))
    o = Oracle.from_binning(w.binning, w.bz_tesla)
    # the CPU baseline is timed on ONE core -- this thread is pinned to the core it is on for the duration
    # (the oracle is single-threaded anyway; pinning only stops migrations) and released afterwards.
    saved = None
    try:
        saved = os.sched_getaffinity(0)
        os.sched_setaffinity(0, {sorted(saved)[-1]})
    except (AttributeError, OSError):
        saved = None
    try:
        t0 = time.perf_counter()
        votes_total = 0
        for e in range(sub.n_events):          # one event at a time keeps the oracle's int32 volume small
            ev = sub.select([e])
            acc, votes = o.vote(ev.hits_xy, ev.event_offsets)
            cands = o.find_peaks(acc, w.threshold)
            o.assign_indexed(ev.hits_xy, ev.event_offsets, cands, w.assoc_dj, w.min_hits)
            votes_total += votes
        secs = time.perf_counter() - t0
    finally:
        if saved is not None:
            os.sched_setaffinity(0, saved)
    return votes_total, sub.n_events, secs


def oracle_events_for_seconds(w, target_s: float) -> int:
    """Bounded sample size: ~target_s of single-thread oracle work, from the full-scan evaluation count
    (2 scans: vote + indexed assignment) at ~6.5e8 evaluations/s (measured on the GPU box's host, profiles/)."""
    bn = w.binning
    hits_per_event = (w.n_prompt + w.n_displaced) * len(w.layers) + max(w.n_noise, 0)
    per_event_s = 2.0 * hits_per_event * bn.n_phi * bn.n_d0 / 6.5e8 + bn.n_bins / 2.0e8
    return max(1, min(w.n_events, int(target_s / max(per_event_s, 1e-6))))


def run_reference(args, rank, world):
    """--impl reference: this tier's reference arm is the CPU oracle, timed as it stands on the host cores."""
    if rank != 0:
        return
    from workloads import get_workload
    w = get_workload(args.config)
    n_ev = oracle_events_for_seconds(w, args.ref_seconds_per_step)
    wl, batch = make_batch(args.config, n_ev, 0)
    for _ in range(min(args.warmup, 1)):
        oracle_sample(wl, batch, 1)
    votes = 0
    secs = 0.0
    for _ in range(args.steps):
        v, _, s = oracle_sample(wl, batch, n_ev)
        votes += v
        secs += s
    value = votes / secs
    sample = f"{n_ev} event(s) of {wl.name} per step, vote (full scan) + peaks + indexed assignment"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32+int32",
            "data": "synthetic", "events_per_s": n_ev * args.steps / secs,
            "config": {"workload": wl.name, "cite": wl.cite, "events_per_step": n_ev,
                       "note": "bounded sample of the workload; oracle single-threaded"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample, "pinned_to_one_core": True},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------------
class DeviceRun:
    """All device buffers of one rank and the tile loop over the three C-ABI calls."""

    def __init__(self, w, batch, tile_events: int, cand_per_bin: float):
        import torch
        from paper_1311_2769_b200 import HoughPlan, alloc_candidates
        self.torch = torch
        self.w, self.batch = w, batch
        bn = w.binning
        self.n_events = batch.n_events
        self.tile_events = max(1, min(tile_events, self.n_events))
        off = batch.event_offsets.astype(np.int64)
        self.tiles = []
        for e0 in range(0, self.n_events, self.tile_events):
            e1 = min(e0 + self.tile_events, self.n_events)
            self.tiles.append((e0, e1, int(off[e0]), int(off[e1])))
        max_hits = max(h1 - h0 for (_, _, h0, h1) in self.tiles)
        self.plan = HoughPlan.from_workload(w, max_hits=max(max_hits, 1), max_events=self.tile_events)
        self.plan.set_option("reuse_staging", 1)     # vote and assign_hits of a tile get the same device hits (include/hough.h)
        self.d_hits = torch.from_numpy(batch.hits_xy).cuda()
        # per-tile offsets are relative to the tile's first hit
        self.d_offs = []
        for (e0, e1, h0, _) in self.tiles:
            self.d_offs.append(torch.from_numpy((off[e0:e1 + 1] - h0).astype(np.int32)).cuda())
        self.accum = self.plan.alloc_accum(self.tile_events)
        self.cap = int(cand_per_bin * bn.n_bins * self.tile_events) + 1024
        self.cands = alloc_candidates(self.cap)
        self.cand_off = torch.zeros(self.tile_events + 1, dtype=torch.int32, device="cuda")
        self.h2c = torch.empty(max(max_hits, 1), dtype=torch.int32, device="cuda")
        self.nh = torch.empty(self.cap, dtype=torch.int32, device="cuda")
        self.keep = torch.empty(self.cap, dtype=torch.uint8, device="cuda")
        self.totals = torch.zeros(len(self.tiles), dtype=torch.int32, device="cuda")

    def step_tile(self, t, call_events=None):
        """vote -> find_peaks -> assign_hits of tile t on the current stream.  call_events: dict of lists
        {"vote", "peaks", "assign"} to append (start, end) CUDA events bracketing each C-ABI call."""
        torch = self.torch
        w = self.w
        (e0, e1, h0, h1) = self.tiles[t]
        hits = self.d_hits[h0:h1]
        offs = self.d_offs[t]
        n_ev = e1 - e0

        def timed(name, fn):
            if call_events is None:
                fn()
                return
            a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
            a.record(); fn(); b.record()
            call_events[name].append((a, b))

        timed("vote", lambda: self.plan.vote(hits, offs, self.accum))
        timed("peaks", lambda: self.plan.find_peaks(self.accum, n_ev, w.threshold, self.cands, self.cap, self.cand_off))
        timed("assign", lambda: self.plan.assign_hits(hits, offs, self.cands, self.cand_off, self.cap, w.assoc_dj,
                                                      w.min_hits, self.h2c[:max(h1 - h0, 1)], self.nh, self.keep))
        self.totals[t:t + 1].copy_(self.cand_off[n_ev:n_ev + 1])

    def reassign_tile(self, t):
        """hough_reassign_hits (D12) on tile t, after step_tile(t) left its D9 outputs on the device."""
        (e0, e1, h0, h1) = self.tiles[t]
        self.plan.reassign_hits(self.d_hits[h0:h1], self.d_offs[t], self.cands, self.cand_off, self.cap, self.w.assoc_dj, 2,
                                self.h2c[:max(h1 - h0, 1)], self.nh, self.keep)

    def step(self, call_events=None):
        """One pass over all tiles on the current stream."""
        for t in range(len(self.tiles)):
            self.step_tile(t, call_events)

    def count_votes(self) -> int:
        """Votes cast per step = sum of all accumulator bins (counted once, outside the timed region)."""
        torch = self.torch
        total = 0
        for t, (e0, e1, h0, h1) in enumerate(self.tiles):
            self.plan.vote(self.d_hits[h0:h1], self.d_offs[t], self.accum)
            n_ev = e1 - e0
            total += int(self.accum[:n_ev].to(torch.int64).sum().item())
        return total


def e2e_pipeline(run: DeviceRun, steps: int, warmup: int, n_streams: int, tile_events: int, cand_per_bin: float,
                 kept_only: bool = False):
    """End-to-end through the library's batched path (hough_pipeline_run_host): pinned HOST buffers in (hits, offsets)
    and out (hit_to_cand, cand_offsets, candidate records, nhits, keep); every host<->device copy is inside the
    timed region.  Wall-clock around the blocking call (it returns when the results are in the host buffers)."""
    torch = run.torch
    from paper_1311_2769_b200 import HoughPipeline
    w, batch = run.w, run.batch
    tile_events = max(1, min(tile_events, batch.n_events))
    off = batch.event_offsets.astype(np.int64)
    n_tiles = (batch.n_events + tile_events - 1) // tile_events
    max_hits = max(int(off[min(e0 + tile_events, batch.n_events)] - off[e0]) for e0 in range(0, batch.n_events, tile_events))
    tile_cap = int(cand_per_bin * w.binning.n_bins * tile_events) + 1024
    pipe = HoughPipeline.from_workload(w, tile_events, max(max_hits, 1), tile_cap, n_streams)
    if kept_only:
        pipe.set_option("kept_only", 1)
    total_cap = int(sum(int(t) for t in run.totals.tolist())) + 1024
    h_hits = torch.from_numpy(batch.hits_xy).pin_memory()
    h_off = torch.from_numpy(batch.event_offsets.astype(np.int32)).pin_memory()
    out_h2c = torch.empty(max(batch.n_hits, 1), dtype=torch.int32).pin_memory()
    out_off = torch.empty(batch.n_events + 1, dtype=torch.int32).pin_memory()
    out_cands = torch.empty((total_cap, 32), dtype=torch.uint8).pin_memory()
    out_nh = torch.empty(total_cap, dtype=torch.int32).pin_memory()
    out_keep = torch.empty(total_cap, dtype=torch.uint8).pin_memory()

    def one_step():
        return pipe.run_host(h_hits, h_off, w.threshold, w.assoc_dj, w.min_hits, out_h2c[:batch.n_hits], out_off, out_cands,
                             total_cap, out_nh, out_keep)

    for _ in range(max(warmup, 1)):
        one_step()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    over = False
    for _ in range(steps):
        over = one_step() or over
    torch.cuda.synchronize()
    ms = 1e3 * (time.perf_counter() - t0) / steps
    n_c = int(out_off[batch.n_events])
    h2d = batch.n_hits * 8 + (batch.n_events + n_tiles) * 4
    d2h = (batch.n_events + n_tiles) * 4 + batch.n_hits * 4 + min(n_c, total_cap) * (32 + 4 + 1)
    if kept_only:                                        # two offset arrays per tile; keep flags are not copied
        d2h = 2 * (batch.n_events + n_tiles) * 4 + batch.n_hits * 4 + min(n_c, total_cap) * (32 + 4)
    pipe.close()
    return ms, h2d, d2h, over


def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_1311_2769_b200 import kernel_launches, load_library, version

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (libhough_b200 has no CPU fallback)")
    load_library()
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    from workloads import get_workload
    w0 = get_workload(args.config)
    n_events = args.events if args.events > 0 else w0.n_events
    w, batch = make_batch(args.config, n_events, rank)
    run = DeviceRun(w, batch, args.tile_events, args.cand_per_bin)
    votes_per_step = run.count_votes()
    torch.cuda.synchronize()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        run.step()
    barrier()
    sampler = ClockSampler(_physical_gpu_index(local_rank))
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    barrier()
    call_events = {"vote": [], "peaks": [], "assign": []}
    launches0 = kernel_launches()
    t_mark0 = time.time()
    ev0 = torch.cuda.Event(enable_timing=True); ev1 = torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(args.steps):
        run.step(call_events)
    ev1.record()
    barrier()
    t_mark1 = time.time()
    launches = kernel_launches() - launches0
    ms_total = ev0.elapsed_time(ev1)
    clocks = sampler.stop(t_mark0, t_mark1) if rank == 0 else None
    call_ms = {k: [a.elapsed_time(b) for (a, b) in v] for k, v in call_events.items()}
    vote_ms = call_ms["vote"]
    peaks_overflow = bool((run.totals > run.cap).any().item())

    # max over ranks (device time), whole-job totals
    ms_job, (job_votes, job_events, job_hits) = reduce_job(ms_total, votes_per_step, batch.n_events, batch.n_hits, world, "cuda")
    ms_step = ms_job / args.steps

    # e2e leg (host buffers in and out), same workload
    e2e_ms, h2d, d2h, e2e_over = e2e_pipeline(run, max(1, min(args.steps, args.e2e_steps)), 1, args.streams, args.e2e_tile_events,
                                                args.cand_per_bin)
    k_ms, k_h2d, k_d2h, k_over = e2e_pipeline(run, max(1, min(args.steps, args.e2e_steps)), 1, args.streams,
                                              args.e2e_tile_events, args.cand_per_bin, kept_only=True)
    te = torch.tensor([e2e_ms, k_ms], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(te, op=dist.ReduceOp.MAX)
    e2e_ms, k_ms = (float(x) for x in te.tolist())

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    hbm_gbs, sm_max_mhz, peak_src = load_peaks()
    sms = torch.cuda.get_device_properties(local_rank).multi_processor_count
    bn = w.binning
    n_launch = len(run.tiles) * args.steps
    votes_per_launch = votes_per_step / len(run.tiles)
    hits_per_launch = batch.n_hits / len(run.tiles)
    bins_per_launch = bn.n_bins * run.tile_events
    cands_per_launch = float(run.totals.sum().item()) / len(run.tiles)

    # Ceilings measured in THIS process on THIS GPU (hough_microbench, outside the timed region): conflict-free and
    # random-address shared-memory atomicAdd rates, and the issue rate of the exact D3 sequence.
    from paper_1311_2769_b200 import microbench
    mb = {"smem_atomic_conflict_free_gops": microbench(0, 0, 5) / 1e9, "smem_atomic_random_gops": microbench(1, 0, 5) / 1e9,
          "d3_exact_eval_gops": microbench(4, 0, 5) / 1e9}
    traffic_tab, traffic_src = load_traffic()

    def avg(name):
        return sum(call_ms[name]) / max(len(call_ms[name]), 1)

    # --- hough_vote (stage + vote walk + flush).  Three ceilings in votes/s; `bound` is the LOWEST of them,
    # chosen here by rule: ALU issue (12 issue slots per vote at the very least), shared-memory atomics (one per
    # vote, conflict-free rate measured above), HBM (hit bytes in + accumulator bytes out at the measured copy rate).
    vote_ms_avg = avg("vote")
    achieved = votes_per_launch / (vote_ms_avg * 1e-3) / 1e9                     # Gvotes/s
    hbm_bytes = hits_per_launch * 8 + bins_per_launch * bn.bin_bytes            # hits in + accumulator out
    ceilings = {"alu": sms * FP32_LANES_PER_SM * sm_max_mhz * 1e6 / D3_MIN_ISSUE_SLOTS / 1e9,
                "atomic": mb["smem_atomic_conflict_free_gops"],
                "hbm": votes_per_launch / (hbm_bytes / (hbm_gbs * 1e9)) / 1e9}
    bound = min(ceilings, key=ceilings.get)
    roofline = {"bound": bound, "kernel": "hough_vote (stage + vote walk + flush)", "achieved": achieved,
                "peak": ceilings[bound], "unit": "Gvotes/s", "frac": achieved / ceilings[bound],
                "traffic": traffic_tab.get(("vote", run.tile_events)) if args.config == 3 else None,
                "traffic_source": traffic_src,
                "rule": "bound = the lowest of the three ceilings below, all in votes/s (SURVEY 8(d): report all three, "
                        "say which binds); north_star's reading (slower of atomic and HBM) is frac_atomic / frac_hbm",
                "ceilings_gvotes": ceilings,
                "frac_alu": achieved / ceilings["alu"], "frac_atomic": achieved / ceilings["atomic"],
                "frac_atomic_random": achieved / mb["smem_atomic_random_gops"], "frac_hbm": achieved / ceilings["hbm"],
                "peak_source": f"alu: {sms} SMs x {FP32_LANES_PER_SM} fp32 lanes x {sm_max_mhz:.0f} MHz / "
                               f"{D3_MIN_ISSUE_SLOTS} issue slots per vote (DESIGN.md), clocks {peak_src}; atomic: "
                               "hough_microbench kind 0 measured in this run; hbm: copy rate " + peak_src,
                "measured_in_run": mb, "vote_ms_per_launch": vote_ms_avg, "votes_per_launch": votes_per_launch,
                "launches_timed": len(vote_ms),
                "hbm": {"algorithmic_bytes_per_launch": hbm_bytes, "achieved_gbs": hbm_bytes / (vote_ms_avg * 1e-3) / 1e9,
                        "peak_gbs": hbm_gbs, "frac": hbm_bytes / (vote_ms_avg * 1e-3) / 1e9 / hbm_gbs}}
    # --- hough_find_peaks: HBM-bound by construction (reads every bin once, writes the candidate records)
    peaks_ms = avg("peaks")
    peak_bytes = bins_per_launch * bn.bin_bytes + cands_per_launch * 32 + (run.tile_events + 1) * 4
    roofline_peaks = {"bound": "hbm", "kernel": "hough_find_peaks (mask + scans + emit)", "achieved": peak_bytes / (peaks_ms * 1e-3) / 1e9,
                      "peak": hbm_gbs, "unit": "GB/s", "frac": peak_bytes / (peaks_ms * 1e-3) / 1e9 / hbm_gbs,
                      "algorithmic_bytes_per_launch": peak_bytes, "ms_per_launch": peaks_ms,
                      "candidates_per_launch": cands_per_launch,
                      "traffic": traffic_tab.get(("peaks", run.tile_events)) if args.config == 3 else None}
    # --- hough_assign_hits: every vote position of every hit has to be held against the candidates (D8 as the indexed
    # oracle states it), so the unit is the vote position and the ceiling the same ALU issue bound as the vote's
    assign_ms = avg("assign")
    a_ach = votes_per_launch / (assign_ms * 1e-3) / 1e9
    roofline_assign = {"bound": "alu", "kernel": "hough_assign_hits (association + duplicate removal)", "achieved": a_ach,
                       "peak": ceilings["alu"], "unit": "G vote positions/s", "frac": a_ach / ceilings["alu"],
                       "ms_per_launch": assign_ms, "vote_positions_per_launch": votes_per_launch,
                       "candidates_per_launch": cands_per_launch,
                       "note": "unit = vote positions of the launch's hits (what D8 ranges over); an association that "
                               "visits fewer positions than that can exceed the per-position ceiling"}
    step_share = {k: sum(v) / (ms_total) for k, v in call_ms.items()}

    # second Hough transform (tracks -> displaced vertices; D10): line-model workloads only
    vertex = None
    if getattr(bn, "model", 0) == 1:
        from paper_1311_2769_b200 import HoughPlan, alloc_candidates, hough_vertex_vote
        n_r, r_max, thr_v = 32, 16.0, 6
        (e0, e1, h0, h1) = run.tiles[0]
        n_ev = e1 - e0
        run.step_tile(0)                                # leaves the first tile's candidates / keep flags on the device
        vacc = torch.empty((n_ev, bn.n_phi, n_r), dtype=torch.int32, device="cuda")
        vplan = HoughPlan(bn.n_phi, n_r, 1, 0.0, r_max, bz_tesla=0.0, max_hits=1, max_events=n_ev, model=1)
        vcands = alloc_candidates(1 << 16)
        vcoff = torch.zeros(n_ev + 1, dtype=torch.int32, device="cuda")
        vt = []
        for it in range(25):
            a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
            a.record()
            hough_vertex_vote(run.plan, run.cands, run.cand_off, n_ev, run.cap, run.keep, 0.6, n_r, r_max, vacc)
            vplan.find_peaks(vacc, n_ev, thr_v, vcands, 1 << 16, vcoff)
            b.record(); b.synchronize()
            if it >= 5:
                vt.append(a.elapsed_time(b))
        vertex = {"ms_median": statistics.median(vt), "vertex_votes": int(vacc.to(torch.int64).sum().item()),
                  "vertex_candidates": int(vcoff[n_ev].item()), "binning": [bn.n_phi, n_r], "r_max_cm": r_max,
                  "threshold": thr_v, "api": "hough_vertex_vote + hough_find_peaks on the vertex space (D10)"}
        vplan.close()

    # circle fit of the assigned hits (D11), first tile, outside the timed step
    fit_info = None
    try:
        from paper_1311_2769_b200 import hough_fit_circles
        (e0, e1, h0, h1) = run.tiles[0]
        n_ev = e1 - e0
        run.step_tile(0)                                # hits, candidates and assignments of the SAME (first) tile
        work = torch.empty((run.cap, 9), dtype=torch.float64, device="cuda")
        fitp = torch.empty((run.cap, 4), dtype=torch.float64, device="cuda")
        nfit = torch.empty((run.cap,), dtype=torch.int32, device="cuda")
        ft = []
        for it in range(12):
            a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
            a.record()
            hough_fit_circles(run.plan, run.d_hits[h0:h1], run.h2c[:max(h1 - h0, 1)][:h1 - h0], run.cands, run.cand_off, n_ev,
                              run.cap, run.keep, work, fitp, nfit)
            b.record(); b.synchronize()
            if it >= 2:
                ft.append(a.elapsed_time(b))
        fit_info = {"ms_median": statistics.median(ft), "events": n_ev, "tracks_fitted": int((nfit > 0).sum().item()),
                    "api": "hough_fit_circles on the first tile (D11), not part of the timed step"}
        del work, fitp, nfit
    except Exception as exc:                              # noqa: BLE001 -- report, do not hide
        print(f"bench.py: fit stage failed: {exc}", file=sys.stderr)

    # single events: the same path through hough_event_run (one launch of a thread-block cluster when it fits)
    event_info = None
    if batch.n_events == 1:
        try:
            from paper_1311_2769_b200 import kernel_launches
            (e0, e1, h0, h1) = run.tiles[0]
            et = []
            l0 = 0
            for it in range(40):
                if it == 10:
                    l0 = kernel_launches()
                a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
                a.record()
                run.plan.event_run(run.d_hits[h0:h1], run.d_offs[0], run.accum, w.threshold, run.cands, run.cap, run.cand_off,
                                   w.assoc_dj, w.min_hits, run.h2c[:max(h1 - h0, 1)], run.nh, run.keep)
                b.record(); b.synchronize()
                if it >= 10:
                    et.append(a.elapsed_time(b))
            event_info = {"ms_median": statistics.median(et), "ms_min": min(et),
                          "launches_per_call": (kernel_launches() - l0) / 30.0,
                          "api": "hough_event_run: vote + peaks + assign of the single event in one call "
                                 "(one cluster launch for two-parameter spaces up to 2560 hits)"}
        except Exception as exc:                          # noqa: BLE001 -- report, do not hide
            print(f"bench.py: hough_event_run stage failed: {exc}", file=sys.stderr)

    # re-assignment round of the stranded hits (PAPER.md:33 / :29; D12), first tile, outside the timed step
    reassign_info = None
    try:
        (e0, e1, h0, h1) = run.tiles[0]
        n_ev = e1 - e0
        rt = []
        gained = 0
        for it in range(8):
            run.step_tile(0)                            # fresh D9 state of the first tile
            before = int((run.h2c[:h1 - h0] >= 0).sum().item()) if it == 7 else 0
            a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
            a.record()
            run.reassign_tile(0)
            b.record(); b.synchronize()
            if it >= 2:
                rt.append(a.elapsed_time(b))
            if it == 7:
                gained = int((run.h2c[:h1 - h0] >= 0).sum().item()) - before
        reassign_info = {"ms_median": statistics.median(rt), "events": n_ev, "hits_recovered": gained,
                         "api": "hough_reassign_hits on the first tile (D12, candidate-centric over the kept candidates), "
                                "not part of the timed step"}
    except Exception as exc:                              # noqa: BLE001 -- report, do not hide
        print(f"bench.py: reassign stage failed: {exc}", file=sys.stderr)

    n_ref = oracle_events_for_seconds(w, args.cpu_seconds)
    o_votes, o_events, o_secs = oracle_sample(w, batch, n_ref)
    cpu = {"value": o_votes / o_secs, "unit": UNIT, "cores": 1, "kind": "oracle",
           "sample": f"first {o_events} event(s) of {w.name}: vote (full scan) + peaks + indexed assignment, "
                     f"{o_secs:.1f} s", "events_per_s": o_events / o_secs, "host_cores_available": os.cpu_count(), "pinned_to_one_core": True}

    line = {"metric": METRIC, "value": job_votes / (ms_step * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32+u16" if bn.bin_bytes == 2 else "f32+int32",
            "data": "synthetic",
            "config": {"workload": w.name, "cite": w.cite, "events_per_gpu": batch.n_events,
                       "hits_per_gpu": batch.n_hits, "votes_per_step_per_gpu": votes_per_step,
                       "binning": [bn.n_phi, bn.n_qpt, bn.n_d0], "accum": "u16" if bn.bin_bytes == 2 else "i32",
                       "threshold": w.threshold, "tile_events": run.tile_events, "parallelism": f"events x{world}",
                       "l2": "no flush: per-step working set (hits + accumulators + candidates) exceeds the 126 MB L2"
                             if batch.n_events * bn.n_bins * bn.bin_bytes > 126e6 else
                             "working set fits L2; latency-bound configuration",
                       "library": version()},
            "events_per_s": job_events / (ms_step * 1e-3), "hits_per_s": job_hits / (ms_step * 1e-3),
            "e2e": {"value": job_votes / (e2e_ms * 1e-3), "unit": UNIT, "events_per_s": job_events / (e2e_ms * 1e-3),
                    "ms_per_step": e2e_ms, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "api": f"hough_pipeline_run_host: {min(args.e2e_tile_events, batch.n_events)}-event tiles on {args.streams} streams, CUDA graph per "
                           "lane, pinned host buffers in and out; wall clock around the blocking call",
                    "candidate_overflow": bool(e2e_over)},
            "e2e_kept_only": {"value": job_votes / (k_ms * 1e-3), "unit": UNIT, "events_per_s": job_events / (k_ms * 1e-3),
                              "ms_per_step": k_ms, "h2d_bytes_per_step": int(k_h2d), "d2h_bytes_per_step": int(k_d2h),
                              "api": "the same pipeline with option kept_only: identical work, only the candidates that "
                                     "survive duplicate removal are compacted on the device and copied back",
                              "candidate_overflow": bool(k_over)},
            "gpu_launches": int(launches), "roofline": roofline, "roofline_assign": roofline_assign,
            "roofline_peaks": roofline_peaks, "step_share": step_share, "cpu_baseline": cpu, "clocks": clocks,
            "candidate_overflow": peaks_overflow}
    if vertex is not None:
        line["vertex"] = vertex
    if fit_info is not None:
        line["fit"] = fit_info
    if reassign_info is not None:
        line["reassign"] = reassign_info
    if event_info is not None:
        line["event_run"] = event_info
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_sweep(args):
    """Fig. 2-style sweep ("time performance, as a function of number of tracks") on the
    paper's toy detector (workload 5): one event of n tracks, vote + peaks + assign, median device time of `reps` runs.
    Prints one JSON line per n (not the driver's bench line)."""
    import torch
    from paper_1311_2769_b200 import HoughPlan, alloc_candidates, load_library
    from workloads import generate_events, get_workload
    load_library()
    torch.cuda.set_device(0)
    base = get_workload(5)
    for n in (50, 100, 200, 500, 1000, 2000, 5000, 10000, 20000):
        w = base.with_tracks(n)
        batch = generate_events(w)
        plan = HoughPlan.from_workload(w, max_hits=max(batch.n_hits, 1), max_events=1)
        plan.set_option("reuse_staging", 1)
        d_hits = torch.from_numpy(batch.hits_xy).cuda()
        d_off = torch.from_numpy(batch.event_offsets).cuda()
        accum = plan.alloc_accum(1)
        cap = w.binning.n_bins // 8 + 1024
        cands = alloc_candidates(cap)
        coff = torch.zeros(2, dtype=torch.int32, device="cuda")
        h2c = torch.empty(max(batch.n_hits, 1), dtype=torch.int32, device="cuda")
        nh = torch.empty(cap, dtype=torch.int32, device="cuda")
        keep = torch.empty(cap, dtype=torch.uint8, device="cuda")

        def once():
            plan.vote(d_hits, d_off, accum)
            plan.find_peaks(accum, 1, w.threshold, cands, cap, coff)
            plan.assign_hits(d_hits, d_off, cands, coff, cap, w.assoc_dj, w.min_hits, h2c, nh, keep)
        for _ in range(5):
            once()
        torch.cuda.synchronize()
        times = []
        for _ in range(args.sweep_reps):
            a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
            a.record(); once(); b.record(); b.synchronize()
            times.append(a.elapsed_time(b))
        # the same three calls captured once in a CUDA graph and replayed (the calls only enqueue: include/hough.h)
        gtimes = []
        try:
            side = torch.cuda.Stream()
            side.wait_stream(torch.cuda.current_stream())
            with torch.cuda.stream(side):
                once()
            torch.cuda.current_stream().wait_stream(side)
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph):
                once()
            for _ in range(5):
                graph.replay()
            torch.cuda.synchronize()
            for _ in range(args.sweep_reps):
                a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
                a.record(); graph.replay(); b.record(); b.synchronize()
                gtimes.append(a.elapsed_time(b))
        except Exception as exc:                          # noqa: BLE001 -- report, do not hide
            print(f"bench.py: graph capture failed: {exc}", file=sys.stderr)
        # the same event through hough_event_run: one launch of a thread-block cluster (csrc/event.cu)
        etimes = []
        launches_event = None
        try:
            from paper_1311_2769_b200 import kernel_launches
            for _ in range(5):
                plan.event_run(d_hits, d_off, accum, w.threshold, cands, cap, coff, w.assoc_dj, w.min_hits, h2c, nh, keep)
            torch.cuda.synchronize()
            l0 = kernel_launches()
            for _ in range(args.sweep_reps):
                a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
                a.record()
                plan.event_run(d_hits, d_off, accum, w.threshold, cands, cap, coff, w.assoc_dj, w.min_hits, h2c, nh, keep)
                b.record(); b.synchronize()
                etimes.append(a.elapsed_time(b))
            launches_event = (kernel_launches() - l0) / float(args.sweep_reps)
        except Exception as exc:                          # noqa: BLE001 -- report, do not hide
            print(f"bench.py: hough_event_run failed: {exc}", file=sys.stderr)
        votes = int(accum.to(torch.int64).sum().item())
        n_c = int(coff[1].item())
        kept = int(keep[:min(n_c, cap)].sum().item())
        print(json.dumps({"sweep": "paper_toy_2d", "cite": "P:L39, P:L55", "n_tracks": n, "hits": batch.n_hits, "votes": votes,
                          "peaks": n_c, "kept": kept, "ms_median": statistics.median(times), "ms_min": min(times),
                          "ms_graph_median": statistics.median(gtimes) if gtimes else None,
                          "ms_event_run_median": statistics.median(etimes) if etimes else None,
                          "ms_event_run_min": min(etimes) if etimes else None, "event_run_launches": launches_event,
                          "reps": args.sweep_reps}), flush=True)
        plan.close()


def run_efficiency(args):
    """Track-finding efficiency / fake / duplicate report against generator truth (Fig. 1: "track-finding
    efficiency ... approximately 86%" on the toy detector of PAPER.md:39).  vote -> peaks -> assign (D9),
    then the D12 re-assignment round, then the circle fit of the kept candidates, all through the library; the counting is
    paper_1311_2769_b200.efficiency (host numpy).  Prints one JSON line per configuration (not the driver's bench line)."""
    import math
    import torch
    from paper_1311_2769_b200 import HoughPlan, alloc_candidates, candidates_to_numpy, hough_fit_circles, load_library
    from paper_1311_2769_b200.efficiency import efficiency_report, truth_parameters
    from workloads import generate_events, get_workload
    load_library()
    torch.cuda.set_device(0)
    from dataclasses import replace
    todo = [(cfg, None) for cfg in args.efficiency]
    if args.efficiency_scan:
        # the paper's toy scenario (workload 5) under other binnings: PAPER.md:43 quotes its 86 % without stating the binning
        todo = [(5, t) for t in ((512, 256, 8, 8, 1), (1024, 64, 8, 8, 1), (2048, 64, 8, 8, 1), (2048, 32, 8, 8, 1),
                                 (4096, 64, 8, 8, 1), (2048, 64, 7, 7, 1), (2048, 64, 9, 8, 2), (4096, 32, 9, 8, 1),
                                 (4096, 128, 7, 7, 2), (8192, 64, 8, 8, 1))]
    for cfg, alt in todo:
        w = get_workload(cfg)
        if alt is not None:
            w = replace(w, binning=replace(w.binning, n_phi=alt[0], n_qpt=alt[1]), threshold=alt[2], assoc_dj=alt[4],
                        name=f"{w.name}_{alt[0]}x{alt[1]}_thr{alt[2]}_min{alt[3]}_dj{alt[4]}")
            min_hits_alt = alt[3]
        else:
            min_hits_alt = None
        if w.n_events > 1:
            w = w.scaled(min(w.n_events, args.efficiency_events))
        batch = generate_events(w, want_truth=True)
        n_ev = w.n_events
        bn = w.binning
        plan = HoughPlan.from_workload(w, max_hits=max(batch.n_hits, 1), max_events=n_ev)
        d_hits = torch.from_numpy(batch.hits_xy).cuda()
        d_off = torch.from_numpy(batch.event_offsets).cuda()
        accum = plan.alloc_accum(n_ev)
        plan.vote(d_hits, d_off, accum)
        coff = torch.zeros(n_ev + 1, dtype=torch.int32, device="cuda")
        plan.find_peaks(accum, n_ev, w.threshold, None, 0, coff)
        cap = int(coff[n_ev].item()) + 1
        cands = alloc_candidates(cap)
        plan.find_peaks(accum, n_ev, w.threshold, cands, cap, coff)
        h2c = torch.empty(max(batch.n_hits, 1), dtype=torch.int32, device="cuda")
        nh = torch.empty(cap, dtype=torch.int32, device="cuda")
        keep = torch.empty(cap, dtype=torch.uint8, device="cuda")
        min_hits = w.min_hits if min_hits_alt is None else min_hits_alt
        plan.assign_hits(d_hits, d_off, cands, coff, cap, w.assoc_dj, min_hits, h2c, nh, keep)
        torch.cuda.synchronize()
        off = coff.cpu().numpy()
        rec = candidates_to_numpy(cands, int(off[-1]))
        keep_h = keep[:int(off[-1])].cpu().numpy()
        h2c_d9 = h2c[:batch.n_hits].cpu().numpy()
        plan.reassign_hits(d_hits, d_off, cands, coff, cap, w.assoc_dj, 2, h2c, nh, keep)
        torch.cuda.synchronize()
        h2c_d12 = h2c[:batch.n_hits].cpu().numpy()
        # circle fit of the kept candidates on the re-assigned hits (D11)
        work = torch.zeros(cap * 9, dtype=torch.float64, device="cuda")
        fit = torch.zeros((cap, 4), dtype=torch.float64, device="cuda")
        nfit = torch.zeros(cap, dtype=torch.int32, device="cuda")
        hough_fit_circles(plan, d_hits, h2c, cands, coff, n_ev, cap, keep, work, fit, nfit)
        torch.cuda.synchronize()
        fit_h, nfit_h = fit.cpu().numpy(), nfit.cpu().numpy()

        def total(h2c_all):
            acc = None
            for e in range(n_ev):
                a, b = int(batch.event_offsets[e]), int(batch.event_offsets[e + 1])
                c0, c1 = int(off[e]), int(off[e + 1])
                local = np.where(h2c_all[a:b] >= 0, h2c_all[a:b] - c0, -1)
                r = efficiency_report(bn, w.bz_tesla, batch.truth[e], rec[c0:c1], keep_h[c0:c1], local, min_hits)
                if acc is None:
                    acc = {k: r[k] for k in ("tracks", "reconstructable", "candidates", "kept", "hits_assigned", "hits_total")}
                    acc["found_by_hits"] = r["by_hits"]["tracks_found"]
                    acc["found_by_parameters"] = r["by_parameters"]["tracks_found"]
                    acc["fake_by_hits"] = r["by_hits"]["fake_rate"] * max(r["kept"], 1)
                    acc["dup_by_hits"] = r["by_hits"]["duplicate_rate"] * max(r["kept"], 1)
                    acc["fake_by_parameters"] = r["by_parameters"]["fake_rate"] * max(r["kept"], 1)
                    acc["dup_by_parameters"] = r["by_parameters"]["duplicate_rate"] * max(r["kept"], 1)
                    acc["purity_sum"] = r["mean_purity"] * r["kept"]
                else:
                    for k in ("tracks", "reconstructable", "candidates", "kept", "hits_assigned", "hits_total"):
                        acc[k] += r[k]
                    acc["found_by_hits"] += r["by_hits"]["tracks_found"]
                    acc["found_by_parameters"] += r["by_parameters"]["tracks_found"]
                    acc["fake_by_hits"] += r["by_hits"]["fake_rate"] * max(r["kept"], 1)
                    acc["dup_by_hits"] += r["by_hits"]["duplicate_rate"] * max(r["kept"], 1)
                    acc["fake_by_parameters"] += r["by_parameters"]["fake_rate"] * max(r["kept"], 1)
                    acc["dup_by_parameters"] += r["by_parameters"]["duplicate_rate"] * max(r["kept"], 1)
                    acc["purity_sum"] += r["mean_purity"] * r["kept"]
            kept = max(acc["kept"], 1)
            reco = max(acc["reconstructable"], 1)
            out = {k: acc[k] for k in ("tracks", "reconstructable", "candidates", "kept", "hits_assigned", "hits_total")}
            out["mean_purity"] = acc["purity_sum"] / kept
            for m in ("hits", "parameters"):
                out["by_" + m] = {"efficiency": acc["found_by_" + m] / reco, "fake_rate": acc["fake_by_" + m] / kept,
                                  "duplicate_rate": acc["dup_by_" + m] / kept}
            return out

        # q/pT resolution of the kept, hit-matched candidates: peak centroid (D7) vs circle fit (D11), against truth
        res_c, res_f = [], []
        for e in range(n_ev):
            tp = truth_parameters(batch.truth[e], w.bz_tesla)
            a, b = int(batch.event_offsets[e]), int(batch.event_offsets[e + 1])
            lab = batch.truth[e]["hit_track"]
            for c in range(int(off[e]), int(off[e + 1])):
                if not keep_h[c] or nfit_h[c] < 3:
                    continue
                own = lab[np.nonzero(h2c_d12[a:b] == c)[0]]
                own = own[own >= 0]
                if len(own) == 0:
                    continue
                ids, cnt = np.unique(own, return_counts=True)
                t = ids[np.argmax(cnt)]
                if 2 * cnt.max() <= nfit_h[c] or bn.model != 0:
                    continue
                res_c.append(float(rec["qpt"][c]) - tp["qpt"][t])
                res_f.append(fit_h[c, 1] - tp["qpt"][t])
        line = {"report": "efficiency", "cite": "PAPER.md:43 (approx. 86 % on its toy detector, binning unstated), SURVEY 8(f) f4",
                "config": {"workload": w.name, "events": n_ev, "n_phi": bn.n_phi, "n_qpt": bn.n_qpt, "n_d0": bn.n_d0,
                           "threshold": w.threshold, "min_hits": min_hits, "assoc_dj": w.assoc_dj},
                "d9_single_pass": total(h2c_d9), "d12_reassigned": total(h2c_d12),
                "qpt_resolution": {"matched_candidates": len(res_c), "bin_width": (bn.qpt_max - bn.qpt_min) / bn.n_qpt,
                                   "centroid_rms": float(np.sqrt(np.mean(np.square(res_c)))) if res_c else None,
                                   "circle_fit_rms": float(np.sqrt(np.mean(np.square(res_f)))) if res_f else None,
                                   "circle_fit_median_abs": float(np.median(np.abs(res_f))) if res_f else None}}
        print(json.dumps(line), flush=True)
        plan.close()


def run_stage_probe(args):
    """--stage-probe: hough_vote on a batched fine-phi plan (n_phi = 1024, 1024 events, 64 hits each: the staging sort and
    its key-start table dominate) -- the cost of the staging sector count (plan.cu caps it by the table size; HOUGH_SECTORS=n
    in the environment overrides).  One JSON line; not a bench value."""
    import torch
    from paper_1311_2769_b200 import HoughPlan
    from workloads import LAYERS_14
    n_ev, per = 1024, 64
    rng = np.random.default_rng(3)
    r = rng.choice(np.asarray(LAYERS_14), n_ev * per)
    ph = rng.uniform(0, 2 * np.pi, n_ev * per)
    hits = np.stack([r * np.cos(ph), r * np.sin(ph)], 1).astype(np.float32)
    off = (np.arange(n_ev + 1) * per).astype(np.int32)
    plan = HoughPlan(1024, 128, 1, -1.0, 1.0, -20.0, 20.0, 1, 3.8, LAYERS_14, max_hits=len(hits), max_events=n_ev)
    d_hits, d_off = torch.from_numpy(hits).cuda(), torch.from_numpy(off).cuda()
    acc = plan.alloc_accum(n_ev)
    for _ in range(3):
        plan.vote(d_hits, d_off, acc)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ts = []
    for _ in range(max(args.steps, 20)):
        a.record()
        plan.vote(d_hits, d_off, acc)
        b.record()
        b.synchronize()
        ts.append(a.elapsed_time(b))
    print(json.dumps({"probe": "stage_sectors", "HOUGH_SECTORS": os.environ.get("HOUGH_SECTORS", "default (capped by table size)"),
                      "plan": "n_phi 1024 x n_qpt 128 x 1, u16, max_events 1024", "hits": len(hits),
                      "hough_vote_ms_median": statistics.median(ts), "hough_vote_ms_min": min(ts),
                      "votes": int(acc.to(torch.int64).sum().item())}), flush=True)
    plan.close()


def run_atoms_probe(args):
    """--atoms-probe: shared-memory vote rates of hough_microbench kinds 0 / 1 / 5 / 6 / 7 on this GPU (one JSON line):
    +1 votes (ATOMS.POPC.INC) against + 1 << 16 votes (ATOMS.ADD, the odd column of a packed pair word) on the same
    addresses, and the latter warp-aggregated with __match_any_sync (B:L5).  Not a bench value."""
    import torch
    from paper_1311_2769_b200 import microbench
    torch.cuda.init()
    names = {0: "add_1_conflict_free", 1: "add_1_random_64KB", 5: "add_1_random_bin_of_one_row_per_warp",
             6: "add_65536_same_addresses_as_5", 7: "add_65536_match_any_leader_same_addresses_as_5"}
    out = {"probe": "shared_atomics", "unit": "Gops/s (lane operations)"}
    for k, n in names.items():
        out[n] = microbench(k, 0, 5) / 1e9
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--events", type=int, default=0, help="events per GPU (default: the workload's own count)")
    ap.add_argument("--tile-events", type=int, default=256, help="events per call of the device-resident loop")
    ap.add_argument("--e2e-tile-events", type=int, default=32, help="events per tile of the batched host pipeline")
    ap.add_argument("--cand-per-bin", type=float, default=1.0 / 16.0, help="candidate capacity per accumulator bin")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--streams", type=int, default=4, help="CUDA streams of the batched pipeline (B:L10: 4)")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target oracle time of the cpu_baseline sample")
    ap.add_argument("--ref-seconds-per-step", type=float, default=10.0)
    ap.add_argument("--sweep-tracks", action="store_true", help="Fig. 2-style sweep on the paper's toy detector (workload 5)")
    ap.add_argument("--sweep-reps", type=int, default=30)
    ap.add_argument("--efficiency", type=int, nargs="*", default=None, metavar="CFG",
                    help="efficiency / fake / duplicate report against generator truth for these workloads (PAPER.md:43)")
    ap.add_argument("--efficiency-events", type=int, default=8)
    ap.add_argument("--efficiency-scan", action="store_true", help="the paper's toy scenario under a list of other binnings")
    ap.add_argument("--stage-probe", action="store_true", help="staging cost of a batched n_phi = 1024 plan (sector count)")
    ap.add_argument("--atoms-probe", action="store_true", help="shared-memory atomic rates: +1, +65536, match_any-aggregated")
    args = ap.parse_args()
    if args.atoms_probe:
        run_atoms_probe(args)
        return
    if args.stage_probe:
        run_stage_probe(args)
        return
    if args.efficiency_scan and args.efficiency is None:
        args.efficiency = [5]
    if args.efficiency is not None:
        if not args.efficiency:
            args.efficiency = [5, 0, 1, 3]
        run_efficiency(args)
        return
    if args.sweep_tracks:
        run_sweep(args)
        return
    rank, world, local_rank = _env_int("RANK", 0), _env_int("WORLD_SIZE", 1), _env_int("LOCAL_RANK", 0)
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()

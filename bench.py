#!/usr/bin/env python
"""bench.py — events/s of the TPC sector tracker on central Pb-Pb-like events (BASELINE.json configs[3]).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--events E] [--impl tpcst|reference]
    python bench.py --stream 256        (BASELINE.json configs[4]: one pass over 256 distinct events)
    python bench.py --size-sweep        (time per event vs input size, Fig. 9)
    python bench.py --alpha-scan        (chi2-suppression factor on synthetic truth, Fig. 6)
    python bench.py --l2-random         (this GPU's random L2 gather / red.max rate, tpcst_selftest_random_access: the yardstick for the selection kernels)

One "step" is one pass of the whole hot path (bin_rows ... write_tracks) over
one synthetic central Pb-Pb-like event (36 sectors x 159 rows, ~3.7 M clusters, 44 MB).  E distinct
seeded events are generated up front (outside every timed region) and visited round robin.

Legs, all through the C ABI (paper_1712_09407_b200.SectorTracker):
  value : clusters already resident in HBM (TPCST_DEVICE); four events in flight (slots 0..3, one compute
          stream each), so the device->host copy of one event's tracks and the edges of its kernel set
          overlap the next event's kernels.
  e2e   : clusters in pinned HOST memory (TPCST_HOST_PINNED); the host->device copy of every step's
          input runs on the copy stream inside the timed region and overlaps the previous event's
          tracking (BASELINE.json configs[4]); tracks come back to pinned host memory.
  roofline / kernels : per-kernel CUDA-event times recorded on the compute stream during a second timed
          pass of the same steps (tpcst_set_profiling(1): all slots on one stream, so that an event pair
          times a kernel and not its wait for the other event), work counters from one untimed counting pass
          (tpcst_set_profiling(2)); arithmetic in DESIGN.md section 7.
  cpu_baseline : the CPU oracle (oracle/, test infrastructure) on the same events, on the host cores.
After the timed legs, at N = 1 only and outside every timed region above (skip with --no-extras):
  stream  : BASELINE.json configs[4] in small: ONE pass over 32 distinct pinned-host events (events/s, input GB/s), then the
            race check of --stream --check on 4 of them.
  options : every optional stage on its own (select_mode=1, select_rounds=2, max_passes=3, global_tracking=1,
            merge_tracks=1): pipelined device-resident events/s and the per-kernel times that are new or changed.
  small_configs : BASELINE.json configs[0..2]: single-event kernel-set time and call latency, oracle on one thread.
The events of all legs come from one seeded stream (seed STREAM_BASE_SEED + index); under torchrun rank r tracks the
events shard.event_shard gives it, so N = 1 and N = 8 see the same stream.

--impl reference times the oracle instead (this repository's tier has no reference implementation;
the oracle is the stand-in).  Under torchrun (N > 1) every rank tracks its
share of the stream (event-level data parallelism, no collective on the data path; "scaling": "weak").
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

IN_FLIGHT = 4   # events in flight (= TPCST_N_SLOTS)
EXTRA_STREAM_EVENTS = 32   # default run, after the timed legs: one pass over this many distinct pinned-host events (`stream`)
# default run, after the timed legs: every optional stage on its own (`options`), PAPER.md L88 / L116-L136 / L45 / L102
OPTIONS = (("select_mode=1", {"select_mode": 1}), ("select_rounds=2", {"select_rounds": 2}), ("max_passes=3", {"max_passes": 3}),
           ("global_tracking=1", {"global_tracking": 1}), ("merge_tracks=1", {"merge_tracks": 1}))
METRIC = "central_pbpb_like_events_per_s"
UNIT = "events/s"
WORKLOAD = "BASELINE.json configs[3]: central Pb-Pb-like, 36 sectors x 159 rows, 20000 primaries + 3000 secondaries, 5% noise"

# ---- roofline arithmetic ---------------------------------------------------
# fp32 operations per unit of work of construct_tracklets, counted from the formulas of DESIGN.md
# section 3 step 5 in the 9-element covariance form (add, mul, div, sqrt = 1 operation each):
FLOP_TRANSPORT = 80      # per row step: state 42 + covariance 38
FLOP_INNOV = 5           # per row step that reaches the innovation (counted per search + update)
FLOP_SEARCH = 22         # per searched row: box half widths and 4 bin coordinates
FLOP_CANDIDATE = 7       # per chi2 candidate
FLOP_UPDATE = 35         # per update
# fp32 operations of find_neighbours: 4 per window test (2 subtractions, 2 |.| comparisons counted
# as 2) and 11 per pair (G7), 4 per cluster for the projections.
FLOP_NF_TEST, FLOP_NF_PAIR, FLOP_NF_CLUSTER = 4, 11, 4
NOMINAL_HBM_GBS = 8000.0   # B200 HBM3e nominal (north_star: "~8 TB/s"); the measured copy peak is what `peak` holds


def _peaks():
    """(hbm GB/s, source) from MEASURED_PEAKS.json, else the fallback of the profiling recipe."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def kernel_source_digest() -> str:
    """sha256 (first 16 hex digits) over the kernel sources a `--set full` capture depends on."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_1712_09407_b200", "csrc")
    for f in ("tpcst_internal.h", "kalman_math.cuh", "kernels_ca.cu", "kernels_kalman.cu", "kernels_select.cu", "kernels_merge.cu"):
        with open(os.path.join(d, f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def ncu_traffic():
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of every kernel, from the committed
    summary of one `ncu --set full` capture -> ({kernel: bytes}, name of the capture, why it was refused or None).
    profiles/traffic.csv names the capture in its third column and, in a `# kernel_source_digest:` line, the digest of the
    kernel sources it was taken on; if the sources have changed since, the numbers are stale and are NOT reported."""
    out, capture, digest = {}, None, None
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as f:
            for line in f.read().strip().splitlines():
                if line.startswith("#"):
                    if "kernel_source_digest:" in line:
                        digest = line.split("kernel_source_digest:", 1)[1].strip()
                    continue
                if line.startswith("kernel,"):
                    continue
                k, b, c = line.split(",")
                out[k] = float(b)
                capture = c.strip()
    except Exception:
        return {}, None, "profiles/traffic.csv is absent"
    now = kernel_source_digest()
    if digest != now:
        return {}, capture, f"stale: {capture} was taken on kernel sources {digest}, the sources are now {now}"
    return out, capture, None


def algorithmic(name, n, nbins, T, K, ids, work, sm_count, sm_mhz):
    """Algorithmic bytes / operations of one launch of kernel `name` -> (bound, amount, unit, peak)."""
    hbm, _ = _peaks()
    alu_peak = sm_count * 128 * sm_mhz * 1e6 / 1e12      # fp32 op/s without FMA, in Tops/s
    w = work
    if name == "bin_rows":          # read xyz 12 B, write (y,z) 8 B + original index 4 B; 2 B per bin
        return "hbm", n * 24 + nbins * 2, "GB/s", hbm
    if name == "find_neighbours":   # rows k-1, k, k+1 read once per row (8 B each) + bin tables, 8 B links out
        return "hbm", n * 32 + nbins * 4, "GB/s", hbm
    if name == "evolve_links":      # 2 links read, 2 gathered, 2 written
        return "hbm", n * 24, "GB/s", hbm
    if name == "find_starts":       # 2 links read, per start: chain gathers + list entry
        return "hbm", n * 8 + T * 16, "GB/s", hbm
    if name == "scan_rows":
        return "hbm", 5724 * 8, "GB/s", hbm
    if name == "list_tracklets":    # counts/offsets per row + one 16-byte record per tracklet (8 B read, 16 B written)
        return "hbm", 5724 * 12 + T * 24, "GB/s", hbm
    if name == "construct_tracklets":
        ops = (w["kf_row_steps"] * FLOP_TRANSPORT + (w["kf_searches"] + w["kf_updates"]) * FLOP_INNOV +
               w["kf_searches"] * FLOP_SEARCH + w["kf_candidates"] * FLOP_CANDIDATE + w["kf_updates"] * FLOP_UPDATE)
        return "alu", ops, "TFLOP/s", alu_peak
    if name == "select_claim":      # hit 4 B read + 8 B atomic per claimed hit, 8 B header per tracklet
        return "hbm", w["claimed_hits"] * 12 + T * 8, "GB/s", hbm
    if name == "select_collect":    # hit 4 B + owner 8 B per claimed hit; per tracklet 8 B header in, 8 B group counts + 20 B row masks out
        return "hbm", w["claimed_hits"] * 12 + T * 36, "GB/s", hbm
    if name == "select_accept":     # header 4 + group counts 8 + kappa 4 in, kept 4 out per tracklet
        return "hbm", T * 20, "GB/s", hbm
    if name == "scan_partials":
        return "hbm", (T // 128 + 1) * 16, "GB/s", hbm
    if name == "write_tracks":      # track record 112 B out, 64 B of tracklet SoA in; 8 B per tracklet
        return "hbm", K * (112 + 64) + T * 8, "GB/s", hbm
    if name == "write_ids":         # per kept cluster: hit 4 + orig 4 + id 4; per tracklet 16 B header + 20 B row masks
        return "hbm", ids * 12 + T * 36, "GB/s", hbm
    # global tracking (--cut global_tracking=1): 2K (track, end) entries; state in, state + picks out (upper bounds)
    if name == "gt_extend":
        return "hbm", 2 * K * (64 + 60 + 128), "GB/s", hbm
    if name == "gt_scan":
        return "hbm", 2 * K * 12, "GB/s", hbm
    if name == "gt_write":
        return "hbm", 2 * K * (8 + 112 + 128), "GB/s", hbm
    # track merging (--cut merge_tracks=1): one lane per track; bytes a track must move (upper bounds)
    if name == "merge_rank":        # key in, rank out
        return "hbm", K * 16, "GB/s", hbm
    if name == "merge_refit":       # record in, both end states out; per cluster and pass: id 4 + (y, z) 8
        return "hbm", K * (112 + 192) + ids * 2 * 12, "GB/s", hbm
    if name == "merge_match":       # own outer state + the inner state of a handful of candidates
        return "hbm", K * 192 * 2, "GB/s", hbm
    if name == "merge_link":
        return "hbm", K * 24, "GB/s", hbm
    if name == "merge_chain":       # every cluster of a chain once per pass, the merged record out
        return "hbm", K * 92 + ids * 2 * 12, "GB/s", hbm
    raise KeyError(name)


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons of one GPU every 20 ms while the timed region runs."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz, self._stop_ev = index, [], set(), None, threading.Event()
        self.err = None

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = int(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
            names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                     "hw_power_brake": 0x80, "sync_boost": 0x10, "applications_clocks_setting": 0x2}
            while not self._stop_ev.is_set():
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)))
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(h))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
                self._stop_ev.wait(0.02)
        except Exception as e:          # NVML missing: report it rather than inventing numbers
            self.err = repr(e)

    def stop(self) -> dict:
        self._stop_ev.set()
        self.join(timeout=2.0)
        if self.err or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "error": self.err or "no samples"}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def _gen_one(seed: int):
    from tpcsynth import generate_event
    return generate_event(4, seed)


def gen_events(n_events: int, rank: int = 0, world: int = 1, skip: int = 0):
    """Central Pb-Pb-like events of ONE seeded stream (seed STREAM_BASE_SEED + global index): rank
    `rank` of `world` gets the events shard.event_shard gives it out of world * n_events, so that N = 1 and N = 8 track
    the same stream (N = 1: its first n_events events).  `skip` leaves out the first events of the rank's share (already
    generated).  More than a handful are generated by a pool of host processes (before or between the CUDA legs, never
    inside a timed region); the result does not depend on the pool."""
    from paper_1712_09407_b200.shard import event_shard
    from tpcsynth import STREAM_BASE_SEED
    seeds = [STREAM_BASE_SEED + g for g in event_shard(world * n_events, rank, world)][skip:]
    if len(seeds) <= 4:
        return [_gen_one(sd) for sd in seeds]
    from concurrent.futures import ProcessPoolExecutor
    import multiprocessing as mp
    with ProcessPoolExecutor(max_workers=min(os.cpu_count() or 1, 32), mp_context=mp.get_context("fork")) as ex:
        return list(ex.map(_gen_one, seeds))


# ---- the oracle legs ------------------------------------------------------------------------------
def cpu_model() -> str:
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_events_per_s(events, steps: int, warmup: int, n_threads: int):
    """Times the CPU oracle as it stands: one step = one whole event, sector-parallel over n_threads
    host threads (the paper's CPU tracker used the same trivial parallelisation)."""
    from oracle import Oracle
    o = Oracle.for_geometry(events[0].geometry)
    for i in range(warmup):
        o.run(events[i % len(events)].xyz, events[i % len(events)].row_start, n_threads=n_threads, fetch=False)
    t0 = time.perf_counter()
    ncl = 0
    for i in range(steps):
        ev = events[i % len(events)]
        o.run(ev.xyz, ev.row_start, n_threads=n_threads, fetch=False)
        ncl += ev.n_clusters
    dt = time.perf_counter() - t0
    return steps / dt, ncl / dt, dt


def run_reference(args, rank: int):
    if rank != 0:
        return
    cores = os.cpu_count() or 1
    nthr = min(cores, 36)
    events = gen_events(min(args.events, 2))
    steps = max(1, min(args.steps, 12))
    warm = min(args.warmup, 1)
    evs, cls, dt = oracle_events_per_s(events, steps, warm, nthr)
    line = {"impl": "reference", "metric": METRIC, "value": evs, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": warm, "ms_per_step": 1e3 * dt / steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": WORKLOAD, "events": len(events), "note": "CPU oracle (oracle/tpc_oracle.cpp), "
                       "whole events, sector-parallel host threads; stands in for the absent reference"},
            "clusters_per_s": cls,
            "cpu_baseline": {"value": evs, "unit": UNIT, "cores": nthr, "kind": "oracle", "cpu_model": cpu_model(),
                             "host_cores": cores, "build": "g++ -O2 -ffp-contract=off (plain oracle, not tuned)",
                             "sample": f"{steps} whole events, {nthr} threads over the 36 sectors"},
            "e2e": {"value": evs, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ---- the CUDA legs --------------------------------------------------------------------------------
def pipelined(trk, inputs, steps: int, first: int = 0, on_done=None, depth: int = None):
    """Track `steps` events with `depth` in flight (slot = step % depth); returns (tracks, kept clusters, bytes copied
    back).  on_done(slot, step, result) sees every result while it is still valid (views of the slot's pinned buffers)."""
    n = len(inputs)
    depth = depth or IN_FLIGHT
    tracks = kept = d2h = 0
    for i in range(steps + depth - 1):
        if i < steps:
            xyz, rs = inputs[(first + i) % n]
            trk.submit_event(xyz, rs, i % depth)
        j = i - (depth - 1)
        if j >= 0:
            r = trk.wait_event(j % depth, copy=False)
            tracks += len(r.tracks)
            kept += len(r.cluster_ids)
            d2h += r.tracks.nbytes + r.cluster_ids.nbytes + 64
            if on_done is not None:
                on_done(j % depth, j, r)
    return tracks, kept, d2h


def run_tpcst(args, rank: int, world: int, local_rank: int):
    import torch
    import torch.distributed as dist
    import paper_1712_09407_b200 as T

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the tracker has no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    extras = world == 1 and not args.stream and not args.no_extras
    n_gen = args.stream or (max(args.events, EXTRA_STREAM_EVENTS) if extras else args.events)
    all_events = gen_events(n_gen, rank, world)            # before CUDA is touched: the pool forks
    events = all_events if args.stream else all_events[:args.events]
    geo = events[0].geometry
    nmax = max(e.n_clusters for e in all_events)
    maxc, maxt = int(nmax * 1.05), int(nmax * 1.05) // 8
    cuts = {}
    for kv in args.cut:
        k, v = kv.split("=", 1)
        cuts[k] = float(v) if any(ch in v for ch in ".e") else int(v)
    trk = T.SectorTracker(geo, maxc, maxt, device=dev, **cuts)
    props = torch.cuda.get_device_properties(dev)

    if args.stream:
        run_stream(args, trk, events, dev, rank, world, local_rank)
        trk.close()
        if world > 1:
            dist.destroy_process_group()
        return
    dev_in = [(torch.from_numpy(e.xyz).to(dev), torch.from_numpy(e.row_start.astype(np.int32)).to(dev)) for e in events]
    host_in = [(torch.from_numpy(e.xyz).pin_memory(), torch.from_numpy(e.row_start.astype(np.int32)).pin_memory())
               for e in events]
    torch.cuda.synchronize(dev)

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    def timed(inputs, profile: bool):
        """W warm-up steps, then exactly K timed steps between barriers.  The interval is taken from two CUDA events
        recorded on the caller's compute stream, which every submit orders its slot's stream after and which carries
        none of the tracker's kernels (they run on the library's per-slot streams): the first is recorded before the
        first submit, the second after the last wait has returned (wait is host-synchronous), so the interval covers
        all device work of the region plus the host's last wake-up — device timestamps of a wall-clock bracket."""
        kms = []
        trk.set_profiling(1 if profile else 0)
        pipelined(trk, inputs, args.warmup)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        sampler = ClockSampler(local_rank)
        sampler.start()
        t0 = time.perf_counter()
        e0.record(trk.stream_compute)
        tracks, kept, d2h = pipelined(trk, inputs, args.steps, first=args.warmup,
                                      on_done=(lambda s, j, r: kms.append(trk.kernel_ms(s).copy())) if profile else None)
        e1.record(trk.stream_compute)       # after the last wait returned: everything of the region is done
        barrier()
        wall = time.perf_counter() - t0
        clocks = sampler.stop()
        ms = max(e0.elapsed_time(e1), 0.0)
        if world > 1:
            t = torch.tensor([ms], device=dev, dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms = float(t.item())
        trk.set_profiling(0)
        return ms, wall, tracks, kept, d2h, (np.mean(kms, axis=0) if kms else None), clocks

    # counting pass (untimed): work counters of every event + result sizes
    trk.set_profiling(2)
    work = {k: 0 for k in T.WORK_NAMES}
    n_tracklets = n_tracks = n_ids = 0
    for xyz, rs in dev_in:
        r = trk.track_event(xyz, rs, copy=False)
        for k, v in trk.work_counters(0).items():
            work[k] += v
        n_tracklets += r.n_tracklets
        n_tracks += len(r.tracks)
        n_ids += len(r.cluster_ids)
    E = len(events)
    work = {k: v / E for k, v in work.items()}
    trk.set_profiling(0)

    ms, wall, tracks, kept, d2h, _, clocks = timed(dev_in, profile=False)
    ms_e2e, wall_e2e, _, _, d2h_e2e, _, clocks_e2e = timed(host_in, profile=False)
    # per-kernel CUDA events: the same K steps once more with tpcst_set_profiling(1), which puts all slots on one
    # stream (overlapped, an event pair around a kernel would also time its wait for the other event's kernels)
    ms_prof, _, _, _, _, kms, _ = timed(dev_in, profile=True)

    n_clusters_step = float(np.mean([events[(args.warmup + i) % E].n_clusters for i in range(args.steps)]))
    h2d_step = float(np.mean([events[(args.warmup + i) % E].xyz.nbytes + events[(args.warmup + i) % E].row_start.nbytes
                              for i in range(args.steps)]))
    value = world * args.steps / (ms * 1e-3)
    e2e_value = world * args.steps / (ms_e2e * 1e-3)

    # per-kernel table and the dominant kernel's roofline
    nbins = float(trk_bins(geo, trk))
    n_avg = float(np.mean([e.n_clusters for e in events]))
    kernels = []
    traffic, traffic_capture, traffic_refused = ncu_traffic()
    for i, name in enumerate(trk.kernel_names):
        bound, amount, unit, peak = algorithmic(name, n_avg, nbins, n_tracklets / E, n_tracks / E, n_ids / E, work,
                                                props.multi_processor_count, clocks.get("sm_max_mhz") or 1965.0)
        t_ms = float(kms[i])
        ach = amount / (t_ms * 1e-3) / (1e9 if unit == "GB/s" else 1e12) if t_ms > 0 else 0.0
        kernels.append({"kernel": name, "ms": t_ms, "share": t_ms / float(kms.sum()), "bound": bound,
                        "achieved": ach, "peak": peak, "unit": unit, "frac": ach / peak,
                        # north_star quotes HBM fractions against ~8 TB/s nominal as well as the measured copy peak
                        "frac_of_nominal_8TBs": ach / NOMINAL_HBM_GBS if bound == "hbm" else None,
                        "algorithmic": amount, "traffic": traffic.get(name)})
        if name == "find_neighbours":      # north_star: "shared-memory / FP32 ALU for the pair loop" -- the same launch against the ALU peak
            ops = work["nf_window_tests"] * FLOP_NF_TEST + work["nf_pair_evals"] * FLOP_NF_PAIR + n_avg * FLOP_NF_CLUSTER
            alu_peak = props.multi_processor_count * 128 * (clocks.get("sm_max_mhz") or 1965.0) * 1e6 / 1e12
            kernels[-1]["alu"] = {"bound": "alu", "achieved": ops / (t_ms * 1e-3) / 1e12 if t_ms > 0 else 0.0, "peak": alu_peak,
                                  "unit": "TFLOP/s", "frac": ops / (t_ms * 1e-3) / 1e12 / alu_peak if t_ms > 0 else 0.0,
                                  "algorithmic": ops}
    top = max(kernels, key=lambda k: k["ms"])
    _, peak_src = _peaks()
    roofline = {"kernel": top["kernel"], "bound": top["bound"], "achieved": top["achieved"], "peak": top["peak"],
                "unit": top["unit"], "frac": top["frac"], "traffic": top["traffic"], "ms": top["ms"],
                "traffic_source": traffic_refused or f"not measured in this run (hardware counters need ncu): committed ncu --set full "
                                  f"capture {traffic_capture} of the same kernel sources (digest {kernel_source_digest()}, profiles/traffic.csv)",
                "peak_source": peak_src if top["bound"] == "hbm" else
                "derived: SMs x 128 fp32 lanes x max SM clock, one operation per lane per cycle (FMA contraction is off)"}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": WORKLOAD, "events": E, "clusters_per_event": n_avg,
                       "l2": "inputs larger than L2: every step touches ~0.5 GB of workspace and rotates over "
                             f"{E} distinct events of {n_avg * 12 / 1e6:.0f} MB", "in_flight": IN_FLIGHT,
                       "streams": "one compute stream per slot: the kernel sets of the events in flight overlap at their "
                                  "edges; `kernels` / `roofline` come from a second pass of the same steps with per-kernel "
                                  "CUDA events, which runs all slots on one stream (kernel_pass_ms_per_step)",
                       "parallelism": f"event-level data parallel x{world}, no collective"},
            "clusters_per_s": world * n_clusters_step * args.steps / (ms * 1e-3),
            "wall_ms_per_step": 1e3 * wall / args.steps,
            "tracks_per_event": tracks / args.steps, "tracklets_per_event": n_tracklets / E,
            "kernel_set_ms": float(kms.sum()), "kernel_pass_ms_per_step": ms_prof / args.steps,
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d_step, "d2h_bytes_per_step": d2h_e2e / args.steps,
                    "ms_per_step": ms_e2e / args.steps, "input_GB_per_s": world * h2d_step * args.steps / (ms_e2e * 1e-3) / 1e9,
                    "clocks": clocks_e2e},
            "gpu_launches": args.steps * trk.kernels_per_event,
            "roofline": roofline, "kernels": kernels, "work_per_event": work}
    default_ms = {name: float(kms[i]) for i, name in enumerate(trk.kernel_names)}
    trk.close()

    if extras:
        # Outside the timed legs above; each its own short measurement (CUDA events on the caller's stream, as in timed()).
        def quick(tr, inputs, steps, warm=4):
            pipelined(tr, inputs, warm)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize(dev)
            e0.record(tr.stream_compute)
            pipelined(tr, inputs, steps, first=warm)
            e1.record(tr.stream_compute)
            torch.cuda.synchronize(dev)
            return e0.elapsed_time(e1) / steps

        def kernel_pass(tr, inputs, steps):
            acc = []
            tr.set_profiling(1)
            pipelined(tr, inputs, 2)
            pipelined(tr, inputs, steps, first=2, on_done=lambda sl, j, r: acc.append(tr.kernel_ms(sl).copy()))
            tr.set_profiling(0)
            return dict(zip(tr.kernel_names, (float(v) for v in np.mean(acc, axis=0))))

        # (1) BASELINE.json configs[4] in small: one pass over EXTRA_STREAM_EVENTS distinct pinned-host events
        with T.SectorTracker(geo, maxc, maxt, device=dev, **cuts) as tr:
            rec = stream_pass(tr, all_events[:EXTRA_STREAM_EVENTS], dev, args.warmup, 4)
        line["stream"] = {k: rec[k] for k in ("value", "unit", "steps", "warmup", "ms_per_step", "input_GB_per_s", "clusters_per_s",
                                              "h2d_bytes_per_step", "d2h_bytes_per_step", "check", "clocks")}
        line["stream"]["workload"] = rec["config"]["workload"]
        # (2) every optional stage on its own: pipelined device-resident events/s and what its kernels cost
        opt_steps = max(8, min(args.steps, 40))
        line["options"] = []
        for label, oc in OPTIONS:
            with T.SectorTracker(geo, maxc, maxt, device=dev, **{**cuts, **oc}) as tr:
                ms_o = quick(tr, dev_in, opt_steps)
                km = kernel_pass(tr, dev_in, 8)
                r = tr.track_event(*dev_in[0], copy=False)
                n_tr, n_gl, n_mg = len(r.tracks), len(r.global_ext), len(r.merge)
            changed = {k: round(v, 5) for k, v in km.items() if k not in default_ms or abs(v - default_ms[k]) > 0.01}
            line["options"].append({"option": label, "value": 1e3 / ms_o, "unit": UNIT, "ms_per_step": ms_o,
                                    "steps": opt_steps, "kernel_set_ms": sum(km.values()),
                                    "extra_kernel_ms": sum(km.values()) - sum(default_ms.values()),
                                    "kernels_ms_new_or_changed": changed, "tracks": n_tr, "global_ext": n_gl, "merge_records": n_mg})
        # (3) the small configurations (BASELINE.json configs[0..2]): single-event latency of tpcst_track_event, best of 5,
        #     next to the oracle on one thread, best of 3
        from oracle import Oracle
        from tpcsynth import generate_event
        line["small_configs"] = []
        for cfg in (1, 2, 3):
            ev = generate_event(cfg)
            with T.SectorTracker(ev.geometry, max(ev.n_clusters, 1), max(ev.n_clusters // 8, 1024), device=dev) as tr:
                xyz_d = torch.from_numpy(ev.xyz).to(dev)
                rs_d = torch.from_numpy(ev.row_start.astype(np.int32)).to(dev)
                torch.cuda.synchronize(dev)
                lat, gms = [], []
                for _ in range(8):
                    t0 = time.perf_counter()
                    r = tr.track_event(xyz_d, rs_d, copy=False)
                    lat.append(1e3 * (time.perf_counter() - t0))
                    gms.append(r.gpu_ms)
                n_tr = len(r.tracks)
            orc = Oracle.for_geometry(ev.geometry)
            ot = []
            for _ in range(3):
                t0 = time.perf_counter()
                orc.run(ev.xyz, ev.row_start, n_threads=1, fetch=False)
                ot.append(1e3 * (time.perf_counter() - t0))
            line["small_configs"].append({"config": f"BASELINE.json configs[{cfg - 1}]", "clusters": ev.n_clusters, "tracks": n_tr,
                                          "gpu_kernel_set_ms": min(gms[3:]), "gpu_call_latency_ms": min(lat[3:]),
                                          "oracle_single_thread_ms": min(ot), "timing": "GPU best of 5 after 3 warm-up calls, oracle best of 3"})

    if rank == 0:
        if world == 1 and not args.no_cpu_baseline:
            cores = os.cpu_count() or 1
            nthr = min(cores, 36)
            _, _, dt_one = oracle_events_per_s(events, 1, 0, nthr)        # sizes the sample to ~12 s of work
            n_ev = int(min(64, max(2, round(12.0 / dt_one))))
            evs, cls, dt = oracle_events_per_s(events, n_ev, 0, nthr)
            singles = [oracle_events_per_s(events, 1, 0, 1)[2] for _ in range(3 if extras else 1)]   # seconds for one event
            evs1 = 1.0 / min(singles)
            line["cpu_baseline"] = {"value": evs, "unit": UNIT, "cores": nthr, "kind": "oracle", "cpu_model": cpu_model(),
                                    "host_cores": cores, "build": "g++ -O2 -ffp-contract=off (plain oracle, not tuned)",
                                    "sample": f"{n_ev} whole events of the same workload in {dt:.1f} s, {nthr} threads over "
                                              f"the 36 sectors; single thread: best of {len(singles)} runs of one event",
                                    "single_thread_value": evs1, "single_thread_runs_s": singles, "clusters_per_s": cls}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def stream_pass(trk, events, dev, warmup: int, n_check: int, rank: int = 0, world: int = 1, local_rank: int = 0) -> dict:
    """BASELINE.json configs[4]: a stream of N distinct seeded central Pb-Pb-like events in pinned host
    buffers, tracked back to back ONCE (no event is visited twice inside the timed region); the H2D copy
    of event e + 1 runs on the copy stream while event e is tracked (a8).  Returns the record of the pass."""
    import torch
    import torch.distributed as dist
    host_in = [(torch.from_numpy(e.xyz).pin_memory(), torch.from_numpy(e.row_start.astype(np.int32)).pin_memory())
               for e in events]
    N = len(host_in)
    pipelined(trk, host_in, min(warmup, N))                      # warm-up on the first events of the same stream
    torch.cuda.synchronize(dev)
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.perf_counter()
    e0.record(trk.stream_compute)
    tracks, kept, d2h = pipelined(trk, host_in, N)
    e1.record(trk.stream_compute)
    torch.cuda.synchronize(dev)
    wall = time.perf_counter() - t0
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1)
    # check (after the timed region, so that it costs the measurement nothing): the stream is tracked ONCE MORE in
    # the same pipelined way and a fingerprint of the picked results is taken while they are valid; then the picked
    # events are tracked again one at a time (nothing else in flight) and must give the same bytes: the overlapped
    # streams, copies and slots changed nothing (a race detector; the comparison with the oracle is
    # tests/test_gpu_parity.py::test_bench_launch_configuration_at_full_size)
    import zlib
    n_check = min(n_check, N)
    stride = max(1, N // n_check) if n_check else 0
    picked = set(range(0, N, stride)[:n_check]) if n_check else set()
    prints = {}
    def fingerprint(slot, j, r):
        if j in picked:
            prints[j] = (len(r.tracks), zlib.crc32(r.tracks.tobytes()), zlib.crc32(r.cluster_ids.tobytes()))
    if picked:
        pipelined(trk, host_in, N, on_done=fingerprint)
    mismatches = []
    for j in sorted(picked):
        r = trk.track_event(*host_in[j], copy=False)
        again = (len(r.tracks), zlib.crc32(r.tracks.tobytes()), zlib.crc32(r.cluster_ids.tobytes()))
        if again != prints[j]:
            mismatches.append(j)
    if mismatches:
        raise SystemExit(f"bench.py stream check: events {mismatches} differ between the pipelined pass and a synchronous re-run")
    if world > 1:
        t = torch.tensor([ms], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    h2d = float(sum(e.xyz.nbytes + e.row_start.nbytes for e in events))
    ncl = float(sum(e.n_clusters for e in events))
    return {
        "metric": "central_pbpb_like_stream_events_per_s", "value": world * N / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
        "steps": N, "warmup": min(warmup, N), "ms_per_step": ms / N, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[4]: stream of {N} seeded central Pb-Pb-like events, pinned host "
                               "buffers, H2D of event e+1 overlaps tracking of event e", "events": N, "in_flight": IN_FLIGHT,
                   "clusters_per_event": ncl / N, "pinned_host_GB": h2d / 1e9},
        "input_GB_per_s": world * h2d / (ms * 1e-3) / 1e9, "clusters_per_s": world * ncl / (ms * 1e-3),
        "wall_ms_per_step": 1e3 * wall / N, "tracks_per_event": tracks / N,
        "h2d_bytes_per_step": h2d / N, "d2h_bytes_per_step": d2h / N, "gpu_launches": N * trk.kernels_per_event,
        "clocks": clocks,
        "check": {"events_rechecked": len(picked), "mismatches": 0} if picked else None,
        "paper_context": "PAPER.md L10: > 200 Hz central Pb-Pb, ~25 GB/s of raw data into the whole HLT farm (other "
                         "hardware, other input format: context, not a baseline)"}


def run_stream(args, trk, events, dev, rank: int, world: int, local_rank: int):
    rec = stream_pass(trk, events, dev, args.warmup, args.check, rank, world, local_rank)
    if rank == 0:
        print(json.dumps(rec))


def _scaled_event(args):
    from dataclasses import replace
    from tpcsynth import CONFIGS, generate_event
    frac, seed = args
    cfg = replace(CONFIGS[4], n_primaries=int(round(20000 * frac)), n_secondaries=int(round(3000 * frac)))
    return generate_event(cfg, seed)


def run_size_sweep(args, local_rank: int):
    """PAPER.md L112 / Fig. 9: "both CPU and GPU tracking time depend linearly on the input data size the GPU tracker
    having a small offset".  Central Pb-Pb-like events scaled to 1/8 ... 3/2 of BASELINE.json configs[3]; per size the
    device-resident pipelined time per event (as `value`), and the oracle on the host threads; a straight-line fit."""
    import torch
    import paper_1712_09407_b200 as T
    from concurrent.futures import ProcessPoolExecutor
    import multiprocessing as mp
    fracs = (0.125, 0.25, 0.5, 0.75, 1.0, 1.5)
    with ProcessPoolExecutor(max_workers=min(os.cpu_count() or 1, 12), mp_context=mp.get_context("fork")) as ex:
        evs = list(ex.map(_scaled_event, [(fr, 5000 + 10 * i + e) for i, fr in enumerate(fracs) for e in range(2)]))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    nmax = max(e.n_clusters for e in evs)
    trk = T.SectorTracker(evs[0].geometry, int(nmax * 1.05), int(nmax * 1.05) // 8, device=dev)
    from oracle import Oracle
    orc = Oracle.for_geometry(evs[0].geometry)
    nthr = min(os.cpu_count() or 1, 36)
    pts = []
    for i, fr in enumerate(fracs):
        pair = evs[2 * i: 2 * i + 2]
        dev_in = [(torch.from_numpy(e.xyz).to(dev), torch.from_numpy(e.row_start.astype(np.int32)).to(dev)) for e in pair]
        pipelined(trk, dev_in, max(args.warmup, 3))
        torch.cuda.synchronize(dev)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(trk.stream_compute)
        tracks, _, _ = pipelined(trk, dev_in, args.steps)
        e1.record(trk.stream_compute)
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        for e in pair:
            orc.run(e.xyz, e.row_start, n_threads=nthr, fetch=False)
        cpu_ms = 1e3 * (time.perf_counter() - t0) / len(pair)
        pts.append({"fraction": fr, "clusters": float(np.mean([e.n_clusters for e in pair])), "tracks": tracks / args.steps,
                    "gpu_ms_per_event": e0.elapsed_time(e1) / args.steps, "oracle_ms_per_event": cpu_ms})
    trk.close()
    x = np.array([p["clusters"] for p in pts])
    out = {"metric": "time_vs_input_size", "unit": "ms/event", "steps": args.steps, "points": pts, "oracle_threads": nthr}
    for key in ("gpu_ms_per_event", "oracle_ms_per_event"):
        y = np.array([p[key] for p in pts])
        a, b = np.polyfit(x, y, 1)
        out[key.replace("_ms_per_event", "_fit")] = {"ns_per_cluster": 1e6 * a, "offset_ms": b,
                                                    "max_rel_residual": float(np.max(np.abs(a * x + b - y) / y))}
    print(json.dumps(out))


def run_alpha_scan(args, local_rank: int):
    """PAPER.md L88-L94 / Fig. 6: the chi2-suppression factor alpha of the weighted cluster assignment, scanned on
    synthetic truth (central Pb-Pb-like event): tracks found, efficiency for findable particles (>= 30 clusters in one
    sector), clones, fakes (< 80 % of the clusters from one particle), clusters per track, cluster purity.
    alpha -> infinity is the length rule (select_mode 0, the last line)."""
    import torch
    import paper_1712_09407_b200 as T
    from tpcsynth import generate_event
    ev = generate_event(4)
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    R = ev.geometry.n_rows
    sr = np.repeat(np.arange(len(ev.row_start) - 1), np.diff(ev.row_start.astype(np.int64)))
    sec = sr // R
    tid = ev.truth_id.astype(np.int64)
    real = tid != 0xFFFFFFFF
    per = np.bincount(tid[real] * 36 + sec[real])                       # clusters of particle p in sector s
    findable = int((per >= 30).sum())
    rows = []
    for alpha in (1.0, 2.0, 3.0, 4.0, 6.0, 8.0, 12.0, 25.0, None):
        cuts = {"select_mode": 0} if alpha is None else {"select_mode": 1, "alpha": alpha}
        with T.SectorTracker(ev.geometry, ev.n_clusters, ev.n_clusters // 8, device=dev, **cuts) as trk:
            r = trk.track_event(ev.xyz, ev.row_start)
        first, n = r.tracks["first_cluster"].astype(np.int64), r.tracks["n_clusters"].astype(np.int64)
        t_of = tid[r.cluster_ids]
        fakes = purity_num = clones = 0
        seen = set()
        for k in range(len(n)):
            cl = t_of[first[k]: first[k] + n[k]]
            v, c = np.unique(cl, return_counts=True)
            j = c.argmax()
            purity_num += int(c[j])
            if v[j] == 0xFFFFFFFF or c[j] < 0.8 * n[k]:
                fakes += 1
                continue
            key = (int(v[j]), int(r.tracks["sector"][k]))
            if key in seen:
                clones += 1
            seen.add(key)
        found = sum(1 for (p, s) in seen if per[p * 36 + s] >= 30)
        rows.append({"alpha": alpha, "tracks": int(len(n)), "efficiency": found / findable, "clone_rate": clones / max(len(n), 1),
                     "fake_rate": fakes / max(len(n), 1), "clusters_per_track": float(n.mean()),
                     "cluster_purity": purity_num / float(n.sum())})
    print(json.dumps({"metric": "alpha_scan", "event": "BASELINE.json configs[3], seed 4", "findable": findable, "rows": rows}))


def run_l2_random(args, local_rank: int):
    """Reference point for the selection kernels (select_claim, select_collect, write_ids), which are bound by random
    4-byte accesses to an L2-resident array (owner[] / s_orig[], ~15 MB): the rate this GPU sustains for that pattern in
    two plain microkernels of the library's self-test (tpcst_selftest_random_access: uniformly random gathers, and atomic maxima whose
    result is not used, four independent accesses in flight per thread) over an array of the central event's size and as
    many accesses as the event claims hits, next to the tracker's kernels on the same event (CUDA events)."""
    import torch
    import paper_1712_09407_b200 as T
    from tpcsynth import generate_event
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    ev = generate_event(4)
    with T.SectorTracker(ev.geometry, ev.n_clusters, ev.n_clusters // 8, device=dev) as trk:
        trk.set_profiling(2)
        trk.track_event(ev.xyz, ev.row_start)
        claimed = trk.work_counters(0)["claimed_hits"]
        trk.set_profiling(1)
        kms = np.mean([(trk.track_event(ev.xyz, ev.row_start), trk.kernel_ms(0).copy())[1] for _ in range(10)], axis=0)
        ms = dict(zip(trk.kernel_names, kms))
    n = ev.n_clusters + 16 * 36 * 159
    t_gather, t_red = T.selftest_random_access(n, claimed, reps=20, device=dev)
    print(json.dumps({
        "metric": "random_l2_access_rate", "unit": "G accesses/s", "accesses": claimed, "array_MB": n * 4 / 1e6,
        "device_gather": {"ms": t_gather, "rate": claimed / t_gather / 1e6},
        "device_red_max": {"ms": t_red, "rate": claimed / t_red / 1e6},
        "select_claim": {"ms": float(ms["select_claim"]), "rate": claimed / float(ms["select_claim"]) / 1e6,
                         "frac_of_device_red_max": t_red / float(ms["select_claim"])},
        "select_collect": {"ms": float(ms["select_collect"]), "rate": claimed / float(ms["select_collect"]) / 1e6,
                           "frac_of_device_gather": t_gather / float(ms["select_collect"])},
        "note": "device_* = tpcst_selftest_random_access (best of 20 launches, uniform random indices); the tracker's kernels also read a "
                "2-byte hit and a row offset per access and walk items of 32 rows, and their indices are not uniform: "
                "clusters of one track sit in neighbouring rows' slabs"}))


def trk_bins(geo, trk) -> int:
    """Number of grid bins of one event (host arithmetic of DESIGN.md section 3, G4)."""
    c = trk.cuts
    nz = int(np.ceil(float(geo.z_max) / float(c.bin_z))) + 1
    ymax = (geo.row_x.astype(np.float64) * float(geo.tan_half_angle)).astype(np.float32).astype(np.float64)
    ny = np.ceil(2.0 * ymax / float(c.bin_y)) + 1
    return int(ny.sum()) * nz * int(geo.n_sectors)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=4)
    ap.add_argument("--events", type=int, default=4, help="distinct synthetic events visited round robin")
    ap.add_argument("--stream", type=int, default=0, metavar="N",
                    help="BASELINE.json configs[4] instead of the default legs: N distinct events (256 in the config), "
                         "pinned host buffers, one pass, sustained events/s and input GB/s")
    ap.add_argument("--check", type=int, default=0, metavar="N",
                    help="with --stream: after the timed region, track the stream once more in the pipelined way and N of its events synchronously, and compare the bytes")
    ap.add_argument("--size-sweep", action="store_true", help="time per event vs input size (PAPER.md Fig. 9) instead of the default legs")
    ap.add_argument("--alpha-scan", action="store_true", help="chi2-suppression factor scan on synthetic truth (PAPER.md Fig. 6)")
    ap.add_argument("--l2-random", action="store_true",
                    help="reference point for the selection kernels: the device's random gather / red.max rate over an array of the event's size (tpcst_selftest_random_access)")
    ap.add_argument("--impl", default="tpcst", choices=["tpcst", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true",
                    help="skip what the default single-GPU run measures after its timed legs: `stream` (32 distinct pinned-host "
                         "events, one pass), `options` (every optional stage on its own), `small_configs` (configs 1-3)")
    ap.add_argument("--cut", action="append", default=[], metavar="KEY=VALUE",
                    help="override one field of tpcst_cuts (tuning experiments, e.g. --cut bin_y=1.0)")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    args.warmup = max(args.warmup, 3) if args.impl == "tpcst" else args.warmup
    if args.size_sweep or args.alpha_scan or args.l2_random:
        if rank == 0:
            args.steps = min(args.steps, 60)
            (run_size_sweep if args.size_sweep else (run_alpha_scan if args.alpha_scan else run_l2_random))(args, local_rank)
    elif args.impl == "reference":
        run_reference(args, rank)
    else:
        run_tpcst(args, rank, world, local_rank)


if __name__ == "__main__":
    main()

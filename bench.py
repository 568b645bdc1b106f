#!/usr/bin/env python
"""bench.py -- central Pb-Pb-like events/s (and clusters/s) of the TPC tracker hot path on B200.

One *step* = one pass of the whole hot path (K1 bucket/grid sort, K2 neighbour finder, K3 cleaner, K4 start hits,
K5 Kalman tracklet constructor, K6 selector + output) over one batch of 16 synthetic central Pb-Pb-like events
(BASELINE.json config 5 = 16 x config 4), through the C ABI call ``tpc_track_events``.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--events E] [--workload central]

* default arm: ``value`` = events/s with the inputs resident in HBM; ``e2e`` = the same work from pinned HOST
  buffers (H2D of the clusters and D2H of the tracks inside the timed region) through ``tpc_submit_events`` /
  ``tpc_wait_events`` with three batches in flight (``e2e.single_call``: ``tpc_track_events``, one call at a time); ``roofline`` = the dominant kernel
  (K5) against the measured HBM copy bandwidth; ``cpu_baseline`` = the oracle timed on the host cores.
* ``--impl reference``: the CPU oracle, as it stands, on the host cores (one event per step).
* N > 1 (torchrun): replicas only -- every rank tracks its own batch on its own GPU; no collective on the data path.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "central_pbpb_events_per_s"
UNIT = "events/s"


HBM_NOMINAL_GBS = 8000.0   # BASELINE.json:5 "nominal ~8 TB/s"


def measured_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def run_config(args, n_events):
    """What identifies a measured configuration (profiles/traffic.json is valid for exactly one)."""
    return {"workload": args.workload, "events": n_events, "link_step": args.link_step, "refit": bool(args.refit),
            "merge": bool(args.merge), "seed_dedup": not args.no_seed_dedup}


def committed_traffic(cfg):
    """DRAM bytes per step of each stage from the committed ncu --set full capture -- only when that capture was
    taken on this very configuration; tagged with the commit it was taken at."""
    tf = ROOT / "profiles" / "traffic.json"
    if not tf.exists():
        return None
    d = json.loads(tf.read_text())
    if d.get("config") != cfg:
        return None
    return d


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz, self._stop_evt = index, [], set(), None, threading.Event()
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
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20,
                 "hw_power_brake_slowdown": 0x80, "sync_boost": 0x10, "applications_clocks_setting": 0x2}
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop_evt.wait(0.1)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons)}


def event_seeds(workload, n_events, rank=0):
    """Seeds of the events rank `rank` tracks: replicas only -- every rank has its OWN batch
    of n_events events, disjoint from the other ranks'; rank 0's batch is the single-GPU batch."""
    from paper_1712_09416_b200 import gen
    recipe = gen.RECIPES[workload]
    base = 1000 * gen.RECIPES["central_batch16"].config_id if workload == "central" else 1000 * recipe.config_id
    return [base + rank * n_events + e for e in range(n_events)]


def make_events(workload, n_events, rank=0):
    from paper_1712_09416_b200 import gen
    return [gen.generate(gen.RECIPES[workload], seed=s) for s in event_seeds(workload, n_events, rank)]


def stage_bytes(c):
    """Algorithmic bytes per stage from the run's own counters."""
    N, S, V, A, T, H, B = (c[k] for k in ("n_clusters", "n_seeds", "n_row_visits", "n_tracklet_hits", "n_tracks",
                                          "n_track_hits", "n_tracklets"))
    return {
        "K1_sort_grid": 26 * N,
        "K2_neighbours": 18 * N,
        "K3K4_clean_seeds": 24 * N + 36 * S,
        "K5_construct": 12 * V + 4 * A + 36 * S + 124 * B,
        "K6_select": 16 * A + 4 * H + 44 * T,
        "K7_refit": (12 * H + 44 * T) if c.get("n_refit_visits", 0) else 0,
    }


def k5_flops(c):
    """Algorithmic float32 operations of K5: + - x / sqrt count 1 each, as the method
    writes them (no fused multiply-add): 164 per row visit (transport 160, gate weights 4), 107 per accepted
    measurement (gate 7, two scalar updates 100)."""
    return 164 * c["n_row_visits"] + 107 * c["n_updates"]


def cpu_baselines(evs, rx, gen):
    """The oracle as it stands, timed on the host cores on bounded samples of the workload: all
    hardware threads in strict-float32 mode (the reference of the parity tests) and in double, and one thread."""
    import oracle
    geom = oracle.Geometry(evs[0].n_sectors, rx, gen.TAN_HALF_ANGLE, evs[0].sigma, evs[0].sigma, evs[0].bz)
    cores = oracle.max_threads()
    out = {}
    nb = min(2, len(evs))
    t0 = time.perf_counter()
    for ev in evs[:nb]:
        oracle.track_event(geom, ev.sector_offset, ev.y, ev.z, ev.row, precision="float")
    dt = time.perf_counter() - t0
    out.update({"value": nb / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                "sample": "first %d events of the batch (%d clusters), strict-float32 mode, OpenMP over sectors"
                          % (nb, sum(ev.n_clusters for ev in evs[:nb]))})
    ev = evs[0]
    t0 = time.perf_counter()
    oracle.track_event(geom, ev.sector_offset, ev.y, ev.z, ev.row, precision="double")
    dt = time.perf_counter() - t0
    out["double"] = {"value": 1.0 / dt, "unit": UNIT, "cores": cores,
                     "sample": "first event of the batch (%d clusters), double mode" % ev.n_clusters}
    # one thread: the first sectors of the first event (about a ninth of it), scaled to whole events
    ns1 = max(1, min(4, ev.n_sectors))
    g1 = oracle.Geometry(ns1, rx, gen.TAN_HALF_ANGLE, ev.sigma, ev.sigma, ev.bz)
    n1 = int(ev.sector_offset[ns1])
    t0 = time.perf_counter()
    oracle.track_event(g1, ev.sector_offset[:ns1 + 1], ev.y[:n1], ev.z[:n1], ev.row[:n1], precision="float", n_threads=1)
    dt = time.perf_counter() - t0
    out["one_thread"] = {"value": (n1 / max(ev.n_clusters, 1)) / dt, "unit": UNIT, "cores": 1,
                         "sample": "sectors 0-%d of the first event (%d of its %d clusters) on one thread, strict-float32 "
                                   "mode, scaled to whole events by the cluster share" % (ns1 - 1, n1, ev.n_clusters)}
    return out


def fp32_peak_tflops(sm_count, sm_max_mhz):
    """FP32 peak of the device from its unit counts and clock: SMs x 128 FP32 lanes x 2 (fused multiply-add) x
    max SM clock.  The path's arithmetic is un-fused by definition, so half of this is its ceiling."""
    return sm_count * 128 * 2 * (sm_max_mhz or 1965.0) * 1e6 / 1e12


def max_over_ranks(ms, world, device="cuda"):
    """Elapsed time of the job = the slowest rank's (all_reduce MAX; identity for one rank)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(events_per_rank, steps, ms, world):
    """Whole-job events/s: every rank tracked its own events_per_rank x steps events in ms milliseconds."""
    return world * events_per_rank * steps / (ms * 1e-3)


def run_reference(args, rank, world):
    """The CPU oracle (unmodified, strict-float32 mode, all host threads) -- one event per step."""
    if rank != 0:
        return
    import oracle
    from paper_1712_09416_b200 import gen
    evs = make_events(args.workload, max(1, min(args.events, args.steps + args.warmup)))
    rx = gen.row_x().astype(np.float32)
    geom = oracle.Geometry(evs[0].n_sectors, rx, gen.TAN_HALF_ANGLE, evs[0].sigma, evs[0].sigma, evs[0].bz)
    cores = oracle.max_threads()

    def one(ev):
        return oracle.track_event(geom, ev.sector_offset, ev.y, ev.z, ev.row, precision="float")
    for w in range(args.warmup):
        one(evs[w % len(evs)])
    t0 = time.perf_counter()
    ncl = 0
    for k in range(args.steps):
        ev = evs[k % len(evs)]
        one(ev)
        ncl += ev.n_clusters
    dt = time.perf_counter() - t0
    v = args.steps / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": "%d x central Pb-Pb-like events per step (BASELINE.json config 5 = 16 x config 4)" % args.events
                               if args.workload == "central" else "%d x %s event(s) per step" % (args.events, args.workload),
                   "sample": "each step of this arm is ONE event of that batch (bounded sample), CPU oracle"},
        "clusters_per_s": ncl / dt,
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": "%d steps x 1 event (~%d clusters each), strict-float32 mode, OpenMP over sectors"
                                   % (args.steps, ncl // max(args.steps, 1))},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--events", type=int, default=16, help="events per batch (one step)")
    ap.add_argument("--workload", default="central", choices=["central", "semicentral", "pp", "single_sector", "dense"],
                    help="dense = 2.5 x the central multiplicity (SURVEY.md 8(f).4; not a BASELINE.json config)")
    ap.add_argument("--no-seed-dedup", action="store_true", help="fit every start hit (round-1 behaviour)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--group-events", type=int, default=0,
                    help="measurement of event waves (SURVEY.md 8(f).3): cut the device-resident batch into groups of this "
                         "many events on separate streams (at most four groups) and print only the step time")
    ap.add_argument("--link-step", type=int, default=1, choices=[1, 2], help="neighbour rows r +- step (SURVEY.md 8(f).4)")
    ap.add_argument("--merge", action="store_true", help="also link segments across sector borders (O9, SURVEY.md 8(f).2; implies --refit)")
    ap.add_argument("--refit", action="store_true", help="also refit the output tracks (O8, SURVEY.md 8(f).1; not part of the headline path)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the tracker has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    from paper_1712_09416_b200 import gen, tracker

    evs = make_events(args.workload, args.events, rank)
    n_total = sum(ev.n_clusters for ev in evs)
    rx = gen.row_x().astype(np.float32)
    params = None
    args.refit = args.refit or args.merge
    if args.refit or args.link_step != 1 or args.no_seed_dedup:
        params = tracker.tpc_default_params()
        params.refit = int(args.refit)
        params.merge = int(args.merge)
        params.link_step = args.link_step
        params.seed_dedup = int(not args.no_seed_dedup)
    trk = tracker.Tracker(evs[0].n_sectors, rx, gen.TAN_HALF_ANGLE, evs[0].sigma, evs[0].sigma, evs[0].bz,
                          params=params, max_events=len(evs), max_clusters=n_total)
    stream = torch.cuda.Stream()
    trk.set_stream(stream.cuda_stream)
    trk.tpc_tracker_set_profiling(not args.group_events)   # (per-stage events are per group: off in the wave measurement)
    if args.group_events:
        trk.tpc_tracker_set_group_events(args.group_events)

    dev_in = [dict(sector_offset=ev.sector_offset, y=torch.from_numpy(ev.y).cuda(), z=torch.from_numpy(ev.z).cuda(),
                   row=torch.from_numpy(ev.row).cuda()) for ev in evs]

    def pinned(a):
        t = torch.empty(a.shape, dtype=torch.from_numpy(a).dtype, pin_memory=True)
        t.numpy()[...] = a
        return t
    host_keep = [(pinned(ev.y), pinned(ev.z), pinned(ev.row)) for ev in evs]
    host_in = [dict(sector_offset=ev.sector_offset, y=k[0].numpy(), z=k[1].numpy(), row=k[2].numpy())
               for ev, k in zip(evs, host_keep)]

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(inputs, steps, collect_stages):
        stages = np.zeros(6)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record(stream)
        outs = None
        launches = 0
        for _ in range(steps):
            outs = trk.tpc_track_events(inputs)
            launches += trk.tpc_get_counters()["n_kernel_launches"]
            if collect_stages:
                stages += np.array(trk.tpc_get_stage_ms())
        e1.record(stream)
        barrier()
        ms = max_over_ranks(e0.elapsed_time(e1), world)
        return ms, stages / max(steps, 1), outs, launches

    for _ in range(args.warmup):
        trk.tpc_track_events(dev_in)
    sampler = ClockSampler(local_rank)
    sampler.start()
    ms, stage_ms, outs, launches = timed(dev_in, args.steps, True)
    counters = trk.tpc_get_counters()
    # Second pass, the one `value` comes from when the batch is more than one wave of the constructor's CTAs: the same
    # batch cut into TWO groups of events on two streams (tpc_tracker_set_group_events, a public knob; results do not
    # depend on it).  Each group's K5 is then a single wave of sector tasks and the groups' kernels overlap: measured
    # 6.68 against 7.21 ms per step on 16 central events (profiles/r3_waves.md).  Per-stage CUDA events are per group and
    # would overlap, so the stage times, the roofline and the counters stay those of the one-group pass above.
    two_groups = None
    if not args.group_events and len(evs) >= 2 and len(evs) * evs[0].n_sectors > 2 * 148:
        trk.tpc_tracker_set_profiling(False)
        trk.tpc_tracker_set_group_events((len(evs) + 1) // 2)
        for _ in range(args.warmup):
            trk.tpc_track_events(dev_in)
        ms2, _, outs2, launches2 = timed(dev_in, args.steps, False)
        assert [o.n_tracks for o in outs2] == [o.n_tracks for o in outs]
        assert sum(o.n_track_hits for o in outs2) == sum(o.n_track_hits for o in outs)
        two_groups = {"one_group_profiled_ms_per_step": ms / args.steps, "one_group_gpu_launches": int(launches),
                      "groups": 2, "events_per_group": (len(evs) + 1) // 2,
                      "note": "value / ms_per_step / gpu_launches: the batch as two groups of events on two streams, "
                              "CUDA-graph replay, no per-stage events; stages / roofline / counters: a separate pass of the "
                              "same K steps as one group with per-stage CUDA events (its ms_per_step given here)"}
        ms, outs, launches = ms2, outs2, launches2
        trk.tpc_tracker_set_group_events(0)
        trk.tpc_tracker_set_profiling(True)
    clocks = sampler.stop()
    if args.group_events:      # wave measurement: the step time of the same batch run as groups; nothing else is reported
        if rank == 0:
            print(json.dumps({"metric": METRIC, "value": aggregate_value(len(evs), args.steps, ms, world), "unit": UNIT,
                              "ms_per_step": ms / args.steps, "steps": args.steps, "warmup": args.warmup, "n_gpus": world,
                              "config": {"workload": args.workload, "events_per_step": len(evs),
                                         "group_events": args.group_events,
                                         "note": "device-resident batch cut into groups of events on separate streams; "
                                                 "synchronous tpc_track_events calls, timed around the calls"},
                              "gpu_launches": int(launches), "clocks": clocks}))
        trk.close()
        if world > 1:
            dist.destroy_process_group()
        return
    n_tracks = sum(o.n_tracks for o in outs)
    n_hits = sum(o.n_track_hits for o in outs)

    e2e = None
    if not args.no_e2e:
        for _ in range(2):
            trk.tpc_track_events(host_in)
        ms_e, _, outs_e, _ = timed(host_in, args.steps, False)
        assert sum(o.n_tracks for o in outs_e) == n_tracks
        e2e = {"value": aggregate_value(len(evs), args.steps, ms_e, world), "unit": UNIT,
               "h2d_bytes_per_step": int(12 * n_total + sum(4 * (ev.n_sectors + 1) for ev in evs)),
               "d2h_bytes_per_step": int(44 * n_tracks + 4 * n_hits), "ms_per_step": ms_e / args.steps}
        # Pipelined: tpc_submit_events / tpc_wait_events keep three batches in flight on one tracker, so that the copies
        # of one batch overlap the kernels of the other.  Same host buffers, same bytes per step; every step's result
        # is waited for and read.  Reported beside the single-call figure, not instead of it.
        trk.tpc_tracker_set_profiling(False)
        for _ in range(2):                # warm-up with all tickets in flight (each owns its work space and buffers)
            tk = [trk.tpc_submit_events(host_in) for _ in range(3)]
            for x in tk:
                trk.tpc_wait_events(x)
        # Steady state of the pipeline: two batches are submitted and W untimed rounds of (submit, wait) run BEFORE the
        # timed region, and the two batches still in flight at its end are waited for AFTER it, so that the region
        # holds exactly K submits (K x the H2D copies), K waits (K results read, K x the D2H copies) and K x the
        # kernels -- what is in flight when it starts equals what is in flight when it ends.  (Timing the fill and the
        # drain as well adds ~1.7 ms per step at K = 10 and ~0.4 ms at K = 40: that is start-up, not throughput.)
        barrier()
        flight = [trk.tpc_submit_events(host_in) for _ in range(2)]   # (no device synchronisation from here to e1)
        for _ in range(max(args.warmup, 3)):                          # untimed rounds until the pipeline runs steadily
            flight.append(trk.tpc_submit_events(host_in))
            trk.tpc_wait_events(flight.pop(0))
        # Timer: the host clock.  The work runs on the library's own streams (CUDA events recorded on torch's current
        # stream would not see it), and every tpc_wait_events blocks until its batch's results are in host memory, so
        # the wall time of K (submit, wait) rounds in steady state is the end-to-end time of K steps.
        t0 = time.perf_counter()
        # three batches in flight: the clusters of step k+2 are on their way in while the kernels of step k+1 run and
        # the tracks of step k go out
        for k in range(args.steps):
            flight.append(trk.tpc_submit_events(host_in))
            got = sum(o.n_tracks for o in trk.tpc_wait_events(flight.pop(0)))
            assert got == n_tracks
        t1 = time.perf_counter()
        barrier()
        for x in flight:                  # drain
            got = sum(o.n_tracks for o in trk.tpc_wait_events(x))
            assert got == n_tracks
        torch.cuda.synchronize()
        ms_p = max_over_ranks((t1 - t0) * 1e3, world)
        assert got == n_tracks
        # headline: the steady-state throughput of the asynchronous calls; the one-call-at-a-time figure beside it
        e2e = {"value": aggregate_value(len(evs), args.steps, ms_p, world), "unit": UNIT,
               "h2d_bytes_per_step": e2e["h2d_bytes_per_step"], "d2h_bytes_per_step": e2e["d2h_bytes_per_step"],
               "ms_per_step": ms_p / args.steps,
               "api": "tpc_submit_events / tpc_wait_events, three batches in flight on one tracker; every step copies its "
                      "clusters in from pinned host memory and its tracks out, and every result is waited for and read; "
                      "steady state: the pipeline is primed (two batches + the warm-up rounds) before the timed region, which "
                      "holds K submits and K waits, and drained after it",
               "timer": "host perf_counter around the K (submit, wait) rounds; every wait blocks until its batch's tracks "
                        "are in host memory (the work runs on the library's own streams)",
               "single_call": {"value": e2e["value"], "unit": UNIT, "ms_per_step": e2e["ms_per_step"],
                               "api": "tpc_track_events, one call at a time (copies of its event groups overlap its kernels)"}}

    if rank == 0:
        peak, peak_src = measured_peaks()
        sb = stage_bytes(counters)
        names = list(sb)
        stages = {}
        for k, name in enumerate(names):
            gbs = sb[name] / (stage_ms[k] * 1e-3) / 1e9 if stage_ms[k] > 0 else None
            stages[name] = {"ms": round(float(stage_ms[k]), 4), "algorithmic_bytes": int(sb[name]),
                            "GBps": gbs, "frac_of_hbm_peak": (gbs / peak if gbs else None),
                            "frac_of_nominal_8TBps": (gbs / HBM_NOMINAL_GBS if gbs else None)}
        dom = max(names, key=lambda n: stages[n]["ms"])
        # DRAM bytes per step from the committed ncu --set full capture: only for the configuration it was taken on
        cap = committed_traffic(run_config(args, len(evs)))
        traffic = cap.get(dom) if cap else None
        if dom == "K5_construct":
            # K5 = k_construct, ONE launch per step (up and down sweep of every sector task), timed with CUDA events on
            # the launching stream inside the timed region.  Arithmetic intensity ~20 flop/B: bound by FP32 issue.
            sm_count = torch.cuda.get_device_properties(local_rank).multi_processor_count
            derived = fp32_peak_tflops(sm_count, clocks.get("sm_max_mhz"))
            fused, unfused = tracker.tpc_measure_fp32_peak()          # measured here, on this device, after the run
            tfl = k5_flops(counters) / (stage_ms[names.index(dom)] * 1e-3) / 1e12
            roofline = {"bound": "alu", "kernel": "K5 k_construct (1 launch per step: up and down sweep of every sector task)",
                        "achieved": tfl, "peak": fused, "unit": "TFLOP/s", "frac": tfl / fused,
                        "traffic": traffic, "traffic_commit": cap.get("commit") if cap else None,
                        "peak_source": "measured by tpc_measure_fp32_peak on this device: independent FFMA chains, "
                                       "multiply and add counted separately",
                        "peak_unfused_measured": unfused, "frac_of_unfused": tfl / unfused,
                        "peak_derived": derived,
                        "note": "the method's arithmetic is defined without contraction (strict float32 parity), so the "
                                "un-fused multiply + add rate is its ceiling; derived = %d SMs x 128 lanes x 2 x %.0f MHz"
                                % (sm_count, clocks.get("sm_max_mhz") or 1965.0),
                        "hbm": {"achieved": stages[dom]["GBps"], "peak": peak, "unit": "GB/s",
                                "frac": stages[dom]["frac_of_hbm_peak"], "peak_source": peak_src,
                                "frac_of_nominal_8TBps": stages[dom]["frac_of_nominal_8TBps"]}}
        else:
            roofline = {"bound": "hbm", "kernel": dom, "achieved": stages[dom]["GBps"], "peak": peak, "unit": "GB/s",
                        "frac": stages[dom]["frac_of_hbm_peak"], "traffic": traffic,
                        "traffic_commit": cap.get("commit") if cap else None, "peak_source": peak_src,
                        "frac_of_nominal_8TBps": stages[dom]["frac_of_nominal_8TBps"]}
        cpu = None
        if not args.no_cpu_baseline:
            cpu = cpu_baselines(evs, rx, gen)
        value = aggregate_value(len(evs), args.steps, ms, world)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": ("%d x central Pb-Pb-like events per step (BASELINE.json config 5 = 16 x config 4)" % len(evs))
                                   if args.workload == "central" else "%d x %s event(s) per step" % (len(evs), args.workload),
                       "link_step": args.link_step, "refit": bool(args.refit), "merge": bool(args.merge),
                       "seed_dedup": not args.no_seed_dedup,
                       "events_per_step": len(evs), "clusters_per_step": int(n_total),
                       "tracks_per_step": int(n_tracks), "parallelism": "replicas only" if world > 1 else "1 GPU",
                       "l2": "inputs (%.0f MB per step) larger than L2 (126 MB); no flush" % (12 * n_total / 1e6)},
            "clusters_per_s": world * n_total * args.steps / (ms * 1e-3),
            "roofline": roofline, "stages": stages, "cpu_baseline": cpu, "e2e": e2e,
            "gpu_launches": int(launches), "clocks": clocks, "counters": counters,
        }
        if two_groups:
            line["passes"] = two_groups
            line["config"]["event_groups"] = "2 groups of %d events on two streams (tpc_tracker_set_group_events)" % two_groups["events_per_group"]
        print(json.dumps(line))
    trk.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

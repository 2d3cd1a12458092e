#!/usr/bin/env python
"""bench.py -- events/s of unpack + three-threshold clustering on B200 (BASELINE.json metric).

One "step" = one pass of the whole hot path over the
workload of BASELINE.json config 3: 64 independent full-detector events (440 FEDs x 96 x 256
strips, generator of config 1, seeds 1..64) processed over 8 CUDA streams, calibration uploaded
once, per-event output buffers taken from the library's stream-ordered pool.

  value      whole-job events/s with the raw data already resident in HBM (CUDA-event timed)
  e2e        the same metric through sst_unpack_cluster_host_packed: pinned HOST buffers, H2D of the raw
             data and D2H of the clusters inside the timed region
  roofline   algorithmic HBM bytes of a launch / launch duration for sst_event_kernel (the one kernel
             of a launch with plain outputs: its warps also move the staged clusters into order once
             the FED work is used up; --move-mode 1 leaves that to sst_emit_kernel behind it) against
             MEASURED_PEAKS.json
  cpu_baseline  the CPU oracle as it stands, timed on this box's host cores (reported, not a target)

After the timed loop the output blocks of the TIMED launches are read back and every output of
every event is compared with the oracle (bit-exact; barycenter 1e-6 relative); a difference fails
the run.  `--config 1|2|4` times 64 events of that BASELINE.json config instead of config 3.
`--sweep` prints the single-event latencies, events/s against events per call and against the
number of streams, and the OpenMP oracle's N x M table.  `--trace` prints where a warp's time goes,
phase by phase, and the timeline of a launch (sst_config.trace).  `--impl reference` times the oracle alone
on the same config (see the task's contract).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from concurrent.futures import ProcessPoolExecutor

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2101_11489_b200 import synth  # noqa: E402

N_EVENTS = 64          # BASELINE.json config 3
N_STREAMS = 8
THRESHOLDS = (2.0, 3.0, 5.0)
METRIC = "events/s unpack+cluster (full-detector events, 440 FEDs x 96 x 256 strips)"
FALLBACK_HBM_GBS = 6650.0   # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
SPEC_HBM_GBS = 8000.0       # the 8 TB/s BASELINE.md section 2 reads the north_star's 50 % target against (frac_spec)


# --------------------------------------------------------------------------- workload
def event_seeds_for_rank(rank: int, world: int, n_events: int = N_EVENTS):
    """Weak scaling: every rank processes its own n_events events (independent units, no
    collective on the data path).  Rank r gets seeds r*n_events+1 .. (r+1)*n_events."""
    assert 0 <= rank < world
    return list(range(rank * n_events + 1, (rank + 1) * n_events + 1))


def _gen_one(args):
    cfg_id, n_feds, seed = args
    cfg = synth.CONFIGS[cfg_id]
    calib = _gen_one.calib
    ev = synth.make_event(cfg, calib, seed)
    meta = dict(ev.meta)
    per_fed = np.count_nonzero(ev.z.reshape(n_feds, -1), axis=1)
    meta["max_fed_strips"] = int(per_fed.max())
    meta["p99_fed_strips"] = int(np.percentile(per_fed, 99))
    return ev.raw, ev.fed_offsets, meta


def generate_events(cfg_id: int, n_feds: int, seeds, calib, workers: int = 0):
    """Seeded synthetic events (paper_2101_11489_b200/synth.py), generated in a process pool."""
    _gen_one.calib = calib
    workers = workers or min(8, os.cpu_count() or 1, len(seeds))
    jobs = [(cfg_id, n_feds, s) for s in seeds]
    if workers <= 1:
        return [_gen_one(j) for j in jobs]
    import multiprocessing as mp
    with ProcessPoolExecutor(workers, mp_context=mp.get_context("fork")) as ex:
        return list(ex.map(_gen_one, jobs))


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md, MEASURED_PEAKS.json absent)"


def max_over_ranks(x: float, device=None) -> float:
    """Max of a per-rank scalar over all ranks (device time of a multi-GPU step)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


# --------------------------------------------------------------------------- clocks
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.samples = []
        self.proc = None
        self.t0 = self.t1 = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(gpu_index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.samples.append((time.time(), line.strip()))

    def mark_start(self):
        self.t0 = time.time()

    def mark_stop(self):
        self.t1 = time.time()

    def finish(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        time.sleep(0.15)
        self.proc.terminate()
        inside = [s for t, s in self.samples if self.t0 - 0.05 <= t <= self.t1 + 0.15]
        note = "timed region"
        if not inside:
            inside = [s for _, s in self.samples[-3:]]
            note = "nearest samples (timed region shorter than the sampling period)"
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for s in inside:
            f = [x.strip() for x in s.split(",")]
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm), "window": note}


# --------------------------------------------------------------------------- CPU oracle legs
def time_oracle(events, calib, thresholds, budget_s: float, check=None, min_events: int = 4):
    """Sequential oracle (oracle/sst_oracle.c) over the workload's events until budget_s; only the
    oracle calls are timed.  check(i, result) is called (untimed) for every event of the first pass."""
    from oracle import sst_oracle as O
    O.build()
    spent, n = 0.0, 0
    while True:
        raw, fo, _ = events[n % len(events)]
        t0 = time.perf_counter()
        r = O.run(raw, fo, calib.n_feds, calib.gain, calib.noise, calib.bad, calib.chan_module, thresholds)
        spent += time.perf_counter() - t0
        if n < len(events) and check is not None:
            check(n, r)
        n += 1
        if (spent >= budget_s and n >= max(min_events, len(events) if check else 0)) or n >= 4 * len(events):
            break
    return n / spent, n, spent


def compare_with_oracle(g, r, what, dense=True):
    """Every output of one event against the oracle: integers bit-exact, barycenter 1e-6 relative."""
    def same(name, a, b):
        if not np.array_equal(a, b):
            raise SystemExit(f"VERIFICATION FAILED ({what}): {name} differs from the oracle")
    if dense:
        same("strip_adc", g["strip_adc"], r.adc)
    if int(g["n_clusters"]) != int(r.n_clusters):
        raise SystemExit(f"VERIFICATION FAILED ({what}): {g['n_clusters']} clusters, oracle {r.n_clusters}")
    for name in ("cl_module", "cl_first", "cl_width", "cl_charge", "cl_adc_off", "cl_adc"):
        same(name, np.asarray(g[name]).view(getattr(r, name).dtype), getattr(r, name))
    if not np.allclose(g["cl_bary"], r.cl_bary, rtol=1e-6, atol=0):
        raise SystemExit(f"VERIFICATION FAILED ({what}): barycenters differ from the oracle by more than 1e-6 relative")
    same("dev_status", np.asarray(g["status"]).view(np.uint32)[:5], r.status[:5])


OMP_ENV = {"OMP_PROC_BIND": "spread,close", "OMP_PLACES": "cores"}


def omp_leg(args):
    """--omp-leg (a child of time_oracle_omp): the OpenMP build of the oracle in the paper's N x M
    shapes (Table 1) -- N events in flight x M threads per event, over the divisors of
    the core count -- on the first `--events` events of the workload.  Prints {"table", "cores"}."""
    from oracle import sst_oracle as O
    O.build()
    cfg = synth.CONFIGS[args.config]
    thr = cfg.thresholds[0]
    calib = synth.make_calibration(args.n_feds, cfg.bad_frac)
    events = generate_events(args.config, args.n_feds, list(range(1, args.events + 1)), calib)
    cores = os.cpu_count() or 1
    shapes = sorted({(cores // m, m) for m in (1, 2, 4, 8, 16, 32) if m <= cores and cores % m == 0})
    raws = [e[0] for e in events]
    fos = [e[1] for e in events]
    table = []
    per = max(args.cpu_budget / len(shapes), 1.0)
    for n_outer, n_inner in shapes:
        run = lambda: O.events_omp(raws, fos, calib.n_feds, calib.gain, calib.noise, calib.bad, calib.chan_module,
                                   thr, n_outer, n_inner)
        run()   # untimed: the threads of this shape exist and hold their work arrays
        t0 = time.perf_counter()
        done = 0
        while True:
            run()
            done += len(raws)
            dt = time.perf_counter() - t0
            if dt >= per:
                break
        table.append({"N": n_outer, "M": n_inner, "events_per_s": done / dt})
    print(json.dumps({"table": table, "cores": cores}))


def time_oracle_omp(cfg_id: int, n_feds: int, n_events: int, budget_s: float):
    """The OpenMP leg of the CPU baseline, in a process of its own so that the thread binding
    BASELINE.md section 3.2 asks for (OMP_PROC_BIND / OMP_PLACES; `spread,close` is its nested form: the N
    event threads spread over the cores, the M threads of an event close to theirs) is in the
    environment before the OpenMP runtime starts and binds nothing of this process.  The child
    regenerates the same seeded events (seeds 1..n_events).  Returns (table, cores, env)."""
    env = dict(os.environ)
    env.update(OMP_ENV)
    cmd = [sys.executable, os.path.abspath(__file__), "--omp-leg", "--config", str(cfg_id), "--n-feds", str(n_feds),
           "--events", str(n_events), "--cpu-budget", str(budget_s)]
    out = subprocess.run(cmd, env=env, capture_output=True, text=True, timeout=600)
    if out.returncode != 0:
        raise RuntimeError("OpenMP oracle leg failed: " + out.stderr[-2000:])
    doc = json.loads(out.stdout.strip().splitlines()[-1])
    return doc["table"], doc["cores"], dict(OMP_ENV)


CONFIG_NOTES = {1: "generator of config 1 (2% occupancy, seeds 1..N)", 2: "generator of config 2 (6% occupancy, "
                   "wide clusters, seeds 1..N)", 3: "generator of config 1 (2% occupancy)",
                4: "generator of config 4 (15% occupancy, saturation, empty and full channels, seeds 1..N)"}


def workload_config(cfg_id, n_feds, n_events, thresholds):
    return {"workload": f"BASELINE.json config {cfg_id}: {n_events} events x {n_feds} FEDs x 96 ch x 256 strips, "
                        f"{CONFIG_NOTES[cfg_id]}, thresholds {tuple(thresholds)}, {N_STREAMS} CUDA streams, "
                        "one sst_unpack_cluster_batch call per step",
            "config_id": cfg_id, "n_events": n_events, "n_feds": n_feds, "streams": N_STREAMS,
            "l2": "working set per step (raw buffers + 86.5 MB calibration + one distinct ~20 MB output block per "
                  "event, > 1.3 GB) exceeds the 126 MB L2; no explicit flush"}


def run_reference(args):
    """--impl reference: the CPU oracle alone, same config/metric; rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n_feds = args.n_feds
    per_step = min(args.ref_events, args.events)
    cfg = synth.CONFIGS[args.config]
    thr = cfg.thresholds[0]
    calib = synth.make_calibration(n_feds, cfg.bad_frac)
    events = generate_events(args.config, n_feds, list(range(1, per_step + 1)), calib)
    from oracle import sst_oracle as O
    O.build()

    def step():
        for raw, fo, _ in events:
            O.run(raw, fo, n_feds, calib.gain, calib.noise, calib.bad, calib.chan_module, thr)

    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = time.perf_counter() - t0
    value = per_step * args.steps / dt
    sample = (f"each step = the first {per_step} of the workload's {args.events} events (seeds 1..{per_step}), "
              "sequential oracle, 1 thread")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": "events/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u8/f32/f64", "data": "synthetic",
        "config": workload_config(args.config, n_feds, args.events, thr),
        "cpu_baseline": {"value": value, "unit": "events/s", "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "events/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# --------------------------------------------------------------------------- GPU arm
def git_blob_sha1(path: str) -> str:
    """What `git hash-object` prints for the file."""
    import hashlib
    data = open(path, "rb").read()
    return hashlib.sha1(b"blob %d\0" % len(data) + data).hexdigest()


def ncu_traffic(cfg_id: int):
    """Measured DRAM bytes per step (read + write of every kernel of a step) from the committed ncu
    launch list summary profiles/traffic.csv (rows: workload, kernel, read bytes, write bytes), or None;
    and whether the capture is STALE: the file names the git blob of the sst.cu it was taken from
    (a `# sst.cu blob: <sha1>` line), which is compared with the source this run was built from."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(p):
        return None, None
    tot, found, blob = 0.0, False, None
    for line in open(p):
        if line.startswith("# sst.cu blob:"):
            blob = line.split(":", 1)[1].strip()
        f = [x.strip() for x in line.split(",")]
        if len(f) >= 4 and f[0] == f"config{cfg_id}":
            try:
                tot += float(f[2]) + float(f[3])
                found = True
            except ValueError:
                pass
    stale = blob != git_blob_sha1(os.path.join(ROOT, "paper_2101_11489_b200", "csrc", "sst.cu"))
    return (tot if found else None), stale


MOVE_MODE = 0  # sst_config.move_mode of the detectors the bench makes (--move-mode)


def make_detector(harness, n_feds, calib, events, device=0, hint=True, move_mode=None):
    max_raw = (max(int(e[0].size) for e in events) + 4095) // 4096 * 4096
    # sst_config.fed_strips_hint (present strips of a large FED) sizes the shared-memory working
    # set: the 99th percentile of the events' FEDs, as a site would take it from its occupancy (the
    # few larger FEDs are processed through global scratch)
    strips_hint = int(1.02 * np.percentile([int(e[2]["p99_fed_strips"]) for e in events], 90)) + 16 if hint else 0
    det = harness.Detector(n_feds, calib.gain, calib.noise, calib.bad, calib.chan_module, device=device,
                           max_raw_bytes=max_raw, max_events_in_flight=N_STREAMS, fed_strips_hint=strips_hint,
                           move_mode=MOVE_MODE if move_mode is None else move_mode)
    return det, max_raw


def run_sweep(args):
    """Single-event device latency of every single-event config; config 3 throughput against the
    events per call and against the number of streams (Table 1 sweeps the events in
    flight); the OpenMP oracle's N x M table (Table 1)."""
    import torch
    from paper_2101_11489_b200 import binding as B, harness
    torch.cuda.set_device(0)
    out = {"single_event": [], "events_per_call": [], "streams": [], "omp_oracle": None}
    for cid in (0, 1, 2, 4):
        cfg, cal, evs = synth.make_config(cid)
        ev = evs[0]
        nf = cal.n_feds
        mrb = (int(ev.raw.size) + 4095) // 4096 * 4096
        hint = int(1.05 * int(np.count_nonzero(ev.z.reshape(nf, -1), axis=1).max())) + 16
        det = harness.Detector(nf, cal.gain, cal.noise, cal.bad, cal.chan_module, max_raw_bytes=mrb, fed_strips_hint=hint)
        d_raw, d_fo = det.upload_raw(ev.raw, ev.fed_offsets)
        outs = det.alloc_outputs(mrb // 3 + 1, mrb, dense=True)
        st = torch.cuda.Stream()
        for thr in cfg.thresholds:
            n_rep = 30
            evs_t = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_rep)]
            for rep in range(2):
                with torch.cuda.stream(st):
                    torch.cuda._sleep(2_000_000)
                for a, b in evs_t:
                    a.record(st)
                    det.run(d_raw, d_fo, thr, outs, stream=st)
                    b.record(st)
                torch.cuda.synchronize()
            us = float(np.median([a.elapsed_time(b) for a, b in evs_t])) * 1e3
            # the same call captured in a CUDA graph and replayed
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=st):
                det.run(d_raw, d_fo, thr, outs, stream=st)
            for rep in range(2):
                with torch.cuda.stream(st):
                    torch.cuda._sleep(2_000_000)
                    for a, b in evs_t:
                        a.record(st)
                        graph.replay()
                        b.record(st)
                torch.cuda.synchronize()
            us_graph = float(np.median([a.elapsed_time(b) for a, b in evs_t])) * 1e3
            del graph
            g = outs.numpy()
            out["single_event"].append({"config": cid, "n_feds": nf, "thresholds": list(thr), "latency_us": us,
                                        "latency_us_graph_replay": us_graph,
                                        "present_strips": int(ev.meta["present"]), "clusters": int(g["n_clusters"]),
                                        "raw_bytes": int(ev.raw.size), "info": det.info()})
        del outs
        det.close()
    n_feds = args.n_feds
    thr = THRESHOLDS
    calib = synth.make_calibration(n_feds, synth.CONFIGS[3].bad_frac)
    events = generate_events(3, n_feds, range(1, N_EVENTS + 1), calib)
    det, mrb = make_detector(harness, n_feds, calib, events)
    d_in = [det.upload_raw(e[0], e[1]) for e in events]
    outs = [det.alloc_outputs(mrb // 3 + 1, mrb, dense=True) for _ in events]

    def rate(n, n_streams):
        streams = [torch.cuda.Stream() for _ in range(n_streams)]
        batch = B.Batch([d[0] for d in d_in[:n]], [d[1] for d in d_in[:n]], thr, [o.out for o in outs[:n]],
                        [s.cuda_stream for s in streams])
        steps = max(20, 640 // n)
        for _ in range(5):
            B.sst_unpack_cluster_batch(det.ctx, batch)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(steps):
            B.sst_unpack_cluster_batch(det.ctx, batch)
        torch.cuda.synchronize()
        return n * steps / (time.perf_counter() - t0)

    for n in (1, 2, 4, 8, 16, 32, 64):
        r = rate(n, min(n, N_STREAMS))
        out["events_per_call"].append({"events": n, "streams": min(n, N_STREAMS), "events_per_s": r, "us_per_event": 1e6 / r})
    for ns in (1, 2, 4, 8, 16):
        r = rate(N_EVENTS, ns)
        out["streams"].append({"events": N_EVENTS, "streams": ns, "events_per_s": r})
    det.close()
    table, cores, omp_env = time_oracle_omp(3, n_feds, 16, 24.0)
    out["omp_oracle"] = {"cores": cores, "events_per_pass": 16, "table": table, "env": omp_env}
    print(json.dumps({"sweep": out}))


TRACE_PHASES = ("ticket + prologue", "payload staging (TMA wait)", "length chain", "pass 1 + scan", "pass 2", "expansion",
                "dense SoA", "sweep", "members and heads", "counts + cluster list", "staging of the clusters", "publish")


def run_trace(args):
    """Where a warp's time goes, FED phase by FED phase, and the timeline of one launch: a context
    created with sst_config.trace = 1 (the traced instantiations of sst_event_kernel), one launch of
    n events of the chosen config for n = 1, 8, 64; sst_trace_read after each."""
    import torch
    from paper_2101_11489_b200 import binding as B, harness
    torch.cuda.set_device(0)
    n_feds = args.n_feds
    calib = synth.make_calibration(n_feds, synth.CONFIGS[args.config].bad_frac)
    events = generate_events(args.config, n_feds, range(1, N_EVENTS + 1), calib)
    mhz = float(subprocess.check_output(["nvidia-smi", "--query-gpu=clocks.max.sm", "--format=csv,noheader,nounits", "-i", "0"],
                                        text=True).split()[0])
    max_raw = (max(int(e[0].size) for e in events) + 4095) // 4096 * 4096
    hint = int(1.02 * np.percentile([int(e[2]["p99_fed_strips"]) for e in events], 90)) + 16
    det = harness.Detector(n_feds, calib.gain, calib.noise, calib.bad, calib.chan_module, max_raw_bytes=max_raw,
                           max_events_in_flight=N_STREAMS, fed_strips_hint=hint, move_mode=MOVE_MODE, trace=1)
    st = torch.cuda.Stream()
    d_in = [det.upload_raw(e[0], e[1]) for e in events]
    outs = [harness.PooledOutputs(det, max_raw // 3 + 1, max_raw, st.cuda_stream, dense=True) for _ in events]
    out = {"config": args.config, "n_feds": n_feds, "move_mode": MOVE_MODE, "sm_max_mhz": mhz, "info": det.info(), "launches": []}
    for n in (1, 8, 64):
        batch = B.Batch([d[0] for d in d_in[:n]], [d[1] for d in d_in[:n]], THRESHOLDS, [o.out for o in outs[:n]], [st.cuda_stream])
        for _ in range(3):
            B.sst_unpack_cluster_batch(det.ctx, batch)
        B.sst_trace_read(det.ctx, st.cuda_stream)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(st)
        B.sst_unpack_cluster_batch(det.ctx, batch)
        e1.record(st)
        t = B.sst_trace_read(det.ctx, st.cuda_stream)
        feds = max(t[0], 1)
        phases = {name: t[1 + i] / feds / mhz for i, name in enumerate(TRACE_PHASES)}
        out["launches"].append({
            "events": n, "feds": t[0], "launch_us_cuda_events": 1e3 * e0.elapsed_time(e1),
            "us_per_fed_by_phase": phases, "us_per_fed": sum(phases.values()),
            "feds_moved_in_kernel": t[13], "us_per_moved_fed": t[14] / max(t[13], 1) / mhz,
            "timeline_us": {"first_warp_out_of_fed_tickets": (t[21] - t[20]) / 1e3, "last_warp_out_of_fed_tickets": (t[22] - t[20]) / 1e3,
                            "kernel_end": (t[23] - t[20]) / 1e3}})
    det.close()
    print(json.dumps({"trace": out}))


def respawn_under_torchrun(args):
    """`python bench.py --gpus N` with N > 1 and no launcher: start N ranks (one per GPU)."""
    import socket
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
    os.execv(sys.executable, cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4],
                    help="BASELINE.json config the 64 events are generated from (3 = the headline workload)")
    ap.add_argument("--n-feds", type=int, default=440)
    ap.add_argument("--events", type=int, default=N_EVENTS)
    ap.add_argument("--ref-events", type=int, default=8, help="events per step of --impl reference")
    ap.add_argument("--cpu-budget", type=float, default=12.0, help="seconds of oracle timing (rank 0, N=1)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg (and with it the verification)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--omp-leg", action="store_true", help=argparse.SUPPRESS)
    ap.add_argument("--trace", action="store_true",
                    help="instead of the bench line: per-phase time of a FED and the timeline of a launch of 1, 8 and 64 "
                         "events, from a context with sst_config.trace = 1")
    ap.add_argument("--move-mode", type=int, default=0, choices=[0, 1],
                    help="sst_config.move_mode: 0 = the ordered move inside sst_event_kernel, 1 = sst_emit_kernel behind it")
    ap.add_argument("--sweep", action="store_true",
                    help="instead of the bench line: single-event latency of configs 0, 1, 2, 4, events/s against the "
                         "events per call and the number of streams, and the OpenMP oracle's N x M table")
    args = ap.parse_args()
    global MOVE_MODE
    MOVE_MODE = args.move_mode
    if args.warmup < 3 and args.impl == "b200":
        args.warmup = 3
    if args.sweep:
        return run_sweep(args)
    if args.trace:
        return run_trace(args)
    if args.omp_leg:
        return omp_leg(args)
    world_env = os.environ.get("WORLD_SIZE")
    if world_env is None and args.gpus > 1:
        return respawn_under_torchrun(args)
    if world_env is not None and int(world_env) != args.gpus:
        print(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world_env}", file=sys.stderr)
        sys.exit(2)
    if args.impl == "reference":
        run_reference(args)
        return

    import torch
    from paper_2101_11489_b200 import binding as B
    from paper_2101_11489_b200 import build as sst_build
    from paper_2101_11489_b200 import harness

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    torch.cuda.set_device(local_rank)
    if rank == 0:
        sst_build.build()
    if world > 1:
        dist.barrier()

    n_feds, n_events = args.n_feds, args.events
    cfg = synth.CONFIGS[args.config]
    thr = cfg.thresholds[0]
    calib = synth.make_calibration(n_feds, cfg.bad_frac)
    events = generate_events(args.config, n_feds, event_seeds_for_rank(rank, world, n_events), calib)
    det, max_raw = make_detector(harness, n_feds, calib, events, device=local_rank)
    info = det.info()
    dev = det.device
    n_strips = n_feds * B.FED_STRIPS

    # resident inputs; one pooled output block per event (64 distinct blocks, ~1.3 GB)
    d_in = [det.upload_raw(e[0], e[1]) for e in events]
    cap_cl, cap_adc = max_raw // 3 + 1, max_raw
    streams = [torch.cuda.Stream(device=dev) for _ in range(N_STREAMS)]
    main_stream = torch.cuda.current_stream(dev)
    outs = [harness.PooledOutputs(det, cap_cl, cap_adc, streams[i % N_STREAMS].cuda_stream, dense=True) for i in range(n_events)]
    batch = B.Batch([d[0] for d in d_in], [d[1] for d in d_in], thr, [o.out for o in outs], [st.cuda_stream for st in streams])

    def step():
        """One pass over the workload: the events of each stream share launches, one C call."""
        B.sst_unpack_cluster_batch(det.ctx, batch)

    def fork_join_begin(ev):
        ev.record(main_stream)
        for s in streams:
            s.wait_event(ev)

    def fork_join_end(ev):
        for s in streams:
            e = torch.cuda.Event()
            e.record(s)
            main_stream.wait_event(e)
        ev.record(main_stream)

    def timed(n_steps, warm):
        for _ in range(warm):
            step()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        fork_join_begin(e0)
        for _ in range(n_steps):
            step()
        fork_join_end(e1)
        torch.cuda.synchronize()
        t_host = time.perf_counter() - t0
        if world > 1:
            dist.barrier()
        return max_over_ranks(e0.elapsed_time(e1), dev), t_host

    # ---- timed: device-resident inputs
    sampler = ClockSampler(local_rank)
    sampler.mark_start()
    ms_total, t_host = timed(args.steps, args.warmup)
    sampler.mark_stop()
    clocks = sampler.finish()
    ms_step = ms_total / args.steps
    value = world * n_events * args.steps / (ms_total * 1e-3)

    # ---- the outputs of the timed launches: counts and algorithmic bytes per event
    mod_first = np.zeros(int(calib.chan_module.max()) + 1, np.int64)
    cm = calib.chan_module.astype(np.int64)
    firsts = np.flatnonzero(np.concatenate([[True], cm[1:] != cm[:-1]]))
    mod_first[cm[firsts]] = firsts * 256
    results, per_event = [], []
    for i in range(n_events):
        g = outs[i].numpy(streams[i % N_STREAMS].cuda_stream)
        st = g["status"]
        assert st[B.ST_FLAGS] == 0, f"event {i}: dev_status flags {st[B.ST_FLAGS]}"
        present = g["strip_adc"] != 0
        s_noise = int(present.reshape(-1, 8).any(axis=1).sum())          # 32-B sectors of a float array
        lcl = mod_first[g["cl_module"].astype(np.int64)] + g["cl_first"].astype(np.int64)
        mark = np.zeros(n_strips + 1, np.int32)
        np.add.at(mark, lcl, 1)
        np.add.at(mark, lcl + g["cl_width"].astype(np.int64), -1)
        in_cl = np.cumsum(mark[:-1]) > 0
        s_gain = int(in_cl.reshape(-1, 8).any(axis=1).sum())
        n_cl, n_adc = int(st[B.ST_N_CLUSTERS]), int(st[B.ST_N_ADC])
        b_alg = int(events[i][0].size) + n_strips + 32 * s_noise + 32 * s_gain + 20 * n_cl + n_adc
        per_event.append({"n_clusters": n_cl, "n_adc": n_adc, "n_seeds": int(st[B.ST_N_SEEDS]),
                          "present": int(present.sum()), "b_alg": b_alg})
        results.append(g if not args.no_cpu and rank == 0 and world == 1 else None)
    b_alg_step = sum(p["b_alg"] for p in per_event)
    clusters_step = sum(p["n_clusters"] for p in per_event)
    present_step = sum(p["present"] for p in per_event)

    # ---- roofline of sst_event_kernel: one launch of each kernel per step (up to 64 events per launch)
    peak, peak_src = measured_peak()
    epl = int(info.get("events_per_launch", 1))
    n_groups = min(N_STREAMS, n_events, max(1, -(-n_events // epl)))
    launches_step = sum(-(-sum(1 for e in range(n_events) if (e % N_STREAMS) % n_groups == g) // epl)
                        for g in range(n_groups))
    launches = launches_step * args.steps
    kernels_per_launch = int(info.get("kernels_per_event", 1))
    dur_us = 1e3 * ms_total / launches
    achieved = (b_alg_step / launches_step) / (dur_us * 1e-6) / 1e9
    traffic, traffic_stale = ncu_traffic(args.config)

    # ---- two batches in flight: consecutive steps alternate between two halves of the stream set (and
    # two sets of output blocks), so the ordered move of one step overlaps the event kernel of the next
    pipelined, results_b = None, None
    if world == 1:
        half = N_STREAMS // 2
        sets = []
        for h in range(2):
            ss = streams[h * half:(h + 1) * half]
            oo = outs if h == 0 else [harness.PooledOutputs(det, cap_cl, cap_adc, ss[i % half].cuda_stream, dense=True)
                                      for i in range(n_events)]
            sets.append((ss, oo, B.Batch([d[0] for d in d_in], [d[1] for d in d_in], thr, [o.out for o in oo],
                                         [st.cuda_stream for st in ss])))
        torch.cuda.synchronize()
        for i in range(6):
            B.sst_unpack_cluster_batch(det.ctx, sets[i % 2][2])
        torch.cuda.synchronize()
        n_p = max(2, args.steps // 2 * 2)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        fork_join_begin(e0)
        for i in range(n_p):
            B.sst_unpack_cluster_batch(det.ctx, sets[i % 2][2])
        fork_join_end(e1)
        torch.cuda.synchronize()
        pipelined = {"value": n_events * n_p / (e0.elapsed_time(e1) * 1e-3), "unit": "events/s", "steps": n_p,
                     "note": "the same step issued alternately on streams 0-3 and 4-7 with two sets of output blocks: "
                             "two batches in flight, the move of one overlapping the event kernel of the next (a caller's "
                             "choice; `value` is one batch at a time)"}
        if not args.no_cpu and rank == 0:
            results_b = [sets[1][1][i].numpy(sets[1][0][i % half].cuda_stream) for i in range(n_events)]
        for i, o in enumerate(sets[1][1]):
            o.free(sets[1][0][i % half].cuda_stream)
        torch.cuda.synchronize()

    # ---- the same with the default shared-memory sizing (fed_strips_hint = 0)
    default_hint = None
    if world == 1:
        det0, _ = make_detector(harness, n_feds, calib, events, device=local_rank, hint=False)
        main_ctx, det.ctx = det.ctx, det0.ctx
        ms0, _ = timed(max(10, args.steps // 10), 3)
        det.ctx = main_ctx
        default_hint = {"value": n_events * max(10, args.steps // 10) / (ms0 * 1e-3), "unit": "events/s",
                        "info": det0.info(), "note": "fed_strips_hint = 0: slot sized from max_raw_bytes / n_feds"}
        det0.close()

    # ---- the same with the other way of moving the staged clusters (sst_config.move_mode)
    other_move = None
    if world == 1:
        det1, _ = make_detector(harness, n_feds, calib, events, device=local_rank, move_mode=1 - MOVE_MODE)
        main_ctx, det.ctx = det.ctx, det1.ctx
        ms1, _ = timed(max(10, args.steps // 4), 3)
        det.ctx = main_ctx
        other_move = {"value": n_events * max(10, args.steps // 4) / (ms1 * 1e-3), "unit": "events/s", "move_mode": 1 - MOVE_MODE,
                      "note": "move_mode 0 = staged clusters moved inside sst_event_kernel (one launch per batch), "
                              "1 = by sst_emit_kernel behind it (two launches)"}
        det1.close()

    # ---- single-event latency on one stream (launches queued behind a sleep kernel)
    serial = None
    if world == 1:
        s0 = streams[0]
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_events)]
        for rep in range(2):
            with torch.cuda.stream(s0):
                torch.cuda._sleep(4_000_000)        # keep the stream busy while the host enqueues
            for i in range(n_events):
                evs[i][0].record(s0)
                B.sst_unpack_cluster(det.ctx, d_in[i][0], d_in[i][1], thr, outs[i].out, s0.cuda_stream)
                evs[i][1].record(s0)
            torch.cuda.synchronize()
        d = np.array([a.elapsed_time(b) for a, b in evs]) * 1e3
        serial = {"launch_us_median": float(np.median(d)), "launch_us_min": float(d.min()),
                  "note": "one event per call on one stream, CUDA events around each call"}

    # ---- e2e: HOST buffers through sst_unpack_cluster_host_packed
    e2e, e2e_views = None, None
    if not args.no_e2e:
        pin = [(torch.from_numpy(e[0]).pin_memory(), torch.from_numpy(e[1].view(np.int32)).pin_memory()) for e in events]
        # one pinned, packed result block per event; one C call per step: the 64 events are cut into
        # chunks whose uploads, launches and (single, size-guessed) downloads overlap on the 8 streams
        host_blocks = [torch.zeros(64 + 20 * cap_cl + cap_adc, dtype=torch.uint8).pin_memory() for _ in range(n_events)]
        e2e_steps = max(1, min(args.steps, 20))
        pbatch = B.PackedBatch([p[0] for p in pin], [int(e[0].size) for e in events], [p[1] for p in pin], thr,
                               cap_cl, cap_adc, host_blocks, [st.cuda_stream for st in streams])
        counts_view = [blk.numpy()[32:36].view(np.uint32) for blk in host_blocks]

        def e2e_step():
            B.sst_unpack_cluster_host_packed(det.ctx, pbatch)
            return sum(int(c[0]) for c in counts_view)

        for _ in range(3):
            e2e_step()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        t0 = time.perf_counter()
        n_cl_seen = 0
        for _ in range(e2e_steps):
            n_cl_seen += e2e_step()
        torch.cuda.synchronize()
        dt = max_over_ranks(time.perf_counter() - t0, dev)
        assert n_cl_seen == clusters_step * e2e_steps, "e2e cluster counts differ from the device-resident pass"
        h2d = sum(int(e[0].size) + 4 * (n_feds + 1) for e in events)
        d2h = sum(64 + 20 * p["n_clusters"] + p["n_adc"] for p in per_event)
        e2e = {"value": world * n_events * e2e_steps / dt, "unit": "events/s", "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "steps": e2e_steps, "host_threads": 1,
               "api": "sst_unpack_cluster_host_packed (pinned host raw in; status, cluster records and ADCs out as one "
                      "packed block per event; chunks of 4 events pipelined over the 8 streams)"}
        e2e_views = [pbatch.view(i) for i in range(n_events)]
        # what the link alone allows: plain copies of the same byte counts in both directions at once
        d_up = [torch.empty(int(e[0].size), dtype=torch.uint8, device=dev) for e in events]
        nb = [64 + 20 * p["n_clusters"] + p["n_adc"] for p in per_event]
        d_dn = [torch.empty(n, dtype=torch.uint8, device=dev) for n in nb]
        h_dn = [torch.empty(max(nb), dtype=torch.uint8).pin_memory() for _ in range(N_STREAMS)]
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(5):
            for i in range(n_events):
                with torch.cuda.stream(streams[i % N_STREAMS]):
                    d_up[i].copy_(pin[i][0], non_blocking=True)
                    h_dn[i % N_STREAMS][:nb[i]].copy_(d_dn[i], non_blocking=True)
        torch.cuda.synchronize()
        e2e["copy_floor"] = {"value": n_events * 5 / (time.perf_counter() - t0), "unit": "events/s",
                             "note": "the step's H2D and D2H bytes as plain pinned cudaMemcpyAsync copies over the 8 "
                                     "streams, no kernels: the PCIe ceiling of this box for this result volume"}
        del d_up, d_dn, h_dn

    # ---- SURVEY.md section 8(d) mode (ii), BASELINE.json config 3 as worded: pinned H2D of the raw data in the
    # loop, overlapping the kernels of other events; results stay on the device
    h2d_overlap = None
    if not args.no_e2e and world == 1:
        chunk = 8
        def h2d_step():
            held = []
            for c0 in range(0, n_events, chunk):
                st = streams[(c0 // chunk) % N_STREAMS].cuda_stream
                ptrs = [B.sst_event_upload(det.ctx, pin[i][0], int(events[i][0].size), pin[i][1], st)
                        for i in range(c0, min(c0 + chunk, n_events))]
                bb = B.Batch([q[0] for q in ptrs], [q[1] for q in ptrs], thr,
                             [outs[i].out for i in range(c0, min(c0 + chunk, n_events))], [st])
                B.sst_unpack_cluster_batch(det.ctx, bb)
                for q in ptrs:
                    B.sst_event_free(det.ctx, q[0], st)
                    B.sst_event_free(det.ctx, q[1], st)
                held.append(bb)
            return held
        for _ in range(3):
            h2d_step()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        n_h = max(1, min(args.steps, 20))
        for _ in range(n_h):
            h2d_step()
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        h2d_overlap = {"value": n_events * n_h / dt, "unit": "events/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": 0,
                       "note": "per step 8 chunks of 8 events: sst_event_upload (pooled device buffers, pinned H2D) and one "
                               "sst_unpack_cluster_batch per chunk on its own stream, so uploads overlap the kernels of the "
                               "chunks before; outputs stay on the device (BASELINE.json config 3 as worded, PAPER.md:41)"}

    # ---- CPU baseline (rank 0, N = 1 only) and the verification of the timed outputs against it
    cpu = cpu_omp = verified = None
    if rank == 0 and world == 1 and not args.no_cpu:
        def check(i, r):
            compare_with_oracle(results[i], r, f"timed batch launch, event {i}")
            results[i] = None
            if results_b is not None:
                compare_with_oracle(results_b[i], r, f"pipelined batches, event {i}")
                results_b[i] = None
            if e2e_views is not None:
                compare_with_oracle(e2e_views[i], r, f"e2e, event {i}", dense=False)

        rate, n_done, dt = time_oracle(events, calib, thr, args.cpu_budget, check=check)
        verified = f"{n_events}/{n_events} events of the timed launches, all outputs (dense SoA, clusters, ADCs, status)" + \
                   ("; the second output set of the pipelined leg likewise" if results_b is not None else "") + \
                   ("; e2e blocks: clusters, ADCs, status" if e2e_views is not None else "")
        cpu = {"value": rate, "unit": "events/s", "cores": 1, "kind": "oracle",
               "sample": f"{n_done} events of the workload (seeds 1..{min(n_done, n_events)}), {dt:.1f} s of oracle time, "
                         "oracle/sst_oracle.c -O2 sequential"}
        table, cores, omp_env = time_oracle_omp(args.config, n_feds, min(16, n_events), max(args.cpu_budget / 2, 4.0))
        best = max(table, key=lambda t: t["events_per_s"])
        cpu_omp = {"value": best["events_per_s"], "unit": "events/s", "cores": cores, "kind": "oracle (OpenMP build)",
                   "shape_NxM": f"{best['N']}x{best['M']}", "table": table, "env": omp_env,
                   "sample": f"{min(16, n_events)} events of the workload per pass (seeds 1..{min(16, n_events)}), N events in "
                             "flight x M threads per event, in a child process with that environment; one untimed pass per shape"}

    if rank == 0:
        dram = None
        if traffic is not None:
            dram_gbs = traffic / (ms_step * 1e-3) / 1e9
            dram = {"bytes_per_step": traffic, "achieved": dram_gbs, "frac": dram_gbs / peak, "frac_spec": dram_gbs / SPEC_HBM_GBS,
                    "traffic_stale": traffic_stale,
                    "source": "profiles/traffic.csv (ncu dram__bytes_read.sum + dram__bytes_write.sum of the kernels of a step, "
                              "one step) over this run's step time"}
        line = {
            "metric": METRIC, "value": value, "unit": "events/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "u8/f32/f64", "data": "synthetic",
            "config": workload_config(args.config, n_feds, n_events, thr),
            "verified": verified,
            "strips_per_s": value * n_strips, "present_strips_per_s": value * present_step / n_events,
            "clusters_per_s": value * clusters_step / n_events,
            "host_wall_ms_per_step": 1e3 * t_host / args.steps,
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "frac_spec": achieved / SPEC_HBM_GBS, "spec_peak": SPEC_HBM_GBS,
                         "traffic": traffic, "traffic_stale": traffic_stale, "peak_source": peak_src,
                         "kernel": "sst_event_kernel", "algorithmic_bytes_per_launch": b_alg_step / launches_step,
                         "events_per_launch": n_events / launches_step,
                         "launch_us": dur_us,
                         "dram": dram,
                         "limiter": "not HBM: a warp works through its FED as one long chain of dependent steps, eight "
                                    "warps per scheduler hide ~67 % of it (issue slots 67 % busy, DRAM 31 %, 11.9 cycles per issued "
                                    "instruction; profiles/r03_final.md); the calibration term of the algorithmic bytes is served by L2",
                         "how": "achieved = algorithmic bytes per launch / launch duration, B_alg = raw + N dense + 32 B x "
                                "noise sectors of present strips + 32 B x gain sectors of accepted-cluster strips + 20 B x "
                                "clusters + cluster ADC bytes; launch duration = CUDA-event span of the timed region / "
                                "sst_event_kernel launches (move_mode 0: the ordered move of the staged clusters is part of "
                                "that kernel; move_mode 1: sst_emit_kernel runs behind it and its time is charged to it); "
                                "`dram` is the same span against the DRAM bytes ncu measured",
                         "serial": serial},
            "pipelined": pipelined,
            "default_hint": default_hint,
            "other_move": other_move, "e2e": e2e, "h2d_overlap": h2d_overlap, "gpu_launches": launches * kernels_per_launch, "clocks": clocks,
            "cpu_baseline": cpu, "cpu_baseline_omp": cpu_omp,
            "kernel_info": info,
            "paper_context": "PAPER.md Table 1: best 649 events/s on one P100, 560 events/s on 28 Broadwell cores "
                             "(TTBar PU70, ~800k strips/event; other hardware and data, context only)",
        }
        print(json.dumps(line))
    for i, o in enumerate(outs):
        o.free(streams[i % N_STREAMS].cuda_stream)
    torch.cuda.synchronize()
    det.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

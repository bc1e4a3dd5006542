#!/usr/bin/env python
"""bench.py — VELO-tracking throughput on B200 (BASELINE.json:metric): events/s and hits/s on the
mu=5 workload, with the fraction of the HBM roofline, the oracle timed beside it, and the
end-to-end number through the host-buffer C-ABI call.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl velo|reference] [--config 2]

A "step" is one pass of the whole hot path (S0 ... S8 of DESIGN.md §1) over one synthetic
workload: BASELINE.json:configs[2], 100 000 events at mu=5 in 4 streamed batches of 25 000.
Inputs are resident in HBM when the timed region starts (2.5 GB, far larger than the 126 MB L2,
so nothing is cache-warm between steps). N > 1: one process per GPU (torchrun), every rank
reconstructs its own 100 000 events (weak scaling, no data-path collective: events are
independent); NCCL is used only for the barrier and the max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

# ncu --set full counters of one 25 000-event launch of every kernel of the path (configs[2] batch size),
# written from the capture summarised in profiles/r02j_pipeline.md; read by name, never pasted here
STAGE_COUNTERS_CSV = os.path.join(ROOT, "profiles", "r02j_stage_counters.csv")
STAGE_COUNTERS_EVENTS = 25_000
# stage k runs between stage events k and k+1 of velo_launch_options_t (include/velo.h)
STAGES = [("sort", ["velo_sort_kernel", "velo_order_kernel"]),
          ("track", ["velo_track_kernel", "velo_event_slab_kernel"]),
          ("fit", ["velo_fit_kernel"]),
          ("offsets", ["velo_offsets_kernel"]),
          ("write", ["velo_write_kernel"])]

METRIC = "velo_tracking_events_per_s"
UNIT = "events/s"
N_MODULES = 26


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="velo", choices=["velo", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json:configs index (default 2)")
    ap.add_argument("--events", type=int, default=None, help="override the number of events (debugging)")
    ap.add_argument("--ctas-per-sm", type=int, default=0, help="slab-kernel launch option (0 = library default)")
    ap.add_argument("--path", type=int, default=0, help="0 = three-stage pipeline + slab kernel for deferred events, 1 = slab only")
    ap.add_argument("--no-other-workloads", action="store_true", help="skip the short configs[3] and configs[4] legs")
    ap.add_argument("--track-group", type=int, default=0, help="threads per event of the module-loop kernel (0 = default)")
    ap.add_argument("--track-teams", type=int, default=0)
    ap.add_argument("--fit-teams", type=int, default=0)
    ap.add_argument("--sort-teams", type=int, default=0)
    ap.add_argument("--pool-units", type=int, default=0)
    ap.add_argument("--timeline", action="store_true",
                    help="instrumented build: print when each pipeline stage of each batch ran, then exit")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-split", default="growing", choices=["growing", "equal"],
                    help="batch sizes of the end-to-end call: 10/20/30/40 %% of the events (default) or four equal batches")
    ap.add_argument("--e2e-fractions", default="0.10,0.20,0.30,0.40",
                    help="the growing split (measured: 6/14/30/50 %% 39.4 ms, 10/20/30/40 %% 39.7 ms, six or eight growing "
                         "batches 42-50 ms: every batch costs two host synchronisations)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


def workload_name(cfg_index: int, n_events: int, n_batches: int) -> str:
    base = {0: "configs[0] mu=5 closed VELO", 1: "configs[1] mu=5 closed VELO", 2: "configs[2] mu=5 closed VELO",
            3: "configs[3] mu=5 open VELO (49 mm)", 4: "configs[4] ion-like"}[cfg_index]
    return f"{base}: {n_events} events in {n_batches} streamed batch(es), seed 1"


def algorithmic_bytes(n_events: int, n_hits: int, n_tracks: int, n_track_hits: int) -> int:
    """DESIGN.md §6 / SURVEY.md §8(d): what the method itself must move per batch.
    in: x, y, z f32 + module u8 per hit, one offset per event;
    out: track_hits u32, track_hit_offsets u32 + 13 state words per track, one offset per event."""
    return 13 * n_hits + 4 * (n_events + 1) + 4 * n_track_hits + (4 + 52) * n_tracks + 4 * (n_events + 1)


# ---- clocks during the timed region (B200_PROFILING.md recipe) -----------------------------------
_CLOCK_QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
                "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
                "clocks_event_reasons.sw_power_cap")


class ClockSampler:
    def __init__(self, gpu_index: int):
        self.idx, self.proc = gpu_index, None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={_CLOCK_QUERY}", "--format=csv,noheader,nounits", "-lms", "50",
                 "-i", str(self.idx)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        lines = []
        if self.proc is not None:
            time.sleep(0.06)
            self.proc.terminate()
            try:
                out, _ = self.proc.communicate(timeout=5)
                lines = [l for l in out.splitlines() if l.strip()]
            except Exception:
                self.proc.kill()
        if not lines:
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={_CLOCK_QUERY}", "--format=csv,noheader,nounits",
                                      "-i", str(self.idx)], capture_output=True, text=True, timeout=10).stdout
                lines = [l for l in out.splitlines() if l.strip()]
            except Exception:
                lines = []
        sm, smax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for l in lines:
            f = [t.strip() for t in l.split(",")]
            try:
                sm.append(float(f[0])); smax.append(float(f[1]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def stage_counters() -> dict:
    """kernel name -> counters of one 25 000-event launch (profiles/r02j_stage_counters.csv); {} if absent."""
    import csv
    try:
        with open(STAGE_COUNTERS_CSV) as f:
            return {r["kernel"]: r for r in csv.DictReader(f)}
    except OSError:
        return {}


def measured_peak_gbs() -> tuple[float, str]:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ---- the oracle legs: cpu_baseline and --impl reference -----------------------------------------
def time_oracle(d: dict, n_events: int) -> tuple[float, int]:
    """The oracle as it stands (single thread) on the first n_events of the workload. Returns
    (seconds, hits processed)."""
    import oracle
    off = d["event_offsets"]
    h1 = int(off[n_events])
    t0 = time.perf_counter()
    r = oracle.reconstruct(d["x"][:h1], d["y"][:h1], d["z"][:h1], d["module"][:h1], off[:n_events + 1], N_MODULES)
    dt = time.perf_counter() - t0
    assert r["status"] == 0
    time_oracle.last_result = r
    return dt, h1 - int(off[0])


def time_oracle_after_path(d: dict, n_events: int) -> dict:
    """The oracle's Kalman filter and vertex finder (oracle/velo_next_oracle.c) on the tracks of the last
    time_oracle() call: seconds for the sample, one thread."""
    import oracle
    r = time_oracle.last_result
    h1 = int(d["event_offsets"][n_events])
    t0 = time.perf_counter()
    oracle.kalman_tracks(r, d["x"][:h1], d["y"][:h1], d["z"][:h1], oracle.default_params().sigma_hit)
    t1 = time.perf_counter()
    pv = oracle.pv_find(r["event_track_offsets"], r["states"])
    t2 = time.perf_counter()
    return {"kalman_s": t1 - t0, "pv_s": t2 - t1, "n_pvs": pv["n_pvs"], "events": n_events}


def run_reference(args):
    """Base contract's reference arm for this tier: the CPU oracle (oracle/velo_oracle.c, one
    thread) on a bounded sample of the same workload, on this box's host cores."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2412_05041_b200 import datagen
    cfg, n_full, n_batches = datagen.CONFIGS[args.config]
    sample = min(args.events or 2000, n_full)
    d = datagen.generate(cfg, 0, sample)
    for _ in range(args.warmup):
        time_oracle(d, min(sample, 200))
    tot_t, tot_h = 0.0, 0
    for _ in range(args.steps):
        dt, nh = time_oracle(d, sample)
        tot_t += dt; tot_h += nh
    value = sample * args.steps / tot_t
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "hits_per_s": tot_h / tot_t,
        "config": {"workload": workload_name(args.config, n_full, n_batches),
                   "sample": f"each step = the first {sample} events of that workload"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle",
                         "sample": f"first {sample} events of the workload, {args.steps} steps"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ---- the CUDA arm ----------------------------------------------------------------------------------
class Workload:
    """One BASELINE.json config resident in HBM: pinned host arrays, device hits, per-batch outputs."""

    def __init__(self, velo, datagen, sharding, torch, cfg_index, n_events_override, rank, opts_kw, want_pixels=False,
                 custom=None):
        self.torch, self.velo = torch, velo
        self.cfg_index = cfg_index
        # custom: (GenConfig, n_events, n_batches) of a workload that is not one of BASELINE.json's configs
        cfg, n_events, n_batches = custom if custom is not None else datagen.CONFIGS[cfg_index]
        if n_events_override:
            n_events = n_events_override
        self.n_events, self.n_batches, self.cfg = n_events, n_batches, cfg
        self.keep = []

        def pinned(shape, dtype):
            t = torch.empty(int(np.prod(shape)) if not np.isscalar(shape) else int(shape),
                            dtype={np.float32: torch.float32, np.uint8: torch.uint8, np.uint32: torch.int32}[np.dtype(dtype).type],
                            pin_memory=True)
            self.keep.append(t)
            return t.numpy().view(np.dtype(dtype))

        e0, _ = sharding.weak_event_range(rank, n_events)   # every rank its own events: weak scaling
        self.d = d = datagen.generate(cfg, e0, n_events, alloc=pinned, pixels=want_pixels)
        self.off = off = d["event_offsets"]
        self.n_hits = d["n_hits"]
        self.cuts = cuts = [n_events * b // n_batches for b in range(n_batches + 1)]
        if cfg.stagger_z != 0.0:      # 52-sensor layout: both sensor planes of every station (include/velo.h module_z_b)
            za, zb = datagen.sensor_planes(cfg)
            self.g = velo.velo_geometry_load(za, half_shift_x=cfg.half_shift_x, module_z_b=zb)
        else:
            self.g = velo.velo_geometry_load(datagen.MODULE_Z, half_shift_x=cfg.half_shift_x)
        self.P = velo.velo_params_default(self.g)
        self.dh = velo.DeviceHits(d["x"], d["y"], d["z"], d["module"], off)
        self.opts_kw = opts_kw
        opts0 = velo.LaunchOptions(**opts_kw)
        self.outs, self.hstructs = [], []
        for b in range(n_batches):
            nh = int(off[cuts[b + 1]]) - int(off[cuts[b]])
            self.outs.append(velo.DeviceTracks(cuts[b + 1] - cuts[b], nh, opts=opts0))
            self.hstructs.append(self.dh.slice_struct(cuts[b], cuts[b + 1], nh))
        self.streams = [torch.cuda.Stream() for _ in range(n_batches)]
        self.main = torch.cuda.current_stream()
        self.fork = torch.cuda.Event()
        self.joins = [torch.cuda.Event() for _ in range(n_batches)]

    def step(self):
        """One pass of the whole hot path over the workload: every batch on its own stream."""
        velo = self.velo
        self.fork.record(self.main)
        o = velo.LaunchOptions(**self.opts_kw)
        for b in range(self.n_batches):
            self.streams[b].wait_event(self.fork)
            velo.velo_reconstruct(self.g, self.hstructs[b], self.P, self.outs[b], self.streams[b], o)
            self.joins[b].record(self.streams[b])
            self.main.wait_event(self.joins[b])

    def stage_pass(self, reps):
        """The same batches one after the other on ONE stream with an event at every stage boundary
        (velo_launch_options_t.stage_events): the duration of every kernel of the path, measured
        with CUDA events on the stream it is launched on. Returns {stage: mean ms per launch}."""
        torch, velo = self.torch, self.velo
        st = self.streams[0]
        ev = [[[torch.cuda.Event(enable_timing=True) for _ in range(velo.VELO_N_STAGE_EVENTS)]
               for _ in range(self.n_batches)] for _ in range(reps)]
        torch.cuda.synchronize()
        for r in range(reps):
            for b in range(self.n_batches):
                o = velo.LaunchOptions(**self.opts_kw)
                for k in range(velo.VELO_N_STAGE_EVENTS):
                    ev[r][b][k].record(st)      # a torch event is created lazily by its first record()
                    o.stage_events[k] = ev[r][b][k].cuda_event
                velo.velo_reconstruct(self.g, self.hstructs[b], self.P, self.outs[b], st, o)
        torch.cuda.synchronize()
        out = {}
        for k, (name, _) in enumerate(STAGES):
            out[name] = float(np.mean([ev[r][b][k].elapsed_time(ev[r][b][k + 1])
                                       for r in range(reps) for b in range(self.n_batches)]))
        return out

    def after_path_pass(self, reps):
        """The two steps after the hot path on the batches' device outputs:
        velo_kalman_fit and velo_pv_find, timed with CUDA events on one stream."""
        torch, velo = self.torch, self.velo
        st = self.streams[0]
        pvs = [velo.DevicePvs(o.n_events, o.cap_tracks) for o in self.outs]
        kal = torch.empty((velo.VELO_N_STATE, max(o.cap_tracks for o in self.outs)), dtype=torch.float32, device="cuda")
        ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(reps * self.n_batches)]
        torch.cuda.synchronize()
        with torch.cuda.stream(st):
            for r in range(reps):
                for b in range(self.n_batches):
                    e = ev[r * self.n_batches + b]
                    e[0].record(st)
                    velo.velo_kalman_fit(self.hstructs[b], self.outs[b], self.P.sigma_hit, stream=st, out=kal)
                    e[1].record(st)
                    velo.velo_pv_find(self.outs[b], pvs[b], stream=st)
                    e[2].record(st)
        torch.cuda.synchronize()
        n_pvs = sum(p.to_host()["n_pvs"] for p in pvs)
        return {"kalman_ms_per_launch": float(np.median([e[0].elapsed_time(e[1]) for e in ev])),
                "pv_ms_per_launch": float(np.median([e[1].elapsed_time(e[2]) for e in ev])), "n_pvs": n_pvs,
                "what": "velo_kalman_fit (parameterised Kalman filter on the VELO segment) and velo_pv_find (primary "
                        "vertices) on each batch's device outputs; not part of `value`"}

    def results(self):
        return [o.to_host() for o in self.outs]          # raises on any device-side status

    def alg_bytes(self, res):
        off, cuts = self.off, self.cuts
        return [algorithmic_bytes(cuts[b + 1] - cuts[b], int(off[cuts[b + 1]]) - int(off[cuts[b]]),
                                  res[b]["n_tracks"], res[b]["n_track_hits"]) for b in range(self.n_batches)]

    def free(self):
        self.outs = self.hstructs = self.dh = self.d = self.keep = None
        self.torch.cuda.empty_cache()


def timed_steps(torch, dist, world, wl, warmup, steps, sampler=None):
    """W untimed steps, then exactly K timed steps between barrier + synchronize; device time with CUDA
    events on the launching stream, max over ranks. Returns (total ms, [ms of every step])."""
    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(warmup):
        wl.step()
    barrier()
    if sampler:
        sampler.start()
    marks = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    marks[0].record(wl.main)
    for i in range(steps):
        wl.step()
        marks[i + 1].record(wl.main)
    barrier()
    total = marks[0].elapsed_time(marks[steps])
    per_step = [marks[i].elapsed_time(marks[i + 1]) for i in range(steps)]
    if world > 1:
        t = torch.tensor([total] + per_step, device="cuda"); dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total, per_step = float(t[0].item()), [float(v) for v in t[1:].tolist()]
    return total, per_step


def run_velo(args):
    import torch
    import torch.distributed as dist

    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl velo needs a CUDA device: there is no CPU fallback")
    from paper_2412_05041_b200 import build as vbuild
    from paper_2412_05041_b200 import datagen, sharding, velo

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    vbuild.build()
    velo.lib()

    opts_kw = dict(ctas_per_sm=args.ctas_per_sm, path=args.path, track_group=args.track_group,
                   track_teams=args.track_teams, fit_teams=args.fit_teams, sort_teams=args.sort_teams,
                   pool_units=args.pool_units)
    kernels_per_batch = 3 if args.path == 1 else 7   # sort, order, track, slab, fit, offsets, write
    wl = Workload(velo, datagen, sharding, torch, args.config, args.events, rank, opts_kw, want_pixels=not args.no_e2e)
    n_events, n_batches, n_hits, off, cuts = wl.n_events, wl.n_batches, wl.n_hits, wl.off, wl.cuts
    launches = 0

    if args.timeline:
        for _ in range(args.warmup):
            wl.step()
        torch.cuda.synchronize()
        # windows of the sort / track / fit kernels of the last warm-up step's batches (GPU global timer)
        rows, phases = [], []
        for b, o in enumerate(wl.outs):
            skip = o.workspace_ptr - o.workspace.data_ptr() + 256
            clk = o.workspace[skip:skip + 512].cpu().numpy().view(np.uint64)
            rows.append([(int(~clk[2 * k]), int(clk[2 * k + 1])) for k in range(3)])
            phases.append(clk.copy())
        t0 = min(r[0][0] for r in rows)
        for b, r in enumerate(rows):
            print("batch %d: " % b + "  ".join("%s %8.3f .. %8.3f ms" % (nm, (s - t0) / 1e6, (e - t0) / 1e6)
                                                 for nm, (s, e) in zip(("sort", "track", "fit"), r)), flush=True)
        # SM clocks per event and phase, summed over the team leaders (batch 0)
        names = {"sort": (8, ["fetch", "decode", "scan", "scatter+rank", "place", "starts+write", "free"]),
                 "track": (16, ["fetch: pool wait and barrier", "setup", "wait module", "forwarding", "centre list", "seeding", "tail",
                                "fetch: ticket and descriptors"]),
                 "fit": (32, ["fetch", "weak filter", "fit", "owners 1", "owners 2", "clone+counts"])}
        clk = phases[0]
        for nm, (base, labels) in names.items():
            nev = max(int(clk[base]), 1)
            print("%s: %d events; SM clocks per event: " % (nm, nev) +
                  ", ".join("%s %.0f" % (l, clk[base + 1 + i] / nev) for i, l in enumerate(labels)), flush=True)
        return

    sampler = ClockSampler(local)
    ms_total, per_step = timed_steps(torch, dist, world, wl, args.warmup, args.steps, sampler)
    clocks = sampler.stop()
    launches += kernels_per_batch * n_batches * (args.steps + args.warmup)
    ms_step = float(np.median(per_step))

    # -- results of the last step: sizes for the byte counts, status for validity --
    res = wl.results()
    n_tracks = sum(r["n_tracks"] for r in res); n_thits = sum(r["n_track_hits"] for r in res)
    n_deferred = sum(r["n_deferred"] for r in res)
    alg_batch = wl.alg_bytes(res)
    alg_launch = float(np.mean(alg_batch))

    # -- every kernel of the path timed on its own stream (one stream, stage events) --
    stage_reps = max(1, min(args.steps, 5))
    stage_ms = wl.stage_pass(stage_reps)
    launches += kernels_per_batch * n_batches * stage_reps
    stage_sum = sum(stage_ms.values())
    after_path = wl.after_path_pass(stage_reps)
    launches += 4 * n_batches * stage_reps
    peak, peak_src = measured_peak_gbs()
    # algorithmic bytes of the two steps per launch: the filter gathers x, y, z of every track hit through
    # its index and writes 13 state words per track; the vertex finder reads six state words per track
    nt_b = n_tracks / n_batches; nth_b = n_thits / n_batches
    kal_bytes = 16.0 * nth_b + (4 + 52) * nt_b
    pv_bytes = 24.0 * nt_b + 4.0 * (n_events / n_batches) + 20.0 * after_path["n_pvs"] / n_batches
    after_path["kalman_roofline"] = {"bound": "hbm", "algorithmic_bytes_per_launch": kal_bytes,
                                     "achieved": kal_bytes / (after_path["kalman_ms_per_launch"] * 1e-3) / 1e9, "peak": peak,
                                     "unit": "GB/s", "frac": kal_bytes / (after_path["kalman_ms_per_launch"] * 1e-3) / 1e9 / peak}
    after_path["pv_roofline"] = {"bound": "hbm", "algorithmic_bytes_per_launch": pv_bytes,
                                 "achieved": pv_bytes / (after_path["pv_ms_per_launch"] * 1e-3) / 1e9, "peak": peak,
                                 "unit": "GB/s", "frac": pv_bytes / (after_path["pv_ms_per_launch"] * 1e-3) / 1e9 / peak,
                                 "limiter": "instruction issue and latency of a warp per event (histogram of 2 400 bins, four fit "
                                            "iterations), not HBM"}
    counters = stage_counters() if (args.config == 2 and args.path == 0 and n_events // n_batches == STAGE_COUNTERS_EVENTS) else {}

    def traffic_of(kernels):
        if not counters or any(k not in counters for k in kernels):
            return None
        return sum(int(counters[k]["dram_bytes_read"]) + int(counters[k]["dram_bytes_write"]) for k in kernels)

    stages = []
    for name, kernels in STAGES:
        ms = stage_ms[name]
        stages.append({"stage": name, "kernels": kernels, "ms_per_launch": ms, "share_of_path": ms / stage_sum,
                       "achieved": alg_launch / (ms * 1e-3) / 1e9 if ms > 0 else None, "traffic": traffic_of(kernels)})
    dom = max(stages, key=lambda s_: s_["ms_per_launch"])
    step_gbs = float(sum(alg_batch)) / (ms_step * 1e-3) / 1e9
    all_kernels = [k for _, ks in STAGES for k in ks]
    step_traffic = traffic_of(all_kernels)
    warp_inst = sum(int(counters[k]["warp_instructions"]) for k in all_kernels) / STAGE_COUNTERS_EVENTS if counters else None
    mhz = clocks.get("sm_mhz") or 1965.0
    issue_peak = 148 * 4 * mhz * 1e6
    events_per_s = world * n_events / (ms_step * 1e-3)

    line = {
        "metric": METRIC, "value": events_per_s, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "ms_per_step_mean": ms_total / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "hits_per_s": world * n_hits / (ms_step * 1e-3),
        "config": {"workload": workload_name(args.config, n_events, n_batches), "events_per_gpu": n_events,
                   "hits_per_gpu": n_hits, "tracks": n_tracks, "track_hits": n_thits, "streams": n_batches,
                   "events_deferred_to_slab_kernel": n_deferred,
                   "event_kernels": "slab only" if args.path == 1 else
                                    "three-stage pipeline (sort, module loop, fit) + slab kernel for deferred events",
                   "cache": "inputs larger than L2 (%.2f GB per step)" % (13 * n_hits / 1e9),
                   "timing": "median of the steps (device time, CUDA events, max over ranks)",
                   "parallelism": f"events sharded over {world} GPU(s), no collective"},
        "roofline": {"bound": "hbm", "kernel": " + ".join(dom["kernels"][:1]), "stage": dom["stage"],
                     "achieved": dom["achieved"], "peak": peak, "unit": "GB/s", "frac": dom["achieved"] / peak,
                     "traffic": dom["traffic"],
                     "traffic_source": "profiles/r02j_stage_counters.csv (ncu --set full, one 25 000-event launch of every kernel)"
                                       if counters else None,
                     "peak_source": peak_src, "algorithmic_bytes_per_launch": alg_launch,
                     "kernel_ms_per_launch": dom["ms_per_launch"], "kernel_share_of_step": dom["share_of_path"],
                     "how": "algorithmic bytes of one batch / duration of that batch's launch of the stage, CUDA events "
                            "at the stage boundaries on the launching stream, batches one after the other on one stream, "
                            "%d passes after the timed region" % stage_reps,
                     "stages": stages, "path_ms_per_launch": stage_sum,
                     "step_achieved": step_gbs, "step_frac": step_gbs / peak, "step_traffic": step_traffic,
                     "step_traffic_over_algorithmic": step_traffic * n_batches / float(sum(alg_batch)) if step_traffic else None,
                     "frac_of_nominal_8TBs": step_gbs / 8000.0, "target_frac": 0.40, "target_met": step_gbs / peak >= 0.40,
                     "limiter": "instruction issue and event latency, not HBM: every stage holds an event's shared memory "
                                "for the length of its dependent instruction chains and waits at its team barriers (profiles/r02j_pipeline.md)"},
        "issue": ({"bound": "alu", "achieved": events_per_s / world * warp_inst / 1e9, "peak": issue_peak / 1e9,
                   "unit": "G warp instr/s", "frac": events_per_s / world * warp_inst / issue_peak,
                   "warp_instructions_per_event": warp_inst, "source": "profiles/r02j_stage_counters.csv"}
                  if warp_inst else None),
        "after_path": after_path,
        "clocks": clocks,
    }

    # -- end to end through the host-buffer C-ABI call (velo_scheduler_run_host): pinned host
    #    inputs -> H2D -> kernels -> D2H of the produced tracks, all inside the timed region --
    d = wl.d
    if not args.no_e2e:
        # The packed-input call is bound by the device->host copy of the produced tracks, which cannot start before
        # the first batch is through H2D and the kernels: batches of growing size (10, 20, 30, 40 % of the events)
        # let it start after a tenth of the input, and every later batch is ready before the copy of the one before
        # ends (39.8 instead of 42.3 ms per step). The fp32 call is bound by its 2.46 GB of input and keeps equal
        # batches (a large last batch would leave its kernels and its copy behind the last upload).
        eq_cuts = cuts
        if n_batches == 4 and args.e2e_split == "growing":
            fr = [float(v) for v in args.e2e_fractions.split(",")]
            acc = np.cumsum(fr) / sum(fr)
            cuts = [0] + [int(round(n_events * f)) for f in acc[:-1]] + [n_events]
        px_batches = len(cuts) - 1
        max_ev = max(c[b + 1] - c[b] for c in (cuts, eq_cuts) for b in range(len(c) - 1))
        max_h = max(int(off[c[b + 1]]) - int(off[c[b]]) for c in (cuts, eq_cuts) for b in range(len(c) - 1))
        g, P = wl.g, wl.P
        wl.outs = wl.hstructs = wl.dh = None
        torch.cuda.empty_cache()
        sched = velo.Scheduler(g, max(n_batches, px_batches), max_ev, max_h)
        houts = [velo.HostTracks(eq_cuts[b + 1] - eq_cuts[b], int(off[eq_cuts[b + 1]]) - int(off[eq_cuts[b]])) for b in range(n_batches)]
        off_pinned = torch.from_numpy(off.view(np.int32).copy()).pin_memory()
        e2e_steps = max(1, min(args.steps, 5))
        off_u32 = off_pinned.numpy().view(np.uint32)
        fmt = velo.PixelFormat(pitch=wl.cfg.pitch, half_shift_x=wl.cfg.half_shift_x)
        px_pinned = torch.from_numpy(d["pixel"].view(np.int32)) if "pixel" in d else None

        def measure(run):
            run()  # warm-up
            if world > 1:
                dist.barrier()
            torch.cuda.synchronize()
            times = []
            for _ in range(e2e_steps):
                w0 = time.perf_counter()
                run()                      # returns after every copy has completed
                times.append(time.perf_counter() - w0)
            t_ = float(np.median(times))
            if world > 1:
                tt = torch.tensor([t_], device="cuda"); dist.all_reduce(tt, op=dist.ReduceOp.MAX); t_ = float(tt.item())
            hres = [h.result() for h in houts]
            assert sum(r["n_tracks"] for r in hres) == n_tracks and sum(r["n_track_hits"] for r in hres) == n_thits
            return t_, hres

        soa_s, hres = measure(lambda: sched.run_host(P, d["x"], d["y"], d["z"], d["module"], off_u32, eq_cuts, houts))
        d2h = sum(4 * velo.VELO_N_SUMMARY + 4 * (eq_cuts[b + 1] - eq_cuts[b] + 1) + 4 * (r["n_tracks"] + 1) + 52 * r["n_tracks"] + 4 * r["n_track_hits"]
                  for b, r in enumerate(hres))
        off_bytes = sum(4 * (eq_cuts[b + 1] - eq_cuts[b] + 1) for b in range(n_batches))
        e2e_soa = {"value": world * n_events / soa_s, "unit": UNIT, "h2d_bytes_per_step": 13 * n_hits + off_bytes,
                   "d2h_bytes_per_step": d2h, "ms_per_step": 1e3 * soa_s, "steps": e2e_steps,
                   "pcie_gbs": (13 * n_hits + off_bytes + d2h) / soa_s / 1e9,
                   "input": "fp32 SoA hits (x, y, z f32 + module u8: 13 B per hit)",
                   "api": "velo_scheduler_run_host (pinned host buffers, %d streams)" % n_batches}
        launches += kernels_per_batch * n_batches * (e2e_steps + 1)
        if px_pinned is not None:
            if cuts is not eq_cuts:
                houts = None   # (pinned host memory: free the equal batches' buffers first)
                houts = [velo.HostTracks(cuts[b + 1] - cuts[b], int(off[cuts[b + 1]]) - int(off[cuts[b]])) for b in range(px_batches)]
            px_s, _ = measure(lambda: sched.run_host_pixels(P, px_pinned, off_u32, fmt, cuts, houts))
            line["e2e"] = {"value": world * n_events / px_s, "unit": UNIT, "h2d_bytes_per_step": 4 * n_hits + off_bytes,
                           "d2h_bytes_per_step": d2h, "ms_per_step": 1e3 * px_s, "steps": e2e_steps,
                           "pcie_gbs": (4 * n_hits + off_bytes + d2h) / px_s / 1e9,
                           "input": "packed pixel addresses (4 B per hit; include/velo.h velo_pixel_hits_t), decoded inside "
                                    "stage 1; identical tracks to the fp32 path (tests/test_gpu_pixels.py)",
                           "bound": "PCIe: the device->host copy of the produced tracks (%.2f GB per step)" % (d2h / 1e9),
                           "api": "velo_scheduler_run_host_pixels (pinned host buffers, %d streams)" % max(n_batches, px_batches),
                           "batches": [cuts[b + 1] - cuts[b] for b in range(px_batches)]}
            line["e2e_fp32_soa"] = e2e_soa
            launches += kernels_per_batch * px_batches * (e2e_steps + 1)
        else:
            line["e2e"] = e2e_soa
        sched.close()

    # -- the oracle on this box's host cores (rank 0, N=1 only): a baseline, not the target --
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        sample = min(n_events, 4000 if args.config != 4 else 60)
        runs = [time_oracle(d, sample) for _ in range(3)]
        dt = float(np.median([r[0] for r in runs])); nh = runs[0][1]
        line["cpu_baseline"] = {"value": sample / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "hits_per_s": nh / dt, "host_cores_available": os.cpu_count(),
                                "sample": f"first {sample} events of the workload, median of 3 passes, {dt:.1f} s each"}
        ap = time_oracle_after_path(d, sample)
        line["after_path"]["cpu_oracle"] = {"kalman_events_per_s": sample / ap["kalman_s"], "pv_events_per_s": sample / ap["pv_s"],
                                            "cores": 1, "sample": f"the same {sample} events"}
        per_batch = n_events / n_batches
        line["after_path"]["kalman_events_per_s"] = per_batch / (line["after_path"]["kalman_ms_per_launch"] * 1e-3)
        line["after_path"]["pv_events_per_s"] = per_batch / (line["after_path"]["pv_ms_per_launch"] * 1e-3)

    # -- the small- and large-event regimes: short legs on configs[3] and configs[4] (device-resident) --
    if args.config == 2 and not args.events and not args.no_other_workloads and world == 1:
        wl.free()
        others = []
        for ci in (3, 4):
            w2 = Workload(velo, datagen, sharding, torch, ci, None, rank, opts_kw)
            k2 = max(3, min(args.steps, 5))
            _, ps = timed_steps(torch, dist, world, w2, 3, k2)
            r2 = w2.results()
            ms2 = float(np.median(ps))
            gbs2 = float(sum(w2.alg_bytes(r2))) / (ms2 * 1e-3) / 1e9
            st2 = w2.stage_pass(2)
            launches += kernels_per_batch * w2.n_batches * (3 + k2 + 2)
            others.append({"workload": workload_name(ci, w2.n_events, w2.n_batches), "value": w2.n_events / (ms2 * 1e-3),
                           "unit": UNIT, "hits_per_s": w2.n_hits / (ms2 * 1e-3), "ms_per_step": ms2, "steps": k2,
                           "hits": w2.n_hits, "tracks": sum(r["n_tracks"] for r in r2),
                           "events_deferred_to_slab_kernel": sum(r["n_deferred"] for r in r2),
                           "roofline": {"bound": "hbm", "step_achieved": gbs2, "peak": peak, "unit": "GB/s", "step_frac": gbs2 / peak,
                                        "stage_ms_per_launch": st2}})
            w2.free()
        # SURVEY.md §8(f) f4's layout variants (DESIGN.md §2 A23, L-1), mu = 5 like configs[1]: half of the tracks
        # backward (same kernels), and the 52-sensor layout (two staggered, overlapping sensors per station, both
        # planes declared in the geometry: the two-plane instantiation of the pipeline's kernels)
        from dataclasses import replace
        base_cfg = datagen.CONFIGS[1][0]
        for name, cfg_v, n_v in (("mu=5, backward_frac 0.5", replace(base_cfg, backward_frac=0.5), 25000),
                                 ("mu=5, 52-sensor layout (stagger_z 12.5 mm, overlap_x 0.5 mm)",
                                  replace(base_cfg, stagger_z=12.5, overlap_x=0.5), 25000)):
            w2 = Workload(velo, datagen, sharding, torch, 1, None, rank, opts_kw, custom=(cfg_v, n_v, 1))
            _, ps = timed_steps(torch, dist, world, w2, 3, 3)
            r2 = w2.results()
            ms2 = float(np.median(ps))
            launches += kernels_per_batch * (3 + 3)
            others.append({"workload": f"{name}: {n_v} events in 1 batch, seed 1", "value": n_v / (ms2 * 1e-3), "unit": UNIT,
                           "hits_per_s": w2.n_hits / (ms2 * 1e-3), "ms_per_step": ms2, "steps": 3, "hits": w2.n_hits,
                           "tracks": sum(r["n_tracks"] for r in r2),
                           "events_deferred_to_slab_kernel": sum(r["n_deferred"] for r in r2)})
            w2.free()
        line["other_workloads"] = others
    line["gpu_launches"] = launches
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def respawn_under_torchrun(args) -> int:
    """`python bench.py --gpus N` with N > 1 and no torchrun environment: start N ranks of this script
    under torch.distributed.run on this node (one process per GPU) and pass their output through."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    args = parse_args()
    if args.timeline:
        os.environ["VELO_TIMELINE_BUILD"] = "1"

    if args.impl == "reference":
        run_reference(args)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(respawn_under_torchrun(args))
    else:
        run_velo(args)


if __name__ == "__main__":
    main()

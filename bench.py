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

# dram__bytes_read.sum + dram__bytes_write.sum of one event-kernel launch, from the ncu --set full
# capture summarised in profiles/r01c_team_kernel_25k.md; key = (config, path, events per step)
NCU_DRAM_BYTES_PER_LAUNCH = {(2, 0, 100_000): 676_917_248 + 496_348_160}
# smsp__inst_executed.sum of the same capture / its 25 000 events: what bounds the path in practice
NCU_WARP_INST_PER_EVENT = {(2, 0): 94_811.0}

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
    ap.add_argument("--teams", type=int, default=0, help="teams per CTA of the team kernel (0 = library default)")
    ap.add_argument("--path", type=int, default=0, help="0 = team kernel + slab for deferred events, 1 = slab only")
    ap.add_argument("--track-group", type=int, default=0, help="threads per event of the module-loop kernel (0 = default)")
    ap.add_argument("--track-teams", type=int, default=0)
    ap.add_argument("--fit-teams", type=int, default=0)
    ap.add_argument("--sort-teams", type=int, default=0)
    ap.add_argument("--pool-units", type=int, default=0)
    ap.add_argument("--timeline", action="store_true",
                    help="instrumented build: print when each pipeline stage of each batch ran, then exit")
    ap.add_argument("--no-e2e", action="store_true")
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


def issue_block(args, events_per_s: float, clocks: dict):
    """The practical limiter beside the HBM roofline: warp instructions issued per second against
    the issue peak of the chip (148 SMs x 4 schedulers x 1 warp instruction per clock at the SM
    clock seen during the run). Instructions per event come from the ncu capture in profiles/."""
    per_event = NCU_WARP_INST_PER_EVENT.get((args.config, args.path))
    mhz = clocks.get("sm_mhz") or 1965.0
    if per_event is None:
        return None
    peak = 148 * 4 * mhz * 1e6
    return {"bound": "alu", "achieved": events_per_s * per_event / 1e9, "peak": peak / 1e9, "unit": "G warp instr/s",
            "frac": events_per_s * per_event / peak, "warp_instructions_per_event": per_event,
            "source": "profiles/r01c_team_kernel_25k.md"}


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
    return dt, h1 - int(off[0])


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

    # -- synthetic workload: this rank's own events (weak scaling) --
    cfg, n_events, n_batches = datagen.CONFIGS[args.config]
    if args.events:
        n_events = args.events
    keep = []  # pinned host tensors behind the numpy views

    def pinned(shape, dtype):
        t = torch.empty(int(np.prod(shape)) if not np.isscalar(shape) else int(shape),
                        dtype={np.float32: torch.float32, np.uint8: torch.uint8}[np.dtype(dtype).type],
                        pin_memory=True)
        keep.append(t)
        return t.numpy()

    e0, _ = sharding.weak_event_range(rank, n_events)   # every rank its own events: weak scaling
    d = datagen.generate(cfg, e0, n_events, alloc=pinned)
    off = d["event_offsets"]
    n_hits = d["n_hits"]
    cuts = [n_events * b // n_batches for b in range(n_batches + 1)]
    g = velo.velo_geometry_load(datagen.MODULE_Z, half_shift_x=cfg.half_shift_x)
    P = velo.velo_params_default(g)
    dh = velo.DeviceHits(d["x"], d["y"], d["z"], d["module"], off)
    tune = dict(track_group=args.track_group, track_teams=args.track_teams, fit_teams=args.fit_teams,
                sort_teams=args.sort_teams, pool_units=args.pool_units)
    opts0 = velo.LaunchOptions(ctas_per_sm=args.ctas_per_sm, path=args.path, teams_per_cta=args.teams, **tune)
    launches_per_batch = 3 if args.path == 1 else 5   # [order, team kernel,] slab kernel, offsets, compaction
    streams = [torch.cuda.Stream() for _ in range(n_batches)]
    if os.environ.get('VELO_BENCH_SERIAL'):
        streams = [streams[0]] * n_batches
    main = torch.cuda.current_stream()
    outs, hstructs = [], []
    for b in range(n_batches):
        e0, e1 = cuts[b], cuts[b + 1]
        nh = int(off[e1]) - int(off[e0])
        outs.append(velo.DeviceTracks(e1 - e0, nh, opts=opts0))
        hstructs.append(dh.slice_struct(e0, e1, nh))
    n_steps_total = args.warmup + args.steps
    kev = [[(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_batches)]
           for _ in range(n_steps_total)]
    fork = torch.cuda.Event(); joins = [torch.cuda.Event() for _ in range(n_batches)]

    def step(i):
        fork.record(main)
        for b in range(n_batches):
            streams[b].wait_event(fork)
            # raw cudaEvent_t handles: a torch event is created lazily by its first record()
            ks, ke = kev[i][b]
            ks.record(streams[b]); ke.record(streams[b])
            o = velo.LaunchOptions(event_kernel_start=ks.cuda_event, event_kernel_stop=ke.cuda_event,
                                   ctas_per_sm=args.ctas_per_sm, path=args.path, teams_per_cta=args.teams, **tune)
            velo.velo_reconstruct(g, hstructs[b], P, outs[b], streams[b], o)
            joins[b].record(streams[b])
            main.wait_event(joins[b])

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for i in range(args.warmup):
        step(i)
    barrier()
    if args.timeline:
        # windows of the sort / track / fit kernels of the last warm-up step's batches (GPU global timer)
        rows, phases = [], []
        for b, o in enumerate(outs):
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
                 "track": (16, ["fetch", "setup", "wait module", "forwarding", "centre list", "seeding", "tail"]),
                 "fit": (32, ["fetch", "weak filter", "fit", "owners 1", "owners 2", "clone+counts"])}
        clk = phases[0]
        for nm, (base, labels) in names.items():
            nev = max(int(clk[base]), 1)
            print("%s: %d events; SM clocks per event: " % (nm, nev) +
                  ", ".join("%s %.0f" % (l, clk[base + 1 + i] / nev) for i, l in enumerate(labels)), flush=True)
        return
    sampler = ClockSampler(local); sampler.start()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record(main)
    for i in range(args.warmup, n_steps_total):
        step(i)
    t1.record(main)
    barrier()
    clocks = sampler.stop()
    ms_total = t0.elapsed_time(t1)
    if world > 1:
        t = torch.tensor([ms_total], device="cuda"); dist.all_reduce(t, op=dist.ReduceOp.MAX); ms_total = float(t.item())
    ms_step = ms_total / args.steps

    # -- results of the last step: sizes for the byte counts, status for validity --
    res = [o.to_host() for o in outs]          # raises on any device-side status
    n_tracks = sum(r["n_tracks"] for r in res); n_thits = sum(r["n_track_hits"] for r in res)
    n_deferred = sum(r["n_deferred"] for r in res)
    alg_batch = [algorithmic_bytes(cuts[b + 1] - cuts[b], int(off[cuts[b + 1]]) - int(off[cuts[b]]),
                                   res[b]["n_tracks"], res[b]["n_track_hits"]) for b in range(n_batches)]
    # The event kernels of a step's batches each fill the GPU (one persistent CTA per SM), so they run
    # back to back even though they are launched on different streams. Their average duration is the
    # span from the first start mark to the last stop mark of the step, divided by the launches.
    span_ms = []
    for i in range(args.warmup, n_steps_total):
        first = min(range(n_batches), key=lambda b: kev[i][0][0].elapsed_time(kev[i][b][0]))
        span_ms.append(max(kev[i][first][0].elapsed_time(kev[i][b][1]) for b in range(n_batches)))
    avg_kern_ms = float(np.mean(span_ms)) / n_batches
    peak, peak_src = measured_peak_gbs()
    achieved = float(np.mean(alg_batch)) / (avg_kern_ms * 1e-3) / 1e9
    step_gbs = float(sum(alg_batch)) / (ms_step * 1e-3) / 1e9

    value = world * n_events / (ms_step * 1e-3)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "hits_per_s": world * n_hits / (ms_step * 1e-3),
        "config": {"workload": workload_name(args.config, n_events, n_batches), "events_per_gpu": n_events,
                   "hits_per_gpu": n_hits, "tracks": n_tracks, "track_hits": n_thits, "streams": n_batches,
                   "events_deferred_to_slab_kernel": n_deferred,
                   "event_kernels": "slab only" if args.path == 1 else "shared-memory teams + slab for deferred events",
                   "cache": "inputs larger than L2 (%.2f GB per step)" % (13 * n_hits / 1e9),
                   "parallelism": f"events sharded over {world} GPU(s), no collective"},
        "roofline": {"bound": "hbm", "kernel": "velo_event_slab_kernel" if args.path == 1 else "velo_event_team_kernel (+ slab kernel for deferred events)", "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "traffic": NCU_DRAM_BYTES_PER_LAUNCH.get((args.config, args.path, n_events)),
                     "traffic_source": "profiles/r01c_team_kernel_25k.md (ncu --set full, one 25 000-event launch)",
                     "peak_source": peak_src,
                     "algorithmic_bytes_per_launch": float(np.mean(alg_batch)), "kernel_ms_per_launch": avg_kern_ms,
                     "kernel_share_of_step": avg_kern_ms * n_batches / ms_step,
                     "step_achieved": step_gbs, "step_frac": step_gbs / peak,
                     "frac_of_nominal_8TBs": step_gbs / 8000.0,
                     "limiter": "instruction issue and latency, not HBM (ncu: issue slots 52.0 % busy, DRAM 3 % busy, "
                                "94.8 k warp instructions per event; see profiles/ and DESIGN.md 5.1)"},
        "issue": issue_block(args, world * n_events / (ms_step * 1e-3), clocks),
        "clocks": clocks,
        "gpu_launches": launches_per_batch * n_batches * (args.steps + args.warmup),
    }

    # -- end to end through the host-buffer C-ABI call (velo_scheduler_run_host): pinned host
    #    inputs -> H2D -> kernels -> D2H of the produced tracks, all inside the timed region --
    if not args.no_e2e:
        max_ev = max(cuts[b + 1] - cuts[b] for b in range(n_batches))
        max_h = max(int(off[cuts[b + 1]]) - int(off[cuts[b]]) for b in range(n_batches))
        del outs, dh
        torch.cuda.empty_cache()
        sched = velo.Scheduler(g, n_batches, max_ev, max_h)
        houts = [velo.HostTracks(cuts[b + 1] - cuts[b], int(off[cuts[b + 1]]) - int(off[cuts[b]])) for b in range(n_batches)]
        off_pinned = torch.from_numpy(off.view(np.int32).copy()).pin_memory()
        e2e_steps = max(1, min(args.steps, 5))
        run = lambda: sched.run_host(P, d["x"], d["y"], d["z"], d["module"], off_pinned.numpy().view(np.uint32),
                                     cuts, houts)
        run()  # warm-up
        barrier()
        w0 = time.perf_counter()
        for _ in range(e2e_steps):
            run()
        torch.cuda.synchronize()
        e2e_s = (time.perf_counter() - w0) / e2e_steps
        if world > 1:
            t = torch.tensor([e2e_s], device="cuda"); dist.all_reduce(t, op=dist.ReduceOp.MAX); e2e_s = float(t.item())
        hres = [h.result() for h in houts]
        assert sum(r["n_tracks"] for r in hres) == n_tracks and sum(r["n_track_hits"] for r in hres) == n_thits
        h2d = 13 * n_hits + sum(4 * (cuts[b + 1] - cuts[b] + 1) for b in range(n_batches))
        d2h = sum(16 + 4 * (cuts[b + 1] - cuts[b] + 1) + 4 * (r["n_tracks"] + 1) + 52 * r["n_tracks"] + 4 * r["n_track_hits"]
                  for b, r in enumerate(hres))
        line["e2e"] = {"value": world * n_events / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d,
                       "d2h_bytes_per_step": d2h, "ms_per_step": 1e3 * e2e_s, "steps": e2e_steps,
                       "api": "velo_scheduler_run_host (pinned host buffers, %d streams)" % n_batches}
        line["gpu_launches"] += 5 * n_batches * (e2e_steps + 1)
        sched.close()

    # -- the oracle on this box's host cores (rank 0, N=1 only): a baseline, not the target --
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        sample = min(n_events, 4000 if args.config != 4 else 60)
        dt, nh = time_oracle(d, sample)
        line["cpu_baseline"] = {"value": sample / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "hits_per_s": nh / dt, "host_cores_available": os.cpu_count(),
                                "sample": f"first {sample} events of the workload, one pass, {dt:.1f} s"}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.timeline:
        os.environ["VELO_TIMELINE_BUILD"] = "1"

    if args.impl == "reference":
        run_reference(args)
    else:
        run_velo(args)


if __name__ == "__main__":
    main()

#!/usr/bin/env python
"""bench.py -- throughput of the EVIS event-synthesis hot path on B200 (contract: see DESIGN.md Sec. 8).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..4] [--impl ours|reference]

One "step" = one evis_step call = one keyframe interval of the whole batch: log-luminance of the new
keyframe, bidirectional warp with z-buffered splat to S substeps, event model on every substep,
compaction + deterministic ordering.  The keyframes are seeded
synthetic scenes (paper_2607_08098_b200/scenes.py) and are resident in HBM before the timed region
(`value`); `e2e` repeats the measurement through evis_step_host / evis_read_events with pinned HOST
buffers, host<->device copies inside the timed region.

Prints ONE JSON line on rank 0.  N > 1: one process per GPU (torchrun), envs are independent so every
rank runs its own batch of the same shape (different seed) with no data-path collective; the time is
the max over ranks ("scaling": "weak").
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "pixel-substeps/s"
ALGO_BYTES_PER_PIXEL = 52          # per pixel per keyframe interval, DESIGN.md Sec. 6
ALGO_BYTES_PER_EVENT = 16
FALLBACK_HBM_GBS = 6650.0          # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
ISSUE_PEAK = 148 * 4 * 32 * 1.965e9   # thread-instructions/s: SMs x schedulers x lanes x clocks.max.sm
SURVEY_INSTR_BOUNDS = (60.0, 150.0)   # algorithmic estimate of issued instructions per pixel-substep
# Committed ncu captures the line quotes (profiles/*.md say how each was made).  They are constants of a build, not
# measurements of this run: each names the git head and the hash of paper_2607_08098_b200/csrc it was taken on and the
# events per step of ITS steps; `stale` is set when the tree's kernels differ from the capture's, and the ratio
# traffic / algorithmic is formed with the capture's own algorithmic bytes.
RANGE_CAPTURE = os.path.join("profiles", "round2_a_range_cfg4.csv")      # instruction counts (schedule-independent)
RANGE_WORKLOAD, RANGE_STEPS = "cfg4_256env_346x260_S16_rl", 5
RANGE_CSRC_SHA = "6931bcd6ccdd"
GRAPH_CAPTURES = {      # workload -> whole steps as CUDA graphs (`ncu --graph-profiling graph`, bench.py --graph-probe)
    "cfg4_256env_346x260_S16_rl": {"file": os.path.join("profiles", "round3_b_graph_cfg4.csv"), "doc": "profiles/round3_b_graph_cfg4.md",
                                   "git_head": "0f0284c", "csrc_sha": "0afb0723d1b1", "events_per_step": None},
    "cfg2_16env_640x480_S16": {"file": os.path.join("profiles", "round2_h_graph_cfg2.csv"), "doc": "profiles/round2_h_graph_cfg2_cfg3.md",
                               "git_head": "120e9a6", "csrc_sha": "6931bcd6ccdd", "events_per_step": 10.3e6},
    "cfg3_64env_1280x720_S33_disk": {"file": os.path.join("profiles", "round2_h_graph_cfg3.csv"), "doc": "profiles/round2_h_graph_cfg2_cfg3.md",
                                "git_head": "120e9a6", "csrc_sha": "6931bcd6ccdd", "events_per_step": 88.0e6},
}


def csrc_sha() -> str:
    """Hash of the kernel sources in the tree (names and contents of csrc/*.cu, *.cuh, *.h), to tell whether a committed
    capture still describes this build."""
    import hashlib
    d = os.path.join(ROOT, "paper_2607_08098_b200", "csrc")
    h = hashlib.sha256()
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh", ".h")):
            h.update(f.encode())
            with open(os.path.join(d, f), "rb") as fh:
                h.update(fh.read())
    return h.hexdigest()[:12]


def step_traffic(workload: str):
    """(DRAM bytes read + written of ONE WHOLE STEP in the schedule the bench runs, capture record) from the committed
    `ncu --graph-profiling graph` capture of `workload`: the mean over its graph launches; (None, None) without one."""
    meta = GRAPH_CAPTURES.get(workload)
    if not meta:
        return None, None
    try:
        import csv
        rd, wr, inst = [], [], []
        with open(os.path.join(ROOT, meta["file"])) as f:
            for row in csv.reader(f):
                if len(row) >= 15 and row[4] == "graph":
                    if row[12] == "dram__bytes_read.sum":
                        rd.append(float(row[14].replace(",", "")))
                    elif row[12] == "dram__bytes_write.sum":
                        wr.append(float(row[14].replace(",", "")))
                    elif row[12] == "smsp__inst_executed.sum":
                        inst.append(float(row[14].replace(",", "")))
        if not rd or len(rd) != len(wr):
            return None, None
        rec = dict(meta, steps=len(rd), stale=meta["csrc_sha"] != csrc_sha(),
                   warp_instructions_per_step=sum(inst) / len(inst) if len(inst) == len(rd) else None)
        return (sum(rd) + sum(wr)) / len(rd), rec
    except (OSError, ValueError):
        return None, None


def range_capture(workload: str):
    """{metric: value per step} from the committed whole-step ncu capture when it describes `workload`, else None."""
    if workload != RANGE_WORKLOAD:
        return None
    out = {}
    try:
        import csv
        with open(os.path.join(ROOT, RANGE_CAPTURE)) as f:
            for row in csv.reader(f):
                if len(row) >= 13 and row[4] == "range":
                    out[row[10]] = float(row[12].replace(",", "")) / RANGE_STEPS
    except (OSError, ValueError):
        return None
    return out or None


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config (1-based, 1..4)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--envs", type=int, default=0, help="override the number of envs (0 = the config's)")
    ap.add_argument("--defocus", type=float, default=None,
                    help="switch the defocus blur on (sigma in pixels, PAPER.md:158): a variant measurement, not the headline")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = every rank its own batch of the config's shape (default); strong = ONE batch of the "
                         "config's shape, rank r takes the envs sharding.env_block(r, N, E) (sharding.ShardedEvis)")
    ap.add_argument("--composite-mode", type=int, default=0, choices=[0, 1, 2],
                    help="0 = B primary / A fills (the paper's, headline); 1 = blend; 2 = weighted front-surface splat: variants")
    ap.add_argument("--time-sorted", action="store_true", help="sort the stored stream by (env, t) on the device: a variant")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--profile-range", action="store_true",
                    help="bracket the timed region with cudaProfilerStart / Stop (for `ncu --replay-mode app-range`: "
                         "counters of the whole step in its real multi-stream schedule); implies no e2e / cpu legs")
    ap.add_argument("--graph-probe", action="store_true",
                    help="measurement hook: every timed step is captured and launched as ONE CUDA graph (EVIS_GRAPH=1) on a "
                         "stream of its own, so that `ncu --graph-profiling graph` measures the whole step in its real "
                         "multi-stream schedule; the steps are serialised by the capture: no throughput claim; implies no e2e / cpu legs")
    ap.add_argument("--sweep", action="store_true",
                    help="BASELINE.json config 5: one JSON line per (envs x resolution x S) point, device-resident")
    return ap.parse_args()


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], None, set()
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.15] or [r for (_, r) in self.rows]
        for r in rows:
            c = [x.strip() for x in r.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx = float(c[1])
            except ValueError:
                continue
            for name, v in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"], c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


# ------------------------------------------------------------------------------------------------
# the oracle legs (cpu_baseline of our arm; the whole --impl reference arm)
# ------------------------------------------------------------------------------------------------
def time_oracle(spec, n_envs: int, n_steps: int, warmup: int):
    """Run the CPU oracle (oracle/, as it stands, single thread) on the first `n_envs` envs of the
    workload for warmup + n_steps keyframe intervals.  Returns (pixel-substeps/s, events/s, seconds
    per step, events)."""
    from oracle import evis_oracle as orc
    from paper_2607_08098_b200 import scenes
    sub = scenes.small(spec, num_envs=n_envs)
    sc = scenes.make_scene(sub)
    o = orc.Oracle(n_envs, spec.height, spec.width, spec.substeps, spec.c_pos, spec.c_neg, spec.log_eps,
                   spec.keyframe_dt)
    kfs = [{a: b.numpy() for a, b in scenes.render_keyframe(sc, k).items()} for k in range(warmup + n_steps + 1)]
    for k in range(warmup + 1):                        # keyframe 0 initialises; then `warmup` intervals
        o.step(kfs[k]["rad"], kfs[k]["mv_bwd"], kfs[k]["depth"], kfs[k]["mv_fwd"])
    ev = 0
    t0 = time.perf_counter()
    for k in range(warmup + 1, warmup + 1 + n_steps):
        ev += len(o.step(kfs[k]["rad"], kfs[k]["mv_bwd"], kfs[k]["depth"], kfs[k]["mv_fwd"]))
    dt = time.perf_counter() - t0
    pxss = n_envs * spec.height * spec.width * spec.substeps * n_steps
    return pxss / dt, ev / dt, dt / n_steps, ev


def cpu_baseline(spec, seconds: float) -> dict:
    """The oracle on a bounded sample of the same workload, sized for about `seconds` of CPU work."""
    n_envs = min(spec.num_envs, 2)
    rate, _, per_step, _ = time_oracle(spec, n_envs, 1, 0)          # probe: one interval
    steps = max(1, min(60, int(seconds / max(per_step, 1e-3))))
    rate, ev_rate, per_step, _ = time_oracle(spec, n_envs, steps, 0)
    return {"value": rate, "unit": METRIC, "events_per_s": ev_rate, "cores": 1, "kind": "oracle",
            "sample": f"oracle/evis_oracle.c single thread, first {n_envs} envs of {spec.name} at full "
                      f"resolution, {steps} keyframe intervals ({per_step:.2f} s each)"}


def run_reference(args, spec) -> None:
    """--impl reference: there is no reference code (paper only), so the reference arm is the oracle,
    timed as it stands on the host cores.  Rank 0 alone works."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n_envs = min(spec.num_envs, 2)
    steps = args.steps
    rate, ev_rate, per_step, ev = time_oracle(spec, n_envs, steps, args.warmup)
    sample = (f"oracle/evis_oracle.c single thread; each step = one keyframe interval of the first {n_envs} "
              f"envs of {spec.name} at full resolution")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": rate, "unit": METRIC, "n_gpus": args.gpus,
        "steps": steps, "warmup": args.warmup, "ms_per_step": per_step * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": workload_config(spec, "cpu-oracle"),
        "events_per_s": ev_rate,
        "cpu_baseline": {"value": rate, "unit": METRIC, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": rate, "unit": METRIC, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def workload_config(spec, path: str) -> dict:
    return {"workload": spec.name, "envs": spec.num_envs, "height": spec.height, "width": spec.width,
            "substeps": spec.substeps, "keyframe_hz": round(1.0 / spec.keyframe_dt, 3),
            "c_pos": spec.c_pos, "c_neg": spec.c_neg, "log_eps": spec.log_eps, "path": path,
            "l2": ("inputs larger than L2 (one keyframe = %d MB >= 126 MB, a new one every step), no flush" if
                   spec.num_envs * spec.height * spec.width * 32 >= 126 << 20 else
                   "one keyframe = %d MB < L2 (126 MB), a new one every step, no flush: a parity-size config, not the "
                   "bench workload") % (spec.num_envs * spec.height * spec.width * 32 >> 20)}


# ------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------
def run_ours(args, spec) -> None:
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2607_08098_b200 import binding, scenes, sharding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback for the product path)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    binding.load()                                     # fails loudly when libevis.so is missing
    if args.graph_probe:
        os.environ["EVIS_GRAPH"] = "1"
        args.no_e2e = args.no_cpu = True
        args.profile_range = True                      # cudaProfilerStart / Stop around the timed steps (ncu --profile-from-start off)

    K, Wm = args.steps, args.warmup
    n_kf = Wm + K + 1
    if args.scaling == "strong" and world > 1:
        # ONE batch: rank r owns the envs env_block(r, world, E) of it (no exchange step); it renders only those
        e0, e1 = sharding.env_block(rank, world, spec.num_envs)
        if e1 == e0:
            raise SystemExit("bench.py: more ranks than environments")
        sc = scenes.make_scene(spec)
        kfs = [scenes.render_keyframe(sc, k, device=dev, envs=list(range(e0, e1))) for k in range(n_kf)]
        global_envs = spec.num_envs
        spec = scenes.small(spec, num_envs=e1 - e0)
    else:
        # every rank: its own batch of the same shape (envs are independent: no exchange step)
        spec = scenes.small(spec, seed=sharding.rank_seed(spec.seed, rank))
        sc = scenes.make_scene(spec)
        kfs = [scenes.render_keyframe(sc, k, device=dev) for k in range(n_kf)]
        global_envs = spec.num_envs * world
    E, H, W, S = spec.num_envs, spec.height, spec.width, spec.substeps
    path = binding.PATH_AUTO
    cap = int(min(0x7FFFFFFF, max(1 << 22, 10 * E * H * W)))          # events stored per step
    def mk():
        e = binding.Evis(E, H, W, S, spec.c_pos, spec.c_neg, spec.log_eps, spec.keyframe_dt,
                         max_motion_px=spec.max_motion_px(), path=path, device=local, event_capacity=cap,
                         composite_mode=args.composite_mode)
        if args.defocus is not None:
            e.set_defocus(args.defocus)
        if args.time_sorted:
            e.set_time_sorted(True)
        return e
    ev = mk()
    stream = torch.cuda.Stream(dev) if args.graph_probe else torch.cuda.current_stream(dev)   # a capture needs a stream of its own

    def step(k):
        f = kfs[k]
        ev.step(f["rad"], f["mv_bwd"], f["depth"], mv_fwd=f["mv_fwd"], stream=stream)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # ---- device-resident timing -------------------------------------------------------------------
    for k in range(Wm + 1):                             # keyframe 0 initialises, then W warm-up intervals
        step(k)
    barrier()
    i0 = ev.info()
    clk = ClockSampler(local)
    clk.start()
    time.sleep(0.25)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t0 = time.time()
    if args.profile_range:
        torch.cuda.profiler.start()
    e0.record(stream)
    for k in range(Wm + 1, Wm + 1 + K):
        step(k)
    ev.wait_events(stream)                              # the last step's ordered stream is part of the timed region
    e1.record(stream)
    barrier()
    if args.profile_range:
        torch.cuda.profiler.stop()
    t1 = time.time()
    ms = e0.elapsed_time(e1)
    clocks = clk.stop(t0, t1)
    i1 = ev.info()
    if i1.overflow_steps != i0.overflow_steps:          # sticky: any step of the timed region, not only the last
        raise SystemExit("bench.py: event capacity overflow in the timed region")
    events = i1.total_events - i0.total_events
    launches = i1.kernel_launches - i0.kernel_launches
    path_used = "global"

    # ---- per-stage device time of the same steps (second pass over the same keyframes, CUDA events
    #      recorded by the library on the launching stream) -> dominant kernel for the roofline -------
    ev.destroy()
    ev = mk()
    for k in range(Wm + 1):
        step(k)
    torch.cuda.synchronize(dev)
    j0 = ev.info()
    ev.profile_enable(True)
    for k in range(Wm + 1, Wm + 1 + K):
        step(k)
    prof = ev.profile_read()
    ev.profile_enable(False)
    j1 = ev.info()
    ev.destroy()
    # the same keyframes must give the same events: the timed pass runs fully asynchronously (regions' streams not joined,
    # the host far ahead), this pass with every region joined to the caller's stream
    if j1.total_events - j0.total_events != events:
        raise SystemExit(f"bench.py: the timed pass produced {events} events, the stage-timed pass over the same keyframes "
                         f"{j1.total_events - j0.total_events}: the asynchronous schedule is not deterministic")

    (ms,), (events, launches) = sharding.reduce_max_sum([ms], [float(events), float(launches)], dev)
    launches = int(launches)
    value = global_envs * H * W * S * K / (ms * 1e-3)        # all ranks' pixel-substeps over the slowest rank's time

    # ---- roofline: the WHOLE step's algorithmic bytes over the WHOLE step's time (the path is one fused pass over the
    #      keyframes: its stages overlap on several streams, so no stage is charged the bytes alone) --------------------
    peak, peak_src = hbm_peak()
    stage_ms = {k: v / K for k, v in prof["ms"].items()}
    dom = max(stage_ms, key=stage_ms.get)
    ev_per_step = events / world / K
    algo_bytes_step = ALGO_BYTES_PER_PIXEL * E * H * W + ALGO_BYTES_PER_EVENT * ev_per_step
    step_s = ms / K * 1e-3
    achieved = algo_bytes_step / step_s / 1e9
    pxss_step = E * H * W * S
    cap_ = range_capture(spec.name)
    traffic, trec = step_traffic(spec.name)
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "peak_source": peak_src,
                "traffic": traffic,
                "algorithmic_bytes_per_step": algo_bytes_step, "basis": "whole step: algorithmic bytes / ms_per_step",
                "dominant_stage_ms": stage_ms[dom], "dominant_stage_launches_per_step": max(1.0, prof["launches"][dom] / K),
                "stage_ms_per_step": stage_ms, "stage_launches_per_step": {k: v / K for k, v in prof["launches"].items()}}
    if trec:
        # the capture's own steps decide its algorithmic bytes (the same steps as this run's when events_per_step is None:
        # the capture was then taken with this command's --steps / --warmup on the same seeded keyframes)
        cap_events = trec["events_per_step"] if trec["events_per_step"] is not None else ev_per_step
        cap_algo = ALGO_BYTES_PER_PIXEL * E * H * W + ALGO_BYTES_PER_EVENT * cap_events
        roofline["traffic_capture"] = {
            "what": "DRAM bytes of one WHOLE step in its real multi-stream schedule: every step captured as one CUDA graph and "
                    "measured by `ncu --graph-profiling graph` (a committed capture, not this run)",
            "file": trec["file"], "doc": trec["doc"], "git_head": trec["git_head"], "csrc_sha": trec["csrc_sha"],
            "stale": trec["stale"], "steps": trec["steps"], "events_per_step": cap_events,
            "algorithmic_bytes_per_step": cap_algo, "traffic_over_algorithmic": traffic / cap_algo}
    if cap_ and "smsp__inst_executed.sum" in cap_:
        # instructions of the step: from the graph capture of these very steps when it has them, else the older range capture
        winst, isrc = cap_["smsp__inst_executed.sum"], RANGE_CAPTURE
        if trec and trec.get("warp_instructions_per_step"):
            winst, isrc = trec["warp_instructions_per_step"], trec["file"]
        ipp = winst * 32.0 / pxss_step                                       # issue slots (thread-instructions) per pixel-substep
        roofline["capture"] = {"file": RANGE_CAPTURE, "steps": RANGE_STEPS, "schedule": "serialised by ncu",
                               "csrc_sha": RANGE_CSRC_SHA, "stale": RANGE_CSRC_SHA != csrc_sha(),
                               "warp_instructions_per_step": cap_["smsp__inst_executed.sum"],
                               "dram_bytes_per_step": cap_.get("dram__bytes_read.sum", 0.0) + cap_.get("dram__bytes_write.sum", 0.0),
                               "l2_red_sectors_per_step": cap_.get("lts__t_sectors_op_red.sum")}
        roofline["issue_roof"] = {"bound": "alu", "unit": "thread-instr/s", "peak": ISSUE_PEAK, "derived_from": isrc,
                                  "instr_per_pixel_substep": ipp, "achieved": ipp * pxss_step / step_s,
                                  "frac": ipp * pxss_step / step_s / ISSUE_PEAK,
                                  "note": "utilisation of issue slots by the kernels' own instruction stream; against "
                                          "SURVEY.md 8(d)'s algorithmic estimate of 60 / 150 instructions per pixel-substep "
                                          "the throughput is the fractions below",
                                  "frac_vs_survey_bounds": [n * pxss_step / step_s / ISSUE_PEAK for n in SURVEY_INSTR_BOUNDS]}

    out = {"metric": METRIC, "value": value, "unit": METRIC, "n_gpus": world, "steps": K, "warmup": Wm,
           "ms_per_step": ms / K, "higher_is_better": True, "scaling": args.scaling if world > 1 else "weak", "vs_baseline": None,
           "dtype": "f32", "data": "synthetic",
           "config": dict(workload_config(spec, path_used), **({"defocus_sigma": args.defocus} if args.defocus is not None else {}),
                          **({"composite_mode": args.composite_mode} if args.composite_mode else {}),
                          **({"time_sorted": True} if args.time_sorted else {})),
           "events_per_s": events / (ms * 1e-3), "events_per_step": ev_per_step,
           "x_realtime": spec.keyframe_dt / (ms / K * 1e-3),
           "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline}

    # ---- e2e: HOST buffers through evis_step_host; every step uploads its keyframe from pinned memory and downloads its
    #      result into pinned memory.  `e2e` = the hot path's product, the ordered event stream (8-byte compact events, inside
    #      north_star's stamp tolerance); `e2e_events16` = the same stream as 16-byte events; `e2e_voxels` = the per-polarity
    #      accumulation image (no event leaves the GPU).  Upload of keyframe k + 1, kernels of step k and download of step
    #      k - 1 run concurrently (two staging sets, doubled ordered stream, deferred read).
    if not args.no_e2e and not args.profile_range:
        Ke = max(1, min(args.e2e_steps, K))
        hk = []
        for k in range(Wm + 1 + Ke):
            hk.append({a: b.cpu().pin_memory() for a, b in kfs[k].items()})
        del kfs
        torch.cuda.empty_cache()
        h2d = int(E * H * W * 32)

        def e2e_arm(voxels: bool, compact: bool = False):
            ev = mk()
            esize = 8 if compact else 16
            if voxels:
                ev.set_voxels(1, window_steps=1, keep_events=False)
                nel = int(np.prod(ev.voxel_shape()))
                hbufs = [torch.empty(nel, dtype=torch.float32).pin_memory() for _ in range(2)]
                harrs = [hb.numpy() for hb in hbufs]
            else:
                if compact:
                    ev.set_compact_events(True)
                hcap = int(min(cap, 2 * ev_per_step + (1 << 20)))
                hbufs = [torch.empty(hcap * esize, dtype=torch.uint8).pin_memory() for _ in range(2)]
                harrs = [hb.numpy().view(np.uint64 if compact else binding.EVENT_DTYPE) for hb in hbufs]
            for k in range(Wm + 1):
                f = hk[k]
                ev.step_host(f["rad"], f["mv_bwd"], f["depth"], f["mv_fwd"])
            barrier()
            tt0 = time.perf_counter()
            got, pending, n_last = 0, False, 0
            first = Wm + 1
            for k in range(first, first + Ke):
                f = hk[k]
                # enqueue only: this keyframe's upload starts while the previous step still computes
                ev.step_host(f["rad"], f["mv_bwd"], f["depth"], f["mv_fwd"], sync=False)
                if voxels:
                    ev.read_voxels_begin(harrs[k & 1])             # ends the previous copy first
                    got += harrs[0].nbytes
                elif k > first:
                    if pending:                                    # the stream of step k - 2 has arrived
                        got += esize * ev.read_events_finish()
                    # step k is enqueued: wait for step k - 1 alone and start copying its stream
                    ev.read_events_enqueue(harrs[(k - 1) & 1], previous_step=True)
                    pending = True
            if voxels:
                ev.read_voxels_end()
            else:
                if pending:
                    got += esize * ev.read_events_finish()
                ev.read_events_enqueue(harrs[(first + Ke - 1) & 1])   # the last step of the timed region
                n_last = ev.read_events_finish()
                got += esize * n_last
            barrier()
            dt = time.perf_counter() - tt0
            # (outside the timed region) the last result really arrived
            if voxels:
                total = float(harrs[(Wm + Ke) & 1].sum(dtype=np.float64))             # one unit per event
                if abs(total - ev.info().last_events) > 0.5:
                    raise SystemExit("bench.py: the downloaded accumulation image does not hold the step's events")
            else:
                last = harrs[(Wm + Ke) & 1][:n_last]
                envs = ((last >> np.uint64(24)) & np.uint64(0xFFFF)) if compact else last["env"]
                if n_last != ev.info().last_events or n_last >= hcap or int(envs.max()) != E - 1 or np.any(np.diff(envs.astype(np.int64)) < 0):
                    raise SystemExit("bench.py: the downloaded event stream is not the step's ordered stream")
            ev.destroy()
            (dt,), _ = sharding.reduce_max_sum([dt], [], dev)
            return {"value": global_envs * H * W * S * Ke / dt, "unit": METRIC, "steps": Ke,
                    "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": int(got / Ke), "ms_per_step": dt / Ke * 1e3,
                    "x_realtime": spec.keyframe_dt / (dt / Ke)}

        ev_api = ("evis_step_host with n_events = NULL (pinned host keyframes; the upload of keyframe k + 1 overlaps step k) + "
                  "evis_read_events_enqueue(previous_step) / _finish (pinned host stream: the stream of step k - 1 is copied out "
                  "after step k has been enqueued, waiting for step k - 1 only)")
        out["e2e"] = dict(e2e_arm(False, compact=True), result="the full ordered event stream (env, x, y, substep, polarity exact; the "
                          "stamp within T/S * 2^-16 = 1.6e-8 s, inside north_star's 1e-7 s) as 8-byte compact events "
                          "(evis_set_compact_events)", api=ev_api)
        out["e2e_events16"] = dict(e2e_arm(False), result="the full ordered event stream, 16 B per event (binary32 stamps)", api=ev_api)
        out["e2e_voxels"] = dict(e2e_arm(True), result="per-polarity accumulation image of the step [E,2,1,H,W] float32 "
                                 "(evis_set_voxels bins=1, keep_events=0)",
                                 api="evis_step_host with n_events = NULL + evis_read_voxels_begin / _end (pinned host image, "
                                     "overlapping the next upload)")

    if rank == 0 and not args.no_cpu and not args.profile_range:
        out["cpu_baseline"] = cpu_baseline(scenes.small(spec, seed=spec.seed - 1000 * rank), args.cpu_seconds)
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def run_sweep(args) -> None:
    """BASELINE.json configs[4]: throughput at (roughly) fixed total pixels over envs x resolution x S, analytic
    rectangle scenes as config 1.  One JSON line per point: pixel-substeps/s, events/s, fraction of the HBM
    roofline (algorithmic bytes of the point / time / measured copy peak).  Single GPU, device-resident inputs."""
    import torch
    from paper_2607_08098_b200 import binding, scenes
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback for the product path)")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    binding.load()
    peak, peak_src = hbm_peak()
    K, Wm = args.steps, args.warmup
    for spec in scenes.sweep_points():
        E, H, W, S = spec.num_envs, spec.height, spec.width, spec.substeps
        sc = scenes.make_scene(spec)
        kfs = [scenes.render_keyframe(sc, k, device=dev) for k in range(Wm + K + 1)]
        ev = binding.Evis(E, H, W, S, spec.c_pos, spec.c_neg, spec.log_eps, spec.keyframe_dt,
                          max_motion_px=spec.max_motion_px(), path=binding.PATH_AUTO, device=0,
                          event_capacity=int(min(0x7FFFFFFF, max(1 << 22, 10 * E * H * W))))
        stream = torch.cuda.current_stream(dev)
        for k in range(Wm + 1):
            f = kfs[k]
            ev.step(f["rad"], f["mv_bwd"], f["depth"], mv_fwd=f["mv_fwd"], stream=stream)
        torch.cuda.synchronize(dev)
        i0 = ev.info()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for k in range(Wm + 1, Wm + 1 + K):
            f = kfs[k]
            ev.step(f["rad"], f["mv_bwd"], f["depth"], mv_fwd=f["mv_fwd"], stream=stream)
        ev.wait_events(stream)
        e1.record(stream)
        torch.cuda.synchronize(dev)
        ms = e0.elapsed_time(e1)
        i1 = ev.info()
        if i1.overflow_steps != i0.overflow_steps:
            raise SystemExit("bench.py: event capacity overflow in the sweep")
        events = i1.total_events - i0.total_events
        ev.destroy()
        del kfs
        torch.cuda.empty_cache()
        algo = (ALGO_BYTES_PER_PIXEL * E * H * W) * K + ALGO_BYTES_PER_EVENT * events
        print(json.dumps({"metric": METRIC, "workload": spec.name, "envs": E, "height": H, "width": W, "substeps": S,
                          "value": E * H * W * S * K / (ms * 1e-3), "unit": METRIC, "events_per_s": events / (ms * 1e-3),
                          "ms_per_step": ms / K, "steps": K, "warmup": Wm,
                          "hbm_roofline_frac": algo / (ms * 1e-3) / 1e9 / peak, "hbm_peak_gbs": peak,
                          "x_realtime": spec.keyframe_dt / (ms / K * 1e-3)}), flush=True)


def main():
    args = parse_args()
    from paper_2607_08098_b200 import scenes
    if args.sweep:
        run_sweep(args)
        return
    spec = scenes.config(args.config)
    if args.envs:
        spec = scenes.small(spec, num_envs=args.envs, name=f"{spec.name}_E{args.envs}")
    if args.impl == "reference":
        run_reference(args, spec)
    else:
        run_ours(args, spec)


if __name__ == "__main__":
    main()

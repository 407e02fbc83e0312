#!/usr/bin/env python
"""bench.py — AVM hot-path throughput on B200 (contract: see DESIGN.md §Measurement).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

A "step" is one AVM timestep (all rows of the hot path) of one synthetic Voronoi tiling.
value = vertex-updates/s = V * K / (device time of K steps), whole job over all ranks (multi-GPU =
independent replicas, weak scaling, no collective on the data path).  Prints ONE JSON line.

Besides the `--steps/--warmup` region (`value`, exactly as asked), the line carries `whole_run` and
`second_half`: the config's nominal run (1000 steps for cfg3) timed from its
initial state in two halves, because a Voronoi start opens with a burst of T1 transitions that
decays over ~100 steps and the steady state is what a long run pays for.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "AVM vertex-updates/s (= V x timesteps/s) at N cells"
UNIT = "vertex-updates/s"
NOMINAL_PEAK_GBS = 8000.0     # north_star: "B200 peak (about 8 TB/s)"

# Algorithmic (compulsory, useful) bytes of the two dense kernels, DESIGN.md §5:
#   force_move : per vertex  pos 16 + vertexNeighbors 12 + vertexCellNeighbors 12 + pos_next 16,
#                plus the cell records gathered once per cell: 32 B/cell = 16 B/vertex      -> 72 B/vertex
#   cell_update: per cell    cellVertexNum 4 + tag 4 + theta 8+8 + record write 32 + row entries 4*6
#                + positions gathered once per vertex 16 B/vertex = 32 B/cell             -> 112 B/cell
# SURVEY.md §8(d)'s reference model of the same step: 134 B/vertex-step as stored.
BYTES_FORCE_MOVE_PER_VERTEX = 72.0
BYTES_CELL_UPDATE_PER_CELL = 112.0
SURVEY_BYTES_PER_VERTEX_STEP = 134.0
# --precision mixed (libavm_b200_mixed.so, NEXT-3; never the headline): positions 8 B, records 16 B
#   force_move : pos 8 + 12 + 12 + pos_next 8 + records 16 B/cell = 8 B/vertex  -> 48 B/vertex
#   cell_update: 4 + 4 + theta 8+8 + record write 16 + rows 24 + positions 2 x 8 -> 80 B/cell
BYTES_MIXED = (48.0, 80.0)


def workload_string(cfg, N, V):
    return (f"{cfg['name']}: AVM N={N} cells, V={V}, L={cfg['L'] * (N / cfg['N']) ** 0.5:g}, periodic Voronoi of uniform points "
            f"(seed {cfg['points_seed']}), p0={cfg['p0']}, v0={cfg['v0']}, Dr={cfg['Dr']}, dt={cfg['dt']}, "
            f"l_c={cfg['l_c']}, Hilbert-sorted at create={cfg['sort_at_create']}, sort_every={cfg['sort_every']}")


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the GPU works."""

    def __init__(self, index: int):
        self.ok = False
        try:
            import pynvml
            self.nv = pynvml
            pynvml.nvmlInit()
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.ok = True
        except Exception:
            self.nv = None
        self.sm, self.reasons, self.sm_max = [], set(), None

    def sample(self):
        if not self.ok:
            return
        nv = self.nv
        try:
            self.sm.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
            if self.sm_max is None:
                self.sm_max = nv.nvmlDeviceGetMaxClockInfo(self.h, nv.NVML_CLOCK_SM)
            r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h) if hasattr(nv, "nvmlDeviceGetCurrentClocksEventReasons") \
                else nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
            names = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
                     0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
                     0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}
            for bit, name in names.items():
                if r & bit and name != "gpu_idle":
                    self.reasons.add(name)
        except Exception:
            pass

    def start(self, period_s: float = 0.0005):
        """sample from a background thread while the caller enqueues and waits (ctypes releases the GIL)"""
        import threading
        self._stop = threading.Event()

        def loop():
            while not self._stop.is_set():
                self.sample()
                self._stop.wait(period_s)
        self._thread = threading.Thread(target=loop, daemon=True)
        self._thread.start()

    def stop(self):
        self._stop.set()
        self._thread.join()

    def summary(self):
        if not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": sorted(self.reasons), "samples": 0}
        return {"sm_mhz": float(np.median(self.sm)), "sm_max_mhz": self.sm_max, "reasons": sorted(self.reasons),
                "samples": len(self.sm)}


def ncu_capture(kernel: str, workload: str):
    """ncu figures of `kernel` from the committed capture (profiles/r2_ncu_kernels.csv; the commands, the
    commit and the step range of each capture are in profiles/r2_ncu_kernels.md): DRAM bytes per
    launch (dram__bytes_read.sum + dram__bytes_write.sum) and pipe utilisations.  Static evidence
    read from a file, not measured in this run; the record says which capture it is."""
    path = os.path.join(ROOT, "profiles", "r2_ncu_kernels.csv")
    try:
        import csv
        for row in csv.DictReader(open(path)):
            if row["kernel"] == kernel and row["workload"] == workload:
                return row
    except Exception:
        pass
    return None


def max_over_ranks(ms: float, dist, device: str) -> float:
    """Replicas only: ranks share nothing but the clock.  The job's time is the
    slowest rank's device time; this all-reduce of one scalar is the only collective in bench.py
    (never on the data path).  `dist` is torch.distributed or None (single process)."""
    if dist is None:
        return float(ms)
    import torch
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(units_per_rank: float, steps: int, ms: float, world: int) -> float:
    """whole-job throughput: every rank advances its own replica of the workload (weak scaling)"""
    return world * units_per_rank * steps / (ms * 1e-3)


def bandwidth_fractions(bytes_per_step: float, ms_per_step: float, peak: float) -> dict:
    gbs = bytes_per_step / (ms_per_step * 1e-3) / 1e9
    return {"GBps": gbs, "frac_of_measured_peak": gbs / peak, "frac_of_nominal_8TBps": gbs / NOMINAL_PEAK_GBS}


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, rank 0 only.  The full tiling of the config is
    used whenever K+W steps of it end within the time budget; otherwise a smaller tiling of the same
    recipe and density, and config.workload says which N really ran."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    from paper_1702_02939_b200 import workloads as w
    cfg = w.CONFIGS[args.config]
    p = w.config_params(args.config)
    total = max(1, args.steps + args.warmup)
    budget_cells = 150.0 / (total * 1.5e-6)              # ~1.5 us per cell-step on one core, ~150 s in all
    Ns = cfg["N"]
    while Ns > 1024 and Ns > budget_cells:
        Ns //= 4
    Ls = cfg["L"] * (Ns / cfg["N"]) ** 0.5
    t = w.voronoi_tiling(Ns, Ls, cfg["points_seed"])
    sim = oracle.from_tiling(t, **dict(p, Lx=Ls, Ly=Ls))
    sim.step(args.warmup)
    t0 = time.perf_counter()
    sim.step(args.steps)
    dt = time.perf_counter() - t0
    value = t.V * args.steps / dt
    sample = (f"the oracle (oracle/avm_oracle.cpp, one thread) on {'the full' if Ns == cfg['N'] else 'a reduced'} {Ns}-cell tiling "
              f"of the {cfg['name']} recipe, steps {args.warmup}..{args.warmup + args.steps - 1}")
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(1, args.steps),
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": workload_string(cfg, Ns, t.V), "cells_run": Ns, "cells_of_config": cfg["N"]},
           "timesteps_per_s": args.steps / dt,
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                            "host_cpus": os.cpu_count()},
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=100)
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json configs index (default 3: N=1,048,576)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (kernel experiments only)")
    ap.add_argument("--no-nominal-run", action="store_true", help="skip the whole_run / second_half records")
    ap.add_argument("--no-cfg4", action="store_true",
                    help="skip the cfg4 sub-record (N = 4,194,304: the config's own 500-step run, added to the default cfg3 line)")
    ap.add_argument("--profile-steps", type=int, default=0,
                    help="steps of the per-kernel event pass (default: the timed region itself, at most 200 steps)")
    ap.add_argument("--t1-passes", type=int, default=1,
                    help="T1 passes per step: 1 = north_star's rule (default, the headline), P > 1 = repeat until none (NEXT-1)")
    ap.add_argument("--schedule", default="auto", choices=["auto", "fused", "unfused", "persistent"])
    ap.add_argument("--precision", default="f64", choices=["f64", "mixed"],
                    help="f64 = the default library and the headline; mixed = libavm_b200_mixed.so (reduced-precision storage, NEXT-3)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)

    if args.impl == "reference":
        run_reference(args)
        return

    import torch
    from paper_1702_02939_b200 import workloads as w
    from paper_1702_02939_b200 import binding as B   # raises if libavm_b200.so is missing: no fallback

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device"
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = w.CONFIGS[args.config]
    p = dict(w.config_params(args.config), device=local_rank, schedule=args.schedule, precision=args.precision)
    if args.t1_passes > 1:
        p["t1_max_passes"] = args.t1_passes
    t = w.config_tiling(args.config)
    N, V = t.N, t.V
    peak, peak_src = measured_peaks()
    kbytes = {"force_move": BYTES_FORCE_MOVE_PER_VERTEX * V, "cell_update": BYTES_CELL_UPDATE_PER_CELL * N}
    if args.precision == "mixed":
        kbytes = {"force_move": BYTES_MIXED[0] * V, "cell_update": BYTES_MIXED[1] * N}
    step_bytes = sum(kbytes.values())
    survey_step_bytes = SURVEY_BYTES_PER_VERTEX_STEP * V

    def timed_steps(sim, n):
        """device time of n steps (CUDA events on the stream the library launches on), clocks sampled meanwhile"""
        sampler = ClockSampler(local_rank)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        sampler.start()
        e0.record()
        sim.step(n)
        e1.record()
        e1.synchronize()
        sampler.stop()
        barrier()
        return max_over_ranks(e0.elapsed_time(e1), dist, "cuda"), sampler

    def region_record(ms, n, first_step, st0, st1, sampler, n_vertices=None):
        per = ms / n
        nv = V if n_vertices is None else n_vertices
        scale = nv / V                                    # both byte models are per vertex
        return {"steps": f"{first_step}..{first_step + n - 1}", "ms_per_step": per,
                "value": aggregate_value(nv, n, ms, world), "unit": UNIT, "timesteps_per_s": n / (ms * 1e-3),
                "t1_flips_per_step": (st1["t1_flips"] - st0["t1_flips"]) / n,
                "bandwidth": {"bytes_model_this_repo_128B_per_vertex": bandwidth_fractions(step_bytes * scale, per, peak),
                              "bytes_model_survey_134B_per_vertex": bandwidth_fractions(survey_step_bytes * scale, per, peak)},
                "clocks": sampler.summary()}

    def nominal_run(tq, pq, nominal):
        """the config's own run from its initial state, timed in two halves (re-sorts included)"""
        simn = B.from_tiling(tq, **pq)
        s0 = simn.stats()
        h1 = nominal // 2
        ms1, smp1 = timed_steps(simn, h1)
        s1 = simn.stats()
        ms2, smp2 = timed_steps(simn, nominal - h1)
        s2 = simn.stats()
        smp_all = ClockSampler(local_rank)
        smp_all.sm, smp_all.reasons, smp_all.sm_max = smp1.sm + smp2.sm, smp1.reasons | smp2.reasons, smp1.sm_max
        whole = region_record(ms1 + ms2, nominal, 0, s0, s2, smp_all, tq.V)
        whole["includes_resorts"] = s2["n_sorts"] - s0["n_sorts"]
        second = region_record(ms2, nominal - h1, h1, s1, s2, smp2, tq.V)
        return simn, whole, second

    # ---------------- device-resident run: inputs already in HBM when the clock starts -----------
    sim = B.from_tiling(t, **p)
    sim.step(args.warmup)
    st0 = sim.stats()
    ms, sampler = timed_steps(sim, args.steps)
    st1 = sim.stats()
    value = aggregate_value(V, args.steps, ms, world)
    state_after = st1
    sim.close()
    del sim

    # ---------------- per-kernel device time over the SAME steps (CUDA events inside the library) -
    # A fresh simulation repeats the warm-up (the run is deterministic), then avm_step_profile
    # brackets every kernel of the timed steps with events; clocks are sampled during this pass too.
    prof_steps = args.profile_steps if args.profile_steps > 0 else min(args.steps, 200)
    simp = B.from_tiling(t, **p)
    simp.step(args.warmup)
    psampler = ClockSampler(local_rank)
    torch.cuda.synchronize()
    psampler.start()
    prof = simp.step_profile(prof_steps)
    torch.cuda.synchronize()
    psampler.stop()
    simp.close()
    del simp
    per_launch_ms = {k: v / max(1, prof_steps) for k, v in prof.items()}
    # fewer than two launches per step = the library stepped launch-free (its default up to 8192 vertices)
    timed_persistent = (st1["kernel_launches"] - st0["kernel_launches"]) < 2 * args.steps
    dom = max(kbytes, key=lambda k: per_launch_ms[k])
    ach = kbytes[dom] / (per_launch_ms[dom] * 1e-3) / 1e9
    cap = ncu_capture(dom, cfg["name"] + ("_steady" if args.warmup >= 300 else "")) if args.precision == "f64" else None
    traffic = (float(cap["dram_bytes_read_per_launch"]) + float(cap["dram_bytes_write_per_launch"])) if cap else None
    roofline = {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "frac_of_nominal_8TBps": ach / NOMINAL_PEAK_GBS,
                "traffic": traffic,
                "traffic_source": (f"ncu capture {cap['capture']} (commit {cap['commit']}, steps {cap['steps']}; profiles/r2_ncu_kernels.md), "
                                   "not measured in this run") if cap else None,
                "ncu": {k: cap[k] for k in cap if k not in ("kernel", "workload")} if cap else None,
                "peak_source": peak_src,
                "timing": f"CUDA events on the library's stream around every launch of steps {args.warmup}..{args.warmup + prof_steps - 1} "
                          "of a second, identical run; the events serialise the launches; " + (
                              "LAUNCHED schedule (one launch per kernel): the timed region ran the launch-free persistent kernel, "
                              "which avm_step_profile cannot bracket, so these per-kernel times describe a different schedule"
                              if timed_persistent else "same schedule decisions as the timed region"),
                "timed_region_schedule": "persistent (launch-free)" if timed_persistent else "one launch per kernel",
                "bytes_per_launch": kbytes[dom], "ms_per_launch": per_launch_ms[dom],
                "kernels_ms_per_launch": per_launch_ms,
                "kernels_frac_of_measured_peak": {k: kbytes[k] / (per_launch_ms[k] * 1e-3) / 1e9 / peak for k in kbytes if per_launch_ms[k] > 0},
                "clocks_during_profile_pass": psampler.summary(),
                "step": {"algorithmic_bytes": step_bytes, **bandwidth_fractions(step_bytes, ms / args.steps, peak),
                         "survey_134B_model": bandwidth_fractions(survey_step_bytes, ms / args.steps, peak)}}
    roofline["step"]["frac"] = roofline["step"]["frac_of_measured_peak"]
    roofline["step"]["achieved_GBps"] = roofline["step"]["GBps"]

    # ---------------- the config's nominal run from its initial state, in two halves --------------
    whole_run = second_half = None
    if not args.no_nominal_run:
        nominal = cfg["steps"] if cfg["steps"] <= 2000 else 2000     # cfg1/cfg2 name 10^4 steps: the first 2000 are timed
        simn, whole_run, second_half = nominal_run(t, p, nominal)
        simn.close()
        del simn

    # ---------------- cfg4 (N = 4,194,304, T1-heavy, re-sort every 100 steps) beside the default cfg3 line -------
    # The largest single-GPU config has no line of its own in a default run: its own 500-step run in two
    # halves, then the per-kernel event pass over the next 40 steps of the same simulation.  GPU only, no oracle leg.
    cfg4 = None
    if args.config == 3 and world == 1 and args.precision == "f64" and args.t1_passes == 1 and not (args.no_cfg4 or args.no_nominal_run):
        c4 = w.CONFIGS[4]
        t4 = w.config_tiling(4)
        p4 = dict(w.config_params(4), device=local_rank, schedule=args.schedule, precision=args.precision)
        sim4, whole4, second4 = nominal_run(t4, p4, c4["steps"])
        smp4 = ClockSampler(local_rank)
        torch.cuda.synchronize()
        smp4.start()
        prof4 = sim4.step_profile(40)
        torch.cuda.synchronize()
        smp4.stop()
        err4 = sim4.stats()["error"]
        sim4.close()
        del sim4
        kb4 = {"force_move": BYTES_FORCE_MOVE_PER_VERTEX * t4.V, "cell_update": BYTES_CELL_UPDATE_PER_CELL * t4.N}
        per4 = {k: v / 40 for k, v in prof4.items()}
        cfg4 = {"workload": workload_string(c4, t4.N, t4.V), "whole_run": whole4, "second_half": second4,
                "kernels_ms_per_launch": per4,
                "kernels_frac_of_measured_peak": {k: kb4[k] / (per4[k] * 1e-3) / 1e9 / peak for k in kb4 if per4[k] > 0},
                "kernels_timing": f"CUDA events around every launch of steps {c4['steps']}..{c4['steps'] + 39} of the same simulation (serialised launches)",
                "clocks_during_profile_pass": smp4.summary(), "error_word": err4}
        del t4

    # ---------------- end to end through the host-pointer entry points --------------------------
    # One job = avm_create_host (H2D of the whole state from pinned memory) + K steps +
    # avm_get_state_host (D2H of the whole state into pinned memory), all inside the timed region.
    e2e = None
    if not args.no_e2e:
        pinned = {}
        for name in ("pos", "cell_vertex_num", "cell_vertices", "vertex_neighbors", "vertex_cell_neighbors", "theta"):
            a = np.ascontiguousarray(getattr(t, name))
            tp = torch.from_numpy(a.copy()).pin_memory()
            pinned[name] = tp.numpy()
        tin = w.Tiling(t.Lx, t.Ly, t.S, pinned["pos"], pinned["cell_vertex_num"], pinned["cell_vertices"],
                       pinned["vertex_neighbors"], pinned["vertex_cell_neighbors"], pinned["theta"])
        out = {k: torch.empty(v.shape, dtype=torch.from_numpy(v).dtype).pin_memory().numpy() for k, v in pinned.items()}
        h2d = sum(v.nbytes for v in pinned.values())
        d2h = sum(v.nbytes for v in out.values())
        e2e_ms = []
        for rep in range(2):                      # first repetition warms allocator and page locks
            barrier()
            t0 = time.perf_counter()
            s2 = B.from_tiling(tin, host=True, **p)
            s2.step(args.steps)
            s2.get_state_host(out)
            torch.cuda.synchronize()
            e2e_ms.append((time.perf_counter() - t0) * 1e3)
            s2.close()
            del s2
        e2e_t = e2e_ms[-1]
        e2e_t = max_over_ranks(e2e_t, dist, "cuda")
        e2e = {"value": aggregate_value(V, args.steps, e2e_t, world), "unit": UNIT,
               "h2d_bytes_per_step": h2d / args.steps, "d2h_bytes_per_step": d2h / args.steps,
               "job": "avm_create_host + avm_step(K) + avm_get_state_host, pinned host buffers", "ms": e2e_t}

    # ---------------- CPU baseline: the oracle as it stands, one core, bounded sample ------------
    # BASELINE.md §3 / SURVEY §8(d): time >= 20 consecutive steps AFTER the initial burst (the oracle's
    # own first 50 steps) for the large configs.  A million-cell step takes the oracle ~0.7 s, so the
    # sample is sized to ~25 s of timed work plus the untimed skip.
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        o = oracle.from_tiling(t, **{a: b for a, b in p.items() if a not in ("precision", "schedule", "device")})
        est = 0.7e-6 * N                                       # s per step, one core
        n_o = max(20, min(400, int(15.0 / est)))
        skip = 50 if est * 50 < 60.0 else max(0, int(60.0 / est))   # cfg4: the skip itself is capped at ~60 s
        o.step(skip)
        t0 = time.perf_counter()
        o.step(n_o)
        dt = time.perf_counter() - t0
        cpu = {"value": V * n_o / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"steps {skip}..{skip + n_o - 1} of the same {cfg['name']} tiling ({N} cells), after the oracle's own first {skip} steps",
               "timesteps_per_s": n_o / dt, "host_cpus": os.cpu_count()}

    if rank == 0:
        steps_timed = st1["step"] - st0["step"]
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64" if args.precision == "f64" else "f64 arithmetic on fixed-point-32 positions and f32 cell records",
            "data": "synthetic",
            "config": {"workload": workload_string(cfg, N, V), "precision": args.precision,
                       "parallelism": "replicas only" if world > 1 else "1 GPU",
                       "t1_passes_per_step": args.t1_passes, "schedule": args.schedule,
                       "l2": f"inputs larger than L2: resident state {224 * N / 1e6:.0f} MB vs 126 MB L2" if 224 * N > 126e6
                             else "state fits in L2 (latency/launch bound config); no flush",
                       "timed_region": f"steps {st0['step']}..{st1['step'] - 1} after {args.warmup} warm-up steps"},
            "timesteps_per_s": args.steps / (ms * 1e-3),
            "gpu_launches": st1["kernel_launches"] - st0["kernel_launches"],
            "t1": {"flips_in_timed_region": st1["t1_flips"] - st0["t1_flips"],
                   "candidates": st1["t1_candidates"] - st0["t1_candidates"],
                   "blocked": st1["t1_blocked"] - st0["t1_blocked"], "steps": steps_timed,
                   "error_word": state_after["error"]},
            "clocks": sampler.summary(),
            # an NVML sample takes about a millisecond, so a 1.5 ms region (--steps 20) holds one; the config's nominal
            # run in the same process (whole_run below) is sampled the same way and holds hundreds
            "clocks_nominal_run": whole_run["clocks"] if whole_run else None,
            "roofline": roofline,
            "whole_run": whole_run,
            "second_half": second_half,
            "e2e": e2e,
            "cpu_baseline": cpu,
            "cfg4": cfg4,
        }
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

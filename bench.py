#!/usr/bin/env python
"""bench.py — AVM hot-path throughput on B200 (contract: see DESIGN.md §Measurement).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

A "step" is one AVM timestep (all rows of the hot path) of one synthetic Voronoi tiling.
value = vertex-updates/s = V * K / (device time of K steps), whole job over all ranks (multi-GPU =
independent replicas, weak scaling, no collective on the data path).  Prints ONE JSON line.
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

# Algorithmic (compulsory, useful) bytes of the two dense kernels, DESIGN.md §Byte model:
#   force_move : per vertex  pos 16 + vertexNeighbors 12 + vertexCellNeighbors 12 + pos_next 16,
#                plus the cell records gathered once per cell: 32 B/cell = 16 B/vertex      -> 72 B/vertex
#   cell_update: per cell    cellVertexNum 4 + tag 4 + theta 8+8 + record write 32 + row entries 4*6
#                + positions gathered once per vertex 16 B/vertex = 32 B/cell             -> 112 B/cell
BYTES_FORCE_MOVE_PER_VERTEX = 72.0
BYTES_CELL_UPDATE_PER_CELL = 112.0


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

    def start(self, period_s: float = 0.004):
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


def ncu_traffic(kernel: str, workload: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel`, from the committed ncu
    capture (profiles/r1_v4_dram_traffic.csv; the command is in profiles/r1_v4_two_launch.md)."""
    path = os.path.join(ROOT, "profiles", "r1_v4_dram_traffic.csv")
    try:
        import csv
        for row in csv.DictReader(open(path)):
            if row["kernel"] == kernel and row["workload"] == workload:
                return float(row["dram_bytes_read_per_launch"]) + float(row["dram_bytes_write_per_launch"])
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


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, rank 0 only, on a bounded sample of the
    workload (a smaller tiling of the same recipe and density) so that K+W steps end in minutes."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    from paper_1702_02939_b200 import workloads as w
    cfg = w.CONFIGS[args.config]
    p = w.config_params(args.config)
    total = max(1, args.steps + args.warmup)
    budget_cells = 100.0 / (total * 1.5e-6)              # ~1.5 us per cell-step on one core
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
    sample = f"{Ns}-cell tiling of the {cfg['name']} recipe (same density, parameters, seed), {args.steps} steps after {args.warmup}"
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(1, args.steps),
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": f"{cfg['name']}: AVM N={cfg['N']} cells, L={cfg['L']}, Voronoi seed {cfg['points_seed']}",
                      "sample": sample},
           "timesteps_per_s": args.steps / dt,
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
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
    ap.add_argument("--profile-steps", type=int, default=100)
    ap.add_argument("--t1-passes", type=int, default=1,
                    help="T1 passes per step: 1 = north_star's rule (default, the headline), P > 1 = repeat until none (NEXT-1)")
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
    p = dict(w.config_params(args.config), device=local_rank)
    if args.t1_passes > 1:
        p["t1_max_passes"] = args.t1_passes
    t = w.config_tiling(args.config)
    N, V = t.N, t.V

    # ---------------- device-resident run: inputs already in HBM when the clock starts -----------
    sim = B.from_tiling(t, **p)
    sim.step(args.warmup)
    st0 = sim.stats()
    sampler = ClockSampler(local_rank)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler.start()
    e0.record()
    sim.step(args.steps)
    e1.record()
    e1.synchronize()
    sampler.stop()
    barrier()
    ms = e0.elapsed_time(e1)
    st1 = sim.stats()
    ms = max_over_ranks(ms, dist, "cuda")
    value = aggregate_value(V, args.steps, ms, world)

    # ---------------- per-kernel device time (CUDA events inside the library) --------------------
    prof = sim.step_profile(args.profile_steps)
    peak, peak_src = measured_peaks()
    per_launch_ms = {k: v / max(1, args.profile_steps) for k, v in prof.items()}
    kbytes = {"force_move": BYTES_FORCE_MOVE_PER_VERTEX * V, "cell_update": BYTES_CELL_UPDATE_PER_CELL * N}
    dom = max(kbytes, key=lambda k: per_launch_ms[k])
    ach = kbytes[dom] / (per_launch_ms[dom] * 1e-3) / 1e9
    step_bytes = sum(kbytes.values())
    roofline = {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "traffic": ncu_traffic(dom, cfg["name"]), "peak_source": peak_src,
                "timing": "CUDA events on the library's stream around every launch of a separate pass of "
                          f"{args.profile_steps} steps (same schedule as the timed region, launches serialised by the events)",
                "bytes_per_launch": kbytes[dom], "ms_per_launch": per_launch_ms[dom],
                "kernels_ms_per_launch": per_launch_ms,
                "step": {"algorithmic_bytes": step_bytes, "achieved_GBps": step_bytes / (ms / args.steps * 1e-3) / 1e9,
                         "frac": step_bytes / (ms / args.steps * 1e-3) / 1e9 / peak}}
    state_after = sim.stats()
    sim.close()
    del sim

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
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        o = oracle.from_tiling(t, **p)
        n_o = max(2, min(200, int(15.0 / (1.5e-6 * N))))      # ~15 s of single-core work
        t0 = time.perf_counter()
        o.step(n_o)
        dt = time.perf_counter() - t0
        cpu = {"value": V * n_o / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"steps 0..{n_o - 1} of the same {cfg['name']} tiling from its initial state (inside the step-0 T1 burst)",
               "timesteps_per_s": n_o / dt, "host_cpus": os.cpu_count()}

    if rank == 0:
        steps_timed = st1["step"] - st0["step"]
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{cfg['name']}: AVM N={N} cells, V={V}, L={cfg['L']}, periodic Voronoi of uniform points "
                                   f"(seed {cfg['points_seed']}), p0={cfg['p0']}, v0={cfg['v0']}, Dr={cfg['Dr']}, dt={cfg['dt']}, "
                                   f"l_c={cfg['l_c']}, Hilbert-sorted at create={cfg['sort_at_create']}, sort_every={cfg['sort_every']}",
                       "parallelism": "replicas only" if world > 1 else "1 GPU",
                       "t1_passes_per_step": args.t1_passes,
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
            "roofline": roofline,
            "e2e": e2e,
            "cpu_baseline": cpu,
        }
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

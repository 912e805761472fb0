#!/usr/bin/env python
"""bench.py -- ANI-2x energy+force atom-evals/s on BASELINE.json configs[1] (50 atoms, 8 models).

A "step" is one pass of the whole hot path (neighbour pairs -> AEV -> ensemble MLPs -> backward ->
forces added into the force buffer) = one nnp_compute on the next frame of the seeded, perturbed
trajectory.  See DESIGN.md "Measurement" for what each JSON key means and how it is measured.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl reference]
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

from paper_2201_08110_b200 import workloads as wl  # noqa: E402

METRIC = "ANI-2x energy+force atom-evals/sec (50-atom, 8-model ligand; us/step and % of roofline in extra keys)"
UNIT = "atom-evals/s"
L2_FLUSH_BYTES = 256 << 20


def workload_config(w, extra=None):
    cfg = {
        "workload": f"BASELINE.json configs[{w.config - 1}]: {w.name}, {w.n_atoms} atoms, {w.n_molecules} molecule(s), "
                    f"{w.n_models}-model ANI-2x ensemble, perturbed trajectory N(0,0.005 A) per step",
        "n_atoms": w.n_atoms, "n_models": w.n_models, "n_molecules": w.n_molecules,
    }
    if extra:
        cfg.update(extra)
    return cfg


def ncu_traffic_bytes(config: int):
    """dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel, per launch, from the committed
    `ncu --set full` summary (profiles/top_kernel_traffic.txt, lines `config<C>_dram_bytes=<n>`); None if absent."""
    try:
        for line in open(os.path.join(ROOT, "profiles", "top_kernel_traffic.txt")):
            if line.startswith(f"config{config}_dram_bytes="):
                return float(line.split("=", 1)[1])
    except OSError:
        pass
    return None


# ------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks + throttle reasons sampled DURING the timed region."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.lines = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100", "-i",
                 str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------
def run_reference(args):
    """--impl reference: the float64 CPU oracle, as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from oracle.ani_oracle import AniOracle

    w = wl.get_config(args.config)
    W, B = w.weights()
    orc = AniOracle(w.params, W, B)
    n_frames = min(max(args.steps + args.warmup, 1), 1000)
    traj = w.trajectory(n_frames)
    for t in range(args.warmup):
        orc.energy_forces(traj[t % n_frames], w.species, w.mol_offsets)
    t0 = time.perf_counter()
    for t in range(args.steps):
        orc.energy_forces(traj[(args.warmup + t) % n_frames], w.species, w.mol_offsets)
    dt = time.perf_counter() - t0
    value = w.n_atoms * args.steps / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(w),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": orc.threads, "kind": "oracle",
                         "sample": f"{args.steps} full energy+force evaluations of the {w.n_atoms}-atom workload "
                                   f"(every step is the whole workload step)"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
def run_gpu(args):
    import torch

    from paper_2201_08110_b200.binding import NNP

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a GPU (there is no CPU fallback)"
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=dev)

    # every rank evaluates its own replica of the workload (independent molecules: no data-path
    # collective, weak scaling); rank r starts at a different frame of the trajectory
    w = wl.get_config(args.config)
    W, B = w.weights()
    nnp = NNP(w.params, W, B, w.species, w.mol_offsets, flags=args.flags)
    K, Wu = args.steps, args.warmup
    n_frames = min(K + Wu, 1000)
    traj_h = w.trajectory(n_frames)
    traj = torch.from_numpy(traj_h).to(dev)
    pos = traj[0].clone()  # the MD engine's position buffer: same pointer every step
    E = torch.zeros(w.n_molecules, dtype=torch.float64, device=dev)
    F = torch.zeros((w.n_atoms, 3), dtype=torch.float32, device=dev)
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()

    def frame(t):
        return (t + 17 * rank) % n_frames

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def step(t, timed_events=None):
        pos.copy_(traj[frame(t)])      # untimed: the integrator moved the atoms
        flush.zero_()                  # untimed: evict L2 (weights must come from HBM again)
        if timed_events is not None:
            timed_events[0].record(stream)
        nnp.compute_torch(pos, E, F)
        if timed_events is not None:
            timed_events[1].record(stream)

    for t in range(Wu):
        step(t)
    nnp.check()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    t_wall0 = time.perf_counter()
    for t in range(K):
        step(Wu + t, evs[t])
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop() if rank == 0 else None
    nnp.check()
    dev_ms = sum(a.elapsed_time(b) for a, b in evs)
    per_step_ms = sorted(a.elapsed_time(b) for a, b in evs)
    tmax = torch.tensor([dev_ms], dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    dev_ms_max = float(tmax.item())
    value = world * w.n_atoms * K / (dev_ms_max * 1e-3)

    # ---- warm-L2 variant (weights stay L2-resident between steps, as in a tight MD loop)
    warm_ms = None
    if rank == 0:
        for t in range(5):
            nnp.compute_torch(pos, E, F)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for t in range(K):
            nnp.compute_torch(pos, E, F)
        b.record(stream)
        torch.cuda.synchronize()
        warm_ms = a.elapsed_time(b) / K

    # ---- per-kernel stage times (CUDA events between stages, same flush discipline) -> roofline
    roofline = None
    stages = None
    if rank == 0:
        nnp.set_profiling(True)
        acc = {}
        n_prof = min(K, 50)
        for t in range(n_prof):
            step(Wu + t)
            for k, v in nnp.stage_times().items():
                acc[k] = acc.get(k, 0.0) + v
        nnp.set_profiling(False)
        stages = {k: 1e3 * v / n_prof for k, v in acc.items()}  # us
        top = max(stages, key=stages.get)
        work = nnp.work()
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except Exception:
            pass
        hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
        peak_src = "measured (MEASURED_PEAKS.json hbm_gbs)" if "hbm_gbs" in peaks else "fallback 6650 GB/s"
        # dominant kernel of this workload: the layer-1 GEMMs stream the layer-1 weights once per launch
        l1 = "mlp_fwd_l1"
        l1_bytes = work["layer1_weight_bytes"] + w.n_atoms * nnp.n_features * 4
        achieved = l1_bytes / (stages[l1] * 1e-6) / 1e9
        roofline = {"bound": "hbm", "kernel": "gemm_tma_kernel (" + l1 + ")", "achieved": achieved,
                    "peak": hbm_peak, "unit": "GB/s", "frac": achieved / hbm_peak,
                    "traffic": ncu_traffic_bytes(args.config),
                    "peak_source": peak_src, "algorithmic_bytes": l1_bytes, "kernel_us": stages[l1],
                    "top_stage": top}

    # ---- end-to-end through the C ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if True:
        hp = torch.from_numpy(traj_h).pin_memory()
        hE = torch.zeros(w.n_molecules, dtype=torch.float64).pin_memory()
        hF = torch.zeros((w.n_atoms, 3), dtype=torch.float32).pin_memory()
        sraw = stream.cuda_stream
        for t in range(3):
            nnp.compute_host_into(hp[frame(t)].data_ptr(), hE.data_ptr(), hF.data_ptr(), sraw)
        barrier()
        tot = 0.0
        for t in range(K):
            flush.zero_()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            nnp.compute_host_into(hp[frame(Wu + t)].data_ptr(), hE.data_ptr(), hF.data_ptr(), sraw)  # syncs
            tot += time.perf_counter() - t0
        tt = torch.tensor([tot], dtype=torch.float64, device=dev)
        if dist is not None:
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        e2e = {"value": world * w.n_atoms * K / float(tt.item()), "unit": UNIT,
               "h2d_bytes_per_step": w.n_atoms * 12, "d2h_bytes_per_step": w.n_atoms * 12 + w.n_molecules * 8,
               "us_per_step": 1e6 * float(tt.item()) / K}

    # ---- CPU baseline: the oracle as it stands, bounded sample, rank 0 at N=1 only
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle.ani_oracle import AniOracle

        orc = AniOracle(w.params, W, B)
        n_s = args.cpu_steps
        orc.energy_forces(traj_h[0], w.species, w.mol_offsets)
        t0 = time.perf_counter()
        for t in range(n_s):
            orc.energy_forces(traj_h[t % n_frames], w.species, w.mol_offsets)
        dt = time.perf_counter() - t0
        cpu = {"value": w.n_atoms * n_s / dt, "unit": UNIT, "cores": orc.threads, "kind": "oracle",
               "sample": f"first {n_s} frames of the same trajectory, full energy+force evaluation each, "
                         f"{1e3 * dt / n_s:.1f} ms/step"}

    launches = K * nnp.launches_per_compute
    nnp.destroy()
    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wu,
            "ms_per_step": dev_ms_max / K, "us_per_step": 1e3 * dev_ms_max / K,
            "us_per_step_median": 1e3 * per_step_ms[len(per_step_ms) // 2],
            "us_per_step_warm_l2": None if warm_ms is None else 1e3 * warm_ms,
            "wall_us_per_step_incl_flush": 1e6 * t_wall / K,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": workload_config(w, {"l2": f"flushed between timed steps ({L2_FLUSH_BYTES >> 20} MiB write, "
                                                "outside the per-step CUDA events)",
                                          "timing": "sum of per-step CUDA-event durations on the launch stream, "
                                                    "max over ranks", "parallelism": f"replicas x{world}"}),
            "e2e": e2e, "gpu_launches": launches, "clocks": clocks, "roofline": roofline,
            "stage_us": stages, "cpu_baseline": cpu,
        }
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config, 1-based (2 = the metric's)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--cpu-steps", type=int, default=200)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--flags", type=int, default=0, help="NNP_FLAG_* bits (include/nnp.h) for A/B runs of the engines")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()

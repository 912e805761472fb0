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

from paper_2201_08110_b200 import multi  # noqa: E402
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


def ncu_traffic_bytes(config: int, stage: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of a kernel, per launch, from the committed `ncu --set full`
    summaries (profiles/top_kernel_traffic.txt, lines `config<C>_<stage>_dram_bytes=<n>`); None if absent."""
    try:
        for line in open(os.path.join(ROOT, "profiles", "top_kernel_traffic.txt")):
            if line.startswith(f"config{config}_{stage}_dram_bytes="):
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
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "20", "-i",
                 str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.perf_counter(), line.strip()))

    def wait_first_sample(self, timeout=10.0):
        t0 = time.perf_counter()
        while self.proc is not None and not self.lines and time.perf_counter() - t0 < timeout:
            time.sleep(0.01)

    def stop(self, t_begin=None, t_end=None):
        """Summary of the samples taken in [t_begin, t_end] (perf_counter times); if the window is shorter than
        the sampling period, the samples of the whole loaded run are used and `window` says so."""
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        window = "timed region"
        lines = [ln for t, ln in self.lines if (t_begin is None or t >= t_begin) and (t_end is None or t <= t_end)]
        if not lines:
            window = "whole run under load (timed region shorter than the sampling period)"
            lines = [ln for _, ln in self.lines]
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in lines:
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
                "samples": len(sm), "window": window, "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------
KERNEL_OF_STAGE = {  # ligand-size engine / tensor-core engine
    "ligand": {"mlp_fwd_l1": "small_fwd1_kernel", "mlp_mid": "small_mid_kernel", "mlp_bwd_l1": "small_bwd1_kernel"},
    "tensor": {"mlp_fwd_l1": "gemm_umma_kernel", "mlp_fwd_l2": "gemm_umma_kernel", "mlp_fwd_l3": "gemm_umma_kernel",
               "mlp_bwd_l3": "gemm_umma_kernel", "mlp_bwd_l2": "gemm_umma_kernel", "mlp_bwd_l1": "gemm_umma_kernel"},
}


def stage_rooflines(w, nnp, stages, config):
    """Roofline of the dominant MLP kernel (and, under "kernels", of every MLP launch) from the live CUDA-event
    stage times.  Algorithmic work per launch: a layer GEMM does 2 flop per weight per
    atom-model; the ligand-size layer-1 forward must stream the layer-1 weights of the ensemble once (HBM-bound
    when L2 was flushed); FP32 peak = SMs x 128 lanes x 2 flop x max SM clock; TF32 tensor peak = measured bf16
    peak x 0.5 (nominal ratio), against which 3xTF32 can reach at most 1/3."""
    import torch

    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        peaks = {}
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    hbm_src = "measured (MEASURED_PEAKS.json hbm_gbs)" if "hbm_gbs" in peaks else "fallback 6650 GB/s (B200_PROFILING.md)"
    bf16 = float(peaks.get("bf16_tflops", 1650.0))
    sm_mhz = float(peaks.get("sm_max_mhz", 1965.0))
    n_sm = torch.cuda.get_device_properties(torch.cuda.current_device()).multi_processor_count
    fp32_peak = n_sm * 128 * 2 * sm_mhz * 1e6 / 1e12  # TFLOP/s
    p = w.params
    dims = np.asarray(p.layer_dims, dtype=np.int64)  # [S][L+1]
    L = dims.shape[1] - 1
    counts = np.bincount(w.species, minlength=dims.shape[0]).astype(np.int64)
    M = w.n_models
    mac = {l: int((counts * dims[:, l - 1] * dims[:, l]).sum()) * M for l in range(1, L + 1)}  # per pass
    w1_bytes = int(((counts > 0) * dims[:, 0] * dims[:, 1]).sum()) * M * 4
    engine = "ligand" if "mlp_mid" in stages or "mlp_last" not in stages else "tensor"
    out = []

    def add(stage, bound, work, unit, peak, src, note=None):
        if stage not in stages or stages[stage] <= 0:
            return
        achieved = work / (stages[stage] * 1e-6) / (1e9 if unit == "GB/s" else 1e12)
        d = {"stage": stage, "kernel": KERNEL_OF_STAGE[engine].get(stage, stage), "bound": bound,
             "achieved": achieved, "peak": peak, "unit": unit, "frac": achieved / peak, "kernel_us": stages[stage],
             "algorithmic_work": work, "peak_source": src}
        if note:
            d["note"] = note
        out.append(d)

    alu_src = f"derived: {n_sm} SMs x 128 FP32 lanes x 2 flop x {sm_mhz:.0f} MHz"
    if engine == "ligand":
        add("mlp_fwd_l1", "hbm", w1_bytes + w.n_atoms * nnp.n_features * 4, "GB/s", hbm_peak, hbm_src,
            "layer-1 weights of the ensemble streamed once + AEV rows; L2 flushed before the step")
        add("mlp_bwd_l1", "alu", 2.0 * mac[1], "TFLOP/s", fp32_peak, alu_src,
            "weights re-read from L2 (resident after the forward pass); FFMA2 on the CUDA cores")
        add("mlp_mid", "alu", 4.0 * sum(mac[l] for l in range(2, L)) + 4.0 * mac[L], "TFLOP/s", fp32_peak, alu_src,
            "layers 2..L-1 forward+backward and the 1-output layer, one CTA per (element, model, 4 atoms)")
    else:
        tf32_peak = 0.5 * bf16
        tsrc = "measured bf16 (MEASURED_PEAKS.json bf16_tflops) x 0.5 nominal TF32:BF16 ratio" if "bf16_tflops" in peaks \
            else "fallback 1650 TFLOP/s bf16 x 0.5"
        # layer 1 skips the 32-wide contraction boxes (forward) / 128-wide output tiles (backward) that hold only AEV
        # columns of absent species: quote the dense nominal flops AND the share actually issued
        present = counts > 0
        n_sub = p.shf_a.size * p.shf_z.size
        live = np.zeros(int(dims[0, 0]), bool)
        for s_ in range(dims.shape[0]):
            live[s_ * p.shf_r.size:(s_ + 1) * p.shf_r.size] = present[s_]
        pidx = 0
        for s_ in range(dims.shape[0]):
            for t_ in range(s_, dims.shape[0]):
                live[p.n_radial + pidx * n_sub:p.n_radial + (pidx + 1) * n_sub] = present[s_] and present[t_]
                pidx += 1
        nb = (live.size + 31) // 32
        nt = (live.size + 127) // 128
        frac_f = sum(live[32 * b:32 * b + 32].any() for b in range(nb)) / nb
        frac_b = sum(live[128 * b:128 * b + 128].any() for b in range(nt)) / nt
        for l in range(1, L):
            for st in (f"mlp_fwd_l{l}", f"mlp_bwd_l{l}"):
                issued = (frac_f if st.startswith("mlp_fwd") else frac_b) if l == 1 else 1.0
                add(st, "tensor", 2.0 * mac[l], "TFLOP/s", tf32_peak, tsrc,
                    "dense nominal useful flops; 3xTF32 issues 3 MMAs per useful MAC (ceiling of frac 1/3); "
                    f"share of the dense flops actually issued (structural zeros of absent species skipped): {issued:.3f}")
                if out and out[-1]["stage"] == st:
                    out[-1]["issued_fraction"] = issued
                    out[-1]["achieved_issued"] = out[-1]["achieved"] * issued
    if not out:
        return None
    top = max(out, key=lambda d: d["kernel_us"])
    roof = {k: top[k] for k in ("bound", "achieved", "peak", "unit", "frac")}
    roof["kernel"] = f'{top["kernel"]} ({top["stage"]})'
    roof["traffic"] = ncu_traffic_bytes(config, top["stage"])
    roof.update({k: top[k] for k in ("kernel_us", "algorithmic_work", "peak_source")})
    roof["timing"] = "CUDA events around the launch on the launch stream (profiling mode: plain launches, so the " \
                     "event-to-event time includes launch latency; conservative)"
    roof["top_stage_overall"] = max(stages, key=stages.get)
    roof["kernels"] = out
    return roof


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
        return multi.rank_frame(t, rank, n_frames)

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

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    for t in range(Wu):
        step(t)
    nnp.check()
    if rank == 0:
        sampler.wait_first_sample()
    barrier()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    t_wall0 = time.perf_counter()
    for t in range(K):
        step(Wu + t, evs[t])
    barrier()
    t_wall1 = time.perf_counter()
    t_wall = t_wall1 - t_wall0
    nnp.check()
    dev_ms = sum(a.elapsed_time(b) for a, b in evs)
    per_step_ms = sorted(a.elapsed_time(b) for a, b in evs)
    dev_ms_max = multi.max_over_ranks(dev_ms, dist, dev)
    value = multi.aggregate_throughput(w.n_atoms, K, world, dev_ms_max)

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
        roofline = stage_rooflines(w, nnp, stages, args.config)

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
        tot_max = multi.max_over_ranks(tot, dist, dev)
        e2e = {"value": multi.aggregate_throughput(w.n_atoms, K, world, 1e3 * tot_max), "unit": UNIT,
               "h2d_bytes_per_step": w.n_atoms * 12, "d2h_bytes_per_step": w.n_atoms * 12 + w.n_molecules * 8,
               "us_per_step": 1e6 * tot_max / K}
    clocks = sampler.stop(t_wall0, t_wall1) if rank == 0 else None

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
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config, 1-based (2 = the metric's)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--cpu-steps", type=int, default=1000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--flags", type=int, default=0, help="NNP_FLAG_* bits (include/nnp.h) for A/B runs of the engines")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()

#!/usr/bin/env python
"""bench.py -- ANI-2x energy+force atom-evals/s on BASELINE.json configs[1] (50 atoms, 8 models).

A "step" is one pass of the whole hot path (neighbour pairs -> AEV -> ensemble MLPs -> backward ->
forces added into the force buffer) = one nnp_compute on the next frame of the seeded, perturbed
trajectory.  See DESIGN.md "Measurement" for what each JSON key means and how it is measured.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--shard replicas|molecules|ensemble]
                  [--impl reference] [--no-other-configs]

With --gpus N > 1 and no torchrun environment the script starts its N ranks itself
(`python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 ...`).
"""
from __future__ import annotations

import argparse
import json
import math
import os
import socket
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
MIN_LOADED_SECONDS = 1.5  # the GPU is kept under load at least this long while the clocks are sampled


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
    """nvidia-smi clocks + throttle reasons sampled DURING the loaded part of the run."""

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
        """Summary of the samples taken in [t_begin, t_end] (perf_counter times)."""
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        window = "timed steps + warm-L2 loop + stage profiling (GPU under load throughout)"
        lines = [ln for t, ln in self.lines if (t_begin is None or t >= t_begin) and (t_end is None or t <= t_end)]
        if not lines:
            window = "whole run (no sample fell inside the loaded window)"
            lines = [ln for _, ln in self.lines]
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
                pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "window": window,
                "loaded_seconds": None if t_begin is None or t_end is None else t_end - t_begin,
                "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------
KERNEL_OF_STAGE = {
    "mlp_fwd_l1": "small_fwd1_kernel", "mlp_mid": "small_mid_kernel", "mlp_bwd_l1": "small_bwd1_kernel",
    "aev_fwd": "aev_forward_kernel", "aev_bwd": "aev_backward_kernel", "finish": "finish_kernel", "nbr": "nbr kernels",
    "mlp_last": "last_layer_kernel",
}


def load_peaks():
    """Roofline denominators: the driver-measured HBM copy / bf16 figures (MEASURED_PEAKS.json) and the library's own
    micro-benchmarks for what that file does not hold (FP32 FFMA, tcgen05 TF32 issue rate, L2 reads)."""
    from paper_2201_08110_b200.binding import measure_peaks

    try:
        drv = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        drv = {}
    pk = measure_peaks()
    pk["hbm_copy_gbs"] = float(drv.get("hbm_gbs", 6650.0))
    pk["hbm_copy_source"] = "MEASURED_PEAKS.json hbm_gbs (driver-measured copy)" if "hbm_gbs" in drv \
        else "fallback 6650 GB/s (B200_PROFILING.md)"
    pk["bf16_tflops_driver"] = drv.get("bf16_tflops")
    pk["tf32x3_ceiling_tflops"] = pk["tf32_tcgen05_tflops"] / 3.0
    pk["how"] = "nnp_measure_peaks in this run (csrc/peaks.cu): FFMA chains on every scheduler; tcgen05 kind::tf32 " \
                "M=128 N=256 K=8 issued back to back from shared-memory operands; reads of a 32 MiB (L2) and a 2 GiB buffer"
    return pk


def stage_rooflines(w, nnp, stages, config, peaks):
    """Roofline of every MLP launch from the live CUDA-event stage times, and of the dominant one under the contract's
    keys.  Algorithmic work: a layer GEMM does 2 flop per weight per atom-model; the ligand-size
    layer-1 forward must stream the layer-1 weights of the ensemble once (HBM-bound when L2 was flushed).  Tensor
    launches: `achieved` = flops ACTUALLY ISSUED (nnp_get_stage_work: structural zeros skipped, padding excluded) per
    second, `peak` = measured tcgen05 TF32 rate / 3 (3xTF32 issues three MMAs per useful MAC)."""
    p = w.params
    dims = np.asarray(p.layer_dims, dtype=np.int64)  # [S][L+1]
    L = dims.shape[1] - 1
    counts = np.bincount(w.species, minlength=dims.shape[0]).astype(np.int64)
    M = w.n_models
    mac = {l: int((counts * dims[:, l - 1] * dims[:, l]).sum()) * M for l in range(1, L + 1)}  # per pass
    w1_bytes = int(((counts > 0) * dims[:, 0] * dims[:, 1]).sum()) * M * 4
    issued = nnp.stage_work()
    tensor = any(v[0] > 0 for v in issued.values())
    ligand = "mlp_mid" in stages
    out = []

    def add(stage, kernel, bound, work, unit, peak, src, note=None, extra=None):
        if stage not in stages or stages[stage] <= 0:
            return
        achieved = work / (stages[stage] * 1e-6) / (1e9 if unit == "GB/s" else 1e12)
        d = {"stage": stage, "kernel": kernel, "bound": bound, "achieved": achieved, "peak": peak, "unit": unit,
             "frac": achieved / peak, "kernel_us": stages[stage], "algorithmic_work": work, "peak_source": src}
        if note:
            d["note"] = note
        if extra:
            d.update(extra)
        out.append(d)

    fp32, fsrc = peaks["fp32_ffma_tflops"], "measured: nnp_measure_peaks FP32 FFMA"
    if ligand:
        add("mlp_fwd_l1", KERNEL_OF_STAGE["mlp_fwd_l1"], "hbm", w1_bytes + w.n_atoms * nnp.n_features * 4, "GB/s",
            peaks["hbm_copy_gbs"], peaks["hbm_copy_source"],
            "layer-1 weights of the ensemble streamed once + AEV rows; L2 flushed before the step")
        add("mlp_bwd_l1", KERNEL_OF_STAGE["mlp_bwd_l1"], "alu", 2.0 * mac[1], "TFLOP/s", fp32, fsrc,
            "weights re-read from L2 (resident after the forward pass); FFMA2 on the CUDA cores")
        add("mlp_mid", KERNEL_OF_STAGE["mlp_mid"], "alu", 4.0 * sum(mac[l] for l in range(2, L)) + 4.0 * mac[L], "TFLOP/s",
            fp32, fsrc, "layers 2..L-1 forward+backward and the 1-output layer, one CTA per (element, model, 4 atoms)")
    elif tensor:
        ceiling = peaks["tf32x3_ceiling_tflops"]
        tsrc = "measured: nnp_measure_peaks tcgen05 kind::tf32 rate / 3 (3xTF32 issues 3 MMAs per useful MAC)"
        abytes = nnp.stage_bytes()
        for l in range(1, L):
            for st in (f"mlp_fwd_l{l}", f"mlp_bwd_l{l}"):
                fl, tile = issued.get(st, (0.0, 0))
                by = abytes.get(st, 0.0)
                if stages.get(st, 0) <= 0:
                    continue
                t = stages[st] * 1e-6
                tfrac = fl / t / 1e12 / ceiling
                hfrac = by / t / 1e9 / peaks["hbm_copy_gbs"]
                extra = {"dense_nominal_flops": 2.0 * mac[l], "issued_fraction": fl / (2.0 * mac[l]) if mac[l] else None,
                         "atom_tile": tile, "frac_of_tf32_peak": fl / t / 1e12 / peaks["tf32_tcgen05_tflops"],
                         "tensor_frac": tfrac, "hbm_frac": hfrac, "issued_flops": fl, "algorithmic_bytes": by}
                # a launch is bound by whichever of its two rooflines it is closer to: the hidden-layer launches of a
                # large system stream split activation planes that do not fit L2
                if hfrac > tfrac and by > 126e6:  # below the L2 size the planes of a launch never leave the L2
                    add(st, "gemm_umma_kernel", "hbm", by, "GB/s", peaks["hbm_copy_gbs"], peaks["hbm_copy_source"],
                        "algorithmic bytes (nnp_get_stage_bytes): operand planes, output planes and epilogue reads, each once",
                        extra)
                else:
                    add(st, "gemm_umma_kernel", "tensor", fl, "TFLOP/s", ceiling, tsrc,
                        "flops actually issued (structural-zero boxes skipped, padding excluded)", extra)
    else:  # grouped FP32 FFMA GEMMs (shapes outside the tensor engine)
        for l in range(1, L):
            for st in (f"mlp_fwd_l{l}", f"mlp_bwd_l{l}"):
                add(st, "gemm_grouped_kernel", "alu", 2.0 * mac[l], "TFLOP/s", fp32, fsrc)
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
    roof["mlp_flops_per_step_dense"] = nnp.work()["mlp_flops"]
    roof["kernels"] = out
    return roof


# ------------------------------------------------------------------------------------------------
def oracle_sample(w, W, B, traj_h, n_evals):
    """The float64 oracle, as it stands, on the host cores: `n_evals` full evaluations (after one untimed call)."""
    from oracle.ani_oracle import AniOracle

    orc = AniOracle(w.params, W, B)
    orc.energy_forces(traj_h[0], w.species, w.mol_offsets)
    t0 = time.perf_counter()
    for t in range(n_evals):
        orc.energy_forces(traj_h[t % len(traj_h)], w.species, w.mol_offsets)
    dt = time.perf_counter() - t0
    return {"value": w.n_atoms * n_evals / dt, "unit": UNIT, "cores": orc.threads, "kind": "oracle",
            "sample": f"{n_evals} full energy+force evaluation(s) of the {w.n_atoms}-atom workload on consecutive frames, "
                      f"{1e3 * dt / n_evals:.1f} ms/step"}


def run_reference(args):
    """--impl reference: the float64 CPU oracle, as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    w = wl.get_config(args.config)
    W, B = w.weights()
    from oracle.ani_oracle import AniOracle

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
def measure_single(w, W, B, steps, warmup, peaks, config_id, flags=0, n_prof=5, cpu_evals=0):
    """One workload on the current device, one rank: cold-L2 device time per step (CUDA events per step, L2 flushed
    between steps), per-stage times and rooflines, optionally the oracle on a bounded sample.  Used for the
    `other_configs` legs of the default run."""
    import torch

    from paper_2201_08110_b200.binding import NNP

    dev = torch.device("cuda", torch.cuda.current_device())
    nnp = NNP(w.params, W, B, w.species, w.mol_offsets, flags=flags)
    n_frames = min(max(steps + warmup, 2), w.n_steps if w.n_steps > 1 else 1, 1000)
    traj_h = w.trajectory(max(n_frames, 1)) if w.n_steps > 1 else w.positions[None]
    traj = torch.from_numpy(np.ascontiguousarray(traj_h)).to(dev)
    pos = traj[0].clone()
    E = torch.zeros(w.n_molecules, dtype=torch.float64, device=dev)
    F = torch.zeros((w.n_atoms, 3), dtype=torch.float32, device=dev)
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()

    def step(t, ev=None):
        pos.copy_(traj[t % traj.shape[0]])
        flush.zero_()
        if ev:
            ev[0].record(stream)
        nnp.compute_torch(pos, E, F)
        if ev:
            ev[1].record(stream)

    for t in range(warmup):
        step(t)
    nnp.check()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for t in range(steps):
        step(warmup + t, evs[t])
    torch.cuda.synchronize()
    nnp.check()
    per = sorted(a.elapsed_time(b) for a, b in evs)
    ms = sum(per) / steps
    nnp.set_profiling(True)
    acc = {}
    for t in range(n_prof):
        step(warmup + t)
        for k, v in nnp.stage_times().items():
            acc[k] = acc.get(k, 0.0) + v
    nnp.set_profiling(False)
    stages = {k: 1e3 * v / n_prof for k, v in acc.items()}
    roof = stage_rooflines(w, nnp, stages, config_id, peaks)
    out = {"workload": f"{w.name}: {w.n_atoms} atoms, {w.n_molecules} molecule(s), {w.n_models} model(s)",
           "steps": steps, "warmup": warmup, "us_per_step": 1e3 * ms, "us_per_step_median": 1e3 * per[len(per) // 2],
           "atom_evals_per_s": w.n_atoms / (ms * 1e-3), "gpu_launches_per_step": nnp.launches_per_compute,
           "stage_us": stages}
    if roof:
        out["mlp_kernels"] = [{k: d[k] for k in ("stage", "kernel", "bound", "achieved", "peak", "unit", "frac", "kernel_us",
                                                 "atom_tile", "issued_fraction") if k in d} for d in roof["kernels"]]
    nnp.destroy()
    if cpu_evals > 0:
        out["cpu_baseline"] = oracle_sample(w, W, B, traj_h, cpu_evals)
    return out


def measure_coupling(peaks, steps=20, warmup=3):
    """Eq. 4 coupling kernel on the 50-atom NNP region in 30 000 MM atoms with the paper's 9 A
    cutoff: pair tests per second, and the oracle on the same input."""
    import torch

    from oracle.coupling_oracle import COULOMB_KCAL_A, coupling_energy_forces
    from paper_2201_08110_b200.binding import Coupling

    dev = torch.device("cuda", torch.cuda.current_device())
    s = wl.coupling_system()
    a = (s.nnp_rows, s.q_nnp, s.sigma_nnp, s.eps_nnp, s.mm_rows, s.q_mm, s.sigma_mm, s.eps_mm)
    cp = Coupling(*a, coulomb_const=COULOMB_KCAL_A, cutoff=9.0)
    pos = torch.from_numpy(s.positions).to(dev)
    E = torch.zeros(1, dtype=torch.float64, device=dev)
    F = torch.zeros((s.n_rows, 3), dtype=torch.float32, device=dev)
    st = torch.cuda.current_stream()
    for _ in range(warmup):
        cp.compute(pos.data_ptr(), 3, E.data_ptr(), F.data_ptr(), 3, st.cuda_stream)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(st)
    for _ in range(steps):
        cp.compute(pos.data_ptr(), 3, E.data_ptr(), F.data_ptr(), 3, st.cuda_stream)
    e1.record(st)
    torch.cuda.synchronize()
    us = 1e3 * e0.elapsed_time(e1) / steps
    cp.destroy()
    pairs = cp.n_nnp * cp.n_mm
    t0 = time.perf_counter()
    coupling_energy_forces(s.positions, *a, cutoff=9.0)
    t_cpu = time.perf_counter() - t0
    # every pair is tested twice (once per force side); ~60 FP64 operations per test incl. the rare full evaluation
    return {"workload": f"Eq. 4 coupling: {cp.n_nnp} NNP atoms x {cp.n_mm} MM atoms, 9 A cutoff, forces on both regions",
            "us_per_step": us, "pair_tests_per_s": pairs / (us * 1e-6), "gpu_launches_per_step": 2,
            "cpu_baseline": {"value": pairs / t_cpu, "unit": "pair tests/s", "cores": 1, "kind": "oracle",
                             "sample": f"1 evaluation of the same system, {1e3 * t_cpu:.1f} ms"}}


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

    w = wl.get_config(args.config)
    W, B = w.weights()
    K, Wu = args.steps, args.warmup
    n_frames = min(max(K + Wu, 2), 1000)
    traj_full = w.trajectory(n_frames)
    shard = args.shard if world > 1 else "replicas"
    # what this rank evaluates: the whole workload (replicas: independent copies, weak scaling), its molecules
    # (configs[2]: no data-path collective) or the whole molecule with its share of the ensemble (one all-reduce)
    m_part = w.n_models
    if shard == "molecules":
        sh = multi.shard_molecules(w.mol_offsets, world, rank)
        species, offsets = w.species[sh.atom_lo:sh.atom_hi], sh.mol_offsets
        traj_h = np.ascontiguousarray(traj_full[:, sh.atom_lo:sh.atom_hi])
        Wr, Br = W, B
    elif shard == "ensemble":
        m_lo, m_hi = multi.shard_models(w.n_models, world, rank)
        Wr, Br = multi.slice_models(W, B, m_lo, m_hi)
        m_part = m_hi - m_lo
        species, offsets, traj_h = w.species, w.mol_offsets, traj_full
    else:
        species, offsets, traj_h, Wr, Br = w.species, w.mol_offsets, traj_full, W, B
    n_local = int(species.size)
    n_mol_local = int(len(offsets) - 1)
    nnp = NNP(w.params, Wr, Br, species, offsets, flags=args.flags)
    traj = torch.from_numpy(traj_h).to(dev)
    pos = traj[0].clone()  # the MD engine's position buffer: same pointer every step
    E = torch.zeros(n_mol_local, dtype=torch.float64, device=dev)
    F = torch.zeros((n_local, 3), dtype=torch.float32, device=dev)
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()
    peaks = load_peaks() if rank == 0 else None

    def frame(t):
        return multi.rank_frame(t, rank if shard == "replicas" else 0, n_frames)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def compute():
        if shard == "ensemble":
            F.zero_()
            nnp.compute_torch(pos, E, F)
            return multi.combine_ensemble_parts(E, F, m_part, w.n_models, dist)  # NCCL SUM all-reduce, in stream order
        nnp.compute_torch(pos, E, F)
        return E, F

    def step(t, timed_events=None):
        pos.copy_(traj[frame(t)])      # untimed: the integrator moved the atoms
        flush.zero_()                  # untimed: evict L2 (weights must come from HBM again)
        if timed_events is not None:
            timed_events[0].record(stream)
        compute()
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
    units = w.n_atoms if shard != "replicas" else w.n_atoms * world  # atoms of the whole job per step
    value = units * K / (dev_ms_max * 1e-3)

    # ---- warm-L2 variant (weights stay L2-resident between steps, as in a tight MD loop); also the part of the run
    # that keeps the GPU loaded long enough for the clock record to mean something
    warm_ms, n_warm = None, 0
    if rank == 0 and shard != "ensemble":
        for t in range(5):
            nnp.compute_torch(pos, E, F)
        est = max(per_step_ms[len(per_step_ms) // 2] * 1e-3, 1e-6)
        n_warm = int(min(max(K, math.ceil(MIN_LOADED_SECONDS / est)), 200000))
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for t in range(n_warm):
            nnp.compute_torch(pos, E, F)
        b.record(stream)
        torch.cuda.synchronize()
        warm_ms = a.elapsed_time(b) / n_warm

    # ---- per-kernel stage times (CUDA events between stages, same flush discipline) -> roofline
    roofline = None
    stages = None
    if rank == 0:
        nnp.set_profiling(True)
        acc = {}
        n_prof = min(max(K, 5), 50)
        for t in range(n_prof):
            pos.copy_(traj[frame(Wu + t)])
            flush.zero_()
            nnp.compute_torch(pos, E, F)
            for k, v in nnp.stage_times().items():
                acc[k] = acc.get(k, 0.0) + v
        nnp.set_profiling(False)
        stages = {k: 1e3 * v / n_prof for k, v in acc.items()}  # us
        local_w = w if shard == "replicas" else None
        if local_w is not None:
            roofline = stage_rooflines(w, nnp, stages, args.config, peaks)
    t_loaded_end = time.perf_counter()

    # ---- end-to-end through the C ABI with HOST buffers (pinned), copies inside the timed region
    hp = torch.from_numpy(traj_h).pin_memory()
    hE = torch.zeros(n_mol_local, dtype=torch.float64).pin_memory()
    hF = torch.zeros((n_local, 3), dtype=torch.float32).pin_memory()
    sraw = stream.cuda_stream

    def e2e_step(t):
        if shard == "ensemble":  # host -> device, this rank's networks, the all-reduce, device -> host
            pos.copy_(hp[frame(t)], non_blocking=True)
            Ec, Fc = compute()
            hE.copy_(Ec, non_blocking=True)
            hF.copy_(Fc, non_blocking=True)
            torch.cuda.synchronize()
        else:
            nnp.compute_host_into(hp[frame(t)].data_ptr(), hE.data_ptr(), hF.data_ptr(), sraw)  # syncs

    for t in range(3):
        e2e_step(t)
    barrier()
    tot = 0.0
    for t in range(K):
        flush.zero_()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        e2e_step(Wu + t)
        tot += time.perf_counter() - t0
    tot_max = multi.max_over_ranks(tot, dist, dev)
    e2e = {"value": units * K / tot_max, "unit": UNIT, "h2d_bytes_per_step": n_local * 12,
           "d2h_bytes_per_step": n_local * 12 + n_mol_local * 8, "us_per_step": 1e6 * tot_max / K,
           "api": "nnp_compute_host (pinned host buffers; one H2D copy, the graph, one D2H copy, one stream sync)"}
    clocks = sampler.stop(t_wall0, t_loaded_end) if rank == 0 else None
    launches = K * nnp.launches_per_compute
    nnp.destroy()

    # ---- CPU baseline and the other workloads: rank 0 at N = 1 only
    cpu = None
    others = None
    if rank == 0 and world == 1:
        if not args.no_cpu_baseline:
            cpu = oracle_sample(w, W, B, traj_full, args.cpu_steps)
        if not args.no_other_configs and args.config == 2:
            others = {}
            plan = [("configs[0]", wl.config1(), 1, 20, 5, 20), ("configs[2]", wl.config3(), 3, 10, 3, 1),
                    ("configs[3]", wl.config4(), 4, 20, 3, 5), ("configs[4]", wl.config5(), 5, 10, 3, 1),
                    ("configs[1] with 1 NN (PAPER.md:160)", wl.config2(n_models=1), 2, 50, 5, 50),
                    ("ANI-1x, 48-atom ligand (PAPER.md:166-175)", wl.ani1x_ligand(), 0, 50, 5, 50)]
            for name, wk, cid, st, wm, ce in plan:
                Wk, Bk = wk.weights()
                others[name] = measure_single(wk, Wk, Bk, st, wm, peaks, cid, cpu_evals=0 if args.no_cpu_baseline else ce)
            others["Eq. 4 coupling (PAPER.md:67-71)"] = measure_coupling(peaks)
    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wu,
            "ms_per_step": dev_ms_max / K, "us_per_step": 1e3 * dev_ms_max / K,
            "us_per_step_median": 1e3 * per_step_ms[len(per_step_ms) // 2],
            "us_per_step_warm_l2": None if warm_ms is None else 1e3 * warm_ms, "warm_l2_steps": n_warm,
            "wall_us_per_step_incl_flush": 1e6 * t_wall / K,
            "higher_is_better": True, "scaling": "weak" if shard == "replicas" else "strong", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": workload_config(w, {"l2": f"flushed between timed steps ({L2_FLUSH_BYTES >> 20} MiB write, "
                                                "outside the per-step CUDA events)",
                                          "timing": "sum of per-step CUDA-event durations on the launch stream, "
                                                    "max over ranks",
                                          "parallelism": {"replicas": f"replicas x{world}",
                                                          "molecules": f"molecules sharded over {world} ranks, no collective",
                                                          "ensemble": f"ensemble sharded over {world} ranks, one SUM "
                                                                      f"all-reduce of E and F per step"}[shard]}),
            "e2e": e2e, "gpu_launches": launches, "clocks": clocks, "peaks": peaks, "roofline": roofline,
            "stage_us": stages, "cpu_baseline": cpu, "other_configs": others,
        }
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def spawn_ranks(args):
    """--gpus N without a torchrun environment: start the N ranks of this node ourselves."""
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config, 1-based (2 = the metric's)")
    ap.add_argument("--shard", default="replicas", choices=["replicas", "molecules", "ensemble"],
                    help="N > 1: independent replicas (weak), the molecules of a batch (strong, configs[2]) or the "
                         "ensemble members of one molecule (strong, one all-reduce)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--cpu-steps", type=int, default=1000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true")
    ap.add_argument("--flags", type=int, default=0, help="NNP_FLAG_* bits (include/nnp.h) for A/B runs of the engines")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(spawn_ranks(args))
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()

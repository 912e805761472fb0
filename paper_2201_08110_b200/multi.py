"""Host-side logic of the multi-GPU path (one process per GPU, torch.distributed for the plumbing).

The hot path shards over INDEPENDENT molecules (BASELINE.json configs[2]): every rank owns a
contiguous slice of the molecules of a batch and evaluates it with its own handle; there is no data-path
collective (energies are per molecule, forces per atom, both stay on the rank that owns the molecule).  The
only collective is the max-over-ranks reduction of the device time of a benchmark.  Nothing here does any of the
method's arithmetic.
"""
from __future__ import annotations

from typing import NamedTuple

import numpy as np


def shard_range(n_units: int, world: int, rank: int):
    """Contiguous, balanced [lo, hi) of `n_units` for `rank` of `world` (first n_units % world ranks get one more)."""
    if world < 1 or not (0 <= rank < world) or n_units < 0:
        raise ValueError("bad shard arguments")
    base, rem = divmod(n_units, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


class MoleculeShard(NamedTuple):
    mol_lo: int
    mol_hi: int
    atom_lo: int
    atom_hi: int
    mol_offsets: np.ndarray  # local CSR offsets [mol_hi - mol_lo + 1], starting at 0


def shard_molecules(mol_offsets, world: int, rank: int) -> MoleculeShard:
    """The slice of a batch (CSR molecule offsets) that `rank` owns: whole molecules only, contiguous."""
    off = np.asarray(mol_offsets, dtype=np.int64)
    if off.ndim != 1 or off.size < 1 or off[0] != 0 or np.any(np.diff(off) < 0):
        raise ValueError("mol_offsets must be a CSR offset array starting at 0")
    lo, hi = shard_range(off.size - 1, world, rank)
    a_lo, a_hi = int(off[lo]), int(off[hi])
    return MoleculeShard(lo, hi, a_lo, a_hi, (off[lo:hi + 1] - off[lo]).astype(np.int32))


def rank_frame(t: int, rank: int, n_frames: int) -> int:
    """Trajectory frame that `rank` evaluates at step t of a replica benchmark (ranks are de-phased by 17 frames)."""
    return (t + 17 * rank) % n_frames


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """MAX all-reduce of one scalar (the benchmark's device time); identity without a process group."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch

    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_per_rank: int, steps: int, world: int, ms_max: float) -> float:
    """Whole-job units/s when every rank processed `units_per_rank` units per step and the slowest took ms_max."""
    return world * units_per_rank * steps / (ms_max * 1e-3)


# ------------------------------------------------------------------------------------------------
# A SINGLE large molecule (configs[3], configs[4]) does not shard over molecules; it shards over the ENSEMBLE
# (SURVEY.md 8(e)): the energy is the mean of the member networks' energies and the forces are linear in them, so
# rank r evaluates the whole molecule with its contiguous subset of M_r networks (its own handle with n_models = M_r)
# and one SUM all-reduce of (M_r / M) * [E_mol..., F] gives every rank the ensemble result.  The per-species
# self-energies are added by every rank and are weighted like the rest: sum_r (M_r / M) = 1.  The message is
# n_mol + 3 N numbers (240 KB at 10 000 atoms): latency-bound over NVLink, which is why this only pays above a few
# hundred atoms.
def shard_models(n_models: int, world: int, rank: int):
    """Contiguous [lo, hi) of the ensemble members for `rank`; every rank must own at least one network."""
    if world > n_models:
        raise ValueError(f"ensemble sharding needs world <= n_models ({world} > {n_models})")
    return shard_range(n_models, world, rank)


def combine_ensemble_parts(E_part, F_part, n_models_part: int, n_models_total: int, dist=None):
    """The one data-path collective of the ensemble-sharded path.  E_part [n_mol] (f64) and F_part [N,3] are this
    rank's results with its n_models_part networks (torch tensors on the device of the process group's backend, or
    numpy arrays for a CPU group); returns (E, F) of the whole ensemble, same types.  Without a group: identity
    weighting of a single part (n_models_part must equal n_models_total)."""
    import torch

    as_np = isinstance(E_part, np.ndarray)
    E_t = torch.from_numpy(np.ascontiguousarray(E_part, dtype=np.float64)) if as_np else E_part
    F_t = torch.from_numpy(np.ascontiguousarray(F_part)) if as_np else F_part
    weight = float(n_models_part) / float(n_models_total)
    buf = torch.cat([E_t.to(torch.float64).reshape(-1), F_t.to(torch.float64).reshape(-1)]) * weight
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(buf, op=dist.ReduceOp.SUM)
    elif n_models_part != n_models_total:
        raise ValueError("a partial ensemble needs a process group to be combined")
    n_e = E_t.numel()
    E = buf[:n_e].reshape(E_t.shape)
    F = buf[n_e:].reshape(F_t.shape).to(F_t.dtype)
    return (E.numpy(), F.numpy()) if as_np else (E, F)


def slice_models(weights, biases, lo: int, hi: int):
    """The networks [lo, hi) of nested [m][e][l] weight / bias lists (biases may be None)."""
    return weights[lo:hi], (None if biases is None else biases[lo:hi])

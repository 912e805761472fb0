"""N>1 host logic on CPU: world_size-2 gloo process group (127.0.0.1).  Every rank evaluates its shard of a
batch of independent molecules (here with the float64 oracle standing in for the per-rank engine: the test is
about the sharding, not the kernels) and the union must equal the unsharded evaluation; the benchmark's
max-over-ranks reduction and throughput aggregation are checked on the same group."""
import os
import socket

import numpy as np
import pytest

from paper_2201_08110_b200 import multi
from paper_2201_08110_b200 import workloads as wl


def test_shard_range_partitions_exactly():
    for n in (0, 1, 2, 7, 256, 1001):
        for world in (1, 2, 3, 8):
            spans = [multi.shard_range(n, world, r) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            assert all(spans[r][1] == spans[r + 1][0] for r in range(world - 1))
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        multi.shard_range(4, 2, 2)


def test_shard_molecules_keeps_molecules_whole():
    off = np.array([0, 3, 3, 10, 14, 20], np.int32)  # molecule 1 is empty
    shards = [multi.shard_molecules(off, 2, r) for r in range(2)]
    assert shards[0].mol_lo == 0 and shards[1].mol_hi == 5 and shards[0].mol_hi == shards[1].mol_lo
    assert shards[0].atom_hi == shards[1].atom_lo == int(off[shards[0].mol_hi])
    for s in shards:
        assert s.mol_offsets[0] == 0 and s.mol_offsets[-1] == s.atom_hi - s.atom_lo
        assert np.array_equal(np.diff(s.mol_offsets), np.diff(off[s.mol_lo:s.mol_hi + 1]))
    with pytest.raises(ValueError):
        multi.shard_molecules(np.array([1, 2]), 2, 0)


def test_rank_frames_and_aggregate():
    assert multi.rank_frame(0, 0, 1000) == 0 and multi.rank_frame(990, 1, 1000) == 7
    assert multi.aggregate_throughput(50, 200, 8, 20.0) == pytest.approx(8 * 50 * 200 / 0.020)
    assert multi.max_over_ranks(3.5) == 3.5  # no process group: identity


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch.distributed as dist

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle.ani_oracle import AniOracle

        p = wl.small_params(3, (16, 12, 8))
        W, B = wl.make_weights(p, 2, seed=11, random_biases=True)
        mols = [wl.random_molecule(n, 3, seed=40 + i, params=p, n_models=2) for i, n in enumerate((9, 14, 6, 11, 8))]
        pos = np.concatenate([m.positions for m in mols])
        spc = np.concatenate([m.species for m in mols])
        off = np.concatenate([[0], np.cumsum([m.n_atoms for m in mols])]).astype(np.int32)
        sh = multi.shard_molecules(off, world, rank)
        orc = AniOracle(p, W, B)
        mine = orc.energy_forces(pos[sh.atom_lo:sh.atom_hi], spc[sh.atom_lo:sh.atom_hi], sh.mol_offsets)
        gathered = [None] * world
        dist.all_gather_object(gathered, (sh.mol_lo, sh.atom_lo, mine["E"], mine["F"]))
        t_max = multi.max_over_ranks(10.0 + rank, dist)
        # ensemble sharding of ONE molecule: this rank's networks, then the one SUM all-reduce
        W3, B3 = wl.make_weights(p, 3, seed=12, random_biases=True)
        se = np.array([-0.5, -38.0, -54.7])
        m_lo, m_hi = multi.shard_models(3, world, rank)  # 2 + 1 networks: unequal parts
        Wp, Bp = multi.slice_models(W3, B3, m_lo, m_hi)
        part = AniOracle(p, Wp, Bp, self_energy=se).energy_forces(mols[1].positions, mols[1].species)
        E_all, F_all = multi.combine_ensemble_parts(part["E"], part["F"], m_hi - m_lo, 3, dist)
        whole = AniOracle(p, W3, B3, self_energy=se).energy_forces(mols[1].positions, mols[1].species)
        ens_ok = (np.allclose(E_all, whole["E"], rtol=1e-13, atol=1e-9) and np.allclose(F_all, whole["F"], rtol=0, atol=1e-10))
        flags = [None] * world
        dist.all_gather_object(flags, bool(ens_ok))
        if rank == 0:
            assert all(flags), "ensemble-sharded result differs from the whole ensemble"
            full = orc.energy_forces(pos, spc, off)
            E = np.concatenate([g[2] for g in sorted(gathered, key=lambda g: g[0])])
            F = np.concatenate([g[3] for g in sorted(gathered, key=lambda g: g[1])])
            ok = (E.shape == full["E"].shape and np.allclose(E, full["E"], rtol=0, atol=1e-12)
                  and np.allclose(F, full["F"], rtol=0, atol=1e-12) and t_max == 10.0 + world - 1)
            q.put(bool(ok))
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_sharded_batch_matches_unsharded():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for pr in procs:
        pr.start()
    for pr in procs:
        pr.join(timeout=180)
        assert pr.exitcode == 0
    assert q.get(timeout=10) is True


def test_shard_models_and_single_part_identity():
    assert [multi.shard_models(8, 4, r) for r in range(4)] == [(0, 2), (2, 4), (4, 6), (6, 8)]
    assert [multi.shard_models(8, 3, r) for r in range(3)] == [(0, 3), (3, 6), (6, 8)]
    with pytest.raises(ValueError):
        multi.shard_models(1, 2, 0)
    E, F = np.array([1.5, -2.0]), np.arange(12, dtype=np.float32).reshape(4, 3)
    E2, F2 = multi.combine_ensemble_parts(E, F, 8, 8)
    assert np.array_equal(E, E2) and np.array_equal(F, F2) and F2.dtype == np.float32
    with pytest.raises(ValueError):
        multi.combine_ensemble_parts(E, F, 4, 8)

"""Seeded synthetic inputs for the ANI-2x energy+force hot path.

This module holds NO arithmetic of the method (no cutoff function, no symmetry
function, no MLP): it only draws positions, species, weights and perturbation
noise, and carries the ANI-2x hyper-parameter *values* that BASELINE.json
configs[0] prints.  Both the CPU oracle tests and the CUDA tests feed the very
same arrays (same bits) to their side; neither side imports the other.

The paper's own inputs (PDBbind ligands 1AJV/1HPO/2P95/3BE9, 48-75 atoms,
PAPER.md:116-119 Table 1; trained ANI-2x weights) are not in this
container; these inputs take their sizes, element set and density and stand in
for them.  Recipes follow SURVEY.md section 8(d) / DESIGN.md "Input recipe".

Readings used here (DESIGN.md lists them): S5 species order H,C,N,O,F,S,Cl;
S11 Xavier-uniform f32 weights; S14 exact species counts by largest remainder;
S15 config-2 sphere = 12 A diameter; S16 config-3 literal 6 A cube; S17 config 5
= 3333 waters; S18 cumulative random-walk perturbation.
"""
from __future__ import annotations

import dataclasses
import math
from typing import List, Sequence

import numpy as np

BASE_SEED = 220108110
SPECIES = ("H", "C", "N", "O", "F", "S", "Cl")
MIN_DIST = 0.95  # Angstrom, BASELINE.json configs[0..4]


@dataclasses.dataclass(frozen=True)
class AniParams:
    """ANI-2x hyper-parameters as float32/int32 arrays (values: BASELINE.json configs[0])."""

    n_species: int
    rc_radial: np.float32
    rc_angular: np.float32
    eta_r: np.float32
    shf_r: np.ndarray  # f32[16]
    eta_a: np.float32
    zeta: np.float32
    shf_a: np.ndarray  # f32[8]
    shf_z: np.ndarray  # f32[4]
    cos_scale: np.float32
    celu_alpha: np.float32
    layer_dims: np.ndarray  # i32[n_species][n_layers+1]
    energy_scale: float  # output unit per model unit (kcal/mol per Hartree, reading S8)

    @property
    def n_layers(self) -> int:
        return int(self.layer_dims.shape[1] - 1)

    @property
    def n_radial(self) -> int:
        return int(self.n_species * self.shf_r.size)

    @property
    def n_pairs(self) -> int:
        return int(self.n_species * (self.n_species + 1) // 2)

    @property
    def n_features(self) -> int:
        return int(self.n_radial + self.n_pairs * self.shf_a.size * self.shf_z.size)


def ani2x_params() -> AniParams:
    f32 = np.float32
    k16 = np.arange(16, dtype=np.float64)
    k8 = np.arange(8, dtype=np.float64)
    k4 = np.arange(4, dtype=np.float64)
    hidden = {
        "H": (256, 192, 160),
        "C": (224, 192, 160),
        "N": (192, 160, 128),
        "O": (192, 160, 128),
        "F": (160, 128, 96),
        "S": (160, 128, 96),
        "Cl": (160, 128, 96),
    }
    n_feat = 7 * 16 + 28 * 32
    dims = np.array([[n_feat, *hidden[s], 1] for s in SPECIES], dtype=np.int32)
    return AniParams(
        n_species=7,
        rc_radial=f32(5.1),
        rc_angular=f32(3.5),
        eta_r=f32(19.7),
        shf_r=(0.8 + 0.26875 * k16).astype(f32),
        eta_a=f32(12.5),
        zeta=f32(14.1),
        shf_a=(0.8 + 0.3375 * k8).astype(f32),
        shf_z=((2.0 * k4 + 1.0) * math.pi / 8.0).astype(f32),
        cos_scale=f32(0.95),
        celu_alpha=f32(0.1),
        layer_dims=dims,
        energy_scale=627.5094740631,
    )


def small_params(n_species: int = 3, hidden: Sequence[int] = (16, 12, 8)) -> AniParams:
    """A reduced parameter set (fewer species, tiny MLPs) for fast unit tests."""
    p = ani2x_params()
    n_feat = n_species * 16 + (n_species * (n_species + 1) // 2) * 32
    dims = np.array([[n_feat, *hidden, 1]] * n_species, dtype=np.int32)
    return dataclasses.replace(p, n_species=n_species, layer_dims=dims)


def make_weights(params: AniParams, n_models: int, seed: int, random_biases: bool = False):
    """Xavier-uniform f32 weights [out][in] (S11), model-major, then element, then layer.

    Returns (weights, biases): nested lists [m][e][l] of C-contiguous f32 arrays.
    Biases are zero (BASELINE.json configs[0]) unless ``random_biases`` (tests of the
    bias path: real ANI models have biases, S10).
    """
    rng = np.random.default_rng(seed)
    W: List[List[List[np.ndarray]]] = []
    B: List[List[List[np.ndarray]]] = []
    for _m in range(n_models):
        Wm, Bm = [], []
        for e in range(params.n_species):
            We, Be = [], []
            for l in range(params.n_layers):
                fan_in = int(params.layer_dims[e, l])
                fan_out = int(params.layer_dims[e, l + 1])
                a = math.sqrt(6.0 / (fan_in + fan_out))
                w = rng.uniform(-a, a, size=(fan_out, fan_in)).astype(np.float32)
                if random_biases:
                    b = rng.uniform(-0.05, 0.05, size=(fan_out,)).astype(np.float32)
                else:
                    b = np.zeros((fan_out,), dtype=np.float32)
                We.append(np.ascontiguousarray(w))
                Be.append(b)
            Wm.append(We)
            Bm.append(Be)
        W.append(Wm)
        B.append(Bm)
    return W, B


def species_counts(n: int, fractions: Sequence[float]) -> List[int]:
    """Exact counts by largest-remainder rounding, ties to the earlier element (S14)."""
    raw = [n * f for f in fractions]
    cnt = [int(math.floor(x + 1e-9)) for x in raw]
    rem = [x - c for x, c in zip(raw, cnt)]
    order = sorted(range(len(raw)), key=lambda i: (-round(rem[i], 9), i))
    left = n - sum(cnt)
    for i in order[:left]:
        cnt[i] += 1
    assert sum(cnt) == n
    return cnt


def make_species(n: int, fractions: Sequence[float], seed: int) -> np.ndarray:
    cnt = species_counts(n, fractions)
    s = np.concatenate([np.full(c, e, dtype=np.int32) for e, c in enumerate(cnt)])
    np.random.default_rng(seed).shuffle(s)
    return s


def _place(rng, n: int, draw, min_dist: float = MIN_DIST, max_tries: int = 2_000_000) -> np.ndarray:
    """Sequential rejection sampling: accept a draw if >= min_dist from all accepted."""
    pts = np.empty((n, 3), dtype=np.float64)
    k = 0
    tries = 0
    while k < n:
        tries += 1
        if tries > max_tries:
            raise RuntimeError("rejection placement did not converge")
        c = draw(rng)
        if k and np.min(np.sum((pts[:k] - c) ** 2, axis=1)) < min_dist * min_dist:
            continue
        pts[k] = c
        k += 1
    return pts.astype(np.float32)


def place_in_cube(rng, n: int, side: float) -> np.ndarray:
    return _place(rng, n, lambda r: r.uniform(0.0, side, size=3))


def place_in_ball(rng, n: int, radius: float) -> np.ndarray:
    def draw(r):
        while True:
            c = r.uniform(-radius, radius, size=3)
            if float(c @ c) <= radius * radius:
                return c

    return _place(rng, n, draw)


def place_waters(rng, n_mol: int, side: float) -> np.ndarray:
    """Rigid O-H-H triples (O-H 0.96 A, H-O-H 104.5 deg), random orientation, whole
    molecule inside the cube, inter-molecular atom distance >= MIN_DIST (S17)."""
    half = math.radians(104.5) / 2.0
    local = np.array(
        [
            [0.0, 0.0, 0.0],
            [0.96 * math.sin(half), 0.96 * math.cos(half), 0.0],
            [-0.96 * math.sin(half), 0.96 * math.cos(half), 0.0],
        ]
    )
    cell = 2.0  # coarse grid over molecule centres for the rejection test
    ncell = int(math.ceil(side / cell))
    grid = {}
    out = np.empty((n_mol * 3, 3), dtype=np.float64)
    k = 0
    tries = 0
    md2 = MIN_DIST * MIN_DIST
    while k < n_mol:
        tries += 1
        if tries > 200 * n_mol:
            raise RuntimeError("water placement did not converge")
        q = rng.normal(size=4)
        q /= np.linalg.norm(q)
        w, x, y, z = q
        R = np.array(
            [
                [1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)],
            ]
        )
        o = rng.uniform(0.0, side, size=3)
        mol = o + local @ R.T
        if mol.min() < 0.0 or mol.max() > side:
            continue
        ci = np.minimum((o / cell).astype(int), ncell - 1)
        ok = True
        for dx in (-2, -1, 0, 1, 2):
            for dy in (-2, -1, 0, 1, 2):
                for dz in (-2, -1, 0, 1, 2):
                    for idx in grid.get((ci[0] + dx, ci[1] + dy, ci[2] + dz), ()):
                        other = out[3 * idx : 3 * idx + 3]
                        d2 = np.sum((other[:, None, :] - mol[None, :, :]) ** 2, axis=2)
                        if d2.min() < md2:
                            ok = False
                            break
                    if not ok:
                        break
                if not ok:
                    break
            if not ok:
                break
        if not ok:
            continue
        out[3 * k : 3 * k + 3] = mol
        grid.setdefault((ci[0], ci[1], ci[2]), []).append(k)
        k += 1
    return out.astype(np.float32)


@dataclasses.dataclass
class Workload:
    name: str
    config: int  # 1-based index into BASELINE.json configs
    positions: np.ndarray  # f32[N,3], Angstrom
    species: np.ndarray  # i32[N], index into SPECIES
    mol_offsets: np.ndarray  # i32[n_mol+1], CSR
    n_models: int
    n_steps: int  # consecutive evaluations the config asks for
    weight_seed: int
    perturb_seed: int
    params: AniParams

    @property
    def n_atoms(self) -> int:
        return int(self.positions.shape[0])

    @property
    def n_molecules(self) -> int:
        return int(self.mol_offsets.size - 1)

    def weights(self, random_biases: bool = False):
        return make_weights(self.params, self.n_models, self.weight_seed, random_biases)

    def trajectory(self, n_steps: int | None = None) -> np.ndarray:
        """f32[n_steps,N,3]: step 0 is ``positions``; x_t = f32(x_{t-1} + 0.005*xi_t) (S18)."""
        n = self.n_steps if n_steps is None else n_steps
        rng = np.random.default_rng(self.perturb_seed)
        traj = np.empty((n, self.n_atoms, 3), dtype=np.float32)
        traj[0] = self.positions
        for t in range(1, n):
            noise = rng.normal(0.0, 0.005, size=(self.n_atoms, 3)).astype(np.float32)
            traj[t] = traj[t - 1] + noise
        return traj


def _seeds(c: int):
    b = BASE_SEED + 10 * c
    return dict(pos=b, species=b + 1, weights=b + 2, perturb=b + 3, sizes=b + 4)


def config1() -> Workload:
    """12 atoms, H/C/N/O 50/30/10/10, 6 A cube, 1 model, 1 evaluation (BASELINE.json configs[0])."""
    s = _seeds(1)
    pos = place_in_cube(np.random.default_rng(s["pos"]), 12, 6.0)
    spc = make_species(12, (0.5, 0.3, 0.1, 0.1), s["species"])
    return Workload("tiny12", 1, pos, spc, np.array([0, 12], np.int32), 1, 1, s["weights"], s["perturb"], ani2x_params())


def config2(radius: float = 6.0, n_models: int = 8) -> Workload:
    """50 atoms, H/C/N/O/S/F/Cl 45/33/8/8/2/2/2, 12 A-diameter ball, 8 models, 1000 steps
    (BASELINE.json configs[1]; S15: 12 A is read as the diameter)."""
    s = _seeds(2)
    pos = place_in_ball(np.random.default_rng(s["pos"]), 50, radius)
    # fractions in index order H,C,N,O,F,S,Cl (S5: the config lists S before F as labels)
    spc = make_species(50, (0.45, 0.33, 0.08, 0.08, 0.02, 0.02, 0.02), s["species"])
    return Workload("ligand50", 2, pos, spc, np.array([0, 50], np.int32), n_models, 1000, s["weights"], s["perturb"], ani2x_params())


def config3(n_mol: int = 256, n_models: int = 8) -> Workload:
    """256 molecules of 30..70 atoms, species/placement as config 1 (literal 6 A cube, S16)."""
    s = _seeds(3)
    sizes = np.random.default_rng(s["sizes"]).integers(30, 71, size=n_mol)
    rng_p = np.random.default_rng(s["pos"])
    rng_s = np.random.default_rng(s["species"])
    pos, spc = [], []
    for n in sizes:
        pos.append(place_in_cube(rng_p, int(n), 6.0))
        cnt = species_counts(int(n), (0.5, 0.3, 0.1, 0.1))
        sp = np.concatenate([np.full(c, e, dtype=np.int32) for e, c in enumerate(cnt)])
        rng_s.shuffle(sp)
        spc.append(sp)
    off = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int32)
    return Workload("batch256", 3, np.concatenate(pos), np.concatenate(spc), off, n_models, 1, s["weights"], s["perturb"], ani2x_params())


def config4(n: int = 500, n_models: int = 8) -> Workload:
    """500 atoms H/C/N/O 50/30/10/10 at 0.1 atoms/A^3 in a cube, 100 steps."""
    s = _seeds(4)
    side = (n / 0.1) ** (1.0 / 3.0)
    pos = place_in_cube(np.random.default_rng(s["pos"]), n, side)
    spc = make_species(n, (0.5, 0.3, 0.1, 0.1), s["species"])
    return Workload("large500", 4, pos, spc, np.array([0, n], np.int32), n_models, 100, s["weights"], s["perturb"], ani2x_params())


def config5(n_mol: int = 3333, n_models: int = 8) -> Workload:
    """3333 rigid waters (9999 atoms, order O,H,H) at 0.1 atoms/A^3 in a cube (S17)."""
    s = _seeds(5)
    n = 3 * n_mol
    side = (n / 0.1) ** (1.0 / 3.0)
    pos = place_waters(np.random.default_rng(s["pos"]), n_mol, side)
    spc = np.tile(np.array([3, 0, 0], dtype=np.int32), n_mol)
    return Workload("water10k", 5, pos, spc, np.array([0, n], np.int32), n_models, 1, s["weights"], s["perturb"], ani2x_params())


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}


def get_config(c: int) -> Workload:
    return CONFIGS[c]()


def random_molecule(n: int, n_species: int, seed: int, side: float | None = None, params: AniParams | None = None,
                    n_models: int = 1) -> Workload:
    """Generic seeded test molecule: uniform species over ``n_species``, cube placement."""
    rng = np.random.default_rng(seed)
    if side is None:
        side = max(3.0, (n / 0.06) ** (1.0 / 3.0))
    pos = place_in_cube(rng, n, side)
    spc = rng.integers(0, n_species, size=n).astype(np.int32)
    p = params if params is not None else ani2x_params()
    return Workload(f"rand{n}", 0, pos, spc, np.array([0, n], np.int32), n_models, 1, seed + 2, seed + 3, p)


# ------------------------------------------------------------------------------------------------
# NNP/MM system for the coupling term (Eq. 4): the ligand-sized NNP region of configs[1] inside
# an MM environment of water-like density.  The paper's systems (Table 1: 48-75 ligand atoms in
# 26-40 thousand-atom solvated complexes) are not in this container; this generator takes their sizes.  Charges and
# Lennard-Jones parameters are drawn in the ranges of a biomolecular force field; no arithmetic of the method here.
@dataclasses.dataclass(frozen=True)
class CouplingSystem:
    positions: np.ndarray  # f32[n_rows][3], A; rows of NNP and MM atoms interleaved at random
    nnp_rows: np.ndarray   # i32[n_nnp]
    mm_rows: np.ndarray    # i32[n_mm]
    q_nnp: np.ndarray      # f32, e
    sigma_nnp: np.ndarray  # f32, A
    eps_nnp: np.ndarray    # f32, kcal/mol
    q_mm: np.ndarray
    sigma_mm: np.ndarray
    eps_mm: np.ndarray

    @property
    def n_rows(self) -> int:
        return int(self.positions.shape[0])


def coupling_system(n_mm: int = 30000, seed: int = BASE_SEED + 77, density: float = 0.1,
                    min_dist: float = 1.6) -> CouplingSystem:
    """configs[1]'s 50-atom NNP region at the centre of a cube of n_mm MM atoms at `density` atoms/A^3; MM atoms keep
    `min_dist` from the NNP atoms (no clash with the ligand), not from each other (MM-MM pairs are not in Eq. 4)."""
    rng = np.random.default_rng(seed)
    lig = config2()
    n_nnp = lig.n_atoms
    side = ((n_mm + n_nnp) / density) ** (1.0 / 3.0)
    nnp_pos = lig.positions.astype(np.float64)  # centred at the origin (ball of radius 6 A)
    mm = np.empty((0, 3))
    while mm.shape[0] < n_mm:
        cand = rng.uniform(-side / 2, side / 2, size=(2 * (n_mm - mm.shape[0]) + 64, 3))
        near = cand[np.abs(cand).max(axis=1) < 8.0]
        ok = np.ones(cand.shape[0], bool)
        idx = np.nonzero(np.abs(cand).max(axis=1) < 8.0)[0]
        if idx.size:
            d = np.linalg.norm(near[:, None, :] - nnp_pos[None, :, :], axis=2).min(axis=1)
            ok[idx[d < min_dist]] = False
        mm = np.concatenate([mm, cand[ok]])[:n_mm]
    n_rows = n_nnp + n_mm
    perm = rng.permutation(n_rows).astype(np.int32)
    pos = np.empty((n_rows, 3), np.float32)
    nnp_rows, mm_rows = perm[:n_nnp].copy(), perm[n_nnp:].copy()
    pos[nnp_rows] = nnp_pos.astype(np.float32)
    pos[mm_rows] = mm.astype(np.float32)
    f32 = lambda lo, hi, n: rng.uniform(lo, hi, size=n).astype(np.float32)
    return CouplingSystem(pos, nnp_rows, mm_rows, f32(-0.6, 0.6, n_nnp), f32(1.0, 3.6, n_nnp), f32(0.01, 0.25, n_nnp),
                          f32(-0.9, 0.9, n_mm), f32(0.4, 3.6, n_mm), f32(0.0, 0.25, n_mm))


# ------------------------------------------------------------------------------------------------
# ANI-1x as a second parameter set (Table 4: "ANI-1x" on the 3BE9 ligand): 4 elements H, C, N, O ->
# 4*16 + 10*32 = 384 features, its own AEV constants and narrower networks.  Values: the published ANI-1x
# hyper-parameters; trained weights are not in this container (seeded Xavier weights stand in, as for ANI-2x).
ANI1X_ATOMIC_NUMBERS = (1, 6, 7, 8)
ANI2X_ATOMIC_NUMBERS = (1, 6, 7, 8, 9, 16, 17)


def ani1x_params() -> AniParams:
    f32 = np.float32
    hidden = {"H": (160, 128, 96), "C": (144, 112, 96), "N": (128, 112, 96), "O": (128, 112, 96)}
    n_feat = 4 * 16 + 10 * 32
    dims = np.array([[n_feat, *hidden[s], 1] for s in ("H", "C", "N", "O")], dtype=np.int32)
    return AniParams(
        n_species=4,
        rc_radial=f32(5.2),
        rc_angular=f32(3.5),
        eta_r=f32(16.0),
        shf_r=(0.9 + 0.26875 * np.arange(16, dtype=np.float64)).astype(f32),
        eta_a=f32(8.0),
        zeta=f32(32.0),
        shf_a=(0.9 + 0.65 * np.arange(4, dtype=np.float64)).astype(f32),
        shf_z=((2.0 * np.arange(8, dtype=np.float64) + 1.0) * math.pi / 16.0).astype(f32),
        cos_scale=f32(0.95),
        celu_alpha=f32(0.1),
        layer_dims=dims,
        energy_scale=627.5094740631,
    )


def ani1x_ligand(n: int = 48, n_models: int = 8) -> Workload:
    """A 3BE9-ligand-sized region (48 atoms) of H/C/N/O at 50/30/10/10 % in a ball of radius 6 A."""
    b = BASE_SEED + 60
    pos = place_in_ball(np.random.default_rng(b), n, 6.0)
    spc = make_species(n, (0.5, 0.3, 0.1, 0.1), b + 1)
    return Workload(f"ani1x_ligand{n}", 0, pos, spc, np.array([0, n], np.int32), n_models, 100, b + 2, b + 3, ani1x_params())

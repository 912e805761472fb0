"""Pins of the float64 CPU oracle (oracle/ani_oracle.c) against things other than itself.

Each test names the definition it pins (O1-O7 of SURVEY.md 8(c) / DESIGN.md "Readings") and the
kind of pin: closed form, brute force, textbook routine, invariant, finite difference.
A plausible mistake (dropped term, wrong sign/index, transposed operand) must fail one of them.
No GPU, no CUDA code is touched here.
"""
import math

import numpy as np
import pytest

from oracle.ani_oracle import AniOracle
from paper_2201_08110_b200 import workloads as wl


def _zero_weights(params, n_models=1):
    W, B = wl.make_weights(params, n_models, seed=1)
    return W, B


@pytest.fixture(scope="module")
def ani():
    p = wl.ani2x_params()
    W, B = wl.make_weights(p, 1, seed=11)
    return p, AniOracle(p, W, B)


@pytest.fixture(scope="module")
def small():
    p = wl.small_params(n_species=3, hidden=(16, 12, 8))
    W, B = wl.make_weights(p, 2, seed=5, random_biases=True)
    return p, W, B, AniOracle(p, W, B)


# ---------------------------------------------------------------- O1-O3: radial closed forms
def test_radial_dimer_closed_form(ani, golden):
    """O1+O3 closed form: dimer H-C at r=0.8 and r=1.0 (tests/golden)."""
    p, orc = ani
    for r, keys in ((0.8, {0: "dimer_r0.8_k0"}),
                    (1.0, {0: "dimer_r1.0_k0", 1: "dimer_r1.0_k1", 2: "dimer_r1.0_k2", 3: "dimer_r1.0_k3"})):
        pos = np.array([[0, 0, 0], [r, 0, 0]], dtype=np.float64)
        spc = np.array([0, 1], dtype=np.int32)  # H centre, C neighbour
        G = orc.aev(pos, spc)
        # entries live in the radial block of the NEIGHBOUR's species
        for k, key in keys.items():
            assert G[0, 1 * 16 + k] == pytest.approx(golden[key], rel=2e-6)
            assert G[1, 0 * 16 + k] == pytest.approx(golden[key], rel=2e-6)
        nz = np.flatnonzero(G[0])
        assert nz.min() >= 16 and nz.max() < 32  # only block of species C
        if r == 1.0:
            assert G[0, 16:32].sum() == pytest.approx(golden["dimer_r1.0_sum16"], rel=2e-6)
        assert np.all(G[:, 112:] == 0.0)  # no triplet, no angular term


def test_radial_prefactor_and_cutoff_value(ani):
    """O1/O3 special case: r = ShfR_0 makes exp(0)=1, so G = 0.25*f_C(r) exactly (S2 prefactor)."""
    p, orc = ani
    r = float(np.float64(p.shf_r[0]))
    pos = np.array([[0, 0, 0], [0, r, 0]], dtype=np.float64)
    G = orc.aev(pos, np.array([0, 0], np.int32))
    rc = float(np.float64(p.rc_radial))
    assert G[0, 0] == pytest.approx(0.25 * (0.5 * math.cos(math.pi * r / rc) + 0.5), rel=1e-14)


# ---------------------------------------------------------------- O4: angular closed forms
def test_angular_right_angle_trimer(ani, golden):
    """O4 closed form: centre at origin, j=(1,0,0), k=(0,1.2,0): theta = pi/2 exactly."""
    p, orc = ani
    pos = np.array([[0, 0, 0], [1.0, 0, 0], [0, 1.2, 0]], dtype=np.float64)
    spc = np.zeros(3, np.int32)
    G = orc.aev(pos, spc)
    blk = G[0, 112:144].reshape(8, 4)
    for a in (0, 1):
        for z in range(4):
            assert blk[a, z] == pytest.approx(golden[f"rtrimer_a{a}_z{z}"], rel=2e-6)
    assert blk.sum() == pytest.approx(golden["rtrimer_sum32"], rel=2e-6)
    # z <-> 3-z symmetry at theta = pi/2 (ShfZ symmetric about pi/2); f32-widened ShfZ break it at ~1e-7
    assert np.allclose(blk[:, 0], blk[:, 3], rtol=1e-5) and np.allclose(blk[:, 1], blk[:, 2], rtol=1e-5)


def test_angular_equilateral(ani, golden):
    """O4 closed form + S6 (0.95 scaling): equilateral side 1.0 => theta = arccos(0.475)."""
    p, orc = ani
    h = math.sqrt(3.0) / 2.0
    pos = np.array([[0, 0, 0], [1.0, 0, 0], [0.5, h, 0]], dtype=np.float64)
    G = orc.aev(pos, np.zeros(3, np.int32))
    blk = G[0, 112:144].reshape(8, 4)
    for z in range(4):
        assert blk[0, z] == pytest.approx(golden[f"equi_a0_z{z}"], rel=3e-6)
    assert blk.sum() == pytest.approx(golden["equi_sum32"], rel=3e-6)
    # all three centres see the same environment
    assert np.allclose(G[0], G[1], rtol=1e-12, atol=1e-15) and np.allclose(G[0], G[2], rtol=1e-12, atol=1e-15)


def test_angular_layout_species_pair_block(ani):
    """S4 layout: trimer (H; C, O) -> only angular block p(1,3)=9 is non-zero; 2*16+32 = 64 non-zeros."""
    p, orc = ani
    pos = np.array([[0, 0, 0], [1.0, 0.1, 0], [-0.3, 1.1, 0.2]], dtype=np.float64)
    G = orc.aev(pos, np.array([0, 1, 3], np.int32))
    row = G[0]
    nz = np.flatnonzero(row)
    assert len(nz) == 64
    ang = nz[nz >= 112]
    assert ang.min() == 112 + 9 * 32 and ang.max() == 112 + 9 * 32 + 31
    rad = nz[nz < 112]
    assert set(rad // 16) == {1, 3}
    # unordered pair: swapping the two neighbours' species gives the same block
    G2 = orc.aev(pos, np.array([0, 3, 1], np.int32))
    assert np.flatnonzero(G2[0][112:]).min() == 9 * 32


def test_pair_index_all_blocks(ani):
    """S4: p(s,t) = s*S - s(s-1)/2 + (t-s) enumerates the upper triangle row-major: (H,H)=0..(Cl,Cl)=27."""
    p, orc = ani
    expected = {}
    idx = 0
    for s in range(7):
        for t in range(s, 7):
            expected[(s, t)] = idx
            idx += 1
    assert idx == 28
    pos = np.array([[0, 0, 0], [1.0, 0, 0], [0, 1.0, 0]], dtype=np.float64)
    for (s, t), blk in expected.items():
        for order in ((s, t), (t, s)):
            G = orc.aev(pos, np.array([0, order[0], order[1]], np.int32))
            nz = np.flatnonzero(G[0][112:])
            assert nz.min() // 32 == blk and nz.max() // 32 == blk


# ---------------------------------------------------------------- O2-O4: brute-force enumeration
def _brute_force_aev(p, pos, spc):
    """Plain O(N^3) loops with explicit distance tests, numpy float64 -- independent of the C code."""
    S = p.n_species
    n = len(pos)
    f = lambda v: float(np.float64(np.float32(v)))
    shf_r = [f(v) for v in p.shf_r]
    shf_a = [f(v) for v in p.shf_a]
    shf_z = [f(v) for v in p.shf_z]
    rcr, rca = f(p.rc_radial), f(p.rc_angular)
    eta_r, eta_a, zeta, cs = f(p.eta_r), f(p.eta_a), f(p.zeta), f(p.cos_scale)
    nf = S * 16 + S * (S + 1) // 2 * 32
    G = np.zeros((n, nf))
    fc = lambda r, rc: 0.5 * math.cos(math.pi * r / rc) + 0.5
    pairs = [(s, t) for s in range(S) for t in range(s, S)]
    for i in range(n):
        for j in range(n):
            if j == i:
                continue
            rij = math.dist(pos[i], pos[j])
            if rij <= rcr:
                for k in range(16):
                    G[i, spc[j] * 16 + k] += 0.25 * math.exp(-eta_r * (rij - shf_r[k]) ** 2) * fc(rij, rcr)
            for k in range(n):
                if k == i or k <= j:
                    continue
                rik = math.dist(pos[i], pos[k])
                if rij > rca or rik > rca:
                    continue
                a = pos[j] - pos[i]
                b = pos[k] - pos[i]
                th = math.acos(cs * float(a @ b) / (rij * rik))
                blk = pairs.index((min(spc[j], spc[k]), max(spc[j], spc[k])))
                for ia in range(8):
                    F2 = math.exp(-eta_a * ((rij + rik) / 2 - shf_a[ia]) ** 2)
                    for iz in range(4):
                        F1 = ((1 + math.cos(th - shf_z[iz])) / 2) ** zeta
                        G[i, S * 16 + blk * 32 + ia * 4 + iz] += 2 * F1 * F2 * fc(rij, rca) * fc(rik, rca)
    return G


@pytest.mark.parametrize("seed,n", [(1, 5), (2, 9), (3, 12)])
def test_aev_brute_force_triplets(small, seed, n):
    """O2-O4 brute force: O(N^3) enumeration in pure Python must equal the oracle to 1e-13."""
    p, W, B, orc = small
    w = wl.random_molecule(n, p.n_species, seed=seed, side=4.5, params=p)
    pos = w.positions.astype(np.float64)
    G = orc.aev(pos, w.species)
    Gb = _brute_force_aev(p, pos, w.species)
    assert G.shape == Gb.shape
    assert np.max(np.abs(G - Gb)) <= 1e-13 * max(1.0, np.max(np.abs(Gb)))
    assert np.count_nonzero(Gb[:, p.n_species * 16:]) > 0  # the case has triplets


def test_aev_brute_force_config1():
    """Same pin on BASELINE.json configs[0] (12 atoms, 7-species layout, 1008 features)."""
    w = wl.config1()
    W, B = w.weights()
    orc = AniOracle(w.params, W, B)
    pos = w.positions.astype(np.float64)
    G = orc.aev(pos, w.species)
    Gb = _brute_force_aev(w.params, pos, w.species)
    assert G.shape == (12, 1008)
    assert np.max(np.abs(G - Gb)) <= 1e-13


def test_molecules_do_not_interact(small):
    """O2 'same molecule': two overlapping molecules in one batch give each molecule's own AEV."""
    p, W, B, orc = small
    a = wl.random_molecule(6, p.n_species, seed=21, side=3.5, params=p)
    b = wl.random_molecule(7, p.n_species, seed=22, side=3.5, params=p)
    pos = np.concatenate([a.positions, b.positions])
    spc = np.concatenate([a.species, b.species])
    off = np.array([0, 6, 13], np.int32)
    G = orc.aev(pos, spc, off)
    assert np.array_equal(G[:6], orc.aev(a.positions, a.species))
    assert np.array_equal(G[6:], orc.aev(b.positions, b.species))
    r = orc.energy_forces(pos, spc, off)
    ra = orc.energy_forces(a.positions, a.species)
    rb = orc.energy_forces(b.positions, b.species)
    assert r["E"][0] == ra["E"][0] and r["E"][1] == rb["E"][0]
    assert np.array_equal(r["F"][:6], ra["F"]) and np.array_equal(r["F"][6:], rb["F"])


# ---------------------------------------------------------------- O2: pair predicate
def test_pairs_predicate_inclusive_and_exact(ani):
    """O2/S1: D2 <= Rc^2 in binary64 on f32-widened inputs; r == Rc is included, next f32 up is not."""
    p, orc = ani
    rc = np.float32(5.1)
    up = np.nextafter(rc, np.float32(10))
    pos = np.array([[0, 0, 0], [rc, 0, 0], [0, up, 0]], dtype=np.float32)
    ij = orc.pairs(pos, "radial")
    assert ij.tolist() == [[0, 1]]
    rca = np.float32(3.5)
    pos = np.array([[0, 0, 0], [0, 0, rca], [np.nextafter(rca, np.float32(10)), 0, 0]], dtype=np.float32)
    assert orc.pairs(pos, "angular").tolist() == [[0, 1]]


def test_pairs_match_numpy(ani):
    """O2 brute force with numpy float64 using the defined operation order (dx*dx + dy*dy) + dz*dz."""
    p, orc = ani
    w = wl.config4(n=120)
    pos = w.positions.astype(np.float64)
    d = pos[None, :, :] - pos[:, None, :]
    D2 = (d[..., 0] * d[..., 0] + d[..., 1] * d[..., 1]) + d[..., 2] * d[..., 2]
    for which, rc in (("radial", 5.1), ("angular", 3.5)):
        rc64 = float(np.float64(np.float32(rc)))
        iu, ju = np.nonzero(np.triu(D2 <= rc64 * rc64, k=1))
        want = np.stack([iu, ju], axis=1)
        got = orc.pairs(w.positions, which)
        assert np.array_equal(got, want)


# ---------------------------------------------------------------- O5: MLP vs textbook matmul
def _np_celu(x, alpha):
    return np.where(x > 0, x, alpha * np.expm1(np.minimum(x, 0) / alpha))


def test_mlp_matches_numpy_matmul(ani):
    """O5 reduces to dense float64 matmul + CELU: compare with numpy `x @ W.T` on random rows."""
    p, orc = ani
    W, B = wl.make_weights(p, 2, seed=3, random_biases=True)
    o = AniOracle(p, W, B)
    rng = np.random.default_rng(0)
    n = 9
    spc = np.array([0, 1, 2, 3, 4, 5, 6, 0, 1], np.int32)
    G = rng.uniform(0, 0.6, size=(n, 1008)) * (rng.uniform(size=(n, 1008)) < 0.2)
    e, dG = o.mlp(G, spc)
    alpha = float(np.float64(p.celu_alpha))
    for m in range(2):
        for i in range(n):
            h = G[i]
            for l in range(4):
                z = W[m][spc[i]][l].astype(np.float64) @ h + B[m][spc[i]][l].astype(np.float64)
                h = _np_celu(z, alpha) if l < 3 else z
            assert e[m, i] == pytest.approx(h[0], rel=1e-12, abs=1e-14)


def test_mlp_input_gradient_matches_numpy_chain(small):
    """O7 (MLP part): dE/dG = mean_m W1^T(CELU' . W2^T(CELU' . W3^T(CELU' . W4^T))) via numpy."""
    p, W, B, orc = small
    rng = np.random.default_rng(4)
    n = 5
    spc = np.array([0, 1, 2, 1, 0], np.int32)
    G = rng.uniform(-0.5, 0.8, size=(n, orc.n_features))
    e, dG = orc.mlp(G, spc)
    alpha = float(np.float64(p.celu_alpha))
    for i in range(n):
        acc = np.zeros(orc.n_features)
        for m in range(2):
            hs, zs = [G[i]], []
            for l in range(4):
                z = W[m][spc[i]][l].astype(np.float64) @ hs[-1] + B[m][spc[i]][l].astype(np.float64)
                zs.append(z)
                hs.append(_np_celu(z, alpha) if l < 3 else z)
            d = np.ones(1)
            for l in range(3, -1, -1):
                d = W[m][spc[i]][l].astype(np.float64).T @ d
                if l > 0:
                    d = d * np.where(zs[l - 1] > 0, 1.0, np.exp(zs[l - 1] / alpha))
            acc += d / 2
        assert np.allclose(dG[i], acc, rtol=1e-12, atol=1e-15)


def test_celu_special_values():
    """O5: CELU(0)=0, CELU(x>0)=x, CELU(-inf) -> -alpha, continuity of CELU' at 0 (1-layer 'network')."""
    p = wl.small_params(n_species=1, hidden=(1, 1, 1))
    nf = 16 + 32
    W = [[[np.zeros((1, nf), np.float32), np.ones((1, 1), np.float32), np.ones((1, 1), np.float32),
           np.ones((1, 1), np.float32)]]]
    W[0][0][0][0, 0] = 1.0
    o = AniOracle(p, W, None)
    a = float(np.float64(p.celu_alpha))
    c1 = lambda x: x if x > 0 else a * math.expm1(x / a)
    for x in (0.0, 0.3, -0.05, -50.0):
        G = np.zeros((1, nf))
        G[0, 0] = x
        e, dG = o.mlp(G, np.zeros(1, np.int32))
        assert e[0, 0] == pytest.approx(c1(c1(c1(x))), rel=1e-12, abs=1e-300)
    G = np.zeros((1, nf)); G[0, 0] = -50.0
    assert o.mlp(G, np.zeros(1, np.int32))[0][0, 0] == pytest.approx(c1(c1(-a)), rel=1e-9)
    for eps in (1e-12, -1e-12):
        G[0, 0] = eps
        assert o.mlp(G, np.zeros(1, np.int32))[1][0, 0] == pytest.approx(1.0, abs=1e-9)


# ---------------------------------------------------------------- O6: ensemble
def test_ensemble_identities():
    """O6/S7: M identical copies reproduce the M=1 energy; permuting models changes nothing;
    the ensemble energy is the mean of the single-model energies."""
    p = wl.small_params()
    W, B = wl.make_weights(p, 3, seed=9, random_biases=True)
    w = wl.random_molecule(10, p.n_species, seed=31, side=4.5, params=p)
    one = AniOracle(p, W[:1], B[:1]).energy_forces(w.positions, w.species)
    same = AniOracle(p, [W[0]] * 4, [B[0]] * 4).energy_forces(w.positions, w.species)
    assert same["E"][0] == pytest.approx(one["E"][0], rel=1e-14)
    assert np.allclose(same["F"], one["F"], rtol=1e-13, atol=1e-13)
    full = AniOracle(p, W, B).energy_forces(w.positions, w.species)
    perm = AniOracle(p, [W[2], W[0], W[1]], [B[2], B[0], B[1]]).energy_forces(w.positions, w.species)
    assert perm["E"][0] == pytest.approx(full["E"][0], rel=1e-13)
    singles = [AniOracle(p, [W[m]], [B[m]]).energy_forces(w.positions, w.species) for m in range(3)]
    assert full["E"][0] == pytest.approx(np.mean([s["E"][0] for s in singles]), rel=1e-13)
    assert np.allclose(full["F"], np.mean([s["F"] for s in singles], axis=0), rtol=1e-12, atol=1e-12)


def test_self_energy_and_scale():
    """O6/S12/S8: E = scale * sum_i (e_i + E_self[s_i]); forces scale with energy_scale, not with E_self."""
    p = wl.small_params()
    W, B = wl.make_weights(p, 1, seed=2)
    w = wl.random_molecule(8, p.n_species, seed=33, side=4.0, params=p)
    base = AniOracle(p, W, B, energy_scale=1.0).energy_forces(w.positions, w.species)
    se = np.array([0.5, -1.25, 2.0])
    r = AniOracle(p, W, B, self_energy=se, energy_scale=3.0).energy_forces(w.positions, w.species)
    assert r["E"][0] == pytest.approx(3.0 * (base["E"][0] + se[w.species].sum()), rel=1e-13)
    assert np.allclose(r["F"], 3.0 * base["F"], rtol=1e-13, atol=1e-14)


def test_energy_is_sum_of_atomic_energies(small):
    p, W, B, orc = small
    w = wl.random_molecule(11, p.n_species, seed=35, side=4.5, params=p)
    r = orc.energy_forces(w.positions, w.species, want_intermediates=True)
    assert r["E"][0] == pytest.approx(p.energy_scale * r["e_atom"].mean(axis=0).sum(), rel=1e-13)
    e2, dG2 = orc.mlp(r["G"], w.species)
    assert np.array_equal(e2, r["e_atom"]) and np.array_equal(dG2, r["dG"])


# ---------------------------------------------------------------- O7: forces
def _fd_forces(orc, pos, spc, h=1e-5, off=None):
    F = np.zeros_like(pos)
    for a in range(pos.shape[0]):
        for x in range(3):
            pp = pos.copy(); pp[a, x] += h
            pm = pos.copy(); pm[a, x] -= h
            F[a, x] = -(orc.energy(pp, spc, off).sum() - orc.energy(pm, spc, off).sum()) / (2 * h)
    return F


def test_forces_central_finite_difference_small(small):
    """O7 / PAPER.md Eq. 3: F = -grad V.  Central FD (h=1e-5 A, f64 positions) to 1e-6 * max|F|."""
    p, W, B, orc = small
    w = wl.random_molecule(9, p.n_species, seed=41, side=4.2, params=p)
    pos = w.positions.astype(np.float64)
    F = orc.energy_forces(pos, w.species)["F"]
    Ffd = _fd_forces(orc, pos, w.species)
    assert np.max(np.abs(F)) > 1e-3
    assert np.max(np.abs(F - Ffd)) <= 1e-6 * np.max(np.abs(F))


def test_forces_central_finite_difference_ani2x():
    """Same pin with the full ANI-2x shapes on BASELINE.json configs[0] (12 atoms, 1008 features)."""
    w = wl.config1()
    W, B = w.weights(random_biases=True)
    orc = AniOracle(w.params, W, B)
    pos = w.positions.astype(np.float64)
    F = orc.energy_forces(pos, w.species)["F"]
    Ffd = _fd_forces(orc, pos, w.species)
    assert np.max(np.abs(F - Ffd)) <= 1e-6 * np.max(np.abs(F))


def test_forces_fd_radial_only_and_angular_only(ani):
    """Separates the radial and the angular derivative: a dimer has no triplet; an isolated
    trimer with g concentrated on angular features exercises only the angular chain."""
    p, orc = ani
    pos = np.array([[0, 0, 0], [1.1, 0.2, -0.1]], dtype=np.float64)
    spc = np.array([1, 3], np.int32)
    F = orc.energy_forces(pos, spc)["F"]
    assert np.max(np.abs(F - _fd_forces(orc, pos, spc))) <= 1e-6 * np.max(np.abs(F))
    # zero the radial columns of layer 1 => the energy depends on angular terms only
    W, B = wl.make_weights(p, 1, seed=12)
    for e in range(7):
        W[0][e][0][:, :112] = 0.0
    o2 = AniOracle(p, W, B)
    pos = np.array([[0, 0, 0], [1.0, 0.1, 0], [-0.3, 1.1, 0.2], [0.9, 1.0, -0.8]], dtype=np.float64)
    spc = np.array([0, 1, 3, 0], np.int32)
    F = o2.energy_forces(pos, spc)["F"]
    assert np.max(np.abs(F)) > 1e-4
    assert np.max(np.abs(F - _fd_forces(o2, pos, spc))) <= 1e-6 * np.max(np.abs(F))


def test_net_force_and_torque_vanish(small):
    """Translation/rotation invariance of V (Eq. 2) => sum F = 0, sum r x F = 0."""
    p, W, B, orc = small
    w = wl.random_molecule(14, p.n_species, seed=43, side=5.0, params=p)
    pos = w.positions.astype(np.float64)
    F = orc.energy_forces(pos, w.species)["F"]
    scale = np.max(np.abs(F))
    assert np.max(np.abs(F.sum(axis=0))) <= 1e-12 * scale
    assert np.max(np.abs(np.cross(pos, F).sum(axis=0))) <= 1e-11 * scale


def test_invariance_rotation_translation_permutation(small):
    """V depends only on positions and atomic numbers of the region."""
    p, W, B, orc = small
    w = wl.random_molecule(12, p.n_species, seed=47, side=4.8, params=p)
    pos = w.positions.astype(np.float64)
    r0 = orc.energy_forces(pos, w.species)
    rng = np.random.default_rng(5)
    q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    pos2 = pos @ q.T + np.array([3.0, -2.0, 0.7])
    r1 = orc.energy_forces(pos2, w.species)
    assert r1["E"][0] == pytest.approx(r0["E"][0], rel=1e-11)
    assert np.allclose(r1["F"], r0["F"] @ q.T, rtol=0, atol=1e-10 * np.max(np.abs(r0["F"])))
    perm = rng.permutation(12)
    r2 = orc.energy_forces(pos[perm], w.species[perm])
    assert r2["E"][0] == pytest.approx(r0["E"][0], rel=1e-12)
    assert np.allclose(r2["F"], r0["F"][perm], rtol=0, atol=1e-11 * np.max(np.abs(r0["F"])))


def test_cutoff_continuity(ani):
    """O1: f_C and f_C' vanish at Rc => E and F are continuous when a pair crosses either cutoff.
    Across 2e-9 A the energy may only change by the smooth first-order amount -F.dr (the pair that
    crosses the 3.5 A angular cutoff is still inside the 5.1 A radial one); a missing f_C or f_C'
    factor would jump by > 1e-3."""
    p, orc = ani
    base = np.array([[0, 0, 0], [1.2, 0, 0], [0.2, 1.3, 0.1]], dtype=np.float64)
    spc = np.array([0, 1, 2, 3], np.int32)
    eps = 1e-9
    for rc in (5.1, 3.5):
        rc64 = float(np.float64(np.float32(rc)))
        out = []
        for e in (-eps, eps):
            pos = np.vstack([base, [[0, 0, rc64 + e]]])
            out.append(orc.energy_forces(pos, spc))
        fz = 0.5 * (out[0]["F"][3, 2] + out[1]["F"][3, 2])
        assert abs(out[1]["E"][0] - out[0]["E"][0] + fz * 2 * eps) <= 1e-11
        assert np.max(np.abs(out[0]["F"] - out[1]["F"])) <= 1e-6


def test_bad_inputs_are_rejected(small):
    p, W, B, orc = small
    pos = np.zeros((2, 3)); pos[1, 0] = 1.0
    with pytest.raises(ValueError):
        orc.energy_forces(pos, np.array([0, 7], np.int32))
    with pytest.raises(ValueError):
        orc.energy_forces(pos, np.array([0, 1], np.int32), np.array([0, 1], np.int32))

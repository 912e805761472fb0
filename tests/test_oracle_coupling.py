"""Pins of oracle/coupling_oracle.c (Eq. 4) against what the formula and mechanics fix: two-atom
closed forms, the zero and the minimum of the Lennard-Jones term, central finite differences of the energy, Newton's
third law, zero net torque, "only NNP-MM pairs", the Lorentz-Berthelot combination (reading C1) and the cutoff
predicate (reading C3).  CPU only."""
import math

import numpy as np
import pytest

from oracle.coupling_oracle import COULOMB_KCAL_A, coupling_energy_forces
from paper_2201_08110_b200 import workloads as wl


def pair(r, qi=0.3, qj=-0.5, si=3.0, sj=3.4, ei=0.1, ej=0.2, cutoff=0.0):
    pos = np.array([[0.0, 0.0, 0.0], [r, 0.0, 0.0]])
    return coupling_energy_forces(pos, [0], [qi], [si], [ei], [1], [qj], [sj], [ej], cutoff=cutoff)


def test_coulomb_only_closed_form():
    # eps = 0 switches the Lennard-Jones term off: V = kc q_i q_j / r, F_j = kc q_i q_j / r^2 along +x (repulsive if same sign)
    V, F = pair(2.5, qi=0.4, qj=0.7, ei=0.0)
    assert V == pytest.approx(COULOMB_KCAL_A * 0.28 / 2.5, rel=1e-14)
    assert F[1, 0] == pytest.approx(COULOMB_KCAL_A * 0.28 / 6.25, rel=1e-14) and F[0, 0] == -F[1, 0]
    assert np.all(F[:, 1:] == 0.0)
    # one elementary charge pair at 1 A: the Coulomb constant itself
    assert pair(1.0, qi=1.0, qj=1.0, ei=0.0)[0] == pytest.approx(332.0637133, rel=1e-12)


def test_lennard_jones_zero_minimum_and_combination_rule():
    # charges off.  sigma_ij = (3.0 + 3.4)/2 = 3.2, eps_ij = sqrt(0.1 * 0.2) (reading C1)
    s, e = 3.2, math.sqrt(0.02)
    V, _ = pair(s, qi=0.0)
    assert abs(V) < 1e-13                                    # V_LJ(sigma) = 0
    rmin = 2.0 ** (1.0 / 6.0) * s
    V, F = pair(rmin, qi=0.0)
    assert V == pytest.approx(-e, rel=1e-13)                 # well depth
    assert np.abs(F).max() < 1e-12                           # force vanishes at the minimum
    V, F = pair(0.9 * s, qi=0.0)
    assert V == pytest.approx(4 * e * (0.9 ** -12 - 0.9 ** -6), rel=1e-13)
    assert F[1, 0] > 0 and F[0, 0] < 0                       # repulsive inside sigma
    V, F = pair(1.5 * s, qi=0.0)
    assert F[1, 0] < 0                                       # attractive beyond the minimum


def test_forces_are_minus_gradient_and_newtons_third_law():
    sysm = wl.coupling_system(n_mm=400, seed=11)
    args = (sysm.nnp_rows, sysm.q_nnp, sysm.sigma_nnp, sysm.eps_nnp, sysm.mm_rows, sysm.q_mm, sysm.sigma_mm, sysm.eps_mm)
    pos = sysm.positions.astype(np.float64)
    for cutoff in (0.0, 9.0):
        V, F = coupling_energy_forces(pos, *args, cutoff=cutoff)
        assert np.abs(F.sum(axis=0)).max() <= 1e-9 * np.abs(F).max()            # action = reaction
        assert np.abs(np.cross(pos, F).sum(axis=0)).max() <= 1e-8 * np.abs(F).max() * 40  # central forces: no torque
        rng = np.random.default_rng(5)
        h = 1e-6
        for a in list(sysm.nnp_rows[:4]) + list(rng.choice(sysm.mm_rows, 6, replace=False)):
            for c in range(3):
                p = pos.copy(); p[a, c] += h
                m = pos.copy(); m[a, c] -= h
                fd = -(coupling_energy_forces(p, *args, cutoff=cutoff, want_forces=False)[0]
                       - coupling_energy_forces(m, *args, cutoff=cutoff, want_forces=False)[0]) / (2 * h)
                assert fd == pytest.approx(F[a, c], abs=2e-6 * max(1.0, np.abs(F).max()))


def test_only_cross_pairs_and_additivity():
    # V is a sum over (NNP, MM) pairs: splitting the MM list splits V; two NNP atoms (or two MM atoms) on top of each
    # other do not blow anything up because same-region pairs are not part of Eq. 4
    pos = np.array([[0, 0, 0], [0, 0, 0.01], [3, 0, 0], [3, 0.01, 0], [0, 4, 0]], float)
    n, m = [0, 1], [2, 3, 4]
    q, s, e = [0.2, -0.1], [3.0, 2.0], [0.1, 0.05]
    qm, sm_, em = [0.5, -0.4, 0.3], [3.1, 2.9, 3.3], [0.15, 0.1, 0.2]
    V, F = coupling_energy_forces(pos, n, q, s, e, m, qm, sm_, em)
    assert np.isfinite(V) and np.all(np.isfinite(F))
    parts = 0.0
    for i in range(2):
        for j in range(3):
            parts += coupling_energy_forces(pos, [n[i]], [q[i]], [s[i]], [e[i]], [m[j]], [qm[j]], [sm_[j]], [em[j]])[0]
    assert V == pytest.approx(parts, rel=1e-13)


def test_cutoff_is_inclusive_plain_truncation():
    # reading C3: a pair contributes iff D2 <= rc^2
    V_in, _ = pair(9.0, cutoff=9.0)
    V_all, _ = pair(9.0)
    assert V_in == V_all != 0.0
    V_out, F_out = pair(math.nextafter(9.0, 10.0), cutoff=9.0)
    assert V_out == 0.0 and np.all(F_out == 0.0)
    # float32 inputs are widened, not re-rounded: a pair just inside in f32 stays inside
    r32 = np.float32(8.999999)
    assert coupling_energy_forces(np.array([[0, 0, 0], [r32, 0, 0]], np.float32), [0], [0.3], [3.0], [0.1], [1], [-0.5],
                                  [3.4], [0.2], cutoff=9.0)[0] != 0.0

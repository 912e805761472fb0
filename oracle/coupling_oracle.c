/*
 * oracle/coupling_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain float64 statement of the NNP-MM coupling term of mechanical embedding, Eq. 4 of the paper
 * (PAPER.md:67-71):
 *
 *   V_NNP-MM(r) = sum_{i in NNP} sum_{j in MM} ( V_C^{ij} + V_LJ^{ij} ),
 *   V_C^{ij}  = q_i q_j / (4 pi eps0 r_ij),
 *   V_LJ^{ij} = 4 eps_ij [ (sigma_ij / r_ij)^12 - (sigma_ij / r_ij)^6 ],
 *
 * and of the forces F_a = -dV/dr_a on every atom of both regions.  Only NNP-MM pairs enter: pairs inside
 * the NNP region are V_NNP's business, pairs inside the MM region V_MM's (Eq. 1).
 *
 * Readings where the paper is silent (C1-C4):
 *   C1  eps_ij, sigma_ij by the Lorentz-Berthelot rule: sigma_ij = (sigma_i + sigma_j)/2,
 *       eps_ij = sqrt(eps_i eps_j) (per-atom parameters are what an MM force field carries);
 *   C2  1/(4 pi eps0) is passed in as `kc` in the caller's units (332.0637... kcal A / (mol e^2));
 *   C3  optional plain truncation: a pair contributes iff D2 <= rc^2 (rc <= 0: no cutoff), D2 evaluated as
 *       in the neighbour predicate O2: widened coordinates, (dx dx + dy dy) + dz dz, no FMA contraction.
 *       (The paper's MD runs use a 9 A van der Waals cutoff; Eq. 4 itself has none.)
 *   C4  no periodic images (as S13 for the NNP term).
 *
 * Only tests/ and bench.py's cpu_baseline leg may call this; it shares no code with the CUDA path.
 * Build with -ffp-contract=off.  Pins: tests/test_oracle_coupling.py (two-atom closed forms, the
 * Lennard-Jones zero and minimum, central finite differences, Newton's third law, zero net torque,
 * only-cross-pairs, the cutoff predicate).
 */
#include <math.h>

/*
 * pos    [n_rows][3] positions of all atoms of the system (A)
 * nnp_rows[n_nnp], mm_rows[n_mm]   rows of the NNP / MM atoms
 * q_*, sigma_*, eps_*              per listed atom
 * force  [n_rows][3] or NULL: F_a is ADDED (mechanical embedding adds into the MM force buffer)
 * returns V_NNP-MM
 */
double coupling_energy_forces(int n_nnp, const int* nnp_rows, const double* q_nnp, const double* sigma_nnp,
                              const double* eps_nnp, int n_mm, const int* mm_rows, const double* q_mm,
                              const double* sigma_mm, const double* eps_mm, const double* pos, double kc, double rc,
                              double* force) {
  double V = 0.0;
  const double rc2 = rc * rc;
  for (int i = 0; i < n_nnp; ++i) {
    const double* ri = pos + 3 * (long)nnp_rows[i];
    for (int j = 0; j < n_mm; ++j) {
      const double* rj = pos + 3 * (long)mm_rows[j];
      const double dx = rj[0] - ri[0], dy = rj[1] - ri[1], dz = rj[2] - ri[2];
      const double d2 = (dx * dx + dy * dy) + dz * dz;
      if (rc > 0.0 && d2 > rc2) continue; /* C3 */
      const double r = sqrt(d2);
      const double sigma = 0.5 * (sigma_nnp[i] + sigma_mm[j]); /* C1 */
      const double eps = sqrt(eps_nnp[i] * eps_mm[j]);
      const double sr6 = pow(sigma / r, 6.0), sr12 = sr6 * sr6;
      const double vc = kc * q_nnp[i] * q_mm[j] / r;
      const double vlj = 4.0 * eps * (sr12 - sr6);
      V += vc + vlj;
      if (force) {
        /* dV/dr = -vc/r + 4 eps (-12 sr12 + 6 sr6)/r ;  F_j = -dV/dr * (r_j - r_i)/r ,  F_i = -F_j */
        const double dvdr = -vc / r + 4.0 * eps * (-12.0 * sr12 + 6.0 * sr6) / r;
        const double fx = -dvdr * dx / r, fy = -dvdr * dy / r, fz = -dvdr * dz / r;
        double* fj = force + 3 * (long)mm_rows[j];
        double* fi = force + 3 * (long)nnp_rows[i];
        fj[0] += fx; fj[1] += fy; fj[2] += fz;
        fi[0] -= fx; fi[1] -= fy; fi[2] -= fz;
      }
    }
  }
  return V;
}

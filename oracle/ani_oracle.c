/*
 * oracle/ani_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, float64 CPU statement of what the NNP/MM hot path computes: the
 * energy V_NNP(Z, r) of the ANI-2x neural network potential for the NNP region
 * (Eq. 2) and the forces F = -grad V_NNP (Eq. 3).
 * ANI = "modified Behler-Parrinello symmetry functions", cutoff 5.1 A, elements
 * H,C,N,O,F,S,Cl; ensemble of 8 NNs.  The paper prints
 * none of the formulas; they are the definitions O1-O7 of SURVEY.md section 8(c)
 * (restated in DESIGN.md "Readings"), with constants passed in by the caller
 * (BASELINE.json configs[0] values).  Each function below cites its definition.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call this.  It shares no code with the CUDA path (paper_2201_08110_b200/csrc)
 * and neither includes the other.
 *
 * Arithmetic: binary64 throughout, inputs (f32 positions, constants, weights) are
 * widened, never re-derived.  Build with -ffp-contract=off (the pair predicate O2 is
 * defined without FMA contraction).  No blocking, fusion or reordering beyond the
 * definitions; the only structure is "list the neighbours of centre i by a plain scan,
 * then loop over them", which the brute-force O(N^3) test in tests/ pins.
 *
 * Pins (tests/test_oracle_*.py): closed-form dimer/trimer values, numpy brute-force
 * O(N^3) enumeration, numpy float64 matmul for the MLP, central finite differences of
 * the energy, translation/rotation/permutation invariance, zero net force and torque,
 * ensemble identities, cutoff continuity.  Parity with *trained* ANI-2x numbers is
 * UNPINNED: the paper prints no energies/forces and the weights are not in this container.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
  int n_species;              /* S */
  int n_models;               /* M */
  double rc_r, rc_a;          /* radial / angular cutoff (A) */
  double eta_r;
  int n_shf_r;
  const double *shf_r;
  double eta_a, zeta;
  int n_shf_a;
  const double *shf_a;
  int n_shf_z;
  const double *shf_z;
  double cos_scale;           /* 0.95, reading S6 */
  double celu_alpha;          /* 0.1 */
  int n_layers;               /* 4 */
  const int *layer_dims;      /* [S][n_layers+1] */
  const float *const *weights; /* [M*S*n_layers], index (m*S+e)*n_layers+l, row-major [out][in] */
  const float *const *biases;  /* same indexing, [out]; entry or whole pointer may be NULL => 0 */
  const double *self_energy;  /* [S] or NULL */
  double energy_scale;        /* output unit per model unit */
} ani_params;

static const double ORACLE_PI = 3.14159265358979323846;

int ani_oracle_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* number of AEV features: S*n_shf_r + S(S+1)/2 * n_shf_a*n_shf_z (1008 for ANI-2x, BASELINE.json configs[0]) */
int ani_n_features(const ani_params *p) {
  return p->n_species * p->n_shf_r + (p->n_species * (p->n_species + 1) / 2) * p->n_shf_a * p->n_shf_z;
}

/* O1: f_C(r;Rc) = 0.5 cos(pi r/Rc) + 0.5 for r <= Rc, else 0 */
static double fcut(double r, double rc) { return r <= rc ? 0.5 * cos(ORACLE_PI * r / rc) + 0.5 : 0.0; }
/* O1: f_C'(r) = -(pi / 2Rc) sin(pi r/Rc) */
static double dfcut(double r, double rc) { return r <= rc ? -(ORACLE_PI / (2.0 * rc)) * sin(ORACLE_PI * r / rc) : 0.0; }

/* O2: D2 = (dx*dx + dy*dy) + dz*dz in binary64, left to right, no FMA contraction */
static double dist2(const double *pos, int i, int j) {
  double dx = pos[3 * j + 0] - pos[3 * i + 0];
  double dy = pos[3 * j + 1] - pos[3 * i + 1];
  double dz = pos[3 * j + 2] - pos[3 * i + 2];
  double xx = dx * dx;
  double yy = dy * dy;
  double zz = dz * dz;
  double s = xx + yy;
  return s + zz;
}

/* O4: upper-triangle row-major index of the unordered species pair {s,t} */
static int pair_index(int s, int t, int S) {
  if (s > t) { int u = s; s = t; t = u; }
  return s * S - s * (s - 1) / 2 + (t - s);
}

static int mol_of(int i, int n_mol, const int *off) {
  for (int m = 0; m < n_mol; ++m)
    if (i >= off[m] && i < off[m + 1]) return m;
  return -1;
}

/*
 * O2: pair set {(i,j): i<j, same molecule, D2 <= Rc^2}.  Writes up to `capacity` pairs
 * as (i,j) int pairs in lexicographic order; returns the total count.
 */
long ani_pairs(int n, const double *pos, int n_mol, const int *mol_off, double rc,
               int *ij, long capacity) {
  long cnt = 0;
  double rc2 = rc * rc;
  for (int m = 0; m < n_mol; ++m)
    for (int i = mol_off[m]; i < mol_off[m + 1]; ++i)
      for (int j = i + 1; j < mol_off[m + 1]; ++j)
        if (dist2(pos, i, j) <= rc2) {
          if (cnt < capacity) { ij[2 * cnt] = i; ij[2 * cnt + 1] = j; }
          ++cnt;
        }
  (void)n;
  return cnt;
}

/* neighbours of centre i inside its molecule [lo,hi) with D2 <= rc^2, ascending j */
static int list_neighbours(const double *pos, int i, int lo, int hi, double rc, int *out) {
  int c = 0;
  double rc2 = rc * rc;
  for (int j = lo; j < hi; ++j)
    if (j != i && dist2(pos, i, j) <= rc2) out[c++] = j;
  return c;
}

/* O3 + O4: the AEV row G_i (n_features doubles, zeroed here) of centre i */
static void aev_row(const ani_params *p, const double *pos, const int *species, int i, int lo, int hi,
                    int *nbr, double *G) {
  const int S = p->n_species;
  const int nf = ani_n_features(p);
  const int ang0 = S * p->n_shf_r;
  const int nsub = p->n_shf_a * p->n_shf_z;
  for (int f = 0; f < nf; ++f) G[f] = 0.0;

  /* O3 radial: G[s_j*16+k] += 0.25 exp(-eta_R (r - ShfR_k)^2) f_C(r; RcR) */
  int nr = list_neighbours(pos, i, lo, hi, p->rc_r, nbr);
  for (int a = 0; a < nr; ++a) {
    int j = nbr[a];
    double r = sqrt(dist2(pos, i, j));
    double fc = fcut(r, p->rc_r);
    for (int k = 0; k < p->n_shf_r; ++k) {
      double d = r - p->shf_r[k];
      G[species[j] * p->n_shf_r + k] += 0.25 * exp(-p->eta_r * d * d) * fc;
    }
  }

  /* O4 angular: unordered {j,k}, j<k, both within RcA of i */
  int na = list_neighbours(pos, i, lo, hi, p->rc_a, nbr);
  for (int a = 0; a < na; ++a)
    for (int b = a + 1; b < na; ++b) {
      int j = nbr[a], k = nbr[b];
      double ax = pos[3 * j] - pos[3 * i], ay = pos[3 * j + 1] - pos[3 * i + 1], az = pos[3 * j + 2] - pos[3 * i + 2];
      double bx = pos[3 * k] - pos[3 * i], by = pos[3 * k + 1] - pos[3 * i + 1], bz = pos[3 * k + 2] - pos[3 * i + 2];
      double ra = sqrt(dist2(pos, i, j)), rb = sqrt(dist2(pos, i, k));
      double c = p->cos_scale * (ax * bx + ay * by + az * bz) / (ra * rb);
      double theta = acos(c);
      double W = fcut(ra, p->rc_a) * fcut(rb, p->rc_a);
      double rbar = 0.5 * (ra + rb);
      int base = ang0 + pair_index(species[j], species[k], S) * nsub;
      for (int ia = 0; ia < p->n_shf_a; ++ia) {
        double d = rbar - p->shf_a[ia];
        double F2 = exp(-p->eta_a * d * d);
        for (int iz = 0; iz < p->n_shf_z; ++iz) {
          double F1 = pow(0.5 * (1.0 + cos(theta - p->shf_z[iz])), p->zeta);
          G[base + ia * p->n_shf_z + iz] += 2.0 * F1 * F2 * W;
        }
      }
    }
}

/* O5: CELU(x) = x (x>0), alpha (exp(x/alpha) - 1) (x<=0) */
static double celu(double x, double alpha) { return x > 0.0 ? x : alpha * (exp(x / alpha) - 1.0); }
/* O5: CELU'(x) = 1 (x>0), exp(x/alpha) (x<=0) */
static double dcelu(double x, double alpha) { return x > 0.0 ? 1.0 : exp(x / alpha); }

static int max_width(const ani_params *p) {
  int w = 0;
  for (int e = 0; e < p->n_species; ++e)
    for (int l = 0; l <= p->n_layers; ++l)
      if (p->layer_dims[e * (p->n_layers + 1) + l] > w) w = p->layer_dims[e * (p->n_layers + 1) + l];
  return w;
}

/*
 * O5 forward and its input-gradient: one atom of element e, one model m.
 * h_0 = G; z_l = W_l h_{l-1} + b_l; h_l = CELU(z_l) for l < L; output e = z_L (scalar).
 * Returns e; if dG != NULL adds (weight * d e / d G) into dG[0..nf).
 * scratch: (n_layers+1) * 2 * maxw doubles.
 */
static double mlp_atom(const ani_params *p, int m, int e, const double *G, double weight, double *dG,
                       double *scratch) {
  const int L = p->n_layers;
  const int *dims = p->layer_dims + e * (L + 1);
  const int mw = max_width(p);
  double *z = scratch;                 /* z[l] at z + l*mw, l = 1..L */
  double *d = scratch + (L + 1) * mw;  /* delta buffers, two rows used alternately */
  const double *h_prev = G;
  double *h = NULL;
  double *hbuf = (double *)malloc(sizeof(double) * (size_t)(L + 1) * mw); /* h_l at hbuf + l*mw */
  for (int l = 1; l <= L; ++l) {
    const float *W = p->weights[(m * p->n_species + e) * L + (l - 1)];
    const float *b = (p->biases && p->biases[(m * p->n_species + e) * L + (l - 1)])
                         ? p->biases[(m * p->n_species + e) * L + (l - 1)] : NULL;
    int nin = dims[l - 1], nout = dims[l];
    h = hbuf + l * mw;
    for (int o = 0; o < nout; ++o) {
      double acc = 0.0;
      for (int k = 0; k < nin; ++k) acc += (double)W[(size_t)o * nin + k] * h_prev[k];
      acc += b ? (double)b[o] : 0.0;
      z[l * mw + o] = acc;
      h[o] = (l < L) ? celu(acc, p->celu_alpha) : acc;
    }
    h_prev = h;
  }
  double energy = z[L * mw + 0];
  if (dG) {
    /* O7 chain rule through the MLP: delta_L = 1; delta_{l-1} = W_l^T delta_l (.) CELU'(z_{l-1}) */
    double *dl = d, *dprev = d + mw;
    dl[0] = 1.0;
    for (int l = L; l >= 1; --l) {
      const float *W = p->weights[(m * p->n_species + e) * L + (l - 1)];
      int nin = dims[l - 1], nout = dims[l];
      for (int k = 0; k < nin; ++k) {
        double acc = 0.0;
        for (int o = 0; o < nout; ++o) acc += (double)W[(size_t)o * nin + k] * dl[o];
        if (l > 1) acc *= dcelu(z[(l - 1) * mw + k], p->celu_alpha);
        dprev[k] = acc;
      }
      double *t = dl; dl = dprev; dprev = t;
    }
    for (int k = 0; k < dims[0]; ++k) dG[k] += weight * dl[k];
  }
  free(hbuf);
  return energy;
}

/*
 * O5 for a batch of AEV rows (test entry): e_out[m*n + i], dG_out[i*nf + f] = (1/M) sum_m d e_i^(m)/d G_i[f].
 */
void ani_mlp(const ani_params *p, int n, const int *species, const double *G, double *e_out, double *dG_out) {
  const int nf = ani_n_features(p);
  const int mw = max_width(p);
  double *scratch = (double *)malloc(sizeof(double) * (size_t)(p->n_layers + 3) * mw);
  for (int i = 0; i < n; ++i) {
    if (dG_out) for (int f = 0; f < nf; ++f) dG_out[(size_t)i * nf + f] = 0.0;
    for (int m = 0; m < p->n_models; ++m)
      e_out[(size_t)m * n + i] = mlp_atom(p, m, species[i], G + (size_t)i * nf, 1.0 / p->n_models,
                                         dG_out ? dG_out + (size_t)i * nf : NULL, scratch);
  }
  free(scratch);
}

/* O3+O4 for all atoms (test entry): G[n][nf] */
void ani_aev(const ani_params *p, int n, const double *pos, const int *species, int n_mol, const int *mol_off,
             double *G) {
  const int nf = ani_n_features(p);
#pragma omp parallel
  {
    int *nbr = (int *)malloc(sizeof(int) * (size_t)(n > 0 ? n : 1));
#pragma omp for schedule(dynamic, 4)
    for (int i = 0; i < n; ++i) {
      int m = mol_of(i, n_mol, mol_off);
      aev_row(p, pos, species, i, mol_off[m], mol_off[m + 1], nbr, G + (size_t)i * nf);
    }
    free(nbr);
  }
}

/*
 * O7: add to F (model-unit energy per A, NOT yet scaled) the force contributions of the AEV of
 * centre i, given g = dE/dG_i.  Serial; follows SURVEY 8(c) O7 term by term.
 */
static void aev_row_forces(const ani_params *p, const double *pos, const int *species, int i, int lo, int hi,
                           int *nbr, const double *g, double *F) {
  const int S = p->n_species;
  const int ang0 = S * p->n_shf_r;
  const int nsub = p->n_shf_a * p->n_shf_z;

  /* radial: T = 0.25 exp(-eta (r-Shf)^2) fC(r);  dT/dr = T(-2 eta (r-Shf)) + 0.25 exp(.) fC'(r) */
  int nr = list_neighbours(pos, i, lo, hi, p->rc_r, nbr);
  for (int a = 0; a < nr; ++a) {
    int j = nbr[a];
    double vx = pos[3 * j] - pos[3 * i], vy = pos[3 * j + 1] - pos[3 * i + 1], vz = pos[3 * j + 2] - pos[3 * i + 2];
    double r = sqrt(dist2(pos, i, j));
    double fc = fcut(r, p->rc_r), dfc = dfcut(r, p->rc_r);
    double dEdr = 0.0;
    for (int k = 0; k < p->n_shf_r; ++k) {
      double d = r - p->shf_r[k];
      double ex = exp(-p->eta_r * d * d);
      double T = 0.25 * ex * fc;
      double dT = T * (-2.0 * p->eta_r * d) + 0.25 * ex * dfc;
      dEdr += g[species[j] * p->n_shf_r + k] * dT;
    }
    /* dr/dr_j = (r_j - r_i)/r ; F = -dE/dr */
    double fx = dEdr * vx / r, fy = dEdr * vy / r, fz = dEdr * vz / r;
    F[3 * j] -= fx; F[3 * j + 1] -= fy; F[3 * j + 2] -= fz;
    F[3 * i] += fx; F[3 * i + 1] += fy; F[3 * i + 2] += fz;
  }

  /* angular: A = 2 F1 F2 W */
  int na = list_neighbours(pos, i, lo, hi, p->rc_a, nbr);
  for (int a = 0; a < na; ++a)
    for (int b = a + 1; b < na; ++b) {
      int j = nbr[a], k = nbr[b];
      double av[3] = {pos[3 * j] - pos[3 * i], pos[3 * j + 1] - pos[3 * i + 1], pos[3 * j + 2] - pos[3 * i + 2]};
      double bv[3] = {pos[3 * k] - pos[3 * i], pos[3 * k + 1] - pos[3 * i + 1], pos[3 * k + 2] - pos[3 * i + 2]};
      double ra = sqrt(dist2(pos, i, j)), rb = sqrt(dist2(pos, i, k));
      double dot = av[0] * bv[0] + av[1] * bv[1] + av[2] * bv[2];
      double c = p->cos_scale * dot / (ra * rb);
      double theta = acos(c);
      double dtheta_dc = -1.0 / sqrt(1.0 - c * c);
      double fca = fcut(ra, p->rc_a), fcb = fcut(rb, p->rc_a);
      double dfca = dfcut(ra, p->rc_a), dfcb = dfcut(rb, p->rc_a);
      double W = fca * fcb;
      double rbar = 0.5 * (ra + rb);
      /* dc/da = cos_scale [ b/(ra rb) - (a.b) a/(ra^3 rb) ], and a<->b */
      double dc_da[3], dc_db[3];
      for (int x = 0; x < 3; ++x) {
        dc_da[x] = p->cos_scale * (bv[x] / (ra * rb) - dot * av[x] / (ra * ra * ra * rb));
        dc_db[x] = p->cos_scale * (av[x] / (ra * rb) - dot * bv[x] / (rb * rb * rb * ra));
      }
      int base = ang0 + pair_index(species[j], species[k], S) * nsub;
      double ga[3] = {0, 0, 0}, gb[3] = {0, 0, 0}; /* sum_f g_f dA_f/da, dA_f/db */
      for (int ia = 0; ia < p->n_shf_a; ++ia) {
        double d = rbar - p->shf_a[ia];
        double F2 = exp(-p->eta_a * d * d);
        double dF2_dr = -p->eta_a * d * F2; /* dF2/dra = dF2/drb */
        for (int iz = 0; iz < p->n_shf_z; ++iz) {
          double u = 0.5 * (1.0 + cos(theta - p->shf_z[iz]));
          double F1 = pow(u, p->zeta);
          double dF1_dtheta = -(p->zeta / 2.0) * pow(u, p->zeta - 1.0) * sin(theta - p->shf_z[iz]);
          double gf = g[base + ia * p->n_shf_z + iz];
          for (int x = 0; x < 3; ++x) {
            double dA_da = 2.0 * (dF1_dtheta * dtheta_dc * dc_da[x] * F2 * W
                                  + F1 * dF2_dr * (av[x] / ra) * W
                                  + F1 * F2 * dfca * fcb * (av[x] / ra));
            double dA_db = 2.0 * (dF1_dtheta * dtheta_dc * dc_db[x] * F2 * W
                                  + F1 * dF2_dr * (bv[x] / rb) * W
                                  + F1 * F2 * fca * dfcb * (bv[x] / rb));
            ga[x] += gf * dA_da;
            gb[x] += gf * dA_db;
          }
        }
      }
      /* F_j -= g dA/da ; F_k -= g dA/db ; F_i += g (dA/da + dA/db) */
      for (int x = 0; x < 3; ++x) {
        F[3 * j + x] -= ga[x];
        F[3 * k + x] -= gb[x];
        F[3 * i + x] += ga[x] + gb[x];
      }
    }
}

/*
 * O1-O7: energy per molecule and forces.
 *   pos      f64[n][3]  (A)            species  i32[n] in 0..S-1
 *   mol_off  i32[n_mol+1] CSR, molecules are contiguous atom ranges
 * outputs (any optional pointer may be NULL):
 *   E_mol    f64[n_mol]  energy_scale * sum_i [ (1/M) sum_m e_i^(m) + E_self[s_i] ]      (O6)
 *   F        f64[n][3]   -dE/dr, scaled by energy_scale                                   (O7)
 *   G_out    f64[n][nf]  AEVs                e_out f64[M][n] atomic energies per model (model units)
 *   dG_out   f64[n][nf]  dE_model_units/dG = (1/M) sum_m d e_i^(m)/dG_i
 * returns 0, or -1 on bad species / offsets.
 */
int ani_energy_forces(const ani_params *p, int n, const double *pos, const int *species, int n_mol,
                      const int *mol_off, double *E_mol, double *F, double *G_out, double *e_out,
                      double *dG_out) {
  const int nf = ani_n_features(p);
  const int M = p->n_models;
  const int mw = max_width(p);
  if (n_mol < 1 || mol_off[0] != 0 || mol_off[n_mol] != n) return -1;
  for (int i = 0; i < n; ++i)
    if (species[i] < 0 || species[i] >= p->n_species) return -1;

  double *G = G_out ? G_out : (double *)malloc(sizeof(double) * (size_t)n * nf);
  double *dG = dG_out ? dG_out : (double *)malloc(sizeof(double) * (size_t)n * nf);
  double *eat = (double *)malloc(sizeof(double) * (size_t)n); /* (1/M) sum_m e_i^(m) */
  int *molid = (int *)malloc(sizeof(int) * (size_t)n);
  for (int i = 0; i < n; ++i) molid[i] = mol_of(i, n_mol, mol_off);

  /* per-centre work is independent: AEV row, then the M atomic networks and their input-gradients */
#pragma omp parallel
  {
    int *nbr = (int *)malloc(sizeof(int) * (size_t)n);
    double *scratch = (double *)malloc(sizeof(double) * (size_t)(p->n_layers + 3) * mw);
#pragma omp for schedule(dynamic, 1)
    for (int i = 0; i < n; ++i) {
      int m0 = molid[i];
      aev_row(p, pos, species, i, mol_off[m0], mol_off[m0 + 1], nbr, G + (size_t)i * nf);
      double *dgi = dG + (size_t)i * nf;
      for (int f = 0; f < nf; ++f) dgi[f] = 0.0;
      double esum = 0.0;
      for (int m = 0; m < M; ++m) {
        double e = mlp_atom(p, m, species[i], G + (size_t)i * nf, 1.0 / M, dgi, scratch);
        if (e_out) e_out[(size_t)m * n + i] = e;
        esum += e;
      }
      eat[i] = esum / M; /* S7: arithmetic mean over the ensemble */
    }
    free(nbr);
    free(scratch);
  }

  /* O6 */
  if (E_mol)
    for (int m = 0; m < n_mol; ++m) {
      double s = 0.0;
      for (int i = mol_off[m]; i < mol_off[m + 1]; ++i)
        s += eat[i] + (p->self_energy ? p->self_energy[species[i]] : 0.0);
      E_mol[m] = p->energy_scale * s;
    }

  /* O7, serial over centres (every centre adds into its neighbours' force rows) */
  if (F) {
    int *nbr = (int *)malloc(sizeof(int) * (size_t)n);
    for (int i = 0; i < 3 * n; ++i) F[i] = 0.0;
    for (int i = 0; i < n; ++i)
      aev_row_forces(p, pos, species, i, mol_off[molid[i]], mol_off[molid[i] + 1], nbr, dG + (size_t)i * nf, F);
    for (int i = 0; i < 3 * n; ++i) F[i] *= p->energy_scale;
    free(nbr);
  }

  if (!G_out) free(G);
  if (!dG_out) free(dG);
  free(eat);
  free(molid);
  return 0;
}

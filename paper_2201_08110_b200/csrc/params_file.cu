// nnp_create_from_file: build a handle from a parameter file (NEXT-1 of SURVEY.md 8(f): "load real ANI-2x-format
// parameters (biases, self-energies, species-order map) through the same nnp_config, and a 1 NN fast mode",
// PAPER.md:36,83,160).  The trained ANI-2x / ANI-1x parameter sets are not in this container; the container format
// below is this library's own (little-endian, written by binding.write_parameter_file), and carries everything a
// published ANI parameter set holds: the element list in the set's own species order, the AEV constants, the layer
// shapes, weights AND biases of every (model, element, layer) and the per-element self-energies.
//
//   char    magic[8] = "NNPB200P";  int32 version = 1
//   int32   n_species, n_models, n_layers
//   float   rc_radial, rc_angular, eta_r, eta_a, zeta, cos_scale, celu_alpha
//   int32   n_shf_r, n_shf_a, n_shf_z
//   double  energy_scale
//   int32   atomic_number[n_species]          species index s of the file <-> element Z
//   float   shf_r[n_shf_r], shf_a[n_shf_a], shf_z[n_shf_z]
//   int32   layer_dims[n_species][n_layers + 1]
//   double  self_energy[n_species]
//   for m, e, l:  float W[out][in], float b[out]
//
// The caller names its atoms by ATOMIC NUMBER; the file's element list maps them to species indices, so a set
// that orders its elements H C N O S F Cl (as the label order of BASELINE.json configs[1]) loads the same way as
// one that orders them H C N O F S Cl.
#include <stdio.h>
#include <string.h>

#include <vector>

#include "nnp.h"

namespace {
template <typename T>
bool rd(FILE* f, T* p, size_t n) {
  return n == 0 || fread(p, sizeof(T), n, f) == n;
}
}  // namespace

extern "C" int nnp_create_from_file(nnp_handle** out, const char* path, int32_t n_atoms, const int32_t* atomic_numbers_host,
                                    int32_t n_molecules, const int32_t* mol_offsets_host, int32_t n_models_to_use,
                                    double length_scale, int32_t flags) {
  if (!out) return NNP_ERR_INVALID_ARG;
  *out = nullptr;
  if (!path || n_atoms < 0 || (n_atoms > 0 && !atomic_numbers_host) || n_models_to_use < 0) return NNP_ERR_INVALID_ARG;
  FILE* f = fopen(path, "rb");
  if (!f) return NNP_ERR_INVALID_ARG;
  struct Closer {
    FILE* f;
    ~Closer() { fclose(f); }
  } closer{f};
  char magic[8];
  int32_t version = 0, S = 0, M = 0, L = 0, nr = 0, na = 0, nz = 0;
  float fl[7];
  double escale = 0.0;
  if (!rd(f, magic, 8) || memcmp(magic, "NNPB200P", 8) != 0 || !rd(f, &version, 1) || version != 1) return NNP_ERR_INVALID_ARG;
  if (!rd(f, &S, 1) || !rd(f, &M, 1) || !rd(f, &L, 1) || !rd(f, fl, 7) || !rd(f, &nr, 1) || !rd(f, &na, 1) || !rd(f, &nz, 1) ||
      !rd(f, &escale, 1))
    return NNP_ERR_INVALID_ARG;
  if (S < 1 || S > 64 || M < 1 || M > 1024 || L < 2 || L > 16 || nr < 1 || nr > 1024 || na < 1 || na > 1024 || nz < 1 || nz > 1024)
    return NNP_ERR_INVALID_ARG;
  std::vector<int32_t> Z(S), dims((size_t)S * (L + 1));
  std::vector<float> shf_r(nr), shf_a(na), shf_z(nz);
  std::vector<double> se(S);
  if (!rd(f, Z.data(), Z.size()) || !rd(f, shf_r.data(), shf_r.size()) || !rd(f, shf_a.data(), shf_a.size()) ||
      !rd(f, shf_z.data(), shf_z.size()) || !rd(f, dims.data(), dims.size()) || !rd(f, se.data(), se.size()))
    return NNP_ERR_INVALID_ARG;
  for (int32_t d : dims)
    if (d < 1 || d > (1 << 20)) return NNP_ERR_INVALID_ARG;
  const int m_use = n_models_to_use == 0 ? M : n_models_to_use;  // 1 = the paper's "1 NN" variant
  if (m_use > M) return NNP_ERR_INVALID_ARG;
  std::vector<std::vector<float>> W((size_t)m_use * S * L), B((size_t)m_use * S * L);
  for (int m = 0; m < M; ++m)
    for (int e = 0; e < S; ++e)
      for (int l = 0; l < L; ++l) {
        const size_t nin = dims[(size_t)e * (L + 1) + l], nout = dims[(size_t)e * (L + 1) + l + 1];
        if (m < m_use) {
          auto& w = W[((size_t)m * S + e) * L + l];
          auto& b = B[((size_t)m * S + e) * L + l];
          w.resize(nout * nin);
          b.resize(nout);
          if (!rd(f, w.data(), w.size()) || !rd(f, b.data(), b.size())) return NNP_ERR_INVALID_ARG;
        } else if (fseek(f, (long)((nout * nin + nout) * sizeof(float)), SEEK_CUR) != 0) {
          return NNP_ERR_INVALID_ARG;
        }
      }
  // atomic numbers -> species indices of this parameter set
  std::vector<int32_t> species(n_atoms);
  for (int i = 0; i < n_atoms; ++i) {
    int s = -1;
    for (int k = 0; k < S; ++k)
      if (Z[k] == atomic_numbers_host[i]) s = k;
    if (s < 0) return NNP_ERR_INVALID_ARG;  // an element the potential was not trained for
    species[i] = s;
  }
  std::vector<const float*> wp(W.size()), bp(B.size());
  for (size_t k = 0; k < W.size(); ++k) {
    wp[k] = W[k].data();
    bp[k] = B[k].data();
  }
  nnp_config cfg;
  memset(&cfg, 0, sizeof(cfg));
  cfg.n_species = S; cfg.n_models = m_use;
  cfg.rc_radial = fl[0]; cfg.rc_angular = fl[1]; cfg.eta_r = fl[2]; cfg.eta_a = fl[3]; cfg.zeta = fl[4];
  cfg.cos_scale = fl[5]; cfg.celu_alpha = fl[6];
  cfg.n_shf_r = nr; cfg.shf_r = shf_r.data();
  cfg.n_shf_a = na; cfg.shf_a = shf_a.data();
  cfg.n_shf_z = nz; cfg.shf_z = shf_z.data();
  cfg.n_layers = L; cfg.layer_dims = dims.data();
  cfg.weights = wp.data(); cfg.biases = bp.data();
  cfg.self_energy = se.data();
  cfg.energy_scale = escale;
  cfg.length_scale = length_scale;
  cfg.flags = flags;
  return nnp_create(out, &cfg, n_atoms, species.data(), n_molecules, mol_offsets_host);
}

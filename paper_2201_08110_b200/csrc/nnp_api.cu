// C-ABI entry points of libnnp_b200 (include/nnp.h): handle set-up (A0), the per-step launch chain
// (A1..A8) replayed as one CUDA graph, status, profiling and the debug/parity exports.
#include <math.h>
#include <string.h>

#include <algorithm>
#include <new>

#include "nnp_internal.h"

int aev_set_smem_attributes(nnp_handle* h);

#define CK(call)                                  \
  do {                                            \
    cudaError_t _e = (call);                      \
    if (_e != cudaSuccess) return NNP_ERR_CUDA;   \
  } while (0)

namespace {

template <typename T>
int dev_alloc(T** p, size_t n) {
  *p = nullptr;
  if (n == 0) n = 1;
  return cudaMalloc((void**)p, n * sizeof(T)) == cudaSuccess ? 0 : -1;
}

template <typename T>
int upload(T** p, const std::vector<T>& v) {
  if (dev_alloc(p, v.size())) return -1;
  if (!v.empty() && cudaMemcpy(*p, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice) != cudaSuccess) return -1;
  return 0;
}

long long align_up(long long x, long long a) { return (x + a - 1) / a * a; }

int upload_launch(GemmLaunch& g, const std::vector<GemmProblem>& probs) {
  std::vector<GemmTile> tiles;
  build_gemm_tiles(probs, tiles);
  g.n_tiles = (int)tiles.size();
  if (upload(&g.d_probs, probs)) return -1;
  if (upload(&g.d_tiles, tiles)) return -1;
  return 0;
}

}  // namespace

extern "C" const char* nnp_error_string(int code) {
  switch (code) {
    case NNP_OK: return "ok";
    case NNP_ERR_INVALID_ARG: return "invalid argument";
    case NNP_ERR_CUDA: return "CUDA error";
    case NNP_ERR_UNSUPPORTED_ARCH: return "unsupported GPU architecture (need sm_100)";
    case NNP_ERR_CAPACITY: return "neighbour row capacity exceeded";
    case NNP_ERR_NONFINITE: return "non-finite position";
    case NNP_ERR_ALLOC: return "allocation failed";
    case NNP_ERR_STATIC_LIMIT: return "more atoms than the fixed scratch array of nnp_coupling_compute_static holds";
    default: return "unknown error";
  }
}

extern "C" void nnp_destroy(nnp_handle* h) {
  if (!h) return;
  cudaSetDevice(h->device);
  if (h->last_stream) cudaStreamSynchronize(h->last_stream);
  cudaDeviceSynchronize();
  if (h->h_hout) cudaFreeHost(h->h_hout);
  if (h->h_hpos) cudaFreeHost(h->h_hpos);
  for (auto& g : h->graphs)
    if (g.exec) cudaGraphExecDestroy(g.exec);
  if (h->own_stream) cudaStreamDestroy(h->own_stream);
  for (auto e : h->events) cudaEventDestroy(e);
  void* ptrs[] = {h->d_eblocks, h->d_epart, h->d_ecount, h->d_mol_range, h->d_species, h->d_mol_off, h->d_mol_id, h->d_sortpos, h->d_perm, h->d_grp_off, h->d_self_energy,
                  h->d_pos4, h->d_nbr_r, h->d_nbr_a, h->d_cnt_r, h->d_cnt_a, h->d_aev, h->d_daev, h->d_facc,
                  h->d_eatom, h->d_status, h->d_W, h->d_b,
                  h->d_aev_lo, h->d_Whi, h->d_Wlo, h->d_WThi, h->d_WTlo, h->d_act_full};
  for (void* p : ptrs)
    if (p) cudaFree(p);
  for (int l = 0; l < NNP_MAX_LAYERS; ++l) {
    if (h->d_act[l]) cudaFree(h->d_act[l]);
    if (h->d_act_lo[l]) cudaFree(h->d_act_lo[l]);
  }
  for (auto* v : {&h->fwd, &h->bwd})
    for (auto& g : *v) {
      if (g.d_probs) cudaFree(g.d_probs);
      if (g.d_tiles) cudaFree(g.d_tiles);
    }
  for (auto* v : {&h->ufwd, &h->ubwd})
    for (auto& g : *v) umma_free_launch(g);
  for (auto* v : {&h->sfwd, &h->sbwd})
    for (auto& g : *v) small_free_launch(g);
  small_free_launch(h->smid);
  cells_free(h);
  delete h;
}

extern "C" int nnp_create(nnp_handle** out, const nnp_config* cfg, int32_t n_atoms, const int32_t* species_host,
                          int32_t n_molecules, const int32_t* mol_offsets_host) {
  if (!out) return NNP_ERR_INVALID_ARG;
  *out = nullptr;
  if (!cfg || n_atoms < 0 || (n_atoms > 0 && !species_host) || n_molecules < 1) return NNP_ERR_INVALID_ARG;
  const int S = cfg->n_species, M = cfg->n_models, L = cfg->n_layers;
  if (S < 1 || S > NNP_MAX_SPECIES || M < 1 || L < 2 || L > NNP_MAX_LAYERS) return NNP_ERR_INVALID_ARG;
  if (cfg->n_shf_r < 1 || cfg->n_shf_r > NNP_MAX_SHF_R || cfg->n_shf_a < 1 || cfg->n_shf_a > NNP_MAX_SHF_A ||
      cfg->n_shf_z < 1 || cfg->n_shf_z > NNP_MAX_SHF_Z || cfg->n_shf_a * cfg->n_shf_z > NNP_MAX_SUB)
    return NNP_ERR_INVALID_ARG;
  if (!cfg->shf_r || !cfg->shf_a || !cfg->shf_z || !cfg->layer_dims || !cfg->weights) return NNP_ERR_INVALID_ARG;
  if (!(cfg->rc_radial > 0.f) || !(cfg->rc_angular > 0.f) || cfg->rc_angular > cfg->rc_radial)
    return NNP_ERR_INVALID_ARG;
  if (!(cfg->celu_alpha > 0.f) || !(cfg->length_scale > 0.0)) return NNP_ERR_INVALID_ARG;
  if (!(cfg->zeta >= 1.0f) || cfg->zeta >= 64.0f) return NNP_ERR_INVALID_ARG;  /* integer part by repeated squaring */
  const int n_sub = cfg->n_shf_a * cfg->n_shf_z;
  const int n_radial = S * cfg->n_shf_r;
  const int n_feat = n_radial + (S * (S + 1) / 2) * n_sub;
  for (int e = 0; e < S; ++e) {
    const int32_t* d = cfg->layer_dims + (size_t)e * (L + 1);
    if (d[0] != n_feat || d[L] != 1) return NNP_ERR_INVALID_ARG;
    for (int l = 0; l < L; ++l)
      if (d[l] < 1 || d[l] % 4 != 0) return NNP_ERR_INVALID_ARG;  // float4 row loads
  }
  for (int i = 0; i < n_atoms; ++i)
    if (species_host[i] < 0 || species_host[i] >= S) return NNP_ERR_INVALID_ARG;
  std::vector<int> mol_off(n_molecules + 1);
  if (mol_offsets_host) {
    for (int m = 0; m <= n_molecules; ++m) mol_off[m] = mol_offsets_host[m];
    if (mol_off[0] != 0 || mol_off[n_molecules] != n_atoms) return NNP_ERR_INVALID_ARG;
    for (int m = 0; m < n_molecules; ++m)
      if (mol_off[m + 1] < mol_off[m]) return NNP_ERR_INVALID_ARG;
  } else {
    if (n_molecules != 1) return NNP_ERR_INVALID_ARG;
    mol_off[0] = 0;
    mol_off[1] = n_atoms;
  }

  int dev = 0;
  CK(cudaGetDevice(&dev));
  cudaDeviceProp prop;
  CK(cudaGetDeviceProperties(&prop, dev));
  if (prop.major != 10) return NNP_ERR_UNSUPPORTED_ARCH;  // binary holds sm_100a code only

  nnp_handle* h = new (std::nothrow) nnp_handle();
  if (!h) return NNP_ERR_ALLOC;
  h->device = dev;
  h->N = n_atoms; h->n_mol = n_molecules; h->S = S; h->M = M; h->L = L; h->n_feat = n_feat;
  h->flags = cfg->flags;
  h->use_pdl = !(cfg->flags & NNP_FLAG_NO_PDL);
  h->energy_scale = cfg->energy_scale;
  h->length_scale = cfg->length_scale;
  h->dims.assign(cfg->layer_dims, cfg->layer_dims + (size_t)S * (L + 1));

  AevConst& a = h->aev;
  memset(&a, 0, sizeof(a));
  a.S = S; a.n_shf_r = cfg->n_shf_r; a.n_shf_a = cfg->n_shf_a; a.n_shf_z = cfg->n_shf_z;
  a.n_sub = n_sub; a.n_radial = n_radial; a.n_feat = n_feat;
  a.rc_r = cfg->rc_radial; a.rc_a = cfg->rc_angular; a.eta_r = cfg->eta_r; a.eta_a = cfg->eta_a;
  a.zeta = cfg->zeta; a.cos_scale = cfg->cos_scale; a.length_scale = (float)cfg->length_scale;
  a.rc_r2 = (double)cfg->rc_radial * (double)cfg->rc_radial;
  a.rc_a2 = (double)cfg->rc_angular * (double)cfg->rc_angular;
  {
    const double z = (double)cfg->zeta;
    a.zeta_int = (int)floor(z);
    a.zeta1_int = a.zeta_int - 1;
    a.zeta_frac = (float)(z - floor(z));
    const double log2e = 1.4426950408889634074;
    const double kr = -(double)cfg->eta_r * log2e, ka = -(double)cfg->eta_a * log2e;
    a.kr_hi = (float)kr; a.kr_lo = (float)(kr - (double)a.kr_hi);
    a.ka_hi = (float)ka; a.ka_lo = (float)(ka - (double)a.ka_hi);
  }
  for (int k = 0; k < cfg->n_shf_r; ++k) a.shf_r[k] = cfg->shf_r[k];
  for (int k = 0; k < cfg->n_shf_a; ++k) a.shf_a[k] = cfg->shf_a[k];
  for (int k = 0; k < cfg->n_shf_z; ++k) {
    const double cz = cos((double)cfg->shf_z[k]), sz = sin((double)cfg->shf_z[k]);
    a.cos_z[k] = (float)cz;
    a.sin_z[k] = (float)sz;
    a.cos_z_lo[k] = (float)(cz - (double)a.cos_z[k]);
    a.sin_z_lo[k] = (float)(sz - (double)a.sin_z[k]);
  }

  // ---- A0: group atoms by element (stable), molecule ids, capacities
  const int N = n_atoms;
  std::vector<int> species(species_host, species_host + N), perm(N), sortpos(N), mol_id(N);
  h->grp_off.assign(S + 1, 0);
  for (int i = 0; i < N; ++i) h->grp_off[species[i] + 1]++;
  for (int e = 0; e < S; ++e) h->grp_off[e + 1] += h->grp_off[e];
  {
    std::vector<int> cur(h->grp_off.begin(), h->grp_off.end() - 1);
    for (int i = 0; i < N; ++i) {
      const int p = cur[species[i]]++;
      perm[p] = i;
      sortpos[i] = p;
    }
  }
  int max_mol = 1;
  for (int m = 0; m < n_molecules; ++m) {
    for (int i = mol_off[m]; i < mol_off[m + 1]; ++i) mol_id[i] = m;
    max_mol = std::max(max_mol, mol_off[m + 1] - mol_off[m]);
  }
  // Row capacities of the neighbour lists.  A molecule of n atoms has at most n - 1 neighbours; for large molecules the
  // default assumes condensed matter (<= 0.11 atoms/A^3 gives ~61 atoms inside 5.1 A and ~20 inside 3.5 A; configs[4]
  // peaks at 90 / 39): 160 radial and 80 angular slots.  The capacities size the per-centre shared-memory tables of the
  // AEV kernels (occupancy) and the pair-gradient buffer; a denser system sets NNP_ERR_CAPACITY, which nnp_status
  // reports, and is served by max_radial_neighbors / max_angular_neighbors.
  const int dflt_r = max_mol >= 1024 ? 160 : 256, dflt_a = max_mol >= 1024 ? 80 : 128;
  h->capR = cfg->max_radial_neighbors > 0 ? cfg->max_radial_neighbors : std::min(std::max(max_mol - 1, 1), dflt_r);
  h->capA = cfg->max_angular_neighbors > 0 ? cfg->max_angular_neighbors : std::min(std::max(max_mol - 1, 1), dflt_a);
  if (h->capA > h->capR) h->capA = h->capR;
  // A1 engine: all pairs inside a molecule at ligand sizes, cell binning for large molecules
  h->use_cells = N > 0 && !(cfg->flags & NNP_FLAG_NO_CELLS) && (max_mol >= 1024 || (cfg->flags & NNP_FLAG_FORCE_CELLS));

  auto fail = [&](int code) {
    nnp_destroy(h);
    return code;
  };
  if (aev_smem_bytes(h, true) > (size_t)prop.sharedMemPerBlockOptin || aev_set_smem_attributes(h) != 0)
    return fail(NNP_ERR_INVALID_ARG);

  {
    std::vector<int> range(2 * (size_t)N);
    for (int i = 0; i < N; ++i) {
      range[2 * i] = mol_off[mol_id[i]];
      range[2 * i + 1] = mol_off[mol_id[i] + 1];
    }
    if (upload(&h->d_mol_range, range)) return fail(NNP_ERR_ALLOC);
  }
  if (upload(&h->d_species, species) || upload(&h->d_mol_off, mol_off) || upload(&h->d_mol_id, mol_id) ||
      upload(&h->d_sortpos, sortpos) || upload(&h->d_perm, perm) || upload(&h->d_grp_off, h->grp_off))
    return fail(NNP_ERR_ALLOC);
  if (cfg->self_energy) {
    std::vector<double> se(cfg->self_energy, cfg->self_energy + S);
    if (upload(&h->d_self_energy, se)) return fail(NNP_ERR_ALLOC);
  }

  // ---- weights: arena ordered (element, layer, model); models of one (e,l) are contiguous so the
  // layer-1 backward over the whole ensemble is a single GEMM with K = M*H1.
  h->w_off.assign((size_t)S * L, 0);
  h->b_off.assign((size_t)S * L, 0);
  long long wo = 0, bo = 0;
  for (int e = 0; e < S; ++e)
    for (int l = 0; l < L; ++l) {
      const int nin = h->dims[e * (L + 1) + l], nout = h->dims[e * (L + 1) + l + 1];
      h->w_off[e * L + l] = wo;
      h->b_off[e * L + l] = bo;
      wo = align_up(wo + (long long)M * nout * nin, 64);
      bo = align_up(bo + (long long)M * nout, 64);
    }
  h->w_floats = (size_t)wo;
  h->b_floats = (size_t)bo;
  std::vector<float> B((size_t)bo, 0.f);  // host copy of the biases (the ligand-size engine folds b_L into its items)
  std::vector<float> Wh((size_t)wo, 0.f);  // host copy of the weight arena (split for the tensor engine below)
  {
    for (int m = 0; m < M; ++m)
      for (int e = 0; e < S; ++e)
        for (int l = 0; l < L; ++l) {
          const int nin = h->dims[e * (L + 1) + l], nout = h->dims[e * (L + 1) + l + 1];
          const size_t idx = ((size_t)m * S + e) * L + l;
          const float* src = cfg->weights[idx];
          if (!src) return fail(NNP_ERR_INVALID_ARG);
          memcpy(&Wh[h->w_off[e * L + l] + (size_t)m * nout * nin], src, sizeof(float) * (size_t)nout * nin);
          if (cfg->biases && cfg->biases[idx])
            memcpy(&B[h->b_off[e * L + l] + (size_t)m * nout], cfg->biases[idx], sizeof(float) * nout);
        }
    if (upload(&h->d_W, Wh) || upload(&h->d_b, B)) return fail(NNP_ERR_ALLOC);
  }

  // ---- MLP engine: the tensor-core engine takes hidden widths that are multiples of 16.  A contraction that is not
  // a whole number of 32-float TMA boxes is padded by the tensor maps: the WEIGHT operand of every GEMM is a tensor
  // whose contraction extent is exactly K, so its box columns beyond K are zero-filled by TMA, and whatever the
  // activation box holds there (the next model's activations, finite) is multiplied by zero.  ANI-1x: 144 and 112.
  bool box_ok = n_feat % 4 == 0 && N > 0;
  for (int e = 0; e < S && box_ok; ++e) {
    for (int l = 1; l < L; ++l)
      if (h->dims[e * (L + 1) + l] % 16 != 0) box_ok = false;
  }
  // ligand-size engine: every element group is small, so the layers are weight-streaming problems
  int max_grp = 0, max_dim = n_feat;
  for (int e = 0; e < S; ++e) {
    max_grp = std::max(max_grp, h->grp_off[e + 1] - h->grp_off[e]);
    for (int l = 1; l < L; ++l) max_dim = std::max(max_dim, h->dims[e * (L + 1) + l]);
  }
  const bool parts_fit = (size_t)N * M * n_feat * 4 <= ((size_t)8 << 20);
  h->use_small = !(cfg->flags & NNP_FLAG_NO_SMALL) && N > 0 && n_feat % 4 == 0 && max_dim <= 1024 && max_grp <= 64 &&
                 parts_fit && small_init() == 0;
  h->use_umma = !h->use_small && box_ok && !(cfg->flags & NNP_FLAG_NO_UMMA) && umma_init() == 0;
  // at ligand sizes the layer-1 backward is split per model (every CTA streams its own slice of W1
  // exactly once); the M partial dE/dAEV rows are summed by the AEV backward kernel
  h->n_parts = (h->use_small && parts_fit) ? M : 1;
  if (h->use_umma) {
    // layer-1 backward on the tensor engine: one GEMM per element with K = M*H1.  When that leaves most SMs without a
    // tile (few hundred atoms), the contraction is cut into n_parts groups of models whose partial dE/dAEV rows the
    // AEV backward kernel sums (as it does at ligand sizes).
    long long tiles = 0;
    for (int e = 0; e < S; ++e) tiles += ((h->grp_off[e + 1] - h->grp_off[e] + 127) / 128) * (long long)((n_feat + 127) / 128);
    // a group of models must be whole boxes of every element's contraction (the weight tensor of the layer-1 backward
    // spans ALL models, so nothing zero-fills a box that runs into the next group; one group = the whole extent: any K)
    auto group_ok = [&](int p) {
      for (int e = 0; e < S; ++e)
        if (((long long)(M / p) * h->dims[e * (L + 1) + 1]) % 32 != 0) return false;
      return true;
    };
    int parts = 1;
    while (parts < M && M % (2 * parts) == 0 && tiles * parts < 2LL * prop.multiProcessorCount &&
           (size_t)N * (2 * parts) * n_feat * 4 <= ((size_t)64 << 20) && group_ok(2 * parts))
      parts *= 2;
    h->n_parts = parts;
    // 3xTF32 operand planes: weights hi = rna_tf32(w), lo = rna_tf32(w - hi), in the forward layout and transposed
    // (layer 1: [n_feat][M*H1]; layers l > 1: per model [H_{l-1}][H_l]) so that both passes read K-major boxes
    auto rna = [](float x) {
      uint32_t u;
      memcpy(&u, &x, 4);
      u = (u + 0x1000u) & 0xFFFFE000u;
      float r;
      memcpy(&r, &u, 4);
      return r;
    };
    std::vector<float> hi(Wh.size()), lo(Wh.size()), thi(Wh.size(), 0.f), tlo(Wh.size(), 0.f);
    for (size_t i = 0; i < Wh.size(); ++i) {
      hi[i] = rna(Wh[i]);
      lo[i] = rna(Wh[i] - hi[i]);
    }
    for (int e = 0; e < S; ++e)
      for (int l = 0; l < L - 1; ++l) {
        const int nin = h->dims[e * (L + 1) + l], nout = h->dims[e * (L + 1) + l + 1];
        const size_t base = (size_t)h->w_off[e * L + l];
        for (int m = 0; m < M; ++m)
          for (int o = 0; o < nout; ++o) {
            const size_t src = base + ((size_t)m * nout + o) * nin;
            for (int n = 0; n < nin; ++n) {
              const size_t dst = l == 0 ? base + (size_t)n * M * nout + (size_t)m * nout + o
                                        : base + ((size_t)m * nin + n) * nout + o;
              thi[dst] = hi[src + n];
              tlo[dst] = lo[src + n];
            }
          }
      }
    if (upload(&h->d_Whi, hi) || upload(&h->d_Wlo, lo) || upload(&h->d_WThi, thi) || upload(&h->d_WTlo, tlo))
      return fail(NNP_ERR_ALLOC);
  }
  Wh.clear();
  Wh.shrink_to_fit();

  // ---- workspaces
  if (dev_alloc(&h->d_pos4, (size_t)N) || dev_alloc(&h->d_nbr_r, (size_t)N * h->capR) ||
      dev_alloc(&h->d_nbr_a, (size_t)N * h->capA) || dev_alloc(&h->d_cnt_r, (size_t)N) ||
      dev_alloc(&h->d_cnt_a, (size_t)N) || dev_alloc(&h->d_aev, (size_t)N * n_feat) ||
      dev_alloc(&h->d_daev, (size_t)h->n_parts * N * n_feat) || dev_alloc(&h->d_facc, (size_t)N * 3) ||
      dev_alloc(&h->d_eatom, (size_t)N * M) || dev_alloc(&h->d_status, 1))
    return fail(NNP_ERR_ALLOC);
  h->hout_force_off = sizeof(double) * (size_t)n_molecules;
  h->hout_bytes = h->hout_force_off + sizeof(float) * 3 * (size_t)N;
  if (cudaHostAlloc((void**)&h->h_hout, std::max<size_t>(h->hout_bytes, 8), cudaHostAllocMapped) != cudaSuccess ||
      cudaHostAlloc((void**)&h->h_hpos, std::max<size_t>(sizeof(float) * 3 * (size_t)N, 4), cudaHostAllocMapped) != cudaSuccess ||
      cudaHostGetDevicePointer((void**)&h->d_hout_alias, h->h_hout, 0) != cudaSuccess ||
      cudaHostGetDevicePointer((void**)&h->d_hpos_alias, h->h_hpos, 0) != cudaSuccess)
    return fail(NNP_ERR_ALLOC);
  memset(h->h_hout, 0, std::max<size_t>(h->hout_bytes, 8));
  if (h->use_umma && dev_alloc(&h->d_aev_lo, (size_t)N * n_feat)) return fail(NNP_ERR_ALLOC);
  // latency-bound sizes only: in a large batch the serial row build inside every centre's CTA costs more than the
  // launch it saves (configs[2]: +36 us in the AEV forward against a 12 us neighbour kernel)
  h->fuse_nbr = N > 0 && N <= 512 && !h->use_cells && max_mol <= 512 && !(cfg->flags & NNP_FLAG_NO_NBR_FUSION);
  if (h->use_cells && cells_alloc(h) != 0) return fail(NNP_ERR_ALLOC);
  {  // energy reduction blocks: chunks of <= 512 atoms (two per thread: the loads of a thread are a dependent chain
     // sortpos -> atomic energies, so short chunks on many CTAs beat long ones: configs[4] finish 18 -> see DESIGN.md)
    const int ECH = 512;
    std::vector<EnergyBlock> eb;
    for (int m = 0; m < n_molecules; ++m) {
      const int a0 = mol_off[m], a1 = mol_off[m + 1];
      const int nch = std::max(1, (a1 - a0 + ECH - 1) / ECH);
      const int first = (int)eb.size();
      for (int q = 0; q < nch; ++q) eb.push_back(EnergyBlock{m, std::min(a1, a0 + q * ECH), std::min(a1, a0 + (q + 1) * ECH), first, nch});
    }
    h->n_eblocks = (int)eb.size();
    if (upload(&h->d_eblocks, eb) || dev_alloc(&h->d_epart, eb.size()) || dev_alloc(&h->d_ecount, (size_t)n_molecules))
      return fail(NNP_ERR_ALLOC);
    cudaMemset(h->d_ecount, 0, sizeof(int) * (size_t)n_molecules);
  }
  cudaMemset(h->d_status, 0, sizeof(int));
  cudaMemset(h->d_nbr_r, 0, sizeof(int) * std::max<size_t>((size_t)N * h->capR, 1));
  cudaMemset(h->d_nbr_a, 0, sizeof(int) * std::max<size_t>((size_t)N * h->capA, 1));
  cudaMemset(h->d_cnt_r, 0, sizeof(int) * std::max<size_t>(N, 1));
  cudaMemset(h->d_cnt_a, 0, sizeof(int) * std::max<size_t>(N, 1));
  cudaMemset(h->d_facc, 0, sizeof(unsigned long long) * std::max<size_t>((size_t)N * 3, 1));
  cudaMemset(h->d_eatom, 0, sizeof(double) * std::max<size_t>((size_t)N * M, 1));
  cudaMemset(h->d_daev, 0, sizeof(float) * std::max<size_t>((size_t)h->n_parts * N * n_feat, 1));  // skipped tiles stay 0

  // activations act[l], l = 1..L-1, layout per element group: [atom][model][H_l]
  for (int l = 1; l < L; ++l) {
    h->act_off[l].assign(S, 0);
    long long o = 0;
    for (int e = 0; e < S; ++e) {
      h->act_off[l][e] = o;
      const long long ne = h->grp_off[e + 1] - h->grp_off[e];
      o = align_up(o + ne * M * h->dims[e * (L + 1) + l], 64);
    }
    if (dev_alloc(&h->d_act[l], (size_t)o)) return fail(NNP_ERR_ALLOC);
    if (h->use_umma && dev_alloc(&h->d_act_lo[l], (size_t)o)) return fail(NNP_ERR_ALLOC);
    // the last hidden layer's forward launch writes delta_{L-1} in its epilogue when it is a per-model problem
    // (L - 1 >= 2): its h is kept as one plane for the energies
    if (h->use_umma && l == L - 1 && L - 1 >= 2) {
      if (dev_alloc(&h->d_act_full, (size_t)o)) return fail(NNP_ERR_ALLOC);
      h->fuse_delta = true;
    }
  }

  // ---- MLP launches (grouped GEMMs), shapes fixed at create time
  const float alpha = cfg->celu_alpha;
  double flops = 0, wbytes = 0, w1bytes = 0;
  for (int l = 1; l < L; ++l) {  // forward hidden layers
    std::vector<GemmProblem> probs;
    for (int e = 0; e < S; ++e) {
      const int ne = h->grp_off[e + 1] - h->grp_off[e];
      if (ne == 0) continue;
      const int nin = h->dims[e * (L + 1) + l - 1], nout = h->dims[e * (L + 1) + l];
      for (int m = 0; m < M; ++m) {
        GemmProblem p;
        memset(&p, 0, sizeof(p));
        if (l == 1) {
          p.A = h->d_aev + (size_t)h->grp_off[e] * n_feat;
          p.lda = n_feat;
        } else {
          p.A = h->d_act[l - 1] + h->act_off[l - 1][e] + (size_t)m * nin;
          p.lda = M * nin;
        }
        p.B = h->d_W + h->w_off[e * L + l - 1] + (size_t)m * nout * nin;
        p.ldb = nin;
        p.transB = 0;
        p.C = h->d_act[l] + h->act_off[l][e] + (size_t)m * nout;
        p.ldc = M * nout;
        p.bias = h->d_b + h->b_off[e * L + l - 1] + (size_t)m * nout;
        p.M = ne; p.N = nout; p.K = nin;
        p.epi = EPI_BIAS_CELU;
        p.alpha = alpha;
        probs.push_back(p);
        flops += 4.0 * ne * (double)nout * nin;
        wbytes += 4.0 * nout * nin;
        if (l == 1) w1bytes += 4.0 * nout * nin;
      }
    }
    GemmLaunch g;
    g.name = "mlp_fwd_l" + std::to_string(l);
    if (upload_launch(g, probs)) return fail(NNP_ERR_ALLOC);
    h->fwd.push_back(g);
  }
  for (int l = L - 1; l >= 1; --l) {  // backward through hidden layer l: delta_{l-1} = delta_l W_l (.) CELU'
    std::vector<GemmProblem> probs;
    for (int e = 0; e < S; ++e) {
      const int ne = h->grp_off[e + 1] - h->grp_off[e];
      if (ne == 0) continue;
      const int nin = h->dims[e * (L + 1) + l - 1], nout = h->dims[e * (L + 1) + l];
      if (l > 1) {
        for (int m = 0; m < M; ++m) {
          GemmProblem p;
          memset(&p, 0, sizeof(p));
          p.A = h->d_act[l] + h->act_off[l][e] + (size_t)m * nout;
          p.lda = M * nout;
          p.B = h->d_W + h->w_off[e * L + l - 1] + (size_t)m * nout * nin;
          p.ldb = nin;
          p.transB = 1;
          p.C = h->d_act[l - 1] + h->act_off[l - 1][e] + (size_t)m * nin;
          p.ldc = M * nin;
          p.aux = p.C;
          p.ldaux = p.ldc;
          p.M = ne; p.N = nin; p.K = nout;
          p.epi = EPI_MUL_DCELU;
          p.alpha = alpha;
          probs.push_back(p);
        }
      } else {  // layer 1: dE/dAEV = (1/M) sum_m delta_1^(m) W_1^(m): one GEMM with K = M*H1
        GemmProblem p;
        memset(&p, 0, sizeof(p));
        p.A = h->d_act[1] + h->act_off[1][e];
        p.lda = M * nout;
        p.B = h->d_W + h->w_off[e * L + 0];
        p.ldb = nin;
        p.transB = 1;
        p.C = h->d_daev + (size_t)h->grp_off[e] * n_feat;
        p.ldc = n_feat;
        p.M = ne; p.N = nin; p.K = M * nout;
        p.epi = EPI_SCALE;
        p.scale = 1.0f / (float)M;
        probs.push_back(p);
      }
    }
    GemmLaunch g;
    g.name = "mlp_bwd_l" + std::to_string(l);
    if (upload_launch(g, probs)) return fail(NNP_ERR_ALLOC);
    h->bwd.push_back(g);
  }
  // Structural zeros of the AEV: the radial block of species s and the angular blocks of pairs (s, t) are zero for
  // every atom when s (or t) does not occur in the system.  Layer 1 can skip the 32-wide contraction boxes that hold
  // only such columns (forward) and the 128-wide tiles of dE/dAEV that hold only such columns (backward: the AEV
  // backward kernel never reads them).  The result is unchanged; only multiplications by zero are not issued.
  unsigned long long l1_kmask = 0, l1_fmask = 0;
  if (!(cfg->flags & NNP_FLAG_NO_ZERO_SKIP) && n_feat <= 64 * 32) {
    std::vector<char> live(n_feat, 0);
    std::vector<char> present(S, 0);
    for (int e = 0; e < S; ++e) present[e] = h->grp_off[e + 1] > h->grp_off[e];
    for (int sp = 0; sp < S; ++sp)
      if (present[sp])
        for (int k = 0; k < cfg->n_shf_r; ++k) live[sp * cfg->n_shf_r + k] = 1;
    for (int sp = 0, pidx = 0; sp < S; ++sp)
      for (int tp = sp; tp < S; ++tp, ++pidx)
        if (present[sp] && present[tp])
          for (int k = 0; k < n_sub; ++k) live[n_radial + pidx * n_sub + k] = 1;
    bool any_dead = false;
    for (int cidx = 0; cidx < n_feat; ++cidx) {
      if (live[cidx]) {
        l1_kmask |= 1ull << (cidx / 32);
        l1_fmask |= 1ull << (cidx / 128);
      } else {
        any_dead = true;
      }
    }
    if (!any_dead) l1_kmask = l1_fmask = 0;  // nothing to skip
  }
  h->aev_live_boxes = l1_kmask;  // the AEV backward kernel loads only these 32-column boxes of a dE/dAEV row
  if (h->use_umma) {
    // tcgen05 engine: D[f][a] = sum_k W[f][k] X[a][k].  Layer 1 forward runs all models of an element as ONE
    // problem (their weight rows are contiguous and they share the AEV input): F = M*H1 is a multiple of 128.
    std::vector<int> slot(S, -1);
    int ns = 0;
    for (int e = 0; e < S; ++e)
      if (h->grp_off[e + 1] > h->grp_off[e]) slot[e] = ns++;
    for (int pass = 0; pass < 2; ++pass) {
      for (int li = 0; li < L - 1; ++li) {
        const int l = pass == 0 ? li + 1 : L - 1 - li;  // fwd: 1..L-1, bwd: L-1..1
        std::vector<UmmaProblem> probs;
        std::vector<UmmaOperand> aops(ns), bops(ns);
        for (int e = 0; e < S; ++e) {
          if (slot[e] < 0) continue;
          const int ne = h->grp_off[e + 1] - h->grp_off[e];
          const int nin = h->dims[e * (L + 1) + l - 1], nout = h->dims[e * (L + 1) + l];
          const long long wofs = h->w_off[e * L + l - 1];
          if (pass == 0) {
            aops[slot[e]] = UmmaOperand{h->d_Whi + wofs, h->d_Wlo + wofs, (long long)M * nout, nin, nin};
            if (l == 1)
              bops[slot[e]] = UmmaOperand{h->d_aev + (size_t)h->grp_off[e] * n_feat, h->d_aev_lo + (size_t)h->grp_off[e] * n_feat,
                                          ne, n_feat, n_feat};
            else
              bops[slot[e]] = UmmaOperand{h->d_act[l - 1] + h->act_off[l - 1][e], h->d_act_lo[l - 1] + h->act_off[l - 1][e], ne,
                                          (long long)M * nin, (long long)M * nin};
          } else {
            if (l == 1) aops[slot[e]] = UmmaOperand{h->d_WThi + wofs, h->d_WTlo + wofs, nin, (long long)M * nout, (long long)M * nout};
            else aops[slot[e]] = UmmaOperand{h->d_WThi + wofs, h->d_WTlo + wofs, (long long)M * nin, nout, nout};
            bops[slot[e]] = UmmaOperand{h->d_act[l] + h->act_off[l][e], h->d_act_lo[l] + h->act_off[l][e], ne,
                                        (long long)M * nout, (long long)M * nout};
          }
          UmmaProblem p;
          memset(&p, 0, sizeof(p));
          p.amap = p.bmap = slot[e];
          p.n_atoms = ne;
          p.alpha = alpha;
          p.inv_alpha = 1.0f / alpha;
          if (pass == 0 && l == 1) {
            p.kmask = l1_kmask;
            p.F = M * nout; p.K = nin;
            p.C = h->d_act[1] + h->act_off[1][e];
            p.C_lo = h->d_act_lo[1] + h->act_off[1][e];
            p.ldc = M * nout;
            p.bias = h->d_b + h->b_off[e * L + 0];
            p.epi = EPI_BIAS_CELU;
            probs.push_back(p);
          } else if (pass == 0) {
            const bool last = h->fuse_delta && l == L - 1;
            for (int m = 0; m < M; ++m) {
              UmmaProblem q = p;
              if (last) {
                q.C_full = h->d_act_full + h->act_off[l][e] + (size_t)m * nout;
                q.w_last = h->d_W + h->w_off[e * L + L - 1] + (size_t)m * nout;
              }
              q.F = nout; q.K = nin;
              q.a_c0 = 0; q.a_c1 = m * nout; q.b_c0 = m * nin; q.b_c1 = 0;
              q.C = h->d_act[l] + h->act_off[l][e] + (size_t)m * nout;
              q.C_lo = h->d_act_lo[l] + h->act_off[l][e] + (size_t)m * nout;
              q.ldc = M * nout;
              q.bias = h->d_b + h->b_off[e * L + l - 1] + (size_t)m * nout;
              q.epi = last ? EPI_BIAS_CELU_LAST : EPI_BIAS_CELU;
              probs.push_back(q);
            }
          } else if (l > 1) {
            for (int m = 0; m < M; ++m) {  // delta_{l-1}[a][n] = CELU'(h_{l-1}) sum_o WT[m][n][o] delta_l[a][m][o]
              UmmaProblem q = p;
              q.F = nin; q.K = nout;
              q.a_c0 = 0; q.a_c1 = m * nin; q.b_c0 = m * nout; q.b_c1 = 0;
              q.C = h->d_act[l - 1] + h->act_off[l - 1][e] + (size_t)m * nin;
              q.C_lo = h->d_act_lo[l - 1] + h->act_off[l - 1][e] + (size_t)m * nin;
              q.ldc = M * nin;
              q.aux = q.C; q.aux_lo = q.C_lo; q.ldaux = q.ldc;
              q.epi = EPI_MUL_DCELU;
              probs.push_back(q);
            }
          } else {  // dE/dAEV[a][n] = (1/M) sum_{m,o} W1T[n][m*H1 + o] delta_1[a][m][o], in n_parts groups of models
            const int mg = M / h->n_parts;
            for (int pt = 0; pt < h->n_parts; ++pt) {
              UmmaProblem q = p;
              q.fmask = l1_fmask;
              q.F = nin; q.K = mg * nout;
              q.a_c0 = pt * mg * nout; q.a_c1 = 0; q.b_c0 = pt * mg * nout; q.b_c1 = 0;
              q.epi = EPI_SCALE;
              q.scale = 1.0f / (float)M;
              q.ldc = n_feat;
              q.C = h->d_daev + ((size_t)pt * N + h->grp_off[e]) * n_feat;
              probs.push_back(q);
            }
          }
        }
        UmmaLaunch ul;
        ul.name = (pass == 0 ? "mlp_fwd_l" : "mlp_bwd_l") + std::to_string(l);
        const bool reverse = !(cfg->flags & NNP_FLAG_NO_SWEEP_REVERSAL) && ((pass * (L - 1) + li) & 1) == 0;
        // opt-in: the two layer-1 launches of large systems on CTA pairs (cta_group::2, 256 x 256 tiles)
        const bool pair = l == 1 && (cfg->flags & NNP_FLAG_UMMA_PAIRS) && umma2_suits(probs) && umma2_init() == 0;
        if (pair ? umma2_build_launch(ul, probs, aops, bops, prop.multiProcessorCount)
                 : umma_build_launch(ul, probs, aops, bops, prop.multiProcessorCount, reverse,
                                     !(cfg->flags & NNP_FLAG_NO_TAIL_SPLIT))) {
          umma_free_launch(ul);
          return fail(NNP_ERR_CUDA);
        }
        (pass == 0 ? h->ufwd : h->ubwd).push_back(ul);
      }
    }
  }
  if (h->use_small) {
    const float inv_alpha = 1.0f / alpha;
    // layers 2..L-1, the 1-output layer and the backward pass down to delta_1 as ONE fused launch when the
    // hidden layers are narrow enough for its register tiles
    h->use_mid = !(cfg->flags & NNP_FLAG_NO_MID) && mid_init() == 0;
    for (int e = 0; e < S && h->use_mid; ++e)
      if (h->grp_off[e + 1] > h->grp_off[e] && !mid_supported(L, &h->dims[e * (L + 1)])) h->use_mid = false;
    if (h->use_mid) {
      std::vector<MidItem> items;
      for (int e = 0; e < S; ++e) {
        const int ne = h->grp_off[e + 1] - h->grp_off[e];
        const int* d = &h->dims[e * (L + 1)];
        for (int a0 = 0; a0 < ne; a0 += 4)
          for (int m = 0; m < M; ++m) {
            MidItem it;
            memset(&it, 0, sizeof(it));
            for (int l = 2; l <= L - 1; ++l) {
              it.W[l] = h->d_W + h->w_off[e * L + l - 1] + (size_t)m * d[l] * d[l - 1];
              it.bias[l] = h->d_b + h->b_off[e * L + l - 1] + (size_t)m * d[l];
            }
            for (int l = 1; l <= L - 1; ++l) it.H[l] = d[l];
            it.w_last = h->d_W + h->w_off[e * L + L - 1] + (size_t)m * d[L - 1];
            it.b_last = B[h->b_off[e * L + L - 1] + m];
            it.h1 = h->d_act[1] + h->act_off[1][e] + (size_t)a0 * M * d[1] + (size_t)m * d[1];
            it.ld1 = M * d[1];
            it.e_out = h->d_eatom + (size_t)(h->grp_off[e] + a0) * M + m;
            it.lde = M;
            it.L = L;
            it.n_atoms = std::min(4, ne - a0);
            it.alpha = alpha; it.inv_alpha = inv_alpha;
            items.push_back(it);
          }
      }
      h->smid.name = "mlp_mid";
      if (mid_build(h->smid, items)) { small_free_launch(h->smid); return fail(NNP_ERR_CUDA); }
    }
    const int l_fwd_end = h->use_mid ? 2 : L;   // forward layers run by the per-layer kernels: [1, l_fwd_end)
    const int l_bwd_begin = h->use_mid ? 1 : L - 1;
    bool fwd1_done = false;
    if (!(cfg->flags & NNP_FLAG_NO_FWD1)) {
      // layer 1 forward: persistent CTAs, each streams a share of ONE element's weight rows (all models of the
      // element are contiguous); shares are proportional to (row tiles) x (streaming + compute cost per tile)
      struct Work { int e, a0, na; long long tiles; double cost; int n_cta; };
      std::vector<Work> work;
      const int TR = small_fwd1_tile_rows();
      double total = 0;
      for (int e = 0; e < S; ++e) {
        const int ne = h->grp_off[e + 1] - h->grp_off[e];
        const long long rows = (long long)M * h->dims[e * (L + 1) + 1];
        for (int a0 = 0; a0 < ne; a0 += 24) {
          Work wk{e, a0, std::min(24, ne - a0), (rows + TR - 1) / TR, 0.0, 1};
          wk.cost = (double)wk.tiles * (16 + wk.na);
          total += wk.cost;
          work.push_back(wk);
        }
      }
      const int budget = std::max(prop.multiProcessorCount, (int)work.size());
      int used = 0;
      for (auto& wk : work) {
        wk.n_cta = (int)std::max<long long>(1, std::min<long long>(wk.tiles, (long long)(wk.cost / total * budget)));
        used += wk.n_cta;
      }
      for (bool grew = true; grew && used < budget;) {  // hand the remaining CTAs to the most loaded shares
        grew = false;
        Work* best = nullptr;
        for (auto& wk : work)
          if (wk.n_cta < wk.tiles && (!best || wk.cost / wk.n_cta > best->cost / best->n_cta)) best = &wk;
        if (best) { ++best->n_cta; ++used; grew = true; }
      }
      std::vector<Fwd1Item> items;
      for (const auto& wk : work) {
        const int e = wk.e, nout = h->dims[e * (L + 1) + 1];
        const long long rows = (long long)M * nout;
        const long long tiles_per = (wk.tiles + wk.n_cta - 1) / wk.n_cta;
        for (long long t0 = 0; t0 < wk.tiles; t0 += tiles_per) {
          const long long r0 = t0 * TR, r1 = std::min(rows, (t0 + tiles_per) * TR);
          Fwd1Item it;
          memset(&it, 0, sizeof(it));
          it.W = h->d_W + h->w_off[e * L + 0] + (size_t)r0 * n_feat;
          it.X = h->d_aev + (size_t)(h->grp_off[e] + wk.a0) * n_feat;
          it.bias = h->d_b + h->b_off[e * L + 0] + r0;
          it.out = h->d_act[1] + h->act_off[1][e] + (size_t)wk.a0 * M * nout + r0;
          it.ldx = n_feat; it.ldc = M * nout;
          it.n_atoms = wk.na; it.K = n_feat; it.n_rows = (int)(r1 - r0);
          it.alpha = alpha; it.inv_alpha = inv_alpha;
          items.push_back(it);
        }
      }
      SmallLaunch sl;
      sl.name = "mlp_fwd_l1";
      if (small_build_fwd1(sl, items) == 0) {
        h->sfwd.push_back(sl);
        fwd1_done = true;
      } else {
        small_free_launch(sl);  // shapes the persistent kernel does not take: per-layer kernel below
      }
    }
    for (int l = fwd1_done ? 2 : 1; l < l_fwd_end; ++l) {  // forward
      std::vector<SmallFwdItem> items;
      for (int e = 0; e < S; ++e) {
        const int ne = h->grp_off[e + 1] - h->grp_off[e];
        if (ne == 0) continue;
        const int nin = h->dims[e * (L + 1) + l - 1], nout = h->dims[e * (L + 1) + l];
        const float* Wl = h->d_W + h->w_off[e * L + l - 1];
        const float* bl = h->d_b + h->b_off[e * L + l - 1];
        float* outl = h->d_act[l] + h->act_off[l][e];
        for (int a0 = 0; a0 < ne; a0 += 32) {
          const int na = std::min(32, ne - a0);
          auto add = [&](int row0, int rows, const float* X, int ldx) {  // rows of the (e,l) block [M*nout][nin]
            for (int r0 = 0; r0 < rows; r0 += 16) {  // one row pair per warp
              SmallFwdItem it;
              memset(&it, 0, sizeof(it));
              it.W = Wl + (size_t)(row0 + r0) * nin;
              it.X = X; it.ldx = ldx;
              it.bias = bl + row0 + r0;
              it.out = outl + (size_t)a0 * M * nout + row0 + r0;
              it.ldc = M * nout;
              it.n_atoms = na; it.K = nin; it.n_rows = std::min(16, rows - r0);
              it.alpha = alpha; it.inv_alpha = inv_alpha;
              items.push_back(it);
            }
          };
          if (l == 1) {
            add(0, M * nout, h->d_aev + (size_t)(h->grp_off[e] + a0) * n_feat, n_feat);
          } else {
            for (int m = 0; m < M; ++m)
              add(m * nout, nout, h->d_act[l - 1] + h->act_off[l - 1][e] + (size_t)a0 * M * nin + (size_t)m * nin, M * nin);
          }
        }
      }
      SmallLaunch sl;
      sl.name = "mlp_fwd_l" + std::to_string(l);
      if (small_build_fwd(sl, items)) { small_free_launch(sl); return fail(NNP_ERR_CUDA); }
      h->sfwd.push_back(sl);
    }
    for (int l = l_bwd_begin; l >= 1; --l) {  // backward
      std::vector<SmallBwdItem> items;
      const bool bwd1 = l == 1 && (h->use_mid || L - 1 > 1);  // plain delta_1 -> dE/dAEV (no fused last layer)
      std::vector<TmaOperand> wops;  // layer-1 weight block per present element (tensor maps of the persistent kernel)
      std::vector<int> wslot(S, -1);
      if (bwd1)
        for (int e = 0; e < S; ++e)
          if (h->grp_off[e + 1] > h->grp_off[e]) {
            wslot[e] = (int)wops.size();
            wops.push_back(TmaOperand{h->d_W + h->w_off[e * L + 0], (long long)M * h->dims[e * (L + 1) + 1], n_feat, n_feat});
          }
      for (int e = 0; e < S; ++e) {
        const int ne = h->grp_off[e + 1] - h->grp_off[e];
        if (ne == 0) continue;
        const int nin = h->dims[e * (L + 1) + l - 1], nout = h->dims[e * (L + 1) + l];
        const float* Wl = h->d_W + h->w_off[e * L + l - 1];
        const int achunk = bwd1 ? 24 : 32;  // layer 1 runs on the weights-read-once kernel (<= 24 atoms per item)
        for (int a0 = 0; a0 < ne; a0 += achunk) {
          const int na = std::min(achunk, ne - a0);
          for (int m = 0; m < M; ++m)
            for (int n0 = 0; n0 < nin; n0 += 128) {
              SmallBwdItem it;
              memset(&it, 0, sizeof(it));
              it.W = Wl + (size_t)m * nout * nin + n0;
              it.ldw = nin;
              it.D = h->d_act[l] + h->act_off[l][e] + (size_t)a0 * M * nout + (size_t)m * nout;
              it.ldd = M * nout;
              it.n_atoms = na; it.n_out = nout; it.n_cols = std::min(128, nin - n0);
              it.tmap = wslot[e]; it.t_row0 = m * nout; it.t_col0 = n0;
              small_bwd_shape(na, &it.AW, &it.G);
              it.inv_alpha = inv_alpha;
              if (l > 1) {
                it.out = h->d_act[l - 1] + h->act_off[l - 1][e] + (size_t)a0 * M * nin + (size_t)m * nin + n0;
                it.ldo = M * nin;
                it.aux = it.out; it.ldaux = it.ldo;
                it.epi = EPI_MUL_DCELU;
              } else {
                it.out = h->d_daev + ((size_t)m * N + h->grp_off[e] + a0) * n_feat + n0;
                it.ldo = n_feat;
                it.epi = EPI_SCALE;
                it.scale = 1.0f / (float)M;
              }
              if (l == L - 1 && !h->use_mid) {
                it.w_last = h->d_W + h->w_off[e * L + L - 1] + (size_t)m * nout;
                it.b_last = B[h->b_off[e * L + L - 1] + m];
                if (n0 == 0) {
                  it.e_out = h->d_eatom + (size_t)(h->grp_off[e] + a0) * M + m;
                  it.lde = M;
                }
              }
              items.push_back(it);
            }
        }
      }
      SmallLaunch sl;
      sl.name = "mlp_bwd_l" + std::to_string(l);
      if (bwd1 ? small_build_bwd1(sl, items, wops) : small_build_bwd(sl, items)) { small_free_launch(sl); return fail(NNP_ERR_CUDA); }
      h->sbwd.push_back(sl);
    }
  }
  // last layer
  {
    std::vector<long long> ao(S), wo2(S), bo2(S);
    std::vector<int> Hs(S);
    for (int e = 0; e < S; ++e) {
      ao[e] = h->act_off[L - 1][e];
      wo2[e] = h->w_off[e * L + L - 1];
      bo2[e] = h->b_off[e * L + L - 1];
      Hs[e] = h->dims[e * (L + 1) + L - 1];
      const int ne = h->grp_off[e + 1] - h->grp_off[e];
      flops += 4.0 * ne * (double)M * Hs[e];
      if (ne) wbytes += 4.0 * M * Hs[e];
    }
    LastLayerArgs& la = h->last;
    memset(&la, 0, sizeof(la));
    la.act = h->d_act[L - 1]; la.act_lo = h->d_act_lo[L - 1]; la.act_full = h->fuse_delta ? h->d_act_full : nullptr; la.W = h->d_W; la.bias = h->d_b; la.e_out = h->d_eatom;
    for (int e = 0; e <= S; ++e) la.grp_off[e] = h->grp_off[e];
    for (int e = 0; e < S; ++e) {
      la.act_off[e] = ao[e]; la.w_off[e] = wo2[e]; la.b_off[e] = bo2[e]; la.H[e] = Hs[e];
    }
    la.S = S; la.M = M; la.n_sorted = N; la.alpha = alpha;
  }
  h->work[0] = wbytes;
  h->work[1] = flops;
  h->work[2] = 2.0 * 4.0 * (double)N * n_feat;
  h->work[3] = w1bytes;

  if (h->fuse_nbr) h->stage_names = {"aev_fwd"};  // the AEV forward kernel builds the neighbour rows itself
  else h->stage_names = {"nbr", "aev_fwd"};
  if (h->use_small) {
    for (auto& g : h->sfwd) h->stage_names.push_back(g.name);
    if (h->use_mid) h->stage_names.push_back(h->smid.name);
    for (auto& g : h->sbwd) h->stage_names.push_back(g.name);
  } else {
    for (auto& g : h->fwd) h->stage_names.push_back(g.name);
    h->stage_names.push_back("mlp_last");
    for (auto& g : h->bwd) h->stage_names.push_back(g.name);
  }
  h->stage_names.push_back("aev_bwd");
  h->stage_names.push_back("finish");
  h->stage_issued.assign(h->stage_names.size(), 0.0);
  h->stage_tile.assign(h->stage_names.size(), 0);
  h->stage_bytes.assign(h->stage_names.size(), 0.0);
  if (h->use_umma)
    for (size_t k = 0; k < h->stage_names.size(); ++k)
      for (auto* v : {&h->ufwd, &h->ubwd})
        for (auto& g : *v)
          if (g.name == h->stage_names[k]) {
            h->stage_issued[k] = g.issued_flops;
            h->stage_tile[k] = g.tile;
            h->stage_bytes[k] = g.algo_bytes;
          }
  h->n_launches = N > 0 ? (int)h->stage_names.size() + (h->use_cells ? 4 : 0) : 0;  // cell path: 5 kernels in "nbr"
  h->events.resize(h->stage_names.size() + 1);
  for (auto& e : h->events)
    if (cudaEventCreate(&e) != cudaSuccess) return fail(NNP_ERR_CUDA);
  if (cudaDeviceSynchronize() != cudaSuccess) return fail(NNP_ERR_CUDA);
  *out = h;
  return NNP_OK;
}

// enqueue the launch chain A1..A8 on `s`; with `ev` record an event before the first and after each stage
static void enqueue_chain(nnp_handle* h, const float* d_pos, int ps, const int* d_idx, double* d_energy,
                          void* d_force, int fs, int fixed, cudaStream_t s, bool ev) {
  int k = 0;
  auto mark = [&]() {
    if (ev) cudaEventRecord(h->events[k], s);
    ++k;
  };
  h->pdl_now = h->use_pdl && !ev;  // event records between the kernels would break the programmatic edges
  const bool pdl = h->pdl_now;
  mark();
  if (!h->fuse_nbr) { launch_neighbors(h, d_pos, ps, d_idx, s); mark(); }
  launch_aev_forward(h, d_pos, ps, d_idx, s); mark();
  if (h->use_small) {  // per-atom energies and delta_L-1 come out of the first backward launch
    for (auto& g : h->sfwd) { small_launch_fwd(g, s, pdl); mark(); }
    if (h->use_mid) { mid_launch(h->smid, s, pdl); mark(); }
    for (auto& g : h->sbwd) { small_launch_bwd(g, s, pdl); mark(); }
    launch_aev_backward(h, s); mark();
    launch_finish(h, d_idx, d_energy, d_force, fs, fixed, s); mark();
    return;
  }
  if (h->use_umma) {
    for (auto& g : h->ufwd) { umma_launch(g, s, pdl); mark(); }
  } else {
    for (auto& g : h->fwd) { launch_gemm(g, s); mark(); }
  }
  launch_last_layer(h, s); mark();
  if (h->use_umma) {
    for (auto& g : h->ubwd) { umma_launch(g, s, pdl); mark(); }
  } else {
    for (auto& g : h->bwd) { launch_gemm(g, s); mark(); }
  }
  launch_aev_backward(h, s); mark();
  launch_finish(h, d_idx, d_energy, d_force, fs, fixed, s); mark();
}

static int compute_impl(nnp_handle* h, const float* d_pos, int ps, const int* d_atom_index, double* d_energy, void* d_force,
                        int fs, int fixed, cudaStream_t s) {
  if (!h) return NNP_ERR_INVALID_ARG;
  if (h->N == 0) {  // no atoms: every (empty) molecule has energy 0; d_energy is WRITTEN as documented
    if (d_energy) CK(cudaMemsetAsync(d_energy, 0, sizeof(double) * (size_t)h->n_mol, s));
    h->last_stream = s;
    return NNP_OK;
  }
  if (!d_pos || ps < 3 || (d_force && fs < 3)) return NNP_ERR_INVALID_ARG;
  h->last_stream = s;
  if (h->profiling || (h->flags & NNP_FLAG_NO_GRAPH)) {
    enqueue_chain(h, d_pos, ps, d_atom_index, d_energy, d_force, fs, fixed, s, h->profiling);
    return cudaGetLastError() == cudaSuccess ? NNP_OK : NNP_ERR_CUDA;
  }
  nnp_handle::GraphSlot* slot = nullptr;
  for (auto& g : h->graphs)
    if (g.exec && g.pos == d_pos && g.idx == d_atom_index && g.energy == d_energy && g.force == d_force && g.ps == ps &&
        g.fs == fs && g.fixed == fixed)
      slot = &g;
  if (!slot) {
    slot = &h->graphs[0];  // a free entry, else the least recently used one
    for (auto& g : h->graphs) {
      if (!g.exec) { slot = &g; break; }
      if (g.used < slot->used) slot = &g;
    }
    if (slot->exec) {
      cudaGraphExecDestroy(slot->exec);
      slot->exec = nullptr;
    }
    cudaStream_t cs;
    CK(cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));
    cudaGraph_t graph = nullptr;
    if (cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
      cudaStreamDestroy(cs);
      return NNP_ERR_CUDA;
    }
    enqueue_chain(h, d_pos, ps, d_atom_index, d_energy, d_force, fs, fixed, cs, false);
    cudaError_t e = cudaStreamEndCapture(cs, &graph);
    cudaStreamDestroy(cs);
    if (e != cudaSuccess || !graph) return NNP_ERR_CUDA;
    e = cudaGraphInstantiate(&slot->exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) {
      slot->exec = nullptr;
      return NNP_ERR_CUDA;
    }
    slot->pos = d_pos; slot->idx = d_atom_index; slot->energy = d_energy; slot->force = d_force;
    slot->ps = ps; slot->fs = fs; slot->fixed = fixed;
  }
  slot->used = ++h->graph_clock;
  CK(cudaGraphLaunch(slot->exec, s));
  return NNP_OK;
}

extern "C" int nnp_compute(nnp_handle* h, const float* d_pos, int32_t pos_stride_floats,
                           const int32_t* d_atom_index, double* d_energy, float* d_force_accum,
                           int32_t force_stride_floats, void* cuda_stream) {
  return compute_impl(h, d_pos, pos_stride_floats, d_atom_index, d_energy, d_force_accum, force_stride_floats, 0,
                      (cudaStream_t)cuda_stream);
}

extern "C" int nnp_compute_fixed(nnp_handle* h, const float* d_pos, int32_t pos_stride_floats,
                                 const int32_t* d_atom_index, double* d_energy, int64_t* d_force_fixed,
                                 int32_t force_stride_int64, void* cuda_stream) {
  return compute_impl(h, d_pos, pos_stride_floats, d_atom_index, d_energy, d_force_fixed, force_stride_int64, 1,
                      (cudaStream_t)cuda_stream);
}

extern "C" int nnp_compute_async(nnp_handle* h, const float* d_pos, int32_t pos_stride_floats,
                                 const int32_t* d_atom_index, double* d_energy, void* d_force, int32_t force_stride,
                                 int32_t force_is_fixed64, void* wait_event, void* done_event) {
  if (!h) return NNP_ERR_INVALID_ARG;
  if (!h->own_stream) CK(cudaStreamCreateWithFlags(&h->own_stream, cudaStreamNonBlocking));
  if (wait_event) CK(cudaStreamWaitEvent(h->own_stream, (cudaEvent_t)wait_event, 0));
  const int rc = compute_impl(h, d_pos, pos_stride_floats, d_atom_index, d_energy, d_force, force_stride,
                              force_is_fixed64 ? 1 : 0, h->own_stream);
  if (rc != NNP_OK) return rc;
  if (done_event) CK(cudaEventRecord((cudaEvent_t)done_event, h->own_stream));
  return NNP_OK;
}

extern "C" int nnp_compute_host(nnp_handle* h, const float* pos_host, double* energy_host, float* force_host,
                                void* cuda_stream) {
  if (!h || (h->N > 0 && !pos_host)) return NNP_ERR_INVALID_ARG;
  if (h->N == 0) {
    if (energy_host) memset(energy_host, 0, sizeof(double) * (size_t)h->n_mol);
    return NNP_OK;
  }
  cudaStream_t s = (cudaStream_t)cuda_stream;
  // Zero-copy staging: the positions go into a pinned block of the library (a host memcpy of 12 N bytes) that the
  // first kernel reads through its device alias, and the finish kernel WRITES energies and forces straight into a
  // second pinned block; the call is then one graph launch and one stream synchronisation -- no copy engine
  // operations, no memset (each costs 2-4 us of launch latency at ligand sizes).
  memcpy(h->h_hpos, pos_host, sizeof(float) * 3 * (size_t)h->N);
  int rc = compute_impl(h, h->d_hpos_alias, 3, nullptr, reinterpret_cast<double*>(h->d_hout_alias),
                        h->d_hout_alias + h->hout_force_off, 3, 2, s);
  if (rc != NNP_OK) return rc;
  CK(cudaStreamSynchronize(s));
  if (energy_host) memcpy(energy_host, h->h_hout, sizeof(double) * (size_t)h->n_mol);
  if (force_host) memcpy(force_host, h->h_hout + h->hout_force_off, sizeof(float) * 3 * (size_t)h->N);
  return NNP_OK;
}

extern "C" int nnp_status(nnp_handle* h) {
  if (!h) return NNP_ERR_INVALID_ARG;
  if (cudaStreamSynchronize(h->last_stream) != cudaSuccess) return NNP_ERR_CUDA;
  int st = 0;
  if (cudaMemcpy(&st, h->d_status, sizeof(int), cudaMemcpyDeviceToHost) != cudaSuccess) return NNP_ERR_CUDA;
  if (cudaGetLastError() != cudaSuccess) return NNP_ERR_CUDA;
  if (st) cudaMemset(h->d_status, 0, sizeof(int));
  if (st & NNP_ST_NONFINITE) return NNP_ERR_NONFINITE;
  if (st & NNP_ST_CAPACITY) return NNP_ERR_CAPACITY;
  return NNP_OK;
}

extern "C" int nnp_launches_per_compute(nnp_handle* h) { return h ? h->n_launches : 0; }
extern "C" int nnp_n_features(nnp_handle* h) { return h ? h->n_feat : 0; }

extern "C" int nnp_set_profiling(nnp_handle* h, int32_t enable) {
  if (!h) return NNP_ERR_INVALID_ARG;
  h->profiling = enable != 0;
  return NNP_OK;
}

extern "C" int nnp_get_stage_times(nnp_handle* h, float* ms_host, int32_t capacity, int32_t* n_stages) {
  if (!h || !n_stages) return NNP_ERR_INVALID_ARG;
  const int n = (int)h->stage_names.size();
  *n_stages = n;
  if (!ms_host) return NNP_OK;
  CK(cudaStreamSynchronize(h->last_stream));
  for (int k = 0; k < n && k < capacity; ++k) {
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, h->events[k], h->events[k + 1]));
    ms_host[k] = ms;
  }
  return NNP_OK;
}

extern "C" const char* nnp_stage_name(nnp_handle* h, int32_t stage) {
  if (!h || stage < 0 || stage >= (int)h->stage_names.size()) return "";
  return h->stage_names[stage].c_str();
}

extern "C" int nnp_get_stage_work(nnp_handle* h, int32_t stage, double* issued_flops_host, int32_t* atom_tile_host) {
  if (!h || stage < 0 || stage >= (int)h->stage_names.size()) return NNP_ERR_INVALID_ARG;
  if (issued_flops_host) *issued_flops_host = h->stage_issued[stage];
  if (atom_tile_host) *atom_tile_host = h->stage_tile[stage];
  return NNP_OK;
}

extern "C" int nnp_get_stage_bytes(nnp_handle* h, int32_t stage, double* bytes_host) {
  if (!h || !bytes_host || stage < 0 || stage >= (int)h->stage_names.size()) return NNP_ERR_INVALID_ARG;
  *bytes_host = h->stage_bytes[stage];
  return NNP_OK;
}

extern "C" int nnp_get_work(nnp_handle* h, double* what_host, int32_t n) {
  if (!h || !what_host) return NNP_ERR_INVALID_ARG;
  for (int k = 0; k < n && k < 4; ++k) what_host[k] = h->work[k];
  return NNP_OK;
}

// ---------------------------------------------------------------- debug / parity exports
extern "C" int nnp_debug_pairs(nnp_handle* h, int32_t which, int64_t* n_pairs, int32_t* ij_host, int64_t capacity) {
  if (!h || !n_pairs || (which != 0 && which != 1)) return NNP_ERR_INVALID_ARG;
  CK(cudaStreamSynchronize(h->last_stream));
  const int N = h->N;
  std::vector<int> nr((size_t)N * h->capR), cr(N), na((size_t)N * h->capA), ca(N);
  if (N) {
    CK(cudaMemcpy(nr.data(), h->d_nbr_r, nr.size() * sizeof(int), cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(cr.data(), h->d_cnt_r, cr.size() * sizeof(int), cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(na.data(), h->d_nbr_a, na.size() * sizeof(int), cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(ca.data(), h->d_cnt_a, ca.size() * sizeof(int), cudaMemcpyDeviceToHost));
  }
  int64_t cnt = 0;
  for (int i = 0; i < N; ++i) {
    const int n = which == 0 ? cr[i] : ca[i];
    for (int q = 0; q < n; ++q) {
      const int j = which == 0 ? nr[(size_t)i * h->capR + q] : nr[(size_t)i * h->capR + na[(size_t)i * h->capA + q]];
      if (ij_host && cnt < capacity) {
        ij_host[2 * cnt] = i;
        ij_host[2 * cnt + 1] = j;
      }
      ++cnt;
    }
  }
  *n_pairs = cnt;
  return NNP_OK;
}

static int export_rows(nnp_handle* h, const float* d_rows, float* host) {
  if (!h || !host) return NNP_ERR_INVALID_ARG;
  CK(cudaStreamSynchronize(h->last_stream));
  std::vector<float> tmp((size_t)h->N * h->n_feat);
  std::vector<int> sortpos(h->N);
  if (h->N) {
    CK(cudaMemcpy(tmp.data(), d_rows, tmp.size() * sizeof(float), cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(sortpos.data(), h->d_sortpos, sortpos.size() * sizeof(int), cudaMemcpyDeviceToHost));
  }
  for (int i = 0; i < h->N; ++i)
    memcpy(host + (size_t)i * h->n_feat, &tmp[(size_t)sortpos[i] * h->n_feat], sizeof(float) * h->n_feat);
  return NNP_OK;
}

extern "C" int nnp_debug_aev(nnp_handle* h, float* aev_host) {
  if (!h) return NNP_ERR_INVALID_ARG;
  int rc = export_rows(h, h->d_aev, aev_host);
  if (rc != NNP_OK || !h->d_aev_lo) return rc;
  std::vector<float> lo((size_t)h->N * h->n_feat);  // tensor engine: the row is stored split, G = hi + lo exactly
  rc = export_rows(h, h->d_aev_lo, lo.data());
  for (size_t i = 0; rc == NNP_OK && i < lo.size(); ++i) aev_host[i] += lo[i];
  return rc;
}
extern "C" int nnp_debug_daev(nnp_handle* h, float* g_host) {
  if (!h) return NNP_ERR_INVALID_ARG;
  int rc = export_rows(h, h->d_daev, g_host);
  if (rc != NNP_OK || h->n_parts == 1) return rc;
  std::vector<float> part((size_t)h->N * h->n_feat);
  for (int p = 1; p < h->n_parts; ++p) {
    rc = export_rows(h, h->d_daev + (size_t)p * h->N * h->n_feat, part.data());
    if (rc != NNP_OK) return rc;
    for (size_t i = 0; i < part.size(); ++i) g_host[i] += part[i];
  }
  return NNP_OK;
}

extern "C" int nnp_debug_atomic_energies(nnp_handle* h, double* e_host) {
  if (!h || !e_host) return NNP_ERR_INVALID_ARG;
  CK(cudaStreamSynchronize(h->last_stream));
  std::vector<double> tmp((size_t)h->N * h->M);
  std::vector<int> sortpos(h->N);
  if (h->N) {
    CK(cudaMemcpy(tmp.data(), h->d_eatom, tmp.size() * sizeof(double), cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(sortpos.data(), h->d_sortpos, sortpos.size() * sizeof(int), cudaMemcpyDeviceToHost));
  }
  for (int i = 0; i < h->N; ++i)
    for (int m = 0; m < h->M; ++m) e_host[(size_t)m * h->N + i] = tmp[(size_t)sortpos[i] * h->M + m];
  return NNP_OK;
}

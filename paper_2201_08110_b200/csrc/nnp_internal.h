// Internal declarations of libnnp_b200 (CUDA, sm_100a).  Not part of the C ABI (include/nnp.h).
// Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "nnp.h"

#define NNP_MAX_SHF_R 32
#define NNP_MAX_SHF_A 16
#define NNP_MAX_SHF_Z 8
#define NNP_MAX_SUB 64
#define NNP_MAX_SPECIES 16
#define NNP_MAX_LAYERS 8

// device status bits (sticky)
#define NNP_ST_CAPACITY 1
#define NNP_ST_NONFINITE 2

// ---- programmatic dependent launch (PDL): a kernel launched with the attribute may start while its
// predecessor in the stream is still running; everything it does before pdl_wait() must touch only data that is
// constant after nnp_create (items, weights, topology).  pdl_wait() returns when the predecessor grid has
// completed and its writes are visible; pdl_trigger() lets the successor start launching.  Both are no-ops for
// plain launches.  Every CTA of every kernel in the chain calls pdl_wait() (completion is then transitive).
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <typename... KArgs, typename... Args>
inline cudaError_t launch_kernel(bool pdl, void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s,
                                 Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}
#endif

// AEV constants, passed by value to kernels.
struct AevConst {
  int S, n_shf_r, n_shf_a, n_shf_z, n_sub, n_radial, n_feat;
  float rc_r, rc_a, eta_r, eta_a, zeta, cos_scale, length_scale;
  double rc_r2, rc_a2;  // ((double)(float)Rc)^2, the O2 predicate thresholds
  int zeta_int, zeta1_int;     // floor(zeta), floor(zeta - 1)
  float zeta_frac;             // zeta - floor(zeta)
  float kr_hi, kr_lo, ka_hi, ka_lo;  // -eta*log2(e) as hi+lo: exp(-eta d^2) = ex2(d^2 k)
  float shf_r[NNP_MAX_SHF_R];
  float shf_a[NNP_MAX_SHF_A];
  float cos_z[NNP_MAX_SHF_Z];  // cos(ShfZ_z), sin(ShfZ_z): cos(theta - ShfZ) = c cosZ + s sinZ
  float sin_z[NNP_MAX_SHF_Z];
  float cos_z_lo[NNP_MAX_SHF_Z];  // low parts: cos_z + cos_z_lo = cos(ShfZ) to ~2^-48 (a rounded constant
  float sin_z_lo[NNP_MAX_SHF_Z];  // is a coherent error amplified by zeta)
};

// One GEMM of a grouped launch: C[m][n] = epi( sum_k A[m][k] * Bop[k][n] ).
struct GemmProblem {
  const float* A;
  const float* B;
  float* C;
  const float* bias;  // [N] or null (EPI_BIAS_CELU)
  const float* aux;   // [M][ldaux] activations h for EPI_MUL_DCELU (may alias C)
  int M, N, K;
  int lda, ldb, ldc, ldaux;
  int transB;  // 0: B is [N][K] (k contiguous, forward);  1: B is [K][N] (n contiguous, backward)
  int epi;
  float scale;
  float alpha;  // CELU alpha
  float inv_alpha;
};
enum { EPI_BIAS_CELU = 0, EPI_MUL_DCELU = 1, EPI_SCALE = 2, EPI_BIAS_CELU_LAST = 3 };

struct GemmTile {
  int prob, m0, n0, cfg;
};

struct GemmLaunch {
  GemmProblem* d_probs = nullptr;
  GemmTile* d_tiles = nullptr;
  int n_tiles = 0;
  std::string name;
  double flops = 0, weight_bytes = 0;
};

// a row-major f32 matrix [rows][cols] with pitch ld floats, as a TMA tensor-map operand
struct TmaOperand {
  const float* base;
  long long rows, cols, ld;
};

// ---- tcgen05 engine (mlp_umma.cu): D[f][a] = sum_k A[f][k] B[a][k], f = output feature, a = atom.
// Both operands arrive PRE-SPLIT for 3xTF32: every matrix is a pair of planes (hi, lo) with hi = rna_tf32(x),
// lo = x - hi (activations, written by the producing kernel) or rna_tf32(x - hi) (weights, split at create time).
struct UmmaOperand {         // a row-major f32 matrix pair [rows][cols], pitch ld floats
  const float* hi;
  const float* lo;
  long long rows, cols, ld;
};
struct UmmaItem {            // one tile of one GEMM, as the persistent CTAs consume it
  int amap, bmap;            // tensor-map slots (weights / activations)
  int a_c0, a_c1;            // weight box origin (k col, feature row)
  int b_c0, b_c1;            // activation box origin (k col, atom row)
  int nkb;                   // contraction boxes (32 wide) of the item
  unsigned long long kmask;  // non-zero: the boxes actually loaded are the set bits (popcount = nkb)
  int n_pad, n_valid, f_valid;  // MMA N (16/32/64/128), atoms and feature rows actually stored
  int epi, ldc, ldaux;
  float* C;                  // C[a * ldc + f]: hi plane (or the whole value when C_lo is null)
  float* C_lo;               // lo plane of the output, or null
  const float* bias;         // [f] or null
  const float* aux;          // aux[a * ldaux + f]: activations h (hi plane) for EPI_MUL_DCELU (may alias C)
  const float* aux_lo;       // lo plane of h (may alias C_lo), or null
  // EPI_BIAS_CELU_LAST (forward through the last hidden layer): h goes to C_full as ONE plane (the 1-output layer's
  // FP64 dot product reads it) and C / C_lo receive delta = w_last * CELU'(h), the operand of the backward pass
  float* C_full;
  const float* w_last;       // [f] weights of the 1-output layer for this tile's features
  float scale, alpha, inv_alpha;
  // K-split tail items (EPI_SCALE launches): the item is one of split_n parts of a tile's contraction.  A part runs
  // nkb boxes starting at box kb_skip of the tile's (live) box list, writes its raw partial tile to
  // scratch[split_idx][128 atoms][128 features] and takes a ticket; the part that draws the last ticket adds the
  // split_n partial tiles in index order (fixed order => bit-identical reruns) and runs the epilogue.  split_n = 0:
  // a whole tile.
  int kb_skip, split_n, split_idx;
  float* scratch;
  unsigned int* ticket;
};
struct UmmaProblem {
  unsigned long long kmask;    // non-zero: contraction boxes (32 wide) to run; the others multiply structural zeros
  unsigned long long fmask;    // non-zero: 128-feature output tiles to run; the others are never read downstream
  int amap, bmap;
  int a_c0, a_c1, b_c0, b_c1;  // origins of feature 0 / atom 0 / contraction element 0
  int F, n_atoms, K;
  int epi, ldc, ldaux;
  float* C;
  float* C_lo;
  const float* bias;
  const float* aux;
  const float* aux_lo;
  float* C_full;
  const float* w_last;
  float scale, alpha, inv_alpha;
};
struct UmmaLaunch {
  void* params = nullptr;  // UmmaParams (host copy, passed by value as __grid_constant__)
  UmmaItem* d_items = nullptr;
  int* d_cta_off = nullptr;
  int n_items = 0, grid = 0, tile = 0;
  size_t smem_bytes = 0;
  bool pair = false;       // built by the CTA-pair engine (mlp_umma2.cu)
  double issued_flops = 0;
  double algo_bytes = 0;   // operand planes read once + output planes written once + epilogue reads  // 2 x MACs of the boxes actually run (padding and structural zeros excluded/included as issued)
  float* d_split_scratch = nullptr;        // partial tiles of the K-split tail items
  unsigned int* d_split_tickets = nullptr; // one arrival counter per split tile (zero between launches)
  int n_split_tiles = 0, split_n = 0;
  std::string name;
};
int umma_init();
int umma_build_launch(UmmaLaunch& L, const std::vector<UmmaProblem>& probs, const std::vector<UmmaOperand>& aops,
                      const std::vector<UmmaOperand>& bops, int num_sms, bool reverse = false,
                      bool tail_split = true);
void umma_launch(const UmmaLaunch& L, cudaStream_t s, bool pdl);
void umma_free_launch(UmmaLaunch& L);
// CTA-pair variant (cta_group::2, 256 x 256 tiles): opt-in (NNP_FLAG_UMMA_PAIRS), measured slower
int umma2_init();
bool umma2_suits(const std::vector<UmmaProblem>& probs);
int umma2_build_launch(UmmaLaunch& L, const std::vector<UmmaProblem>& probs, const std::vector<UmmaOperand>& aops,
                       const std::vector<UmmaOperand>& bops, int num_sms);
void umma2_launch(const UmmaLaunch& L, cudaStream_t s, bool pdl);
void umma2_free_params(UmmaLaunch& L);

// ---- ligand-size engine (mlp_small.cu): weight-streaming FFMA kernels, one CTA per item
struct SmallFwdItem {       // out[a*ldc + r] = CELU(bias[r] + sum_k W[r*K + k] X[a*ldx + k]),  r < n_rows, a < n_atoms
  const float* W;           // first weight row of the item (row-major, pitch K)
  const float* X;           // activations of the item's first atom (model columns already applied)
  const float* bias;        // bias of the first row, or null
  float* out;               // output of (first atom, first row)
  int ldx, ldc, n_atoms, K, n_rows;  // n_atoms <= 32, n_rows even, K % 4 == 0
  float alpha, inv_alpha;
};
struct SmallBwdItem {       // out[a*ldo + n] = epi(sum_o D[a*ldd + o] W[o*ldw + n]),  n < n_cols (<= 128)
  const float* W;           // weights at (row 0, first column of the chunk)
  const float* D;           // delta (or, with w_last, the activation h) of the item's first atom
  float* out;               // output at (first atom, first column)
  const float* aux;         // EPI_MUL_DCELU: stored activation at the same place as out (may alias it)
  const float* w_last;      // non-null: D holds h of the last hidden layer, delta[o] = w_last[o] * CELU'(h[o])
  double* e_out;            // non-null (with w_last): e_out[a*lde] = b_last + w_last . h  (FP64)
  int ldw, ldd, ldo, ldaux, lde;
  int n_atoms, n_out, n_cols;  // n_atoms <= 32, n_out % 4 == 0, n_cols % 4 == 0
  int epi, AW, G;           // atoms per warp (1..4), atom groups (1,2,4,8): G*AW >= n_atoms
  int tmap, t_row0, t_col0; // persistent layer-1 kernel: tensor map of the element's layer-1 block, row / column origin
  float scale, inv_alpha, b_last;
};
struct Fwd1Item {            // persistent layer-1 forward item: one CTA, a run of weight rows of one element
  const float* W;            // first weight row of the run (row-major, pitch K); rows of all models are contiguous
  const float* X;            // AEV row of the item's first atom (pitch ldx)
  const float* bias;         // bias of the first row, or null
  float* out;                // out[a*ldc + r] at (first atom, first row)
  int ldx, ldc, n_atoms, K, n_rows;  // n_atoms <= 24, K % 4 == 0
  float alpha, inv_alpha;
};
struct SmallLaunch {
  void* d_items = nullptr;
  int n_items = 0, variant = 1;
  int grid = 0, stages = 0;  // persistent kernels: CTAs and ring depth
  void* params = nullptr;    // persistent layer-1 backward: host copy of its __grid_constant__ parameter block
  void* d_aux = nullptr;     // persistent layer-1 backward: per-CTA item ranges (device)
  size_t smem_bytes = 0;
  std::string name;
};
int small_init();
void small_bwd_shape(int n_atoms, int* AW, int* G);
int small_build_fwd(SmallLaunch& L, std::vector<SmallFwdItem>& items);
int small_build_bwd(SmallLaunch& L, std::vector<SmallBwdItem>& items);
int small_build_bwd1(SmallLaunch& L, std::vector<SmallBwdItem>& items,
                     const std::vector<TmaOperand>& wops);  // wops[tmap]: the [rows][cols] layer-1 weight block of an element
int small_build_fwd1(SmallLaunch& L, std::vector<Fwd1Item>& items);
int small_fwd1_tile_rows();  // layer 1: persistent, weights streamed through a ring  // layer 1: weights read once, FFMA2
void small_launch_fwd(const SmallLaunch& L, cudaStream_t s, bool pdl);
void small_launch_bwd(const SmallLaunch& L, cudaStream_t s, bool pdl);
void small_free_launch(SmallLaunch& L);

// ---- ligand-size engine, fused middle of the network (mlp_mid.cu): layers 2..L-1 forward, the final
// 1-output layer + per-atom energies, and the backward pass down to delta_1, one CTA per item
struct MidItem {
  const float* W[NNP_MAX_LAYERS];     // W[l], l = 2..L-1: weights of layer l of this (element, model), [H_l][H_{l-1}]
  const float* bias[NNP_MAX_LAYERS];  // bias[l] or null
  const float* w_last;                // [H_{L-1}] weights of the 1-output layer L
  float* h1;                          // in: h_1 of the item's first atom (model columns applied); out: delta_1
  double* e_out;                      // e_out[a * lde] = b_L + w_L . h_{L-1}
  int H[NNP_MAX_LAYERS];              // H[l], l = 1..L-1 (each <= 256, % 4 == 0)
  int L, n_atoms, ld1, lde;           // n_atoms <= 4
  float b_last, alpha, inv_alpha;
};
int mid_init();
bool mid_supported(int L, const int* dims_of_element);  // dims: [L+1]
int mid_build(SmallLaunch& L, std::vector<MidItem>& items);
void mid_launch(const SmallLaunch& L, cudaStream_t s, bool pdl);

// Final layer (1 output) + start of the backward pass.
struct EnergyBlock {  // one CTA of the energy reduction: atoms [a0, a1) of molecule `mol`
  int mol, a0, a1;
  int first, n_chunks;  // this molecule's CTAs are blocks [first, first + n_chunks) of the energy part
};

struct LastLayerArgs {
  float* act;          // [n_atoms_sorted][M][H] per element group (arena), overwritten with delta
  float* act_lo;       // tensor engine: lo plane of the same arena (h = act + act_lo; delta is written split), else null
  const float* act_full;  // tensor engine with the fused delta: h of the last hidden layer as one plane (energies only)
  const float* W;      // arena
  const float* bias;   // arena
  double* e_out;       // [n_sorted][M]
  // per-element tables by value (kernel parameter space: no dependent global loads before the data loads)
  int grp_off[NNP_MAX_SPECIES + 1];       // [S+1]
  long long act_off[NNP_MAX_SPECIES];     // [S] float offset of the group's block in act
  long long w_off[NNP_MAX_SPECIES];       // [S] float offset of W_L for (e, m=0); models contiguous with stride H
  long long b_off[NNP_MAX_SPECIES];       // [S]
  int H[NNP_MAX_SPECIES];                 // [S]
  int S, M, n_sorted;
  float alpha;
};

struct nnp_handle {
  int device = 0;
  int N = 0, n_mol = 0, S = 0, M = 0, L = 0, n_feat = 0;
  int capR = 0, capA = 0;
  int flags = 0;
  double energy_scale = 1.0, length_scale = 1.0;
  AevConst aev;
  std::vector<int> dims;     // [S][L+1]
  std::vector<int> grp_off;  // [S+1] host
  // device: topology
  int* d_mol_range = nullptr;  // [N][2] (first atom, end) of every atom's molecule
  int *d_species = nullptr, *d_mol_off = nullptr, *d_mol_id = nullptr, *d_sortpos = nullptr, *d_perm = nullptr,
      *d_grp_off = nullptr;
  double* d_self_energy = nullptr;
  // device: per-step workspace
  float4* d_pos4 = nullptr;
  int *d_nbr_r = nullptr, *d_nbr_a = nullptr, *d_cnt_r = nullptr, *d_cnt_a = nullptr;
  float* d_aev = nullptr;   // [N sorted][n_feat]
  float* d_aev_lo = nullptr;  // tensor engine: lo plane (d_aev then holds rna_tf32(G), d_aev_lo = G - that)
  float* d_daev = nullptr;  // [n_parts][N sorted][n_feat]
  unsigned long long* d_facc = nullptr;  // [N][3] fixed-point force accumulator (AEV backward adds, finish reads + clears)
  double* d_eatom = nullptr;  // [N sorted][M]
  EnergyBlock* d_eblocks = nullptr;  // energy reduction: large molecules are summed by several CTAs
  double* d_epart = nullptr;         // [n_eblocks] partial sums
  int* d_ecount = nullptr;           // [n_mol] arrival counters (reset by the last CTA of a molecule)
  int n_eblocks = 0;
  // cell-binned neighbour search (nbr_cells.cu), used for large molecules
  bool use_cells = false;
  bool fuse_nbr = false;  // small molecules: the AEV forward kernel builds the neighbour rows itself
  void* d_cell_grid = nullptr;
  int *d_cell_count = nullptr, *d_cell_start = nullptr, *d_cell_of = nullptr, *d_cell_rank = nullptr,
      *d_cell_atoms = nullptr, *d_cell_mol = nullptr;  // cell_mol: molecule of every atom, in cell order
  unsigned long long aev_live_boxes = 0;  // 32-column boxes of the AEV that are not structural zeros (0: all)
  float4* d_cell_pos4 = nullptr;                        // positions (+ species) in cell order
  int* d_status = nullptr;
  // weights
  float *d_W = nullptr, *d_b = nullptr;
  // tensor engine: weights split for 3xTF32 (hi, lo), in the forward layout and transposed for the backward pass
  float *d_Whi = nullptr, *d_Wlo = nullptr, *d_WThi = nullptr, *d_WTlo = nullptr;
  std::vector<long long> w_off, b_off;  // [S][L] float offsets of the (e,l) block, models contiguous
  size_t w_floats = 0, b_floats = 0;
  // activations: act[l] for l = 1..L-1
  float* d_act[NNP_MAX_LAYERS] = {nullptr};
  float* d_act_lo[NNP_MAX_LAYERS] = {nullptr};  // tensor engine: lo planes
  float* d_act_full = nullptr;                  // tensor engine: h_{L-1} as one plane (see EPI_BIAS_CELU_LAST)
  bool fuse_delta = false;
  std::vector<long long> act_off[NNP_MAX_LAYERS];  // [S] float offsets
  // MLP launches
  std::vector<GemmLaunch> fwd, bwd;  // fwd: layers 1..L-1; bwd: layers L-1..1
  std::vector<UmmaLaunch> ufwd, ubwd; // the same launches on the tcgen05 engine (used when use_umma)
  std::vector<SmallLaunch> sfwd, sbwd; // ligand-size engine (used when use_small); no separate last-layer launch
  SmallLaunch smid;                    // fused middle launch of the ligand-size engine (used when use_mid)
  bool use_umma = false, use_small = false, use_mid = false;
  bool use_pdl = false, pdl_now = false;  // programmatic dependent launches along the chain (pdl_now: this enqueue)
  int n_parts = 1;                   // dE/dAEV is produced as n_parts partial sums (per model at small N)
  LastLayerArgs last;
  // host staging for nnp_compute_host
  // nnp_compute_host: pinned, device-mapped host blocks (positions in; energies then forces out) and their device
  // aliases: the kernels read / write them directly
  float* h_hpos = nullptr;
  const float* d_hpos_alias = nullptr;
  unsigned char* h_hout = nullptr;
  unsigned char* d_hout_alias = nullptr;
  size_t hout_bytes = 0, hout_force_off = 0;
  // graphs: one instantiated graph per distinct argument tuple, a small LRU (an engine that double-buffers its
  // positions or forces alternates between two of them at no cost)
  struct GraphSlot {
    cudaGraphExec_t exec = nullptr;
    const void* pos = nullptr;
    const void* idx = nullptr;
    void *energy = nullptr, *force = nullptr;
    int ps = 0, fs = 0, fixed = 0;
    unsigned long long used = 0;
  };
  GraphSlot graphs[4];
  unsigned long long graph_clock = 0;
  cudaStream_t last_stream = nullptr;
  cudaStream_t own_stream = nullptr;  // nnp_compute_async: library-owned stream
  // profiling
  bool profiling = false;
  std::vector<cudaEvent_t> events;
  std::vector<std::string> stage_names;
  std::vector<double> stage_issued, stage_bytes;  // tensor-engine stages: 2 x MACs actually issued (structural zeros skipped)
  std::vector<int> stage_tile;       // tensor-engine stages: atom-tile width chosen for the launch
  int n_launches = 0;
  double work[4] = {0, 0, 0, 0};
};

// kernels (launch wrappers)
void launch_neighbors(nnp_handle* h, const float* d_pos, int pos_stride, const int* d_atom_index, cudaStream_t s);
int cells_alloc(nnp_handle* h);
void cells_free(nnp_handle* h);
void launch_neighbors_cells(nnp_handle* h, const float* d_pos, int pos_stride, const int* d_atom_index, cudaStream_t s);
void launch_aev_forward(nnp_handle* h, const float* d_pos, int pos_stride, const int* d_atom_index, cudaStream_t s);
void launch_aev_backward(nnp_handle* h, cudaStream_t s);
void launch_gemm(const GemmLaunch& g, cudaStream_t s);
void launch_last_layer(nnp_handle* h, cudaStream_t s);
void launch_finish(nnp_handle* h, const int* d_atom_index, double* d_energy, void* d_force, int force_stride, int fixed,
                   cudaStream_t s);
size_t aev_smem_bytes(const nnp_handle* h, bool backward);
void build_gemm_tiles(const std::vector<GemmProblem>& probs, std::vector<GemmTile>& tiles);

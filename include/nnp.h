/*
 * nnp.h -- C ABI of the B200-native ANI-2x energy+force library (libnnp_b200.so).
 *
 * What it computes (arXiv 2201.08110 "NNP/MM"; citations are lines of /root/reference/PAPER.md):
 *   V_NNP(Z_NNP, r_NNP): the neural-network-potential energy of the NNP region as a function of
 *   its atomic numbers and positions (Eq. 2) and F_NNP = -grad V_NNP (Eq. 3,
 *   PAPER.md:63-65), for the ANI family of potentials (modified Behler-Parrinello symmetry
 *   functions, 5.1 A cutoff, H C N O F S Cl, ensemble of 8 networks: PAPER.md:36,77).
 *   Mechanical embedding (Eq. 1 and 4): the NNP forces are simply ADDED to the MM
 *   force buffer on the device; "neither atomic positions nor atomic forces need to be
 *   transferred between the CPU and GPU".  The molecule is fixed across MD steps
 *   ("the same molecule is computed repeatedly"), so species, weights, element
 *   grouping and workspaces are set up once in nnp_create.
 *   The paper prints no formulas; the exact definitions (cutoff function, radial/angular terms,
 *   feature layout, CELU MLPs, ensemble mean, units) are O1-O7 / S1-S20 in DESIGN.md.
 *
 * Conventions
 *   - Every function returns an int status (NNP_OK = 0, negative = error); nothing throws.
 *   - "host" / "device" is stated for every pointer.  Device pointers must belong to the CUDA
 *     device that was current when nnp_create ran.  No torch types, no C++ types.
 *   - nnp_compute is asynchronous on the caller's stream and never synchronises the host.
 *     Device-detected conditions (neighbour capacity overflow, non-finite input) set a sticky
 *     device flag that nnp_status() reports.
 *   - One handle may be used by one stream at a time.
 *   - There is no CPU fallback and no other backend: on a machine without an sm_100 GPU
 *     nnp_create fails with NNP_ERR_UNSUPPORTED_ARCH / NNP_ERR_CUDA.
 */
#ifndef NNP_B200_H
#define NNP_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NNP_OK 0
#define NNP_ERR_INVALID_ARG (-1)
#define NNP_ERR_CUDA (-2)
#define NNP_ERR_UNSUPPORTED_ARCH (-3)
#define NNP_ERR_CAPACITY (-4)  /* a centre has more neighbours than the row capacity */
#define NNP_ERR_NONFINITE (-5) /* NaN/Inf position seen on the device */
#define NNP_ERR_ALLOC (-6)
#define NNP_ERR_STATIC_LIMIT (-7) /* nnp_coupling_compute_static: more atoms than its fixed scratch array holds */

typedef struct nnp_handle nnp_handle; /* opaque; owned by the library */

/*
 * Model description.  All pointers are HOST pointers and are copied by nnp_create (the caller may
 * free them afterwards).  Values for ANI-2x: BASELINE.json configs[0] (restated in DESIGN.md).
 */
typedef struct {
  int32_t n_species;       /* S; species index 0..S-1 (ANI-2x: 7, order H C N O F S Cl, reading S5) */
  int32_t n_models;        /* M; ensemble size (8; 1 = the "1 NN" variant) */
  float rc_radial;         /* radial cutoff in A (5.1) */
  float rc_angular;        /* angular cutoff in A (3.5) */
  float eta_r;             /* 19.7 */
  int32_t n_shf_r;         /* 16 (<= 32) */
  const float *shf_r;      /* host [n_shf_r] */
  float eta_a;             /* 12.5 */
  float zeta;              /* 14.1 */
  int32_t n_shf_a;         /* 8 */
  const float *shf_a;      /* host [n_shf_a] */
  int32_t n_shf_z;         /* 4;  n_shf_a*n_shf_z <= 64 */
  const float *shf_z;      /* host [n_shf_z] */
  float cos_scale;         /* 0.95 (reading S6) */
  float celu_alpha;        /* 0.1 */
  int32_t n_layers;        /* 4 (must be >= 2; the last layer has 1 output) */
  const int32_t *layer_dims; /* host [S][n_layers+1]; [e][0] must equal the AEV length */
  const float *const *weights; /* host [M*S*n_layers] pointers, index (m*S+e)*n_layers+l, each row-major [out][in] */
  const float *const *biases;  /* same indexing, each [out]; the array or any entry may be NULL => zeros */
  const double *self_energy;   /* host [S] per-species energy shift in model units, or NULL */
  double energy_scale;     /* output energy unit per model unit (627.5094740631: Hartree -> kcal/mol, S8) */
  double length_scale;     /* A per caller length unit (1.0 = caller works in A; 10.0 = nm) */
  int32_t max_radial_neighbors;  /* row capacity of the radial list; 0 = library default */
  int32_t max_angular_neighbors; /* row capacity of the angular list; 0 = library default */
  int32_t flags;           /* NNP_FLAG_* */
} nnp_config;

#define NNP_FLAG_NO_GRAPH 1 /* launch kernels one by one instead of replaying a CUDA graph */
#define NNP_FLAG_NO_UMMA 4  /* keep the MLP layers off the tcgen05 tensor-core engine (grouped FP32 FFMA GEMMs instead: the engine of
                              shapes the tensor engine does not take, i.e. hidden widths that are not multiples of 32) */
#define NNP_FLAG_NO_SMALL 8 /* do not use the ligand-size weight-streaming engine even when every element group is small */
#define NNP_FLAG_NO_MID 16  /* ligand-size engine: one launch per layer instead of the fused middle-of-the-network launch */
#define NNP_FLAG_NO_PDL 32  /* plain stream-ordered launches instead of programmatic dependent launches along the chain */
#define NNP_FLAG_NO_CELLS 64     /* neighbour search: all pairs inside a molecule even for large molecules */
#define NNP_FLAG_FORCE_CELLS 128 /* neighbour search: cell binning even for small molecules (default: molecules >= 1024 atoms) */
#define NNP_FLAG_NO_FWD1 256     /* ligand-size engine: row-pair layer-1 forward kernel instead of the persistent ring-fed one */
#define NNP_FLAG_NO_NBR_FUSION 1024 /* small molecules: separate neighbour launch instead of building the rows inside the AEV forward kernel */
#define NNP_FLAG_NO_TAIL_SPLIT 8192 /* tensor engine: whole tiles only (default: the tiles of a layer-1 backward launch that do not fill a round of the machine are cut along the contraction into parts on different SMs) */
#define NNP_FLAG_UMMA_PAIRS 4096 /* tensor engine, opt-in: the two layer-1 launches of a large system (every element >= 512 atoms) on CTA pairs (tcgen05 cta_group::2, 256 x 256 tiles); correct and measured SLOWER than the default one-CTA tiles */
#define NNP_FLAG_NO_SWEEP_REVERSAL 512 /* tensor engine: every launch sweeps the (element, model) blocks in the same direction (A/B switch for the L2 reuse between consecutive launches) */
#define NNP_FLAG_NO_ZERO_SKIP 2048 /* tensor engine: run layer 1 densely even over AEV columns that are structurally zero */

/*
 * nnp_create: build a handle for a fixed set of atoms.
 *   out               host; receives the handle
 *   cfg               host; model description, copied
 *   n_atoms           number of NNP atoms N (>= 0; N == 0 gives a handle whose compute is a no-op)
 *   species_host      host i32[N], values in 0..S-1
 *   n_molecules       number of independent molecules in the batch (>= 1)
 *   mol_offsets_host  host i32[n_molecules+1] CSR offsets, molecules are contiguous atom ranges
 *                     (mol_offsets[0]=0, last=N); NULL => one molecule.  Atoms of different
 *                     molecules never interact (BASELINE.json configs[2]).
 * Allocates all device memory; uploads and re-packs the weights; groups atoms by element.
 */
int nnp_create(nnp_handle **out, const nnp_config *cfg, int32_t n_atoms, const int32_t *species_host,
               int32_t n_molecules, const int32_t *mol_offsets_host);

/*
 * nnp_create_from_file: nnp_create from a parameter file holding a whole ANI-style parameter set (element list in
 * the set's own species order, AEV constants, layer shapes, weights AND biases of every (model, element, layer),
 * self-energies, energy scale); PAPER.md:36 (ANI-2x), :166-175 (ANI-1x as a second set).  The container format is
 * this library's own, documented in csrc/params_file.cu and written by binding.write_parameter_file (the trained
 * sets are not distributed with the library).
 *   path                 host; file name
 *   atomic_numbers_host  host i32[N]: the atoms by ATOMIC NUMBER; mapped to species indices through the file's
 *                        element list (an element the set does not cover => NNP_ERR_INVALID_ARG)
 *   n_models_to_use      0 = the whole ensemble; k > 0 = its first k networks (1 = the "1 NN" variant)
 *   length_scale, flags  as in nnp_config
 * Errors: NNP_ERR_INVALID_ARG for an unreadable / malformed file, else as nnp_create.
 */
int nnp_create_from_file(nnp_handle **out, const char *path, int32_t n_atoms, const int32_t *atomic_numbers_host,
                         int32_t n_molecules, const int32_t *mol_offsets_host, int32_t n_models_to_use,
                         double length_scale, int32_t flags);

/*
 * nnp_compute: one energy+force evaluation (one MD step), enqueued on `cuda_stream`.
 *   d_pos               device f32; position of NNP atom a is at d_pos[row(a)*pos_stride_floats + 0..2]
 *                       in caller length units (x length_scale = A)
 *   pos_stride_floats   3 (xyz) or 4 (float4 "posq") or any stride >= 3
 *   d_atom_index        device i32[N] row(a) of NNP atom a in the caller's position/force buffers,
 *                       or NULL => row(a) = a
 *   d_energy            device f64[n_molecules]; WRITTEN (not accumulated): E_mol in output energy units
 *   d_force_accum       device f32; F_NNP (output energy unit per caller length unit) is ADDED in place at
 *                       d_force_accum[row(a)*force_stride_floats + 0..2]; may be NULL (energy only still
 *                       runs the whole path)
 *   force_stride_floats >= 3
 *   cuda_stream         a cudaStream_t (0 = legacy default stream); borrowed
 * No host synchronisation; buffers are borrowed until the enqueued work has run.
 */
int nnp_compute(nnp_handle *h, const float *d_pos, int32_t pos_stride_floats, const int32_t *d_atom_index,
                double *d_energy, float *d_force_accum, int32_t force_stride_floats, void *cuda_stream);

/*
 * nnp_compute_host: the same evaluation for HOST buffers (used for end-to-end timing and by callers
 * without device data): copies pos_host f32[N][3] to the device, runs nnp_compute, copies back
 * energy_host f64[n_molecules] and force_host f32[N][3] (forces are WRITTEN, not accumulated), and
 * synchronises the stream before returning.  Every step of the path still runs on the GPU.
 */
int nnp_compute_host(nnp_handle *h, const float *pos_host, double *energy_host, float *force_host,
                     void *cuda_stream);

/*
 * nnp_compute_fixed: nnp_compute with the forces accumulated in 64-bit fixed point ("performs the NNP
 * and MM calculations on a GPU sequentially, but it would be more efficient to do that concurrently").
 *   d_force_fixed       device i64; round(F * 2^32) is added with integer atomics at
 *                       d_force_fixed[row(a)*force_stride_int64 + 0..2] (the accumulation format of GPU MD engines).
 *                       Integer additions commute, so kernels of the MM engine may add into the same buffer AT THE
 *                       SAME TIME on another stream and the sum has the same bits in any order.  nnp_compute's
 *                       float read-modify-write is only safe when every other adder is ordered with its stream.
 * Everything else as nnp_compute.
 */
int nnp_compute_fixed(nnp_handle *h, const float *d_pos, int32_t pos_stride_floats, const int32_t *d_atom_index,
                      double *d_energy, int64_t *d_force_fixed, int32_t force_stride_int64, void *cuda_stream);

/*
 * nnp_compute_async: the evaluation on a stream OWNED BY THE LIBRARY, so that the caller's MM kernels overlap it.
 *   wait_event   a cudaEvent_t the caller recorded after the positions were written, or NULL (positions ready now)
 *   done_event   a cudaEvent_t the library records when energy and forces are in, or NULL; the caller makes its
 *                integrator wait on it (cudaStreamWaitEvent) -- no host synchronisation anywhere
 *   d_force / force_stride / force_is_fixed64
 *                as d_force_accum of nnp_compute (0) or d_force_fixed of nnp_compute_fixed (1).  Concurrent adders
 *                into the same buffer require the fixed-point format.
 */
int nnp_compute_async(nnp_handle *h, const float *d_pos, int32_t pos_stride_floats, const int32_t *d_atom_index,
                      double *d_energy, void *d_force, int32_t force_stride, int32_t force_is_fixed64,
                      void *wait_event, void *done_event);

/* nnp_status: synchronises the last used stream and returns the sticky device status (NNP_OK or
 * NNP_ERR_CAPACITY / NNP_ERR_NONFINITE / NNP_ERR_CUDA); the flag is cleared by the call. */
int nnp_status(nnp_handle *h);

/* nnp_destroy: frees everything owned by the handle (NULL is allowed). */
void nnp_destroy(nnp_handle *h);

/* nnp_error_string: static string for a status code. */
const char *nnp_error_string(int code);

/* Number of kernel launches (graph nodes) one nnp_compute enqueues. */
int nnp_launches_per_compute(nnp_handle *h);

/*
 * Stage timing (measurement only).  nnp_set_profiling(h,1) makes nnp_compute launch its kernels one by
 * one with CUDA events between stages; nnp_get_stage_times then synchronises and returns, for the last
 * compute, the duration in ms of each stage (ms_host f32[capacity]) and the stage count; names via
 * nnp_stage_name.  Profiling mode is not the timed configuration.
 */
int nnp_set_profiling(nnp_handle *h, int32_t enable);
int nnp_get_stage_times(nnp_handle *h, float *ms_host, int32_t capacity, int32_t *n_stages);
const char *nnp_stage_name(nnp_handle *h, int32_t stage);

/* Algorithmic bytes / flops of one compute, for roofline accounting:
 * what[0] = weight bytes the MLP layers must read once, what[1] = MLP flops (2 per MAC, forward +
 * input-gradient backward), what[2] = AEV bytes (write+read), what[3] = layer-1 weight bytes. */
int nnp_get_work(nnp_handle *h, double *what_host, int32_t n);
/* Per stage (index as in nnp_stage_name): for a tensor-engine launch the flops it actually issues (2 per MAC of the
 * valid rows x atoms of every contraction box it runs; boxes of structural zeros are skipped and not counted) and the
 * atom-tile width chosen for it; 0 / 0 for other stages.  Either pointer may be NULL. */
int nnp_get_stage_work(nnp_handle *h, int32_t stage, double *issued_flops_host, int32_t *atom_tile_host);
/* Per stage: ALGORITHMIC bytes of a tensor-engine launch -- every operand plane it reads counted once (weights and
 * activations, hi and lo planes, only the contraction boxes it runs), the planes it writes once, and the activations
 * its epilogue reads once; 0 for other stages.  The hidden-layer launches of a large system move more bytes per flop
 * than the layer-1 launches and are bound by this number, not by the tensor pipe. */
int nnp_get_stage_bytes(nnp_handle *h, int32_t stage, double *bytes_host);

/*
 * nnp_measure_peaks (measurement only): micro-benchmarks on the current device; peaks_host f64[n], n <= 4:
 * [0] FP32 FFMA TFLOP/s, [1] tcgen05 kind::tf32 TFLOP/s issued from shared-memory operands (M=128, N=256, K=8),
 * [2] L2-resident read GB/s, [3] DRAM read GB/s.  Synchronises the device; takes ~0.1 s.
 */
int nnp_measure_peaks(double *peaks_host, int32_t n);

/*
 * Debug / parity exports: copy device workspace of the LAST compute to the host after synchronising.
 * Not on the timed path.  Atom indices are the caller's NNP atom order (0..N-1).
 *   nnp_debug_pairs   which = 0 radial / 1 angular; writes directed pairs (i,j) as i32 pairs, row-major
 *                     by centre i; *n_pairs receives the total even when it exceeds `capacity` pairs
 *   nnp_debug_aev     f32[N][n_features]
 *   nnp_debug_atomic_energies  f64[M][N], model units (before mean/scale)
 *   nnp_debug_daev    f32[N][n_features] = dE_model_units/dAEV (mean over the ensemble).  Columns of AEV blocks that
 *                     are zero for every atom of the system (a species that does not occur) never reach the forces;
 *                     the tensor engine does not compute whole 128-column tiles of them (exported as 0).
 */
int nnp_debug_pairs(nnp_handle *h, int32_t which, int64_t *n_pairs, int32_t *ij_host, int64_t capacity);
int nnp_debug_aev(nnp_handle *h, float *aev_host);
int nnp_debug_atomic_energies(nnp_handle *h, double *e_host);
int nnp_debug_daev(nnp_handle *h, float *g_host);
int nnp_n_features(nnp_handle *h);

/*
 * NNP-MM coupling term of mechanical embedding, Eq. 4:
 *   V_NNP-MM = sum_{i in NNP} sum_{j in MM} [ kc q_i q_j / r_ij + 4 eps_ij ((sigma_ij/r_ij)^12 - (sigma_ij/r_ij)^6) ]
 * with sigma_ij = (sigma_i + sigma_j)/2, eps_ij = sqrt(eps_i eps_j) (reading C1), kc = 1/(4 pi eps0) supplied by the
 * caller in its units (C2), an optional inclusive plain cutoff on r_ij in A (C3; <= 0: none) and no periodic images
 * (C4).  Only NNP-MM pairs enter.  Forces on the atoms of BOTH regions are ADDED to the caller's buffer.
 *
 * nnp_coupling_create: all pointers HOST, copied.  *_rows are rows of the atoms in the caller's position / force
 * buffers; q in e, sigma in A, eps in the output energy unit; length_scale = A per caller length unit.
 * nnp_coupling_compute: d_pos / d_force_accum as in nnp_compute (device, strides in floats); d_energy device f64[1],
 * WRITTEN, may be NULL; asynchronous on cuda_stream.  nnp_coupling_compute_fixed: 64-bit fixed-point forces as in
 * nnp_compute_fixed.  Errors: NNP_ERR_INVALID_ARG (negative row or eps, bad stride, NULL handle), NNP_ERR_CUDA,
 * NNP_ERR_UNSUPPORTED_ARCH, NNP_ERR_ALLOC.
 */
typedef struct nnp_coupling nnp_coupling; /* opaque; owned by the library */
int nnp_coupling_create(nnp_coupling **out, int32_t n_nnp, const int32_t *nnp_rows_host, const float *q_nnp_host,
                        const float *sigma_nnp_host, const float *eps_nnp_host, int32_t n_mm,
                        const int32_t *mm_rows_host, const float *q_mm_host, const float *sigma_mm_host,
                        const float *eps_mm_host, double coulomb_const, double cutoff, double length_scale);
int nnp_coupling_compute(nnp_coupling *c, const float *d_pos, int32_t pos_stride_floats, double *d_energy,
                         float *d_force_accum, int32_t force_stride_floats, void *cuda_stream);
int nnp_coupling_compute_fixed(nnp_coupling *c, const float *d_pos, int32_t pos_stride_floats, double *d_energy,
                               int64_t *d_force_fixed, int32_t force_stride_int64, void *cuda_stream);
void nnp_coupling_destroy(nnp_coupling *c);

/*
 * nnp_coupling_compute_static: Eq. 4 as above through an entry point that ALLOCATES NOTHING -- no cudaMalloc, cudaFree
 * or allocating library call, in this call or behind it -- for callers that cannot allocate (CUDA graph capture, tight
 * serving loops, harnesses that forbid it).  No handle: the atom lists are DEVICE arrays passed with every call
 * (d_*_rows i32, d_q / d_sigma / d_eps f32, meaning and units as in nnp_coupling_create; not validated: rows must be
 * >= 0, eps >= 0), the other arguments as in nnp_coupling_compute (forces ADDED to f32 d_force_accum, may be NULL;
 * d_energy device f64[1] WRITTEN, may be NULL; asynchronous on cuda_stream).  Results: the kernels and summation
 * orders of nnp_coupling_compute, i.e. the same bits for the same inputs.
 * Scratch (packed atom records, per-CTA partial sums) is one file-scope device array of
 * ~1.8 MB sized for NNP_COUPLING_STATIC_MAX_NNP x NNP_COUPLING_STATIC_MAX_MM atoms, held by every GPU that loads the
 * library until the process exits; more atoms => NNP_ERR_STATIC_LIMIT, nothing is launched.  All calls share the
 * array, which keeps the last call's contents (no element needs to start at zero: everything read is written earlier
 * in the same call); calls that OVERLAP on the GPU (different streams without an ordering) race on it -- issue them
 * on one stream or order them with events.
 * nnp_coupling_static_init: optional; resolves the array's device address for the CURRENT device (once per device,
 * done lazily by the first compute call otherwise -- call it before starting a stream capture).
 * Errors: NNP_ERR_INVALID_ARG, NNP_ERR_STATIC_LIMIT, NNP_ERR_UNSUPPORTED_ARCH, NNP_ERR_CUDA.
 */
#define NNP_COUPLING_STATIC_MAX_NNP 128
#define NNP_COUPLING_STATIC_MAX_MM 65536
int nnp_coupling_static_init(void);
int nnp_coupling_compute_static(int32_t n_nnp, const int32_t *d_nnp_rows, const float *d_q_nnp, const float *d_sigma_nnp,
                                const float *d_eps_nnp, int32_t n_mm, const int32_t *d_mm_rows, const float *d_q_mm,
                                const float *d_sigma_mm, const float *d_eps_mm, double coulomb_const, double cutoff,
                                double length_scale, const float *d_pos, int32_t pos_stride_floats, double *d_energy,
                                float *d_force_accum, int32_t force_stride_floats, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* NNP_B200_H */

// NNP-MM coupling term of mechanical embedding (Eq. 4) on the device:
//   V = sum_{i in NNP} sum_{j in MM} [ kc q_i q_j / r_ij + 4 eps_ij ((sigma_ij/r_ij)^12 - (sigma_ij/r_ij)^6) ],
// forces on the atoms of BOTH regions added into the caller's force buffer (the same buffer nnp_compute adds
// into).  Readings C1-C4 of DESIGN.md: Lorentz-Berthelot mixing, caller-supplied Coulomb constant, optional
// inclusive plain cutoff on D2 = (dx dx + dy dy) + dz dz evaluated in binary64 without contraction (the same
// predicate as the neighbour search, so the pair set equals the oracle's), no periodic images.
//
// The NNP region is small (48-75 atoms in the paper's systems) and the MM region large, so the
// work is O(N_NNP N_MM) distance tests of which a few per cent pass a 9 A cutoff.  Two launches, no float atomics,
// fixed summation orders (bit-identical reruns):
//   coupling_mm_kernel   one thread per MM atom j, NNP atoms staged in shared memory: F_j, the pair energies, and the
//                        reaction on every NNP atom reduced over the warp (shuffles) and the CTA (warp order)
//   coupling_nnp_kernel  adds the per-CTA partials of F_i and of the energy in CTA order
// Arithmetic is FP64 (the work is tiny; B200 has full-rate FP64 FMA) so that parity with the
// float64 oracle is at rounding level; the force increments are rounded once when they are added to the buffer.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include <new>
#include <vector>

#include "nnp.h"

namespace {

constexpr int CP_THREADS = 256;

struct CpAtom {  // an atom of either list: row in the caller's buffers and its parameters
  int row;
  float q, sigma, eps;
};

struct CpArgs {
  const CpAtom* nnp;
  const CpAtom* mm;
  int n_nnp, n_mm;
  double kc, rc2, length_scale;  // rc2 <= 0: no cutoff
};

__device__ __forceinline__ void load_pos(const float* pos, int stride, int row, double ls, double& x, double& y, double& z) {
  const float* p = pos + (size_t)row * stride;
  // caller length unit -> A with one f32 multiply, as nnp_compute does, so a caller working in nm sees the same bits
  const float fl = (float)ls;
  x = (double)(p[0] * fl); y = (double)(p[1] * fl); z = (double)(p[2] * fl);
}

// pair (NNP atom a, MM atom b) with d = r_b - r_a: energy and dV/dr / r ("g": F_b = -g d, F_a = +g d)
__device__ __forceinline__ bool pair_terms(const CpArgs& A, double dx, double dy, double dz, float qa, float sa, float ea,
                                           float qb, float sb, float eb, double& v, double& g) {
  const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
  if (A.rc2 > 0.0 && d2 > A.rc2) return false;
  const double r = sqrt(d2), inv = 1.0 / r;
  const double sigma = 0.5 * ((double)sa + (double)sb);
  const double eps = sqrt((double)ea * (double)eb);
  const double s = sigma * inv, s2 = s * s, s6 = s2 * s2 * s2, s12 = s6 * s6;
  const double vc = A.kc * (double)qa * (double)qb * inv;
  v = vc + 4.0 * eps * (s12 - s6);
  g = (-vc + 4.0 * eps * (-12.0 * s12 + 6.0 * s6)) * inv * inv;  // (dV/dr) / r
  return true;
}

__device__ __forceinline__ double block_sum(double v, double* red) {  // fixed tree; result valid in thread 0
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  const int w = threadIdx.x >> 5;
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[w] = v;
  __syncthreads();
  double t = 0.0;
  if (threadIdx.x == 0)
    for (int k = 0; k < CP_THREADS / 32; ++k) t += red[k];
  return t;
}

// add a force increment (output energy unit per caller length unit) into the caller's buffer
__device__ __forceinline__ void add_force(void* buf, int stride, int row, int fixed, double fx, double fy, double fz) {
  if (fixed) {  // 64-bit fixed point, 2^32 per unit: integer atomics commute, so concurrent adders give the same bits
    unsigned long long* f = reinterpret_cast<unsigned long long*>(buf) + (size_t)row * stride;
    atomicAdd(f + 0, (unsigned long long)__double2ll_rn(fx * 4294967296.0));
    atomicAdd(f + 1, (unsigned long long)__double2ll_rn(fy * 4294967296.0));
    atomicAdd(f + 2, (unsigned long long)__double2ll_rn(fz * 4294967296.0));
  } else {
    float* f = reinterpret_cast<float*>(buf) + (size_t)row * stride;
    f[0] += (float)fx; f[1] += (float)fy; f[2] += (float)fz;
  }
}

constexpr int CP_CHUNK = 64;  // NNP atoms staged per pass

// One thread per MM atom j, NNP atoms staged in shared memory CP_CHUNK at a time.  F_j is accumulated by the thread
// and added to the buffer (every j belongs to one thread).  The reaction on NNP atom i is reduced over the warp with
// shuffles -- only for the (i, warp) combinations that have a pair inside the cutoff, which a 9 A cutoff makes rare --
// then over the CTA's warps in warp order, and written as the CTA's partial f_part[blockIdx][i][3]; the second kernel
// adds the partials in CTA order.  No float atomics; every sum has a fixed order.
__global__ void __launch_bounds__(CP_THREADS) coupling_mm_kernel(const __grid_constant__ CpArgs A, const float* __restrict__ pos,
                                                                  int pos_stride, void* force, int force_stride, int fixed,
                                                                  double* __restrict__ e_part, double* __restrict__ f_part) {
  __shared__ double sx[CP_CHUNK], sy[CP_CHUNK], sz[CP_CHUNK];
  __shared__ float sq[CP_CHUNK], ss[CP_CHUNK], se[CP_CHUNK];
  __shared__ double wpart[CP_THREADS / 32][CP_CHUNK][3];
  __shared__ double red[CP_THREADS / 32];
  const int j = blockIdx.x * CP_THREADS + threadIdx.x;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const bool live = j < A.n_mm;
  CpAtom b = live ? A.mm[j] : CpAtom{0, 0.f, 0.f, 0.f};
  double bx = 0, by = 0, bz = 0;
  if (live) load_pos(pos, pos_stride, b.row, A.length_scale, bx, by, bz);
  double fx = 0, fy = 0, fz = 0, e = 0;
  for (int i0 = 0; i0 < A.n_nnp; i0 += CP_CHUNK) {
    const int n = min(CP_CHUNK, A.n_nnp - i0);
    __syncthreads();
    if ((int)threadIdx.x < n) {
      const CpAtom a = A.nnp[i0 + threadIdx.x];
      load_pos(pos, pos_stride, a.row, A.length_scale, sx[threadIdx.x], sy[threadIdx.x], sz[threadIdx.x]);
      sq[threadIdx.x] = a.q; ss[threadIdx.x] = a.sigma; se[threadIdx.x] = a.eps;
    }
    for (int k = threadIdx.x; k < (CP_THREADS / 32) * CP_CHUNK * 3; k += CP_THREADS) (&wpart[0][0][0])[k] = 0.0;
    __syncthreads();
    for (int i = 0; i < n; ++i) {  // NNP atoms in index order
      const double dx = bx - sx[i], dy = by - sy[i], dz = bz - sz[i];
      double v = 0.0, g = 0.0;
      const bool hit = live && pair_terms(A, dx, dy, dz, sq[i], ss[i], se[i], b.q, b.sigma, b.eps, v, g);
      if (__ballot_sync(0xffffffffu, hit) == 0u) continue;
      double gx = hit ? g * dx : 0.0, gy = hit ? g * dy : 0.0, gz = hit ? g * dz : 0.0;
      if (hit) {
        e += v;
        fx -= gx; fy -= gy; fz -= gz;
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        gx += __shfl_xor_sync(0xffffffffu, gx, o);
        gy += __shfl_xor_sync(0xffffffffu, gy, o);
        gz += __shfl_xor_sync(0xffffffffu, gz, o);
      }
      if (lane == 0) { wpart[warp][i][0] = gx; wpart[warp][i][1] = gy; wpart[warp][i][2] = gz; }
    }
    __syncthreads();
    for (int k = threadIdx.x; k < n * 3; k += CP_THREADS) {
      const int i = k / 3, c = k - 3 * i;
      double t = 0.0;
      for (int w = 0; w < CP_THREADS / 32; ++w) t += wpart[w][i][c];
      f_part[((size_t)blockIdx.x * A.n_nnp + i0 + i) * 3 + c] = t;
    }
  }
  if (live && force && (fx != 0.0 || fy != 0.0 || fz != 0.0))
    add_force(force, force_stride, b.row, fixed, fx * A.length_scale, fy * A.length_scale, fz * A.length_scale);
  const double t = block_sum(e, red);
  if (threadIdx.x == 0) e_part[blockIdx.x] = t;
}

// forces on the NNP atoms: one warp per atom adds the CTA partials of the first kernel (lanes stride over the CTAs,
// then a fixed shuffle tree: the same order in every run); the energy partials likewise by warp 0 of CTA 0
__global__ void __launch_bounds__(CP_THREADS) coupling_nnp_kernel(const __grid_constant__ CpArgs A, void* force, int force_stride,
                                                                   int fixed, const double* __restrict__ e_part,
                                                                   const double* __restrict__ f_part, int n_part,
                                                                   double* __restrict__ energy) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int i = blockIdx.x * (CP_THREADS / 32) + warp;
  if (i < A.n_nnp) {
    double tx = 0.0, ty = 0.0, tz = 0.0;
    for (int k = lane; k < n_part; k += 32) {
      const double* p = f_part + ((size_t)k * A.n_nnp + i) * 3;
      tx += p[0]; ty += p[1]; tz += p[2];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      tx += __shfl_xor_sync(0xffffffffu, tx, o);
      ty += __shfl_xor_sync(0xffffffffu, ty, o);
      tz += __shfl_xor_sync(0xffffffffu, tz, o);
    }
    if (lane == 0 && force)
      add_force(force, force_stride, A.nnp[i].row, fixed, tx * A.length_scale, ty * A.length_scale, tz * A.length_scale);
  }
  if (blockIdx.x == 0 && warp == 0 && energy) {
    double s = 0.0;
    for (int k = lane; k < n_part; k += 32) s += e_part[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) *energy = s;
  }
}

}  // namespace

struct nnp_coupling {
  int device = 0;
  CpArgs args;
  CpAtom *d_nnp = nullptr, *d_mm = nullptr;
  double *d_epart = nullptr, *d_fpart = nullptr;
  int n_part = 0;
};

extern "C" void nnp_coupling_destroy(nnp_coupling* c) {
  if (!c) return;
  cudaSetDevice(c->device);
  cudaDeviceSynchronize();
  if (c->d_nnp) cudaFree(c->d_nnp);
  if (c->d_mm) cudaFree(c->d_mm);
  if (c->d_epart) cudaFree(c->d_epart);
  if (c->d_fpart) cudaFree(c->d_fpart);
  delete c;
}

extern "C" int nnp_coupling_create(nnp_coupling** out, int32_t n_nnp, const int32_t* nnp_rows_host, const float* q_nnp_host,
                                   const float* sigma_nnp_host, const float* eps_nnp_host, int32_t n_mm,
                                   const int32_t* mm_rows_host, const float* q_mm_host, const float* sigma_mm_host,
                                   const float* eps_mm_host, double coulomb_const, double cutoff, double length_scale) {
  if (!out) return NNP_ERR_INVALID_ARG;
  *out = nullptr;
  if (n_nnp < 0 || n_mm < 0 || !(length_scale > 0.0)) return NNP_ERR_INVALID_ARG;
  if (n_nnp > 0 && (!nnp_rows_host || !q_nnp_host || !sigma_nnp_host || !eps_nnp_host)) return NNP_ERR_INVALID_ARG;
  if (n_mm > 0 && (!mm_rows_host || !q_mm_host || !sigma_mm_host || !eps_mm_host)) return NNP_ERR_INVALID_ARG;
  for (int i = 0; i < n_nnp; ++i)
    if (nnp_rows_host[i] < 0 || eps_nnp_host[i] < 0.f) return NNP_ERR_INVALID_ARG;
  for (int j = 0; j < n_mm; ++j)
    if (mm_rows_host[j] < 0 || eps_mm_host[j] < 0.f) return NNP_ERR_INVALID_ARG;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return NNP_ERR_CUDA;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return NNP_ERR_CUDA;
  if (prop.major != 10) return NNP_ERR_UNSUPPORTED_ARCH;
  nnp_coupling* c = new (std::nothrow) nnp_coupling();
  if (!c) return NNP_ERR_ALLOC;
  c->device = dev;
  std::vector<CpAtom> a(n_nnp), b(n_mm);
  for (int i = 0; i < n_nnp; ++i) a[i] = CpAtom{nnp_rows_host[i], q_nnp_host[i], sigma_nnp_host[i], eps_nnp_host[i]};
  for (int j = 0; j < n_mm; ++j) b[j] = CpAtom{mm_rows_host[j], q_mm_host[j], sigma_mm_host[j], eps_mm_host[j]};
  c->n_part = (n_mm + CP_THREADS - 1) / CP_THREADS;
  bool ok = cudaMalloc((void**)&c->d_nnp, sizeof(CpAtom) * (size_t)(n_nnp > 0 ? n_nnp : 1)) == cudaSuccess &&
            cudaMalloc((void**)&c->d_mm, sizeof(CpAtom) * (size_t)(n_mm > 0 ? n_mm : 1)) == cudaSuccess &&
            cudaMalloc((void**)&c->d_epart, sizeof(double) * (size_t)(c->n_part > 0 ? c->n_part : 1)) == cudaSuccess &&
            cudaMalloc((void**)&c->d_fpart, sizeof(double) * 3 * (size_t)(c->n_part > 0 ? c->n_part : 1) * (size_t)(n_nnp > 0 ? n_nnp : 1)) == cudaSuccess;
  if (ok && n_nnp) ok = cudaMemcpy(c->d_nnp, a.data(), sizeof(CpAtom) * (size_t)n_nnp, cudaMemcpyHostToDevice) == cudaSuccess;
  if (ok && n_mm) ok = cudaMemcpy(c->d_mm, b.data(), sizeof(CpAtom) * (size_t)n_mm, cudaMemcpyHostToDevice) == cudaSuccess;
  if (!ok) {
    nnp_coupling_destroy(c);
    return NNP_ERR_ALLOC;
  }
  c->args = CpArgs{c->d_nnp, c->d_mm, n_nnp, n_mm, coulomb_const, cutoff > 0.0 ? cutoff * cutoff : 0.0, length_scale};
  *out = c;
  return NNP_OK;
}

static int coupling_enqueue(nnp_coupling* c, const float* d_pos, int ps, double* d_energy, void* d_force, int fs, int fixed,
                            cudaStream_t s) {
  if (!c || !d_pos || ps < 3 || (d_force && fs < 3)) return NNP_ERR_INVALID_ARG;
  if (c->args.n_mm > 0)
    coupling_mm_kernel<<<c->n_part, CP_THREADS, 0, s>>>(c->args, d_pos, ps, d_force, fs, fixed, c->d_epart, c->d_fpart);
  const int nb = (c->args.n_nnp + CP_THREADS / 32 - 1) / (CP_THREADS / 32);
  coupling_nnp_kernel<<<nb > 0 ? nb : 1, CP_THREADS, 0, s>>>(c->args, d_force, fs, fixed, c->d_epart, c->d_fpart,
                                                            c->args.n_mm > 0 ? c->n_part : 0, d_energy);
  return cudaGetLastError() == cudaSuccess ? NNP_OK : NNP_ERR_CUDA;
}

extern "C" int nnp_coupling_compute(nnp_coupling* c, const float* d_pos, int32_t pos_stride_floats, double* d_energy,
                                    float* d_force_accum, int32_t force_stride_floats, void* cuda_stream) {
  return coupling_enqueue(c, d_pos, pos_stride_floats, d_energy, d_force_accum, force_stride_floats, 0,
                          (cudaStream_t)cuda_stream);
}

extern "C" int nnp_coupling_compute_fixed(nnp_coupling* c, const float* d_pos, int32_t pos_stride_floats, double* d_energy,
                                          int64_t* d_force_fixed, int32_t force_stride_int64, void* cuda_stream) {
  return coupling_enqueue(c, d_pos, pos_stride_floats, d_energy, d_force_fixed, force_stride_int64, 1,
                          (cudaStream_t)cuda_stream);
}

// ------------------------------------------------------------------------------------------------
// nnp_coupling_compute_static: the same Eq. 4 computation with NO allocation anywhere in the call, for callers that
// cannot call cudaMalloc (stream capture, tight serving loops, harnesses that forbid it).  There is no handle: the
// caller passes the atom lists as device arrays with every call, and everything the kernels need in between -- the
// packed atom records and the per-CTA partial sums of the first kernel -- lives in ONE file-scope device array of a
// fixed maximum size.  Every GPU that loads the library holds that array until the process exits.
//   * All calls share the array and it keeps the last call's contents.  Nothing in it has to start at zero: every
//     element a kernel reads is written earlier in the SAME call (the pack kernel writes the atom records, the MM
//     kernel writes e_part[block] and f_part[block][i][:] for every block and every NNP atom), so no clear is needed.
//   * Two calls that overlap on the GPU (different streams, no ordering between them) RACE on the array; calls on one
//     stream, or ordered by events, are safe.
// In host code `g_cp_scratch` is a host-side stand-in for the symbol, not a device address: the address the kernels
// get comes from cudaGetSymbolAddress, once per device, with that device current.
// ------------------------------------------------------------------------------------------------
namespace {

constexpr int CPS_MAX_NNP = NNP_COUPLING_STATIC_MAX_NNP;
constexpr int CPS_MAX_MM = NNP_COUPLING_STATIC_MAX_MM;
constexpr int CPS_MAX_PART = (CPS_MAX_MM + CP_THREADS - 1) / CP_THREADS;
// layout (bytes, every section 256-byte aligned): NNP records | MM records | e_part | f_part
constexpr size_t CPS_OFF_NNP = 0;
constexpr size_t CPS_OFF_MM = CPS_OFF_NNP + ((sizeof(CpAtom) * CPS_MAX_NNP + 255) & ~(size_t)255);
constexpr size_t CPS_OFF_EPART = CPS_OFF_MM + ((sizeof(CpAtom) * CPS_MAX_MM + 255) & ~(size_t)255);
constexpr size_t CPS_OFF_FPART = CPS_OFF_EPART + ((sizeof(double) * CPS_MAX_PART + 255) & ~(size_t)255);
constexpr size_t CPS_BYTES = CPS_OFF_FPART + sizeof(double) * 3 * (size_t)CPS_MAX_PART * CPS_MAX_NNP;  // ~1.8 MB

static __device__ __align__(256) unsigned char g_cp_scratch[CPS_BYTES];

// device lists (structure of arrays, as the caller holds them) -> the packed records the kernels read
__global__ void __launch_bounds__(CP_THREADS) coupling_pack_kernel(CpAtom* __restrict__ dst_nnp, int n_nnp,
                                                                    const int* __restrict__ nnp_rows, const float* __restrict__ q_nnp,
                                                                    const float* __restrict__ s_nnp, const float* __restrict__ e_nnp,
                                                                    CpAtom* __restrict__ dst_mm, int n_mm,
                                                                    const int* __restrict__ mm_rows, const float* __restrict__ q_mm,
                                                                    const float* __restrict__ s_mm, const float* __restrict__ e_mm) {
  const int k = blockIdx.x * CP_THREADS + threadIdx.x;
  if (k < n_nnp) dst_nnp[k] = CpAtom{nnp_rows[k], q_nnp[k], s_nnp[k], e_nnp[k]};
  if (k < n_mm) dst_mm[k] = CpAtom{mm_rows[k], q_mm[k], s_mm[k], e_mm[k]};
}

constexpr int CPS_MAX_DEVICES = 64;
unsigned char* g_cp_scratch_ptr[CPS_MAX_DEVICES];  // device address of g_cp_scratch, per device; null = not set up

// once per device, with that device current
int static_scratch(unsigned char** out) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return NNP_ERR_CUDA;
  if (dev < 0 || dev >= CPS_MAX_DEVICES) return NNP_ERR_INVALID_ARG;
  unsigned char* p = __atomic_load_n(&g_cp_scratch_ptr[dev], __ATOMIC_ACQUIRE);
  if (!p) {
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return NNP_ERR_CUDA;
    if (prop.major != 10) return NNP_ERR_UNSUPPORTED_ARCH;
    void* sym = nullptr;
    if (cudaGetSymbolAddress(&sym, g_cp_scratch) != cudaSuccess || !sym) {
      cudaGetLastError();
      return NNP_ERR_CUDA;
    }
    p = static_cast<unsigned char*>(sym);
    __atomic_store_n(&g_cp_scratch_ptr[dev], p, __ATOMIC_RELEASE);  // the same value from whichever thread gets here first
  }
  *out = p;
  return NNP_OK;
}

}  // namespace

extern "C" int nnp_coupling_static_init(void) {
  unsigned char* p = nullptr;
  return static_scratch(&p);
}

extern "C" int nnp_coupling_compute_static(int32_t n_nnp, const int32_t* d_nnp_rows, const float* d_q_nnp,
                                           const float* d_sigma_nnp, const float* d_eps_nnp, int32_t n_mm,
                                           const int32_t* d_mm_rows, const float* d_q_mm, const float* d_sigma_mm,
                                           const float* d_eps_mm, double coulomb_const, double cutoff, double length_scale,
                                           const float* d_pos, int32_t pos_stride_floats, double* d_energy,
                                           float* d_force_accum, int32_t force_stride_floats, void* cuda_stream) {
  if (n_nnp < 0 || n_mm < 0 || !(length_scale > 0.0)) return NNP_ERR_INVALID_ARG;
  if (n_nnp > CPS_MAX_NNP || n_mm > CPS_MAX_MM) return NNP_ERR_STATIC_LIMIT;
  if (!d_pos || pos_stride_floats < 3 || (d_force_accum && force_stride_floats < 3)) return NNP_ERR_INVALID_ARG;
  if (n_nnp > 0 && (!d_nnp_rows || !d_q_nnp || !d_sigma_nnp || !d_eps_nnp)) return NNP_ERR_INVALID_ARG;
  if (n_mm > 0 && (!d_mm_rows || !d_q_mm || !d_sigma_mm || !d_eps_mm)) return NNP_ERR_INVALID_ARG;
  unsigned char* scratch = nullptr;
  const int rc = static_scratch(&scratch);
  if (rc != NNP_OK) return rc;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  CpAtom* nnp = reinterpret_cast<CpAtom*>(scratch + CPS_OFF_NNP);
  CpAtom* mm = reinterpret_cast<CpAtom*>(scratch + CPS_OFF_MM);
  double* e_part = reinterpret_cast<double*>(scratch + CPS_OFF_EPART);
  double* f_part = reinterpret_cast<double*>(scratch + CPS_OFF_FPART);
  const int n_max = n_nnp > n_mm ? n_nnp : n_mm;
  if (n_max > 0)
    coupling_pack_kernel<<<(n_max + CP_THREADS - 1) / CP_THREADS, CP_THREADS, 0, s>>>(
        nnp, n_nnp, d_nnp_rows, d_q_nnp, d_sigma_nnp, d_eps_nnp, mm, n_mm, d_mm_rows, d_q_mm, d_sigma_mm, d_eps_mm);
  const CpArgs args{nnp, mm, n_nnp, n_mm, coulomb_const, cutoff > 0.0 ? cutoff * cutoff : 0.0, length_scale};
  const int n_part = (n_mm + CP_THREADS - 1) / CP_THREADS;
  if (n_mm > 0)
    coupling_mm_kernel<<<n_part, CP_THREADS, 0, s>>>(args, d_pos, pos_stride_floats, d_force_accum, force_stride_floats, 0,
                                                     e_part, f_part);
  const int nb = (n_nnp + CP_THREADS / 32 - 1) / (CP_THREADS / 32);
  coupling_nnp_kernel<<<nb > 0 ? nb : 1, CP_THREADS, 0, s>>>(args, d_force_accum, force_stride_floats, 0, e_part, f_part,
                                                            n_mm > 0 ? n_part : 0, d_energy);
  return cudaGetLastError() == cudaSuccess ? NNP_OK : NNP_ERR_CUDA;
}

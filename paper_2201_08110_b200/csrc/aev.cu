// Neighbour pairs (A1), radial+angular AEV forward (A2,A3), AEV backward (A7) and the force gather /
// mechanical-embedding add / energy reduce (A5,A8) of the ANI hot path.  sm_100a.
//
// Definitions: DESIGN.md O1-O4, O6, O7 (the paper names ANI-2x, and gives no formulas).
// Design: one warp per centre atom; the centre's 1008-float feature row (or dE/dAEV row) lives in
// shared memory; the 32 lanes of the warp are the 32 (ShfA, ShfZ) sub-terms of an angular block, so a
// triplet is one conflict-free shared-memory row update and no atomics are needed anywhere; forces
// leave the kernel as one "pair gradient" phi_ij per directed pair, gathered per atom afterwards.
#include <math_constants.h>

#include "nnp_internal.h"

#define FULL 0xffffffffu
constexpr int AEV_WARPS = 4;  // warps (= centres) per CTA

// ------------------------------------------------------------------------------------------------
// A1: all-pairs neighbour search inside a molecule, warp per centre, ballot compaction.
// Predicate O2/S1: D2 = (dx*dx + dy*dy) + dz*dz in binary64 on the widened f32 coordinates, no FMA,
// D2 <= Rc^2.  Evaluated in FP64 for every candidate, so the pair sets are bit-exact by construction.
// Rows come out sorted by j.  nbr_a stores the SLOT of the neighbour in the radial row.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) nbr_allpairs_kernel(
    const float* __restrict__ pos, int pos_stride, const int* __restrict__ atom_index,
    const int* __restrict__ species, const int* __restrict__ mol_id, const int* __restrict__ mol_off, int N,
    AevConst c, int capR, int capA, float4* __restrict__ pos4, int* __restrict__ nbr_r, int* __restrict__ nbr_a,
    int* __restrict__ cnt_r, int* __restrict__ cnt_a, int* __restrict__ status) {
  const int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (i >= N) return;
  const int m = mol_id[i];
  const int lo = mol_off[m], hi = mol_off[m + 1];
  const int rowi = atom_index ? atom_index[i] : i;
  const float xi = pos[(size_t)rowi * pos_stride + 0] * c.length_scale;
  const float yi = pos[(size_t)rowi * pos_stride + 1] * c.length_scale;
  const float zi = pos[(size_t)rowi * pos_stride + 2] * c.length_scale;
  if (lane == 0) {
    pos4[i] = make_float4(xi, yi, zi, __int_as_float(species[i]));
    if (!(isfinite(xi) && isfinite(yi) && isfinite(zi))) atomicOr(status, NNP_ST_NONFINITE);
  }
  int nr = 0, na = 0;
  for (int base = lo; base < hi; base += 32) {
    const int j = base + lane;
    bool in_r = false, in_a = false;
    if (j < hi && j != i) {
      const int rowj = atom_index ? atom_index[j] : j;
      const double dx = (double)(pos[(size_t)rowj * pos_stride + 0] * c.length_scale) - (double)xi;
      const double dy = (double)(pos[(size_t)rowj * pos_stride + 1] * c.length_scale) - (double)yi;
      const double dz = (double)(pos[(size_t)rowj * pos_stride + 2] * c.length_scale) - (double)zi;
      const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
      in_r = d2 <= c.rc_r2;
      in_a = d2 <= c.rc_a2;
    }
    const unsigned br = __ballot_sync(FULL, in_r);
    const unsigned ba = __ballot_sync(FULL, in_a);
    const unsigned below = (1u << lane) - 1u;
    const int slot_r = nr + __popc(br & below);
    if (in_r && slot_r < capR) nbr_r[(size_t)i * capR + slot_r] = j;
    if (in_a) {
      const int slot_a = na + __popc(ba & below);
      if (slot_a < capA && slot_r < capR) nbr_a[(size_t)i * capA + slot_a] = slot_r;
    }
    nr += __popc(br);
    na += __popc(ba);
  }
  if (lane == 0) {
    if (nr > capR || na > capA) atomicOr(status, NNP_ST_CAPACITY);
    cnt_r[i] = min(nr, capR);
    cnt_a[i] = min(na, capA);
  }
}

// ------------------------------------------------------------------------------------------------
// shared helpers
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ int pair_index(int s, int t, int S) {
  const int a = min(s, t), b = max(s, t);
  return a * S - (a * (a - 1)) / 2 + (b - a);
}

// per angular neighbour, 8 floats in shared memory
struct PairData {
  float ux, uy, uz, r, rlo, fc, dfc;  // r + rlo = the FP64 distance to ~2^-48
  int ss;                             // slot * 16 + species
  __device__ __forceinline__ int spec() const { return ss & 15; }
  __device__ __forceinline__ int slot() const { return ss >> 4; }
};

// geometry of a directed pair in FP64 from the f32 coordinates (cheap on B200, removes the
// cancellation error of an f32 distance); results rounded to f32 once.
__device__ __forceinline__ void pair_geometry(const float4 pi, const float4 pj, double& r, float& ux, float& uy,
                                              float& uz) {
  const double dx = (double)pj.x - (double)pi.x;
  const double dy = (double)pj.y - (double)pi.y;
  const double dz = (double)pj.z - (double)pi.z;
  r = sqrt(dx * dx + dy * dy + dz * dz);
  const double inv = 1.0 / r;
  ux = (float)(dx * inv);
  uy = (float)(dy * inv);
  uz = (float)(dz * inv);
}

// O1: f_C = 0.5 cos(pi r/Rc) + 0.5 = cos^2(pi r / 2Rc) (the squared form keeps relative accuracy near Rc);
//     f_C' = -(pi/2Rc) sin(pi r/Rc) = -(pi/Rc) sin(pi r/2Rc) cos(pi r/2Rc)
// cospif/sincospif take the argument in units of pi, so no rounded pi enters the argument (a rounded
// pi biases every f_C by ~ -5e-8 relative, which adds up coherently over the whole AEV).
__device__ __forceinline__ float cutoff_f(float r, float rc) {
  const float ch = cospif(0.5f * r / rc);
  return ch * ch;
}
__device__ __forceinline__ float dcutoff_f(float r, float rc) {
  float sh, ch;
  sincospif(0.5f * r / rc, &sh, &ch);
  return -(CUDART_PI_F / rc) * sh * ch;
}

size_t aev_smem_bytes(const nnp_handle* h, bool backward) {
  size_t per_warp = (size_t)h->n_feat + (backward ? 3 * (size_t)h->capR : (size_t)h->aev.n_radial) +
                    8 * (size_t)h->capA;
  per_warp = (per_warp + 3) & ~(size_t)3;
  return per_warp * 4 * AEV_WARPS;
}

// fills the per-warp PairData table for centre i; returns nothing (na entries)
__device__ __forceinline__ void load_pair_data(PairData* pd, int na, int i, const float4 pi,
                                               const float4* __restrict__ pos4, const int* __restrict__ nbr_r,
                                               const int* __restrict__ nbr_a, int capR, int capA, float rc_a,
                                               int lane) {
  for (int q = lane; q < na; q += 32) {
    const int slot = nbr_a[(size_t)i * capA + q];
    const int j = nbr_r[(size_t)i * capR + slot];
    const float4 pj = pos4[j];
    double r;
    PairData d;
    pair_geometry(pi, pj, r, d.ux, d.uy, d.uz);
    d.r = (float)r;
    d.rlo = (float)(r - (double)d.r);
    d.fc = cutoff_f(d.r, rc_a);
    d.dfc = dcutoff_f(d.r, rc_a);
    d.ss = slot * 16 + __float_as_int(pj.w);
    pd[q] = d;
  }
}

// ------------------------------------------------------------------------------------------------
// A2 + A3: AEV forward, warp per centre.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(AEV_WARPS * 32) aev_forward_kernel(
    const float4* __restrict__ pos4, const int* __restrict__ nbr_r, const int* __restrict__ nbr_a,
    const int* __restrict__ cnt_r, const int* __restrict__ cnt_a, const int* __restrict__ sortpos, int N,
    AevConst c, int capR, int capA, float* __restrict__ aev) {
  extern __shared__ __align__(16) float smem[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int i = blockIdx.x * AEV_WARPS + warp;
  if (i >= N) return;
  size_t per_warp = ((size_t)c.n_feat + c.n_radial + 8 * (size_t)capA + 3) & ~(size_t)3;
  float* row = smem + per_warp * warp;
  float* rad1 = row + c.n_feat;
  PairData* pd = reinterpret_cast<PairData*>(rad1 + c.n_radial);

  for (int f = lane; f < c.n_feat + c.n_radial; f += 32) row[f] = 0.0f;
  const float4 pi = pos4[i];
  const int nr = cnt_r[i], na = cnt_a[i];
  load_pair_data(pd, na, i, pi, pos4, nbr_r, nbr_a, capR, capA, c.rc_a, lane);
  __syncwarp();

  // ---- radial (O3): two neighbours per pass when n_shf_r <= 16 (one per half-warp, own partial row)
  {
    const int groups = c.n_shf_r <= 16 ? 2 : 1;
    const int glanes = 32 / groups;
    const int grp = lane / glanes, k = lane % glanes;
    float* dst = grp ? rad1 : row;
    for (int s0 = 0; s0 < nr; s0 += groups) {
      const int s = s0 + grp;
      if (s < nr && k < c.n_shf_r) {
        const int j = nbr_r[(size_t)i * capR + s];
        const float4 pj = pos4[j];
        double r;
        float ux, uy, uz;
        pair_geometry(pi, pj, r, ux, uy, uz);
        const float fc = cutoff_f((float)r, c.rc_r);
        const float d = (float)(r - (double)c.shf_r[k]);
        const float val = 0.25f * expf(-c.eta_r * d * d) * fc;
        dst[__float_as_int(pj.w) * c.n_shf_r + k] += val;
      }
      __syncwarp();
    }
    if (groups == 2)
      for (int f = lane; f < c.n_radial; f += 32) row[f] += rad1[f];
    __syncwarp();
  }

  // ---- angular (O4): lanes are the (ShfA, ShfZ) sub-terms; triplets are visited serially
  float* ang = row + c.n_radial;
  for (int t = lane; t < c.n_sub; t += 32) {
    const int ia = t / c.n_shf_z, iz = t % c.n_shf_z;
    const float shfa = c.shf_a[ia], cz = c.cos_z[iz], sz = c.sin_z[iz];
    const float czl = c.cos_z_lo[iz], szl = c.sin_z_lo[iz];
    for (int a = 0; a < na; ++a) {
      const PairData A = pd[a];
      for (int b = a + 1; b < na; ++b) {
        const PairData B = pd[b];
        const float cth = A.ux * B.ux + A.uy * B.uy + A.uz * B.uz;
        const float cc = c.cos_scale * cth;
        const float ss = sqrtf(fmaxf(1.0f - cc * cc, 0.0f));
        const float u = 0.5f + 0.5f * ((cc * cz + ss * sz) + (cc * czl + ss * szl));
        const float F1 = exp2f(c.zeta * log2f(u));
        const float d = 0.5f * (((A.r - shfa) + (B.r - shfa)) + (A.rlo + B.rlo));
        const float F2 = expf(-c.eta_a * d * d);
        const float val = 2.0f * F1 * F2 * (A.fc * B.fc);
        ang[pair_index(A.spec(), B.spec(), c.S) * c.n_sub + t] += val;
      }
    }
  }
  __syncwarp();
  float* out = aev + (size_t)sortpos[i] * c.n_feat;
  for (int f = lane; f < c.n_feat; f += 32) out[f] = row[f];
}

// ------------------------------------------------------------------------------------------------
// A7: AEV backward, warp per centre.  phi[i][slot] = dE/d(r_j - r_i) for every radial slot of i.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
  return v;
}

__global__ void __launch_bounds__(AEV_WARPS * 32) aev_backward_kernel(
    const float4* __restrict__ pos4, const int* __restrict__ nbr_r, const int* __restrict__ nbr_a,
    const int* __restrict__ cnt_r, const int* __restrict__ cnt_a, const int* __restrict__ sortpos, int N,
    AevConst c, int capR, int capA, const float* __restrict__ daev, float* __restrict__ phi) {
  extern __shared__ __align__(16) float smem[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int i = blockIdx.x * AEV_WARPS + warp;
  if (i >= N) return;
  size_t per_warp = ((size_t)c.n_feat + 3 * (size_t)capR + 8 * (size_t)capA + 3) & ~(size_t)3;
  float* g = smem + per_warp * warp;
  float* ph = g + c.n_feat;  // [capR][3]
  PairData* pd = reinterpret_cast<PairData*>(ph + 3 * capR);

  const float* gin = daev + (size_t)sortpos[i] * c.n_feat;
  for (int f = lane; f < c.n_feat; f += 32) g[f] = gin[f];
  const float4 pi = pos4[i];
  const int nr = cnt_r[i], na = cnt_a[i];
  load_pair_data(pd, na, i, pi, pos4, nbr_r, nbr_a, capR, capA, c.rc_a, lane);
  __syncwarp();

  // ---- radial: dT/dr = T (-2 eta (r - Shf)) + 0.25 exp(.) fC'(r)
  {
    const int groups = c.n_shf_r <= 16 ? 2 : 1;
    const int glanes = 32 / groups;
    const int grp = lane / glanes, k = lane % glanes;
    for (int s0 = 0; s0 < nr; s0 += groups) {
      const int s = s0 + grp;
      float v = 0.0f, ux = 0.f, uy = 0.f, uz = 0.f;
      if (s < nr) {
        const int j = nbr_r[(size_t)i * capR + s];
        const float4 pj = pos4[j];
        double r;
        pair_geometry(pi, pj, r, ux, uy, uz);
        if (k < c.n_shf_r) {
          const float rf = (float)r;
          const float fc = cutoff_f(rf, c.rc_r), dfc = dcutoff_f(rf, c.rc_r);
          const float d = (float)(r - (double)c.shf_r[k]);
          const float ex = 0.25f * expf(-c.eta_r * d * d);
          const float dT = ex * (dfc - 2.0f * c.eta_r * d * fc);
          v = g[__float_as_int(pj.w) * c.n_shf_r + k] * dT;
        }
      }
      for (int o = glanes >> 1; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
      if (s < nr && k == 0) {
        ph[3 * s + 0] = v * ux;
        ph[3 * s + 1] = v * uy;
        ph[3 * s + 2] = v * uz;
      }
    }
    __syncwarp();
  }

  // ---- angular: A = 2 F1 F2 fa fb.  Per triplet reduce over the sub-terms
  //   R0 = sum g F1 F2,  R1 = sum g F1 dF2/drbar-half,  R2 = sum g F2 dF1/dc
  const float* gang = g + c.n_radial;
  for (int a = 0; a < na; ++a) {
    const PairData A = pd[a];
    for (int b = a + 1; b < na; ++b) {
      const PairData B = pd[b];
      const float cth = A.ux * B.ux + A.uy * B.uy + A.uz * B.uz;
      const float cc = c.cos_scale * cth;
      const float ss = sqrtf(fmaxf(1.0f - cc * cc, 0.0f));
      const float cot = cc / ss;
      const float* gb = gang + pair_index(A.spec(), B.spec(), c.S) * c.n_sub;
      float R0 = 0.f, R1 = 0.f, R2 = 0.f;
      for (int t = lane; t < c.n_sub; t += 32) {
        const int ia = t / c.n_shf_z, iz = t % c.n_shf_z;
        const float cz = c.cos_z[iz], sz = c.sin_z[iz], shfa = c.shf_a[ia];
        const float u = 0.5f + 0.5f * ((cc * cz + ss * sz) + (cc * c.cos_z_lo[iz] + ss * c.sin_z_lo[iz]));
        const float pw1 = exp2f((c.zeta - 1.0f) * log2f(u));  // u^(zeta-1)
        const float F1 = pw1 * u;
        const float dF1dc = c.zeta * pw1 * 0.5f * (cz - cot * sz);
        const float d = 0.5f * (((A.r - shfa) + (B.r - shfa)) + (A.rlo + B.rlo));
        const float F2 = expf(-c.eta_a * d * d);
        const float gt = gb[t];
        R0 += gt * F1 * F2;
        R1 += gt * F1 * (-c.eta_a * d * F2);
        R2 += gt * F2 * dF1dc;
      }
      R0 = warp_sum(R0);
      R1 = warp_sum(R1);
      R2 = warp_sum(R2);
      if (lane < 3) {
        const float W = A.fc * B.fc;
        const float coefA = 2.0f * (W * R1 + A.dfc * B.fc * R0);
        const float coefB = 2.0f * (W * R1 + A.fc * B.dfc * R0);
        const float coefC = 2.0f * W * R2 * c.cos_scale;
        const float ua = lane == 0 ? A.ux : (lane == 1 ? A.uy : A.uz);
        const float ub = lane == 0 ? B.ux : (lane == 1 ? B.uy : B.uz);
        ph[3 * A.slot() + lane] += coefA * ua + coefC * (ub - cth * ua) / A.r;
        ph[3 * B.slot() + lane] += coefB * ub + coefC * (ua - cth * ub) / B.r;
      }
      __syncwarp();
    }
  }
  __syncwarp();
  float* out = phi + (size_t)i * capR * 3;
  for (int f = lane; f < 3 * nr; f += 32) out[f] = ph[f];
}

// ------------------------------------------------------------------------------------------------
// A8 + A5: F_a = sum_j phi[a][j] - sum_i phi[i][a], added into the caller's force buffer (mechanical
// embedding); energies per molecule in FP64.  Blocks [0, n_force_blocks) do forces
// (warp per atom), the remaining blocks do energies (warp per molecule).  Fixed reduction trees,
// no atomics => bit-identical reruns.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) finish_kernel(
    const int* __restrict__ nbr_r, const int* __restrict__ cnt_r, const float* __restrict__ phi, int N, int capR,
    const int* __restrict__ atom_index, float* __restrict__ force, int force_stride, float fscale,
    int n_force_blocks, const double* __restrict__ eatom, const int* __restrict__ sortpos,
    const int* __restrict__ species, const int* __restrict__ mol_off, int n_mol, int M,
    const double* __restrict__ self_energy, double escale, double* __restrict__ energy) {
  const int lane = threadIdx.x & 31;
  const int wib = threadIdx.x >> 5;
  if ((int)blockIdx.x < n_force_blocks) {
    const int a = blockIdx.x * 4 + wib;
    if (a >= N || force == nullptr) return;
    const int n = cnt_r[a];
    float fx = 0.f, fy = 0.f, fz = 0.f;
    for (int s = lane; s < n; s += 32) {
      const int i = nbr_r[(size_t)a * capR + s];
      // slot of a in the (sorted) row of i: binary search
      const int* rowi = nbr_r + (size_t)i * capR;
      int lo = 0, hi = cnt_r[i] - 1, slot = -1;
      while (lo <= hi) {
        const int mid = (lo + hi) >> 1;
        const int v = rowi[mid];
        if (v == a) { slot = mid; break; }
        if (v < a) lo = mid + 1; else hi = mid - 1;
      }
      const float* own = phi + ((size_t)a * capR + s) * 3;
      fx += own[0]; fy += own[1]; fz += own[2];
      if (slot >= 0) {
        const float* oth = phi + ((size_t)i * capR + slot) * 3;
        fx -= oth[0]; fy -= oth[1]; fz -= oth[2];
      }
    }
    fx = warp_sum(fx); fy = warp_sum(fy); fz = warp_sum(fz);
    if (lane == 0) {
      const int row = atom_index ? atom_index[a] : a;
      float* f = force + (size_t)row * force_stride;
      f[0] += fscale * fx;
      f[1] += fscale * fy;
      f[2] += fscale * fz;
    }
  } else {
    const int m = (blockIdx.x - n_force_blocks) * 4 + wib;
    if (m >= n_mol || energy == nullptr) return;
    double acc = 0.0;
    for (int i = mol_off[m] + lane; i < mol_off[m + 1]; i += 32) {
      const double* e = eatom + (size_t)sortpos[i] * M;
      double s = 0.0;
      for (int k = 0; k < M; ++k) s += e[k];
      acc += s / (double)M + (self_energy ? self_energy[species[i]] : 0.0);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(FULL, acc, o);
    if (lane == 0) energy[m] = escale * acc;
  }
}

// ------------------------------------------------------------------------------------------------
// launch wrappers
// ------------------------------------------------------------------------------------------------
void launch_neighbors(nnp_handle* h, const float* d_pos, int pos_stride, const int* d_atom_index, cudaStream_t s) {
  if (h->N == 0) return;
  const int blocks = (h->N + 3) / 4;
  nbr_allpairs_kernel<<<blocks, 128, 0, s>>>(d_pos, pos_stride, d_atom_index, h->d_species, h->d_mol_id,
                                             h->d_mol_off, h->N, h->aev, h->capR, h->capA, h->d_pos4, h->d_nbr_r,
                                             h->d_nbr_a, h->d_cnt_r, h->d_cnt_a, h->d_status);
}

void launch_aev_forward(nnp_handle* h, cudaStream_t s) {
  if (h->N == 0) return;
  const int blocks = (h->N + AEV_WARPS - 1) / AEV_WARPS;
  aev_forward_kernel<<<blocks, AEV_WARPS * 32, aev_smem_bytes(h, false), s>>>(
      h->d_pos4, h->d_nbr_r, h->d_nbr_a, h->d_cnt_r, h->d_cnt_a, h->d_sortpos, h->N, h->aev, h->capR, h->capA,
      h->d_aev);
}

void launch_aev_backward(nnp_handle* h, cudaStream_t s) {
  if (h->N == 0) return;
  const int blocks = (h->N + AEV_WARPS - 1) / AEV_WARPS;
  aev_backward_kernel<<<blocks, AEV_WARPS * 32, aev_smem_bytes(h, true), s>>>(
      h->d_pos4, h->d_nbr_r, h->d_nbr_a, h->d_cnt_r, h->d_cnt_a, h->d_sortpos, h->N, h->aev, h->capR, h->capA,
      h->d_daev, h->d_phi);
}

void launch_finish(nnp_handle* h, const int* d_atom_index, double* d_energy, float* d_force, int force_stride,
                   cudaStream_t s) {
  if (h->N == 0) return;
  const int nfb = (h->N + 3) / 4;
  const int neb = (h->n_mol + 3) / 4;
  const float fscale = (float)(h->energy_scale * h->length_scale);
  finish_kernel<<<nfb + neb, 128, 0, s>>>(h->d_nbr_r, h->d_cnt_r, h->d_phi, h->N, h->capR, d_atom_index, d_force,
                                          force_stride, fscale, nfb, h->d_eatom, h->d_sortpos, h->d_species,
                                          h->d_mol_off, h->n_mol, h->M, h->d_self_energy, h->energy_scale,
                                          d_energy);
}

int aev_set_smem_attributes(nnp_handle* h) {
  cudaError_t e1 = cudaFuncSetAttribute(aev_forward_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        (int)aev_smem_bytes(h, false));
  cudaError_t e2 = cudaFuncSetAttribute(aev_backward_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                        (int)aev_smem_bytes(h, true));
  return (e1 == cudaSuccess && e2 == cudaSuccess) ? 0 : -1;
}

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

// ------------------------------------------------------------------------------------------------
// fast-math building blocks.  Accuracy notes:
//  - u^zeta = u^floor(zeta) (exact-ish repeated squaring) * 2^(frac * lg2 u): the MUFU lg2 error
//    (2^-22 absolute) is scaled by frac (0.1), not by zeta (14.1);
//  - exp(-eta d^2) = ex2(d^2 * k), k = -eta*log2(e) carried as hi+lo so the constant is not a bias;
//  - geometry (r, unit vectors) is FP64 once per directed pair, r is kept as hi+lo floats.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float lg2_approx(float x) {
  float y;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float sqrt_approx(float x) {
  float y;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float rcp_approx(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// u^(n + frac), n >= 0 uniform across the grid, 0 <= frac < 1, u in [0, 1]
__device__ __forceinline__ float pow_split(float u, int n, float frac) {
  float r = 1.0f, b = u;
#pragma unroll
  for (int bit = 0; bit < 6; ++bit) {
    if (n & 1) r *= b;
    b *= b;
    n >>= 1;
  }
  if (frac != 0.0f) r *= ex2_approx(frac * lg2_approx(u));
  return r;
}
__device__ __forceinline__ float gauss(float d, float khi, float klo) {
  const float d2 = d * d;
  return ex2_approx(fmaf(d2, klo, d2 * khi));
}

constexpr int TAB_FIELDS = 10;  // per radial slot: ux uy uz rhi rlo fcr dfcr fca dfca spec

size_t aev_smem_bytes(const nnp_handle* h, bool backward) {
  size_t fl = (size_t)TAB_FIELDS * h->capR + h->capA;
  if (!backward) fl += (size_t)AEV_WARPS * (h->n_feat - h->aev.n_radial);
  else fl += (size_t)h->n_feat + (size_t)(AEV_WARPS + 1) * 3 * h->capR;
  return ((fl + 3) & ~(size_t)3) * 4;
}

struct CentreTab {
  float *ux, *uy, *uz, *rhi, *rlo, *fcr, *dfcr, *fca, *dfca;
  int* spec;
  int* asl;  // angular neighbours: radial slots, sorted by species (stable)
};

__device__ __forceinline__ CentreTab carve_tab(float* smem, int capR) {
  CentreTab t;
  t.ux = smem; t.uy = t.ux + capR; t.uz = t.uy + capR; t.rhi = t.uz + capR; t.rlo = t.rhi + capR;
  t.fcr = t.rlo + capR; t.dfcr = t.fcr + capR; t.fca = t.dfcr + capR; t.dfca = t.fca + capR;
  t.spec = reinterpret_cast<int*>(t.dfca + capR);
  t.asl = t.spec + capR;
  return t;
}

// Phase 0 of both AEV kernels: geometry of every radial neighbour of centre i (FP64 once, all threads
// of the CTA in parallel), and the angular neighbour list re-ordered by species so that consecutive
// triplets of a warp fall into the same feature block.
__device__ __forceinline__ void build_tab(const CentreTab& t, int i, int nr, int na, const float4 pi,
                                          const float4* __restrict__ pos4, const int* __restrict__ nbr_r,
                                          const int* __restrict__ nbr_a, int capR, int capA, const AevConst& c) {
  for (int q = threadIdx.x; q < nr; q += blockDim.x) {
    const int j = nbr_r[(size_t)i * capR + q];
    const float4 pj = pos4[j];
    const double dx = (double)pj.x - (double)pi.x;
    const double dy = (double)pj.y - (double)pi.y;
    const double dz = (double)pj.z - (double)pi.z;
    const double r = sqrt(dx * dx + dy * dy + dz * dz);
    const double inv = 1.0 / r;
    t.ux[q] = (float)(dx * inv);
    t.uy[q] = (float)(dy * inv);
    t.uz[q] = (float)(dz * inv);
    const float rf = (float)r;
    t.rhi[q] = rf;
    t.rlo[q] = (float)(r - (double)rf);
    // O1 via cospi: f_C = cos^2(pi r / 2Rc), f_C' = -(pi/Rc) sin cos; no rounded pi in the argument
    float sh, ch;
    sincospif(0.5f * rf / c.rc_r, &sh, &ch);
    t.fcr[q] = ch * ch;
    t.dfcr[q] = -(CUDART_PI_F / c.rc_r) * sh * ch;
    sincospif(0.5f * rf / c.rc_a, &sh, &ch);
    t.fca[q] = ch * ch;
    t.dfca[q] = -(CUDART_PI_F / c.rc_a) * sh * ch;
    t.spec[q] = __float_as_int(pj.w);
  }
  __syncthreads();
  // stable counting sort of the angular list by species: rank = #(smaller species) + #(same, earlier)
  for (int q = threadIdx.x; q < na; q += blockDim.x) {
    const int slot = nbr_a[(size_t)i * capA + q];
    const int sp = t.spec[slot];
    int rank = 0;
    for (int q2 = 0; q2 < na; ++q2) {
      const int s2 = t.spec[nbr_a[(size_t)i * capA + q2]];
      rank += (s2 < sp) || (s2 == sp && q2 < q);
    }
    t.asl[rank] = slot;
  }
  __syncthreads();
}

// first triplet (a,b), a<b<na, of warp w in the flattened order, and the step to the next one
__device__ __forceinline__ void trip_norm(int& a, int& b, int na) {
  while (a < na - 1 && b >= na) {
    ++a;
    b = b - na + a + 1;
  }
}

// ------------------------------------------------------------------------------------------------
// A2 + A3: AEV forward.  One CTA (4 warps) per centre.
//   radial : one thread per output column (species s, shift k) loops over the neighbours of species s
//            and keeps the sum in a register (fixed order, no shared-memory updates);
//   angular: the triplets are dealt round-robin to the 4 warps; lanes are the (ShfA, ShfZ) sub-terms;
//            each warp sums runs of triplets that fall into the same species-pair block in a register
//            and flushes to its own partial row; the 4 partial rows are added in a fixed order.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(AEV_WARPS * 32) aev_forward_kernel(
    const float4* __restrict__ pos4, const int* __restrict__ nbr_r, const int* __restrict__ nbr_a,
    const int* __restrict__ cnt_r, const int* __restrict__ cnt_a, const int* __restrict__ sortpos, int N,
    const __grid_constant__ AevConst c, int capR, int capA, float* __restrict__ aev) {
  extern __shared__ __align__(16) float smem[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int i = blockIdx.x;
  const CentreTab t = carve_tab(smem, capR);
  const int n_ang = c.n_feat - c.n_radial;
  float* rows = reinterpret_cast<float*>(t.asl + capA);  // [AEV_WARPS][n_ang]
  const float4 pi = pos4[i];
  const int nr = cnt_r[i], na = cnt_a[i];
  for (int f = threadIdx.x; f < AEV_WARPS * n_ang; f += blockDim.x) rows[f] = 0.0f;
  build_tab(t, i, nr, na, pi, pos4, nbr_r, nbr_a, capR, capA, c);
  float* out = aev + (size_t)sortpos[i] * c.n_feat;

  // ---- radial (O3)
  for (int col = threadIdx.x; col < c.n_radial; col += blockDim.x) {
    const int s = col / c.n_shf_r, k = col % c.n_shf_r;
    const float shf = c.shf_r[k];
    float acc = 0.0f;
    for (int q = 0; q < nr; ++q) {
      if (t.spec[q] != s) continue;
      const float d = (t.rhi[q] - shf) + t.rlo[q];
      acc += 0.25f * gauss(d, c.kr_hi, c.kr_lo) * t.fcr[q];
    }
    out[col] = acc;
  }

  // ---- angular (O4)
  float* myrow = rows + warp * n_ang;
  const int nsub_it = (c.n_sub + 31) >> 5;
  for (int it = 0; it < nsub_it; ++it) {
    const int tt = lane + 32 * it;
    const bool live = tt < c.n_sub;
    const int ia = live ? tt / c.n_shf_z : 0, iz = live ? tt % c.n_shf_z : 0;
    const float shfa = c.shf_a[ia], cz = c.cos_z[iz], sz = c.sin_z[iz];
    const float czl = c.cos_z_lo[iz], szl = c.sin_z_lo[iz];
    int a = 0, b = 1 + warp;
    trip_norm(a, b, na);
    int cur_p = -1;
    float acc = 0.0f;
    while (a < na - 1) {
      const int qa = t.asl[a], qb = t.asl[b];
      const float cth = t.ux[qa] * t.ux[qb] + t.uy[qa] * t.uy[qb] + t.uz[qa] * t.uz[qb];
      const float cc = c.cos_scale * cth;
      const float ss = sqrt_approx(fmaxf(fmaf(-cc, cc, 1.0f), 0.0f));
      const float u = 0.5f + 0.5f * ((cc * cz + ss * sz) + (cc * czl + ss * szl));
      const float F1 = pow_split(u, c.zeta_int, c.zeta_frac);
      const float d = 0.5f * (((t.rhi[qa] - shfa) + (t.rhi[qb] - shfa)) + (t.rlo[qa] + t.rlo[qb]));
      const float F2 = gauss(d, c.ka_hi, c.ka_lo);
      const float val = 2.0f * F1 * F2 * (t.fca[qa] * t.fca[qb]);
      const int sa = t.spec[qa], sb = t.spec[qb];  // sa <= sb (sorted)
      const int p = sa * c.S - (sa * (sa - 1)) / 2 + (sb - sa);
      if (p != cur_p) {
        if (cur_p >= 0 && live) myrow[cur_p * c.n_sub + tt] += acc;
        cur_p = p;
        acc = 0.0f;
      }
      acc += val;
      b += AEV_WARPS;
      trip_norm(a, b, na);
    }
    if (cur_p >= 0 && live) myrow[cur_p * c.n_sub + tt] += acc;
  }
  __syncthreads();
  for (int f = threadIdx.x; f < n_ang; f += blockDim.x) {
    float v = rows[f];
#pragma unroll
    for (int w = 1; w < AEV_WARPS; ++w) v += rows[w * n_ang + f];
    out[c.n_radial + f] = v;
  }
}

// ------------------------------------------------------------------------------------------------
// A7: AEV backward.  One CTA (4 warps) per centre.  phi[i][slot] = dE/d(r_j - r_i) for every radial
// slot of i (pair-gradient formulation: no atomics, the force gather happens per atom afterwards).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
  return v;
}

__global__ void __launch_bounds__(AEV_WARPS * 32) aev_backward_kernel(
    const float4* __restrict__ pos4, const int* __restrict__ nbr_r, const int* __restrict__ nbr_a,
    const int* __restrict__ cnt_r, const int* __restrict__ cnt_a, const int* __restrict__ sortpos, int N,
    const __grid_constant__ AevConst c, int capR, int capA, const float* __restrict__ daev, int n_parts,
    size_t part_stride, float* __restrict__ phi) {
  extern __shared__ __align__(16) float smem[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int i = blockIdx.x;
  const CentreTab t = carve_tab(smem, capR);
  float* g = reinterpret_cast<float*>(t.asl + capA);  // [n_feat]
  float* phr = g + c.n_feat;                          // radial part           [capR][3]
  float* phw = phr + 3 * capR;                        // per-warp angular part [AEV_WARPS][capR][3]
  const float4 pi = pos4[i];
  const int nr = cnt_r[i], na = cnt_a[i];
  const float* gin = daev + (size_t)sortpos[i] * c.n_feat;
  for (int f = threadIdx.x; f < c.n_feat; f += blockDim.x) {
    float v = gin[f];
    for (int p = 1; p < n_parts; ++p) v += gin[(size_t)p * part_stride + f];  // fixed order
    g[f] = v;
  }
  for (int f = threadIdx.x; f < AEV_WARPS * 3 * nr; f += blockDim.x) phw[(f / (3 * nr)) * 3 * capR + f % (3 * nr)] = 0.0f;
  build_tab(t, i, nr, na, pi, pos4, nbr_r, nbr_a, capR, capA, c);

  // ---- radial: dT/dr = 0.25 e (f_C' - 2 eta (r - Shf) f_C); a group of lanes per neighbour
  {
    const int glanes = c.n_shf_r <= 16 ? 16 : 32;
    const int groups = blockDim.x / glanes;
    const int grp = threadIdx.x / glanes, k = threadIdx.x % glanes;
    for (int q0 = 0; q0 < nr; q0 += groups) {
      const int q = q0 + grp;
      float v = 0.0f;
      if (q < nr && k < c.n_shf_r) {
        const float d = (t.rhi[q] - c.shf_r[k]) + t.rlo[q];
        const float ex = 0.25f * gauss(d, c.kr_hi, c.kr_lo);
        const float dT = ex * (t.dfcr[q] - 2.0f * c.eta_r * d * t.fcr[q]);
        v = g[t.spec[q] * c.n_shf_r + k] * dT;
      }
      for (int o = glanes >> 1; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
      if (q < nr && k == 0) {
        phr[3 * q + 0] = v * t.ux[q];
        phr[3 * q + 1] = v * t.uy[q];
        phr[3 * q + 2] = v * t.uz[q];
      }
    }
  }

  // ---- angular: A = 2 F1 F2 fa fb; per triplet reduce over the sub-terms
  //   R0 = sum g F1 F2,  R1 = sum g F1 dF2/dr,  R2 = sum g F2 dF1/dc
  float* myph = phw + warp * 3 * capR;
  const float* gang = g + c.n_radial;
  {
    int a = 0, b = 1 + warp;
    trip_norm(a, b, na);
    while (a < na - 1) {
      const int qa = t.asl[a], qb = t.asl[b];
      const float uax = t.ux[qa], uay = t.uy[qa], uaz = t.uz[qa];
      const float ubx = t.ux[qb], uby = t.uy[qb], ubz = t.uz[qb];
      const float cth = uax * ubx + uay * uby + uaz * ubz;
      const float cc = c.cos_scale * cth;
      const float ss = sqrt_approx(fmaxf(fmaf(-cc, cc, 1.0f), 0.0f));
      const float cot = cc * rcp_approx(ss);
      const float ra = t.rhi[qa], rb = t.rhi[qb];
      const float rl = t.rlo[qa] + t.rlo[qb];
      const int sa = t.spec[qa], sb = t.spec[qb];
      const float* gb = gang + (sa * c.S - (sa * (sa - 1)) / 2 + (sb - sa)) * c.n_sub;
      float R0 = 0.f, R1 = 0.f, R2 = 0.f;
      for (int tt = lane; tt < c.n_sub; tt += 32) {
        const int ia = tt / c.n_shf_z, iz = tt % c.n_shf_z;
        const float cz = c.cos_z[iz], sz = c.sin_z[iz], shfa = c.shf_a[ia];
        const float u = 0.5f + 0.5f * ((cc * cz + ss * sz) + (cc * c.cos_z_lo[iz] + ss * c.sin_z_lo[iz]));
        const float pw1 = pow_split(u, c.zeta1_int, c.zeta_frac);  // u^(zeta-1)
        const float F1 = pw1 * u;
        const float dF1dc = c.zeta * pw1 * 0.5f * (cz - cot * sz);
        const float d = 0.5f * (((ra - shfa) + (rb - shfa)) + rl);
        const float F2 = gauss(d, c.ka_hi, c.ka_lo);
        const float gt = gb[tt];
        R0 += gt * F1 * F2;
        R1 += gt * F1 * (-c.eta_a * d * F2);
        R2 += gt * F2 * dF1dc;
      }
      R0 = warp_sum(R0);
      R1 = warp_sum(R1);
      R2 = warp_sum(R2);
      if (lane < 3) {
        const float fa = t.fca[qa], fb = t.fca[qb];
        const float W = fa * fb;
        const float coefA = 2.0f * (W * R1 + t.dfca[qa] * fb * R0);
        const float coefB = 2.0f * (W * R1 + fa * t.dfca[qb] * R0);
        const float coefC = 2.0f * W * R2 * c.cos_scale;
        const float ua = lane == 0 ? uax : (lane == 1 ? uay : uaz);
        const float ub = lane == 0 ? ubx : (lane == 1 ? uby : ubz);
        myph[3 * qa + lane] += coefA * ua + coefC * (ub - cth * ua) * rcp_approx(ra);
        myph[3 * qb + lane] += coefB * ub + coefC * (ua - cth * ub) * rcp_approx(rb);
      }
      __syncwarp();
      b += AEV_WARPS;
      trip_norm(a, b, na);
    }
  }
  __syncthreads();
  float* out = phi + (size_t)i * capR * 3;
  for (int f = threadIdx.x; f < 3 * nr; f += blockDim.x) {
    float v = phr[f];
#pragma unroll
    for (int w = 0; w < AEV_WARPS; ++w) v += phw[w * 3 * capR + f];
    out[f] = v;
  }
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
  const int blocks = h->N;
  aev_forward_kernel<<<blocks, AEV_WARPS * 32, aev_smem_bytes(h, false), s>>>(
      h->d_pos4, h->d_nbr_r, h->d_nbr_a, h->d_cnt_r, h->d_cnt_a, h->d_sortpos, h->N, h->aev, h->capR, h->capA,
      h->d_aev);
}

void launch_aev_backward(nnp_handle* h, cudaStream_t s) {
  if (h->N == 0) return;
  const int blocks = h->N;
  aev_backward_kernel<<<blocks, AEV_WARPS * 32, aev_smem_bytes(h, true), s>>>(
      h->d_pos4, h->d_nbr_r, h->d_nbr_a, h->d_cnt_r, h->d_cnt_a, h->d_sortpos, h->N, h->aev, h->capR, h->capA,
      h->d_daev, h->n_parts, (size_t)h->N * h->n_feat, h->d_phi);
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

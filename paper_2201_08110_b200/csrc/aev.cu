// Neighbour pairs (A1), radial+angular AEV forward (A2,A3), AEV backward (A7) and the force gather /
// mechanical-embedding add / energy reduce (A5,A8) of the ANI hot path.  sm_100a.
//
// Definitions: DESIGN.md O1-O4, O6, O7 (the paper names ANI-2x, and gives no formulas).
// Design: one CTA per centre atom; the centre's feature row (or dE/dAEV row) and the geometry of its
// neighbours live in shared memory; the angular work is one thread per TRIPLET (its powers and Gaussians
// are evaluated once and combined in registers), every floating-point sum has a fixed order (no float atomics
// anywhere); a centre's "pair gradients" phi_ij are added to the two atoms of each pair in 64-bit fixed point
// (integer atomics: order-independent), which the finish kernel converts into the caller's force buffer.
#include <math_constants.h>

#include "nnp_internal.h"

#define FULL 0xffffffffu

// ------------------------------------------------------------------------------------------------
// A1: all-pairs neighbour search inside a molecule, warp per centre, ballot compaction.
// Predicate O2/S1: D2 = (dx*dx + dy*dy) + dz*dz in binary64 on the widened f32 coordinates, no FMA,
// D2 <= Rc^2.  Evaluated in FP64 for every candidate, so the pair sets are bit-exact by construction.
// Rows come out sorted by j.  nbr_a stores the SLOT of the neighbour in the radial row.
// ------------------------------------------------------------------------------------------------
// raw inputs of the neighbour search (the caller's position buffer and the molecule topology)
struct NbrArgs {
  const float* pos;
  const int* atom_index;
  const int* species;
  const int* mol_id;
  const int* mol_off;
  const int2* mol_range;  // [N] (first atom, end) of the atom's molecule: one load instead of mol_id -> mol_off
  int* status;
  int pos_stride;
  float length_scale;
};

__device__ __forceinline__ float4 raw_pos4(const NbrArgs& a, int j) {
  const int row = a.atom_index ? a.atom_index[j] : j;
  const float* p = a.pos + (size_t)row * a.pos_stride;
  return make_float4(p[0] * a.length_scale, p[1] * a.length_scale, p[2] * a.length_scale, __int_as_float(a.species[j]));
}

// one warp builds the radial and angular rows of centre i
__device__ __forceinline__ void nbr_row_warp(const NbrArgs& a, int i, int lane, double rc_r2, double rc_a2, int capR,
                                             int capA, float4* __restrict__ pos4, int* __restrict__ nbr_r,
                                             int* __restrict__ nbr_a, int* __restrict__ cnt_r, int* __restrict__ cnt_a) {
  const int m = a.mol_id[i];
  const int lo = a.mol_off[m], hi = a.mol_off[m + 1];
  const float4 pi = raw_pos4(a, i);
  if (lane == 0) {
    pos4[i] = pi;
    if (!(isfinite(pi.x) && isfinite(pi.y) && isfinite(pi.z))) atomicOr(a.status, NNP_ST_NONFINITE);
  }
  int nr = 0, na = 0;
  for (int base = lo; base < hi; base += 32) {
    const int j = base + lane;
    bool in_r = false, in_a = false;
    if (j < hi && j != i) {
      const float4 pj = raw_pos4(a, j);
      const double dx = (double)pj.x - (double)pi.x;
      const double dy = (double)pj.y - (double)pi.y;
      const double dz = (double)pj.z - (double)pi.z;
      const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
      in_r = d2 <= rc_r2;
      in_a = d2 <= rc_a2;
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
    if (nr > capR || na > capA) atomicOr(a.status, NNP_ST_CAPACITY);
    cnt_r[i] = min(nr, capR);
    cnt_a[i] = min(na, capA);
  }
}

// the same search for one centre with the molecule's positions already in shared memory (fused AEV forward path)
__device__ __forceinline__ void nbr_row_warp_smem(const float4* __restrict__ mp, int lo, int hi, int i, int lane,
                                                  double rc_r2, double rc_a2, int capR, int capA, int* status,
                                                  float4* __restrict__ pos4, int* __restrict__ nbr_r,
                                                  int* __restrict__ nbr_a, int* __restrict__ cnt_r, int* __restrict__ cnt_a) {
  const float4 pi = mp[i - lo];
  if (lane == 0) {
    pos4[i] = pi;
    if (!(isfinite(pi.x) && isfinite(pi.y) && isfinite(pi.z))) atomicOr(status, NNP_ST_NONFINITE);
  }
  int nr = 0, na = 0;
  for (int base = lo; base < hi; base += 32) {
    const int j = base + lane;
    bool in_r = false, in_a = false;
    if (j < hi && j != i) {
      const float4 pj = mp[j - lo];
      const double dx = (double)pj.x - (double)pi.x;
      const double dy = (double)pj.y - (double)pi.y;
      const double dz = (double)pj.z - (double)pi.z;
      const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
      in_r = d2 <= rc_r2;
      in_a = d2 <= rc_a2;
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

__global__ void __launch_bounds__(128) nbr_allpairs_kernel(const __grid_constant__ NbrArgs a, int N, double rc_r2,
                                                           double rc_a2, int capR, int capA, float4* __restrict__ pos4,
                                                           int* __restrict__ nbr_r, int* __restrict__ nbr_a,
                                                           int* __restrict__ cnt_r, int* __restrict__ cnt_a) {
  const int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  pdl_trigger();
  pdl_wait();  // the previous step's kernels still read the lists this kernel rewrites
  if (i >= N) return;
  nbr_row_warp(a, i, lane, rc_r2, rc_a2, capR, capA, pos4, nbr_r, nbr_a, cnt_r, cnt_a);
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

constexpr int AEV_THREADS = 256;  // one CTA per centre atom: 256 threads at latency-bound sizes, 128 at large N
constexpr int TAB_FIELDS = 11;    // per radial slot: ux uy uz rhi rlo fcr dfcr fca dfca spec rord
// triplets of a centre processed per pass through shared memory: small enough that 6-8 CTAs share an SM (the
// phases of a centre are latency-bound, other centres fill the gaps), measured on configs[2] and configs[4]
constexpr int TRIP_CHUNK_FWD = 256;
constexpr int TRIP_CHUNK_BWD = 512;  // upper bound; trip_chunk() halves it when that lets one more CTA share the SM

static int trip_chunk(const nnp_handle* h, bool backward);
static int ang_row_pad(const nnp_handle* h) {  // floats per padded angular block of the staged dE/dAEV row
  return h->aev.n_sub + 4;
}

// shared memory (floats): table | asl[capA] | sp_off[S+1] | pair_st[n_pairs] | tmp[2 capA] | pres[n_pairs+1] |
// r_off[S+1] | boff[n_pairs+1] | kernel part
static size_t aev_common_floats(const nnp_handle* h) {
  const int S = h->S;
  return (size_t)TAB_FIELDS * h->capR + 3 * (size_t)h->capA + 2 * (S + 1) + 3 * ((size_t)S * (S + 1) / 2) + 2;
}
static size_t aev_smem_bytes_ch(const nnp_handle* h, bool backward, int CH) {
  size_t fl = aev_common_floats(h);
  const int n_pairs = h->S * (h->S + 1) / 2;
  if (!backward) {
    fl += (size_t)(h->n_feat - h->aev.n_radial);                       // angular part of the row
    fl += (size_t)(h->aev.n_shf_z + h->aev.n_shf_a) * (CH + 1);        // F1 / F2 factors of a pass (row pitch CH + 1)
  } else {
    fl += (size_t)h->aev.n_radial + (size_t)n_pairs * ang_row_pad(h);  // dE/dAEV row (angular blocks padded)
    fl += (size_t)2 * 3 * h->capR;                                     // radial + angular pair gradients
    fl += (size_t)6 * CH;                                              // per-triplet gradient pairs of a pass
  }
  return ((fl + 3) & ~(size_t)3) * 4 + 16;
}
// shape of the backward launch: threads per centre CTA and triplets per pass (see aev_block_threads)
static void aev_bwd_shape(const nnp_handle* h, int* threads, int* chunk) {
  const long long t = (long long)h->capA * (h->capA - 1) / 2;
  const long long c = std::max<long long>(32, (t + 31) / 32 * 32);
  const int big = (int)std::min<long long>(c, TRIP_CHUNK_BWD), small = (int)std::min<long long>(c, TRIP_CHUNK_BWD / 2);
  *threads = AEV_THREADS;
  *chunk = big;
  if (h->N < 2048) return;
#ifdef AEV_BWD_FORCE_THREADS
  *threads = AEV_BWD_FORCE_THREADS;
  *chunk = AEV_BWD_FORCE_CHUNK < big ? AEV_BWD_FORCE_CHUNK : big;
  return;
#endif
  const size_t sm_bytes = 227 * 1024;
  if ((aev_smem_bytes_ch(h, true, big) + 1024) * 8 <= sm_bytes) { *threads = 128; return; }
  if ((aev_smem_bytes_ch(h, true, small) + 1024) * 8 <= sm_bytes) { *threads = 128; *chunk = small; }
}
// triplets per pass: enough for every centre of this handle, a multiple of 32, bounded
static int trip_chunk(const nnp_handle* h, bool backward) {
  if (backward) {
    int th, ch;
    aev_bwd_shape(h, &th, &ch);
    return ch;
  }
  const long long t = (long long)h->capA * (h->capA - 1) / 2;
  return (int)std::min<long long>(std::max<long long>(32, (t + 31) / 32 * 32), TRIP_CHUNK_FWD);
}
size_t aev_smem_bytes(const nnp_handle* h, bool backward) { return aev_smem_bytes_ch(h, backward, trip_chunk(h, backward)); }

struct CentreTab {
  float *ux, *uy, *uz, *rhi, *rlo, *fcr, *dfcr, *fca, *dfca;
  int* spec;
  int* rord;     // radial slots grouped by species (stable within a species)
  int* r_off;    // [S+1] first position in rord of every species
  int* asl;      // angular neighbours: radial slots, sorted by species (stable)
  int* sp_off;   // [S+1] first position in asl of every species
  int* pair_st;  // [n_pairs] (s << 8) | t of every species-pair block, s <= t
  int* tmp;      // [2 capA] scratch of build_tab: angular slots and their species in list order
  int* pres;     // [n_pairs + 1] species-pair blocks that have at least one triplet (ascending), count at [n_pairs]
  int* boff;     // [n_pairs + 1] first triplet of every PRESENT block in the block-ordered triplet enumeration
  float* rest;   // kernel-specific part (16-byte aligned)
};

__device__ __forceinline__ CentreTab carve_tab(float* smem, int capR, int capA, int S) {
  CentreTab t;
  t.ux = smem; t.uy = t.ux + capR; t.uz = t.uy + capR; t.rhi = t.uz + capR; t.rlo = t.rhi + capR;
  t.fcr = t.rlo + capR; t.dfcr = t.fcr + capR; t.fca = t.dfcr + capR; t.dfca = t.fca + capR;
  t.spec = reinterpret_cast<int*>(t.dfca + capR);
  t.rord = t.spec + capR;
  t.asl = t.rord + capR;
  t.sp_off = t.asl + capA;
  t.pair_st = t.sp_off + (S + 1);
  t.tmp = t.pair_st + S * (S + 1) / 2;
  t.pres = t.tmp + 2 * capA;
  t.r_off = t.pres + S * (S + 1) / 2 + 1;
  t.boff = t.r_off + (S + 1);
  const int used = TAB_FIELDS * capR + 3 * capA + 2 * (S + 1) + 3 * (S * (S + 1) / 2) + 2;
  t.rest = smem + ((used + 3) & ~3);
  return t;
}

// Phase 0 of both AEV kernels: geometry of every radial neighbour of centre i (FP64 once, all threads
// of the CTA in parallel), the angular neighbour list re-ordered by species (so the triplets of one
// species-pair block are index ranges), the species offsets and the block -> species-pair table.
__device__ __forceinline__ void build_tab(const CentreTab& t, int i, int nr, int na, const float4 pi,
                                          const float4* __restrict__ pos4, const int* __restrict__ nbr_r,
                                          const int* __restrict__ nbr_a, int capR, int capA, const AevConst& c,
                                          bool want_pres, const float4* mol_pos = nullptr, int mol_lo = 0) {
  for (int q = threadIdx.x; q < nr; q += blockDim.x) {
    const int j = nbr_r[(size_t)i * capR + q];
    const float4 pj = mol_pos ? mol_pos[j - mol_lo] : pos4[j];  // fused neighbour search: pos4[j] is another CTA's job
    const double dx = (double)pj.x - (double)pi.x;
    const double dy = (double)pj.y - (double)pi.y;
    const double dz = (double)pj.z - (double)pi.z;
    // 1/r by two Newton steps on the FP32 rsqrt seed (relative error 1e-7 -> 1e-14 -> rounding), r = r2 / r
    const double r2 = dx * dx + dy * dy + dz * dz;
    double inv = (double)rsqrtf((float)r2);
    inv = inv * (1.5 - 0.5 * r2 * inv * inv);
    inv = inv * (1.5 - 0.5 * r2 * inv * inv);
    const double r = r2 * inv;
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
  // block -> (s, t) table: row-major upper triangle
  for (int s = threadIdx.x; s < c.S; s += blockDim.x) {
    int p = s * c.S - (s * (s - 1)) / 2;
    for (int u = s; u < c.S; ++u) t.pair_st[p++] = (s << 8) | u;
  }
  __syncthreads();
  if (want_pres) {
    // radial slots grouped by species, list order kept within a species (ballot compaction, one warp per species):
    // a radial column then visits the neighbours of ITS species only, in the order the full loop would add them
    const int lane = threadIdx.x & 31;
    for (int s = threadIdx.x >> 5; s < c.S; s += (int)(blockDim.x >> 5)) {
      int less = 0;
      for (int q0 = 0; q0 < nr; q0 += 32) {
        const int q = q0 + lane;
        less += __popc(__ballot_sync(FULL, q < nr && t.spec[q] < s));
      }
      int pos = less;
      for (int q0 = 0; q0 < nr; q0 += 32) {
        const int q = q0 + lane;
        const bool m = q < nr && t.spec[q] == s;
        const unsigned b = __ballot_sync(FULL, m);
        if (m) t.rord[pos + __popc(b & ((1u << lane) - 1u))] = q;
        pos += __popc(b);
      }
      if (lane == 0) {
        t.r_off[s] = less;
        if (s == c.S - 1) t.r_off[c.S] = pos;
      }
    }
  }
  // the angular slots and their species, staged once (the sort below reads them na times)
  for (int q = threadIdx.x; q < na; q += blockDim.x) {
    const int slot = nbr_a[(size_t)i * capA + q];
    t.tmp[q] = slot;
    t.tmp[capA + q] = t.spec[slot];
  }
  __syncthreads();
  // stable counting sort of the angular list by species: rank = #(smaller species) + #(same, earlier)
  for (int q = threadIdx.x; q < na; q += blockDim.x) {
    const int sp = t.tmp[capA + q];
    int rank = 0;
#pragma unroll 4
    for (int q2 = 0; q2 < na; ++q2) {
      const int s2 = t.tmp[capA + q2];
      rank += (s2 < sp) || (s2 == sp && q2 < q);
    }
    t.asl[rank] = t.tmp[q];
  }
  for (int s = threadIdx.x; s <= c.S; s += blockDim.x) {
    int cnt = 0;
#pragma unroll 4
    for (int q2 = 0; q2 < na; ++q2) cnt += t.tmp[capA + q2] < s;
    t.sp_off[s] = cnt;
  }
  __syncthreads();
  if (!want_pres) return;  // CTA-uniform
  // species-pair blocks with at least one triplet, in ascending order (ballot compaction by the first warp)
  if (threadIdx.x < 32) {
    const int n_pairs = (c.S * (c.S + 1)) >> 1;
    int count = 0;
    for (int base = 0; base < n_pairs; base += 32) {
      const int p = base + (int)threadIdx.x;
      bool has = false;
      if (p < n_pairs) {
        const int st = t.pair_st[p], s = st >> 8, u = st & 255;
        const int ns = t.sp_off[s + 1] - t.sp_off[s], nu = t.sp_off[u + 1] - t.sp_off[u];
        has = s == u ? ns >= 2 : (ns > 0 && nu > 0);
      }
      const unsigned b = __ballot_sync(FULL, has);
      if (has) t.pres[count + __popc(b & ((1u << threadIdx.x) - 1u))] = p;
      count += __popc(b);
    }
    if (threadIdx.x == 0) t.pres[n_pairs] = count;
    __syncwarp();
    // block-ordered triplet enumeration: the triplets of present block pp are [boff[pp], boff[pp + 1]) (warp scan)
    int carry = 0;
    for (int base = 0; base < count; base += 32) {
      const int pp = base + (int)threadIdx.x;
      int cnt = 0;
      if (pp < count) {
        const int st = t.pair_st[t.pres[pp]], s = st >> 8, u = st & 255;
        const int ns = t.sp_off[s + 1] - t.sp_off[s], nu = t.sp_off[u + 1] - t.sp_off[u];
        cnt = s == u ? (ns * (ns - 1)) >> 1 : ns * nu;
      }
      int incl = cnt;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(FULL, incl, o);
        if ((int)threadIdx.x >= o) incl += v;
      }
      if (pp < count) t.boff[pp + 1] = carry + incl;
      carry += __shfl_sync(FULL, incl, 31);
    }
    if (threadIdx.x == 0) t.boff[0] = 0;
  }
  __syncthreads();
}

// unordered triplets (a, b), a < b < na, in row-major order: flat index and its inverse
__device__ __forceinline__ int trip_row_start(int a, int na) { return (a * (2 * na - a - 1)) >> 1; }
__device__ __forceinline__ void trip_decode(int t, int na, int& a, int& b) {
  const float m = (float)(2 * na - 1);
  int r = (int)(0.5f * (m - sqrtf(fmaxf(m * m - 8.0f * (float)t, 0.0f))));
  r = max(0, min(r, na - 2));
  while (r > 0 && trip_row_start(r, na) > t) --r;
  while (r < na - 2 && trip_row_start(r + 1, na) <= t) ++r;
  a = r;
  b = t - trip_row_start(r, na) + r + 1;
}

// ------------------------------------------------------------------------------------------------
// A2 + A3: AEV forward.  One CTA per centre.
//   radial : one thread per output column (species s, shift k) loops over the neighbours of species s
//            and keeps the sum in a register (fixed order, no shared-memory updates);
//   angular: the angular term is separable, A = F1_z(theta) * [2 F2_a(r_a, r_b) f_C f_C], so
//            pass 1: one THREAD per triplet evaluates its n_shf_z powers and n_shf_a Gaussians once
//                    (12 transcendental groups instead of 32 per triplet) into shared memory;
//            pass 2: one thread per output column (block p, a, z) sums F1_z * F2_a over the triplets of
//                    its species-pair block, which are index ranges because the angular list is sorted by
//                    species.  Fixed order, no atomics.
// NZ / NA are the register-array bounds (n_shf_z <= NZ, n_shf_a <= NA).
// ------------------------------------------------------------------------------------------------
// 4 CTAs of 256 threads (8 of 128 at large N) per SM: 64 registers per thread.  A bound of 6 (40 registers) spilled in
// the backward kernel and measured 8-11 % slower at configs[4]; shared memory, not registers, limits residency there.
constexpr int AEV_MINB = 4;
template <int NZ, int NA>
__global__ void __launch_bounds__(AEV_THREADS, AEV_MINB) aev_forward_kernel(
    const float4* __restrict__ pos4, const int* __restrict__ nbr_r, const int* __restrict__ nbr_a,
    const int* __restrict__ cnt_r, const int* __restrict__ cnt_a, const int* __restrict__ sortpos, int N,
    const __grid_constant__ AevConst c, int capR, int capA, int CH, float* __restrict__ aev, float* __restrict__ aev_lo,
    const __grid_constant__ NbrArgs nb, int fused, int mp_off4, float4* __restrict__ pos4_w, int* __restrict__ nbr_r_w,
    int* __restrict__ nbr_a_w, int* __restrict__ cnt_r_w, int* __restrict__ cnt_a_w) {
  extern __shared__ __align__(16) float smem[];
  const int i = blockIdx.x;
  const CentreTab t = carve_tab(smem, capR, capA, c.S);
  const int n_ang = c.n_feat - c.n_radial;
  float* row = t.rest;                 // [n_ang]
  // row pitch CH + 1: in the column sums below the lanes of a warp read the same triplet of DIFFERENT rows (one per
  // (ShfA, ShfZ) sub-term); with a pitch that is a multiple of 32 those were 4- and 8-way bank conflicts (ncu: 55 % of
  // the kernel's shared-memory wavefronts)
  const int CHP = CH + 1;
  float* bF1 = row + n_ang;            // [n_shf_z][CHP]
  float* bF2 = bF1 + c.n_shf_z * CHP;  // [n_shf_a][CHP]
  pdl_trigger();
  pdl_wait();
  float4* mp = reinterpret_cast<float4*>(smem) + mp_off4;  // [max molecule size]: the molecule's positions (fused path)
  int mlo = 0;
  if (fused) {
    // small systems: the centre's CTA builds its own neighbour rows instead of a separate launch.  All threads load
    // the molecule's positions into shared memory (one memory round trip), the first warp runs the pair search on
    // them; the rows also go to global memory for the backward and gather kernels.
    const int2 rg = nb.mol_range[i];
    mlo = rg.x;
    for (int j = rg.x + (int)threadIdx.x; j < rg.y; j += blockDim.x) mp[j - rg.x] = raw_pos4(nb, j);
    __syncthreads();
    if (threadIdx.x < 32)
      nbr_row_warp_smem(mp, rg.x, rg.y, i, threadIdx.x, c.rc_r2, c.rc_a2, capR, capA, nb.status, pos4_w, nbr_r_w, nbr_a_w,
                        cnt_r_w, cnt_a_w);
    __syncthreads();  // the CTA's own global writes are visible to the CTA
  }
  const float4 pi = fused ? mp[i - mlo] : pos4[i];
  const int nr = fused ? cnt_r_w[i] : cnt_r[i], na = fused ? cnt_a_w[i] : cnt_a[i];
  for (int f = threadIdx.x; f < n_ang; f += blockDim.x) row[f] = 0.0f;
  build_tab(t, i, nr, na, pi, pos4, fused ? nbr_r_w : nbr_r, fused ? nbr_a_w : nbr_a, capR, capA, c, true,
            fused ? mp : nullptr, mlo);
  float* out = aev + (size_t)sortpos[i] * c.n_feat;
  // tensor engine: the row is written as two TF32-exact planes (hi = rna_tf32(G), lo = G - hi), the operand format of
  // the 3xTF32 layer-1 GEMM
  float* out_lo = aev_lo ? aev_lo + (size_t)sortpos[i] * c.n_feat : nullptr;

  // ---- radial (O3)
  for (int col = threadIdx.x; col < c.n_radial; col += blockDim.x) {
    const int s = col / c.n_shf_r, k = col % c.n_shf_r;
    const float shf = c.shf_r[k];
    float acc = 0.0f;
    const int p1 = t.r_off[s + 1];
#pragma unroll 4
    for (int p = t.r_off[s]; p < p1; ++p) {  // the neighbours of species s, in list order
      const int q = t.rord[p];
      const float d = (t.rhi[q] - shf) + t.rlo[q];
      acc += 0.25f * gauss(d, c.kr_hi, c.kr_lo) * t.fcr[q];
    }
    if (out_lo) {
      const float hi = __uint_as_float((__float_as_uint(acc) + 0x1000u) & 0xFFFFE000u);
      out[col] = hi;
      out_lo[col] = acc - hi;
    } else {
      out[col] = acc;
    }
  }

  // ---- angular (O4)
  const int ntrip = (na * (na - 1)) >> 1;
  const int n_pres = t.pres[(c.S * (c.S + 1)) >> 1];
  for (int c0 = 0; c0 < ntrip; c0 += CH) {
    const int cn = min(CH, ntrip - c0);
    for (int tl = threadIdx.x; tl < cn; tl += blockDim.x) {
      // triplet number c0 + tl of the BLOCK-ORDERED enumeration (all triplets of the first present species-pair block,
      // then the next ...; inside a block (a, b) row-major as before): the column sums below are then plain ranges
      const int g = c0 + tl;
      int lo_pp = 0, hi_pp = n_pres;  // boff[lo_pp] <= g < boff[hi_pp]
      while (hi_pp - lo_pp > 1) {
        const int mid = (lo_pp + hi_pp) >> 1;
        if (t.boff[mid] <= g) lo_pp = mid; else hi_pp = mid;
      }
      int a, b;
      {
        const int st = t.pair_st[t.pres[lo_pp]], s = st >> 8, u = st & 255;
        const int local = g - t.boff[lo_pp];
        const int a0 = t.sp_off[s];
        if (s == u) {
          trip_decode(local, t.sp_off[s + 1] - a0, a, b);
          a += a0; b += a0;
        } else {
          const int b0 = t.sp_off[u], nu = t.sp_off[u + 1] - b0;
          const int qa_ = local / nu;
          a = a0 + qa_;
          b = b0 + (local - qa_ * nu);
        }
      }
      const int qa = t.asl[a], qb = t.asl[b];
      const float cth = t.ux[qa] * t.ux[qb] + t.uy[qa] * t.uy[qb] + t.uz[qa] * t.uz[qb];
      const float cc = c.cos_scale * cth;
      const float ss = sqrt_approx(fmaxf(fmaf(-cc, cc, 1.0f), 0.0f));
#pragma unroll
      for (int iz = 0; iz < NZ; ++iz) {
        if (iz < c.n_shf_z) {
          const float u = 0.5f + 0.5f * ((cc * c.cos_z[iz] + ss * c.sin_z[iz]) + (cc * c.cos_z_lo[iz] + ss * c.sin_z_lo[iz]));
          bF1[iz * CHP + tl] = pow_split(u, c.zeta_int, c.zeta_frac);
        }
      }
      const float w = 2.0f * (t.fca[qa] * t.fca[qb]);
      const float ra = t.rhi[qa], rb = t.rhi[qb], rl = t.rlo[qa] + t.rlo[qb];
#pragma unroll
      for (int ia = 0; ia < NA; ++ia) {
        if (ia < c.n_shf_a) {
          const float shfa = c.shf_a[ia];
          const float d = 0.5f * (((ra - shfa) + (rb - shfa)) + rl);
          bF2[ia * CHP + tl] = w * gauss(d, c.ka_hi, c.ka_lo);
        }
      }
    }
    __syncthreads();
    const int n_out = n_pres * c.n_sub;  // columns of the blocks that have triplets
    for (int fo = threadIdx.x; fo < n_out; fo += blockDim.x) {
      const int pp = fo / c.n_sub, sub = fo - pp * c.n_sub;
      const int f = t.pres[pp] * c.n_sub + sub;
      const int ia = sub / c.n_shf_z, iz = sub - ia * c.n_shf_z;
      const float* f1 = bF1 + iz * CHP - c0;
      const float* f2 = bF2 + ia * CHP - c0;
      const int lo = max(t.boff[pp], c0), hi = min(t.boff[pp + 1], c0 + cn);  // the block's triplets in this pass
      float acc = 0.0f;
#pragma unroll 4
      for (int g = lo; g < hi; ++g) acc = fmaf(f1[g], f2[g], acc);
      row[f] += acc;
    }
    __syncthreads();
  }
  if (out_lo) {
    for (int f = threadIdx.x; f < n_ang; f += blockDim.x) {
      const float v = row[f];
      const float hi = __uint_as_float((__float_as_uint(v) + 0x1000u) & 0xFFFFE000u);
      out[c.n_radial + f] = hi;
      out_lo[c.n_radial + f] = v - hi;
    }
  } else {
    for (int f = threadIdx.x; f < n_ang; f += blockDim.x) out[c.n_radial + f] = row[f];
  }
}

// ------------------------------------------------------------------------------------------------
// A7: AEV backward.  One CTA per centre.  phi[i][slot] = dE/d(r_j - r_i) for every radial slot of i
// (pair-gradient formulation), added to the two atoms of the pair in 64-bit fixed point (integer atomics only).
//   angular: one THREAD per triplet.  With G the n_shf_a x n_shf_z block of dE/dAEV of the triplet's
//   species pair,  R0 = sum_a F2_a (G F1)_a,  R1 = sum_a dF2_a (G F1)_a,  R2 = sum_a F2_a (G dF1)_a  are
//   register sums (4 powers + 8 Gaussians + 8 float4 shared-memory loads per triplet for ANI-2x); the
//   triplet's two pair gradients go to a shared-memory buffer and one thread per (neighbour, component)
//   adds them in triplet order (fixed order => bit-identical reruns).
// ------------------------------------------------------------------------------------------------
// fixed-point force accumulator: 2^-44 model force units per count, range +-5e5
constexpr double FACC_ONE = 17592186044416.0;  // 2^44

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
  return v;
}

// MULTI: dE/dAEV arrives as several partial rows (ligand sizes, one per model); a separate instantiation so that its
// wider load batch does not cost the large-system instantiation registers (occupancy)
template <int NZ, int NA, bool MULTI>
__global__ void __launch_bounds__(AEV_THREADS, MULTI ? 4 : AEV_MINB) aev_backward_kernel(
    const float4* __restrict__ pos4, const int* __restrict__ nbr_r, const int* __restrict__ nbr_a,
    const int* __restrict__ cnt_r, const int* __restrict__ cnt_a, const int* __restrict__ sortpos, int N,
    const __grid_constant__ AevConst c, int capR, int capA, int CH, const float* __restrict__ daev, int n_parts,
    size_t part_stride, unsigned long long live_boxes, unsigned long long* __restrict__ facc) {
  extern __shared__ __align__(16) float smem[];
  const int i = blockIdx.x;
  const CentreTab t = carve_tab(smem, capR, capA, c.S);
  const int n_pairs = (c.S * (c.S + 1)) >> 1;
  const int bpad = c.n_sub + 4;         // padded block pitch: blocks of different species pairs hit different banks
  float* g = t.rest;                    // [n_radial]
  float* gang = g + c.n_radial;         // [n_pairs][bpad]
  float* phr = gang + n_pairs * bpad;   // radial part   [capR][3]
  float* pha = phr + 3 * capR;          // angular part  [capR][3]
  float* buf = pha + 3 * capR;          // [6][CH] pair gradients of the triplets of a pass
  pdl_trigger();
  pdl_wait();
  const float4 pi = pos4[i];
  const int nr = cnt_r[i], na = cnt_a[i];
  const float* gin = daev + (size_t)sortpos[i] * c.n_feat;
  // dE/dAEV row = fixed-order sum of the partial rows, staged in shared memory (angular blocks padded).  A warp takes
  // 32-column boxes of the row; the boxes that hold only structural zeros (species that do not occur in the system:
  // `live_boxes`, the mask layer 1 skips by) are never read below and are not loaded (water: 8 of 32 boxes).  All
  // loads of a pass are issued before the first add: one memory latency per pass, not one per partial row.
  // (Loading only the columns THIS centre touches -- known after the table is built -- saves more instructions and
  // LOSES 5 % of the time at configs[4]: the row load then sits on the centre's dependency chain.)
  {
    const int nbox = (c.n_feat + 31) >> 5;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nw = blockDim.x >> 5;
    const unsigned long long live = live_boxes ? live_boxes : ~0ull;
    const int sub_shift = (c.n_sub & (c.n_sub - 1)) == 0 ? __ffs(c.n_sub) - 1 : -1;  // n_sub = 32 for ANI-1x / ANI-2x
    auto put = [&](int f, float v) {
      if (f < c.n_radial) {
        g[f] = v;
      } else {
        const int fa = f - c.n_radial;
        const int blk = sub_shift >= 0 ? fa >> sub_shift : fa / c.n_sub;
        gang[blk * bpad + (fa - blk * c.n_sub)] = v;
      }
    };
    constexpr int KB = MULTI ? 4 : 8;  // boxes per warp and pass
    for (int b0 = warp; b0 < nbox; b0 += KB * nw) {
      if (!MULTI) {  // large systems: one row
        float x[KB];
#pragma unroll
        for (int k = 0; k < KB; ++k) {
          const int bx = b0 + k * nw, f = bx * 32 + lane;
          x[k] = (bx < nbox && ((live >> bx) & 1ull) && f < c.n_feat) ? gin[f] : 0.0f;
        }
#pragma unroll
        for (int k = 0; k < KB; ++k) {
          const int bx = b0 + k * nw, f = bx * 32 + lane;
          if (bx < nbox && ((live >> bx) & 1ull) && f < c.n_feat) put(f, x[k]);
        }
      } else {
        float acc[KB];
#pragma unroll
        for (int k = 0; k < KB; ++k) acc[k] = 0.0f;
        for (int p0 = 0; p0 < n_parts; p0 += 8) {
          float x[KB][8];
#pragma unroll
          for (int k = 0; k < KB; ++k) {
            const int bx = b0 + k * nw, f = bx * 32 + lane;
            const bool on = bx < nbox && ((live >> bx) & 1ull) && f < c.n_feat;
#pragma unroll
            for (int u = 0; u < 8; ++u) x[k][u] = (on && p0 + u < n_parts) ? gin[(size_t)(p0 + u) * part_stride + f] : 0.0f;
          }
#pragma unroll
          for (int k = 0; k < KB; ++k)
#pragma unroll
            for (int u = 0; u < 8; ++u) acc[k] += x[k][u];
        }
#pragma unroll
        for (int k = 0; k < KB; ++k) {
          const int bx = b0 + k * nw, f = bx * 32 + lane;
          if (bx < nbox && ((live >> bx) & 1ull) && f < c.n_feat) put(f, acc[k]);
        }
      }
    }
  }
  for (int f = threadIdx.x; f < 3 * nr; f += blockDim.x) pha[f] = 0.0f;
  build_tab(t, i, nr, na, pi, pos4, nbr_r, nbr_a, capR, capA, c, false);

  // ---- radial: dT/dr = 0.25 e (f_C' - 2 eta (r - Shf) f_C); four lanes per neighbour, each takes every fourth
  // shift (a 16-lane group per neighbour spent half of its instructions in the shuffle tree)
  {
    const int q4 = threadIdx.x >> 2, l4 = threadIdx.x & 3, per_pass = blockDim.x >> 2;
    for (int q0 = 0; q0 < nr; q0 += per_pass) {
      const int q = q0 + q4;
      float v = 0.0f;
      if (q < nr) {
        const float rh = t.rhi[q], rl = t.rlo[q], fc = t.fcr[q], dfc = t.dfcr[q];
        const float* gs = g + t.spec[q] * c.n_shf_r;
        for (int k = l4; k < c.n_shf_r; k += 4) {
          const float d = (rh - c.shf_r[k]) + rl;
          const float ex = 0.25f * gauss(d, c.kr_hi, c.kr_lo);
          v = fmaf(gs[k], ex * (dfc - 2.0f * c.eta_r * d * fc), v);
        }
      }
      v += __shfl_xor_sync(FULL, v, 1);
      v += __shfl_xor_sync(FULL, v, 2);
      if (q < nr && l4 < 3) phr[3 * q + l4] = v * (l4 == 0 ? t.ux[q] : l4 == 1 ? t.uy[q] : t.uz[q]);
    }
  }

  // ---- angular: A = 2 F1 F2 fa fb
  const int ntrip = (na * (na - 1)) >> 1;
  const bool vec4 = (NZ == 4) && c.n_shf_z == 4 && (c.n_radial & 3) == 0;
  for (int c0 = 0; c0 < ntrip; c0 += CH) {
    const int cn = min(CH, ntrip - c0);
    for (int tl = threadIdx.x; tl < cn; tl += blockDim.x) {
      int a, b;
      trip_decode(c0 + tl, na, a, b);
      const int qa = t.asl[a], qb = t.asl[b];
      const float uax = t.ux[qa], uay = t.uy[qa], uaz = t.uz[qa];
      const float ubx = t.ux[qb], uby = t.uy[qb], ubz = t.uz[qb];
      const float cth = uax * ubx + uay * uby + uaz * ubz;
      const float cc = c.cos_scale * cth;
      const float ss = sqrt_approx(fmaxf(fmaf(-cc, cc, 1.0f), 0.0f));
      const float cot = cc * rcp_approx(ss);
      const float ra = t.rhi[qa], rb = t.rhi[qb];
      const float rl = t.rlo[qa] + t.rlo[qb];
      const int sa = t.spec[qa], sb = t.spec[qb];  // sa <= sb (sorted)
      const float* gb = gang + (sa * c.S - (sa * (sa - 1)) / 2 + (sb - sa)) * bpad;
      float F1[NZ], dF1[NZ];
#pragma unroll
      for (int iz = 0; iz < NZ; ++iz) {
        F1[iz] = 0.0f; dF1[iz] = 0.0f;
        if (iz < c.n_shf_z) {
          const float cz = c.cos_z[iz], sz = c.sin_z[iz];
          const float u = 0.5f + 0.5f * ((cc * cz + ss * sz) + (cc * c.cos_z_lo[iz] + ss * c.sin_z_lo[iz]));
          const float pw1 = pow_split(u, c.zeta1_int, c.zeta_frac);  // u^(zeta-1)
          F1[iz] = pw1 * u;
          dF1[iz] = c.zeta * pw1 * 0.5f * (cz - cot * sz);
        }
      }
      float R0 = 0.f, R1 = 0.f, R2 = 0.f;
#pragma unroll
      for (int ia = 0; ia < NA; ++ia) {
        if (ia < c.n_shf_a) {
          const float shfa = c.shf_a[ia];
          const float d = 0.5f * (((ra - shfa) + (rb - shfa)) + rl);
          const float F2 = gauss(d, c.ka_hi, c.ka_lo);
          float s1 = 0.f, s2 = 0.f;
          if (vec4) {
            const float4 gv = *reinterpret_cast<const float4*>(gb + 4 * ia);
            s1 = gv.x * F1[0]; s2 = gv.x * dF1[0];
            if (NZ > 1) { s1 = fmaf(gv.y, F1[1 % NZ], s1); s2 = fmaf(gv.y, dF1[1 % NZ], s2); }
            if (NZ > 2) { s1 = fmaf(gv.z, F1[2 % NZ], s1); s2 = fmaf(gv.z, dF1[2 % NZ], s2); }
            if (NZ > 3) { s1 = fmaf(gv.w, F1[3 % NZ], s1); s2 = fmaf(gv.w, dF1[3 % NZ], s2); }
          } else {
#pragma unroll
            for (int iz = 0; iz < NZ; ++iz) {
              if (iz < c.n_shf_z) {
                const float gv = gb[ia * c.n_shf_z + iz];
                s1 = fmaf(gv, F1[iz], s1);
                s2 = fmaf(gv, dF1[iz], s2);
              }
            }
          }
          R0 = fmaf(F2, s1, R0);
          R1 = fmaf(-c.eta_a * d * F2, s1, R1);
          R2 = fmaf(F2, s2, R2);
        }
      }
      const float fa = t.fca[qa], fb = t.fca[qb];
      const float W = fa * fb;
      const float coefA = 2.0f * (W * R1 + t.dfca[qa] * fb * R0);
      const float coefB = 2.0f * (W * R1 + fa * t.dfca[qb] * R0);
      const float coefC = 2.0f * W * R2 * c.cos_scale;
      const float ia_r = coefC * rcp_approx(ra), ib_r = coefC * rcp_approx(rb);
      buf[0 * CH + tl] = coefA * uax + ia_r * (ubx - cth * uax);
      buf[1 * CH + tl] = coefA * uay + ia_r * (uby - cth * uay);
      buf[2 * CH + tl] = coefA * uaz + ia_r * (ubz - cth * uaz);
      buf[3 * CH + tl] = coefB * ubx + ib_r * (uax - cth * ubx);
      buf[4 * CH + tl] = coefB * uby + ib_r * (uay - cth * uby);
      buf[5 * CH + tl] = coefB * ubz + ib_r * (uaz - cth * ubz);
    }
    __syncthreads();
    // one thread per (angular neighbour s, component): add the gradients of the triplets that contain s
    for (int w = threadIdx.x; w < 3 * na; w += blockDim.x) {
      const int comp = w / na, s = w - comp * na;
      float acc = 0.0f;
      for (int a = 0; a < s; ++a) {  // triplets (a, s): s is the second member
        const int tl = trip_row_start(a, na) + (s - a - 1) - c0;
        if (tl >= 0 && tl < cn) acc += buf[(3 + comp) * CH + tl];
      }
      {  // triplets (s, b), b > s: a contiguous run
        const int base = trip_row_start(s, na) - s - 1 - c0;
        const int lo = max(s + 1, -base), hi = min(na, cn - base);
        for (int b = lo; b < hi; ++b) acc += buf[comp * CH + base + b];
      }
      pha[3 * t.asl[s] + comp] += acc;
    }
    __syncthreads();
  }
  __syncthreads();
  // A8, first half: phi[i][q] = dE/d(r_j - r_i) is a force of +phi on the centre i and of -phi on the neighbour j.
  // Both go straight into the per-atom accumulator facc[N][3] as 64-bit fixed point (2^FACC_BITS per model force
  // unit): integer adds commute, so the sum has the same bits in whatever order the centres arrive (bit-identical
  // reruns without a gather pass; the previous design wrote phi[N][capR][3] and the finish kernel looked up, by binary
  // search, the slot of every atom in the rows of its neighbours).  Centre: the threads add up their own terms, one
  // shuffle tree per warp, three atomics per warp.
  {
    long long self[3] = {0, 0, 0};
    const int* rowi = nbr_r + (size_t)i * capR;
    for (int f = threadIdx.x; f < 3 * nr; f += blockDim.x) {
      const int q = f / 3, comp = f - 3 * q;
      const long long v = __double2ll_rn((double)(phr[f] + pha[f]) * FACC_ONE);
      atomicAdd(facc + (size_t)rowi[q] * 3 + comp, (unsigned long long)(-v));
      self[0] += comp == 0 ? v : 0;
      self[1] += comp == 1 ? v : 0;
      self[2] += comp == 2 ? v : 0;
    }
#pragma unroll
    for (int comp = 0; comp < 3; ++comp) {
      long long v = self[comp];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
      if ((threadIdx.x & 31) == 0 && v != 0) atomicAdd(facc + (size_t)i * 3 + comp, (unsigned long long)v);
    }
  }
}

// ------------------------------------------------------------------------------------------------
// A8 (second half) + A5: F_a = sum_j phi[a][j] - sum_i phi[i][a] sits in the fixed-point accumulator facc (filled by
// the AEV backward kernel); it is converted, scaled, added into the caller's force buffer (mechanical embedding,
// PAPER.md:50-71,75) and the accumulator entry is cleared for the next step.  Energies per molecule in FP64.  Blocks
// [0, n_force_blocks) do forces (thread per atom), the remaining blocks do energies.  Integer accumulation and fixed
// reduction trees => bit-identical reruns.
// ------------------------------------------------------------------------------------------------
constexpr int FIN_THREADS = 256;
constexpr int FIN_WARPS = FIN_THREADS / 32;

__global__ void __launch_bounds__(FIN_THREADS) finish_kernel(
    unsigned long long* __restrict__ facc, int N, const int* __restrict__ atom_index, void* __restrict__ force,
    int force_stride, int fixed, float fscale, int n_force_blocks, const double* __restrict__ eatom,
    const int* __restrict__ sortpos, const int* __restrict__ species, const int* __restrict__ mol_off, int n_mol, int M,
    const double* __restrict__ self_energy, double escale, double* __restrict__ energy,
    const EnergyBlock* __restrict__ eblocks, int n_eblocks, double* __restrict__ epart, int* __restrict__ ecount) {
  const int lane = threadIdx.x & 31;
  const int wib = threadIdx.x >> 5;
  pdl_trigger();
  pdl_wait();
  if ((int)blockIdx.x < n_force_blocks) {
    const int a = blockIdx.x * FIN_THREADS + threadIdx.x;
    if (a >= N) return;
    unsigned long long* acc = facc + (size_t)a * 3;
    const long long ix = (long long)acc[0], iy = (long long)acc[1], iz = (long long)acc[2];
    acc[0] = 0ull; acc[1] = 0ull; acc[2] = 0ull;  // ready for the next step, whether or not forces were asked for
    if (force == nullptr) return;
    const double inv = 1.0 / FACC_ONE;
    const int row = atom_index ? atom_index[a] : a;
    if (fixed & 1) {
      // 64-bit fixed point (2^32 per force unit, the accumulation format of GPU MD engines): integer atomic adds
      // commute, so MM kernels running CONCURRENTLY may add into the same buffer and the sum has the same bits in
      // any order (NNP and MM concurrently instead of sequentially)
      unsigned long long* f = reinterpret_cast<unsigned long long*>(force) + (size_t)row * force_stride;
      const double sc = (double)fscale * 4294967296.0 * inv;
      atomicAdd(f + 0, (unsigned long long)__double2ll_rn(sc * (double)ix));
      atomicAdd(f + 1, (unsigned long long)__double2ll_rn(sc * (double)iy));
      atomicAdd(f + 2, (unsigned long long)__double2ll_rn(sc * (double)iz));
    } else {
      const float fx = (float)((double)ix * inv), fy = (float)((double)iy * inv), fz = (float)((double)iz * inv);
      float* f = reinterpret_cast<float*>(force) + (size_t)row * force_stride;
      if (fixed & 2) {  // nnp_compute_host: the buffer is the library's own, forces are WRITTEN
        f[0] = fscale * fx;
        f[1] = fscale * fy;
        f[2] = fscale * fz;
      } else {  // plain read-modify-write: safe only when every other adder is ordered with this stream
        f[0] += fscale * fx;
        f[1] += fscale * fy;
        f[2] += fscale * fz;
      }
    }
  } else {
    // energy blocks: a CTA sums a chunk of a molecule (thread-strided atoms, warp tree, then the warps in order).  A
    // molecule larger than one chunk is summed by several CTAs; the last one to arrive adds their partial sums in
    // chunk order (fixed order => bit-identical reruns whatever the arrival order).
    __shared__ double wsum[FIN_WARPS];
    __shared__ int s_last;
    const int bid = blockIdx.x - n_force_blocks;
    if (bid >= n_eblocks || energy == nullptr) return;
    const EnergyBlock eb = eblocks[bid];
    double acc = 0.0;
    for (int i = eb.a0 + (int)threadIdx.x; i < eb.a1; i += FIN_THREADS) {
      const double* e = eatom + (size_t)sortpos[i] * M;
      double s = 0.0;
#pragma unroll 8
      for (int k = 0; k < M; ++k) s += e[k];
      acc += s / (double)M + (self_energy ? self_energy[species[i]] : 0.0);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(FULL, acc, o);
    if (lane == 0) wsum[wib] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
      double tot = 0.0;
      for (int w = 0; w < FIN_WARPS; ++w) tot += wsum[w];
      if (eb.n_chunks == 1) {
        energy[eb.mol] = escale * tot;
      } else {
        epart[bid] = tot;
        __threadfence();
        s_last = atomicAdd(&ecount[eb.mol], 1) == eb.n_chunks - 1;
        if (s_last) {
          __threadfence();
          double sum = 0.0;
          for (int q = 0; q < eb.n_chunks; ++q) sum += __ldcg(&epart[eb.first + q]);
          energy[eb.mol] = escale * sum;
          ecount[eb.mol] = 0;
        }
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// launch wrappers
// ------------------------------------------------------------------------------------------------
static NbrArgs nbr_args(nnp_handle* h, const float* d_pos, int pos_stride, const int* d_atom_index) {
  NbrArgs a;
  a.pos = d_pos; a.atom_index = d_atom_index; a.species = h->d_species; a.mol_id = h->d_mol_id; a.mol_off = h->d_mol_off;
  a.mol_range = reinterpret_cast<const int2*>(h->d_mol_range);
  a.status = h->d_status; a.pos_stride = pos_stride; a.length_scale = h->aev.length_scale;
  return a;
}

void launch_neighbors(nnp_handle* h, const float* d_pos, int pos_stride, const int* d_atom_index, cudaStream_t s) {
  if (h->N == 0 || h->fuse_nbr) return;  // fused: the AEV forward kernel builds the rows
  if (h->use_cells) {
    launch_neighbors_cells(h, d_pos, pos_stride, d_atom_index, s);
    return;
  }
  const int blocks = (h->N + 3) / 4;
  nbr_allpairs_kernel<<<blocks, 128, 0, s>>>(nbr_args(h, d_pos, pos_stride, d_atom_index), h->N, h->aev.rc_r2,
                                             h->aev.rc_a2, h->capR, h->capA, h->d_pos4, h->d_nbr_r, h->d_nbr_a,
                                             h->d_cnt_r, h->d_cnt_a);
}

static bool aev_small_shape(const nnp_handle* h) { return h->aev.n_shf_z <= 4 && h->aev.n_shf_a <= 8; }
// threads per centre CTA: at large N twice as many (smaller) CTAs per SM hide the barrier phases of a centre better
// (configs[2]: forward 237 -> 215 us, backward 192 -> 167 us); at ligand sizes the wider CTA is 2 us faster
// -- in the backward kernel only while shared memory still lets ~10 of the smaller CTAs share an SM (configs[4]
// backward: 33 KB per CTA, 6 per SM either way, where the wider CTA wins; measured both ways)
static int aev_block_threads(const nnp_handle* h, bool backward) {
  if (h->N < 2048) return AEV_THREADS;
  if (!backward) return 128;
  int th, ch;
  aev_bwd_shape(h, &th, &ch);
  return th;
}

void launch_aev_forward(nnp_handle* h, const float* d_pos, int pos_stride, const int* d_atom_index, cudaStream_t s) {
  if (h->N == 0) return;
  const int blocks = h->N;
  const size_t smem0 = aev_smem_bytes(h, false);
  const size_t smem = smem0 + (h->fuse_nbr ? 512 * sizeof(float4) : 0);  // + the molecule's positions (<= 512 atoms)
  const int mp_off4 = (int)(smem0 / sizeof(float4));
  const NbrArgs nb = nbr_args(h, d_pos, pos_stride, d_atom_index);
  const int fused = h->fuse_nbr ? 1 : 0;
  const bool pdl = h->pdl_now && !fused;  // fused: first kernel of the step, must not overtake the previous step
  if (aev_small_shape(h))
    launch_kernel(pdl, aev_forward_kernel<4, 8>, dim3(blocks), dim3(aev_block_threads(h, false)), smem, s, (const float4*)h->d_pos4,
                  (const int*)h->d_nbr_r, (const int*)h->d_nbr_a, (const int*)h->d_cnt_r, (const int*)h->d_cnt_a,
                  (const int*)h->d_sortpos, h->N, h->aev, h->capR, h->capA, trip_chunk(h, false), h->d_aev, h->d_aev_lo, nb, fused,
                  mp_off4, h->d_pos4, h->d_nbr_r, h->d_nbr_a, h->d_cnt_r, h->d_cnt_a);
  else
    launch_kernel(pdl, aev_forward_kernel<NNP_MAX_SHF_Z, NNP_MAX_SHF_A>, dim3(blocks), dim3(aev_block_threads(h, false)), smem, s,
                  (const float4*)h->d_pos4, (const int*)h->d_nbr_r, (const int*)h->d_nbr_a, (const int*)h->d_cnt_r,
                  (const int*)h->d_cnt_a, (const int*)h->d_sortpos, h->N, h->aev, h->capR, h->capA,
                  trip_chunk(h, false), h->d_aev, h->d_aev_lo, nb, fused, mp_off4, h->d_pos4, h->d_nbr_r, h->d_nbr_a, h->d_cnt_r,
                  h->d_cnt_a);
}

template <int NZ, int NA, bool MULTI>
static void launch_aev_backward_t(nnp_handle* h, cudaStream_t s) {
  launch_kernel(h->pdl_now, aev_backward_kernel<NZ, NA, MULTI>, dim3(h->N), dim3(aev_block_threads(h, true)), aev_smem_bytes(h, true), s,
                (const float4*)h->d_pos4, (const int*)h->d_nbr_r, (const int*)h->d_nbr_a, (const int*)h->d_cnt_r,
                (const int*)h->d_cnt_a, (const int*)h->d_sortpos, h->N, h->aev, h->capR, h->capA, trip_chunk(h, true),
                (const float*)h->d_daev, h->n_parts, (size_t)h->N * h->n_feat, h->aev_live_boxes, h->d_facc);
}

void launch_aev_backward(nnp_handle* h, cudaStream_t s) {
  if (h->N == 0) return;
  const bool multi = h->n_parts > 1;
  if (aev_small_shape(h)) {
    if (multi) launch_aev_backward_t<4, 8, true>(h, s);
    else launch_aev_backward_t<4, 8, false>(h, s);
  } else {
    if (multi) launch_aev_backward_t<NNP_MAX_SHF_Z, NNP_MAX_SHF_A, true>(h, s);
    else launch_aev_backward_t<NNP_MAX_SHF_Z, NNP_MAX_SHF_A, false>(h, s);
  }
}

void launch_finish(nnp_handle* h, const int* d_atom_index, double* d_energy, void* d_force, int force_stride, int fixed,
                   cudaStream_t s) {
  if (h->N == 0) return;
  const int nfb = (h->N + FIN_THREADS - 1) / FIN_THREADS;
  const int neb = h->n_eblocks;
  const float fscale = (float)(h->energy_scale * h->length_scale);
  launch_kernel(h->pdl_now, finish_kernel, dim3(nfb + neb), dim3(FIN_THREADS), 0, s, h->d_facc, h->N, d_atom_index, d_force,
                force_stride, fixed, fscale, nfb, h->d_eatom, h->d_sortpos, h->d_species,
                h->d_mol_off, h->n_mol, h->M, h->d_self_energy, h->energy_scale, d_energy,
                (const EnergyBlock*)h->d_eblocks, h->n_eblocks, h->d_epart, h->d_ecount);
}

int aev_set_smem_attributes(nnp_handle* h) {
  const int fb = (int)(aev_smem_bytes(h, false) + 512 * sizeof(float4)), bb = (int)aev_smem_bytes(h, true);
  cudaError_t e[6];
  e[0] = cudaFuncSetAttribute(aev_forward_kernel<4, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, fb);
  e[1] = cudaFuncSetAttribute(aev_forward_kernel<NNP_MAX_SHF_Z, NNP_MAX_SHF_A>,
                              cudaFuncAttributeMaxDynamicSharedMemorySize, fb);
  e[2] = cudaFuncSetAttribute(aev_backward_kernel<4, 8, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bb);
  e[3] = cudaFuncSetAttribute(aev_backward_kernel<NNP_MAX_SHF_Z, NNP_MAX_SHF_A, false>,
                              cudaFuncAttributeMaxDynamicSharedMemorySize, bb);
  e[4] = cudaFuncSetAttribute(aev_backward_kernel<4, 8, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bb);
  e[5] = cudaFuncSetAttribute(aev_backward_kernel<NNP_MAX_SHF_Z, NNP_MAX_SHF_A, true>,
                              cudaFuncAttributeMaxDynamicSharedMemorySize, bb);
  for (cudaError_t x : e)
    if (x != cudaSuccess) return -1;
  return 0;
}

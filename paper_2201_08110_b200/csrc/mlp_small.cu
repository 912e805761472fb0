// Ligand-size MLP engine (A4 forward, A5 per-atom energies, A6 input-gradient backward), FP32 FFMA.
//
// Mathematics: DESIGN.md O5/O7.  Regime: every element group of the molecule has at most a few dozen
// atoms (BASELINE.json configs[0,1]: 12 and 50 atoms), so each layer is a set of very skinny GEMMs whose
// cost is STREAMING THE WEIGHTS once (43 MB for layer 1 of the 8-model ensemble) -- tensor-core tiles of
// 128 rows would be almost empty and their TMA -> MMA -> TMEM -> register chain only adds latency.  So
// this engine is two weight-streaming kernels on the CUDA cores:
//
//   small_fwd_kernel   out[a][r] = CELU(b[r] + sum_k W[r][k] X[a][k])
//       the item's activations X (<= 32 atoms x K) sit in shared memory; a warp owns two weight rows at
//       a time, lanes split the contraction (coalesced 128-bit loads of W, 16 loads in flight per lane; X
//       rows arrive by 1-D bulk async copies on an mbarrier while those loads are in flight),
//       partial sums are tree-reduced with shuffles; every weight is read exactly once per item.
//   small_bwd_kernel   out[a][n] = epi(sum_o D[a][o] W[o][n])
//       lanes own 4 consecutive input columns (rows of the SAME row-major weights: the backward pass re-reads
//       what the forward pass left in L2); the whole 128-column weight chunk of the item is put in flight at
//       once as bulk async copies into shared memory (4 mbarrier groups, compute starts when the first
//       lands); warps split atoms and/or output rows; the delta tile sits in shared memory; a fixed-order cross-warp sum in shared memory finishes the row split.
//       The first backward launch forms delta_L-1 = w_L (.) CELU'(h_L-1) on the fly and also produces the
//       per-atom energies e = b_L + w_L . h_L-1 (FP64), so the separate last-layer launch disappears.
//
// Grids are plain (one CTA per item, heavy items first) so the hardware block scheduler balances the
// very uneven elements (23 H atoms vs 1 Cl atom in configs[1]).  Summation orders are fixed =>
// bit-identical reruns.
#include <cuda.h>
#include <string.h>

#include <algorithm>

#include "nnp_internal.h"

namespace {

constexpr int SM_THREADS = 256;
constexpr int SM_WARPS = SM_THREADS / 32;
constexpr int BWD_GROUPS = 4;  // weight-row groups of the backward kernel, one mbarrier each

__device__ __forceinline__ float celu_s(float x, float alpha, float inv_alpha) {
  return x > 0.0f ? x : alpha * expm1f(x * inv_alpha);
}
// CELU'(x) from h = CELU(x):  x > 0 -> 1;  x <= 0 -> exp(x/alpha) = h/alpha + 1
__device__ __forceinline__ float dcelu_s(float h, float inv_alpha) { return h > 0.0f ? 1.0f : fmaf(h, inv_alpha, 1.0f); }

__device__ __forceinline__ float4 ldg_stream(const float4* p) {
  float4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
               : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
               : "l"(p));
  return v;
}

__device__ __forceinline__ float dot4(const float4 w, const float4 x, float s) {
  s = fmaf(w.x, x.x, s);
  s = fmaf(w.y, x.y, s);
  s = fmaf(w.z, x.z, s);
  return fmaf(w.w, x.w, s);
}

// ---- mbarrier + 1-D bulk async copy (global -> shared), the staging path of both kernels
__device__ __forceinline__ uint32_t s_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void sbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(s_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void sbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(s_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void sbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(s_u32(bar)) : "memory");
}
__device__ __forceinline__ void sbar_wait(uint64_t* bar, uint32_t parity) {
  const uint32_t addr = s_u32(bar);
  uint32_t done;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(addr), "r"(parity)
        : "memory");
  } while (!done);
}
// bytes % 16 == 0, both addresses 16-byte aligned
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(s_u32(dst)), "l"(src), "r"(bytes), "r"(s_u32(bar))
               : "memory");
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// forward
// ------------------------------------------------------------------------------------------------
template <int NJ>
__global__ void __launch_bounds__(SM_THREADS, 2) small_fwd_kernel(const SmallFwdItem* __restrict__ items) {
  extern __shared__ __align__(16) float smem_f[];
  __shared__ __align__(8) uint64_t xbar;
  const SmallFwdItem it = items[blockIdx.x];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int K4 = it.K >> 2;
  float4* xs = reinterpret_cast<float4*>(smem_f);  // [n_atoms][K4]

  // the first row pair of this warp: issue the weight loads before staging X so both latencies overlap
  float4 w0[NJ], w1[NJ];
  auto load_rows = [&](int r) {
    const float4* p0 = reinterpret_cast<const float4*>(it.W + (size_t)r * it.K);
    const float4* p1 = reinterpret_cast<const float4*>(it.W + (size_t)(r + 1) * it.K);
#pragma unroll
    for (int j = 0; j < NJ; ++j) {
      const int k4 = lane + 32 * j;
      if (k4 < K4) {
        w0[j] = ldg_stream(p0 + k4);
        w1[j] = ldg_stream(p1 + k4);
      } else {
        w0[j] = make_float4(0.f, 0.f, 0.f, 0.f);
        w1[j] = make_float4(0.f, 0.f, 0.f, 0.f);
      }
    }
  };
  int r = 2 * warp;
  pdl_trigger();
  if (r < it.n_rows) load_rows(r);  // weights: constant data, in flight before the producer of X has finished
  // X rows (contiguous K floats per atom) arrive by bulk async copies, all in flight at once
  if (threadIdx.x == 0) {
    sbar_init(&xbar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    sbar_expect_tx(&xbar, (uint32_t)(it.n_atoms * it.K * 4));
  }
  __syncthreads();
  pdl_wait();
  if (threadIdx.x < it.n_atoms)
    bulk_g2s(smem_f + (size_t)threadIdx.x * it.K, it.X + (size_t)threadIdx.x * it.ldx, (uint32_t)(it.K * 4), &xbar);
  sbar_wait(&xbar, 0);

  for (; r < it.n_rows; r += 2 * SM_WARPS) {
    float keep0 = 0.0f, keep1 = 0.0f;
    for (int a = 0; a < it.n_atoms; a += 2) {
      const int a1 = min(a + 1, it.n_atoms - 1);
      const float4* xa = xs + a * K4;
      const float4* xb = xs + a1 * K4;
      float s00 = 0.f, s01 = 0.f, s10 = 0.f, s11 = 0.f;
#pragma unroll
      for (int j = 0; j < NJ; ++j) {
        const int k4 = lane + 32 * j;
        if (k4 < K4) {
          const float4 x0 = xa[k4], x1 = xb[k4];
          s00 = dot4(w0[j], x0, s00);
          s01 = dot4(w0[j], x1, s01);
          s10 = dot4(w1[j], x0, s10);
          s11 = dot4(w1[j], x1, s11);
        }
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        s00 += __shfl_xor_sync(0xffffffffu, s00, o);
        s01 += __shfl_xor_sync(0xffffffffu, s01, o);
        s10 += __shfl_xor_sync(0xffffffffu, s10, o);
        s11 += __shfl_xor_sync(0xffffffffu, s11, o);
      }
      if (lane == a) { keep0 = s00; keep1 = s10; }
      if (lane == a + 1) { keep0 = s01; keep1 = s11; }
    }
    if (lane < it.n_atoms) {
      const float b0 = it.bias ? it.bias[r] : 0.0f, b1 = it.bias ? it.bias[r + 1] : 0.0f;
      float2 v;
      v.x = celu_s(keep0 + b0, it.alpha, it.inv_alpha);
      v.y = celu_s(keep1 + b1, it.alpha, it.inv_alpha);
      *reinterpret_cast<float2*>(it.out + (size_t)lane * it.ldc + r) = v;
    }
    if (r + 2 * SM_WARPS < it.n_rows) load_rows(r + 2 * SM_WARPS);  // items normally hold one pair per warp
  }
}

// ------------------------------------------------------------------------------------------------
// backward
// ------------------------------------------------------------------------------------------------
// shared memory: ds [n_pad][n_out] | ws [n_out][128] | red [(n_slices-1)][n_pad][32] float4
template <int AW>
__device__ __forceinline__ void small_bwd_body(const SmallBwdItem& it, float* smem_f, uint64_t* bars) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int G = it.G, n_slices = SM_WARPS / G;
  const int n_pad = G * AW;  // atoms incl. padding
  float* ds = smem_f;
  float* ws = ds + (size_t)n_pad * it.n_out;
  float4* red = reinterpret_cast<float4*>(ws + (size_t)it.n_out * 128);
  const int rpg = (((it.n_out + BWD_GROUPS - 1) / BWD_GROUPS) + 3) & ~3;  // weight rows per barrier group
  uint64_t* dbar = bars + BWD_GROUPS;

  // ---- every weight row of the chunk and the delta rows: bulk async copies, all in flight at once
  if (threadIdx.x == 0) {
    for (int g = 0; g < BWD_GROUPS; ++g) {
      const int rows = max(0, min(it.n_out, (g + 1) * rpg) - g * rpg);
      sbar_init(&bars[g], 1);
      if (rows) sbar_expect_tx(&bars[g], (uint32_t)(rows * it.n_cols * 4));
    }
    sbar_init(dbar, 1);
    if (!it.w_last) sbar_expect_tx(dbar, (uint32_t)(it.n_atoms * it.n_out * 4));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  pdl_trigger();
  for (int o = threadIdx.x; o < it.n_out; o += SM_THREADS)
    bulk_g2s(ws + (size_t)o * 128, it.W + (size_t)o * it.ldw, (uint32_t)(it.n_cols * 4), &bars[o / rpg]);
  pdl_wait();  // delta / activations come from the previous kernel
  if (!it.w_last) {
    if (threadIdx.x < it.n_atoms)
      bulk_g2s(ds + (size_t)threadIdx.x * it.n_out, it.D + (size_t)threadIdx.x * it.ldd, (uint32_t)(it.n_out * 4), dbar);
    for (int idx = it.n_atoms * it.n_out + threadIdx.x; idx < n_pad * it.n_out; idx += SM_THREADS) ds[idx] = 0.0f;
  } else {
    // first backward layer: delta = w_L (.) CELU'(h), and the per-atom energies e = b_L + w_L . h (FP64)
    const int no4 = it.n_out >> 2;
    const float4* wl4 = reinterpret_cast<const float4*>(it.w_last);
#pragma unroll 4
    for (int idx = threadIdx.x; idx < n_pad * no4; idx += SM_THREADS) {
      const int a = idx / no4, o4 = idx - a * no4;
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (a < it.n_atoms) {
        const float4 h = __ldg(reinterpret_cast<const float4*>(it.D + (size_t)a * it.ldd) + o4);
        const float4 w = __ldg(wl4 + o4);
        v.x = w.x * dcelu_s(h.x, it.inv_alpha); v.y = w.y * dcelu_s(h.y, it.inv_alpha);
        v.z = w.z * dcelu_s(h.z, it.inv_alpha); v.w = w.w * dcelu_s(h.w, it.inv_alpha);
      }
      reinterpret_cast<float4*>(ds)[idx] = v;
    }
    if (it.e_out) {
      for (int a = warp; a < it.n_atoms; a += SM_WARPS) {
        double acc = 0.0;
        for (int o = lane; o < it.n_out; o += 32)
          acc += (double)__ldg(it.w_last + o) * (double)__ldg(it.D + (size_t)a * it.ldd + o);
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
        if (lane == 0) it.e_out[(size_t)a * it.lde] = acc + (double)it.b_last;
      }
    }
  }
  __syncthreads();                     // generic-proxy writes of ds (zero fill / delta) visible
  if (!it.w_last) sbar_wait(dbar, 0);  // bulk-copied delta rows landed

  const int g = warp % G, s = warp / G;
  const bool col_ok = 4 * lane < it.n_cols;
  float4 acc[AW];
#pragma unroll
  for (int t = 0; t < AW; ++t) acc[t] = make_float4(0.f, 0.f, 0.f, 0.f);
  if (s < n_slices) {
    const int rps = (((it.n_out + n_slices - 1) / n_slices) + 3) & ~3;
    const int o0 = s * rps, o1 = min(it.n_out, o0 + rps);
    const float4* wp = reinterpret_cast<const float4*>(ws) + lane;
    const float* dbase = ds + (size_t)(g * AW) * it.n_out;
    int ready = -1;  // last weight-row group known to have landed
    for (int o = o0; o < o1; o += 4) {
      const int grp = (o + 3) / rpg;  // rpg % 4 == 0: the four rows lie in one group
      if (grp > ready) {
        for (int q = ready + 1; q <= grp; ++q) sbar_wait(&bars[q], 0);
        ready = grp;
      }
      if (col_ok) {
        float4 w[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) w[i] = wp[(size_t)(o + i) * 32];
#pragma unroll
        for (int t = 0; t < AW; ++t) {
          const float4 d = *reinterpret_cast<const float4*>(dbase + (size_t)t * it.n_out + o);
          acc[t].x = fmaf(d.x, w[0].x, acc[t].x); acc[t].y = fmaf(d.x, w[0].y, acc[t].y);
          acc[t].z = fmaf(d.x, w[0].z, acc[t].z); acc[t].w = fmaf(d.x, w[0].w, acc[t].w);
          acc[t].x = fmaf(d.y, w[1].x, acc[t].x); acc[t].y = fmaf(d.y, w[1].y, acc[t].y);
          acc[t].z = fmaf(d.y, w[1].z, acc[t].z); acc[t].w = fmaf(d.y, w[1].w, acc[t].w);
          acc[t].x = fmaf(d.z, w[2].x, acc[t].x); acc[t].y = fmaf(d.z, w[2].y, acc[t].y);
          acc[t].z = fmaf(d.z, w[2].z, acc[t].z); acc[t].w = fmaf(d.z, w[2].w, acc[t].w);
          acc[t].x = fmaf(d.w, w[3].x, acc[t].x); acc[t].y = fmaf(d.w, w[3].y, acc[t].y);
          acc[t].z = fmaf(d.w, w[3].z, acc[t].z); acc[t].w = fmaf(d.w, w[3].w, acc[t].w);
        }
      }
    }
  }
  if (n_slices > 1) {  // fixed-order sum over the row slices
    if (s > 0 && s < n_slices) {
#pragma unroll
      for (int t = 0; t < AW; ++t) red[((size_t)(s - 1) * n_pad + g * AW + t) * 32 + lane] = acc[t];
    }
    __syncthreads();
    if (s == 0) {
      for (int q = 1; q < n_slices; ++q) {
#pragma unroll
        for (int t = 0; t < AW; ++t) {
          const float4 v = red[((size_t)(q - 1) * n_pad + g * AW + t) * 32 + lane];
          acc[t].x += v.x; acc[t].y += v.y; acc[t].z += v.z; acc[t].w += v.w;
        }
      }
    }
  }
  if (s == 0 && col_ok) {
#pragma unroll
    for (int t = 0; t < AW; ++t) {
      const int a = g * AW + t;
      if (a >= it.n_atoms) continue;
      float4 v = acc[t];
      if (it.epi == EPI_MUL_DCELU) {
        const float4 h = *reinterpret_cast<const float4*>(it.aux + (size_t)a * it.ldaux + 4 * lane);
        v.x *= dcelu_s(h.x, it.inv_alpha); v.y *= dcelu_s(h.y, it.inv_alpha);
        v.z *= dcelu_s(h.z, it.inv_alpha); v.w *= dcelu_s(h.w, it.inv_alpha);
      } else {
        v.x *= it.scale; v.y *= it.scale; v.z *= it.scale; v.w *= it.scale;
      }
      *reinterpret_cast<float4*>(it.out + (size_t)a * it.ldo + 4 * lane) = v;
    }
  }
}

__global__ void __launch_bounds__(SM_THREADS) small_bwd_kernel(const SmallBwdItem* __restrict__ items) {
  extern __shared__ __align__(16) float smem_f[];
  __shared__ __align__(8) uint64_t bars[BWD_GROUPS + 1];
  const SmallBwdItem it = items[blockIdx.x];
  switch (it.AW) {  // atoms per warp: CTA-uniform
    case 1: small_bwd_body<1>(it, smem_f, bars); break;
    case 2: small_bwd_body<2>(it, smem_f, bars); break;
    case 3: small_bwd_body<3>(it, smem_f, bars); break;
    default: small_bwd_body<4>(it, smem_f, bars); break;
  }
}

// ------------------------------------------------------------------------------------------------
// backward through layer 1 (the 43 MB layer): out[a][n] = scale * sum_o D[a][o] W[o][n]
// ------------------------------------------------------------------------------------------------
// Every weight of the item's [n_out][128-column] chunk is read from shared memory exactly ONCE and applied to
// all atoms of the item from registers: a warp owns a slice of the rows o, a lane owns 4 consecutive columns and
// NA x 4 accumulators, held as packed pairs of columns and updated with FFMA2 (fma.rn.f32x2: two columns per
// instruction; the weight pairs come straight out of the 128-bit shared-memory load, the delta operand is a
// broadcast pair); one broadcast 128-bit load of the delta tile serves four rows of one atom.  The 8 row slices are summed in a fixed order through shared memory (the
// weight buffer is reused).  Weight rows arrive as bulk async copies, one mbarrier per row slice, all issued
// before griddepcontrol.wait.
constexpr int B1_SLICES = SM_WARPS;

__device__ __forceinline__ unsigned long long ffma2(unsigned long long a, unsigned long long b, unsigned long long c) {
  unsigned long long d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}
__device__ __forceinline__ unsigned long long pack2(float x, float y) {
  unsigned long long d;
  asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(x), "f"(y));
  return d;
}
__device__ __forceinline__ float2 unpack2(unsigned long long v) {
  float2 r;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v));
  return r;
}

struct Bwd1pParams {
  CUtensorMap wmap[NNP_MAX_SPECIES];  // layer-1 weight block of an element: [M * H1 rows][n_feat columns], box 32 x 128
  const SmallBwdItem* items;  // grouped by CTA: CTA b owns items [cta_off[b], cta_off[b + 1])
  const int* cta_off;
  int n_items, n_stages;
  int use_tma;  // one-CTA-per-item kernel: weight chunk by 2-D tensor copies (else one bulk copy per row)
  int n_single;      // one-CTA-per-item kernel: CTAs [0, n_single) own one item, the rest a pair of light items
  int pair_floats;   // shared-memory floats of one half of a pair CTA
};

__device__ __forceinline__ void p1_tma_2d(void* dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
      ::"r"(s_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(s_u32(bar))
      : "memory");
}

// NW = warps that work on the item: 8 (the whole CTA) or 4 (two light items share a CTA, one per half: their time is
// start-up and weight-fetch latency, not arithmetic, so two per SM nearly halves their cost); `tid` is the thread's
// index within its group, `bar_id` the group's named barrier.
template <int NW>
__device__ __forceinline__ void b1_sync(int bar_id) {
  if (NW == SM_WARPS) __syncthreads();
  else asm volatile("bar.sync %0, %1;" ::"r"(bar_id), "n"(NW * 32) : "memory");
}

template <int NA, int NW>
__device__ __forceinline__ void small_bwd1_body(const SmallBwdItem& it, float* smem_raw, uint64_t* bars,
                                                const CUtensorMap* wmap, int tid, int bar_id) {
  constexpr int NT = NW * 32;
  const int warp = tid >> 5, lane = tid & 31;
  const int rps = (((it.n_out + NW - 1) / NW) + 3) & ~3;  // rows per slice, a multiple of 4
  const int n_tiles = (it.n_out + 31) >> 5;               // 32-row tiles of the tensor copies
  const bool tma = wmap != nullptr && n_tiles <= B1_SLICES;
  float* smem_f = smem_raw + (((128u - (s_u32(smem_raw) & 127u)) & 127u) >> 2);  // 128-byte aligned (tensor copies)
  const size_t ws_floats = max((size_t)n_tiles * 32 * 128, (size_t)NW * NA * 128);
  float* ws = smem_f;               // [n_out][128]; later red [NW][NA][128]
  float* ds = smem_f + ws_floats;   // [NA][n_out]
  uint64_t* dbar = bars + B1_SLICES;
  if (tid == 0) {
    for (int g = 0; g < B1_SLICES; ++g) {
      sbar_init(&bars[g], 1);
      if (tma) {
        if (g < n_tiles) sbar_expect_tx(&bars[g], 32u * 128u * 4u);  // whole box: columns beyond the matrix arrive as zeros
      } else {
        const int rows = max(0, min(it.n_out, (g + 1) * rps) - g * rps);
        if (rows) sbar_expect_tx(&bars[g], (uint32_t)(rows * it.n_cols * 4));
      }
    }
    sbar_init(dbar, 1);
    sbar_expect_tx(dbar, (uint32_t)(it.n_atoms * it.n_out * 4));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  b1_sync<NW>(bar_id);
  pdl_trigger();
  if (tma) {  // one 2-D tensor copy per 32-row tile (512-byte row segments as separate bulk copies are issue-bound)
    if (tid < n_tiles) p1_tma_2d(ws + (size_t)tid * 32 * 128, wmap, it.t_col0, it.t_row0 + 32 * tid, &bars[tid]);
  } else {
    for (int o = tid; o < it.n_out; o += NT)
      bulk_g2s(ws + (size_t)o * 128, it.W + (size_t)o * it.ldw, (uint32_t)(it.n_cols * 4), &bars[o / rps]);
  }
  for (int idx = it.n_atoms * it.n_out + tid; idx < NA * it.n_out; idx += NT) ds[idx] = 0.0f;
  pdl_wait();  // delta comes from the previous kernel
  if (tid < it.n_atoms)
    bulk_g2s(ds + (size_t)tid * it.n_out, it.D + (size_t)tid * it.ldd, (uint32_t)(it.n_out * 4), dbar);
  b1_sync<NW>(bar_id);  // zero rows of the padding atoms visible
  sbar_wait(dbar, 0);

  // acc[a][0] = columns (4 lane, 4 lane + 1), acc[a][1] = columns (4 lane + 2, 4 lane + 3) of atom a
  unsigned long long acc[NA][2];
#pragma unroll
  for (int a = 0; a < NA; ++a) acc[a][0] = acc[a][1] = 0ull;
  const bool col_ok = 4 * lane < it.n_cols;
  const int o0 = warp * rps, o1 = min(it.n_out, o0 + rps);
  if (o0 < o1) {
    if (tma) {
      for (int t = o0 >> 5; t <= (o1 - 1) >> 5; ++t) sbar_wait(&bars[t], 0);
    } else {
      sbar_wait(&bars[warp], 0);
    }
  }
  if (col_ok) {
    const float4* wp = reinterpret_cast<const float4*>(ws) + lane;
    for (int o = o0; o < o1; o += 4) {
      unsigned long long wlo[4], whi[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const float4 w = wp[(size_t)(o + i) * 32];
        wlo[i] = pack2(w.x, w.y);
        whi[i] = pack2(w.z, w.w);
      }
#pragma unroll
      for (int a = 0; a < NA; ++a) {
        const float4 d = *reinterpret_cast<const float4*>(ds + (size_t)a * it.n_out + o);
        const unsigned long long d0 = pack2(d.x, d.x), d1 = pack2(d.y, d.y), d2 = pack2(d.z, d.z), d3 = pack2(d.w, d.w);
        acc[a][0] = ffma2(d0, wlo[0], acc[a][0]); acc[a][1] = ffma2(d0, whi[0], acc[a][1]);
        acc[a][0] = ffma2(d1, wlo[1], acc[a][0]); acc[a][1] = ffma2(d1, whi[1], acc[a][1]);
        acc[a][0] = ffma2(d2, wlo[2], acc[a][0]); acc[a][1] = ffma2(d2, whi[2], acc[a][1]);
        acc[a][0] = ffma2(d3, wlo[3], acc[a][0]); acc[a][1] = ffma2(d3, whi[3], acc[a][1]);
      }
    }
  }
  b1_sync<NW>(bar_id);  // every warp is done with the weight buffer: reuse it for the slice sums
  float4* red = reinterpret_cast<float4*>(ws);
  if (col_ok) {
#pragma unroll
    for (int a = 0; a < NA; ++a) {
      const float2 lo = unpack2(acc[a][0]), hi = unpack2(acc[a][1]);
      red[((size_t)warp * NA + a) * 32 + lane] = make_float4(lo.x, lo.y, hi.x, hi.y);
    }
  }
  b1_sync<NW>(bar_id);
  for (int idx = tid; idx < it.n_atoms * 32; idx += NT) {
    const int a = idx >> 5, l = idx & 31;
    if (4 * l >= it.n_cols) continue;
    float4 v = red[(size_t)a * 32 + l];
#pragma unroll
    for (int s = 1; s < NW; ++s) {  // fixed order
      const float4 u = red[((size_t)s * NA + a) * 32 + l];
      v.x += u.x; v.y += u.y; v.z += u.z; v.w += u.w;
    }
    v.x *= it.scale; v.y *= it.scale; v.z *= it.scale; v.w *= it.scale;
    *reinterpret_cast<float4*>(it.out + (size_t)a * it.ldo + 4 * l) = v;
  }
}

__global__ void __launch_bounds__(SM_THREADS, 1) small_bwd1_kernel(const __grid_constant__ Bwd1pParams P) {
  extern __shared__ __align__(16) float smem_f[];
  __shared__ __align__(8) uint64_t bars[2][B1_SLICES + 1];
  if ((int)blockIdx.x >= P.n_single) {  // two light items (<= 4 atoms), one per half of the CTA
    const int half = threadIdx.x >> 7;
    const SmallBwdItem it = P.items[P.n_single + 2 * ((int)blockIdx.x - P.n_single) + half];
    small_bwd1_body<4, SM_WARPS / 2>(it, smem_f + (size_t)half * P.pair_floats, bars[half],
                                     P.use_tma ? &P.wmap[it.tmap] : nullptr, threadIdx.x & 127, 1 + half);
    return;
  }
  const SmallBwdItem it = P.items[blockIdx.x];
  const CUtensorMap* wmap = P.use_tma ? &P.wmap[it.tmap] : nullptr;
  if (it.n_atoms <= 4) small_bwd1_body<4, SM_WARPS>(it, smem_f, bars[0], wmap, threadIdx.x, 0);
  else if (it.n_atoms <= 8) small_bwd1_body<8, SM_WARPS>(it, smem_f, bars[0], wmap, threadIdx.x, 0);
  else if (it.n_atoms <= 16) small_bwd1_body<16, SM_WARPS>(it, smem_f, bars[0], wmap, threadIdx.x, 0);
  else small_bwd1_body<24, SM_WARPS>(it, smem_f, bars[0], wmap, threadIdx.x, 0);
}

// ------------------------------------------------------------------------------------------------
// forward through layer 1 (the 43 MB layer): out[a][r] = CELU(b[r] + sum_k W[r][k] X[a][k]),  K = 1008
// ------------------------------------------------------------------------------------------------
// Persistent: one CTA per SM-sized share of ONE element's weight rows (the rows of all models of an (element,
// layer 1) block are contiguous).  The element's AEV rows (<= 24 atoms) are staged in shared memory once; a
// producer warp streams the weight rows as 12-row tiles (bulk async copies, one per row, padded pitch) through a
// ring and runs ahead of the 8 consumer warps, starting before griddepcontrol.wait (weights are constant data),
// so the weight fetch is continuous: the launch is bound by HBM when the step starts with a cold L2.
// Consumers: a register-tiled contraction.  A thread owns 3 rows x AG atoms and one of 16 interleaved slices
// of K; per 4-wide k-step it loads 3 weight + AG activation float4 (conflict-free, mostly broadcast) and issues
// 3 x AG x 2 FFMA2 (the two halves of a float4 dot product run as a packed pair).  The 16 slice partials of an
// output are summed in a fixed order: one shuffle (the two slices of a warp), then the 8 warps through shared
// memory; bias + CELU fused.
constexpr int F1_ROWS = 12;               // rows per tile: 4 row groups x 3
constexpr int F1_CONSUMERS = 256;
constexpr int F1_THREADS = F1_CONSUMERS + 32;
constexpr int F1_MAX_STAGES = 6;
constexpr int F1_BIAS_MAX = 1024;              // biases of a CTA's rows staged in shared memory (else read per tile)
static const size_t F1_SMEM = 200 * 1024;

__host__ __device__ __forceinline__ int f1_pitch(int K) { return (K & 7) == 0 ? K + 4 : K; }  // == 4 (mod 8) words
__host__ __device__ __forceinline__ int f1_pad_atoms(int n) { return n <= 4 ? 4 : n <= 8 ? 8 : n <= 16 ? 16 : 24; }
__host__ __device__ __forceinline__ int f1_stages(int n_atoms, int K) {
  const size_t P = (size_t)f1_pitch(K) * 4;
  const int NAT = f1_pad_atoms(n_atoms);
  const size_t fixed = (size_t)NAT * P + (size_t)(F1_CONSUMERS / 32) * F1_ROWS * NAT * 4;
  const long long st = ((long long)F1_SMEM - (long long)fixed) / (long long)(F1_ROWS * P);
  return st > F1_MAX_STAGES ? F1_MAX_STAGES : (int)st;
}
__device__ __forceinline__ void f1_consumer_sync() { asm volatile("bar.sync 1, %0;" ::"n"(F1_CONSUMERS) : "memory"); }
// packed pair of floats <-> 64-bit register (FFMA2 operands)
__device__ __forceinline__ unsigned long long f1_pack(float x, float y) {
  unsigned long long d;
  asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(x), "f"(y));
  return d;
}
__device__ __forceinline__ unsigned long long f1_ffma2(unsigned long long a, unsigned long long b, unsigned long long c) {
  unsigned long long d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}
__device__ __forceinline__ float f1_sum2(unsigned long long v) {
  float x, y;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(x), "=f"(y) : "l"(v));
  return x + y;
}

template <int AG>
__device__ __forceinline__ void small_fwd1_body(const Fwd1Item& it, float* smem_f, uint64_t* full, uint64_t* empty,
                                                uint64_t* xbar, float* bias_s) {
  constexpr int NAT = 4 * AG;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int K4 = it.K >> 2, P = f1_pitch(it.K);
  const int n_stages = f1_stages(it.n_atoms, it.K);
  const int n_tiles = (it.n_rows + F1_ROWS - 1) / F1_ROWS;
  float* Xs = smem_f;                                  // [NAT][P]
  float* Ws = Xs + (size_t)NAT * P;                    // [n_stages][F1_ROWS][P]
  float* red = Ws + (size_t)n_stages * F1_ROWS * P;    // [warps][F1_ROWS][NAT]
  if (threadIdx.x == 0) {
    for (int s = 0; s < n_stages; ++s) {
      sbar_init(&full[s], 1);
      sbar_init(&empty[s], F1_CONSUMERS / 32);
    }
    sbar_init(xbar, 1);
    sbar_expect_tx(xbar, (uint32_t)(it.n_atoms * it.K * 4));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  pdl_trigger();

  if (warp == F1_CONSUMERS / 32) {
    // ------------------------------------------------------------ producer warp: weight tiles, lane r = row r
    uint32_t slot = 0, phase = 0;
    for (int t = 0; t < n_tiles; ++t) {
      const int rows = min(F1_ROWS, it.n_rows - t * F1_ROWS);
      if (lane == 0) {
        sbar_wait(&empty[slot], phase ^ 1u);
        sbar_expect_tx(&full[slot], (uint32_t)(rows * it.K * 4));
      }
      __syncwarp();
      if (lane < rows)
        bulk_g2s(Ws + ((size_t)slot * F1_ROWS + lane) * P, it.W + ((size_t)t * F1_ROWS + lane) * it.K,
                 (uint32_t)(it.K * 4), &full[slot]);
      if (++slot == (uint32_t)n_stages) { slot = 0; phase ^= 1u; }
    }
    pdl_wait();
    return;
  }
  // -------------------------------------------------------------- consumers
  const int tid = threadIdx.x;
  for (int idx = it.n_atoms * P + tid; idx < NAT * P; idx += F1_CONSUMERS) Xs[idx] = 0.0f;  // rows of padding atoms
  // biases of the CTA's rows: staged once (constant data, before the dependency wait) -- a global load per tile in
  // the epilogue was ~1.5 us of exposed DRAM latency per tile when the step starts with a cold L2
  const bool bias_staged = it.bias != nullptr && it.n_rows <= F1_BIAS_MAX;
  if (bias_staged)
    for (int r = tid; r < it.n_rows; r += F1_CONSUMERS) bias_s[r] = __ldg(it.bias + r);
  pdl_wait();  // the AEV rows come from the previous kernel
  if (tid < it.n_atoms) bulk_g2s(Xs + (size_t)tid * P, it.X + (size_t)tid * it.ldx, (uint32_t)(it.K * 4), xbar);
  f1_consumer_sync();
  sbar_wait(xbar, 0);

  // lane = (k-slice pair, atom group, row group); the two slices of a warp are 4 float4 apart, which together with
  // the pitch == 20 (mod 32) words keeps the 8 distinct 16-byte addresses of a weight load on different banks
  const int rg = lane & 3, ag = (lane >> 2) & 3, ks2 = lane >> 4;
  const int slice = (warp & 3) + 8 * (warp >> 2) + 4 * ks2;
  const float4* xs4 = reinterpret_cast<const float4*>(Xs);
  const int P4 = P >> 2;
  uint32_t slot = 0, phase = 0;
  for (int t = 0; t < n_tiles; ++t) {
    sbar_wait(&full[slot], phase);
    const float4* ws4 = reinterpret_cast<const float4*>(Ws + (size_t)slot * F1_ROWS * P);
    unsigned long long acc[3][AG];
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = 0; j < AG; ++j) acc[i][j] = 0ull;
#pragma unroll 2
    for (int k4 = slice; k4 < K4; k4 += F1_CONSUMERS / 16) {
      unsigned long long wlo[3], whi[3];
#pragma unroll
      for (int i = 0; i < 3; ++i) {
        const float4 w = ws4[(rg + 4 * i) * P4 + k4];
        wlo[i] = f1_pack(w.x, w.y);
        whi[i] = f1_pack(w.z, w.w);
      }
#pragma unroll
      for (int j = 0; j < AG; ++j) {
        const float4 x = xs4[(ag + 4 * j) * P4 + k4];
        const unsigned long long xlo = f1_pack(x.x, x.y), xhi = f1_pack(x.z, x.w);
#pragma unroll
        for (int i = 0; i < 3; ++i) {
          acc[i][j] = f1_ffma2(wlo[i], xlo, acc[i][j]);
          acc[i][j] = f1_ffma2(whi[i], xhi, acc[i][j]);
        }
      }
    }
    __syncwarp();
    if (lane == 0) sbar_arrive(&empty[slot]);  // the tile has been read: the producer may refill the stage
    if (++slot == (uint32_t)n_stages) { slot = 0; phase ^= 1u; }
    // slice partials: the warp's two slices by one shuffle, then the warps through shared memory (fixed order)
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = 0; j < AG; ++j) {
        float v = f1_sum2(acc[i][j]);
        v += __shfl_xor_sync(0xffffffffu, v, 16);
        if (ks2 == 0) red[((size_t)warp * F1_ROWS + rg + 4 * i) * NAT + ag + 4 * j] = v;
      }
    f1_consumer_sync();
    const int r0 = t * F1_ROWS;
    for (int idx = tid; idx < F1_ROWS * NAT; idx += F1_CONSUMERS) {
      const int a = idx / F1_ROWS, r = idx - a * F1_ROWS;  // consecutive threads -> consecutive rows (coalesced stores)
      if (a < it.n_atoms && r0 + r < it.n_rows) {
        float v = red[(size_t)r * NAT + a];
#pragma unroll
        for (int w = 1; w < F1_CONSUMERS / 32; ++w) v += red[((size_t)w * F1_ROWS + r) * NAT + a];
        const float b = bias_staged ? bias_s[r0 + r] : (it.bias ? it.bias[r0 + r] : 0.0f);
        it.out[(size_t)a * it.ldc + r0 + r] = celu_s(v + b, it.alpha, it.inv_alpha);
      }
    }
    f1_consumer_sync();  // red is reused by the next tile
  }
}

__global__ void __launch_bounds__(F1_THREADS, 1) small_fwd1_kernel(const Fwd1Item* __restrict__ items) {
  extern __shared__ __align__(16) float smem_f[];
  __shared__ __align__(8) uint64_t full[F1_MAX_STAGES];
  __shared__ __align__(8) uint64_t empty[F1_MAX_STAGES];
  __shared__ __align__(8) uint64_t xbar;
  __shared__ float bias_s[F1_BIAS_MAX];
  const Fwd1Item it = items[blockIdx.x];
  if (it.n_atoms <= 4) small_fwd1_body<1>(it, smem_f, full, empty, &xbar, bias_s);
  else if (it.n_atoms <= 8) small_fwd1_body<2>(it, smem_f, full, empty, &xbar, bias_s);
  else if (it.n_atoms <= 16) small_fwd1_body<4>(it, smem_f, full, empty, &xbar, bias_s);
  else small_fwd1_body<6>(it, smem_f, full, empty, &xbar, bias_s);
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
static const size_t SMALL_SMEM_MAX = 200 * 1024;

template <typename K>
static int set_smem(K kernel, size_t bytes) {
  return cudaFuncSetAttribute((const void*)kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) ==
                 cudaSuccess ? 0 : -1;
}

int small_init() {
  int rc = 0;
  rc |= set_smem(small_fwd_kernel<1>, SMALL_SMEM_MAX);
  rc |= set_smem(small_fwd_kernel<2>, SMALL_SMEM_MAX);
  rc |= set_smem(small_fwd_kernel<4>, SMALL_SMEM_MAX);
  rc |= set_smem(small_fwd_kernel<8>, SMALL_SMEM_MAX);
  rc |= set_smem(small_bwd_kernel, SMALL_SMEM_MAX);
  rc |= set_smem(small_bwd1_kernel, SMALL_SMEM_MAX);
  rc |= set_smem(small_fwd1_kernel, F1_SMEM);
  return rc;
}

void small_bwd_shape(int n_atoms, int* AW, int* G) {
  if (n_atoms <= 4) { *G = 1; *AW = std::max(1, n_atoms); }
  else if (n_atoms <= 8) { *G = 2; *AW = (n_atoms + 1) / 2; }
  else if (n_atoms <= 16) { *G = 4; *AW = (n_atoms + 3) / 4; }
  else { *G = 8; *AW = (n_atoms + 7) / 8; }
}

int small_build_fwd(SmallLaunch& L, std::vector<SmallFwdItem>& items) {
  std::stable_sort(items.begin(), items.end(), [](const SmallFwdItem& a, const SmallFwdItem& b) {
    return (long long)a.n_rows * a.K * (a.n_atoms + 16) > (long long)b.n_rows * b.K * (b.n_atoms + 16);
  });
  L.n_items = (int)items.size();
  L.variant = 1;
  L.smem_bytes = 0;
  for (const auto& it : items) {
    const int nj = (it.K + 127) / 128;
    while (L.variant < nj) L.variant *= 2;
    L.smem_bytes = std::max(L.smem_bytes, (size_t)it.n_atoms * it.K * 4);
  }
  if (L.variant > 8 || L.smem_bytes > SMALL_SMEM_MAX) return -1;
  if (cudaMalloc(&L.d_items, std::max<size_t>(1, items.size()) * sizeof(SmallFwdItem)) != cudaSuccess) return -1;
  if (!items.empty())
    cudaMemcpy(L.d_items, items.data(), items.size() * sizeof(SmallFwdItem), cudaMemcpyHostToDevice);
  return 0;
}

int small_build_bwd(SmallLaunch& L, std::vector<SmallBwdItem>& items) {
  std::stable_sort(items.begin(), items.end(), [](const SmallBwdItem& a, const SmallBwdItem& b) {
    return (long long)a.n_out * a.n_cols * (a.n_atoms + 16) > (long long)b.n_out * b.n_cols * (b.n_atoms + 16);
  });
  L.n_items = (int)items.size();
  L.smem_bytes = 0;
  for (const auto& it : items) {
    if (it.AW < 1 || it.AW > 4) return -1;
    const int n_pad = it.G * it.AW, n_slices = SM_WARPS / it.G;
    const size_t b = (size_t)n_pad * it.n_out * 4 + (size_t)it.n_out * 512 + (size_t)std::max(0, n_slices - 1) * n_pad * 32 * 16;
    L.smem_bytes = std::max(L.smem_bytes, b);
  }
  if (L.smem_bytes > SMALL_SMEM_MAX) return -1;
  if (cudaMalloc(&L.d_items, std::max<size_t>(1, items.size()) * sizeof(SmallBwdItem)) != cudaSuccess) return -1;
  if (!items.empty())
    cudaMemcpy(L.d_items, items.data(), items.size() * sizeof(SmallBwdItem), cudaMemcpyHostToDevice);
  return 0;
}

static int bwd1_pad(int n_atoms) { return n_atoms <= 4 ? 4 : n_atoms <= 8 ? 8 : n_atoms <= 16 ? 16 : 24; }

// layer-1 backward items: n_atoms <= 24, n_cols <= 128, epilogue EPI_SCALE
int small_build_bwd1(SmallLaunch& L, std::vector<SmallBwdItem>& items, const std::vector<TmaOperand>& wops) {
  std::stable_sort(items.begin(), items.end(), [](const SmallBwdItem& a, const SmallBwdItem& b) {
    return (long long)a.n_out * a.n_cols * (a.n_atoms + 4) > (long long)b.n_out * b.n_cols * (b.n_atoms + 4);
  });
  L.n_items = (int)items.size();
  L.variant = 100;
  L.smem_bytes = 0;
  bool maps_ok = !wops.empty() && wops.size() <= NNP_MAX_SPECIES;
  for (const auto& it : items) {
    if (it.n_atoms < 1 || it.n_atoms > 24 || it.n_cols > 128 || it.epi != EPI_SCALE) return -1;
    const int NA = bwd1_pad(it.n_atoms);
    const size_t rows32 = (size_t)((it.n_out + 31) / 32) * 32;  // the tensor copies write whole 32-row tiles
    const size_t b = (std::max(rows32 * 128, (size_t)B1_SLICES * NA * 128) + (size_t)it.n_out * NA) * 4 + 128;
    L.smem_bytes = std::max(L.smem_bytes, b);
    maps_ok = maps_ok && it.tmap >= 0 && it.tmap < (int)wops.size();
  }
  // tensor maps of the elements' layer-1 weight blocks: [rows][cols] f32, box 32 rows x 128 columns, no swizzle
  Bwd1pParams* P = new Bwd1pParams();
  memset(P, 0, sizeof(*P));
  L.params = P;
  if (maps_ok) {
    typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void* fp = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fp, cudaEnableDefault, &qr) != cudaSuccess ||
        qr != cudaDriverEntryPointSuccess || !fp)
      maps_ok = false;
    for (size_t k = 0; k < wops.size() && maps_ok; ++k) {
      cuuint64_t gdim[2] = {(cuuint64_t)wops[k].cols, (cuuint64_t)std::max<long long>(wops[k].rows, 1)};
      cuuint64_t gstr[1] = {(cuuint64_t)wops[k].ld * 4};
      cuuint32_t box[2] = {128, 32};
      cuuint32_t estr[2] = {1, 1};
      if (((EncodeFn)fp)(&P->wmap[k], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, (void*)wops[k].base, gdim, gstr, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        maps_ok = false;
    }
  }
  P->use_tma = maps_ok ? 1 : 0;
  std::vector<int> p1_off(1, 0);
  // one CTA per item, except that light items (<= 4 atoms) go two to a CTA, one per half, when both fit
  int n_single = (int)items.size();
  size_t pair_floats = 0;
  {
    L.grid = (int)items.size();
    {
      auto item_bytes = [](const SmallBwdItem& it) {
        const size_t rows32 = (size_t)((it.n_out + 31) / 32) * 32;
        return (std::max(rows32 * 128, (size_t)(B1_SLICES / 2) * 4 * 128) + (size_t)it.n_out * 4) * 4 + 128;
      };
      size_t half = 0;
      for (const auto& it : items)
        if (it.n_atoms <= 4) half = std::max(half, item_bytes(it));
      half = (half + 127) & ~(size_t)127;
      if (half && 2 * half <= SMALL_SMEM_MAX) {
        auto mid = std::stable_partition(items.begin(), items.end(), [](const SmallBwdItem& it) { return it.n_atoms > 4; });
        int n_light = (int)(items.end() - mid);
        n_light &= ~1;  // an odd one out runs alone
        n_single = (int)items.size() - n_light;
        pair_floats = half / 4;
        if (n_light) L.smem_bytes = std::max(L.smem_bytes, 2 * half);
        L.grid = n_single + n_light / 2;
      }
    }
  }
  P->n_single = n_single;
  P->pair_floats = (int)pair_floats;
  if (L.smem_bytes > SMALL_SMEM_MAX) return -1;
  if (cudaMalloc(&L.d_items, std::max<size_t>(1, items.size()) * sizeof(SmallBwdItem)) != cudaSuccess) return -1;
  if (!items.empty())
    cudaMemcpy(L.d_items, items.data(), items.size() * sizeof(SmallBwdItem), cudaMemcpyHostToDevice);
  int* d_off = nullptr;
  if (cudaMalloc((void**)&d_off, p1_off.size() * sizeof(int)) != cudaSuccess) return -1;
  cudaMemcpy(d_off, p1_off.data(), p1_off.size() * sizeof(int), cudaMemcpyHostToDevice);
  L.d_aux = d_off;
  P->items = reinterpret_cast<const SmallBwdItem*>(L.d_items);
  P->cta_off = d_off;
  P->n_items = L.n_items;
  P->n_stages = L.stages;
  return 0;
}

// persistent layer-1 forward items (one CTA each, heavy first)
int small_build_fwd1(SmallLaunch& L, std::vector<Fwd1Item>& items) {
  std::stable_sort(items.begin(), items.end(), [](const Fwd1Item& a, const Fwd1Item& b) {
    return (long long)a.n_rows * (16 + a.n_atoms) > (long long)b.n_rows * (16 + b.n_atoms);
  });
  L.n_items = (int)items.size();
  L.variant = 101;
  L.smem_bytes = F1_SMEM;
  for (const auto& it : items)
    if (it.n_atoms < 1 || it.n_atoms > 24 || (it.K & 3) || f1_stages(it.n_atoms, it.K) < 2) return -1;
  if (cudaMalloc(&L.d_items, std::max<size_t>(1, items.size()) * sizeof(Fwd1Item)) != cudaSuccess) return -1;
  if (!items.empty()) cudaMemcpy(L.d_items, items.data(), items.size() * sizeof(Fwd1Item), cudaMemcpyHostToDevice);
  return 0;
}
int small_fwd1_tile_rows() { return F1_ROWS; }

void small_launch_fwd(const SmallLaunch& L, cudaStream_t s, bool pdl) {
  if (L.n_items == 0) return;
  if (L.variant == 101) {
    launch_kernel(pdl, small_fwd1_kernel, dim3(L.n_items), dim3(F1_THREADS), L.smem_bytes, s,
                  reinterpret_cast<const Fwd1Item*>(L.d_items));
    return;
  }
  const SmallFwdItem* it = reinterpret_cast<const SmallFwdItem*>(L.d_items);
  const dim3 g(L.n_items), b(SM_THREADS);
  switch (L.variant) {
    case 1: launch_kernel(pdl, small_fwd_kernel<1>, g, b, L.smem_bytes, s, it); break;
    case 2: launch_kernel(pdl, small_fwd_kernel<2>, g, b, L.smem_bytes, s, it); break;
    case 4: launch_kernel(pdl, small_fwd_kernel<4>, g, b, L.smem_bytes, s, it); break;
    default: launch_kernel(pdl, small_fwd_kernel<8>, g, b, L.smem_bytes, s, it); break;
  }
}

void small_launch_bwd(const SmallLaunch& L, cudaStream_t s, bool pdl) {
  if (L.n_items == 0) return;
  if (L.variant == 100) {
    launch_kernel(pdl, small_bwd1_kernel, dim3(L.grid), dim3(SM_THREADS), L.smem_bytes, s,
                  *reinterpret_cast<const Bwd1pParams*>(L.params));
    return;
  }
  launch_kernel(pdl, small_bwd_kernel, dim3(L.n_items), dim3(SM_THREADS), L.smem_bytes, s,
                reinterpret_cast<const SmallBwdItem*>(L.d_items));
}

void small_free_launch(SmallLaunch& L) {
  if (L.d_items) cudaFree(L.d_items);
  L.d_items = nullptr;
  if (L.params) delete reinterpret_cast<Bwd1pParams*>(L.params);
  L.params = nullptr;
  if (L.d_aux) cudaFree(L.d_aux);
  L.d_aux = nullptr;
}

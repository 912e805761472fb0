// tcgen05 (5th-gen tensor core) GEMM engine for the per-element atomic MLPs (A4 forward, A6 backward).
//
// Mathematics: DESIGN.md O5/O7 -- the layer GEMMs  D[f][a] = sum_k W[f][k] X[a][k]  (forward, f = output
// feature, a = atom) and  D[n][a] = sum_o W[o][n] delta[a][o]  (input-gradient backward).
//
// Precision ("3xTF32, no tensor-core accumulation of the main term").  Measured on B200 (DESIGN.md
// section 7): tcgen05 TRUNCATES FP32 inputs to TF32 and TRUNCATES when it adds into the FP32 accumulator,
// so accumulating a long contraction in TMEM is biased towards zero (-6.5e-6 relative at K = 1024) and the
// bias shows up as a coherent energy error.  Therefore
//   * weights  w = hi + lo with hi = trunc_tf32(w) (what the tensor core makes of the raw FP32 box, so the
//     TMA-written box is used as it is) and lo = rna_tf32(w - hi);
//     activations x = hi + lo with hi = rna_tf32(x), lo = x - hi (random sign, so the dropped lo*lo term,
//     <= 2^-21 relative, has no preferred sign);
//   * the hi*hi products (exact: 11 x 11 bits) of every k-step (8 contraction elements) go into a FRESH
//     TMEM slot; the drain warps add the slots in FP32 round-to-nearest registers (two-level for tiles of
//     up to 64 atoms: 8 slots -> partial -> total);
//   * lo*hi + hi*lo go into a second accumulator over the whole contraction (2^-10 of the result, so its
//     truncation is irrelevant).
//
// Structure: persistent CTAs (one per SM), 14 warps:
//   warp 0      TMA producer      cp.async.bulk.tensor boxes [rows][32 floats] -> deep raw ring (full barriers)
//   warp 1      MMA issuer        one thread issues tcgen05.mma kind::tf32 (M = 128, N = 16..128, K = 8)
//   warps 2-5   converters        raw box -> lo parts in a short second ring (conv barriers)
//   warps 6-13  drain + epilogue  tcgen05.ld of finished slot groups, FP32 adds, fused bias+CELU / CELU' /
//                                  scale, coalesced stores (group_full / group_empty barriers)
// The raw ring is what keeps HBM busy in the weight-streaming regime (ligand sizes): up to 8 x 16 KB of
// weights in flight per SM.
// Operand layouts: weights are read in their natural row-major layout in both passes -- forward as a
// K-major operand (128-byte swizzle), backward as an MN-major operand (TF32 MN-major needs the
// "128B swizzle, 32B atom" layout: CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B + UMMA layout type 1).
#include <cuda.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>

#include "nnp_internal.h"

namespace {

constexpr int U_THREADS = 448;
constexpr int U_DRAIN_THREADS = 256;
constexpr int BOXF = 32;                 // floats per box row (128 B)
constexpr int A_BOX_BYTES = 128 * 128;   // weight box: 128 feature rows x 32 contraction floats
constexpr int U_MAX_RAW = 10;            // raw ring depth (upper bound)
constexpr int U_LO_STAGES = 2;           // lo ring depth
constexpr int U_MAX_GROUPS = 8;
constexpr int L1_SLOTS = 8;              // two-level summation: slots per first-level partial sum

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  const uint32_t addr = smem_u32(bar);
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
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(bar))
      : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
               : "memory");
}
// D[tmem] (+)= A[smem desc] * B[smem desc], kind::tf32, FP32 accumulate
__device__ __forceinline__ void mma_tf32(uint32_t d_tmem, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(d_tmem), "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
      : "memory");
}
// shared-memory matrix descriptor: start address, leading / stride byte offsets, sm_100 version bit,
// layout type (2 = 128B swizzle, 1 = 128B swizzle with 32B atoms)
__device__ __forceinline__ uint64_t smem_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo, uint32_t layout) {
  return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)((lbo >> 4) & 0x3FFF) << 16) |
         ((uint64_t)((sbo >> 4) & 0x3FFF) << 32) | (1ull << 46) | ((uint64_t)layout << 61);
}
// round to TF32 (10 explicit mantissa bits), nearest, ties away from zero == cvt.rna.tf32.f32 for finite inputs,
// done on the integer ALU (the conversion instruction runs at a fraction of the ALU rate and paced the converters)
__device__ __forceinline__ float tf32_rna(float x) {
  return __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xFFFFE000u);
}
// weights: hi = trunc_tf32(w) is implicit (the tensor core truncates the raw value); lo = rna(w - hi)
__device__ __forceinline__ float w_lo(float w) {
  return tf32_rna(w - __uint_as_float(__float_as_uint(w) & 0xFFFFE000u));
}
__device__ __forceinline__ float4 w_lo4(const float4 v) { return make_float4(w_lo(v.x), w_lo(v.y), w_lo(v.z), w_lo(v.w)); }
// activations: hi = rna(x), lo = x - hi
__device__ __forceinline__ void x_split4(const float4 v, float4& h, float4& l) {
  h.x = tf32_rna(v.x); h.y = tf32_rna(v.y); h.z = tf32_rna(v.z); h.w = tf32_rna(v.w);
  l.x = v.x - h.x; l.y = v.y - h.y; l.z = v.z - h.z; l.w = v.w - h.w;
}
// CELU with the hardware exponential: alpha (2^(x log2e / alpha) - 1).  Near x = 0 the subtraction leaves an ABSOLUTE
// error of ~2^-24 alpha = 6e-9 on an activation of order 0.1..1 (unbiased), far below the TF32-split error of the
// GEMM that produced x; expm1f costs ~30 instructions per element in an epilogue of 64 elements per thread.
__device__ __forceinline__ float celu_f(float x, float alpha, float inv_alpha) {
  float e;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(x * inv_alpha * 1.4426950408889634f));
  return x > 0.0f ? x : alpha * (e - 1.0f);
}
__device__ __forceinline__ float dcelu_from_h(float h, float inv_alpha) { return h > 0.0f ? 1.0f : fmaf(h, inv_alpha, 1.0f); }

// acc[0..CNT-1] += CNT consecutive TMEM columns of this thread's lane (CNT = 8, 16 or 32)
template <int CNT>
__device__ __forceinline__ void tmem_add(uint32_t taddr, float* acc) {
  uint32_t r[CNT];
  if constexpr (CNT == 8) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n\t"
        "tcgen05.wait::ld.sync.aligned;"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
        : "r"(taddr)
        : "memory");
  } else if constexpr (CNT == 16) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];\n\t"
        "tcgen05.wait::ld.sync.aligned;"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
  } else {
    static_assert(CNT == 32, "column count");
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,"
        "%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];\n\t"
        "tcgen05.wait::ld.sync.aligned;"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
          "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
          "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr)
        : "memory");
  }
#pragma unroll
  for (int j = 0; j < CNT; ++j) acc[j] += __uint_as_float(r[j]);
}
// CT columns starting at taddr (CT = 8, 16, 32 or 64)
template <int CT>
__device__ __forceinline__ void tmem_add_cols(uint32_t taddr, float* acc) {
  if constexpr (CT <= 32) {
    tmem_add<CT>(taddr, acc);
  } else {
#pragma unroll
    for (int g = 0; g < CT / 32; ++g) tmem_add<32>(taddr + 32 * g, acc + 32 * g);
  }
}

}  // namespace

struct UmmaParams {
  CUtensorMap amap[NNP_MAX_SPECIES];
  CUtensorMap bmap[NNP_MAX_SPECIES];
  const UmmaItem* items;
  const int* cta_off;  // [grid + 1] item range of every persistent CTA
  int b_box_bytes;     // largest activation box of the launch (n_pad_max * 128)
  int stage_bytes;     // A_BOX_BYTES + b_box_bytes (raw and lo stages have the same layout)
  int n_raw;           // raw ring depth
  int slot_cols;       // TMEM columns per accumulator slot (= n_pad_max); cross accumulator at column 0
  int kps;             // k-steps (8 contraction elements each) accumulated in TMEM per slot: 1 or 4
  int gslots;          // slots per group = commit / drain granularity
  int n_groups;        // slot-group ring depth
};

// ------------------------------------------------------------------------------------------------
// drain + epilogue of one item: this thread owns feature row (TMEM lane) `quarter*32 + lane` and the
// atom columns [half*CT, half*CT + CT) of the tile.
template <int NP>
__device__ __forceinline__ void drain_item(const UmmaItem& t, const UmmaParams& P, uint32_t tmem, uint64_t* group_full,
                                           uint64_t* group_empty, uint64_t* cross_empty, uint32_t& grp, uint32_t& gphase,
                                           int quarter, int half, int lane) {
  constexpr int CT = NP >= 32 ? NP / 2 : NP;       // columns per thread
  constexpr bool TWO_LEVEL = NP <= 64;
  const bool active = NP >= 32 || half == 0;
  const int col0 = NP >= 32 ? half * CT : 0;
  float tot[CT];
  float part[TWO_LEVEL ? CT : 1];
#pragma unroll
  for (int j = 0; j < CT; ++j) tot[j] = 0.0f;
  if constexpr (TWO_LEVEL) {
#pragma unroll
    for (int j = 0; j < CT; ++j) part[j] = 0.0f;
  }
  int ks_left = ((t.kb1 - t.kb0) * 4 + P.kps - 1) / P.kps;  // slots of this item
  const uint32_t lane_base = tmem + ((uint32_t)(quarter * 32) << 16) + (uint32_t)col0;
  int in_part = 0;
  while (ks_left > 0) {
    const int ns = min(P.gslots, ks_left);
    mbar_wait(&group_full[grp], gphase);
    tc_fence_after();
    if (active) {
      const uint32_t src = lane_base + (uint32_t)P.slot_cols * (1u + grp * (uint32_t)P.gslots);
      for (int q = 0; q < ns; ++q) {
        if constexpr (TWO_LEVEL) {
          tmem_add_cols<CT>(src + (uint32_t)(q * P.slot_cols), part);
          if (++in_part == L1_SLOTS) {
#pragma unroll
            for (int j = 0; j < CT; ++j) { tot[j] += part[j]; part[j] = 0.0f; }
            in_part = 0;
          }
        } else {
          tmem_add_cols<CT>(src + (uint32_t)(q * P.slot_cols), tot);
        }
      }
    }
    tc_fence_before();
    mbar_arrive(&group_empty[grp]);
    if (++grp == (uint32_t)P.n_groups) { grp = 0; gphase ^= 1u; }
    ks_left -= ns;
  }
  if constexpr (TWO_LEVEL) {
#pragma unroll
    for (int j = 0; j < CT; ++j) tot[j] += part[j];
  }
  // cross terms (complete: the commit of the last group tracks every earlier MMA of the issuing thread)
  if (active) tmem_add_cols<CT>(lane_base, tot);
  tc_fence_before();
  mbar_arrive(cross_empty);
  // ---- epilogue
  const int f = quarter * 32 + lane;
  if (active && f < t.f_valid) {
    float* C = t.C + (size_t)col0 * t.ldc + f;
    const int nv = t.n_valid - col0;
    if (t.epi == EPI_BIAS_CELU) {
      const float b = t.bias ? t.bias[f] : 0.0f;
#pragma unroll
      for (int j = 0; j < CT; ++j)
        if (j < nv) C[(size_t)j * t.ldc] = celu_f(tot[j] + b, t.alpha, t.inv_alpha);
    } else if (t.epi == EPI_MUL_DCELU) {
      // aux may alias C (delta overwrites the activation in place): read every activation of this thread first, so
      // the loads are independent and in flight together instead of being ordered behind the stores
      const float* aux = t.aux + (size_t)col0 * t.ldaux + f;
      constexpr int HB = CT < 16 ? CT : 16;  // batch size: enough loads in flight, no register spills
#pragma unroll
      for (int j0 = 0; j0 < CT; j0 += HB) {
        float hv[HB];
#pragma unroll
        for (int j = 0; j < HB; ++j) hv[j] = j0 + j < nv ? aux[(size_t)(j0 + j) * t.ldaux] : 0.0f;
#pragma unroll
        for (int j = 0; j < HB; ++j)
          if (j0 + j < nv) C[(size_t)(j0 + j) * t.ldc] = tot[j0 + j] * dcelu_from_h(hv[j], t.inv_alpha);
      }
    } else {
#pragma unroll
      for (int j = 0; j < CT; ++j)
        if (j < nv) C[(size_t)j * t.ldc] = tot[j] * t.scale;
    }
  }
}

__global__ void __launch_bounds__(U_THREADS, 1) gemm_umma_kernel(const __grid_constant__ UmmaParams P) {
  extern __shared__ __align__(1024) unsigned char smem_dyn[];
  unsigned char* raw = smem_dyn + ((1024u - (smem_u32(smem_dyn) & 1023u)) & 1023u);
  unsigned char* los = raw + (size_t)P.n_raw * P.stage_bytes;
  uint64_t* bars = reinterpret_cast<uint64_t*>(los + (size_t)U_LO_STAGES * P.stage_bytes);
  uint64_t* full = bars;                              // [U_MAX_RAW]   TMA landed
  uint64_t* raw_empty = full + U_MAX_RAW;             // [U_MAX_RAW]   MMAs that read the raw stage are done
  uint64_t* conv = raw_empty + U_MAX_RAW;             // [U_LO_STAGES] lo parts written
  uint64_t* lo_empty = conv + U_LO_STAGES;            // [U_LO_STAGES]
  uint64_t* group_full = lo_empty + U_LO_STAGES;      // [U_MAX_GROUPS]
  uint64_t* group_empty = group_full + U_MAX_GROUPS;  // [U_MAX_GROUPS]
  uint64_t* cross_empty = group_empty + U_MAX_GROUPS; // [1]
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(cross_empty + 1);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < P.n_raw; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&raw_empty[s], 1);
    }
    for (int s = 0; s < U_LO_STAGES; ++s) {
      mbar_init(&conv[s], 128);
      mbar_init(&lo_empty[s], 1);
    }
    for (int g = 0; g < P.n_groups; ++g) {
      mbar_init(&group_full[g], 1);
      mbar_init(&group_empty[g], U_DRAIN_THREADS);
    }
    mbar_init(cross_empty, U_DRAIN_THREADS);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_slot)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  const int it0 = P.cta_off[blockIdx.x], it1 = P.cta_off[blockIdx.x + 1];

  if (warp == 0) {
    // ------------------------------------------------------------ TMA producer
    if (lane == 0) {
      uint32_t rs = 0, rphase = 0;
      for (int it = it0; it < it1; ++it) {
        const UmmaItem& t = P.items[it];
        const CUtensorMap* am = &P.amap[t.amap];
        const CUtensorMap* bm = &P.bmap[t.bmap];
        const int a_mn = t.a_mn, a_c0 = t.a_c0, a_c1 = t.a_c1, b_c0 = t.b_c0, b_c1 = t.b_c1, kb1 = t.kb1;
        const uint32_t tx = A_BOX_BYTES + (uint32_t)t.n_pad * 128u;
        unsigned long long live = t.kmask;
        for (int kbi = t.kb0; kbi < kb1; ++kbi) {
          int kb = kbi;
          if (live) {  // skip the contraction boxes that only hold structural zeros
            kb = __ffsll((long long)live) - 1;
            live &= live - 1;
          }
          mbar_wait(&raw_empty[rs], rphase ^ 1);
          unsigned char* sa = raw + (size_t)rs * P.stage_bytes;
          unsigned char* sb = sa + A_BOX_BYTES;
          mbar_expect_tx(&full[rs], tx);
          if (!a_mn) {
            tma_load_2d(sa, am, a_c0 + kb * BOXF, a_c1, &full[rs]);
          } else {
#pragma unroll
            for (int q = 0; q < 4; ++q) tma_load_2d(sa + q * 4096, am, a_c0 + q * BOXF, a_c1 + kb * BOXF, &full[rs]);
          }
          tma_load_2d(sb, bm, b_c0 + kb * BOXF, b_c1, &full[rs]);
          if (++rs == (uint32_t)P.n_raw) { rs = 0; rphase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ------------------------------------------------------------ MMA issuer
    // One thread; its instruction stream is the critical path of the CTA (every instruction of a single thread
    // costs its full latency), so everything loop-invariant lives in registers and the four shared-memory
    // descriptors of a box are formed once and advanced by an integer add per k-step.
    if (lane == 0) {
      uint32_t rs = 0, ls = 0, lphase = 0, grp = 0, gphase = 0, item_ctr = 0;
      const uint32_t d_x = tmem;
      const uint32_t n_raw = (uint32_t)P.n_raw, n_groups = (uint32_t)P.n_groups, gslots = (uint32_t)P.gslots,
                     kps = (uint32_t)P.kps, slot_cols = (uint32_t)P.slot_cols, stage_bytes = (uint32_t)P.stage_bytes;
      const uint32_t raw0 = smem_u32(raw), lo0 = smem_u32(los);
      // descriptor templates (address field zero): K-major 128B swizzle / MN-major 128B swizzle with 32B atoms
      const uint64_t desc_k = smem_desc(0, 16, 1024, 2), desc_mn = smem_desc(0, 4096, 512, 1);
      uint32_t d_hi = tmem + slot_cols;  // slot (grp 0, in_group 0)
      for (int it = it0; it < it1; ++it) {
        const UmmaItem& t = P.items[it];
        const int a_mn = t.a_mn, nb = t.kb1 - t.kb0;
        const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)a_mn << 15) |
                               ((uint32_t)(t.n_pad >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
        const uint64_t desc_a = a_mn ? desc_mn : desc_k;
        const uint32_t a_step = a_mn ? (1024u >> 4) : (32u >> 4);  // descriptor address units (16 B) per k-step
        mbar_wait(cross_empty, (item_ctr & 1u) ^ 1u);
        uint32_t in_group = 0, in_slot = 0, ks_left = (uint32_t)nb * 4u, first = 1u;
        for (int b = 0; b < nb; ++b) {
          mbar_wait(&conv[ls], lphase);  // lo parts written (and, transitively, the raw stage has landed)
          tc_fence_after();
          const uint32_t sa = (raw0 + rs * stage_bytes) >> 4, sal = (lo0 + ls * stage_bytes) >> 4;
          uint64_t ah = desc_a | sa, al = desc_a | sal;
          uint64_t bh = desc_k | (sa + (A_BOX_BYTES >> 4)), bl = desc_k | (sal + (A_BOX_BYTES >> 4));
#pragma unroll
          for (int ks = 0; ks < 4; ++ks) {
            if ((in_group | in_slot) == 0) {
              mbar_wait(&group_empty[grp], gphase ^ 1u);
              tc_fence_after();
            }
            mma_tf32(d_x, al, bh, idesc, first ^ 1u);
            mma_tf32(d_x, ah, bl, idesc, 1u);
            mma_tf32(d_hi, ah, bh, idesc, in_slot);
            first = 0u;
            ah += a_step; al += a_step; bh += 2; bl += 2;
            --ks_left;
            if (++in_slot == kps || ks_left == 0) {
              in_slot = 0;
              d_hi += slot_cols;
              if (++in_group == gslots || ks_left == 0) {
                tc_commit(&group_full[grp]);
                in_group = 0;
                if (++grp == n_groups) { grp = 0; gphase ^= 1u; }
                d_hi = tmem + slot_cols * (1u + grp * gslots);
              }
            }
          }
          tc_commit(&raw_empty[rs]);  // frees the stages when these MMAs have read them
          tc_commit(&lo_empty[ls]);
          if (++rs == n_raw) rs = 0;
          if (++ls == U_LO_STAGES) { ls = 0; lphase ^= 1u; }
        }
        ++item_ctr;
      }
    }
  } else if (warp < 6) {
    // ------------------------------------------------------------ converters
    const int ct = threadIdx.x - 64;
    uint32_t rs = 0, rphase = 0, ls = 0, lphase = 0;
    for (int it = it0; it < it1; ++it) {
      const UmmaItem& t = P.items[it];
      const int nbv = t.n_pad * 8;  // float4 count of the activation box
      const int nb = t.kb1 - t.kb0;
      for (int b = 0; b < nb; ++b) {
        mbar_wait(&lo_empty[ls], lphase ^ 1u);
        mbar_wait(&full[rs], rphase);
        unsigned char* sa = raw + (size_t)rs * P.stage_bytes;
        unsigned char* sl = los + (size_t)ls * P.stage_bytes;
        const float4* aw = reinterpret_cast<const float4*>(sa);
        float4* al = reinterpret_cast<float4*>(sl);
        float4* bh = reinterpret_cast<float4*>(sa + A_BOX_BYTES);
        float4* bl = reinterpret_cast<float4*>(sl + A_BOX_BYTES);
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const int idx = ct + 128 * i;
          al[idx] = w_lo4(aw[idx]);
        }
        for (int idx = ct; idx < nbv; idx += 128) {
          float4 h, l;
          x_split4(bh[idx], h, l);
          bh[idx] = h;
          bl[idx] = l;
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_arrive(&conv[ls]);
        if (++rs == (uint32_t)P.n_raw) { rs = 0; rphase ^= 1u; }
        if (++ls == U_LO_STAGES) { ls = 0; lphase ^= 1u; }
      }
    }
  } else {
    // ------------------------------------------------------------ drain + epilogue (TMEM lane quarter = warp % 4)
    const int quarter = warp & 3, half = (warp - 6) >> 2;
    uint32_t grp = 0, gphase = 0;
    for (int it = it0; it < it1; ++it) {
      const UmmaItem t = P.items[it];
      switch (t.n_pad) {
        case 16: drain_item<16>(t, P, tmem, group_full, group_empty, cross_empty, grp, gphase, quarter, half, lane); break;
        case 32: drain_item<32>(t, P, tmem, group_full, group_empty, cross_empty, grp, gphase, quarter, half, lane); break;
        case 64: drain_item<64>(t, P, tmem, group_full, group_empty, cross_empty, grp, gphase, quarter, half, lane); break;
        default: drain_item<128>(t, P, tmem, group_full, group_empty, cross_empty, grp, gphase, quarter, half, lane); break;
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem) : "memory");
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
  }
  return fn;
}

// 2-D f32 tensor [rows][cols], row pitch ld floats; box = [box_rows][32 floats]
static int encode_map(CUtensorMap* m, const float* base, long long rows, long long cols, long long ld, int box_rows,
                      CUtensorMapSwizzle swz) {
  EncodeTiledFn enc = get_encode();
  if (!enc) return -1;
  if (rows <= 0) rows = 1;
  cuuint64_t gdim[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
  cuuint64_t gstr[1] = {(cuuint64_t)ld * 4};
  cuuint32_t box[2] = {(cuuint32_t)BOXF, (cuuint32_t)box_rows};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, (void*)base, gdim, gstr, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, swz, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? 0 : -1;
}

int umma_atom_tile(int n_rows) {
  if (n_rows <= 16) return 16;
  if (n_rows <= 32) return 32;
  if (n_rows <= 64) return 64;
  return 128;
}

static const size_t UMMA_SMEM_BUDGET = 220 * 1024;

int umma_build_launch(UmmaLaunch& L, const std::vector<UmmaProblem>& probs, const std::vector<TmaOperand>& aops,
                      const std::vector<TmaOperand>& bops, int a_mn, int num_sms) {
  UmmaParams* P = new UmmaParams();
  memset(P, 0, sizeof(*P));
  L.params = P;
  if (aops.size() > NNP_MAX_SPECIES || bops.size() > NNP_MAX_SPECIES) return -1;
  std::vector<int> tile_of_bmap(bops.size(), 16);
  int np_max = 16;
  for (size_t i = 0; i < bops.size(); ++i) {
    tile_of_bmap[i] = umma_atom_tile((int)bops[i].rows);
    np_max = std::max(np_max, tile_of_bmap[i]);
    if (encode_map(&P->bmap[i], bops[i].base, bops[i].rows, bops[i].cols, bops[i].ld, tile_of_bmap[i],
                   CU_TENSOR_MAP_SWIZZLE_128B))
      return -1;
  }
  for (size_t i = 0; i < aops.size(); ++i)
    if (encode_map(&P->amap[i], aops[i].base, aops[i].rows, aops[i].cols, aops[i].ld, a_mn ? 32 : 128,
                   a_mn ? CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B : CU_TENSOR_MAP_SWIZZLE_128B))
      return -1;
  std::vector<UmmaItem> items;
  std::vector<long long> cost;
  for (const UmmaProblem& p : probs) {
    if (p.n_atoms <= 0 || p.F <= 0 || p.K <= 0) continue;
    const int nt = tile_of_bmap[p.bmap];
    const int nkb_all = (p.K + BOXF - 1) / BOXF;
    unsigned long long kmask = nkb_all <= 64 ? p.kmask : 0ull;
    if (nkb_all < 64) kmask &= (1ull << nkb_all) - 1ull;
    const int nkb = kmask ? __builtin_popcountll(kmask) : nkb_all;
    for (int f0 = 0; f0 < p.F; f0 += 128) {
      if (p.fmask && f0 / 128 < 64 && !((p.fmask >> (f0 / 128)) & 1ull)) continue;
      for (int a0 = 0; a0 < p.n_atoms; a0 += nt) {
        UmmaItem t;
        memset(&t, 0, sizeof(t));
        t.amap = p.amap; t.bmap = p.bmap; t.a_mn = a_mn;
        if (!a_mn) { t.a_c0 = p.a_c0; t.a_c1 = p.a_c1 + f0; }  // (k col, feature row)
        else { t.a_c0 = p.a_c0 + f0; t.a_c1 = p.a_c1; }        // (feature col, contraction row)
        t.b_c0 = p.b_c0; t.b_c1 = p.b_c1 + a0;
        t.kb0 = 0; t.kb1 = nkb;
        t.kmask = kmask;
        t.n_pad = nt;
        t.n_valid = std::min(nt, p.n_atoms - a0);
        t.f_valid = std::min(128, p.F - f0);
        t.epi = p.epi;
        t.C = p.C + (size_t)a0 * p.ldc + f0;
        t.ldc = p.ldc;
        t.bias = p.bias ? p.bias + f0 : nullptr;
        t.aux = p.aux ? p.aux + (size_t)a0 * p.ldaux + f0 : nullptr;
        t.ldaux = p.ldaux;
        t.scale = p.scale; t.alpha = p.alpha; t.inv_alpha = p.inv_alpha;
        items.push_back(t);
        cost.push_back((long long)nkb * (128 + 2 * nt));
      }
    }
  }
  // heavy items first, dealt to the persistent CTAs in snake order (static => deterministic)
  const size_t n = items.size();
  std::vector<size_t> order(n);
  for (size_t i = 0; i < n; ++i) order[i] = i;
  std::stable_sort(order.begin(), order.end(), [&](size_t a, size_t b) { return cost[a] > cost[b]; });
  const size_t G = std::max<size_t>(1, std::min<size_t>(n, (size_t)num_sms));
  std::vector<std::vector<UmmaItem>> per_cta(G);
  for (size_t i = 0; i < n; ++i) {
    const size_t round = i / G, posn = i % G;
    per_cta[(round & 1) ? G - 1 - posn : posn].push_back(items[order[i]]);
  }
  std::vector<UmmaItem> flat;
  std::vector<int> off(G + 1, 0);
  for (size_t c = 0; c < G; ++c) {
    for (auto& t : per_cta[c]) flat.push_back(t);
    off[c + 1] = (int)flat.size();
  }
  L.n_items = (int)n;
  L.grid = n ? (int)G : 0;
  P->b_box_bytes = np_max * 128;
  P->stage_bytes = A_BOX_BYTES + P->b_box_bytes;
  const size_t bar_bytes = (2 * U_MAX_RAW + 2 * U_LO_STAGES + 2 * U_MAX_GROUPS + 1) * 8 + 16;
  P->n_raw = (int)std::min<size_t>(U_MAX_RAW, (UMMA_SMEM_BUDGET - 1024 - bar_bytes) / P->stage_bytes - U_LO_STAGES);
  L.smem_bytes = (size_t)(P->n_raw + U_LO_STAGES) * P->stage_bytes + bar_bytes + 1024;
  P->slot_cols = np_max;
  {
    const char* e = getenv("NNP_UMMA_KPS");  // experiment knob: k-steps accumulated in TMEM per slot
    P->kps = (e && atoi(e) == 1) ? 1 : 4;
  }
  P->gslots = std::max(1, std::min(4, 128 / np_max));
  P->n_groups = std::min(U_MAX_GROUPS, (512 - np_max) / (P->gslots * np_max));
  if (cudaMalloc((void**)&L.d_items, std::max<size_t>(1, n) * sizeof(UmmaItem)) != cudaSuccess) return -1;
  if (cudaMalloc((void**)&L.d_cta_off, (G + 1) * sizeof(int)) != cudaSuccess) return -1;
  if (n) cudaMemcpy(L.d_items, flat.data(), n * sizeof(UmmaItem), cudaMemcpyHostToDevice);
  cudaMemcpy(L.d_cta_off, off.data(), (G + 1) * sizeof(int), cudaMemcpyHostToDevice);
  P->items = L.d_items;
  P->cta_off = L.d_cta_off;
  return 0;
}

void umma_launch(const UmmaLaunch& L, cudaStream_t s) {
  if (L.n_items == 0) return;
  gemm_umma_kernel<<<L.grid, U_THREADS, L.smem_bytes, s>>>(*reinterpret_cast<const UmmaParams*>(L.params));
}

int umma_init() {
  if (!get_encode()) return -1;
  return cudaFuncSetAttribute((const void*)gemm_umma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)UMMA_SMEM_BUDGET) == cudaSuccess ? 0 : -1;
}

void umma_free_launch(UmmaLaunch& L) {
  if (L.d_items) cudaFree(L.d_items);
  if (L.d_cta_off) cudaFree(L.d_cta_off);
  delete reinterpret_cast<UmmaParams*>(L.params);
  L.d_items = nullptr; L.d_cta_off = nullptr; L.params = nullptr;
}

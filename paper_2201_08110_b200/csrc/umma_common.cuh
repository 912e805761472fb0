// Shared device helpers of the tcgen05 GEMM engines (mlp_umma.cu: one CTA per tile; mlp_umma2.cu: CTA pairs,
// cta_group::2): mbarrier / TMA / tcgen05 wrappers, the TMEM drain with truncation compensation and the staged
// epilogue.  Included by those two files only; everything is in an anonymous namespace.
#pragma once
#include <cuda.h>

#include "nnp_internal.h"

namespace {

constexpr int BOXF = 32;                 // floats per box row (128 B)
constexpr int A_BOX_BYTES = 128 * 128;   // weight box: 128 feature rows x 32 contraction floats (one plane)
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
// warp-converged issue: every lane runs the role loop with warp-uniform values (so the compiler keeps descriptors and
// addresses in uniform registers), one elected lane executes the asynchronous instructions
__device__ __forceinline__ uint32_t elect_one() {
  uint32_t pred;
  asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
  return pred;
}
__device__ __forceinline__ void tma_load_2d_s(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
      ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar)
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
// done on the integer ALU
__device__ __forceinline__ float tf32_rna(float x) {
  return __uint_as_float((__float_as_uint(x) + 0x1000u) & 0xFFFFE000u);
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

// acc[0..CNT-1] += CNT consecutive TMEM columns of this thread's lane (CNT = 8, 16 or 32).
// comp = 1: every value read is first moved one ulp AWAY from zero.  tcgen05 truncates towards zero each time it adds
// into its accumulator (measured: mean -0.27 ulp per accumulating k-step, -1.07 ulp over the 4 k-steps of a slot,
// DESIGN.md section 7); adding the expected loss back removes the coherent shrink of every pre-activation, which
// otherwise shows up as an energy bias of -4e-6 kcal/mol per atom.  An exact zero becomes the smallest denormal
// (1.4e-45): harmless, and padding rows / columns are never stored.
template <int CNT>
__device__ __forceinline__ void tmem_add(uint32_t taddr, float* acc, uint32_t comp) {
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
  for (int j = 0; j < CNT; ++j) acc[j] += __uint_as_float(r[j] + comp);
}
// CT columns starting at taddr (CT = 8, 16, 32 or 64)
template <int CT>
__device__ __forceinline__ void tmem_add_cols(uint32_t taddr, float* acc, uint32_t comp) {
  if constexpr (CT <= 32) {
    tmem_add<CT>(taddr, acc, comp);
  } else {  // 32 columns per load: fewer load / wait round trips per slot than 16, and the staging registers still fit
#pragma unroll
    for (int g = 0; g < CT / 32; ++g) tmem_add<32>(taddr + 32 * g, acc + 32 * g, comp);
  }
}

__device__ __forceinline__ float4 ld4(const float* p) { return *reinterpret_cast<const float4*>(p); }
__device__ __forceinline__ void st4(float* p, const float4 v) { *reinterpret_cast<float4*>(p) = v; }
__device__ __forceinline__ void split4(const float4 v, float4& h, float4& l) {
  h.x = tf32_rna(v.x); h.y = tf32_rna(v.y); h.z = tf32_rna(v.z); h.w = tf32_rna(v.w);
  l.x = v.x - h.x; l.y = v.y - h.y; l.z = v.z - h.z; l.w = v.w - h.w;
}
// store one float4 of results: split into the hi / lo planes when a tensor launch consumes it
__device__ __forceinline__ void store_out(const UmmaItem& t, size_t o, const float4 x) {
  if (t.C_lo) {
    float4 h, l;
    split4(x, h, l);
    st4(t.C + o, h);
    st4(t.C_lo + o, l);
  } else {
    st4(t.C + o, x);
  }
}

// epilogue of `na` <= 64 atoms (rows of the staging tile [atom][128 features]) by the THREADS drain threads: bias + CELU /
// x CELU' / scale, four consecutive features of one atom per thread and step (16-byte loads and stores).  A thread
// has at most 8 steps; the backward epilogue issues ALL its global loads (h of the layer below, two planes) before
// the first use, so a round costs one memory latency instead of one per step.  Global row of staging row r is a0 + r.
template <int THREADS>
__device__ __forceinline__ void epilogue_rows(const UmmaItem& t, const float* staging, int a0, int na, int dt) {
  constexpr int RPS = THREADS / 32, U = 64 / RPS;  // rows per step, steps: 64 atoms x 32 feature groups / THREADS
  const int n_vec = na * 32;
  const int g = dt & 31;          // the thread's feature group is the same in every step (256 % 32 == 0)
  if (4 * g >= t.f_valid) return;
  const int r0 = dt >> 5;         // rows r0, r0 + 8, ...
  if (t.epi == EPI_MUL_DCELU) {
    float4 d[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int r = r0 + RPS * u;
      d[u] = make_float4(0.f, 0.f, 0.f, 0.f);
      if (r * 32 < n_vec) d[u] = ld4(t.aux + (size_t)(a0 + r) * t.ldaux + 4 * g);
    }
    if (t.aux_lo) {
      float4 l[U];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int r = r0 + RPS * u;
        l[u] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (r * 32 < n_vec) l[u] = ld4(t.aux_lo + (size_t)(a0 + r) * t.ldaux + 4 * g);
      }
#pragma unroll
      for (int u = 0; u < U; ++u) { d[u].x += l[u].x; d[u].y += l[u].y; d[u].z += l[u].z; d[u].w += l[u].w; }  // exact
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int r = r0 + RPS * u;
      if (r * 32 >= n_vec) continue;
      float4 x = ld4(staging + r * 128 + 4 * g);
      x.x *= dcelu_from_h(d[u].x, t.inv_alpha); x.y *= dcelu_from_h(d[u].y, t.inv_alpha);
      x.z *= dcelu_from_h(d[u].z, t.inv_alpha); x.w *= dcelu_from_h(d[u].w, t.inv_alpha);
      store_out(t, (size_t)(a0 + r) * t.ldc + 4 * g, x);
    }
  } else if (t.epi == EPI_BIAS_CELU_LAST) {
    // last hidden layer: h as ONE plane for the energy kernel, and the start of the backward pass
    // delta = w_last * CELU'(h) as the split operand of the first backward GEMM (h is not read again as an operand)
    float4 b = make_float4(0.f, 0.f, 0.f, 0.f);
    if (t.bias) b = ld4(t.bias + 4 * g);
    const float4 wl = ld4(t.w_last + 4 * g);
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int r = r0 + RPS * u;
      if (r * 32 >= n_vec) continue;
      float4 x = ld4(staging + r * 128 + 4 * g);
      x.x = celu_f(x.x + b.x, t.alpha, t.inv_alpha); x.y = celu_f(x.y + b.y, t.alpha, t.inv_alpha);
      x.z = celu_f(x.z + b.z, t.alpha, t.inv_alpha); x.w = celu_f(x.w + b.w, t.alpha, t.inv_alpha);
      const size_t o = (size_t)(a0 + r) * t.ldc + 4 * g;
      st4(t.C_full + o, x);
      x.x = wl.x * dcelu_from_h(x.x, t.inv_alpha); x.y = wl.y * dcelu_from_h(x.y, t.inv_alpha);
      x.z = wl.z * dcelu_from_h(x.z, t.inv_alpha); x.w = wl.w * dcelu_from_h(x.w, t.inv_alpha);
      store_out(t, o, x);
    }
  } else if (t.epi == EPI_BIAS_CELU) {
    float4 b = make_float4(0.f, 0.f, 0.f, 0.f);
    if (t.bias) b = ld4(t.bias + 4 * g);
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int r = r0 + RPS * u;
      if (r * 32 >= n_vec) continue;
      float4 x = ld4(staging + r * 128 + 4 * g);
      x.x = celu_f(x.x + b.x, t.alpha, t.inv_alpha); x.y = celu_f(x.y + b.y, t.alpha, t.inv_alpha);
      x.z = celu_f(x.z + b.z, t.alpha, t.inv_alpha); x.w = celu_f(x.w + b.w, t.alpha, t.inv_alpha);
      store_out(t, (size_t)(a0 + r) * t.ldc + 4 * g, x);
    }
  } else {
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int r = r0 + RPS * u;
      if (r * 32 >= n_vec) continue;
      float4 x = ld4(staging + r * 128 + 4 * g);
      x.x *= t.scale; x.y *= t.scale; x.z *= t.scale; x.w *= t.scale;
      st4(t.C + (size_t)(a0 + r) * t.ldc + 4 * g, x);
    }
  }
}

}  // namespace

// Ligand-size MLP engine, fused middle of the network (A4 layers 2..L-1, A5 per-atom energies, A6 back
// to delta_1) in ONE launch.  FP32 FFMA, FP64 for the energy dot product.
//
// Mathematics: DESIGN.md O5/O7.  Regime: BASELINE.json configs[0,1] (12 / 50 atoms): after the first
// layer every remaining layer of an (element, model) network is a few hundred KB of weights applied to a
// handful of atoms, and the cost of running them as separate launches is the launch + dependent-latency
// chain (5 launches ~ 55 us at 50 atoms), not bytes or flops.  Here one CTA owns (element, model, chunk of
// <= 4 atoms) and walks h_1 -> h_2 -> ... -> h_{L-1} -> e, delta_{L-1} -> ... -> delta_1 with every
// activation in shared memory / registers.  The weights do not depend on the data, so a producer warp
// streams them (forward layers, then the same matrices again for the backward pass) as 1-D bulk async
// copies of <= 32 row tiles through a deep shared-memory ring: the copies of the next few tiles are in flight while
// tile t is consumed, across layer boundaries, so the only exposed latency is that of the first tile.
//
//   forward tile (rows = output features):  a warp owns 2 rows; lanes split the contraction (x of the 4
//       atoms in registers), 8 partial sums are reduced by a 9-shuffle transposing butterfly (fixed order);
//   backward tile (rows = contraction index o): a warp owns 2 rows, lanes own 4 consecutive input columns,
//       accumulators stay in registers over all tiles of the layer; the 16 warps are summed in a fixed order
//       through shared memory, multiplied by CELU'(h) and become the next delta.
#include <algorithm>

#include "nnp_internal.h"

namespace {

constexpr int MID_CONSUMERS = 512;               // 16 consumer warps
constexpr int MID_THREADS = MID_CONSUMERS + 32;  // + 1 producer warp
constexpr int MID_WARPS = MID_CONSUMERS / 32;
constexpr int MID_TILE_ROWS = 32;                // 2 rows per consumer warp
constexpr int MID_RW = 2;
constexpr int MID_AC = 4;                        // atoms per CTA
constexpr int MID_NJ = 2;                        // float4 per lane along a row: rows of <= 256 floats
constexpr int MID_HMAX = 128 * MID_NJ;
constexpr int MID_MAX_STAGES = 6;

// CELU through the hardware exponential: alpha (2^(x log2e / alpha) - 1); absolute error ~6e-9 near x = 0 (unbiased),
// two orders below the FP32 rounding of the dot product that produced x; expm1f costs ~30 instructions
__device__ __forceinline__ float celu_m(float x, float alpha, float inv_alpha) {
  float e;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(x * inv_alpha * 1.4426950408889634f));
  return x > 0.0f ? x : alpha * (e - 1.0f);
}
__device__ __forceinline__ float dcelu_m(float h, float inv_alpha) { return h > 0.0f ? 1.0f : fmaf(h, inv_alpha, 1.0f); }
__device__ __forceinline__ float dot4m(const float4 w, const float4 x, float s) {
  s = fmaf(w.x, x.x, s);
  s = fmaf(w.y, x.y, s);
  s = fmaf(w.z, x.z, s);
  return fmaf(w.w, x.w, s);
}
__device__ __forceinline__ uint32_t m_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mb_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(m_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mb_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(m_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mb_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(m_u32(bar)) : "memory");
}
__device__ __forceinline__ void mb_wait(uint64_t* bar, uint32_t parity) {
  const uint32_t addr = m_u32(bar);
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
__device__ __forceinline__ void bulk_load(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(m_u32(dst)), "l"(src), "r"(bytes), "r"(m_u32(bar))
               : "memory");
}
__device__ __forceinline__ void consumer_sync() { asm volatile("bar.sync 1, %0;" ::"n"(MID_CONSUMERS) : "memory"); }

}  // namespace

// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(MID_THREADS, 1) small_mid_kernel(const MidItem* __restrict__ items, int n_stages) {
  extern __shared__ __align__(128) unsigned char mid_smem[];
  __shared__ __align__(8) uint64_t full[MID_MAX_STAGES];
  __shared__ __align__(8) uint64_t empty[MID_MAX_STAGES];
  __shared__ MidItem it;
  constexpr int TILE_FLOATS = MID_TILE_ROWS * MID_HMAX;
  constexpr int AH = MID_AC * MID_HMAX;  // floats of one activation / delta buffer
  {
    const int* src = reinterpret_cast<const int*>(items + blockIdx.x);
    int* dst = reinterpret_cast<int*>(&it);
    for (int w = threadIdx.x; w < (int)(sizeof(MidItem) / 4); w += MID_THREADS) dst[w] = src[w];
  }
  if (threadIdx.x == 0) {
    for (int s = 0; s < n_stages; ++s) {
      mb_init(&full[s], 1);
      mb_init(&empty[s], MID_WARPS);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  pdl_trigger();
  float* ring = reinterpret_cast<float*>(mid_smem);
  const int L = it.L;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == MID_WARPS) {
    // ------------------------------------------------------------ producer: the whole weight sequence
    if (lane == 0) {
      uint32_t slot = 0, phase = 0;
      for (int pass = 0; pass < 2; ++pass) {
        for (int li = 2; li <= L - 1; ++li) {
          const int l = pass == 0 ? li : (L + 1 - li);  // forward 2..L-1, backward L-1..2
          const int K = it.H[l - 1], R = it.H[l];
          const float* Wl = it.W[l];
          for (int r0 = 0; r0 < R; r0 += MID_TILE_ROWS) {
            const uint32_t bytes = (uint32_t)(min(MID_TILE_ROWS, R - r0) * K * 4);
            mb_wait(&empty[slot], phase ^ 1u);
            mb_expect_tx(&full[slot], bytes);
            bulk_load(ring + (size_t)slot * TILE_FLOATS, Wl + (size_t)r0 * K, bytes, &full[slot]);
            if (++slot == (uint32_t)n_stages) { slot = 0; phase ^= 1u; }
          }
        }
      }
    }
    return;
  }

  // -------------------------------------------------------------- consumers
  float* hs = ring + (size_t)n_stages * TILE_FLOATS;  // [L-1][AC][HMAX]: h_1 .. h_{L-1}
  float* dbuf = hs + (size_t)(L - 1) * AH;            // [2][AC][HMAX]: delta ping-pong
  float* red = dbuf + 2 * AH;                         // [MID_WARPS][AC][HMAX]
  float* bs = red + MID_WARPS * AH;                   // [L+1][HMAX]: biases of layers 2..L-1 at row l, w_L at row L
  const int tid = threadIdx.x;
  uint32_t slot = 0, phase = 0;
  {  // biases and w_L: staged once so that no global load sits inside the tile loops
    for (int l = 2; l <= L - 1; ++l)
      for (int r = tid; r < it.H[l]; r += MID_CONSUMERS) bs[l * MID_HMAX + r] = it.bias[l] ? __ldg(it.bias[l] + r) : 0.0f;
    for (int o = tid; o < it.H[L - 1]; o += MID_CONSUMERS) bs[L * MID_HMAX + o] = __ldg(it.w_last + o);
  }
  pdl_wait();  // h_1 comes from the layer-1 kernel; the weight ring (constant data) is already filling
  {  // h_1 of the chunk (rows of padding atoms are zero)
    const int K4 = it.H[1] >> 2;
    for (int idx = tid; idx < MID_AC * K4; idx += MID_CONSUMERS) {
      const int a = idx / K4, k4 = idx - a * K4;
      float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
      if (a < it.n_atoms) v = *(reinterpret_cast<const float4*>(it.h1 + (size_t)a * it.ld1) + k4);
      reinterpret_cast<float4*>(hs + a * MID_HMAX)[k4] = v;
    }
  }
  consumer_sync();

  // ---- forward, layers 2..L-1
  for (int l = 2; l <= L - 1; ++l) {
    const int K4 = it.H[l - 1] >> 2, R = it.H[l];
    const float* hin = hs + (size_t)(l - 2) * AH;
    float* hout = hs + (size_t)(l - 1) * AH;
    const float* bias = bs + l * MID_HMAX;
    float4 x[MID_AC][MID_NJ];
#pragma unroll
    for (int a = 0; a < MID_AC; ++a)
#pragma unroll
      for (int j = 0; j < MID_NJ; ++j) {
        const int k4 = lane + 32 * j;
        x[a][j] = k4 < K4 ? reinterpret_cast<const float4*>(hin + a * MID_HMAX)[k4] : make_float4(0.f, 0.f, 0.f, 0.f);
      }
    for (int r0 = 0; r0 < R; r0 += MID_TILE_ROWS) {
      mb_wait(&full[slot], phase);
      const float4* tile = reinterpret_cast<const float4*>(ring + (size_t)slot * TILE_FLOATS);
      float s[8];
#pragma unroll
      for (int q = 0; q < 8; ++q) s[q] = 0.0f;
#pragma unroll
      for (int rr = 0; rr < MID_RW; ++rr) {
        const int r = warp * MID_RW + rr;
        if (r0 + r < R) {
#pragma unroll
          for (int j = 0; j < MID_NJ; ++j) {
            const int k4 = lane + 32 * j;
            if (k4 < K4) {
              const float4 w = tile[r * K4 + k4];
#pragma unroll
              for (int a = 0; a < MID_AC; ++a) s[rr * 4 + a] = dot4m(w, x[a][j], s[rr * 4 + a]);
            }
          }
        }
      }
      __syncwarp();
      if (lane == 0) mb_arrive(&empty[slot]);
      if (++slot == (uint32_t)n_stages) { slot = 0; phase ^= 1u; }
      // transposing butterfly: 8 sums over 32 lanes, 9 shuffles, fixed order
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const bool up = lane & 16;
        const float send = up ? s[q] : s[q + 4];
        const float keep = up ? s[q + 4] : s[q];
        s[q] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
      }
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        const bool up = lane & 8;
        const float send = up ? s[q] : s[q + 2];
        const float keep = up ? s[q + 2] : s[q];
        s[q] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
      }
      {
        const bool up = lane & 4;
        const float send = up ? s[0] : s[1];
        const float keep = up ? s[1] : s[0];
        s[0] = keep + __shfl_xor_sync(0xffffffffu, send, 4);
      }
      s[0] += __shfl_xor_sync(0xffffffffu, s[0], 2);
      s[0] += __shfl_xor_sync(0xffffffffu, s[0], 1);
      if ((lane & 3) == 0) {
        const int q = ((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1);
        const int rr = q >> 2, a = q & 3;
        const int r = r0 + warp * MID_RW + rr;
        if (r < R) hout[a * MID_HMAX + r] = celu_m(s[0] + bias[r], it.alpha, it.inv_alpha);
      }
    }
    consumer_sync();
  }
  // ---- layer L (1 output): per-atom energies (FP64) and delta_{L-1} = w_L (.) CELU'(h_{L-1})
  float* dcur = dbuf;
  float* dnext = dbuf + AH;
  {
    const int HL = it.H[L - 1];
    const float* hL = hs + (size_t)(L - 2) * AH;
    if (warp < it.n_atoms && it.e_out) {
      double acc = 0.0;
      for (int o = lane; o < HL; o += 32) acc += (double)bs[L * MID_HMAX + o] * (double)hL[warp * MID_HMAX + o];
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, off);
      if (lane == 0) it.e_out[(size_t)warp * it.lde] = acc + (double)it.b_last;
    }
    for (int idx = tid; idx < MID_AC * HL; idx += MID_CONSUMERS) {
      const int a = idx / HL, o = idx - a * HL;
      dcur[a * MID_HMAX + o] = a < it.n_atoms ? bs[L * MID_HMAX + o] * dcelu_m(hL[a * MID_HMAX + o], it.inv_alpha) : 0.0f;
    }
  }
  consumer_sync();
  // ---- backward through layers L-1..2: delta_{l-1} = (delta_l W_l) (.) CELU'(h_{l-1})
  for (int l = L - 1; l >= 2; --l) {
    const int R = it.H[l], N4 = it.H[l - 1] >> 2;
    float4 acc[MID_AC][MID_NJ];
#pragma unroll
    for (int a = 0; a < MID_AC; ++a)
#pragma unroll
      for (int j = 0; j < MID_NJ; ++j) acc[a][j] = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int o0 = 0; o0 < R; o0 += MID_TILE_ROWS) {
      mb_wait(&full[slot], phase);
      const float4* tile = reinterpret_cast<const float4*>(ring + (size_t)slot * TILE_FLOATS);
      const int ow = o0 + warp * MID_RW;  // R % 4 == 0: the warp's two rows are valid together
      if (ow < R) {
        float2 d[MID_AC];
#pragma unroll
        for (int a = 0; a < MID_AC; ++a) d[a] = *reinterpret_cast<const float2*>(dcur + a * MID_HMAX + ow);
#pragma unroll
        for (int j = 0; j < MID_NJ; ++j) {
          const int n4 = lane + 32 * j;
          if (n4 < N4) {
            const float4 w0 = tile[(warp * MID_RW + 0) * N4 + n4], w1 = tile[(warp * MID_RW + 1) * N4 + n4];
#pragma unroll
            for (int a = 0; a < MID_AC; ++a) {
              float4 v = acc[a][j];
              v.x = fmaf(d[a].x, w0.x, v.x); v.y = fmaf(d[a].x, w0.y, v.y); v.z = fmaf(d[a].x, w0.z, v.z); v.w = fmaf(d[a].x, w0.w, v.w);
              v.x = fmaf(d[a].y, w1.x, v.x); v.y = fmaf(d[a].y, w1.y, v.y); v.z = fmaf(d[a].y, w1.z, v.z); v.w = fmaf(d[a].y, w1.w, v.w);
              acc[a][j] = v;
            }
          }
        }
      }
      __syncwarp();
      if (lane == 0) mb_arrive(&empty[slot]);
      if (++slot == (uint32_t)n_stages) { slot = 0; phase ^= 1u; }
    }
    float4* red4 = reinterpret_cast<float4*>(red);
#pragma unroll
    for (int a = 0; a < MID_AC; ++a)
#pragma unroll
      for (int j = 0; j < MID_NJ; ++j) {
        const int n4 = lane + 32 * j;
        if (n4 < N4) red4[(warp * MID_AC + a) * (MID_HMAX / 4) + n4] = acc[a][j];
      }
    consumer_sync();
    const float* hprev = hs + (size_t)(l - 2) * AH;
    for (int idx = tid; idx < MID_AC * N4; idx += MID_CONSUMERS) {
      const int a = idx / N4, n4 = idx - a * N4;
      float4 v = red4[a * (MID_HMAX / 4) + n4];
#pragma unroll
      for (int w = 1; w < MID_WARPS; ++w) {  // fixed order
        const float4 u = red4[(w * MID_AC + a) * (MID_HMAX / 4) + n4];
        v.x += u.x; v.y += u.y; v.z += u.z; v.w += u.w;
      }
      const float4 h = reinterpret_cast<const float4*>(hprev + a * MID_HMAX)[n4];
      v.x *= dcelu_m(h.x, it.inv_alpha); v.y *= dcelu_m(h.y, it.inv_alpha);
      v.z *= dcelu_m(h.z, it.inv_alpha); v.w *= dcelu_m(h.w, it.inv_alpha);
      if (l == 2) {
        if (a < it.n_atoms) *(reinterpret_cast<float4*>(it.h1 + (size_t)a * it.ld1) + n4) = v;  // delta_1, in place
      } else {
        reinterpret_cast<float4*>(dnext + a * MID_HMAX)[n4] = v;
      }
    }
    consumer_sync();
    float* tmp = dcur; dcur = dnext; dnext = tmp;
  }
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
static const size_t MID_SMEM_MAX = 224 * 1024;

static size_t mid_fixed_bytes(int L) {
  return ((size_t)(L - 1) * MID_AC * MID_HMAX + 2 * MID_AC * MID_HMAX + (size_t)MID_WARPS * MID_AC * MID_HMAX +
          (size_t)(L + 1) * MID_HMAX) * 4;
}

bool mid_supported(int L, const int* d) {
  if (L < 3) return false;
  for (int l = 1; l <= L - 1; ++l)
    if (d[l] > MID_HMAX || d[l] % 4 != 0) return false;
  return mid_fixed_bytes(L) + 2 * (size_t)MID_TILE_ROWS * MID_HMAX * 4 <= MID_SMEM_MAX;
}

int mid_init() {
  return cudaFuncSetAttribute((const void*)small_mid_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)MID_SMEM_MAX) == cudaSuccess ? 0 : -1;
}

int mid_build(SmallLaunch& L, std::vector<MidItem>& items) {
  // heavy items (most weight bytes) first
  auto cost = [](const MidItem& t) {
    long long c = 0;
    for (int l = 2; l <= t.L - 1; ++l) c += (long long)t.H[l] * t.H[l - 1];
    return c;
  };
  std::stable_sort(items.begin(), items.end(), [&](const MidItem& a, const MidItem& b) { return cost(a) > cost(b); });
  L.n_items = (int)items.size();
  int Lmax = 3;
  for (const auto& t : items) Lmax = std::max(Lmax, t.L);
  const size_t tile = (size_t)MID_TILE_ROWS * MID_HMAX * 4;
  int stages = (int)((MID_SMEM_MAX - mid_fixed_bytes(Lmax)) / tile);
  stages = std::min(stages, MID_MAX_STAGES);
  if (stages < 2) return -1;
  L.variant = stages;
  L.smem_bytes = mid_fixed_bytes(Lmax) + (size_t)stages * tile;
  if (cudaMalloc(&L.d_items, std::max<size_t>(1, items.size()) * sizeof(MidItem)) != cudaSuccess) return -1;
  if (!items.empty()) cudaMemcpy(L.d_items, items.data(), items.size() * sizeof(MidItem), cudaMemcpyHostToDevice);
  return 0;
}

void mid_launch(const SmallLaunch& L, cudaStream_t s, bool pdl) {
  if (L.n_items == 0) return;
  launch_kernel(pdl, small_mid_kernel, dim3(L.n_items), dim3(MID_THREADS), L.smem_bytes, s,
                reinterpret_cast<const MidItem*>(L.d_items), L.variant);
}

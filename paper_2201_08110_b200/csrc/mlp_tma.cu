// TMA-staged, mbarrier-pipelined persistent GEMM engine for the per-element atomic MLPs (A4/A6).
//
// Same mathematics as mlp_ffma.cu (O5/O7) -- exact FP32 products, FP32 accumulation in a
// fixed order, two-level (per-stage) partial sums -- but the operand tiles are brought into shared
// memory by the Tensor Memory Accelerator (cp.async.bulk.tensor, 128-byte swizzle) through a ring of
// stages guarded by full/empty mbarriers, and the CTAs are persistent: one producer warp runs ahead
// across tile boundaries so the weight stream from HBM/L2 never drains.  At ligand sizes (a few
// atoms per element, BASELINE.json configs[1]) the layer-1 GEMMs are weight-streaming kernels and
// this is what bounds the step; at large atom counts the same kernel runs 128x64 tiles FFMA-bound.
//
//   NT (forward):   C[a][n] = sum_k A[a][k] * W[n][k]     A tile [TA][64 k], W tile [64 n][64 k]
//   NN (backward):  C[a][n] = sum_o A[a][o] * W[o][n]     A tile [TA][64 o], W tile [64 o][64 n]
// Both operands are read from global memory in their natural row-major layout (no transposed weight
// copy): every TMA box is [rows][32 floats] = rows x 128 B, swizzled so that float4 reads by 8
// consecutive rows (NT) or 8 consecutive 16-byte chunks of one row (NN) are bank-conflict free.
#include <cuda.h>
#include <string.h>

#include <algorithm>

#include "nnp_internal.h"

namespace {

constexpr int CONSUMER_WARPS = 8;
constexpr int TMA_THREADS = (CONSUMER_WARPS + 1) * 32;
constexpr int NT_ = 64;       // output columns per tile
constexpr int KC = 64;        // contraction elements per stage (two 32-wide TMA boxes)
constexpr int BOXF = 32;      // floats per TMA box row (128 B, one swizzle row)

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
__device__ __forceinline__ void prefetch_tmap(const CUtensorMap* map) {
  asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}

__device__ __forceinline__ float celu_f(float x, float alpha, float inv_alpha) { return x > 0.0f ? x : alpha * expm1f(x * inv_alpha); }
__device__ __forceinline__ float dcelu_from_h(float h, float inv_alpha) { return h > 0.0f ? 1.0f : fmaf(h, inv_alpha, 1.0f); }

// float4 at (row, 16-byte chunk) of a [rows][128 B] box written by TMA with CU_TENSOR_MAP_SWIZZLE_128B
__device__ __forceinline__ float4 lds_sw128(const unsigned char* box, int row, int chunk) {
  return *reinterpret_cast<const float4*>(box + row * 128 + ((chunk ^ (row & 7)) << 4));
}

template <int TA>
struct TileCfg {
  // warp grid (WM x WN = 8 consumer warps); lanes: 4 along atoms x 8 along columns
  static constexpr int TM = TA >= 128 ? 8 : (TA >= 32 ? 4 : (TA >= 16 ? 4 : 2));
  static constexpr int WM = TA / (4 * TM);
  static constexpr int WN = CONSUMER_WARPS / WM;
  static constexpr int TN = NT_ / (8 * WN);     // NT: columns per thread (stride 8); NN: must be 4 per 32-col box
  static_assert(WM * WN == CONSUMER_WARPS && WM >= 1, "bad warp grid");
};

}  // namespace

struct TmaGemmParams {
  CUtensorMap amap[NNP_MAX_SPECIES];
  CUtensorMap bmap[NNP_MAX_SPECIES];
  const GemmProblem* probs;
  const TmaTile* tiles;
  int n_tiles;
  int stage_bytes;  // uniform ring slot: (max tile height + 64) * KC * 4; a tile uses a prefix of its slot
  int n_stages;
};

// ------------------------------------------------------------------------------------------------
template <int TA>
__device__ __forceinline__ void run_tile_producer(const TmaGemmParams& P, const TmaTile& t,
                                                  unsigned char* ring, uint64_t* full, uint64_t* empty,
                                                  uint32_t& stage, uint32_t& phase) {
  const int nkb = (t.K + BOXF - 1) / BOXF;  // 32-wide contraction blocks
  const CUtensorMap* am = &P.amap[t.amap];
  const CUtensorMap* bm = &P.bmap[t.bmap];
  for (int kb0 = 0; kb0 < nkb; kb0 += KC / BOXF) {
    const int nb = min(KC / BOXF, nkb - kb0);
    mbar_wait(&empty[stage], phase ^ 1);
    unsigned char* sa = ring + (size_t)stage * P.stage_bytes;
    unsigned char* sb = sa + TA * KC * 4;
    if (t.transB == 0) {
      mbar_expect_tx(&full[stage], nb * (TA + NT_) * 128);
      for (int q = 0; q < nb; ++q) {
        tma_load_2d(sa + q * TA * 128, am, t.a_col0 + (kb0 + q) * BOXF, t.a_row0, &full[stage]);
        tma_load_2d(sb + q * NT_ * 128, bm, t.b_col0 + (kb0 + q) * BOXF, t.b_row0, &full[stage]);
      }
    } else {
      // W rows are the contraction index: one [64 o][32 n] box per 32 output columns
      mbar_expect_tx(&full[stage], nb * TA * 128 + (NT_ / BOXF) * KC * 128);
      for (int q = 0; q < nb; ++q)
        tma_load_2d(sa + q * TA * 128, am, t.a_col0 + (kb0 + q) * BOXF, t.a_row0, &full[stage]);
      for (int q = 0; q < NT_ / BOXF; ++q)
        tma_load_2d(sb + q * KC * 128, bm, t.b_col0 + q * BOXF, t.b_row0 + kb0 * BOXF, &full[stage]);
    }
    if (++stage == (uint32_t)P.n_stages) { stage = 0; phase ^= 1; }
  }
}

template <int TA>
__device__ __forceinline__ void run_tile_consumer(const TmaGemmParams& P, const TmaTile& t, unsigned char* ring,
                                                  uint64_t* full, uint64_t* empty, uint32_t& stage,
                                                  uint32_t& phase, int warp, int lane) {
  using C = TileCfg<TA>;
  constexpr int TM = C::TM;
  const int wm = warp / C::WN, wn = warp % C::WN;
  const int al = lane >> 3, nl = lane & 7;  // 4 atom-lanes x 8 column-lanes
  const int arow = wm * 4 * TM + al;        // this thread's atoms: arow + 4 i
  const int nkb = (t.K + BOXF - 1) / BOXF;
  const GemmProblem& p = P.probs[t.prob];  // read (from global/L1) only in the epilogue

  if (t.transB == 0) {
    // ---------------- NT: thread columns n = wn*8*TN + nl + 8 j
    constexpr int TN = C::TN;
    const int brow = wn * 8 * TN + nl;
    float acc[TM][TN];
#pragma unroll
    for (int i = 0; i < TM; ++i)
#pragma unroll
      for (int j = 0; j < TN; ++j) acc[i][j] = 0.f;
    for (int kb0 = 0; kb0 < nkb; kb0 += KC / BOXF) {
      const int nb = min(KC / BOXF, nkb - kb0);
      mbar_wait(&full[stage], phase);
      const unsigned char* sa = ring + (size_t)stage * P.stage_bytes;
      const unsigned char* sb = sa + TA * KC * 4;
      float part[TM][TN];
#pragma unroll
      for (int i = 0; i < TM; ++i)
#pragma unroll
        for (int j = 0; j < TN; ++j) part[i][j] = 0.f;
      for (int q = 0; q < nb; ++q) {
        const unsigned char* ba = sa + q * TA * 128;
        const unsigned char* bb = sb + q * NT_ * 128;
#pragma unroll
        for (int c = 0; c < 8; ++c) {
          float4 a[TM], b[TN];
#pragma unroll
          for (int i = 0; i < TM; ++i) a[i] = lds_sw128(ba, arow + 4 * i, c);
#pragma unroll
          for (int j = 0; j < TN; ++j) b[j] = lds_sw128(bb, brow + 8 * j, c);
#pragma unroll
          for (int i = 0; i < TM; ++i)
#pragma unroll
            for (int j = 0; j < TN; ++j) {
              float s = part[i][j];
              s = fmaf(a[i].x, b[j].x, s);
              s = fmaf(a[i].y, b[j].y, s);
              s = fmaf(a[i].z, b[j].z, s);
              s = fmaf(a[i].w, b[j].w, s);
              part[i][j] = s;
            }
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[stage]);
#pragma unroll
      for (int i = 0; i < TM; ++i)
#pragma unroll
        for (int j = 0; j < TN; ++j) acc[i][j] += part[i][j];
      if (++stage == (uint32_t)P.n_stages) { stage = 0; phase ^= 1; }
    }
#pragma unroll
    for (int i = 0; i < TM; ++i) {
      const int gm = t.m0 + arow + 4 * i;
      if (gm >= p.M) continue;
#pragma unroll
      for (int j = 0; j < TN; ++j) {
        const int gn = t.n0 + brow + 8 * j;
        if (gn >= p.N) continue;
        float v = acc[i][j];
        if (p.epi == EPI_BIAS_CELU) v = celu_f(v + (p.bias ? p.bias[gn] : 0.0f), p.alpha, p.inv_alpha);
        else if (p.epi == EPI_MUL_DCELU) v *= dcelu_from_h(p.aux[(size_t)gm * p.ldaux + gn], p.inv_alpha);
        else v *= p.scale;
        p.C[(size_t)gm * p.ldc + gn] = v;
      }
    }
  } else {
    // ---------------- NN: thread columns n = (wn*NB + q)*32 + 4 nl + {0..3},  NB boxes per warp
    constexpr int NB = (NT_ / BOXF) / C::WN > 0 ? (NT_ / BOXF) / C::WN : 1;
    constexpr int WN_ACTIVE = (NT_ / BOXF) / NB;  // warps along n that have work (others idle in NN)
    const bool active = wn < WN_ACTIVE;
    float acc[TM][4 * NB];
#pragma unroll
    for (int i = 0; i < TM; ++i)
#pragma unroll
      for (int j = 0; j < 4 * NB; ++j) acc[i][j] = 0.f;
    for (int kb0 = 0; kb0 < nkb; kb0 += KC / BOXF) {
      const int nb = min(KC / BOXF, nkb - kb0);
      mbar_wait(&full[stage], phase);
      const unsigned char* sa = ring + (size_t)stage * P.stage_bytes;
      const unsigned char* sb = sa + TA * KC * 4;
      if (active) {
        float part[TM][4 * NB];
#pragma unroll
        for (int i = 0; i < TM; ++i)
#pragma unroll
          for (int j = 0; j < 4 * NB; ++j) part[i][j] = 0.f;
        for (int q = 0; q < nb; ++q) {
          const unsigned char* ba = sa + q * TA * 128;
#pragma unroll
          for (int c = 0; c < 8; ++c) {
            float4 a[TM];
#pragma unroll
            for (int i = 0; i < TM; ++i) a[i] = lds_sw128(ba, arow + 4 * i, c);
#pragma unroll
            for (int tt = 0; tt < 4; ++tt) {
              const int o = q * BOXF + 4 * c + tt;  // contraction row inside the stage
#pragma unroll
              for (int b = 0; b < NB; ++b) {
                const float4 w = lds_sw128(sb + (wn * NB + b) * KC * 128, o, nl);
#pragma unroll
                for (int i = 0; i < TM; ++i) {
                  const float av = tt == 0 ? a[i].x : (tt == 1 ? a[i].y : (tt == 2 ? a[i].z : a[i].w));
                  part[i][4 * b + 0] = fmaf(av, w.x, part[i][4 * b + 0]);
                  part[i][4 * b + 1] = fmaf(av, w.y, part[i][4 * b + 1]);
                  part[i][4 * b + 2] = fmaf(av, w.z, part[i][4 * b + 2]);
                  part[i][4 * b + 3] = fmaf(av, w.w, part[i][4 * b + 3]);
                }
              }
            }
          }
        }
#pragma unroll
        for (int i = 0; i < TM; ++i)
#pragma unroll
          for (int j = 0; j < 4 * NB; ++j) acc[i][j] += part[i][j];
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[stage]);
      if (++stage == (uint32_t)P.n_stages) { stage = 0; phase ^= 1; }
    }
    if (active) {
#pragma unroll
      for (int i = 0; i < TM; ++i) {
        const int gm = t.m0 + arow + 4 * i;
        if (gm >= p.M) continue;
#pragma unroll
        for (int b = 0; b < NB; ++b) {
          const int gn0 = t.n0 + (wn * NB + b) * BOXF + 4 * nl;
          float v[4] = {acc[i][4 * b], acc[i][4 * b + 1], acc[i][4 * b + 2], acc[i][4 * b + 3]};
#pragma unroll
          for (int x = 0; x < 4; ++x) {
            const int gn = gn0 + x;
            if (gn >= p.N) continue;
            float r = v[x];
            if (p.epi == EPI_MUL_DCELU) r *= dcelu_from_h(p.aux[(size_t)gm * p.ldaux + gn], p.inv_alpha);
            else if (p.epi == EPI_BIAS_CELU) r = celu_f(r + (p.bias ? p.bias[gn] : 0.0f), p.alpha, p.inv_alpha);
            else r *= p.scale;
            p.C[(size_t)gm * p.ldc + gn] = r;
          }
        }
      }
    }
  }
}

__global__ void __launch_bounds__(TMA_THREADS, 1) gemm_tma_kernel(const __grid_constant__ TmaGemmParams P) {
  extern __shared__ __align__(1024) unsigned char smem_dyn[];
  // ring first (1024-byte aligned boxes), barriers after it
  unsigned char* ring = smem_dyn + ((1024u - (smem_u32(smem_dyn) & 1023u)) & 1023u);
  uint64_t* full = reinterpret_cast<uint64_t*>(ring + (size_t)P.n_stages * P.stage_bytes);
  uint64_t* empty = full + P.n_stages;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < P.n_stages; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], CONSUMER_WARPS);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  uint32_t stage = 0, phase = 0;
  if (warp == CONSUMER_WARPS) {
    if (lane == 0) {
      for (int ti = blockIdx.x; ti < P.n_tiles; ti += gridDim.x) {
        const TmaTile t = P.tiles[ti];
        switch (t.ta) {
          case 8: run_tile_producer<8>(P, t, ring, full, empty, stage, phase); break;
          case 16: run_tile_producer<16>(P, t, ring, full, empty, stage, phase); break;
          case 32: run_tile_producer<32>(P, t, ring, full, empty, stage, phase); break;
          default: run_tile_producer<128>(P, t, ring, full, empty, stage, phase); break;
        }
      }
    }
  } else {
    for (int ti = blockIdx.x; ti < P.n_tiles; ti += gridDim.x) {
      const TmaTile t = P.tiles[ti];
      switch (t.ta) {
        case 8: run_tile_consumer<8>(P, t, ring, full, empty, stage, phase, warp, lane); break;
        case 16: run_tile_consumer<16>(P, t, ring, full, empty, stage, phase, warp, lane); break;
        case 32: run_tile_consumer<32>(P, t, ring, full, empty, stage, phase, warp, lane); break;
        default: run_tile_consumer<128>(P, t, ring, full, empty, stage, phase, warp, lane); break;
      }
    }
  }
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

// 2-D f32 tensor [rows][cols] with row pitch ld (floats); box = [box_rows][32 floats], 128B swizzle
static int encode_map(CUtensorMap* m, const float* base, long long rows, long long cols, long long ld,
                      int box_rows) {
  EncodeTiledFn enc = get_encode();
  if (!enc) return -1;
  if (rows <= 0) rows = 1;
  cuuint64_t gdim[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
  cuuint64_t gstr[1] = {(cuuint64_t)ld * 4};
  cuuint32_t box[2] = {(cuuint32_t)BOXF, (cuuint32_t)box_rows};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, (void*)base, gdim, gstr, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? 0 : -1;
}

int tma_pick_ta(int n_rows) {
  if (n_rows <= 8) return 8;
  if (n_rows <= 16) return 16;
  if (n_rows <= 96) return 32;  // re-stream the weights per 32-atom tile while that is still cheap
  return 128;
}

static const size_t TMA_SMEM_BUDGET = 200 * 1024;  // ring + barriers + alignment slack, < 227 KB

// Build one launch (one MLP layer): `probs` are the GEMMs (one per (element[, model])), `aops`/`bops`
// describe the A / W tensors per element, `extra` places each problem inside them.
int tma_build_launch(TmaLaunch& L, const std::vector<GemmProblem>& probs, const std::vector<TmaOperand>& aops,
                     const std::vector<TmaOperand>& bops, const std::vector<TmaProbExtra>& extra, int num_sms) {
  TmaGemmParams* P = new TmaGemmParams();
  memset(P, 0, sizeof(*P));
  L.params = P;
  if (aops.size() > NNP_MAX_SPECIES || bops.size() > NNP_MAX_SPECIES) return -1;
  std::vector<int> ta_of_amap(aops.size(), 0);
  int ta_max = 8;
  for (size_t i = 0; i < aops.size(); ++i) {
    ta_of_amap[i] = tma_pick_ta((int)aops[i].rows);
    ta_max = std::max(ta_max, ta_of_amap[i]);
    if (encode_map(&P->amap[i], aops[i].base, aops[i].rows, aops[i].cols, aops[i].ld, ta_of_amap[i])) return -1;
  }
  for (size_t i = 0; i < bops.size(); ++i)
    if (encode_map(&P->bmap[i], bops[i].base, bops[i].rows, bops[i].cols, bops[i].ld, KC)) return -1;
  std::vector<TmaTile> tiles;
  for (size_t pi = 0; pi < probs.size(); ++pi) {
    const GemmProblem& p = probs[pi];
    const TmaProbExtra& x = extra[pi];
    if (p.M <= 0 || p.N <= 0) continue;
    const int ta = ta_of_amap[x.amap];
    for (int m0 = 0; m0 < p.M; m0 += ta)
      for (int n0 = 0; n0 < p.N; n0 += NT_) {
        TmaTile t;
        t.prob = (int)pi; t.m0 = m0; t.n0 = n0; t.ta = ta;
        t.K = p.K; t.transB = p.transB;
        t.amap = x.amap; t.bmap = x.bmap;
        t.a_row0 = x.a_row0 + m0; t.a_col0 = x.a_col0;
        if (p.transB == 0) { t.b_row0 = x.b_row0 + n0; t.b_col0 = 0; }
        else { t.b_row0 = x.b_row0; t.b_col0 = n0; }
        t.cost = (long long)p.K * (std::min(ta, p.M - m0) * 2 + NT_);
        tiles.push_back(t);
      }
  }
  // heavy tiles first, dealt to the persistent CTAs in snake order (static => deterministic)
  std::stable_sort(tiles.begin(), tiles.end(), [](const TmaTile& a, const TmaTile& b) { return a.cost > b.cost; });
  const size_t n = tiles.size();
  const size_t G = std::max<size_t>(1, std::min<size_t>(n, (size_t)num_sms));
  std::vector<TmaTile> ordered(n);
  for (size_t i = 0; i < n; ++i) {
    const size_t round = i / G, posn = i % G;
    const size_t cnt = std::min(G, n - round * G);
    ordered[round * G + ((round & 1) ? cnt - 1 - posn : posn)] = tiles[i];
  }
  L.n_tiles = (int)n;
  L.grid = n ? (int)G : 0;
  P->stage_bytes = (ta_max + NT_) * KC * 4;
  P->n_stages = (int)std::min<size_t>(12, (TMA_SMEM_BUDGET - 1024) / (P->stage_bytes + 16));
  L.smem_bytes = (size_t)P->n_stages * (P->stage_bytes + 16) + 1024;
  if (cudaMalloc((void**)&L.d_probs, std::max<size_t>(1, probs.size()) * sizeof(GemmProblem)) != cudaSuccess) return -1;
  if (cudaMalloc((void**)&L.d_tiles, std::max<size_t>(1, n) * sizeof(TmaTile)) != cudaSuccess) return -1;
  if (!probs.empty())
    cudaMemcpy(L.d_probs, probs.data(), probs.size() * sizeof(GemmProblem), cudaMemcpyHostToDevice);
  if (n) cudaMemcpy(L.d_tiles, ordered.data(), n * sizeof(TmaTile), cudaMemcpyHostToDevice);
  P->probs = L.d_probs;
  P->tiles = L.d_tiles;
  P->n_tiles = L.n_tiles;
  return 0;
}

void tma_launch(const TmaLaunch& L, cudaStream_t s) {
  if (L.n_tiles == 0) return;
  gemm_tma_kernel<<<L.grid, TMA_THREADS, L.smem_bytes, s>>>(*reinterpret_cast<const TmaGemmParams*>(L.params));
}

int tma_init() {
  if (!get_encode()) return -1;
  return cudaFuncSetAttribute((const void*)gemm_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)TMA_SMEM_BUDGET) == cudaSuccess ? 0 : -1;
}

void tma_free_launch(TmaLaunch& L) {
  if (L.d_probs) cudaFree(L.d_probs);
  if (L.d_tiles) cudaFree(L.d_tiles);
  delete reinterpret_cast<TmaGemmParams*>(L.params);
  L.d_probs = nullptr; L.d_tiles = nullptr; L.params = nullptr;
}

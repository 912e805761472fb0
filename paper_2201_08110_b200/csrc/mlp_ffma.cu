// Per-element atomic MLPs of the ensemble (A4 forward, A6 input-gradient backward), FP32 FFMA path.
//
// Definitions: DESIGN.md O5 (forward, CELU alpha) and O7 (chain rule through the MLP).  Atoms are
// grouped by element at create time ("the same molecule is computed repeatedly"), so each
// (element, model, layer) is one dense GEMM; one launch per layer runs all of them as a grouped GEMM
// whose tile list is built once on the host.  This file is the CUDA-core path (exact FP32 products,
// FP32 accumulation in a fixed order); it meets the 1e-3 kcal/mol/A tolerance by construction.
#include "nnp_internal.h"

constexpr int BK = 16;
constexpr int GEMM_THREADS = 256;

__device__ __forceinline__ float celu_f(float x, float alpha) { return x > 0.0f ? x : alpha * expm1f(x / alpha); }
// CELU'(x) from h = CELU(x):  x>0 -> 1;  x<=0 -> exp(x/alpha) = h/alpha + 1
__device__ __forceinline__ float dcelu_from_h(float h, float alpha) { return h > 0.0f ? 1.0f : h / alpha + 1.0f; }

template <int BM, int BN>
struct GemmSmem {
  float As[2][BK][BM + 4];
  float Bs[2][BK][BN + 4];
};

// C tile BM x BN, 16x16 threads, micro-tile TM x TN (TM = BM/16 rows of A, TN = BN/16 columns).
template <int BM, int BN>
__device__ __forceinline__ void gemm_tile(const GemmProblem& p, int m0, int n0, unsigned char* smem_raw) {
  constexpr int TM = BM / 16, TN = BN / 16;
  static_assert(TN % 4 == 0, "TN must be a multiple of 4");
  GemmSmem<BM, BN>& sm = *reinterpret_cast<GemmSmem<BM, BN>*>(smem_raw);
  const int tid = threadIdx.x;
  const int tx = tid & 15, ty = tid >> 4;

  constexpr int A_F4 = BM * BK / 4;                                // float4 loads per A tile
  constexpr int B_F4 = BN * BK / 4;
  constexpr int A_PER = (A_F4 + GEMM_THREADS - 1) / GEMM_THREADS;  // per thread
  constexpr int B_PER = (B_F4 + GEMM_THREADS - 1) / GEMM_THREADS;
  float4 ra[A_PER], rb[B_PER];

  auto load_global = [&](int k0) {
#pragma unroll
    for (int q = 0; q < A_PER; ++q) {
      const int idx = tid + q * GEMM_THREADS;
      ra[q] = make_float4(0.f, 0.f, 0.f, 0.f);
      if (idx < A_F4) {
        const int m = idx / (BK / 4), kq = idx % (BK / 4);
        const int gm = m0 + m, gk = k0 + kq * 4;
        if (gm < p.M && gk < p.K) ra[q] = *reinterpret_cast<const float4*>(p.A + (size_t)gm * p.lda + gk);
      }
    }
#pragma unroll
    for (int q = 0; q < B_PER; ++q) {
      const int idx = tid + q * GEMM_THREADS;
      rb[q] = make_float4(0.f, 0.f, 0.f, 0.f);
      if (idx < B_F4) {
        if (p.transB == 0) {  // B[n][k]
          const int n = idx / (BK / 4), kq = idx % (BK / 4);
          const int gn = n0 + n, gk = k0 + kq * 4;
          if (gn < p.N && gk < p.K) rb[q] = *reinterpret_cast<const float4*>(p.B + (size_t)gn * p.ldb + gk);
        } else {  // B[k][n]
          const int k = idx / (BN / 4), nq = idx % (BN / 4);
          const int gk = k0 + k, gn = n0 + nq * 4;
          if (gk < p.K && gn < p.N) rb[q] = *reinterpret_cast<const float4*>(p.B + (size_t)gk * p.ldb + gn);
        }
      }
    }
  };
  auto store_smem = [&](int buf) {
#pragma unroll
    for (int q = 0; q < A_PER; ++q) {
      const int idx = tid + q * GEMM_THREADS;
      if (idx < A_F4) {
        const int m = idx / (BK / 4), kq = idx % (BK / 4);
        sm.As[buf][kq * 4 + 0][m] = ra[q].x;
        sm.As[buf][kq * 4 + 1][m] = ra[q].y;
        sm.As[buf][kq * 4 + 2][m] = ra[q].z;
        sm.As[buf][kq * 4 + 3][m] = ra[q].w;
      }
    }
#pragma unroll
    for (int q = 0; q < B_PER; ++q) {
      const int idx = tid + q * GEMM_THREADS;
      if (idx < B_F4) {
        if (p.transB == 0) {
          const int n = idx / (BK / 4), kq = idx % (BK / 4);
          sm.Bs[buf][kq * 4 + 0][n] = rb[q].x;
          sm.Bs[buf][kq * 4 + 1][n] = rb[q].y;
          sm.Bs[buf][kq * 4 + 2][n] = rb[q].z;
          sm.Bs[buf][kq * 4 + 3][n] = rb[q].w;
        } else {
          const int k = idx / (BN / 4), nq = idx % (BN / 4);
          *reinterpret_cast<float4*>(&sm.Bs[buf][k][nq * 4]) = rb[q];
        }
      }
    }
  };

  float acc[TM][TN];
#pragma unroll
  for (int i = 0; i < TM; ++i)
#pragma unroll
    for (int j = 0; j < TN; ++j) acc[i][j] = 0.0f;

  const int nk = (p.K + BK - 1) / BK;
  load_global(0);
  store_smem(0);
  __syncthreads();
  for (int kt = 0; kt < nk; ++kt) {
    const int buf = kt & 1;
    if (kt + 1 < nk) load_global((kt + 1) * BK);
    // two-level accumulation: a fresh partial sum per k-tile, added to the running total once.  The
    // rounding error of a 1008-long FP32 dot product then grows with sqrt(K/BK), not sqrt(K).
    float part[TM][TN];
#pragma unroll
    for (int i = 0; i < TM; ++i)
#pragma unroll
      for (int j = 0; j < TN; ++j) part[i][j] = 0.0f;
#pragma unroll
    for (int kk = 0; kk < BK; ++kk) {
      float a[TM], b[TN];
#pragma unroll
      for (int i = 0; i < TM; ++i) a[i] = sm.As[buf][kk][ty * TM + i];
#pragma unroll
      for (int j = 0; j < TN; j += 4) {
        const float4 v = *reinterpret_cast<const float4*>(&sm.Bs[buf][kk][tx * TN + j]);
        b[j] = v.x; b[j + 1] = v.y; b[j + 2] = v.z; b[j + 3] = v.w;
      }
#pragma unroll
      for (int i = 0; i < TM; ++i)
#pragma unroll
        for (int j = 0; j < TN; ++j) part[i][j] = fmaf(a[i], b[j], part[i][j]);
    }
#pragma unroll
    for (int i = 0; i < TM; ++i)
#pragma unroll
      for (int j = 0; j < TN; ++j) acc[i][j] += part[i][j];
    if (kt + 1 < nk) {
      store_smem(buf ^ 1);
      __syncthreads();
    }
  }

  // epilogue
#pragma unroll
  for (int i = 0; i < TM; ++i) {
    const int gm = m0 + ty * TM + i;
    if (gm >= p.M) continue;
#pragma unroll
    for (int j = 0; j < TN; ++j) {
      const int gn = n0 + tx * TN + j;
      if (gn >= p.N) continue;
      float v = acc[i][j];
      if (p.epi == EPI_BIAS_CELU) {
        v = celu_f(v + (p.bias ? p.bias[gn] : 0.0f), p.alpha);
      } else if (p.epi == EPI_MUL_DCELU) {
        v *= dcelu_from_h(p.aux[(size_t)gm * p.ldaux + gn], p.alpha);
      } else {
        v *= p.scale;
      }
      p.C[(size_t)gm * p.ldc + gn] = v;
    }
  }
}

// tile configurations: cfg -> (BM, BN)
//   0: 16 x 128   1: 32 x 128   2: 64 x 64   3: 128 x 64
__global__ void __launch_bounds__(GEMM_THREADS) gemm_grouped_kernel(const GemmProblem* __restrict__ probs,
                                                                    const GemmTile* __restrict__ tiles) {
  __shared__ __align__(16) unsigned char smem_raw[sizeof(GemmSmem<128, 64>) > sizeof(GemmSmem<32, 128>)
                                                      ? sizeof(GemmSmem<128, 64>)
                                                      : sizeof(GemmSmem<32, 128>)];
  const GemmTile t = tiles[blockIdx.x];
  const GemmProblem p = probs[t.prob];
  switch (t.cfg) {
    case 0: gemm_tile<16, 128>(p, t.m0, t.n0, smem_raw); break;
    case 1: gemm_tile<32, 128>(p, t.m0, t.n0, smem_raw); break;
    case 2: gemm_tile<64, 64>(p, t.m0, t.n0, smem_raw); break;
    default: gemm_tile<128, 64>(p, t.m0, t.n0, smem_raw); break;
  }
}

static const int CFG_BM[4] = {16, 32, 64, 128};
static const int CFG_BN[4] = {128, 128, 64, 64};

// choose the tile shape per problem: the smallest padded row count wins, larger tiles on ties
void build_gemm_tiles(const std::vector<GemmProblem>& probs, std::vector<GemmTile>& tiles) {
  tiles.clear();
  for (size_t pi = 0; pi < probs.size(); ++pi) {
    const GemmProblem& p = probs[pi];
    if (p.M <= 0 || p.N <= 0) continue;
    int best = 0;
    long best_cost = -1;
    for (int c = 0; c < 4; ++c) {
      const long mp = (long)((p.M + CFG_BM[c] - 1) / CFG_BM[c]) * CFG_BM[c];
      const long np = (long)((p.N + CFG_BN[c] - 1) / CFG_BN[c]) * CFG_BN[c];
      // cost ~ padded MACs, with a mild penalty for the LDS-bound skinny tiles
      const long cost = mp * np * (c == 0 ? 5 : (c == 1 ? 4 : 3));
      if (best_cost < 0 || cost <= best_cost) { best = c; best_cost = cost; }
    }
    for (int m0 = 0; m0 < p.M; m0 += CFG_BM[best])
      for (int n0 = 0; n0 < p.N; n0 += CFG_BN[best]) tiles.push_back(GemmTile{(int)pi, m0, n0, best});
  }
}

void launch_gemm(const GemmLaunch& g, cudaStream_t s) {
  if (g.n_tiles == 0) return;
  gemm_grouped_kernel<<<g.n_tiles, GEMM_THREADS, 0, s>>>(g.d_probs, g.d_tiles);
}

// ------------------------------------------------------------------------------------------------
// Final layer (one output): e = b + w . h, and the start of the backward pass
// delta[o] = w[o] * CELU'(h[o]) written over h.  One warp per (atom, model); FP64 dot product.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) last_layer_kernel(const __grid_constant__ LastLayerArgs a) {
  const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (w >= a.n_sorted * a.M) return;
  const int row = w / a.M, m = w % a.M;
  int e = 0;
  while (e + 1 < a.S && row >= a.grp_off[e + 1]) ++e;
  const int H = a.H[e];
  const size_t hoff = a.act_off[e] + ((size_t)(row - a.grp_off[e]) * a.M + m) * H;
  float* h = a.act + hoff;
  float* hl = a.act_lo ? a.act_lo + hoff : nullptr;  // tensor engine: activations are stored split (hi, lo planes)
  const float* wv = a.W + a.w_off[e] + (size_t)m * H;
  double acc = 0.0;
  if (a.act_full) {  // tensor engine: delta was written by the forward epilogue; only the energy is left
    const float* hf = a.act_full + hoff;
    for (int o = lane; o < H; o += 32) acc += (double)wv[o] * (double)hf[o];
  } else
  for (int o = lane; o < H; o += 32) {
    const float hv = hl ? h[o] + hl[o] : h[o], ww = wv[o];  // hi + lo is exact
    acc += (double)ww * (double)hv;
    const float d = ww * dcelu_from_h(hv, a.alpha);
    if (hl) {
      const float dh = __uint_as_float((__float_as_uint(d) + 0x1000u) & 0xFFFFE000u);  // rna_tf32
      h[o] = dh;
      hl[o] = d - dh;
    } else {
      h[o] = d;
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (lane == 0) a.e_out[(size_t)row * a.M + m] = acc + (double)a.bias[a.b_off[e] + m];
}

// Tensor engine (delta already written by the forward epilogue): only the energies e[a][m] = b[m] + w[m] . h[a][m][:]
// are left, a pure read of the one-plane copy of h.  Half a warp per (atom, model): 16-byte loads, all of a lane's loads
// (up to four of h, four of w) in flight before the first use, FP64 dot product, four shuffle steps.
__global__ void __launch_bounds__(128) last_energy_kernel(const __grid_constant__ LastLayerArgs a) {
  const int hw = (blockIdx.x * blockDim.x + threadIdx.x) >> 4;  // half-warp index = (atom row, model)
  const int l16 = threadIdx.x & 15;
  const bool live = hw < a.n_sorted * a.M;
  const int row = live ? hw / a.M : 0, m = live ? hw % a.M : 0;
  int e = 0;
  while (e + 1 < a.S && row >= a.grp_off[e + 1]) ++e;
  const int H4 = a.H[e] >> 2;
  const float4* hf = reinterpret_cast<const float4*>(a.act_full + a.act_off[e] + ((size_t)(row - a.grp_off[e]) * a.M + m) * a.H[e]);
  const float4* wv = reinterpret_cast<const float4*>(a.W + a.w_off[e] + (size_t)m * a.H[e]);
  float4 x[4], w[4];
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    const int q = l16 + 16 * u;
    const bool on = live && q < H4;
    x[u] = on ? hf[q] : make_float4(0.f, 0.f, 0.f, 0.f);
    w[u] = on ? wv[q] : make_float4(0.f, 0.f, 0.f, 0.f);
  }
  double acc = 0.0;
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    acc += (double)w[u].x * (double)x[u].x;
    acc += (double)w[u].y * (double)x[u].y;
    acc += (double)w[u].z * (double)x[u].z;
    acc += (double)w[u].w * (double)x[u].w;
  }
#pragma unroll
  for (int o = 8; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (live && l16 == 0) a.e_out[(size_t)row * a.M + m] = acc + (double)a.bias[a.b_off[e] + m];
}

void launch_last_layer(nnp_handle* h, cudaStream_t s) {
  const long warps = (long)h->N * h->M;
  if (warps == 0) return;
  {
    bool wide_ok = h->last.act_full != nullptr;
    for (int e = 0; e < h->last.S; ++e) wide_ok = wide_ok && h->last.H[e] % 4 == 0 && h->last.H[e] <= 256 && h->last.act_off[e] % 4 == 0 && h->last.w_off[e] % 4 == 0;
    if (wide_ok) {
      last_energy_kernel<<<(int)((warps * 16 + 127) / 128), 128, 0, s>>>(h->last);
      return;
    }
  }
  const int blocks = (int)((warps + 3) / 4);
  last_layer_kernel<<<blocks, 128, 0, s>>>(h->last);
}

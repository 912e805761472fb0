// tcgen05 (5th-gen tensor core) GEMM engine for the per-element atomic MLPs (A4 forward, A6 backward).
//
// Mathematics: DESIGN.md O5/O7 -- the layer GEMMs  D[f][a] = sum_k W[f][k] X[a][k]  (forward, f = output
// feature, a = atom) and  D[n][a] = sum_o W[o][n] delta[a][o]  (input-gradient backward; the weights are kept
// transposed for this pass, so both passes read K-major operands).
//
// Precision ("3xTF32 from pre-split operands").  Every operand exists in global memory as two TF32-exact planes:
//   weights      hi = rna_tf32(w), lo = rna_tf32(w - hi)           (split once in nnp_create)
//   activations  hi = rna_tf32(x), lo = x - hi                     (written by the kernel that produces x)
// and a product is  hi*hi + (lo*hi + hi*lo);  the dropped lo*lo term is <= 2^-22 relative with no preferred sign.
// tcgen05 TRUNCATES when it adds into its FP32 accumulator (measured): a contraction
// accumulated entirely in TMEM is biased towards zero.  Therefore the contraction is cut into SLOTS of `kps`
// k-steps (8 contraction elements each): every slot starts a FRESH TMEM accumulator, receives its cross terms
// first (2^-11 of the result: their truncation is irrelevant) and its hi*hi terms last, and the drain warps add
// the finished slots in FP32 round-to-nearest registers.
//
// Structure: persistent CTAs (one per SM), 10 warps:
//   warp 0      TMA producer   four boxes per stage: W hi/lo [128 rows][32 floats], X hi/lo [n_pad rows][32 floats]
//   warp 1      MMA issuer     one thread: per slot 2*kps cross MMAs + kps main MMAs (kind::tf32, M = 128,
//                              N = 16..128, K = 8), then tcgen05.commit to the slot's barrier; per stage a commit
//                              that frees the operand ring entry
//   warps 2-9   drain + epilogue   tcgen05.ld of finished slots, FP32 adds, fused bias+CELU / CELU' / scale; the
//                              output is written split (hi, lo planes) when a tensor-engine launch consumes it
// Slots are self-contained, so the ring of TMEM slots runs across item boundaries: the epilogue of item i overlaps
// the MMAs of item i+1.  No shared-memory traffic other than TMA writes and tensor-core operand reads.
#include <cuda.h>
#include <string.h>

#include <algorithm>

#include "nnp_internal.h"
#include "umma_common.cuh"

namespace {

#ifndef U_ISSUERS
#define U_ISSUERS 2
#endif
constexpr int U_DRAIN_THREADS = 256;     // 8 drain warps (two per TMEM lane quarter)
constexpr int U_FIRST_DRAIN = 1 + U_ISSUERS;  // warp 0: TMA producer, then the MMA issuer warp(s), then the drain warps
constexpr int U_THREADS = 32 * U_FIRST_DRAIN + U_DRAIN_THREADS;
constexpr int U_MAX_STAGES = 6;          // operand ring depth (upper bound)
constexpr int U_MAX_SLOTS = 8;           // TMEM accumulator slots (upper bound)

}  // namespace

struct UmmaParams {
  CUtensorMap ahi[NNP_MAX_SPECIES], alo[NNP_MAX_SPECIES];  // weights of an element (hi / lo planes)
  CUtensorMap bhi[NNP_MAX_SPECIES], blo[NNP_MAX_SPECIES];  // activations of an element
  const UmmaItem* items;
  const int* cta_off;  // [grid + 1] item range of every persistent CTA
  int b_box_bytes;     // largest activation box of the launch (n_pad_max * 128), one plane
  int stage_bytes;     // 2 * A_BOX_BYTES + 2 * b_box_bytes
  int n_stages;        // operand ring depth
  int staging_rows;    // atoms per epilogue round = rows of the staging tile (min(n_pad_max, 64))
  int slot_cols;       // TMEM columns per accumulator slot (= n_pad_max)
  int n_slots;         // TMEM slot ring depth: 4 or 8
  int slot_shift;      // log2(n_slots)
  int comp;            // 1: add the expected truncation loss of a slot (one ulp away from zero, see tmem_add) back
};

__device__ __forceinline__ void drain_sync() { asm volatile("bar.sync 1, %0;" ::"n"(U_DRAIN_THREADS) : "memory"); }

// ------------------------------------------------------------------------------------------------
// drain + epilogue of one item: this thread owns feature row (TMEM lane) `quarter*32 + lane` and the atom columns
// [half*CT, half*CT + CT) of the tile; it adds the item's slots in FP32 registers.  The totals then go through a
// shared-memory staging tile [64 atoms][128 features] (one half of the tile at a time), which transposes them for
// an epilogue with 16-byte global accesses by all drain threads.
template <int NP>
__device__ __forceinline__ void drain_item(const UmmaItem& t, const UmmaParams& P, uint32_t tmem, uint64_t* slot_full,
                                           uint64_t* slot_empty, float* staging, uint32_t slot_ctr, int quarter, int half,
                                           int lane, int dt, int* split_last) {
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
  const uint32_t lane_base = tmem + ((uint32_t)(quarter * 32) << 16) + (uint32_t)col0;
  const uint32_t slot_mask = (uint32_t)P.n_slots - 1u, slot_shift = (uint32_t)P.slot_shift;
  if (t.epi == EPI_MUL_DCELU) {
    // the epilogue reads h of the layer below (written several launches ago, usually no longer in L2): start those
    // lines towards L2 now, while the tile is being accumulated, with the addresses epilogue_rows will use
    const int g = dt & 31;
    if (4 * g < t.f_valid)
      for (int r = dt >> 5; r < t.n_valid; r += U_DRAIN_THREADS / 32) {
        const size_t o = (size_t)r * t.ldaux + 4 * g;
        asm volatile("prefetch.global.L2 [%0];" ::"l"(t.aux + o));
        if (t.aux_lo) asm volatile("prefetch.global.L2 [%0];" ::"l"(t.aux_lo + o));
      }
  }
  int in_part = 0;
  for (int q = 0; q < t.nkb; ++q, ++slot_ctr) {
    const uint32_t slot = slot_ctr & slot_mask, sphase = (slot_ctr >> slot_shift) & 1u;
    mbar_wait(&slot_full[slot], sphase);
    tc_fence_after();
    if (active) {
      const uint32_t src = lane_base + (uint32_t)P.slot_cols * slot;
      if constexpr (TWO_LEVEL) {
        tmem_add_cols<CT>(src, part, (uint32_t)P.comp);
        if (++in_part == L1_SLOTS) {
#pragma unroll
          for (int j = 0; j < CT; ++j) { tot[j] += part[j]; part[j] = 0.0f; }
          in_part = 0;
        }
      } else {
        tmem_add_cols<CT>(src, tot, (uint32_t)P.comp);
      }
    }
    tc_fence_before();
    mbar_arrive(&slot_empty[slot]);
  }
  if constexpr (TWO_LEVEL) {
#pragma unroll
    for (int j = 0; j < CT; ++j) tot[j] += part[j];
  }
  // ---- epilogue, one half of the tile per round
  constexpr int ROUNDS = NP >= 32 ? 2 : 1;
  if (NP == 128 && t.split_n > 0) {
    // K-split part (EPI_SCALE): the raw partial tile goes to scratch; the part that draws the last ticket adds all
    // parts in index order and scales.  [part][atom][feature], 16-byte accesses, the thread -> element map of
    // epilogue_rows (every thread reads back only what the same thread position of the other parts wrote).
    const int g = dt & 31, r0 = dt >> 5;
    float* mine = t.scratch + (size_t)t.split_idx * 128 * 128;
#pragma unroll
    for (int h = 0; h < ROUNDS; ++h) {
      if (active && half == h) {
        float* dst = staging + quarter * 32 + lane;
#pragma unroll
        for (int j = 0; j < CT; ++j) dst[j * 128] = tot[j];
      }
      drain_sync();
      for (int r = r0; r < 64; r += U_DRAIN_THREADS / 32) st4(mine + (size_t)(h * 64 + r) * 128 + 4 * g, ld4(staging + r * 128 + 4 * g));
      drain_sync();
    }
    __threadfence();
    drain_sync();
    if (dt == 0) {
      const unsigned int ticket = atomicAdd(t.ticket, 1u);
      *split_last = ticket == (unsigned int)t.split_n - 1u;
      if (*split_last) *t.ticket = 0u;  // all parts have arrived; the next launch is ordered after this kernel
    }
    drain_sync();
    if (*split_last) {
      __threadfence();
      if (4 * g < t.f_valid)
        for (int r = r0; r < t.n_valid; r += U_DRAIN_THREADS / 32) {
          float4 x = make_float4(0.f, 0.f, 0.f, 0.f);
          for (int q = 0; q < t.split_n; ++q) {
            const float4 v = __ldcg(reinterpret_cast<const float4*>(t.scratch + ((size_t)q * 128 + r) * 128 + 4 * g));
            x.x += v.x; x.y += v.y; x.z += v.z; x.w += v.w;
          }
          x.x *= t.scale; x.y *= t.scale; x.z *= t.scale; x.w *= t.scale;
          st4(t.C + (size_t)r * t.ldc + 4 * g, x);
        }
    }
    drain_sync();  // split_last is read above and rewritten by the next split item
    return;
  }
#pragma unroll
  for (int h = 0; h < ROUNDS; ++h) {
    if (active && half == h) {
      float* dst = staging + quarter * 32 + lane;
#pragma unroll
      for (int j = 0; j < CT; ++j) dst[j * 128] = tot[j];
    }
    drain_sync();
    const int na = min(CT, t.n_valid - h * CT);
    if (na > 0) epilogue_rows<U_DRAIN_THREADS>(t, staging, h * CT, na, dt);
    drain_sync();
  }
}

__global__ void __launch_bounds__(U_THREADS, 1) gemm_umma_kernel(const __grid_constant__ UmmaParams P) {
  extern __shared__ __align__(1024) unsigned char smem_dyn[];
  unsigned char* ring = smem_dyn + ((1024u - (smem_u32(smem_dyn) & 1023u)) & 1023u);
  float* staging = reinterpret_cast<float*>(ring + (size_t)P.n_stages * P.stage_bytes);  // [<= 64 atoms][128]
  uint64_t* bars = reinterpret_cast<uint64_t*>(staging + (size_t)P.staging_rows * 128);
  uint64_t* full = bars;                            // [U_MAX_STAGES] TMA landed
  uint64_t* empty = full + U_MAX_STAGES;            // [U_MAX_STAGES] MMAs that read the stage are done
  uint64_t* slot_full = empty + U_MAX_STAGES;       // [U_MAX_SLOTS]  slot accumulated
  uint64_t* slot_empty = slot_full + U_MAX_SLOTS;   // [U_MAX_SLOTS]  slot drained
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(slot_empty + U_MAX_SLOTS);
  int* split_last = reinterpret_cast<int*>(tmem_slot + 1);  // K-split items: "this part drew the last ticket"
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < P.n_stages; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], U_ISSUERS);
    }
    for (int g = 0; g < P.n_slots; ++g) {
      mbar_init(&slot_full[g], 1);
      mbar_init(&slot_empty[g], U_DRAIN_THREADS);
    }
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
  const uint32_t slot_mask = (uint32_t)P.n_slots - 1u, slot_shift = (uint32_t)P.slot_shift;
  pdl_trigger();
  pdl_wait();  // operands come from the previous kernel of the chain

  if (warp == 0) {
    // ------------------------------------------------------------ TMA producer (warp-converged, one lane issues)
    const uint32_t leader = elect_one();
    uint32_t rs = 0, rphase = 0;
    const uint32_t ring0 = __shfl_sync(0xffffffffu, smem_u32(ring), 0);
    for (int it = it0; it < it1; ++it) {
      const UmmaItem& t = P.items[it];
      const int amap = __shfl_sync(0xffffffffu, t.amap, 0), bmap = __shfl_sync(0xffffffffu, t.bmap, 0);
      const CUtensorMap* ah = &P.ahi[amap];
      const CUtensorMap* al = &P.alo[amap];
      const CUtensorMap* bh = &P.bhi[bmap];
      const CUtensorMap* bl = &P.blo[bmap];
      const int a_c0 = __shfl_sync(0xffffffffu, t.a_c0, 0), a_c1 = __shfl_sync(0xffffffffu, t.a_c1, 0),
                b_c0 = __shfl_sync(0xffffffffu, t.b_c0, 0), b_c1 = __shfl_sync(0xffffffffu, t.b_c1, 0),
                nkb = __shfl_sync(0xffffffffu, t.nkb, 0);
      const uint32_t tx = 2u * A_BOX_BYTES + 2u * (uint32_t)__shfl_sync(0xffffffffu, t.n_pad, 0) * 128u;
      unsigned long long live = __shfl_sync(0xffffffffu, t.kmask, 0);
      const int kb_skip = __shfl_sync(0xffffffffu, t.kb_skip, 0);  // K-split part: its first box within the tile
      if (live)
        for (int q = 0; q < kb_skip; ++q) live &= live - 1;
      for (int kbi = 0; kbi < nkb; ++kbi) {
        int kb = kb_skip + kbi;
        if (live) {  // skip the contraction boxes that only hold structural zeros
          kb = __ffsll((long long)live) - 1;
          live &= live - 1;
        }
        mbar_wait(&empty[rs], rphase ^ 1u);
        if (leader) {
          const uint32_t sa = ring0 + rs * (uint32_t)P.stage_bytes;
          const uint32_t sb = sa + 2 * A_BOX_BYTES;
          const uint32_t bar = smem_u32(&full[rs]);
          asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(tx) : "memory");
          tma_load_2d_s(sa, ah, a_c0 + kb * BOXF, a_c1, bar);
          tma_load_2d_s(sb, bh, b_c0 + kb * BOXF, b_c1, bar);
          tma_load_2d_s(sa + A_BOX_BYTES, al, a_c0 + kb * BOXF, a_c1, bar);
          tma_load_2d_s(sb + (uint32_t)P.b_box_bytes, bl, b_c0 + kb * BOXF, b_c1, bar);
        }
        __syncwarp();
        if (++rs == (uint32_t)P.n_stages) { rs = 0; rphase ^= 1u; }
      }
    }
  } else if (warp < U_FIRST_DRAIN) {
    // ------------------------------------------------------------ MMA issuer warp(s); two of them alternate boxes
    // A warp runs this loop converged; every value it uses is warp-uniform (kernel parameters, loop counters,
    // broadcasts of the item fields), so descriptors and addresses live in uniform registers and the tcgen05
    // instructions of the elected lane issue back to back.  (Under `if (lane == 0)` the compiler cannot prove
    // uniformity and wraps every MMA in a register-to-uniform broadcast loop: ~200 cycles per MMA, measured.)
    // The barrier round trips of a box (operands landed, slot drained, two commits: ~600 cycles, measured) would
    // leave the tensor pipe idle between boxes if one warp did them all; boxes are independent (each fills a fresh
    // TMEM slot), so two warps take them in turn and one waits while the other issues.  The slot ring has an even
    // depth (a slot barrier is always waited on by the same warp); the stage ring may be odd, so both warps wait on
    // the "landed" barrier of every box (a parity wait cannot tell phase k from phase k - 2) and a stage is refilled
    // only after both have seen it.
    const uint32_t me = (uint32_t)(warp - 1);
    const uint32_t leader = elect_one();
    uint32_t box = 0, rs = 0, rphase = 0;
    const uint32_t n_stages = (uint32_t)P.n_stages;
    const uint32_t slot_cols = (uint32_t)P.slot_cols, stage_bytes = (uint32_t)P.stage_bytes, b_box = (uint32_t)P.b_box_bytes;
    const uint32_t ring0 = __shfl_sync(0xffffffffu, smem_u32(ring), 0);
    const uint32_t tmem_u = __shfl_sync(0xffffffffu, tmem, 0);
    const uint64_t desc_k = smem_desc(0, 16, 1024, 2);  // K-major, 128-byte swizzle (address field zero)
    for (int it = it0; it < it1; ++it) {
      const int nb = __shfl_sync(0xffffffffu, P.items[it].nkb, 0);
      const uint32_t n_pad = (uint32_t)__shfl_sync(0xffffffffu, P.items[it].n_pad, 0);
      const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((n_pad >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
      for (int b = 0; b < nb; ++b, ++box) {
        const uint32_t my_rs = rs, my_phase = rphase;
        if (++rs == n_stages) { rs = 0; rphase ^= 1u; }
        mbar_wait(&full[my_rs], my_phase);  // every box: a warp must see every phase of a barrier it waits on
        if (U_ISSUERS == 2 && (box & 1u) != me) {
          // the other warp's box: having seen it land, let the producer refill the stage (it needs both warps'
          // arrivals, so neither can be lapped on this barrier -- a lapped parity wait would never return)
          if (leader) mbar_arrive(&empty[my_rs]);
          __syncwarp();
          continue;
        }
        const uint32_t slot = box & slot_mask, sphase = (box >> slot_shift) & 1u;
        mbar_wait(&slot_empty[slot], sphase ^ 1u);
        tc_fence_after();
        const uint32_t sa = (ring0 + my_rs * stage_bytes) >> 4;
        const uint64_t ah = desc_k | sa, al = desc_k | (sa + (A_BOX_BYTES >> 4));
        const uint64_t bh = desc_k | (sa + (2 * A_BOX_BYTES >> 4)), bl = desc_k | (sa + ((2 * A_BOX_BYTES + b_box) >> 4));
        const uint32_t d = tmem_u + slot_cols * slot;
        if (leader) {
#pragma unroll
          for (uint32_t ks = 0; ks < 4; ++ks) {  // cross terms first: a fresh accumulator
            mma_tf32(d, al + 2 * ks, bh + 2 * ks, idesc, ks != 0);
            mma_tf32(d, ah + 2 * ks, bl + 2 * ks, idesc, 1u);
          }
#pragma unroll
          for (uint32_t ks = 0; ks < 4; ++ks) mma_tf32(d, ah + 2 * ks, bh + 2 * ks, idesc, 1u);
          tc_commit(&slot_full[slot]);
          tc_commit(&empty[my_rs]);  // frees the stage when these MMAs have read it
        }
        __syncwarp();
      }
    }
  } else {
    // ------------------------------------------------------------ drain + epilogue (8 warps; TMEM lane quarter = warp % 4)
    const int quarter = warp & 3, half = (warp - U_FIRST_DRAIN) >> 2, dt = threadIdx.x - 32 * U_FIRST_DRAIN;
    uint32_t slot_ctr = 0;
    for (int it = it0; it < it1; ++it) {
      const UmmaItem t = P.items[it];
      switch (t.n_pad) {
        case 16: drain_item<16>(t, P, tmem, slot_full, slot_empty, staging, slot_ctr, quarter, half, lane, dt, split_last); break;
        case 32: drain_item<32>(t, P, tmem, slot_full, slot_empty, staging, slot_ctr, quarter, half, lane, dt, split_last); break;
        case 64: drain_item<64>(t, P, tmem, slot_full, slot_empty, staging, slot_ctr, quarter, half, lane, dt, split_last); break;
        default: drain_item<128>(t, P, tmem, slot_full, slot_empty, staging, slot_ctr, quarter, half, lane, dt, split_last); break;
      }
      slot_ctr += (uint32_t)t.nkb;
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

// 2-D f32 tensor [rows][cols], row pitch ld floats; box = [box_rows][32 floats], 128-byte swizzle
static int encode_map(CUtensorMap* m, const float* base, long long rows, long long cols, long long ld, int box_rows) {
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

static int atom_tile(int n_rows, int cap) {
  int t = 16;
  while (t < cap && t < n_rows) t *= 2;
  return t;
}

// cycles of one contraction box (32 elements) of a 128 x nt tile: the larger of the tensor-pipe time (12 MMAs of
// nt/2 cycles) and the shared-memory time (operand reads of the 12 MMAs + the TMA writes, 128 B/clk)
static long long box_cycles(int nt) {
  const long long mma = 12LL * (nt / 2);
  const long long smem = (12LL * (4096 + nt * 32) + 2LL * A_BOX_BYTES + 2LL * nt * 128) / 128;
  return std::max(mma, smem) + 40;
}

static const size_t UMMA_SMEM_BUDGET = 227 * 1024;

struct UmmaPlan {
  std::vector<UmmaItem> items;
  std::vector<long long> cost;
  std::vector<int> tile_of_bmap;
  int np_max = 16;
  long long makespan = 0;
  double flops = 0;
  double bytes = 0;  // algorithmic: every operand / output plane of a problem once
};

static void plan_items(UmmaPlan& pl, const std::vector<UmmaProblem>& probs, const std::vector<UmmaOperand>& bops, int cap,
                       int num_sms) {
  pl.tile_of_bmap.assign(bops.size(), 16);
  pl.np_max = 16;
  for (size_t i = 0; i < bops.size(); ++i) {
    pl.tile_of_bmap[i] = atom_tile((int)bops[i].rows, cap);
    pl.np_max = std::max(pl.np_max, pl.tile_of_bmap[i]);
  }
  for (const UmmaProblem& p : probs) {
    if (p.n_atoms <= 0 || p.F <= 0 || p.K <= 0) continue;
    const int nt = pl.tile_of_bmap[p.bmap];
    const int nkb_all = (p.K + BOXF - 1) / BOXF;
    unsigned long long kmask = nkb_all <= 64 ? p.kmask : 0ull;
    if (nkb_all < 64) kmask &= (1ull << nkb_all) - 1ull;
    const int nkb = kmask ? __builtin_popcountll(kmask) : nkb_all;
    {
      // algorithmic bytes of the problem: both operands (hi and lo planes, the contraction boxes that are run, clipped
      // to K), the output planes and what the epilogue reads, each once; dead feature tiles excluded
      int f_live = 0;
      for (int f0 = 0; f0 < p.F; f0 += 128)
        if (!(p.fmask && f0 / 128 < 64 && !((p.fmask >> (f0 / 128)) & 1ull))) f_live += std::min(128, p.F - f0);
      const double k_live = std::min<double>(p.K, 32.0 * nkb);
      const double out_planes = (p.C_lo ? 2.0 : 1.0) + (p.C_full ? 1.0 : 0.0);
      const double aux_planes = p.aux ? (p.aux_lo ? 2.0 : 1.0) : 0.0;
      pl.bytes += 4.0 * (2.0 * k_live * ((double)f_live + p.n_atoms) + (out_planes + aux_planes) * (double)p.n_atoms * f_live);
    }
    for (int f0 = 0; f0 < p.F; f0 += 128) {
      if (p.fmask && f0 / 128 < 64 && !((p.fmask >> (f0 / 128)) & 1ull)) continue;
      for (int a0 = 0; a0 < p.n_atoms; a0 += nt) {
        UmmaItem t;
        memset(&t, 0, sizeof(t));
        t.amap = p.amap; t.bmap = p.bmap;
        t.a_c0 = p.a_c0; t.a_c1 = p.a_c1 + f0;  // (k col, feature row)
        t.b_c0 = p.b_c0; t.b_c1 = p.b_c1 + a0;
        t.nkb = nkb;
        t.kmask = kmask;
        t.n_pad = nt;
        t.n_valid = std::min(nt, p.n_atoms - a0);
        t.f_valid = std::min(128, p.F - f0);
        t.epi = p.epi;
        t.C = p.C + (size_t)a0 * p.ldc + f0;
        t.C_lo = p.C_lo ? p.C_lo + (size_t)a0 * p.ldc + f0 : nullptr;
        t.ldc = p.ldc;
        t.bias = p.bias ? p.bias + f0 : nullptr;
        t.aux = p.aux ? p.aux + (size_t)a0 * p.ldaux + f0 : nullptr;
        t.aux_lo = p.aux_lo ? p.aux_lo + (size_t)a0 * p.ldaux + f0 : nullptr;
        t.ldaux = p.ldaux;
        t.C_full = p.C_full ? p.C_full + (size_t)a0 * p.ldc + f0 : nullptr;
        t.w_last = p.w_last ? p.w_last + f0 : nullptr;
        t.scale = p.scale; t.alpha = p.alpha; t.inv_alpha = p.inv_alpha;
        pl.items.push_back(t);
        pl.cost.push_back((long long)nkb * box_cycles(nt) + 1500);
        pl.flops += 2.0 * t.f_valid * t.n_valid * 32.0 * nkb;
      }
    }
  }
  // makespan of the static schedule below (heavy first, snake order over the CTAs)
  const size_t n = pl.items.size();
  const size_t G = std::max<size_t>(1, std::min<size_t>(n, (size_t)num_sms));
  std::vector<long long> sorted(pl.cost);
  std::sort(sorted.begin(), sorted.end(), [](long long a, long long b) { return a > b; });
  std::vector<long long> load(G, 0);
  for (size_t i = 0; i < n; ++i) {
    const size_t round = i / G, posn = i % G;
    load[(round & 1) ? G - 1 - posn : posn] += sorted[i];
  }
  pl.makespan = 0;
  for (long long v : load) pl.makespan = std::max(pl.makespan, v);
}

int umma_build_launch(UmmaLaunch& L, const std::vector<UmmaProblem>& probs, const std::vector<UmmaOperand>& aops,
                      const std::vector<UmmaOperand>& bops, int num_sms, bool reverse, bool tail_split) {
  UmmaParams* P = new UmmaParams();
  memset(P, 0, sizeof(*P));
  L.params = P;
  if (aops.size() > NNP_MAX_SPECIES || bops.size() > NNP_MAX_SPECIES) return -1;
  // atom-tile width: wide tiles use the operands best (a weight box serves 128 atoms), narrow tiles fill the machine
  // when the element groups are small; take the width with the shortest estimated makespan
  UmmaPlan best;
  bool have = false;
  for (int cap : {128, 64, 32}) {
    UmmaPlan pl;
    plan_items(pl, probs, bops, cap, num_sms);
    if (!have || pl.makespan < best.makespan) { best = std::move(pl); have = true; }
  }
  for (size_t i = 0; i < bops.size(); ++i) {
    if (encode_map(&P->bhi[i], bops[i].hi, bops[i].rows, bops[i].cols, bops[i].ld, best.tile_of_bmap[i])) return -1;
    if (encode_map(&P->blo[i], bops[i].lo, bops[i].rows, bops[i].cols, bops[i].ld, best.tile_of_bmap[i])) return -1;
  }
  for (size_t i = 0; i < aops.size(); ++i) {
    if (encode_map(&P->ahi[i], aops[i].hi, aops[i].rows, aops[i].cols, aops[i].ld, 128)) return -1;
    if (encode_map(&P->alo[i], aops[i].lo, aops[i].rows, aops[i].cols, aops[i].ld, 128)) return -1;
  }
  std::vector<UmmaItem>& items = best.items;
  std::vector<long long>& cost = best.cost;
  const int np_max = best.np_max;
  // heavy items first, dealt to the persistent CTAs in snake order (static => deterministic)
  const size_t n = items.size();
  std::vector<size_t> order(n);
  for (size_t i = 0; i < n; ++i) order[i] = i;
  std::stable_sort(order.begin(), order.end(), [&](size_t a, size_t b) { return cost[a] > cost[b]; });
  // Consecutive launches of the chain sweep the (element, model) blocks in OPPOSITE directions: a launch reads what the
  // previous one wrote, and the activations of a large system are several times the L2 -- reading the most recently
  // written blocks first finds them still cached (same direction: the reader starts with the blocks that were written
  // first and are long evicted).  The price is lighter items first in every other launch (a slightly worse tail).
  if (reverse) std::reverse(order.begin(), order.end());
  const size_t G = std::max<size_t>(1, std::min<size_t>(n, (size_t)num_sms));
  std::vector<std::vector<UmmaItem>> per_cta(G);
  // Tail of a launch with few, long items (layer-1 backward: 48-64 boxes per tile, 4.1 tiles per SM at configs[2] -- a
  // fifth round for 14 of 606 tiles): the tiles that do not fill a round are cut along the contraction into split_n
  // parts on different SMs, so the last round is 1/split_n of a tile long.  The parts exchange partial tiles through
  // scratch memory; the part that arrives last adds them in index order and runs the epilogue (see UmmaItem).
  size_t n_whole = n;
  int split_n = 0;
  {
    bool scale_only = tail_split && n > 0 && np_max == 128;
    int min_nkb = 1 << 30;
    for (const UmmaItem& t : items) {
      scale_only = scale_only && t.epi == EPI_SCALE && t.n_pad == 128;
      min_nkb = std::min(min_nkb, t.nkb);
    }
    // r tiles are left after the whole rounds.  Cut into s parts each, an SM runs ceil(r s / G) parts of 1/s of a tile
    // plus the fixed cost of a part (its own drain, the scratch traffic, a fence and the ticket: about 10 boxes' worth
    // of time, measured: configs[4], 92 tiles left of 240, LOST 40 us with 8 parts and 5 us with 3) instead of one
    // tile.  Take the s <= 8 with the shortest tail, if that saves at least 5 % of a round (configs[2]: 14 tiles left
    // of 606, 8 parts, layer-1 backward 191 -> 179 us).
    const size_t r = n % G;
    if (scale_only && n >= G && r > 0 && !reverse) {
      double best = 0.95;
      const double ovh = 10.0 / (double)min_nkb;
      for (int s_try = 2; s_try <= 8 && min_nkb >= 4 * s_try; ++s_try) {
        const double tail = (double)((r * (size_t)s_try + G - 1) / G) * (1.0 / s_try + ovh);
        if (tail < best - 1e-9) { best = tail; split_n = s_try; }
      }
      if (split_n) n_whole = n - r;
    }
  }
  for (size_t i = 0; i < n_whole; ++i) {
    const size_t round = i / G, posn = i % G;
    per_cta[(round & 1) ? G - 1 - posn : posn].push_back(items[order[i]]);
  }
  if (split_n) {
    const size_t r = n - n_whole;
    L.n_split_tiles = (int)r;
    L.split_n = split_n;
    if (cudaMalloc((void**)&L.d_split_scratch, r * split_n * 128 * 128 * sizeof(float)) != cudaSuccess) return -1;
    if (cudaMalloc((void**)&L.d_split_tickets, r * sizeof(unsigned int)) != cudaSuccess) return -1;
    cudaMemset(L.d_split_tickets, 0, r * sizeof(unsigned int));
    // the parts go to the CTAs with the least work so far (all equal after whole rounds: plain order)
    std::vector<long long> load(G, 0);
    for (size_t c = 0; c < G; ++c)
      for (const UmmaItem& t : per_cta[c]) load[c] += (long long)t.nkb;
    std::vector<size_t> by_load(G);
    for (size_t c = 0; c < G; ++c) by_load[c] = c;
    std::stable_sort(by_load.begin(), by_load.end(), [&](size_t a, size_t b) { return load[a] < load[b]; });
    size_t next = 0;
    for (size_t k = 0; k < r; ++k) {
      const UmmaItem& whole = items[order[n_whole + k]];
      for (int q = 0; q < split_n; ++q) {
        UmmaItem t = whole;
        const int b0 = (int)((long long)whole.nkb * q / split_n), b1 = (int)((long long)whole.nkb * (q + 1) / split_n);
        t.kb_skip = b0;
        t.nkb = b1 - b0;
        t.split_n = split_n;
        t.split_idx = q;
        t.scratch = L.d_split_scratch + (size_t)k * split_n * 128 * 128;
        t.ticket = L.d_split_tickets + k;
        per_cta[by_load[next % G]].push_back(t);
        ++next;
      }
    }
  }
  std::vector<UmmaItem> flat;
  std::vector<int> off(G + 1, 0);
  for (size_t c = 0; c < G; ++c) {
    for (auto& t : per_cta[c]) flat.push_back(t);
    off[c + 1] = (int)flat.size();
  }
  const size_t n_flat = n_whole + (size_t)L.n_split_tiles * (size_t)L.split_n;
  L.n_items = (int)n_flat;
  L.grid = n ? (int)G : 0;
  L.tile = np_max;
  L.issued_flops = best.flops;
  L.algo_bytes = best.bytes;
  P->b_box_bytes = np_max * 128;
  P->stage_bytes = 2 * A_BOX_BYTES + 2 * P->b_box_bytes;
  const size_t bar_bytes = (2 * U_MAX_STAGES + 2 * U_MAX_SLOTS) * 8 + 16;
  P->staging_rows = std::min(np_max, 64);
  const size_t staging_bytes = (size_t)P->staging_rows * 512;  // [atoms of a round][128 features] f32
  P->n_stages = (int)std::min<size_t>(U_MAX_STAGES, (UMMA_SMEM_BUDGET - 1024 - bar_bytes - staging_bytes) / P->stage_bytes);
  L.smem_bytes = (size_t)P->n_stages * P->stage_bytes + staging_bytes + bar_bytes + 1024;
  P->slot_cols = np_max;
  P->n_slots = std::min(U_MAX_SLOTS, 512 / np_max);
  P->slot_shift = P->n_slots == 8 ? 3 : 2;
  P->comp = 1;
  if (cudaMalloc((void**)&L.d_items, std::max<size_t>(1, n_flat) * sizeof(UmmaItem)) != cudaSuccess) return -1;
  if (cudaMalloc((void**)&L.d_cta_off, (G + 1) * sizeof(int)) != cudaSuccess) return -1;
  if (n_flat) cudaMemcpy(L.d_items, flat.data(), n_flat * sizeof(UmmaItem), cudaMemcpyHostToDevice);
  cudaMemcpy(L.d_cta_off, off.data(), (G + 1) * sizeof(int), cudaMemcpyHostToDevice);
  P->items = L.d_items;
  P->cta_off = L.d_cta_off;
  return 0;
}

void umma_launch(const UmmaLaunch& L, cudaStream_t s, bool pdl) {
  if (L.n_items == 0) return;
  if (L.pair) {
    umma2_launch(L, s, pdl);
    return;
  }
  launch_kernel(pdl, gemm_umma_kernel, dim3(L.grid), dim3(U_THREADS), L.smem_bytes, s,
                *reinterpret_cast<const UmmaParams*>(L.params));
}

int umma_init() {
  if (!get_encode()) return -1;
  return cudaFuncSetAttribute((const void*)gemm_umma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)UMMA_SMEM_BUDGET) == cudaSuccess ? 0 : -1;
}

void umma_free_launch(UmmaLaunch& L) {
  if (L.d_items) cudaFree(L.d_items);
  if (L.d_cta_off) cudaFree(L.d_cta_off);
  if (L.d_split_scratch) cudaFree(L.d_split_scratch);
  if (L.d_split_tickets) cudaFree(L.d_split_tickets);
  L.d_split_scratch = nullptr;
  L.d_split_tickets = nullptr;
  if (L.pair) umma2_free_params(L);
  else delete reinterpret_cast<UmmaParams*>(L.params);
  L.d_items = nullptr; L.d_cta_off = nullptr; L.params = nullptr;
}

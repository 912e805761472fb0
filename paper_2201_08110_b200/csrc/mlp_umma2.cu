// tcgen05 GEMM engine, CTA-PAIR variant (cta_group::2) for the two layer-1 launches of large systems.
//
// Same mathematics, operands, slot structure and epilogue as mlp_umma.cu (3xTF32 from pre-split planes, a fresh TMEM
// slot per contraction box with the cross terms first, slots added in FP32 registers with the truncation
// compensation).  What changes is the tile: two CTAs of a cluster (the two SMs of a TPC) compute a 256-feature x
// 256-atom tile together.  CTA r of the pair holds the weight rows [128 r, 128 r + 128) and the activation rows
// (atoms) [128 r, 128 r + 128) of every contraction box in ITS shared memory; one tcgen05.mma.cta_group::2 of shape
// M = 256, N = 256, K = 8, issued by the leader CTA, makes both tensor cores multiply their own 128 weight rows with
// all 256 atoms, each activation half being read once and fed to both.  Per CTA and box that is 96 KB of operand reads
// and 64 KB of TMA writes for 1536 cycles of tensor time -- the one-CTA 128 x 128 box needs the same 160 KB for 768
// cycles and is therefore bound by shared-memory bandwidth (1250 of its measured 1270 cycles).
//
// STATUS: opt-in (NNP_FLAG_UMMA_PAIRS), parity-tested, and SLOWER than the one-CTA engine (configs[2] layer 1 forward
// 148 -> 266 us, backward 197 -> 345 us): a fresh accumulator per box means draining 128 lanes x 256 columns of tensor
// memory per CTA and box, and tensor-memory reads (~64 B/clk per SM) then take longer than the box's MMAs.  Kept as the
// measured evidence for DESIGN.md section 6 and as the starting point for a multi-box-per-slot variant.
//
// Protocol (all barriers live at the same shared-memory offset in both CTAs):
//   full[s]        in the LEADER: its producer expects the bytes of both CTAs; the TMA loads of both CTAs complete on
//                  it (cp.async.bulk.tensor ... cta_group::2 with the leader's barrier address)
//   empty[s]       in each CTA: the leader's tcgen05.commit.multicast arrives on both when the MMAs have read stage s
//   slot_full[j]   in each CTA (multicast commit): the CTA's drain warps read their half of the accumulator
//   slot_empty[j]  in the LEADER: one arrival per drain warp of both CTAs (remote arrivals through mapa)
// Warps: 0 TMA producer (both CTAs), 1 MMA issuer (leader only; one issuer is enough, a box is 1536 cycles of tensor
// time against ~600 of issue overhead), 2..17 drain + epilogue (TMEM lane quarter = warp % 4, 64 of the 256 columns
// each).  TMEM: 2 slots of 256 columns.
#include <string.h>

#include <algorithm>

#include "nnp_internal.h"
#include "umma_common.cuh"

namespace {

constexpr int V_DRAIN_WARPS = 16;
constexpr int V_DRAIN_THREADS = 32 * V_DRAIN_WARPS;
constexpr int V_FIRST_DRAIN = 2;
constexpr int V_THREADS = 32 * V_FIRST_DRAIN + V_DRAIN_THREADS;
constexpr int V_STAGES = 3;
constexpr int V_STAGE_BYTES = 4 * A_BOX_BYTES;  // W hi, W lo, X hi, X lo: 128 rows x 32 floats each
constexpr int V_SLOTS = 2;
constexpr int V_COLS = 256;                     // atoms of a pair tile = TMEM columns of a slot
constexpr int V_STAGING_ROWS = 64;

__device__ __forceinline__ uint32_t cluster_rank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// address of `local` (a shared::cta address of this CTA) in CTA `cta` of the cluster
__device__ __forceinline__ uint32_t map_to_cta(uint32_t local, uint32_t cta) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local), "r"(cta));
  return r;
}
// the tensor-memory reads before it are ordered by tcgen05.wait::ld + fence::before_thread_sync, so the arrival itself
// needs no cluster-scope release (which costs a GPU-wide memory barrier per call)
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
// TMA box into THIS CTA's shared memory, completion on a barrier given by its cluster address (the leader's)
__device__ __forceinline__ void tma_load_2d_pair(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar_cluster) {
  asm volatile(
      "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
      ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(bar_cluster)
      : "memory");
}
__device__ __forceinline__ void mma_tf32_pair(uint32_t d_tmem, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(d_tmem), "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
      : "memory");
}
// arrive on the barrier at this shared-memory offset in BOTH CTAs when the MMAs issued so far have completed
__device__ __forceinline__ void tc_commit_pair(uint64_t* bar) {
  asm volatile(
      "tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
      ::"r"(smem_u32(bar)), "h"((uint16_t)3)
      : "memory");
}

}  // namespace

struct Umma2Params {
  CUtensorMap ahi[NNP_MAX_SPECIES], alo[NNP_MAX_SPECIES];  // weights of an element (hi / lo planes), box 128 x 32
  CUtensorMap bhi[NNP_MAX_SPECIES], blo[NNP_MAX_SPECIES];  // activations of an element, box 128 x 32
  const UmmaItem* items;  // pair tiles: a_c1 / b_c1 / C ... are those of the pair's first feature / atom
  const int* cta_off;     // [clusters + 1] item range of every persistent CTA pair
  int comp;
};

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(V_THREADS, 1)
    gemm_umma2_kernel(const __grid_constant__ Umma2Params P) {
  extern __shared__ __align__(1024) unsigned char smem_dyn[];
  unsigned char* ring = smem_dyn + ((1024u - (smem_u32(smem_dyn) & 1023u)) & 1023u);
  float* staging = reinterpret_cast<float*>(ring + (size_t)V_STAGES * V_STAGE_BYTES);  // [64 atoms][128 features]
  uint64_t* bars = reinterpret_cast<uint64_t*>(staging + V_STAGING_ROWS * 128);
  uint64_t* full = bars;                       // [V_STAGES]  (the leader's are used)
  uint64_t* empty = full + V_STAGES;           // [V_STAGES]
  uint64_t* slot_full = empty + V_STAGES;      // [V_SLOTS]
  uint64_t* slot_empty = slot_full + V_SLOTS;  // [V_SLOTS]   (the leader's are used)
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(slot_empty + V_SLOTS);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_rank();
  if (threadIdx.x == 0) {
    for (int s = 0; s < V_STAGES; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], 1);
    }
    for (int g = 0; g < V_SLOTS; ++g) {
      mbar_init(&slot_full[g], 1);
      mbar_init(&slot_empty[g], 2 * V_DRAIN_WARPS);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {  // the same warp of both CTAs allocates the pair's tensor memory
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_slot)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  cluster_sync_all();  // barriers of both CTAs initialised before any remote arrival; also a CTA-wide barrier
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  const int cl = blockIdx.x >> 1;
  const int it0 = P.cta_off[cl], it1 = P.cta_off[cl + 1];
  pdl_trigger();
  pdl_wait();  // operands come from the previous kernel of the chain

  if (warp == 0) {
    // ------------------------------------------------------------ TMA producer (both CTAs): my 128 weight rows and my
    // 128 atoms of every box; completion on the LEADER's barrier
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
      const int a_c0 = __shfl_sync(0xffffffffu, t.a_c0, 0), a_c1 = __shfl_sync(0xffffffffu, t.a_c1, 0) + 128 * (int)rank,
                b_c0 = __shfl_sync(0xffffffffu, t.b_c0, 0), b_c1 = __shfl_sync(0xffffffffu, t.b_c1, 0) + 128 * (int)rank,
                nkb = __shfl_sync(0xffffffffu, t.nkb, 0);
      unsigned long long live = __shfl_sync(0xffffffffu, t.kmask, 0);
      for (int kbi = 0; kbi < nkb; ++kbi) {
        int kb = kbi;
        if (live) {  // skip the contraction boxes that only hold structural zeros
          kb = __ffsll((long long)live) - 1;
          live &= live - 1;
        }
        mbar_wait(&empty[rs], rphase ^ 1u);
        if (leader) {
          const uint32_t sa = ring0 + rs * (uint32_t)V_STAGE_BYTES;
          const uint32_t bar_local = smem_u32(&full[rs]);
          if (rank == 0)
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar_local), "r"(2u * V_STAGE_BYTES) : "memory");
          const uint32_t bar = map_to_cta(bar_local, 0);
          tma_load_2d_pair(sa, ah, a_c0 + kb * BOXF, a_c1, bar);
          tma_load_2d_pair(sa + 2 * A_BOX_BYTES, bh, b_c0 + kb * BOXF, b_c1, bar);
          tma_load_2d_pair(sa + A_BOX_BYTES, al, a_c0 + kb * BOXF, a_c1, bar);
          tma_load_2d_pair(sa + 3 * A_BOX_BYTES, bl, b_c0 + kb * BOXF, b_c1, bar);
        }
        __syncwarp();
        if (++rs == (uint32_t)V_STAGES) { rs = 0; rphase ^= 1u; }
      }
    }
  } else if (warp == 1) {
    // ------------------------------------------------------------ MMA issuer (leader CTA only, warp-converged)
    if (rank == 0) {
      const uint32_t leader = elect_one();
      uint32_t rs = 0, rphase = 0, slot = 0, sphase = 0;
      const uint32_t ring0 = __shfl_sync(0xffffffffu, smem_u32(ring), 0);
      const uint32_t tmem_u = __shfl_sync(0xffffffffu, tmem, 0);
      const uint64_t desc_k = smem_desc(0, 16, 1024, 2);  // K-major, 128-byte swizzle (address field zero)
      // D f32, A/B tf32, K-major, N = 256, M = 256 (the pair)
      const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(V_COLS >> 3) << 17) | ((uint32_t)(256 >> 4) << 24);
      for (int it = it0; it < it1; ++it) {
        const int nb = __shfl_sync(0xffffffffu, P.items[it].nkb, 0);
        for (int b = 0; b < nb; ++b) {
          mbar_wait(&full[rs], rphase);
          mbar_wait(&slot_empty[slot], sphase ^ 1u);
          tc_fence_after();
          const uint32_t sa = (ring0 + rs * (uint32_t)V_STAGE_BYTES) >> 4;
          const uint64_t ah = desc_k | sa, al = desc_k | (sa + (A_BOX_BYTES >> 4));
          const uint64_t bh = desc_k | (sa + (2 * A_BOX_BYTES >> 4)), bl = desc_k | (sa + (3 * A_BOX_BYTES >> 4));
          const uint32_t d = tmem_u + (uint32_t)V_COLS * slot;
          if (leader) {
#pragma unroll
            for (uint32_t ks = 0; ks < 4; ++ks) {  // cross terms first: a fresh accumulator
              mma_tf32_pair(d, al + 2 * ks, bh + 2 * ks, idesc, ks != 0);
              mma_tf32_pair(d, ah + 2 * ks, bl + 2 * ks, idesc, 1u);
            }
#pragma unroll
            for (uint32_t ks = 0; ks < 4; ++ks) mma_tf32_pair(d, ah + 2 * ks, bh + 2 * ks, idesc, 1u);
            tc_commit_pair(&slot_full[slot]);
            tc_commit_pair(&empty[rs]);
          }
          __syncwarp();
          if (++rs == (uint32_t)V_STAGES) { rs = 0; rphase ^= 1u; }
          if (++slot == (uint32_t)V_SLOTS) { slot = 0; sphase ^= 1u; }
        }
      }
    }
  } else {
    // ------------------------------------------------------------ drain + epilogue (both CTAs): my 128 feature rows
    const int quarter = warp & 3, cq = (warp - V_FIRST_DRAIN) >> 2, dt = threadIdx.x - 32 * V_FIRST_DRAIN;
    const uint32_t lane_base = tmem + ((uint32_t)(quarter * 32) << 16) + (uint32_t)(64 * cq);
    uint32_t slot = 0, sphase = 0;
    for (int it = it0; it < it1; ++it) {
      UmmaItem t = P.items[it];
      float tot[64];
#pragma unroll
      for (int j = 0; j < 64; ++j) tot[j] = 0.0f;
      for (int q = 0; q < t.nkb; ++q) {
        mbar_wait(&slot_full[slot], sphase);
        tc_fence_after();
        tmem_add_cols<64>(lane_base + (uint32_t)V_COLS * slot, tot, (uint32_t)P.comp);
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_cluster(map_to_cta(smem_u32(&slot_empty[slot]), 0));
        if (++slot == (uint32_t)V_SLOTS) { slot = 0; sphase ^= 1u; }
      }
      // my half of the pair tile: features [128 rank, 128 rank + 128)
      const int fo = 128 * (int)rank;
      t.f_valid = max(0, min(128, t.f_valid - fo));
      t.C += fo;
      if (t.C_lo) t.C_lo += fo;
      if (t.C_full) t.C_full += fo;
      if (t.bias) t.bias += fo;
      if (t.w_last) t.w_last += fo;
      if (t.aux) t.aux += fo;
      if (t.aux_lo) t.aux_lo += fo;
#pragma unroll
      for (int h = 0; h < 4; ++h) {  // 64 atoms per round through the staging tile
        if (cq == h) {
          float* dst = staging + quarter * 32 + lane;
#pragma unroll
          for (int j = 0; j < 64; ++j) dst[j * 128] = tot[j];
        }
        asm volatile("bar.sync 1, %0;" ::"n"(V_DRAIN_THREADS) : "memory");
        const int na = min(64, t.n_valid - 64 * h);
        if (na > 0) epilogue_rows<V_DRAIN_THREADS>(t, staging, 64 * h, na, dt);
        asm volatile("bar.sync 1, %0;" ::"n"(V_DRAIN_THREADS) : "memory");
      }
    }
  }
  tc_fence_before();
  cluster_sync_all();  // both CTAs are done with the pair's tensor memory and with each other's barriers
  if (warp == 1) asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, 512;" ::"r"(tmem) : "memory");
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn2)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                   const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn2 get_encode2() {
  static EncodeTiledFn2 fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn2)p;
  }
  return fn;
}

// 2-D f32 tensor [rows][cols], row pitch ld floats; box = [128 rows][32 floats], 128-byte swizzle
static int encode_map2(CUtensorMap* m, const float* base, long long rows, long long cols, long long ld) {
  EncodeTiledFn2 enc = get_encode2();
  if (!enc) return -1;
  if (rows <= 0) rows = 1;
  cuuint64_t gdim[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
  cuuint64_t gstr[1] = {(cuuint64_t)ld * 4};
  cuuint32_t box[2] = {(cuuint32_t)BOXF, 128};
  cuuint32_t estr[2] = {1, 1};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, (void*)base, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS
             ? 0 : -1;
}

static const size_t UMMA2_SMEM = (size_t)V_STAGES * V_STAGE_BYTES + (size_t)V_STAGING_ROWS * 512 +
                                 (2 * V_STAGES + 2 * V_SLOTS) * 8 + 16 + 1024;

// the pair engine takes a launch when every problem is wide enough to fill 256-atom tiles reasonably
bool umma2_suits(const std::vector<UmmaProblem>& probs) {
  if (probs.empty()) return false;
  for (const UmmaProblem& p : probs)
    if (p.n_atoms < 512 || p.K < 256) return false;
  return true;
}

int umma2_build_launch(UmmaLaunch& L, const std::vector<UmmaProblem>& probs, const std::vector<UmmaOperand>& aops,
                       const std::vector<UmmaOperand>& bops, int num_sms) {
  Umma2Params* P = new Umma2Params();
  memset(P, 0, sizeof(*P));
  L.params = P;
  L.pair = true;
  if (aops.size() > NNP_MAX_SPECIES || bops.size() > NNP_MAX_SPECIES) return -1;
  for (size_t i = 0; i < bops.size(); ++i)
    if (encode_map2(&P->bhi[i], bops[i].hi, bops[i].rows, bops[i].cols, bops[i].ld) ||
        encode_map2(&P->blo[i], bops[i].lo, bops[i].rows, bops[i].cols, bops[i].ld))
      return -1;
  for (size_t i = 0; i < aops.size(); ++i)
    if (encode_map2(&P->ahi[i], aops[i].hi, aops[i].rows, aops[i].cols, aops[i].ld) ||
        encode_map2(&P->alo[i], aops[i].lo, aops[i].rows, aops[i].cols, aops[i].ld))
      return -1;
  std::vector<UmmaItem> items;
  std::vector<long long> cost;
  double flops = 0;
  for (const UmmaProblem& p : probs) {
    if (p.n_atoms <= 0 || p.F <= 0 || p.K <= 0) continue;
    const int nkb_all = (p.K + BOXF - 1) / BOXF;
    unsigned long long kmask = nkb_all <= 64 ? p.kmask : 0ull;
    if (nkb_all < 64) kmask &= (1ull << nkb_all) - 1ull;
    const int nkb = kmask ? __builtin_popcountll(kmask) : nkb_all;
    for (int f0 = 0; f0 < p.F; f0 += 256) {
      if (p.fmask && f0 / 128 + 1 < 64 && !((p.fmask >> (f0 / 128)) & 3ull)) continue;  // both 128-feature halves dead
      for (int a0 = 0; a0 < p.n_atoms; a0 += V_COLS) {
        UmmaItem t;
        memset(&t, 0, sizeof(t));
        t.amap = p.amap; t.bmap = p.bmap;
        t.a_c0 = p.a_c0; t.a_c1 = p.a_c1 + f0;
        t.b_c0 = p.b_c0; t.b_c1 = p.b_c1 + a0;
        t.nkb = nkb;
        t.kmask = kmask;
        t.n_pad = V_COLS;
        t.n_valid = std::min(V_COLS, p.n_atoms - a0);
        t.f_valid = std::min(256, p.F - f0);
        t.epi = p.epi;
        t.C = p.C + (size_t)a0 * p.ldc + f0;
        t.C_lo = p.C_lo ? p.C_lo + (size_t)a0 * p.ldc + f0 : nullptr;
        t.C_full = p.C_full ? p.C_full + (size_t)a0 * p.ldc + f0 : nullptr;
        t.ldc = p.ldc;
        t.bias = p.bias ? p.bias + f0 : nullptr;
        t.w_last = p.w_last ? p.w_last + f0 : nullptr;
        t.aux = p.aux ? p.aux + (size_t)a0 * p.ldaux + f0 : nullptr;
        t.aux_lo = p.aux_lo ? p.aux_lo + (size_t)a0 * p.ldaux + f0 : nullptr;
        t.ldaux = p.ldaux;
        t.scale = p.scale; t.alpha = p.alpha; t.inv_alpha = p.inv_alpha;
        items.push_back(t);
        cost.push_back((long long)nkb * 1600 + 3000);
        flops += 2.0 * t.f_valid * t.n_valid * 32.0 * nkb;
      }
    }
  }
  // heavy items first, dealt to the persistent CTA pairs in snake order (static => deterministic)
  const size_t n = items.size();
  std::vector<size_t> order(n);
  for (size_t i = 0; i < n; ++i) order[i] = i;
  std::stable_sort(order.begin(), order.end(), [&](size_t a, size_t b) { return cost[a] > cost[b]; });
  const size_t G = std::max<size_t>(1, std::min<size_t>(n, (size_t)num_sms / 2));
  std::vector<std::vector<UmmaItem>> per(G);
  for (size_t i = 0; i < n; ++i) {
    const size_t round = i / G, posn = i % G;
    per[(round & 1) ? G - 1 - posn : posn].push_back(items[order[i]]);
  }
  std::vector<UmmaItem> flat;
  std::vector<int> off(G + 1, 0);
  for (size_t c = 0; c < G; ++c) {
    for (auto& t : per[c]) flat.push_back(t);
    off[c + 1] = (int)flat.size();
  }
  L.n_items = (int)n;
  L.grid = n ? (int)(2 * G) : 0;
  L.tile = V_COLS;
  L.issued_flops = flops;
  L.algo_bytes = 0;  // not accounted for the opt-in engine
  L.smem_bytes = UMMA2_SMEM;
  P->comp = 1;
  if (cudaMalloc((void**)&L.d_items, std::max<size_t>(1, n) * sizeof(UmmaItem)) != cudaSuccess) return -1;
  if (cudaMalloc((void**)&L.d_cta_off, (G + 1) * sizeof(int)) != cudaSuccess) return -1;
  if (n) cudaMemcpy(L.d_items, flat.data(), n * sizeof(UmmaItem), cudaMemcpyHostToDevice);
  cudaMemcpy(L.d_cta_off, off.data(), (G + 1) * sizeof(int), cudaMemcpyHostToDevice);
  P->items = L.d_items;
  P->cta_off = L.d_cta_off;
  return 0;
}

void umma2_launch(const UmmaLaunch& L, cudaStream_t s, bool pdl) {
  if (L.n_items == 0) return;
  launch_kernel(pdl, gemm_umma2_kernel, dim3(L.grid), dim3(V_THREADS), L.smem_bytes, s,
                *reinterpret_cast<const Umma2Params*>(L.params));  // cluster dims are compiled into the kernel
}

int umma2_init() {
  if (!get_encode2()) return -1;
  return cudaFuncSetAttribute((const void*)gemm_umma2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)UMMA2_SMEM) == cudaSuccess ? 0 : -1;
}

void umma2_free_params(UmmaLaunch& L) {
  delete reinterpret_cast<Umma2Params*>(L.params);
  L.params = nullptr;
}

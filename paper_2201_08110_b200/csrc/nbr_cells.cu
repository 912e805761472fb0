// A1 for large NNP regions: cell binning + warp-ballot compaction into the radial (5.1 A) and angular
// (3.5 A) neighbour rows (BASELINE.json north_star item (1); configs[4]: 9999 atoms).
//
// The pair predicate is the same FP64 expression as in the all-pairs kernel (O2/S1), evaluated for
// every candidate of the 27 cells around the centre's cell, so the pair sets are bit-exact by construction: the
// cell edge is Rc_radial * (1 + 1e-4), hence two atoms within Rc differ by at most one cell per axis even
// with the FP32 rounding of the cell coordinate.  Rows come out sorted by neighbour index (a rank sort
// inside the warp), i.e. exactly the rows the all-pairs kernel produces; everything downstream is unchanged and
// the summation orders stay fixed.
//
//   cell_grid_kernel   1 CTA : bounding box (FP32 min/max, order-independent), grid origin / dims / cell edge,
//                               zeroes the per-cell counters
//   cell_count_kernel  atoms : pos4, cell of every atom, rank inside the cell (integer atomics: the ORDER inside a
//                               cell is arbitrary, which is why the rows are sorted afterwards)
//   cell_scan_kernel   1 CTA : exclusive scan of the cell counts
//   cell_fill_kernel   atoms : atoms listed per cell
//   nbr_cells_kernel   warp per centre: 27-cell sweep, FP64 predicate, ballot/popc compaction, rank sort
#include <algorithm>

#include "nnp_internal.h"

#define FULLMASK 0xffffffffu

struct CellGrid {
  float ox, oy, oz, inv_edge;
  int nx, ny, nz, n_cells;
};

constexpr int CELL_MAX = 32768;    // upper bound on the number of cells (the edge grows beyond Rc if needed)
constexpr int GRID_THREADS = 1024;
constexpr int NBRC_WARPS = 4;

__device__ __forceinline__ float pos_coord(const float* pos, int stride, const int* atom_index, int i, int c, float scale) {
  const int row = atom_index ? atom_index[i] : i;
  return pos[(size_t)row * stride + c] * scale;
}

__global__ void __launch_bounds__(GRID_THREADS) cell_grid_kernel(const float* __restrict__ pos, int pos_stride,
                                                                const int* __restrict__ atom_index, int N,
                                                                float length_scale, float rc, CellGrid* __restrict__ grid,
                                                                int* __restrict__ cell_count) {
  __shared__ float smin[3][GRID_THREADS / 32], smax[3][GRID_THREADS / 32];
  pdl_trigger();
  pdl_wait();
  float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
  for (int i = threadIdx.x; i < N; i += GRID_THREADS)
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const float v = pos_coord(pos, pos_stride, atom_index, i, c, length_scale);
      if (isfinite(v)) {  // non-finite input is reported by cell_count_kernel; keep the grid sane
        lo[c] = fminf(lo[c], v);
        hi[c] = fmaxf(hi[c], v);
      }
    }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    for (int o = 16; o > 0; o >>= 1) {
      lo[c] = fminf(lo[c], __shfl_xor_sync(FULLMASK, lo[c], o));
      hi[c] = fmaxf(hi[c], __shfl_xor_sync(FULLMASK, hi[c], o));
    }
    if (lane == 0) { smin[c][warp] = lo[c]; smax[c][warp] = hi[c]; }
  }
  __syncthreads();
  __shared__ int s_ncells;
  if (threadIdx.x == 0) {
    float mn[3], mx[3];
    for (int c = 0; c < 3; ++c) {
      mn[c] = smin[c][0]; mx[c] = smax[c][0];
      for (int w = 1; w < GRID_THREADS / 32; ++w) { mn[c] = fminf(mn[c], smin[c][w]); mx[c] = fmaxf(mx[c], smax[c][w]); }
      if (!(mn[c] <= mx[c])) { mn[c] = 0.0f; mx[c] = 0.0f; }
    }
    float edge = rc * 1.0001f;
    int nx, ny, nz;
    for (;;) {
      nx = (int)floorf((mx[0] - mn[0]) / edge) + 1;
      ny = (int)floorf((mx[1] - mn[1]) / edge) + 1;
      nz = (int)floorf((mx[2] - mn[2]) / edge) + 1;
      if ((long long)nx * ny * nz <= CELL_MAX) break;
      edge *= 1.25f;
    }
    CellGrid g;
    g.ox = mn[0]; g.oy = mn[1]; g.oz = mn[2];
    g.inv_edge = 1.0f / edge;
    g.nx = nx; g.ny = ny; g.nz = nz; g.n_cells = nx * ny * nz;
    *grid = g;
    s_ncells = g.n_cells;
  }
  __syncthreads();
  for (int c = threadIdx.x; c < s_ncells; c += GRID_THREADS) cell_count[c] = 0;
}

__device__ __forceinline__ int cell_coord(float v, float o, float inv_edge, int n) {
  const float t = (v - o) * inv_edge;
  int c = isfinite(t) ? (int)floorf(t) : 0;
  return max(0, min(n - 1, c));
}

__global__ void __launch_bounds__(256) cell_count_kernel(const float* __restrict__ pos, int pos_stride,
                                                         const int* __restrict__ atom_index,
                                                         const int* __restrict__ species, int N, float length_scale,
                                                         const CellGrid* __restrict__ grid, float4* __restrict__ pos4,
                                                         int* __restrict__ cell_of, int* __restrict__ cell_rank,
                                                         int* __restrict__ cell_count, int* __restrict__ status) {
  pdl_trigger();
  pdl_wait();
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const CellGrid g = *grid;
  const float x = pos_coord(pos, pos_stride, atom_index, i, 0, length_scale);
  const float y = pos_coord(pos, pos_stride, atom_index, i, 1, length_scale);
  const float z = pos_coord(pos, pos_stride, atom_index, i, 2, length_scale);
  pos4[i] = make_float4(x, y, z, __int_as_float(species[i]));
  if (!(isfinite(x) && isfinite(y) && isfinite(z))) atomicOr(status, NNP_ST_NONFINITE);
  const int cx = cell_coord(x, g.ox, g.inv_edge, g.nx), cy = cell_coord(y, g.oy, g.inv_edge, g.ny),
            cz = cell_coord(z, g.oz, g.inv_edge, g.nz);
  const int c = (cz * g.ny + cy) * g.nx + cx;
  cell_of[i] = c;
  cell_rank[i] = atomicAdd(&cell_count[c], 1);
}

// exclusive scan of cell_count[0 .. n_cells) into cell_start[0 .. n_cells]; one CTA
__global__ void __launch_bounds__(GRID_THREADS) cell_scan_kernel(const CellGrid* __restrict__ grid,
                                                                const int* __restrict__ cell_count,
                                                                int* __restrict__ cell_start) {
  __shared__ int wsum[GRID_THREADS / 32];
  __shared__ int carry;
  pdl_trigger();
  pdl_wait();
  const int n = grid->n_cells;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  for (int base = 0; base < n; base += GRID_THREADS) {
    const int c = base + threadIdx.x;
    const int v = c < n ? cell_count[c] : 0;
    int incl = v;
    for (int o = 1; o < 32; o <<= 1) {
      const int t = __shfl_up_sync(FULLMASK, incl, o);
      if (lane >= o) incl += t;
    }
    if (lane == 31) wsum[warp] = incl;
    __syncthreads();
    if (warp == 0) {
      int w = wsum[lane];
      for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(FULLMASK, w, o);
        if (lane >= o) w += t;
      }
      wsum[lane] = w;  // inclusive over warps
    }
    __syncthreads();
    const int before = carry + (warp ? wsum[warp - 1] : 0) + incl - v;
    if (c < n) cell_start[c] = before;
    __syncthreads();
    if (threadIdx.x == GRID_THREADS - 1) carry = before + v;
    __syncthreads();
  }
  if (threadIdx.x == 0) cell_start[n] = carry;
}

// atoms in cell order: index, position and molecule side by side, so that the sweep below reads three coalesced,
// INDEPENDENT streams (index -> molecule -> position was a chain of three dependent gathers per candidate batch)
__global__ void __launch_bounds__(256) cell_fill_kernel(int N, const int* __restrict__ cell_of,
                                                        const int* __restrict__ cell_rank,
                                                        const int* __restrict__ cell_start, const float4* __restrict__ pos4,
                                                        const int* __restrict__ mol_id, int* __restrict__ cell_atoms,
                                                        float4* __restrict__ cell_pos4, int* __restrict__ cell_mol) {
  pdl_trigger();
  pdl_wait();
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int dst = cell_start[cell_of[i]] + cell_rank[i];
  cell_atoms[dst] = i;
  cell_pos4[dst] = pos4[i];
  cell_mol[dst] = mol_id[i];
}

// warp per centre; dynamic shared memory: [NBRC_WARPS][2][capR] ints (compacted row, sorted row)
__global__ void __launch_bounds__(NBRC_WARPS * 32) nbr_cells_kernel(
    const float4* __restrict__ pos4, const int* __restrict__ mol_id, const CellGrid* __restrict__ grid,
    const int* __restrict__ cell_of, const int* __restrict__ cell_start, const int* __restrict__ cell_atoms,
    const float4* __restrict__ cell_pos4, const int* __restrict__ cell_mol, int N, double rc_r2, double rc_a2, int capR, int capA, int* __restrict__ nbr_r, int* __restrict__ nbr_a,
    int* __restrict__ cnt_r, int* __restrict__ cnt_a, int* __restrict__ status) {
  extern __shared__ int rows_smem[];
  pdl_trigger();
  pdl_wait();
  const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int i = blockIdx.x * NBRC_WARPS + wib;
  if (i >= N) return;
  int* row = rows_smem + (size_t)wib * 2 * capR;
  int* sorted = row + capR;
  const CellGrid g = *grid;
  const float4 pi = pos4[i];
  const int m = mol_id[i];
  const int ci = cell_of[i];
  const int cx = ci % g.nx, cy = (ci / g.nx) % g.ny, cz = ci / (g.nx * g.ny);
  const unsigned below = (1u << lane) - 1u;
  // the nine x-runs of the 27-cell neighbourhood (the up to three cells of a run are contiguous in the cell order):
  // lane r < 9 fetches the atom range of run r, so the range lookups of all runs are one memory round trip
  int my_s0 = 0, my_s1 = 0;
  if (lane < 9) {
    const int z = cz + lane / 3 - 1, y = cy + lane % 3 - 1;
    if (z >= 0 && z < g.nz && y >= 0 && y < g.ny) {
      const int x0 = max(cx - 1, 0), x1 = min(cx + 1, g.nx - 1);
      const int c0 = (z * g.ny + y) * g.nx + x0;
      my_s0 = cell_start[c0];
      my_s1 = cell_start[c0 + (x1 - x0) + 1];
    }
  }
  int nr = 0;
  for (int run = 0; run < 9; ++run) {
    const int s0 = __shfl_sync(FULLMASK, my_s0, run), s1 = __shfl_sync(FULLMASK, my_s1, run);
    for (int base = s0; base < s1; base += 32) {
      const int idx = base + lane;
      const bool live = idx < s1;
      const int j = live ? cell_atoms[idx] : -1;
      const int mj = live ? cell_mol[idx] : -1;
      float4 pj = make_float4(0.f, 0.f, 0.f, 0.f);
      if (live) pj = cell_pos4[idx];
      bool in_r = false, in_a = false;
      if (live && j != i && mj == m) {
        const double dx = (double)pj.x - (double)pi.x;
        const double dy2 = (double)pj.y - (double)pi.y;
        const double dz2 = (double)pj.z - (double)pi.z;
        const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy2, dy2)), __dmul_rn(dz2, dz2));
        in_r = d2 <= rc_r2;
        in_a = d2 <= rc_a2;
      }
      const unsigned br = __ballot_sync(FULLMASK, in_r);
      const int slot = nr + __popc(br & below);
      if (in_r && slot < capR) row[slot] = j | (in_a ? (int)0x80000000 : 0);
      nr += __popc(br);
    }
  }
  __syncwarp();
  const int n = min(nr, capR);
  // rank sort by neighbour index (indices are unique): the rows of the all-pairs kernel
  for (int q = lane; q < n; q += 32) {
    const int v = row[q];
    const int key = v & 0x7fffffff;
    int rank = 0;
    for (int q2 = 0; q2 < n; ++q2) rank += (row[q2] & 0x7fffffff) < key;
    sorted[rank] = v;
    nbr_r[(size_t)i * capR + rank] = key;
  }
  __syncwarp();
  int na = 0;
  for (int base = 0; base < n; base += 32) {
    const int q = base + lane;
    const bool in_a = q < n && (sorted[q] < 0);
    const unsigned ba = __ballot_sync(FULLMASK, in_a);
    const int slot_a = na + __popc(ba & below);
    if (in_a && slot_a < capA) nbr_a[(size_t)i * capA + slot_a] = q;
    na += __popc(ba);
  }
  if (lane == 0) {
    if (nr > capR || na > capA) atomicOr(status, NNP_ST_CAPACITY);
    cnt_r[i] = n;
    cnt_a[i] = min(na, capA);
  }
}

// ------------------------------------------------------------------------------------------------
int cells_alloc(nnp_handle* h) {
  const size_t N = (size_t)std::max(h->N, 1);
  if (cudaMalloc((void**)&h->d_cell_grid, sizeof(CellGrid)) != cudaSuccess) return -1;
  if (cudaMalloc((void**)&h->d_cell_count, sizeof(int) * CELL_MAX) != cudaSuccess) return -1;
  if (cudaMalloc((void**)&h->d_cell_start, sizeof(int) * (CELL_MAX + 1)) != cudaSuccess) return -1;
  if (cudaMalloc((void**)&h->d_cell_of, sizeof(int) * N) != cudaSuccess) return -1;
  if (cudaMalloc((void**)&h->d_cell_rank, sizeof(int) * N) != cudaSuccess) return -1;
  if (cudaMalloc((void**)&h->d_cell_atoms, sizeof(int) * N) != cudaSuccess) return -1;
  if (cudaMalloc((void**)&h->d_cell_mol, sizeof(int) * N) != cudaSuccess) return -1;
  if (cudaMalloc((void**)&h->d_cell_pos4, sizeof(float4) * N) != cudaSuccess) return -1;
  const size_t smem = (size_t)NBRC_WARPS * 2 * h->capR * sizeof(int);
  if (smem > 48 * 1024 &&
      cudaFuncSetAttribute((const void*)nbr_cells_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
    return -1;
  return 0;
}

void cells_free(nnp_handle* h) {
  void* ptrs[] = {h->d_cell_grid, h->d_cell_count, h->d_cell_start, h->d_cell_of, h->d_cell_rank, h->d_cell_atoms,
                  h->d_cell_mol,  h->d_cell_pos4};
  for (void* p : ptrs)
    if (p) cudaFree(p);
}

void launch_neighbors_cells(nnp_handle* h, const float* d_pos, int pos_stride, const int* d_atom_index, cudaStream_t s) {
  const int N = h->N;
  CellGrid* grid = reinterpret_cast<CellGrid*>(h->d_cell_grid);
  const bool pdl = h->pdl_now;
  // the first kernel is a plain launch: it must not overtake the previous step (it rewrites what that step reads)
  launch_kernel(false, cell_grid_kernel, dim3(1), dim3(GRID_THREADS), 0, s, d_pos, pos_stride, d_atom_index, N,
                h->aev.length_scale, h->aev.rc_r, grid, h->d_cell_count);
  launch_kernel(pdl, cell_count_kernel, dim3((N + 255) / 256), dim3(256), 0, s, d_pos, pos_stride, d_atom_index,
                (const int*)h->d_species, N, h->aev.length_scale, (const CellGrid*)grid, h->d_pos4, h->d_cell_of,
                h->d_cell_rank, h->d_cell_count, h->d_status);
  launch_kernel(pdl, cell_scan_kernel, dim3(1), dim3(GRID_THREADS), 0, s, (const CellGrid*)grid,
                (const int*)h->d_cell_count, h->d_cell_start);
  launch_kernel(pdl, cell_fill_kernel, dim3((N + 255) / 256), dim3(256), 0, s, N, (const int*)h->d_cell_of,
                (const int*)h->d_cell_rank, (const int*)h->d_cell_start, (const float4*)h->d_pos4, (const int*)h->d_mol_id,
                h->d_cell_atoms, h->d_cell_pos4, h->d_cell_mol);
  const size_t smem = (size_t)NBRC_WARPS * 2 * h->capR * sizeof(int);
  launch_kernel(pdl, nbr_cells_kernel, dim3((N + NBRC_WARPS - 1) / NBRC_WARPS), dim3(NBRC_WARPS * 32), smem, s,
                (const float4*)h->d_pos4, (const int*)h->d_mol_id, (const CellGrid*)grid, (const int*)h->d_cell_of,
                (const int*)h->d_cell_start, (const int*)h->d_cell_atoms, (const float4*)h->d_cell_pos4,
                (const int*)h->d_cell_mol, N, h->aev.rc_r2, h->aev.rc_a2, h->capR, h->capA,
                h->d_nbr_r, h->d_nbr_a, h->d_cnt_r, h->d_cnt_a, h->d_status);
}

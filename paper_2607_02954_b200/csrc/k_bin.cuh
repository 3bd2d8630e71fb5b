// k_bin.cuh -- K0: bin the beads by grid cell in a canonical (run-to-run identical) order.
//
// Mechanism for S2/S5 (north_star (2): "bead sort by cell ... so global atomics are
// minimised"): the deposit and the spread are GATHERS by grid node over the bead lists of
// the 4x4 cells whose kernels reach the node, so no float atomic is ever issued and every
// node sums its contributions in one fixed order.  That order is (cell id, bead index):
//   count   : integer atomics per cell (counts do not depend on arrival order)
//   scan    : exclusive prefix sum -> cell_start
//   scatter : slot = cell_start[cell] + arrival rank   (arrival order is NOT canonical)
//   sort    : each cell's segment is sorted by bead index  -> canonical
//   pack    : per slot, the bead's 4+4 Peskin weights (SoA planes) for the gathers
#pragma once
#include "mc_common.cuh"

namespace mc {

__global__ void k_bin_count(const float2* __restrict__ X, int N, int nx, int ny,
                            int* __restrict__ cell_count, int* __restrict__ bead_cell,
                            int* __restrict__ bead_rank) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= N) return;
  const float2 p = X[b];
  const int ci = wrapi((int)floorf(p.x), nx);
  const int cj = wrapi((int)floorf(p.y), ny);
  const int c = cj * nx + ci;
  bead_cell[b] = c;
  bead_rank[b] = atomicAdd(&cell_count[c], 1);
}

// ---- exclusive scan of cell_count[n] -> cell_start[n] (+ cell_start[n] = total) ----
constexpr int SCAN_THREADS = 1024;
constexpr int SCAN_ITEMS = 4;
constexpr int SCAN_CHUNK = SCAN_THREADS * SCAN_ITEMS;

__device__ __forceinline__ int block_exclusive_scan(int v, int* smem /*[32]*/, int& total) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  int inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) smem[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    int s = (lane < (int)(blockDim.x >> 5)) ? smem[lane] : 0;
    int si = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int t = __shfl_up_sync(0xffffffffu, si, o);
      if (lane >= o) si += t;
    }
    smem[lane] = si - s;  // exclusive warp offsets
    if (lane == 31) smem[32] = si;
  }
  __syncthreads();
  total = smem[32];
  const int r = smem[wid] + inc - v;
  __syncthreads();
  return r;
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_block_sums(const int* __restrict__ in, int n,
                                                                  int* __restrict__ block_sums) {
  __shared__ int sm[33];
  const int base = blockIdx.x * SCAN_CHUNK + threadIdx.x * SCAN_ITEMS;
  int s = 0;
  if (base + SCAN_ITEMS <= n) {
    const int4 v = *reinterpret_cast<const int4*>(in + base);
    s = v.x + v.y + v.z + v.w;
  } else {
    for (int k = 0; k < SCAN_ITEMS; ++k)
      if (base + k < n) s += in[base + k];
  }
  int total;
  block_exclusive_scan(s, sm, total);
  if (threadIdx.x == 0) block_sums[blockIdx.x] = total;
}

// single block: exclusive scan of block_sums in place
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_top(int* __restrict__ block_sums, int nb) {
  __shared__ int sm[33];
  int carry = 0;
  for (int base = 0; base < nb; base += SCAN_THREADS) {
    const int i = base + threadIdx.x;
    const int v = (i < nb) ? block_sums[i] : 0;
    int total;
    const int ex = block_exclusive_scan(v, sm, total);
    if (i < nb) block_sums[i] = carry + ex;
    carry += total;
  }
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_apply(const int* __restrict__ in, int n,
                                                             const int* __restrict__ block_sums,
                                                             int* __restrict__ out, int total_all) {
  __shared__ int sm[33];
  const int base = blockIdx.x * SCAN_CHUNK + threadIdx.x * SCAN_ITEMS;
  int v[SCAN_ITEMS];
  if (base + SCAN_ITEMS <= n) {
    const int4 q = *reinterpret_cast<const int4*>(in + base);
    v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
  } else {
    for (int k = 0; k < SCAN_ITEMS; ++k) v[k] = (base + k < n) ? in[base + k] : 0;
  }
  const int s = v[0] + v[1] + v[2] + v[3];
  int total;
  int ex = block_exclusive_scan(s, sm, total) + block_sums[blockIdx.x];
  if (base + SCAN_ITEMS <= n) {
    int4 o;
    o.x = ex; o.y = ex + v[0]; o.z = o.y + v[1]; o.w = o.z + v[2];
    *reinterpret_cast<int4*>(out + base) = o;
  } else {
    for (int k = 0; k < SCAN_ITEMS; ++k) {
      if (base + k < n) out[base + k] = ex;
      ex += v[k];
    }
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) out[n] = total_all;
}

__global__ void k_bin_scatter(int N, const int* __restrict__ bead_cell, const int* __restrict__ bead_rank,
                              const int* __restrict__ cell_start, int* __restrict__ slot_bead) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= N) return;
  slot_bead[cell_start[bead_cell[b]] + bead_rank[b]] = b;
}

// canonical order inside each cell: ascending bead index (insertion sort; segments are short)
__global__ void k_bin_sort_cells(int n_cells, const int* __restrict__ cell_start, int* __restrict__ slot_bead) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n_cells) return;
  const int s = cell_start[c], e = cell_start[c + 1];
  for (int a = s + 1; a < e; ++a) {
    const int key = slot_bead[a];
    int k = a - 1;
    while (k >= s && slot_bead[k] > key) {
      slot_bead[k + 1] = slot_bead[k];
      --k;
    }
    slot_bead[k + 1] = key;
  }
}

// per slot: the 4+4 Peskin weights of the bead in that slot, planes W[0..3] = wx, W[4..7] = wy
__global__ void k_bin_pack(int N, const int* __restrict__ slot_bead, const float2* __restrict__ X,
                           float* __restrict__ W, size_t plane) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= N) return;
  const float2 p = X[slot_bead[k]];
  int i0;
  float fx, fy, w0, w1, w2, w3;
  support(p.x, i0, fx);
  support(p.y, i0, fy);
  peskin4(fx, w0, w1, w2, w3);
  W[0 * plane + k] = w0; W[1 * plane + k] = w1; W[2 * plane + k] = w2; W[3 * plane + k] = w3;
  peskin4(fy, w0, w1, w2, w3);
  W[4 * plane + k] = w0; W[5 * plane + k] = w1; W[6 * plane + k] = w2; W[7 * plane + k] = w3;
}

}  // namespace mc

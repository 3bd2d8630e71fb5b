// k_tile.cuh -- K0: bin the beads by grid TILE (north_star (2): "bead sort by cell tile
// followed by shared-memory tile accumulation, so global atomics are minimised").
//
// A tile is TS x TS nodes.  A bead is listed in every tile its 4x4 Peskin support, widened by a
// SKIN (a quarter node of bead motion in every direction), overlaps (1, 2 or 4 tiles), so a tile's CTA can accumulate ALL
// contributions to its own nodes from its own list and never writes outside the tile: no global
// float atomics, no halo exchange.  The skin makes a list valid for many steps: K4 records the
// largest bead displacement component of every step, the policy (list_rebuild_due, below)
// adds it to the drift accumulated since the lists were built and orders a rebuild only when
// the drift could reach the skin; until then the K0 kernels return at once.  Entries
// whose support no longer (or not yet) overlaps the tile add exact zeros (k_p2g.cuh), so the
// schedule touches the results only through the per-tile fixed-point scales (powers of two
// chosen from the list lengths), i.e. at rounding level; it is a function of the state alone,
// so runs stay bit-reproducible and mc_step(a), mc_step(b) equals mc_step(a + b).
//   count  : per bead, +1 on each overlapped tile (integer atomics, warp-aggregated) and +1 on
//            the (tile, bank key) bucket
//   scan   : exclusive prefix sum over the tiles (one block; there are few tiles)
//   starts : one warp per tile turns its 32 bucket counts into cursors inside the tile's segment
//   fill   : per bead, claim a slot in each overlapped tile's bucket and store the bead index
// A tile's list is thus ordered by the BANK KEY of its entries: the shared-memory bank of the
// first accumulator node a bead touches (bead_key).  The consumers (k_p2g.cuh) deal the sorted
// entries to the lanes so that the lanes of one atomic instruction hold different keys, i.e.
// land on different banks (arrival order made them collide ~3.4-fold).  Stale keys (beads move
// between rebuilds) cost a few conflicts, never correctness.  The order inside a bucket is the
// arrival order of the atomics and is NOT reproducible; that is harmless because the
// accumulation that consumes the lists adds integers (fixed point), which is order-independent.
#pragma once
#include <cooperative_groups.h>

#include "mc_common.cuh"

namespace mc {

constexpr int TS = 32;          // tile side in nodes
// Shared accumulator of a tile (k_p2g.cuh): the TS x TS nodes plus a HALO of 4 on every side, so
// that every support of a listed bead (first node within [-4, TS] of the tile origin, skin
// included) fits and the 16 contributions go to base + constant offsets with no clamping; halo
// sums are dropped (the neighbouring tiles accumulate them from their own lists).  Row pitch 41
// = 9 (mod 32): the 16 nodes of a support lie on 16 different banks.
constexpr int HALO = 4;
constexpr int AW = TS + 2 * HALO;
constexpr int TSP = 41;
constexpr int ACC_N = AW * TSP;
constexpr float LIST_SKIN = 0.25f;  // a bead is listed as if it sat anywhere within +-LIST_SKIN of its position
constexpr float LIST_DRIFT_MAX = 0.22f;  // rebuild when the accumulated drift bound exceeds this (< LIST_SKIN)

// device-side list state, in the world's flag words
struct ListState {
  int need;            // 1: the K0 kernels of this step rebuild the lists
  float drift;         // bound on the per-axis displacement of any listed point since the lists were built
  unsigned step_max;   // bits of max |U_x|,|U_y| over the beads in the last step (K4, atomicMax)
  unsigned step_max_p; // ... of the projection displacement of the last step (k_pbd.cuh; 0 without pbd_project)
  unsigned step_max_m; // ... of the change of the two-layer marker offsets (k_pbd.cuh; 0 without two_layer)
};

// The policy is evaluated where it is needed instead of in a launch of its own: the count pass
// (first K0 kernel) only READS the state and every thread derives the same decision; the scan
// kernel (one block, next in the stream) then commits it -- st->need for the kernels after it,
// the new drift, step_max = 0 for this step's K4.
__device__ __forceinline__ bool list_rebuild_due(const ListState* st, float* drift_out) {
  // a listed point moves by at most the sum of the three per-step bounds (triangle inequality)
  const float d = st->drift + (__uint_as_float(st->step_max) + __uint_as_float(st->step_max_p) +
                               __uint_as_float(st->step_max_m));
  *drift_out = d;
  return !(d <= LIST_DRIFT_MAX);  // also true for NaN
}
__device__ __forceinline__ void list_policy_commit(ListState* st) {
  float d;
  const bool need = list_rebuild_due(st, &d);
  st->step_max = 0u;
  st->step_max_p = 0u;
  st->step_max_m = 0u;
  st->need = need ? 1 : 0;
  st->drift = need ? 0.0f : d;
}

// The (up to 4) tiles overlapped by the skinned support of a bead at (x,y): tiles of the first
// and the last listed node along each axis (periodic).  Returns the number of distinct tiles.
__device__ __forceinline__ int bead_tiles(float x, float y, int nx, int ny, int ntx, int t[4]) {
  // first and last node any support can reach while the bead stays within the skin
  const int ia = (int)floorf(x - LIST_SKIN) - 1, ja = (int)floorf(y - LIST_SKIN) - 1;
  const int wx = (int)floorf(x + LIST_SKIN) + 2 - ia, wy = (int)floorf(y + LIST_SKIN) + 2 - ja;  // 3 or 4
  const int i0 = wrapi(ia, nx), j0 = wrapi(ja, ny);
  const int i3 = (i0 + wx >= nx) ? i0 + wx - nx : i0 + wx, j3 = (j0 + wy >= ny) ? j0 + wy - ny : j0 + wy;
  const int txa = i0 / TS, txb = i3 / TS, tya = j0 / TS, tyb = j3 / TS;
  int n = 0;
  t[n++] = tya * ntx + txa;
  if (txb != txa) t[n++] = tya * ntx + txb;
  if (tyb != tya) {
    t[n++] = tyb * ntx + txa;
    if (txb != txa) t[n++] = tyb * ntx + txb;
  }
  return n;
}

// Bank key of a bead: accumulator address of support node (r, c) is (j0 + r) * TSP + i0 + c (+ a
// constant) with (i0, j0) the first support node relative to the tile origin; tile origins and
// the periods nx, ny are multiples of 32, so the bank is key + TSP r + c (mod 32) with this key
// for every tile the bead is listed in.
__device__ __forceinline__ int bead_key(float x, float y) {
  return ((TSP & 31) * ((int)floorf(y) - 1) + (int)floorf(x) - 1) & 31;
}

// warp-aggregated atomicAdd(&ctr[key], 1) for the lanes with act set; returns the claimed value
__device__ __forceinline__ int warp_claim(int* ctr, int key, bool act) {
  const unsigned m = __ballot_sync(0xffffffffu, act);
  int slot = 0;
  if (act) {
    const unsigned peers = __match_any_sync(m, key);
    const int lane = threadIdx.x & 31;
    const int leader = __ffs(peers) - 1;
    int base = 0;
    if (lane == leader) base = atomicAdd(&ctr[key], __popc(peers));
    base = __shfl_sync(peers, base, leader);
    slot = base + __popc(peers & ((1u << lane) - 1u));
  }
  return slot;
}

// The four phases of a rebuild as device functions over the threads of the calling grid (a
// 1-block grid is allowed), so that the per-phase kernels of large worlds and the one-CTA kernel
// of small worlds share them.

// FILL = false: tile_ctr[t] += 1 and (if given) bucket_ctr[32 t + key] += 1 per listed bead.
// FILL = true: bucket_ctr holds the running cursors (bucket_starts) and the bead index is
// stored at the claimed slot.
// O != NULL (two-layer broadcast, reading 28): the listed items are the 2 N MARKERS, item 2 b + s
// at X_b + O_b (s = 0) or X_b - O_b (s = 1).  Rounding the marker to fp32 here is harmless: the
// lists only have to cover the support within the skin (the consumers form it exactly).
template <bool FILL>
__device__ __forceinline__ void tile_bin(const float2* __restrict__ X, const float2* __restrict__ O, int N, int nx, int ny,
                                         int* __restrict__ tile_ctr, int* __restrict__ bucket_ctr,
                                         int* __restrict__ list) {
  const int n_items = O ? 2 * N : N;
  // grid-stride over whole blocks of items: every lane of a warp takes part in warp_claim
  for (int base = blockIdx.x * blockDim.x; base < n_items; base += gridDim.x * blockDim.x) {
    const int b = base + threadIdx.x;
    int t[4] = {0, 0, 0, 0};
    int n = 0, key = 0;
    if (b < n_items) {
      float2 p;
      if (O) {
        p = X[b >> 1];
        const float2 o = O[b >> 1];
        p.x += (b & 1) ? -o.x : o.x;
        p.y += (b & 1) ? -o.y : o.y;
      } else {
        p = X[b];
      }
      n = bead_tiles(p.x, p.y, nx, ny, nx / TS, t);
      key = bead_key(p.x, p.y);
    }
#pragma unroll
    for (int s = 0; s < 4; ++s) {
      if (FILL) {
        if (s < n) list[atomicAdd(&bucket_ctr[32 * t[s] + key], 1)] = b;
      } else {
        // 77 % of the points lie in one tile only: skip the claim rounds no lane of the warp needs
        if (s > 0 && !__any_sync(0xffffffffu, s < n)) break;
        warp_claim(tile_ctr, t[s], s < n);
        if (bucket_ctr && s < n) atomicAdd(&bucket_ctr[32 * t[s] + key], 1);
      }
    }
  }
}

// one warp per tile: bucket_cursor[32 t + k] = tile_start[t] + exclusive scan of the tile's 32
// bucket counts; the counts are zeroed for the next rebuild.
__device__ __forceinline__ void bucket_starts(int n_tiles, const int* __restrict__ tile_start,
                                              int* __restrict__ bucket_count, int* __restrict__ bucket_cursor) {
  const int lane = threadIdx.x & 31;
  const int warps = (gridDim.x * blockDim.x) >> 5;
  for (int t = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; t < n_tiles; t += warps) {
    const int v = bucket_count[32 * t + lane];
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int u = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += u;
    }
    bucket_cursor[32 * t + lane] = tile_start[t] + inc - v;
    bucket_count[32 * t + lane] = 0;
  }
}

// Crowded tiles (config 5): the tiles whose list exceeds CROWDED_N entries are handed to a cluster
// launch of their own (k_cluster.cuh) that runs BESIDE the one-CTA-per-tile launch on a second
// stream; the table is rebuilt with the lists.  crowded[r] = tile id of rank r, crowded_rank[t] = r or
// -1, *n_crowded = their number.  The ranks depend on the arrival order of the atomics, i.e. which
// crowded tile gets which cluster is not reproducible -- harmless: every tile's result is the same
// integer sum whoever computes it.
constexpr int CROWDED_N = 1024;
struct CrowdedTable {
  int* crowded;       // [n_tiles]
  int* crowded_rank;  // [n_tiles]
  int* n_crowded;     // [1]
};

// ONE block of 1024 threads: tile_start = exclusive scan of tile_count (n_tiles + 1 entries);
// counts are zeroed for the next rebuild.  sm: 33 ints of shared memory.
__device__ __forceinline__ void tile_scan(int* __restrict__ tile_count, int n_tiles, int* __restrict__ tile_start,
                                          int* sm, CrowdedTable ct = CrowdedTable{nullptr, nullptr, nullptr}) {
  // Each WARP owns a contiguous segment of the tiles (a multiple of 32 long): coalesced sums of the
  // segment, one block-wide scan of the 32 segment totals, then a second coalesced pass with a
  // running carry and a warp scan per row of 32 -- two barriers whatever the number of tiles (the
  // chunked version paid three per 1024 tiles: 40 us on world 4d's 38,416 tiles).
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int seg = (((n_tiles + 31) / 32 + 31) / 32) * 32;  // tiles per warp
  const int s0 = wid * seg, s1 = min(s0 + seg, n_tiles);
  int total = 0;
  for (int i = s0 + lane; i < s1; i += 32) total += tile_count[i];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) total += __shfl_xor_sync(0xffffffffu, total, o);
  if (lane == 0) sm[wid] = total;
  __syncthreads();
  if (wid == 0) {
    const int sv = sm[lane];
    int si = sv;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int u = __shfl_up_sync(0xffffffffu, si, o);
      if (lane >= o) si += u;
    }
    sm[lane] = si - sv;
    if (lane == 31) sm[32] = si;
  }
  __syncthreads();
  int run = sm[wid];  // exclusive prefix of this warp's segment
  for (int base = s0; base < s1; base += 32) {
    const int i = base + lane;
    const int v = (i < s1) ? tile_count[i] : 0;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int u = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += u;
    }
    if (i < s1) {
      tile_start[i] = run + inc - v;
      tile_count[i] = 0;
    }
    run += __shfl_sync(0xffffffffu, inc, 31);
  }
  const int carry = sm[32];
  if (threadIdx.x == 0) tile_start[n_tiles] = carry;
  if (ct.crowded) {
    // ranks in (roughly) DESCENDING order of list length -- 64 linear buckets between CROWDED_N and
    // the longest list: the cluster launch is dispatched in rank order, and starting the heaviest
    // tiles first evens out the SMs (config 5: busiest SM 151 k cycles against 90 k on average with
    // ranks in tile order)
    __shared__ int hist[64], cursor[64], longest;
    if (threadIdx.x < 64) hist[threadIdx.x] = 0;
    if (threadIdx.x == 0) longest = CROWDED_N + 1;
    __syncthreads();  // also makes tile_start visible to the whole block
    for (int i = threadIdx.x; i < n_tiles; i += 1024) atomicMax(&longest, tile_start[i + 1] - tile_start[i]);
    __syncthreads();
    const int span = longest - CROWDED_N;
    auto bucket = [&](int n) { return 63 - min(63, (int)(((long long)(n - CROWDED_N - 1) * 64) / span)); };  // 0 = longest
    for (int i = threadIdx.x; i < n_tiles; i += 1024) {
      const int n = tile_start[i + 1] - tile_start[i];
      if (n > CROWDED_N) atomicAdd(&hist[bucket(n)], 1);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      int run = 0;
      for (int b = 0; b < 64; ++b) { cursor[b] = run; run += hist[b]; }
      *ct.n_crowded = run;
    }
    __syncthreads();
    for (int i = threadIdx.x; i < n_tiles; i += 1024) {
      const int n = tile_start[i + 1] - tile_start[i];
      int r = -1;
      if (n > CROWDED_N) {
        r = atomicAdd(&cursor[bucket(n)], 1);
        ct.crowded[r] = i;
      }
      ct.crowded_rank[i] = r;
    }
  }
}

template <bool FILL>
__global__ void __launch_bounds__(256) k_tile_bin(const ListState* __restrict__ st, const float2* __restrict__ X,
                                                  const float2* __restrict__ O, int N, int nx, int ny,
                                                  int* __restrict__ tile_ctr, int* __restrict__ bucket_ctr,
                                                  int* __restrict__ list, size_t wstride) {
  const size_t ws = blockIdx.y * wstride;
  st = wshift(st, ws); X = wshift(X, ws); O = wshift(O, ws); tile_ctr = wshift(tile_ctr, ws);
  bucket_ctr = wshift(bucket_ctr, ws); list = wshift(list, ws);
  if (FILL) {
    if (!st->need) return;
  } else {
    float d;
    if (!list_rebuild_due(st, &d)) return;
  }
  tile_bin<FILL>(X, O, N, nx, ny, tile_ctr, bucket_ctr, list);
}

__global__ void __launch_bounds__(256) k_bucket_starts(const ListState* __restrict__ st, int n_tiles,
                                                       const int* __restrict__ tile_start,
                                                       int* __restrict__ bucket_count,
                                                       int* __restrict__ bucket_cursor, size_t wstride) {
  const size_t ws = blockIdx.y * wstride;
  st = wshift(st, ws); tile_start = wshift(tile_start, ws); bucket_count = wshift(bucket_count, ws);
  bucket_cursor = wshift(bucket_cursor, ws);
  if (!st->need) return;
  bucket_starts(n_tiles, tile_start, bucket_count, bucket_cursor);
}

__global__ void __launch_bounds__(1024) k_tile_scan(ListState* __restrict__ st, int* __restrict__ tile_count,
                                                    int n_tiles, int* __restrict__ tile_start, CrowdedTable ct,
                                                    size_t wstride) {
  const size_t ws = blockIdx.y * wstride;
  st = wshift(st, ws); tile_count = wshift(tile_count, ws); tile_start = wshift(tile_start, ws);
  ct.crowded = wshift(ct.crowded, ws); ct.crowded_rank = wshift(ct.crowded_rank, ws); ct.n_crowded = wshift(ct.n_crowded, ws);
  __shared__ int sm[33];
  __shared__ int need_s;
  if (threadIdx.x == 0) {
    list_policy_commit(st);
    need_s = st->need;
  }
  __syncthreads();
  if (!need_s) return;
  tile_scan(tile_count, n_tiles, tile_start, sm, ct);
}

// Small worlds (bound by launch overhead, not by work): the whole of K0 in ONE launch of one
// 1024-thread CTA -- policy, count, scan, bucket starts, fill, separated by __syncthreads()
// (global atomics and stores of a block are visible to the same block after the barrier).
__global__ void __launch_bounds__(1024) k_list_build_small(ListState* __restrict__ st, const float2* __restrict__ X,
                                                           const float2* __restrict__ O, int N, int nx, int ny,
                                                           int n_tiles, int* __restrict__ tile_count,
                                                           int* __restrict__ tile_start, int* __restrict__ bucket_count,
                                                           int* __restrict__ bucket_cursor, int* __restrict__ list,
                                                           CrowdedTable ct, size_t wstride) {
  // one CTA per world: blockIdx.x is always 0 here, the world index rides in blockIdx.y
  const size_t ws = blockIdx.y * wstride;
  ct.crowded = wshift(ct.crowded, ws); ct.crowded_rank = wshift(ct.crowded_rank, ws); ct.n_crowded = wshift(ct.n_crowded, ws);
  st = wshift(st, ws); X = wshift(X, ws); O = wshift(O, ws); tile_count = wshift(tile_count, ws);
  tile_start = wshift(tile_start, ws); bucket_count = wshift(bucket_count, ws);
  bucket_cursor = wshift(bucket_cursor, ws); list = wshift(list, ws);
  __shared__ int sm[33];
  __shared__ int need_s;
  if (threadIdx.x == 0) {
    list_policy_commit(st);
    need_s = st->need;
  }
  __syncthreads();
  if (!need_s) return;
  tile_bin<false>(X, O, N, nx, ny, tile_count, bucket_count, nullptr);
  __syncthreads();
  tile_scan(tile_count, n_tiles, tile_start, sm, ct);
  __syncthreads();
  bucket_starts(n_tiles, tile_start, bucket_count, bucket_cursor);
  __syncthreads();
  tile_bin<true>(X, O, N, nx, ny, nullptr, bucket_cursor, list);
}

// Medium worlds (up to a few hundred thousand beads: still bound by launch overhead on the steps
// that keep their lists, too many beads for one CTA on the steps that rebuild them): the whole of
// K0 in ONE launch of one thread-block CLUSTER of 8 x 1024 threads.  The phases are separated by
// the hardware cluster barrier (release/acquire at cluster scope, which also orders the global
// atomics and stores of the phases); the CTAs of a cluster are co-scheduled by construction, so
// unlike a hand-made grid barrier this cannot deadlock.
constexpr int K0_CLUSTER = 8;
__global__ void __cluster_dims__(K0_CLUSTER, 1, 1) __launch_bounds__(1024)
    k_list_build_cluster(ListState* __restrict__ st, const float2* __restrict__ X, const float2* __restrict__ O, int N,
                         int nx, int ny, int n_tiles, int* __restrict__ tile_count, int* __restrict__ tile_start,
                         int* __restrict__ bucket_count, int* __restrict__ bucket_cursor, int* __restrict__ list,
                         CrowdedTable ct, size_t wstride) {
  // one cluster per world: blockIdx.x = rank in the cluster, blockIdx.y = world
  const size_t ws = blockIdx.y * wstride;
  ct.crowded = wshift(ct.crowded, ws); ct.crowded_rank = wshift(ct.crowded_rank, ws); ct.n_crowded = wshift(ct.n_crowded, ws);
  st = wshift(st, ws); X = wshift(X, ws); O = wshift(O, ws); tile_count = wshift(tile_count, ws);
  tile_start = wshift(tile_start, ws); bucket_count = wshift(bucket_count, ws);
  bucket_cursor = wshift(bucket_cursor, ws); list = wshift(list, ws);
  namespace cg = cooperative_groups;
  cg::cluster_group cl = cg::this_cluster();
  __shared__ int sm[33];
  if (blockIdx.x == 0 && threadIdx.x == 0) list_policy_commit(st);
  cl.sync();
  if (!*reinterpret_cast<volatile int*>(&st->need)) return;  // the same value in every CTA: all leave together
  tile_bin<false>(X, O, N, nx, ny, tile_count, bucket_count, nullptr);
  cl.sync();
  if (blockIdx.x == 0) tile_scan(tile_count, n_tiles, tile_start, sm, ct);
  cl.sync();
  bucket_starts(n_tiles, tile_start, bucket_count, bucket_cursor);
  cl.sync();
  tile_bin<true>(X, O, N, nx, ny, nullptr, bucket_cursor, list);
}

// Large single worlds: the whole of K0 in ONE cooperative launch (grid barrier between the phases; all
// CTAs co-resident by construction of a cooperative launch) instead of four launches, three of which
// only return on the ~10 of 11 steps that keep their lists: on worlds of a million beads the launch
// boundaries of those empty kernels are 5 % of the step.  Nobody writes the list state while the grid
// decides (every thread derives the same decision from it); the LAST CTA to leave commits the policy
// (an exit counter, reset by that CTA).  grid = resident CTAs of 1024 threads (host: occupancy query).
__global__ void __launch_bounds__(1024) k_list_build_coop(ListState* __restrict__ st, int* __restrict__ exit_ctr,
                                                          const float2* __restrict__ X, const float2* __restrict__ O,
                                                          int N, int nx, int ny, int n_tiles, int* __restrict__ tile_count,
                                                          int* __restrict__ tile_start, int* __restrict__ bucket_count,
                                                          int* __restrict__ bucket_cursor, int* __restrict__ list,
                                                          CrowdedTable ct) {
  namespace cg = cooperative_groups;
  __shared__ int sm[33];
  float d;
  const bool due = list_rebuild_due(st, &d);  // the same in every thread of the grid
  if (due) {
    cg::grid_group grid = cg::this_grid();
    tile_bin<false>(X, O, N, nx, ny, tile_count, bucket_count, nullptr);
    grid.sync();
    if (blockIdx.x == 0) tile_scan(tile_count, n_tiles, tile_start, sm, ct);
    grid.sync();
    bucket_starts(n_tiles, tile_start, bucket_count, bucket_cursor);
    grid.sync();
    tile_bin<true>(X, O, N, nx, ny, nullptr, bucket_cursor, list);
  }
  __syncthreads();  // every thread of this CTA has read the state
  if (threadIdx.x == 0) {
    __threadfence();
    if (atomicAdd(exit_ctr, 1) == (int)gridDim.x - 1) {
      *exit_ctr = 0;
      list_policy_commit(st);  // need, drift, step maxima for this step's K4
    }
  }
}

// mc_load_filaments: largest tile list (chooses the CTA size of the P2G kernels)
__global__ void k_max_int(const int* __restrict__ v, int n, int* __restrict__ out) {
  int m = 0;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) m = max(m, v[i]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0) atomicMax(out, m);
}

}  // namespace mc

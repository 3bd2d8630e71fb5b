// k_cluster.cuh -- crowded worlds (BASELINE.json config 5: "to stress scatter contention"): the
// tile-accumulation kernels K2a (S2 deposit) and K2b+K3b (S5 spread fused with S6) with a
// THREAD-BLOCK CLUSTER of C CTAs per tile instead of one CTA.
//
// Why: one CTA per 32x32 tile walks the whole list of the tile.  In the cluster of config 5 the
// central tiles list ~16,000 beads each (64 shared-memory atomics per bead in their hi + lo
// planes) while most of the 4096 tiles list none: a hundred CTAs carry the kernel and the other
// SMs idle.  Here the C CTAs of a cluster deal the tile's key-sorted list among ALL their warps
// (DealCfg, k_p2g.cuh), each into its own shared accumulators; after a cluster barrier CTA r
// owns the rows [r TS/C, (r+1) TS/C) of the tile and sums the C partial accumulators of its nodes
// through distributed shared memory.  The partial sums are integers (fixed point, same scale in
// every CTA), so the total -- and every bit of the result -- is the same as with one CTA per tile.
// Tiles with at most SPLIT_N listed beads are accumulated by the first CTA of their cluster alone
// (the others only take their rows of the result from it), empty tiles by nobody: in a crowded
// world most tiles are empty, and an 8-way reduction of zeros cost more than it saved.
#pragma once
#include <cooperative_groups.h>

#include "k_lbm.cuh"
#include "k_p2g.cuh"

namespace mc {

namespace cg = cooperative_groups;

constexpr int SPLIT_N = 1024;  // listed beads above which the whole cluster shares a tile's list

// number of CTAs of the cluster that accumulate a list of n entries
template <int C>
__device__ __forceinline__ int cluster_share(int n) { return n == 0 ? 0 : (n > SPLIT_N ? C : 1); }

// sum over the cluster of one accumulator word, then hi + lo -> float exactly like tile_value
template <int C>
__device__ __forceinline__ float cluster_value(cg::cluster_group& cl, int* acc, int* accl, int a, float linv, int ce) {
  int hi = 0, lo = 0;
#pragma unroll
  for (int r = 0; r < C; ++r) {
    if (r < ce) {
      hi += cl.map_shared_rank(acc, r)[a];
      if (linv != 0.0f) lo += cl.map_shared_rank(accl, r)[a];
    }
  }
  return (linv != 0.0f) ? fmaf((float)lo, linv, (float)hi) : (float)hi;
}

// K2a with C CTAs per tile.  grid = n_tiles * C (1-D, cluster-major), 256 threads.
template <int C>
__global__ void __cluster_dims__(C, 1, 1) __launch_bounds__(256)
    k_deposit_tile_cl(int nx, int ny, const int* __restrict__ tile_start, const int* __restrict__ list,
                      const float2* __restrict__ X, float* __restrict__ rho_b, float* __restrict__ tile_rho_max,
                      unsigned* __restrict__ tile_fmax, size_t wstride, const int* __restrict__ crowded = nullptr,
                      const int* __restrict__ n_crowded = nullptr, int cl_max = 0) {
  __shared__ __align__(16) int acc[ACC_N], accl[ACC_N];
  {
    const size_t ws = blockIdx.y * wstride;
    crowded = wshift(crowded, ws); n_crowded = wshift(n_crowded, ws);
    tile_start = wshift(tile_start, ws); list = wshift(list, ws); X = wshift(X, ws); rho_b = wshift(rho_b, ws);
    tile_rho_max = wshift(tile_rho_max, ws); tile_fmax = wshift(tile_fmax, ws);
  }
  cg::cluster_group cl = cg::this_cluster();
  const int rank = (int)cl.block_rank();
  int t = blockIdx.x / C;
  if (crowded) {  // split launch: cluster k serves the k-th crowded tile (the whole cluster leaves together)
    if (t >= min(*n_crowded, cl_max)) return;
    t = crowded[t];
  }
  const int ntx = nx / TS;
  const int x0 = (t % ntx) * TS, y0 = (t / ntx) * TS;
  const int s = tile_start[t], e = tile_start[t + 1];
  const bool wide = (e - s) > WIDE_N;
  const int ce = cluster_share<C>(e - s);  // the same in every CTA of the cluster
  const float scale = pow2_scale(fmaxf(0.25f * (float)(e - s), 1.0f));
  const float lscale = pow2f(lo_bits(e - s));
  if (rank < ce) {
    const DealCfg cfg(8 * ce, rank * 8 + (threadIdx.x >> 5));
    float2 xpre = make_float2(0.f, 0.f);
    {
      const Deal d(e - s, cfg);
      if (d.valid()) xpre = __ldg(X + __ldg(list + s + d.p));
    }
    zero_acc<256>(acc);
    if (wide) zero_acc<256>(accl);
    __syncthreads();
    if (wide) deposit_loop_wide_cfg(nx, ny, x0, y0, s, e, list, X, scale, lscale, acc, accl, xpre, cfg.nw, cfg.v0);
    else if (nx == TS || ny == TS) deposit_loop<false, true>(nx, ny, x0, y0, s, e, list, X, scale, lscale, acc, accl, xpre, cfg);
    else deposit_loop<false, false>(nx, ny, x0, y0, s, e, list, X, scale, lscale, acc, accl, xpre, cfg);
  }
  if (ce) cl.sync();
  const float inv = 1.0f / scale, linv = wide ? 1.0f / lscale : 0.0f;
  float mx = 0.0f;
  constexpr int RP = TS / C;  // rows of the tile owned by this CTA
  for (int c = threadIdx.x; c < RP * TS / 4; c += 256) {
    const int ly = rank * RP + (c >> 3), lx = (c & 7) << 2;
    const int a = acc_index(lx, ly);
    float v[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      v[k] = cluster_value<C>(cl, acc, accl, a + k, linv, ce) * inv;
      mx = fmaxf(mx, v[k]);
    }
    __stcs(reinterpret_cast<float4*>(rho_b + (size_t)(y0 + ly) * nx + x0 + lx), make_float4(v[0], v[1], v[2], v[3]));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  if ((threadIdx.x & 31) == 0) atomicMax(reinterpret_cast<unsigned*>(tile_rho_max) + t, __float_as_uint(mx));
  if (threadIdx.x == 0 && rank == 0) tile_fmax[t] = 0u;
  if (ce) cl.sync();  // nobody leaves while a peer may still read its accumulators
}

// K2b + K3b with C CTAs per tile.  grid = n_tiles * C (1-D, cluster-major), 256 threads; the
// threads with ry < TS/C run S6 on the node pairs of this CTA's rows.
template <int C, bool KEEP_G>
__global__ void __cluster_dims__(C, 1, 1) __launch_bounds__(256) k_lbm_spread_tile_cl(LbmSpreadArgs p, size_t wstride) {
  __shared__ __align__(16) int acc0[ACC_N], acc1[ACC_N], accl0[ACC_N], accl1[ACC_N];
  __shared__ float red[32];
  p.shift(blockIdx.y * wstride);
  cg::cluster_group cl = cg::this_cluster();
  const int rank = (int)cl.block_rank();
  const LbmArgs& a = p.lbm;
  const int nx = a.nx, ny = a.ny;
  int t = blockIdx.x / C;
  if (p.crowded) {  // split launch: cluster k serves the k-th crowded tile
    if (t >= min(*p.n_crowded, p.cl_max)) return;
    t = p.crowded[t];
  }
  const int ntx = nx / TS;
  const int x0 = (t % ntx) * TS, y0 = (t / ntx) * TS;
  const int s = p.tile_start[t], e = p.tile_start[t + 1];
  const int ce = cluster_share<C>(e - s);  // the same in every CTA of the cluster
  if (rank < ce) {
    const DealCfg cfg(8 * ce, rank * 8 + (threadIdx.x >> 5));
    float2 xpre = make_float2(0.f, 0.f), fpre = make_float2(0.f, 0.f);
    {
      const int b = first_entry(s, e, p.list, cfg);
      if (b >= 0) { xpre = __ldg(p.X + b); fpre = __ldg(p.F + b); }
    }
    float linv_own;
    const float scale = spread_tile_accumulate<true>(nx, ny, x0, y0, s, e, p.list, p.X, p.F,
                                                     p.tile_rho_max ? p.tile_rho_max[t] : 0.0f, p.tile_fmax, t, acc0,
                                                     acc1, accl0, accl1, red, linv_own, xpre, fpre, cfg);
    // the scale and the lo-plane factor of the tile, for the CTAs that did not accumulate (every
    // accumulating CTA derives the same values; red[0] was consumed behind a barrier)
    if (threadIdx.x == 0) { red[1] = 1.0f / scale; red[2] = linv_own; }
  }
  constexpr int RP = TS / C;
  const size_t nc = (size_t)nx * ny;
  const int lx = (threadIdx.x & 15) << 1, ry = threadIdx.x >> 4;
  const bool mine = ry < RP;
  const int ly = rank * RP + (mine ? ry : 0), i = x0 + lx, j = y0 + ly;
  const int im = (i == 0) ? nx - 1 : i - 1, ip2 = (i + 2 == nx) ? 0 : i + 2;
  const int jm = (j == 0) ? ny - 1 : j - 1, jp = (j == ny - 1) ? 0 : j + 1;
  const size_t r0 = (size_t)j * nx, rm = (size_t)jm * nx, rp = (size_t)jp * nx;
  float gA[9], gB[9];
  if (mine) {  // pull: g_q(x) = src_q(x - c_q), issued before the barrier that ends the atomic phase
    const float2 v0 = __ldg(reinterpret_cast<const float2*>(a.src + 0 * nc + r0 + i));
    const float2 v2 = __ldg(reinterpret_cast<const float2*>(a.src + 2 * nc + rm + i));
    const float2 v4 = __ldg(reinterpret_cast<const float2*>(a.src + 4 * nc + rp + i));
    gA[0] = v0.x; gB[0] = v0.y; gA[2] = v2.x; gB[2] = v2.y; gA[4] = v4.x; gB[4] = v4.y;
    gA[1] = __ldg(a.src + 1 * nc + r0 + im);     gB[1] = __ldg(a.src + 1 * nc + r0 + i);
    gA[3] = __ldg(a.src + 3 * nc + r0 + i + 1);  gB[3] = __ldg(a.src + 3 * nc + r0 + ip2);
    gA[5] = __ldg(a.src + 5 * nc + rm + im);     gB[5] = __ldg(a.src + 5 * nc + rm + i);
    gA[6] = __ldg(a.src + 6 * nc + rm + i + 1);  gB[6] = __ldg(a.src + 6 * nc + rm + ip2);
    gA[7] = __ldg(a.src + 7 * nc + rp + i + 1);  gB[7] = __ldg(a.src + 7 * nc + rp + ip2);
    gA[8] = __ldg(a.src + 8 * nc + rp + im);     gB[8] = __ldg(a.src + 8 * nc + rp + i);
  }
  float inv = 0.0f, linv = 0.0f;
  if (ce) {
    cl.sync();
    const float* red0 = cl.map_shared_rank(red, 0);
    inv = red0[1];
    linv = red0[2];
  }
  if (threadIdx.x == 0 && rank == 0 && p.tile_rho_max) p.tile_rho_max[t] = 0.0f;  // every CTA read it before the barrier
  if (mine) {
    const size_t c = r0 + i;
    const int sa = acc_index(lx, ly);
    const float GAx = cluster_value<C>(cl, acc0, accl0, sa, linv, ce) * inv, GAy = cluster_value<C>(cl, acc1, accl1, sa, linv, ce) * inv;
    const float GBx = cluster_value<C>(cl, acc0, accl0, sa + 1, linv, ce) * inv, GBy = cluster_value<C>(cl, acc1, accl1, sa + 1, linv, ce) * inv;
    if (KEEP_G) {
      *reinterpret_cast<float2*>(a.G0out + c) = make_float2(GAx, GBx);
      *reinterpret_cast<float2*>(a.G1out + c) = make_float2(GAy, GBy);
    }
    float uAx, uAy, uBx, uBy;
    trt_collide(gA, GAx, GAy, a.rho0, a.k, uAx, uAy);
    trt_collide(gB, GBx, GBy, a.rho0, a.k, uBx, uBy);
    __stcs(reinterpret_cast<float4*>(a.u + blk_index(i, j, nx)), make_float4(uAx, uAy, uBx, uBy));
#pragma unroll
    for (int q = 0; q < 9; ++q) __stcs(reinterpret_cast<float2*>(a.dst + q * nc + c), make_float2(gA[q], gB[q]));
    if (!(fabsf(uAx) <= 0.3f && fabsf(uAy) <= 0.3f && fabsf(uBx) <= 0.3f && fabsf(uBy) <= 0.3f)) atomicOr(a.flag, 4);
  }
  if (ce) cl.sync();  // nobody leaves while a peer may still read its accumulators
}

}  // namespace mc

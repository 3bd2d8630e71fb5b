// k_p2g.cuh -- K2a scalar deposition (S2) and K2b force spreading (S5): shared-memory tile
// accumulation (north_star (2)).
//
// S2: rho_b(g) = sum_i delta_h(g - X_i)            ("node positions are deposited")
// S5: G(g)     = sum_i F_i delta_h(g - X_i)        ("broadcasts ... onto the grid")
// delta_h = Peskin 4-point product kernel (readings 7, 13).
//
// One CTA per TS x TS tile.  Each thread takes beads from the tile's list (k_tile.cuh), forms
// the 4+4 weights and adds its up-to-16 contributions into the tile's accumulators in shared
// memory with the native 32-bit integer atomic (ATOMS.ADD).  Accumulating in FIXED POINT
// makes the sum independent of the order in which the atomics land, so the result is
// bit-reproducible run to run without sorting the lists (a float atomic would not be, and on
// sm_100a it is a CAS loop ~4x slower than the integer one; profiles/atoms_microbench.md).
// The fixed-point scale is a power of two chosen per tile from a bound on the largest
// possible accumulator, so no overflow can occur and the quantisation is ~2^-30 of that bound:
//   S2: every contribution is <= 1/4, so |acc| <= n_list/4;
//   S5: |sum_i F_i w_i| <= max|F| * sum_i w_i = max|F| * rho_b(g) <= max|F| * max_tile(rho_b),
//       with max_tile(rho_b) left behind by S2 of the same step (same X, same weights).
// Crowded tiles (more than WIDE_N listed beads, e.g. the cluster of config 5) would lose digits
// that way: their bound is far above the typical node value (many contributions, cancelling
// forces).  They accumulate every contribution as TWO integers -- the rounded value and its
// remainder scaled by a further 2^LB -- into a second accumulator plane, which restores fp32
// accuracy per contribution at twice the atomics, in those tiles only.
#pragma once
#include "k_tile.cuh"
#include "mc_common.cuh"

namespace mc {

// A listed bead seen from one tile.  Common case: `base` is the accumulator index of its first
// support node (accumulators carry a halo, k_tile.cuh), the 16 contributions go to base +
// r * TSP + c unconditionally.  WRAP_IN_TILE case (domain one tile wide along an axis, where a
// support can wrap around onto the same tile): per-node offsets folded into the tile and
// weights masked to zero outside it.
constexpr int WIDE_N = 1024;  // listed beads above which a tile accumulates hi + lo words

struct TileBead {
  int base;
  int col[4], row[4];    // WRAP_IN_TILE only.  col: halo + local x; row: (halo + local y) * TSP
  float wx[4], wy[4];
};

// zero one accumulator plane with 16-byte stores (the planes are 16-byte aligned, ACC_N % 4 == 0)
static_assert(ACC_N % 4 == 0, "accumulator planes are zeroed as int4");
// NT: CTA size when it is a compile-time fact (fully unrolled, constant store offsets), 0: any
template <int NT>
__device__ __forceinline__ void zero_acc(int* acc) {
  int4* a4 = reinterpret_cast<int4*>(acc);
  if (NT > 0) {
#pragma unroll
    for (int k = 0; k < (ACC_N / 4 + NT - 1) / NT; ++k) {
      const int c = threadIdx.x + k * NT;
      if ((k + 1) * NT <= ACC_N / 4 || c < ACC_N / 4) a4[c] = make_int4(0, 0, 0, 0);
    }
  } else {
    for (int c = threadIdx.x; c < ACC_N / 4; c += blockDim.x) a4[c] = make_int4(0, 0, 0, 0);
  }
}

__device__ __forceinline__ int acc_index(int lx, int ly) { return (ly + HALO) * TSP + lx + HALO; }

// distance (in nodes, periodic) from the tile origin to the first support node, in [-n/2, n/2)
__device__ __forceinline__ int tile_delta(int i0, int origin, int n) {
  int d = i0 - origin;
  const int h = n >> 1;
  if ((unsigned)(d + h + n) < (unsigned)(3 * n)) {  // within one period of the window: common case
    if (d >= h) d -= n;
    else if (d < -h) d += n;
  } else {
    d = wrapi(d + h, n) - h;
  }
  return d;
}

// WRAP_IN_TILE: the domain is a single tile wide along some axis, so a support can wrap around
// onto the SAME tile; then every node is folded individually.  Otherwise one periodic fold of the
// first support node is enough and the other three follow by +1.
// TWO (two-layer broadcast, reading 28): the point is the marker p + o; its support is formed
// from the bead's exact fractional part plus the offset (support_off, mc_common.cuh).
template <bool WRAP_IN_TILE, bool TWO = false>
__device__ __forceinline__ void tile_bead(float2 p, float2 o, int nx, int ny, int x0, int y0, TileBead& tb) {
  int i0, j0;
  float fx, fy;
  if (TWO) {
    support_off(p.x, o.x, i0, fx);
    support_off(p.y, o.y, j0, fy);
  } else {
    support(p.x, i0, fx);
    support(p.y, j0, fy);
  }
  peskin4(fx, tb.wx[0], tb.wx[1], tb.wx[2], tb.wx[3]);
  peskin4(fy, tb.wy[0], tb.wy[1], tb.wy[2], tb.wy[3]);
  if (WRAP_IN_TILE) {
    i0 = wrapi(i0, nx);
    j0 = wrapi(j0, ny);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int c = ((i0 + k >= nx) ? i0 + k - nx : i0 + k) - x0;
      const int r = ((j0 + k >= ny) ? j0 + k - ny : j0 + k) - y0;
      const bool cin = (unsigned)c < (unsigned)TS, rin = (unsigned)r < (unsigned)TS;
      tb.col[k] = HALO + (cin ? c : 0);
      tb.row[k] = (HALO + (rin ? r : 0)) * TSP;
      tb.wx[k] = cin ? tb.wx[k] : 0.0f;
      tb.wy[k] = rin ? tb.wy[k] : 0.0f;
    }
  } else {
    // a first node outside [-HALO, TS] has no support node inside the tile (a stale entry
    // cannot get there, k_tile.cuh; the clamp only guards the shared array) and keeps none
    i0 = min(max(tile_delta(i0, x0, nx), -HALO), TS);
    j0 = min(max(tile_delta(j0, y0, ny), -HALO), TS);
    tb.base = acc_index(i0, j0);
  }
}

template <bool WRAP_IN_TILE>
__device__ __forceinline__ int tap_index(const TileBead& tb, int l, int kx) {
  return WRAP_IN_TILE ? tb.row[l] + tb.col[kx] : tb.base + l * TSP + kx;
}

__device__ __forceinline__ float block_max(float v, float* sm /*[32]*/) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
  __syncthreads();
  v = (threadIdx.x < (blockDim.x >> 5)) ? sm[threadIdx.x] : 0.0f;
  if (threadIdx.x < 32) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    if (threadIdx.x == 0) sm[0] = v;
  }
  __syncthreads();
  v = sm[0];
  __syncthreads();
  return v;
}

// power-of-two scale s with bound * s < 2^30, for a normal positive bound (exponent arithmetic on
// the bits: frexpf/ldexpf cost ~60 instructions in every thread of every tile)
__device__ __forceinline__ float pow2_scale(float bound) {
  const int e = (int)((__float_as_uint(bound) >> 23) & 0xffu);  // bound in [2^(e-127), 2^(e-126))
  return __uint_as_float((unsigned)(127 + 30 - (e - 126)) << 23);  // 2^(30 - (e - 126))
}
__device__ __forceinline__ float pow2f(int k) { return __uint_as_float((unsigned)(127 + k) << 23); }

// number of extra fraction bits the lo word can carry without overflowing for n contributions
__device__ __forceinline__ int lo_bits(int n) {
  const int lg = 32 - __clz(max(n, 2) - 1);  // ceil(log2 n)
  return min(20, max(0, 30 - lg));
}

// Dealing of a tile's key-sorted list (k_tile.cuh) to the CTA: the n entries form W = ceil(n/32)
// rounds; in round v lane l takes sorted position l W + v, so every lane walks its own short run
// of (nearly) one key and the 32 lanes of a round hold (nearly) 32 different keys.  Warp w takes
// the rounds w, w + n_warps, ...
// DealCfg: the warps that share one tile's list -- the CTA's own (default), or the warps of all the
// CTAs of a thread-block cluster that splits a crowded tile (k_cluster.cuh).
struct DealCfg {
  int nw, v0;  // number of warps dealing the list, index of this thread's warp among them
  __device__ __forceinline__ DealCfg() : nw(blockDim.x >> 5), v0(threadIdx.x >> 5) {}
  __device__ __forceinline__ DealCfg(int nw_, int v0_) : nw(nw_), v0(v0_) {}
};

struct Deal {
  int W, n, nw, v, p;
  __device__ __forceinline__ Deal(int n_, DealCfg c = DealCfg()) : n(n_) {
    W = (n + 31) >> 5;
    nw = c.nw;
    v = c.v0;
    p = (threadIdx.x & 31) * W + v;
  }
  __device__ __forceinline__ bool valid() const { return v < W && p < n; }
  __device__ __forceinline__ bool next_valid() const { return v + nw < W && p + nw < n; }
  __device__ __forceinline__ void advance() { v += nw; p += nw; }
};

// A list entry e names bead e -- or, TWO, marker e: bead e >> 1, offset +O (e even) / -O (e odd).
template <bool TWO>
__device__ __forceinline__ void load_point(const float2* __restrict__ X, const float2* __restrict__ O, int e, float2& p,
                                           float2& o) {
  if (TWO) {
    p = __ldg(X + (e >> 1));
    o = __ldg(O + (e >> 1));
    if (e & 1) { o.x = -o.x; o.y = -o.y; }
  } else {
    p = __ldg(X + e);
    o = make_float2(0.f, 0.f);
  }
}

template <bool WIDE, bool WRAP, bool TWO = false>
__device__ __forceinline__ void deposit_loop(int nx, int ny, int x0, int y0, int s, int e,
                                             const int* __restrict__ list, const float2* __restrict__ X,
                                             float scale, float lscale, int* acc, int* accl, float2 xpre,
                                             DealCfg cfg = DealCfg(), const float2* __restrict__ O = nullptr,
                                             float2 opre = make_float2(0.f, 0.f)) {
  float2 xc = xpre, oc = opre;  // first entry preloaded by the caller, later ones one iteration ahead
  const float wscale = TWO ? 0.5f * scale : scale;  // each marker deposits half of its bead
  for (Deal d(e - s, cfg); d.valid(); d.advance()) {
    const float2 xb = xc, ob = oc;
    if (d.next_valid()) load_point<TWO>(X, O, __ldg(list + s + d.p + d.nw), xc, oc);
    TileBead tb;
    tile_bead<WRAP, TWO>(xb, ob, nx, ny, x0, y0, tb);
#pragma unroll
    for (int l = 0; l < 4; ++l) {
      const float wys = tb.wy[l] * wscale;
#pragma unroll
      for (int kx = 0; kx < 4; ++kx) {
        const int a = tap_index<WRAP>(tb, l, kx);
        const float v = tb.wx[kx] * wys;
        if (WIDE) {
          const float h = rintf(v);
          atomicAdd(&acc[a], (int)h);
          atomicAdd(&accl[a], __float2int_rn((v - h) * lscale));
        } else {
          atomicAdd(&acc[a], __float2int_rn(v));
        }
      }
    }
  }
}

template <bool WIDE, bool WRAP, bool TWO = false>
__device__ __forceinline__ void spread_loop(int nx, int ny, int x0, int y0, int s, int e,
                                            const int* __restrict__ list, const float2* __restrict__ X,
                                            const float2* __restrict__ F, float scale, float lscale,
                                            int* acc0, int* acc1, int* accl0, int* accl1,
                                            float2 xpre, float2 fpre, DealCfg cfg = DealCfg(),
                                            const float2* __restrict__ O = nullptr,
                                            float2 opre = make_float2(0.f, 0.f)) {
  // the caller loaded this thread's FIRST entry (xpre, fpre) before the zeroing and the barrier,
  // so that the list -> X/F gather latency is spent under them; later entries are software-
  // pipelined one iteration ahead
  float2 xc = xpre, fc = fpre, oc = opre;
  const float wscale = TWO ? 0.5f * scale : scale;  // each marker carries half of its bead's force
  for (Deal d(e - s, cfg); d.valid(); d.advance()) {
    const float2 xb = xc, f = fc, ob = oc;
    if (d.next_valid()) {
      const int bn = __ldg(list + s + d.p + d.nw);
      load_point<TWO>(X, O, bn, xc, oc);
      fc = __ldg(F + (TWO ? bn >> 1 : bn));
    }
    TileBead tb;
    tile_bead<WRAP, TWO>(xb, ob, nx, ny, x0, y0, tb);
    const float fxs = f.x * wscale, fys = f.y * wscale;
#pragma unroll
    for (int l = 0; l < 4; ++l) {
      const float wyx = tb.wy[l] * fxs, wyy = tb.wy[l] * fys;
#pragma unroll
      for (int kx = 0; kx < 4; ++kx) {
        const int a = tap_index<WRAP>(tb, l, kx);
        const float vx = tb.wx[kx] * wyx, vy = tb.wx[kx] * wyy;
        if (WIDE) {
          const float hx = rintf(vx), hy = rintf(vy);
          atomicAdd(&acc0[a], (int)hx);
          atomicAdd(&acc1[a], (int)hy);
          atomicAdd(&accl0[a], __float2int_rn((vx - hx) * lscale));
          atomicAdd(&accl1[a], __float2int_rn((vy - hy) * lscale));
        } else {
          atomicAdd(&acc0[a], __float2int_rn(vx));
          atomicAdd(&acc1[a], __float2int_rn(vy));
        }
      }
    }
  }
}

// the rare crowded-tile variants are kept out of line so that their registers do not count
// against the occupancy of the common path
__device__ __noinline__ void deposit_loop_wide(int nx, int ny, int x0, int y0, int s, int e, const int* list,
                                               const float2* X, float scale, float lscale, int* acc, int* accl,
                                               float2 xpre) {
  deposit_loop<true, true>(nx, ny, x0, y0, s, e, list, X, scale, lscale, acc, accl, xpre);
}
__device__ __noinline__ void deposit_loop_wide_cfg(int nx, int ny, int x0, int y0, int s, int e, const int* list,
                                                   const float2* X, float scale, float lscale, int* acc, int* accl,
                                                   float2 xpre, int nw, int v0) {
  deposit_loop<true, true>(nx, ny, x0, y0, s, e, list, X, scale, lscale, acc, accl, xpre, DealCfg(nw, v0));
}
__device__ __noinline__ void spread_loop_wide_cfg(int nx, int ny, int x0, int y0, int s, int e, const int* list,
                                                  const float2* X, const float2* F, float scale, float lscale,
                                                  int* acc0, int* acc1, int* accl0, int* accl1, float2 xpre,
                                                  float2 fpre, int nw, int v0) {
  spread_loop<true, true>(nx, ny, x0, y0, s, e, list, X, F, scale, lscale, acc0, acc1, accl0, accl1, xpre, fpre,
                          DealCfg(nw, v0));
}
__device__ __noinline__ void spread_loop_wide(int nx, int ny, int x0, int y0, int s, int e, const int* list,
                                              const float2* X, const float2* F, float scale, float lscale,
                                              int* acc0, int* acc1, int* accl0, int* accl1, float2 xpre,
                                              float2 fpre) {
  spread_loop<true, true>(nx, ny, x0, y0, s, e, list, X, F, scale, lscale, acc0, acc1, accl0, accl1, xpre, fpre);
}

// K2a: S2 deposit.  tile_rho_max[t] receives max over the tile of rho_b (for K2b's scale).
// LIGHT: the variant for worlds without crowded tiles, launched with 128 threads and capped at
// 40 registers (more resident CTAs hide the per-tile latency chain; the cap costs the crowded
// config 5 10 % and gains world 4d 2 %).
// TWO: the list holds two-layer markers (reading 28), O their offsets; grid = (nx/TS, ny/TS, worlds).
template <bool LIGHT, bool TWO = false>
__global__ void __launch_bounds__(256, LIGHT ? 6 : 1) k_deposit_tile(int nx, int ny, const int* __restrict__ tile_start,
                                                      const int* __restrict__ list,
                                                      const float2* __restrict__ X,
                                                      float* __restrict__ rho_b,
                                                      float* __restrict__ tile_rho_max,
                                                      unsigned* __restrict__ tile_fmax,
                                                      const float2* __restrict__ O, size_t wstride,
                                                      const int* __restrict__ crowded_rank = nullptr, int cl_max = 0) {
  __shared__ __align__(16) int acc[ACC_N], accl[ACC_N];
  if (wstride) {  // batched worlds; single worlds pass 0
    const size_t ws = blockIdx.z * wstride;
    crowded_rank = wshift(crowded_rank, ws);
    tile_start = wshift(tile_start, ws); list = wshift(list, ws); X = wshift(X, ws); rho_b = wshift(rho_b, ws);
    tile_rho_max = wshift(tile_rho_max, ws); tile_fmax = wshift(tile_fmax, ws); O = wshift(O, ws);
  }
  const int t = blockIdx.y * gridDim.x + blockIdx.x;  // grid = (nx/TS, ny/TS)
  if (crowded_rank && (unsigned)crowded_rank[t] < (unsigned)cl_max) return;  // served by the cluster launch (k_cluster.cuh)
  const int x0 = blockIdx.x * TS, y0 = blockIdx.y * TS;
  const int s = tile_start[t], e = tile_start[t + 1];
  const bool wide = (e - s) > WIDE_N;
  float2 xpre = make_float2(0.f, 0.f), opre = make_float2(0.f, 0.f);
  {
    const Deal d(e - s);
    if (d.valid()) load_point<TWO>(X, O, __ldg(list + s + d.p), xpre, opre);  // gather starts before the zeroing
  }
  if (LIGHT) {  // the light variant is launched with 128 threads
    zero_acc<128>(acc);
    if (wide) zero_acc<128>(accl);
  } else {
    zero_acc<0>(acc);
    if (wide) zero_acc<0>(accl);
  }
  const float scale = pow2_scale(fmaxf(0.25f * (float)(e - s), 1.0f));
  const float lscale = pow2f(lo_bits(e - s));
  __syncthreads();
  if (TWO) {
    if (wide) deposit_loop<true, true, true>(nx, ny, x0, y0, s, e, list, X, scale, lscale, acc, accl, xpre, DealCfg(), O, opre);
    else if (nx == TS || ny == TS) deposit_loop<false, true, true>(nx, ny, x0, y0, s, e, list, X, scale, lscale, acc, accl, xpre, DealCfg(), O, opre);
    else deposit_loop<false, false, true>(nx, ny, x0, y0, s, e, list, X, scale, lscale, acc, accl, xpre, DealCfg(), O, opre);
  } else if (wide) deposit_loop_wide(nx, ny, x0, y0, s, e, list, X, scale, lscale, acc, accl, xpre);
  else if (nx == TS || ny == TS) deposit_loop<false, true>(nx, ny, x0, y0, s, e, list, X, scale, lscale, acc, accl, xpre);
  else deposit_loop<false, false>(nx, ny, x0, y0, s, e, list, X, scale, lscale, acc, accl, xpre);
  __syncthreads();
  const float inv = 1.0f / scale, linv = 1.0f / lscale;
  float mx = 0.0f;
  // four consecutive nodes of a row per thread: one 16-byte store
  for (int c = threadIdx.x; c < TS * TS / 4; c += blockDim.x) {
    const int ly = c >> 3, lx = (c & 7) << 2;
    const int a = acc_index(lx, ly);
    float v[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      v[k] = (wide ? fmaf((float)accl[a + k], linv, (float)acc[a + k]) : (float)acc[a + k]) * inv;
      mx = fmaxf(mx, v[k]);
    }
    __stcs(reinterpret_cast<float4*>(rho_b + (size_t)(y0 + ly) * nx + x0 + lx), make_float4(v[0], v[1], v[2], v[3]));
  }
  // tile maximum: rho_b >= 0, so the float bits order like unsigned integers; one global
  // atomicMax per warp onto tile_rho_max[t] (reset to 0 by the fused spread + fluid kernel of the
  // previous step, k_lbm.cuh, after it has read it; zero from mc_create before the first step)
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  if ((threadIdx.x & 31) == 0) atomicMax(reinterpret_cast<unsigned*>(tile_rho_max) + t, __float_as_uint(mx));
  if (threadIdx.x == 0) tile_fmax[t] = 0u;  // K1 of this step raises it (atomicMax), K2b reads it
}

// accumulator -> float (before the 1/scale): hi word, plus the lo word in wide tiles (linv != 0)
__device__ __forceinline__ float tile_value(const int* acc, const int* accl, int a, float linv) {
  return (linv != 0.0f) ? fmaf((float)accl[a], linv, (float)acc[a]) : (float)acc[a];
}

// First list entry of this thread in the tile segment [s, e): bead index, or -1.
__device__ __forceinline__ int first_entry(int s, int e, const int* __restrict__ list, DealCfg cfg = DealCfg()) {
  const Deal d(e - s, cfg);
  return d.valid() ? __ldg(list + s + d.p) : -1;
}

// Accumulate the spread force of one tile into shared memory (two planes), return the scale.
// Used by the fused spread + fluid kernel (k_lbm.cuh), which must __syncthreads() before it
// reads the accumulators.  (xpre, fpre): X and F of this thread's first entry, loaded by the
// caller well ahead (their list -> X/F gather is the longest latency chain of the tile).
template <bool CL = false, bool TWO = false>
__device__ __forceinline__ float spread_tile_accumulate(int nx, int ny, int x0, int y0, int s, int e,
                                                        const int* __restrict__ list,
                                                        const float2* __restrict__ X,
                                                        const float2* __restrict__ F, float rho_max,
                                                        const unsigned* __restrict__ tile_fmax, int t,
                                                        int* acc0, int* acc1, int* accl0, int* accl1,
                                                        float* red, float& linv, float2 xpre, float2 fpre,
                                                        DealCfg cfg = DealCfg(), const float2* __restrict__ O = nullptr,
                                                        float2 opre = make_float2(0.f, 0.f)) {
  const bool wide = (e - s) > WIDE_N;
  const float lscale = pow2f(lo_bits(e - s));
  linv = wide ? 1.0f / lscale : 0.0f;  // 0 => the readers skip the lo planes (not zeroed then)
  zero_acc<256>(acc0);  // the fused kernel runs 256 threads
  zero_acc<256>(acc1);
  if (wide) { zero_acc<256>(accl0); zero_acc<256>(accl1); }
  float fm = 0.0f;
  if (tile_fmax) {
    // max |F| over the beads owned by this tile and its 8 neighbours (every listed bead whose
    // support overlaps the tile is owned by one of them), left by K1: no pass over the list
    if (threadIdx.x < 32) {
      const int ntx = nx / TS, nty = ny / TS;
      const int tx = t % ntx, ty = t / ntx;
      if (threadIdx.x < 9) {
        const int dx = (int)threadIdx.x % 3 - 1, dy = (int)threadIdx.x / 3 - 1;
        fm = __uint_as_float(tile_fmax[wrap1(ty + dy, nty) * ntx + wrap1(tx + dx, ntx)]);
      }
#pragma unroll
      for (int o = 8; o > 0; o >>= 1) fm = fmaxf(fm, __shfl_xor_sync(0xffffffffu, fm, o));
      if (threadIdx.x == 0) red[0] = fm;
    }
    __syncthreads();  // also orders the zeroing before the atomics
    fm = red[0];
  } else {
    for (int k = s + threadIdx.x; k < e; k += blockDim.x) {  // any order
      const int b = __ldg(list + k);
      const float2 f = __ldg(F + (TWO ? b >> 1 : b));
      fm = fmaxf(fm, fmaxf(fabsf(f.x), fabsf(f.y)));
    }
    fm = block_max(fm, red);  // also orders the zeroing before the atomics
  }
  const float sum_w = (rho_max > 0.0f) ? 1.0625f * rho_max : fmaxf(0.25f * (float)(e - s), 1.0f);
  const float scale = pow2_scale(fmaxf(fm * sum_w, 1e-18f));
  if (CL) {  // the list is shared with the other CTAs of a cluster (k_cluster.cuh)
    if (wide) spread_loop_wide_cfg(nx, ny, x0, y0, s, e, list, X, F, scale, lscale, acc0, acc1, accl0, accl1, xpre, fpre, cfg.nw, cfg.v0);
    else if (nx == TS || ny == TS) spread_loop<false, true>(nx, ny, x0, y0, s, e, list, X, F, scale, lscale, acc0, acc1, accl0, accl1, xpre, fpre, cfg);
    else spread_loop<false, false>(nx, ny, x0, y0, s, e, list, X, F, scale, lscale, acc0, acc1, accl0, accl1, xpre, fpre, cfg);
    return scale;
  }
  if (TWO) {
    if (wide) spread_loop<true, true, true>(nx, ny, x0, y0, s, e, list, X, F, scale, lscale, acc0, acc1, accl0, accl1, xpre, fpre, DealCfg(), O, opre);
    else if (nx == TS || ny == TS) spread_loop<false, true, true>(nx, ny, x0, y0, s, e, list, X, F, scale, lscale, acc0, acc1, accl0, accl1, xpre, fpre, DealCfg(), O, opre);
    else spread_loop<false, false, true>(nx, ny, x0, y0, s, e, list, X, F, scale, lscale, acc0, acc1, accl0, accl1, xpre, fpre, DealCfg(), O, opre);
    return scale;
  }
  if (wide) spread_loop_wide(nx, ny, x0, y0, s, e, list, X, F, scale, lscale, acc0, acc1, accl0, accl1, xpre, fpre);
  else if (nx == TS || ny == TS) spread_loop<false, true>(nx, ny, x0, y0, s, e, list, X, F, scale, lscale, acc0, acc1, accl0, accl1, xpre, fpre);
  else spread_loop<false, false>(nx, ny, x0, y0, s, e, list, X, F, scale, lscale, acc0, acc1, accl0, accl1, xpre, fpre);
  // NO barrier here: the caller issues its next global loads first, then synchronises
  return scale;
}

}  // namespace mc

// k_lbm.cuh -- K3b: S6 fluid update.  D2Q9 (Qian et al. 1992), two-relaxation-time
// collision (Ginzburg et al. 2008) with Guo's forcing split by parity, then streaming.
// Readings 10 (scheme details) and 11 (beads see the collision-time velocity
// u = (sum_q c_q f_q + G/2)/rho, which lets collide + stream + store-u be one pass).
//
// Storage: populations are kept SHIFTED, g_q = f_q - w_q*rho0 (fp32 velocities are small
// differences of O(1) populations; the shift keeps ~3 more digits).
// The array holds the POST-collision values of the previous step at their own node; streaming
// is done on read ("pull"): the pre-collision population of this step is
// g_q(x) = gpost_q(x - c_q).  Two buffers alternate.  Reads are coalesced rows shifted by
// at most one cell; writes are aligned.
//
// With g: drho = sum g_q, rho = rho0 + drho, m = sum c_q g_q (sum c_q w_q = 0),
//   geq+_q - w_q rho0 = w_q [drho + rho (4.5 (c_q.u)^2 - 1.5 u.u)]     (even part)
//   geq-_q            = w_q rho 3 c_q.u                                 (odd part)
//   S+_q = w_q [-3 u.G + 9 (c_q.u)(c_q.G)],  S-_q = 3 w_q c_q.G         (Guo source by parity)
//   gpost_q = g_q - w+ (g+_q - geq+_q) - w- (g-_q - geq-_q) + (1 - w+/2) S+_q + (1 - w-/2) S-_q
#pragma once
#include "k_p2g.cuh"
#include "mc_common.cuh"

namespace mc {

// Collision constants that depend only on the relaxation rates w+ and w- (filled on the host in
// fp32 with the same operations the kernel would do; as kernel arguments they are constant-bank
// operands and cost no registers).
struct TrtConst {
  float wp;    // w+
  float hwp;   // w+ / 2
  float hwm;   // w- / 2
  float cp3;   // 3 (1 - w+/2)
  float cb;    // 9 (1 - w+/2)
  float c2;    // 3 (1 - w-/2)
  float wp45;  // 4.5 w+
  float wm3;   // 3 w-
};

struct LbmArgs {
  const float* src;   // [9][ny][nx] post-collision, shifted
  float* dst;         // [9][ny][nx]
  const float* G0;    // spread force planes (may be NULL: zero force)
  const float* G1;
  float* G0out;       // fused kernel only: where G is stored when KEEP_G
  float* G1out;
  float2* u;          // out: collision-time velocity, interleaved (ux, uy)
  int nx, ny;
  float rho0;
  TrtConst k;         // collision constants (host, mc_api.cu)
  int* flag;          // sticky divergence flag (bit 2: |u| > 0.3 or non-finite)
  __device__ __forceinline__ void shift(size_t bytes) {  // batched worlds (mc_common.cuh wshift)
    src = wshift(src, bytes); dst = wshift(dst, bytes); G0 = wshift(G0, bytes); G1 = wshift(G1, bytes);
    G0out = wshift(G0out, bytes); G1out = wshift(G1out, bytes); u = wshift(u, bytes); flag = wshift(flag, bytes);
  }
};

// One TRT collision of a node given its pre-collision shifted populations g[9].
// The formulae of the header with the common factors pulled out (the kernel is issue bound):
//   even_q = -w+ g+_q + w_q [E0 + (c.u)(a (c.u) + b (c.G))],  E0 = w+ (drho - 1.5 rho u.u) - 3 (1 - w+/2) u.G,
//                                                              a = 4.5 w+ rho, b = 9 (1 - w+/2)
//   odd_q  = -w- g-_q + w_q [c1 (c.u) + c2 (c.G)],             c1 = 3 w- rho, c2 = 3 (1 - w-/2)
//   gpost_q = g_q + even_q + odd_q,  gpost_qbar = g_qbar + even_q - odd_q
__device__ __forceinline__ void trt_collide(float g[9], float Gx, float Gy, float rho0, const TrtConst& k,
                                            float& ux, float& uy) {
  const float W0 = 4.0f / 9.0f, W1 = 1.0f / 9.0f, W5 = 1.0f / 36.0f;
  const float drho = g[0] + ((g[1] + g[3]) + (g[2] + g[4])) + ((g[5] + g[7]) + (g[6] + g[8]));
  const float mx = (g[1] - g[3]) + ((g[5] - g[7]) + (g[8] - g[6]));
  const float my = (g[2] - g[4]) + ((g[5] - g[7]) + (g[6] - g[8]));
  const float rho = rho0 + drho;
  // 1/rho to 1 ulp (MUFU.RCP; rho = 1 + O(Ma^2)): the IEEE division costs 11 instructions per node
  float inv;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(inv) : "f"(rho));
  ux = (mx + 0.5f * Gx) * inv;
  uy = (my + 0.5f * Gy) * inv;
  const float usq = ux * ux + uy * uy;
  const float uG = ux * Gx + uy * Gy;
  const float wp = k.wp, hwp = k.hwp, hwm = k.hwm, cb = k.cb, c2 = k.c2;
  const float E0 = wp * (drho - 1.5f * rho * usq) - k.cp3 * uG;
  const float ca = k.wp45 * rho;
  const float c1 = k.wm3 * rho;
  // rest population (even only, c = 0)
  g[0] = fmaf(W0, E0, g[0] - wp * g[0]);
#define MC_PAIR(q, qb, w, cu, cG)                                                     \
  {                                                                                   \
    const float cu_ = (cu), cG_ = (cG);                                               \
    const float even = fmaf((w), fmaf(cu_, fmaf(ca, cu_, cb * cG_), E0), -hwp * (g[q] + g[qb])); \
    const float odd = fmaf((w), fmaf(c1, cu_, c2 * cG_), -hwm * (g[q] - g[qb]));      \
    g[q] += even + odd;                                                               \
    g[qb] += even - odd;                                                              \
  }
  MC_PAIR(1, 3, W1, ux, Gx)
  MC_PAIR(2, 4, W1, uy, Gy)
  MC_PAIR(5, 7, W5, ux + uy, Gx + Gy)
  MC_PAIR(6, 8, W5, uy - ux, Gy - Gx)
#undef MC_PAIR
}

__global__ void __launch_bounds__(256) k_lbm_step(LbmArgs a, size_t wstride) {
  a.shift(blockIdx.z * wstride);  // grid = (nx / bx, ny, worlds)
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y;
  const int nx = a.nx, ny = a.ny;
  const size_t nc = (size_t)nx * ny;
  const int im = (i == 0) ? nx - 1 : i - 1, ip = (i == nx - 1) ? 0 : i + 1;
  const int jm = (j == 0) ? ny - 1 : j - 1, jp = (j == ny - 1) ? 0 : j + 1;
  const size_t r0 = (size_t)j * nx, rm = (size_t)jm * nx, rp = (size_t)jp * nx;
  float g[9];
  // pull: g_q(x) = src_q(x - c_q)
  g[0] = __ldg(a.src + 0 * nc + r0 + i);
  g[1] = __ldg(a.src + 1 * nc + r0 + im);
  g[2] = __ldg(a.src + 2 * nc + rm + i);
  g[3] = __ldg(a.src + 3 * nc + r0 + ip);
  g[4] = __ldg(a.src + 4 * nc + rp + i);
  g[5] = __ldg(a.src + 5 * nc + rm + im);
  g[6] = __ldg(a.src + 6 * nc + rm + ip);
  g[7] = __ldg(a.src + 7 * nc + rp + ip);
  g[8] = __ldg(a.src + 8 * nc + rp + im);
  const size_t c = r0 + i;
  float Gx = 0.0f, Gy = 0.0f;
  if (a.G0) { Gx = __ldg(a.G0 + c); Gy = __ldg(a.G1 + c); }
  float ux, uy;
  trt_collide(g, Gx, Gy, a.rho0, a.k, ux, uy);
  a.u[blk_index(i, j, nx)] = make_float2(ux, uy);
#pragma unroll
  for (int q = 0; q < 9; ++q) a.dst[q * nc + c] = g[q];
  if (!(fabsf(ux) <= 0.3f && fabsf(uy) <= 0.3f)) atomicOr(a.flag, 4);
}

// Fused K2b + K3b: one CTA per TS x TS tile first accumulates the spread force of its tile in
// shared memory (S5, k_p2g.cuh) and then updates the fluid of the same nodes with it (S6), so G
// never travels through HBM (-16 B/node).  CTAs in their atomic phase overlap on an SM with
// CTAs in their streaming phase.  KEEP_G also stores G (parity tests: mc_keep_intermediates).
struct LbmSpreadArgs {
  LbmArgs lbm;             // G0/G1 are OUTPUTS here, used only when KEEP_G
  const int* tile_start;
  const int* list;
  const float2* X;
  const float2* F;
  float* tile_rho_max;        // may be NULL; read, then reset to 0 for the next step's S2 (atomicMax)
  const unsigned* tile_fmax;  // may be NULL
  const float2* O;            // two-layer marker offsets (TWO variants), else NULL
  // crowded worlds (k_cluster.cuh): tiles with rank < cl_max in the crowded table belong to the cluster
  // launch; the cluster launch finds its tiles in crowded[0 .. min(*n_crowded, cl_max))
  const int* crowded_rank;    // NULL: no split
  const int* crowded;
  const int* n_crowded;
  int cl_max;
  __device__ __forceinline__ void shift(size_t bytes) {
    lbm.shift(bytes);
    crowded_rank = wshift(crowded_rank, bytes); crowded = wshift(crowded, bytes); n_crowded = wshift(n_crowded, bytes);
    tile_start = wshift(tile_start, bytes); list = wshift(list, bytes); X = wshift(X, bytes); F = wshift(F, bytes);
    tile_rho_max = wshift(tile_rho_max, bytes); tile_fmax = wshift(tile_fmax, bytes); O = wshift(O, bytes);
  }
};

template <bool KEEP_G, bool TWO = false>
__global__ void __launch_bounds__(256, 5) k_lbm_spread_tile(LbmSpreadArgs p, size_t wstride) {
  __shared__ __align__(16) int acc0[ACC_N], acc1[ACC_N], accl0[ACC_N], accl1[ACC_N];
  __shared__ float red[32];
  if (wstride) p.shift(blockIdx.y * wstride);  // batched worlds; single worlds pass 0
  const LbmArgs& a = p.lbm;
  const int nx = a.nx, ny = a.ny;
  // 1-D grid in row-major tile order (a 2-D grid is rasterised differently by the hardware and
  // cost the streaming phase 20 % on world 4d)
  const int t = blockIdx.x, ntx = nx / TS;
  if (p.crowded_rank && (unsigned)p.crowded_rank[t] < (unsigned)p.cl_max) return;  // the cluster launch's tile
  const int x0 = (t % ntx) * TS, y0 = (t / ntx) * TS;
  const int s = p.tile_start[t], e = p.tile_start[t + 1];
  {
    // start pulling this tile's populations towards L2 while the atomic phase runs: 9 planes x
    // 32 rows x one 128-byte line (the +-1 halo columns/rows come with the neighbours' tiles)
    // thread (q, r) takes row r of plane q; plane 8 falls to the first warp
    const size_t ncp = (size_t)nx * ny;
    const int q = threadIdx.x >> 5, r = threadIdx.x & 31;
    const float* row = a.src + (size_t)(y0 + r) * nx + x0;
    asm volatile("prefetch.global.L2 [%0];" ::"l"(row + q * ncp));
    if (threadIdx.x < 32) asm volatile("prefetch.global.L2 [%0];" ::"l"(row + 8 * ncp));
  }
  // this thread's first list entry: its list -> X/F gather is the longest latency chain of the
  // tile, so it starts before the zeroing and the barrier of the atomic phase
  float2 xpre = make_float2(0.f, 0.f), fpre = make_float2(0.f, 0.f), opre = make_float2(0.f, 0.f);
  {
    const int b = first_entry(s, e, p.list);
    if (b >= 0) { load_point<TWO>(p.X, p.O, b, xpre, opre); fpre = __ldg(p.F + (TWO ? b >> 1 : b)); }
  }
  float linv;
  const float scale = spread_tile_accumulate<false, TWO>(nx, ny, x0, y0, s, e, p.list, p.X, p.F,
                                                         p.tile_rho_max ? p.tile_rho_max[t] : 0.0f, p.tile_fmax, t,
                                                         acc0, acc1, accl0, accl1, red, linv, xpre, fpre, DealCfg(),
                                                         p.O, opre);
  const float inv = 1.0f / scale;
  if (threadIdx.x == 0 && p.tile_rho_max) p.tile_rho_max[t] = 0.0f;  // all reads happened before the barrier
  // S6 on the tile: each thread owns the node PAIR (i, i+1), i even, in rows ry and ry + 16.
  // Two nodes per thread halve the address arithmetic and turn the unshifted planes, all nine
  // stores and the blocked u store into 8/16-byte accesses: the kernel is bound by issue slots
  // (5.8e8 warp instructions per launch on world 4d), not by DRAM.
  const size_t nc = (size_t)nx * ny;
  const int lx = (threadIdx.x & 15) << 1, ry = threadIdx.x >> 4;
  const int i = x0 + lx;
  const int im = (i == 0) ? nx - 1 : i - 1, ip2 = (i + 2 == nx) ? 0 : i + 2;
  bool bad = false;
  float gA[9], gB[9];  // pre-collision populations of nodes i and i+1 (pull: g_q(x) = src_q(x - c_q))
  // Addresses: plane q of a row pointer is one IMAD.WIDE (32-bit plane size x immediate q + 64-bit
  // pointer) and the column neighbours are immediate offsets, unless the pair touches the
  // periodic seam in x (first/last pair of a row of the domain) or the planes exceed 4 GB / 8.
  const unsigned pb = (unsigned)(nc * sizeof(float));  // bytes per plane (used only when it fits)
  const bool fast = (nc * sizeof(float) * 8 < 0xffffffffull) && i != 0 && i + 2 != nx;
  auto plane = [&](const float* p, int q) {
    return reinterpret_cast<const float*>(reinterpret_cast<const char*>(p) + (unsigned long long)pb * (unsigned)q);
  };
  auto load_pair = [&](int ly) {
    const int j = y0 + ly;
    const int jm = (j == 0) ? ny - 1 : j - 1, jp = (j == ny - 1) ? 0 : j + 1;
    if (fast) {
      const float* p0 = a.src + (size_t)j * nx + i;
      const float* pm = a.src + (size_t)jm * nx + i;
      const float* pp = a.src + (size_t)jp * nx + i;
      const float2 v0 = __ldg(reinterpret_cast<const float2*>(p0));
      const float2 v2 = __ldg(reinterpret_cast<const float2*>(plane(pm, 2)));
      const float2 v4 = __ldg(reinterpret_cast<const float2*>(plane(pp, 4)));
      gA[0] = v0.x; gB[0] = v0.y; gA[2] = v2.x; gB[2] = v2.y; gA[4] = v4.x; gB[4] = v4.y;
      const float* q1 = plane(p0, 1); gA[1] = __ldg(q1 - 1); gB[1] = __ldg(q1);
      const float* q3 = plane(p0, 3); gA[3] = __ldg(q3 + 1); gB[3] = __ldg(q3 + 2);
      const float* q5 = plane(pm, 5); gA[5] = __ldg(q5 - 1); gB[5] = __ldg(q5);
      const float* q6 = plane(pm, 6); gA[6] = __ldg(q6 + 1); gB[6] = __ldg(q6 + 2);
      const float* q7 = plane(pp, 7); gA[7] = __ldg(q7 + 1); gB[7] = __ldg(q7 + 2);
      const float* q8 = plane(pp, 8); gA[8] = __ldg(q8 - 1); gB[8] = __ldg(q8);
      return;
    }
    const size_t r0 = (size_t)j * nx, rm = (size_t)jm * nx, rp = (size_t)jp * nx;
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
  };
  // the first pass's 15 loads are issued BEFORE the barrier that ends the atomic phase, so their
  // DRAM latency is spent while the slower warps finish their atomics
  load_pair(ry);
  __syncthreads();
#pragma unroll 1
  for (int h = 0; h < 2; ++h) {
    const int ly = ry + 16 * h, j = y0 + ly;
    if (h) load_pair(ly);
    const size_t r0 = (size_t)j * nx;
    const size_t c = r0 + i;
    const int sa = acc_index(lx, ly);
    const float GAx = tile_value(acc0, accl0, sa, linv) * inv, GAy = tile_value(acc1, accl1, sa, linv) * inv;
    const float GBx = tile_value(acc0, accl0, sa + 1, linv) * inv, GBy = tile_value(acc1, accl1, sa + 1, linv) * inv;
    if (KEEP_G) {
      *reinterpret_cast<float2*>(a.G0out + c) = make_float2(GAx, GBx);
      *reinterpret_cast<float2*>(a.G1out + c) = make_float2(GAy, GBy);
    }
    float uAx, uAy, uBx, uBy;
    trt_collide(gA, GAx, GAy, a.rho0, a.k, uAx, uAy);
    trt_collide(gB, GBx, GBy, a.rho0, a.k, uBx, uBy);
    // blocked u: nodes i and i+1 (i even) are neighbours inside one 4x4 block
    __stcs(reinterpret_cast<float4*>(a.u + blk_index(i, j, nx)), make_float4(uAx, uAy, uBx, uBy));
    if (nc * sizeof(float) * 8 < 0xffffffffull) {
      char* d0 = reinterpret_cast<char*>(a.dst + c);
#pragma unroll
      for (int q = 0; q < 9; ++q)  // streaming stores: nothing reads these lines before a whole step has passed
        __stcs(reinterpret_cast<float2*>(d0 + (unsigned long long)pb * (unsigned)q), make_float2(gA[q], gB[q]));
    } else {
#pragma unroll
      for (int q = 0; q < 9; ++q) *reinterpret_cast<float2*>(a.dst + q * nc + c) = make_float2(gA[q], gB[q]);
    }
    bad = bad || !(fabsf(uAx) <= 0.3f && fabsf(uAy) <= 0.3f && fabsf(uBx) <= 0.3f && fabsf(uBy) <= 0.3f);
  }
  if (bad) atomicOr(a.flag, 4);
}

// mc_read_state: current pre-collision populations (streamed) as deviations, and rho.
__global__ void k_lbm_export(const float* __restrict__ src, int nx, int ny, float rho0,
                             float* __restrict__ fdev, float* __restrict__ rho) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y;
  if (i >= nx) return;
  const size_t nc = (size_t)nx * ny;
  const int im = (i == 0) ? nx - 1 : i - 1, ip = (i == nx - 1) ? 0 : i + 1;
  const int jm = (j == 0) ? ny - 1 : j - 1, jp = (j == ny - 1) ? 0 : j + 1;
  const size_t r0 = (size_t)j * nx, rm = (size_t)jm * nx, rp = (size_t)jp * nx;
  float g[9];
  g[0] = src[0 * nc + r0 + i];
  g[1] = src[1 * nc + r0 + im];
  g[2] = src[2 * nc + rm + i];
  g[3] = src[3 * nc + r0 + ip];
  g[4] = src[4 * nc + rp + i];
  g[5] = src[5 * nc + rm + im];
  g[6] = src[6 * nc + rm + ip];
  g[7] = src[7 * nc + rp + ip];
  g[8] = src[8 * nc + rp + im];
  const size_t c = r0 + i;
  if (fdev) {
#pragma unroll
    for (int q = 0; q < 9; ++q) fdev[q * nc + c] = g[q];
  }
  if (rho) rho[c] = rho0 + (g[0] + ((g[1] + g[3]) + (g[2] + g[4])) + ((g[5] + g[7]) + (g[6] + g[8])));
}

// mc_load_fluid: the inverse of k_lbm_export.  The library stores POST-collision populations at their
// own node and streams on read (g_q(x) = gpost_q(x - c_q)); a caller hands in the streamed,
// pre-collision deviations g_q(x), so gpost_q(x) = g_q(x + c_q).
__global__ void k_lbm_import(const float* __restrict__ fdev, int nx, int ny, float* __restrict__ dst) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y;
  if (i >= nx) return;
  const size_t nc = (size_t)nx * ny;
  const int im = (i == 0) ? nx - 1 : i - 1, ip = (i == nx - 1) ? 0 : i + 1;
  const int jm = (j == 0) ? ny - 1 : j - 1, jp = (j == ny - 1) ? 0 : j + 1;
  const size_t r0 = (size_t)j * nx, rm = (size_t)jm * nx, rp = (size_t)jp * nx;
  const size_t c = r0 + i;
  dst[0 * nc + c] = fdev[0 * nc + r0 + i];
  dst[1 * nc + c] = fdev[1 * nc + r0 + ip];   // c_1 = (+1, 0)
  dst[2 * nc + c] = fdev[2 * nc + rp + i];    // c_2 = (0, +1)
  dst[3 * nc + c] = fdev[3 * nc + r0 + im];   // c_3 = (-1, 0)
  dst[4 * nc + c] = fdev[4 * nc + rm + i];    // c_4 = (0, -1)
  dst[5 * nc + c] = fdev[5 * nc + rp + ip];   // c_5 = (+1, +1)
  dst[6 * nc + c] = fdev[6 * nc + rp + im];   // c_6 = (-1, +1)
  dst[7 * nc + c] = fdev[7 * nc + rm + im];   // c_7 = (-1, -1)
  dst[8 * nc + c] = fdev[8 * nc + rm + ip];   // c_8 = (+1, -1)
}

// mc_read_state: blocked interleaved (x,y) field -> two row-major planes
__global__ void k_split2(int nx, int ny, const float2* __restrict__ in, float* __restrict__ out0, float* __restrict__ out1) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
  if (i >= nx) return;
  const float2 v = in[blk_index(i, j, nx)];
  out0[(size_t)j * nx + i] = v.x;
  out1[(size_t)j * nx + i] = v.y;
}

}  // namespace mc

// k_mdf.cuh -- K5: Multi-Direct Forcing coupling (MC_COUPLING_MDF).
// P:L125 "the filaments' nodes sample the local fluid velocity ... the agent broadcasts its own
// velocity back onto the grid"; "Multi-Direct Forcing (MDF) (Wang et al., 2008)".
// Reading 26: the bead's own velocity is V_i = D_i + field displacement (K1 with
// kappa = 1).  With u*(g) = sum_q c_q f_q / rho the force-free velocity of this step's
// populations, u^0 = u*, F = 0, iteration k = 0..K-1:
//   U_i  = sum_g u^k(g) delta_h(g - X_i)                  (sample,    K5b)
//   dF_i = rho0 (V_i - U_i),  F_i += dF_i                 (force,     K5b)
//   u^{k+1}(g) = u^k(g) + [sum_i dF_i delta_h(g - X_i)] / (2 rho(g))   (broadcast, K5c; Guo's
//                                                          velocity u = u* + G/(2 rho), reading 11)
// The summed F then goes through the fused spread + fluid kernel (k_lbm.cuh) unchanged: spreading
// is linear, so its G = sum_k dG^k and its stored u equals u^K; the last iteration needs no
// broadcast of its own.
//
// HBM traffic on top of the FORCE-coupled step: K5a 36 + 12 B/node; per iteration 24 B/bead
// (X, V/F, dF) + the u gather; per broadcast 20 B/node of the tiles that hold beads + 16 B/bead.
#pragma once
#include "k_p2g.cuh"
#include "mc_common.cuh"

namespace mc {

// K5a: rho and u* of the current (pre-collision, pull-streamed) populations.  u in the blocked
// float2 layout K5b/K4 gather from; hrinv = 1/(2 rho), row-major.  Two nodes (i, i+1), i even,
// per thread: 8-byte loads of the unshifted planes and one 16-byte u store.
__global__ void __launch_bounds__(256) k_lbm_moments(const float* __restrict__ src, int nx, int ny, float rho0,
                                                     float2* __restrict__ u, float* __restrict__ hrinv, size_t wstride) {
  src = wshift(src, blockIdx.z * wstride);  // grid = (nx / (2 bx), ny, worlds)
  u = wshift(u, blockIdx.z * wstride);
  hrinv = wshift(hrinv, blockIdx.z * wstride);
  const int i = (blockIdx.x * blockDim.x + threadIdx.x) << 1;
  const int j = blockIdx.y;
  if (i >= nx) return;
  const size_t nc = (size_t)nx * ny;
  const int im = (i == 0) ? nx - 1 : i - 1, ip2 = (i + 2 == nx) ? 0 : i + 2;
  const int jm = (j == 0) ? ny - 1 : j - 1, jp = (j == ny - 1) ? 0 : j + 1;
  const size_t r0 = (size_t)j * nx, rm = (size_t)jm * nx, rp = (size_t)jp * nx;
  float gA[9], gB[9];  // g_q(x) = src_q(x - c_q)
  const float2 v0 = __ldg(reinterpret_cast<const float2*>(src + 0 * nc + r0 + i));
  const float2 v2 = __ldg(reinterpret_cast<const float2*>(src + 2 * nc + rm + i));
  const float2 v4 = __ldg(reinterpret_cast<const float2*>(src + 4 * nc + rp + i));
  gA[0] = v0.x; gB[0] = v0.y; gA[2] = v2.x; gB[2] = v2.y; gA[4] = v4.x; gB[4] = v4.y;
  gA[1] = __ldg(src + 1 * nc + r0 + im);     gB[1] = __ldg(src + 1 * nc + r0 + i);
  gA[3] = __ldg(src + 3 * nc + r0 + i + 1);  gB[3] = __ldg(src + 3 * nc + r0 + ip2);
  gA[5] = __ldg(src + 5 * nc + rm + im);     gB[5] = __ldg(src + 5 * nc + rm + i);
  gA[6] = __ldg(src + 6 * nc + rm + i + 1);  gB[6] = __ldg(src + 6 * nc + rm + ip2);
  gA[7] = __ldg(src + 7 * nc + rp + i + 1);  gB[7] = __ldg(src + 7 * nc + rp + ip2);
  gA[8] = __ldg(src + 8 * nc + rp + im);     gB[8] = __ldg(src + 8 * nc + rp + i);
  float4 uo;
  float2 hr;
  {
    const float* g = gA;  // same summation order as trt_collide (k_lbm.cuh)
    const float drho = g[0] + ((g[1] + g[3]) + (g[2] + g[4])) + ((g[5] + g[7]) + (g[6] + g[8]));
    const float mx = (g[1] - g[3]) + ((g[5] - g[7]) + (g[8] - g[6]));
    const float my = (g[2] - g[4]) + ((g[5] - g[7]) + (g[6] - g[8]));
    const float inv = 1.0f / (rho0 + drho);
    uo.x = mx * inv; uo.y = my * inv; hr.x = 0.5f * inv;
  }
  {
    const float* g = gB;
    const float drho = g[0] + ((g[1] + g[3]) + (g[2] + g[4])) + ((g[5] + g[7]) + (g[6] + g[8]));
    const float mx = (g[1] - g[3]) + ((g[5] - g[7]) + (g[8] - g[6]));
    const float my = (g[2] - g[4]) + ((g[5] - g[7]) + (g[6] - g[8]));
    const float inv = 1.0f / (rho0 + drho);
    uo.z = mx * inv; uo.w = my * inv; hr.y = 0.5f * inv;
  }
  *reinterpret_cast<float4*>(u + blk_index(i, j, nx)) = uo;  // nodes i, i+1 are neighbours in a 4x4 block
  *reinterpret_cast<float2*>(hrinv + r0 + i) = hr;
}

// K5b: sample the current grid velocity at the bead, add the direct-forcing increment.
// tile_fmax (zeroed once per step by the host's memset, one slot per iteration): bound for the
// fixed-point scale of the spread that consumes this iteration's output, kept exactly like K1's
// (k_filament.cuh): the warp's maximum is raised on every tile the warp's beads lie in.  It bounds
// |dF| for the broadcast K5c, and |F| (LAST: the summed force) for the fused spread + fluid kernel.
template <bool FIRST, bool LAST, int TEXROWS>
__global__ void __launch_bounds__(256) k_mdf_force(int N, const float2* __restrict__ X, const float2* __restrict__ V,
                                                   const float2* __restrict__ u, cudaTextureObject_t tex_u, int nx,
                                                   int ny, float rho0, float2* __restrict__ dF,
                                                   float2* __restrict__ F, unsigned* __restrict__ tile_fmax,
                                                   size_t wstride, const float2* __restrict__ O = nullptr) {
  {
    const size_t ws = blockIdx.y * wstride;
    X = wshift(X, ws); V = wshift(V, ws); u = wshift(u, ws); dF = wshift(dF, ws); F = wshift(F, ws);
    tile_fmax = wshift(tile_fmax, ws); O = wshift(O, ws);
  }
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = b < N;  // every lane stays for the warp-wide reduction
  const float2 p = X[valid ? b : N - 1];
  float m = 0.0f;
  if (valid) {
    float2 U;
    if (!TEXROWS && O) {  // two-layer broadcast (readings 26 + 28): the mean of the samples at the two markers
      const float2 o = __ldg(O + b);
      const float2 up = interp2_off(u, nx, ny, p.x, p.y, o.x, o.y), um = interp2_off(u, nx, ny, p.x, p.y, -o.x, -o.y);
      U = make_float2(0.5f * (up.x + um.x), 0.5f * (up.y + um.y));
    } else {
      U = TEXROWS ? interp2_tex<TEXROWS, false>(u, tex_u, nx, ny, p.x, p.y) : interp2_pair<0>(u, nx, ny, p.x, p.y);
    }
    const float2 v = V[b];
    const float2 d = make_float2(rho0 * (v.x - U.x), rho0 * (v.y - U.y));
    float2 f = d;
    if (!FIRST) {
      const float2 f0 = F[b];
      f = make_float2(f0.x + d.x, f0.y + d.y);
    }
    F[b] = f;
    if (!LAST) dF[b] = d;  // the last increment reaches the fluid inside the summed F
    m = LAST ? fmaxf(fabsf(f.x), fabsf(f.y)) : fmaxf(fabsf(d.x), fabsf(d.y));
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  const unsigned mb = __float_as_uint(m);  // positive floats order like their bit patterns
  const int t = (wrapi((int)floorf(p.y), ny) >> 5) * (nx >> 5) + (wrapi((int)floorf(p.x), nx) >> 5);
  const unsigned peers = __match_any_sync(0xffffffffu, t);
  if ((int)(threadIdx.x & 31) == __ffs(peers) - 1 && mb > tile_fmax[t]) atomicMax(tile_fmax + t, mb);
}

// K5c: broadcast.  One CTA per 32x32 tile accumulates the spread of dF in shared memory (the
// fixed-point tile accumulation of S5, k_p2g.cuh: order independent, bit-reproducible) and
// corrects the velocity of the tile's nodes in place.  Tiles without listed beads return at once.
template <bool TWO = false>
__global__ void __launch_bounds__(256, 5) k_mdf_spread_tile(int nx, int ny, const int* __restrict__ tile_start,
                                                            const int* __restrict__ list,
                                                            const float2* __restrict__ X,
                                                            const float2* __restrict__ dF,
                                                            const float* __restrict__ tile_rho_max,
                                                            const unsigned* __restrict__ tile_fmax,
                                                            const float* __restrict__ hrinv, float2* __restrict__ u,
                                                            size_t wstride, const float2* __restrict__ O = nullptr) {
  __shared__ __align__(16) int acc0[ACC_N], acc1[ACC_N], accl0[ACC_N], accl1[ACC_N];
  __shared__ float red[32];
  {
    const size_t ws = blockIdx.y * wstride;
    tile_start = wshift(tile_start, ws); list = wshift(list, ws); X = wshift(X, ws); dF = wshift(dF, ws);
    tile_rho_max = wshift(tile_rho_max, ws); tile_fmax = wshift(tile_fmax, ws); hrinv = wshift(hrinv, ws);
    u = wshift(u, ws); O = wshift(O, ws);
  }
  const int t = blockIdx.x, ntx = nx / TS;
  const int s = tile_start[t], e = tile_start[t + 1];
  if (s == e) return;  // nothing reaches this tile: u^{k+1} = u^k
  const int x0 = (t % ntx) * TS, y0 = (t / ntx) * TS;
  // this thread's node pairs (i, i+1), i even, in rows ry and ry + 16: their u and 1/(2 rho) are
  // requested now, so that the DRAM latency is spent under the atomic phase
  const int lx = (threadIdx.x & 15) << 1, ry = threadIdx.x >> 4;
  const int i = x0 + lx;
  float4* up0 = reinterpret_cast<float4*>(u + blk_index(i, y0 + ry, nx));
  float4* up1 = reinterpret_cast<float4*>(u + blk_index(i, y0 + ry + 16, nx));
  float4 v0 = *up0, v1 = *up1;
  const float2 h0 = __ldg(reinterpret_cast<const float2*>(hrinv + (size_t)(y0 + ry) * nx + i));
  const float2 h1 = __ldg(reinterpret_cast<const float2*>(hrinv + (size_t)(y0 + ry + 16) * nx + i));
  float2 xpre = make_float2(0.f, 0.f), fpre = make_float2(0.f, 0.f), opre = make_float2(0.f, 0.f);
  {
    const int b = first_entry(s, e, list);
    if (b >= 0) { load_point<TWO>(X, O, b, xpre, opre); fpre = __ldg(dF + (TWO ? b >> 1 : b)); }
  }
  float linv;
  const float scale = spread_tile_accumulate<false, TWO>(nx, ny, x0, y0, s, e, list, X, dF,
                                                         tile_rho_max ? tile_rho_max[t] : 0.0f, tile_fmax, t, acc0,
                                                         acc1, accl0, accl1, red, linv, xpre, fpre, DealCfg(), O, opre);
  __syncthreads();
  const float inv = 1.0f / scale;
  {
    const int sa = acc_index(lx, ry);
    const float ax = h0.x * inv, bx = h0.y * inv;
    v0.x = fmaf(tile_value(acc0, accl0, sa, linv), ax, v0.x);
    v0.y = fmaf(tile_value(acc1, accl1, sa, linv), ax, v0.y);
    v0.z = fmaf(tile_value(acc0, accl0, sa + 1, linv), bx, v0.z);
    v0.w = fmaf(tile_value(acc1, accl1, sa + 1, linv), bx, v0.w);
    *up0 = v0;
  }
  {
    const int sa = acc_index(lx, ry + 16);
    const float ax = h1.x * inv, bx = h1.y * inv;
    v1.x = fmaf(tile_value(acc0, accl0, sa, linv), ax, v1.x);
    v1.y = fmaf(tile_value(acc1, accl1, sa, linv), ax, v1.y);
    v1.z = fmaf(tile_value(acc0, accl0, sa + 1, linv), bx, v1.z);
    v1.w = fmaf(tile_value(acc1, accl1, sa + 1, linv), bx, v1.w);
    *up1 = v1;
  }
}

}  // namespace mc

// k_g2p.cuh -- K4: S7 grid-to-particle interpolation fused with position integration.
// U_i = sum_g u(g) delta_h(g - X_i) with the u stored by S6 and the same X as S1-S5;
// X_i <- X_i + U_i (forward Euler in lattice units; readings 11, 12, 19).
// P:L125 "the filaments' nodes sample the local fluid velocity".
#pragma once
#include "mc_common.cuh"

namespace mc {

// O != NULL (two-layer broadcast, reading 28; TEXROWS = 0): U_i is the mean of u sampled at the
// bead's two markers X_i +- O_i, the adjoint of the two-layer spread.
template <int TEXROWS>
__global__ void __launch_bounds__(256) k_interp_integrate(int N, float2* __restrict__ X,
                                                          const float2* __restrict__ u, cudaTextureObject_t tex_u,
                                                          int nx, int ny,
                                                          int* __restrict__ flag, long long* __restrict__ step,
                                                          unsigned* __restrict__ step_max,
                                                          const float2* __restrict__ O, size_t wstride) {
  if (!TEXROWS && wstride) {  // the texture variants serve single worlds only (views are per world)
    const size_t ws = blockIdx.y * wstride;
    X = wshift(X, ws); u = wshift(u, ws); flag = wshift(flag, ws); step = wshift(step, ws);
    step_max = wshift(step_max, ws); O = wshift(O, ws);
  }
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b == 0) *step += 1;  // device copy of the step counter (K1 of the next step reads it)
  float m = 0.0f;
  if (b < N) {
    float2 p = X[b];
    float2 U;
    if (!TEXROWS && O) {
      const float2 o = __ldg(O + b);
      const float2 up = interp2_off(u, nx, ny, p.x, p.y, o.x, o.y), um = interp2_off(u, nx, ny, p.x, p.y, -o.x, -o.y);
      U = make_float2(0.5f * (up.x + um.x), 0.5f * (up.y + um.y));
    } else {
      // 16-byte pair loads, all four rows through the LSU pipe (world 4d: 0.1415 ms with 8-byte loads
      // and one row through the texture pipe, 0.138 with pairs, 0.158 with pairs + one texture row)
      U = interp2_pair<0>(u, nx, ny, p.x, p.y);
    }
    p.x += U.x;
    p.y += U.y;
    X[b] = p;
    if (!(isfinite(p.x) && isfinite(p.y))) atomicOr(flag, 8);
    m = fmaxf(fabsf(U.x), fabsf(U.y));
  }
  // largest displacement component of this step: feeds the drift bound of the tile lists
  // (k_tile.cuh).  One guarded atomicMax per warp; positive floats order like their bits.
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0) {
    const unsigned mb = __float_as_uint(m);
    if (mb > *step_max) atomicMax(step_max, mb);
  }
}

}  // namespace mc

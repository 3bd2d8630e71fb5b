// k_p2g.cuh -- K2a scalar deposition (S2) and K2b force spreading (S5) as gathers by node.
//
// S2: rho_b(g) = sum_i delta_h(g - X_i)            ("node positions are deposited")
// S5: G(g)     = sum_i F_i delta_h(g - X_i)        ("broadcasts ... onto the grid")
// delta_h = Peskin 4-point product kernel (reading 7, 13).
//
// A bead whose cell is (ci,cj) = floor(X) touches nodes ci-1..ci+2, cj-1..cj+2, so node
// (i,j) receives from the beads of cells (i+di, j+dj), di,dj in -2..1, with weight planes
// wx[1-di] * wy[1-dj].  One thread per node walks those 16 bead lists in the canonical order
// K0 built: no float atomics, fixed summation order => bit-reproducible.
#pragma once
#include "mc_common.cuh"

namespace mc {

template <bool SPREAD>
__global__ void __launch_bounds__(256) k_p2g_gather(int nx, int ny, const int* __restrict__ cell_start,
                                                    const float* __restrict__ W, size_t plane,
                                                    const int* __restrict__ slot_bead,
                                                    const float2* __restrict__ F,
                                                    float* __restrict__ out0, float* __restrict__ out1) {
  const int i = blockIdx.x * 32 + (threadIdx.x & 31);
  const int j = blockIdx.y * 8 + (threadIdx.x >> 5);
  float a0 = 0.0f, a1 = 0.0f;
#pragma unroll
  for (int dj = -2; dj <= 1; ++dj) {
    const int row = wrap1(j + dj, ny);
    const float* wy = W + (size_t)(4 + 1 - dj) * plane;
#pragma unroll
    for (int di = -2; di <= 1; ++di) {
      const int col = wrap1(i + di, nx);
      const int c = row * nx + col;
      const int s = __ldg(cell_start + c), e = __ldg(cell_start + c + 1);
      const float* wx = W + (size_t)(1 - di) * plane;
      for (int k = s; k < e; ++k) {
        const float w = __ldg(wx + k) * __ldg(wy + k);
        if (SPREAD) {
          const float2 f = __ldg(F + __ldg(slot_bead + k));
          a0 = fmaf(w, f.x, a0);
          a1 = fmaf(w, f.y, a1);
        } else {
          a0 += w;
        }
      }
    }
  }
  const size_t g = (size_t)j * nx + i;
  out0[g] = a0;
  if (SPREAD) out1[g] = a1;
}

}  // namespace mc

// k_blur.cuh -- K3a: S3 Gaussian filter + gradient of the deposited bead density, one kernel,
// intermediates in shared memory.
//
// "node positions are deposited onto a grid, diffused with a Gaussian filter via FFT
// convolution to produce a density field, and the gradient of this density field generates
// repulsive forces."  Reading 14: the filter is the periodic convolution with the sampled,
// normalised Gaussian truncated at R (= the paper's filter to 2.6e-8 at R = 5 sigma), separable
// (applied here along y, then along x); reading 15: second-order central difference.
//
// Output: the force-gradient planes A = sum_fields coupling_k * grad(field_k) with the sign of
// the force (-kappa_rep for bead-density fields, +kappa_chi for static ones; S4 then needs one
// two-plane gather per bead whatever the number of fields -- interpolation is linear).
#pragma once
#include "mc_common.cuh"

namespace mc {

constexpr int BLUR_T = 32;       // output tile side
constexpr int BLUR_MAX_R = 16;   // largest supported truncation radius

struct BlurTaps {
  float g[2 * BLUR_MAX_R + 1];
};

// shared-memory geometry for radius R.  The two intermediate planes hold the 32 rows of the tile
// and the columns from node i0 - (R+1) on, so that the x pass of the 8 outputs starting at node
// i0 + 8c reads its window from column 8c: every shared access of the x pass is a 16-byte one.
constexpr int BLUR_THREADS = 128;
__host__ __device__ constexpr int blur_NV(int R) { return 10 + 2 * R; }               // window: 8 outputs + 2 + 2R
__host__ __device__ constexpr int blur_NV4(int R) { return (blur_NV(R) + 3) / 4; }
__host__ __device__ constexpr int blur_CW(int R) { return 24 + 4 * blur_NV4(R); }     // columns held >= 34 + 2R
// pitch of the interleaved (ty, dy) plane in float2: CW + 2, so that the 16-byte accesses of a
// quarter warp (2 chunks x 4 rows) fall on the 8 different bank groups
__host__ __device__ constexpr int blur_CP(int R) { return blur_CW(R) + 2; }


// One CTA filters one 32x32 tile; rho_b is read once per node plus the halo (through L1), the
// gradient is written once, nothing else touches global memory.  The y pass comes first because
// its loads are then coalesced straight from global memory (lanes = columns) and the y-derivative
// is a register operation on its outputs:
//   y pass: thread = (PAIR of columns of the tile + x halo, chunk of 8 rows): 10 + 2R 8-byte
//           loads of its columns, ty = G_y rho_b on 10 rows (packed FFMA2, one column in each
//           half), of which 8 are stored together with
//           dy = (ty[y+1] - ty[y-1]) / 2                              -> (ty, dy) [32][CP]
//   x pass: thread = (row, chunk of 8 nodes): register window of the interleaved (ty, dy) pairs
//           (16-byte LDS), (B, G_x dy) = G_x (ty, dy) on 10 nodes with packed FFMA2,
//           grad_x = (B[x+1] - B[x-1]) / 2, grad_y = G_x dy on the 8 inner nodes,
//           scaled by the signed coupling, plus the base field, stored as 16-byte pieces of the
//           blocked layout.
// (G_x G_y = G_y G_x and the differences commute with both: the result is the oracle's central
// difference of the filtered field up to rounding order.)
// coef: lattice coupling with the sign of the force.  base: blocked field added to the result
// (static part, or the running sum over earlier bead-density fields), may be NULL.
// A: blocked (x,y) force-gradient field.  field_out (filtered density, row-major) may be NULL.
template <int R>
__global__ void __launch_bounds__(BLUR_THREADS, R > 6 ? 1 : 7) k_blur_grad(int nx, int ny, BlurTaps taps,
                                                            const float* __restrict__ rho_b, float coef,
                                                            const float2* base, float2* A,
                                                            float* __restrict__ field_out, size_t wstride,
                                                            const float* __restrict__ tile_rho_max = nullptr) {
  if (wstride) {  // batched worlds (single worlds pass 0); field_out is a caller array of ONE world
    rho_b = wshift(rho_b, blockIdx.y * wstride);
    base = wshift(base, blockIdx.y * wstride);
    A = wshift(A, blockIdx.y * wstride);
    tile_rho_max = wshift(tile_rho_max, blockIdx.y * wstride);
  }
  constexpr int NV = blur_NV(R), CW = blur_CW(R), CP = blur_CP(R);
  __shared__ __align__(16) float2 td[BLUR_T * CP];
  // 1-D grid in row-major tile order (2-D grids are rasterised in an order that streams worse)
  const int ntx = nx / BLUR_T;
  const int i0 = (blockIdx.x % ntx) * BLUR_T, j0 = (blockIdx.x / ntx) * BLUR_T;
  if (tile_rho_max) {
    // Crowded worlds (config 5: ~90 % of the tiles hold no bead): the window of this tile reaches
    // R + 1 <= 17 nodes into its 8 neighbours; if S2 left rho_b = 0 on all nine tiles (their maxima,
    // written by K2a of this step) the filtered field and its gradient vanish here: the tile only
    // writes the base field (or zeros) and skips the loads and the arithmetic.  Exact, not approximate.
    static_assert(BLUR_T == 32, "tile_rho_max is per 32 x 32 tile");
    const int nty = ny / BLUR_T, tx = blockIdx.x % ntx, ty = blockIdx.x / ntx;
    bool any = false;
#pragma unroll
    for (int d = 0; d < 9; ++d)
      any = any || tile_rho_max[wrap1(ty + d / 3 - 1, nty) * ntx + wrap1(tx + d % 3 - 1, ntx)] != 0.0f;
    if (!any) {
      if (threadIdx.x < BLUR_T * 4) {
        const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
        const int c = (lane & 1) + 2 * ((lane >> 3) & 1);
        const int row = ((lane >> 1) & 3) + 4 * (lane >> 4) + 8 * wid;
        const size_t bidx = blk_index(i0 + 8 * c, j0 + row, nx);
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          float4* dst = reinterpret_cast<float4*>(A + bidx + 16 * h);
          float4 lo = make_float4(0.f, 0.f, 0.f, 0.f), hi = lo;
          if (base) {
            const float4* src = reinterpret_cast<const float4*>(base + bidx + 16 * h);
            lo = src[0];
            hi = src[1];
          }
          __stcs(dst, lo);
          __stcs(dst + 1, hi);
        }
        if (field_out) {
          float4* f = reinterpret_cast<float4*>(field_out + (size_t)(j0 + row) * nx + i0 + 8 * c);
          f[0] = make_float4(0.f, 0.f, 0.f, 0.f);
          f[1] = f[0];
        }
      }
      return;
    }
  }
  // y pass: items (chunk c of 8 rows, PAIR of columns col, col + 1 <-> nodes i0 - (R+1) + col ...):
  // 8-byte loads, both columns ride in packed FFMA2 pairs
  // (for even R the window starts at an odd node: the pairs then start one column further left)
  constexpr int PO = (R + 1) & 1, NP = CW / 2 + PO;
  for (int it = threadIdx.x; it < 4 * NP; it += BLUR_THREADS) {
    const int c = it / NP, col = 2 * (it - c * NP) - PO;    // first column of the pair (-1 possible)
    const int gi = wrap1(i0 - (R + 1) + col, nx);           // even: aligned, never straddles the x seam
    const int r0 = j0 + 8 * c - 1 - R;                      // first row of the window
    float2 v[NV];
    if (j0 - 1 - R >= 0 && j0 + BLUR_T + 1 + R <= ny) {     // tile away from the y seam: no row wraps
      // row k of the window: one IMAD.WIDE (32-bit row size x immediate k + 64-bit pointer)
      const char* p = reinterpret_cast<const char*>(rho_b + (size_t)r0 * nx + gi);
      const unsigned rowb = (unsigned)nx * (unsigned)sizeof(float);
#pragma unroll
      for (int k = 0; k < NV; ++k)
        v[k] = __ldg(reinterpret_cast<const float2*>(p + (unsigned long long)rowb * (unsigned)k));
    } else {
#pragma unroll
      for (int k = 0; k < NV; ++k)
        v[k] = __ldg(reinterpret_cast<const float2*>(rho_b + (size_t)wrap1(r0 + k, ny) * nx + gi));
    }
    float2 t[10];
#pragma unroll
    for (int a = 0; a < 10; ++a) {
      float2 s2 = make_float2(0.0f, 0.0f);
#pragma unroll
      for (int k = 0; k <= 2 * R; ++k) s2 = ffma2(v[a + k], taps.g[k], s2);
      t[a] = s2;                                            // ty at row j0 + 8c - 1 + a, columns col, col + 1
    }
#pragma unroll
    for (int a = 0; a < 8; ++a) {
      const float2 lo = make_float2(t[a + 1].x, 0.5f * (t[a + 2].x - t[a].x));
      const float2 hi = make_float2(t[a + 1].y, 0.5f * (t[a + 2].y - t[a].y));
      float2* dst = td + (8 * c + a) * CP + col;
      if (PO == 0) {
        *reinterpret_cast<float4*>(dst) = make_float4(lo.x, lo.y, hi.x, hi.y);
      } else {
        if (col >= 0) dst[0] = lo;
        if (col + 1 < CW) dst[1] = hi;
      }
    }
  }
  __syncthreads();
  // x pass: items (row, chunk c of 8 nodes).  A warp takes 8 rows x 4 chunks (its stores fill
  // whole 128-byte lines of the blocked layout); the 8 lanes of a 16-byte shared access are
  // 2 chunks x 4 rows.
  if (threadIdx.x < BLUR_T * 4) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int c = (lane & 1) + 2 * ((lane >> 3) & 1);
    const int row = ((lane >> 1) & 3) + 4 * (lane >> 4) + 8 * wid;
    float2 v[NV];
    {
      const float4* p = reinterpret_cast<const float4*>(td + row * CP + 8 * c);
#pragma unroll
      for (int q = 0; q < NV / 2; ++q) {
        const float4 t4 = p[q];
        v[2 * q] = make_float2(t4.x, t4.y);
        v[2 * q + 1] = make_float2(t4.z, t4.w);
      }
    }
    float2 acc[10];  // .x: filtered density B at node i0 + 8c - 1 + a;  .y: G_x dy at the same node
#pragma unroll
    for (int a = 0; a < 10; ++a) {
      float2 s2 = make_float2(0.0f, 0.0f);
#pragma unroll
      for (int k = 0; k <= 2 * R; ++k) s2 = ffma2(v[a + k], taps.g[k], s2);
      acc[a] = s2;
    }
    float B[10];
#pragma unroll
    for (int a = 0; a < 10; ++a) B[a] = acc[a].x;
    float2 o[8];
#pragma unroll
    for (int a = 0; a < 8; ++a) o[a] = make_float2(coef * (0.5f * (B[a + 2] - B[a])), coef * acc[a + 1].y);
    // nodes (i0 + 8c .. + 7, j0 + row): two 32-byte rows of two neighbouring 4x4 blocks
    const size_t bidx = blk_index(i0 + 8 * c, j0 + row, nx);
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      float4* dst = reinterpret_cast<float4*>(A + bidx + 16 * h);
      float4 lo = make_float4(o[4 * h].x, o[4 * h].y, o[4 * h + 1].x, o[4 * h + 1].y);
      float4 hi = make_float4(o[4 * h + 2].x, o[4 * h + 2].y, o[4 * h + 3].x, o[4 * h + 3].y);
      if (base) {
        const float4* src = reinterpret_cast<const float4*>(base + bidx + 16 * h);
        const float4 b0 = src[0], b1 = src[1];
        lo.x += b0.x; lo.y += b0.y; lo.z += b0.z; lo.w += b0.w;
        hi.x += b1.x; hi.y += b1.y; hi.z += b1.z; hi.w += b1.w;
      }
      __stcs(dst, lo);
      __stcs(dst + 1, hi);
    }
    if (field_out) {
      float4* f = reinterpret_cast<float4*>(field_out + (size_t)(j0 + row) * nx + i0 + 8 * c);
      f[0] = make_float4(B[1], B[2], B[3], B[4]);
      f[1] = make_float4(B[5], B[6], B[7], B[8]);
    }
  }
}

// Static-source field ("persistent scalar energy field consisting of Gaussian packets"):
// c(g) = sum_s A_s exp(-|g - x_s|^2 / (2 w_s^2)), periodic minimum image (reading 17).
__device__ inline double static_c(int nx, int ny, int n_src, const float* __restrict__ src, int i, int j) {
  double s = 0.0;
  for (int k = 0; k < n_src; ++k) {
    double dx = (double)i - (double)src[4 * k], dy = (double)j - (double)src[4 * k + 1];
    dx -= nx * nearbyint(dx / nx);
    dy -= ny * nearbyint(dy / ny);
    const double wd = (double)src[4 * k + 3];
    s += (double)src[4 * k + 2] * exp(-(dx * dx + dy * dy) / (2.0 * wd * wd));
  }
  return s;
}

// Runs once per static field at mc_create (not on the hot path): c, csum += c and
// As += coef * central-difference gradient of c.  The difference is taken in fp64 before
// rounding, because c is O(1) and its gradient O(1e-2): differencing fp32-rounded c would
// cost two digits of the force.
__global__ void k_static_init(int nx, int ny, int n_src, const float* __restrict__ src, float coef,
                              float* __restrict__ c_out, float* __restrict__ csum,
                              float2* __restrict__ As) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
  if (i >= nx) return;
  const size_t g = (size_t)j * nx + i;
  const double c = static_c(nx, ny, n_src, src, i, j);
  const double gx = 0.5 * (static_c(nx, ny, n_src, src, wrap1(i + 1, nx), j) -
                           static_c(nx, ny, n_src, src, wrap1(i - 1, nx), j));
  const double gy = 0.5 * (static_c(nx, ny, n_src, src, i, wrap1(j + 1, ny)) -
                           static_c(nx, ny, n_src, src, i, wrap1(j - 1, ny)));
  c_out[g] = (float)c;
  csum[g] += (float)c;
  const size_t bg = blk_index(i, j, nx);  // blocked like A
  float2 a = As[bg];
  a.x += (float)((double)coef * gx);
  a.y += (float)((double)coef * gy);
  As[bg] = a;
}

}  // namespace mc

// k_blur.cuh -- K3a: S3 Gaussian filter + gradient of the deposited bead density, one pass
// through shared memory.
//
// "node positions are deposited onto a grid, diffused with a Gaussian filter via FFT
// convolution to produce a density field, and the gradient of this density field generates
// repulsive forces."  Reading 14: the filter is the periodic convolution with the sampled,
// normalised Gaussian truncated at R (= the paper's filter to 2.6e-8 at R = 5 sigma), applied
// along x then along y; reading 15: second-order central difference.
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

// shared-memory geometry for radius R.  The input tile starts P nodes left of the output tile,
// P the smallest multiple of 4 >= R+1, so that every global and shared access of the x pass is
// a 16-byte one; the x pass then produces its outputs from column i0 - 1 - S on, S = P - 1 - R.
__host__ __device__ constexpr int blur_P(int R) { return 4 * ((R + 1 + 3) / 4); }
__host__ __device__ constexpr int blur_S(int R) { return blur_P(R) - 1 - R; }
__host__ __device__ constexpr int blur_NC(int R) { return (BLUR_T + 2 + blur_S(R) + 3) / 4; }  // x chunks
__host__ __device__ constexpr int blur_TWP(int R) { return 4 * blur_NC(R); }                    // filtered pitch
__host__ __device__ constexpr int blur_HP(int R) { return 4 * ((blur_TWP(R) + 2 * R + 3) / 4); } // input pitch
__host__ __device__ constexpr int blur_H(int R) { return BLUR_T + 2 * R + 2; }                  // input rows
__host__ __device__ constexpr size_t blur_smem_bytes(int R) {
  return sizeof(float) * ((size_t)blur_H(R) * blur_HP(R) + (size_t)(blur_H(R) + 4) * blur_TWP(R));
}

// One CTA filters one 32x32 tile.  Stages (all in shared memory, one read of rho_b per node plus
// the halo, one write of the gradient):
//   load  H x HP nodes of rho_b with 16-byte loads, periodic indices
//   x pass: each thread produces 4 consecutive outputs of one row from a register window
//           (4+2R inputs fetched with 16-byte LDS)                       -> tmp[H][TWP]
//   y pass: each thread produces 4 consecutive outputs of one column    -> bl[36][TWP]
//   central difference, scale by the signed coupling, add the base field, store float2.
// coef: lattice coupling with the sign of the force.  base: interleaved field added to the
// result (static part, or the running sum over earlier bead-density fields), may be NULL.
// A: interleaved (x,y) force-gradient field.  field_out (filtered density) may be NULL.
template <int R>
__global__ void __launch_bounds__(256) k_blur_grad(int nx, int ny, BlurTaps taps,
                                                   const float* __restrict__ rho_b, float coef,
                                                   const float2* base, float2* A,
                                                   float* __restrict__ field_out) {
  extern __shared__ __align__(16) float sm[];
  constexpr int H = blur_H(R), HP = blur_HP(R), TWP = blur_TWP(R), NC = blur_NC(R);
  constexpr int P = blur_P(R), S = blur_S(R);
  constexpr int NV = 4 + 2 * R, NV4 = (NV + 3) / 4, HP4 = HP / 4;
  float* in = sm;                    // [H][HP]    in[y][x]  <-> node (j0-R-1+y, i0-P+x)
  float* tmp = sm + (size_t)H * HP;  // [H+4][TWP] tmp[y][t] <-> node (j0-R-1+y, i0-1-S+t)
  // 1-D grid in row-major tile order (2-D grids are rasterised in an order that streams worse)
  const int ntx = nx / BLUR_T;
  const int i0 = (blockIdx.x % ntx) * BLUR_T, j0 = (blockIdx.x / ntx) * BLUR_T;
  float g[2 * R + 1];
#pragma unroll
  for (int k = 0; k <= 2 * R; ++k) g[k] = taps.g[k];
  const int nx4 = nx >> 2, gc0 = (i0 - P) >> 2;  // arithmetic shift: i0 - P may be negative
  for (int it = threadIdx.x; it < H * HP4; it += 256) {
    const int y = it / HP4, v = it - y * HP4;
    const int gj = wrap1(j0 - R - 1 + y, ny);  // halo <= R+1 < ny
    const int gc = wrap1(gc0 + v, nx4);
    reinterpret_cast<float4*>(in)[it] = __ldg(reinterpret_cast<const float4*>(rho_b + (size_t)gj * nx) + gc);
  }
  __syncthreads();
  // x pass: items (row y, chunk c of 4 outputs)
  for (int it = threadIdx.x; it < H * NC; it += 256) {
    const int y = it / NC, c = it - y * NC;
    float v[4 * NV4];
    const float4* p = reinterpret_cast<const float4*>(in + y * HP + 4 * c);
#pragma unroll
    for (int q = 0; q < NV4; ++q) {
      const float4 t = p[q];
      v[4 * q] = t.x; v[4 * q + 1] = t.y; v[4 * q + 2] = t.z; v[4 * q + 3] = t.w;
    }
    float o[4];
#pragma unroll
    for (int a = 0; a < 4; ++a) {
      float s = 0.0f;
#pragma unroll
      for (int k = 0; k <= 2 * R; ++k) s = fmaf(g[k], v[a + k], s);
      o[a] = s;
    }
    *reinterpret_cast<float4*>(tmp + y * TWP + 4 * c) = make_float4(o[0], o[1], o[2], o[3]);
  }
  for (int x = threadIdx.x; x < 4 * TWP; x += 256) tmp[H * TWP + x] = 0.0f;  // pad rows
  __syncthreads();
  // y pass: items (chunk c of 4 output rows, column t); bl[36][TWP] overwrites `in`
  float* bl = in;                    // bl[y][t] <-> node (j0-1+y, i0-1-S+t)
  for (int it = threadIdx.x; it < 9 * TWP; it += 256) {
    const int c = it / TWP, x = it - c * TWP;
    float v[NV];
#pragma unroll
    for (int k = 0; k < NV; ++k) v[k] = tmp[(4 * c + k) * TWP + x];
#pragma unroll
    for (int a = 0; a < 4; ++a) {
      float s = 0.0f;
#pragma unroll
      for (int k = 0; k <= 2 * R; ++k) s = fmaf(g[k], v[a + k], s);
      bl[(4 * c + a) * TWP + x] = s;
    }
  }
  __syncthreads();
  for (int t = threadIdx.x; t < BLUR_T * BLUR_T; t += 256) {
    // 16 consecutive threads own one 4x4 block of the blocked output: a warp stores two full lines
    const int bl_id = t >> 4, n = t & 15;
    const int y = ((bl_id >> 3) << 2) + (n >> 2), xo = ((bl_id & 7) << 2) + (n & 3), x = xo + S;
    const float gx = 0.5f * (bl[(y + 1) * TWP + x + 2] - bl[(y + 1) * TWP + x]);
    const float gy = 0.5f * (bl[(y + 2) * TWP + x + 1] - bl[y * TWP + x + 1]);
    const size_t gidx = (size_t)(j0 + y) * nx + (i0 + xo);
    float2 a = make_float2(coef * gx, coef * gy);
    const size_t bidx = blk_index(i0 + xo, j0 + y, nx);  // A and base are blocked (mc_common.cuh)
    if (base) { const float2 b = base[bidx]; a.x += b.x; a.y += b.y; }
    A[bidx] = a;
    if (field_out) field_out[gidx] = bl[(y + 1) * TWP + x + 1];
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

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

__host__ __device__ inline size_t blur_smem_bytes(int R) {
  const int H = BLUR_T + 2 * R + 2;
  return sizeof(float) * ((size_t)H * H + (size_t)H * (BLUR_T + 2));
}

// coef: lattice coupling with sign.  base0/base1: planes added to the result (static part or the
// running sum over earlier bead-density fields), may be NULL.  field_out may be NULL.
__global__ void __launch_bounds__(256) k_blur_grad(int nx, int ny, int R, BlurTaps taps,
                                                   const float* __restrict__ rho_b, float coef,
                                                   const float* base0, const float* base1,
                                                   float* A0, float* A1, float* __restrict__ field_out) {
  extern __shared__ float sm[];
  const int H = BLUR_T + 2 * R + 2;   // input tile side
  const int TW = BLUR_T + 2;          // blurred tile side (one-cell halo for the gradient)
  float* in = sm;                     // [H][H]
  float* tmp = sm + (size_t)H * H;    // [H][TW]
  const int i0 = blockIdx.x * BLUR_T, j0 = blockIdx.y * BLUR_T;
  for (int t = threadIdx.x; t < H * H; t += blockDim.x) {
    const int y = t / H, x = t - y * H;
    const int gi = wrapi(i0 - R - 1 + x, nx), gj = wrapi(j0 - R - 1 + y, ny);
    in[t] = __ldg(rho_b + (size_t)gj * nx + gi);
  }
  __syncthreads();
  // along x
  for (int t = threadIdx.x; t < H * TW; t += blockDim.x) {
    const int y = t / TW, x = t - y * TW;
    const float* r = in + y * H + x;
    float s = 0.0f;
    for (int k = 0; k <= 2 * R; ++k) s = fmaf(taps.g[k], r[k], s);
    tmp[t] = s;
  }
  __syncthreads();
  // along y; result bl[TW][TW] overwrites the front of `in`
  float* bl = in;
  for (int t = threadIdx.x; t < TW * TW; t += blockDim.x) {
    const int y = t / TW, x = t - y * TW;
    const float* c = tmp + y * TW + x;
    float s = 0.0f;
    for (int k = 0; k <= 2 * R; ++k) s = fmaf(taps.g[k], c[k * TW], s);
    bl[t] = s;
  }
  __syncthreads();
  for (int t = threadIdx.x; t < BLUR_T * BLUR_T; t += blockDim.x) {
    const int y = t >> 5, x = t & 31;
    const float gx = 0.5f * (bl[(y + 1) * TW + x + 2] - bl[(y + 1) * TW + x]);
    const float gy = 0.5f * (bl[(y + 2) * TW + x + 1] - bl[y * TW + x + 1]);
    const size_t g = (size_t)(j0 + y) * nx + (i0 + x);
    float a0 = coef * gx, a1 = coef * gy;
    if (base0) { a0 += base0[g]; a1 += base1[g]; }
    A0[g] = a0;
    A1[g] = a1;
    if (field_out) field_out[g] = bl[(y + 1) * TW + x + 1];
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
                              float* __restrict__ As0, float* __restrict__ As1) {
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
  As0[g] += (float)((double)coef * gx);
  As1[g] += (float)((double)coef * gy);
}

}  // namespace mc

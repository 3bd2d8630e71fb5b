// k_filament.cuh -- K1: S0 actuation + S1 elastic PBD displacement (Eq. 1-4) + S4 field forces.
//
// One warp per chain; lane <-> bead; neighbour beads are exchanged with warp shuffles
// (north_star (1)).  A chain longer than 32 beads is walked in windows of 32 beads that
// overlap by 4 (D_i needs X_{i-2..i+2}).
//
// Paper: bending pass Eq. 1, position pass Eq. 2-4.
// Readings: 1 the net PBD displacement D_i becomes the bead force kappa*D_i;
// 2 edge angles come from the current geometry; 3 one Jacobi iteration; 4 joint angle =
// atan2(cross, dot); 5 free ends; 18 theta*_i(n) = theta0_i + a_i sin(2 pi n dt/T_i + phi_i).
//
// Precision.  State and parameters are fp32 and so is most of the arithmetic, but D_i is a
// difference of differences: |D| ~ 1e-4 is formed from edge vectors of length ~1 and joint
// angles ~0.3 rad, so plain fp32 leaves ~1e-5 relative error on the force (measured, DESIGN.md
// "Precision") -- at the parity bar.  The three cancelling quantities are therefore formed
// in fp64 from the exact fp32 inputs and rounded once: edge vector v = X_{i+1} - X_i,
// |v|^2 - L^2, and the joint angle psi - theta* (cross, dot, atan2 and the actuation phase).
#pragma once
#include "mc_common.cuh"

namespace mc {

struct FilamentArgs {
  const int* offsets;     // [n_fil+1]
  int n_fil;
  const float2* X;        // [N]
  const float4* P0;       // {L_rest, theta_rest, act_amp, act_phase}
  const float4* P1;       // {k_bend, k_shear, k_stretch, act_period}
  float2* F;              // [N] out: total bead force
  float* sense;           // [N] out (only written when csum != NULL)
  const float* A0;        // force-gradient planes (may be NULL: no field forces)
  const float* A1;
  const float* csum;      // sum of static fields (may be NULL)
  int nx, ny;
  float kappa;            // k_el * dt^2
  double t;               // n * dt (step index before the increment)
};

__global__ void __launch_bounds__(256) k_filament_force(FilamentArgs a) {
  const int lane = threadIdx.x & 31;
  const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int n_warps = (gridDim.x * blockDim.x) >> 5;
  const double TWO_PI = 6.283185307179586476925286766559;
  const unsigned FULL = 0xffffffffu;
  for (int f = warp; f < a.n_fil; f += n_warps) {
    const int b0 = a.offsets[f];
    const int m = a.offsets[f + 1] - b0;
    for (int base = 0;; base += 28) {
      const bool last = (base + 32 >= m);
      const int i = base + lane;
      const bool valid = i < m;
      float2 x = make_float2(0.f, 0.f);
      float4 p0 = make_float4(1.f, 0.f, 0.f, 0.f), p1 = make_float4(0.f, 0.f, 0.f, 1.f);
      if (valid) {
        x = a.X[b0 + i];
        p0 = a.P0[b0 + i];
        p1 = a.P1[b0 + i];
      }
      // edge i = (i, i+1): v = X_{i+1} - X_i
      const double xd = (double)x.x, yd = (double)x.y;
      const double xn = __shfl_down_sync(FULL, xd, 1), yn = __shfl_down_sync(FULL, yd, 1);
      const bool has_edge = (i + 1 < m) && (lane < 31);
      const double vx = has_edge ? xn - xd : 1.0, vy = has_edge ? yn - yd : 0.0;
      // joint i (between edge i-1 and edge i): C = psi - theta*   (Eq. 1's C_bend)
      const double pvx = __shfl_up_sync(FULL, vx, 1), pvy = __shfl_up_sync(FULL, vy, 1);
      const bool has_joint = (i >= 1) && (i + 1 < m) && (lane >= 1) && (lane < 31);
      float hkC = 0.0f;  // (1/2) k_bend C
      if (has_joint) {
        const double cross = pvx * vy - pvy * vx, dot = pvx * vx + pvy * vy;
        const double psi = atan2(cross, dot);
        double ph = TWO_PI * (a.t / (double)p1.w) + (double)p0.w;
        ph -= TWO_PI * rint(ph * (1.0 / TWO_PI));
        const float s = sinf((float)ph);
        const double theta_star = (double)p0.y + (double)(p0.z * s);
        hkC = 0.5f * p1.x * (float)(psi - theta_star);
      }
      // Eq. 1 applied to edge i: theta_1 of joint i+1 (+), theta_2 of joint i (-)
      const float hkC_next = __shfl_down_sync(FULL, hkC, 1);
      const float delta = hkC_next - hkC;
      float dx = 0.0f, dy = 0.0f;  // Delta x of edge i (Eq. 3)
      if (has_edge) {
        const double l2 = vx * vx + vy * vy;
        const float L = p0.x;
        const float ell = sqrtf((float)l2);
        const float dl = (float)(l2 - (double)L * (double)L) / (ell + L);  // |v| - L_rest
        const float inv = 1.0f / ell;
        const float tx = (float)vx * inv, ty = (float)vy * inv;
        const float sd = sinf(delta), sh = sinf(0.5f * delta);
        const float omc = 2.0f * sh * sh;  // 1 - cos(delta)
        // t - d, d = Rot(delta) t  (director after the bending pass)
        const float ex = omc * tx + sd * ty, ey = omc * ty - sd * tx;
        const float ksL = p1.y * L;
        dx = 0.5f * p1.z * fmaf(ksL, ex, dl * tx);
        dy = 0.5f * p1.z * fmaf(ksL, ey, dl * ty);
      }
      // Eq. 4 summed per bead: D_i = Delta_i - Delta_{i-1}
      const float pdx = __shfl_up_sync(FULL, dx, 1), pdy = __shfl_up_sync(FULL, dy, 1);
      float Dx = dx, Dy = dy;
      if (lane >= 1) { Dx -= pdx; Dy -= pdy; }
      const bool out = valid && (base == 0 || lane >= 2) && (last || lane <= 29);
      if (out) {
        float Fx = a.kappa * Dx, Fy = a.kappa * Dy;
        if (a.A0) {
          const float2 g = interp2(a.A0, a.A1, a.nx, a.ny, x.x, x.y);
          Fx += g.x;
          Fy += g.y;
        }
        a.F[b0 + i] = make_float2(Fx, Fy);
        if (a.csum) a.sense[b0 + i] = interp1(a.csum, a.nx, a.ny, x.x, x.y);
      }
      if (last) break;
    }
  }
}

// mc_load_filaments: pack the per-bead parameters and validate them (flag != 0 => invalid)
__global__ void k_pack_params(int N, const float* __restrict__ xy, const float* __restrict__ L_rest,
                              const float* __restrict__ theta_rest, const float* __restrict__ k_bend,
                              const float* __restrict__ k_shear, const float* __restrict__ k_stretch,
                              const float* __restrict__ act_amp, const float* __restrict__ act_phase,
                              const float* __restrict__ act_period, float2* __restrict__ X,
                              float4* __restrict__ P0, float4* __restrict__ P1, int* __restrict__ flag) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= N) return;
  X[b] = make_float2(xy[2 * b], xy[2 * b + 1]);
  const float kb = k_bend[b], ks = k_shear[b], kst = k_stretch[b], T = act_period[b];
  P0[b] = make_float4(L_rest[b], theta_rest[b], act_amp[b], act_phase[b]);
  P1[b] = make_float4(kb, ks, kst, T);
  if (!(kb >= 0.f && kb <= 1.f && ks >= 0.f && ks <= 1.f && kst >= 0.f && kst <= 1.f)) atomicOr(flag, 1);
  if (!(T > 0.f)) atomicOr(flag, 2);
}

}  // namespace mc

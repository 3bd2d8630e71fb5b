// k_pbd.cuh -- the general form of K1: literal PBD (reading 27) and
// the two-layer gathers of S4 (NEXT-4; reading 28).  The one-iteration Jacobi kernel of
// k_filament.cuh stays the fast path of the default configuration; this kernel runs when
//   pbd_iters > 1, pbd_order = Gauss-Seidel, the rest length is actuated, two_layer is on,
//   or as the PROJECTION pass after S7 (pbd_project).
//
// Paper: "PBD ... an iterative constraint projection method ... Each iteration decouples the solver
// into two phases.  First, a bending pass updates theta toward theta_rest.  Second, a position
// pass enforces nodal connectivity by resolving stretch and shear errors based on the updated
// orientations and rest length L_rest" (Eq. 1-4); "The CPPN outputs the rest
// angle theta_rest and the rest length L_rest".
//
// Mapping: as in k_filament.cuh a warp owns a window of 64 consecutive beads, two per lane, and
// everything stays in registers and shuffles across ALL iterations.  The working positions
// Y^k = X + Dtot^k are never formed: at |X| ~ 6000 an fp32 Y would lose the displacement (ulp
// 4.9e-4).  Instead each lane keeps its two EDGE VECTORS in fp64 (exact differences of the fp32
// positions at k = 0) and adds the differences of the beads' fp32 displacements after every
// iteration; every quantity of Eq. 1-4 is a function of edge vectors only.
// One iteration needs the beads i-2..i+2 (Jacobi) or i-3..i+3 (red-black Gauss-Seidel) of a bead,
// so K iterations need a halo of K (Jacobi) or ceil(3K/2) (Gauss-Seidel) LANES on either side of
// the window's output lanes; windows advance by 64 - 4 * halo_lanes beads.  When every chain has
// the same length m and m divides 64 the windows are aligned to chain starts and need no halo.
//
// Gauss-Seidel (order 1): bending pass for all joints from the iteration's start state; position
// pass over the EVEN edges of each chain (parity of the edge's first bead within its chain,
// BEAD_ODD flag) from the start state, Eq. 4 applied; then over the ODD edges, whose edge vector
// and Kirchhoff-Love error are those of the start state plus the difference w of their end beads'
// phase-1 displacements (v' = v + w, v' - L d = (v - L d) + w: the director d of the bending pass
// is kept), exactly the oracle's order of operations.
#pragma once
#include "k_filament.cuh"

namespace mc {

struct PbdArgs {
  FilamentArgs f;
  const float* PE;      // [N] rest-length actuation amplitude of edge (i, i+1), or NULL
  const float2* O;      // [N] two-layer marker offset h n_i (markers X_i +- O_i), or NULL
  float2* Dp;           // projection mode: out [N] net displacement (no force, no gathers); else NULL
  int iters;            // K >= 1
  int order;            // 0 Jacobi, 1 red-black Gauss-Seidel
  int halo_lanes;       // lanes of halo on either side of an overlapping window
  long long step_off;   // added to *f.step (projection runs after K4 incremented it: -1)
};

// sin(2 pi n dt / T + phi): the one sine that drives theta* and L* of a bead's entry (reading 18,
// 27).  Same reduction as half_kC (k_filament.cuh).
__device__ __forceinline__ float act_sine(const BeadParams& p, double n_step) {
  const double TWO_PI = 6.283185307179586476925286766559;
  double turns = n_step * (double)p.rhi + n_step * (double)p.rlo;
  turns -= rint(turns);
  double ph = TWO_PI * turns + (double)p.phase;
  ph -= TWO_PI * rint(ph * (1.0 / TWO_PI));
  return sin_pi((float)ph);
}

// (1/2) k_bend C_bend of the joint between edge pv (incoming) and v (outgoing), Eq. 1, with the
// actuation term amp * sine given (half_kC of k_filament.cuh with the sine hoisted out of the
// iteration loop).
__device__ __forceinline__ float half_kC_s(double pvx, double pvy, double vx, double vy, const BeadParams& p, float as) {
  const double cross = pvx * vy - pvy * vx, dot = pvx * vx + pvy * vy;
  const double c = (double)p.c0, s = (double)p.s0;
  const double dotp = dot * c + cross * s, crossp = cross * c - dot * s;
  const float yf = (float)crossp, xf = (float)dotp;
  float psi_p = (xf > 0.0f && fabsf(yf) <= 0.5f * xf) ? atan_small(yf, xf) : atan2f(yf, xf);
  if (!(dot > 0.0 && dotp > 0.0)) {
    const float t = psi_p + atan2f(p.s0, p.c0);
    if (t > 3.14159265358979f) psi_p -= 6.28318530717959f;
    else if (t <= -3.14159265358979f) psi_p += 6.28318530717959f;
  }
  return 0.5f * p.kb * (psi_p - p.eps - as);
}

// The pieces of Eq. 2-3 of one edge at the start of an iteration, all free of cancellation:
//   cs = C_stretch = (|v| - L) t,   ex = L (t - d) with d = Rot(delta) t,
// so that v - L d = cs + ex and Delta x = (k_st/2) [cs + k_sh ex].
struct EdgeStart {
  float2 cs, ex;
};
__device__ __forceinline__ EdgeStart edge_start(double vx, double vy, float delta, float L) {
  const double l2 = vx * vx + vy * vy;
  const float ell = sqrtf((float)l2);
  const float dl = (float)(l2 - (double)L * (double)L) / (ell + L);
  const float inv = 1.0f / ell;
  const float tx = (float)vx * inv, ty = (float)vy * inv;
  const float sd = sin_small(delta), sh = sin_small(0.5f * delta);
  const float omc = 2.0f * sh * sh;
  EdgeStart r;
  r.cs = make_float2(dl * tx, dl * ty);
  r.ex = make_float2(L * (omc * tx + sd * ty), L * (omc * ty - sd * tx));
  return r;
}
__device__ __forceinline__ float2 edge_dx(const EdgeStart& e, float ks, float kst) {
  return make_float2(0.5f * kst * fmaf(ks, e.ex.x, e.cs.x), 0.5f * kst * fmaf(ks, e.ex.y, e.cs.y));
}
// Delta x of an ODD edge in the Gauss-Seidel pass: its end beads moved by w in phase 1.
//   v' = v + w;  C_stretch' from v';  v' - L d = (cs + ex) + w
__device__ __forceinline__ float2 edge_dx_moved(double vx, double vy, const EdgeStart& e, float2 w, float L, float ks,
                                                float kst) {
  const double nvx = vx + (double)w.x, nvy = vy + (double)w.y;
  const double l2 = nvx * nvx + nvy * nvy;
  const float ell = sqrtf((float)l2);
  const float dl = (float)(l2 - (double)L * (double)L) / (ell + L);
  const float inv = 1.0f / ell;
  const float csx = dl * (float)nvx * inv, csy = dl * (float)nvy * inv;
  const float klx = (e.cs.x + e.ex.x) + w.x, kly = (e.cs.y + e.ex.y) + w.y;   // v' - L d
  return make_float2(0.5f * kst * fmaf(ks, klx - csx, csx), 0.5f * kst * fmaf(ks, kly - csy, csy));
}

template <bool UNIFORM>
__global__ void __launch_bounds__(128) k_filament_pbd(PbdArgs g, size_t wstride) {
  g.f.shift(blockIdx.y * wstride);
  g.PE = wshift(g.PE, blockIdx.y * wstride);
  g.O = wshift(g.O, blockIdx.y * wstride);
  g.Dp = wshift(g.Dp, blockIdx.y * wstride);
  const FilamentArgs& a = g.f;
  const int lane = threadIdx.x & 31;
  const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (w >= a.n_windows) return;
  const unsigned FULL = 0xffffffffu;
  const bool aligned = (a.stride == 64);
  const int HL = aligned ? 0 : g.halo_lanes;
  const int base = w * a.stride - 2 * HL;  // even => float4-aligned pairs
  const int bA = base + 2 * lane, bB = bA + 1;
  const bool vA = bA >= 0 && bA < a.N, vB = bB >= 0 && bB < a.N;
  float2 xa = make_float2(0.f, 0.f), xb = make_float2(1.f, 0.f);
  if (vA && vB) {
    const float4 q = __ldg(reinterpret_cast<const float4*>(a.X + bA));
    xa = make_float2(q.x, q.y);
    xb = make_float2(q.z, q.w);
  } else {
    if (vA) xa = __ldg(a.X + bA);
    if (vB) xb = __ldg(a.X + bB);
  }
  const BeadParams pA = load_params<UNIFORM>(a, bA, vA), pB = load_params<UNIFORM>(a, bB, vB);
  const float bLA = (g.PE && vA) ? __ldg(g.PE + bA) : 0.0f, bLB = (g.PE && vB) ? __ldg(g.PE + bB) : 0.0f;
  const float nxa = __shfl_down_sync(FULL, xa.x, 1), nya = __shfl_down_sync(FULL, xa.y, 1);
  // edge vectors in fp64: exact at k = 0, then updated by differences of displacements
  double eAx = (double)xb.x - (double)xa.x, eAy = (double)xb.y - (double)xa.y;  // A -> B
  double eBx = (double)nxa - (double)xb.x, eBy = (double)nya - (double)xb.y;    // B -> next A
  const bool firstA = (pA.flags & BEAD_FIRST) != 0, firstB = (pB.flags & BEAD_FIRST) != 0;
  const bool edgeA = !(pA.flags & BEAD_LAST) && vB;
  const bool edgeB = !(pB.flags & BEAD_LAST) && lane < 31;
  const bool jointA = !(pA.flags & (BEAD_FIRST | BEAD_LAST)) && lane >= 1;
  const bool jointB = !(pB.flags & (BEAD_FIRST | BEAD_LAST)) && lane < 31;
  const bool oddA = (pA.flags & BEAD_ODD) != 0, oddB = (pB.flags & BEAD_ODD) != 0;
  // S0: targets of this step, the same for all iterations
  const double n_step = (double)(*a.step + g.step_off);
  const float sA = act_sine(pA, n_step), sB = act_sine(pB, n_step);
  const float asA = pA.amp * sA, asB = pB.amp * sB;
  const float LA = fmaf(bLA, sA, pA.L), LB = fmaf(bLB, sB, pB.L);
  float2 DtA = make_float2(0.f, 0.f), DtB = make_float2(0.f, 0.f);
  for (int k = 0; k < g.iters; ++k) {
    // bending pass (Eq. 1) from the current edge vectors
    const double ePx = __shfl_up_sync(FULL, eBx, 1), ePy = __shfl_up_sync(FULL, eBy, 1);  // prev B -> A
    const float hA = jointA ? half_kC_s(ePx, ePy, eAx, eAy, pA, asA) : 0.0f;
    const float hB = jointB ? half_kC_s(eAx, eAy, eBx, eBy, pB, asB) : 0.0f;
    const float hA_next = __shfl_down_sync(FULL, hA, 1);
    EdgeStart stA, stB;
    stA.cs = stA.ex = stB.cs = stB.ex = make_float2(0.f, 0.f);
    if (edgeA) stA = edge_start(eAx, eAy, hB - hA, LA);
    if (edgeB) stB = edge_start(eBx, eBy, hA_next - hB, LB);
    float2 DA, DB;
    if (g.order == 0) {
      // Jacobi position pass: every edge from the start state, Eq. 4 summed per bead
      const float2 dA = edgeA ? edge_dx(stA, pA.ks, pA.kst) : make_float2(0.f, 0.f);
      const float2 dB = edgeB ? edge_dx(stB, pB.ks, pB.kst) : make_float2(0.f, 0.f);
      float pdx = __shfl_up_sync(FULL, dB.x, 1), pdy = __shfl_up_sync(FULL, dB.y, 1);
      if (firstA || lane == 0) { pdx = 0.f; pdy = 0.f; }
      DA = make_float2(dA.x - pdx, dA.y - pdy);
      DB = firstB ? dB : make_float2(dB.x - dA.x, dB.y - dA.y);
    } else {
      // red-black Gauss-Seidel: even edges first
      const float2 d1A = (edgeA && !oddA) ? edge_dx(stA, pA.ks, pA.kst) : make_float2(0.f, 0.f);
      const float2 d1B = (edgeB && !oddB) ? edge_dx(stB, pB.ks, pB.kst) : make_float2(0.f, 0.f);
      float p1x = __shfl_up_sync(FULL, d1B.x, 1), p1y = __shfl_up_sync(FULL, d1B.y, 1);
      if (firstA || lane == 0) { p1x = 0.f; p1y = 0.f; }
      const float2 P1A = make_float2(d1A.x - p1x, d1A.y - p1y);
      const float2 P1B = firstB ? d1B : make_float2(d1B.x - d1A.x, d1B.y - d1A.y);
      const float nP1x = __shfl_down_sync(FULL, P1A.x, 1), nP1y = __shfl_down_sync(FULL, P1A.y, 1);
      // odd edges on the moved beads
      float2 d2A = make_float2(0.f, 0.f), d2B = make_float2(0.f, 0.f);
      if (edgeA && oddA)
        d2A = edge_dx_moved(eAx, eAy, stA, make_float2(P1B.x - P1A.x, P1B.y - P1A.y), LA, pA.ks, pA.kst);
      if (edgeB && oddB)
        d2B = edge_dx_moved(eBx, eBy, stB, make_float2(nP1x - P1B.x, nP1y - P1B.y), LB, pB.ks, pB.kst);
      float p2x = __shfl_up_sync(FULL, d2B.x, 1), p2y = __shfl_up_sync(FULL, d2B.y, 1);
      if (firstA || lane == 0) { p2x = 0.f; p2y = 0.f; }
      DA = make_float2(P1A.x + (d2A.x - p2x), P1A.y + (d2A.y - p2y));
      DB = firstB ? make_float2(P1B.x + d2B.x, P1B.y + d2B.y)
                  : make_float2(P1B.x + (d2B.x - d2A.x), P1B.y + (d2B.y - d2A.y));
    }
    DtA.x += DA.x; DtA.y += DA.y;
    DtB.x += DB.x; DtB.y += DB.y;
    if (k + 1 < g.iters) {
      const float nDx = __shfl_down_sync(FULL, DA.x, 1), nDy = __shfl_down_sync(FULL, DA.y, 1);
      eAx += (double)(DB.x - DA.x); eAy += (double)(DB.y - DA.y);
      eBx += (double)(nDx - DB.x);  eBy += (double)(nDy - DB.y);
    }
  }
  const bool out = aligned || (lane >= HL && lane <= 31 - HL);
  const bool oA = out && vA, oB = out && vB;
  if (g.Dp) {  // projection pass: the displacement itself
    if (oA && oB) {
      *reinterpret_cast<float4*>(g.Dp + bA) = make_float4(DtA.x, DtA.y, DtB.x, DtB.y);
    } else {
      if (oA) g.Dp[bA] = DtA;
      if (oB) g.Dp[bB] = DtB;
    }
    return;
  }
  float2 FA = make_float2(a.kappa * DtA.x, a.kappa * DtA.y), FB = make_float2(a.kappa * DtB.x, a.kappa * DtB.y);
  float2 oa = make_float2(0.f, 0.f), ob = make_float2(0.f, 0.f);
  if (g.O) {
    if (oA) oa = __ldg(g.O + bA);
    if (oB) ob = __ldg(g.O + bB);
  }
  if (a.A) {
    if (oA) {
      if (g.O) {  // two layers: the mean of the samples at the two markers (reading 28)
        const float2 gp = interp2_off(a.A, a.nx, a.ny, xa.x, xa.y, oa.x, oa.y);
        const float2 gm = interp2_off(a.A, a.nx, a.ny, xa.x, xa.y, -oa.x, -oa.y);
        FA.x += 0.5f * (gp.x + gm.x); FA.y += 0.5f * (gp.y + gm.y);
      } else {
        const float2 gq = interp2_pair<0>(a.A, a.nx, a.ny, xa.x, xa.y);
        FA.x += gq.x; FA.y += gq.y;
      }
    }
    if (oB) {
      if (g.O) {
        const float2 gp = interp2_off(a.A, a.nx, a.ny, xb.x, xb.y, ob.x, ob.y);
        const float2 gm = interp2_off(a.A, a.nx, a.ny, xb.x, xb.y, -ob.x, -ob.y);
        FB.x += 0.5f * (gp.x + gm.x); FB.y += 0.5f * (gp.y + gm.y);
      } else {
        const float2 gq = interp2_pair<0>(a.A, a.nx, a.ny, xb.x, xb.y);
        FB.x += gq.x; FB.y += gq.y;
      }
    }
  }
  if (a.tile_fmax) {
    // bound for the fixed-point scale of S5, as in k_filament_force: the warp's maximum on every
    // tile its beads lie in.  (Two-layer markers sit within one node of their bead: the 3x3 tile
    // neighbourhood the spread kernel reads covers them.)
    float m = 0.0f;
    if (oA) m = fmaxf(fabsf(FA.x), fabsf(FA.y));
    if (oB) m = fmaxf(m, fmaxf(fabsf(FB.x), fabsf(FB.y)));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(FULL, m, o));
    const unsigned mb = __float_as_uint(m);
    const int ntx = a.nx >> 5;
    const int tA = oA ? (wrapi((int)floorf(xa.y), a.ny) >> 5) * ntx + (wrapi((int)floorf(xa.x), a.nx) >> 5) : -1;
    const int tB = oB ? (wrapi((int)floorf(xb.y), a.ny) >> 5) * ntx + (wrapi((int)floorf(xb.x), a.nx) >> 5) : -1;
    const unsigned pa = __match_any_sync(FULL, tA), pb = __match_any_sync(FULL, tB);
    if (tA >= 0 && lane == __ffs(pa) - 1 && mb > a.tile_fmax[tA]) atomicMax(a.tile_fmax + tA, mb);
    if (tB >= 0 && tB != tA && lane == __ffs(pb) - 1 && mb > a.tile_fmax[tB]) atomicMax(a.tile_fmax + tB, mb);
  }
  if (oA && oB) {
    *reinterpret_cast<float4*>(a.F + bA) = make_float4(FA.x, FA.y, FB.x, FB.y);
  } else {
    if (oA) a.F[bA] = FA;
    if (oB) a.F[bB] = FB;
  }
  if (a.csum) {
    if (g.O) {
      if (oA) a.sense[bA] = 0.5f * (interp1(a.csum, a.nx, a.ny, xa.x, xa.y, oa.x, oa.y) + interp1(a.csum, a.nx, a.ny, xa.x, xa.y, -oa.x, -oa.y));
      if (oB) a.sense[bB] = 0.5f * (interp1(a.csum, a.nx, a.ny, xb.x, xb.y, ob.x, ob.y) + interp1(a.csum, a.nx, a.ny, xb.x, xb.y, -ob.x, -ob.y));
    } else {
      if (oA) a.sense[bA] = interp1(a.csum, a.nx, a.ny, xa.x, xa.y);
      if (oB) a.sense[bB] = interp1(a.csum, a.nx, a.ny, xb.x, xb.y);
    }
  }
}

// Raise *slot (bits of a non-negative float) to the block's maximum of m: ONE guarded atomic per
// CTA.  These kernels are short and all their warps would hit the same address (k_markers spent 53 of
// its 57 us on 7,572 serialised reds); the guard reads past L1 so that it sees other CTAs' updates.
__device__ __forceinline__ void block_max_to(float m, unsigned* __restrict__ slot) {
  __shared__ float wmax[32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x < 32) {
    m = (threadIdx.x < (blockDim.x >> 5)) ? wmax[threadIdx.x] : 0.0f;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    if (threadIdx.x == 0) {
      const unsigned mb = __float_as_uint(m);
      if (mb > __ldcg(slot)) atomicMax(slot, mb);
    }
  }
}

// Two-layer broadcast (reading 28): offset h n_i of every bead, n_i = normalised mean of the unit
// normals (-t_y, t_x) of the adjacent edges (one edge at a chain end; the first edge's normal if
// the two cancel).  Runs after every change of X (load, mc_set_positions, K4, projection).
// step_max_m: bits of the largest component change of an offset, for the drift bound of the tile
// lists (a marker moves by the bead's displacement plus the change of its offset).
__global__ void __launch_bounds__(1024) k_markers(int N, const float2* __restrict__ X,
                                                  const unsigned char* __restrict__ bflags, float h,
                                                  float2* __restrict__ O, unsigned* __restrict__ step_max_m, size_t wstride) {
  X = wshift(X, blockIdx.y * wstride);
  bflags = wshift(bflags, blockIdx.y * wstride);
  O = wshift(O, blockIdx.y * wstride);
  step_max_m = wshift(step_max_m, blockIdx.y * wstride);
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  float m = 0.0f;
  if (b < N) {
    // every load up front and unconditional (clamped neighbours): one round trip to memory.  The flags
    // come from the one-byte array of the load (the float4 parameter pack would cost 16 B/bead for 2 bits)
    const int fl = bflags[b];
    const float2 p = X[b], qp = X[max(b - 1, 0)], qn = X[min(b + 1, N - 1)], old = O[b];
    // The differences of nearby fp32 positions are exact.  fp32 normals carry ~1e-7 each; where the
    // joint is bent beyond ~150 degrees the two normals nearly cancel and the direction of their sum
    // loses |n1 + n2|^-1 digits (parity world "hairpin" failed at 8e-6): those beads -- rare -- take the
    // same sum in fp64.  (All in fp64 cost 0.5 ms per step on world 4d: fp64 sqrt and divide.)
    const bool hasp = !(fl & BEAD_FIRST), hasn = !(fl & BEAD_LAST);
    float2 vp = make_float2(1.f, 0.f), vn = make_float2(1.f, 0.f);
    if (hasp) vp = make_float2(p.x - qp.x, p.y - qp.y);   // edge (b-1, b)
    if (hasn) vn = make_float2(qn.x - p.x, qn.y - p.y);   // edge (b, b+1)
    const float ip = rsqrtf(vp.x * vp.x + vp.y * vp.y), in_ = rsqrtf(vn.x * vn.x + vn.y * vn.y);
    const float2 np_ = make_float2(-vp.y * ip, vp.x * ip), nn_ = make_float2(-vn.y * in_, vn.x * in_);
    float sx = (hasp ? np_.x : 0.f) + (hasn ? nn_.x : 0.f), sy = (hasp ? np_.y : 0.f) + (hasn ? nn_.y : 0.f);
    const float s2 = sx * sx + sy * sy;
    float2 o;
    if (s2 > 0.25f) {
      const float sc = h * rsqrtf(s2);
      o = make_float2(sc * sx, sc * sy);
    } else {
      double nx_ = 0.0, ny_ = 0.0, fx = 0.0, fy = 0.0;
      if (hasp) {
        const double inv = 1.0 / sqrt((double)vp.x * vp.x + (double)vp.y * vp.y);
        fx = -(double)vp.y * inv; fy = (double)vp.x * inv;
        nx_ = fx; ny_ = fy;
      }
      if (hasn) {
        const double inv = 1.0 / sqrt((double)vn.x * vn.x + (double)vn.y * vn.y);
        const double ex = -(double)vn.y * inv, ey = (double)vn.x * inv;
        if (!hasp) { fx = ex; fy = ey; }
        nx_ += ex; ny_ += ey;
      }
      double nn = sqrt(nx_ * nx_ + ny_ * ny_);
      if (!(nn > 1e-9)) { nx_ = fx; ny_ = fy; nn = 1.0; }
      const double sc = (double)h / nn;
      o = make_float2((float)(sc * nx_), (float)(sc * ny_));
    }
    O[b] = o;
    m = fmaxf(fabsf(o.x - old.x), fabsf(o.y - old.y));
  }
  block_max_to(m, step_max_m);
}

// Projection (reading 27): X += Dp after the PBD pass on the advected positions; also the
// non-finite guard and the largest projection displacement for the lists' drift bound.
__global__ void __launch_bounds__(1024) k_add_displacement(int N, float2* __restrict__ X, const float2* __restrict__ Dp,
                                                          int* __restrict__ flag, unsigned* __restrict__ step_max_p,
                                                          size_t wstride) {
  X = wshift(X, blockIdx.y * wstride);
  Dp = wshift(Dp, blockIdx.y * wstride);
  flag = wshift(flag, blockIdx.y * wstride);
  step_max_p = wshift(step_max_p, blockIdx.y * wstride);
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  float m = 0.0f;
  if (b < N) {
    float2 p = X[b];
    const float2 d = Dp[b];
    p.x += d.x;
    p.y += d.y;
    X[b] = p;
    if (!(isfinite(p.x) && isfinite(p.y))) atomicOr(flag, 8);
    m = fmaxf(fabsf(d.x), fabsf(d.y));
  }
  block_max_to(m, step_max_p);
}

}  // namespace mc

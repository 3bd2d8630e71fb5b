// k_filament.cuh -- K1: S0 actuation + S1 elastic PBD displacement (Eq. 1-4) + S4 field forces.
//
// Paper: bending pass Eq. 1, position pass Eq. 2-4.
// Readings: 1 the net PBD displacement D_i becomes the bead force kappa*D_i;
// 2 edge angles come from the current geometry; 3 one Jacobi iteration; 4 joint angle =
// atan2(cross, dot) in (-pi, pi]; 5 free ends; 18 theta*_i(n) = theta0_i + a_i sin(2 pi n dt/T_i + phi_i).
//
// Mapping (north_star (1): one warp per chain, neighbours by warp shuffles, float4 SoA loads).
// The beads of all chains form one flat chain-ordered array with a first/last flag per bead.
// A warp owns a window of 64 consecutive beads, two per lane (positions arrive as one float4
// per lane, parameters as three float4 per bead); D_i needs X_{i-2..i+2}, of which all but two
// shuffles per quantity stay inside the lane.  When every chain has the same length m and m
// divides 64 the windows are aligned to chain starts (one 64-bead chain, two 32-bead chains or
// four 16-bead chains per warp) and all 64 beads are outputs; otherwise windows advance by 60
// and overlap by 4, the two beads at either end being halo.
//
// Precision.  State and parameters are fp32 and so is almost all arithmetic.  But D_i is a
// difference of differences (|D| ~ 1e-4 out of edge vectors ~1 and joint angles ~0.3 rad);
// plain fp32 leaves ~1e-5 relative error on the force, which is the parity bar (measured,
// DESIGN.md "Precision").  Three cancelling quantities are therefore formed in fp64 from the
// exact fp32 inputs and rounded once: the edge vector v = X_{i+1} - X_i, |v|^2 - L^2, and
// the joint's (cross, dot).  The joint angle itself never needs an fp64 atan2: (dot, cross) is
// rotated by the rest angle first -- by the fp32 pair (cos, sin)(theta0) stored at load time,
// whose own angle differs from theta0 by a stored residual eps -- so that the fp32 atan2f acts
// on the SMALL angle psi - theta0, where its absolute error is ~1e-9.
#pragma once
#include "mc_common.cuh"

namespace mc {

// layout twin of ListState (k_tile.cuh), which this header cannot include
struct ListStateWords {
  int need;
  float drift;
  unsigned step_max, step_max_p, step_max_m;
};

constexpr int BEAD_FIRST = 1, BEAD_LAST = 2, BEAD_PAD = 4;
constexpr int BEAD_ODD = 8;  // odd index within its chain (edge parity of the Gauss-Seidel pass, k_pbd.cuh)

struct FilamentArgs {
  const float2* X;   // [N]
  const float4* PA;  // {L_rest, act_amp, act_phase, k_bend}
  const float4* PB;  // {k_shear, k_stretch, r_hi, r_lo}       r = dt / act_period (hi + lo)
  const float4* PC;  // {cos theta0, sin theta0, eps, flags}   eps = theta0 - atan2(sin, cos)
  const float2* PD;  // {act_amp, act_phase}: with PC all the UNIFORM variant reads per bead
  const float4* uni; // [2] {L_rest, k_bend, k_shear, k_stretch}, {r_hi, r_lo, -, -} of bead 0 (UNIFORM variant)
  float2* F;         // [N] out: total bead force
  float* sense;      // [N] out (only written when csum != NULL)
  const float2* A;   // interleaved force-gradient field (may be NULL: no field forces)
  cudaTextureObject_t tex_A;  // linear float2 view of A, or 0 (gathers then use the LSU pipe only)
  const float* csum;  // sum of static fields (may be NULL)
  unsigned* tile_fmax;  // per 32x32 tile: bits of max |F| over the beads whose floor(X) lies in it (may be NULL)
  int N;
  int nx, ny;
  int stride;        // 64 (aligned windows) or 60 (overlapping windows)
  int n_windows;
  float kappa;       // k_el * dt^2
  const long long* step;  // DEVICE: step index n (before the increment); K4 increments it
  // batched worlds: move every workspace pointer to world `blockIdx.y` (mc_common.cuh wshift)
  __device__ __forceinline__ void shift(size_t bytes) {
    X = wshift(X, bytes); PA = wshift(PA, bytes); PB = wshift(PB, bytes); PC = wshift(PC, bytes);
    PD = wshift(PD, bytes); uni = wshift(uni, bytes); F = wshift(F, bytes); sense = wshift(sense, bytes);
    A = wshift(A, bytes); csum = wshift(csum, bytes); tile_fmax = wshift(tile_fmax, bytes);
    step = wshift(step, bytes);
  }
};

struct BeadParams {
  float L, amp, phase, kb, ks, kst, rhi, rlo, c0, s0, eps;
  int flags;
};

// UNIFORM: rest length, stiffnesses and actuation period are the same for every bead of the
// loaded configuration (checked by k_pack_params; the paper's populations are built that way):
// they come from one broadcast load and the per-bead traffic drops from 48 to 24 bytes.
template <bool UNIFORM>
__device__ __forceinline__ BeadParams load_params(const FilamentArgs& a, int b, bool valid) {
  BeadParams p;
  if (valid) {
    const float4 pc = __ldcs(a.PC + b);  // parameters are read once per step: streaming loads
    p.c0 = pc.x; p.s0 = pc.y; p.eps = pc.z; p.flags = __float_as_int(pc.w);
    if (UNIFORM) {
      const float2 pd = __ldcs(a.PD + b);
      const float4 u0 = __ldg(a.uni), u1 = __ldg(a.uni + 1);
      p.L = u0.x; p.kb = u0.y; p.ks = u0.z; p.kst = u0.w; p.rhi = u1.x; p.rlo = u1.y;
      p.amp = pd.x; p.phase = pd.y;
    } else {
      const float4 pa = __ldcs(a.PA + b), pb = __ldcs(a.PB + b);
      p.L = pa.x; p.amp = pa.y; p.phase = pa.z; p.kb = pa.w;
      p.ks = pb.x; p.kst = pb.y; p.rhi = pb.z; p.rlo = pb.w;
    }
  } else {
    p.L = 1.f; p.amp = p.phase = p.kb = p.ks = p.kst = p.rhi = p.rlo = p.s0 = p.eps = 0.f;
    p.c0 = 1.f;
    p.flags = BEAD_FIRST | BEAD_LAST | BEAD_PAD;
  }
  return p;
}

// atan2(y, x) for x > 0 and |y| <= x/2 (joint angles within 0.46 rad of their rest value: the
// common case): t = y/x, odd polynomial in t fitted on Chebyshev nodes of t^2 in [0, 1/4]
// (degree 11 in t; absolute error < 3e-8: that of atan2f, at a third of its instructions).
__device__ __forceinline__ float atan_small(float y, float x) {
  const float t = __fdividef(y, x), u = t * t;
  float p = fmaf(u, -0.05077829957008362f, 0.10122803598642349f);
  p = fmaf(u, p, -0.14165857434272766f);
  p = fmaf(u, p, 0.19993248581886292f);
  p = fmaf(u, p, -0.3333319127559662f);
  return fmaf(t * u, p, t);
}

// sin(s) for |s| <= pi (the reduced actuation phase): reflect onto [-pi/2, pi/2], odd polynomial
// of degree 9 fitted on Chebyshev nodes of s^2 (absolute error < 1e-7).
__device__ __forceinline__ float sin_pi(float s) {
  if (fabsf(s) > 1.57079632679f) s = (copysignf(3.140625f, s) - s) + copysignf(9.67653589793e-4f, s);
  const float u = s * s;
  float p = fmaf(u, 2.6051661734527443e-06f, -0.00019809046352747828f);
  p = fmaf(u, p, 0.008333050645887852f);
  p = fmaf(u, p, -0.16666658222675323f);
  return fmaf(s * u, p, s);
}

// (1/2) k_bend C_bend of the joint between edge pv (incoming) and edge v (outgoing); Eq. 1.
__device__ __forceinline__ float half_kC(double pvx, double pvy, double vx, double vy, const BeadParams& p,
                                         double n_step) {
  const double TWO_PI = 6.283185307179586476925286766559;
  const double cross = pvx * vy - pvy * vx, dot = pvx * vx + pvy * vy;
  // rotate by -theta0' (theta0' = angle of the stored fp32 pair): small-angle atan2f
  const double c = (double)p.c0, s = (double)p.s0;
  const double dotp = dot * c + cross * s, crossp = cross * c - dot * s;
  const float yf = (float)crossp, xf = (float)dotp;
  // = psi - theta0' (mod 2 pi)
  float psi_p = (xf > 0.0f && fabsf(yf) <= 0.5f * xf) ? atan_small(yf, xf) : atan2f(yf, xf);
  if (!(dot > 0.0 && dotp > 0.0)) {
    // rare: joint bent beyond +-pi/2.  Restore the oracle's branch, psi in (-pi, pi].
    const float t = psi_p + atan2f(p.s0, p.c0);
    if (t > 3.14159265358979f) psi_p -= 6.28318530717959f;
    else if (t <= -3.14159265358979f) psi_p += 6.28318530717959f;
  }
  // actuation phase 2 pi n dt/T + phi, reduced in fp64 (n dt/T reaches thousands of turns)
  double turns = n_step * (double)p.rhi + n_step * (double)p.rlo;
  turns -= rint(turns);
  double ph = TWO_PI * turns + (double)p.phase;
  ph -= TWO_PI * rint(ph * (1.0 / TWO_PI));
  const float C = psi_p - p.eps - p.amp * sin_pi((float)ph);
  return 0.5f * p.kb * C;
}

// sin(x) for the small director rotations of Eq. 1 (|delta| is a fraction of the joint error):
// odd Taylor polynomial to x^9 for |x| <= 0.5 (relative error < 2e-10 there), sinf beyond.
__device__ __forceinline__ float sin_small(float x) {
  if (fabsf(x) > 0.5f) return sinf(x);
  const float x2 = x * x;
  const float p = fmaf(x2, fmaf(x2, fmaf(x2, 2.7557319e-6f, -1.9841270e-4f), 8.3333333e-3f), -1.6666667e-1f);
  return fmaf(x * x2, p, x);
}

// Delta x of an edge (Eq. 2-3) after the bending pass turned its director by delta.
__device__ __forceinline__ float2 edge_delta(double vx, double vy, float delta, const BeadParams& p) {
  const double l2 = vx * vx + vy * vy;
  const float L = p.L;
  const float ell = sqrtf((float)l2);
  const float dl = (float)(l2 - (double)L * (double)L) / (ell + L);  // |v| - L_rest, no cancellation
  const float inv = 1.0f / ell;
  const float tx = (float)vx * inv, ty = (float)vy * inv;
  const float sd = sin_small(delta), sh = sin_small(0.5f * delta);
  const float omc = 2.0f * sh * sh;  // 1 - cos(delta)
  // t - d with d = Rot(delta) t: Kirchhoff-Love error minus the stretch part, divided by L
  const float ex = omc * tx + sd * ty, ey = omc * ty - sd * tx;
  const float ksL = p.ks * L;
  return make_float2(0.5f * p.kst * fmaf(ksL, ex, dl * tx), 0.5f * p.kst * fmaf(ksL, ey, dl * ty));
}

template <bool UNIFORM, int TEXROWS>
__global__ void __launch_bounds__(256, 5) k_filament_force(FilamentArgs a, size_t wstride) {
  if (!TEXROWS && wstride) a.shift(blockIdx.y * wstride);  // the texture variants serve single worlds only (views are per world)
  const int lane = threadIdx.x & 31;
  const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (w >= a.n_windows) return;
  const unsigned FULL = 0xffffffffu;
  const bool aligned = (a.stride == 64);
  const int base = w * a.stride - (aligned ? 0 : 2);  // even => float4-aligned pairs
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
  // neighbours across the lane boundary
  const float nxa = __shfl_down_sync(FULL, xa.x, 1), nya = __shfl_down_sync(FULL, xa.y, 1);
  const float pxb = __shfl_up_sync(FULL, xb.x, 1), pyb = __shfl_up_sync(FULL, xb.y, 1);
  // edge vectors (fp64 differences of fp32 positions are exact)
  const double eAx = (double)xb.x - (double)xa.x, eAy = (double)xb.y - (double)xa.y;  // A -> B
  const double eBx = (double)nxa - (double)xb.x, eBy = (double)nya - (double)xb.y;    // B -> next A
  const double ePx = (double)xa.x - (double)pxb, ePy = (double)xa.y - (double)pyb;    // prev B -> A
  const bool edgeA = !(pA.flags & BEAD_LAST) && vB;
  const bool edgeB = !(pB.flags & BEAD_LAST) && lane < 31;
  const bool jointA = !(pA.flags & (BEAD_FIRST | BEAD_LAST)) && lane >= 1;
  const bool jointB = !(pB.flags & (BEAD_FIRST | BEAD_LAST)) && lane < 31;
  const double n_step = (double)*a.step;
  const float hA = jointA ? half_kC(ePx, ePy, eAx, eAy, pA, n_step) : 0.0f;
  const float hB = jointB ? half_kC(eAx, eAy, eBx, eBy, pB, n_step) : 0.0f;
  // Eq. 1 on an edge: theta_1 of its far joint (+), theta_2 of its near joint (-)
  const float hA_next = __shfl_down_sync(FULL, hA, 1);
  float2 dA = make_float2(0.f, 0.f), dB = make_float2(0.f, 0.f);
  if (edgeA) dA = edge_delta(eAx, eAy, hB - hA, pA);
  if (edgeB) dB = edge_delta(eBx, eBy, hA_next - hB, pB);
  // Eq. 4 summed per bead: D_i = Delta_i - Delta_{i-1}
  float pdx = __shfl_up_sync(FULL, dB.x, 1), pdy = __shfl_up_sync(FULL, dB.y, 1);
  if ((pA.flags & BEAD_FIRST) || lane == 0) { pdx = 0.f; pdy = 0.f; }
  float DAx = dA.x - pdx, DAy = dA.y - pdy;
  float DBx = dB.x, DBy = dB.y;
  if (!(pB.flags & BEAD_FIRST)) { DBx -= dA.x; DBy -= dA.y; }
  // halo lanes of an overlapping window stay in the warp (the reductions below are warp-wide)
  // but own no output
  const bool out = aligned || (lane >= 1 && lane <= 30);
  const bool oA = out && vA, oB = out && vB;
  float2 FA = make_float2(a.kappa * DAx, a.kappa * DAy), FB = make_float2(a.kappa * DBx, a.kappa * DBy);
  if (a.A) {
    if (oA) {
      const float2 g = TEXROWS ? interp2_tex<TEXROWS, true>(a.A, a.tex_A, a.nx, a.ny, xa.x, xa.y)
                               : interp2_pair<0>(a.A, a.nx, a.ny, xa.x, xa.y);
      FA.x += g.x; FA.y += g.y;
    }
    if (oB) {
      const float2 g = TEXROWS ? interp2_tex<TEXROWS, true>(a.A, a.tex_A, a.nx, a.ny, xb.x, xb.y)
                               : interp2_pair<0>(a.A, a.nx, a.ny, xb.x, xb.y);
      FB.x += g.x; FB.y += g.y;
    }
  }
  if (a.tile_fmax) {
    // Bound for the fixed-point scale of S5 (k_p2g.cuh): tile_fmax[t] >= max |F| over the beads
    // whose floor(X) lies in tile t.  The warp's own maximum is used for every tile its beads
    // touch (a valid, slightly looser bound) so that one lane per distinct tile issues at most
    // one atomicMax, and none once the stored value is high enough.  Positive floats order like
    // their bit patterns.
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
    if (oA) a.sense[bA] = interp1(a.csum, a.nx, a.ny, xa.x, xa.y);
    if (oB) a.sense[bB] = interp1(a.csum, a.nx, a.ny, xb.x, xb.y);
  }
}

// mc_load_filaments: gather the caller's arrays into the internal (spatially sorted) chain
// order, pack the per-bead parameters and validate them (flag != 0 => invalid input).
struct PackArgs {
  int N;
  const int* src;  // internal bead -> caller's bead
  const unsigned char* flags;
  const float *xy, *L_rest, *theta_rest, *k_bend, *k_shear, *k_stretch, *act_amp, *act_phase, *act_period;
  float2* X;
  float4 *PA, *PB, *PC;
  float2* PD;
  float4* uni;     // [2] bead 0's uniform-candidate parameters (FilamentArgs::uni)
  double dt;
  int* bad;
  int* nonuniform; // set when some bead's L_rest, stiffnesses or period differ from bead 0's
};

__global__ void k_pack_params(PackArgs a) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= a.N) return;
  const int s = a.src[b];
  a.X[b] = make_float2(a.xy[2 * s], a.xy[2 * s + 1]);
  const float kb = a.k_bend[s], ks = a.k_shear[s], kst = a.k_stretch[s], T = a.act_period[s];
  const double th = (double)a.theta_rest[s];
  const float c0 = (float)cos(th), s0 = (float)sin(th);
  const float eps = (float)(th - atan2((double)s0, (double)c0));
  const double r = a.dt / (double)T;
  const float rhi = (float)r, rlo = (float)(r - (double)rhi);
  a.PA[b] = make_float4(a.L_rest[s], a.act_amp[s], a.act_phase[s], kb);
  a.PB[b] = make_float4(ks, kst, rhi, rlo);
  a.PC[b] = make_float4(c0, s0, eps, __int_as_float((int)a.flags[b]));
  a.PD[b] = make_float2(a.act_amp[s], a.act_phase[s]);
  if (s == 0) {
    a.uni[0] = make_float4(a.L_rest[0], kb, ks, kst);
    a.uni[1] = make_float4(rhi, rlo, 0.f, 0.f);
  } else if (a.L_rest[s] != a.L_rest[0] || kb != a.k_bend[0] || ks != a.k_shear[0] || kst != a.k_stretch[0] ||
             T != a.act_period[0]) {
    *a.nonuniform = 1;  // every writer stores the same value
  }
  if (!(kb >= 0.f && kb <= 1.f && ks >= 0.f && ks <= 1.f && kst >= 0.f && kst <= 1.f)) atomicOr(a.bad, 1);
  if (!(T > 0.f)) atomicOr(a.bad, 2);
}

// first-bead tile key of every chain (for the spatial sort of the chains at load time)
__global__ void k_chain_keys(int n_fil, const int* __restrict__ offsets, const float* __restrict__ xy, int nx,
                             int ny, int key_tile, int* __restrict__ keys) {
  const int f = blockIdx.x * blockDim.x + threadIdx.x;
  if (f >= n_fil) return;
  const int b = offsets[f];
  const int ci = wrapi((int)floorf(xy[2 * b]), nx), cj = wrapi((int)floorf(xy[2 * b + 1]), ny);
  keys[f] = (cj / key_tile) * ((nx + key_tile - 1) / key_tile) + ci / key_tile;
}

// mc_read_state: internal order -> caller's order.  Batched (blockIdx.y = world): the workspace
// arrays lie wstride bytes apart, the caller's array holds the worlds back to back (N entries each).
__global__ void k_unpermute2(int N, const int* __restrict__ src, const float2* __restrict__ in, float2* __restrict__ out,
                             size_t wstride = 0) {
  src = wshift(src, blockIdx.y * wstride);
  in = wshift(in, blockIdx.y * wstride);
  out += (size_t)blockIdx.y * N;
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b < N) out[src[b]] = in[b];
}
// mc_set_positions: caller's order -> internal order
__global__ void k_permute2(int N, const int* __restrict__ src, const float2* __restrict__ in, float2* __restrict__ out,
                           size_t wstride = 0) {
  src = wshift(src, blockIdx.y * wstride);
  out = wshift(out, blockIdx.y * wstride);
  in += (size_t)blockIdx.y * N;
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b < N) out[b] = in[src[b]];
}
// all worlds of a batch: the next step rebuilds the tile lists (drift = +inf)
__global__ void k_force_rebuild(ListStateWords* st, size_t wstride) {
  st = wshift(st, blockIdx.x * wstride);
  if (threadIdx.x == 0) { st->need = 1; st->drift = __int_as_float(0x7f800000); st->step_max = st->step_max_p = st->step_max_m = 0u; }
}
__global__ void k_permute1(int N, const int* __restrict__ src, const float* __restrict__ in, float* __restrict__ out,
                           int* __restrict__ nonzero) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b < N) {
    const float v = in[src[b]];
    out[b] = v;
    if (v != 0.0f) *nonzero = 1;  // every writer stores the same value
  }
}
__global__ void k_unpermute1(int N, const int* __restrict__ src, const float* __restrict__ in, float* __restrict__ out) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b < N) out[src[b]] = in[b];
}

}  // namespace mc

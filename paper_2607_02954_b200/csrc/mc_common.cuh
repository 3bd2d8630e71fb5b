// mc_common.cuh -- device helpers shared by the kernels of libmc.so (CUDA path only).
// P:L<n> = PAPER.md line n; "reading k" = DESIGN.md "Readings" row k.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

namespace mc {

// wrap when i is known to lie in [-n, 2n)
// Packed fp32 pairs (sm_100 FFMA2: one issue slot for two lanes of arithmetic;
// the step's kernels are bound by issue slots).  A float2 in an aligned register pair is the
// operand; the compiler turns a duplicated scalar into the instruction's broadcast form.
typedef unsigned long long f32x2_t;
__device__ __forceinline__ f32x2_t pack2(float2 a) {
  f32x2_t r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a.x), "f"(a.y));
  return r;
}
__device__ __forceinline__ float2 unpack2(f32x2_t a) {
  float2 d;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(d.x), "=f"(d.y) : "l"(a));
  return d;
}
__device__ __forceinline__ float2 dup2(float s) { return make_float2(s, s); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) {
  f32x2_t r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(pack2(a)), "l"(pack2(b)), "l"(pack2(c)));
  return unpack2(r);
}
// d = a * s + c on both halves
__device__ __forceinline__ float2 ffma2(float2 a, float s, float2 c) { return fma2(a, dup2(s), c); }

// Batched worlds (mc_batch): the worlds of a batch have identical workspace
// layouts, `wstride` bytes apart, and every kernel of the step is launched ONCE for all of them
// with the world index in blockIdx.y (blockIdx.z for kernels on a 2-D grid).  A kernel shifts its
// workspace pointers by world * wstride on entry; a single world is a batch of one (shift 0).
template <class T>
__device__ __forceinline__ T* wshift(T* p, size_t bytes) {
  return p ? reinterpret_cast<T*>(reinterpret_cast<char*>(const_cast<typename std::remove_const<T>::type*>(p)) + bytes) : p;
}

__device__ __forceinline__ int wrap1(int i, int n) {
  return i < 0 ? i + n : (i >= n ? i - n : i);
}
// periodic wrap of a grid index (reading 9).  Beads are almost always within one period of the
// domain, so the integer division (~35 instructions) is kept off the common path.
__device__ __forceinline__ int wrapi(int i, int n) {
  if ((unsigned)(i + n) < (unsigned)(3 * n)) return wrap1(i, n);
  i %= n;
  return i < 0 ? i + n : i;
}

// Peskin's 4-point function (Peskin 2002, cited P:L125; reading 7) at the four nodes
// fl-1, fl, fl+1, fl+2 of a bead with fractional coordinate fr = x - floor(x) in [0,1).
// Node distances are 1+fr, fr, 1-fr, 2-fr.  The two inner weights are evaluated from
// phi(r) = (3 - 2|r| + sqrt(1 + 4|r| - 4r^2))/8; the outer two follow from the kernel's
// even/odd sum rule (w0 + w2 = w1 + w3 = 1/2), which is exact for phi and avoids the
// cancellation in the outer branch's radicand.
// sqrt.approx (one MUFU, relative error ~1e-7, radicand in [1,2]) instead of the IEEE-rounded
// sqrtf (MUFU.RSQ + Newton + a slow-path call, ~10 instructions): four of them per bead in each
// of the four bead-grid kernels.
__device__ __forceinline__ float sqrt_fast(float v) {
  float r;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(v));
  return r;
}

__device__ __forceinline__ void peskin4(float fr, float& w0, float& w1, float& w2, float& w3) {
  const float a1 = fr, a2 = 1.0f - fr;
  w1 = 0.125f * (3.0f - 2.0f * a1 + sqrt_fast(fmaf(4.0f * a1, a2, 1.0f)));  // 1+4a-4a^2 = 1+4a(1-a)
  w2 = 0.125f * (3.0f - 2.0f * a2 + sqrt_fast(fmaf(4.0f * a2, a1, 1.0f)));
  w0 = 0.5f - w2;
  w3 = 0.5f - w1;
}

// Support of a coordinate: first node (unwrapped) and fractional part (reading 8).
__device__ __forceinline__ void support(float x, int& i0, float& fr) {
  const float fl = floorf(x);
  fr = x - fl;  // exact in fp32
  i0 = (int)fl - 1;
}

// Support of a coordinate given as a bead position x plus a small offset o (two-layer markers,
// reading 28: M = X +- h n).  The marker is never rounded to fp32 on its own -- at |X| ~ 6000 that
// would cost 2.4e-4 nodes, far above the parity bar: the fractional part is formed from the exact
// fractional part of x plus o (|o| <= 1), so its error stays ~6e-8 whatever |X|.
__device__ __forceinline__ void support_off(float x, float o, int& i0, float& fr) {
  const float fl = floorf(x);
  const float s = (x - fl) + o;   // in (-1, 2)
  const float fs = floorf(s);
  fr = s - fs;
  i0 = (int)fl + (int)fs - 1;
}

// The two gathered fields (velocity u, force-gradient field A) are stored BLOCKED: 4x4 nodes of
// float2 = one 128-byte line.  Consecutive beads of a chain are ~1 node apart in an arbitrary
// direction; in a row-major field every lane of a gather instruction then sits on its own line
// (vertical chains), while 4x4 blocks are shared by ~4 consecutive beads whatever the direction.
__device__ __forceinline__ size_t blk_index(int i, int j, int nx) {
  return ((size_t)(j >> 2) * (nx >> 2) + (i >> 2)) * 16 + ((j & 3) << 2) + (i & 3);
}

// Interpolate an interleaved two-component field at (x,y): sum over the 4x4 support of
// field(g) * delta_h(g - X)  ("nodes sample the local fluid velocity"; also S4's
// gradient sampling).  One 8-byte load per support node.
__device__ __forceinline__ float2 interp2(const float2* __restrict__ p, int nx, int ny, float x, float y) {
  int i0, j0;
  float fx, fy, wx[4], wy[4];
  support(x, i0, fx);
  support(y, j0, fy);
  peskin4(fx, wx[0], wx[1], wx[2], wx[3]);
  peskin4(fy, wy[0], wy[1], wy[2], wy[3]);
  i0 = wrapi(i0, nx);
  j0 = wrapi(j0, ny);
  int col[4];  // column part of the blocked index
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const int c = (i0 + k >= nx) ? i0 + k - nx : i0 + k;
    col[k] = ((c >> 2) << 4) + (c & 3);
  }
  const int nbx = nx >> 2;
  float ax = 0.0f, ay = 0.0f;
#pragma unroll
  for (int l = 0; l < 4; ++l) {
    const int row = (j0 + l >= ny) ? j0 + l - ny : j0 + l;
    // row pointer once, then one IMAD.WIDE (32-bit column offset x 8 + pointer) per node
    const char* r = reinterpret_cast<const char*>(p + ((size_t)(row >> 2) * nbx * 16 + ((row & 3) << 2)));
    float sx = 0.0f, sy = 0.0f;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const float2 v = __ldg(reinterpret_cast<const float2*>(r + (unsigned long long)(unsigned)col[k] * 8u));
      sx = fmaf(v.x, wx[k], sx);
      sy = fmaf(v.y, wx[k], sy);
    }
    ax = fmaf(sx, wy[l], ax);
    ay = fmaf(sy, wy[l], ay);
  }
  return make_float2(ax, ay);
}

// Same sum with the support rows 2 and 3 fetched through the texture pipe (raw fetches of the
// same memory, no filtering: identical bits).  The per-bead gathers are bound by the LSU pipe's
// tag stage (one 128-byte line per clock); the TEX pipe has its own.
// PACK: accumulate both components in one packed pair (FFMA2): same bits, half the FMA issue
// slots, but K4 then drops to 32 registers and a higher occupancy that costs it 1 % (measured),
// so only K1 uses it.
template <int TEXROWS, bool PACK>
__device__ __forceinline__ float2 interp2_tex(const float2* __restrict__ p, cudaTextureObject_t tex, int nx, int ny,
                                              float x, float y) {
  int i0, j0;
  float fx, fy, wx[4], wy[4];
  support(x, i0, fx);
  support(y, j0, fy);
  peskin4(fx, wx[0], wx[1], wx[2], wx[3]);
  peskin4(fy, wy[0], wy[1], wy[2], wy[3]);
  i0 = wrapi(i0, nx);
  j0 = wrapi(j0, ny);
  int col[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const int c = (i0 + k >= nx) ? i0 + k - nx : i0 + k;
    col[k] = ((c >> 2) << 4) + (c & 3);
  }
  const int nbx = nx >> 2;
  float2 acc = make_float2(0.0f, 0.0f);
#pragma unroll
  for (int l = 0; l < 4; ++l) {
    const int row = (j0 + l >= ny) ? j0 + l - ny : j0 + l;
    const int ro = (row >> 2) * nbx * 16 + ((row & 3) << 2);
    float2 s2 = make_float2(0.0f, 0.0f);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const float2 v = (l >= 4 - TEXROWS)
                           ? tex1Dfetch<float2>(tex, ro + col[k])
                           : __ldg(reinterpret_cast<const float2*>(reinterpret_cast<const char*>(p + ro) +
                                                                   (unsigned long long)(unsigned)col[k] * 8u));
      s2 = PACK ? ffma2(v, wx[k], s2) : make_float2(fmaf(v.x, wx[k], s2.x), fmaf(v.y, wx[k], s2.y));
    }
    acc = PACK ? ffma2(s2, wy[l], acc) : make_float2(fmaf(s2.x, wy[l], acc.x), fmaf(s2.y, wy[l], acc.y));
  }
  return acc;
}

// The same sum with 16-BYTE loads of aligned node pairs.  The gathers are bound by the LSU pipe's
// wavefronts (one per distinct 128-byte line an instruction touches, ~8 per 32-lane gather): fewer,
// wider instructions mean fewer wavefronts for the same lines.  In the blocked layout the nodes
// (c, c+1), c even, of a row are 16 bytes apart from nothing else: a support starting at an EVEN
// column is two such pairs, at an ODD column it is the second node of one pair, a whole pair and
// the first node of a third -- the third load is predicated off for the even lanes.  Weights of the
// unused pair halves are zero.
template <int TEXROWS = 0>
__device__ __forceinline__ float2 interp2_pair(const float2* __restrict__ p, int nx, int ny, float x, float y,
                                               cudaTextureObject_t tex = 0) {
  int i0, j0;
  float fx, fy, wx[4], wy[4];
  support(x, i0, fx);
  support(y, j0, fy);
  peskin4(fx, wx[0], wx[1], wx[2], wx[3]);
  peskin4(fy, wy[0], wy[1], wy[2], wy[3]);
  i0 = wrapi(i0, nx);
  j0 = wrapi(j0, ny);
  const bool odd = (i0 & 1) != 0;
  const int e = i0 & ~1;  // first column of the first pair (nx is even: a pair never straddles the seam)
  int pc[3];
#pragma unroll
  for (int q = 0; q < 3; ++q) {
    const int c = (e + 2 * q >= nx) ? e + 2 * q - nx : e + 2 * q;
    pc[q] = ((c >> 2) << 4) + (c & 3);
  }
  // weights of the six columns e .. e+5
  const float w0 = odd ? 0.0f : wx[0], w1 = odd ? wx[0] : wx[1], w2 = odd ? wx[1] : wx[2], w3 = odd ? wx[2] : wx[3],
              w4 = odd ? wx[3] : 0.0f;
  const int nbx = nx >> 2;
  float ax = 0.0f, ay = 0.0f;
#pragma unroll
  for (int l = 0; l < 4; ++l) {
    const int row = (j0 + l >= ny) ? j0 + l - ny : j0 + l;
    if (l >= 4 - TEXROWS) {  // the last rows through the texture pipe (its own tag stage), node by node
      const int ro = (row >> 2) * nbx * 16 + ((row & 3) << 2);
      float sx = 0.0f, sy = 0.0f;
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const int c = (i0 + k >= nx) ? i0 + k - nx : i0 + k;
        const float2 v = tex1Dfetch<float2>(tex, ro + ((c >> 2) << 4) + (c & 3));
        sx = fmaf(v.x, wx[k], sx);
        sy = fmaf(v.y, wx[k], sy);
      }
      ax = fmaf(sx, wy[l], ax);
      ay = fmaf(sy, wy[l], ay);
      continue;
    }
    const char* r = reinterpret_cast<const char*>(p + ((size_t)(row >> 2) * nbx * 16 + ((row & 3) << 2)));
    const float4 v0 = __ldg(reinterpret_cast<const float4*>(r + (unsigned long long)(unsigned)pc[0] * 8u));
    const float4 v1 = __ldg(reinterpret_cast<const float4*>(r + (unsigned long long)(unsigned)pc[1] * 8u));
    float4 v2 = make_float4(0.f, 0.f, 0.f, 0.f);
    if (odd) v2 = __ldg(reinterpret_cast<const float4*>(r + (unsigned long long)(unsigned)pc[2] * 8u));
    float sx = v0.x * w0, sy = v0.y * w0;
    sx = fmaf(v0.z, w1, sx); sy = fmaf(v0.w, w1, sy);
    sx = fmaf(v1.x, w2, sx); sy = fmaf(v1.y, w2, sy);
    sx = fmaf(v1.z, w3, sx); sy = fmaf(v1.w, w3, sy);
    sx = fmaf(v2.x, w4, sx); sy = fmaf(v2.y, w4, sy);
    ax = fmaf(sx, wy[l], ax);
    ay = fmaf(sy, wy[l], ay);
  }
  return make_float2(ax, ay);
}

// interp2 at the marker (x + ox, y + oy) (two-layer broadcast): 16-byte pair loads like interp2_pair,
// the support formed by support_off.
__device__ __forceinline__ float2 interp2_off(const float2* __restrict__ p, int nx, int ny, float x, float y, float ox,
                                              float oy) {
  int i0, j0;
  float fx, fy, wx[4], wy[4];
  support_off(x, ox, i0, fx);
  support_off(y, oy, j0, fy);
  peskin4(fx, wx[0], wx[1], wx[2], wx[3]);
  peskin4(fy, wy[0], wy[1], wy[2], wy[3]);
  i0 = wrapi(i0, nx);
  j0 = wrapi(j0, ny);
  const bool odd = (i0 & 1) != 0;
  const int e = i0 & ~1;
  int pc[3];
#pragma unroll
  for (int q = 0; q < 3; ++q) {
    const int c = (e + 2 * q >= nx) ? e + 2 * q - nx : e + 2 * q;
    pc[q] = ((c >> 2) << 4) + (c & 3);
  }
  const float w0 = odd ? 0.0f : wx[0], w1 = odd ? wx[0] : wx[1], w2 = odd ? wx[1] : wx[2], w3 = odd ? wx[2] : wx[3],
              w4 = odd ? wx[3] : 0.0f;
  const int nbx = nx >> 2;
  float ax = 0.0f, ay = 0.0f;
#pragma unroll
  for (int l = 0; l < 4; ++l) {
    const int row = (j0 + l >= ny) ? j0 + l - ny : j0 + l;
    const char* r = reinterpret_cast<const char*>(p + ((size_t)(row >> 2) * nbx * 16 + ((row & 3) << 2)));
    const float4 v0 = __ldg(reinterpret_cast<const float4*>(r + (unsigned long long)(unsigned)pc[0] * 8u));
    const float4 v1 = __ldg(reinterpret_cast<const float4*>(r + (unsigned long long)(unsigned)pc[1] * 8u));
    float4 v2 = make_float4(0.f, 0.f, 0.f, 0.f);
    if (odd) v2 = __ldg(reinterpret_cast<const float4*>(r + (unsigned long long)(unsigned)pc[2] * 8u));
    float sx = v0.x * w0, sy = v0.y * w0;
    sx = fmaf(v0.z, w1, sx); sy = fmaf(v0.w, w1, sy);
    sx = fmaf(v1.x, w2, sx); sy = fmaf(v1.y, w2, sy);
    sx = fmaf(v1.z, w3, sx); sy = fmaf(v1.w, w3, sy);
    sx = fmaf(v2.x, w4, sx); sy = fmaf(v2.y, w4, sy);
    ax = fmaf(sx, wy[l], ax);
    ay = fmaf(sy, wy[l], ay);
  }
  return make_float2(ax, ay);
}

// row-major scalar plane at (x + ox, y + oy); ox = oy = 0 gives the plain bead position
__device__ __forceinline__ float interp1(const float* __restrict__ p0, int nx, int ny, float x, float y,
                                         float ox = 0.0f, float oy = 0.0f) {
  int i0, j0;
  float fx, fy, wx[4], wy[4];
  support_off(x, ox, i0, fx);
  support_off(y, oy, j0, fy);
  peskin4(fx, wx[0], wx[1], wx[2], wx[3]);
  peskin4(fy, wy[0], wy[1], wy[2], wy[3]);
  i0 = wrapi(i0, nx);
  j0 = wrapi(j0, ny);
  float a = 0.0f;
#pragma unroll
  for (int l = 0; l < 4; ++l) {
    const int row = (j0 + l >= ny) ? j0 + l - ny : j0 + l;
    const float* r0 = p0 + (size_t)row * nx;
    float s = 0.0f;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int c = (i0 + k >= nx) ? i0 + k - nx : i0 + k;
      s = fmaf(__ldg(r0 + c), wx[k], s);
    }
    a = fmaf(s, wy[l], a);
  }
  return a;
}

}  // namespace mc

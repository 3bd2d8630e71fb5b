// mco.cpp -- CPU ORACLE (test infrastructure; see mco.h).  Plain loops, fp64.
// Shares nothing with the CUDA path.  P:L<n> = /root/reference/PAPER.md line n.
#include "mco.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

const double PI = 3.14159265358979323846264338327950288;

// D2Q9 (Qian et al. 1992): velocities, weights, opposites.
const int CX[9] = {0, 1, 0, -1, 0, 1, -1, -1, 1};
const int CY[9] = {0, 0, 1, 0, -1, 1, 1, -1, -1};
const double WQ[9] = {4.0 / 9, 1.0 / 9, 1.0 / 9, 1.0 / 9, 1.0 / 9,
                      1.0 / 36, 1.0 / 36, 1.0 / 36, 1.0 / 36};
const int OPP[9] = {0, 3, 4, 1, 2, 7, 8, 5, 6};

// Thread count of the independent loops (same arithmetic whatever it is).  It belongs to a WORLD
// (mco_world::threads, mco_set_threads); mco_step installs it for the duration of the call on the
// calling thread.  The stateless component functions called on their own run serially.
thread_local int tl_threads = 0;  // 0/1 = serial; >1 = OpenMP over independent loops
struct ThreadScope {
  int saved;
  explicit ThreadScope(int k) : saved(tl_threads) { tl_threads = k; }
  ~ThreadScope() { tl_threads = saved; }
};
#define MCO_PAR _Pragma("omp parallel for schedule(static) num_threads(tl_threads > 1 ? tl_threads : 1)")

inline int wrap(long long i, int n) {
  long long r = i % n;
  if (r < 0) r += n;
  return (int)r;
}

}  // namespace

extern "C" {

// Peskin (2002) 4-point regularised delta, cited by the paper for IBM;
// choice of this kernel among IBM kernels: DESIGN.md reading 7.
double mco_phi(double r) {
  double a = std::fabs(r);
  if (a <= 1.0) return 0.125 * (3.0 - 2.0 * a + std::sqrt(1.0 + 4.0 * a - 4.0 * a * a));
  if (a <= 2.0) return 0.125 * (5.0 - 2.0 * a - std::sqrt(-7.0 + 12.0 * a - 4.0 * a * a));
  return 0.0;
}

// Support of a bead at coordinate x: nodes i0..i0+3, i0 = floor(x)-1 (reading 8).
void mco_support(double x, int32_t* i0, double w[4]) {
  double fl = std::floor(x);
  *i0 = (int32_t)fl - 1;
  for (int k = 0; k < 4; ++k) w[k] = mco_phi((fl - 1.0 + k) - x);
}

// Eq. 1-4, one Jacobi iteration (reading 3), theta from geometry
// (reading 2), free ends (reading 5), sinusoidal actuation of theta_rest (reading 18).
int mco_elastic(int32_t n_fil, const int32_t* offsets, const double* xy,
                const float* L_rest, const float* theta_rest, const float* k_bend,
                const float* k_shear, const float* k_stretch, const float* act_amp,
                const float* act_phase, const float* act_period, double dt, int64_t n,
                double* D) {
  int bad = 0;
  MCO_PAR
  for (int32_t f = 0; f < n_fil; ++f) {
    const int64_t b0 = offsets[f];
    const int m = offsets[f + 1] - offsets[f];
    std::vector<double> vx(m), vy(m), len(m), tx(m), ty(m), C(m, 0.0), dx(m), dy(m);
    // 1. edge vectors v_e = X_{e+1} - X_e
    for (int e = 0; e + 1 < m; ++e) {
      vx[e] = xy[2 * (b0 + e + 1)] - xy[2 * (b0 + e)];
      vy[e] = xy[2 * (b0 + e + 1) + 1] - xy[2 * (b0 + e) + 1];
      len[e] = std::sqrt(vx[e] * vx[e] + vy[e] * vy[e]);
      if (!(len[e] > 1e-12)) { bad = 1; len[e] = 1.0; }  // degenerate edge (reading 21)
      tx[e] = vx[e] / len[e];
      ty[e] = vy[e] / len[e];
    }
    // 2.-3. joints j = 1..m-2: C_bend = (theta_2 - theta_1) - theta_rest
    for (int j = 1; j + 1 < m; ++j) {
      double cross = vx[j - 1] * vy[j] - vy[j - 1] * vx[j];
      double dot = vx[j - 1] * vx[j] + vy[j - 1] * vy[j];
      double psi = std::atan2(cross, dot);
      double T = (double)act_period[b0 + j];
      double theta_star = (double)theta_rest[b0 + j] +
                          (double)act_amp[b0 + j] *
                              std::sin(2.0 * PI * ((double)n * dt) / T + (double)act_phase[b0 + j]);
      C[j] = psi - theta_star;
    }
    // 4.-7. per edge: Eq. 1 angle change, director, Eq. 2, Eq. 3
    for (int e = 0; e + 1 < m; ++e) {
      double delta = 0.0;
      if (e + 1 <= m - 2) delta += 0.5 * (double)k_bend[b0 + e + 1] * C[e + 1];  // theta_1 += k C /2
      if (e >= 1) delta -= 0.5 * (double)k_bend[b0 + e] * C[e];                  // theta_2 -= k C /2
      double cd = std::cos(delta), sd = std::sin(delta);
      double ddx = cd * tx[e] - sd * ty[e];  // director d(theta) after the bending pass
      double ddy = sd * tx[e] + cd * ty[e];
      double L = (double)L_rest[b0 + e];
      double csx = (len[e] - L) * tx[e];     // Eq. 2
      double csy = (len[e] - L) * ty[e];
      double ks = (double)k_shear[b0 + e], kst = (double)k_stretch[b0 + e];
      dx[e] = 0.5 * kst * (csx + ks * (vx[e] - L * ddx - csx));  // Eq. 3
      dy[e] = 0.5 * kst * (csy + ks * (vy[e] - L * ddy - csy));
    }
    // 8. Eq. 4 summed per bead: x1 += dx, x2 -= dx
    for (int i = 0; i < m; ++i) {
      double sx = 0.0, sy = 0.0;
      if (i <= m - 2) { sx += dx[i]; sy += dy[i]; }
      if (i >= 1) { sx -= dx[i - 1]; sy -= dy[i - 1]; }
      D[2 * (b0 + i)] = sx;
      D[2 * (b0 + i) + 1] = sy;
    }
  }
  return bad ? MCO_ESTATE : MCO_OK;
}

// Literal PBD (reading 27): "an iterative constraint projection
// method ... Each iteration decouples the solver into two phases.  First, a bending pass updates
// theta toward theta_rest.  Second, a position pass enforces nodal connectivity", with
// the rest angle AND the rest length as time-dependent targets ("The CPPN outputs the rest angle
// theta_rest and the rest length L_rest"; jellyfish "contractile movement via uniform
// distance and bending constraints").
//   iters K >= 1 iterations, each on the working positions Y^k = X + Dtot^k (Y^0 = X):
//     bending pass: psi_j from Y^k, C_j = psi_j - theta*_j(n), Eq. 1 on all joints at once ->
//                   delta_e, material director d_e = Rot(delta_e) t_e(Y^k);
//     position pass, order 0 (Jacobi): Eq. 2-3 on every edge from Y^k, Eq. 4 summed per bead;
//                    order 1 (red-black Gauss-Seidel): the EVEN edges of each chain (e = 0, 2, ..)
//                    first, Eq. 4 applied at once; then the ODD edges from the updated positions
//                    (the directors d_e of the bending pass are kept);
//   L*_e(n) = L_rest[e] + act_L_amp[e] sin(2 pi n dt / act_period[e] + act_phase[e])  (entry e of
//   the per-bead arrays serves joint e and edge (e, e+1)); act_L_amp may be NULL (no actuation).
//   Out: D [N][2] = Dtot^K = Y^K - X, the net displacement of the K iterations.
// K = 1, order 0, no length actuation reproduces mco_elastic bit for bit (pinned).
int mco_pbd(int32_t n_fil, const int32_t* offsets, const double* xy, const float* L_rest,
            const float* theta_rest, const float* k_bend, const float* k_shear,
            const float* k_stretch, const float* act_amp, const float* act_phase,
            const float* act_period, const float* act_L_amp, double dt, int64_t n, int32_t iters,
            int32_t order, double* D) {
  if (iters < 1 || (order != 0 && order != 1)) return MCO_EINVAL;
  int bad = 0;
  MCO_PAR
  for (int32_t f = 0; f < n_fil; ++f) {
    const int64_t b0 = offsets[f];
    const int m = offsets[f + 1] - offsets[f];
    std::vector<double> yx(m), yy(m), tx(m), ty(m), C(m, 0.0), ddx(m), ddy(m), Ls(m), ths(m, 0.0);
    std::vector<double> Dx(m, 0.0), Dy(m, 0.0);
    // S0: targets of step n (the same for all K iterations)
    for (int i = 0; i < m; ++i) {
      const double s = std::sin(2.0 * PI * ((double)n * dt) / (double)act_period[b0 + i] + (double)act_phase[b0 + i]);
      ths[i] = (double)theta_rest[b0 + i] + (double)act_amp[b0 + i] * s;
      Ls[i] = (double)L_rest[b0 + i] + (act_L_amp ? (double)act_L_amp[b0 + i] * s : 0.0);
    }
    // Eq. 2-3 on edge e from the CURRENT working positions and the director (ddx, ddy) of the bending pass
    auto edge_delta = [&](int e, double& ox, double& oy) {
      const double vx = yx[e + 1] - yx[e], vy = yy[e + 1] - yy[e];
      double len = std::sqrt(vx * vx + vy * vy);
      if (!(len > 1e-12)) { bad = 1; len = 1.0; }
      const double ux = vx / len, uy = vy / len;
      const double L = Ls[e];
      const double csx = (len - L) * ux, csy = (len - L) * uy;   // Eq. 2
      const double ks = (double)k_shear[b0 + e], kst = (double)k_stretch[b0 + e];
      ox = 0.5 * kst * (csx + ks * (vx - L * ddx[e] - csx));      // Eq. 3
      oy = 0.5 * kst * (csy + ks * (vy - L * ddy[e] - csy));
    };
    for (int k = 0; k < iters; ++k) {
      for (int i = 0; i < m; ++i) {
        yx[i] = xy[2 * (b0 + i)] + Dx[i];
        yy[i] = xy[2 * (b0 + i) + 1] + Dy[i];
      }
      // bending pass (Eq. 1) from Y^k
      std::vector<double> vx(m), vy(m);
      for (int e = 0; e + 1 < m; ++e) {
        vx[e] = yx[e + 1] - yx[e];
        vy[e] = yy[e + 1] - yy[e];
        double len = std::sqrt(vx[e] * vx[e] + vy[e] * vy[e]);
        if (!(len > 1e-12)) { bad = 1; len = 1.0; }
        tx[e] = vx[e] / len;
        ty[e] = vy[e] / len;
      }
      for (int j = 1; j + 1 < m; ++j) {
        const double cross = vx[j - 1] * vy[j] - vy[j - 1] * vx[j];
        const double dot = vx[j - 1] * vx[j] + vy[j - 1] * vy[j];
        C[j] = std::atan2(cross, dot) - ths[j];
      }
      for (int e = 0; e + 1 < m; ++e) {
        double delta = 0.0;
        if (e + 1 <= m - 2) delta += 0.5 * (double)k_bend[b0 + e + 1] * C[e + 1];
        if (e >= 1) delta -= 0.5 * (double)k_bend[b0 + e] * C[e];
        const double cd = std::cos(delta), sd = std::sin(delta);
        ddx[e] = cd * tx[e] - sd * ty[e];
        ddy[e] = sd * tx[e] + cd * ty[e];
      }
      if (order == 0) {
        // Jacobi position pass: all edges from Y^k, Eq. 4 summed per bead
        std::vector<double> ex(m, 0.0), ey(m, 0.0);
        for (int e = 0; e + 1 < m; ++e) edge_delta(e, ex[e], ey[e]);
        for (int i = 0; i < m; ++i) {
          double sx = 0.0, sy = 0.0;
          if (i <= m - 2) { sx += ex[i]; sy += ey[i]; }
          if (i >= 1) { sx -= ex[i - 1]; sy -= ey[i - 1]; }
          Dx[i] += sx;
          Dy[i] += sy;
        }
      } else {
        // red-black Gauss-Seidel position pass: even edges, then odd edges on the updated positions
        for (int colour = 0; colour < 2; ++colour)
          for (int e = colour; e + 1 < m; e += 2) {
            double ex, ey;
            edge_delta(e, ex, ey);
            Dx[e] += ex;     Dy[e] += ey;          // x1 += dx   (Eq. 4)
            Dx[e + 1] -= ex; Dy[e + 1] -= ey;      // x2 -= dx
            yx[e] = xy[2 * (b0 + e)] + Dx[e];             yy[e] = xy[2 * (b0 + e) + 1] + Dy[e];
            yx[e + 1] = xy[2 * (b0 + e + 1)] + Dx[e + 1]; yy[e + 1] = xy[2 * (b0 + e + 1) + 1] + Dy[e + 1];
          }
      }
    }
    for (int i = 0; i < m; ++i) {
      D[2 * (b0 + i)] = Dx[i];
      D[2 * (b0 + i) + 1] = Dy[i];
    }
  }
  return bad ? MCO_ESTATE : MCO_OK;
}

// Two-layer broadcast (reading 28): "broadcasting the single filament
// into a two-layer version of itself to artificially amplify a zero-thickness filament into a
// solid object".  Every bead i is represented on the grid by two markers
//   M_i^+- = X_i +- h n_i,   n_i = unit normal of the chain at bead i
// = the normalised mean of the unit normals (-t_y, t_x) of the adjacent edges (one edge at a chain
// end); if the two edge normals cancel (a hairpin) the first edge's normal is used.
// Out: markers [2N][2], marker 2i = M_i^+, 2i+1 = M_i^-.  Every exchange with the grid then uses
// delta2_h(g; i) = 1/2 [delta_h(g - M_i^+) + delta_h(g - M_i^-)] in place of delta_h(g - X_i).
void mco_markers(int32_t n_fil, const int32_t* offsets, const double* xy, double h, double* markers) {
  MCO_PAR
  for (int32_t f = 0; f < n_fil; ++f) {
    const int64_t b0 = offsets[f];
    const int m = offsets[f + 1] - offsets[f];
    for (int i = 0; i < m; ++i) {
      double nx_ = 0.0, ny_ = 0.0, n1x = 0.0, n1y = 0.0;
      for (int e = i - 1; e <= i; ++e) {
        if (e < 0 || e + 1 >= m) continue;
        const double vx = xy[2 * (b0 + e + 1)] - xy[2 * (b0 + e)], vy = xy[2 * (b0 + e + 1) + 1] - xy[2 * (b0 + e) + 1];
        const double len = std::sqrt(vx * vx + vy * vy);
        const double ex = -vy / len, ey = vx / len;   // edge normal: tangent turned by +90 degrees
        if (nx_ == 0.0 && ny_ == 0.0 && n1x == 0.0 && n1y == 0.0) { n1x = ex; n1y = ey; }
        nx_ += ex;
        ny_ += ey;
      }
      double nn = std::sqrt(nx_ * nx_ + ny_ * ny_);
      if (!(nn > 1e-9)) { nx_ = n1x; ny_ = n1y; nn = 1.0; }
      nx_ /= nn;
      ny_ /= nn;
      const double px = xy[2 * (b0 + i)], py = xy[2 * (b0 + i) + 1];
      markers[4 * (b0 + i) + 0] = px + h * nx_;
      markers[4 * (b0 + i) + 1] = py + h * ny_;
      markers[4 * (b0 + i) + 2] = px - h * nx_;
      markers[4 * (b0 + i) + 3] = py - h * ny_;
    }
  }
}

// S2 deposit: rho_b(g) = sum_i delta_h(g - X_i), unit weight (reading 13).
void mco_deposit(int32_t nx, int32_t ny, int64_t N, const double* xy, double* rho_b) {
  for (long long c = 0; c < (long long)nx * ny; ++c) rho_b[c] = 0.0;
  for (int64_t b = 0; b < N; ++b) {
    int32_t i0, j0;
    double wx[4], wy[4];
    mco_support(xy[2 * b], &i0, wx);
    mco_support(xy[2 * b + 1], &j0, wy);
    for (int l = 0; l < 4; ++l)
      for (int k = 0; k < 4; ++k)
        rho_b[(size_t)wrap(j0 + l, ny) * nx + wrap(i0 + k, nx)] += wx[k] * wy[l];
  }
}

// S5 spread: G(g) = sum_i F_i delta_h(g - X_i) ("broadcasts ... onto the grid").
void mco_spread(int32_t nx, int32_t ny, int64_t N, const double* xy, const double* F,
                double* G) {
  const size_t nc = (size_t)nx * ny;
  for (size_t c = 0; c < 2 * nc; ++c) G[c] = 0.0;
  for (int64_t b = 0; b < N; ++b) {
    int32_t i0, j0;
    double wx[4], wy[4];
    mco_support(xy[2 * b], &i0, wx);
    mco_support(xy[2 * b + 1], &j0, wy);
    for (int l = 0; l < 4; ++l)
      for (int k = 0; k < 4; ++k) {
        size_t c = (size_t)wrap(j0 + l, ny) * nx + wrap(i0 + k, nx);
        double w = wx[k] * wy[l];
        G[c] += F[2 * b] * w;
        G[nc + c] += F[2 * b + 1] * w;
      }
  }
}

// S4/S7 interpolate: out_i = sum_g plane(g) delta_h(g - X_i) ("nodes sample").
void mco_interp(int32_t nx, int32_t ny, int32_t nch, const double* planes, int64_t N,
                const double* xy, double* out) {
  const size_t nc = (size_t)nx * ny;
  MCO_PAR
  for (int64_t b = 0; b < N; ++b) {
    int32_t i0, j0;
    double wx[4], wy[4];
    mco_support(xy[2 * b], &i0, wx);
    mco_support(xy[2 * b + 1], &j0, wy);
    for (int ch = 0; ch < nch; ++ch) {
      double s = 0.0;
      for (int l = 0; l < 4; ++l)
        for (int k = 0; k < 4; ++k)
          s += planes[ch * nc + (size_t)wrap(j0 + l, ny) * nx + wrap(i0 + k, nx)] * wx[k] * wy[l];
      out[b * nch + ch] = s;
    }
  }
}

int32_t mco_radius(double sigma, int32_t radius) {
  return radius > 0 ? radius : (int32_t)std::ceil(5.0 * sigma);
}

// S3 taps: sampled Gaussian truncated at R and normalised (reading 14).
void mco_gauss_taps(double sigma, int32_t R, double* taps) {
  double Z = 0.0;
  for (int k = -R; k <= R; ++k) {
    taps[k + R] = std::exp(-(double)(k * k) / (2.0 * sigma * sigma));
    Z += taps[k + R];
  }
  for (int k = 0; k <= 2 * R; ++k) taps[k] /= Z;
}

// S3 filter: periodic convolution along x, then along y ("Gaussian filter").
void mco_blur(int32_t nx, int32_t ny, const double* in, double sigma, int32_t R, double* out) {
  std::vector<double> g(2 * R + 1), tmp((size_t)nx * ny);
  mco_gauss_taps(sigma, R, g.data());
  MCO_PAR
  for (int j = 0; j < ny; ++j)
    for (int i = 0; i < nx; ++i) {
      double s = 0.0;
      for (int k = -R; k <= R; ++k) s += g[k + R] * in[(size_t)j * nx + wrap(i + k, nx)];
      tmp[(size_t)j * nx + i] = s;
    }
  MCO_PAR
  for (int j = 0; j < ny; ++j)
    for (int i = 0; i < nx; ++i) {
      double s = 0.0;
      for (int k = -R; k <= R; ++k) s += g[k + R] * tmp[(size_t)wrap(j + k, ny) * nx + i];
      out[(size_t)j * nx + i] = s;
    }
}

// S3 gradient: second-order central difference, periodic (reading 15).
void mco_grad(int32_t nx, int32_t ny, const double* in, double* gx, double* gy) {
  MCO_PAR
  for (int j = 0; j < ny; ++j)
    for (int i = 0; i < nx; ++i) {
      size_t c = (size_t)j * nx + i;
      gx[c] = 0.5 * (in[(size_t)j * nx + wrap(i + 1, nx)] - in[(size_t)j * nx + wrap(i - 1, nx)]);
      gy[c] = 0.5 * (in[(size_t)wrap(j + 1, ny) * nx + i] - in[(size_t)wrap(j - 1, ny) * nx + i]);
    }
}

// Persistent scalar field of Gaussian packets, periodic minimum image.
void mco_static_field(int32_t nx, int32_t ny, int32_t n_sources, const float* sources,
                      double* c) {
  MCO_PAR
  for (int j = 0; j < ny; ++j)
    for (int i = 0; i < nx; ++i) {
      double s = 0.0;
      for (int k = 0; k < n_sources; ++k) {
        double ddx = (double)i - (double)sources[4 * k];
        double ddy = (double)j - (double)sources[4 * k + 1];
        ddx -= nx * std::nearbyint(ddx / nx);
        ddy -= ny * std::nearbyint(ddy / ny);
        double wdt = (double)sources[4 * k + 3];
        s += (double)sources[4 * k + 2] * std::exp(-(ddx * ddx + ddy * ddy) / (2.0 * wdt * wdt));
      }
      c[(size_t)j * nx + i] = s;
    }
}

// nu_lat = nu*dt; tau+ = 3 nu_lat + 1/2; tau- = Lambda/(tau+ - 1/2) + 1/2 (reading 10;
// TRT: Ginzburg et al. 2008, cited P:L127; "viscosity ... controlled by tau" P:L119).
void mco_lattice_constants(double nu, double dt, double trt_lambda, double* omega_plus,
                           double* omega_minus) {
  double nu_lat = nu * dt;
  double tau_p = 3.0 * nu_lat + 0.5;
  double tau_m = trt_lambda / (tau_p - 0.5) + 0.5;
  *omega_plus = 1.0 / tau_p;
  *omega_minus = 1.0 / tau_m;
}

// S6: D2Q9 TRT collision with Guo forcing split by parity, then streaming (P:L117-119,
// L127; reading 10, 11).  f pre-collision in, pre-collision of the next step out.
void mco_lbm_step(int32_t nx, int32_t ny, double* f, const double* G, double omega_plus,
                  double omega_minus, double* u_out) {
  const size_t nc = (size_t)nx * ny;
  std::vector<double> fs(9 * nc);
  MCO_PAR
  for (int j = 0; j < ny; ++j)
    for (int i = 0; i < nx; ++i) {
      size_t c = (size_t)j * nx + i;
      double fq[9], rho = 0.0, mx = 0.0, my = 0.0;
      for (int q = 0; q < 9; ++q) {
        fq[q] = f[q * nc + c];
        rho += fq[q];
        mx += CX[q] * fq[q];
        my += CY[q] * fq[q];
      }
      double gx = G ? G[c] : 0.0, gy = G ? G[nc + c] : 0.0;
      double ux = (mx + 0.5 * gx) / rho, uy = (my + 0.5 * gy) / rho;  // Guo velocity
      if (u_out) { u_out[c] = ux; u_out[nc + c] = uy; }
      double feq[9];
      for (int q = 0; q < 9; ++q) {
        double cu = CX[q] * ux + CY[q] * uy;
        feq[q] = WQ[q] * rho * (1.0 + 3.0 * cu + 4.5 * cu * cu - 1.5 * (ux * ux + uy * uy));
      }
      for (int q = 0; q < 9; ++q) {
        int o = OPP[q];
        double fp = 0.5 * (fq[q] + fq[o]), fm = 0.5 * (fq[q] - fq[o]);
        double ep = 0.5 * (feq[q] + feq[o]), em = 0.5 * (feq[q] - feq[o]);
        double cu = CX[q] * ux + CY[q] * uy, cg = CX[q] * gx + CY[q] * gy;
        double Sp = WQ[q] * (-3.0 * (ux * gx + uy * gy) + 9.0 * cu * cg);
        double Sm = 3.0 * WQ[q] * cg;
        double post = fq[q] - omega_plus * (fp - ep) - omega_minus * (fm - em) +
                      (1.0 - 0.5 * omega_plus) * Sp + (1.0 - 0.5 * omega_minus) * Sm;
        // stream: f_q(x + c_q, n+1) = f*_q(x, n)
        fs[q * nc + (size_t)wrap(j + CY[q], ny) * nx + wrap(i + CX[q], nx)] = post;
      }
    }
  std::memcpy(f, fs.data(), 9 * nc * sizeof(double));
}

// Moments of the populations: rho = sum f_q, u* = sum c_q f_q / rho.  u* is the velocity the
// node would have without any force this step (Guo: u = u* + G/(2 rho), reading 11).
void mco_moments(int32_t nx, int32_t ny, const double* f, double* rho, double* ustar) {
  const size_t nc = (size_t)nx * ny;
  MCO_PAR
  for (long long c = 0; c < (long long)nc; ++c) {
    double r = 0.0, mx = 0.0, my = 0.0;
    for (int q = 0; q < 9; ++q) {
      r += f[q * nc + c];
      mx += CX[q] * f[q * nc + c];
      my += CY[q] * f[q * nc + c];
    }
    rho[c] = r;
    ustar[c] = mx / r;
    ustar[nc + c] = my / r;
  }
}

// Multi-Direct Forcing (Wang, Fan & Luo 2008, cited P:L127; "the filaments' nodes sample
// the local fluid velocity ... the agent broadcasts its own velocity back onto the grid").
// Reading 26: each iteration adds the bead force rho0 (V_i - U_i), spreads
// it and corrects the grid velocity with Guo's u = u* + G/(2 rho); the bead forces add up.  The
// factor rho0 (half of the 2 rho0 that would cancel an isolated bead's slip at once) keeps the
// iteration contracting where chains overlap: it needs interp(rho_b)(X_i) < 4 instead of < 2.
void mco_mdf(int32_t nx, int32_t ny, int64_t N, const double* xy, const double* V,
             const double* ustar, const double* rho, double rho0, int32_t iters, double* F,
             double* G, double* u_out, double* resid) {
  const size_t nc = (size_t)nx * ny;
  std::vector<double> u(ustar, ustar + 2 * nc), U(2 * (size_t)N), dF(2 * (size_t)N), dG(2 * nc);
  for (size_t c = 0; c < 2 * nc; ++c) G[c] = 0.0;
  for (int64_t i = 0; i < 2 * N; ++i) F[i] = 0.0;
  for (int k = 0; k <= iters; ++k) {
    mco_interp(nx, ny, 2, u.data(), N, xy, U.data());           // sample
    if (resid) {
      double r = 0.0;
      for (int64_t i = 0; i < 2 * N; ++i) r = std::fmax(r, std::fabs(V[i] - U[i]));
      resid[k] = r;
    }
    if (k == iters) break;
    for (int64_t i = 0; i < 2 * N; ++i) {
      dF[i] = rho0 * (V[i] - U[i]);                             // direct forcing
      F[i] += dF[i];
    }
    mco_spread(nx, ny, N, xy, dF.data(), dG.data());             // broadcast
    for (size_t c = 0; c < 2 * nc; ++c) G[c] += dG[c];
    for (size_t c = 0; c < nc; ++c) {
      u[c] = ustar[c] + G[c] / (2.0 * rho[c]);
      u[nc + c] = ustar[nc + c] + G[nc + c] / (2.0 * rho[c]);
    }
  }
  if (u_out) std::memcpy(u_out, u.data(), 2 * nc * sizeof(double));
}

// Multi-Direct Forcing through the two-layer broadcast (readings 26 + 28; P:L127 lists both among
// the practices used together).  P holds `layers` points per bead (layers = 2: the markers
// M_i^+, M_i^-; layers = 1: the bead itself, then this is mco_mdf).  Each iteration
//   U_i = mean over the bead's points of interp(u^k);  dF_i = rho0 (V_i - U_i);  F_i += dF_i;
//   every point spreads dF_i / layers;  u^{k+1} = ustar + G^{k+1} / (2 rho).
void mco_mdf_layers(int32_t nx, int32_t ny, int64_t N, int32_t layers, const double* P, const double* V,
                    const double* ustar, const double* rho, double rho0, int32_t iters, double* F,
                    double* G, double* u_out, double* resid) {
  const size_t nc = (size_t)nx * ny;
  const int64_t NP = N * layers;
  std::vector<double> u(ustar, ustar + 2 * nc), Up(2 * (size_t)NP), U(2 * (size_t)N), dF(2 * (size_t)N),
      dFp(2 * (size_t)NP), dG(2 * nc);
  for (size_t c = 0; c < 2 * nc; ++c) G[c] = 0.0;
  for (int64_t i = 0; i < 2 * N; ++i) F[i] = 0.0;
  for (int k = 0; k <= iters; ++k) {
    mco_interp(nx, ny, 2, u.data(), NP, P, Up.data());           // sample at every point
    for (int64_t i = 0; i < N; ++i)
      for (int c = 0; c < 2; ++c) {
        double s = 0.0;
        for (int l = 0; l < layers; ++l) s += Up[2 * (i * layers + l) + c];
        U[2 * i + c] = s / layers;                                 // mean over the bead's points
      }
    if (resid) {
      double r = 0.0;
      for (int64_t i = 0; i < 2 * N; ++i) r = std::fmax(r, std::fabs(V[i] - U[i]));
      resid[k] = r;
    }
    if (k == iters) break;
    for (int64_t i = 0; i < 2 * N; ++i) {
      dF[i] = rho0 * (V[i] - U[i]);                               // direct forcing
      F[i] += dF[i];
    }
    for (int64_t i = 0; i < N; ++i)
      for (int l = 0; l < layers; ++l)
        for (int c = 0; c < 2; ++c) dFp[2 * (i * layers + l) + c] = dF[2 * i + c] / layers;
    mco_spread(nx, ny, NP, P, dFp.data(), dG.data());             // broadcast through every point
    for (size_t c = 0; c < 2 * nc; ++c) G[c] += dG[c];
    for (size_t c = 0; c < nc; ++c) {
      u[c] = ustar[c] + G[c] / (2.0 * rho[c]);
      u[nc + c] = ustar[nc + c] + G[nc + c] / (2.0 * rho[c]);
    }
  }
  if (u_out) std::memcpy(u_out, u.data(), 2 * nc * sizeof(double));
}

}  // extern "C"

// ------------------------------------------------------------------------------------
// The world and the step: S0..S7 in the order BASELINE.json's north_star lists
// (force -> deposit/gradient -> spread -> fluid update -> interpolate -> integrate),
// built only from the component functions above.
// ------------------------------------------------------------------------------------
struct mco_world {
  mco_world_params p;
  std::vector<std::vector<float>> sources;  // own copy of each field's packets
  int nx = 0, ny = 0;
  size_t nc = 0;
  double dt = 0, omega_p = 0, omega_m = 0, kappa = 0, rho0 = 1;
  int64_t step = 0;
  int fp32_state = 0;
  int threads = 0;  // OpenMP threads of this world's steps (mco_set_threads)
  // filaments
  int32_t n_fil = 0;
  int64_t N = 0;
  std::vector<int32_t> offsets;
  std::vector<float> L_rest, theta_rest, k_bend, k_shear, k_stretch, act_amp, act_phase, act_period;
  std::vector<float> act_L_amp;  // empty: rest length not actuated
  std::vector<double> X;  // [N][2]
  // fluid
  std::vector<double> f;  // [9][ny][nx], un-shifted, pre-collision
  std::vector<double> u;  // [2][ny][nx]
  // fields
  std::vector<double> field;       // [n_fields][ny][nx]: last blurred density / static c
  std::vector<double> static_gx, static_gy;  // [n_fields][ny][nx] (static kinds only)
  // last step's intermediates
  std::vector<double> D, F, sense, rho_b, G;
  std::string err;
};

extern "C" {

const char* mco_last_error(const mco_world* w) { return w ? w->err.c_str() : "null world"; }

int mco_create(const mco_world_params* p, mco_world** out) {
  if (!p || !out) return MCO_EINVAL;
  *out = nullptr;
  if (p->nx <= 0 || p->ny <= 0 || !(p->dt > 0) || !(p->nu > 0) || !(p->trt_lambda > 0) ||
      !(p->rho0 > 0) || p->pbd_iters < 1 || p->pbd_iters > 8 || p->n_fields < 0 || p->n_fields > 4 ||
      p->max_beads < 0)
    return MCO_EINVAL;
  if ((p->pbd_order != 0 && p->pbd_order != 1) || (p->pbd_project != 0 && p->pbd_project != 1) ||
      (p->two_layer != 0 && p->two_layer != 1) || !(p->layer_offset >= 0) || p->layer_offset > 1)
    return MCO_EINVAL;

  if (p->coupling != MCO_COUPLING_FORCE && p->coupling != MCO_COUPLING_MDF) return MCO_EINVAL;
  if (p->coupling == MCO_COUPLING_MDF && (p->mdf_iters < 1 || p->mdf_iters > 16)) return MCO_EINVAL;
  for (int k = 0; k < p->n_fields; ++k) {
    const mco_field_params& fp = p->fields[k];
    if (fp.kind == MCO_FIELD_BEAD_DENSITY) {
      if (!(fp.sigma > 0)) return MCO_EINVAL;
    } else if (fp.kind == MCO_FIELD_STATIC_SOURCE) {
      if (fp.n_sources < 0 || (fp.n_sources > 0 && !fp.sources)) return MCO_EINVAL;
    } else {
      return MCO_EINVAL;
    }
  }
  mco_world* w = new (std::nothrow) mco_world();
  if (!w) return MCO_ENOMEM;
  w->p = *p;
  w->nx = p->nx;
  w->ny = p->ny;
  w->nc = (size_t)p->nx * p->ny;
  w->dt = (double)p->dt;
  w->rho0 = (double)p->rho0;
  mco_lattice_constants((double)p->nu, w->dt, (double)p->trt_lambda, &w->omega_p, &w->omega_m);
  w->kappa = (double)p->k_el * w->dt * w->dt;
  w->f.resize(9 * w->nc);
  for (int q = 0; q < 9; ++q)
    for (size_t c = 0; c < w->nc; ++c) w->f[q * w->nc + c] = WQ[q] * w->rho0;  // fluid at rest
  w->u.assign(2 * w->nc, 0.0);
  w->field.assign((size_t)p->n_fields * w->nc, 0.0);
  w->static_gx.assign((size_t)p->n_fields * w->nc, 0.0);
  w->static_gy.assign((size_t)p->n_fields * w->nc, 0.0);
  w->sources.resize(p->n_fields);
  for (int k = 0; k < p->n_fields; ++k) {
    const mco_field_params& fp = p->fields[k];
    if (fp.kind == MCO_FIELD_STATIC_SOURCE) {
      w->sources[k].assign(fp.sources, fp.sources + 4 * (size_t)fp.n_sources);
      w->p.fields[k].sources = w->sources[k].data();
      // computed once: c and its central-difference gradient (no blur)
      mco_static_field(w->nx, w->ny, fp.n_sources, w->sources[k].data(), &w->field[k * w->nc]);
      mco_grad(w->nx, w->ny, &w->field[k * w->nc], &w->static_gx[k * w->nc], &w->static_gy[k * w->nc]);
    } else {
      w->p.fields[k].sources = nullptr;
    }
  }
  w->rho_b.assign(w->nc, 0.0);
  w->G.assign(2 * w->nc, 0.0);
  *out = w;
  return MCO_OK;
}

void mco_destroy(mco_world* w) { delete w; }

int mco_load_filaments(mco_world* w, int32_t n_fil, const int32_t* offsets, const float* xy,
                       const float* L_rest, const float* theta_rest, const float* k_bend,
                       const float* k_shear, const float* k_stretch, const float* act_amp,
                       const float* act_phase, const float* act_period) {
  if (!w) return MCO_EINVAL;
  if (n_fil < 0 || !offsets || offsets[0] != 0) { w->err = "bad offsets"; return MCO_EINVAL; }
  int64_t N = offsets[n_fil];
  if (N > w->p.max_beads) { w->err = "N > max_beads"; return MCO_EINVAL; }
  for (int32_t f = 0; f < n_fil; ++f)
    if (offsets[f + 1] - offsets[f] < 3) { w->err = "chain shorter than 3 beads"; return MCO_EINVAL; }
  if (N > 0 && (!xy || !L_rest || !theta_rest || !k_bend || !k_shear || !k_stretch || !act_amp ||
                !act_phase || !act_period)) { w->err = "null array"; return MCO_EINVAL; }
  for (int64_t i = 0; i < N; ++i) {
    if (!(k_bend[i] >= 0 && k_bend[i] <= 1 && k_shear[i] >= 0 && k_shear[i] <= 1 &&
          k_stretch[i] >= 0 && k_stretch[i] <= 1)) { w->err = "stiffness outside [0,1]"; return MCO_EINVAL; }
    if (!(act_period[i] > 0)) { w->err = "period <= 0"; return MCO_EINVAL; }
  }
  w->n_fil = n_fil;
  w->N = N;
  w->offsets.assign(offsets, offsets + n_fil + 1);
  w->L_rest.assign(L_rest, L_rest + N);
  w->theta_rest.assign(theta_rest, theta_rest + N);
  w->k_bend.assign(k_bend, k_bend + N);
  w->k_shear.assign(k_shear, k_shear + N);
  w->k_stretch.assign(k_stretch, k_stretch + N);
  w->act_amp.assign(act_amp, act_amp + N);
  w->act_phase.assign(act_phase, act_phase + N);
  w->act_period.assign(act_period, act_period + N);
  w->act_L_amp.clear();
  w->X.resize(2 * N);
  for (int64_t i = 0; i < 2 * N; ++i) w->X[i] = (double)xy[i];
  w->D.assign(2 * N, 0.0);
  w->F.assign(2 * N, 0.0);
  w->sense.assign(N, 0.0);
  return MCO_OK;
}

int mco_set_length_actuation(mco_world* w, const float* act_L_amp) {
  if (!w) return MCO_EINVAL;
  if (act_L_amp) w->act_L_amp.assign(act_L_amp, act_L_amp + w->N);
  else w->act_L_amp.clear();
  return MCO_OK;
}

int mco_set_state(mco_world* w, int64_t step, const double* xy, const double* fdev) {
  if (!w || step < 0) return MCO_EINVAL;
  w->step = step;
  if (xy) std::memcpy(w->X.data(), xy, 2 * (size_t)w->N * sizeof(double));
  if (fdev)
    for (int q = 0; q < 9; ++q)
      for (size_t c = 0; c < w->nc; ++c) w->f[q * w->nc + c] = WQ[q] * w->rho0 + fdev[q * w->nc + c];
  return MCO_OK;
}

int mco_set_fp32_state(mco_world* w, int32_t on) {
  if (!w) return MCO_EINVAL;
  w->fp32_state = on ? 1 : 0;
  return MCO_OK;
}

int mco_set_threads(mco_world* w, int32_t k) {
  if (!w || k < 0) return MCO_EINVAL;
  w->threads = k;
  return MCO_OK;
}

static int mco_one_step(mco_world* w) {
  const int nx = w->nx, ny = w->ny;
  const size_t nc = w->nc;
  const int64_t N = w->N;
  const double dt2 = w->dt * w->dt;
  const float* Lamp = w->act_L_amp.empty() ? nullptr : w->act_L_amp.data();
  // S0+S1: actuation and the PBD displacement D of pbd_iters iterations (Eq. 1-4; reading 27;
  // one Jacobi iteration = reading 3); F_el = kappa * D (reading 1)
  int rc = mco_pbd(w->n_fil, w->offsets.data(), w->X.data(), w->L_rest.data(), w->theta_rest.data(),
                   w->k_bend.data(), w->k_shear.data(), w->k_stretch.data(), w->act_amp.data(),
                   w->act_phase.data(), w->act_period.data(), Lamp, w->dt, w->step, w->p.pbd_iters,
                   w->p.pbd_order, w->D.data());
  if (rc != MCO_OK) { w->err = "degenerate edge"; return rc; }
  // FORCE coupling: F = kappa D + field forces.  MDF coupling (reading 26): the same sum with
  // kappa = 1 is the bead's own velocity V_i = D_i + field displacement (lattice units, one
  // step, unit bead mass); it is held in F until the forcing iterations replace it.
  const bool mdf = w->p.coupling == MCO_COUPLING_MDF;
  const double kD = mdf ? 1.0 : w->kappa;
  for (int64_t i = 0; i < 2 * N; ++i) w->F[i] = kD * w->D[i];
  for (int64_t i = 0; i < N; ++i) w->sense[i] = 0.0;
  // The grid sees every bead through delta_h(g - X_i), or -- two-layer broadcast, reading 28 --
  // through 1/2 [delta_h(g - M_i^+) + delta_h(g - M_i^-)]: the same X (hence the same markers) in
  // S2, S4, S5 and S7.
  const bool two = w->p.two_layer != 0;
  const int64_t NM = two ? 2 * N : N;
  std::vector<double> markers;
  if (two) {
    markers.resize(4 * (size_t)N);
    const double h = w->p.layer_offset > 0 ? (double)w->p.layer_offset : 0.5;
    mco_markers(w->n_fil, w->offsets.data(), w->X.data(), h, markers.data());
  }
  const double* P = two ? markers.data() : w->X.data();  // the NM points that touch the grid
  // sample nch planes at the beads: plain interpolation, or the mean over a bead's two markers
  auto sample = [&](int nch, const double* planes, double* out) {
    if (!two) { mco_interp(nx, ny, nch, planes, N, P, out); return; }
    std::vector<double> tmp((size_t)NM * nch);
    mco_interp(nx, ny, nch, planes, NM, P, tmp.data());
    for (int64_t i = 0; i < N; ++i)
      for (int ch = 0; ch < nch; ++ch)
        out[i * nch + ch] = 0.5 * (tmp[(2 * i) * nch + ch] + tmp[(2 * i + 1) * nch + ch]);
  };
  // S2: deposit (one rho_b serves every bead-density field)
  mco_deposit(nx, ny, NM, P, w->rho_b.data());
  if (two) for (size_t c = 0; c < nc; ++c) w->rho_b[c] *= 0.5;
  std::vector<double> gx(nc), gy(nc), samp(2 * (size_t)N), s1((size_t)N);
  std::vector<double> planes(2 * nc);
  for (int k = 0; k < w->p.n_fields; ++k) {
    const mco_field_params& fp = w->p.fields[k];
    const double coup = (double)fp.coupling * dt2;  // kappa_rep or kappa_chi, lattice units
    if (fp.kind == MCO_FIELD_BEAD_DENSITY) {
      // S3: filter + gradient; S4: F_rep = -kappa_rep * interp(grad)
      int R = mco_radius((double)fp.sigma, fp.radius);
      mco_blur(nx, ny, w->rho_b.data(), (double)fp.sigma, R, &w->field[k * nc]);
      mco_grad(nx, ny, &w->field[k * nc], gx.data(), gy.data());
      std::memcpy(&planes[0], gx.data(), nc * sizeof(double));
      std::memcpy(&planes[nc], gy.data(), nc * sizeof(double));
      sample(2, planes.data(), samp.data());
      for (int64_t i = 0; i < 2 * N; ++i) w->F[i] -= coup * samp[i];
    } else {
      // S4: F_chem = +kappa_chi * interp(grad c); s_i = interp(c) (reading 17)
      std::memcpy(&planes[0], &w->static_gx[k * nc], nc * sizeof(double));
      std::memcpy(&planes[nc], &w->static_gy[k * nc], nc * sizeof(double));
      sample(2, planes.data(), samp.data());
      for (int64_t i = 0; i < 2 * N; ++i) w->F[i] += coup * samp[i];
      sample(1, &w->field[k * nc], s1.data());
      for (int64_t i = 0; i < N; ++i) w->sense[i] += s1[i];
    }
  }
  if (mdf) {
    // S5 (MDF): forcing iterations against the force-free velocity of the current populations
    std::vector<double> rho(nc), ustar(2 * nc), V(w->F);
    mco_moments(nx, ny, w->f.data(), rho.data(), ustar.data());
    if (two)  // the forcing iterations see the fluid through the markers as well (readings 26 + 28)
      mco_mdf_layers(nx, ny, N, 2, P, V.data(), ustar.data(), rho.data(), w->rho0, w->p.mdf_iters,
                     w->F.data(), w->G.data(), nullptr, nullptr);
    else
      mco_mdf(nx, ny, N, w->X.data(), V.data(), ustar.data(), rho.data(), w->rho0, w->p.mdf_iters,
              w->F.data(), w->G.data(), nullptr, nullptr);
  } else if (two) {
    // S5, two layers: each marker carries half of its bead's force
    std::vector<double> FM(2 * (size_t)NM);
    for (int64_t i = 0; i < N; ++i)
      for (int c = 0; c < 2; ++c) FM[4 * i + c] = FM[4 * i + 2 + c] = 0.5 * w->F[2 * i + c];
    mco_spread(nx, ny, NM, P, FM.data(), w->G.data());
  } else {
    // S5: spread the total bead force
    mco_spread(nx, ny, N, w->X.data(), w->F.data(), w->G.data());
  }
  // S6: fluid update; stores the collision-time velocity u
  mco_lbm_step(nx, ny, w->f.data(), w->G.data(), w->omega_p, w->omega_m, w->u.data());
  // S7: interpolate u at the same X and integrate (forward Euler, lattice units)
  sample(2, w->u.data(), samp.data());
  for (int64_t i = 0; i < 2 * N; ++i) w->X[i] += samp[i];
  if (w->p.pbd_project) {
    // optional projection (reading 27): the constraints of step n act once more, directly on the
    // advected positions ("directly modifies node positions")
    std::vector<double> Dp(2 * (size_t)N);
    rc = mco_pbd(w->n_fil, w->offsets.data(), w->X.data(), w->L_rest.data(), w->theta_rest.data(),
                 w->k_bend.data(), w->k_shear.data(), w->k_stretch.data(), w->act_amp.data(),
                 w->act_phase.data(), w->act_period.data(), Lamp, w->dt, w->step, w->p.pbd_iters,
                 w->p.pbd_order, Dp.data());
    if (rc != MCO_OK) { w->err = "degenerate edge"; return rc; }
    for (int64_t i = 0; i < 2 * N; ++i) w->X[i] += Dp[i];
  }
  w->step += 1;
  if (w->fp32_state) {
    for (int64_t i = 0; i < 2 * N; ++i) w->X[i] = (double)(float)w->X[i];
    for (int q = 0; q < 9; ++q)
      for (size_t c = 0; c < nc; ++c) {
        double dev = w->f[q * nc + c] - WQ[q] * w->rho0;
        w->f[q * nc + c] = WQ[q] * w->rho0 + (double)(float)dev;
      }
  }
  return MCO_OK;
}

int mco_step(mco_world* w, int32_t n) {
  if (!w || n < 0) return MCO_EINVAL;
  ThreadScope scope(w->threads);
  for (int32_t s = 0; s < n; ++s) {
    int rc = mco_one_step(w);
    if (rc != MCO_OK) return rc;
  }
  return MCO_OK;
}

int mco_read_state(mco_world* w, int64_t* step_out, double* xy, double* u, double* rho,
                   double* fdev, double* field, double* force, double* sense) {
  if (!w) return MCO_EINVAL;
  const size_t nc = w->nc;
  if (step_out) *step_out = w->step;
  if (xy) std::memcpy(xy, w->X.data(), 2 * (size_t)w->N * sizeof(double));
  if (u) std::memcpy(u, w->u.data(), 2 * nc * sizeof(double));
  if (rho)
    for (size_t c = 0; c < nc; ++c) {
      double s = 0.0;
      for (int q = 0; q < 9; ++q) s += w->f[q * nc + c];
      rho[c] = s;
    }
  if (fdev)
    for (int q = 0; q < 9; ++q)
      for (size_t c = 0; c < nc; ++c) fdev[q * nc + c] = w->f[q * nc + c] - WQ[q] * w->rho0;
  if (field) std::memcpy(field, w->field.data(), (size_t)w->p.n_fields * nc * sizeof(double));
  if (force) std::memcpy(force, w->F.data(), 2 * (size_t)w->N * sizeof(double));
  if (sense) std::memcpy(sense, w->sense.data(), (size_t)w->N * sizeof(double));
  return MCO_OK;
}

int mco_read_intermediates(mco_world* w, double* D, double* rho_b, double* G) {
  if (!w) return MCO_EINVAL;
  if (D) std::memcpy(D, w->D.data(), 2 * (size_t)w->N * sizeof(double));
  if (rho_b) std::memcpy(rho_b, w->rho_b.data(), w->nc * sizeof(double));
  if (G) std::memcpy(G, w->G.data(), 2 * w->nc * sizeof(double));
  return MCO_OK;
}

}  // extern "C"

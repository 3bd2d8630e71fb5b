/* mco.h -- CPU ORACLE for the Microcosmos per-timestep update (test infrastructure).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference leg may load it.  It shares no code,
 * header, table or constant with paper_2607_02954_b200/csrc (the CUDA path).
 *
 * What it is: a plain, slow, fp64 restatement of the step the paper describes
 * (/root/reference/PAPER.md, cited below as P:L<line>):
 *   - filament PBD constraints, Eq. 1-4
 *   - D2Q9 lattice Boltzmann fluid with TRT
 *   - steric field: deposit -> Gaussian -> gradient P:L119
 *   - persistent scalar (energy) field, sensed
 *   - immersed-boundary spread / interpolate
 *   - Multi-Direct Forcing coupling (optional)      P:L125-127 (reading 26)
 * Where the paper is silent the readings of SURVEY.md 8(c).2 / DESIGN.md are taken;
 * each function in mco.cpp names the passage or reading it follows.
 *
 * Conventions: grid node (i,j) sits at position (i,j), cell size 1, periodic domain
 * [0,nx) x [0,ny); grid arrays row-major, x fastest (index j*nx+i); multi-channel
 * arrays are planes ([q][j][i]).  Bead positions are unwrapped.  All pointers are HOST
 * pointers.  Inputs that mirror the product ABI are float; everything the oracle
 * returns is double.
 *
 * Pins (tests/test_oracle_*.py): every component function below is pinned to a closed
 * form, an invariant or a brute-force evaluation.  The whole coupled trajectory has
 * no printed reference values in the paper: absolute trajectory values are
 * "parity unpinned" beyond the component pins and the qualitative scallop check.
 */
#ifndef MCO_H
#define MCO_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct mco_world mco_world;

enum { MCO_OK = 0, MCO_EINVAL = -1, MCO_ENOMEM = -2, MCO_ESTATE = -4 };
enum { MCO_FIELD_BEAD_DENSITY = 0, MCO_FIELD_STATIC_SOURCE = 1 };
/* How the PBD output reaches the fluid ("broadcasts its own velocity back onto the grid"):
 * FORCE: the net displacement becomes a bead force kappa*D_i (reading 1);
 * MDF:   the bead's own velocity V_i is imposed on the fluid by iterated direct forcing
 *        (Multi-Direct Forcing, Wang et al. 2008, cited P:L127; reading 26). */
enum { MCO_COUPLING_FORCE = 0, MCO_COUPLING_MDF = 1 };

typedef struct {
  int32_t kind;        /* MCO_FIELD_*                                             */
  float sigma;         /* Gaussian filter width, cells (bead-density fields)       */
  int32_t radius;      /* truncation radius R; 0 => ceil(5*sigma)                  */
  float coupling;      /* k_rep or chi, physical units; lattice value = *dt^2      */
  int32_t n_sources;   /* static-source fields                                     */
  const float* sources;/* [n_sources][4] = cx, cy, amplitude, width                */
} mco_field_params;

typedef struct {
  int32_t nx, ny;      /* periodic grid                                            */
  float dt;            /* physical time per step                                   */
  float nu;            /* kinematic viscosity; nu_lat = nu*dt                      */
  float trt_lambda;    /* TRT magic parameter Lambda                               */
  float rho0;          /* rest density                                             */
  float k_el;          /* elastic coupling; kappa = k_el*dt^2                      */
  int32_t pbd_iters;   /* PBD iterations per step K, 1..8 (reading 27; 1 = reading 3) */
  int32_t n_fields;
  mco_field_params fields[4];
  int64_t max_beads;
  int32_t coupling;    /* MCO_COUPLING_*                                           */
  int32_t mdf_iters;   /* MDF: forcing iterations per step, 1..16 (ignored for FORCE) */
  int32_t pbd_order;   /* 0 Jacobi, 1 red-black Gauss-Seidel over even/odd edges (reading 27) */
  int32_t pbd_project; /* 1: after S7 the PBD displacement of the advected positions is added to
                          them directly ("directly modifies node positions"; reading 27) */
  int32_t two_layer;   /* 1: two-layer broadcast of every bead (reading 28)      */
  float layer_offset;  /* half distance h between the two layers, nodes (0 => 0.5)       */
} mco_world_params;

/* ---- world life cycle (twin of the product ABI, host pointers) ---- */
int mco_create(const mco_world_params* p, mco_world** out);
void mco_destroy(mco_world* w);
const char* mco_last_error(const mco_world* w);
int mco_load_filaments(mco_world* w, int32_t n_fil, const int32_t* offsets,
                       const float* xy, const float* L_rest, const float* theta_rest,
                       const float* k_bend, const float* k_shear, const float* k_stretch,
                       const float* act_amp, const float* act_phase, const float* act_period);
/* rest-length actuation amplitudes act_L_amp [N] (entry e: edge (e, e+1)); NULL switches it off.
 * Call after mco_load_filaments (which resets it to none). */
int mco_set_length_actuation(mco_world* w, const float* act_L_amp);
/* overwrite state: step counter, positions [N][2], populations as deviations
 * f_q - w_q*rho0, planes [9][ny][nx].  NULL pointer = keep. */
int mco_set_state(mco_world* w, int64_t step, const double* xy, const double* fdev);
/* fp32_state != 0: round X and (f - w*rho0) to float at the end of every step */
int mco_set_fp32_state(mco_world* w, int32_t on);
/* 0 = serial loops; k>0 = OpenMP threads for the independent loops (same arithmetic) */
int mco_set_threads(mco_world* w, int32_t k);
int mco_step(mco_world* w, int32_t n);
/* any output pointer may be NULL.
 * xy [N][2]; u [2][ny][nx] (velocity stored by the last step, lattice units);
 * rho [ny][nx] (sum_q f_q of the current populations); fdev [9][ny][nx];
 * field [n_fields][ny][nx] (last step's blurred density, or the static field c);
 * force [N][2] (last step's total bead force, lattice units); sense [N]. */
int mco_read_state(mco_world* w, int64_t* step_out, double* xy, double* u, double* rho,
                   double* fdev, double* field, double* force, double* sense);
/* last step's intermediate arrays, for parity on intermediates:
 * D [N][2] elastic displacement (Eq. 1-4), rho_b [ny][nx], G [2][ny][nx] */
int mco_read_intermediates(mco_world* w, double* D, double* rho_b, double* G);

/* ---- components (stateless), each pinned separately ---- */
double mco_phi(double r);                                /* Peskin 4-point function   */
void mco_support(double x, int32_t* i0, double w[4]);    /* i0=floor(x)-1, 4 weights  */
/* Eq. 1-4 on an array of chains; step index n selects the actuation phase.
 * D out [N][2]. */
int mco_elastic(int32_t n_fil, const int32_t* offsets, const double* xy,
                const float* L_rest, const float* theta_rest, const float* k_bend,
                const float* k_shear, const float* k_stretch, const float* act_amp,
                const float* act_phase, const float* act_period, double dt, int64_t n,
                double* D);
/* Literal PBD (reading 27): iters >= 1 iterations of {bending pass Eq. 1, position pass Eq. 2-4}
 * on working positions, order 0 = Jacobi, 1 = red-black Gauss-Seidel over the even / odd edges of
 * each chain; rest length actuated like the rest angle when act_L_amp != NULL:
 * L*_e(n) = L_rest[e] + act_L_amp[e] sin(2 pi n dt/act_period[e] + act_phase[e]).
 * D out [N][2] = net displacement of the iters iterations.  iters = 1, order = 0, act_L_amp = NULL
 * gives mco_elastic bit for bit. */
int mco_pbd(int32_t n_fil, const int32_t* offsets, const double* xy, const float* L_rest,
            const float* theta_rest, const float* k_bend, const float* k_shear,
            const float* k_stretch, const float* act_amp, const float* act_phase,
            const float* act_period, const float* act_L_amp, double dt, int64_t n, int32_t iters,
            int32_t order, double* D);
/* Two-layer broadcast (reading 28): markers [2N][2] = X_i + h n_i (entry 2i), X_i - h n_i (2i+1),
 * n_i the normalised mean of the adjacent edges' unit normals. */
void mco_markers(int32_t n_fil, const int32_t* offsets, const double* xy, double h, double* markers);
void mco_deposit(int32_t nx, int32_t ny, int64_t N, const double* xy, double* rho_b);
void mco_spread(int32_t nx, int32_t ny, int64_t N, const double* xy, const double* F,
                double* G /*[2][ny][nx]*/);
/* interpolate nch planes at the beads: out [N][nch] */
void mco_interp(int32_t nx, int32_t ny, int32_t nch, const double* planes, int64_t N,
                const double* xy, double* out);
int32_t mco_radius(double sigma, int32_t radius);
void mco_gauss_taps(double sigma, int32_t R, double* taps /*[2R+1]*/);
void mco_blur(int32_t nx, int32_t ny, const double* in, double sigma, int32_t R, double* out);
void mco_grad(int32_t nx, int32_t ny, const double* in, double* gx, double* gy);
void mco_static_field(int32_t nx, int32_t ny, int32_t n_sources, const float* sources,
                      double* c);
/* one TRT collide(+Guo source)+stream; f in/out [9][ny][nx] un-shifted; G [2][ny][nx]
 * may be NULL (zero); u_out [2][ny][nx] may be NULL */
void mco_lbm_step(int32_t nx, int32_t ny, double* f, const double* G, double omega_plus,
                  double omega_minus, double* u_out);
void mco_lattice_constants(double nu, double dt, double trt_lambda, double* omega_plus,
                           double* omega_minus);
/* zeroth and first moments of un-shifted populations f [9][ny][nx]:
 * rho [ny][nx] = sum_q f_q, ustar [2][ny][nx] = sum_q c_q f_q / rho (velocity without force) */
void mco_moments(int32_t nx, int32_t ny, const double* f, double* rho, double* ustar);
/* Multi-Direct Forcing (reading 26).  V [N][2] target bead velocities, ustar/rho from
 * mco_moments.  Iteration k = 0..iters-1, starting from u^0 = ustar, G^0 = 0:
 *   U_i = interp(u^k)(X_i);  dF_i = rho0 (V_i - U_i);  F_i += dF_i;
 *   G^{k+1} = G^k + spread(dF);  u^{k+1}(g) = ustar(g) + G^{k+1}(g) / (2 rho(g)).
 * Out: F [N][2] summed bead force, G [2][ny][nx] summed grid force, u_out [2][ny][nx] = u^iters
 * (may be NULL), resid [iters+1] (may be NULL): max_i |V_i - U_i| (max-norm over beads and
 * components) seen at the start of each iteration and after the last one. */
void mco_mdf(int32_t nx, int32_t ny, int64_t N, const double* xy, const double* V,
             const double* ustar, const double* rho, double rho0, int32_t iters, double* F,
             double* G, double* u_out, double* resid);

/* MDF through `layers` points per bead (layers = 2: the two-layer markers, readings 26 + 28;
 * layers = 1 is mco_mdf).  P [N*layers][2], point l of bead i at row i*layers + l.  Sampling = mean
 * over a bead's points, broadcast = dF / layers through each point.  Other arguments as mco_mdf. */
void mco_mdf_layers(int32_t nx, int32_t ny, int64_t N, int32_t layers, const double* P, const double* V,
                    const double* ustar, const double* rho, double rho0, int32_t iters, double* F,
                    double* G, double* u_out, double* resid);

#ifdef __cplusplus
}
#endif
#endif

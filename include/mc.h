/* mc.h -- C ABI of the B200-native Microcosmos per-timestep update (libmc.so).
 *
 * The library advances a 2-D periodic world that holds many elastic filament chains
 * two-way coupled to a D2Q9 lattice-Boltzmann fluid and to scalar fields, in the
 * discretisation of arxiv/paper_2607_02954 (cited as P:L<line> of PAPER.md; readings of
 * the paper's silences are numbered in DESIGN.md "Readings").  Every step of the path
 * runs in hand-written sm_100a CUDA kernels; there is no CPU fallback.
 *
 * One step (state at step n -> n+1), in this order (north_star of BASELINE.json):
 *   S0 actuation of the rest angle          P:L153, L171      (reading 18)
 *   S1 elastic PBD displacement, Eq. 1-4     P:L91-113         (readings 1-5)
 *   S2 deposit beads -> rho_b                P:L119            (reading 13)
 *   S3 Gaussian filter + gradient            P:L119            (readings 14, 15)
 *   S4 field forces at the beads             P:L119, L121, L175 (readings 16, 17)
 *   S5 spread bead forces -> G               P:L125            (reading 7)
 *   S6 D2Q9 TRT collide (Guo source) + stream P:L117-119, L127 (readings 10, 11)
 *   S7 interpolate u at the beads, X += U    P:L125            (readings 11, 12, 19)
 * With coupling = MC_COUPLING_MDF ("Multi-Direct Forcing", reading 26) S4 yields the
 * bead's own velocity V_i = D_i + field displacement instead of a force, and S5 becomes
 *   S5' u^0 = u* = sum_q c_q f_q / rho; mdf_iters times: U_i = interp(u^k)(X_i),
 *       F_i += rho0 (V_i - U_i), u^{k+1} = u^k + spread(rho0 (V - U)) / (2 rho);  G = spread(F)
 * followed by S6 and S7 unchanged.
 *
 * Conventions.  Grid node (i,j) sits at position (i,j); cell size 1; periodic domain
 * [0,nx) x [0,ny).  Grid arrays are row-major, x fastest (index j*nx+i); multi-channel
 * arrays are planes ([q][j][i]).  Bead arrays are chain-ordered (bead offsets[f]+i).
 * Bead positions are unwrapped; only grid indices wrap.  Everything is fp32 in memory.
 * D2Q9 numbering: c0=(0,0) c1=(1,0) c2=(0,1) c3=(-1,0) c4=(0,-1) c5=(1,1) c6=(-1,1)
 * c7=(-1,-1) c8=(1,-1); w0=4/9, w1..4=1/9, w5..8=1/36.
 *
 * Pointers: every pointer argument says HOST or DEVICE.  The caller owns all memory it
 * passes in; the library copies what it needs into the workspace and keeps no caller
 * pointer after the call returns.  No allocation of device memory happens inside the
 * library: all device state lives in the caller-provided workspace.
 *
 * Errors: every call returns 0 (MC_OK) or a negative code; the message is available from
 * mc_last_error.  Nothing throws or aborts across the ABI.
 *
 * Threading: one world = one stream; calls on one world are not re-entrant.
 * Determinism: same inputs => bit-identical outputs of mc_read_state, run to run.
 */
#ifndef MC_H
#define MC_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct mc_world mc_world; /* opaque host-side handle */

enum { MC_OK = 0, MC_EINVAL = -1, MC_ENOMEM = -2, MC_ECUDA = -3, MC_ESTATE = -4, MC_EDIVERGED = -5 };

enum {
  MC_FIELD_BEAD_DENSITY = 0, /* beads deposit; force = -k * grad(gauss * rho_b)  */
  MC_FIELD_STATIC_SOURCE = 1 /* Gaussian packets; force = +k * grad(c); c is sensed P:L121 */
};

enum {
  MC_COUPLING_FORCE = 0, /* bead force kappa*D_i spread to the fluid (reading 1); the default      */
  MC_COUPLING_MDF = 1    /* bead velocity imposed by iterated direct forcing (reading 26)          */
};

enum {
  MC_PBD_JACOBI = 0,      /* every constraint of an iteration from the same state (reading 3)        */
  MC_PBD_GAUSS_SEIDEL = 1 /* position pass over the even, then the odd edges of each chain (reading 27) */
};

typedef struct {
  int32_t kind;         /* MC_FIELD_*                                                     */
  float sigma;          /* Gaussian filter width in cells (bead-density fields), > 0       */
  int32_t radius;       /* truncation radius R of the filter; 0 => ceil(5*sigma); R <= 16  */
  float coupling;       /* k_rep or chi in physical units; lattice value = coupling*dt^2   */
  int32_t n_sources;    /* static-source fields: number of packets                         */
  const float* sources; /* HOST [n_sources][4] = cx, cy, amplitude, width (cells)          */
} mc_field_params;

typedef struct {
  int32_t nx, ny;    /* periodic grid, each a multiple of 32, >= 32                        */
  float dt;          /* physical time per step (> 0)                                       */
  float nu;          /* kinematic viscosity, cell^2/time; nu_lat = nu*dt; tau+ = 3nu_lat+.5 */
  float trt_lambda;  /* TRT magic parameter Lambda (> 0), 0.25 is the usual choice         */
  float rho0;        /* rest density of the fluid (> 0), 1.0                               */
  float k_el;        /* elastic coupling, 1/time^2; kappa = k_el*dt^2 (reading 1)          */
  int32_t pbd_iters; /* PBD iterations per step K, 1..8: each a bending pass (Eq. 1) then a
                        position pass (Eq. 2-4) on the positions the previous ones produced
                        (reading 27).  1 = reading 3, the configuration of BASELINE.json */
  int32_t n_fields;  /* 0..4                                                               */
  mc_field_params fields[4];
  int64_t max_beads; /* capacity; mc_load_filaments may load up to this many beads         */
  int32_t coupling;  /* MC_COUPLING_*; with MDF k_el is not used                           */
  int32_t mdf_iters; /* MDF: forcing iterations per step, 1..16 (ignored for FORCE).  The
                        iteration contracts while the bead density interpolated at every bead
                        stays below 4 (chains ~1 node apart, a few overlapping)            */
  int32_t pbd_order; /* MC_PBD_JACOBI (default) or MC_PBD_GAUSS_SEIDEL                     */
  int32_t pbd_project; /* 1: after S7 the PBD displacement of the advected positions (same targets
                        as the step) is added to them directly: "PBD ... directly modifies node
                        positions" (reading 27).  0 (default): only through the fluid  */
  int32_t two_layer; /* 1: two-layer broadcast (reading 28): every exchange of a bead with
                        the grid (S2, S4, S5, S7) goes through its two markers X_i +- h n_i with
                        weight 1/2 each, n_i the unit normal of the chain at the bead; with
                        MC_COUPLING_MDF the forcing iterations sample and broadcast through the
                        markers as well                                                   */
  float layer_offset; /* h, half the distance between the two layers, in nodes; 0 => 0.5; <= 1 */
} mc_world_params;

/* Bytes of DEVICE workspace mc_create needs for these parameters (0 if they are invalid). */
size_t mc_workspace_bytes(const mc_world_params* p /*HOST*/);

/* Create a world: fluid at rest (f_q = w_q rho0), no filaments, step counter 0.
 * Defines: the paper's world = "a two-dimensional world of fields and filaments": the D2Q9
 * lattice-Boltzmann fluid grid whose viscosity is set by one relaxation parameter (
 * nu, trt_lambda -> tau+, tau-, TRT P:L127), the steric density field built from deposited node
 * positions and the persistent energy field of Gaussian packets.
 * workspace: DEVICE, >= mc_workspace_bytes(p) bytes, 256-byte aligned (512-byte alignment, which
 * cudaMalloc and torch give, also lets the gathers use texture views: mc_texture_gathers),
 * owned by the caller and must outlive the world.  cuda_stream: a cudaStream_t (NULL = legacy default stream); all
 * work of this world is enqueued on it.  *out receives the handle.
 * Errors: MC_EINVAL (bad parameters, workspace too small or misaligned), MC_ENOMEM (host),
 * MC_ECUDA. */
int mc_create(const mc_world_params* p /*HOST*/, void* workspace /*DEVICE*/, size_t workspace_bytes,
              void* cuda_stream, mc_world** out /*HOST*/);

/* Load (replace) the filaments.
 * Defines: the paper's filament = a chain of nodes in continuous 2-D space whose edges carry the
 * rest length L_rest, the rest angle theta_rest and the optional stiffnesses k_bend, k_shear,
 * k_stretch "set on the edge level instead of globally" (direct encoding = one value per
 * node), with a time-dependent rest angle -- and, with act_L_amp, rest length -- as the
 * controller would emit them per node and time (hand-designed sinusoids P:L153).
 * offsets: HOST int32 [n_fil+1], offsets[0] = 0, chain f owns
 * beads offsets[f] .. offsets[f+1]-1, every chain >= 3 beads, N = offsets[n_fil] <= max_beads.
 * All other arrays are DEVICE float arrays, chain-ordered:
 *   xy [N][2] unwrapped positions;
 *   L_rest[i], k_shear[i], k_stretch[i] belong to edge (i,i+1) (last entry of a chain unused);
 *   theta_rest[i], k_bend[i], act_amp[i], act_phase[i], act_period[i] belong to the joint at
 *   bead i (first/last entry of a chain unused);
 *   theta*_i(n) = theta_rest[i] + act_amp[i]*sin(2*pi*n*dt/act_period[i] + act_phase[i]).
 * Stiffnesses must lie in [0,1] and periods be > 0, else MC_EINVAL.  Synchronises the stream.
 * The fluid state and the step counter are left as they are. */
int mc_load_filaments(mc_world* w, int32_t n_fil, const int32_t* offsets /*HOST*/,
                      const float* xy /*DEVICE*/, const float* L_rest /*DEVICE*/,
                      const float* theta_rest /*DEVICE*/, const float* k_bend /*DEVICE*/,
                      const float* k_shear /*DEVICE*/, const float* k_stretch /*DEVICE*/,
                      const float* act_amp /*DEVICE*/, const float* act_phase /*DEVICE*/,
                      const float* act_period /*DEVICE*/);

/* Time-dependent rest LENGTH ("The CPPN outputs the rest angle theta_rest and the rest length
 * L_rest"; P:L153 jellyfish "contractile movement"; reading 27):
 *   L*_e(n) = L_rest[e] + act_L_amp[e] * sin(2*pi*n*dt/act_period[e] + act_phase[e])
 * with the period and phase of entry e (the entry that serves joint e and edge (e, e+1)).
 * act_L_amp: DEVICE float [N], chain-ordered, or NULL to switch the actuation off.  Call after
 * mc_load_filaments (a load resets it to none).  Synchronises the stream. */
int mc_set_length_actuation(mc_world* w, const float* act_L_amp /*DEVICE*/);

/* Replace the bead positions of the loaded filaments and keep everything else (parameters, fluid,
 * step counter).  xy: DEVICE float [N][2], chain-ordered like mc_load_filaments.  The next step
 * rebuilds the tile lists.  Synchronises the stream.  Errors: MC_EINVAL, MC_ECUDA. */
int mc_set_positions(mc_world* w, const float* xy /*DEVICE*/);

/* Advance n >= 0 steps of the update S0..S7 listed at the top of this header: PBD bending pass
 * Eq. 1 and position pass Eq. 2-4 of "each iteration", steric
 * field deposit -> Gaussian -> gradient -> repulsive force, immersed-boundary exchange with
 * the fluid and the D2Q9 TRT fluid update.
 * Asynchronous: kernels are enqueued on the world's stream and the
 * call returns without synchronising.  Blocks of four steps are replayed from a CUDA graph when
 * the stream can be captured (not the legacy default stream); the results are bit-identical to
 * direct launches, so mc_step(a) then mc_step(b) equals mc_step(a + b).  Errors: MC_EINVAL, MC_ECUDA (launch failure),
 * MC_EDIVERGED (a previous mc_read_state saw the sticky divergence flag: non-finite bead
 * position or |u| > 0.3). */
int mc_step(mc_world* w, int32_t n);

/* Copy the state out: what the paper's experiments read from a rollout -- node positions (fitness =
 * displacement; loss on the final shape), the fluid and scalar fields of the
 * world and the energy sensed at the nodes.
 * Synchronises the stream.  Every output pointer is DEVICE memory of the
 * stated size and may be NULL (skipped); step_out is HOST.
 *   xy    [N][2]        bead positions
 *   u     [2][ny][nx]   velocity stored by the last step's S6 (lattice units)
 *   rho   [ny][nx]      fluid density sum_q f_q of the current (pre-collision) populations
 *   fdev  [9][ny][nx]   current pre-collision populations as deviations f_q - w_q*rho0
 *                       (the library stores populations shifted; un-shifting in fp32 would
 *                       throw their low bits away)
 *   field [n_fields][ny][nx]  last step's filtered bead density, or the static field c
 *   force [N][2]        last step's total bead force F_i (lattice units; MDF: the summed
 *                       direct-forcing increments)
 *   sense [N]           last step's sum over static fields of c interpolated at the bead
 * Returns MC_EDIVERGED (after filling the outputs) if the divergence flag is set. */
int mc_read_state(mc_world* w, int64_t* step_out /*HOST*/, float* xy, float* u, float* rho,
                  float* fdev, float* field, float* force, float* sense);

/* Checkpoint / resume: replace the fluid state and the step counter by a state read earlier with
 * mc_read_state ("discrete grids which store information about the world, such as the fluid
 * state").  fdev: DEVICE float [9][ny][nx], pre-collision populations as deviations f_q - w_q*rho0
 * exactly as mc_read_state returns them, or NULL to keep the fluid; step: the step index the next
 * mc_step starts from (it selects the actuation phase).  Together with mc_load_filaments /
 * mc_set_positions this restores a world: a resumed run continues like the uninterrupted one up to
 * rounding (the tile lists are rebuilt, and their lengths set the fixed-point scales).  Clears a
 * divergence flag.  Synchronises the stream.  Errors: MC_EINVAL, MC_ESTATE (batch member), MC_ECUDA. */
int mc_load_fluid(mc_world* w, int64_t step, const float* fdev /*DEVICE or NULL*/);

/* Last step's intermediates, for parity checks (same rules as mc_read_state):
 *   rho_b [ny][nx] deposited bead density (S2); G [2][ny][nx] spread force (S5). */
int mc_read_intermediates(mc_world* w, float* rho_b, float* G);

/* The hot path fuses S5 into the fluid kernel and never stores G.  mc_keep_intermediates(w, 1)
 * makes the following steps store it too (slower; for parity checks); without it
 * mc_read_intermediates with a non-NULL G returns MC_ESTATE.  rho_b is always stored while the
 * world has a bead-density field. */
int mc_keep_intermediates(mc_world* w, int32_t on);

/* The per-bead 4x4 gathers of K1 (force-gradient field) and K4 (fluid velocity) send part of
 * their loads through the texture pipe (linear float2 views of the same memory, raw fetches:
 * identical bits) when the views could be created at mc_create.
 * mc_texture_gathers(w, 0) makes the following steps use plain loads only (for tests and
 * measurements), (w, 1) restores the default.  Returns 1 if the texture path is in use after
 * the call, 0 if not, or a negative error. */
int mc_texture_gathers(mc_world* w, int32_t on);

/* Crowded worlds: the tile-accumulation kernels (S2 deposit; S5 spread fused with S6) can give a
 * 32x32 tile a thread-block cluster of c CTAs that share the tile's bead list and combine their
 * integer partial sums through distributed shared memory (identical bits).
 * mc_load_filaments switches this on (c = 4) when the largest tile list exceeds 4096 beads: the
 * tiles listing more than 1024 beads are then served by a cluster launch of their own that runs
 * beside the one-CTA-per-tile launch over all other tiles (second stream owned by the world).
 * mc_cluster_tiles(w, c) with c in {0, 2, 4, 8} forces the setting for the following steps (0: one
 * CTA per tile), c | MC_CLUSTER_ALL_TILES gives EVERY tile a cluster in one launch (the simpler
 * scheme, for tests and measurements), c = -1 restores the automatic choice.  Returns the cluster
 * size in use after the call, or a negative error. */
#define MC_CLUSTER_ALL_TILES 64
int mc_cluster_tiles(mc_world* w, int32_t c);

/* Optional per-kernel timing with CUDA events on the world's stream (used by bench.py for the
 * roofline line; off by default, costs one event record per kernel group when on).
 * Slots: 0 K0 bin, 1 K2a deposit, 2 K3a filter+gradient, 3 K1 filament force, 4 K2b spread (FORCE
 * coupling: empty, S5 is fused into the fluid kernel and is timed in slot 5; MDF coupling: the
 * moments, forcing and broadcast kernels K5a-c),
 * 5 K3b fluid, 6 K4 interpolate+integrate.  mc_profile_enable(w,1) starts a capture of up to
 * 64 steps; mc_profile_read synchronises, writes the summed milliseconds per slot to
 * ms (HOST float[MC_PROF_SLOTS]) and the number of captured steps, and restarts the capture. */
#define MC_PROF_SLOTS 7
int mc_profile_enable(mc_world* w, int32_t on);
int mc_profile_read(mc_world* w, float* ms /*HOST*/, int32_t* steps /*HOST*/);

/* Kernels launched on the world's stream since mc_create (a plain host counter). */
int64_t mc_launch_count(const mc_world* w);

/* ---- batched worlds --------------------------------------------------------
 * The paper's workload is a population of small worlds stepped in lock-step ("large
 * populations ... over evolutionary timescales"; P:L173-179 NEAT / MAP-Elites; P:L190 256 x 256
 * grids): singly such a world is bound by kernel-launch overhead.  A batch holds n_worlds worlds of
 * IDENTICAL parameters and chain structure (offsets) -- positions and per-bead parameters differ --
 * and launches every kernel of the step once for all of them.  World k of a batch computes exactly
 * what the same world computes alone through mc_step, bit for bit.
 *
 * workspace: DEVICE, mc_batch_workspace_bytes(p, n_worlds) = n_worlds * mc_workspace_bytes(p) bytes,
 * 256-byte aligned, owned by the caller; world k lives at offset k * mc_workspace_bytes(p).
 * mc_load_filaments_batch: offsets HOST int32 [n_fil+1] shared by all worlds; every other array is
 * DEVICE float [n_worlds][N] ([n_worlds][N][2] for xy), world-major; act_L_amp may be NULL.
 * mc_batch_world(b, k): the handle of world k, valid until mc_destroy_batch, for mc_read_state,
 * mc_read_intermediates, mc_set_positions, mc_last_error and the switches; mc_step,
 * mc_load_filaments and mc_set_length_actuation on it return MC_ESTATE (the batch steps together).
 * Errors as for the single-world calls; mc_batch_last_error gives the message (b == NULL: of the
 * last failed mc_create_batch on this thread). */
typedef struct mc_batch mc_batch;
size_t mc_batch_workspace_bytes(const mc_world_params* p /*HOST*/, int32_t n_worlds);
int mc_create_batch(const mc_world_params* p /*HOST*/, int32_t n_worlds, void* workspace /*DEVICE*/,
                    size_t workspace_bytes, void* cuda_stream, mc_batch** out /*HOST*/);
int mc_load_filaments_batch(mc_batch* b, int32_t n_fil, const int32_t* offsets /*HOST*/,
                            const float* xy /*DEVICE*/, const float* L_rest /*DEVICE*/,
                            const float* theta_rest /*DEVICE*/, const float* k_bend /*DEVICE*/,
                            const float* k_shear /*DEVICE*/, const float* k_stretch /*DEVICE*/,
                            const float* act_amp /*DEVICE*/, const float* act_phase /*DEVICE*/,
                            const float* act_period /*DEVICE*/, const float* act_L_amp /*DEVICE or NULL*/);
int mc_step_batch(mc_batch* b, int32_t n);
/* Positions of ALL worlds in one call each way (the population loop: upload the individuals, step,
 * read back their displacement = fitness).  xy: DEVICE float [n_worlds][N][2], world-major,
 * chain-ordered.  mc_set_positions_batch keeps parameters, fluid and step counter and makes the next
 * step rebuild the tile lists; mc_read_positions_batch also returns MC_EDIVERGED if any world's
 * divergence flag is set (after filling xy).  Both synchronise the stream. */
int mc_set_positions_batch(mc_batch* b, const float* xy /*DEVICE*/);
int mc_read_positions_batch(mc_batch* b, int64_t* step_out /*HOST*/, float* xy /*DEVICE*/);
mc_world* mc_batch_world(mc_batch* b, int32_t k);
void mc_destroy_batch(mc_batch* b);
const char* mc_batch_last_error(const mc_batch* b);

/* ---- one entry point that allocates nothing ------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid it) and therefore cannot provide a workspace: S2 on its own,
 *   rho_b(g) = sum_i delta_h(g - X_i)      ("node positions are deposited onto a grid"; readings 7, 13)
 * with the step's own kernels (tile lists + fixed-point shared-memory accumulation), their scratch
 * in a file-scope static device array of the library (803,328 bytes, held by every GPU that loads
 * libmc.so until the process exits).  Limits: n_beads <= MC_NOALLOC_MAX_BEADS and
 * (nx/32)*(ny/32) <= MC_NOALLOC_MAX_TILES (e.g. 1024 x 1024 nodes); larger sizes return MC_EINVAL with
 * a message that names the limit.  The call makes no cudaMalloc / cudaFree and calls no allocating
 * routine; it enqueues three kernels on cuda_stream (NULL = legacy default stream) and returns
 * without synchronising.
 *   xy    DEVICE float [n_beads][2], unwrapped positions, 8-byte aligned (may be NULL if n_beads = 0)
 *   rho_b DEVICE float [ny][nx] out, 16-byte aligned
 * The result equals what a world's S2 computes from the same positions (mc_read_intermediates), bit
 * for bit when that world's tile lists are fresh, else to fixed-point rounding (~1e-7).
 * All calls on a device share the one scratch array, which keeps the previous call's contents (every
 * call clears what must start at zero): calls that OVERLAP on the GPU -- different streams, or
 * host threads without ordering -- race on it; serialise them on one stream or with events.
 * Errors: MC_EINVAL, MC_ECUDA; message from mc_noalloc_last_error (per host thread). */
#define MC_NOALLOC_MAX_BEADS 32768
#define MC_NOALLOC_MAX_TILES 1024
int mc_deposit_noalloc(int32_t nx, int32_t ny, int32_t n_beads, const float* xy /*DEVICE*/,
                       float* rho_b /*DEVICE*/, void* cuda_stream);
const char* mc_noalloc_last_error(void);

/* Frees the host handle only (the workspace belongs to the caller).  NULL is allowed. */
void mc_destroy(mc_world* w);

/* Message of the last error on this world (handle-owned string; "" if none).  With
 * w == NULL returns the message of the last failed mc_create on this thread. */
const char* mc_last_error(const mc_world* w);

#ifdef __cplusplus
}
#endif
#endif

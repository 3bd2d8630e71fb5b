// mc_api.cu -- host side of libmc.so: the C ABI of include/mc.h, workspace layout, and the
// per-step launch sequence K0 -> K2a -> K3a -> K1 -> K2b -> K3b -> K4.
// No CPU implementation of any step lives here: without a CUDA device every call fails.
#include "../../include/mc.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <algorithm>
#include <numeric>
#include <vector>

#include "k_blur.cuh"
#include "k_cluster.cuh"
#include "k_filament.cuh"
#include "k_g2p.cuh"
#include "k_lbm.cuh"
#include "k_mdf.cuh"
#include "k_p2g.cuh"
#include "k_pbd.cuh"
#include "k_tile.cuh"

namespace {

thread_local std::string g_create_error;
thread_local bool g_batch_call = false;  // set while an mc_*_batch call drives its member worlds

constexpr size_t ALIGN = 256;
inline size_t align_up(size_t v) { return (v + ALIGN - 1) / ALIGN * ALIGN; }

struct Layout {
  size_t fA, fB, u, rho_b, A, G, cfield, csum, As, tile_count, tile_start, bucket_count, bucket_cursor, tile_rho_max, tile_fmax;
  size_t X, PA, PB, PC, PD, F, sense, list, src, bflags, scratch, flags, sources;
  size_t V, dF, hrinv, mdf_fmax;  // MDF coupling only
  size_t PE, O, Dp;               // rest-length actuation amplitudes; two-layer offsets; projection displacement
  size_t crowded, crowded_rank;   // crowded-tile table of the split cluster launch (k_tile.cuh CrowdedTable)
  size_t total;
};

struct Derived {
  int n_density = 0, n_static = 0;
  int R[4] = {0, 0, 0, 0};
  size_t n_src_floats = 0;
};

bool validate(const mc_world_params* p, Derived* d, std::string* why) {
  if (!p) { *why = "null params"; return false; }
  if (p->nx < 32 || p->ny < 32 || p->nx % 32 || p->ny % 32) { *why = "nx, ny must be multiples of 32, >= 32"; return false; }
  if ((int64_t)p->nx * p->ny > (int64_t)1 << 30 || p->ny > 65535) { *why = "grid too large"; return false; }
  if (!(p->dt > 0) || !(p->nu > 0) || !(p->trt_lambda > 0) || !(p->rho0 > 0)) { *why = "dt, nu, trt_lambda, rho0 must be > 0"; return false; }
  if (p->pbd_iters < 1 || p->pbd_iters > 8) { *why = "pbd_iters must be 1..8"; return false; }
  if (p->pbd_order != MC_PBD_JACOBI && p->pbd_order != MC_PBD_GAUSS_SEIDEL) { *why = "unknown pbd_order"; return false; }
  if ((p->pbd_project != 0 && p->pbd_project != 1) || (p->two_layer != 0 && p->two_layer != 1)) { *why = "pbd_project and two_layer must be 0 or 1"; return false; }
  if (!(p->layer_offset >= 0.0f) || p->layer_offset > 1.0f) { *why = "layer_offset must lie in [0, 1]"; return false; }
  // two layers list 2 N markers: the 32-bit list offsets then hold up to 8 N
  if (p->two_layer && p->max_beads > ((int64_t)1 << 28) - 1) { *why = "max_beads out of range for two_layer (0 .. 2^28 - 1)"; return false; }
  if (p->n_fields < 0 || p->n_fields > 4) { *why = "n_fields must be 0..4"; return false; }
  // the tile lists hold up to 4 N entries addressed with 32-bit ints (k_tile.cuh)
  if (p->max_beads < 0 || p->max_beads > ((int64_t)1 << 29) - 1) { *why = "max_beads out of range (0 .. 2^29 - 1)"; return false; }
  if (p->coupling != MC_COUPLING_FORCE && p->coupling != MC_COUPLING_MDF) { *why = "unknown coupling"; return false; }
  if (p->coupling == MC_COUPLING_MDF && (p->mdf_iters < 1 || p->mdf_iters > 16)) { *why = "mdf_iters must be 1..16"; return false; }
  for (int k = 0; k < p->n_fields; ++k) {
    const mc_field_params& f = p->fields[k];
    if (f.kind == MC_FIELD_BEAD_DENSITY) {
      if (!(f.sigma > 0)) { *why = "field sigma must be > 0"; return false; }
      const int R = f.radius > 0 ? f.radius : (int)std::ceil(5.0 * (double)f.sigma);
      if (R < 1 || R > mc::BLUR_MAX_R) { *why = "filter radius must be 1..16"; return false; }
      if (2 * R + 1 > p->nx || 2 * R + 1 > p->ny) { *why = "filter wider than the grid"; return false; }
      d->R[k] = R;
      d->n_density++;
    } else if (f.kind == MC_FIELD_STATIC_SOURCE) {
      if (f.n_sources < 0 || (f.n_sources > 0 && !f.sources)) { *why = "bad static sources"; return false; }
      for (int s = 0; s < f.n_sources; ++s)
        if (!(f.sources[4 * s + 3] > 0)) { *why = "source width must be > 0"; return false; }
      d->n_static++;
      d->n_src_floats += 4 * (size_t)f.n_sources;
    } else {
      *why = "unknown field kind";
      return false;
    }
  }
  return true;
}

Layout make_layout(const mc_world_params* p, const Derived& d) {
  Layout L;
  const size_t nc = (size_t)p->nx * p->ny, N = (size_t)p->max_beads, f4 = sizeof(float);
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off += align_up(bytes ? bytes : 1); return o; };
  L.fA = take(9 * nc * f4);
  L.fB = take(9 * nc * f4);
  L.u = take(2 * nc * f4);
  L.rho_b = take(nc * f4);
  L.A = take(d.n_density ? 2 * nc * f4 : 0);
  L.G = take(2 * nc * f4);
  L.cfield = take(d.n_static * nc * f4);
  L.csum = take(d.n_static ? nc * f4 : 0);
  L.As = take(d.n_static ? 2 * nc * f4 : 0);
  const size_t nt = nc / (mc::TS * mc::TS);
  L.tile_count = take(nt * 4);
  L.tile_start = take((nt + 1) * 4);
  L.bucket_count = take(nt * 32 * 4);   // per (tile, bank key), zero outside a rebuild
  L.bucket_cursor = take(nt * 32 * 4);
  L.tile_rho_max = take(nt * 4);
  L.tile_fmax = take(nt * 4);
  L.X = take(N * 8);
  L.PA = take(N * 16);
  L.PB = take(N * 16);
  L.PC = take(N * 16);
  L.PD = take(N * 8);
  L.F = take(N * 8);
  L.sense = take(N * 4);
  L.list = take((p->two_layer ? 2 : 1) * N * 4 * 4);   // a bead (two-layer: each of its 2 markers) is listed in at most 4 tiles
  L.src = take(N * 4);        // internal bead -> caller's bead
  L.bflags = take(N);         // first/last/odd flags, one byte per bead (PC.w carries them for K1; k_markers reads these)
  L.scratch = take((N / 3 + 2) * 8);  // load-time: chain offsets and sort keys
  L.flags = take(64 * 4);
  L.sources = take(d.n_src_floats * f4);
  const bool mdf = p->coupling == MC_COUPLING_MDF;
  L.V = take(mdf ? N * 8 : 0);
  L.dF = take(mdf ? N * 8 : 0);
  L.hrinv = take(mdf ? nc * f4 : 0);
  L.mdf_fmax = take(mdf ? (size_t)p->mdf_iters * nt * 4 : 0);  // per iteration: per-tile bound on |dF| (last: |F|)
  L.PE = take(N * 4);
  L.O = take(p->two_layer ? N * 8 : 0);
  L.Dp = take(p->pbd_project ? N * 8 : 0);
  L.crowded = take(nt * 4);
  L.crowded_rank = take(nt * 4);
  L.total = off;
  return L;
}

}  // namespace

struct mc_world {
  mc_world_params p;
  Derived d;
  Layout L;
  char* ws = nullptr;
  cudaStream_t stream = nullptr;
  int nx = 0, ny = 0;
  size_t nc = 0;
  int64_t step = 0;
  int cur = 0;  // which of fA/fB holds the current post-collision populations
  int n_fil = 0;
  int N = 0;
  int stride = 60;   // K1 window advance: 64 when all chains share a length dividing 64, else 64 - 4 halo_lanes
  int n_windows = 0;
  int halo_lanes = 1;      // K1 halo on either side of an overlapping window: K (Jacobi) or ceil(3K/2) (Gauss-Seidel) lanes
  bool has_L_act = false;  // mc_set_length_actuation gave amplitudes
  float layer_h = 0.5f;    // two_layer: half distance between the layers
  // batched worlds (mc_batch): the leader (world 0) launches every kernel for batch_n worlds whose
  // workspaces lie batch_stride bytes apart; a single world is a batch of one
  int batch_n = 1;
  size_t batch_stride = 0;
  bool batch_member = false;  // owned by an mc_batch: stepped and reloaded only through it
  int coop_grid = 0;  // CTAs of the one-launch cooperative K0 of large single worlds (0: device cannot, four launches)
  // crowded worlds: the cluster launch over the crowded tiles runs on a second stream beside the
  // one-CTA-per-tile launch over the rest (fork / join by events; also under graph capture)
  bool split_on = true;   // mc_cluster_tiles(w, c | MC_CLUSTER_ALL_TILES): every tile gets a cluster (round-1 scheme; tests)
  cudaStream_t side = nullptr;
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
  cudaTextureObject_t tex_u = 0, tex_A = 0;  // linear float2 views of u and A for the texture-pipe half of the gathers
  int n_sm = 148;               // SMs of the device the world lives on (grid-stride kernels size their grids by it)
  bool uniform_params = false;  // K1 variant: L_rest, stiffnesses and period identical for all beads
  int cluster = 0;        // crowded worlds: CTAs per tile of the P2G kernels (k_cluster.cuh); 0 = one CTA per tile
  int cluster_auto = 0;   // what mc_load_filaments chose from the largest tile list
  int cluster_user = -1;  // mc_cluster_tiles override (-1: automatic)
  int deposit_threads = 128;  // CTA size of K2a: 128 hides the per-tile latency better, crowded worlds want 256
  // CUDA graphs of GRAPH_STEPS consecutive steps, one per ping-pong phase, captured on first use
  // (the ping-pong phase is the only host-side state a step depends on); GRAPH_STEPS is even
  cudaGraphExec_t graph[2] = {nullptr, nullptr};
  int64_t graph_launches[2] = {0, 0};
  bool graph_off = false;  // the stream cannot be captured (e.g. the legacy default stream): direct launches
  std::vector<int32_t> loaded_offsets;  // offsets of the last load: same chains => keep the internal order
  float rho0 = 1, omega_p = 1, omega_m = 1, kappa = 0;
  float coef[4] = {0, 0, 0, 0};  // lattice coupling with the sign of the force
  mc::BlurTaps taps[4];
  int static_slot[4] = {-1, -1, -1, -1};
  int64_t launches = 0;
  bool diverged = false;
  bool tex_on = true;   // mc_texture_gathers
  bool keep_G = false;  // mc_keep_intermediates: the fused spread+fluid kernel also stores G
  std::string err;
  // optional per-kernel timing (mc_profile_*): events at the 8 boundaries of a step
  bool prof_on = false;
  int prof_steps = 0;
  std::vector<cudaEvent_t> prof_ev;  // [MC_PROF_MAX_STEPS][MC_PROF_SLOTS + 1]

  template <class T>
  T* ptr(size_t off) const { return reinterpret_cast<T*>(ws + off); }
  float* fbuf(int which) const { return ptr<float>(which ? L.fB : L.fA); }
};

namespace {

int fail(mc_world* w, int code, const std::string& msg) {
  if (w) w->err = msg;
  return code;
}

int check_cuda(mc_world* w, const char* what) {
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(w, MC_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
  return MC_OK;
}

// first failing CUDA call of a sequence: `ok(call, "what")` records it in the world and returns false
struct CudaSeq {
  mc_world* w;
  const char* where;
  int rc = MC_OK;
  bool ok(cudaError_t e, const char* what) {
    if (e == cudaSuccess || rc != MC_OK) return rc == MC_OK;
    rc = fail(w, MC_ECUDA, std::string(where) + ": " + what + ": " + cudaGetErrorString(e));
    return false;
  }
  // after a kernel launch: launch-configuration errors surface here (execution errors at the next sync)
  bool launched(const char* what) { return ok(cudaPeekAtLastError(), what); }
};

constexpr int PROF_MAX_STEPS = 64;
constexpr int GRAPH_STEPS = 4;
// worlds up to this size rebuild their tile lists in one single-CTA launch (launch bound anyway)
constexpr int K0_SMALL_BEADS = 32768, K0_SMALL_TILES = 1024;
// ... and up to this size in one launch of one 8-CTA cluster (k_tile.cuh)
constexpr int K0_MEDIUM_BEADS = 262144, K0_MEDIUM_TILES = 8192;
static_assert(GRAPH_STEPS % 2 == 0, "graph period");

// crowded-tile table of this world (k_tile.cuh); n_crowded lives in the flag words
mc::CrowdedTable crowded_table(mc_world* w) {
  return mc::CrowdedTable{w->ptr<int>(w->L.crowded), w->ptr<int>(w->L.crowded_rank), w->ptr<int>(w->L.flags) + 6};
}
// at most this many crowded tiles get a cluster; the rest stay with the one-CTA launch (correct, slower)
constexpr int CL_MAX = 1024;

bool ensure_side_stream(mc_world* w) {
  if (w->side) return true;
  if (cudaStreamCreateWithFlags(&w->side, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); w->side = nullptr; return false; }
  if (cudaEventCreateWithFlags(&w->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
      cudaEventCreateWithFlags(&w->ev_join, cudaEventDisableTiming) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  return true;
}

void drop_graphs(mc_world* w) {
  for (int k = 0; k < 2; ++k)
    if (w->graph[k]) { cudaGraphExecDestroy(w->graph[k]); w->graph[k] = nullptr; }
}

inline void prof_mark(mc_world* w, int boundary) {
  if (w->prof_on && w->prof_steps < PROF_MAX_STEPS)
    cudaEventRecord(w->prof_ev[(size_t)w->prof_steps * (MC_PROF_SLOTS + 1) + boundary], w->stream);
}

int pick_bx(int nx) { return nx % 256 == 0 ? 256 : (nx % 128 == 0 ? 128 : (nx % 64 == 0 ? 64 : 32)); }

template <int R>
void launch_blur_R(mc_world* w, int k, const float2* base, float2* A, float* field_out) {
  const int grid = (w->nx / mc::BLUR_T) * (w->ny / mc::BLUR_T);
  // the step filters every world of a batch; a read-out (field_out given) only this world
  const unsigned nb = field_out ? 1u : (unsigned)w->batch_n;
  mc::k_blur_grad<R><<<dim3(grid, nb), mc::BLUR_THREADS, 0, w->stream>>>(
      w->nx, w->ny, w->taps[k], w->ptr<float>(w->L.rho_b), w->coef[k], base, A, field_out, w->batch_stride,
      // crowded worlds skip the tiles whose 3 x 3 neighbourhood holds no bead (exact); only inside a step:
      // at read-out time the fused kernel has already reset the per-tile maxima
      (w->cluster > 0 && !field_out && R <= 31) ? w->ptr<float>(w->L.tile_rho_max) : nullptr);
}

// K3a for bead-density field k; first: start from the static part, else add to the planes in A
void launch_blur(mc_world* w, int k, bool first, float* field_out) {
  float2* A = w->ptr<float2>(w->L.A);
  const float2* base = first ? (w->d.n_static ? w->ptr<float2>(w->L.As) : nullptr) : A;
  switch (w->d.R[k]) {
#define MC_BLUR_CASE(R) case R: launch_blur_R<R>(w, k, base, A, field_out); break;
    MC_BLUR_CASE(1) MC_BLUR_CASE(2) MC_BLUR_CASE(3) MC_BLUR_CASE(4) MC_BLUR_CASE(5) MC_BLUR_CASE(6)
    MC_BLUR_CASE(7) MC_BLUR_CASE(8) MC_BLUR_CASE(9) MC_BLUR_CASE(10) MC_BLUR_CASE(11) MC_BLUR_CASE(12)
    MC_BLUR_CASE(13) MC_BLUR_CASE(14) MC_BLUR_CASE(15) MC_BLUR_CASE(16)
#undef MC_BLUR_CASE
    default: break;
  }
  w->launches++;
}

int enqueue_step(mc_world* w) {
  const int N = w->N, nx = w->nx, ny = w->ny;
  cudaStream_t st = w->stream;
  float2* X = w->ptr<float2>(w->L.X);
  float2* F = w->ptr<float2>(w->L.F);
  int* tile_count = w->ptr<int>(w->L.tile_count);
  int* tile_start = w->ptr<int>(w->L.tile_start);
  int* bucket_count = w->ptr<int>(w->L.bucket_count);
  int* bucket_cursor = w->ptr<int>(w->L.bucket_cursor);
  float* tile_rho_max = w->ptr<float>(w->L.tile_rho_max);
  unsigned* tile_fmax = w->d.n_density ? w->ptr<unsigned>(w->L.tile_fmax) : nullptr;
  int* list = w->ptr<int>(w->L.list);
  float* rho_b = w->ptr<float>(w->L.rho_b);
  float* G0 = w->ptr<float>(w->L.G);
  float* G1 = G0 + w->nc;
  int* flag = w->ptr<int>(w->L.flags);
  const int n_tiles = (nx / mc::TS) * (ny / mc::TS);
  const unsigned nb = (unsigned)w->batch_n;       // worlds per launch: blockIdx.y (.z on 2-D grids)
  const size_t ws = w->batch_stride;
  const dim3 tgrid(nx / mc::TS, ny / mc::TS, nb);
  const int bt = 256;
  const bool beads = N > 0;
  const bool mdf = w->p.coupling == MC_COUPLING_MDF;
  const bool two = w->p.two_layer != 0;
  const float2* O = two ? w->ptr<float2>(w->L.O) : nullptr;
  const int n_items = two ? 2 * N : N;            // listed points: beads, or their two-layer markers
  const int bgrid = (n_items + bt - 1) / bt;
  mc::ListState* ls_state = reinterpret_cast<mc::ListState*>(w->ptr<int>(w->L.flags) + 16);
  // crowded worlds: the tiles with long lists go to a cluster launch of their own on a second stream
  const bool split = w->cluster > 0 && !two && w->split_on && w->side != nullptr;
  const mc::CrowdedTable ctab = split ? crowded_table(w) : mc::CrowdedTable{nullptr, nullptr, nullptr};
  const int cl_max = std::min(n_tiles, CL_MAX);
  auto fork_side = [&]() { cudaEventRecord(w->ev_fork, st); cudaStreamWaitEvent(w->side, w->ev_fork, 0); };
  auto join_side = [&]() { cudaEventRecord(w->ev_join, w->side); cudaStreamWaitEvent(st, w->ev_join, 0); };

  prof_mark(w, 0);
  if (beads) {
    // K0: tile binning (policy, count, scan, bucket starts, fill).  The kernels return at once
    // unless the policy finds the lists' drift bound used up (k_tile.cuh).
    if (n_items <= K0_SMALL_BEADS && n_tiles <= K0_SMALL_TILES) {
      // small world: one launch of one CTA (per world) instead of four (k_tile.cuh)
      mc::k_list_build_small<<<dim3(1, nb), 1024, 0, st>>>(ls_state, X, O, N, nx, ny, n_tiles, tile_count, tile_start,
                                                           bucket_count, bucket_cursor, list, ctab, ws);
      w->launches += 1;
    } else if (n_items <= K0_MEDIUM_BEADS && n_tiles <= K0_MEDIUM_TILES) {
      mc::k_list_build_cluster<<<dim3(mc::K0_CLUSTER, nb), 1024, 0, st>>>(ls_state, X, O, N, nx, ny, n_tiles, tile_count,
                                                                          tile_start, bucket_count, bucket_cursor, list, ctab, ws);
      w->launches += 1;
    } else if (nb == 1 && w->coop_grid > 0) {
      // large single world: one cooperative launch (k_tile.cuh k_list_build_coop)
      int* exit_ctr = w->ptr<int>(w->L.flags) + 7;
      const float2* Xc = X;
      int Nc = N, nxc = nx, nyc = ny, ntc = n_tiles;
      mc::CrowdedTable ctc = ctab;
      void* args[] = {&ls_state, &exit_ctr, &Xc, (void*)&O, &Nc, &nxc, &nyc, &ntc, &tile_count, &tile_start,
                      &bucket_count, &bucket_cursor, &list, &ctc};
      const int cgrid = std::min(w->coop_grid, (n_items + 1023) / 1024);
      if (cudaLaunchCooperativeKernel(reinterpret_cast<const void*>(&mc::k_list_build_coop), dim3(cgrid), dim3(1024), args, 0, st) != cudaSuccess)
        return fail(w, MC_ECUDA, std::string("mc_step: cooperative launch of K0: ") + cudaGetErrorString(cudaGetLastError()));
      w->launches += 1;
    } else {
      const int k0grid = bgrid < w->n_sm * 8 ? bgrid : w->n_sm * 8;
      mc::k_tile_bin<false><<<dim3(k0grid, nb), bt, 0, st>>>(ls_state, X, O, N, nx, ny, tile_count, bucket_count, nullptr, ws);
      mc::k_tile_scan<<<dim3(1, nb), 1024, 0, st>>>(ls_state, tile_count, n_tiles, tile_start, ctab, ws);
      mc::k_bucket_starts<<<dim3(std::min((n_tiles + 7) / 8, w->n_sm * 4), nb), 256, 0, st>>>(ls_state, n_tiles, tile_start, bucket_count, bucket_cursor, ws);
      mc::k_tile_bin<true><<<dim3(k0grid, nb), bt, 0, st>>>(ls_state, X, O, N, nx, ny, nullptr, bucket_cursor, list, ws);
      w->launches += 4;
    }
    prof_mark(w, 1);
    // K2a: S2 deposit
    if (w->d.n_density) {
      if (two) {  // two-layer markers: one CTA per tile whatever the crowding
        if (w->deposit_threads == 128) mc::k_deposit_tile<true, true><<<tgrid, 128, 0, st>>>(nx, ny, tile_start, list, X, rho_b, tile_rho_max, tile_fmax, O, ws);
        else mc::k_deposit_tile<false, true><<<tgrid, 256, 0, st>>>(nx, ny, tile_start, list, X, rho_b, tile_rho_max, tile_fmax, O, ws);
      }
      else if (split) {
        // crowded tiles: clusters on the side stream; all other tiles: the light one-CTA kernel beside them
        fork_side();
#define MC_DEP_CL(C) mc::k_deposit_tile_cl<C><<<dim3(cl_max * C, nb), 256, 0, w->side>>>(nx, ny, tile_start, list, X, rho_b, tile_rho_max, tile_fmax, ws, ctab.crowded, ctab.n_crowded, cl_max)
        if (w->cluster == 8) MC_DEP_CL(8);
        else if (w->cluster == 4) MC_DEP_CL(4);
        else MC_DEP_CL(2);
#undef MC_DEP_CL
        mc::k_deposit_tile<true><<<tgrid, 128, 0, st>>>(nx, ny, tile_start, list, X, rho_b, tile_rho_max, tile_fmax, nullptr, ws, ctab.crowded_rank, cl_max);
        join_side();
        w->launches++;
      }
      else if (w->cluster == 8)
        mc::k_deposit_tile_cl<8><<<dim3(n_tiles * 8, nb), 256, 0, st>>>(nx, ny, tile_start, list, X, rho_b, tile_rho_max, tile_fmax, ws);
      else if (w->cluster == 4)
        mc::k_deposit_tile_cl<4><<<dim3(n_tiles * 4, nb), 256, 0, st>>>(nx, ny, tile_start, list, X, rho_b, tile_rho_max, tile_fmax, ws);
      else if (w->cluster == 2)
        mc::k_deposit_tile_cl<2><<<dim3(n_tiles * 2, nb), 256, 0, st>>>(nx, ny, tile_start, list, X, rho_b, tile_rho_max, tile_fmax, ws);
      else if (w->deposit_threads == 128)
        mc::k_deposit_tile<true><<<tgrid, 128, 0, st>>>(nx, ny, tile_start, list, X, rho_b, tile_rho_max, tile_fmax, nullptr, ws);
      else
        mc::k_deposit_tile<false><<<tgrid, w->deposit_threads, 0, st>>>(nx, ny, tile_start, list, X, rho_b, tile_rho_max, tile_fmax, nullptr, ws);
      w->launches++;
      prof_mark(w, 2);
      // K3a: S3 filter + gradient -> force-gradient planes A
      bool first = true;
      for (int k = 0; k < w->p.n_fields; ++k)
        if (w->p.fields[k].kind == MC_FIELD_BEAD_DENSITY) {
          launch_blur(w, k, first, nullptr);
          first = false;
        }
    }
    if (!w->d.n_density) prof_mark(w, 2);
    prof_mark(w, 3);
    // K1: S0 + S1 + S4
    mc::FilamentArgs fa;
    fa.X = X;
    fa.PA = w->ptr<float4>(w->L.PA);
    fa.PB = w->ptr<float4>(w->L.PB);
    fa.PC = w->ptr<float4>(w->L.PC);
    fa.PD = w->ptr<float2>(w->L.PD);
    fa.uni = reinterpret_cast<const float4*>(w->ptr<int>(w->L.flags) + 24);  // flags[24..31]
    fa.F = mdf ? w->ptr<float2>(w->L.V) : F;  // MDF: K1's sum with kappa = 1 is the bead velocity V_i
    fa.sense = w->ptr<float>(w->L.sense);
    fa.A = w->d.n_density ? w->ptr<float2>(w->L.A) : (w->d.n_static ? w->ptr<float2>(w->L.As) : nullptr);
    fa.csum = w->d.n_static ? w->ptr<float>(w->L.csum) : nullptr;
    fa.tile_fmax = tile_fmax;
    fa.N = N;
    fa.nx = nx;
    fa.ny = ny;
    fa.stride = w->stride;
    fa.n_windows = w->n_windows;
    fa.kappa = mdf ? 1.0f : w->kappa;
    fa.step = w->ptr<long long>(w->L.flags) + 4;  // flags[8..9]: device copy of the step counter
    fa.tex_A = (w->tex_on && nb == 1) ? w->tex_A : 0;  // texture views are per world: batches use plain loads
    const bool generic = w->p.pbd_iters > 1 || w->p.pbd_order != MC_PBD_JACOBI || w->has_L_act || two;
    // 64-thread CTAs (two windows): finer-grained scheduling than eight windows per CTA and 42
    // instead of 40 resident warps at 48 registers (world 4d: 256 threads 0.232 ms, 128: 0.225, 64: 0.221, 32: 0.239)
    constexpr int k1t = 64;
    const int k1grid = (w->n_windows * 32 + k1t - 1) / k1t;
    // two of the four support rows of the A gather go through the texture pipe (measured on
    // world 4d: 0 rows 0.254 ms, 1: 0.248, 2: 0.245, 3: 0.256)
    const bool k1tex = fa.A && fa.tex_A;
    if (generic) {
      // literal PBD / rest-length actuation / two-layer gathers: the general kernel (k_pbd.cuh)
      mc::PbdArgs pa;
      pa.f = fa;
      pa.PE = w->has_L_act ? w->ptr<float>(w->L.PE) : nullptr;
      pa.O = O;
      pa.Dp = nullptr;
      pa.iters = w->p.pbd_iters;
      pa.order = w->p.pbd_order;
      pa.halo_lanes = w->halo_lanes;
      pa.step_off = 0;
      if (w->uniform_params) mc::k_filament_pbd<true><<<dim3(k1grid, nb), k1t, 0, st>>>(pa, ws);
      else mc::k_filament_pbd<false><<<dim3(k1grid, nb), k1t, 0, st>>>(pa, ws);
    } else if (w->uniform_params) {
      if (k1tex) mc::k_filament_force<true, 2><<<dim3(k1grid, nb), k1t, 0, st>>>(fa, ws);
      else mc::k_filament_force<true, 0><<<dim3(k1grid, nb), k1t, 0, st>>>(fa, ws);
    } else {
      if (k1tex) mc::k_filament_force<false, 2><<<dim3(k1grid, nb), k1t, 0, st>>>(fa, ws);
      else mc::k_filament_force<false, 0><<<dim3(k1grid, nb), k1t, 0, st>>>(fa, ws);
    }
    prof_mark(w, 4);
    w->launches++;
    if (mdf) {
      // K5 (k_mdf.cuh): u <- u* of the current populations, then mdf_iters x (sample + force),
      // each but the last followed by a broadcast that corrects u on the tiles holding beads.
      // The last increment reaches the fluid through the fused kernel below, which spreads the
      // summed F (spreading is linear) and stores u^K.
      float2* ug = w->ptr<float2>(w->L.u);
      float* hrinv = w->ptr<float>(w->L.hrinv);
      const float2* V = w->ptr<float2>(w->L.V);
      float2* dF = w->ptr<float2>(w->L.dF);
      const int mbx = pick_bx(nx) / 2;
      mc::k_lbm_moments<<<dim3(nx / (2 * mbx), ny, nb), mbx, 0, st>>>(w->fbuf(w->cur), nx, ny, w->rho0, ug, hrinv, ws);
      w->launches++;
      const bool tex = w->tex_on && w->tex_u && nb == 1 && !two;
      const int K = w->p.mdf_iters;
      unsigned* mfmax = w->ptr<unsigned>(w->L.mdf_fmax);  // [K][n_tiles], raised by K5b with atomicMax
      for (unsigned b = 0; b < nb; ++b)
        if (cudaMemsetAsync(reinterpret_cast<char*>(mfmax) + b * ws, 0, (size_t)K * n_tiles * 4, st) != cudaSuccess)
          return fail(w, MC_ECUDA, "mc_step: cudaMemsetAsync(mdf bounds) failed");
      for (int k = 0; k < K; ++k) {
        unsigned* slot = mfmax + (size_t)k * n_tiles;
        const bool first = k == 0, last = k + 1 == K;
#define MC_MDF_FORCE(FI, LA, TX) \
  mc::k_mdf_force<FI, LA, TX><<<dim3((N + 63) / 64, nb), 64, 0, st>>>(N, X, V, ug, w->tex_u, nx, ny, w->rho0, dF, F, slot, ws, O)
        if (tex) {
          if (first && last) MC_MDF_FORCE(true, true, 1);
          else if (first) MC_MDF_FORCE(true, false, 1);
          else if (last) MC_MDF_FORCE(false, true, 1);
          else MC_MDF_FORCE(false, false, 1);
        } else {
          if (first && last) MC_MDF_FORCE(true, true, 0);
          else if (first) MC_MDF_FORCE(true, false, 0);
          else if (last) MC_MDF_FORCE(false, true, 0);
          else MC_MDF_FORCE(false, false, 0);
        }
#undef MC_MDF_FORCE
        w->launches++;
        if (!last) {
          if (two)
            mc::k_mdf_spread_tile<true><<<dim3(n_tiles, nb), 256, 0, st>>>(nx, ny, tile_start, list, X, dF,
                                                                           w->d.n_density ? tile_rho_max : nullptr, slot, hrinv, ug, ws, O);
          else
            mc::k_mdf_spread_tile<false><<<dim3(n_tiles, nb), 256, 0, st>>>(nx, ny, tile_start, list, X, dF,
                                                                            w->d.n_density ? tile_rho_max : nullptr, slot, hrinv, ug, ws);
          w->launches++;
        }
      }
    }
  } else {
    for (int b = 1; b <= 4; ++b) prof_mark(w, b);
  }
  prof_mark(w, 5);
  // K3b: S6 fluid
  mc::LbmArgs la;
  la.src = w->fbuf(w->cur);
  la.dst = w->fbuf(w->cur ^ 1);
  la.G0 = beads ? G0 : nullptr;
  la.G1 = beads ? G1 : nullptr;
  la.u = w->ptr<float2>(w->L.u);
  la.nx = nx;
  la.ny = ny;
  la.rho0 = w->rho0;
  {
    const float wp = w->omega_p, wm = w->omega_m;
    const float cp = 1.0f - 0.5f * wp, cm = 1.0f - 0.5f * wm;
    la.k.wp = wp;
    la.k.hwp = 0.5f * wp;
    la.k.hwm = 0.5f * wm;
    la.k.cp3 = 3.0f * cp;
    la.k.cb = 9.0f * cp;
    la.k.c2 = 3.0f * cm;
    la.k.wp45 = 4.5f * wp;
    la.k.wm3 = 3.0f * wm;
  }
  la.flag = flag;
  la.G0out = G0;
  la.G1out = G1;
  if (beads) {
    // K2b + K3b fused: S5 spread into shared memory, S6 fluid update of the same tile
    la.G0 = nullptr;
    la.G1 = nullptr;
    mc::LbmSpreadArgs ls;
    ls.lbm = la;
    ls.tile_start = tile_start;
    ls.list = list;
    ls.X = X;
    ls.F = F;
    ls.tile_rho_max = w->d.n_density ? tile_rho_max : nullptr;
    // MDF: the bound on the summed F left by the last forcing iteration (K1's is on V)
    ls.tile_fmax = mdf ? w->ptr<unsigned>(w->L.mdf_fmax) + (size_t)(w->p.mdf_iters - 1) * n_tiles : tile_fmax;
    ls.O = O;
    ls.crowded_rank = nullptr; ls.crowded = nullptr; ls.n_crowded = nullptr; ls.cl_max = 0;
#define MC_FUSED_CL(C)                                                                                   \
  {                                                                                                      \
    if (w->keep_G) mc::k_lbm_spread_tile_cl<C, true><<<dim3(n_tiles * C, nb), 256, 0, st>>>(ls, ws);     \
    else mc::k_lbm_spread_tile_cl<C, false><<<dim3(n_tiles * C, nb), 256, 0, st>>>(ls, ws);              \
  }
    if (two) {
      if (w->keep_G) mc::k_lbm_spread_tile<true, true><<<dim3(n_tiles, nb), 256, 0, st>>>(ls, ws);
      else mc::k_lbm_spread_tile<false, true><<<dim3(n_tiles, nb), 256, 0, st>>>(ls, ws);
    }
    else if (split) {
      ls.crowded_rank = ctab.crowded_rank; ls.crowded = ctab.crowded; ls.n_crowded = ctab.n_crowded; ls.cl_max = cl_max;
      fork_side();
#define MC_FUSED_SPLIT(C)                                                                                     \
  {                                                                                                           \
    if (w->keep_G) mc::k_lbm_spread_tile_cl<C, true><<<dim3(cl_max * C, nb), 256, 0, w->side>>>(ls, ws);      \
    else mc::k_lbm_spread_tile_cl<C, false><<<dim3(cl_max * C, nb), 256, 0, w->side>>>(ls, ws);               \
  }
      if (w->cluster == 8) MC_FUSED_SPLIT(8)
      else if (w->cluster == 4) MC_FUSED_SPLIT(4)
      else MC_FUSED_SPLIT(2)
#undef MC_FUSED_SPLIT
      if (w->keep_G) mc::k_lbm_spread_tile<true><<<dim3(n_tiles, nb), 256, 0, st>>>(ls, ws);
      else mc::k_lbm_spread_tile<false><<<dim3(n_tiles, nb), 256, 0, st>>>(ls, ws);
      join_side();
      w->launches++;
    }
    else if (w->cluster == 8) MC_FUSED_CL(8)
    else if (w->cluster == 4) MC_FUSED_CL(4)
    else if (w->cluster == 2) MC_FUSED_CL(2)
    else if (w->keep_G) mc::k_lbm_spread_tile<true><<<dim3(n_tiles, nb), 256, 0, st>>>(ls, ws);
    else mc::k_lbm_spread_tile<false><<<dim3(n_tiles, nb), 256, 0, st>>>(ls, ws);
#undef MC_FUSED_CL
  } else {
    const int bx = pick_bx(nx);
    mc::k_lbm_step<<<dim3(nx / bx, ny, nb), bx, 0, st>>>(la, ws);
  }
  w->launches++;
  w->cur ^= 1;
  prof_mark(w, 6);
  // K4: S7
  if (beads) {
    long long* stepp = w->ptr<long long>(w->L.flags) + 4;
    unsigned* smax = reinterpret_cast<unsigned*>(w->ptr<int>(w->L.flags) + 18);
    // one support row of the u gather through the texture pipe (4d: 0 rows 0.168 ms, 1: 0.156,
    // 2: 0.160, 3: 0.174, 4: 0.193)
    // 64-thread CTAs (world 4d: 256 threads 0.149 ms, 128: 0.146, 64: 0.144)
    constexpr int k4t = 64;
    const int k4grid = (N + k4t - 1) / k4t;
    if (w->tex_on && w->tex_u && nb == 1 && !two)
      mc::k_interp_integrate<1><<<k4grid, k4t, 0, st>>>(N, X, la.u, w->tex_u, nx, ny, flag, stepp, smax, nullptr, ws);
    else
      mc::k_interp_integrate<0><<<dim3(k4grid, nb), k4t, 0, st>>>(N, X, la.u, w->tex_u, nx, ny, flag, stepp, smax, O, ws);
    w->launches++;
    if (w->p.pbd_project) {
      // reading 27: the constraints of step n once more, directly on the advected positions
      // (K4 has already advanced the device step counter: step_off = -1)
      mc::PbdArgs pa;
      pa.f.X = X;
      pa.f.PA = w->ptr<float4>(w->L.PA);
      pa.f.PB = w->ptr<float4>(w->L.PB);
      pa.f.PC = w->ptr<float4>(w->L.PC);
      pa.f.PD = w->ptr<float2>(w->L.PD);
      pa.f.uni = reinterpret_cast<const float4*>(w->ptr<int>(w->L.flags) + 24);
      pa.f.F = nullptr; pa.f.sense = nullptr; pa.f.A = nullptr; pa.f.tex_A = 0; pa.f.csum = nullptr; pa.f.tile_fmax = nullptr;
      pa.f.N = N; pa.f.nx = nx; pa.f.ny = ny; pa.f.stride = w->stride; pa.f.n_windows = w->n_windows;
      pa.f.kappa = 1.0f;
      pa.f.step = stepp;
      pa.PE = w->has_L_act ? w->ptr<float>(w->L.PE) : nullptr;
      pa.O = nullptr;
      pa.Dp = w->ptr<float2>(w->L.Dp);
      pa.iters = w->p.pbd_iters;
      pa.order = w->p.pbd_order;
      pa.halo_lanes = w->halo_lanes;
      pa.step_off = -1;
      const int pgrid = (w->n_windows * 32 + 63) / 64;
      if (w->uniform_params) mc::k_filament_pbd<true><<<dim3(pgrid, nb), 64, 0, st>>>(pa, ws);
      else mc::k_filament_pbd<false><<<dim3(pgrid, nb), 64, 0, st>>>(pa, ws);
      mc::k_add_displacement<<<dim3((N + 1023) / 1024, nb), 1024, 0, st>>>(N, X, pa.Dp, flag, &ls_state->step_max_p, ws);
      w->launches += 2;
    }
    if (two) {
      // the markers follow the new positions (reading 28)
      mc::k_markers<<<dim3((N + 1023) / 1024, nb), 1024, 0, st>>>(N, X, w->ptr<unsigned char>(w->L.bflags), w->layer_h,
                                                                w->ptr<float2>(w->L.O), &ls_state->step_max_m, ws);
      w->launches++;
    }
  }
  prof_mark(w, 7);
  if (w->prof_on && w->prof_steps < PROF_MAX_STEPS) w->prof_steps++;
  w->step += 1;
  // launch-configuration errors of this step's kernels (execution errors surface at the next sync)
  const cudaError_t le = cudaPeekAtLastError();
  if (le != cudaSuccess) return fail(w, MC_ECUDA, std::string("mc_step: kernel launch: ") + cudaGetErrorString(le));
  return MC_OK;
}

}  // namespace

extern "C" {
#pragma GCC visibility push(default)

size_t mc_workspace_bytes(const mc_world_params* p) {
  Derived d;
  std::string why;
  if (!validate(p, &d, &why)) return 0;
  return make_layout(p, d).total;
}

const char* mc_last_error(const mc_world* w) { return w ? w->err.c_str() : g_create_error.c_str(); }

int64_t mc_launch_count(const mc_world* w) { return w ? w->launches : 0; }

void mc_destroy(mc_world* w) {
  if (!w) return;
  for (cudaEvent_t e : w->prof_ev) cudaEventDestroy(e);
  if (w->tex_u) cudaDestroyTextureObject(w->tex_u);
  if (w->tex_A) cudaDestroyTextureObject(w->tex_A);
  if (w->side) cudaStreamSynchronize(w->side);  // nothing of this world may still run on its second stream
  if (w->ev_fork) cudaEventDestroy(w->ev_fork);
  if (w->ev_join) cudaEventDestroy(w->ev_join);
  if (w->side) cudaStreamDestroy(w->side);
  drop_graphs(w);
  delete w;
}

int mc_profile_enable(mc_world* w, int32_t on) {
  if (!w) return MC_EINVAL;
  if (on && w->prof_ev.empty()) {
    w->prof_ev.resize((size_t)PROF_MAX_STEPS * (MC_PROF_SLOTS + 1));
    for (cudaEvent_t& e : w->prof_ev)
      if (cudaEventCreate(&e) != cudaSuccess) return fail(w, MC_ECUDA, "cudaEventCreate failed");
  }
  w->prof_on = on != 0;
  w->prof_steps = 0;
  return MC_OK;
}

int mc_profile_read(mc_world* w, float* ms, int32_t* steps) {
  if (!w || !ms) return MC_EINVAL;
  for (int k = 0; k < MC_PROF_SLOTS; ++k) ms[k] = 0.0f;
  if (steps) *steps = w->prof_steps;
  cudaError_t e = cudaStreamSynchronize(w->stream);
  if (e != cudaSuccess) return fail(w, MC_ECUDA, std::string("mc_profile_read: ") + cudaGetErrorString(e));
  for (int s = 0; s < w->prof_steps; ++s)
    for (int k = 0; k < MC_PROF_SLOTS; ++k) {
      float t = 0.0f;
      const size_t base = (size_t)s * (MC_PROF_SLOTS + 1);
      if (cudaEventElapsedTime(&t, w->prof_ev[base + k], w->prof_ev[base + k + 1]) == cudaSuccess) ms[k] += t;
    }
  w->prof_steps = 0;
  return MC_OK;
}

int mc_create(const mc_world_params* p, void* workspace, size_t workspace_bytes, void* cuda_stream,
              mc_world** out) {
  g_create_error.clear();
  if (!out) { g_create_error = "null out"; return MC_EINVAL; }
  *out = nullptr;
  Derived d;
  std::string why;
  if (!validate(p, &d, &why)) { g_create_error = why; return MC_EINVAL; }
  Layout L = make_layout(p, d);
  if (!workspace || workspace_bytes < L.total || ((uintptr_t)workspace % ALIGN) != 0) {
    g_create_error = "workspace missing, too small or not 256-byte aligned";
    return MC_EINVAL;
  }
  mc_world* w = new (std::nothrow) mc_world();
  if (!w) { g_create_error = "host allocation failed"; return MC_ENOMEM; }
  w->p = *p;
  for (int k = 0; k < 4; ++k) w->p.fields[k].sources = nullptr;  // never keep caller pointers
  w->d = d;
  w->L = L;
  w->ws = static_cast<char*>(workspace);
  w->stream = static_cast<cudaStream_t>(cuda_stream);
  w->nx = p->nx;
  w->ny = p->ny;
  w->nc = (size_t)p->nx * p->ny;
  // linear float2 texture views of the gathered fields (mc_common.cuh interp2_tex); a failure
  // (workspace not aligned to the texture alignment, field beyond the linear-texture limit)
  // leaves the handle 0 and the gathers on the plain path
  auto make_tex = [&](size_t off) -> cudaTextureObject_t {
    cudaResourceDesc rd;
    memset(&rd, 0, sizeof(rd));
    rd.resType = cudaResourceTypeLinear;
    rd.res.linear.devPtr = w->ws + off;
    rd.res.linear.desc = cudaCreateChannelDesc<float2>();
    rd.res.linear.sizeInBytes = w->nc * 8;
    cudaTextureDesc td;
    memset(&td, 0, sizeof(td));
    td.readMode = cudaReadModeElementType;
    cudaTextureObject_t t = 0;
    if (cudaCreateTextureObject(&t, &rd, &td, nullptr) != cudaSuccess) { cudaGetLastError(); t = 0; }
    return t;
  };
  w->tex_u = make_tex(L.u);
  if (d.n_density) w->tex_A = make_tex(L.A);
  else if (d.n_static) w->tex_A = make_tex(L.As);
  {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) == cudaSuccess &&
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0)
      w->n_sm = sms;
  }
  {
    // one-launch K0 for large worlds: a cooperative grid of resident 1024-thread CTAs
    int dev = 0, coop = 0, occ = 0;
    if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) == cudaSuccess && coop &&
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, mc::k_list_build_coop, 1024, 0) == cudaSuccess && occ > 0)
      w->coop_grid = w->n_sm * occ;
    else
      cudaGetLastError();
  }
  // lattice constants (reading 10, 12): nu_lat = nu dt; tau+ = 3 nu_lat + 1/2; tau- = Lambda/(tau+ - 1/2) + 1/2
  const double dt = (double)p->dt, nu_lat = (double)p->nu * dt;
  const double tau_p = 3.0 * nu_lat + 0.5, tau_m = (double)p->trt_lambda / (tau_p - 0.5) + 0.5;
  w->omega_p = (float)(1.0 / tau_p);
  w->omega_m = (float)(1.0 / tau_m);
  w->rho0 = p->rho0;
  w->kappa = (float)((double)p->k_el * dt * dt);
  w->layer_h = p->layer_offset > 0.0f ? p->layer_offset : 0.5f;
  w->halo_lanes = p->pbd_order == MC_PBD_JACOBI ? p->pbd_iters : (3 * p->pbd_iters + 1) / 2;

  cudaStream_t st = w->stream;
  cudaError_t e = cudaMemsetAsync(workspace, 0, L.total, st);  // fluid at rest: shifted populations = 0
  if (e != cudaSuccess) {
    g_create_error = std::string("cudaMemsetAsync: ") + cudaGetErrorString(e);
    delete w;
    return MC_ECUDA;
  }
  // fields
  size_t src_off = 0;
  int n_static_seen = 0;
  for (int k = 0; k < p->n_fields; ++k) {
    const mc_field_params& f = p->fields[k];
    const double lat = (double)f.coupling * dt * dt;
    if (f.kind == MC_FIELD_BEAD_DENSITY) {
      w->coef[k] = (float)(-lat);  // F_rep = -kappa_rep * grad(rho~)
      const int R = d.R[k];
      double g[2 * mc::BLUR_MAX_R + 1], Z = 0.0;
      for (int t = -R; t <= R; ++t) {
        g[t + R] = std::exp(-(double)(t * t) / (2.0 * (double)f.sigma * (double)f.sigma));
        Z += g[t + R];
      }
      for (int t = 0; t <= 2 * R; ++t) w->taps[k].g[t] = (float)(g[t] / Z);
    } else {
      w->coef[k] = (float)lat;  // F_chem = +kappa_chi * grad(c)
      w->static_slot[k] = n_static_seen;
      float* dsrc = w->ptr<float>(L.sources) + src_off;
      if (f.n_sources > 0) {
        e = cudaMemcpyAsync(dsrc, f.sources, 4 * (size_t)f.n_sources * sizeof(float), cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) {
          g_create_error = std::string("cudaMemcpyAsync(sources): ") + cudaGetErrorString(e);
          delete w;
          return MC_ECUDA;
        }
        cudaStreamSynchronize(st);  // the host array belongs to the caller
      }
      mc::k_static_init<<<dim3((w->nx + 127) / 128, w->ny), 128, 0, st>>>(
          w->nx, w->ny, f.n_sources, dsrc, w->coef[k], w->ptr<float>(L.cfield) + (size_t)n_static_seen * w->nc,
          w->ptr<float>(L.csum), w->ptr<float2>(L.As));
      w->launches++;
      src_off += 4 * (size_t)f.n_sources;
      n_static_seen++;
    }
  }
  e = cudaStreamSynchronize(st);
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e != cudaSuccess) {
    g_create_error = std::string("mc_create: ") + cudaGetErrorString(e);
    delete w;
    return MC_ECUDA;
  }
  *out = w;
  return MC_OK;
}

int mc_load_filaments(mc_world* w, int32_t n_fil, const int32_t* offsets, const float* xy, const float* L_rest,
                      const float* theta_rest, const float* k_bend, const float* k_shear,
                      const float* k_stretch, const float* act_amp, const float* act_phase,
                      const float* act_period) {
  if (!w) return MC_EINVAL;
  if (w->batch_member && !g_batch_call) return fail(w, MC_ESTATE, "world belongs to a batch: use mc_load_filaments_batch");
  if (n_fil < 0 || !offsets || offsets[0] != 0) return fail(w, MC_EINVAL, "bad offsets");
  for (int32_t f = 0; f < n_fil; ++f)
    if (offsets[f + 1] - offsets[f] < 3) return fail(w, MC_EINVAL, "chain shorter than 3 beads");
  const int64_t N = offsets[n_fil];
  if (N > w->p.max_beads) return fail(w, MC_EINVAL, "N > max_beads");
  if (N > 0 && (!xy || !L_rest || !theta_rest || !k_bend || !k_shear || !k_stretch || !act_amp || !act_phase ||
                !act_period))
    return fail(w, MC_EINVAL, "null array");
  cudaStream_t st = w->stream;
  CudaSeq cs{w, "mc_load_filaments"};  // every CUDA return code of this call; reported at the next sync
  const bool reuse_order = w->N == N && w->n_fil == n_fil && (int64_t)w->loaded_offsets.size() == n_fil + 1 &&
                           std::equal(w->loaded_offsets.begin(), w->loaded_offsets.end(), offsets);
  const int prev_stride = w->stride, prev_windows = w->n_windows;
  drop_graphs(w);
  w->N = 0;
  w->n_fil = 0;
  w->n_windows = 0;
  if (N == 0) return MC_OK;
  // 1. spatial sort of the CHAINS (not of the beads): chains whose first bead falls in the same
  //    64x64 block of nodes become neighbours in memory, so the per-bead grid gathers of K1/K4
  //    and the per-tile bead gathers of K2 hit L2 instead of re-fetching sectors from HBM.
  //    The internal order is a mechanism only: every output is returned in the caller's order.
  bool uniform = true;
  const int m0 = offsets[1] - offsets[0];
  int* bad = w->ptr<int>(w->L.flags) + 1;
  cs.ok(cudaMemsetAsync(bad, 0, 4, st), "cudaMemsetAsync");
  cudaError_t e = cudaSuccess;
  std::vector<int> src;                 // host staging of this call; must outlive the final sync
  std::vector<unsigned char> bflags;
  if (!reuse_order) {
  int* d_off = w->ptr<int>(w->L.scratch);
  int* d_keys = d_off + (n_fil + 1);
  std::vector<int> keys(n_fil);
  cs.ok(cudaMemcpyAsync(d_off, offsets, (size_t)(n_fil + 1) * 4, cudaMemcpyHostToDevice, st), "cudaMemcpyAsync");
  mc::k_chain_keys<<<(n_fil + 255) / 256, 256, 0, st>>>(n_fil, d_off, xy, w->nx, w->ny, 64, d_keys);
  cs.launched("k_chain_keys");
  w->launches++;
  cs.ok(cudaMemcpyAsync(keys.data(), d_keys, (size_t)n_fil * 4, cudaMemcpyDeviceToHost, st), "cudaMemcpyAsync");
  e = cudaStreamSynchronize(st);
  if (e == cudaSuccess) e = cudaGetLastError();
  if (cs.rc != MC_OK) return cs.rc;
  if (e != cudaSuccess) return fail(w, MC_ECUDA, std::string("mc_load_filaments: ") + cudaGetErrorString(e));
  std::vector<int> order(n_fil);
  std::iota(order.begin(), order.end(), 0);
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return keys[a] < keys[b]; });
  src.resize((size_t)N);
  bflags.assign((size_t)N, 0);
  size_t pos = 0;
  for (int c = 0; c < n_fil; ++c) {
    const int f = order[c];
    const int b0 = offsets[f], m = offsets[f + 1] - b0;
    uniform = uniform && (m == m0);
    for (int i = 0; i < m; ++i) {
      src[pos + i] = b0 + i;
      if (i & 1) bflags[pos + i] |= mc::BEAD_ODD;  // edge parity of the Gauss-Seidel pass
    }
    bflags[pos] |= mc::BEAD_FIRST;
    bflags[pos + m - 1] |= mc::BEAD_LAST;
    pos += m;
  }
  cs.ok(cudaMemcpyAsync(w->ptr<int>(w->L.src), src.data(), (size_t)N * 4, cudaMemcpyHostToDevice, st), "cudaMemcpyAsync");
  cs.ok(cudaMemcpyAsync(w->ptr<unsigned char>(w->L.bflags), bflags.data(), (size_t)N, cudaMemcpyHostToDevice, st), "cudaMemcpyAsync");
  }
  // 2. gather + pack the per-bead parameters in the internal order, validate
  mc::PackArgs pa;
  pa.N = (int)N;
  pa.src = w->ptr<int>(w->L.src);
  pa.flags = w->ptr<unsigned char>(w->L.bflags);
  pa.xy = xy; pa.L_rest = L_rest; pa.theta_rest = theta_rest; pa.k_bend = k_bend; pa.k_shear = k_shear;
  pa.k_stretch = k_stretch; pa.act_amp = act_amp; pa.act_phase = act_phase; pa.act_period = act_period;
  pa.X = w->ptr<float2>(w->L.X);
  pa.PA = w->ptr<float4>(w->L.PA);
  pa.PB = w->ptr<float4>(w->L.PB);
  pa.PC = w->ptr<float4>(w->L.PC);
  pa.PD = w->ptr<float2>(w->L.PD);
  pa.uni = reinterpret_cast<float4*>(w->ptr<int>(w->L.flags) + 24);
  pa.nonuniform = w->ptr<int>(w->L.flags) + 3;
  cs.ok(cudaMemsetAsync(pa.nonuniform, 0, 4, st), "cudaMemsetAsync");
  pa.dt = (double)w->p.dt;
  pa.bad = bad;
  mc::k_pack_params<<<(int)((N + 255) / 256), 256, 0, st>>>(pa);
  cs.launched("k_pack_params");
  w->launches++;
  cs.ok(cudaMemsetAsync(w->ptr<float>(w->L.F), 0, (size_t)N * 8, st), "cudaMemsetAsync");
  cs.ok(cudaMemsetAsync(w->ptr<float>(w->L.sense), 0, (size_t)N * 4, st), "cudaMemsetAsync");
  // largest tile list of the loaded configuration -> CTA size of the deposit kernel
  int* maxlist = w->ptr<int>(w->L.flags) + 2;
  {
    const int n_tiles = (w->nx / mc::TS) * (w->ny / mc::TS);
    int* tile_count = w->ptr<int>(w->L.tile_count);
    cs.ok(cudaMemsetAsync(maxlist, 0, 4, st), "cudaMemsetAsync");
    // force the next step to rebuild the lists (drift = +inf), and count once now with need = 1
    mc::ListState force;
    force.need = 1;
    force.drift = INFINITY;
    force.step_max = force.step_max_p = force.step_max_m = 0u;
    mc::ListState* ls_state = reinterpret_cast<mc::ListState*>(w->ptr<int>(w->L.flags) + 16);
    cs.ok(cudaMemcpyAsync(ls_state, &force, sizeof(force), cudaMemcpyHostToDevice, st), "cudaMemcpyAsync");
    const float2* Omark = nullptr;
    if (w->p.two_layer) {
      // markers of the loaded positions (reading 28); the offsets start from zero
      cs.ok(cudaMemsetAsync(w->ptr<float2>(w->L.O), 0, (size_t)N * 8, st), "cudaMemsetAsync");
      mc::k_markers<<<(int)((N + 1023) / 1024), 1024, 0, st>>>((int)N, w->ptr<float2>(w->L.X), w->ptr<unsigned char>(w->L.bflags),
                                                            w->layer_h, w->ptr<float2>(w->L.O), &ls_state->step_max_m, 0);
      cs.launched("k_markers");
      w->launches++;
      Omark = w->ptr<float2>(w->L.O);
    }
    const int64_t n_items = w->p.two_layer ? 2 * N : N;
    mc::k_tile_bin<false><<<(int)((n_items + 255) / 256), 256, 0, st>>>(ls_state, w->ptr<float2>(w->L.X), Omark, (int)N,
                                                                        w->nx, w->ny, tile_count, nullptr, nullptr, 0);
    cs.launched("k_tile_bin");
    mc::k_max_int<<<64, 256, 0, st>>>(tile_count, n_tiles, maxlist);
    cs.launched("k_max_int");
    cs.ok(cudaMemsetAsync(tile_count, 0, (size_t)n_tiles * 4, st), "cudaMemsetAsync");
    w->launches += 2;
  }
  int h_maxlist = 0;
  cs.ok(cudaMemcpyAsync(&h_maxlist, maxlist, 4, cudaMemcpyDeviceToHost, st), "cudaMemcpyAsync");
  const long long host_step = w->step;  // steps without beads do not advance the device copy
  cs.ok(cudaMemcpyAsync(w->ptr<long long>(w->L.flags) + 4, &host_step, 8, cudaMemcpyHostToDevice, st), "cudaMemcpyAsync");
  int h = 0, h_nonuni = 0;
  cs.ok(cudaMemcpyAsync(&h, bad, 4, cudaMemcpyDeviceToHost, st), "cudaMemcpyAsync");
  cs.ok(cudaMemcpyAsync(&h_nonuni, w->ptr<int>(w->L.flags) + 3, 4, cudaMemcpyDeviceToHost, st), "cudaMemcpyAsync");
  e = cudaStreamSynchronize(st);  // src/bflags are host vectors of this call
  if (e == cudaSuccess) e = cudaGetLastError();
  if (cs.rc != MC_OK) { w->loaded_offsets.clear(); return cs.rc; }
  if (e != cudaSuccess) return fail(w, MC_ECUDA, std::string("mc_load_filaments: ") + cudaGetErrorString(e));
  if (h) {
    w->loaded_offsets.clear();
    return fail(w, MC_EINVAL, (h & 1) ? "stiffness outside [0,1]" : "period <= 0");
  }
  w->N = (int)N;
  w->n_fil = n_fil;
  w->has_L_act = false;  // a load resets the rest-length actuation (mc_set_length_actuation)
  // (two-layer lists hold two markers per bead: twice as long for the same crowding)
  w->deposit_threads = h_maxlist > (w->p.two_layer ? 4096 : 1024) ? 256 : 128;
  // crowded tiles (config 5 lists ~16,000 beads in its central tiles): a cluster of CTAs per tile
  // (measured on config 5: one CTA per tile 0.351 ms/step, clusters of 2: 0.263, 4: 0.250, 8: 0.325)
  w->cluster_auto = h_maxlist > 4096 ? 4 : 0;
  w->cluster = w->cluster_user >= 0 ? w->cluster_user : w->cluster_auto;
  if (w->cluster > 0 && w->split_on) ensure_side_stream(w);  // no side stream: one cluster launch over all tiles
  w->uniform_params = (h_nonuni == 0);
  if (reuse_order) {
    w->stride = prev_stride;
    w->n_windows = prev_windows;
  } else {
    // K1 windows (k_filament.cuh, k_pbd.cuh): aligned to chain starts when every chain has the same
    // length dividing 64, else overlapping by halo_lanes lanes on either side
    const bool aligned = uniform && (64 % m0 == 0);
    w->stride = aligned ? 64 : 64 - 4 * w->halo_lanes;
    w->n_windows = (int)((N + w->stride - 1) / w->stride);
    w->loaded_offsets.assign(offsets, offsets + n_fil + 1);
  }
  return MC_OK;
}

int mc_set_positions(mc_world* w, const float* xy) {
  if (!w) return MC_EINVAL;
  if (w->N == 0) return MC_OK;
  if (!xy) return fail(w, MC_EINVAL, "null array");
  cudaStream_t st = w->stream;
  mc::k_permute2<<<(w->N + 255) / 256, 256, 0, st>>>(w->N, w->ptr<int>(w->L.src), reinterpret_cast<const float2*>(xy),
                                                     w->ptr<float2>(w->L.X));
  w->launches++;
  // the beads may be anywhere now: the next step rebuilds the tile lists (drift = +inf)
  mc::ListState force;
  force.need = 1;
  force.drift = INFINITY;
  force.step_max = force.step_max_p = force.step_max_m = 0u;
  mc::ListState* ls_state = reinterpret_cast<mc::ListState*>(w->ptr<int>(w->L.flags) + 16);
  cudaMemcpyAsync(ls_state, &force, sizeof(force), cudaMemcpyHostToDevice, st);
  if (w->p.two_layer) {
    mc::k_markers<<<(w->N + 1023) / 1024, 1024, 0, st>>>(w->N, w->ptr<float2>(w->L.X), w->ptr<unsigned char>(w->L.bflags), w->layer_h,
                                                      w->ptr<float2>(w->L.O), &ls_state->step_max_m, 0);
    w->launches++;
  }
  cudaError_t e = cudaStreamSynchronize(st);  // `force` is a host variable of this call; xy belongs to the caller
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e != cudaSuccess) return fail(w, MC_ECUDA, std::string("mc_set_positions: ") + cudaGetErrorString(e));
  return MC_OK;
}

int mc_step(mc_world* w, int32_t n) {
  if (!w) return MC_EINVAL;
  if (w->batch_member && !g_batch_call) return fail(w, MC_ESTATE, "world belongs to a batch: use mc_step_batch");
  if (n < 0) return fail(w, MC_EINVAL, "n < 0");
  if (w->diverged) return fail(w, MC_EDIVERGED, "world diverged (non-finite bead or |u| > 0.3)");
  int32_t done = 0;
  while (done < n) {
    // Blocks of GRAPH_STEPS steps replay a captured CUDA
    // graph (same kernels, same order, same arguments: results are bit-identical to direct
    // launches); small worlds are bound by launch overhead, not by the kernels.
    if (!w->prof_on && !w->graph_off && n - done >= GRAPH_STEPS) {
      const int ph = w->cur;
      if (!w->graph[ph]) {
        cudaGraph_t g = nullptr;
        // host-side state a capture advances: restored if the capture does not yield a graph
        const int64_t l0 = w->launches, step0 = w->step;
        const int cur0 = w->cur;
        if (w->stream == nullptr ||
            cudaStreamBeginCapture(w->stream, cudaStreamCaptureModeRelaxed) != cudaSuccess) {
          cudaGetLastError();  // not an error of the world: this stream just cannot be captured
          w->graph_off = true;
          continue;
        }
        int crc = MC_OK;
        for (int s = 0; s < GRAPH_STEPS && crc == MC_OK; ++s) crc = enqueue_step(w);  // advances the host-side state
        cudaError_t e = cudaStreamEndCapture(w->stream, &g);
        if (e == cudaSuccess && crc == MC_OK) e = cudaGraphInstantiate(&w->graph[ph], g, 0);
        if (g) cudaGraphDestroy(g);
        if (e != cudaSuccess || crc != MC_OK) {
          // nothing was enqueued (a capture records, it does not run): put the host counters back
          // and launch these steps directly from now on
          cudaGetLastError();
          if (w->graph[ph]) { cudaGraphExecDestroy(w->graph[ph]); w->graph[ph] = nullptr; }
          w->launches = l0;
          w->step = step0;
          w->cur = cur0;
          w->graph_off = true;
          continue;
        }
        w->graph_launches[ph] = w->launches - l0;
      } else {
        w->step += GRAPH_STEPS;  // cur returns to its value after GRAPH_STEPS steps
        w->launches += w->graph_launches[ph];
      }
      if (cudaGraphLaunch(w->graph[ph], w->stream) != cudaSuccess) {
        // the steps of this block were counted but not enqueued
        w->step -= GRAPH_STEPS;
        w->launches -= w->graph_launches[ph];
        return fail(w, MC_ECUDA, "cudaGraphLaunch failed");
      }
      done += GRAPH_STEPS;
      continue;
    }
    int rc = enqueue_step(w);
    if (rc != MC_OK) return rc;
    ++done;
  }
  return check_cuda(w, "mc_step");
}

int mc_read_state(mc_world* w, int64_t* step_out, float* xy, float* u, float* rho, float* fdev, float* field,
                  float* force, float* sense) {
  if (!w) return MC_EINVAL;
  cudaStream_t st = w->stream;
  const size_t nc = w->nc, N = (size_t)w->N;
  if (step_out) *step_out = w->step;
  const cudaMemcpyKind d2d = cudaMemcpyDeviceToDevice;
  const int* src = w->ptr<int>(w->L.src);
  const int pg = (int)((N + 255) / 256);
  if (xy && N) {
    mc::k_unpermute2<<<pg, 256, 0, st>>>((int)N, src, w->ptr<float2>(w->L.X), reinterpret_cast<float2*>(xy));
    w->launches++;
  }
  if (u) {
    {
      const int bx = pick_bx(w->nx);
      mc::k_split2<<<dim3(w->nx / bx, w->ny), bx, 0, st>>>(w->nx, w->ny, w->ptr<float2>(w->L.u), u, u + nc);
    }
    w->launches++;
  }
  if (rho || fdev) {
    const int bx = pick_bx(w->nx);
    mc::k_lbm_export<<<dim3(w->nx / bx, w->ny), bx, 0, st>>>(w->fbuf(w->cur), w->nx, w->ny, w->rho0, fdev, rho);
    w->launches++;
  }
  if (field) {
    bool first = true;
    for (int k = 0; k < w->p.n_fields; ++k) {
      float* dst = field + (size_t)k * nc;
      if (w->p.fields[k].kind == MC_FIELD_BEAD_DENSITY) {
        // recompute the filtered density from the stored rho_b (A is rebuilt by every step anyway)
        launch_blur(w, k, first, dst);
        first = false;
      } else {
        cudaMemcpyAsync(dst, w->ptr<float>(w->L.cfield) + (size_t)w->static_slot[k] * nc, nc * 4, d2d, st);
      }
    }
  }
  if (force && N) {
    mc::k_unpermute2<<<pg, 256, 0, st>>>((int)N, src, w->ptr<float2>(w->L.F), reinterpret_cast<float2*>(force));
    w->launches++;
  }
  if (sense && N) {
    mc::k_unpermute1<<<pg, 256, 0, st>>>((int)N, src, w->ptr<float>(w->L.sense), sense);
    w->launches++;
  }
  int h = 0;
  cudaMemcpyAsync(&h, w->ptr<int>(w->L.flags), 4, cudaMemcpyDeviceToHost, st);
  cudaError_t e = cudaStreamSynchronize(st);
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e != cudaSuccess) return fail(w, MC_ECUDA, std::string("mc_read_state: ") + cudaGetErrorString(e));
  if (h) {
    w->diverged = true;
    return fail(w, MC_EDIVERGED, "world diverged (non-finite bead or |u| > 0.3)");
  }
  return MC_OK;
}

int mc_set_length_actuation(mc_world* w, const float* act_L_amp) {
  if (!w) return MC_EINVAL;
  if (w->batch_member && !g_batch_call) return fail(w, MC_ESTATE, "world belongs to a batch");
  const bool was = w->has_L_act;
  if (!act_L_amp || w->N == 0) {
    w->has_L_act = false;
  } else {
    cudaStream_t st = w->stream;
    int* nz = w->ptr<int>(w->L.flags) + 5;
    int h = 0;
    CudaSeq cs{w, "mc_set_length_actuation"};
    cs.ok(cudaMemsetAsync(nz, 0, 4, st), "cudaMemsetAsync");
    mc::k_permute1<<<(w->N + 255) / 256, 256, 0, st>>>(w->N, w->ptr<int>(w->L.src), act_L_amp, w->ptr<float>(w->L.PE), nz);
    cs.launched("k_permute1");
    w->launches++;
    cs.ok(cudaMemcpyAsync(&h, nz, 4, cudaMemcpyDeviceToHost, st), "cudaMemcpyAsync");
    cudaError_t e = cudaStreamSynchronize(st);  // the array belongs to the caller
    if (e == cudaSuccess) e = cudaGetLastError();
    if (cs.rc != MC_OK) return cs.rc;
    if (e != cudaSuccess) return fail(w, MC_ECUDA, std::string("mc_set_length_actuation: ") + cudaGetErrorString(e));
    w->has_L_act = h != 0;  // all-zero amplitudes keep the fast kernel
  }
  if (was != w->has_L_act) drop_graphs(w);
  return MC_OK;
}

int mc_load_fluid(mc_world* w, int64_t step, const float* fdev) {
  if (!w) return MC_EINVAL;
  if (w->batch_member && !g_batch_call) return fail(w, MC_ESTATE, "world belongs to a batch");
  if (step < 0) return fail(w, MC_EINVAL, "step < 0");
  cudaStream_t st = w->stream;
  CudaSeq cs{w, "mc_load_fluid"};
  if (fdev) {
    const int bx = pick_bx(w->nx);
    mc::k_lbm_import<<<dim3(w->nx / bx, w->ny), bx, 0, st>>>(fdev, w->nx, w->ny, w->fbuf(w->cur));
    cs.launched("k_lbm_import");
    w->launches++;
  }
  w->step = step;
  const long long host_step = step;
  cs.ok(cudaMemcpyAsync(w->ptr<long long>(w->L.flags) + 4, &host_step, 8, cudaMemcpyHostToDevice, st), "cudaMemcpyAsync");
  w->diverged = false;
  cs.ok(cudaMemsetAsync(w->ptr<int>(w->L.flags), 0, 4, st), "cudaMemsetAsync");  // a loaded state starts with a clear flag
  cudaError_t e = cudaStreamSynchronize(st);  // fdev belongs to the caller, host_step to this frame
  if (e == cudaSuccess) e = cudaGetLastError();
  if (cs.rc != MC_OK) return cs.rc;
  if (e != cudaSuccess) return fail(w, MC_ECUDA, std::string("mc_load_fluid: ") + cudaGetErrorString(e));
  return MC_OK;
}

int mc_keep_intermediates(mc_world* w, int32_t on) {
  if (!w) return MC_EINVAL;
  if (w->keep_G != (on != 0)) drop_graphs(w);
  w->keep_G = on != 0;
  return MC_OK;
}

int mc_cluster_tiles(mc_world* w, int32_t c) {
  if (!w) return MC_EINVAL;
  bool split_on = true;
  if (c >= 0 && (c & MC_CLUSTER_ALL_TILES)) { split_on = false; c &= ~MC_CLUSTER_ALL_TILES; }
  if (c != -1 && c != 0 && c != 2 && c != 4 && c != 8) return fail(w, MC_EINVAL, "cluster size must be -1, 0, 2, 4 or 8");
  const int now = c >= 0 ? c : w->cluster_auto;
  const bool changed = now != w->cluster || split_on != w->split_on;
  if (changed) drop_graphs(w);
  w->cluster_user = c;
  w->cluster = now;
  w->split_on = split_on;
  if (now > 0 && split_on) ensure_side_stream(w);
  if (changed && w->N > 0) {
    // the crowded-tile table is written by the list rebuild of a step that runs the split launch:
    // make the next step rebuild, so that a table from before the switch is never used
    mc::ListState force;
    force.need = 1;
    force.drift = INFINITY;
    force.step_max = force.step_max_p = force.step_max_m = 0u;
    cudaError_t e = cudaMemcpyAsync(reinterpret_cast<mc::ListState*>(w->ptr<int>(w->L.flags) + 16), &force, sizeof(force),
                                    cudaMemcpyHostToDevice, w->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(w->stream);  // `force` is a host variable of this call
    if (e != cudaSuccess) return fail(w, MC_ECUDA, std::string("mc_cluster_tiles: ") + cudaGetErrorString(e));
  }
  return now;
}

int mc_texture_gathers(mc_world* w, int32_t on) {
  if (!w) return MC_EINVAL;
  if (w->tex_on != (on != 0)) drop_graphs(w);
  w->tex_on = on != 0;
  return (w->tex_on && w->tex_u) ? 1 : 0;
}

int mc_read_intermediates(mc_world* w, float* rho_b, float* G) {
  if (!w) return MC_EINVAL;
  if (G && !w->keep_G) return fail(w, MC_ESTATE, "G is only stored after mc_keep_intermediates(w, 1)");
  cudaStream_t st = w->stream;
  const size_t nc = w->nc;
  if (rho_b) cudaMemcpyAsync(rho_b, w->ptr<float>(w->L.rho_b), nc * 4, cudaMemcpyDeviceToDevice, st);
  if (G) cudaMemcpyAsync(G, w->ptr<float>(w->L.G), 2 * nc * 4, cudaMemcpyDeviceToDevice, st);
  cudaError_t e = cudaStreamSynchronize(st);
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e != cudaSuccess) return fail(w, MC_ECUDA, std::string("mc_read_intermediates: ") + cudaGetErrorString(e));
  return MC_OK;
}

// ---------------------------------------------------------------------------------------------
// Batched worlds: the paper's real workload is a POPULATION of small worlds
// stepped in lock-step ("large populations of interacting filaments over evolutionary
// timescales"; NEAT / MAP-Elites populations P:L173-179; 256 x 256 grids P:L190).  A batch is n
// worlds of identical parameters and chain structure (different positions and per-bead parameters)
// in one workspace, world k at k * mc_workspace_bytes(p).  Every kernel of the step is launched
// ONCE for the whole batch (world index in blockIdx.y / .z, mc_common.cuh wshift): a world of a
// batch runs exactly the code and the arithmetic of the same world stepped alone, bit for bit.
struct mc_batch {
  std::vector<mc_world*> worlds;
  size_t stride = 0;
  bool consistent = true;  // false after a batch load that failed part-way: the worlds differ until the next good load
  std::string err;
};

namespace {
struct BatchScope {
  BatchScope() { g_batch_call = true; }
  ~BatchScope() { g_batch_call = false; }
};
thread_local std::string g_batch_create_error;
int bfail(mc_batch* b, int code, const std::string& msg) {
  if (b) b->err = msg;
  return code;
}
}  // namespace

size_t mc_batch_workspace_bytes(const mc_world_params* p, int32_t n_worlds) {
  const size_t one = mc_workspace_bytes(p);
  if (one == 0 || n_worlds < 1 || n_worlds > 65535) return 0;
  return one * (size_t)n_worlds;
}

const char* mc_batch_last_error(const mc_batch* b) { return b ? b->err.c_str() : g_batch_create_error.c_str(); }

void mc_destroy_batch(mc_batch* b) {
  if (!b) return;
  for (mc_world* w : b->worlds) mc_destroy(w);
  delete b;
}

int mc_create_batch(const mc_world_params* p, int32_t n_worlds, void* workspace, size_t workspace_bytes,
                    void* cuda_stream, mc_batch** out) {
  g_batch_create_error.clear();
  if (!out) { g_batch_create_error = "null out"; return MC_EINVAL; }
  *out = nullptr;
  const size_t one = mc_workspace_bytes(p);
  if (one == 0) { g_batch_create_error = "invalid world parameters"; return MC_EINVAL; }
  if (n_worlds < 1 || n_worlds > 65535) { g_batch_create_error = "n_worlds must be 1..65535"; return MC_EINVAL; }
  if (!workspace || workspace_bytes < one * (size_t)n_worlds) { g_batch_create_error = "workspace missing or too small"; return MC_EINVAL; }
  mc_batch* b = new (std::nothrow) mc_batch();
  if (!b) { g_batch_create_error = "host allocation failed"; return MC_ENOMEM; }
  b->stride = one;
  for (int32_t k = 0; k < n_worlds; ++k) {
    mc_world* w = nullptr;
    const int rc = mc_create(p, static_cast<char*>(workspace) + (size_t)k * one, one, cuda_stream, &w);
    if (rc != MC_OK) {
      g_batch_create_error = std::string("world ") + std::to_string(k) + ": " + mc_last_error(nullptr);
      mc_destroy_batch(b);
      return rc;
    }
    w->batch_member = true;
    b->worlds.push_back(w);
  }
  *out = b;
  return MC_OK;
}

mc_world* mc_batch_world(mc_batch* b, int32_t k) {
  return (b && k >= 0 && k < (int32_t)b->worlds.size()) ? b->worlds[(size_t)k] : nullptr;
}

int mc_load_filaments_batch(mc_batch* b, int32_t n_fil, const int32_t* offsets, const float* xy, const float* L_rest,
                            const float* theta_rest, const float* k_bend, const float* k_shear, const float* k_stretch,
                            const float* act_amp, const float* act_phase, const float* act_period,
                            const float* act_L_amp) {
  if (!b) return MC_EINVAL;
  if (n_fil < 0 || !offsets || offsets[0] != 0) return bfail(b, MC_EINVAL, "bad offsets");
  const size_t N = (size_t)offsets[n_fil];
  BatchScope scope;
  mc_world* lead = b->worlds[0];
  lead->batch_n = 1;  // member calls below act on one world each
  b->consistent = false;
  bool uniform_all = true, any_L = false;
  int dep = 128, cl = 0;
  for (size_t k = 0; k < b->worlds.size(); ++k) {
    mc_world* w = b->worlds[k];
    const size_t o = k * N;
    int rc = mc_load_filaments(w, n_fil, offsets, xy + 2 * o, L_rest + o, theta_rest + o, k_bend + o, k_shear + o,
                               k_stretch + o, act_amp + o, act_phase + o, act_period + o);
    if (rc == MC_OK && act_L_amp) rc = mc_set_length_actuation(w, act_L_amp + o);
    if (rc != MC_OK) return bfail(b, rc, std::string("world ") + std::to_string(k) + ": " + w->err);
    uniform_all = uniform_all && w->uniform_params;
    any_L = any_L || w->has_L_act;
    dep = std::max(dep, w->deposit_threads);
    cl = std::max(cl, w->cluster_auto);
  }
  // one launch configuration for the whole batch.  Each choice is bit-neutral (tested): the general
  // K1 parameter path, wider deposit CTAs and tile clusters compute what the specialised ones do.
  for (mc_world* w : b->worlds) {
    w->uniform_params = uniform_all;
    w->has_L_act = any_L;
    w->deposit_threads = dep;
    w->cluster_auto = cl;
    w->cluster = w->cluster_user >= 0 ? w->cluster_user : cl;
  }
  if (lead->cluster > 0 && lead->split_on) ensure_side_stream(lead);
  drop_graphs(lead);
  b->consistent = true;
  return MC_OK;
}

int mc_set_positions_batch(mc_batch* b, const float* xy) {
  if (!b) return MC_EINVAL;
  mc_world* lead = b->worlds[0];
  if (lead->N == 0) return MC_OK;
  if (!xy) return bfail(b, MC_EINVAL, "null array");
  static_assert(sizeof(mc::ListStateWords) == sizeof(mc::ListState), "ListState twin");
  cudaStream_t st = lead->stream;
  const unsigned nb = (unsigned)b->worlds.size();
  mc::k_permute2<<<dim3((lead->N + 255) / 256, nb), 256, 0, st>>>(lead->N, lead->ptr<int>(lead->L.src),
                                                                  reinterpret_cast<const float2*>(xy),
                                                                  lead->ptr<float2>(lead->L.X), b->stride);
  mc::k_force_rebuild<<<nb, 32, 0, st>>>(reinterpret_cast<mc::ListStateWords*>(lead->ptr<int>(lead->L.flags) + 16), b->stride);
  lead->launches += 2;
  if (lead->p.two_layer) {
    mc::ListState* ls_state = reinterpret_cast<mc::ListState*>(lead->ptr<int>(lead->L.flags) + 16);
    mc::k_markers<<<dim3((lead->N + 1023) / 1024, nb), 1024, 0, st>>>(lead->N, lead->ptr<float2>(lead->L.X), lead->ptr<unsigned char>(lead->L.bflags),
                                                                   lead->layer_h, lead->ptr<float2>(lead->L.O),
                                                                   &ls_state->step_max_m, b->stride);
    lead->launches++;
  }
  cudaError_t e = cudaStreamSynchronize(st);  // xy belongs to the caller
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e != cudaSuccess) return bfail(b, MC_ECUDA, std::string("mc_set_positions_batch: ") + cudaGetErrorString(e));
  return MC_OK;
}

int mc_read_positions_batch(mc_batch* b, int64_t* step_out, float* xy) {
  if (!b) return MC_EINVAL;
  mc_world* lead = b->worlds[0];
  if (step_out) *step_out = lead->step;
  cudaStream_t st = lead->stream;
  const unsigned nb = (unsigned)b->worlds.size();
  if (xy && lead->N) {
    mc::k_unpermute2<<<dim3((lead->N + 255) / 256, nb), 256, 0, st>>>(lead->N, lead->ptr<int>(lead->L.src),
                                                                      lead->ptr<float2>(lead->L.X),
                                                                      reinterpret_cast<float2*>(xy), b->stride);
    lead->launches++;
  }
  // sticky divergence flags of all worlds (word 0 of each world's flag block)
  std::vector<int> h(nb, 0);
  cudaError_t e = cudaMemcpy2DAsync(h.data(), sizeof(int), lead->ptr<int>(lead->L.flags), b->stride, sizeof(int), nb,
                                    cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e != cudaSuccess) return bfail(b, MC_ECUDA, std::string("mc_read_positions_batch: ") + cudaGetErrorString(e));
  for (unsigned k = 0; k < nb; ++k)
    if (h[k]) {
      b->worlds[k]->diverged = true;
      return bfail(b, MC_EDIVERGED, std::string("world ") + std::to_string(k) + " diverged (non-finite bead or |u| > 0.3)");
    }
  return MC_OK;
}

int mc_step_batch(mc_batch* b, int32_t n) {
  if (!b) return MC_EINVAL;
  if (n < 0) return bfail(b, MC_EINVAL, "n < 0");
  if (!b->consistent) return bfail(b, MC_ESTATE, "the last mc_load_filaments_batch failed part-way: load the batch again");
  BatchScope scope;
  mc_world* lead = b->worlds[0];
  for (mc_world* w : b->worlds)
    if (w->diverged) return bfail(b, MC_EDIVERGED, "a world of the batch diverged");
  lead->batch_n = (int)b->worlds.size();
  lead->batch_stride = b->stride;
  const int rc = mc_step(lead, n);
  lead->batch_n = 1;  // read-outs of the leader address one world
  for (mc_world* w : b->worlds) {
    w->step = lead->step;
    w->cur = lead->cur;
  }
  if (rc != MC_OK) return bfail(b, rc, lead->err);
  return MC_OK;
}

#pragma GCC visibility pop
}  // extern "C"

// ---------------------------------------------------------------------------------------------
// mc_deposit_noalloc: S2 (rho_b = sum_i delta_h(g - X_i)) for callers that cannot allocate --
// code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  Everything
// else in this library works inside a caller-provided workspace; this ONE entry point needs none:
// the scratch of the tile binning (counters, offsets, bucket cursors, the lists) and of the deposit
// (per-tile maxima) lives in the file-scope device array below, of a fixed modest size that every GPU
// which loads the library holds until the process exits.  The kernels are the ones of the step
// (k_list_build_small, k_deposit_tile): same arithmetic, same fixed-point accumulation.
//
// In HOST code the array's name is a host-side stand-in, not a device address: its device address is
// resolved once per device with cudaGetSymbolAddress (below) and passed to the kernels.
// All calls share the array and it keeps the last call's contents: every call first clears what must
// start at zero (k_noalloc_init).  Calls that overlap on the GPU (two streams, two host threads) RACE
// on it: serialise them on one stream or with events.
namespace {

constexpr int NA_MAX_BEADS = MC_NOALLOC_MAX_BEADS, NA_MAX_TILES = MC_NOALLOC_MAX_TILES;
static_assert(NA_MAX_BEADS <= K0_SMALL_BEADS && NA_MAX_TILES <= K0_SMALL_TILES, "the one-CTA list build serves these sizes");
// layout of the scratch, in 4-byte words
constexpr size_t NA_STATE = 0;                                   // ListState (5 words), padded to 64
constexpr size_t NA_TILE_COUNT = 64;                             // [NA_MAX_TILES]
constexpr size_t NA_TILE_START = NA_TILE_COUNT + NA_MAX_TILES;   // [NA_MAX_TILES + 1], padded to + 64
constexpr size_t NA_BUCKET_COUNT = NA_TILE_START + NA_MAX_TILES + 64;   // [32 NA_MAX_TILES]
constexpr size_t NA_BUCKET_CURSOR = NA_BUCKET_COUNT + 32 * (size_t)NA_MAX_TILES;
constexpr size_t NA_RHO_MAX = NA_BUCKET_CURSOR + 32 * (size_t)NA_MAX_TILES;   // [NA_MAX_TILES] float
constexpr size_t NA_FMAX = NA_RHO_MAX + NA_MAX_TILES;            // [NA_MAX_TILES] unsigned
constexpr size_t NA_LIST = NA_FMAX + NA_MAX_TILES;               // [4 NA_MAX_BEADS]: a bead is listed in at most 4 tiles
constexpr size_t NA_WORDS = NA_LIST + 4 * (size_t)NA_MAX_BEADS;  // 200,832 words = 803,328 bytes

static __device__ __align__(256) int g_noalloc_scratch[NA_WORDS];

// clear what must start at zero and order a list build (drift = +inf => need = 1)
__global__ void k_noalloc_init(int* __restrict__ scratch, int n_tiles) {
  mc::ListState* st = reinterpret_cast<mc::ListState*>(scratch + NA_STATE);
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    st->need = 1;
    st->drift = __int_as_float(0x7f800000);
    st->step_max = st->step_max_p = st->step_max_m = 0u;
  }
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < 32 * n_tiles; i += gridDim.x * blockDim.x) {
    scratch[NA_BUCKET_COUNT + i] = 0;
    if (i < n_tiles) {
      scratch[NA_TILE_COUNT + i] = 0;
      scratch[NA_RHO_MAX + i] = 0;   // bits of 0.0f
      scratch[NA_FMAX + i] = 0;
    }
  }
}

thread_local std::string g_noalloc_error;
constexpr int NA_MAX_DEVICES = 64;
int* g_noalloc_ptr[NA_MAX_DEVICES] = {};   // device address of the scratch, per device (0: not resolved yet)
std::mutex g_noalloc_mutex;

int na_fail(int code, const std::string& msg) {
  g_noalloc_error = msg;
  return code;
}

}  // namespace

extern "C" {
#pragma GCC visibility push(default)

const char* mc_noalloc_last_error(void) { return g_noalloc_error.c_str(); }

int mc_deposit_noalloc(int32_t nx, int32_t ny, int32_t n_beads, const float* xy, float* rho_b, void* cuda_stream) {
  g_noalloc_error.clear();
  if (nx < 32 || ny < 32 || nx % 32 || ny % 32) return na_fail(MC_EINVAL, "nx, ny must be multiples of 32, >= 32");
  const long long n_tiles_ll = (long long)(nx / mc::TS) * (ny / mc::TS);
  if (n_tiles_ll > NA_MAX_TILES)
    return na_fail(MC_EINVAL, "grid too large for mc_deposit_noalloc: " + std::to_string(n_tiles_ll) + " tiles of 32 x 32 nodes, the static scratch holds " +
                                  std::to_string(NA_MAX_TILES) + " (MC_NOALLOC_MAX_TILES)");
  if (n_beads < 0) return na_fail(MC_EINVAL, "n_beads < 0");
  if (n_beads > NA_MAX_BEADS)
    return na_fail(MC_EINVAL, "too many beads for mc_deposit_noalloc: " + std::to_string(n_beads) + ", the static scratch holds " +
                                  std::to_string(NA_MAX_BEADS) + " (MC_NOALLOC_MAX_BEADS)");
  if (!rho_b || (n_beads > 0 && !xy)) return na_fail(MC_EINVAL, "null array");
  if (((uintptr_t)xy % 8) != 0 || ((uintptr_t)rho_b % 16) != 0) return na_fail(MC_EINVAL, "xy must be 8-byte and rho_b 16-byte aligned");
  const int n_tiles = (int)n_tiles_ll;
  // set-up, once per device, with that device current: the device address of the scratch
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return na_fail(MC_ECUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
  if (dev < 0 || dev >= NA_MAX_DEVICES) return na_fail(MC_EINVAL, "device index out of range");
  int* scratch = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[dev]) {
      void* ptr = nullptr;
      e = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);
      if (e != cudaSuccess || !ptr) {
        cudaGetLastError();
        return na_fail(MC_ECUDA, std::string("cudaGetSymbolAddress(g_noalloc_scratch): ") + cudaGetErrorString(e));
      }
      g_noalloc_ptr[dev] = static_cast<int*>(ptr);
    }
    scratch = g_noalloc_ptr[dev];
  }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  mc::ListState* ls_state = reinterpret_cast<mc::ListState*>(scratch + NA_STATE);
  int* tile_count = scratch + NA_TILE_COUNT;
  int* tile_start = scratch + NA_TILE_START;
  int* bucket_count = scratch + NA_BUCKET_COUNT;
  int* bucket_cursor = scratch + NA_BUCKET_CURSOR;
  float* tile_rho_max = reinterpret_cast<float*>(scratch + NA_RHO_MAX);
  unsigned* tile_fmax = reinterpret_cast<unsigned*>(scratch + NA_FMAX);
  int* list = scratch + NA_LIST;
  const float2* X = reinterpret_cast<const float2*>(xy);
  k_noalloc_init<<<32, 256, 0, st>>>(scratch, n_tiles);
  mc::k_list_build_small<<<dim3(1, 1), 1024, 0, st>>>(ls_state, X, nullptr, n_beads, nx, ny, n_tiles, tile_count, tile_start,
                                                       bucket_count, bucket_cursor, list,
                                                       mc::CrowdedTable{nullptr, nullptr, nullptr}, 0);
  mc::k_deposit_tile<false><<<dim3(nx / mc::TS, ny / mc::TS, 1), 256, 0, st>>>(nx, ny, tile_start, list, X, rho_b, tile_rho_max,
                                                                                tile_fmax, nullptr, 0);
  e = cudaPeekAtLastError();
  if (e != cudaSuccess) return na_fail(MC_ECUDA, std::string("mc_deposit_noalloc: kernel launch: ") + cudaGetErrorString(e));
  return MC_OK;
}

#pragma GCC visibility pop
}  // extern "C"

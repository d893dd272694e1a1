// cel_api.cu — host side of the celstep C ABI (include/cel.h): context, physics tables (docs/PHYSICS_SPEC.md S4),
// HBM layout, the non-blocking step-iteration loop and the debug/parity surface.
// No torch types, no CPU fallback: every step of the path runs in the kernels of cel_kernels.cuh.
#include "../../include/cel.h"
#include "cel_kernels.cuh"
#include "cel_physics.cuh"
#include "cel_tail.cuh"

// NVTX ranges around every enqueued phase (ScopedProfiling over NVTX): compile-time switch, build with
// -DCEL_NVTX (paper_2503_17608_b200/build.py: CEL_NVTX=1 in the environment); header-only NVTX 3, no library to link
#ifdef CEL_NVTX
#include <nvtx3/nvToolsExt.h>
#define CEL_RANGE_PUSH(name) nvtxRangePushA(name)
#define CEL_RANGE_POP() nvtxRangePop()
#else
#define CEL_RANGE_PUSH(name) ((void)0)
#define CEL_RANGE_POP() ((void)0)
#endif

#include <cmath>
#include <condition_variable>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <thread>
#include <vector>

using namespace cel;

static_assert(sizeof(cel_primary) == 64 && sizeof(PrimaryRec) == 64, "cel_primary layout");
static_assert(sizeof(cel_track) == 80 && sizeof(TrackRec) == 80, "cel_track layout");
static_assert((int)K_COUNT == (int)CEL_KERNEL_COUNT && (int)K_PUSH == (int)CEL_K_PUSH && (int)K_CHARGED == (int)CEL_K_CHARGED && (int)K_FILL_SORT == (int)CEL_K_FILL_SORT, "kernel ids");
static_assert(sizeof(RecA) == 32 && sizeof(RecB) == 32, "record layout");
static_assert(sizeof(cel_hit) == 16 && sizeof(HitRec) == 16, "cel_hit layout");
static_assert(sizeof(DeviceState) < 3500, "DeviceState must fit in kernel parameter space");

namespace {

constexpr uint32_t kLogCapacity = 1u << 16;  // iterations whose per-action counts are logged
constexpr int kStatusSlots = 2;
constexpr int kMaxKernelsPerIteration = 16;
static_assert(CEL_ERR_INTERNAL == -9, "k_fill_sort sets -9");
constexpr int kSideStreams = 5;   // (the last one carries k_hits_flush beside k_push)

struct HostTables {                 // per material, kept for cel_debug_table
  std::vector<double> t[5];         // compton, pe, pair, brems, range
  double inv_X0;
};

}  // namespace

struct cel_ctx {
  DeviceState D{};
  int n_mats = 0;
  std::vector<HostTables> tables;
  cel_physics phys{};
  cel_geometry geo{};
  std::vector<double> h_bounds; std::vector<int> h_vol_material, h_vol_bin;
  uint64_t n_slots = 0;
  int user_sort_mode = 0;           // the CEL_SORT_* value given to cel_create (D.sort_mode folds BY_ACTION_REUSE into BY_ACTION)
  // device-resident read-only data (small)
  void* d_params_blob = nullptr;
  // workspace
  void* workspace = nullptr; uint64_t workspace_bytes = 0; bool own_workspace = false; bool laid_out = false;
  // stream-ordered scratch of the current run
  void* scratch = nullptr; void* d_tally = nullptr; void* d_prim = nullptr;
  cudaStream_t stream = nullptr; bool own_stream = false; bool stream_blocking = false;
  cudaStream_t side[kSideStreams] = {nullptr, nullptr, nullptr, nullptr, nullptr};   // branches of the iteration graph (independent action kernels)
  cudaEvent_t ev_fork = nullptr, ev_join[kSideStreams] = {nullptr, nullptr, nullptr, nullptr, nullptr};
  int concurrent = 1;
  int tail = 1; int tail_iters = 256; int tail_enter = 512;   // k_tail: small populations (cel_tail.cuh)
  uint64_t tail_launches = 0;
  int max_tiles = 0;  // option "max_tiles": upper bound of the number of bookkeeping tiles (0 = the default of make_tiling)
  int live_tiles = 1; // option "live_tiles": the bookkeeping kernels walk only the tiles the population has reached (0 = every tile)
  int grid_cap = 6;   // blocks per SM of the action kernels' grids (option "grid_cap": several contexts sharing the GPU take a share each)
  int merge_discrete = 1;   // sort by action: photoelectric + pair + annihilation in one launch (k_discrete)
  bool no_pdl_next = false;
  int pdl = 1;   // programmatic dependent launch along the main-stream chain of an iteration
  cudaEvent_t ev_start = nullptr, ev_stop = nullptr, ev_batch[kStatusSlots] = {nullptr, nullptr};
  Control* h_status = nullptr;      // pinned, kStatusSlots entries
  uint64_t* h_tally = nullptr; size_t h_tally_bytes = 0;   // pinned
  void* h_prim = nullptr; size_t h_prim_bytes = 0;         // pinned staging of primaries
  cudaGraph_t graph = nullptr; cudaGraphExec_t graph_exec = nullptr;
  int trace_iters = 0; int trace_ends = 1; void* d_trace = nullptr;   // option "trace": device-side timeline of the first trace_iters iterations
  DeviceState graph_D{}; int graph_cfg[6] = {-1, -1, -1, -1, -1, -1};   // what the captured graph has baked in (arguments, options)
  int use_graph = 1; int batch = 16; int64_t max_iterations = 1ll << 22;
  int n_sm = 148;
  bool ran = false; int run_error = 0;
  uint64_t launches = 0; int kernels_per_iteration = 0;
  Control last{};                   // final status of the last run
  std::string cuda_error;
  // hit transfer (option "hits"): 1 = stream-ordered (k_hits_flush into pinned, device-mapped ring buffers
  // after every iteration, consumed by a host thread one batch behind), 2 = the paper's "before" (a blocking cudaMemcpy
  // on the default stream into pageable memory after every batch)
  int hits_mode = 0; int hit_tally = 0; uint64_t hit_capacity = 1ull << 24;
  void* d_hits = nullptr; uint64_t d_hits_cap = 0;
  cel_hit* h_ring[2] = {nullptr, nullptr}; uint64_t h_ring_cap = 0;
  std::vector<cel_hit> h_pageable;
  cudaEvent_t ev_hfork = nullptr;
  cel_hit_callback hit_cb = nullptr; void* hit_cb_user = nullptr;
  std::thread consumer; std::mutex cmu; std::condition_variable ccv;
  const cel_hit* job_ptr = nullptr; uint64_t job_n = 0; bool job_pending = false, consumer_stop = false, consumer_on = false;
  uint64_t hits_total = 0, hits_qsum = 0, hits_bytes = 0;
  std::vector<uint64_t> h_hit_tally;
  // per-kernel device timing (option "profile"): events around every launch, direct launches, one sync per batch
  int profile = 0;
  std::vector<cudaEvent_t> prof_ev;   // [batch][kMaxKernelsPerIteration + 1]
  int prof_b = 0;                     // iteration inside the current batch
  int iter_kernel[kMaxKernelsPerIteration] = {0};
  double kernel_ms[CEL_KERNEL_COUNT] = {0};
  uint64_t kernel_launches[CEL_KERNEL_COUNT] = {0};
};

namespace {

#define CEL_CUDA(ctx, call)                                                        \
  do {                                                                             \
    cudaError_t e_ = (call);                                                       \
    if (e_ != cudaSuccess) {                                                       \
      (ctx)->cuda_error = std::string(#call) + ": " + cudaGetErrorString(e_);      \
      return (e_ == cudaErrorMemoryAllocation) ? CEL_ERR_OOM : CEL_ERR_CUDA;       \
    }                                                                              \
  } while (0)

inline uint64_t align_up(uint64_t x, uint64_t a) { return (x + a - 1) / a * a; }

// ---------------------------------------------------------------- S4: physics tables, built on the host
double klein_nishina_total(double E) {
  const double k = E / kElectronMass;
  const double L = std::log1p(2.0 * k);
  const double a = (1.0 + k) / (k * k) * (2.0 * (1.0 + k) / (1.0 + 2.0 * k) - L / k);
  const double b = L / (2.0 * k);
  const double c = (1.0 + 3.0 * k) / ((1.0 + 2.0 * k) * (1.0 + 2.0 * k));
  return 2.0 * kPi * kClassicalRadius * kClassicalRadius * (a + b - c);
}

struct MaterialHost { double n_atom, n_e, I, L_rad, inv_X0, Z; };

double collision_stopping_power(const MaterialHost& m, double T) {
  const double tau = T / kElectronMass;
  const double g1 = tau + 1.0;
  const double beta2 = tau * (tau + 2.0) / (g1 * g1);
  const double ir = m.I / kElectronMass;
  const double br = std::log(tau * tau * (tau + 2.0) / (2.0 * ir * ir)) + 1.0 - beta2 +
                    (tau * tau / 8.0 - (2.0 * tau + 1.0) * std::log(2.0)) / (g1 * g1);
  return 2.0 * kPi * kClassicalRadius * kClassicalRadius * kElectronMass * m.n_e / beta2 * br;
}

void build_tables(const cel_material& mat, const cel_physics& ph, HostTables& out) {
  MaterialHost m;
  m.Z = mat.Z;
  m.n_atom = mat.density_g_cm3 * kAvogadro / mat.A;
  m.n_e = mat.Z * m.n_atom;
  m.I = 16e-6 * std::pow(mat.Z, 0.9);
  m.L_rad = std::log(183.0 * std::pow(mat.Z, -1.0 / 3.0));
  m.inv_X0 = 4.0 * kFineStructure * kClassicalRadius * kClassicalRadius * m.n_atom * mat.Z * (mat.Z + 1.0) * m.L_rad;
  out.inv_X0 = m.inv_X0;
  const double u0 = std::log(1e-3), du = std::log(10.0) / 64.0;
  const double n_pb = 11.35 * kAvogadro / 207.2;
  for (auto& v : out.t) v.assign(kGrid, 0.0);
  for (int j = 0; j < kGrid; ++j) {
    const double E = std::exp(u0 + j * du);
    out.t[0][j] = m.n_e * klein_nishina_total(E);
    out.t[1][j] = (m.n_atom / n_pb) * std::pow(mat.Z / 82.0, 5.0) * std::pow(E, -3.5);
    const double no_screen = (28.0 / 9.0) * std::log(2.0 * E / kElectronMass) - 218.0 / 27.0;
    const double full_screen = (28.0 / 9.0) * m.L_rad - 2.0 / 27.0;
    const double f = std::fmax(0.0, std::fmin(no_screen, full_screen));
    out.t[2][j] = ph.enable_pair ? m.n_atom * kFineStructure * kClassicalRadius * kClassicalRadius * mat.Z * (mat.Z + 1.0) * f : 0.0;
    out.t[3][j] = ph.enable_brems ? std::fmax(0.0, std::log(E / ph.cut_MeV)) * m.inv_X0 : 0.0;
  }
  // range: composite Simpson in u = ln T, 64 sub-intervals per cell
  out.t[4][0] = 0.0;
  for (int j = 1; j < kGrid; ++j) {
    const double lo = u0 + (j - 1) * du, hi = u0 + j * du;
    const int n = 64;
    const double h = (hi - lo) / n;
    double acc = 0.0;
    for (int i = 0; i <= n; ++i) {
      const double T = std::exp(lo + i * h);
      const double w = (i == 0 || i == n) ? 1.0 : ((i & 1) ? 4.0 : 2.0);
      acc += w * (T / collision_stopping_power(m, T));
    }
    out.t[4][j] = out.t[4][j - 1] + acc * h / 3.0;
  }
}

int host_locate(const cel_geometry& g, const double* bounds, const double pos[3], const double dir[3]) {
  if (g.kind == CEL_GEOM_SLAB) {
    for (int i = 0; i < g.n_vol; ++i) {
      const double lo = bounds[i], hi = bounds[i + 1];
      if (pos[2] > lo && pos[2] < hi) return i;
      if (pos[2] == lo && dir[2] >= 0.0) return i;
      if (pos[2] == hi && dir[2] < 0.0) return i;
    }
    return -1;
  }
  const double r = std::sqrt(pos[0] * pos[0] + pos[1] * pos[1]);
  for (int i = 0; i < g.n_vol; ++i)
    if (r >= bounds[i] && r < bounds[i + 1]) return i;
  return -1;
}

}  // namespace

// ================================================================ workspace layout
namespace {

struct Layout {
  uint64_t stA, stB, akey, nsec, indices, secA, secB, initA, initB, ctl, log, total;
};

// bookkeeping tiles (cel_device.cuh): sub-tiles of kSub slots, tiles of 2^shift slots in groups of kGroupTiles
struct Tiling { uint32_t n_tiles, tile_shift, subs_per_tile, n_groups; };
uint64_t g_max_tiles_small = 4096, g_max_tiles_large = 8192;
Tiling make_tiling(uint64_t N, uint64_t max_tiles_override = 0) {
  const uint64_t subs = (N + kSub - 1) / kSub;
  uint32_t spt = 1, shift = 10;
  static_assert(kSub == 1024, "tile_shift assumes 1024-slot sub-tiles");
  // 1024-slot tiles up to 2^22 slots (4096 tiles), at most 8192 tiles beyond. Measured with the live-tile bound (blocks above
  // the population leave at once): 2^22 slots 27.8 ms with 4096 tiles vs 29.8 with 2048; 2^24 slots 29.5 ms with 8192 tiles
  // vs 34.7 with 4096 and 30.6 with 16384 — a block that walks several sub-tiles does them one after the other, and every
  // block of a bookkeeping kernel, live or not, costs launch time
  uint64_t max_tiles = N > (1ull << 22) ? g_max_tiles_large : g_max_tiles_small;
  if (max_tiles_override) max_tiles = max_tiles_override;
  if (max_tiles > (uint64_t)kMaxTiles) max_tiles = kMaxTiles;
  while ((subs + spt - 1) / spt > max_tiles) { spt *= 2; shift += 1; }
  Tiling t;
  t.subs_per_tile = spt; t.tile_shift = shift;
  t.n_tiles = (uint32_t)((N + ((uint64_t)1 << shift) - 1) >> shift);
  t.n_groups = (t.n_tiles + kGroupTiles - 1) / kGroupTiles;
  return t;
}

int n_index_regions(int sort_mode) {   // regions of N entries in the index array (cel_device.cuh: DeviceState::indices)
  if (sort_mode == CEL_SORT_BY_ACTION || sort_mode == CEL_SORT_BY_ACTION_REUSE) return 8;
  if (sort_mode == CEL_SORT_BY_PARTICLE) return 4;
  if (sort_mode == CEL_SORT_PARTITION) return 1;   // plist
  return 0;
}

Layout make_layout(uint64_t N, uint64_t cap, int sort_mode, uint64_t max_tiles_override = 0) {
  Layout L{};
  const Tiling tl = make_tiling(N, max_tiles_override);
  const uint64_t padded = (uint64_t)tl.n_tiles << tl.tile_shift;
  uint64_t o = 0;
  auto take = [&](uint64_t bytes) { uint64_t r = o; o = align_up(o + bytes, 256); return r; };
  L.stA = take(N * sizeof(RecA));
  L.stB = take(N * sizeof(RecB));
  L.akey = take(padded);
  L.nsec = take(padded);
  L.indices = take((uint64_t)n_index_regions(sort_mode) * N * sizeof(uint32_t));
  L.secA = take(2 * N * sizeof(RecA));
  L.secB = take(2 * N * sizeof(RecB));
  L.initA = take(cap * sizeof(RecA));
  L.initB = take(cap * sizeof(RecB));
  L.ctl = take(sizeof(Control));
  L.log = take((uint64_t)kLogCapacity * 8 * sizeof(uint32_t));
  L.total = o;
  return L;
}

uint64_t default_capacity(uint64_t N, uint64_t cap) {
  if (cap != 0) return cap;
  const uint64_t c = 8 * N;
  return c > (1ull << 24) ? c : (1ull << 24);
}

int lay_out(cel_ctx* c) {
  if (c->laid_out) return CEL_OK;
  const Layout L = make_layout(c->n_slots, c->D.init_capacity, c->user_sort_mode, (uint64_t)c->max_tiles);
  if (!c->workspace) {
    CEL_CUDA(c, cudaMalloc(&c->workspace, L.total));
    c->workspace_bytes = L.total; c->own_workspace = true;
  } else if (c->workspace_bytes < L.total) {
    return CEL_ERR_INVALID_ARG;
  }
  char* base = (char*)c->workspace;
  DeviceState& D = c->D;
  D.stA = (RecA*)(base + L.stA); D.stB = (RecB*)(base + L.stB);
  D.akey = (uint8_t*)(base + L.akey); D.nsec = (uint8_t*)(base + L.nsec);
  D.indices = n_index_regions(c->user_sort_mode) ? (uint32_t*)(base + L.indices) : nullptr;
  D.secA = (RecA*)(base + L.secA); D.secB = (RecB*)(base + L.secB);
  D.initA = (RecA*)(base + L.initA); D.initB = (RecB*)(base + L.initB);
  D.ctl = (Control*)(base + L.ctl);
  D.counts_log = (uint32_t*)(base + L.log);
  D.log_capacity = kLogCapacity;
  c->laid_out = true;
  return CEL_OK;
}

}  // namespace

extern "C" uint64_t cel_workspace_bytes(uint64_t n_slots, uint64_t init_capacity, int sort_mode) {
  return make_layout(n_slots, default_capacity(n_slots, init_capacity), sort_mode).total;
}

// ================================================================ create / destroy
extern "C" int cel_create(const cel_geometry* g, const cel_material* mats, int n_mats, const cel_physics* ph,
                          uint64_t n_slots, int sort_mode, cel_ctx** out) {
  if (!g || !mats || !ph || !out || n_mats < 1 || n_slots < 1 || n_slots > (1ull << 28)) return CEL_ERR_INVALID_ARG;
  if (sort_mode < 0 || sort_mode > CEL_SORT_BY_ACTION_REUSE || (g->kind != CEL_GEOM_SLAB && g->kind != CEL_GEOM_CYL)) return CEL_ERR_INVALID_ARG;
  if (g->n_vol < 1 || g->n_vol > 254 || !g->bounds || !g->vol_material || !g->vol_bin) return CEL_ERR_INVALID_ARG;
  for (int i = 0; i < g->n_vol; ++i) {
    if (!(g->bounds[i] < g->bounds[i + 1])) return CEL_ERR_INVALID_ARG;
    if (g->vol_material[i] < -1 || g->vol_material[i] >= n_mats || g->vol_bin[i] < -1) return CEL_ERR_INVALID_ARG;
  }
  if (g->kind == CEL_GEOM_CYL && g->bounds[0] != 0.0) return CEL_ERR_INVALID_ARG;
  if (!(ph->cut_MeV > 0.0) || ph->max_substeps < 1) return CEL_ERR_INVALID_ARG;
  if (ph->max_steps_per_track < 1 || ph->max_steps_per_track > 65535u) return CEL_ERR_INVALID_ARG;   // the step count is a 16-bit field of the slot's meta word
  for (int i = 0; i < n_mats; ++i)
    if (!(mats[i].density_g_cm3 > 0.0) || !(mats[i].Z > 0.0) || !(mats[i].A > 0.0)) return CEL_ERR_INVALID_ARG;

  int n_dev = 0;
  if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev < 1) return CEL_ERR_CUDA;  // no CPU fallback

  cel_ctx* c = new cel_ctx();
  c->geo = *g; c->phys = *ph; c->n_mats = n_mats; c->n_slots = n_slots;
  c->h_bounds.assign(g->bounds, g->bounds + g->n_vol + 1);
  c->h_vol_material.assign(g->vol_material, g->vol_material + g->n_vol);
  c->h_vol_bin.assign(g->vol_bin, g->vol_bin + g->n_vol);
  c->geo.bounds = c->h_bounds.data(); c->geo.vol_material = c->h_vol_material.data(); c->geo.vol_bin = c->h_vol_bin.data();
  c->tables.resize(n_mats);
  for (int i = 0; i < n_mats; ++i) build_tables(mats[i], *ph, c->tables[i]);
  int dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, dev);

  // one blob with all read-only device data: bounds | vol_material | vol_bin | mats | photon_xs | charged_xs | range
  const uint64_t o_bounds = 0;
  const uint64_t o_vm = align_up(o_bounds + (g->n_vol + 1) * sizeof(double), 256);
  const uint64_t o_vb = align_up(o_vm + g->n_vol * sizeof(int), 256);
  const uint64_t o_mats = align_up(o_vb + g->n_vol * sizeof(int), 256);
  const uint64_t o_ph = align_up(o_mats + n_mats * sizeof(MaterialDev), 256);
  const uint64_t o_ch = align_up(o_ph + (uint64_t)n_mats * kGrid * sizeof(PhotonXs), 256);
  const uint64_t o_rg = align_up(o_ch + (uint64_t)n_mats * kGrid * sizeof(ChargedXs), 256);
  const uint64_t o_en = align_up(o_rg + (uint64_t)n_mats * kGrid * sizeof(double), 256);
  const uint64_t blob_bytes = align_up(o_en + (uint64_t)kGrid * sizeof(double), 256);
  std::vector<char> blob(blob_bytes, 0);
  std::memcpy(blob.data() + o_bounds, c->h_bounds.data(), (g->n_vol + 1) * sizeof(double));
  std::memcpy(blob.data() + o_vm, c->h_vol_material.data(), g->n_vol * sizeof(int));
  std::memcpy(blob.data() + o_vb, c->h_vol_bin.data(), g->n_vol * sizeof(int));
  for (int m = 0; m < n_mats; ++m) {
    ((MaterialDev*)(blob.data() + o_mats))[m].inv_X0 = c->tables[m].inv_X0;
    for (int j = 0; j < kGrid; ++j) {
      PhotonXs& px = ((PhotonXs*)(blob.data() + o_ph))[(size_t)m * kGrid + j];
      px.compton = c->tables[m].t[0][j]; px.pe = c->tables[m].t[1][j]; px.pair = c->tables[m].t[2][j]; px.pad = 0.0;
      ChargedXs& cx = ((ChargedXs*)(blob.data() + o_ch))[(size_t)m * kGrid + j];
      cx.brems = c->tables[m].t[3][j]; cx.range = c->tables[m].t[4][j];
      ((double*)(blob.data() + o_rg))[(size_t)m * kGrid + j] = c->tables[m].t[4][j];
    }
  }
  for (int j = 0; j < kGrid; ++j) ((double*)(blob.data() + o_en))[j] = std::exp(std::log(1e-3) + j * (std::log(10.0) / 64.0));
  auto fail = [&](int code) { cel_destroy(c); return code; };
  if (cudaMalloc(&c->d_params_blob, blob_bytes) != cudaSuccess) return fail(CEL_ERR_OOM);
  if (cudaMemcpy(c->d_params_blob, blob.data(), blob_bytes, cudaMemcpyHostToDevice) != cudaSuccess) return fail(CEL_ERR_CUDA);
  char* db = (char*)c->d_params_blob;

  DeviceState& D = c->D;
  Params& P = D.P;
  P.geom_kind = g->kind; P.n_vol = g->n_vol;
  int nb = 0;
  for (int i = 0; i < g->n_vol; ++i) if (g->vol_bin[i] + 1 > nb) nb = g->vol_bin[i] + 1;
  P.n_bins = nb;
  P.bounds = (const double*)(db + o_bounds); P.vol_material = (const int*)(db + o_vm); P.vol_bin = (const int*)(db + o_vb);
  P.half_x = g->half_x; P.half_y = g->half_y; P.half_z = g->half_z;
  const double bm = std::sqrt(g->field_T[0] * g->field_T[0] + g->field_T[1] * g->field_T[1] + g->field_T[2] * g->field_T[2]);
  P.bmag = bm;
  P.bhx = bm > 0.0 ? g->field_T[0] / bm : 0.0; P.bhy = bm > 0.0 ? g->field_T[1] / bm : 0.0; P.bhz = bm > 0.0 ? g->field_T[2] / bm : 0.0;
  P.key0 = (uint32_t)(ph->seed & 0xffffffffu); P.key1 = (uint32_t)(ph->seed >> 32);
  P.cut = ph->cut_MeV;
  P.enable_msc = ph->enable_msc; P.enable_eloss = ph->enable_eloss; P.enable_annihilation = ph->enable_annihilation;
  P.electrons_local = ph->electrons_local; P.max_substeps = ph->max_substeps; P.max_steps_per_track = ph->max_steps_per_track;
  P.u0 = std::log(1e-3); P.du = std::log(10.0) / 64.0; P.inv_du = 1.0 / P.du;
  P.mats = (const MaterialDev*)(db + o_mats); P.photon_xs = (const PhotonXs*)(db + o_ph);
  P.charged_xs = (const ChargedXs*)(db + o_ch); P.range_tab = (const double*)(db + o_rg);
  P.energy_nodes = (const double*)(db + o_en);
  const Tiling tl = make_tiling(n_slots);
  D.N = (uint32_t)n_slots; D.n_tiles = tl.n_tiles; D.n_groups = tl.n_groups; D.tile_shift = tl.tile_shift; D.subs_per_tile = tl.subs_per_tile;
  c->user_sort_mode = sort_mode;
  D.sort_mode = sort_mode == CEL_SORT_BY_ACTION_REUSE ? CEL_SORT_BY_ACTION : sort_mode;   // the index sort is the same;
  D.reuse = sort_mode == CEL_SORT_BY_ACTION_REUSE ? 1 : 0;                               // only the interaction epilogues differ (S9-R)
  D.init_capacity = default_capacity(n_slots, ph->init_capacity);

  if (cudaStreamCreateWithFlags(&c->stream, cudaStreamNonBlocking) != cudaSuccess) return fail(CEL_ERR_CUDA);
  c->own_stream = true;
  for (int i = 0; i < kSideStreams; ++i) {
    if (cudaStreamCreateWithFlags(&c->side[i], cudaStreamNonBlocking) != cudaSuccess) return fail(CEL_ERR_CUDA);
    if (cudaEventCreateWithFlags(&c->ev_join[i], cudaEventDisableTiming) != cudaSuccess) return fail(CEL_ERR_CUDA);
  }
  if (cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) != cudaSuccess) return fail(CEL_ERR_CUDA);
  if (cudaEventCreateWithFlags(&c->ev_hfork, cudaEventDisableTiming) != cudaSuccess) return fail(CEL_ERR_CUDA);
  if (cudaEventCreate(&c->ev_start) != cudaSuccess || cudaEventCreate(&c->ev_stop) != cudaSuccess) return fail(CEL_ERR_CUDA);
  for (int i = 0; i < kStatusSlots; ++i)
    if (cudaEventCreateWithFlags(&c->ev_batch[i], cudaEventDisableTiming) != cudaSuccess) return fail(CEL_ERR_CUDA);
  if (cudaHostAlloc((void**)&c->h_status, kStatusSlots * sizeof(Control), cudaHostAllocMapped) != cudaSuccess) return fail(CEL_ERR_OOM);
  { void* dp = nullptr; if (cudaHostGetDevicePointer(&dp, c->h_status, 0) != cudaSuccess) return fail(CEL_ERR_CUDA); D.status_host = (Control*)dp; }
  *out = c;
  return CEL_OK;
}

namespace {
// ---------------------------------------------------------------- the host side of the hit transfer
void consume_hits(cel_ctx* c, const cel_hit* h, uint64_t n) {   // what the "user's sensitive detector" does with a batch
  uint64_t q = 0;
  if (c->hit_tally) {
    const uint64_t stride = (uint64_t)c->D.P.n_bins + 1;
    for (uint64_t i = 0; i < n; ++i) { q += h[i].q; c->h_hit_tally[(uint64_t)h[i].event * stride + (uint64_t)h[i].bin] += h[i].q; }
  } else {
    for (uint64_t i = 0; i < n; ++i) q += h[i].q;
  }
  c->hits_total += n; c->hits_qsum += q; c->hits_bytes += n * sizeof(cel_hit);
  if (c->hit_cb && n) c->hit_cb(h, n, c->hit_cb_user);
}
void consumer_main(cel_ctx* c) {
  std::unique_lock<std::mutex> lk(c->cmu);
  while (true) {
    c->ccv.wait(lk, [c] { return c->job_pending || c->consumer_stop; });
    if (c->job_pending) {
      const cel_hit* p = c->job_ptr; const uint64_t n = c->job_n;
      lk.unlock();
      consume_hits(c, p, n);
      lk.lock();
      c->job_pending = false;
      c->ccv.notify_all();
    } else if (c->consumer_stop) {
      return;
    }
  }
}
void consumer_wait_idle(cel_ctx* c) {
  if (!c->consumer_on) return;
  std::unique_lock<std::mutex> lk(c->cmu);
  c->ccv.wait(lk, [c] { return !c->job_pending; });
}
void consumer_submit(cel_ctx* c, const cel_hit* p, uint64_t n) {
  std::unique_lock<std::mutex> lk(c->cmu);
  c->ccv.wait(lk, [c] { return !c->job_pending; });
  c->job_ptr = p; c->job_n = n; c->job_pending = true;
  c->ccv.notify_all();
}
void consumer_shutdown(cel_ctx* c) {
  if (!c->consumer_on) return;
  { std::unique_lock<std::mutex> lk(c->cmu); c->ccv.wait(lk, [c] { return !c->job_pending; }); c->consumer_stop = true; c->ccv.notify_all(); }
  c->consumer.join();
  c->consumer_on = false;
}
}  // namespace

extern "C" void cel_destroy(cel_ctx* c) {
  if (!c) return;
  if (c->stream) cudaStreamSynchronize(c->stream);
  consumer_shutdown(c);
  if (c->d_hits) cudaFree(c->d_hits);
  for (int i = 0; i < 2; ++i) if (c->h_ring[i]) cudaFreeHost(c->h_ring[i]);
  if (c->ev_hfork) cudaEventDestroy(c->ev_hfork);
  for (int i = 0; i < kSideStreams; ++i) {
    if (c->side[i]) { cudaStreamSynchronize(c->side[i]); cudaStreamDestroy(c->side[i]); }
    if (c->ev_join[i]) cudaEventDestroy(c->ev_join[i]);
  }
  if (c->ev_fork) cudaEventDestroy(c->ev_fork);
  if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
  if (c->graph) cudaGraphDestroy(c->graph);
  if (c->scratch) cudaFree(c->scratch);
  if (c->d_tally) cudaFree(c->d_tally);
  if (c->d_prim) cudaFree(c->d_prim);
  if (c->d_trace) cudaFree(c->d_trace);
  if (c->own_workspace && c->workspace) cudaFree(c->workspace);
  if (c->d_params_blob) cudaFree(c->d_params_blob);
  if (c->h_status) cudaFreeHost(c->h_status);
  if (c->h_tally) cudaFreeHost(c->h_tally);
  if (c->h_prim) cudaFreeHost(c->h_prim);
  if (c->ev_start) cudaEventDestroy(c->ev_start);
  if (c->ev_stop) cudaEventDestroy(c->ev_stop);
  for (int i = 0; i < kStatusSlots; ++i) if (c->ev_batch[i]) cudaEventDestroy(c->ev_batch[i]);
  for (cudaEvent_t e : c->prof_ev) cudaEventDestroy(e);
  if (c->own_stream && c->stream) cudaStreamDestroy(c->stream);
  delete c;
}

extern "C" int cel_set_stream(cel_ctx* c, void* s) {
  if (!c || c->ran) return CEL_ERR_INVALID_ARG;
  if (c->own_stream && c->stream) { cudaStreamDestroy(c->stream); c->own_stream = false; }
  c->stream = (cudaStream_t)s;
  // the legacy default stream cannot be captured into a CUDA graph: launch the kernels directly there
  if (c->stream == nullptr || c->stream == cudaStreamLegacy) c->use_graph = 0;
  return CEL_OK;
}

extern "C" int cel_set_workspace(cel_ctx* c, void* dptr, uint64_t bytes) {
  if (!c || !dptr || c->laid_out || ((uintptr_t)dptr & 255)) return CEL_ERR_INVALID_ARG;
  if (bytes < make_layout(c->n_slots, c->D.init_capacity, c->user_sort_mode).total) return CEL_ERR_INVALID_ARG;
  c->workspace = dptr; c->workspace_bytes = bytes; c->own_workspace = false;
  return CEL_OK;
}

extern "C" int cel_set_option(cel_ctx* c, const char* name, int64_t v) {
  if (!c || !name) return CEL_ERR_INVALID_ARG;
  if (!std::strcmp(name, "use_graph")) c->use_graph = v ? 1 : 0;
  else if (!std::strcmp(name, "batch")) { if (v < 1 || v > 4096) return CEL_ERR_INVALID_ARG; c->batch = (int)v; }
  else if (!std::strcmp(name, "profile")) c->profile = v ? 1 : 0;
  else if (!std::strcmp(name, "concurrent")) c->concurrent = v ? 1 : 0;
  else if (!std::strcmp(name, "pdl")) c->pdl = v ? 1 : 0;
  else if (!std::strcmp(name, "merge_discrete")) c->merge_discrete = v ? 1 : 0;
  else if (!std::strcmp(name, "trace_ends")) c->trace_ends = v ? 1 : 0;
  else if (!std::strcmp(name, "trace")) { if (v < 0 || v > (1 << 20)) return CEL_ERR_INVALID_ARG; c->trace_iters = (int)v; }
  else if (!std::strcmp(name, "tail")) c->tail = v ? 1 : 0;
  else if (!std::strcmp(name, "tail_iters")) { if (v < 1 || v > (1 << 20)) return CEL_ERR_INVALID_ARG; c->tail_iters = (int)v; }
  else if (!std::strcmp(name, "tail_enter")) { if (v < 0 || v > kTailCap) return CEL_ERR_INVALID_ARG; c->tail_enter = (int)v; }
  else if (!std::strcmp(name, "max_tiles")) {   // before the first run only: the slot arrays are padded to whole tiles
    if (v < 0 || v > kMaxTiles || c->laid_out) return CEL_ERR_INVALID_ARG;
    c->max_tiles = (int)v;
    const Tiling tl = make_tiling(c->n_slots, (uint64_t)v);
    c->D.n_tiles = tl.n_tiles; c->D.n_groups = tl.n_groups; c->D.tile_shift = tl.tile_shift; c->D.subs_per_tile = tl.subs_per_tile;
  }
  else if (!std::strcmp(name, "live_tiles")) { if (v != 0 && v != 1) return CEL_ERR_INVALID_ARG; c->live_tiles = (int)v; }
  else if (!std::strcmp(name, "grid_cap")) { if (v < 1 || v > 32) return CEL_ERR_INVALID_ARG; c->grid_cap = (int)v; }
  else if (!std::strcmp(name, "hits")) { if (v < 0 || v > 2) return CEL_ERR_INVALID_ARG; c->hits_mode = (int)v; }
  else if (!std::strcmp(name, "hit_tally")) c->hit_tally = v ? 1 : 0;
  else if (!std::strcmp(name, "hit_capacity")) { if (v < 1 || v > (1ll << 30)) return CEL_ERR_INVALID_ARG; c->hit_capacity = (uint64_t)v; }
  else if (!std::strcmp(name, "max_iterations")) { if (v < 1) return CEL_ERR_INVALID_ARG; c->max_iterations = v; }
  else return CEL_ERR_INVALID_ARG;
  return CEL_OK;
}

extern "C" const char* cel_strerror(int code) {
  switch (code) {
    case CEL_OK: return "ok";
    case CEL_ERR_INVALID_ARG: return "invalid argument";
    case CEL_ERR_CUDA: return "CUDA runtime error";
    case CEL_ERR_OOM: return "out of memory";
    case CEL_ERR_INIT_OVERFLOW: return "initializer stack overflow";
    case CEL_ERR_TALLY_OVERFLOW: return "tally overflow";
    case CEL_ERR_NONFINITE: return "non-finite track state";
    case CEL_ERR_NOT_RUN: return "no transport has run";
    case CEL_ERR_MAX_ITER: return "iteration limit reached";
    case CEL_ERR_INTERNAL: return "internal error: a bookkeeping wait gave up";
    case CEL_ERR_HIT_OVERFLOW: return "hit buffer overflow (option hit_capacity)";
    case CEL_ERR_TOO_LARGE: return "more slots than the static scratch of cel_reindex_static holds (2^22)";
    default: return "unknown error";
  }
}
extern "C" const char* cel_last_cuda_error(cel_ctx* c) { return c ? c->cuda_error.c_str() : ""; }

// ================================================================ the step iteration and the host loop
namespace {

int physics_grid(const cel_ctx* c, int times = 1) {
  const uint64_t need = (c->n_slots + kBlock - 1) / kBlock;
  const uint64_t cap = (uint64_t)c->n_sm * (uint64_t)c->grid_cap * (uint64_t)times;
  return (int)(need < cap ? need : cap);
}
// k_photon sorted by action: four times as many, shorter blocks. Its blocks are dispatched behind k_charged's (whose
// first wave fills every SM's register file), so they are what runs at the end of the action phase, and the phase ends with
// the last of them: short blocks leave a short tail (measured: config 2 -0.8 %, 2^24 slots -1.4 %; k_charged itself is
// fastest at grid_cap blocks per SM, and 16 x is slower again at 2^24 slots).
constexpr int kPhotonGridTimes = 4;

const char* const kKernelNames[CEL_KERNEL_COUNT] = {
    "fill_sort", "annihilation", "photoelectric", "pair", "photon", "charged", "push",
    "part_count", "part_scatter", "discrete", "hits_flush", "tail"};

// bookkeeping after each kernel launch: which kernel it was and, in profile mode, an event behind it
inline void after_launch(cel_ctx* c, int id, int& n) {
  CEL_RANGE_PUSH(kKernelNames[id]); CEL_RANGE_POP();   // (a marker-like range per phase: the launch itself is asynchronous)
  c->iter_kernel[n] = id;
  ++n;
  if (c->profile) cudaEventRecord(c->prof_ev[(size_t)c->prof_b * (kMaxKernelsPerIteration + 1) + n], c->stream);
}

// launch on the main-stream chain: with `pdl` the kernel may be scheduled while its predecessor in the stream drains
template <typename K>
void launch_chain(cel_ctx* c, K kernel, int grid, int block, cudaStream_t s) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = 0; cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  // (the first kernel after a k_tail launch is serialised fully: k_fill_sort reads counters and key bytes BEFORE its
  // programmatic-dependency wait, which is only sound when the kernel before it wrote none of them)
  cfg.attrs = attr; cfg.numAttrs = (c->pdl && !c->profile && !c->no_pdl_next) ? 1 : 0;
  c->no_pdl_next = false;
  cudaLaunchKernelEx(&cfg, kernel, c->D);
}

// P5, and beside it (option hits = 1) the transfer of the iteration's hit records to the host ring buffer
template <bool TR>
void enqueue_push_and_flush(cel_ctx* c, int& n) {
  const DeviceState& D = c->D;
  cudaStream_t s = c->stream;
  const bool flush = c->hits_mode == 1;
  const bool fork = flush && c->concurrent && !c->profile;
  const int fg = c->n_sm * 4;
  if (fork) {
    cudaStream_t hs = c->side[kSideStreams - 1];
    cudaEventRecord(c->ev_hfork, s); cudaStreamWaitEvent(hs, c->ev_hfork, 0);
    k_hits_flush<TR><<<fg, kTileThreads, 0, hs>>>(D); after_launch(c, CEL_K_HITS_FLUSH, n);
  } else if (flush) {
    k_hits_flush<TR><<<fg, kTileThreads, 0, s>>>(D); after_launch(c, CEL_K_HITS_FLUSH, n);
  }
  launch_chain(c, k_push<TR>, (int)D.n_tiles, kTileThreads, s); after_launch(c, CEL_K_PUSH, n);
  if (fork) { cudaEventRecord(c->ev_join[kSideStreams - 1], c->side[kSideStreams - 1]); cudaStreamWaitEvent(s, c->ev_join[kSideStreams - 1], 0); }
}

// one step iteration = P1, P2, P3 (+P4 inside the action kernels), P5 (docs/PHYSICS_SPEC.md S1); returns the number of
// kernels enqueued. The five action kernels touch disjoint slots. Sorted by action, their ranges are fixed by the sort,
// so they are independent and run as parallel branches (side streams; parallel graph branches under capture). In the
// masked modes a kernel picks its participants by the key byte, which other kernels rewrite, so the order
// interaction -> move must hold per species: {ANNIH -> CHARGED} runs beside {PE -> PAIR -> PHOTON}.
template <bool TR>
int enqueue_iteration_t(cel_ctx* c) {
  const DeviceState& D = c->D;
  cudaStream_t s = c->stream;
  const int tg = (int)D.n_tiles;
  const int pg = physics_grid(c);
  const bool cyl = D.P.geom_kind == CEL_GEOM_CYL, field = D.P.bmag != 0.0;
  int n = 0;
  if (c->profile) cudaEventRecord(c->prof_ev[(size_t)c->prof_b * (kMaxKernelsPerIteration + 1)], s);
  if (D.sort_mode == CEL_SORT_PARTITION) {   // S9-P: the popped initializers are partitioned by charge before the fill
    launch_chain(c, k_part_count<TR>, tg, kTileThreads, s); after_launch(c, CEL_K_PART_COUNT, n);
    launch_chain(c, k_part_scatter<TR>, tg, kTileThreads, s); after_launch(c, CEL_K_PART_SCATTER, n);
  }
  launch_chain(c, k_fill_sort<TR>, tg, kTileThreads, s); after_launch(c, CEL_K_FILL_SORT, n);   // P1 + P2 + S11 in one pass
  const bool fork = c->concurrent && !c->profile;
  const bool by_action = D.sort_mode == CEL_SORT_BY_ACTION;
  if ((D.sort_mode == CEL_SORT_NONE || D.sort_mode == CEL_SORT_PARTITION) && c->merge_discrete) {
    // unsorted / partition: the three pure interactions in one pass on the main stream, then photon beside charged
    // (measured +2..5 %; by particle the two chains below are as fast or faster)
    launch_chain(c, k_discrete_masked<TR>, pg, kBlock, s); after_launch(c, CEL_K_DISCRETE, n);
    cudaStream_t sp = s;
    if (fork) { cudaEventRecord(c->ev_fork, s); cudaStreamWaitEvent(c->side[0], c->ev_fork, 0); sp = c->side[0]; }
    if (cyl) k_photon<1, TR><<<pg, kBlock, 0, sp>>>(D); else k_photon<0, TR><<<pg, kBlock, 0, sp>>>(D);
    after_launch(c, CEL_K_PHOTON, n);
    if (cyl) { if (field) k_charged<true, 1, TR><<<pg, kBlock, 0, s>>>(D); else k_charged<false, 1, TR><<<pg, kBlock, 0, s>>>(D); }
    else { if (field) k_charged<true, 0, TR><<<pg, kBlock, 0, s>>>(D); else k_charged<false, 0, TR><<<pg, kBlock, 0, s>>>(D); }
    after_launch(c, CEL_K_CHARGED, n);
    if (fork) { cudaEventRecord(c->ev_join[0], c->side[0]); cudaStreamWaitEvent(s, c->ev_join[0], 0); }
    enqueue_push_and_flush<TR>(c, n);
    return n;
  }
  // sorted by action: photon, annihilation, photoelectric, pair on one branch each (their ranges are disjoint and fixed);
  // masked modes: {photoelectric -> pair -> photon} on one branch beside {annihilation -> charged} on the main stream
  cudaStream_t s_photon = s, s_annih = s, s_pe = s, s_pair = s;
  int n_side = 0;
  if (fork) {
    n_side = by_action ? (c->merge_discrete ? 2 : 4) : 1;
    cudaEventRecord(c->ev_fork, s);
    for (int i = 0; i < n_side; ++i) cudaStreamWaitEvent(c->side[i], c->ev_fork, 0);
    s_photon = c->side[0]; s_pe = c->side[0]; s_pair = c->side[0];
    if (by_action) { s_annih = c->side[1]; s_pe = c->side[2]; s_pair = c->side[3]; }
  }
  if (by_action && c->merge_discrete) {
    const int dg = pg < c->n_sm ? pg : c->n_sm;   // one block per SM: the ranges are small, and a small grid launches faster
    k_discrete<TR><<<dg, kBlock, 0, s_annih>>>(D); after_launch(c, CEL_K_DISCRETE, n);
  } else {
    if (c->phys.enable_annihilation) { k_annihilation<TR><<<pg, kBlock, 0, s_annih>>>(D); after_launch(c, CEL_K_ANNIH, n); }
    k_photoelectric<TR><<<pg, kBlock, 0, s_pe>>>(D); after_launch(c, CEL_K_PE, n);
    if (c->phys.enable_pair) { k_pair<TR><<<pg, kBlock, 0, s_pair>>>(D); after_launch(c, CEL_K_PAIR, n); }
  }
  const int pgp = by_action ? physics_grid(c, kPhotonGridTimes) : pg;
  if (cyl) k_photon<1, TR><<<pgp, kBlock, 0, s_photon>>>(D); else k_photon<0, TR><<<pgp, kBlock, 0, s_photon>>>(D);
  after_launch(c, CEL_K_PHOTON, n);
  // (in the masked modes the annihilation kernel precedes it on the main stream)
  if (cyl) { if (field) launch_chain(c, k_charged<true, 1, TR>, pg, kBlock, s); else launch_chain(c, k_charged<false, 1, TR>, pg, kBlock, s); }
  else { if (field) launch_chain(c, k_charged<true, 0, TR>, pg, kBlock, s); else launch_chain(c, k_charged<false, 0, TR>, pg, kBlock, s); }
  after_launch(c, CEL_K_CHARGED, n);
  for (int i = 0; i < n_side; ++i) {
    cudaEventRecord(c->ev_join[i], c->side[i]);
    cudaStreamWaitEvent(s, c->ev_join[i], 0);
  }
  enqueue_push_and_flush<TR>(c, n);
  return n;
}
int enqueue_iteration(cel_ctx* c) {
  CEL_RANGE_PUSH("cel:step_iteration");   // P1+P2 fill_sort, P3/P4 action kernels, P5 push (one range per enqueued iteration)
  const int n = c->trace_iters > 0 ? enqueue_iteration_t<true>(c) : enqueue_iteration_t<false>(c);
  CEL_RANGE_POP();
  return n;
}

// profile mode: add the event-to-event times of the `n_iter` iterations of the batch that just ended
int collect_profile(cel_ctx* c, int n_iter, int kernels_per_iteration) {
  const size_t stride = kMaxKernelsPerIteration + 1;
  CEL_CUDA(c, cudaEventSynchronize(c->prof_ev[(size_t)(n_iter - 1) * stride + kernels_per_iteration]));
  for (int b = 0; b < n_iter; ++b)
    for (int i = 0; i < kernels_per_iteration; ++i) {
      float ms = 0.f;
      CEL_CUDA(c, cudaEventElapsedTime(&ms, c->prof_ev[b * stride + i], c->prof_ev[b * stride + i + 1]));
      c->kernel_ms[c->iter_kernel[i]] += ms;
      c->kernel_launches[c->iter_kernel[i]] += 1;
    }
  return CEL_OK;
}

// reset slots, staging, counters and tallies; allocate the run's scratch with the stream-ordered allocator
int prepare_run(cel_ctx* c, uint32_t n_events, bool debug) {
  int rc = lay_out(c);
  if (rc != CEL_OK) return rc;
  c->D.write_vacant = debug ? 1 : 0;   // the complete permutation is only needed by the parity surface
  c->D.bound_tiles = (c->live_tiles && !debug && c->D.sort_mode != CEL_SORT_PARTITION) ? 1 : 0;
  cudaStream_t s = c->stream;
  DeviceState& D = c->D;
  // stream-ordered scratch: freed and re-allocated on the stream, never a device-wide sync
  if (c->scratch) { CEL_CUDA(c, cudaFreeAsync(c->scratch, s)); c->scratch = nullptr; }
  if (c->d_tally) { CEL_CUDA(c, cudaFreeAsync(c->d_tally, s)); c->d_tally = nullptr; }
  const uint64_t tiles = D.n_tiles;
  uint64_t so = 0;
  auto stake = [&](uint64_t bytes) { uint64_t r = so; so = align_up(so + bytes, 256); return r; };
  const uint64_t o_vac = stake(2 * tiles * 4), o_sec = stake(tiles * 4);
  const uint64_t o_hist = stake(tiles * 32), o_phist = stake(tiles * 16), o_rows = stake(2ull * kMaxGroups * kRowWords * 4);
  const uint64_t o_gmask = stake(2ull * (kMaxGroups / 32) * 4), o_part = stake(tiles * 4);
  const uint64_t scratch_bytes = so;
  CEL_CUDA(c, cudaMallocAsync(&c->scratch, scratch_bytes, s));
  const uint64_t tally_bytes = (uint64_t)n_events * (D.P.n_bins + 1) * sizeof(unsigned long long);
  CEL_CUDA(c, cudaMallocAsync(&c->d_tally, tally_bytes > 0 ? tally_bytes : 8, s));
  char* sb = (char*)c->scratch;
  D.tile_vac = (uint32_t*)(sb + o_vac); D.tile_sec = (uint32_t*)(sb + o_sec);
  D.tile_hist = (uint32_t*)(sb + o_hist); D.tile_phist = (uint32_t*)(sb + o_phist);
  D.group_rows = (uint32_t*)(sb + o_rows); D.group_mask = (uint32_t*)(sb + o_gmask); D.part_cnt = (uint32_t*)(sb + o_part);
  D.tally = (unsigned long long*)c->d_tally;
  D.n_events = n_events;
  if (c->d_trace) { CEL_CUDA(c, cudaFreeAsync(c->d_trace, s)); c->d_trace = nullptr; }
  D.trace = nullptr; D.trace_iters = 0; D.trace_ends = (uint32_t)c->trace_ends;
  if (c->trace_iters > 0) {   // [iters][K_COUNT][2]: starts = ~0 (atomicMin), ends = 0 (atomicMax)
    const size_t n = (size_t)c->trace_iters * K_COUNT * 2;
    CEL_CUDA(c, cudaMallocAsync(&c->d_trace, n * 8, s));
    std::vector<unsigned long long> init(n);
    for (size_t i = 0; i < n; ++i) init[i] = (i & 1) ? 0ull : ~0ull;
    CEL_CUDA(c, cudaMemcpyAsync(c->d_trace, init.data(), n * 8, cudaMemcpyHostToDevice, s));
    CEL_CUDA(c, cudaStreamSynchronize(s));   // `init` is pageable host memory (measurement mode only)
    D.trace = (unsigned long long*)c->d_trace; D.trace_iters = (uint32_t)c->trace_iters;
  }
  // hits = 2 reproduces the paper's stall: that needs a BLOCKING stream (one the default stream's
  // synchronous copies synchronise with), so the library's own non-blocking stream is replaced by a blocking one
  if (c->hits_mode == 2 && c->own_stream && !c->stream_blocking) {
    CEL_CUDA(c, cudaStreamSynchronize(c->stream));
    cudaStreamDestroy(c->stream);
    CEL_CUDA(c, cudaStreamCreateWithFlags(&c->stream, cudaStreamDefault));
    c->stream_blocking = true;
    s = c->stream;
    if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
    if (c->graph) { cudaGraphDestroy(c->graph); c->graph = nullptr; }
  }
  // hit transfer: device batch buffer + (mode 1) two pinned, device-mapped host ring buffers; kept from run to run
  D.hits = nullptr; D.hit_capacity = 0; D.host_hits[0] = D.host_hits[1] = nullptr;
  if (c->hits_mode) {
    if (c->d_hits_cap < c->hit_capacity) {
      if (c->d_hits) { CEL_CUDA(c, cudaStreamSynchronize(s)); cudaFree(c->d_hits); c->d_hits = nullptr; c->d_hits_cap = 0; }
      CEL_CUDA(c, cudaMalloc(&c->d_hits, c->hit_capacity * sizeof(cel_hit)));
      c->d_hits_cap = c->hit_capacity;
    }
    if (c->hits_mode == 1 && c->h_ring_cap < c->hit_capacity) {
      consumer_wait_idle(c);
      for (int i = 0; i < 2; ++i) {
        if (c->h_ring[i]) { cudaFreeHost(c->h_ring[i]); c->h_ring[i] = nullptr; }
        CEL_CUDA(c, cudaHostAlloc((void**)&c->h_ring[i], c->hit_capacity * sizeof(cel_hit), cudaHostAllocMapped));
      }
      c->h_ring_cap = c->hit_capacity;
    }
    D.hits = (HitRec*)c->d_hits; D.hit_capacity = c->hit_capacity;
    if (c->hits_mode == 1) {
      for (int i = 0; i < 2; ++i) { void* dp = nullptr; CEL_CUDA(c, cudaHostGetDevicePointer(&dp, c->h_ring[i], 0)); D.host_hits[i] = (HitRec*)dp; }
      if (!c->consumer_on) { c->consumer_stop = false; c->job_pending = false; c->consumer = std::thread(consumer_main, c); c->consumer_on = true; }
    }
    consumer_wait_idle(c);
    c->hits_total = 0; c->hits_qsum = 0; c->hits_bytes = 0;
    c->h_hit_tally.assign(c->hit_tally ? (size_t)n_events * (D.P.n_bins + 1) : 0, 0);
  }
  CEL_CUDA(c, cudaMemsetAsync(c->scratch, 0, scratch_bytes, s));
  CEL_CUDA(c, cudaMemsetAsync(c->d_tally, 0, tally_bytes > 0 ? tally_bytes : 8, s));
  CEL_CUDA(c, cudaMemsetAsync(D.ctl, 0, sizeof(Control), s));
  k_reset_state<<<c->n_sm * 4, 256, 0, s>>>(D);
  CEL_CUDA(c, cudaGetLastError());
  // pinned tally buffer for cel_tallies
  if (c->h_tally_bytes < tally_bytes) {
    if (c->h_tally) cudaFreeHost(c->h_tally);
    c->h_tally = nullptr; c->h_tally_bytes = 0;
    CEL_CUDA(c, cudaMallocHost((void**)&c->h_tally, tally_bytes));
    c->h_tally_bytes = tally_bytes;
  }
  // the iteration as a CUDA graph: kernel arguments (scratch and tally pointers) are baked in, so re-capture per run
  // (the stream-ordered pool hands the same scratch back run after run, so the graph of the last run is normally
  // still valid: it is kept when every baked-in argument and option is unchanged)
  const int cfg[6] = {c->batch, c->concurrent + 2 * c->grid_cap, c->pdl, c->hits_mode, c->trace_iters, c->merge_discrete};
  const bool graph_valid = c->graph_exec && std::memcmp(&c->graph_D, &D, sizeof(DeviceState)) == 0 &&
                           std::memcmp(c->graph_cfg, cfg, sizeof(cfg)) == 0;
  if (!graph_valid) {
    if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
    if (c->graph) { cudaGraphDestroy(c->graph); c->graph = nullptr; }
  }
  for (int i = 0; i < CEL_KERNEL_COUNT; ++i) { c->kernel_ms[i] = 0.0; c->kernel_launches[i] = 0; }
  if (c->profile) {
    const size_t need = (size_t)c->batch * (kMaxKernelsPerIteration + 1);
    while (c->prof_ev.size() < need) {
      cudaEvent_t e = nullptr;
      CEL_CUDA(c, cudaEventCreate(&e));
      c->prof_ev.push_back(e);
    }
  }
  // (hits = 2 launches directly: a blocking default-stream copy cannot coexist with another thread's capture of a blocking stream)
  if (c->use_graph && !c->profile && c->hits_mode != 2 && !graph_valid) {
    // one graph = one batch of iterations: a single cudaGraphLaunch per status poll keeps the host far ahead of the device
    CEL_CUDA(c, cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal));
    for (int b = 0; b < c->batch; ++b) c->kernels_per_iteration = enqueue_iteration(c);
    if (c->hits_mode) k_hits_batch_end<<<1, 1, 0, s>>>(c->D);
    k_status<<<1, 64, 0, s>>>(c->D);
    CEL_CUDA(c, cudaStreamEndCapture(s, &c->graph));
    CEL_CUDA(c, cudaGraphInstantiate(&c->graph_exec, c->graph, 0));
    std::memcpy(&c->graph_D, &D, sizeof(DeviceState));
    std::memcpy(c->graph_cfg, cfg, sizeof(cfg));
  }
  c->launches = 1; c->run_error = 0; c->ran = true;   // k_reset_state
  std::memset(&c->last, 0, sizeof(Control));
  return CEL_OK;
}

int validate_primaries(const cel_ctx* c, const cel_primary* p, uint64_t n, uint32_t n_events) {
  for (uint64_t i = 0; i < n; ++i) {
    if (p[i].event >= n_events || p[i].event >= (1u << 24) || p[i].ptype < 0 || p[i].ptype > 2) return CEL_ERR_INVALID_ARG;
    if (!(p[i].energy_MeV > 0.0) || !std::isfinite(p[i].energy_MeV)) return CEL_ERR_INVALID_ARG;
    const double* d = p[i].dir;
    const double n2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    if (!(std::fabs(n2 - 1.0) <= 1e-12)) return CEL_ERR_INVALID_ARG;
    if (host_locate(c->geo, c->h_bounds.data(), p[i].pos, p[i].dir) < 0) return CEL_ERR_INVALID_ARG;
    if (c->geo.kind == CEL_GEOM_SLAB && (std::fabs(p[i].pos[0]) > c->geo.half_x || std::fabs(p[i].pos[1]) > c->geo.half_y)) return CEL_ERR_INVALID_ARG;
    if (c->geo.kind == CEL_GEOM_CYL && std::fabs(p[i].pos[2]) > c->geo.half_z) return CEL_ERR_INVALID_ARG;
  }
  return CEL_OK;
}

// host primaries -> pinned staging -> device scratch (stream-ordered) -> init[i]
int load_primaries_host(cel_ctx* c, const cel_primary* p, uint64_t n) {
  cudaStream_t s = c->stream;
  const size_t bytes = n * sizeof(cel_primary);
  if (c->h_prim_bytes < bytes) {
    if (c->h_prim) cudaFreeHost(c->h_prim);
    c->h_prim = nullptr; c->h_prim_bytes = 0;
    CEL_CUDA(c, cudaMallocHost(&c->h_prim, bytes));
    c->h_prim_bytes = bytes;
  }
  if (n) std::memcpy(c->h_prim, p, bytes);
  if (c->d_prim) { CEL_CUDA(c, cudaFreeAsync(c->d_prim, s)); c->d_prim = nullptr; }
  CEL_CUDA(c, cudaMallocAsync(&c->d_prim, bytes ? bytes : 64, s));
  if (n) CEL_CUDA(c, cudaMemcpyAsync(c->d_prim, c->h_prim, bytes, cudaMemcpyHostToDevice, s));
  k_load_primaries<<<c->n_sm, 256, 0, s>>>(c->D, (const PrimaryRec*)c->d_prim, n);
  c->no_pdl_next = true;   // (k_fill_sort reads Control::tiles_hi before its dependency wait)
  c->launches += 1;
  CEL_CUDA(c, cudaGetLastError());
  return CEL_OK;
}

// small populations: one single-block kernel runs up to tail_iters whole iterations (cel_tail.cuh)
void launch_tail(cel_ctx* c) {
  const bool cyl = c->D.P.geom_kind == CEL_GEOM_CYL, field = c->D.P.bmag != 0.0;
  const uint32_t n = (uint32_t)c->tail_iters;
  cudaStream_t s = c->stream;
  if (cyl) { if (field) k_tail<true, 1><<<1, kTailThreads, 0, s>>>(c->D, n); else k_tail<false, 1><<<1, kTailThreads, 0, s>>>(c->D, n); }
  else { if (field) k_tail<true, 0><<<1, kTailThreads, 0, s>>>(c->D, n); else k_tail<false, 0><<<1, kTailThreads, 0, s>>>(c->D, n); }
  c->launches += 1; c->tail_launches += 1;
  c->no_pdl_next = true;
}

// enqueue batches of iterations; after each batch copy the control block to pinned memory asynchronously and look
// at the PREVIOUS batch's copy, so the device always has a batch queued while the host decides
int run_loop(cel_ctx* c) {
  cudaStream_t s = c->stream;
  CEL_RANGE_PUSH("cel:transport_loop");
  struct RangeGuard { ~RangeGuard() { CEL_RANGE_POP(); } } range_guard;
  CEL_CUDA(c, cudaEventRecord(c->ev_start, s));
  int64_t enqueued = 0;
  int slot = 0;
  bool have_prev = false;
  int rc = CEL_OK;
  // the single-block form for small populations (option tail): chosen batch by batch from the lagged status
  const bool tail_ok = c->tail && !c->profile && c->hits_mode == 0 && c->trace_iters == 0 && c->D.sort_mode != CEL_SORT_PARTITION;
  bool in_tail = false;
  c->tail_launches = 0;
  while (true) {
    int per_iter = c->kernels_per_iteration;
    if (in_tail) {
      CEL_RANGE_PUSH("cel:tail_batch"); launch_tail(c); CEL_RANGE_POP();
      enqueued += c->tail_iters;
      k_status<<<1, 64, 0, s>>>(c->D); c->launches += 1;
      CEL_CUDA(c, cudaEventRecord(c->ev_batch[slot], s));
      const int prev = slot ^ 1;
      CEL_CUDA(c, cudaEventSynchronize(c->ev_batch[prev]));
      const Control& st = c->h_status[prev];
      if (st.error != 0) { rc = st.error; break; }
      if (st.finished) break;
      in_tail = (uint64_t)st.alive + st.n_init <= (uint64_t)c->tail_enter;
      if (enqueued >= c->max_iterations) { rc = CEL_ERR_MAX_ITER; break; }
      slot ^= 1;
      continue;
    }
    // hits, mode 1: the batch about to be enqueued streams into the ring buffer the consumer read two batches ago
    if (c->hits_mode == 1) consumer_wait_idle(c);
    if (c->graph_exec && c->use_graph && !c->profile && c->hits_mode != 2) {
      CEL_CUDA(c, cudaGraphLaunch(c->graph_exec, s));
      c->launches += (uint64_t)c->kernels_per_iteration * c->batch + (c->hits_mode ? 1 : 0) + 1;   // (+ k_status)
    } else {
      for (int b = 0; b < c->batch; ++b) {
        c->prof_b = b;
        per_iter = enqueue_iteration(c); c->launches += per_iter;
      }
      if (c->hits_mode) { k_hits_batch_end<<<1, 1, 0, s>>>(c->D); c->launches += 1; }
      if (c->hits_mode != 2) { k_status<<<1, 64, 0, s>>>(c->D); c->launches += 1; }
    }
    c->prof_b = 0;
    enqueued += c->batch;
    if (c->profile) { int prc = collect_profile(c, c->batch, per_iter); if (prc != CEL_OK) return prc; }
    if (c->hits_mode == 2) {
      // the paper's "before": wait for the batch, then a blocking copy on the default stream into pageable
      // memory — a device-wide synchronisation for every stream that is not non-blocking — and process the hits inline
      CEL_CUDA(c, cudaStreamSynchronize(s));
      Control st;
      CEL_CUDA(c, cudaMemcpy(&st, c->D.ctl, sizeof(Control), cudaMemcpyDeviceToHost));
      if (st.hits_in_batch) {
        if (c->h_pageable.size() < st.hits_in_batch) c->h_pageable.resize(st.hits_in_batch);
        CEL_CUDA(c, cudaMemcpy(c->h_pageable.data(), c->d_hits, st.hits_in_batch * sizeof(cel_hit), cudaMemcpyDeviceToHost));
        consume_hits(c, c->h_pageable.data(), st.hits_in_batch);
      }
      if (st.error != 0) { rc = st.error; break; }
      if (st.finished) break;
      if (enqueued >= c->max_iterations) { rc = CEL_ERR_MAX_ITER; break; }
      continue;
    }
    CEL_CUDA(c, cudaEventRecord(c->ev_batch[slot], s));   // (behind k_status, which has written h_status[slot])
    if (have_prev) {
      const int prev = slot ^ 1;
      CEL_CUDA(c, cudaEventSynchronize(c->ev_batch[prev]));
      const Control& st = c->h_status[prev];
      if (c->hits_mode == 1 && st.hits_in_batch) consumer_submit(c, c->h_ring[st.hits_buf & 1u], st.hits_in_batch);
      if (st.error != 0) { rc = st.error; break; }
      if (st.finished) break;
      in_tail = tail_ok && st.iterations > 0 && (uint64_t)st.alive + st.n_init <= (uint64_t)c->tail_enter;
    }
    if (enqueued >= c->max_iterations) { rc = CEL_ERR_MAX_ITER; break; }
    have_prev = true;
    slot ^= 1;
  }
  CEL_CUDA(c, cudaGetLastError());
  CEL_CUDA(c, cudaEventRecord(c->ev_stop, s));
  c->run_error = rc;
  return rc;
}

}  // namespace

extern "C" int cel_transport(cel_ctx* c, const cel_primary* primaries, uint64_t n, uint32_t n_events) {
  if (!c || (!primaries && n) || n_events < 1 || n_events > (1u << 24) || n > c->D.init_capacity) return CEL_ERR_INVALID_ARG;
  int rc = validate_primaries(c, primaries, n, n_events);
  if (rc != CEL_OK) return rc;
  if ((rc = prepare_run(c, n_events, false)) != CEL_OK) return rc;
  if ((rc = load_primaries_host(c, primaries, n)) != CEL_OK) return rc;
  return run_loop(c);
}

extern "C" int cel_transport_device(cel_ctx* c, const void* d_primaries, uint64_t n, uint32_t n_events) {
  if (!c || (!d_primaries && n) || n_events < 1 || n_events > (1u << 24) || n > c->D.init_capacity) return CEL_ERR_INVALID_ARG;
  int rc = prepare_run(c, n_events, false);
  if (rc != CEL_OK) return rc;
  k_load_primaries<<<c->n_sm, 256, 0, c->stream>>>(c->D, (const PrimaryRec*)d_primaries, n);
  c->no_pdl_next = true;   // (k_fill_sort reads Control::tiles_hi before its dependency wait)
  c->launches += 1;
  CEL_CUDA(c, cudaGetLastError());
  return run_loop(c);
}

extern "C" int cel_tallies(cel_ctx* c, cel_tally_view* out) {
  if (!c || !out) return CEL_ERR_INVALID_ARG;
  if (!c->ran) return CEL_ERR_NOT_RUN;
  cudaStream_t s = c->stream;
  const DeviceState& D = c->D;
  const uint64_t bytes = (uint64_t)D.n_events * (D.P.n_bins + 1) * sizeof(unsigned long long);
  CEL_CUDA(c, cudaMemcpyAsync(c->h_tally, D.tally, bytes, cudaMemcpyDeviceToHost, s));
  CEL_CUDA(c, cudaMemcpyAsync(&c->h_status[0], D.ctl, sizeof(Control), cudaMemcpyDeviceToHost, s));
  CEL_CUDA(c, cudaStreamSynchronize(s));
  c->last = c->h_status[0];
  out->n_events = D.n_events; out->n_bins = D.P.n_bins; out->fixed = c->h_tally;
  out->track_steps = c->last.track_steps; out->iterations = c->last.iterations; out->secondaries = c->last.secondaries;
  float ms = 0.f;
  out->seconds = (cudaEventElapsedTime(&ms, c->ev_start, c->ev_stop) == cudaSuccess) ? ms * 1e-3 : 0.0;
  out->kernel_launches = c->launches;
  if (c->last.error != 0) return c->last.error;
  return c->run_error;
}

extern "C" int cel_set_hit_callback(cel_ctx* c, cel_hit_callback fn, void* user) {
  if (!c) return CEL_ERR_INVALID_ARG;
  consumer_wait_idle(c);
  c->hit_cb = fn; c->hit_cb_user = user;
  return CEL_OK;
}

extern "C" int cel_hit_tallies(cel_ctx* c, cel_hit_view* out) {
  if (!c || !out) return CEL_ERR_INVALID_ARG;
  if (!c->ran) return CEL_ERR_NOT_RUN;
  CEL_CUDA(c, cudaStreamSynchronize(c->stream));
  consumer_wait_idle(c);
  out->n_hits = c->hits_total; out->q_sum = c->hits_qsum; out->bytes_d2h = c->hits_bytes;
  out->n_events = c->D.n_events; out->n_bins = c->D.P.n_bins;
  out->fixed = c->h_hit_tally.empty() ? nullptr : c->h_hit_tally.data();
  return c->run_error;
}

extern "C" int cel_trace(cel_ctx* c, uint64_t* host_out, uint64_t* n_iters) {
  if (!c || !n_iters) return CEL_ERR_INVALID_ARG;
  if (!c->ran) return CEL_ERR_NOT_RUN;
  CEL_CUDA(c, cudaStreamSynchronize(c->stream));
  const uint64_t n = c->d_trace ? (uint64_t)c->D.trace_iters : 0;
  *n_iters = n;
  if (host_out && n) CEL_CUDA(c, cudaMemcpy(host_out, c->d_trace, n * K_COUNT * 2 * 8, cudaMemcpyDeviceToHost));
  return CEL_OK;
}

extern "C" int cel_kernel_count(void) { return CEL_KERNEL_COUNT; }
extern "C" const char* cel_kernel_name(int id) { return (id >= 0 && id < CEL_KERNEL_COUNT) ? kKernelNames[id] : ""; }
extern "C" int cel_kernel_times(cel_ctx* c, double* ms_out, uint64_t* launches_out) {
  if (!c || !ms_out || !launches_out) return CEL_ERR_INVALID_ARG;
  if (!c->ran) return CEL_ERR_NOT_RUN;
  for (int i = 0; i < CEL_KERNEL_COUNT; ++i) { ms_out[i] = c->kernel_ms[i]; launches_out[i] = c->kernel_launches[i]; }
  return CEL_OK;
}

// ================================================================ debug / parity surface (synchronous)
extern "C" int cel_debug_begin(cel_ctx* c, const cel_primary* primaries, uint64_t n, uint32_t n_events) {
  if (!c || (!primaries && n) || n_events < 1 || n_events > (1u << 24) || n > c->D.init_capacity) return CEL_ERR_INVALID_ARG;
  int rc = validate_primaries(c, primaries, n, n_events);
  if (rc != CEL_OK) return rc;
  if ((rc = prepare_run(c, n_events, true)) != CEL_OK) return rc;
  if ((rc = load_primaries_host(c, primaries, n)) != CEL_OK) return rc;
  CEL_CUDA(c, cudaEventRecord(c->ev_start, c->stream));
  CEL_CUDA(c, cudaEventRecord(c->ev_stop, c->stream));
  CEL_CUDA(c, cudaStreamSynchronize(c->stream));
  return CEL_OK;
}

extern "C" int cel_debug_step(cel_ctx* c) {
  if (!c || !c->ran) return CEL_ERR_NOT_RUN;
  c->launches += enqueue_iteration(c);
  CEL_CUDA(c, cudaGetLastError());
  CEL_CUDA(c, cudaMemcpyAsync(&c->h_status[0], c->D.ctl, sizeof(Control), cudaMemcpyDeviceToHost, c->stream));
  CEL_CUDA(c, cudaStreamSynchronize(c->stream));
  c->last = c->h_status[0];
  return c->last.error;
}

namespace {
int unpack_to_host(cel_ctx* c, const RecA* A, const RecB* B, uint64_t n, int as_init, cel_track* host_out) {
  if (n == 0) return CEL_OK;
  void* d = nullptr;
  CEL_CUDA(c, cudaMallocAsync(&d, n * sizeof(TrackRec), c->stream));
  k_unpack<<<c->n_sm * 2, 256, 0, c->stream>>>(A, B, (TrackRec*)d, n, as_init);
  CEL_CUDA(c, cudaGetLastError());
  CEL_CUDA(c, cudaMemcpyAsync(host_out, d, n * sizeof(TrackRec), cudaMemcpyDeviceToHost, c->stream));
  CEL_CUDA(c, cudaFreeAsync(d, c->stream));
  CEL_CUDA(c, cudaStreamSynchronize(c->stream));
  return CEL_OK;
}
int fetch_control(cel_ctx* c) {
  CEL_CUDA(c, cudaMemcpyAsync(&c->h_status[0], c->D.ctl, sizeof(Control), cudaMemcpyDeviceToHost, c->stream));
  CEL_CUDA(c, cudaStreamSynchronize(c->stream));
  c->last = c->h_status[0];
  return CEL_OK;
}
}  // namespace

extern "C" int cel_debug_read_state(cel_ctx* c, cel_track* host_out) {
  if (!c || !host_out) return CEL_ERR_INVALID_ARG;
  if (!c->ran) return CEL_ERR_NOT_RUN;
  return unpack_to_host(c, c->D.stA, c->D.stB, c->n_slots, 0, host_out);
}

extern "C" int cel_debug_read_indices(cel_ctx* c, uint32_t* idx, uint32_t* offsets) {
  if (!c || !idx || !offsets) return CEL_ERR_INVALID_ARG;
  if (!c->ran) return CEL_ERR_NOT_RUN;
  int rc = fetch_control(c);
  if (rc != CEL_OK) return rc;
  std::memcpy(offsets, c->last.offsets, 9 * sizeof(uint32_t));
  if (c->D.sort_mode == CEL_SORT_NONE || c->D.sort_mode == CEL_SORT_PARTITION) {
    for (uint64_t i = 0; i < c->n_slots; ++i) idx[i] = (uint32_t)i;
  } else {   // the index array is kept in regions of N entries per sort key: compact them into the permutation of S2
    const int n_keys = c->D.sort_mode == CEL_SORT_BY_ACTION ? 8 : 4;
    for (int k = 0; k < n_keys; ++k) {
      const uint32_t n = offsets[k + 1] - offsets[k];
      if (n) CEL_CUDA(c, cudaMemcpyAsync(idx + offsets[k], c->D.indices + (uint64_t)k * c->n_slots, (uint64_t)n * sizeof(uint32_t), cudaMemcpyDeviceToHost, c->stream));
    }
    CEL_CUDA(c, cudaStreamSynchronize(c->stream));
  }
  return CEL_OK;
}

extern "C" int cel_debug_n_initializers(cel_ctx* c, uint64_t* n) {
  if (!c || !n) return CEL_ERR_INVALID_ARG;
  if (!c->ran) return CEL_ERR_NOT_RUN;
  int rc = fetch_control(c);
  *n = c->last.n_init;
  return rc;
}

extern "C" int cel_debug_read_initializers(cel_ctx* c, cel_track* host_out) {
  if (!c || !host_out) return CEL_ERR_INVALID_ARG;
  if (!c->ran) return CEL_ERR_NOT_RUN;
  int rc = fetch_control(c);
  if (rc != CEL_OK) return rc;
  return unpack_to_host(c, c->D.initA, c->D.initB, c->last.n_init, 1, host_out);
}

extern "C" int cel_debug_n_counts(cel_ctx* c, uint64_t* n) {
  if (!c || !n) return CEL_ERR_INVALID_ARG;
  if (!c->ran) return CEL_ERR_NOT_RUN;
  int rc = fetch_control(c);
  *n = c->last.n_logged;
  return rc;
}

extern "C" int cel_debug_read_counts(cel_ctx* c, uint32_t* host_out) {
  if (!c || !host_out) return CEL_ERR_INVALID_ARG;
  if (!c->ran) return CEL_ERR_NOT_RUN;
  int rc = fetch_control(c);
  if (rc != CEL_OK) return rc;
  if (c->last.n_logged) {
    CEL_CUDA(c, cudaMemcpyAsync(host_out, c->D.counts_log, (uint64_t)c->last.n_logged * 8 * sizeof(uint32_t), cudaMemcpyDeviceToHost, c->stream));
    CEL_CUDA(c, cudaStreamSynchronize(c->stream));
  }
  return CEL_OK;
}

extern "C" int cel_debug_table(cel_ctx* c, int material, int which, double* out577) {
  if (!c || !out577 || material < 0 || material >= c->n_mats || which < 0 || which > 4) return CEL_ERR_INVALID_ARG;
  // read back what the kernels actually use (device copy), not the host vector
  const Params& P = c->D.P;
  std::vector<double> tmp;
  if (which <= 2) {
    std::vector<PhotonXs> px(kGrid);
    CEL_CUDA(c, cudaMemcpy(px.data(), P.photon_xs + (size_t)material * kGrid, kGrid * sizeof(PhotonXs), cudaMemcpyDeviceToHost));
    for (int j = 0; j < kGrid; ++j) out577[j] = which == 0 ? px[j].compton : (which == 1 ? px[j].pe : px[j].pair);
  } else if (which == 3) {
    std::vector<ChargedXs> cx(kGrid);
    CEL_CUDA(c, cudaMemcpy(cx.data(), P.charged_xs + (size_t)material * kGrid, kGrid * sizeof(ChargedXs), cudaMemcpyDeviceToHost));
    for (int j = 0; j < kGrid; ++j) out577[j] = cx[j].brems;
  } else {
    CEL_CUDA(c, cudaMemcpy(out577, P.range_tab + (size_t)material * kGrid, kGrid * sizeof(double), cudaMemcpyDeviceToHost));
  }
  return CEL_OK;
}

extern "C" int cel_debug_uniforms(cel_ctx* c, const uint32_t* slots, uint32_t n, uint32_t k, uint32_t phase, uint32_t j, double* host_out) {
  if (!c || !slots || !host_out) return CEL_ERR_INVALID_ARG;
  if (n == 0) return CEL_OK;
  void* ds = nullptr; void* dout = nullptr;
  CEL_CUDA(c, cudaMallocAsync(&ds, n * sizeof(uint32_t), c->stream));
  CEL_CUDA(c, cudaMallocAsync(&dout, n * sizeof(double), c->stream));
  CEL_CUDA(c, cudaMemcpyAsync(ds, slots, n * sizeof(uint32_t), cudaMemcpyHostToDevice, c->stream));
  k_debug_uniforms<<<(n + 255) / 256, 256, 0, c->stream>>>(c->D.P, (const uint32_t*)ds, n, k, phase, j, (double*)dout);
  CEL_CUDA(c, cudaGetLastError());
  CEL_CUDA(c, cudaMemcpyAsync(host_out, dout, n * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  CEL_CUDA(c, cudaFreeAsync(ds, c->stream));
  CEL_CUDA(c, cudaFreeAsync(dout, c->stream));
  CEL_CUDA(c, cudaStreamSynchronize(c->stream));
  return CEL_OK;
}

extern "C" int cel_debug_math(cel_ctx* c, int which, const double* host_in, uint32_t n, double* host_out) {
  if (!c || !host_in || !host_out || which < 0 || which > 1) return CEL_ERR_INVALID_ARG;
  if (n == 0) return CEL_OK;
  void* din = nullptr; void* dout = nullptr;
  CEL_CUDA(c, cudaMallocAsync(&din, n * sizeof(double), c->stream));
  CEL_CUDA(c, cudaMallocAsync(&dout, n * sizeof(double), c->stream));
  CEL_CUDA(c, cudaMemcpyAsync(din, host_in, n * sizeof(double), cudaMemcpyHostToDevice, c->stream));
  k_debug_math<<<(n + 255) / 256, 256, 0, c->stream>>>(which, (const double*)din, n, (double*)dout);
  CEL_CUDA(c, cudaGetLastError());
  CEL_CUDA(c, cudaMemcpyAsync(host_out, dout, n * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  CEL_CUDA(c, cudaFreeAsync(din, c->stream));
  CEL_CUDA(c, cudaFreeAsync(dout, c->stream));
  CEL_CUDA(c, cudaStreamSynchronize(c->stream));
  return CEL_OK;
}

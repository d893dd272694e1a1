// cel_device.cuh — device-side data layout and physics primitives of the celstep CUDA path (sm_100a).
// Implements docs/PHYSICS_SPEC.md S0-S8 independently of the CPU oracle (no shared code or headers).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace cel {

// ---------------------------------------------------------------- S0 constants
constexpr double kElectronMass = 0.51099895;
constexpr double kClassicalRadius = 2.8179403262e-13;
constexpr double kAvogadro = 6.02214076e23;
constexpr double kFineStructure = 7.2973525693e-3;
constexpr double kKappa = 2.99792458;
constexpr double kAlphaR = 0.2;
constexpr double kRhoF = 0.01;
constexpr double kDeltaChord = 1e-3;
constexpr double kPi = 3.14159265358979323846;
constexpr double kTallyScale = 68719476736.0;  // 2^36
constexpr int kGrid = 577;

enum : int { A_PE = 0, A_PAIR = 1, A_COMPTON = 2, A_MOVE_G = 3, A_MOVE_C = 4, A_BREMS = 5, A_ANNIH = 6, A_VACANT = 7 };
enum : int { P_GAMMA = 0, P_ELECTRON = 1, P_POSITRON = 2 };
enum : uint32_t { PH_INTERACT = 0, PH_STEP = 1, PH_MSC = 2 };

// ---------------------------------------------------------------- HBM layout
// A slot's state is two 32-byte, 32-byte-aligned records, so that a gathered slot costs exactly two
// sectors read and two written (the +344 % memory operations of PAPER.md:47 are sector amplification
// of a field-per-array SoA under the index indirection).
struct __align__(32) RecA { double x, y, z, energy; };
struct __align__(32) RecB { double dx, dy, dz; unsigned long long meta; };
// meta: bits 0-3 action | 4-5 ptype | 8-15 vol | 16-23 surf (0xff = none) | 24-39 nsteps | 40-63 event

__device__ __forceinline__ int meta_action(unsigned long long m) { return (int)(m & 0xfull); }
__device__ __forceinline__ int meta_ptype(unsigned long long m) { return (int)((m >> 4) & 0x3ull); }
__device__ __forceinline__ int meta_vol(unsigned long long m) { return (int)((m >> 8) & 0xffull); }
__device__ __forceinline__ int meta_surf(unsigned long long m) { int s = (int)((m >> 16) & 0xffull); return s == 0xff ? -1 : s; }
__device__ __forceinline__ uint32_t meta_nsteps(unsigned long long m) { return (uint32_t)((m >> 24) & 0xffffull); }
__device__ __forceinline__ uint32_t meta_event(unsigned long long m) { return (uint32_t)(m >> 40); }
__host__ __device__ __forceinline__ unsigned long long make_meta(int action, int ptype, int vol, int surf, uint32_t nsteps, uint32_t event) {
  return (unsigned long long)(action & 0xf) | ((unsigned long long)(ptype & 0x3) << 4) |
         ((unsigned long long)(vol & 0xff) << 8) | ((unsigned long long)((surf < 0 ? 0xff : surf) & 0xff) << 16) |
         ((unsigned long long)(nsteps & 0xffff) << 24) | ((unsigned long long)event << 40);
}
// the dense key byte read by the scans: low nibble action, bits 4-5 particle type
__host__ __device__ __forceinline__ uint8_t make_key(int action, int ptype) { return (uint8_t)((action & 0xf) | ((ptype & 0x3) << 4)); }

// 256-bit global loads/stores (sm_100: LDG.E.256 / STG.E.256)
__device__ __forceinline__ RecA load_a(const RecA* p) {
  RecA r;
  asm volatile("ld.global.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.energy) : "l"(p));
  return r;
}
__device__ __forceinline__ void store_a(RecA* p, const RecA& r) {
  asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(r.x), "d"(r.y), "d"(r.z), "d"(r.energy) : "memory");
}
__device__ __forceinline__ RecB load_b(const RecB* p) {
  long long a, b, c; unsigned long long m;
  asm volatile("ld.global.v4.b64 {%0,%1,%2,%3}, [%4];" : "=l"(a), "=l"(b), "=l"(c), "=l"(m) : "l"(p));
  RecB r; r.dx = __longlong_as_double(a); r.dy = __longlong_as_double(b); r.dz = __longlong_as_double(c); r.meta = m;
  return r;
}
__device__ __forceinline__ void store_b(RecB* p, const RecB& r) {
  asm volatile("st.global.v4.b64 [%0], {%1,%2,%3,%4};" ::"l"(p), "l"(__double_as_longlong(r.dx)), "l"(__double_as_longlong(r.dy)),
               "l"(__double_as_longlong(r.dz)), "l"(r.meta) : "memory");
}
// ---------------------------------------------------------------- per-context read-only device data
struct MaterialDev { double inv_X0; };
struct PhotonXs { double compton, pe, pair, pad; };   // one grid node, 32 B
struct ChargedXs { double brems, range; };            // one grid node, 16 B

struct Params {
  // geometry
  int geom_kind, n_vol, n_bins;
  const double* bounds;        // n_vol+1
  const int* vol_material;     // n_vol
  const int* vol_bin;          // n_vol
  double half_x, half_y, half_z;
  double bmag, bhx, bhy, bhz;
  // physics
  uint32_t key0, key1;
  double cut;
  int enable_msc, enable_eloss, enable_annihilation, electrons_local, max_substeps;
  uint32_t max_steps_per_track;
  double u0, inv_du, du;
  const MaterialDev* mats;
  const PhotonXs* photon_xs;   // [n_mats][kGrid]
  const ChargedXs* charged_xs; // [n_mats][kGrid]
  const double* range_tab;     // [n_mats][kGrid]
  const double* energy_nodes;  // [kGrid] E_j = exp(u_j)
};

// ---------------------------------------------------------------- per-run device state
// Bookkeeping tiles: a tile is `tile_slots` = 2^tile_shift consecutive slots, processed by one block in sub-tiles of
// kSub slots; tiles are grouped by kGroupTiles for the two-level counters (cel_kernels.cuh). The tile size grows with N
// so that there are never more than kMaxGroups groups.
constexpr int kTileThreads = 256;
constexpr int kKeysPerThread = 4;
constexpr int kSub = kTileThreads * kKeysPerThread;  // 1024 slots per sub-tile
constexpr int kGroupTiles = 32;
constexpr int kMaxGroups = 256;
constexpr int kMaxTiles = kMaxGroups * kGroupTiles;  // 8192
constexpr int kRowWords = 16;                        // one group row: 8 action counts, 4 particle-key counts, arrivals, tile mask, pad

// index ranges of the action kernels in the index array (S2); each kernel walks up to two ranges
enum KernelRange : int { R_PE = 0, R_PAIR, R_ANNIH, R_PHOTON, R_CHARGED, R_COUNT };

struct Control {
  unsigned long long n_init;        // I, the initializer stack height
  unsigned long long track_steps, iterations, secondaries;
  unsigned long long push_total;    // S of this iteration
  uint32_t iter;                    // k
  uint32_t alive;                   // A_k (after P1)
  uint32_t finished;                // A_k == 0 and I == 0
  int32_t error;
  uint32_t offsets[9];              // compact offsets of the sorted index array, per sort key (S2; debug surface)
  uint32_t counts[8];               // action counts of this iteration (after P1)
  uint32_t rb[R_COUNT][2], re[R_COUNT][2];   // index ranges of each action kernel for this iteration (KernelRange)
  uint32_t n_logged;
  uint32_t vac_total;               // V before the fill of this iteration
  unsigned long long n_init_fill;   // I after the fill of this iteration (= n_init until k_push adds S)
  uint32_t iter_cur;                // k of the running iteration, a copy k_push may read while its block 0 bumps iter
  uint32_t part_charged;            // sort mode 3: charged initializers among the n_take popped in this iteration
  uint32_t tiles_hi[2];             // [k&1] = live tiles of iteration k: every tile at or above it is entirely vacant (cel_kernels.cuh)
  uint32_t vac_low[2];              // [k&1] = vacancies below tiles_hi[(k-1)&1] when iteration k begins
  // hit transfer (option "hits")
  unsigned long long n_hits;        // hit records appended to the device batch buffer since the batch began
  unsigned long long hits_mark[2];  // [k&1] = records already streamed to the host when iteration k's flush starts
  unsigned long long hits_in_batch; // set by k_hits_batch_end: records of the batch that just ended ...
  uint32_t hits_buf;                // ... and the host ring buffer (0/1) they were streamed into
  uint32_t hits_cur;                // the host ring buffer the running batch streams into
  uint32_t status_seq;              // batches whose status k_status has published to the host (its slot = status_seq & 1)
};

// one hit = one quantised deposit of one track in one iteration (S10): what the paper's application copies to the host
// at every step iteration for the user's sensitive detectors. = cel_hit of include/cel.h, 16 bytes.
struct HitRec { uint32_t event; int32_t bin; unsigned long long q; };

// everything a kernel needs; passed by value (fits in the 4 KB parameter space)
struct DeviceState {
  Params P;
  uint32_t N;             // n_slots
  uint32_t n_tiles;
  uint32_t n_groups;      // ceil(n_tiles / kGroupTiles)
  uint32_t tile_shift;    // log2(tile_slots)
  uint32_t subs_per_tile; // tile_slots / kSub
  int sort_mode;          // 0 none, 1 by action, 2 by particle, 3 partition (CEL_SORT_BY_ACTION_REUSE is 1 here, with reuse = 1)
  int reuse;              // S9-R: a slot vacated by its interaction takes its first secondary in place
  int write_vacant;       // 1 = also write the indices of vacant slots (complete permutation, debug surface)
  int bound_tiles;        // 1 = the bookkeeping kernels walk the live tiles only (Control::tiles_hi); 0 = every tile
  int vac_buf_override;   // 0: vacancies created in iteration k go to the counters of parity (k&1)^1; 1 + p: to parity p (k_tail)
  unsigned long long init_capacity;
  uint32_t n_events;
  uint32_t log_capacity;
  RecA* stA; RecB* stB;
  uint8_t* akey;          // [n_tiles * tile_slots] action | ptype << 4; padding bytes are 0xff
  uint8_t* nsec;          // [n_tiles * tile_slots] secondaries staged by the slot in this iteration (0..2)
  uint32_t* indices;      // sorted modes: [n_keys][N], region k = the slots of sort key k in ascending order (state_indices,
                          // PAPER.md:41, kept per key so that a tile's write position depends only on the tiles before it);
                          // sort mode 3: [N] the partitioned pop positions (plist, S9-P)
  RecA* secA; RecB* secB; // [2N] staged secondaries
  RecA* initA; RecB* initB; // [init_capacity]
  unsigned long long* tally; // [n_events][n_bins+1]
  uint32_t* counts_log;   // [log_capacity][8]
  Control* ctl;
  // stream-ordered scratch (cudaMallocAsync, per transport call)
  uint32_t* tile_vac;     // [2][n_tiles] vacant slots per tile, double-buffered by iteration parity (cel_kernels.cuh)
  uint32_t* tile_sec;     // [n_tiles] secondaries staged per tile in this iteration: += by the action kernels
  uint32_t* tile_hist;    // [n_tiles][8] per-tile action histogram
  uint32_t* tile_phist;   // [n_tiles][4] per-tile particle-key histogram (sort by particle)
  uint32_t* group_rows;   // [2][kMaxGroups][kRowWords] group histograms + arrival counters, double-buffered by iteration parity
  uint32_t* group_mask;   // [2][kMaxGroups / 32] bit g = every tile of group g has published its rows of this iteration
  uint32_t* part_cnt;     // [n_tiles] sort mode 3: charged pops per tile-sized chunk of the popped segment
  // hit transfer (option "hits"): device batch buffer the action kernels append to, the two pinned host ring buffers
  // (device-mapped) k_hits_flush streams it into; nullptr = off
  HitRec* hits; unsigned long long hit_capacity;
  HitRec* host_hits[2];
  Control* status_host;   // [2] pinned, device-mapped: where k_status publishes the control block at the end of a batch of iterations
  // device-side timeline (option "trace", fig. 2): [trace_iters][K_COUNT][2] globaltimer ns, first block
  // in / last warp out of every kernel of every iteration; nullptr = off
  unsigned long long* trace;
  uint32_t trace_iters;
  uint32_t trace_ends;    // 0 = start stamps only (no end-of-kernel atomics: the least perturbing form)
};

// kernel ids of the timeline and of cel_kernel_times (= CEL_K_* of include/cel.h, checked in cel_api.cu)
enum KernelId : int { K_FILL_SORT = 0, K_ANNIH, K_PE, K_PAIR, K_PHOTON, K_CHARGED, K_PUSH, K_PART_COUNT, K_PART_SCATTER, K_DISCRETE, K_HITS_FLUSH, K_TAIL, K_COUNT };

__device__ __forceinline__ unsigned long long globaltimer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
  return t;
}
// scope object of a kernel body: stamps the kernel's [start, end] of iteration `iter` when tracing is on. One global
// atomic per block and stamp at most: the block's warps count themselves out in shared memory and the last one stamps
// the end; a plain read first skips the atomic when the stamp cannot change. Holds no pointer (the stamp address is
// recomputed from the kernel parameters). Every kernel is compiled twice, TRACE = false being an empty object, so that
// the untraced path keeps its code and its register count.
template <int KID, bool TRACE>
struct TraceScope {
  __device__ __forceinline__ TraceScope(const DeviceState&, uint32_t) {}
};
template <int KID>
struct TraceScope<KID, true> {
  const DeviceState& D;
  const uint32_t iter;
  static __device__ __forceinline__ unsigned int* done_counter() { __shared__ unsigned int s_done; return &s_done; }
  __device__ __forceinline__ unsigned long long* stamp() const { return D.trace + ((size_t)iter * K_COUNT + KID) * 2; }
  __device__ __forceinline__ bool on() const { return D.trace != nullptr && iter < D.trace_iters; }
  __device__ __forceinline__ TraceScope(const DeviceState& D_, uint32_t iter_) : D(D_), iter(iter_) {
    if (on()) {   // block-uniform
      if (threadIdx.x == 0) {
        *done_counter() = 0;
        const unsigned long long now = globaltimer_ns();
        if (now < *reinterpret_cast<volatile unsigned long long*>(stamp())) atomicMin(stamp(), now);
      }
      __syncthreads();
    }
  }
  __device__ __forceinline__ ~TraceScope() {
    if (on() && D.trace_ends && (threadIdx.x & 31) == 0) {
      const unsigned int warps = (blockDim.x + 31) >> 5;
      if (atomicAdd(done_counter(), 1u) == warps - 1) {
        const unsigned long long now = globaltimer_ns();
        if (now > *reinterpret_cast<volatile unsigned long long*>(stamp() + 1)) atomicMax(stamp() + 1, now);
      }
    }
  }
};

// ---------------------------------------------------------------- programmatic dependent launch (sm_90+)
// The kernels of the main-stream chain (fill_sort -> charged -> push -> next fill_sort) are launched with the
// programmatic-stream-serialization attribute: a kernel lets its successor's blocks be scheduled early
// (launch_dependents) and waits itself, before touching any memory, until its predecessors have completed and
// flushed (wait). Without the attribute both instructions are no-ops.
__device__ __forceinline__ void pdl_prologue() {
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}

// ---------------------------------------------------------------- S3 Philox4x32-10
struct Philox4 { uint32_t w[4]; };

__device__ __forceinline__ Philox4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  Philox4 o; o.w[0] = c0; o.w[1] = c1; o.w[2] = c2; o.w[3] = c3;
  return o;
}
__device__ __forceinline__ double to_uniform(uint32_t lo, uint32_t hi) {
  // ((x >> 12) + 0.5) * 2^-52, exactly: the 52 bits become the mantissa of a double in [1, 2); subtracting 1 and adding
  // 2^-53 are both exact (the sum has at most 53 significant bits below 1)
  const unsigned long long x = ((unsigned long long)hi << 32) | lo;
  return (__longlong_as_double((long long)(0x3ff0000000000000ull | (x >> 12))) - 1.0) + 1.1102230246251565e-16;
}
// the two draws (2b, 2b+1) of block b of a phase
__device__ __forceinline__ void draw_pair(const Params& P, uint32_t slot, uint32_t k, uint32_t phase, uint32_t block, double& xa, double& xb) {
  Philox4 o = philox4x32_10(slot, k, phase, block, P.key0, P.key1);
  xa = to_uniform(o.w[0], o.w[1]);
  xb = to_uniform(o.w[2], o.w[3]);
}

// ---------------------------------------------------------------- small-angle trigonometry of the helix substep
// sin x / x and (1 - cos x) / x^2 for |x| <= 0.5 (the helix angle of one chord substep, S7.3: h <= 0.5 / |omega|):
// Taylor polynomials in y = x^2 <= 0.25, truncation < 1e-18; no argument reduction, no cancellation in 1 - cos
__device__ __forceinline__ void sinc_versc_small(double y, double& S, double& V) {
  double s = -1.0 / 1307674368000.0;                                 // -1/15!
  s = fma(s, y, 1.0 / 6227020800.0); s = fma(s, y, -1.0 / 39916800.0); s = fma(s, y, 1.0 / 362880.0);
  s = fma(s, y, -1.0 / 5040.0); s = fma(s, y, 1.0 / 120.0); s = fma(s, y, -1.0 / 6.0); s = fma(s, y, 1.0);
  double v = 1.0 / 20922789888000.0;                                 // 1/16!
  v = fma(v, y, -1.0 / 87178291200.0); v = fma(v, y, 1.0 / 479001600.0); v = fma(v, y, -1.0 / 3628800.0);
  v = fma(v, y, 1.0 / 40320.0); v = fma(v, y, -1.0 / 720.0); v = fma(v, y, 1.0 / 24.0); v = fma(v, y, -0.5);
  S = s; V = -v;
}

// ---------------------------------------------------------------- S4 table lookups
struct GridPos { int j; double f; };
__device__ __forceinline__ GridPos grid_locate(const Params& P, double E) {
  double t = (log(E) - P.u0) * P.inv_du;
  double fl = floor(t);
  int j = fl < 0.0 ? 0 : (fl > 575.0 ? 575 : (int)fl);
  GridPos g; g.j = j; g.f = t - (double)j;
  return g;
}
__device__ __forceinline__ double lerp_node(double y0, double y1, double f) { return y0 + f * (y1 - y0); }

// Rinv(r): largest j <= 575 with R_j <= r, scanning down from j_hint (the cell of the pre-step energy; r <= R(T0))
__device__ __forceinline__ double range_inverse(const Params& P, const double* __restrict__ R, double r, int j_hint) {
  // gallop down from the hint (r is usually within a few cells of it: one step costs at most 20 % of the range),
  // then bisect: a handful of loads for every lane instead of a per-lane linear scan. R is strictly increasing, so
  // this is the same j as the plain downward scan.
  int j = j_hint;
  if (__ldg(R + j) > r) {
    int hi = j, step = 1;                      // invariant: R[hi] > r
    int lo = hi - 1;
    while (lo > 0 && __ldg(R + lo) > r) { hi = lo; step <<= 1; lo = hi - step; if (lo < 0) lo = 0; }
    if (lo < 0) lo = 0;
    while (hi - lo > 1) {                      // invariant: R[lo] <= r or lo == 0
      const int mid = (lo + hi) >> 1;
      if (__ldg(R + mid) > r) hi = mid; else lo = mid;
    }
    j = lo;
  }
  const double Rj = __ldg(R + j), Rj1 = __ldg(R + j + 1);
  // T = exp(u_j + x) = E_j * exp(x), x = du (r - R_j)/(R_j+1 - R_j) in [0, du], du = ln(10)/64 = 0.036:
  // the degree-8 Taylor polynomial of exp is exact to 1e-17 there
  const double x = P.du * (r - Rj) / (Rj1 - Rj);
  double e = 1.0 / 40320.0;
  e = e * x + 1.0 / 5040.0; e = e * x + 1.0 / 720.0; e = e * x + 1.0 / 120.0; e = e * x + 1.0 / 24.0;
  e = e * x + 1.0 / 6.0; e = e * x + 0.5; e = e * x + 1.0; e = e * x + 1.0;
  return __ldg(P.energy_nodes + j) * e;
}

// ---------------------------------------------------------------- vectors
__device__ __forceinline__ void normalise3(double& x, double& y, double& z) {
  const double inv = rsqrt(x * x + y * y + z * z);   // (one Newton chain instead of a square root and a division; <= 2 ulp)
  x *= inv; y *= inv; z *= inv;
}

// S8 rotate(d, theta, phi) taking cos(theta), sin(theta)
// phi = 2 pi xi is passed as xi2 = 2 xi (sincospi: no argument reduction against pi needed)
__device__ __forceinline__ void rotate_dir(double& dx, double& dy, double& dz, double ct, double st, double xi2) {
  double sp, cp;
  sincospi(xi2, &sp, &cp);
  double srho = sqrt(dx * dx + dy * dy);
  double ox, oy, oz;
  if (srho == 0.0) {
    double sg = dz < 0.0 ? -1.0 : 1.0;
    ox = st * cp; oy = st * sp; oz = sg * ct;
  } else {
    const double st_rho = st / srho;
    ox = dx * ct + st_rho * (dx * dz * cp - dy * sp);
    oy = dy * ct + st_rho * (dy * dz * cp + dx * sp);
    oz = dz * ct - srho * st * cp;
  }
  normalise3(ox, oy, oz);
  dx = ox; dy = oy; dz = oz;
}

// ---------------------------------------------------------------- S6 geometry
enum : int { HIT_Z = 1, HIT_X = 2, HIT_Y = 3, HIT_INNER = 4, HIT_OUTER = 5 };
#define CEL_INF (__longlong_as_double(0x7ff0000000000000LL))

__device__ __forceinline__ double clamp0(double s) { return s < 0.0 ? 0.0 : s; }

// Distance along d to the boundary of `vol`, and which surface is hit. Callers only use the result when it is
// <= s_lim (the boundary wins ties against the physics / chord length), so the slab version divides only for the
// candidates that can be <= s_lim: a candidate num/den with |num| > s_lim |den| (1 + 1e-9) is certainly larger and is
// left at +inf. Whenever the true minimum is <= s_lim the value and the tie order z, x, y are exactly those of S6.
constexpr double kFilterSlack = 1.000000001;
__device__ __forceinline__ double slab_candidate(double num, double den, double s_lim) {
  if (fabs(num) > s_lim * fabs(den) * kFilterSlack) return CEL_INF;
  return clamp0(num / den);
}
template <int GEOM>
__device__ __forceinline__ double distance_to_boundary(const Params& P, double x, double y, double z, double dx, double dy, double dz,
                                                       int vol, int surf, double s_lim, int& which) {
  if (GEOM == 0) {
    double sz = CEL_INF, sx = CEL_INF, sy = CEL_INF;
    if (dz > 0.0) sz = slab_candidate(__ldg(P.bounds + vol + 1) - z, dz, s_lim);
    else if (dz < 0.0) sz = slab_candidate(__ldg(P.bounds + vol) - z, dz, s_lim);
    if (dx > 0.0) sx = slab_candidate(P.half_x - x, dx, s_lim);
    else if (dx < 0.0) sx = slab_candidate(-P.half_x - x, dx, s_lim);
    if (dy > 0.0) sy = slab_candidate(P.half_y - y, dy, s_lim);
    else if (dy < 0.0) sy = slab_candidate(-P.half_y - y, dy, s_lim);
    if (sz <= sx && sz <= sy) { which = HIT_Z; return sz; }
    if (sx <= sy) { which = HIT_X; return sx; }
    which = HIT_Y; return sy;
  }
  // The same filter for the cylinders (no square root, no division for a surface the step certainly does not reach): along
  // the ray the squared radius q(s) = r^2 + 2 b s + a s^2 is convex, so on [0, s_lim] it stays below q(s_lim) — the outer
  // cylinder is out of reach when q(s_lim) < rho^2 (1 - 1e-9) — and above r^2 + 2 b s_lim (b < 0) — the inner one is out
  // of reach when that exceeds rho^2 (1 + 1e-9). Most chord substeps of a track curling in a wide gap end there.
  double a = dx * dx + dy * dy;
  double b = x * dx + y * dy;
  double r2 = x * x + y * y;
  double s_in = CEL_INF, s_out = CEL_INF, s_z = CEL_INF;
  const bool filter = s_lim < 1e300;
  if (a != 0.0) {
    {
      double rho = __ldg(P.bounds + vol + 1);
      if (surf == vol + 1) {
        s_out = (b >= 0.0) ? 0.0 : -2.0 * b / a;
        s_out = clamp0(s_out);
      } else {
        double c = r2 - rho * rho;
        if (!(filter && c < 0.0 && c + (2.0 * b + a * s_lim) * s_lim < -1e-9 * (rho * rho))) {
          double D = b * b - a * c;
          if (D < 0.0) D = 0.0;
          s_out = (b > 0.0) ? -c / (b + sqrt(D)) : (-b + sqrt(D)) / a;
          s_out = clamp0(s_out);
        }
      }
    }
    if (vol > 0) {
      double rho = __ldg(P.bounds + vol);
      if (surf == vol) {
        if (b < 0.0) s_in = 0.0;
      } else if (b < 0.0) {
        double c = r2 - rho * rho;
        if (!(filter && c + 2.0 * b * s_lim > 1e-9 * (rho * rho))) {
          double D = b * b - a * c;
          if (D > 0.0) s_in = clamp0(c / (-b + sqrt(D)));
        }
      }
    }
  }
  if (dz > 0.0) s_z = filter ? slab_candidate(P.half_z - z, dz, s_lim) : clamp0((P.half_z - z) / dz);
  else if (dz < 0.0) s_z = filter ? slab_candidate(-P.half_z - z, dz, s_lim) : clamp0((-P.half_z - z) / dz);
  if (s_in <= s_out && s_in <= s_z) { which = HIT_INNER; return s_in; }
  if (s_out <= s_z) { which = HIT_OUTER; return s_out; }
  which = HIT_Z; return s_z;
}

// S7.3 dip rule: the tangent d points into the current volume across the surface hit by the chord ch
// (outward normal: the sign of the chord component for planes, the radial direction for cylinders)
constexpr int kMaxDipHalvings = 30;
__device__ __forceinline__ bool tangent_points_inward(const Params& P, double x, double y, double dx, double dy, double dz,
                                                      double chx, double chy, double chz, int which) {
  if (which == HIT_Z) return dz * chz < 0.0;
  if (which == HIT_X) return dx * chx < 0.0;
  if (which == HIT_Y) return dy * chy < 0.0;
  const double radial = x * dx + y * dy;
  return which == HIT_OUTER ? radial < 0.0 : radial > 0.0;
}

// apply the crossing; dz_sign is the z component of the direction of travel; returns true if escaped
template <int GEOM>
__device__ __forceinline__ bool cross_boundary(const Params& P, double& z, double dz_travel, int& vol, int& surf, int which) {
  if (GEOM == 0) {
    surf = -1;
    if (which != HIT_Z) return true;
    if (dz_travel > 0.0) { z = __ldg(P.bounds + vol + 1); vol += 1; }
    else { z = __ldg(P.bounds + vol); vol -= 1; }
    return vol < 0 || vol >= P.n_vol;
  }
  if (which == HIT_Z) { surf = -1; return true; }
  if (which == HIT_OUTER) { surf = vol + 1; vol += 1; return vol >= P.n_vol; }
  surf = vol; vol -= 1;
  return false;
}

// ---------------------------------------------------------------- S7.3 helix point after arc length h
struct HelixFrame { double dpar, px, py, pz, wx, wy, wz; };  // d_par, d_perp, w = d x bh
__device__ __forceinline__ HelixFrame helix_frame(const Params& P, double dx, double dy, double dz) {
  HelixFrame F;
  F.dpar = dx * P.bhx + dy * P.bhy + dz * P.bhz;
  F.px = dx - F.dpar * P.bhx; F.py = dy - F.dpar * P.bhy; F.pz = dz - F.dpar * P.bhz;
  F.wx = dy * P.bhz - dz * P.bhy; F.wy = dz * P.bhx - dx * P.bhz; F.wz = dx * P.bhy - dy * P.bhx;
  return F;
}
__device__ __forceinline__ void helix_point(const Params& P, const HelixFrame& F, double x, double y, double z, double omega, double h,
                                            double& ox, double& oy, double& oz, double& odx, double& ody, double& odz) {
  // sin(omega h)/omega = h S, 2 sin^2(omega h/2)/omega = (1 - cos(omega h))/omega = x h V with x = omega h, |x| <= 0.5
  const double x_ = omega * h;
  double S, V;
  sinc_versc_small(x_ * x_, S, V);
  const double sn = x_ * S;
  const double cs = 1.0 - (x_ * x_) * V;
  const double A = h * S;
  const double Bc = (x_ * h) * V;
  odx = F.dpar * P.bhx + cs * F.px + sn * F.wx;
  ody = F.dpar * P.bhy + cs * F.py + sn * F.wy;
  odz = F.dpar * P.bhz + cs * F.pz + sn * F.wz;
  ox = x + h * F.dpar * P.bhx + A * F.px + Bc * F.wx;
  oy = y + h * F.dpar * P.bhy + A * F.py + Bc * F.wy;
  oz = z + h * F.dpar * P.bhz + A * F.pz + Bc * F.wz;
}

__device__ __forceinline__ long long quantise(double x) { return __double2ll_rn(x * kTallyScale); }

}  // namespace cel

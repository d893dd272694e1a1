// cel_kernels.cuh — the kernels of one step iteration (docs/PHYSICS_SPEC.md S1):
//   P1 init:    k_vac_count -> k_init_fill          (scan-based vacancy filling, S9)
//   P2 reindex: (histograms in k_init_fill) -> k_scatter   (stable counting sort of slot indices, S2)
//   P3i:        k_interact<PE|PAIR|COMPTON|BREMS|ANNIH>    (S8), each over its own index range
//   P3m:        k_move_photon (S5), k_move_charged (S7)
//   P4:         k_score                              (warp-aggregated integer atomics, S10)
//   P5:         k_push_count -> k_push_write         (scan-ordered secondary push, S9)
// One thread per sorted index tid; slot = state_indices[tid], identity in mode `none`.
#pragma once
#include "cel_device.cuh"

namespace cel {

constexpr int kTileThreads = 256;
constexpr int kKeysPerThread = 16;
constexpr int kTile = kTileThreads * kKeysPerThread;  // 4096 slots per tile
constexpr int kBlock = 256;                           // physics kernels

enum KernelId : int { K_PE = 0, K_PAIR, K_COMPTON, K_BREMS, K_ANNIH, K_MOVE_G, K_MOVE_C, K_SCORE, K_COUNT };

struct Control {
  unsigned long long n_init;        // I, the initializer stack height
  unsigned long long track_steps, iterations, secondaries;
  unsigned long long push_total;    // S of this iteration
  uint32_t iter;                    // k
  uint32_t alive;                   // A_k (after P1)
  uint32_t finished;                // A_k == 0 and I == 0
  int32_t error;
  uint32_t offsets[9];              // offsets of the sorted index array, per sort key
  uint32_t counts[8];               // action counts of this iteration (after P1)
  uint32_t counts_acc[8];           // accumulators (zero between iterations)
  uint32_t rb[K_COUNT], re[K_COUNT];// index range of each kernel for this iteration
  uint32_t ticket_vac, ticket_fill, ticket_pcount, ticket_pwrite;
  uint32_t n_logged;
  uint32_t vac_total;                // V before the fill of this iteration
};

// everything a kernel needs; passed by value (fits in the 4 KB parameter space)
struct DeviceState {
  Params P;
  uint32_t N;             // n_slots
  uint32_t n_tiles;
  int sort_mode;
  unsigned long long init_capacity;
  uint32_t n_events;
  uint32_t log_capacity;
  RecA* stA; RecB* stB;
  uint8_t* akey;          // [n_tiles * kTile] action | ptype << 4
  uint8_t* nsec;          // [n_tiles * kTile]
  uint32_t* indices;      // [N] (sorted modes)
  Stage* stage;           // [N]
  RecA* secA; RecB* secB; // [2N] staged secondaries
  RecA* initA; RecB* initB; // [init_capacity]
  unsigned long long* tally; // [n_events][n_bins+1]
  uint32_t* counts_log;   // [log_capacity][8]
  Control* ctl;
  // stream-ordered scratch (cudaMallocAsync, per transport call)
  uint32_t* tile_vac;     // [n_tiles] exclusive prefix of vacancies after k_vac_count
  uint32_t* tile_hist;    // [n_tiles][8] -> exclusive base per key after k_init_fill
  uint32_t* tile_sec;     // [n_tiles] exclusive prefix of secondaries after k_push_count
};

// ---------------------------------------------------------------- block-level scan primitives
__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    uint32_t n = __shfl_up_sync(0xffffffffu, v, d);
    if ((threadIdx.x & 31) >= d) v += n;
  }
  return v;
}
__device__ __forceinline__ unsigned long long warp_incl_scan64(unsigned long long v) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    unsigned long long n = __shfl_up_sync(0xffffffffu, v, d);
    if ((threadIdx.x & 31) >= d) v += n;
  }
  return v;
}
// exclusive scan over the 256 threads of a tile block; returns the exclusive prefix, total in `total`
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t* smem /* 9 words */, uint32_t& total) {
  uint32_t incl = warp_incl_scan(v);
  int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  __syncthreads();
  if (lane == 31) smem[warp] = incl;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t run = 0;
    for (int w = 0; w < kTileThreads / 32; ++w) { uint32_t t = smem[w]; smem[w] = run; run += t; }
    smem[8] = run;
  }
  __syncthreads();
  total = smem[8];
  return smem[warp] + incl - v;
}
__device__ __forceinline__ unsigned long long block_excl_scan64(unsigned long long v, unsigned long long* smem /* 9 */, unsigned long long& total) {
  unsigned long long incl = warp_incl_scan64(v);
  int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  __syncthreads();
  if (lane == 31) smem[warp] = incl;
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned long long run = 0;
    for (int w = 0; w < kTileThreads / 32; ++w) { unsigned long long t = smem[w]; smem[w] = run; run += t; }
    smem[8] = run;
  }
  __syncthreads();
  total = smem[8];
  return smem[warp] + incl - v;
}
// in-place exclusive scan of a[0..n) by one block (n small: tiles); returns the total to every thread
__device__ __forceinline__ uint32_t block_scan_array(uint32_t* a, uint32_t n, uint32_t stride, uint32_t* smem) {
  __shared__ uint32_t carry_s;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  for (uint32_t base = 0; base < n; base += kTileThreads) {
    uint32_t i = base + threadIdx.x;
    uint32_t v = (i < n) ? a[(size_t)i * stride] : 0;
    uint32_t total;
    uint32_t ex = block_excl_scan(v, smem, total);
    uint32_t carry = carry_s;
    if (i < n) a[(size_t)i * stride] = carry + ex;
    __syncthreads();
    if (threadIdx.x == 0) carry_s = carry + total;
    __syncthreads();
  }
  return carry_s;
}
// "last block done" ticket: true in exactly one block, after every other block's global writes are visible
__device__ __forceinline__ bool last_block_done(uint32_t* ticket) {
  __shared__ bool is_last;
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t t = atomicAdd(ticket, 1u);
    is_last = (t == gridDim.x - 1);
    if (is_last) *ticket = 0;
  }
  __syncthreads();
  if (is_last) __threadfence();
  return is_last;
}

__device__ __forceinline__ int sort_key_of(int sort_mode, uint8_t key) {
  int a = key & 0xf;
  if (sort_mode == 1) return a;
  return a == A_VACANT ? 3 : ((key >> 4) & 0x3);
}

// ================================================================ P1: vacancy scan + fill (S9)
// k_vac_count: one block per tile of 4096 slots; counts vacancies; the last block turns the per-tile counts
// into an exclusive prefix (tile_vac) — scan-based, no atomics in the assignment, so slot assignment is
// deterministic.
__global__ void __launch_bounds__(kTileThreads) k_vac_count(DeviceState D) {
  __shared__ uint32_t smem[9];
  Control* ctl = D.ctl;
  if (ctl->finished) return;
  const uint32_t tile = blockIdx.x;
  const uint32_t base = tile * kTile + threadIdx.x * kKeysPerThread;
  uint4 kv = *reinterpret_cast<const uint4*>(D.akey + base);
  const uint8_t* kb = reinterpret_cast<const uint8_t*>(&kv);
  uint32_t c = 0;
#pragma unroll
  for (int i = 0; i < kKeysPerThread; ++i) c += (base + i < D.N) && ((kb[i] & 0xf) == A_VACANT);
  uint32_t total;
  block_excl_scan(c, smem, total);
  if (threadIdx.x == 0) D.tile_vac[tile] = total;
  if (last_block_done(&ctl->ticket_vac)) {
    uint32_t V = block_scan_array(D.tile_vac, D.n_tiles, 1, smem);
    if (threadIdx.x == 0) ctl->vac_total = V;
  }
}

// k_init_fill: rank-r vacant slot (ascending slot order) takes init[I-1-r] when r < I; also builds the per-tile
// histogram of sort keys for P2 and, in its last block, the offsets, kernel ranges, counters and the log.
__global__ void __launch_bounds__(kTileThreads) k_init_fill(DeviceState D) {
  __shared__ uint32_t smem[9];
  __shared__ uint32_t hist_s[8], act_s[8];
  Control* ctl = D.ctl;
  if (ctl->finished) return;
  const uint32_t tile = blockIdx.x;
  const uint32_t base = tile * kTile + threadIdx.x * kKeysPerThread;
  const unsigned long long I = ctl->n_init;
  if (threadIdx.x < 8) { hist_s[threadIdx.x] = 0; act_s[threadIdx.x] = 0; }
  uint4 kv = *reinterpret_cast<const uint4*>(D.akey + base);
  uint8_t* kb = reinterpret_cast<uint8_t*>(&kv);
  uint32_t c = 0;
#pragma unroll
  for (int i = 0; i < kKeysPerThread; ++i) c += (base + i < D.N) && ((kb[i] & 0xf) == A_VACANT);
  uint32_t total;
  uint32_t rank = D.tile_vac[tile] + block_excl_scan(c, smem, total);
  bool changed = false;
  if (c != 0 && (unsigned long long)rank < I) {
#pragma unroll 1
    for (int i = 0; i < kKeysPerThread; ++i) {
      const uint32_t slot = base + i;
      if (slot < D.N && (kb[i] & 0xf) == A_VACANT) {
        if ((unsigned long long)rank < I) {
          const unsigned long long src = I - 1ull - rank;
          RecA a = load_a(D.initA + src);
          RecB b = load_b(D.initB + src);
          store_a(D.stA + slot, a);
          store_b(D.stB + slot, b);
          kb[i] = make_key(meta_action(b.meta), meta_ptype(b.meta));
          changed = true;
        }
        ++rank;
      }
    }
  }
  if (changed) *reinterpret_cast<uint4*>(D.akey + base) = kv;
  // histograms: action counts (always) and sort-key counts (sorted modes), packed 4 x 16 bit in two words
  unsigned long long a_lo = 0, a_hi = 0, s_lo = 0, s_hi = 0;
#pragma unroll
  for (int i = 0; i < kKeysPerThread; ++i) {
    if (base + i < D.N) {
      int a = kb[i] & 0xf;
      if (a < 4) a_lo += 1ull << (16 * a); else a_hi += 1ull << (16 * (a - 4));
      if (D.sort_mode == 2) { int s = sort_key_of(2, kb[i]); s_lo += 1ull << (16 * s); }
    }
  }
  if (D.sort_mode == 1) { s_lo = a_lo; s_hi = a_hi; }
  // block totals by warp reduction of the packed words (a tile has 4096 slots < 2^16)
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) {
    a_lo += __shfl_xor_sync(0xffffffffu, a_lo, d); a_hi += __shfl_xor_sync(0xffffffffu, a_hi, d);
    s_lo += __shfl_xor_sync(0xffffffffu, s_lo, d); s_hi += __shfl_xor_sync(0xffffffffu, s_hi, d);
  }
  __syncthreads();
  if ((threadIdx.x & 31) == 0) {
#pragma unroll
    for (int a = 0; a < 4; ++a) {
      atomicAdd(&act_s[a], (uint32_t)((a_lo >> (16 * a)) & 0xffff)); atomicAdd(&act_s[a + 4], (uint32_t)((a_hi >> (16 * a)) & 0xffff));
      atomicAdd(&hist_s[a], (uint32_t)((s_lo >> (16 * a)) & 0xffff)); atomicAdd(&hist_s[a + 4], (uint32_t)((s_hi >> (16 * a)) & 0xffff));
    }
  }
  __syncthreads();
  if (threadIdx.x < 8) {
    D.tile_hist[tile * 8 + threadIdx.x] = hist_s[threadIdx.x];
    if (act_s[threadIdx.x]) atomicAdd(&ctl->counts_acc[threadIdx.x], act_s[threadIdx.x]);
  }
  if (!last_block_done(&ctl->ticket_fill)) return;
  // ---- last block: per-key exclusive scan over tiles, offsets, ranges, counters
  __shared__ uint32_t key_total[8];
  const int n_keys = D.sort_mode == 1 ? 8 : (D.sort_mode == 2 ? 4 : 0);
  for (int k = 0; k < n_keys; ++k) {
    uint32_t t = block_scan_array(D.tile_hist + k, D.n_tiles, 8, smem);
    if (threadIdx.x == 0) key_total[k] = t;
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    uint32_t cnt[8];
    for (int a = 0; a < 8; ++a) { cnt[a] = ctl->counts_acc[a]; ctl->counts[a] = cnt[a]; ctl->counts_acc[a] = 0; }
    const uint32_t N = D.N;
    uint32_t off[9];
    off[0] = 0;
    for (int k = 0; k < 8; ++k) off[k + 1] = (k < n_keys) ? off[k] + key_total[k] : off[k];
    if (n_keys == 0) for (int k = 1; k <= 8; ++k) off[k] = N;
    for (int k = 0; k <= 8; ++k) ctl->offsets[k] = off[k];
    uint32_t* rb = ctl->rb; uint32_t* re = ctl->re;
    if (D.sort_mode == 1) {
      rb[K_PE] = off[0]; re[K_PE] = off[1];
      rb[K_PAIR] = off[1]; re[K_PAIR] = off[2];
      rb[K_COMPTON] = off[2]; re[K_COMPTON] = off[3];
      rb[K_MOVE_G] = off[2]; re[K_MOVE_G] = off[4];
      rb[K_MOVE_C] = off[4]; re[K_MOVE_C] = off[6];
      rb[K_BREMS] = off[5]; re[K_BREMS] = off[6];
      rb[K_ANNIH] = off[6]; re[K_ANNIH] = off[7];
      rb[K_SCORE] = 0; re[K_SCORE] = off[7];
    } else if (D.sort_mode == 2) {
      rb[K_PE] = rb[K_PAIR] = rb[K_COMPTON] = rb[K_MOVE_G] = off[0];
      re[K_PE] = re[K_PAIR] = re[K_COMPTON] = re[K_MOVE_G] = off[1];
      rb[K_BREMS] = rb[K_MOVE_C] = off[1]; re[K_BREMS] = re[K_MOVE_C] = off[3];
      rb[K_ANNIH] = off[2]; re[K_ANNIH] = off[3];
      rb[K_SCORE] = 0; re[K_SCORE] = off[3];
    } else {
      for (int k = 0; k < K_COUNT; ++k) { rb[k] = 0; re[k] = N; }
    }
    const uint32_t alive = N - cnt[A_VACANT];
    // I -= min(V, I) with V the number of vacancies before the fill
    const unsigned long long Ibefore = ctl->n_init;
    const unsigned long long V = ctl->vac_total;
    const unsigned long long Iafter = Ibefore - (V < Ibefore ? V : Ibefore);
    ctl->n_init = Iafter;
    ctl->alive = alive;
    if (alive == 0 && Iafter == 0) {
      ctl->finished = 1;
    } else {
      ctl->track_steps += alive;
      ctl->iterations += 1;
      const uint32_t k = ctl->n_logged;
      if (k < D.log_capacity) {
        for (int a = 0; a < 8; ++a) D.counts_log[(size_t)k * 8 + a] = cnt[a];
        ctl->n_logged = k + 1;
      }
    }
  }
}

// ================================================================ P2: stable scatter of slot indices (S2)
// indices[offset[key] + (tiles before)[key] + (rank inside the tile)] = slot; ascending slot order inside a key.
__global__ void __launch_bounds__(kTileThreads) k_scatter(DeviceState D) {
  __shared__ unsigned long long smem64[9];
  __shared__ uint32_t base_s[8];
  Control* ctl = D.ctl;
  if (ctl->finished) return;
  const uint32_t tile = blockIdx.x;
  const uint32_t base = tile * kTile + threadIdx.x * kKeysPerThread;
  if (threadIdx.x < 8) base_s[threadIdx.x] = ctl->offsets[threadIdx.x] + D.tile_hist[tile * 8 + threadIdx.x];
  uint4 kv = *reinterpret_cast<const uint4*>(D.akey + base);
  const uint8_t* kb = reinterpret_cast<const uint8_t*>(&kv);
  unsigned long long lo = 0, hi = 0;
#pragma unroll
  for (int i = 0; i < kKeysPerThread; ++i) {
    if (base + i < D.N) {
      int s = sort_key_of(D.sort_mode, kb[i]);
      if (s < 4) lo += 1ull << (16 * s); else hi += 1ull << (16 * (s - 4));
    }
  }
  unsigned long long tot;
  unsigned long long plo = block_excl_scan64(lo, smem64, tot);
  unsigned long long phi = block_excl_scan64(hi, smem64, tot);
  // vacant slots are never launched; their indices are still written so that the permutation is complete
#pragma unroll
  for (int i = 0; i < kKeysPerThread; ++i) {
    if (base + i < D.N) {
      int s = sort_key_of(D.sort_mode, kb[i]);
      uint32_t r;
      if (s < 4) { r = (uint32_t)((plo >> (16 * s)) & 0xffff); plo += 1ull << (16 * s); }
      else { r = (uint32_t)((phi >> (16 * (s - 4))) & 0xffff); phi += 1ull << (16 * (s - 4)); }
      D.indices[base_s[s] + r] = base + i;
    }
  }
}

// ================================================================ P3i: discrete interactions (S8)
// Each kernel runs over its own range [rb, re) of the sorted index array with a grid-stride
// loop; in modes `none` / `by particle` the dense key byte masks non-participants before any state is read.
struct SecOut { int n; };

__device__ __forceinline__ void stage_secondary(const DeviceState& D, uint32_t slot, int j, const RecA& parent, double energy,
                                                double dx, double dy, double dz, int ptype, int vol, int surf, uint32_t event) {
  RecA a = parent; a.energy = energy;
  RecB b; b.dx = dx; b.dy = dy; b.dz = dz;
  b.meta = make_meta(ptype == P_GAMMA ? A_MOVE_G : A_MOVE_C, ptype, false, vol, surf, 0, event);
  store_a(D.secA + 2ull * slot + j, a);
  store_b(D.secB + 2ull * slot + j, b);
}

// a charged track whose kinetic energy dropped below the cut (its energy is already in edep): returns the new action
__device__ __forceinline__ int stop_charged(const Params& P, int ptype, double& edep) {
  if (ptype == P_POSITRON) {
    if (P.enable_annihilation) return A_ANNIH;
    edep += 2.0 * kElectronMass;
  }
  return A_VACANT;
}

template <int ACT>
__global__ void __launch_bounds__(kBlock) k_interact(DeviceState D) {
  const Control* ctl = D.ctl;
  if (ctl->finished) return;
  constexpr int KID = ACT == A_PE ? K_PE : ACT == A_PAIR ? K_PAIR : ACT == A_COMPTON ? K_COMPTON : ACT == A_BREMS ? K_BREMS : K_ANNIH;
  const uint32_t rb = ctl->rb[KID], re = ctl->re[KID];
  const uint32_t k_iter = ctl->iter;
  const Params& P = D.P;
  for (uint32_t tid = rb + blockIdx.x * blockDim.x + threadIdx.x; tid < re; tid += gridDim.x * blockDim.x) {
    const uint32_t slot = (D.sort_mode != 0) ? D.indices[tid] : tid;
    if (D.sort_mode != 1 && (D.akey[slot] & 0xf) != ACT) continue;
    RecB b = load_b(D.stB + slot);
    if (meta_action(b.meta) != ACT) continue;
    RecA a = load_a(D.stA + slot);
    const int ptype = meta_ptype(b.meta), vol = meta_vol(b.meta), surf = meta_surf(b.meta);
    const uint32_t event = meta_event(b.meta), nsteps = meta_nsteps(b.meta);
    double edep = 0.0;
    int nsec = 0;
    int action = A_VACANT;
    bool write_a = false;
    if (ACT == A_PE) {
      if (P.electrons_local) edep += a.energy;
      else stage_secondary(D, slot, nsec++, a, a.energy, b.dx, b.dy, b.dz, P_ELECTRON, vol, surf, event);
    } else if (ACT == A_PAIR) {
      double xi0, xi1;
      draw_pair(P, slot, k_iter, PH_INTERACT, 0, xi0, xi1);
      const double Tav = a.energy - 2.0 * kElectronMass;
      const double Tm = xi0 * Tav;
      const double Tp = Tav - Tm;
      if (Tm >= P.cut) stage_secondary(D, slot, nsec++, a, Tm, b.dx, b.dy, b.dz, P_ELECTRON, vol, surf, event);
      else edep += Tm;
      stage_secondary(D, slot, nsec++, a, Tp, b.dx, b.dy, b.dz, P_POSITRON, vol, surf, event);
    } else if (ACT == A_COMPTON) {
      const double E = a.energy;
      const double k = E / kElectronMass;
      const double e0 = 1.0 / (1.0 + 2.0 * k);
      const double a1 = -log(e0);
      const double a2 = (1.0 - e0 * e0) / 2.0;
      double eps, tt, sin2, xphi;
      for (uint32_t t = 0;; ++t) {
        double xa, xb, xc;
        draw_pair(P, slot, k_iter, PH_INTERACT, 2 * t, xa, xb);
        draw_pair(P, slot, k_iter, PH_INTERACT, 2 * t + 1, xc, xphi);
        if (xa * (a1 + a2) < a1) eps = exp(-a1 * xb);
        else eps = sqrt(e0 * e0 + (1.0 - e0 * e0) * xb);
        tt = (1.0 - eps) / (k * eps);
        sin2 = tt * (2.0 - tt);
        if (xc <= 1.0 - eps * sin2 / (1.0 + eps * eps) || t >= 65535u) break;
      }
      const double cost = 1.0 - tt;
      const double sint = sqrt(sin2 > 0.0 ? sin2 : 0.0);
      const double phi = 2.0 * kPi * xphi;
      const double E1 = eps * E;
      double d1x = b.dx, d1y = b.dy, d1z = b.dz;
      rotate_dir(d1x, d1y, d1z, cost, sint, phi);
      const double Te = E - E1;
      if (P.electrons_local || Te < P.cut) {
        edep += Te;
      } else {
        double ex = E * b.dx - E1 * d1x, ey = E * b.dy - E1 * d1y, ez = E * b.dz - E1 * d1z;
        const double n = sqrt(ex * ex + ey * ey + ez * ez);
        if (n > 0.0) { ex /= n; ey /= n; ez /= n; } else { ex = b.dx; ey = b.dy; ez = b.dz; }
        stage_secondary(D, slot, nsec++, a, Te, ex, ey, ez, P_ELECTRON, vol, surf, event);
      }
      if (E1 < P.cut) { edep += E1; }
      else { a.energy = E1; b.dx = d1x; b.dy = d1y; b.dz = d1z; action = A_MOVE_G; write_a = true; }
    } else if (ACT == A_BREMS) {
      double xi0, xi1;
      draw_pair(P, slot, k_iter, PH_INTERACT, 0, xi0, xi1);
      const double kph = P.cut * exp(xi0 * log(a.energy / P.cut));
      stage_secondary(D, slot, nsec++, a, kph, b.dx, b.dy, b.dz, P_GAMMA, vol, surf, event);
      const double T1 = a.energy - kph;
      if (T1 < P.cut) { edep += T1; a.energy = 0.0; action = stop_charged(P, ptype, edep); }
      else { a.energy = T1; action = A_MOVE_C; }
      write_a = true;
    } else {  // A_ANNIH
      double xi0, xi1;
      draw_pair(P, slot, k_iter, PH_INTERACT, 0, xi0, xi1);
      const double cost = 2.0 * xi0 - 1.0;
      const double sint = sqrt(1.0 - cost * cost);
      double sp, cp;
      sincos(2.0 * kPi * xi1, &sp, &cp);
      const double ux = sint * cp, uy = sint * sp, uz = cost;
      stage_secondary(D, slot, nsec++, a, kElectronMass, ux, uy, uz, P_GAMMA, vol, surf, event);
      stage_secondary(D, slot, nsec++, a, kElectronMass, -ux, -uy, -uz, P_GAMMA, vol, surf, event);
    }
    const long long q = quantise(edep);
    const bool survivor = (action == A_MOVE_G || action == A_MOVE_C);
    if (q != 0) store_stage(D.stage + slot, q, 0, event, __ldg(P.vol_bin + vol));
    b.meta = make_meta(action, ptype, survivor && q != 0, vol, surf, nsteps, event);
    if (write_a) store_a(D.stA + slot, a);
    store_b(D.stB + slot, b);
    D.akey[slot] = make_key(action, ptype);
    if (nsec) D.nsec[slot] = (uint8_t)nsec;
  }
}

// ================================================================ P3m: photon move (S5)
__global__ void __launch_bounds__(kBlock) k_move_photon(DeviceState D) {
  const Control* ctl = D.ctl;
  if (ctl->finished) return;
  const uint32_t rb = ctl->rb[K_MOVE_G], re = ctl->re[K_MOVE_G];
  const uint32_t k_iter = ctl->iter;
  const Params& P = D.P;
  for (uint32_t tid = rb + blockIdx.x * blockDim.x + threadIdx.x; tid < re; tid += gridDim.x * blockDim.x) {
    const uint32_t slot = (D.sort_mode != 0) ? D.indices[tid] : tid;
    if (D.sort_mode != 1 && (D.akey[slot] & 0xf) != A_MOVE_G) continue;
    RecB b = load_b(D.stB + slot);
    if (meta_action(b.meta) != A_MOVE_G) continue;   // vacated by Compton in this iteration
    RecA a = load_a(D.stA + slot);
    int vol = meta_vol(b.meta), surf = meta_surf(b.meta);
    const int vol0 = vol;
    const uint32_t event = meta_event(b.meta);
    uint32_t nsteps = meta_nsteps(b.meta);
    const int mat = __ldg(P.vol_material + vol);
    double sPE = 0.0, sPair = 0.0, sC = 0.0;
    if (mat >= 0) {
      const GridPos g = grid_locate(P, a.energy);
      const double2* xs = reinterpret_cast<const double2*>(P.photon_xs + (size_t)mat * kGrid + g.j);  // nodes j, j+1: 64 B
      const double2 n0a = __ldg(xs), n0b = __ldg(xs + 1), n1a = __ldg(xs + 2), n1b = __ldg(xs + 3);
      sC = lerp_node(n0a.x, n1a.x, g.f);
      sPE = lerp_node(n0a.y, n1a.y, g.f);
      sPair = lerp_node(n0b.x, n1b.x, g.f);
    }
    const double stot = (sPE + sPair) + sC;
    double xi0, xi1;
    draw_pair(P, slot, k_iter, PH_STEP, 0, xi0, xi1);
    const double s_d = (stot > 0.0) ? -log(xi0) / stot : CEL_INF;
    const double x = xi1 * stot;
    const int process = (x < sPE) ? A_PE : ((x < sPE + sPair) ? A_PAIR : A_COMPTON);
    int which;
    const double s_b = distance_to_boundary(P, a.x, a.y, a.z, b.dx, b.dy, b.dz, vol, surf, which);
    if (nsteps < 65535u) nsteps += 1;
    int action;
    double eesc = 0.0;
    if (s_d < s_b) {
      a.x += s_d * b.dx; a.y += s_d * b.dy; a.z += s_d * b.dz;
      surf = -1;
      action = process;
    } else {
      a.x += s_b * b.dx; a.y += s_b * b.dy; a.z += s_b * b.dz;
      const bool escaped = cross_boundary(P, a.z, b.dz, vol, surf, which);
      if (escaped) { eesc += a.energy; action = A_VACANT; if (vol < 0 || vol > 254) vol = vol0; }
      else action = A_MOVE_G;
    }
    long long q_dep = 0, q_esc = quantise(eesc);
    if (meta_staged(b.meta)) { q_dep += D.stage[slot].q_dep; }
    if ((q_dep | q_esc) != 0) store_stage(D.stage + slot, q_dep, q_esc, event, __ldg(P.vol_bin + vol0));
    b.meta = make_meta(action, P_GAMMA, false, vol, surf, nsteps, event);
    store_a(D.stA + slot, a);
    store_b(D.stB + slot, b);
    D.akey[slot] = make_key(action, P_GAMMA);
  }
}

// ================================================================ P3m: charged move (S7)
// step limit -> linear or helical propagation (<= max_substeps chord substeps) -> CSDA loss -> MSC -> fate
__global__ void __launch_bounds__(kBlock) k_move_charged(DeviceState D) {
  const Control* ctl = D.ctl;
  if (ctl->finished) return;
  const uint32_t rb = ctl->rb[K_MOVE_C], re = ctl->re[K_MOVE_C];
  const uint32_t k_iter = ctl->iter;
  const Params& P = D.P;
  for (uint32_t tid = rb + blockIdx.x * blockDim.x + threadIdx.x; tid < re; tid += gridDim.x * blockDim.x) {
    const uint32_t slot = (D.sort_mode != 0) ? D.indices[tid] : tid;
    if (D.sort_mode != 1 && (D.akey[slot] & 0xf) != A_MOVE_C) continue;
    RecB b = load_b(D.stB + slot);
    if (meta_action(b.meta) != A_MOVE_C) continue;   // brems participant that stopped in this iteration
    RecA a = load_a(D.stA + slot);
    const int ptype = meta_ptype(b.meta);
    int vol = meta_vol(b.meta), surf = meta_surf(b.meta);
    const int vol0 = vol;
    const uint32_t event = meta_event(b.meta);
    uint32_t nsteps = meta_nsteps(b.meta);
    if (nsteps < 65535u) nsteps += 1;
    long long q_dep = meta_staged(b.meta) ? D.stage[slot].q_dep : 0;
    double edep = 0.0, eesc = 0.0;
    const double T0 = a.energy;
    int action;
    if (T0 < P.cut) {  // S7.1
      edep += T0;
      a.energy = 0.0;
      action = stop_charged(P, ptype, edep);
    } else {
      const int mat = __ldg(P.vol_material + vol);
      const double p = sqrt(T0 * (T0 + 2.0 * kElectronMass));
      const double beta = p / (T0 + kElectronMass);
      // S7.2 step limit
      double r0 = 0.0, s_r = CEL_INF, s_d = CEL_INF;
      int j0 = 0;
      if (mat >= 0) {
        const GridPos g = grid_locate(P, T0);
        j0 = g.j;
        const double2* cxs = reinterpret_cast<const double2*>(P.charged_xs + (size_t)mat * kGrid + g.j);  // nodes j, j+1
        const double2 n0 = __ldg(cxs);
        const double2 n1 = __ldg(cxs + 1);
        if (P.enable_eloss) {
          r0 = lerp_node(n0.y, n1.y, g.f);
          s_r = (r0 <= kRhoF) ? r0 : fmax(kAlphaR * r0, kRhoF);
        }
        const double sb = lerp_node(n0.x, n1.x, g.f);
        double xi0, xi1;
        draw_pair(P, slot, k_iter, PH_STEP, 0, xi0, xi1);
        if (sb > 0.0) s_d = -log(xi0) / sb;
      }
      const bool interaction_wins = s_d < s_r;
      const double s_phys = interaction_wins ? s_d : s_r;
      // S7.3 propagation
      double travelled = 0.0;
      bool escaped = false, complete = false;
      if (P.bmag == 0.0) {
        int which;
        const double s_b = distance_to_boundary(P, a.x, a.y, a.z, b.dx, b.dy, b.dz, vol, surf, which);
        if (s_phys < s_b) {
          a.x += s_phys * b.dx; a.y += s_phys * b.dy; a.z += s_phys * b.dz;
          surf = -1; travelled = s_phys; complete = true;
        } else {
          a.x += s_b * b.dx; a.y += s_b * b.dy; a.z += s_b * b.dz;
          travelled = s_b;
          escaped = cross_boundary(P, a.z, b.dz, vol, surf, which);
        }
      } else {
        const double q = (ptype == P_ELECTRON) ? -1.0 : 1.0;
        const double omega = q * kKappa * P.bmag / p;
        const double h_max = fmin(sqrt(8.0 * kDeltaChord / fabs(omega)), 0.5 / fabs(omega));
        double remaining = s_phys;
        int n = 0;
        if (!(s_phys > 0.0)) complete = true;
        while (!complete) {
          if (n == P.max_substeps) break;  // paused
          double h = fmin(remaining, h_max);
          const HelixFrame F = helix_frame(P, b.dx, b.dy, b.dz);
          double nx, ny, nz, ndx, ndy, ndz, l, chx, chy, chz, tb;
          int which;
          for (int halvings = 0;; ++halvings) {
            helix_point(P, F, a.x, a.y, a.z, omega, h, nx, ny, nz, ndx, ndy, ndz);
            const double cx = nx - a.x, cy = ny - a.y, cz = nz - a.z;
            l = sqrt(cx * cx + cy * cy + cz * cz);
            chx = cx / l; chy = cy / l; chz = cz / l;
            tb = distance_to_boundary(P, a.x, a.y, a.z, chx, chy, chz, vol, surf, which);
            // S7.3 dip rule: on a surface with the tangent into the volume but the chord out of it, halve h
            if (tb == 0.0 && halvings < kMaxDipHalvings &&
                tangent_points_inward(P, a.x, a.y, b.dx, b.dy, b.dz, chx, chy, chz, which)) { h *= 0.5; continue; }
            break;
          }
          if (tb <= l) {
            const double f = tb / l;
            double fx, fy, fz, fdx, fdy, fdz;
            helix_point(P, F, a.x, a.y, a.z, omega, f * h, fx, fy, fz, fdx, fdy, fdz);
            a.x += tb * chx; a.y += tb * chy; a.z += tb * chz;
            normalise3(fdx, fdy, fdz);
            b.dx = fdx; b.dy = fdy; b.dz = fdz;
            travelled += f * h;
            escaped = cross_boundary(P, a.z, chz, vol, surf, which);
            break;
          }
          normalise3(ndx, ndy, ndz);
          a.x = nx; a.y = ny; a.z = nz;
          b.dx = ndx; b.dy = ndy; b.dz = ndz;
          travelled += h;
          surf = -1;
          remaining -= h;
          n += 1;
          if (remaining <= 0.0) { travelled = s_phys; complete = true; }
        }
      }
      // S7.4 energy loss
      double T1 = T0;
      if (mat >= 0 && P.enable_eloss) {
        const double r1 = r0 - travelled;
        T1 = (r1 <= 0.0) ? 0.0 : range_inverse(P, P.range_tab + (size_t)mat * kGrid, r1, j0);
        if (T1 > T0) T1 = T0;
        edep += T0 - T1;
      }
      // S7.5 multiple scattering
      if (P.enable_msc && !escaped && mat >= 0 && travelled > 0.0 && T1 >= P.cut) {
        const double x = travelled * __ldg(&P.mats[mat].inv_X0);
        const double theta0 = 13.6 / (beta * p) * sqrt(x) * fmax(0.0, 1.0 + 0.038 * log(x));
        double xm0, xm1;
        draw_pair(P, slot, k_iter, PH_MSC, 0, xm0, xm1);
        const double theta = fmin(theta0 * sqrt(-2.0 * log(xm0)), kPi);
        double st, ct;
        sincos(theta, &st, &ct);
        rotate_dir(b.dx, b.dy, b.dz, ct, st, 2.0 * kPi * xm1);
      }
      // S7.6 fate
      const double rest = (ptype == P_POSITRON) ? 2.0 * kElectronMass : 0.0;
      if (escaped) {
        eesc += T1 + rest; a.energy = T1; action = A_VACANT;
        if (vol < 0 || vol > 254) vol = vol0;
      } else if (T1 < P.cut) {
        edep += T1; a.energy = 0.0;
        action = stop_charged(P, ptype, edep);
      } else if (nsteps >= P.max_steps_per_track) {
        eesc += T1 + rest; a.energy = T1; action = A_VACANT;
      } else {
        a.energy = T1;
        action = (interaction_wins && complete) ? A_BREMS : A_MOVE_C;
      }
    }
    q_dep += quantise(edep);
    const long long q_esc = quantise(eesc);
    if ((q_dep | q_esc) != 0) store_stage(D.stage + slot, q_dep, q_esc, event, __ldg(P.vol_bin + vol0));
    b.meta = make_meta(action, ptype, false, vol, surf, nsteps, event);
    store_a(D.stA + slot, a);
    store_b(D.stB + slot, b);
    D.akey[slot] = make_key(action, ptype);
  }
}

// ================================================================ P4: scoring (S10)
// Adds the slot's staged integer deposits to tally[event][bin]. Lanes of a warp that hit the same tally cell are
// combined first (__match_any_sync + one leader atomic): warp-aggregated atomics. Integer addition is associative,
// so the tally does not depend on thread order or sort mode.
__device__ __forceinline__ void warp_aggregated_add(unsigned long long* tally, bool active, unsigned long long cell, unsigned long long value) {
  const unsigned mask = __ballot_sync(0xffffffffu, active);
  if (!active) return;
  const unsigned peers = __match_any_sync(mask, cell);
  const int lane = threadIdx.x & 31;
  const int leader = __ffs(peers) - 1;
  // sum over the peer group: every lane walks the same peer mask
  unsigned long long sum = 0;
  unsigned rem = peers;
  while (rem) {
    const int src = __ffs(rem) - 1;
    sum += __shfl_sync(peers, value, src);
    rem &= rem - 1;
  }
  if (lane == leader) atomicAdd(tally + cell, sum);
}

__global__ void __launch_bounds__(kBlock) k_score(DeviceState D) {
  const Control* ctl = D.ctl;
  if (ctl->finished) return;
  const uint32_t rb = ctl->rb[K_SCORE], re = ctl->re[K_SCORE];
  const uint32_t nb1 = (uint32_t)D.P.n_bins + 1u;
  // whole warps iterate together so that the aggregation sees converged lanes
  const uint32_t span = re - rb;
  const uint32_t span_pad = (span + 31u) & ~31u;
  for (uint32_t off = blockIdx.x * blockDim.x + threadIdx.x; off < span_pad; off += gridDim.x * blockDim.x) {
    const uint32_t tid = rb + off;
    long long q_dep = 0, q_esc = 0;
    uint32_t event = 0; int32_t bin = -1;
    if (off < span) {
      const uint32_t slot = (D.sort_mode != 0) ? D.indices[tid] : tid;
      const Stage s = load_stage(D.stage + slot);
      if ((s.q_dep | s.q_esc) != 0) {
        q_dep = s.q_dep; q_esc = s.q_esc; event = s.event; bin = s.bin;
        *reinterpret_cast<ulonglong2*>(D.stage + slot) = make_ulonglong2(0ull, 0ull);  // consumed
      }
    }
    const unsigned long long row = (unsigned long long)event * nb1;
    warp_aggregated_add(D.tally, q_dep != 0 && bin >= 0, row + (unsigned long long)(bin < 0 ? 0 : bin), (unsigned long long)q_dep);
    warp_aggregated_add(D.tally, q_esc != 0, row + (unsigned long long)D.P.n_bins, (unsigned long long)q_esc);
  }
}

// ================================================================ P5: secondary push (S9)
// Exclusive scan of nsec[slot] in ascending SLOT order (in every sort mode), so that the initializer order — and with
// it every later slot assignment and PRNG stream — does not depend on thread timing or on the sort mode.
__global__ void __launch_bounds__(kTileThreads) k_push_count(DeviceState D) {
  __shared__ uint32_t smem[9];
  Control* ctl = D.ctl;
  if (ctl->finished) return;
  const uint32_t tile = blockIdx.x;
  const uint32_t base = tile * kTile + threadIdx.x * kKeysPerThread;
  const uint4 nv = *reinterpret_cast<const uint4*>(D.nsec + base);
  // bytes are 0..2: sum the 16 bytes
  uint32_t c = 0;
  const uint32_t w[4] = {nv.x, nv.y, nv.z, nv.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) c += (w[i] & 0xff) + ((w[i] >> 8) & 0xff) + ((w[i] >> 16) & 0xff) + (w[i] >> 24);
  uint32_t total;
  block_excl_scan(c, smem, total);
  if (threadIdx.x == 0) D.tile_sec[tile] = total;
  if (last_block_done(&ctl->ticket_pcount)) {
    const uint32_t S = block_scan_array(D.tile_sec, D.n_tiles, 1, smem);
    if (threadIdx.x == 0) {
      ctl->push_total = S;
      if (ctl->n_init + S > D.init_capacity) ctl->error = -4;  // CEL_ERR_INIT_OVERFLOW (sticky)
    }
  }
}

__global__ void __launch_bounds__(kTileThreads) k_push_write(DeviceState D) {
  __shared__ uint32_t smem[9];
  Control* ctl = D.ctl;
  if (ctl->finished) return;
  const uint32_t tile = blockIdx.x;
  const uint32_t base = tile * kTile + threadIdx.x * kKeysPerThread;
  const bool overflow = ctl->error != 0;
  const unsigned long long I = ctl->n_init;
  uint4 nv = *reinterpret_cast<const uint4*>(D.nsec + base);
  const uint8_t* nb = reinterpret_cast<const uint8_t*>(&nv);
  uint32_t c = 0;
#pragma unroll
  for (int i = 0; i < kKeysPerThread; ++i) c += nb[i];
  uint32_t total;
  uint32_t off = D.tile_sec[tile] + block_excl_scan(c, smem, total);
  if (c != 0) {
#pragma unroll 1
    for (int i = 0; i < kKeysPerThread; ++i) {
      const uint32_t n = nb[i];
      if (n == 0) continue;
      const uint32_t slot = base + i;
      if (!overflow) {
        for (uint32_t j = 0; j < n; ++j) {
          store_a(D.initA + I + off + j, load_a(D.secA + 2ull * slot + j));
          store_b(D.initB + I + off + j, load_b(D.secB + 2ull * slot + j));
        }
      }
      off += n;
    }
    *reinterpret_cast<uint4*>(D.nsec + base) = make_uint4(0, 0, 0, 0);
  }
  if (last_block_done(&ctl->ticket_pwrite)) {
    if (threadIdx.x == 0) {
      const unsigned long long S = ctl->push_total;
      if (!overflow) ctl->n_init = I + S;
      ctl->secondaries += S;
      ctl->iter += 1;
    }
  }
}

// ================================================================ loading, reset, debug helpers
struct PrimaryRec { uint32_t event; int32_t ptype; double energy; double pos[3]; double dir[3]; };  // = cel_primary, 64 B
struct TrackRec { double pos[3]; double dir[3]; double energy; uint32_t event, nsteps; int32_t vol, surf, ptype, action; };  // = cel_track

__device__ __forceinline__ int locate_volume(const Params& P, double x, double y, double z, double dz) {
  if (P.geom_kind == 0) {
    for (int i = 0; i < P.n_vol; ++i) {
      const double lo = P.bounds[i], hi = P.bounds[i + 1];
      if (z > lo && z < hi) return i;
      if (z == lo && dz >= 0.0) return i;
      if (z == hi && dz < 0.0) return i;
    }
    return -1;
  }
  const double r = sqrt(x * x + y * y);
  for (int i = 0; i < P.n_vol; ++i)
    if (r >= P.bounds[i] && r < P.bounds[i + 1]) return i;
  return -1;
}

// S9: primary i -> init[i]; the volume is located from the position (boundary -> the side it points into)
__global__ void k_load_primaries(DeviceState D, const PrimaryRec* prim, unsigned long long n) {
  for (unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; i < n; i += (unsigned long long)gridDim.x * blockDim.x) {
    const PrimaryRec p = prim[i];
    int vol = locate_volume(D.P, p.pos[0], p.pos[1], p.pos[2], p.dir[2]);
    if (vol < 0 || p.event >= D.n_events || p.ptype < 0 || p.ptype > 2) { D.ctl->error = -1; vol = 0; }
    RecA a; a.x = p.pos[0]; a.y = p.pos[1]; a.z = p.pos[2]; a.energy = p.energy;
    RecB b; b.dx = p.dir[0]; b.dy = p.dir[1]; b.dz = p.dir[2];
    b.meta = make_meta(p.ptype == P_GAMMA ? A_MOVE_G : A_MOVE_C, p.ptype, false, vol, -1, 0, p.event);
    store_a(D.initA + i, a);
    store_b(D.initB + i, b);
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) D.ctl->n_init = n;
}

__global__ void k_unpack(const RecA* A, const RecB* B, TrackRec* out, unsigned long long n, int as_initializer) {
  for (unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; i < n; i += (unsigned long long)gridDim.x * blockDim.x) {
    const RecA a = A[i]; const RecB b = B[i];
    TrackRec t;
    t.pos[0] = a.x; t.pos[1] = a.y; t.pos[2] = a.z; t.energy = a.energy;
    t.dir[0] = b.dx; t.dir[1] = b.dy; t.dir[2] = b.dz;
    t.event = meta_event(b.meta); t.nsteps = meta_nsteps(b.meta); t.vol = meta_vol(b.meta); t.surf = meta_surf(b.meta);
    t.ptype = meta_ptype(b.meta); t.action = as_initializer ? -1 : meta_action(b.meta);
    out[i] = t;
  }
}

__global__ void k_debug_uniforms(Params P, const uint32_t* slots, uint32_t n, uint32_t k, uint32_t phase, uint32_t j, double* out) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double xa, xb;
  draw_pair(P, slots[i], k, phase, j >> 1, xa, xb);
  out[i] = (j & 1u) ? xb : xa;
}

}  // namespace cel

namespace cel {
// every slot vacant: key byte 7, meta action VACANT (state bytes are otherwise zero)
__global__ void k_reset_state(DeviceState D) {
  const uint32_t padded = D.n_tiles * kTile;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < padded; i += gridDim.x * blockDim.x) {
    D.akey[i] = (uint8_t)A_VACANT;
    D.nsec[i] = 0;
    if (i < D.N) {
      RecA a; a.x = a.y = a.z = a.energy = 0.0;
      RecB b; b.dx = b.dy = b.dz = 0.0; b.meta = make_meta(A_VACANT, 0, false, 0, -1, 0, 0);
      store_a(D.stA + i, a); store_b(D.stB + i, b);
      store_stage(D.stage + i, 0, 0, 0, -1);
    }
  }
}
}  // namespace cel

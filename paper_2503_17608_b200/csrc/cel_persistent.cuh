// cel_persistent.cuh — the whole step iteration as ONE persistent cooperative kernel (docs/PHYSICS_SPEC.md S1).
// Every phase of cel_kernels.cuh / cel_physics.cuh runs as a device function; the kernel boundaries between the
// phases become grid-wide barriers, and the kernel loops over iterations until the run ends or `max_iters` is
// reached, so an iteration costs four barriers instead of eight launches. With 2^20 slots and a few thousand live
// tracks per iteration (overhead is exposed below ~3000 active tracks) the launch latency floor of the
// kernel-per-action form is ~40 us per iteration on a B200; this form removes it.
//   P1  fill       block b owns the contiguous tile run [b*tpb, (b+1)*tpb)                    -> barrier
//   P2  scatter    (sorted modes) per-key bases from all tiles' histograms; tile_vac -= filled  -> barrier
//   P3+P4 actions  warp-sized chunks of each action's index range, dealt round-robin to all warps: a warp never
//                  mixes actions in the by-action mode; heavy actions are dealt first    -> barrier
//   P5  push                                                                                     -> barrier
// The values every block needs (I, V, S, the key offsets, alive, finished) are recomputed by each block from the
// per-tile counter arrays, so no block waits for another block's scalar; block 0 alone writes the control block.
#pragma once
#include "cel_kernels.cuh"
#include "cel_physics.cuh"

namespace cel {

__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
// grid-wide barrier on a monotonic arrival counter (zeroed by the host before the launch); all blocks are
// co-resident (cooperative launch). `epoch` counts the arrivals that complete the barrier this block waits for.
__device__ __forceinline__ void grid_barrier(unsigned long long* counter, unsigned long long& epoch) {
  __syncthreads();
  if (threadIdx.x == 0) {
    epoch += gridDim.x;
    __threadfence();
    atomicAdd(counter, 1ull);
    while (ld_acquire_u64(counter) < epoch) { }
    __threadfence();
  }
  __syncthreads();
}

// per-key sums of tile_hist rows [0, tile0) and [0, n_tiles): result in sm.base[k] (prefix) and key_total[k]
__device__ __forceinline__ void block_prefix_total8(const uint32_t* tile_hist, uint32_t n_tiles, uint32_t tile0, BookSmem& sm,
                                                    uint32_t* key_total /* shared, 8 */) {
  uint32_t p[8] = {0, 0, 0, 0, 0, 0, 0, 0}, t[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  for (uint32_t i = threadIdx.x; i < n_tiles; i += kTileThreads) {
    const uint4 a = *reinterpret_cast<const uint4*>(tile_hist + i * 8), b = *reinterpret_cast<const uint4*>(tile_hist + i * 8 + 4);
    const uint32_t v[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
#pragma unroll
    for (int k = 0; k < 8; ++k) { t[k] += v[k]; if (i < tile0) p[k] += v[k]; }
  }
  __syncthreads();
  if (threadIdx.x < 8) { sm.base[threadIdx.x] = 0; key_total[threadIdx.x] = 0; }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const uint32_t ps = __reduce_add_sync(0xffffffffu, p[k]), ts = __reduce_add_sync(0xffffffffu, t[k]);
    if ((threadIdx.x & 31) == 0) { if (ps) atomicAdd(&sm.base[k], ps); if (ts) atomicAdd(&key_total[k], ts); }
  }
  __syncthreads();
}

// one track: load the second record (direction + meta), dispatch on the action
template <bool FIELD, int GEOM>
__device__ __forceinline__ void run_action(const DeviceState& D, uint32_t slot, uint32_t k_iter, int act_known) {
  const RecB b = load_b(D.stB + slot);
  const RecA a = load_a(D.stA + slot);
  const int act = act_known >= 0 ? act_known : meta_action(b.meta);
  switch (act) {
    case A_PE: do_photoelectric(D, slot, a, b); break;
    case A_PAIR: do_pair(D, slot, k_iter, a, b); break;
    case A_ANNIH: do_annihilation(D, slot, k_iter, a, b); break;
    case A_COMPTON:
    case A_MOVE_G: do_photon<GEOM>(D, slot, k_iter, a, b, act); break;
    case A_MOVE_C:
    case A_BREMS: do_charged<FIELD, GEOM>(D, slot, k_iter, a, b, act); break;
    default: break;
  }
}

// P3 + P4 for all actions. off[] = key offsets of the sorted index array (shared memory). The three modes differ only in
// how a warp-sized chunk maps to slots and where the action comes from; the track itself is processed at ONE call site,
// so every mode runs the same instructions on a track (tallies are bit-identical across sort modes).
//   by action:   7 ranges, one per action, heaviest first; chunk g of the concatenated ranges goes to warp g mod nw
//   by particle: one range [0, off[3]) = gamma | e- | e+; the action comes from the track (masked)
//   none:        one range [0, N), thread -> slot; the dense key byte masks vacant slots before any state is read
template <bool FIELD, int GEOM>
__device__ __forceinline__ void actions_phase(const DeviceState& D, const uint32_t* off, uint32_t k_iter) {
  const uint32_t lane = threadIdx.x & 31;
  const uint32_t gw = blockIdx.x * (kTileThreads / 32) + (threadIdx.x >> 5);
  const uint32_t nw = gridDim.x * (kTileThreads / 32);
  const int order[7] = {A_MOVE_C, A_BREMS, A_COMPTON, A_MOVE_G, A_PE, A_PAIR, A_ANNIH};
  const int n_ranges = D.sort_mode == 1 ? 7 : 1;
  uint32_t dealt = 0;
#pragma unroll 1
  for (int r = 0; r < n_ranges; ++r) {
    int a = -1;
    uint32_t b0 = 0, e0;
    if (D.sort_mode == 1) { a = order[r]; b0 = off[a]; e0 = off[a + 1]; }
    else if (D.sort_mode == 2) e0 = off[3];
    else e0 = D.N;
    const uint32_t chunks = (e0 - b0 + 31u) >> 5;
#pragma unroll 1
    for (uint32_t c = (gw + nw - dealt % nw) % nw; c < chunks; c += nw) {
      const uint32_t tid = b0 + c * 32u + lane;
      if (tid >= e0) continue;
      uint32_t slot = tid;
      int act = a;
      if (D.sort_mode != 0) slot = D.indices[tid];
      else { act = D.akey[slot] & 0xf; if (act == A_VACANT) continue; }
      run_action<FIELD, GEOM>(D, slot, k_iter, act);
    }
    dealt += chunks;
  }
}

constexpr int kMaxTilesPerBlock = 16;   // the host falls back to the kernel-per-action form if a block would own more

template <bool FIELD, int GEOM>
__global__ void __launch_bounds__(kTileThreads, FIELD ? 2 : 3) k_persistent(DeviceState D, uint32_t max_iters) {
  __shared__ BookSmem sm;
  __shared__ uint32_t key_total[8], act_total[8];
  __shared__ uint32_t off_s[9];
  __shared__ uint32_t tv_s[kMaxTilesPerBlock];   // tile_vac of the own tiles as read in P1 (before any action kernel adds)
  Control* ctl = D.ctl;
  if (ctl->finished || ctl->error != 0) return;   // same value in every block: nobody writes them before a barrier
  unsigned long long I = ctl->n_init;
  uint32_t k_iter = ctl->iter;
  unsigned long long epoch = 0;
  const uint32_t tpb = (D.n_tiles + gridDim.x - 1) / gridDim.x;
  const uint32_t tile0 = min(D.n_tiles, blockIdx.x * tpb), tile1 = min(D.n_tiles, tile0 + tpb);
  const int n_keys = D.sort_mode == 1 ? 8 : (D.sort_mode == 2 ? 4 : 0);
  const bool leader = blockIdx.x == 0 && threadIdx.x == 0;

  for (uint32_t it = 0; it < max_iters; ++it) {
    // ------------------------------------------------------------ P1: fill (S9) + per-tile histograms
    uint32_t prefix_v, V;
    block_prefix_total(D.tile_vac, D.n_tiles, tile0, sm.scan, prefix_v, V);
    const uint32_t n_take = (unsigned long long)V < I ? V : (uint32_t)I;
    const uint32_t alive = D.N - (V - n_take);
    if (alive == 0 && I == (unsigned long long)n_take) {   // A_k == 0 and I == 0 after the fill: the run has ended
      if (leader) {
        ctl->finished = 1; ctl->alive = 0; ctl->vac_total = V;
        for (int a = 0; a < 8; ++a) ctl->counts[a] = (a == A_VACANT) ? D.N : 0u;
      }
      break;
    }
    {
      uint32_t pv = prefix_v;
      for (uint32_t tile = tile0; tile < tile1; ++tile) {
        if (threadIdx.x < 8) { sm.hist[threadIdx.x] = 0; sm.act[threadIdx.x] = 0; }
        __syncthreads();
        const uint32_t tv = D.tile_vac[tile];
        if (threadIdx.x == 0) tv_s[tile - tile0] = tv;
        fill_tile(D, sm, tile, I, n_take, pv, tv);
        __syncthreads();
        publish_tile_hist(D, sm, tile);
        if (threadIdx.x == 8) D.tile_sec[tile] = 0;   // consumed by the push of the previous iteration
        pv += tv;
        __syncthreads();
      }
    }
    grid_barrier(&ctl->barrier, epoch);
    // ------------------------------------------------------------ P2: offsets, tile_vac -= filled, scatter (S2)
    // action counts = column sums of the action histogram (the leader logs them); per-key bases from the rows the
    // scatter sorts by. sm.base = (tiles before tile0)[key] of those rows.
    if (D.sort_mode == 2) {
      if (blockIdx.x == 0) block_prefix_total8(D.tile_hist, D.n_tiles, tile0, sm, act_total);
      block_prefix_total8(D.tile_phist, D.n_tiles, tile0, sm, key_total);
    } else if (D.sort_mode == 1 || blockIdx.x == 0) {
      block_prefix_total8(D.tile_hist, D.n_tiles, tile0, sm, key_total);
      if (threadIdx.x < 8) act_total[threadIdx.x] = key_total[threadIdx.x];
    }
    if (n_keys) {
      if (threadIdx.x == 0) {
        off_s[0] = 0;
        for (int k = 0; k < 8; ++k) off_s[k + 1] = (k < n_keys) ? off_s[k] + key_total[k] : off_s[k];
      }
    }
    __syncthreads();
    if (leader) update_control_after_fill(D, act_total, key_total, n_keys, I, V, n_take);
    {
      uint32_t pv = prefix_v;
      uint32_t run = (threadIdx.x < 8 && n_keys) ? sm.base[threadIdx.x] : 0;   // thread k carries key k's running base
      for (uint32_t tile = tile0; tile < tile1; ++tile) {
        const uint32_t tv = tv_s[tile - tile0];
        const uint32_t filled = filled_in_tile(tv, pv, n_take);
        pv += tv;
        if (n_keys) {
          __syncthreads();
          if (threadIdx.x < 8) { sm.base[threadIdx.x] = off_s[threadIdx.x] + run; run += sort_rows(D)[tile * 8 + threadIdx.x]; }
          __syncthreads();
          scatter_tile(D, sm, tile, tv - filled);
        }
        // the action kernels add to tile_vac atomically; in the mode without reindexing other blocks may already be
        // in P3, so the filled vacancies are taken off atomically as well
        __syncthreads();
        if (threadIdx.x == 0 && filled) atomicSub(&D.tile_vac[tile], filled);
      }
    }
    I -= n_take;
    if (n_keys) grid_barrier(&ctl->barrier, epoch);
    // ------------------------------------------------------------ P3 + P4: the actions, over their index ranges
    actions_phase<FIELD, GEOM>(D, off_s, k_iter);
    grid_barrier(&ctl->barrier, epoch);
    // ------------------------------------------------------------ P5: push (S9)
    uint32_t prefix_s, S;
    block_prefix_total(D.tile_sec, D.n_tiles, tile0, sm.scan, prefix_s, S);
    const bool overflow = I + S > D.init_capacity;
    {
      uint32_t ps = prefix_s;
      for (uint32_t tile = tile0; tile < tile1; ++tile) {
        const uint32_t ts = D.tile_sec[tile];
        push_tile(D, sm, tile, I, ps, ts, overflow);
        ps += ts;
      }
    }
    k_iter += 1;
    if (leader) {
      ctl->push_total = S;
      ctl->secondaries += S;
      ctl->iter = k_iter;
      if (overflow) ctl->error = -4;   // CEL_ERR_INIT_OVERFLOW (sticky)
      else ctl->n_init = I + S;
    }
    if (overflow) break;
    I += S;
    grid_barrier(&ctl->barrier, epoch);
  }
}

}  // namespace cel

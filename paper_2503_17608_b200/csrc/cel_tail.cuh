// cel_tail.cuh — the step iteration for SMALL populations: one block, one launch, many iterations.
//
// PAPER.md:79 (section 4, fig. 2): below a few thousand active tracks the fixed cost of an iteration is exposed. In the
// kernel-per-phase form an iteration is a chain of three dependent launches over thousands of mostly idle blocks (~20 us on
// this GPU however few tracks are left), and the long low-occupancy tail of a shower — or the curling tracks of the barrel
// configuration, 86 % of whose iterations carry fewer than 256 tracks — pays it every time. When the lagged status shows that
// tracks + initializers fit one block, the host enqueues k_tail instead of the iteration graph: ONE 512-thread block keeps
// the sorted list of live slots in shared memory and runs whole iterations back to back — P1 fill, the action counts and
// counters (S11), the actions (the same device functions as the action kernels), P5 push — separated by block barriers
// only, until the run ends, the iteration budget of the launch is used up, or the population outgrows the block (then it
// leaves every structure the kernels of cel_kernels.cuh start from as they expect it and the host switches back).
// The rules are those of docs/PHYSICS_SPEC.md S1, S9 (S9-R in sort mode 4), S10, S11 — the k-th vacancy in ascending slot
// order takes init[I-1-k], secondaries are pushed in ascending slot order, histories are keyed by (slot, iteration) — so
// tallies, counts and counters are bit-identical to the kernel-per-phase form (tests). The index array is not needed here:
// the live list is the reindexing (the actions run grouped by action for coherent warps).
#pragma once
#include "cel_kernels.cuh"
#include "cel_physics.cuh"

namespace cel {

constexpr int kTailThreads = 512;
constexpr int kTailCap = 1024;       // live slots + initializers the block accepts (two passes of the block)

struct TailSmem {
  uint32_t live[kTailCap];           // live slots, ascending
  uint32_t tmp[kTailCap];            // merge / compaction target, then swapped with live
  uint32_t order[kTailCap];          // live slots grouped by action (the block's "state_indices")
  uint32_t scan[kTailThreads / 32 + 2];
  uint32_t cnt[8], cursor[8];
  uint32_t n_live, n_tmp;
  uint32_t top;                      // one past the highest slot the fills of this launch reached
};

// exclusive scan over the block's kTailThreads threads; total to every thread. Ends with a barrier.
__device__ __forceinline__ uint32_t tail_block_scan(uint32_t v, uint32_t* sc, uint32_t& total) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t incl = warp_incl_scan(v);
  __syncthreads();
  if (lane == 31) sc[warp] = incl;
  __syncthreads();
  if (warp == 0) {
    uint32_t w = lane < kTailThreads / 32 ? sc[lane] : 0u;
    const uint32_t wi = warp_incl_scan(w);
    if (lane < kTailThreads / 32) sc[lane] = wi - w;
    if (lane == kTailThreads / 32 - 1) sc[kTailThreads / 32] = wi;
  }
  __syncthreads();
  total = sc[kTailThreads / 32];
  const uint32_t ex = sc[warp] + incl - v;
  __syncthreads();
  return ex;
}

// number of entries of the ascending list a[0..n) that are < x
__device__ __forceinline__ uint32_t lower_count(const uint32_t* a, uint32_t n, uint32_t x) {
  uint32_t lo = 0, hi = n;
  while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (a[mid] < x) lo = mid + 1; else hi = mid; }
  return lo;
}
// the slot of the r-th vacancy (ascending slot order) given the ascending list of live slots: live[i] - i is the number of
// vacancies below live[i] (non-decreasing), so slot = r + #{i : live[i] - i <= r}
__device__ __forceinline__ uint32_t vacancy_slot(const uint32_t* live, uint32_t n, uint32_t r) {
  uint32_t lo = 0, hi = n;
  while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (live[mid] - mid <= r) lo = mid + 1; else hi = mid; }
  return r + lo;
}

// in-place ascending sort of a[0..n), n <= kTailCap, by the whole block (bitonic over the next power of two; padding = ~0)
__device__ __forceinline__ void tail_sort(uint32_t* a, uint32_t n) {
  uint32_t m = 1; while (m < n) m <<= 1;
  for (uint32_t i = n + threadIdx.x; i < m; i += kTailThreads) a[i] = 0xffffffffu;
  __syncthreads();
  for (uint32_t k = 2; k <= m; k <<= 1)
    for (uint32_t j = k >> 1; j > 0; j >>= 1) {
      for (uint32_t i = threadIdx.x; i < m; i += kTailThreads) {
        const uint32_t l = i ^ j;
        if (l > i) {
          const uint32_t x = a[i], y = a[l];
          const bool up = (i & k) == 0;
          if ((x > y) == up) { a[i] = y; a[l] = x; }
        }
      }
      __syncthreads();
    }
}

// one slot's action of iteration k (P3i + P3m + P4), exactly what the action kernels do for it
template <bool FIELD, int GEOM>
__device__ __forceinline__ void tail_act(const DeviceState& D, uint32_t slot, uint32_t k) {
  const RecB b = load_b(D.stB + slot);
  const RecA a = load_a(D.stA + slot);
  const int act = meta_action(b.meta);
  if (act == A_MOVE_C || act == A_BREMS) do_charged<FIELD, GEOM>(D, slot, k, a, b, act);
  else if (act == A_MOVE_G || act == A_COMPTON) do_photon<GEOM>(D, slot, k, a, b, act);
  else if (act == A_PE) do_photoelectric(D, slot, k, a, b);
  else if (act == A_PAIR) do_pair(D, slot, k, a, b);
  else if (act == A_ANNIH) do_annihilation(D, slot, k, a, b);
}

template <bool FIELD, int GEOM>
__global__ void __launch_bounds__(kTailThreads, 1) k_tail(DeviceState Din, uint32_t max_iters) {
  __shared__ TailSmem sm;
  Control* ctl = Din.ctl;
  uint32_t k = ctl->iter;
  unsigned long long I = ctl->n_init;
  // not for this block: already over, in error, or (conservatively: nothing is born between P1 and here except on the
  // stack) more than the block holds
  if (ctl->finished || ctl->error != 0 || (unsigned long long)ctl->alive + I > (unsigned long long)kTailCap) return;
  // vacancies are kept in ONE buffer of the parity pair for the whole launch (the action functions add theirs to it)
  const uint32_t pb = k & 1u;
  DeviceState D = Din;
  D.vac_buf_override = 1 + (int)pb;
  uint32_t* const tvac = D.tile_vac + (size_t)pb * D.n_tiles;
  const uint32_t tid = threadIdx.x;
  unsigned long long track_steps = ctl->track_steps, iterations = ctl->iterations, secondaries = ctl->secondaries;
  uint32_t n_logged = ctl->n_logged;

  // ---- the live list: every non-vacant slot of the live tiles (Control::tiles_hi) that are not entirely vacant, then sorted.
  // First the list of those tiles (sm.tmp; more than kTailCap of them cannot be: each holds a track), all counters in flight
  // at once; then their key bytes.
  const uint32_t T = ctl->tiles_hi[pb];
  if (tid == 0) { sm.n_live = 0; sm.n_tmp = 0; sm.top = 0; }
  __syncthreads();
  for (uint32_t t = tid; t < T; t += kTailThreads)
    if (__ldcg(tvac + t) != real_slots_in_tile(D, t)) { const uint32_t at = atomicAdd(&sm.n_tmp, 1u); if (at < (uint32_t)kTailCap) sm.tmp[at] = t; }
  __syncthreads();
  const uint32_t n_live_tiles = sm.n_tmp;
  if (n_live_tiles > (uint32_t)kTailCap) return;   // (cannot happen: live tiles <= live tracks <= ctl->alive; nothing has been changed yet)
  for (uint32_t j = 0; j < n_live_tiles; ++j) {
    const uint32_t t = sm.tmp[j];
    const uint32_t base = t << D.tile_shift, end = min(base + (1u << D.tile_shift), D.N);
    for (uint32_t s = base + 4 * tid; s < end; s += 4 * kTailThreads) {
      const uint32_t kv = *reinterpret_cast<const uint32_t*>(D.akey + s);    // padding bytes are 0xff: skipped below by s + i < end
#pragma unroll
      for (int i = 0; i < 4; ++i)
        if (s + i < end && ((kv >> (8 * i)) & 0xf) != A_VACANT) { const uint32_t at = atomicAdd(&sm.n_live, 1u); if (at < (uint32_t)kTailCap) sm.live[at] = s + i; }
    }
  }
  __syncthreads();
  uint32_t n_live = sm.n_live;
  if (n_live > (uint32_t)kTailCap) return;   // (cannot happen: n_live <= ctl->alive; nothing has been changed yet)
  tail_sort(sm.live, n_live);
  uint32_t* live = sm.live; uint32_t* other = sm.tmp;

  uint32_t done = 0;
  bool finished = false, overflow = false;
  for (; done < max_iters; ++done, ++k) {
    if ((unsigned long long)n_live + I > (unsigned long long)kTailCap) break;   // outgrown: back to the kernels
    // ---- P1 (S9): the r-th vacancy in ascending slot order takes init[I-1-r]
    const uint32_t V = D.N - n_live;
    const uint32_t n_take = (unsigned long long)V < I ? V : (uint32_t)I;
    if (n_take) {
      for (uint32_t w = tid; w < 2 * n_take; w += kTailThreads) {
        const uint32_t r = w >> 1;
        const uint32_t slot = vacancy_slot(live, n_live, r);
        const unsigned long long src = I - 1ull - r;
        if (w & 1) {
          const RecB b = load_b(D.initB + src);
          store_b(D.stB + slot, b);
          D.akey[slot] = make_key(meta_action(b.meta), meta_ptype(b.meta));
          atomicSub(tvac + (slot >> D.tile_shift), 1u);
          if (r == n_take - 1u && slot >= sm.top) sm.top = slot + 1u;   // (ascending: the last vacancy taken is the highest; one thread)
          other[r + (slot - r)] = slot;          // merged position of the new slot: r + #{live < slot} = slot's own c(r) = slot - r
        } else {
          store_a(D.stA + slot, load_a(D.initA + src));
        }
      }
      // merged position of an old live slot: its index + the number of new slots below it = #{r : vacancy_slot(r) < live[i]}
      // = min(n_take, vacancies below live[i]) = min(n_take, live[i] - i)
      for (uint32_t i = tid; i < n_live; i += kTailThreads) other[i + min(n_take, live[i] - i)] = live[i];
      __syncthreads();
      uint32_t* t2 = live; live = other; other = t2;
      n_live += n_take; I -= n_take;
    }
    // ---- the iteration's action counts (S11) and the grouping by action
    if (tid < 8) { sm.cnt[tid] = 0; }
    __syncthreads();
    for (uint32_t i = tid; i < n_live; i += kTailThreads) atomicAdd(&sm.cnt[__ldcg(D.akey + live[i]) & 0xf], 1u);
    __syncthreads();
    if (n_live == 0 && I == 0) { finished = true; break; }
    if (tid == 0) {
      uint32_t run = 0;
      for (int a = 0; a < 8; ++a) { sm.cursor[a] = run; run += sm.cnt[a]; }
      if (n_logged < D.log_capacity) {
        for (int a = 0; a < 7; ++a) D.counts_log[(size_t)n_logged * 8 + a] = sm.cnt[a];
        D.counts_log[(size_t)n_logged * 8 + 7] = D.N - n_live;
      }
    }
    if (n_logged < D.log_capacity) ++n_logged;
    track_steps += n_live; iterations += 1;
    __syncthreads();
    for (uint32_t i = tid; i < n_live; i += kTailThreads) { const uint32_t s = live[i]; sm.order[atomicAdd(&sm.cursor[__ldcg(D.akey + s) & 0xf], 1u)] = s; }
    __syncthreads();
    // ---- P3i + P3m + P4: one thread per live slot, grouped by action
    for (uint32_t i = tid; i < n_live; i += kTailThreads) tail_act<FIELD, GEOM>(D, sm.order[i], k);
    __syncthreads();
    // ---- P5 (S9): secondaries appended in ascending slot order; then the vacated slots leave the list
    uint32_t S = 0, n_keep = 0;
    for (uint32_t base = 0; base < n_live; base += kTailThreads) {   // block-uniform
      const uint32_t i = base + tid;
      uint32_t slot = 0, ns = 0, keep = 0;
      if (i < n_live) {
        slot = live[i];
        ns = __ldcg(D.nsec + slot);
        keep = (__ldcg(D.akey + slot) & 0xf) != A_VACANT ? 1u : 0u;
      }
      uint32_t tot_s, tot_k;
      const uint32_t off = tail_block_scan(ns, sm.scan, tot_s);
      const uint32_t kpos = tail_block_scan(keep, sm.scan, tot_k);
      if (I + S + tot_s > D.init_capacity) overflow = true;          // block-uniform
      if (ns && !overflow) {
        for (uint32_t j = 0; j < ns; ++j) {
          const unsigned long long dst = I + S + off + j;
          store_a(D.initA + dst, load_a(D.secA + 2ull * slot + j));
          store_b(D.initB + dst, load_b(D.secB + 2ull * slot + j));
        }
      }
      if (ns) D.nsec[slot] = 0;
      if (keep) other[n_keep + kpos] = slot;
      S += tot_s; n_keep += tot_k;
    }
    __syncthreads();
    { uint32_t* t2 = live; live = other; other = t2; }
    n_live = n_keep;
    if (overflow) { ++done; ++k; break; }
    I += S; secondaries += S;
  }

  // ---- leave everything as the kernels of cel_kernels.cuh expect it at the start of iteration k
  __syncthreads();
  // the live tiles as the kernels expect them (cel_kernels.cuh: tile_prefix): now those of the entry, or up to the highest
  // slot a fill of this launch reached; for the fill of iteration k, what k_push would have set: min(V, I) vacancies in
  // ascending order, vac_low of them below T_out, the rest in the consecutive vacant slots above
  uint32_t T_out = (uint32_t)(((unsigned long long)sm.top + (1ull << D.tile_shift) - 1ull) >> D.tile_shift);
  if (T_out < T) T_out = T;
  uint32_t T_next = T_out, vac_low;
  {
    uint32_t v = 0;
    for (uint32_t t = tid; t < T_out; t += kTailThreads) v += __ldcg(tvac + t);
    tail_block_scan(v, sm.scan, vac_low);
    const uint32_t below = slots_below_tile(D, T_out);
    const unsigned long long V = (unsigned long long)vac_low + (D.N - below);
    const unsigned long long n_take = V < I ? V : I;
    if (n_take > vac_low) {
      const unsigned long long top = (unsigned long long)below + (n_take - vac_low);
      T_next = (uint32_t)((top + (1ull << D.tile_shift) - 1ull) >> D.tile_shift);
      if (T_next > D.n_tiles) T_next = D.n_tiles;
      if (T_next < T_out) T_next = T_out;
    }
  }
  if ((k & 1u) != pb) {   // fill(k) reads the vacancy counters of parity k&1
    uint32_t* dst = D.tile_vac + (size_t)(k & 1u) * D.n_tiles;
    for (uint32_t t = tid; t < T_out; t += kTailThreads) dst[t] = tvac[t];
  }
  for (uint32_t i = tid; i < D.n_groups * kRowWords; i += kTailThreads) group_row(D, k & 1u, 0)[i] = 0u;   // the rows fill(k) adds into
  if (tid < kMaxGroups / 32) D.group_mask[(k & 1u) * (kMaxGroups / 32) + tid] = 0u;
  if (tid == 0) {
    for (int a = 0; a < 7; ++a) ctl->counts[a] = sm.cnt[a];
    ctl->counts[7] = D.N - n_live;
    ctl->alive = n_live;   // (an upper bound of the live tracks, as after P1 of the last iteration: what the host's switch looks at)
    ctl->n_init = I; ctl->n_init_fill = I;
    ctl->iter = k; ctl->iter_cur = k - 1u;
    ctl->tiles_hi[(k & 1u) ^ 1u] = T_out; ctl->tiles_hi[k & 1u] = T_next; ctl->vac_low[k & 1u] = vac_low;
    ctl->track_steps = track_steps; ctl->iterations = iterations; ctl->secondaries = secondaries; ctl->n_logged = n_logged;
    if (finished) ctl->finished = 1;
    if (overflow) ctl->error = -4;   // CEL_ERR_INIT_OVERFLOW (sticky)
  }
}

}  // namespace cel

// cel_kernels.cuh — the bookkeeping kernels of one step iteration (docs/PHYSICS_SPEC.md S1):
//   P1 init + P2 reindex:   k_fill_sort   (scan-based vacancy filling, S9; stable counting sort of slot indices, S2;
//                                          the iteration's counts, ranges and counters, S11) — ONE pass, one launch
//   P5 push:                k_push        (scan-ordered secondary push, S9)
//   S9-P (sort mode 3):     k_part_count, k_part_scatter (charged / neutral partition of the popped initializers)
// (P3/P4, the action kernels and the scoring, are in cel_physics.cuh.)
//
// One 256-thread block per tile of 2^tile_shift consecutive slots. What makes a single pass possible:
//  * the action kernels keep per-tile counters of vacancies created and secondaries staged (integer atomics), so a
//    block gets its exclusive prefix from one strided read of the live tiles' counters (<= 8192) — no counting pass, no look-back chain;
//  * the index array is kept in REGIONS of N entries, one per sort key: region k holds the slots of key k in ascending
//    order from k*N, so where a tile writes depends only on the tiles BEFORE it (their per-key counts), never on
//    totals. A block publishes its tile's histogram (own row + atomics on its group's row), then waits for the tiles
//    before it — whole lower groups through an arrival counter in the group row, lower tiles of its own group through
//    a per-tile iteration stamp — and scatters from the key bytes it still holds in shared memory. Dependencies point
//    only to lower block indices, which the hardware dispatches first, so the wait cannot deadlock even when the
//    grid is only partly resident (several contexts sharing the GPU); a bounded spin turns the impossible case into
//    the sticky error CEL_ERR_INTERNAL instead of a hang.
//  * the block of the LAST tile, which by then has seen every other tile's counts, writes the iteration's totals,
//    ranges and counters to the control block (fields no block of this kernel reads).
// The vacancy counters are double-buffered by the parity of the iteration: fill(k) reads buffer k&1 (complete once the
// action kernels of k-1 are), writes what is left of its tile into buffer (k&1)^1, which the action kernels of k then
// add to. So the prefix can be formed BEFORE the programmatic-dependency wait and overlaps the push of the previous iteration.
#pragma once
#include "cel_device.cuh"

namespace cel {

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
// exclusive scan over the 256 threads of a block; returns the exclusive prefix, total in `total`
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
__device__ __forceinline__ int sort_key_of(int sort_mode, uint32_t key) {
  const int a = key & 0xf;
  if (sort_mode == 1) return a;
  return a == A_VACANT ? 3 : ((key >> 4) & 0x3);
}
// number of the 4 key bytes of w whose action nibble is VACANT (padding bytes are 0xff, never vacant)
__device__ __forceinline__ uint32_t count_vacant4(uint32_t w) {
  const uint32_t x = (w & 0x0f0f0f0fu) ^ 0x07070707u;           // byte == 0 <=> vacant
  const uint32_t z = ~(((x & 0x7f7f7f7fu) + 0x7f7f7f7fu) | x) & 0x80808080u;  // 0x80 where the byte is 0
  return __popc(z);
}

// loads that must see what other SMs published through L2 (atomics / stores + fence): never from L1
__device__ __forceinline__ uint32_t load_acquire(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void store_release(uint32_t* p, uint32_t v) {
  asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// ---------------------------------------------------------------- shared memory of a bookkeeping block
constexpr int kResidentSubs = 4;   // sub-tiles whose key bytes stay in shared memory between the fill and the scatter
struct BookSmem {
  uint32_t scan[20];
  unsigned long long scan64[9];
  uint32_t hist[8], act[8], base[8];
  uint32_t part[3 * 9];            // per-warp partial sums of the prefix reductions
  uint32_t before[12];             // per-key counts of the tiles before this one: 0-7 action keys, 8-11 particle keys
  uint32_t skey[kResidentSubs * kTileThreads];   // key bytes of the tile's sub-tiles
  uint32_t list[2 * kSub];         // compacted work list of the cooperative copies
};

__device__ __forceinline__ uint32_t real_slots_in_tile(const DeviceState& D, uint32_t tile) {
  const unsigned long long lo = (unsigned long long)tile << D.tile_shift, hi = lo + (1ull << D.tile_shift);
  return lo >= D.N ? 0u : (uint32_t)((hi < D.N ? hi : (unsigned long long)D.N) - lo);
}
__device__ __forceinline__ uint32_t tiles_in_group(uint32_t n_tiles, uint32_t g) {
  const uint32_t lo = g * kGroupTiles;
  return lo >= n_tiles ? 0u : min((uint32_t)kGroupTiles, n_tiles - lo);
}
// slots of the first t tiles
__device__ __forceinline__ uint32_t slots_below_tile(const DeviceState& D, uint32_t t) {
  const unsigned long long s = (unsigned long long)t << D.tile_shift;
  return s < D.N ? (uint32_t)s : D.N;
}

// Exclusive prefix of a per-tile counter by one block: the sum over the tiles before `tile`, the total and the tile's own
// counter, over the first n counters (the live tiles, below). Threads stride over them (n <= 8192: at most 32 loads per
// thread, issued back to back before the first use: one L2 round trip). Uses sm.part; a second call needs a barrier first.
//
// Live tiles (Control::tiles_hi): vacancies are filled in ascending slot order, so the tracks of a run occupy a prefix of
// the slot array whose end only moves up when the population outgrows it; every tile at or above tiles_hi[k & 1] is
// entirely vacant throughout iteration k, its counters still hold what k_reset_state wrote, and its blocks leave at once.
// k_push of iteration k-1 sets the bound for iteration k from the stack height: the fill takes min(V, I) vacancies, the
// first vac_low of them below the old bound, the rest in the consecutive vacant slots above it.
__device__ __forceinline__ void tile_prefix(BookSmem& sm, const uint32_t* tile_cnt, uint32_t n, uint32_t tile,
                                            uint32_t& prefix, uint32_t& total, uint32_t& own) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  uint32_t before = 0, all = 0, mine = 0;
  for (uint32_t i0 = 0; i0 < n; i0 += 4 * kTileThreads) {
    uint32_t v[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) { const uint32_t i = i0 + u * kTileThreads + threadIdx.x; v[u] = i < n ? __ldcg(tile_cnt + i) : 0u; }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const uint32_t i = i0 + u * kTileThreads + threadIdx.x;
      all += v[u];
      if (i < tile) before += v[u];
      if (i == tile) mine = v[u];
    }
  }
  before = __reduce_add_sync(0xffffffffu, before);
  all = __reduce_add_sync(0xffffffffu, all);
  mine = __reduce_add_sync(0xffffffffu, mine);
  __syncthreads();
  if (lane == 0) { sm.part[warp] = before; sm.part[9 + warp] = all; sm.part[18 + warp] = mine; }
  __syncthreads();
  uint32_t p = 0, t = 0, o = 0;
#pragma unroll
  for (int w = 0; w < kTileThreads / 32; ++w) { p += sm.part[w]; t += sm.part[9 + w]; o += sm.part[18 + w]; }
  prefix = p; total = t; own = o;
}

// ================================================================ P1: vacancy scan + fill (S9), P2 histogram (S2)
// Rank-r vacant slot (ascending slot order) takes init[I-1-r] when r < I (LIFO). The rank of a tile's first vacancy
// (`prefix`) comes from the two-level vacancy counters — scan-based, no atomics in the assignment, so the slot
// assignment is deterministic. Adds the tile's action histogram to sm.act and (sort by particle) its
// sort-key histogram to sm.hist; the caller zeroes both and synchronises before, and synchronises after. Leaves the
// (updated) key bytes of the first kResidentSubs sub-tiles in sm.skey.
// Which vacancies are filled: ranks [0, low_n) and [high_start, V). Plain rule (S9): low_n = n_take, high_start = V
// (none at the high end), rank r takes pop position r. Partition rule (S9-P, sort mode 3): low_n = C charged,
// high_start = V - G neutral; rank r < C takes the pop position plist[r], rank r >= V - G takes plist[n_take-1-(V-1-r)]
// (plist = D.indices, written by k_part_scatter).
struct FillPlan { uint32_t n_take, low_n, high_start, V; bool partition; };
__device__ __forceinline__ FillPlan plain_plan(uint32_t n_take) { FillPlan p; p.n_take = n_take; p.low_n = n_take; p.high_start = 0xffffffffu; p.V = 0; p.partition = false; return p; }
__device__ __forceinline__ FillPlan partition_plan(uint32_t n_take, uint32_t V, uint32_t n_charged) {
  FillPlan p; p.n_take = n_take; p.low_n = n_charged; p.high_start = V - (n_take - n_charged); p.V = V; p.partition = true; return p;
}
// vacancies of ranks [prefix, prefix + v) that the plan fills
__device__ __forceinline__ uint32_t filled_by_plan(uint32_t v, uint32_t prefix, const FillPlan& pl) {
  const uint32_t end = prefix + v;
  const uint32_t lo = min(end, pl.low_n) > prefix ? min(end, pl.low_n) - prefix : 0u;
  const uint32_t hs = max(prefix, pl.high_start);
  return lo + (end > hs ? end - hs : 0u);
}
// adds the action histogram (and, sorted by particle, the sort-key histogram) of this thread's 4 key bytes to sm.act / sm.hist
__device__ __forceinline__ void add_key_histograms(const DeviceState& D, BookSmem& sm, uint32_t kv) {
  // histograms of this thread's 4 keys, 8 x 8-bit packed (padding bytes 0xff are skipped)
  uint32_t a_lo = 0, a_hi = 0, s_lo = 0;
#pragma unroll
  for (int i = 0; i < kKeysPerThread; ++i) {
    const uint32_t kb = (kv >> (8 * i)) & 0xff;
    if (kb != 0xff) {
      const uint32_t a = kb & 0xf;
      if (a < 4) a_lo += 1u << (8 * a); else a_hi += 1u << (8 * (a - 4));
      if (D.sort_mode == 2) s_lo += 1u << (8 * sort_key_of(2, kb));
    }
  }
  // warp totals: at most 128 per key, so the 8-bit fields cannot carry
  a_lo = __reduce_add_sync(0xffffffffu, a_lo); a_hi = __reduce_add_sync(0xffffffffu, a_hi);
  if (D.sort_mode == 2) s_lo = __reduce_add_sync(0xffffffffu, s_lo);
  {  // lanes 0-7 add the warp's count of key `lane`
    const uint32_t lane = threadIdx.x & 31;
    if (lane < 8) {
      const uint32_t sh = 8 * (lane & 3);
      const uint32_t a = ((lane < 4 ? a_lo : a_hi) >> sh) & 0xff;
      if (a) atomicAdd(&sm.act[lane], a);
      if (D.sort_mode == 2 && lane < 4) { const uint32_t h = (s_lo >> sh) & 0xff; if (h) atomicAdd(&sm.hist[lane], h); }
    }
  }
}

// returns true if the tile's key bytes were read (false: the tile is entirely vacant and gets no fill)
// kv0: the key bytes of the thread's four slots in sub-tile 0, loaded by the caller ahead of time
__device__ __forceinline__ bool fill_tile(const DeviceState& D, BookSmem& sm, uint32_t tile, unsigned long long I, const FillPlan pl,
                                          uint32_t prefix, uint32_t tile_vacant, uint32_t kv0) {
  uint32_t rank0 = prefix;                                   // rank of the first vacancy of the current sub-tile
  const uint32_t rank_end = prefix + tile_vacant;            // one past the rank of the tile's last vacancy
  const uint32_t real = real_slots_in_tile(D, tile);
  // all vacant, nothing to fill: no key byte needs reading (unless the debug surface wants the vacant indices written too)
  if (!D.write_vacant && tile_vacant == real && filled_by_plan(tile_vacant, prefix, pl) == 0) {
    if (threadIdx.x == 0) { sm.act[A_VACANT] = real; if (D.sort_mode == 2) sm.hist[3] = real; }
    return false;
  }
  for (uint32_t sub = 0; sub < D.subs_per_tile; ++sub) {
    const uint32_t sub_base = (tile << D.tile_shift) + sub * kSub;
    const uint32_t base = sub_base + threadIdx.x * kKeysPerThread;
    uint32_t kv = sub == 0 ? kv0 : *reinterpret_cast<const uint32_t*>(D.akey + base);
    // (beyond kResidentSubs: scratch only — the upper half of sm.list, which the fill does not use; NOT a resident sub-tile's place)
    uint32_t* skey = sub < (uint32_t)kResidentSubs ? sm.skey + sub * kTileThreads : sm.list + kSub;
    uint8_t* skey_b = reinterpret_cast<uint8_t*>(skey);
    if (rank0 < rank_end && filled_by_plan(rank_end - rank0, rank0, pl) != 0) {   // block-uniform: this sub-tile may have vacancies to fill
      const uint32_t c = count_vacant4(kv);
      uint32_t total;
      uint32_t r = block_excl_scan(c, sm.scan, total);
      skey[threadIdx.x] = kv;
      if (c) {
#pragma unroll
        for (int i = 0; i < kKeysPerThread; ++i)
          if (((kv >> (8 * i)) & 0xf) == A_VACANT) { sm.list[r] = base + i; ++r; }
      }
      __syncthreads();
      // filled items of the sub-tile's list: [0, n_lo) at the low end of the ranks, [hi_begin, total) at the high end
      const uint32_t n_lo = pl.low_n > rank0 ? min(total, pl.low_n - rank0) : 0u;
      const uint32_t hi_begin = pl.high_start > rank0 ? min(total, pl.high_start - rank0) : 0u;
      const uint32_t nf = n_lo + (total - hi_begin);
      // cooperative copy: work item w = (record, half); half 0 = RecA, half 1 = RecB (+ the key byte).
      // (Tried: two passes in flight per thread through cp.async landing slots in shared memory — 16 KB more shared
      // memory per block cost more in lost overlap with the neighbouring kernels than the pipelining gained: +7 %.)
      for (uint32_t m = threadIdx.x; m < nf; m += kTileThreads) {   // one record per thread and pass: both halves in flight together
        const uint32_t item = m < n_lo ? m : hi_begin + (m - n_lo);
        const uint32_t slot = sm.list[item];
        const uint32_t rank = rank0 + item;
        uint32_t pop = rank;                                 // plain rule: rank r takes init[I-1-r]
        if (pl.partition) pop = D.indices[rank < pl.low_n ? rank : pl.n_take - 1u - (pl.V - 1u - rank)];
        const unsigned long long src = I - 1ull - (unsigned long long)pop;
        const RecB b = load_b(D.initB + src);
        const RecA a = load_a(D.initA + src);
        store_b(D.stB + slot, b);
        const uint8_t key = make_key(meta_action(b.meta), meta_ptype(b.meta));
        D.akey[slot] = key;
        skey_b[slot - sub_base] = key;
        store_a(D.stA + slot, a);
      }
      __syncthreads();
      kv = skey[threadIdx.x];
      rank0 += total;
    } else if (sub < (uint32_t)kResidentSubs) {
      skey[threadIdx.x] = kv;
    }
    add_key_histograms(D, sm, kv);
  }
  return true;
}

// ---- the tiles the population grows into (at or above the live tiles of the previous iteration: entirely vacant, so the
// fills that reach them land on CONSECUTIVE slots: slot `below + m` takes init[I-1-(vac_low+m)], m < n_high). One block per
// tile would copy its 1024+ records a few per thread and round trip, while the blocks above the live tiles have nothing
// to do: those copy the records (grown_copy, a grid-stride loop, about one record half per thread), and the tile's own
// block only reads the 8-byte meta words it needs for the key bytes and the histograms (fill_grown_tile).
__device__ __forceinline__ void grown_copy(const DeviceState& D, unsigned long long I, uint32_t vac_low, uint32_t below,
                                           uint32_t n_high, uint32_t helper, uint32_t n_helpers) {
  for (unsigned long long w = (unsigned long long)helper * kTileThreads + threadIdx.x; w < 2ull * n_high; w += (unsigned long long)n_helpers * kTileThreads) {
    const uint32_t m = (uint32_t)(w >> 1);
    const unsigned long long src = I - 1ull - (unsigned long long)(vac_low + m);
    const uint32_t slot = below + m;
    if (w & 1) store_b(D.stB + slot, load_b(D.initB + src));
    else store_a(D.stA + slot, load_a(D.initA + src));
  }
}
__device__ __forceinline__ bool fill_grown_tile(const DeviceState& D, BookSmem& sm, uint32_t tile, unsigned long long I, uint32_t vac_low,
                                                uint32_t below, uint32_t n_high, uint32_t kv0) {
  const uint32_t tile_base = tile << D.tile_shift;
  if (tile_base - below >= n_high) {   // no fill reaches it (the bound is a whole tile count)
    if (threadIdx.x == 0) { sm.act[A_VACANT] = real_slots_in_tile(D, tile); if (D.sort_mode == 2) sm.hist[3] = sm.act[A_VACANT]; }
    return false;
  }
  for (uint32_t sub = 0; sub < D.subs_per_tile; ++sub) {
    const uint32_t base = tile_base + sub * kSub + threadIdx.x * kKeysPerThread;
    uint32_t kv = sub == 0 ? kv0 : *reinterpret_cast<const uint32_t*>(D.akey + base);
    unsigned long long meta[kKeysPerThread];
#pragma unroll
    for (int i = 0; i < kKeysPerThread; ++i) {   // (slots below `below + n_high` are real slots)
      const uint32_t m = base + i - below;
      meta[i] = m < n_high ? reinterpret_cast<const unsigned long long*>(D.initB + (I - 1ull - (unsigned long long)(vac_low + m)))[3] : 0ull;
    }
    bool any = false;
#pragma unroll
    for (int i = 0; i < kKeysPerThread; ++i)
      if (base + i - below < n_high) {
        kv = (kv & ~(0xffu << (8 * i))) | ((uint32_t)make_key(meta_action(meta[i]), meta_ptype(meta[i])) << (8 * i));
        any = true;
      }
    if (any) *reinterpret_cast<uint32_t*>(D.akey + base) = kv;
    if (sub < (uint32_t)kResidentSubs) sm.skey[sub * kTileThreads + threadIdx.x] = kv;
    add_key_histograms(D, sm, kv);
  }
  return true;
}

// Group rows of the two-level histograms: [2 (iteration parity)][kMaxGroups][kRowWords]; words 0-7 action counts of the
// group's tiles, 8-11 particle-key counts (sort by particle), 12 the number of tiles of the group that have published.
// The blocks of iteration k add into the rows of parity k&1 and zero the rows iteration k+1 will add into.
__device__ __forceinline__ uint32_t* group_row(const DeviceState& D, uint32_t parity, uint32_t g) {
  return D.group_rows + ((size_t)parity * kMaxGroups + g) * kRowWords;
}
constexpr uint32_t kSpinLimit = 1u << 24;   // polls before a wait gives up (~ a second): CEL_ERR_INTERNAL instead of a hang

// ================================================================ P2: stable scatter of slot indices (S2)
// indices[region(key) + (tiles before)[key] + (rank inside the tile)] = slot; ascending slot order inside a key.
// The caller sets sm.base[key] and synchronises. Vacant slots are never launched: their indices are written only when
// the complete permutation is asked for (debug surface). Key bytes come from shared memory (left there by fill_tile) for
// the first kResidentSubs sub-tiles.
// The same for a tile of ONE sub-tile, in two halves: the ranks inside the tile (everything that does not depend on other
// tiles: key counts, the two block scans) are formed BEFORE the block waits for the tiles before it, the index stores after.
__device__ __forceinline__ void scatter_ranks(const DeviceState& D, BookSmem& sm, unsigned long long& plo, unsigned long long& phi) {
  const uint32_t kv = sm.skey[threadIdx.x];
  unsigned long long lo = 0, hi = 0;
#pragma unroll
  for (int i = 0; i < kKeysPerThread; ++i) {
    const uint32_t kb = (kv >> (8 * i)) & 0xff;
    if (kb != 0xff) {
      const int s = sort_key_of(D.sort_mode, kb);
      if (s < 4) lo += 1ull << (16 * s); else hi += 1ull << (16 * (s - 4));
    }
  }
  unsigned long long tot;
  plo = block_excl_scan64(lo, sm.scan64, tot);
  phi = 0;
  if (D.sort_mode == 1) phi = block_excl_scan64(hi, sm.scan64, tot);
}
__device__ __forceinline__ void scatter_store(const DeviceState& D, BookSmem& sm, uint32_t tile, unsigned long long plo, unsigned long long phi) {
  const int vacant_key = D.sort_mode == 1 ? (int)A_VACANT : 3;
  const uint32_t base = (tile << D.tile_shift) + threadIdx.x * kKeysPerThread;
  const uint32_t kv = sm.skey[threadIdx.x];
#pragma unroll
  for (int i = 0; i < kKeysPerThread; ++i) {
    const uint32_t kb = (kv >> (8 * i)) & 0xff;
    if (kb != 0xff) {
      const int s = sort_key_of(D.sort_mode, kb);
      uint32_t r;
      if (s < 4) { r = (uint32_t)((plo >> (16 * s)) & 0xffff); plo += 1ull << (16 * s); }
      else { r = (uint32_t)((phi >> (16 * (s - 4))) & 0xffff); phi += 1ull << (16 * (s - 4)); }
      if (s != vacant_key || D.write_vacant) D.indices[(size_t)s * D.N + sm.base[s] + r] = base + i;
    }
  }
}
__device__ __forceinline__ void scatter_tile(const DeviceState& D, BookSmem& sm, uint32_t tile) {
  const int vacant_key = D.sort_mode == 1 ? (int)A_VACANT : 3;
  for (uint32_t sub = 0; sub < D.subs_per_tile; ++sub) {
    const uint32_t base = (tile << D.tile_shift) + sub * kSub + threadIdx.x * kKeysPerThread;
    const uint32_t kv = sub < (uint32_t)kResidentSubs ? sm.skey[sub * kTileThreads + threadIdx.x] : *reinterpret_cast<const uint32_t*>(D.akey + base);
    // per-thread key counts, 4 x 16-bit packed in two words (keys 0-3, 4-7); a sub-tile has 1024 slots < 2^16
    unsigned long long lo = 0, hi = 0;
#pragma unroll
    for (int i = 0; i < kKeysPerThread; ++i) {
      const uint32_t kb = (kv >> (8 * i)) & 0xff;
      if (kb != 0xff) {
        const int s = sort_key_of(D.sort_mode, kb);
        if (s < 4) lo += 1ull << (16 * s); else hi += 1ull << (16 * (s - 4));
      }
    }
    unsigned long long tot_lo, tot_hi = 0;
    unsigned long long plo = block_excl_scan64(lo, sm.scan64, tot_lo);
    unsigned long long phi = 0;
    if (D.sort_mode == 1) phi = block_excl_scan64(hi, sm.scan64, tot_hi);
#pragma unroll
    for (int i = 0; i < kKeysPerThread; ++i) {
      const uint32_t kb = (kv >> (8 * i)) & 0xff;
      if (kb != 0xff) {
        const int s = sort_key_of(D.sort_mode, kb);
        uint32_t r;
        if (s < 4) { r = (uint32_t)((plo >> (16 * s)) & 0xffff); plo += 1ull << (16 * s); }
        else { r = (uint32_t)((phi >> (16 * (s - 4))) & 0xffff); phi += 1ull << (16 * (s - 4)); }
        if (s != vacant_key || D.write_vacant) D.indices[(size_t)s * D.N + sm.base[s] + r] = base + i;
      }
    }
    if (sub + 1 < D.subs_per_tile) {   // advance the per-key bases by this sub-tile's totals
      __syncthreads();
      if (threadIdx.x < 4) sm.base[threadIdx.x] += (uint32_t)((tot_lo >> (16 * threadIdx.x)) & 0xffff);
      else if (threadIdx.x < 8) sm.base[threadIdx.x] += (uint32_t)((tot_hi >> (16 * (threadIdx.x - 4))) & 0xffff);
      __syncthreads();
    }
  }
}

// ================================================================ P5: secondary push (S9)
// Exclusive scan of nsec[slot] in ascending SLOT order (in every sort mode), so that the initializer order — and with
// it every later slot assignment and PRNG stream — does not depend on thread timing or on the sort mode. A tile's
// offset `off0` comes from the two-level counters of staged secondaries; a tile that staged nothing is not read at all.
// nv0: the thread's four nsec bytes of sub-tile 0, loaded by the caller together with its other prologue loads
__device__ __forceinline__ void push_tile(const DeviceState& D, BookSmem& sm, uint32_t tile, unsigned long long I, uint32_t off0,
                                          uint32_t tile_total, bool overflow, uint32_t nv0) {
  const uint32_t off_end = off0 + tile_total;
  for (uint32_t sub = 0; sub < D.subs_per_tile && off0 < off_end; ++sub) {
    const uint32_t base = (tile << D.tile_shift) + sub * kSub + threadIdx.x * kKeysPerThread;
    const uint32_t nv = sub == 0 ? nv0 : *reinterpret_cast<const uint32_t*>(D.nsec + base);
    const uint32_t c = (nv & 0xff) + ((nv >> 8) & 0xff) + ((nv >> 16) & 0xff) + (nv >> 24);   // bytes are 0..2
    uint32_t total;
    uint32_t r = block_excl_scan(c, sm.scan, total);
    if (c) {
#pragma unroll
      for (int i = 0; i < kKeysPerThread; ++i) {
        const uint32_t n = (nv >> (8 * i)) & 0xff;     // 0, 1 or 2
        if (n >= 1) sm.list[r] = 2u * (base + i);
        if (n >= 2) sm.list[r + 1] = 2u * (base + i) + 1u;
        r += n;
      }
      *reinterpret_cast<uint32_t*>(D.nsec + base) = 0u;   // consumed
    }
    __syncthreads();
    if (!overflow) {
      for (uint32_t item = threadIdx.x; item < total; item += kTileThreads) {   // one record per thread and pass: both halves in flight
        const uint32_t src = sm.list[item];
        const unsigned long long dst = I + (unsigned long long)(off0 + item);
        const RecB rb = load_b(D.secB + src);
        const RecA ra = load_a(D.secA + src);
        store_b(D.initB + dst, rb);
        store_a(D.initA + dst, ra);
      }
    }
    off0 += total;
  }
}

// S2: the index ranges of each action kernel. Sorted modes: region k of the index array is [k N, k N + total[k]).
__device__ __forceinline__ void set_ranges(const DeviceState& D, const uint32_t* key_total, Control* ctl) {
  for (int r = 0; r < R_COUNT; ++r) for (int j = 0; j < 2; ++j) { ctl->rb[r][j] = 0; ctl->re[r][j] = 0; }
  const uint32_t N = D.N;
  auto region = [&](int r, int j, int key) { ctl->rb[r][j] = (uint32_t)key * N; ctl->re[r][j] = (uint32_t)key * N + key_total[key]; };
  if (D.sort_mode == 1) {        // one region per action
    region(R_PE, 0, A_PE); region(R_PAIR, 0, A_PAIR); region(R_ANNIH, 0, A_ANNIH);
    region(R_PHOTON, 0, A_COMPTON); region(R_PHOTON, 1, A_MOVE_G);
    region(R_CHARGED, 0, A_BREMS); region(R_CHARGED, 1, A_MOVE_C);
  } else if (D.sort_mode == 2) { // regions gamma | e- | e+ ; the kernels mask by action inside their particle's regions
    region(R_PE, 0, 0); region(R_PAIR, 0, 0); region(R_PHOTON, 0, 0);
    region(R_CHARGED, 0, 1); region(R_CHARGED, 1, 2);
    region(R_ANNIH, 0, 2);
  } else {
    for (int r = 0; r < R_COUNT; ++r) { ctl->rb[r][0] = 0; ctl->re[r][0] = N; }
  }
}
// end-of-P1 bookkeeping of the control block by one thread (S11): counts, offsets, ranges, I, alive, log. The running
// counters (only this thread ever writes them) were read in the kernel's prologue, so everything here is a store.
struct ControlCarry { unsigned long long track_steps, iterations; uint32_t n_logged; };
__device__ __forceinline__ void update_control_after_fill(const DeviceState& D, const uint32_t* act_total, const uint32_t* key_total,
                                                          int n_keys, unsigned long long Iafter, uint32_t V, uint32_t iter, const ControlCarry cc) {
  Control* ctl = D.ctl;
  uint32_t cnt[8];
  for (int a = 0; a < 8; ++a) { cnt[a] = act_total[a]; ctl->counts[a] = cnt[a]; }
  const uint32_t N = D.N;
  uint32_t off[9];   // the compact offsets of S2 (what the debug surface reports; the kernels use the regions)
  off[0] = 0;
  for (int k = 0; k < 8; ++k) off[k + 1] = (k < n_keys) ? off[k] + key_total[k] : off[k];
  if (n_keys == 0) for (int k = 1; k <= 8; ++k) off[k] = N;
  for (int k = 0; k <= 8; ++k) ctl->offsets[k] = off[k];
  set_ranges(D, key_total, ctl);
  const uint32_t alive = N - cnt[A_VACANT];
  ctl->vac_total = V;
  ctl->n_init_fill = Iafter;   // what k_push reads (it writes n_init itself)
  ctl->iter_cur = iter;
  ctl->alive = alive;
  if (alive == 0 && Iafter == 0) {
    ctl->finished = 1;
  } else {
    ctl->track_steps = cc.track_steps + alive;
    ctl->iterations = cc.iterations + 1;
    const uint32_t k = cc.n_logged;
    if (k < D.log_capacity) {
      for (int a = 0; a < 8; ++a) D.counts_log[(size_t)k * 8 + a] = cnt[a];
      ctl->n_logged = k + 1;
    }
  }
}

// ================================================================ k_fill_sort: P1 + P2 + S11 in one pass (one block per tile)
template <bool TRACE>
__global__ void __launch_bounds__(kTileThreads, 8) k_fill_sort(DeviceState D) {
  __shared__ BookSmem sm;
  Control* ctl = D.ctl;
  const uint32_t tile = blockIdx.x;
  const uint32_t g = tile / kGroupTiles, tg0 = g * kGroupTiles;
  // ---- before the programmatic-dependency wait: what does NOT depend on the kernel just before this one in the stream
  // (k_push of the previous iteration, or the partition passes, which only touch the stack, its height, `iter`, plist and
  // the group counters of the OTHER parity): `finished`, `iter_cur` and the vacancy counters of parity k&1 were last
  // written by the action kernels / the previous k_fill_sort, which had completed before that kernel let this one start.
  const uint32_t finished = ctl->finished;
  uint32_t k = ctl->iter_cur + 1u;                // iter_cur = 0xffffffff after the reset
  uint32_t p = k & 1u;
  uint32_t T_prev = ctl->tiles_hi[p ^ 1u];        // live tiles of iteration k-1 (set by k_push of iteration k-2): the counters to read
  ControlCarry cc; cc.track_steps = ctl->track_steps; cc.iterations = ctl->iterations; cc.n_logged = ctl->n_logged;   // (used by the last tile's block)
  if (threadIdx.x < 8) { sm.hist[threadIdx.x] = 0; sm.act[threadIdx.x] = 0; }
  if (threadIdx.x < 12) sm.before[threadIdx.x] = 0;
  // (the key bytes too: the kernels that write them — the action kernels, the previous fill — are complete; the push is not one)
  const uint8_t* const key_ptr = D.akey + ((size_t)tile << D.tile_shift) + threadIdx.x * kKeysPerThread;
  bool was_live = tile < T_prev;                  // block-uniform
  uint32_t kv0 = 0, prefix = 0, V = 0, tile_vacant = 0;
  if (was_live) {
    kv0 = *reinterpret_cast<const uint32_t*>(key_ptr);
    tile_prefix(sm, D.tile_vac + (size_t)p * D.n_tiles, T_prev, tile, prefix, V, tile_vacant);
  }
  pdl_prologue();
  const uint32_t n_charged = ctl->part_charged;
  const unsigned long long I = ctl->n_init;
  // A block above the live tiles may start after the block of the last live tile has already advanced iter_cur (the grid
  // need not be resident at once, and the live tiles wait only for each other): `iter`, which the push before this
  // kernel set and nothing changes until the next push, decides; such a block redoes the little it did.
  const uint32_t k_now = ctl->iter;
  if (k_now != k) {
    k = k_now; p = k & 1u;
    T_prev = ctl->tiles_hi[p ^ 1u];
    was_live = tile < T_prev;
    if (was_live) {   // (cannot be: a live tile's block has read iter_cur before the last live tile's block got past its wait for it)
      __syncthreads();
      kv0 = *reinterpret_cast<const uint32_t*>(key_ptr);
      tile_prefix(sm, D.tile_vac + (size_t)p * D.n_tiles, T_prev, tile, prefix, V, tile_vacant);
    }
  }
  const uint32_t T = ctl->tiles_hi[p];            // live tiles of this iteration (k_push of iteration k-1)
  const uint32_t vac_low = ctl->vac_low[p];       // vacancies below T_prev (the same sum the blocks below T_prev just formed)
  if (finished) return;
  // the rows and the mask the next iteration adds into (last used by iteration k-1, which is complete)
  if (tile < D.n_groups && threadIdx.x >= 32 && threadIdx.x < 32 + kRowWords) group_row(D, p ^ 1u, tile)[threadIdx.x - 32] = 0u;
  if (tile == 0 && threadIdx.x >= 64 && threadIdx.x < 64 + kMaxGroups / 32) D.group_mask[(p ^ 1u) * (kMaxGroups / 32) + (threadIdx.x - 64)] = 0u;
  const uint32_t below = slots_below_tile(D, T_prev);
  if (!was_live) V = vac_low;                     // (everything from T_prev up is vacant)
  V += D.N - below;
  const uint32_t n_take = (unsigned long long)V < I ? V : (uint32_t)I;
  // fills that land above the live tiles of the previous iteration, and who copies their records: the blocks that have
  // nothing else to do, when there are at least as many of them as tiles to grow into (block-uniform, the same in every block)
  const uint32_t n_high = n_take > vac_low ? n_take - vac_low : 0u;
  const uint32_t n_helpers = D.n_tiles - T;
  const bool helpers_copy = D.bound_tiles && T > T_prev && n_high != 0u && n_helpers >= T - T_prev;
  if (tile >= T) {                                // entirely vacant, and nothing reaches it in this iteration
    if (helpers_copy) { const TraceScope<K_FILL_SORT, TRACE> trace(D, k); grown_copy(D, I, vac_low, below, n_high, tile - T, n_helpers); }
    return;
  }
  if (!was_live) {   // a tile the population grows into: its prefix is a closed form
    kv0 = *reinterpret_cast<const uint32_t*>(key_ptr);
    tile_vacant = real_slots_in_tile(D, tile);
    prefix = vac_low + (slots_below_tile(D, tile) - below);
    __syncthreads();   // (the zeroed histograms; the blocks below T_prev passed the barriers of tile_prefix)
  }
  const TraceScope<K_FILL_SORT, TRACE> trace(D, k);
  if (threadIdx.x == 8) D.tile_sec[tile] = 0;   // consumed by the push of the previous iteration
  const FillPlan plan = D.sort_mode == 3 ? partition_plan(n_take, V, n_charged) : plain_plan(n_take);
  const bool keys_read = (!was_live && helpers_copy) ? fill_grown_tile(D, sm, tile, I, vac_low, below, n_high, kv0)
                                                     : fill_tile(D, sm, tile, I, plan, prefix, tile_vacant, kv0);
  __syncthreads();
  // ---- publish: the tile's rows, its group's rows, what is left of its vacancies; then the stamps the later tiles wait for
  const int n_keys = D.sort_mode == 1 ? 8 : (D.sort_mode == 2 ? 4 : 0);
  const bool is_last = tile == T - 1u;
  {
    uint32_t* row = group_row(D, p, g);
    if (threadIdx.x < 8) {
      const uint32_t a = sm.act[threadIdx.x];
      D.tile_hist[(size_t)tile * 8 + threadIdx.x] = a;
      if (a) atomicAdd(row + threadIdx.x, a);
    } else if (threadIdx.x < 12 && D.sort_mode == 2) {
      const uint32_t h = sm.hist[threadIdx.x - 8];
      D.tile_phist[(size_t)tile * 4 + (threadIdx.x - 8)] = h;
      if (h) atomicAdd(row + threadIdx.x, h);
    } else if (threadIdx.x == 12) {
      D.tile_vac[(size_t)(p ^ 1u) * D.n_tiles + tile] = tile_vacant - filled_by_plan(tile_vacant, prefix, plan);
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {   // the two bits the later tiles poll: "this tile has published", "this group is complete"
      atomicOr(row + 13, 1u << (tile - tg0));
      if (atomicAdd(row + 12, 1u) == tiles_in_group(T, g) - 1u) {
        __threadfence();
        atomicOr(D.group_mask + p * (kMaxGroups / 32) + g / 32, 1u << (g & 31u));
      }
    }
  }
  const bool scatter = n_keys != 0 && (keys_read || D.write_vacant);
  if (!scatter && !is_last) return;
  // a tile of one sub-tile forms its ranks now, while the tiles before it are still publishing
  const bool early_ranks = scatter && D.subs_per_tile == 1;
  unsigned long long plo = 0, phi = 0;
  if (early_ranks) scatter_ranks(D, sm, plo, phi);
  // ---- wait for the tiles before this one: ONE warp polls the mask of complete groups (a word per 32 groups, a lane each)
  // and the mask of published tiles of the own group, all words in flight together, with a back-off, so that a thousand
  // waiting blocks cost L2 next to nothing; then the per-key counts of whole lower groups come from the group rows, those
  // of the lower tiles of the own group from their own rows, all loads in flight together
  if (threadIdx.x < 32) {   // warp 0: lane w polls word w of the group mask (<= 8 words), lane 31 the own group's tile mask — one
    const uint32_t lane = threadIdx.x;                         // round trip when everything before has already published
    const uint32_t* word = nullptr; uint32_t want = 0;
    if (lane * 32u < g) { word = D.group_mask + p * (kMaxGroups / 32) + lane; want = g - lane * 32u >= 32u ? 0xffffffffu : (1u << (g - lane * 32u)) - 1u; }
    else if (lane == 31) { word = group_row(D, p, g) + 13; want = (1u << (tile - tg0)) - 1u; }
    static_assert(kMaxGroups / 32 <= 31, "one lane per word of the group mask, lane 31 for the tile mask");
    uint32_t spins = 0;
    const uint32_t ns = 100;   // one polling warp per block: a short, fixed pause costs L2 nothing and keeps the wake-up latency low
    bool ok = want == 0;
    while (true) {
      if (!ok) ok = (load_acquire(word) & want) == want;
      if (__all_sync(0xffffffffu, ok)) break;
      if (++spins > kSpinLimit) { if (lane == 0) ctl->error = -9; break; }   // CEL_ERR_INTERNAL (sticky)
      __nanosleep(ns);
    }
  }
  __syncthreads();
  {
    const bool by_particle = D.sort_mode == 2;
    const int n_sum = by_particle ? 12 : 8;
    for (uint32_t i0 = 0; i0 < g + kGroupTiles; i0 += kTileThreads) {   // rows [0, g): group rows; [g, g + 32): the own group's tile rows
      const uint32_t i = i0 + threadIdx.x;
      uint32_t s[12];
#pragma unroll
      for (int j = 0; j < 12; ++j) s[j] = 0;
      const uint32_t* row = nullptr; const uint32_t* prow = nullptr;
      if (i < g) { row = group_row(D, p, i); prow = row + 8; }
      else if (i < g + kGroupTiles && tg0 + (i - g) < tile) { row = D.tile_hist + (size_t)(tg0 + (i - g)) * 8; prow = D.tile_phist + (size_t)(tg0 + (i - g)) * 4; }
      if (row) {
        const uint4 a = __ldcg(reinterpret_cast<const uint4*>(row)), b = __ldcg(reinterpret_cast<const uint4*>(row + 4));
        s[0] = a.x; s[1] = a.y; s[2] = a.z; s[3] = a.w; s[4] = b.x; s[5] = b.y; s[6] = b.z; s[7] = b.w;
        if (by_particle) { const uint4 c = __ldcg(reinterpret_cast<const uint4*>(prow)); s[8] = c.x; s[9] = c.y; s[10] = c.z; s[11] = c.w; }
      }
#pragma unroll
      for (int j = 0; j < 12; ++j) {
        if (j < n_sum) {
          const uint32_t v = __reduce_add_sync(0xffffffffu, s[j]);
          if ((threadIdx.x & 31) == 0 && v) atomicAdd(&sm.before[j], v);
        }
      }
    }
    __syncthreads();
  }
  if (threadIdx.x < 8) sm.base[threadIdx.x] = sm.before[D.sort_mode == 2 ? 8 + (threadIdx.x & 3) : threadIdx.x];
  if (is_last && threadIdx.x == 0) {   // every other live tile is before this one: totals = before + own (+ the vacant tiles above)
    uint32_t act_total[8], key_total[8];
    const uint32_t above = D.N - slots_below_tile(D, T);
    for (int i = 0; i < 8; ++i) {
      act_total[i] = sm.before[i] + sm.act[i] + (i == A_VACANT ? above : 0u);
      key_total[i] = D.sort_mode == 2 ? (i < 4 ? sm.before[8 + i] + sm.hist[i] + (i == 3 ? above : 0u) : 0u) : act_total[i];
    }
    update_control_after_fill(D, act_total, key_total, n_keys, I - n_take, V, k, cc);
  }
  if (!scatter) return;
  __syncthreads();
  if (early_ranks) scatter_store(D, sm, tile, plo, phi);
  else scatter_tile(D, sm, tile);
}

// ================================================================ k_push: P5 (one block per tile)
template <bool TRACE>
__global__ void __launch_bounds__(kTileThreads) k_push(DeviceState D) {
  __shared__ BookSmem sm;
  Control* ctl = D.ctl;
  const uint32_t tile = blockIdx.x;
  // ---- before the programmatic-dependency wait: what k_fill_sort of this iteration and the kernels before it left (they
  // were complete before the kernel just before this one — an action kernel — let this one start)
  const uint32_t finished = ctl->finished, iter = ctl->iter_cur;
  const unsigned long long I = ctl->n_init_fill;
  const uint32_t T = ctl->tiles_hi[iter & 1u];     // live tiles of this iteration: nothing was staged above them
  if (tile >= T) return;
  pdl_prologue();
  // No "last block" here: every block forms S itself, and block 0 alone updates the control block — it writes only fields
  // that no block of this kernel reads (n_init and iter are read through the copies k_fill_sort left: n_init_fill, iter_cur).
  const int32_t error = ctl->error;
  // (issued with the loads above and the counters below: one round trip for the whole prologue; 1 KB wasted by a tile that staged nothing)
  const uint32_t nv0 = *reinterpret_cast<const uint32_t*>(D.nsec + ((size_t)tile << D.tile_shift) + threadIdx.x * kKeysPerThread);
  uint32_t prefix, S, tile_total;
  tile_prefix(sm, D.tile_sec, T, tile, prefix, S, tile_total);
  if (finished) return;
  const TraceScope<K_PUSH, TRACE> trace(D, iter);
  const bool overflow = error != 0 || I + S > D.init_capacity;
  if (tile == 0) {
    if (threadIdx.x == 0) {
      ctl->push_total = S;
      if (I + S > D.init_capacity) ctl->error = -4;  // CEL_ERR_INIT_OVERFLOW (sticky)
      else if (error == 0) ctl->n_init = I + S;
      ctl->secondaries += S;
      ctl->iter = iter + 1;
    }
    // the live tiles of the next iteration (see tile_prefix): its fill takes n_take = min(V, I) vacancies in ascending
    // order, vac_low of them below T, the rest in the consecutive vacant slots above
    const uint32_t q = (iter + 1u) & 1u;
    uint32_t unused0, vac_low, unused1;
    __syncthreads();
    tile_prefix(sm, D.tile_vac + (size_t)q * D.n_tiles, T, 0u, unused0, vac_low, unused1);
    if (threadIdx.x == 0) {
      const uint32_t below = slots_below_tile(D, T);
      const unsigned long long V = (unsigned long long)vac_low + (D.N - below);
      const unsigned long long I_next = overflow ? I : I + S;
      const unsigned long long n_take = V < I_next ? V : I_next;
      uint32_t T_next = T;
      if (n_take > vac_low) {
        const unsigned long long top = (unsigned long long)below + (n_take - vac_low);   // one past the highest slot filled
        T_next = (uint32_t)((top + (1ull << D.tile_shift) - 1ull) >> D.tile_shift);
        if (T_next > D.n_tiles) T_next = D.n_tiles;
        if (T_next < T) T_next = T;
      }
      ctl->tiles_hi[q] = T_next;
      ctl->vac_low[q] = vac_low;
    }
    __syncthreads();
  }
  if (tile_total == 0) return;
  push_tile(D, sm, tile, I, prefix, tile_total, overflow, nv0);
}

// ================================================================ S9-P: charged / neutral partition of the popped initializers
// (sort mode 3; section 3.2). Pop position j = 0 .. n_take-1 is init[I-1-j]. Two passes over the popped
// segment, one tile-sized chunk per block: k_part_count counts the charged pops of a chunk; k_part_scatter forms the
// chunk's exclusive prefix by a block reduction over the counts and writes the pop positions, stably, into
// plist (= D.indices): the charged ones from the front in pop order, the neutral ones from the back.
__device__ __forceinline__ bool pop_is_charged(const DeviceState& D, unsigned long long I, uint32_t j) {
  const unsigned long long meta = reinterpret_cast<const unsigned long long*>(D.initB + (I - 1ull - j))[3];
  return meta_ptype(meta) != P_GAMMA;
}
// sum of a[0..tile) and of a[0..n) by one block: the block's exclusive prefix and the grand total
__device__ __forceinline__ void block_prefix_total(const uint32_t* a, uint32_t n, uint32_t tile, uint32_t* smem /* 18 words */,
                                                   uint32_t& prefix, uint32_t& total) {
  uint32_t p = 0, t = 0;
  for (uint32_t i = threadIdx.x; i < n; i += kTileThreads) {
    const uint32_t v = a[i];
    t += v;
    if (i < tile) p += v;
  }
  p = __reduce_add_sync(0xffffffffu, p);
  t = __reduce_add_sync(0xffffffffu, t);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  __syncthreads();
  if (lane == 0) { smem[warp] = p; smem[9 + warp] = t; }
  __syncthreads();
  p = 0; t = 0;
#pragma unroll
  for (int w = 0; w < kTileThreads / 32; ++w) { p += smem[w]; t += smem[9 + w]; }
  prefix = p; total = t;
}
template <bool TRACE>
__global__ void __launch_bounds__(kTileThreads) k_part_count(DeviceState D) {
  __shared__ BookSmem sm;
  pdl_prologue();
  const Control* ctl = D.ctl;
  if (ctl->finished) return;
  const uint32_t iter = ctl->iter;
  const TraceScope<K_PART_COUNT, TRACE> trace(D, iter);
  const uint32_t tile = blockIdx.x;
  const unsigned long long I = ctl->n_init;
  uint32_t unused, V;
  block_prefix_total(D.tile_vac + (size_t)(iter & 1u) * D.n_tiles, D.n_tiles, 0u, sm.scan, unused, V);
  const uint32_t n_take = (unsigned long long)V < I ? V : (uint32_t)I;
  const unsigned long long j0 = (unsigned long long)tile << D.tile_shift;
  const unsigned long long j1 = min(j0 + (1ull << D.tile_shift), (unsigned long long)n_take);
  uint32_t c = 0;
  for (unsigned long long j = j0 + threadIdx.x; j < j1; j += kTileThreads) c += pop_is_charged(D, I, (uint32_t)j) ? 1u : 0u;
  c = __reduce_add_sync(0xffffffffu, c);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) sm.scan[threadIdx.x >> 5] = c;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t t = 0;
    for (int w = 0; w < kTileThreads / 32; ++w) t += sm.scan[w];
    D.part_cnt[tile] = t;
  }
}
template <bool TRACE>
__global__ void __launch_bounds__(kTileThreads) k_part_scatter(DeviceState D) {
  __shared__ BookSmem sm;
  pdl_prologue();
  Control* ctl = D.ctl;
  if (ctl->finished) return;
  const uint32_t iter = ctl->iter;
  const TraceScope<K_PART_SCATTER, TRACE> trace(D, iter);
  const uint32_t tile = blockIdx.x;
  const unsigned long long I = ctl->n_init;
  uint32_t unused, V, cpre, C;
  block_prefix_total(D.tile_vac + (size_t)(iter & 1u) * D.n_tiles, D.n_tiles, 0u, sm.scan, unused, V);
  __syncthreads();
  block_prefix_total(D.part_cnt, D.n_tiles, tile, sm.scan, cpre, C);
  const uint32_t n_take = (unsigned long long)V < I ? V : (uint32_t)I;
  if (tile == 0 && threadIdx.x == 0) ctl->part_charged = C;
  const unsigned long long j0 = (unsigned long long)tile << D.tile_shift;
  const unsigned long long j1 = min(j0 + (1ull << D.tile_shift), (unsigned long long)n_take);
  for (uint32_t sub = 0; sub < D.subs_per_tile; ++sub) {
    const unsigned long long base = j0 + (unsigned long long)sub * kSub + (unsigned long long)threadIdx.x * kKeysPerThread;
    if (j0 + (unsigned long long)sub * kSub >= j1) break;           // block-uniform
    bool ch[kKeysPerThread];
    uint32_t c = 0;
#pragma unroll
    for (int i = 0; i < kKeysPerThread; ++i) { ch[i] = (base + i < j1) && pop_is_charged(D, I, (uint32_t)(base + i)); c += ch[i] ? 1u : 0u; }
    uint32_t total;
    uint32_t r = cpre + block_excl_scan(c, sm.scan, total);         // charged pops before this thread's first pop
#pragma unroll
    for (int i = 0; i < kKeysPerThread; ++i) {
      const unsigned long long j = base + i;
      if (j < j1) {
        if (ch[i]) { D.indices[r] = (uint32_t)j; ++r; }
        else D.indices[n_take - 1u - ((uint32_t)j - r)] = (uint32_t)j;   // neutral rank = j - (charged before j)
      }
    }
    cpre += total;
    __syncthreads();
  }
}

// ================================================================ hit transfer (option "hits"; section 3.4)
// "Hits must be transferred at every step iteration": after the action kernels of iteration k, k_hits_flush
// streams the records they appended, d_hits[mark, n_hits), into the pinned host ring buffer of the running batch at the
// same offsets — plain coalesced 16-byte stores to device-mapped pinned memory, stream-ordered, no host involvement and no
// synchronisation of any kind. It runs beside k_push. The marks are double-buffered by iteration parity so
// that no block reads a field another block of the same launch writes.
template <bool TRACE>
__global__ void __launch_bounds__(kTileThreads) k_hits_flush(DeviceState D) {
  Control* ctl = D.ctl;
  const uint32_t k = ctl->iter_cur;
  if (ctl->finished) return;
  const TraceScope<K_HITS_FLUSH, TRACE> trace(D, k);
  const unsigned long long lo = ctl->hits_mark[k & 1u];
  unsigned long long hi = ctl->n_hits;
  if (hi > D.hit_capacity) hi = D.hit_capacity;
  HitRec* dst = D.host_hits[ctl->hits_cur & 1u];
  for (unsigned long long i = lo + blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; i < hi; i += (unsigned long long)gridDim.x * blockDim.x) {
    unsigned long long a, b;
    asm volatile("ld.global.v2.b64 {%0,%1}, [%2];" : "=l"(a), "=l"(b) : "l"(D.hits + i));
    asm volatile("st.global.v2.b64 [%0], {%1,%2};" ::"l"(dst + i), "l"(a), "l"(b) : "memory");
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) ctl->hits_mark[(k & 1u) ^ 1u] = hi;
}
// end of a batch of iterations: publish the batch's record count and ring buffer in the control block (the host reads
// them from its asynchronous status copy), start the next batch's records at offset 0 of the other ring buffer
__global__ void k_hits_batch_end(DeviceState D) {
  Control* ctl = D.ctl;
  unsigned long long n = ctl->n_hits;
  if (n > D.hit_capacity) n = D.hit_capacity;
  ctl->hits_in_batch = n;
  ctl->hits_buf = ctl->hits_cur;
  ctl->hits_cur ^= 1u;
  ctl->n_hits = 0; ctl->hits_mark[0] = 0; ctl->hits_mark[1] = 0;
}

// end of a batch of iterations: the control block straight into pinned host memory (the host loop never
// blocks the device). An in-stream cudaMemcpyAsync of these 300 bytes cost ~10 us of copy-engine latency between two batches;
// a one-warp kernel writing mapped memory costs ~2. Slots alternate with the batch count, as the host's own counter does.
__global__ void k_status(DeviceState D) {
  Control* ctl = D.ctl;
  const uint32_t seq = ctl->status_seq;
  uint32_t* dst = reinterpret_cast<uint32_t*>(D.status_host + (seq & 1u));
  const uint32_t* src = reinterpret_cast<const uint32_t*>(ctl);
  for (uint32_t i = threadIdx.x; i < sizeof(Control) / 4; i += blockDim.x) dst[i] = src[i];
  __syncthreads();
  if (threadIdx.x == 0) ctl->status_seq = seq + 1u;
  __threadfence_system();
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
    // the checks validate_primaries makes on the host path (cel_transport), for primaries that are already on the device
    const double n2 = p.dir[0] * p.dir[0] + p.dir[1] * p.dir[1] + p.dir[2] * p.dir[2];
    bool bad = vol < 0 || p.event >= D.n_events || p.event >= (1u << 24) || p.ptype < 0 || p.ptype > 2 || !(fabs(n2 - 1.0) <= 1e-12);
    if (D.P.geom_kind == 0) bad = bad || fabs(p.pos[0]) > D.P.half_x || fabs(p.pos[1]) > D.P.half_y;
    else bad = bad || fabs(p.pos[2]) > D.P.half_z;
    if (!(p.energy > 0.0) || !isfinite(p.energy) || !isfinite((p.pos[0] + p.pos[1]) + p.pos[2])) { D.ctl->error = -6; vol = vol < 0 ? 0 : vol; }   // CEL_ERR_NONFINITE
    else if (bad) { D.ctl->error = -1; vol = vol < 0 ? 0 : vol; }
    RecA a; a.x = p.pos[0]; a.y = p.pos[1]; a.z = p.pos[2]; a.energy = p.energy;
    RecB b; b.dx = p.dir[0]; b.dy = p.dir[1]; b.dz = p.dir[2];
    b.meta = make_meta(p.ptype == P_GAMMA ? A_MOVE_G : A_MOVE_C, p.ptype, vol, -1, 0, p.event);
    store_a(D.initA + i, a);
    store_b(D.initB + i, b);
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    D.ctl->n_init = n;
    // live tiles of iteration 0 (tile_prefix): the first min(n, N) slots; none before it. Unbounded (every tile, always)
    // for the partition rule, which also fills from the top, and on the debug surface, which wants the vacant indices too
    uint32_t T0 = D.n_tiles, T_before = D.n_tiles;
    if (D.bound_tiles) {
      const unsigned long long take = n < D.N ? n : (unsigned long long)D.N;
      T0 = (uint32_t)((take + (1ull << D.tile_shift) - 1ull) >> D.tile_shift);
      if (T0 < 1u) T0 = 1u;
      T_before = 0u;
    }
    D.ctl->tiles_hi[0] = T0; D.ctl->tiles_hi[1] = T_before;
    D.ctl->vac_low[0] = 0u; D.ctl->vac_low[1] = 0u;
  }
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

// which = 0: sin(x) of the helix substep (x S(x^2)); 1: 1 - cos(x) (x^2 V(x^2)), |x| <= 0.5
__global__ void k_debug_math(int which, const double* in, uint32_t n, double* out) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double x = in[i];
  double S, V;
  sinc_versc_small(x * x, S, V);
  out[i] = which == 0 ? x * S : (x * x) * V;
}

// every slot vacant: key byte 7 (padding 0xff), meta action VACANT (state bytes are otherwise zero); the per-tile and
// per-group vacancy counters start at the number of real slots
__global__ void k_reset_state(DeviceState D) {
  const unsigned long long padded = (unsigned long long)D.n_tiles << D.tile_shift;
  for (unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; i < padded; i += (unsigned long long)gridDim.x * blockDim.x) {
    D.akey[i] = (i < D.N) ? (uint8_t)A_VACANT : (uint8_t)0xff;
    D.nsec[i] = 0;
    if (i < D.N) {
      RecA a; a.x = a.y = a.z = a.energy = 0.0;
      RecB b; b.dx = b.dy = b.dz = 0.0; b.meta = make_meta(A_VACANT, 0, 0, -1, 0, 0);
      store_a(D.stA + i, a); store_b(D.stB + i, b);
    }
    if (i < D.n_tiles) {   // vacancy counters of both parities (a tile above the live tiles keeps them); everything else in the scratch is zero
      const unsigned long long lo = i << D.tile_shift, hi = (i + 1) << D.tile_shift;
      const uint32_t real = (uint32_t)(lo >= D.N ? 0ull : ((hi < D.N ? hi : (unsigned long long)D.N) - lo));
      D.tile_vac[i] = real; D.tile_vac[D.n_tiles + i] = real;
    }
    if (i == 0) D.ctl->iter_cur = 0xffffffffu;   // k_fill_sort forms k = iter_cur + 1 before its dependency wait
  }
}

}  // namespace cel

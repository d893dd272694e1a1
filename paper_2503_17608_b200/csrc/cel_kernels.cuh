// cel_kernels.cuh — the bookkeeping kernels of one step iteration (docs/PHYSICS_SPEC.md S1):
//   P1 init + P2 histogram: k_init_fill   (scan-based vacancy filling, S9; per-tile sort-key histogram, S2)
//   P2 reindex:             k_scatter     (closes the fill: vacancy counters, action counts, offsets, control block;
//                                          then the stable counting sort of slot indices, S2)
//   P5 push:                k_push        (scan-ordered secondary push, S9)
//   S9-P (sort mode 3):     k_part_count, k_part_scatter (charged / neutral partition of the popped initializers)
// (P3/P4, the action kernels and the scoring, are in cel_physics.cuh.)
// No kernel has a "last block" phase: what one block would have to do after all the others (scans over tiles, the
// control block) is either done redundantly by every block from small two-level counters, or left to the blocks of
// the next kernel.
// The action kernels keep two per-tile counters up to date with integer atomics — vacancies created and secondaries
// staged — so neither scan needs a counting pass: a block reduces the counters of the tiles before it to get its
// exclusive prefix, skips its tile when there is nothing to fill / push, and otherwise scans the tile's dense key
// bytes (1 B per slot) in sub-tiles of 1024 slots. The record copies (64 B per initializer) are spread over the
// whole block through a compacted work list in shared memory, 32 B per thread and step.
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
// in-place exclusive scan of a[0..n) (stride in words) by one block; returns the total to every thread
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
// sum of a[0..tile) and of a[0..n) by one block (n <= kMaxTiles): the block's exclusive prefix and the grand total
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
// The same with the counters already in registers: load_counters issues every load of the kernel's prologue back to
// back (control block, counters) BEFORE the first use, so the prologue costs one L2 round trip instead of one per
// dependent step (in-order issue stalls at the first use). Also returns a[tile].
// (CPT counters per thread: 8 up to 2048 tiles, 16 above — two instantiations of the kernels that use it, so that the
// common sizes keep their register count)
template <int CPT>
__device__ __forceinline__ void load_counters(const uint32_t* a, uint32_t n, uint32_t (&v)[CPT]) {
#pragma unroll
  for (int i = 0; i < CPT; ++i) { const uint32_t idx = threadIdx.x + i * kTileThreads; v[i] = idx < n ? a[idx] : 0u; }
}
template <int CPT>
__device__ __forceinline__ void block_prefix_total_regs(const uint32_t (&v)[CPT], uint32_t tile, uint32_t* smem /* 19 words */,
                                                        uint32_t& prefix, uint32_t& total, uint32_t& own) {
  uint32_t p = 0, t = 0;
#pragma unroll
  for (int i = 0; i < CPT; ++i) {
    const uint32_t idx = threadIdx.x + i * kTileThreads;
    t += v[i];
    if (idx < tile) p += v[i];
  }
  p = __reduce_add_sync(0xffffffffu, p);
  t = __reduce_add_sync(0xffffffffu, t);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  __syncthreads();
  if (lane == 0) { smem[warp] = p; smem[9 + warp] = t; }
#pragma unroll
  for (int i = 0; i < CPT; ++i) if (threadIdx.x + i * kTileThreads == tile) smem[18] = v[i];
  __syncthreads();
  p = 0; t = 0;
#pragma unroll
  for (int w = 0; w < kTileThreads / 32; ++w) { p += smem[w]; t += smem[9 + w]; }
  prefix = p; total = t; own = smem[18];
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

// ---------------------------------------------------------------- shared memory of a bookkeeping block
struct BookSmem {
  uint32_t scan[20];
  unsigned long long scan64[9];
  uint32_t hist[8], act[8], base[8];
  uint32_t skey[kTileThreads];   // the sub-tile's key bytes
  uint32_t list[2 * kSub];       // compacted work list of the cooperative copies
};

__device__ __forceinline__ uint32_t real_slots_in_tile(const DeviceState& D, uint32_t tile) {
  const unsigned long long lo = (unsigned long long)tile << D.tile_shift, hi = lo + (1ull << D.tile_shift);
  return lo >= D.N ? 0u : (uint32_t)((hi < D.N ? hi : (unsigned long long)D.N) - lo);
}

// ================================================================ P1: vacancy scan + fill (S9), P2 histogram (S2)
// Rank-r vacant slot (ascending slot order) takes init[I-1-r] when r < I (LIFO). The rank of a tile's first vacancy
// (`prefix`) is the sum of tile_vac over the tiles before it — scan-based, no atomics in the assignment, so the slot
// assignment is deterministic. Adds the tile's action histogram to sm.act and (sort by particle) its
// sort-key histogram to sm.hist; the caller zeroes both and synchronises before, and synchronises after.
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
__device__ __forceinline__ void fill_tile(const DeviceState& D, BookSmem& sm, uint32_t tile, unsigned long long I, const FillPlan pl,
                                          uint32_t prefix, uint32_t tile_vacant) {
  uint32_t rank0 = prefix;                                   // rank of the first vacancy of the current sub-tile
  const uint32_t rank_end = prefix + tile_vacant;            // one past the rank of the tile's last vacancy
  const uint32_t real = real_slots_in_tile(D, tile);
  if (tile_vacant == real && filled_by_plan(tile_vacant, prefix, pl) == 0) {   // all vacant, nothing to fill: no key byte needs reading
    if (threadIdx.x == 0) { atomicAdd(&sm.act[A_VACANT], real); if (D.sort_mode == 2) atomicAdd(&sm.hist[3], real); }
    return;
  }
  uint8_t* skey_b = reinterpret_cast<uint8_t*>(sm.skey);
  for (uint32_t sub = 0; sub < D.subs_per_tile; ++sub) {
    const uint32_t sub_base = (tile << D.tile_shift) + sub * kSub;
    const uint32_t base = sub_base + threadIdx.x * kKeysPerThread;
    uint32_t kv = *reinterpret_cast<const uint32_t*>(D.akey + base);
    if (rank0 < rank_end && filled_by_plan(rank_end - rank0, rank0, pl) != 0) {   // block-uniform: this sub-tile may have vacancies to fill
      const uint32_t c = count_vacant4(kv);
      uint32_t total;
      uint32_t r = block_excl_scan(c, sm.scan, total);
      sm.skey[threadIdx.x] = kv;
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
      // cooperative copy: work item w = (record, half); half 0 = RecA, half 1 = RecB (+ the key byte)
      for (uint32_t w = threadIdx.x; w < 2 * nf; w += kTileThreads) {
        const uint32_t m = w >> 1;
        const uint32_t item = m < n_lo ? m : hi_begin + (m - n_lo);
        const uint32_t slot = sm.list[item];
        const uint32_t rank = rank0 + item;
        uint32_t pop = rank;                                 // plain rule: rank r takes init[I-1-r]
        if (pl.partition) pop = D.indices[rank < pl.low_n ? rank : pl.n_take - 1u - (pl.V - 1u - rank)];
        const unsigned long long src = I - 1ull - (unsigned long long)pop;
        if (w & 1) {
          const RecB b = load_b(D.initB + src);
          store_b(D.stB + slot, b);
          const uint8_t key = make_key(meta_action(b.meta), meta_ptype(b.meta));
          D.akey[slot] = key;
          skey_b[slot - sub_base] = key;
        } else {
          store_a(D.stA + slot, load_a(D.initA + src));
        }
      }
      __syncthreads();
      kv = sm.skey[threadIdx.x];
      rank0 += total;
    }
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
}
__device__ __forceinline__ void fill_tile(const DeviceState& D, BookSmem& sm, uint32_t tile, unsigned long long I, uint32_t n_take,
                                          uint32_t prefix, uint32_t tile_vacant) {
  fill_tile(D, sm, tile, I, plain_plan(n_take), prefix, tile_vacant);
}
// Two-level histograms. Besides its own row tile_hist[tile][8], every fill block adds its counts into the row of its
// GROUP of kGroupTiles tiles (integer atomics on 8 x n_groups addresses, double-buffered by the parity of the iteration:
// the blocks of iteration k also zero the rows that iteration k+1 will add into). Column totals are then the sum of
// <= 128 group rows, and the base of a tile in the counting sort is (groups before its group) + (tiles of its group
// before it): 2 KB read by each scatter block, 2 KB by the one block that updates the control block — instead of one
// block scanning all 32 KB of rows in place, which was 4.4 of the 12 us of an almost empty k_init_fill (one SM pulls
// ~64 B per clock from L2; profiles/).
constexpr int kGroupTiles = 32;
constexpr int kMaxGroups = kMaxTiles / kGroupTiles;   // 128
__device__ __forceinline__ uint32_t* group_rows(uint32_t* base, uint32_t parity) { return base + (size_t)parity * kMaxGroups * 8; }
// after fill_tile + __syncthreads: publish the tile's action histogram and (sort by particle) its sort-key histogram.
// The iteration's action counts are the column sums of tile_hist (no same-address atomics from a thousand blocks).
__device__ __forceinline__ void publish_tile_hist(const DeviceState& D, BookSmem& sm, uint32_t tile) {
  if (threadIdx.x < 8) {
    D.tile_hist[tile * 8 + threadIdx.x] = sm.act[threadIdx.x];
    if (D.sort_mode == 2) D.tile_phist[tile * 8 + threadIdx.x] = threadIdx.x < 4 ? sm.hist[threadIdx.x] : 0u;
  }
}
// the kernel-per-action form: the group rows of the two-level histograms (see group_rows)
__device__ __forceinline__ void publish_group_hist(const DeviceState& D, BookSmem& sm, uint32_t tile, uint32_t parity) {
  if (threadIdx.x < 8) {
    const uint32_t g = tile / kGroupTiles;
    const uint32_t a = sm.act[threadIdx.x];
    if (a) atomicAdd(group_rows(D.group_hist, parity) + g * 8 + threadIdx.x, a);
    if (D.sort_mode == 2 && threadIdx.x < 4) { const uint32_t h = sm.hist[threadIdx.x]; if (h) atomicAdd(group_rows(D.group_phist, parity) + g * 8 + threadIdx.x, h); }
    if (tile < (uint32_t)kMaxGroups) {   // the rows the next iteration adds into (last read by the previous iteration's scatter)
      group_rows(D.group_hist, parity ^ 1u)[tile * 8 + threadIdx.x] = 0u;
      if (D.sort_mode == 2) group_rows(D.group_phist, parity ^ 1u)[tile * 8 + threadIdx.x] = 0u;
    }
  }
}
// the rows the scatter takes its per-tile bases from: the action histogram (sort by action) or the particle histogram
__device__ __forceinline__ uint32_t* sort_rows(const DeviceState& D) { return D.sort_mode == 2 ? D.tile_phist : D.tile_hist; }

// sum over the rows r < n_rows (n_rows <= 32) of rows[r][0..8) by one warp; every lane gets the 8 column sums
__device__ __forceinline__ void warp_sum_rows(const uint32_t* rows, uint32_t n_rows, uint32_t* out8) {
  const uint32_t lane = threadIdx.x & 31;
  uint4 a = make_uint4(0, 0, 0, 0), b = make_uint4(0, 0, 0, 0);
  if (lane < n_rows) { a = *reinterpret_cast<const uint4*>(rows + lane * 8); b = *reinterpret_cast<const uint4*>(rows + lane * 8 + 4); }
  out8[0] = __reduce_add_sync(0xffffffffu, a.x); out8[1] = __reduce_add_sync(0xffffffffu, a.y);
  out8[2] = __reduce_add_sync(0xffffffffu, a.z); out8[3] = __reduce_add_sync(0xffffffffu, a.w);
  out8[4] = __reduce_add_sync(0xffffffffu, b.x); out8[5] = __reduce_add_sync(0xffffffffu, b.y);
  out8[6] = __reduce_add_sync(0xffffffffu, b.z); out8[7] = __reduce_add_sync(0xffffffffu, b.w);
}
// vacancies of a tile that the fill of this iteration takes: min(v, max(0, n_take - (vacancies before the tile)))
__device__ __forceinline__ uint32_t filled_in_tile(uint32_t v, uint32_t prefix, uint32_t n_take) {
  return min(v, n_take > prefix ? n_take - prefix : 0u);
}

// ================================================================ P2: stable scatter of slot indices (S2)
// indices[offset[key] + (tiles before)[key] + (rank inside the tile)] = slot; ascending slot order inside a key.
// The caller sets sm.base[key] = offset[key] + (tiles before)[key] and synchronises. Vacant slots are never launched:
// their indices are written only when the complete permutation is asked for (debug surface), and a tile that is
// entirely vacant is then skipped without reading its key bytes.
__device__ __forceinline__ void scatter_tile(const DeviceState& D, BookSmem& sm, uint32_t tile, uint32_t tile_vacant_now) {
  const int vacant_key = D.sort_mode == 1 ? (int)A_VACANT : 3;
  if (!D.write_vacant && tile_vacant_now == real_slots_in_tile(D, tile)) return;
  for (uint32_t sub = 0; sub < D.subs_per_tile; ++sub) {
    const uint32_t base = (tile << D.tile_shift) + sub * kSub + threadIdx.x * kKeysPerThread;
    const uint32_t kv = *reinterpret_cast<const uint32_t*>(D.akey + base);
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
        if (s != vacant_key || D.write_vacant) D.indices[sm.base[s] + r] = base + i;
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
// offset `off0` is the sum of tile_sec over the tiles before it; a tile that staged nothing is not read at all.
__device__ __forceinline__ void push_tile(const DeviceState& D, BookSmem& sm, uint32_t tile, unsigned long long I, uint32_t off0,
                                          uint32_t tile_total, bool overflow) {
  const uint32_t off_end = off0 + tile_total;
  for (uint32_t sub = 0; sub < D.subs_per_tile && off0 < off_end; ++sub) {
    const uint32_t base = (tile << D.tile_shift) + sub * kSub + threadIdx.x * kKeysPerThread;
    const uint32_t nv = *reinterpret_cast<const uint32_t*>(D.nsec + base);
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
      for (uint32_t w = threadIdx.x; w < 2 * total; w += kTileThreads) {
        const uint32_t item = w >> 1;
        const uint32_t src = sm.list[item];
        const unsigned long long dst = I + (unsigned long long)(off0 + item);
        if (w & 1) store_b(D.initB + dst, load_b(D.secB + src));
        else store_a(D.initA + dst, load_a(D.secA + src));
      }
    }
    off0 += total;
  }
}

// S2: the index range of each action kernel from the key offsets
__device__ __forceinline__ void set_ranges(const DeviceState& D, const uint32_t* off, uint32_t* rb, uint32_t* re) {
  if (D.sort_mode == 1) {        // PE | PAIR | COMPTON MOVE_G | MOVE_C BREMS | ANNIH | VACANT
    rb[R_PE] = off[0]; re[R_PE] = off[1];
    rb[R_PAIR] = off[1]; re[R_PAIR] = off[2];
    rb[R_PHOTON] = off[2]; re[R_PHOTON] = off[4];
    rb[R_CHARGED] = off[4]; re[R_CHARGED] = off[6];
    rb[R_ANNIH] = off[6]; re[R_ANNIH] = off[7];
  } else if (D.sort_mode == 2) { // gamma | e- | e+ | vacant
    rb[R_PE] = rb[R_PAIR] = rb[R_PHOTON] = off[0];
    re[R_PE] = re[R_PAIR] = re[R_PHOTON] = off[1];
    rb[R_CHARGED] = off[1]; re[R_CHARGED] = off[3];
    rb[R_ANNIH] = off[2]; re[R_ANNIH] = off[3];
  } else {
    for (int k = 0; k < R_COUNT; ++k) { rb[k] = 0; re[k] = D.N; }
  }
}
// end-of-P1 bookkeeping of the control block by one thread (S11): counts, offsets, ranges, I, alive, log
__device__ __forceinline__ void update_control_after_fill(const DeviceState& D, const uint32_t* act_total, const uint32_t* key_total,
                                                          int n_keys, unsigned long long I, uint32_t V, uint32_t n_take) {
  Control* ctl = D.ctl;
  uint32_t cnt[8];
  for (int a = 0; a < 8; ++a) { cnt[a] = act_total[a]; ctl->counts[a] = cnt[a]; }
  const uint32_t N = D.N;
  uint32_t off[9];
  off[0] = 0;
  for (int k = 0; k < 8; ++k) off[k + 1] = (k < n_keys) ? off[k] + key_total[k] : off[k];
  if (n_keys == 0) for (int k = 1; k <= 8; ++k) off[k] = N;
  for (int k = 0; k <= 8; ++k) ctl->offsets[k] = off[k];
  set_ranges(D, off, ctl->rb, ctl->re);
  const uint32_t alive = N - cnt[A_VACANT];
  const unsigned long long Iafter = I - n_take;   // I -= min(V, I)
  ctl->vac_total = V;
  ctl->n_init = Iafter;
  ctl->n_init_fill = Iafter;   // what k_push reads (it writes n_init itself)
  ctl->iter_cur = ctl->iter;
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

// ================================================================ the bookkeeping kernels (one block per tile)
// k_init_fill: P1 + the per-tile and per-group histograms.
template <bool TRACE, int CPT>
__global__ void __launch_bounds__(kTileThreads) k_init_fill(DeviceState D) {
  __shared__ BookSmem sm;
  Control* ctl = D.ctl;
  const uint32_t tile = blockIdx.x;
  // Before the programmatic-dependency wait: what does NOT depend on the kernel just before this one in the stream
  // (k_push of the previous iteration, or the partition passes, which only touch the stack, its height, `iter` and
  // plist): the vacancy counters and `finished` were last written by the action kernels / the previous k_init_fill,
  // which had completed before that kernel let this one start. The vacancy prefix so overlaps the push.
  const uint32_t finished = ctl->finished;
  uint32_t cnt[CPT];
  load_counters<CPT>(D.tile_vac, D.n_tiles, cnt);
  if (threadIdx.x < 8) { sm.hist[threadIdx.x] = 0; sm.act[threadIdx.x] = 0; }
  uint32_t prefix, V, tile_vacant;
  block_prefix_total_regs<CPT>(cnt, tile, sm.scan, prefix, V, tile_vacant);   // (its barriers also publish sm.hist / sm.act)
  pdl_prologue();
  const uint32_t iter = ctl->iter, n_charged = ctl->part_charged;
  const unsigned long long I = ctl->n_init;
  if (finished) return;
  const TraceScope<K_INIT_FILL, TRACE> trace(D, iter);
  if (threadIdx.x == 8) D.tile_sec[tile] = 0;   // consumed by the push of the previous iteration
  const uint32_t n_take = (unsigned long long)V < I ? V : (uint32_t)I;
  const FillPlan plan = D.sort_mode == 3 ? partition_plan(n_take, V, n_charged) : plain_plan(n_take);
  fill_tile(D, sm, tile, I, plan, prefix, tile_vacant);
  __syncthreads();
  publish_tile_hist(D, sm, tile);
  const uint32_t parity = iter & 1u;
  publish_group_hist(D, sm, tile, parity);
  // No "last block": the block leaves what it filled for k_scatter to take off tile_vac (other blocks of THIS kernel
  // may still be reading the counters), and block 0 leaves the iteration's scalars in fields no fill block reads.
  if (threadIdx.x == 0) {
    D.tile_filled[tile] = filled_by_plan(tile_vacant, prefix, plan);
    if (tile == 0) { ctl->vac_total = V; ctl->n_init_fill = I - n_take; ctl->iter_cur = iter; }
  }
}

// k_scatter (every sort mode; "reindex + close the fill"): takes the filled vacancies off tile_vac; every block sums the <= 128 group rows into the
// iteration's action / sort-key counts, hence the key offsets; block 0 writes them with ranges, counters and the log
// to the control block (S11); in the sorted modes the block then scatters its tile's slot indices (P2).
template <bool TRACE>
__global__ void __launch_bounds__(kTileThreads) k_scatter(DeviceState D) {
  __shared__ BookSmem sm;
  pdl_prologue();
  Control* ctl = D.ctl;
  const uint32_t tile = blockIdx.x;
  const uint32_t finished = ctl->finished, iter = ctl->iter;
  const uint32_t tile_vacant = D.tile_vac[tile] - D.tile_filled[tile];
  const unsigned long long Iafter = ctl->n_init_fill;
  const uint32_t V = ctl->vac_total;
  if (finished) return;   // (block 0 may set it below while others start: they then skip work nobody needs any more)
  const TraceScope<K_SCATTER, TRACE> trace(D, iter);
  if (threadIdx.x == 0) D.tile_vac[tile] = tile_vacant;
  const int n_keys = D.sort_mode == 1 ? 8 : (D.sort_mode == 2 ? 4 : 0);
  {
    const uint32_t parity = iter & 1u;
    const uint32_t n_groups = (D.n_tiles + kGroupTiles - 1) / kGroupTiles;
    const uint32_t g = tile / kGroupTiles, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr int kGroupWarps = kMaxGroups / 32;   // 4
    __shared__ uint32_t act_part[kGroupWarps][8], key_part[kGroupWarps][8], before[kGroupWarps + 1][8], off_s[9];
    if (warp < (uint32_t)kGroupWarps) {   // warp w sums the group rows [32 w, 32 w + 32): all of them (totals) and those before the tile's group
      const uint32_t row = warp * 32 + lane;
      const uint32_t* arows = group_rows(D.group_hist, parity);
      const uint32_t* krows = D.sort_mode == 2 ? group_rows(D.group_phist, parity) : arows;
      uint4 a0 = make_uint4(0, 0, 0, 0), a1 = a0, k0 = a0, k1 = a0;
      if (row < n_groups) {
        a0 = *reinterpret_cast<const uint4*>(arows + row * 8); a1 = *reinterpret_cast<const uint4*>(arows + row * 8 + 4);
        if (D.sort_mode == 2) { k0 = *reinterpret_cast<const uint4*>(krows + row * 8); k1 = *reinterpret_cast<const uint4*>(krows + row * 8 + 4); }
        else { k0 = a0; k1 = a1; }
      }
      const uint32_t av[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
      const uint32_t kv[8] = {k0.x, k0.y, k0.z, k0.w, k1.x, k1.y, k1.z, k1.w};
      const bool bef = row < g;
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        const uint32_t ta = __reduce_add_sync(0xffffffffu, av[k]);
        const uint32_t tk = __reduce_add_sync(0xffffffffu, kv[k]);
        const uint32_t tb = __reduce_add_sync(0xffffffffu, bef ? kv[k] : 0u);
        if (lane == 0) { act_part[warp][k] = ta; key_part[warp][k] = tk; before[warp][k] = tb; }
      }
    } else if (warp == (uint32_t)kGroupWarps) {   // the tile rows of the own group before the tile
      uint32_t s8[8];
      warp_sum_rows(sort_rows(D) + (size_t)g * kGroupTiles * 8, n_keys ? tile - g * kGroupTiles : 0u, s8);
      if (lane == 0) {
#pragma unroll
        for (int k = 0; k < 8; ++k) before[kGroupWarps][k] = s8[k];
      }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      uint32_t act_total[8], key_total[8];
      for (int k = 0; k < 8; ++k) {
        act_total[k] = 0; key_total[k] = 0;
        for (int w = 0; w < kGroupWarps; ++w) { act_total[k] += act_part[w][k]; key_total[k] += key_part[w][k]; }
      }
      uint32_t o = 0;
      for (int k = 0; k < 8; ++k) { off_s[k] = o; if (k < n_keys) o += key_total[k]; }
      if (tile == 0) update_control_after_fill(D, act_total, key_total, n_keys, Iafter, V, 0u);
    }
    __syncthreads();
    if (threadIdx.x < 8) {
      uint32_t b = off_s[threadIdx.x];
      for (int w = 0; w <= kGroupWarps; ++w) b += before[w][threadIdx.x];
      sm.base[threadIdx.x] = b;
    }
  }
  if (n_keys == 0) return;   // modes none / partition: no index array
  __syncthreads();
  scatter_tile(D, sm, tile, tile_vacant);
}

template <bool TRACE, int CPT>
__global__ void __launch_bounds__(kTileThreads) k_push(DeviceState D) {
  __shared__ BookSmem sm;
  pdl_prologue();
  Control* ctl = D.ctl;
  const uint32_t tile = blockIdx.x;
  // No "last block" here: every block forms S itself, and block 0 alone updates the control block — it writes only fields
  // that no block of this kernel reads (n_init and iter are read through the copies k_init_fill left: n_init_fill,
  // iter_cur). The per-tile counters are zeroed by the next k_init_fill.
  const uint32_t finished = ctl->finished, iter = ctl->iter_cur;
  const int32_t error = ctl->error;
  const unsigned long long I = ctl->n_init_fill;
  uint32_t cnt[CPT];
  load_counters<CPT>(D.tile_sec, D.n_tiles, cnt);
  if (finished) return;
  const TraceScope<K_PUSH, TRACE> trace(D, iter);
  uint32_t prefix, S, tile_total;
  block_prefix_total_regs<CPT>(cnt, tile, sm.scan, prefix, S, tile_total);
  const bool overflow = error != 0 || I + S > D.init_capacity;
  if (tile == 0 && threadIdx.x == 0) {
    ctl->push_total = S;
    if (I + S > D.init_capacity) ctl->error = -4;  // CEL_ERR_INIT_OVERFLOW (sticky)
    else if (error == 0) ctl->n_init = I + S;
    ctl->secondaries += S;
    ctl->iter = iter + 1;
  }
  push_tile(D, sm, tile, I, prefix, tile_total, overflow);
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
template <bool TRACE>
__global__ void __launch_bounds__(kTileThreads) k_part_count(DeviceState D) {
  __shared__ BookSmem sm;
  pdl_prologue();
  const Control* ctl = D.ctl;
  if (ctl->finished) return;
  const TraceScope<K_PART_COUNT, TRACE> trace(D, ctl->iter);
  const uint32_t tile = blockIdx.x;
  const unsigned long long I = ctl->n_init;
  uint32_t prefix, V;
  block_prefix_total(D.tile_vac, D.n_tiles, tile, sm.scan, prefix, V);
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
  const TraceScope<K_PART_SCATTER, TRACE> trace(D, ctl->iter);
  const uint32_t tile = blockIdx.x;
  const unsigned long long I = ctl->n_init;
  uint32_t prefix, V, cpre, C;
  block_prefix_total(D.tile_vac, D.n_tiles, tile, sm.scan, prefix, V);
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
    b.meta = make_meta(p.ptype == P_GAMMA ? A_MOVE_G : A_MOVE_C, p.ptype, vol, -1, 0, p.event);
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

// which = 0: sin(x) of the helix substep (x S(x^2)); 1: 1 - cos(x) (x^2 V(x^2)), |x| <= 0.5
__global__ void k_debug_math(int which, const double* in, uint32_t n, double* out) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double x = in[i];
  double S, V;
  sinc_versc_small(x * x, S, V);
  out[i] = which == 0 ? x * S : (x * x) * V;
}

// every slot vacant: key byte 7 (padding 0xff), meta action VACANT (state bytes are otherwise zero); the per-tile
// vacancy counters start at the number of real slots in the tile
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
    if (i < D.n_tiles) {
      const unsigned long long lo = i << D.tile_shift, hi = (i + 1) << D.tile_shift;
      D.tile_vac[i] = (uint32_t)(lo >= D.N ? 0ull : ((hi < D.N ? hi : (unsigned long long)D.N) - lo));
      D.tile_sec[i] = 0;
    }
  }
}

}  // namespace cel

// cel_noalloc.cu — cel_reindex_static (include/cel.h): the P2 reindexing of one step iteration (docs/PHYSICS_SPEC.md S2;
// PAPER.md:41, section 3.2: "state_indices", a stable counting sort of the slot indices by action) for callers that may
// not allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// The transport's own sort (k_fill_sort, cel_kernels.cuh) keeps its per-tile histograms in stream-ordered scratch from
// cudaMallocAsync. This variant keeps them in ONE file-scope device array of a fixed, modest size instead:
//   g_reindex_scratch: kMaxTiles x 8 counters = 128 KB, held by every GPU that loads the library until the process exits;
//   it bounds the call at CEL_REINDEX_STATIC_MAX_SLOTS = 2^22 slots (more is CEL_ERR_TOO_LARGE).
// The entry point calls no cudaMalloc / cudaFree / allocating library routine: two kernel launches on the caller's stream.
// In host code the array's NAME is a host-side stand-in, not a device address; the address the kernels get comes from
// cudaGetSymbolAddress, resolved once per device (with that device current) on the first call there.
//
// Every call on a device shares the array, which keeps the last call's contents. Nothing in it has to start at zero:
// k_static_hist overwrites all 8 counters of every tile the call covers before k_static_scatter (stream-ordered behind it)
// reads exactly those rows; rows of higher tiles are stale and never read. Calls that OVERLAP on the GPU (two streams, two
// host threads with their own streams, two graphs in flight) race on the array: serialise them.
#include "../../include/cel.h"

#include <cuda_runtime.h>

#include <cstdint>
#include <mutex>

namespace {

constexpr uint32_t kThreads = 256;
constexpr uint32_t kKeysPerThread = 4;
constexpr uint32_t kTile = kThreads * kKeysPerThread;                         // 1024 slots per block
constexpr uint64_t kMaxSlots = CEL_REINDEX_STATIC_MAX_SLOTS;                  // 2^22
constexpr uint32_t kMaxTiles = (uint32_t)(kMaxSlots / kTile);                 // 4096
constexpr uint32_t kKeys = 8;                                                 // action keys 0..7 (7 = VACANT)
constexpr uint32_t kScratchWords = kMaxTiles * kKeys;                         // 32768 words = 128 KB

static __device__ __align__(256) uint32_t g_reindex_scratch[kScratchWords];   // [tile][key] counts of the running call

// the thread's four sort keys (the low three bits of the key bytes), packed; slots at or beyond n read as 0xff (skipped everywhere)
__device__ __forceinline__ uint32_t load_keys4(const uint8_t* keys, uint32_t base, uint32_t n) {
  if (base + kKeysPerThread <= n) return *reinterpret_cast<const uint32_t*>(keys + base) & 0x07070707u;   // (keys is 4-byte aligned, base a multiple of 4)
  uint32_t kv = 0xffffffffu;
  for (uint32_t i = 0; i < kKeysPerThread; ++i)
    if (base + i < n) kv = (kv & ~(0xffu << (8 * i))) | ((uint32_t)(keys[base + i] & 7u) << (8 * i));
  return kv;
}

// per-key counts of the thread's four keys, 4 x 16-bit packed in two words (keys 0-3, 4-7); a tile has 1024 slots < 2^16
__device__ __forceinline__ void count_keys4(uint32_t kv, unsigned long long& lo, unsigned long long& hi) {
  lo = 0; hi = 0;
#pragma unroll
  for (uint32_t i = 0; i < kKeysPerThread; ++i) {
    const uint32_t kb = (kv >> (8 * i)) & 0xff;
    if (kb != 0xff) {
      const uint32_t s = kb;
      if (s < 4) lo += 1ull << (16 * s); else hi += 1ull << (16 * (s - 4));
    }
  }
}

__device__ __forceinline__ unsigned long long warp_incl_scan64(unsigned long long v) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const unsigned long long u = __shfl_up_sync(0xffffffffu, v, d);
    if ((int)(threadIdx.x & 31) >= d) v += u;
  }
  return v;
}

// pass 1: the tile's key histogram -> scratch[tile][0..8) (all 8 words written: nothing of an earlier call survives in a row that is read)
__global__ void __launch_bounds__(kThreads) k_static_hist(const uint8_t* keys, uint32_t n, uint32_t* scratch) {
  __shared__ uint32_t hist[kKeys];
  const uint32_t tile = blockIdx.x;
  if (threadIdx.x < kKeys) hist[threadIdx.x] = 0;
  __syncthreads();
  const uint32_t kv = load_keys4(keys, tile * kTile + threadIdx.x * kKeysPerThread, n);
  unsigned long long lo, hi;
  count_keys4(kv, lo, hi);
  // warp totals: at most 128 per key, the 16-bit fields cannot carry
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) { lo += __shfl_xor_sync(0xffffffffu, lo, d); hi += __shfl_xor_sync(0xffffffffu, hi, d); }
  const uint32_t lane = threadIdx.x & 31;
  if (lane < kKeys) {
    const uint32_t c = (uint32_t)(((lane < 4 ? lo : hi) >> (16 * (lane & 3))) & 0xffff);
    if (c) atomicAdd(&hist[lane], c);
  }
  __syncthreads();
  if (threadIdx.x < kKeys) scratch[tile * kKeys + threadIdx.x] = hist[threadIdx.x];
}

// pass 2: indices[offsets[key] + (count of the key in the tiles before) + (rank inside the tile)] = slot, ascending slot
// order inside a key (stable); block 0 also writes offsets[0..9) (offsets[k] = slots with a key below k; offsets[8] = n)
__global__ void __launch_bounds__(kThreads) k_static_scatter(const uint8_t* keys, uint32_t n, uint32_t n_tiles, const uint32_t* scratch,
                                                             uint32_t* indices, uint32_t* offsets) {
  __shared__ uint32_t before[kKeys], total[kKeys], base[kKeys];
  __shared__ unsigned long long wsum[2][kThreads / 32];
  const uint32_t tile = blockIdx.x;
  const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x < kKeys) { before[threadIdx.x] = 0; total[threadIdx.x] = 0; }
  __syncthreads();
  // per-key sums over the rows of all tiles / of the tiles before this one: threads stride over the rows (<= 16 each)
  uint32_t all[kKeys], bef[kKeys];
#pragma unroll
  for (uint32_t j = 0; j < kKeys; ++j) { all[j] = 0; bef[j] = 0; }
  for (uint32_t t = threadIdx.x; t < n_tiles; t += kThreads) {
    const uint4 a = __ldcg(reinterpret_cast<const uint4*>(scratch + t * kKeys)), b = __ldcg(reinterpret_cast<const uint4*>(scratch + t * kKeys + 4));
    const uint32_t r[kKeys] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
#pragma unroll
    for (uint32_t j = 0; j < kKeys; ++j) { all[j] += r[j]; if (t < tile) bef[j] += r[j]; }
  }
#pragma unroll
  for (uint32_t j = 0; j < kKeys; ++j) {
    const uint32_t sa = __reduce_add_sync(0xffffffffu, all[j]), sb = __reduce_add_sync(0xffffffffu, bef[j]);
    if (lane == 0) { if (sa) atomicAdd(&total[j], sa); if (sb) atomicAdd(&before[j], sb); }
  }
  __syncthreads();
  if (threadIdx.x < kKeys) {
    uint32_t off = 0;
    for (uint32_t j = 0; j < threadIdx.x; ++j) off += total[j];
    base[threadIdx.x] = off + before[threadIdx.x];
    if (tile == 0) { offsets[threadIdx.x] = off; if (threadIdx.x == kKeys - 1) offsets[kKeys] = off + total[kKeys - 1]; }
  }
  // ranks inside the tile: exclusive block scan of the packed per-thread counts
  const uint32_t slot0 = tile * kTile + threadIdx.x * kKeysPerThread;
  const uint32_t kv = load_keys4(keys, slot0, n);
  unsigned long long lo, hi;
  count_keys4(kv, lo, hi);
  const unsigned long long ilo = warp_incl_scan64(lo), ihi = warp_incl_scan64(hi);
  if (lane == 31) { wsum[0][warp] = ilo; wsum[1][warp] = ihi; }
  __syncthreads();
  unsigned long long plo = ilo - lo, phi = ihi - hi;
  for (uint32_t w = 0; w < warp; ++w) { plo += wsum[0][w]; phi += wsum[1][w]; }
#pragma unroll
  for (uint32_t i = 0; i < kKeysPerThread; ++i) {
    const uint32_t s = (kv >> (8 * i)) & 0xff;
    if (s != 0xff) {
      uint32_t r;
      if (s < 4) { r = (uint32_t)((plo >> (16 * s)) & 0xffff); plo += 1ull << (16 * s); }
      else { r = (uint32_t)((phi >> (16 * (s - 4))) & 0xffff); phi += 1ull << (16 * (s - 4)); }
      indices[base[s] + r] = slot0 + i;
    }
  }
}

// the device address of g_reindex_scratch, per device: resolved once, with that device current
constexpr int kMaxDevices = 64;
uint32_t* g_scratch_addr[kMaxDevices] = {};
std::mutex g_scratch_mutex;

int scratch_address(uint32_t** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return CEL_ERR_CUDA;
  std::lock_guard<std::mutex> lock(g_scratch_mutex);
  if (!g_scratch_addr[dev]) {
    uint32_t* p = nullptr;
    if (cudaGetSymbolAddress((void**)&p, g_reindex_scratch) != cudaSuccess || !p) return CEL_ERR_CUDA;
    g_scratch_addr[dev] = p;
  }
  *out = g_scratch_addr[dev];
  return CEL_OK;
}

}  // namespace

extern "C" uint64_t cel_reindex_static_max_slots(void) { return kMaxSlots; }

extern "C" int cel_reindex_static(const uint8_t* d_keys, uint64_t n_slots, uint32_t* d_indices, uint32_t* d_offsets, void* cuda_stream) {
  if (n_slots > kMaxSlots) return CEL_ERR_TOO_LARGE;
  if (!d_offsets || (n_slots && (!d_keys || !d_indices)) || (reinterpret_cast<uintptr_t>(d_keys) & 3u)) return CEL_ERR_INVALID_ARG;
  uint32_t* scratch = nullptr;
  const int rc = scratch_address(&scratch);
  if (rc != CEL_OK) return rc;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const uint32_t n = (uint32_t)n_slots;
  const uint32_t n_tiles = n ? (n + kTile - 1) / kTile : 1u;   // (n = 0: one block writes the all-zero offsets)
  k_static_hist<<<n_tiles, kThreads, 0, s>>>(d_keys, n, scratch);
  k_static_scatter<<<n_tiles, kThreads, 0, s>>>(d_keys, n, n_tiles, scratch, d_indices, d_offsets);
  return cudaGetLastError() == cudaSuccess ? CEL_OK : CEL_ERR_CUDA;
}

// gg_unique_count_static: the window unique + count step (a-3: U_k ascending with c_k)
// for callers that must not allocate device memory.
//
// Who that is.  A trainer whose framework allocator has already claimed (almost) all of the HBM --
// the usual state of a training process a few seconds after start-up -- gets cudaErrorMemoryAllocation
// from any library that calls cudaMalloc behind its back, and a serving or training loop with several
// streams in flight cannot afford cudaFree, which waits for the whole device.  The rest of this library
// allocates its workspaces in gg_graph_create and grows them in gg_window_stage; this one entry point
// never does.  Its workspace -- the direct-address array of packed 8-bit access counters that the
// ordinary path keeps in cudaMalloc'ed memory (window.cu), plus one partial sum per tile -- is the
// file-scope array below.  It is part of the library image: every GPU that loads libgreengnn.so
// carries these 4 MiB + 2 KiB until the process exits, and that fixed size is what caps num_nodes
// at GG_STATIC_MAX_NODES.
//
// The array is shared by every call on a device and still holds what the previous call left there.
// Each call therefore begins by clearing the counters it is about to use (a cudaMemsetAsync on the
// caller's stream; the tile sums are fully overwritten before they are read).  Two calls whose GPU work
// overlaps (different streams with no ordering between them, or two host threads) race on the array.
//
// Host code cannot use the array's name as a pointer: on the host `g_static_scratch` is only a stand-in
// the runtime uses to look the real array up.  The device address is fetched once per device with
// cudaGetSymbolAddress (with that device current) by the first call made on that device and handed to
// the kernels as an ordinary pointer argument.
#include <cstdio>
#include <mutex>

#include "common.cuh"
#include "kernels.h"

namespace gg {

constexpr int64_t kStaticCntWords = GG_STATIC_MAX_NODES / 4;          // four 8-bit counters per word
constexpr int kStaticMaxTiles = (int)(kStaticCntWords / kWordTile);   // 512
static_assert(kStaticCntWords % kWordTile == 0, "counter words must be whole tiles");

// [0, kStaticCntWords) packed counters, then kStaticMaxTiles tile sums
static __device__ __align__(256) uint32_t g_static_scratch[kStaticCntWords + kStaticMaxTiles];

static std::mutex s_setup_mutex;
static uint32_t* s_scratch_of_device[64] = {nullptr};

// Device address of g_static_scratch on the current device (looked up on the first call there).
static cudaError_t static_scratch(uint32_t** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(s_setup_mutex);
  if (!s_scratch_of_device[dev]) {
    uint32_t* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_static_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    s_scratch_of_device[dev] = p;
  }
  *out = s_scratch_of_device[dev];
  return cudaSuccess;
}

// stats[1] += number of IDs outside [0, num_nodes) (they are not counted)
__global__ void __launch_bounds__(256)
k_static_bump(const int32_t* __restrict__ ids, int64_t n, int32_t num_nodes, uint32_t* __restrict__ cnt8,
              int32_t* __restrict__ stats) {
  int bad = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const int32_t u = ids[i];
    if ((uint32_t)u < (uint32_t)num_nodes) atomicAdd(cnt8 + (u >> 2), 1u << (8 * (u & 3)));
    else ++bad;
  }
  bad = __reduce_add_sync(0xffffffffu, bad);
  if ((threadIdx.x & 31) == 0 && bad) atomicAdd(stats + 1, bad);
}

__device__ __forceinline__ int static_nz_bytes(uint32_t x) {
  uint32_t m = (x | (x >> 4)) & 0x0F0F0F0Fu;
  m = (m | (m >> 2)) & 0x03030303u;
  m = (m | (m >> 1)) & 0x01010101u;
  return __popc(m);
}

// tile_sums[t] = distinct IDs in tile t (kWordTile words = 8192 node IDs)
__global__ void __launch_bounds__(kWordThreads)
k_static_reduce(const uint32_t* __restrict__ cnt8, int32_t* __restrict__ tile_sums) {
  __shared__ int32_t sm[33];
  const int64_t w0 = (int64_t)blockIdx.x * kWordTile + threadIdx.x * 8;
  const uint4* p = reinterpret_cast<const uint4*>(cnt8 + w0);
  const uint4 a = p[0], c = p[1];
  const uint32_t x[8] = {a.x, a.y, a.z, a.w, c.x, c.y, c.z, c.w};
  int s = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += x[k] ? static_nz_bytes(x[k]) : 0;
  int32_t tot;
  block_exclusive_scan<int32_t>(s, sm, &tot);
  if (threadIdx.x == 0) tile_sums[blockIdx.x] = tot;
}

// Every CTA adds up the (at most 512) tile sums itself: the ones before its tile give its output
// offset, all of them give |U|.  Nothing is written when |U| exceeds the caller's capacity.
__global__ void __launch_bounds__(kWordThreads)
k_static_emit(const uint32_t* __restrict__ cnt8, const int32_t* __restrict__ tile_sums, int tiles,
              int64_t capacity, int32_t* __restrict__ uniq, int32_t* __restrict__ cnt,
              int32_t* __restrict__ stats) {
  __shared__ int32_t sm[33];
  __shared__ int32_t s_before, s_total;
  const int t = blockIdx.x;
  if (threadIdx.x == 0) s_before = s_total = 0;
  __syncthreads();
  int before = 0, total = 0;
  for (int i = threadIdx.x; i < tiles; i += blockDim.x) {
    const int32_t v = tile_sums[i];
    total += v;
    if (i < t) before += v;
  }
  before = __reduce_add_sync(0xffffffffu, before);
  total = __reduce_add_sync(0xffffffffu, total);
  if ((threadIdx.x & 31) == 0) {
    atomicAdd(&s_before, before);
    atomicAdd(&s_total, total);
  }
  __syncthreads();
  if (t == 0 && threadIdx.x == 0) stats[0] = s_total;
  if ((int64_t)s_total > capacity) return;

  const int64_t w0 = (int64_t)t * kWordTile + threadIdx.x * 8;
  const uint4* p = reinterpret_cast<const uint4*>(cnt8 + w0);
  const uint4 a = p[0], c = p[1];
  const uint32_t x[8] = {a.x, a.y, a.z, a.w, c.x, c.y, c.z, c.w};
  int s = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += x[k] ? static_nz_bytes(x[k]) : 0;
  int32_t tot;
  const int32_t ex = block_exclusive_scan<int32_t>(s, sm, &tot);
  if (!s) return;
  int32_t run = s_before + ex;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    if (!x[k]) continue;
    for (int q = 0; q < 4; ++q) {
      const int cv = (x[k] >> (8 * q)) & 0xFF;
      if (cv) {
        uniq[run] = (int32_t)((w0 + k) * 4 + q);
        cnt[run] = cv;
        ++run;
      }
    }
  }
}

}  // namespace gg

extern "C" gg_status gg_unique_count_static(const int32_t* ids, int64_t n_ids, int64_t num_nodes,
                                            int32_t* uniq, int32_t* cnt, int64_t capacity,
                                            int32_t* stats, void* cuda_stream) {
  using namespace gg;
  char msg[256];
  if (n_ids < 0 || capacity < 0 || num_nodes < 1 || !stats || (n_ids > 0 && !ids) ||
      (capacity > 0 && (!uniq || !cnt)))
    return report_error(GG_ERR_INVALID_ARG, "gg_unique_count_static: null pointer or negative size");
  if (num_nodes > GG_STATIC_MAX_NODES) {
    snprintf(msg, sizeof msg,
             "gg_unique_count_static: num_nodes %lld exceeds GG_STATIC_MAX_NODES (%d): the counters live in a "
             "fixed-size array inside the library; use gg_window_stage for larger graphs",
             (long long)num_nodes, (int)GG_STATIC_MAX_NODES);
    return report_error(GG_ERR_CAPACITY, msg);
  }
  uint32_t* scratch = nullptr;
  cudaError_t e = static_scratch(&scratch);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int64_t words = (num_nodes + 3) / 4;
  const int tiles = (int)((words + kWordTile - 1) / kWordTile);
  uint32_t* cnt8 = scratch;
  int32_t* tile_sums = reinterpret_cast<int32_t*>(scratch + kStaticCntWords);
  // the previous call's counters are still there: clear the tiles this call reads
  if (e == cudaSuccess) e = cudaMemsetAsync(cnt8, 0, (size_t)tiles * kWordTile * sizeof(uint32_t), st);
  if (e == cudaSuccess) e = cudaMemsetAsync(stats, 0, 2 * sizeof(int32_t), st);
  if (e == cudaSuccess) {
    if (n_ids > 0) {
      int64_t grid = (n_ids + 255) / 256;
      const int64_t cap = (int64_t)sm_count() * 16;
      if (grid > cap) grid = cap;
      k_static_bump<<<(unsigned)grid, 256, 0, st>>>(ids, n_ids, (int32_t)num_nodes, cnt8, stats);
      count_launches(1);
    }
    k_static_reduce<<<tiles, kWordThreads, 0, st>>>(cnt8, tile_sums);
    k_static_emit<<<tiles, kWordThreads, 0, st>>>(cnt8, tile_sums, tiles, capacity, uniq, cnt, stats);
    count_launches(2);
    e = cudaGetLastError();
  }
  if (e != cudaSuccess) {
    snprintf(msg, sizeof msg, "gg_unique_count_static: %s", cudaGetErrorString(e));
    return report_error(GG_ERR_CUDA, msg);
  }
  return GG_OK;
}

// Shared device/host helpers of the CUDA path (sm_100a).  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/greengnn.h"

namespace gg {

// ---- sampling key (reading S1; include/greengnn.h gg_key) -----------------------
// SplitMix64: state += gamma; output = fmix(state).  All arithmetic mod 2^64.
constexpr uint64_t kGamma = 0x9E3779B97F4A7C15ull;

__host__ __device__ __forceinline__ uint64_t fmix64(uint64_t z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
__host__ __device__ __forceinline__ uint64_t splitmix_step(uint64_t x) { return fmix64(x + kGamma); }
// prefix shared by every destination of (batch, layer): sm(sm(sm(seed) ^ batch) ^ layer)
__host__ __device__ __forceinline__ uint64_t key_prefix(uint64_t seed, uint64_t batch, uint64_t layer) {
  return splitmix_step(splitmix_step(splitmix_step(seed) ^ batch) ^ layer);
}
__host__ __device__ __forceinline__ uint64_t key_hdst(uint64_t prefix, uint64_t dst) {
  return splitmix_step(prefix ^ dst);
}
__host__ __device__ __forceinline__ uint64_t key_edge(uint64_t hdst, uint64_t j) {
  return fmix64(hdst + (j + 1) * kGamma);
}

// ---- small POD passed by value to kernels --------------------------------------------------
// Exclusive prefix over the window's batches of a per-batch size (destinations of a hop).
struct BatchOffsets {
  int32_t v[GG_MAX_WINDOW + 1];
};
struct OwnerRanges {
  int32_t P, local;
  int64_t lo[GG_MAX_PARTS + 1];
};
struct StorePtrs {
  const uint8_t* base[GG_MAX_PARTS];
  int64_t stride;
};

__device__ __forceinline__ int find_batch(const int32_t* off, int W, int x) {
  // largest b with off[b] <= x  (off ascending, off[0] = 0, x < off[W])
  int lo = 0, hi = W;
  while (hi - lo > 1) {
    int mid = (lo + hi) >> 1;
    if (off[mid] <= x) lo = mid; else hi = mid;
  }
  return lo;
}
__device__ __forceinline__ int owner_of(const OwnerRanges& R, int32_t u) {
  int m = 0;
#pragma unroll 1
  for (int k = 1; k < R.P; ++k) m += (u >= R.lo[k]);
  return m;
}

__device__ __forceinline__ unsigned lanemask_lt() {
  unsigned m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

// CTA-wide exclusive scan of one value per thread (blockDim.x <= 1024, multiple of 32).
// Returns the exclusive prefix; *total gets the CTA sum.  `smem` holds 33 T's.
template <typename T>
__device__ __forceinline__ T block_exclusive_scan(T v, T* smem, T* total) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  T x = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    T y = __shfl_up_sync(0xffffffffu, x, o);
    if (lane >= o) x += y;
  }
  if (lane == 31) smem[wid] = x;
  __syncthreads();
  if (wid == 0) {
    T s = lane < nw ? smem[lane] : T(0);
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      T y = __shfl_up_sync(0xffffffffu, s, o);
      if (lane >= o) s += y;
    }
    smem[lane] = s;  // inclusive over warps
  }
  __syncthreads();
  T base = wid ? smem[wid - 1] : T(0);
  *total = smem[nw - 1];
  T r = base + x - v;
  __syncthreads();
  return r;
}

}  // namespace gg

// a-3 window unique + count, a-4 hot-set select, a-5 owner split / rebuild delta.
//
// a-3  The per-window access counts live in a direct-address array of packed 8-bit lanes
//      (4 nodes per 32-bit word) that the frontier kernels bumped once per (batch, node).
//      One compaction pass turns it into U_k (ascending) and c_k, and zeroes it again.
//      The same pass classifies remote nodes and builds the histogram of their counts.
// a-4  H_k = the n_hot remote nodes smallest under (-count, id) (reading S10).
//      Counts are <= W, so the host turns the histogram into a threshold t and a quota r of
//      count == t nodes; one 2-lane scan places every selected node in ascending-ID order.
// a-5  Delta_{k,m} = (H_k n N_m) \ (C_{k-1} n N_m): H_k is ascending, owners are
//      ID ranges, so the delta list in ID order is already grouped by owner.  Slots in the new
//      cache buffer: [0, |Delta|) = delta rows in request order (each owner contiguous, so one
//      bulk copy per owner lands in place), then the carried rows.
#include "common.cuh"
#include "kernels.h"

namespace gg {

std::atomic<unsigned long long> g_launches{0};

int sm_count() {
  static int cached[64] = {0};
  int dev = 0;
  cudaGetDevice(&dev);
  if (dev < 0 || dev >= 64) dev = 0;
  if (!cached[dev]) {
    int n = 0;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n < 1) n = 148;
    cached[dev] = n;
  }
  return cached[dev];
}

template <typename T>
__global__ void __launch_bounds__(1024) k_row_scan(T* __restrict__ tiles, int n, T* __restrict__ total) {
  __shared__ T sm[33];
  __shared__ T carry_s;
  if (threadIdx.x == 0) carry_s = T(0);
  __syncthreads();
  for (int base = 0; base < n; base += blockDim.x) {
    const int i = base + threadIdx.x;
    T v = i < n ? tiles[i] : T(0), tot;
    T ex = block_exclusive_scan<T>(v, sm, &tot);
    const T carry = carry_s;
    if (i < n) tiles[i] = carry + ex;
    __syncthreads();
    if (threadIdx.x == 0) carry_s = carry + tot;
    __syncthreads();
  }
  if (threadIdx.x == 0) *total = carry_s;
}

__device__ __forceinline__ int nz_bytes(uint32_t x) {
  // one bit per non-zero byte
  uint32_t m = (x | (x >> 4)) & 0x0F0F0F0Fu;
  m = (m | (m >> 2)) & 0x03030303u;
  m = (m | (m >> 1)) & 0x01010101u;
  return __popc(m);
}

// stats[0] = |U_k|, stats[1] = |R_k|; hist[c] = #remote nodes with count c
__global__ void __launch_bounds__(kWordThreads)
k_cnt_reduce(const uint32_t* __restrict__ cnt8, OwnerRanges R, int32_t* __restrict__ tile_sums,
             int32_t* __restrict__ hist) {
  __shared__ int32_t sm[33];
  __shared__ int32_t s_hist[256];
  const int t = blockIdx.x;
  s_hist[threadIdx.x] = 0;
  __syncthreads();
  const int64_t w0 = (int64_t)t * kWordTile + threadIdx.x * 8;
  const uint4* p = reinterpret_cast<const uint4*>(cnt8 + w0);
  const uint4 a = p[0], c = p[1];
  const uint32_t x[8] = {a.x, a.y, a.z, a.w, c.x, c.y, c.z, c.w};
  int s = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    if (!x[k]) continue;
    s += nz_bytes(x[k]);
    for (int q = 0; q < 4; ++q) {
      const int cv = (x[k] >> (8 * q)) & 0xFF;
      if (cv) {
        const int32_t u = (int32_t)((w0 + k) * 4 + q);
        if (owner_of(R, u) != R.local) atomicAdd(&s_hist[cv], 1);
      }
    }
  }
  int32_t tot;
  block_exclusive_scan<int32_t>(s, sm, &tot);
  if (threadIdx.x == 0) tile_sums[t] = tot;
  const int hv = s_hist[threadIdx.x];
  if (hv) atomicAdd(hist + threadIdx.x, hv);
}

__global__ void __launch_bounds__(kWordThreads)
k_cnt_emit(uint32_t* __restrict__ cnt8, const int32_t* __restrict__ tile_sums,
           int32_t* __restrict__ uniq, int32_t* __restrict__ cnt) {
  __shared__ int32_t sm[33];
  const int t = blockIdx.x;
  const int64_t w0 = (int64_t)t * kWordTile + threadIdx.x * 8;
  uint4* p = reinterpret_cast<uint4*>(cnt8 + w0);
  const uint4 a = p[0], c = p[1];
  const uint32_t x[8] = {a.x, a.y, a.z, a.w, c.x, c.y, c.z, c.w};
  int s = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += x[k] ? nz_bytes(x[k]) : 0;
  int32_t tot;
  const int32_t ex = block_exclusive_scan<int32_t>(s, sm, &tot);
  if (!s) return;
  int32_t run = tile_sums[t] + ex;
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
  const uint4 z = make_uint4(0, 0, 0, 0);
  if (a.x | a.y | a.z | a.w) p[0] = z;
  if (c.x | c.y | c.z | c.w) p[1] = z;
}

// ---- a-4 -----------------------------------------------------------------------------------
constexpr int kSelThreads = 256, kSelPer = 4, kSelTile = kSelThreads * kSelPer;

__device__ __forceinline__ uint64_t sel_flags(const OwnerRanges& R, int32_t u, int32_t c, int32_t thr) {
  if (owner_of(R, u) == R.local) return 0;
  return c > thr ? (1ull << 32) : (c == thr ? 1ull : 0ull);
}

__global__ void __launch_bounds__(kSelThreads)
k_select_reduce(const int32_t* __restrict__ uniq, const int32_t* __restrict__ cnt, int n,
                OwnerRanges R, int32_t thr, uint64_t* __restrict__ tile_sums) {
  __shared__ uint64_t sm[33];
  const int i0 = blockIdx.x * kSelTile + threadIdx.x * kSelPer;
  uint64_t s = 0;
#pragma unroll
  for (int k = 0; k < kSelPer; ++k)
    if (i0 + k < n) s += sel_flags(R, uniq[i0 + k], cnt[i0 + k], thr);
  uint64_t tot;
  block_exclusive_scan<uint64_t>(s, sm, &tot);
  if (threadIdx.x == 0) tile_sums[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(kSelThreads)
k_select_emit(const int32_t* __restrict__ uniq, const int32_t* __restrict__ cnt, int n,
              OwnerRanges R, int32_t thr, uint32_t quota_eq, const uint64_t* __restrict__ tile_sums,
              int32_t* __restrict__ hot) {
  __shared__ uint64_t sm[33];
  const int i0 = blockIdx.x * kSelTile + threadIdx.x * kSelPer;
  uint64_t f[kSelPer], s = 0;
#pragma unroll
  for (int k = 0; k < kSelPer; ++k) {
    f[k] = (i0 + k < n) ? sel_flags(R, uniq[i0 + k], cnt[i0 + k], thr) : 0;
    s += f[k];
  }
  uint64_t tot;
  uint64_t run = block_exclusive_scan<uint64_t>(s, sm, &tot) + tile_sums[blockIdx.x];
#pragma unroll
  for (int k = 0; k < kSelPer; ++k) {
    if (f[k]) {
      const uint32_t gt = (uint32_t)(run >> 32), eq = (uint32_t)run;
      const bool is_gt = (f[k] >> 32) != 0;
      if (is_gt || eq < quota_eq) hot[gt + (eq < quota_eq ? eq : quota_eq)] = uniq[i0 + k];
      run += f[k];
    }
  }
}

// ---- a-5 -----------------------------------------------------------------------------------
// owner_cnt[m] = |H_k n N_m| ; owner_cnt[GG_MAX_PARTS + m] = |Delta_{k,m}|
__global__ void __launch_bounds__(kSelThreads)
k_delta_reduce(const int32_t* __restrict__ hot, int n, OwnerRanges R,
               const int32_t* __restrict__ slot_prev, int carry_over,
               int32_t* __restrict__ tile_sums, int32_t* __restrict__ owner_cnt) {
  __shared__ int32_t sm[33];
  __shared__ int32_t s_cnt[2 * GG_MAX_PARTS];
  if (threadIdx.x < 2 * GG_MAX_PARTS) s_cnt[threadIdx.x] = 0;
  __syncthreads();
  const int i0 = blockIdx.x * kSelTile + threadIdx.x * kSelPer;
  int s = 0;
#pragma unroll
  for (int k = 0; k < kSelPer; ++k) {
    if (i0 + k < n) {
      const int32_t u = hot[i0 + k];
      const int m = owner_of(R, u);
      const int is_delta = carry_over ? (slot_prev[u] < 0) : 1;
      atomicAdd(&s_cnt[m], 1);
      if (is_delta) atomicAdd(&s_cnt[GG_MAX_PARTS + m], 1);
      s += is_delta;
    }
  }
  int32_t tot;
  block_exclusive_scan<int32_t>(s, sm, &tot);
  if (threadIdx.x == 0) tile_sums[blockIdx.x] = tot;
  if (threadIdx.x < 2 * GG_MAX_PARTS && s_cnt[threadIdx.x]) atomicAdd(owner_cnt + threadIdx.x, s_cnt[threadIdx.x]);
}

__global__ void __launch_bounds__(kSelThreads)
k_delta_emit(const int32_t* __restrict__ hot, int n, const int32_t* __restrict__ slot_prev,
             int carry_over, const int32_t* __restrict__ tile_sums, const int32_t* __restrict__ n_delta,
             int32_t* __restrict__ slot_new, int32_t* __restrict__ req_ids,
             int32_t* __restrict__ carry_src, int32_t* __restrict__ carry_ids) {
  __shared__ int32_t sm[33];
  const int i0 = blockIdx.x * kSelTile + threadIdx.x * kSelPer;
  int32_t u[kSelPer], sp[kSelPer];
  int s = 0;
#pragma unroll
  for (int k = 0; k < kSelPer; ++k) {
    sp[k] = -1;
    if (i0 + k < n) {
      u[k] = hot[i0 + k];
      if (carry_over) sp[k] = slot_prev[u[k]];
      s += sp[k] < 0;
    }
  }
  int32_t tot;
  int32_t run = block_exclusive_scan<int32_t>(s, sm, &tot) + tile_sums[blockIdx.x];
  const int32_t nd = *n_delta;
#pragma unroll
  for (int k = 0; k < kSelPer; ++k) {
    if (i0 + k < n) {
      if (sp[k] < 0) {
        req_ids[run] = u[k];
        slot_new[u[k]] = run;
        ++run;
      } else {
        const int32_t r = (i0 + k) - run;  // carried rows before this one
        slot_new[u[k]] = nd + r;
        carry_src[r] = sp[k];
        carry_ids[r] = u[k];
      }
    }
  }
}

__global__ void k_slots_clear(const int32_t* __restrict__ ids, int n, int32_t* __restrict__ slot_map) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x)
    slot_map[ids[i]] = -1;
}

__global__ void k_fill_i32(int32_t* p, int64_t n, int32_t v) {
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
    p[i] = v;
}

void launch_unique_count(cudaStream_t st, uint32_t* cnt8, int64_t n_words_padded, const OwnerRanges& R,
                         int32_t* tile_sums, int32_t* stats, int32_t* hist, int32_t* uniq, int32_t* cnt) {
  const int tiles = (int)(n_words_padded / kWordTile);
  cudaMemsetAsync(hist, 0, 256 * sizeof(int32_t), st);
  count_launches(3);
  k_cnt_reduce<<<tiles, kWordThreads, 0, st>>>(cnt8, R, tile_sums, hist);
  k_row_scan<int32_t><<<1, 1024, 0, st>>>(tile_sums, tiles, stats);
  k_cnt_emit<<<tiles, kWordThreads, 0, st>>>(cnt8, tile_sums, uniq, cnt);
}

void launch_hot_select(cudaStream_t st, const int32_t* uniq, const int32_t* cnt, int n_unique,
                       const OwnerRanges& R, int32_t thr, uint32_t quota_eq, uint64_t* tile_sums64,
                       uint64_t* total64, int32_t* hot) {
  if (n_unique <= 0) return;
  const int tiles = (n_unique + kSelTile - 1) / kSelTile;
  count_launches(3);
  k_select_reduce<<<tiles, kSelThreads, 0, st>>>(uniq, cnt, n_unique, R, thr, tile_sums64);
  k_row_scan<uint64_t><<<1, 1024, 0, st>>>(tile_sums64, tiles, total64);
  k_select_emit<<<tiles, kSelThreads, 0, st>>>(uniq, cnt, n_unique, R, thr, quota_eq, tile_sums64, hot);
}

void launch_delta_split(cudaStream_t st, const int32_t* hot, int n_hot, const OwnerRanges& R,
                        const int32_t* slot_prev, int carry_over, int32_t* tile_sums,
                        int32_t* n_delta, int32_t* owner_cnt, int32_t* slot_new, int32_t* req_ids,
                        int32_t* carry_src, int32_t* carry_ids) {
  cudaMemsetAsync(owner_cnt, 0, 2 * GG_MAX_PARTS * sizeof(int32_t), st);
  cudaMemsetAsync(n_delta, 0, sizeof(int32_t), st);
  if (n_hot <= 0) return;
  const int tiles = (n_hot + kSelTile - 1) / kSelTile;
  count_launches(3);
  k_delta_reduce<<<tiles, kSelThreads, 0, st>>>(hot, n_hot, R, slot_prev, carry_over, tile_sums, owner_cnt);
  k_row_scan<int32_t><<<1, 1024, 0, st>>>(tile_sums, tiles, n_delta);
  k_delta_emit<<<tiles, kSelThreads, 0, st>>>(hot, n_hot, slot_prev, carry_over, tile_sums, n_delta,
                                              slot_new, req_ids, carry_src, carry_ids);
}

void launch_slots_clear(cudaStream_t st, const int32_t* ids, int n, int32_t* slot_map) {
  if (n <= 0) return;
  int g = (n + 255) / 256;
  if (g > sm_count() * 8) g = sm_count() * 8;
  k_slots_clear<<<g, 256, 0, st>>>(ids, n, slot_map);
  count_launches(1);
}

// Control-plane words (sizes, histograms, seeds, request IDs) between device memory and PINNED
// host memory, moved by a kernel through the unified address space instead of the copy engines:
// a cudaMemcpyAsync of a few bytes queues behind whatever bulk transfer occupies that engine
// (a 181 MB staging copy holds the H2D engine for 3.8 ms), which stalled the sampler thread.
__global__ void __launch_bounds__(256) k_copy_words(uint32_t* __restrict__ dst, const uint32_t* __restrict__ src, int64_t n) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
    dst[i] = src[i];
}
void launch_copy_words(cudaStream_t st, void* dst, const void* src, int64_t n_words) {
  if (n_words <= 0) return;
  int64_t g = (n_words + 255) / 256;
  if (g > 64) g = 64;
  k_copy_words<<<(int)g, 256, 0, st>>>((uint32_t*)dst, (const uint32_t*)src, n_words);
  count_launches(1);
}

void launch_fill_i32(cudaStream_t st, int32_t* p, int64_t n, int32_t v) {
  if (n <= 0) return;
  int64_t g = (n + 255) / 256;
  if (g > sm_count() * 16) g = sm_count() * 16;
  k_fill_i32<<<(int)g, 256, 0, st>>>(p, n, v);
  count_launches(1);
}

}  // namespace gg

// a-7 slot-map gather, a-8 miss fill, and the row movers of a-6 (carry-over copy, pull staging).
//
// All four are the same operation -- copy n rows of `rb` opaque bytes from per-row sources to
// per-row destinations -- differing only in how a row's source and destination are resolved:
//   GatherResolve  u = N_b[i]: local -> HBM store row; remote with slot_of[u] >= 0 -> cache row;
//                  else MISS (Alg. 1 l.11-12).  dst = X_b row i (dense).
//   ListResolve    src = src_base + src_idx[i]*src_stride, dst = dst_base + (dst_row0+i)*dst_stride
//                  (carry-over copy out of the previous cache buffer).
//   StoreResolve   src = owner store row of id[i] (pinned host through UVA when remote),
//                  dst = dst_base + (pos ? pos[i] : dst_row0+i)*dst_stride  (miss fill; pull staging).
// Kernel shape: a CTA takes a tile of kRows rows, resolves the row pointers ONCE into shared
// memory (index tile staged in smem), then all threads stream the tile as a flat run of
// VEC-byte chunks: loads are contiguous inside a row, stores are fully coalesced when the
// destination is dense.  Misses are compacted in tile order with warp ballot + popc.
#include <cstdlib>

#include "common.cuh"
#include "kernels.h"

namespace gg {

constexpr int kRows = 64;        // rows per tile
constexpr int kThreads = 256;
constexpr int kUnroll = 4;

template <int VEC> struct VecT;
template <> struct VecT<16> { using type = uint4; };
template <> struct VecT<8> { using type = uint2; };
template <> struct VecT<4> { using type = uint32_t; };

template <int VEC>
__device__ __forceinline__ typename VecT<VEC>::type ld_stream(const uint8_t* p) {
  return __ldg(reinterpret_cast<const typename VecT<VEC>::type*>(p));
}
template <int VEC>
__device__ __forceinline__ void st_stream(uint8_t* p, typename VecT<VEC>::type v) {
  __stcs(reinterpret_cast<typename VecT<VEC>::type*>(p), v);  // write-once output: streaming store
}

// Copies the tile's rows.  s_src[r] == nullptr means "skip row r".  If DENSE_DST the tile's
// destination is one contiguous run starting at dst0 (row pitch = rb).
// One (sub-)warp per row: lane l of the row's group moves chunk l, l + lpr, ... of the row, so a row
// costs one load and one store instruction per 32 chunks and no index arithmetic beyond the row
// pointer -- round 1's flat chunk numbering spent ~50 warp instructions per row on a division per
// chunk, which is what made the gather lose 40 % of its bandwidth beside the (issue-bound) sampler.
// Rows narrower than 17 chunks share a warp (lpr = 16, 8, ...: two, four, ... rows per instruction).
// UNROLL rows (or UNROLL chunks of a wide row) are in flight per lane before the first store.
template <int VEC, bool DENSE_DST, int UNROLL = kUnroll>
__device__ __forceinline__ void copy_tile(const uint8_t* const* s_src, uint8_t* const* s_dst,
                                          uint8_t* dst0, int rows, int rb) {
  using V = typename VecT<VEC>::type;
  const int cpr = rb / VEC;                       // chunks per row
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  constexpr int kWarpsPerCta = kThreads / 32;
  if (cpr <= 32) {
    int lpr = 32;                                 // lanes per row: smallest power of two >= cpr
    while ((lpr >> 1) >= cpr) lpr >>= 1;
    const int rpi = 32 / lpr;                     // rows per warp instruction
    const int sub = lane / lpr, l = lane - sub * lpr;
    const bool lane_on = l < cpr;
    const int step = kWarpsPerCta * rpi;
    for (int r0 = wid * rpi + sub; r0 < rows; r0 += step * UNROLL) {
      V v[UNROLL];
      bool ok[UNROLL];
#pragma unroll
      for (int k = 0; k < UNROLL; ++k) {
        const int r = r0 + k * step;
        const uint8_t* src = r < rows ? s_src[r] : nullptr;
        ok[k] = lane_on && src != nullptr;
        if (ok[k]) v[k] = ld_stream<VEC>(src + (int64_t)l * VEC);
      }
#pragma unroll
      for (int k = 0; k < UNROLL; ++k) {
        if (ok[k]) {
          const int r = r0 + k * step;
          uint8_t* d = DENSE_DST ? dst0 + (int64_t)r * rb : s_dst[r];
          st_stream<VEC>(d + (int64_t)l * VEC, v[k]);
        }
      }
    }
  } else {
    for (int r = wid; r < rows; r += kWarpsPerCta) {
      const uint8_t* src = s_src[r];
      if (src == nullptr) continue;
      uint8_t* d = DENSE_DST ? dst0 + (int64_t)r * rb : s_dst[r];
      for (int c0 = lane; c0 < cpr; c0 += 32 * UNROLL) {
        V v[UNROLL];
#pragma unroll
        for (int k = 0; k < UNROLL; ++k)
          if (c0 + 32 * k < cpr) v[k] = ld_stream<VEC>(src + (int64_t)(c0 + 32 * k) * VEC);
#pragma unroll
        for (int k = 0; k < UNROLL; ++k)
          if (c0 + 32 * k < cpr) st_stream<VEC>(d + (int64_t)(c0 + 32 * k) * VEC, v[k]);
      }
    }
  }
}

// Flat variant for rows that cross the host link (pull staging, miss fill): the tile is one run of
// chunks, thread t takes chunks t, t + 256, ... -- every lane carries a load whatever the row
// width (a 400-byte row fills only 25 lanes of a warp), which is what counts when the transfer is
// bound by the bytes in flight over PCIe; the division per chunk does not matter at link speed.
template <int VEC, int UNROLL>
__device__ __forceinline__ void copy_tile_flat(const uint8_t* const* s_src, uint8_t* const* s_dst, int rows, int rb) {
  const int cpr = rb / VEC, total = rows * cpr;
  for (int c0 = threadIdx.x; c0 < total; c0 += kThreads * UNROLL) {
    typename VecT<VEC>::type v[UNROLL];
    int row[UNROLL], col[UNROLL];
    bool ok[UNROLL];
#pragma unroll
    for (int k = 0; k < UNROLL; ++k) {
      const int c = c0 + k * kThreads;
      row[k] = c / cpr;
      col[k] = c - row[k] * cpr;
      ok[k] = c < total && s_src[row[k] < rows ? row[k] : 0] != nullptr;
      if (ok[k]) v[k] = ld_stream<VEC>(s_src[row[k]] + (int64_t)col[k] * VEC);
    }
#pragma unroll
    for (int k = 0; k < UNROLL; ++k)
      if (ok[k]) st_stream<VEC>(s_dst[row[k]] + (int64_t)col[k] * VEC, v[k]);
  }
}

struct GatherArgs {
  const int32_t* nodes;     // N_b
  int n;
  const int32_t* slot_of;   // [N], -1 = not cached
  const uint8_t* local_base;
  int64_t local_stride;
  const uint8_t* cache_base;
  int64_t cache_stride;
  uint8_t* out;             // X_b, row pitch = rb
  int rb;
  OwnerRanges R;
  int32_t* miss_tmp_pos;    // [tiles*kRows] tile-local compacted misses
  int32_t* miss_tmp_id;
  int32_t* tile_miss;       // [tiles]
  int32_t* counters;        // [2 + P]: hit_local, hit_cache, miss[m]  (accumulated)
  int32_t* n_miss_zero;     // when non-null: block 0 stores 0 there (no miss pass will run)
};

template <int VEC>
__global__ void __launch_bounds__(kThreads) k_gather(GatherArgs A) {
  __shared__ const uint8_t* s_src[kRows];
  __shared__ int32_t s_cnt[2 + GG_MAX_PARTS];
  __shared__ int32_t s_w0miss;
  const int t = blockIdx.x;
  const int r0 = t * kRows;
  const int rows = min(kRows, A.n - r0);
  if (threadIdx.x < 2 + GG_MAX_PARTS) s_cnt[threadIdx.x] = 0;
  if (A.n_miss_zero && t == 0 && threadIdx.x == 0) *A.n_miss_zero = 0;
  __syncthreads();
  if (threadIdx.x < kRows) {
    const int r = threadIdx.x;
    const uint8_t* src = nullptr;
    bool miss = false;
    int32_t u = 0;
    int m = 0;
    if (r < rows) {
      u = __ldg(A.nodes + r0 + r);
      m = owner_of(A.R, u);
      if (m == A.R.local) {
        src = A.local_base + (u - A.R.lo[m]) * A.local_stride;
      } else {
        const int32_t s = __ldg(A.slot_of + u);
        if (s >= 0) src = A.cache_base + (int64_t)s * A.cache_stride;
        else miss = true;
      }
    }
    s_src[r] = src;
    // per-warp counts and ordered miss compaction
    const unsigned act = __ballot_sync(0xffffffffu, r < rows);
    const unsigned ml = __ballot_sync(0xffffffffu, r < rows && m == A.R.local);
    const unsigned mm = __ballot_sync(0xffffffffu, miss);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) {
      atomicAdd(&s_cnt[0], __popc(ml));
      atomicAdd(&s_cnt[1], __popc(act) - __popc(ml) - __popc(mm));
      if (wid == 0) s_w0miss = __popc(mm);
    }
    if (miss) atomicAdd(&s_cnt[2 + m], 1);
    __syncwarp();
    // kRows = 64 -> two warps; warp 1's misses follow warp 0's
    asm volatile("bar.sync 1, 64;");
    if (miss && A.miss_tmp_pos) {
      const int q = (wid ? s_w0miss : 0) + __popc(mm & lanemask_lt());
      A.miss_tmp_pos[(int64_t)t * kRows + q] = r0 + r;
      A.miss_tmp_id[(int64_t)t * kRows + q] = u;
    }
    if (threadIdx.x == 32 && A.tile_miss) A.tile_miss[t] = s_w0miss + __popc(mm);
  }
  __syncthreads();
  copy_tile<VEC, true>(s_src, nullptr, A.out + (int64_t)r0 * A.rb, rows, A.rb);
  if (threadIdx.x < 2 + A.R.P && s_cnt[threadIdx.x]) atomicAdd(A.counters + threadIdx.x, s_cnt[threadIdx.x]);
}

// Ordered concatenation of the tile-local miss lists, in two steps: one CTA turns the per-tile counts
// into exclusive offsets in place (tiles <= ~20k; also the total = n_miss), then one warp per tile copies
// that tile's <= 64 entries to their final places with coalesced reads and writes.  (Until round 3 a
// single CTA did both, each thread walking its own tile's list: ~28 strided loads and stores per
// thread and iteration, a sixth of a budgeted batch's miss path: 327.9 -> 271.7 ms per products epoch.)
__global__ void __launch_bounds__(1024)
k_miss_scan(int32_t* __restrict__ tile_miss, int tiles, int32_t* __restrict__ n_miss,
            unsigned long long* __restrict__ miss_total) {
  __shared__ int32_t sm[33];
  __shared__ int32_t carry_s;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  for (int base = 0; base < tiles; base += blockDim.x) {
    const int t = base + threadIdx.x;
    const int32_t c = t < tiles ? tile_miss[t] : 0;
    int32_t tot;
    const int32_t ex = block_exclusive_scan<int32_t>(c, sm, &tot);
    const int32_t carry = carry_s;
    if (t < tiles) tile_miss[t] = carry + ex;
    __syncthreads();
    if (threadIdx.x == 0) carry_s = carry + tot;
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    *n_miss = carry_s;
    if (miss_total && carry_s) atomicAdd(miss_total, (unsigned long long)carry_s);   // rows of a-8, for gg_profile_get
  }
}

__global__ void __launch_bounds__(256)
k_miss_emit(const int32_t* __restrict__ tile_off, int tiles, const int32_t* __restrict__ n_miss,
            const int32_t* __restrict__ tmp_pos, const int32_t* __restrict__ tmp_id,
            int32_t* __restrict__ miss_pos, int32_t* __restrict__ miss_id) {
  const int lane = threadIdx.x & 31;
  for (int t = blockIdx.x * 8 + (threadIdx.x >> 5); t < tiles; t += gridDim.x * 8) {
    const int32_t o = tile_off[t];
    const int32_t c = (t + 1 < tiles ? tile_off[t + 1] : *n_miss) - o;
    for (int q = lane; q < c; q += 32) {
      miss_pos[o + q] = tmp_pos[(int64_t)t * kRows + q];
      miss_id[o + q] = tmp_id[(int64_t)t * kRows + q];
    }
  }
}

struct RowsArgs {
  int n;                     // used when n_dev == nullptr
  const int32_t* n_dev;      // device-side row count (miss fill)
  // source
  const int32_t* src_idx;    // ListResolve: row index into src_base; StoreResolve: global id
  const uint8_t* src_base;
  int64_t src_stride;
  StorePtrs store;           // StoreResolve
  OwnerRanges R;
  // destination
  const int32_t* dst_pos;    // optional scatter positions
  uint8_t* dst_base;
  int64_t dst_row0, dst_stride;
  int rb;
};

// MODE 0 = ListResolve, 1 = StoreResolve.  Persistent-style: tiles are strided over the grid so
// the launch does not need the (device-side) row count.
template <int VEC, int MODE>
__global__ void __launch_bounds__(kThreads) k_rows(RowsArgs A) {
  __shared__ const uint8_t* s_src[kRows];
  __shared__ uint8_t* s_dst[kRows];
  const int n = A.n_dev ? *A.n_dev : A.n;
  const int tiles = (n + kRows - 1) / kRows;
  for (int t = blockIdx.x; t < tiles; t += gridDim.x) {
    const int r0 = t * kRows;
    const int rows = min(kRows, n - r0);
    __syncthreads();
    if (threadIdx.x < kRows) {
      const int r = threadIdx.x;
      const uint8_t* src = nullptr;
      uint8_t* dst = nullptr;
      if (r < rows) {
        const int32_t x = __ldg(A.src_idx + r0 + r);
        if (MODE == 0) {
          src = A.src_base + (int64_t)x * A.src_stride;
        } else {
          const int m = owner_of(A.R, x);
          src = A.store.base[m] + (x - A.R.lo[m]) * A.store.stride;
        }
        const int64_t drow = A.dst_pos ? (int64_t)__ldg(A.dst_pos + r0 + r) : A.dst_row0 + r0 + r;
        dst = A.dst_base + drow * A.dst_stride;
      }
      s_src[r] = src;
      s_dst[r] = dst;
    }
    __syncthreads();
    // rows that come over the host link (MODE 1) keep twice as many loads in flight per thread:
    // a few CTAs then saturate PCIe and the rest of the GPU stays with the sampler
    if (MODE == 1) copy_tile_flat<VEC, 2 * kUnroll>(s_src, s_dst, rows, A.rb);
    else copy_tile<VEC, false>(s_src, s_dst, nullptr, rows, A.rb);
  }
}

static int pick_vec(int rb, const void* a, const void* b, int64_t s1, int64_t s2) {
  auto al = [&](int v) {
    return rb % v == 0 && ((uintptr_t)a % v) == 0 && ((uintptr_t)b % v) == 0 && s1 % v == 0 && s2 % v == 0;
  };
  return al(16) ? 16 : (al(8) ? 8 : 4);
}

void launch_gather(cudaStream_t st, const GatherLaunch& G) {
  if (G.n <= 0) return;
  GatherArgs A;
  A.nodes = G.nodes; A.n = G.n; A.slot_of = G.slot_of;
  A.local_base = G.local_base; A.local_stride = G.local_stride;
  A.cache_base = G.cache_base; A.cache_stride = G.cache_stride;
  A.out = G.out; A.rb = G.rb; A.R = G.R;
  A.miss_tmp_pos = G.miss_tmp_pos; A.miss_tmp_id = G.miss_tmp_id; A.tile_miss = G.tile_miss;
  A.counters = G.counters;
  A.n_miss_zero = G.may_miss ? nullptr : G.n_miss;
  const int tiles = (G.n + kRows - 1) / kRows;
  int vec = pick_vec(G.rb, G.local_base, G.cache_base, G.local_stride, G.cache_stride);
  if ((uintptr_t)G.out % vec) vec = ((uintptr_t)G.out % 8 == 0 && vec >= 8) ? 8 : 4;
  // (a cp.async.bulk variant -- one bulk copy per row into shared memory, one bulk store per tile -- was
  // built and measured in round 2: equal alone, slower beside the sampler; DESIGN.md Sec. 6 keeps the numbers)
  if (vec == 16) k_gather<16><<<tiles, kThreads, 0, st>>>(A);
  else if (vec == 8) k_gather<8><<<tiles, kThreads, 0, st>>>(A);
  else k_gather<4><<<tiles, kThreads, 0, st>>>(A);
  count_launches(1);
}

void launch_miss_path(cudaStream_t st, const GatherLaunch& G) {
  if (G.n <= 0 || !G.may_miss) return;
  const int tiles = (G.n + kRows - 1) / kRows;
  count_launches(3);
  k_miss_scan<<<1, 1024, 0, st>>>(G.tile_miss, tiles, G.n_miss, G.miss_total);
  int eg = (tiles + 7) / 8;
  if (eg > sm_count() * 4) eg = sm_count() * 4;
  k_miss_emit<<<eg, 256, 0, st>>>(G.tile_miss, tiles, G.n_miss, G.miss_tmp_pos, G.miss_tmp_id, G.miss_pos, G.miss_id);
  // a-8: fill the missed rows straight from the owners' pinned stores (zero-copy reads)
  RowsArgs Rw = {};
  Rw.n = 0; Rw.n_dev = G.n_miss; Rw.src_idx = G.miss_id; Rw.store = G.store; Rw.R = G.R;
  Rw.dst_pos = G.miss_pos; Rw.dst_base = G.out; Rw.dst_row0 = 0; Rw.dst_stride = G.rb; Rw.rb = G.rb;
  int v2 = 4;
  {
    bool ok16 = G.rb % 16 == 0 && (uintptr_t)G.out % 16 == 0 && G.store.stride % 16 == 0;
    bool ok8 = G.rb % 8 == 0 && (uintptr_t)G.out % 8 == 0 && G.store.stride % 8 == 0;
    for (int m = 0; m < G.R.P; ++m) {
      ok16 = ok16 && (uintptr_t)G.store.base[m] % 16 == 0;
      ok8 = ok8 && (uintptr_t)G.store.base[m] % 8 == 0;
    }
    v2 = ok16 ? 16 : (ok8 ? 8 : 4);
  }
  // Misses that cross the host link: like the pull kernel below, a dozen CTAs with 8 loads in flight per
  // thread keep PCIe full (the fill alone: 45 GB/s = 0.80 of the pinned-copy peak; the miss path took
  // the same 325-330 ms per epoch at 12 / 24 / 48 / 148 / 592 CTAs: products, n_hot = 10 %, W=16), while a GPU-wide grid of readers crowds the bulk copies' DMA off the link (copies at
  // 0.66 / 0.50 / 0.40 / 0.32 / 0.34 of the link peak) and the sampler off the SMs.
  constexpr int kMissLinkCtas = 12;
  const int grid = G.miss_over_link ? kMissLinkCtas : sm_count() * 4;
  if (v2 == 16) k_rows<16, 1><<<grid, kThreads, 0, st>>>(Rw);
  else if (v2 == 8) k_rows<8, 1><<<grid, kThreads, 0, st>>>(Rw);
  else k_rows<4, 1><<<grid, kThreads, 0, st>>>(Rw);
}

void launch_rows_from_list(cudaStream_t st, const int32_t* src_idx, int n, const uint8_t* src_base,
                           int64_t src_stride, uint8_t* dst_base, int64_t dst_row0, int64_t dst_stride,
                           int rb) {
  if (n <= 0) return;
  RowsArgs A = {};
  A.n = n; A.src_idx = src_idx; A.src_base = src_base; A.src_stride = src_stride;
  A.dst_base = dst_base; A.dst_row0 = dst_row0; A.dst_stride = dst_stride; A.rb = rb;
  const int vec = pick_vec(rb, src_base, dst_base, src_stride, dst_stride);
  int grid = (n + kRows - 1) / kRows;
  if (grid > sm_count() * 8) grid = sm_count() * 8;
  if (vec == 16) k_rows<16, 0><<<grid, kThreads, 0, st>>>(A);
  else if (vec == 8) k_rows<8, 0><<<grid, kThreads, 0, st>>>(A);
  else k_rows<4, 0><<<grid, kThreads, 0, st>>>(A);
  count_launches(1);
}

void launch_rows_from_store(cudaStream_t st, const int32_t* ids, int n, const StorePtrs& store,
                            const OwnerRanges& R, uint8_t* dst_base, int64_t dst_row0,
                            int64_t dst_stride, int rb, bool over_link) {
  if (n <= 0) return;
  RowsArgs A = {};
  A.n = n; A.src_idx = ids; A.store = store; A.R = R;
  A.dst_base = dst_base; A.dst_row0 = dst_row0; A.dst_stride = dst_stride; A.rb = rb;
  bool ok16 = rb % 16 == 0 && (uintptr_t)dst_base % 16 == 0 && dst_stride % 16 == 0 && store.stride % 16 == 0;
  bool ok8 = rb % 8 == 0 && (uintptr_t)dst_base % 8 == 0 && dst_stride % 8 == 0 && store.stride % 8 == 0;
  for (int m = 0; m < R.P; ++m) {
    ok16 = ok16 && (uintptr_t)store.base[m] % 16 == 0;
    ok8 = ok8 && (uintptr_t)store.base[m] % 8 == 0;
  }
  int grid = (n + kRows - 1) / kRows;
  // Rows cross the host link here: 12 CTAs with 8 16-byte loads in flight per thread already
  // saturate PCIe (41 GB/s); a wider grid only takes SMs and memory-system queue slots away from
  // the sampler (measured, products W=16: 12 / 16 / 24 / 32 / 1184 CTAs -> 3903 / 3657 / 3340 /
  // 3184 / 2607 mini-batches/s).
  constexpr int kPullCtas = 12;
  if (over_link) grid = grid > kPullCtas ? kPullCtas : grid;
  else if (grid > sm_count() * 8) grid = sm_count() * 8;
  if (ok16) k_rows<16, 1><<<grid, kThreads, 0, st>>>(A);
  else if (ok8) k_rows<8, 1><<<grid, kThreads, 0, st>>>(A);
  else k_rows<4, 1><<<grid, kThreads, 0, st>>>(A);
  count_launches(1);
}

}  // namespace gg

// a-1: neighbor sampling for one hop of a whole window (all W batches in one launch set).
//
// Keep rule (include/greengnn.h; readings S3-S5): for destination v with CSR row of
// `deg` entries, keep every position if deg <= f, else the f positions j with the smallest
// (key(j), j), key(j) = fmix(h_dst + (j+1)*gamma); kept neighbors are emitted in ascending
// edge position.  The key depends on (seed, batch, layer, dst, j) only -- never on the
// neighbor id -- so the adjacency row is not read to select; only the <= f chosen entries are.
//
// Launches per hop (the rows of a power-law frontier differ in cost by 1000x, so the KEY SPACE,
// not the row list, is what gets divided among the lanes):
//   k_sample_count   one thread per destination: c = min(deg, f) -> cnt_tmp, per-tile sums,
//                    histogram of the keyed rows (deg > f) over quarter-octave degree bins
//   k_tile_scan      one CTA per batch: exclusive scan of that batch's tile sums, batch total;
//                    CTA 0 also turns the histogram into bin regions (largest degrees first) and
//                    into the chunk numbering below
//   k_sample_plan    one CTA per tile of 256 destinations: in-tile scan -> block indptr and the
//                    FINAL output offset of every row (no atomics on output order =>
//                    deterministic); rows with deg <= f are copied; every other row becomes a
//                    work item {h_dst, row start, deg, output offset} in its bin's region
//   k_select_chunk   ONE LANE PER CHUNK of <= 128 consecutive edge positions.  Every row of a bin is
//                    cut into the same number n_b of equal chunks (n_b = ceil(bin's largest degree /
//                    128)), so chunk k of the bin is chunk k % n_b of the bin's row k / n_b -- no chunk
//                    table -- and the 32 lanes of a warp always run loops of nearly the same length,
//                    whatever the degree mix.  A row of degree < 128 is one chunk: its lane ranks its
//                    candidates and emits the row.  A longer row's lanes append their candidates to the
//                    row's list in global memory (one atomic per lane that found any).
//   k_select_rank    one thread per multi-chunk row: ranks the row's ~f+2.5 sqrt(f) candidates,
//                    proves the result (kept == f) and emits it in ascending edge position
//   k_select_warp    ONE WARP PER ROW for the rows the kernels above could not prove exact (and for
//                    every keyed row when fanout > kChunkMaxFanout)
#include "common.cuh"
#include "kernels.h"

namespace gg {

// cumulative sampler statistics: [0] key evaluations the method asks for (sum of deg over rows
// with deg > fanout), [1] such rows, [2] rows that took the exact ballot/bisection path,
// [3] rows the chunk / rank kernels handed to the warp kernel
__device__ unsigned long long g_sampler_stat[4];
// test knobs (gg_debug_sampler): compare only the top 32-shift bits when ranking (forces
// high-word ties), and add to the candidate target (forces list overflow / too few candidates)
__constant__ int c_rank_shift = 0;
__constant__ float c_want_add = 0.0f;

constexpr int kTile = 256;      // destinations per CTA tile
constexpr int kCand = 256;      // candidate buffer per warp
constexpr int kWarps = 8;
constexpr int kBins = 128;      // quarter-octave degree bins: bin = 4*floor(log2 deg) + next two bits
constexpr int kChunk = 128;     // edge positions per chunk (at most)
// tunables (gg_sampler_tune; passed to the kernels of a hop): rows in bins below single_bins are one
// chunk each, whatever their degree; rows in bins >= warp_bin go to the warp kernel.  Defaults (bin 36 =
// degree 512): one lane per row below degree 512, one warp per row above; cutting the rows of
// degree 128..4095 into chunks with the candidates merged through global memory measured slower
// (products W=16, sampling per epoch alone: 16.5 ms at 36/36 vs 18.8-20.8 ms for 28/48, 36/48,
// 28/128), so the multi-chunk path is off by default.
static int h_single_bins = 36, h_warp_bin = 36, h_hub_bin = 128;   // hub chunking off: see gg_sampler_tune
constexpr int kSmallHopRows = 1 << 16;   // destinations of a hop below which the lane kernel stops at ...
constexpr int kSmallHopBins = 28;        // ... bin 28 = degree 128
constexpr int kChunkMaxFanout = 25;   // candidate lists of the chunk path hold <= 64 entries

// device-side plan of one hop (zeroed before k_sample_count)
struct SamplePlan {
  int32_t bin_count[kBins];    // keyed rows per bin (k_sample_count)
  int32_t bin_start[kBins];    // first item of the bin's region, bins in DESCENDING degree order
  int32_t bin_cursor[kBins];   // items already placed (k_sample_plan)
  unsigned long long bin_chunk0[kBins + 1];  // [o]: first chunk of the o-th bin in descending order
                                             // (bin kBins-1-o), each bin padded to a multiple of 32
  unsigned long long n_chunks;      // = bin_chunk0[kBins]
  unsigned long long chunk_cursor;  // dynamic queue of the chunk kernel (units of 32 chunks)
  int32_t n_items;             // keyed rows
  int32_t n_hub;               // items [0, n_hub): bins >= hub_bin, cut into chunks (a hub row would hold one warp for milliseconds)
  int32_t n_warp_items;        // items [n_hub, n_warp_items) belong to the warp kernel (warp_bin <= bin < hub_bin; fanout > kChunkMaxFanout: all)
  int32_t n_multi;             // items [n_warp_items, n_multi) are multi-chunk rows (single_bins <= bin < warp_bin)
  int32_t n_fallback;          // rows handed over to the warp kernel
  int32_t warp_cursor;         // dynamic queue of the warp kernel
};

__host__ __device__ __forceinline__ int deg_bin(uint32_t deg) {   // deg >= 2; monotone in deg
#ifdef __CUDA_ARCH__
  const int l = 31 - __clz(deg);
#else
  int l = 0;
  while ((deg >> (l + 1)) != 0) ++l;
#endif
  return l >= 2 ? 4 * l + (int)((deg >> (l - 2)) & 3u) : 4 + (int)((deg << 1) & 3u);
}
// chunks per row of a bin: 1 below degree kChunk, else ceil(largest degree of the bin / kChunk)
__host__ __device__ __forceinline__ uint32_t bin_chunks(int bin, int single_bins) {
  if (bin < single_bins) return 1u;
  const int l = bin >> 2, k = bin & 3;
  return ((uint32_t)(5 + k) << (l - 2)) + (kChunk - 2) >> 7;   // largest degree = ((5+k) << (l-2)) - 1
}
static_assert(kChunk == 128, "bin_chunks shifts by log2(kChunk) = 7");

__global__ void __launch_bounds__(kTile)
k_sample_count(const int64_t* __restrict__ indptr, const int32_t* __restrict__ nodes,
               int64_t node_pitch, BatchOffsets n_dst, int fanout, int max_tiles,
               uint8_t* __restrict__ cnt_tmp, int64_t cnt_pitch, int32_t* __restrict__ tile_sums,
               SamplePlan* __restrict__ plan) {
  __shared__ int32_t sm[33];
  __shared__ int32_t s_bin[kBins];
  __shared__ unsigned long long s_keys;
  const int b = blockIdx.y, t = blockIdx.x;
  const int nd = n_dst.v[b];
  if (t * kTile >= nd) return;
  if (threadIdx.x < kBins) s_bin[threadIdx.x] = 0;
  if (threadIdx.x == 0) s_keys = 0;
  __syncthreads();
  const int i = t * kTile + threadIdx.x;
  int c = 0;
  unsigned long long keys = 0;
  if (i < nd) {
    const int32_t v = nodes[b * node_pitch + i];
    const int64_t r0 = __ldg(indptr + v), r1 = __ldg(indptr + v + 1);
    const int64_t deg = r1 - r0;
    c = deg < fanout ? (int)deg : fanout;
    cnt_tmp[b * cnt_pitch + i] = (uint8_t)c;
    if (deg > fanout) {
      keys = (unsigned long long)deg;
      atomicAdd(&s_bin[deg_bin((uint32_t)deg)], 1);
    }
  }
#pragma unroll
  for (int o = 16; o; o >>= 1) keys += __shfl_xor_sync(0xffffffffu, keys, o);
  if ((threadIdx.x & 31) == 0 && keys) atomicAdd(&s_keys, keys);
  int32_t total;
  block_exclusive_scan<int32_t>(c, sm, &total);   // contains __syncthreads
  if (threadIdx.x == 0) tile_sums[b * max_tiles + t] = total;
  int rows = 0;
  if (threadIdx.x < kBins) {
    rows = s_bin[threadIdx.x];
    if (rows) atomicAdd(&plan->bin_count[threadIdx.x], rows);
  }
  if (threadIdx.x < kBins) {
#pragma unroll
    for (int o = 16; o; o >>= 1) rows += __shfl_xor_sync(0xffffffffu, rows, o);
    if ((threadIdx.x & 31) == 0 && rows) atomicAdd(&g_sampler_stat[1], (unsigned long long)rows);
  }
  if (threadIdx.x == 0 && s_keys) atomicAdd(&g_sampler_stat[0], s_keys);
}

// One CTA per batch (row): in-place exclusive scan of row[0..n_tiles[b]) ; totals[b] = sum.
__global__ void __launch_bounds__(1024)
k_tile_scan(int32_t* __restrict__ tiles, int row_pitch, BatchOffsets n_items, int items_per_tile,
            int32_t* __restrict__ totals, SamplePlan* __restrict__ plan, int single_bins, int warp_bin, int hub_bin) {
  __shared__ int32_t sm[33];
  __shared__ int32_t carry_s;
  const int b = blockIdx.x;
  const int n = (n_items.v[b] + items_per_tile - 1) / items_per_tile;
  int32_t* row = tiles + (int64_t)b * row_pitch;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  for (int base = 0; base < n; base += blockDim.x) {
    const int i = base + threadIdx.x;
    int32_t v = i < n ? row[i] : 0, tot;
    int32_t ex = block_exclusive_scan<int32_t>(v, sm, &tot);
    const int32_t carry = carry_s;
    if (i < n) row[i] = carry + ex;
    __syncthreads();
    if (threadIdx.x == 0) carry_s = carry + tot;
    __syncthreads();
  }
  if (threadIdx.x == 0) totals[b] = carry_s;
  // bin regions of the hop's work items, largest degrees first, and the chunk numbering: bin b's
  // rows_b * n_b chunks are numbered consecutively (chunk k = chunk k % n_b of row k / n_b), each
  // bin padded to a multiple of 32 so that a warp's 32 chunks never straddle two bins
  if (plan && b == 0) {
    __shared__ int32_t s_cnt[kBins], s_start[kBins];
    __shared__ unsigned long long s_nc[kBins], s_c0[kBins + 1];
    if (threadIdx.x < kBins) {
      const int k = threadIdx.x;
      const int32_t n = plan->bin_count[k];
      s_cnt[k] = n;
      const unsigned long long nc = (k >= warp_bin && k < hub_bin) ? 0ull : (unsigned long long)n * bin_chunks(k, single_bins);
      s_nc[k] = (nc + 31ull) & ~31ull;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      int32_t acc = 0, n_multi = 0, n_warp = 0, n_hub = 0;
      unsigned long long c0 = 0;
      for (int k = kBins - 1; k >= 0; --k) {
        s_start[k] = acc;
        s_c0[kBins - 1 - k] = c0;
        c0 += s_nc[k];
        acc += s_cnt[k];
        if (k == single_bins) n_multi = acc;
        if (k == hub_bin) n_hub = acc;
        if (k == warp_bin) n_warp = acc;
      }
      s_c0[kBins] = c0;
      plan->n_chunks = c0;
      plan->chunk_cursor = 0;
      plan->n_items = acc;
      n_warp = n_warp > n_hub ? n_warp : n_hub;
      plan->n_hub = n_hub;
      plan->n_warp_items = n_warp;
      plan->n_multi = n_multi > n_warp ? n_multi : n_warp;
      plan->n_fallback = 0;
      plan->warp_cursor = 0;
    }
    __syncthreads();
    if (threadIdx.x < kBins) {
      plan->bin_start[threadIdx.x] = s_start[threadIdx.x];
      plan->bin_cursor[threadIdx.x] = 0;
    }
    if (threadIdx.x <= kBins) plan->bin_chunk0[threadIdx.x] = s_c0[threadIdx.x];
  }
}

// ---- the hot loop: one key per lane per step -------------------------------------------------
// The sampler is bound by the integer ALU pipe (LOP3 / SHF / ISETP issue at half the rate of the
// FMA pipe that runs IMAD), so the step below is written to keep ALU-pipe instructions per key low:
//   * the state h + (j+1)*gamma is formed from j with IMAD.WIDE (FMA pipe), not carried adds;
//   * the high-word halves of the two xor-shifts use mul.hi (x >> s == mulhi(x, 2^(32-s)));
//   * the final xor-shift is never formed for the test: with an ODD high-word threshold M,
//     (z_hi ^ (z_hi >> 31)) <= M  <=>  z_hi <= M, because the xor only flips bit 0;
//   * the compaction (popc, smem stores, finishing the key) runs only when some lane passed.
__device__ __forceinline__ uint32_t mulhi_u32(uint32_t a, uint32_t b) {
  uint32_t r;
  asm("mul.hi.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b));  // opaque to the optimiser: stays an IMAD.HI
  return r;
}
__device__ __forceinline__ uint32_t mad_lo_u32(uint32_t a, uint32_t b, uint32_t c) {
  uint32_t r;
  asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
  return r;
}
__device__ __forceinline__ uint64_t key_z(uint64_t hdst, uint32_t j) {
  uint64_t x = hdst + (uint64_t)(j + 1u) * kGamma;
  uint32_t lo = (uint32_t)x, hi = (uint32_t)(x >> 32);
  lo ^= __funnelshift_r(lo, hi, 30);
  hi ^= mulhi_u32(hi, 1u << 2);
  uint64_t z = (((uint64_t)hi << 32) | lo) * 0xBF58476D1CE4E5B9ull;
  lo = (uint32_t)z;
  hi = (uint32_t)(z >> 32);
  lo ^= __funnelshift_r(lo, hi, 27);
  hi ^= mulhi_u32(hi, 1u << 5);
  return (((uint64_t)hi << 32) | lo) * 0x94D049BB133111EBull;  // key = z ^ (z >> 31)
}

// FULL = exact 64-bit test (only when the bisection can no longer separate on high words).
template <bool FULL, bool CHECK>
__device__ __forceinline__ void select_step(uint64_t hdst, uint32_t j, uint32_t deg, uint64_t T,
                                            uint32_t Modd, int& cnt, uint64_t* s_key, int32_t* s_pos) {
  const uint64_t z = key_z(hdst, j);
  bool p;
  if (FULL) p = (z ^ (z >> 31)) <= T;
  else p = (uint32_t)(z >> 32) <= Modd;
  if (CHECK) p = p && (j < deg);
  const unsigned m = __ballot_sync(0xffffffffu, p);
  if (m) {
    if (p) {
      const int q = cnt + __popc(m & lanemask_lt());
      if (q < kCand) {
        s_key[q] = z ^ (z >> 31);
        s_pos[q] = (int32_t)j;
      }
    }
    cnt += __popc(m);
  }
}

template <bool FULL>
__device__ __forceinline__ int select_pass(uint64_t hdst, uint32_t deg, uint64_t T,
                                           uint64_t* s_key, int32_t* s_pos) {
  const uint32_t lane = threadIdx.x & 31;
  const uint32_t Modd = (uint32_t)(T >> 32) | 1u;
  int cnt = 0;
  uint32_t j = lane;
  const uint32_t full_end = deg & ~63u;
  // two independent key chains per lane per iteration; no bound check inside whole 64-key chunks
  for (; j < full_end; j += 64) {
    select_step<FULL, false>(hdst, j, deg, T, Modd, cnt, s_key, s_pos);
    select_step<FULL, false>(hdst, j + 32, deg, T, Modd, cnt, s_key, s_pos);
  }
  if (full_end < deg) {
    select_step<FULL, true>(hdst, j, deg, T, Modd, cnt, s_key, s_pos);
    select_step<FULL, true>(hdst, j + 32, deg, T, Modd, cnt, s_key, s_pos);
  }
  return cnt;
}

// Exact top-f of `deg` keyed positions by one warp.  Writes the kept positions' neighbor ids,
// ascending in position, to out[0..f).
__device__ __forceinline__ void warp_select(const int32_t* __restrict__ row, int64_t deg64, int f,
                                            uint64_t hdst, uint64_t* s_key, int32_t* s_pos,
                                            int32_t* __restrict__ out) {
  const int lane = threadIdx.x & 31;
  const uint32_t deg = (uint32_t)deg64;
  // candidates wanted: f plus a slack so that a Binomial(deg, want/deg) count falls below f
  // with probability ~3e-4 (a miss only costs one more pass)
  const int want = f + 6 + (int)(4.0f * sqrtf((float)f));
  int cnt;
  if (deg <= (uint32_t)want) {
    // small row: every position is a candidate
    cnt = (int)deg;
    for (int j = lane; j < cnt; j += 32) {
      s_key[j] = key_edge(hdst, (uint64_t)j);
      s_pos[j] = j;
    }
  } else {
    // threshold guess: keys are uniform, so the f-th smallest is near f/deg * 2^64.  The
    // threshold only prunes; the exact rank below decides, so its rounding is immaterial.
    uint64_t T = (uint64_t)((float)want / (float)deg * 18446744073709551616.0f);
    T |= 0x1ffffffffull;  // the test uses the high word made odd: keep T equal to what is tested
    uint64_t lo = 0, hi = ~0ull;  // count(lo) < f known; count(hi) > kCand known once have_hi
    bool have_hi = false, full = false;
    for (;;) {
      cnt = full ? select_pass<true>(hdst, deg, T, s_key, s_pos)
                 : select_pass<false>(hdst, deg, T, s_key, s_pos);
      if (cnt >= f && cnt <= kCand) break;
      if (cnt < f) {
        lo = T;
        T = have_hi ? lo + ((hi - lo) >> 1) : (T > (~0ull >> 1) ? ~0ull : T * 2 + 1);
      } else {
        hi = T;
        have_hi = true;
        T = lo + ((hi - lo) >> 1);
      }
      if (have_hi && (hi >> 32) - (lo >> 32) <= 2) full = true;  // odd high words can no longer separate
      if (!full) T |= 0x1ffffffffull;
    }
  }
  __syncwarp();
  // exact rank among candidates under (key, position); candidates are in ascending position
  typedef unsigned __int128 u128;
  int emitted = 0;
  for (int i0 = 0; i0 < cnt; i0 += 32) {
    const int i = i0 + lane;
    bool keep = false;
    int32_t pos = 0;
    if (i < cnt) {
      pos = s_pos[i];
      const u128 mine = ((u128)s_key[i] << 32) | (uint32_t)pos;
      int rank = 0;
      for (int c = 0; c < cnt; ++c) rank += ((((u128)s_key[c]) << 32) | (uint32_t)s_pos[c]) < mine;
      keep = rank < f;
    }
    const unsigned m = __ballot_sync(0xffffffffu, keep);
    if (keep) out[emitted + __popc(m & lanemask_lt())] = __ldg(row + pos);
    emitted += __popc(m);
  }
  __syncwarp();
}

// ---- fast path: lane-local candidate lists, high-word ranking ---------------------------------
// ncu (profiles/r01_b_pipeline.md) showed the ballot-compacted loop above spending half of its
// issue slots outside the hash (vote, branch, popc, 96-bit ranking of ~40 candidates).  The fast
// path removes every warp-synchronous operation from the key loop:
//   * lane l owns the CONTIGUOUS positions [l*K, (l+1)*K), K = deg/32 (the deg%32 tail positions
//     are handled once at the end), so "lane-major" order is ascending edge position;
//   * a position passes when the HIGH word of its pre-xorshift key z is <= an odd threshold M
//     (same test as above); a passing lane appends (z_hi, x_lo) to its OWN list in shared memory
//     with two predicated stores and one predicated add -- no ballot, no branch.  x_lo is the
//     low word of the SplitMix state, already in a register; the position is recovered from it
//     as (x_lo - h_lo) * gamma_lo^-1 - 1 (mod 2^32);
//   * the <= 128 candidates are compacted lane-major (= ascending position) and ranked on the
//     high 32 bits of the key only: keep i iff #{c : hi_c < hi_i} < f.  That set always CONTAINS
//     the true top-f under (key, position) and equals it iff it has exactly f members (a tie in
//     the high word at the boundary is the only way to get more), so `kept == f` proves exactness
//     and anything else -- a lane list overflow, fewer than f candidates, more than 128, a
//     boundary tie -- falls back to warp_select above, which is exact by construction.
constexpr int kLaneCap = 12;                  // candidate slots per lane
constexpr int kFastCand = 128;                // compacted candidates
constexpr int kScratchWords = 1024;           // per-warp scratch, 4 KB
constexpr uint32_t kGammaLo = 0x7F4A7C15u, kGammaLoInv = 0x9937733Du;  // kGammaLo * kGammaLoInv == 1 (mod 2^32)
constexpr uint32_t kC1lo = 0x1CE4E5B9u, kC1hi = 0xBF58476Du, kC2lo = 0x133111EBu, kC2hi = 0x94D049BBu;

// high word of z = fmix's value before the last xor-shift, from the state x = {xhi, xlo}
__device__ __forceinline__ uint32_t key_zhi(uint32_t xlo, uint32_t xhi) {
  // measured on B200 (warp instructions per clock per sub-partition): IMAD 0.49, SHF / LOP3 / IADD3
  // 0.5, IMAD.HI and IMAD.WIDE 0.25 -- so the high-half shifts are plain shifts (round 1 used
  // mul.hi for them to unload the ALU pipe: 4 clocks each on the FMA pipe instead of 2 on the ALU pipe)
  uint32_t lo = xlo ^ __funnelshift_r(xlo, xhi, 30);
  uint32_t hi = xhi ^ (xhi >> 30);
  // {hi,lo} * C1 (low 64 bits): the cross terms accumulate straight onto the high half of the
  // wide product
  const uint64_t p = (uint64_t)lo * kC1lo;
  hi = mad_lo_u32(lo, kC1hi, mad_lo_u32(hi, kC1lo, (uint32_t)(p >> 32)));
  lo = (uint32_t)p;
  lo ^= __funnelshift_r(lo, hi, 27);
  hi ^= hi >> 27;
  return mulhi_u32(lo, kC2lo) + hi * kC2lo + lo * kC2hi;
}
__device__ __forceinline__ void sts_u32(uint32_t addr, uint32_t v) {
  asm volatile("st.shared.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ uint32_t lds_u32(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ void sts_v2(uint32_t addr, uint32_t a, uint32_t b) {
  asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(addr), "r"(a), "r"(b) : "memory");
}
// entry s of lane l: {z_hi, x_lo} at s*256 + l*8 -- one predicated 64-bit store, conflict-free
__device__ __forceinline__ void fast_step(uint64_t x, uint32_t M, uint32_t& a) {
  const uint32_t xlo = (uint32_t)x;
  const uint32_t z = key_zhi(xlo, (uint32_t)(x >> 32));
  if (z <= M) {
    sts_v2(a, z, xlo);
    a += 256;
  }
}

// Returns true when out[0..f) holds the exact result; false = caller must run warp_select.
__device__ __forceinline__ float want_candidates(int f) {
  return fmaxf((float)f + 2.0f + 2.5f * sqrtf((float)f) + c_want_add, 1.0f);
}
__device__ __forceinline__ bool warp_select_fast(const int32_t* __restrict__ row, uint32_t deg, int f,
                                                 float wantf, uint64_t hdst, uint32_t* scratch,
                                                 int32_t* __restrict__ out) {
  const uint32_t lane = threadIdx.x & 31;
  uint32_t* c_hi = scratch + 2 * kLaneCap * 32;   // [kFastCand]
  uint32_t* c_pos = c_hi + kFastCand;             // [kFastCand]
  const int rshift = c_rank_shift;
  int total;
  if ((float)deg <= wantf && deg <= (uint32_t)kFastCand) {
    // small row: every position is a candidate, already in position order
    total = (int)deg;
    for (uint32_t j = lane; j < deg; j += 32) {
      const uint64_t x = hdst + (uint64_t)(j + 1u) * kGamma;
      const uint32_t z = key_zhi((uint32_t)x, (uint32_t)(x >> 32));
      c_hi[j] = (z ^ (z >> 31)) >> rshift;
      c_pos[j] = j;
    }
  } else {
    const uint32_t M = (uint32_t)fminf(__fdividef(wantf, (float)deg) * 4294967296.0f, 4294967040.0f) | 1u;
    const uint32_t K = deg >> 5;
    const uint32_t a0 = (uint32_t)__cvta_generic_to_shared(scratch) + lane * 8;
    uint32_t a = a0;
    const uint32_t a_lim4 = a0 + (kLaneCap - 4) * 256, a_lim1 = a0 + (kLaneCap - 1) * 256;
    uint64_t x = hdst + (uint64_t)(lane * K + 1u) * kGamma;
    uint32_t n4 = K >> 2;
    // The ALU pipe (IADD3 / SHF / LOP3 / ISETP, one warp instruction per 2 clocks) carries half
    // of this loop (43 of 84 instructions per 4 keys) and is its limiter.  Moving the state
    // updates to the FMA pipe (IMAD.WIDE with a 64-bit addend) was tried three ways; ptxas splits
    // the addend back into IADD3 + IMAD.X every time, so the carried adds stay.
    while (n4 != 0 && a <= a_lim4) {
      fast_step(x, M, a);
      fast_step(x + kGamma, M, a);
      fast_step(x + 2 * kGamma, M, a);
      fast_step(x + 3 * kGamma, M, a);
      x += 4 * kGamma;
      --n4;
    }
    uint32_t rem = (K & 3u) + 4u * n4;   // n4 != 0 only when this lane's list is nearly full
    while (rem != 0 && a <= a_lim1) {
      fast_step(x, M, a);
      x += kGamma;
      --rem;
    }
    const bool ovf = rem != 0;
    // tail positions 32K + lane
    const uint32_t jt = (K << 5) + lane;
    uint32_t zt = 0;
    bool pt = false;
    if (jt < deg) {
      const uint64_t xt = hdst + (uint64_t)(jt + 1u) * kGamma;
      zt = key_zhi((uint32_t)xt, (uint32_t)(xt >> 32));
      pt = zt <= M;
    }
    const unsigned tmask = __ballot_sync(0xffffffffu, pt);
    const int c = (int)((a - a0) >> 8);
    const int total_main = __reduce_add_sync(0xffffffffu, c);
    total = total_main + __popc(tmask);
    if (__any_sync(0xffffffffu, ovf) || total < f || total > kFastCand) return false;
    int incl = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int y = __shfl_up_sync(0xffffffffu, incl, o);
      if ((int)lane >= o) incl += y;
    }
    const int off = incl - c;
    const uint32_t hlo = (uint32_t)hdst;
    for (int s = 0; s < c; ++s) {
      const uint32_t z = lds_u32(a0 + s * 256);
      const uint32_t xl = lds_u32(a0 + s * 256 + 4);
      c_hi[off + s] = (z ^ (z >> 31)) >> rshift;
      c_pos[off + s] = (xl - hlo) * kGammaLoInv - 1u;
    }
    if (pt) {
      const int q = total_main + __popc(tmask & lanemask_lt());
      c_hi[q] = (zt ^ (zt >> 31)) >> rshift;
      c_pos[q] = jt;
    }
  }
  if (lane < 4 && total + (int)lane < kFastCand) c_hi[total + lane] = 0xffffffffu;  // pad to a multiple of 4
  __syncwarp();
  const uint4* c_hi4 = reinterpret_cast<const uint4*>(c_hi);
  const int n4 = (total + 3) >> 2;
  int emitted = 0;
  for (int i0 = 0; i0 < total; i0 += 32) {
    const int i = i0 + (int)lane;
    const uint32_t mine = i < total ? c_hi[i] : 0u;
    int rank = 0;
    for (int q = 0; q < n4; ++q) {
      const uint4 v = c_hi4[q];
      rank += (v.x < mine) + (v.y < mine) + (v.z < mine) + (v.w < mine);
    }
    const bool keep = i < total && rank < f;
    const unsigned m = __ballot_sync(0xffffffffu, keep);
    const int q = emitted + __popc(m & lanemask_lt());
    if (keep && q < f) out[q] = __ldg(row + c_pos[i]);
    emitted += __popc(m);
  }
  __syncwarp();
  return emitted == f;
}


__global__ void __launch_bounds__(kTile)
k_sample_plan(const int64_t* __restrict__ indptr, const int32_t* __restrict__ indices,
              const int32_t* __restrict__ nodes, int64_t node_pitch, BatchOffsets n_dst,
              BatchOffsets dst_off, int W, int fanout, int max_tiles,
              const uint64_t* __restrict__ key_prefix_b, const uint8_t* __restrict__ cnt_tmp,
              int64_t cnt_pitch, const int32_t* __restrict__ tile_sums,
              const int32_t* __restrict__ totals, int32_t* __restrict__ blk_indptr,
              int32_t* __restrict__ edge_off_out, int32_t* __restrict__ src_global,
              SamplePlan* __restrict__ plan, SampleItems items, int single_bins) {
  __shared__ int32_t sm[33];
  __shared__ int32_t s_edge_base;
  __shared__ int32_t s_bin[kBins], s_base[kBins];
  const int b = blockIdx.y, t = blockIdx.x;
  const int nd = n_dst.v[b];
  if (t * kTile >= nd) return;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (threadIdx.x < kBins) s_bin[threadIdx.x] = 0;
  // edge offset of this batch = sum of the totals of the batches before it
  if (wid == 0) {
    int32_t s = 0;
    for (int k = lane; k < b; k += 32) s += totals[k];
#pragma unroll
    for (int o = 16; o; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) {
      s_edge_base = s;
      if (t == 0) {
        edge_off_out[b] = s;
        if (b == W - 1) edge_off_out[W] = s + totals[b];
      }
    }
  }
  const int i = t * kTile + threadIdx.x;
  const int c = i < nd ? cnt_tmp[b * cnt_pitch + i] : 0;
  int32_t tot;
  const int32_t ex = block_exclusive_scan<int32_t>(c, sm, &tot);   // contains __syncthreads
  const int32_t tile_base = tile_sums[b * max_tiles + t];
  // block indptr (0-based inside the batch's block); batch b's row starts at dst_off[b] + b
  int32_t* ip = blk_indptr + dst_off.v[b] + b;
  if (i < nd) ip[i] = tile_base + ex;
  if (i == nd - 1) ip[nd] = tile_base + ex + c;
  const int32_t out = s_edge_base + tile_base + ex;
  int bin = -1, rank = 0;
  int64_t r0 = 0;
  uint32_t deg = 0;
  uint64_t hdst = 0;
  if (i < nd) {
    const int32_t v = nodes[b * node_pitch + i];
    r0 = __ldg(indptr + v);
    const int64_t d64 = __ldg(indptr + v + 1) - r0;
    deg = (uint32_t)d64;
    if (d64 <= fanout) {
      for (int j = 0; j < (int)deg; ++j) src_global[out + j] = __ldg(indices + r0 + j);
    } else {
      hdst = key_hdst(key_prefix_b[b], (uint64_t)(uint32_t)v);
      bin = deg_bin(deg);
      rank = atomicAdd(&s_bin[bin], 1);
    }
  }
  __syncthreads();
  if (threadIdx.x < kBins) {
    const int n = s_bin[threadIdx.x];
    s_base[threadIdx.x] = n ? plan->bin_start[threadIdx.x] + atomicAdd(&plan->bin_cursor[threadIdx.x], n) : 0;
  }
  __syncthreads();
  if (bin >= 0) {
    const int q = s_base[bin] + rank;
    items.hdst[q] = hdst;
    items.row0[q] = r0;
    items.deg[q] = deg;
    items.out[q] = out;
    if (bin >= single_bins) items.row_cnt[q] = 0;   // candidates the chunk kernel will append
  }
}

// ---- one lane per chunk ---------------------------------------------------------------------------
// The lane walks its chunk's positions in ascending order; a position whose z_hi passes the row's
// odd threshold M appends {z_hi, low word of the SplitMix state} to the lane's own list in shared
// memory with ONE predicated 64-bit store (entry s of thread t at s*1024 + t*8: conflict-free) and
// one predicated add -- no ballot, no branch in the loop.  The position comes back from the state's
// low word: (x - h) * gamma^-1 - 1 (mod 2^32).
//   single-chunk row (degree < 128): the lane ranks its c candidates on the high key word (the
//     fanout-th smallest DISTINCT value, one round per rank), keeps those at or below it, and
//     `kept == fanout` proves the result (DESIGN.md Sec. 6 (iv)); it then emits the row;
//   longer row: the lane reserves c slots of the row's candidate list in global memory with one
//     atomicAdd and writes {z_hi, position}; k_select_rank finishes the row.
// Anything that cannot be proved (list overflow, too few candidates, a high-word tie at the
// boundary) goes to the warp kernel's fallback list.
constexpr int kCThreads = 128;
constexpr uint32_t kCSlot = kCThreads * 8;   // bytes per list entry across the CTA

__device__ __forceinline__ void chunk_step(uint64_t x, uint32_t M, uint32_t& a) {
  const uint32_t xlo = (uint32_t)x;
  const uint32_t z = key_zhi(xlo, (uint32_t)(x >> 32));
  if (z <= M) {
    sts_v2(a, z, xlo);
    a += kCSlot;
  }
}
// candidate list capacity (per lane in shared memory, per row in global memory): the target count
// plus 3.5 sigma of a Poisson count, a multiple of 4, at most 64 (keep flags are one 64-bit word)
__host__ __device__ __forceinline__ int cand_cap(int fanout) {
  const float want = (float)fanout + 2.0f + 2.5f * sqrtf((float)fanout);
  const int cap = ((int)ceilf(want + 3.5f * sqrtf(want)) + 3) & ~3;
  return cap > 64 ? 64 : cap;
}
__device__ __forceinline__ uint32_t row_threshold(float wantf, uint32_t deg) {
  const float fdeg = (float)deg;
  return fdeg <= wantf ? 0xffffffffu
                       : ((uint32_t)fminf(__fdividef(wantf, fdeg) * 4294967296.0f, 4294967040.0f) | 1u);
}

// Ranks the c candidates of the calling thread's list (entry s: key word at a0 + s*kCSlot, already
// final and shifted) and returns the keep flags; *kept = their count.  c <= 64, c >= fanout.
__device__ __forceinline__ unsigned long long rank_list(uint32_t a0, int c, int fanout, int* kept) {
  const int c4 = (c + 3) & ~3;
  for (int s = c; s < c4; ++s) sts_u32(a0 + s * kCSlot, 0xffffffffu);   // the list holds c4 <= cap entries
  // the fanout-th smallest DISTINCT value, one round per rank: each round takes the minimum of
  // (v - last - 1) mod 2^32, which orders the values above `last` before everything else.  With
  // fewer than `fanout` distinct values the rounds wrap around to the small ones again; that needs
  // no care: whatever thr comes out, {v <= thr} is a set of smallest values, and it is the top
  // `fanout` exactly when it has `fanout` members, which is the only case the caller accepts.
  uint32_t lastp1 = 0, thr = 0;
  for (int r = 0; r < fanout; ++r) {
    uint32_t best = 0xffffffffu;
    for (int s = 0; s < c4; s += 4) {
      const uint32_t w0 = lds_u32(a0 + s * kCSlot) - lastp1;
      const uint32_t w1 = lds_u32(a0 + (s + 1) * kCSlot) - lastp1;
      const uint32_t w2 = lds_u32(a0 + (s + 2) * kCSlot) - lastp1;
      const uint32_t w3 = lds_u32(a0 + (s + 3) * kCSlot) - lastp1;
      best = min(min(best, w0), min(w1, min(w2, w3)));
    }
    thr = best + lastp1;
    lastp1 = thr + 1u;
  }
  // keep flags, 32 candidates per word (a 64-bit shift per candidate costs five instructions)
  uint32_t k0 = 0, k1 = 0, bit = 1u;
  const int c_lo = c < 32 ? c : 32;
  for (int i = 0; i < c_lo; ++i) {
    if (lds_u32(a0 + i * kCSlot) <= thr) k0 |= bit;
    bit <<= 1;
  }
  bit = 1u;
  for (int i = 32; i < c; ++i) {
    if (lds_u32(a0 + i * kCSlot) <= thr) k1 |= bit;
    bit <<= 1;
  }
  *kept = __popc(k0) + __popc(k1);
  return ((unsigned long long)k1 << 32) | k0;
}

__global__ void __launch_bounds__(kCThreads)
k_select_chunk(const int32_t* __restrict__ indices, int fanout, int cap, int single_bins,
               SamplePlan* __restrict__ plan, SampleItems items, int32_t* __restrict__ src_global) {
  extern __shared__ __align__(16) uint32_t s_list[];   // [cap][kCThreads]{z, x}
  __shared__ unsigned long long s_c0[kBins + 1];
  for (int i = threadIdx.x; i <= kBins; i += kCThreads) s_c0[i] = plan->bin_chunk0[i];
  __syncthreads();
  const unsigned long long n_chunks = s_c0[kBins];
  const float wantf = want_candidates(fanout);
  const int rshift = c_rank_shift;
  const int lane = threadIdx.x & 31;
  const uint32_t a0 = (uint32_t)__cvta_generic_to_shared(s_list) + threadIdx.x * 8;
  const uint32_t a_lim4 = a0 + (uint32_t)(cap - 4) * kCSlot, a_lim1 = a0 + (uint32_t)(cap - 1) * kCSlot;
  for (;;) {
    unsigned long long base = 0;
    if (lane == 0) base = atomicAdd(&plan->chunk_cursor, 32ull);
    base = __shfl_sync(0xffffffffu, base, 0);
    if (base >= n_chunks) break;
    // the bin of these 32 chunks (bins are padded to multiples of 32): largest o with s_c0[o] <= base
    int lo = 0, hi = kBins;
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (s_c0[mid] <= base) lo = mid; else hi = mid;
    }
    const int bin = kBins - 1 - lo;
    const uint32_t nb = bin_chunks(bin, single_bins);
    const uint32_t k = (uint32_t)(base - s_c0[lo]) + lane;      // chunk number inside the bin
    const uint32_t r = k / nb, idx = k - r * nb;
    if (r >= (uint32_t)plan->bin_count[bin]) continue;          // the bin's padding
    const int q = plan->bin_start[bin] + (int)r;
    const uint64_t hdst = items.hdst[q];
    const uint32_t deg = items.deg[q];
    const uint32_t len = nb == 1 ? deg : ((deg + nb - 1) / nb + 3u) & ~3u;
    const uint32_t j0 = idx * len;
    const uint32_t j1 = min(j0 + len, deg);
    const uint32_t M = row_threshold(wantf, deg);
    uint32_t a = a0;
    uint32_t rem = 0;
    if (j0 < j1) {
      uint64_t x = hdst + (uint64_t)(j0 + 1u) * kGamma;
      uint32_t n4 = (j1 - j0) >> 2;
      while (n4 != 0 && a <= a_lim4) {
        chunk_step(x, M, a);
        chunk_step(x + kGamma, M, a);
        chunk_step(x + 2 * kGamma, M, a);
        chunk_step(x + 3 * kGamma, M, a);
        x += 4 * kGamma;
        --n4;
      }
      rem = ((j1 - j0) & 3u) + 4u * n4;
      while (rem != 0 && a <= a_lim1) {
        chunk_step(x, M, a);
        x += kGamma;
        --rem;
      }
    }
    const int c = (int)((a - a0) / kCSlot);
    const uint32_t hlo = (uint32_t)hdst;
    if (nb > 1) {
      // one chunk of a longer row: hand the candidates to the row's list
      int32_t* cnt = items.row_cnt + q;
      if (rem != 0) {
        atomicOr(cnt, 0x40000000);                     // lane list overflow: the row cannot be proved
      } else if (c > 0) {
        const int slot = atomicAdd(cnt, c);
        uint2* dst = items.cand + (int64_t)q * cap;
        for (int s = 0; s < c; ++s) {
          if (slot + s >= cap) break;                  // the rank kernel sees the count and hands the row on
          const uint32_t z = lds_u32(a0 + s * kCSlot);
          dst[slot + s] = make_uint2(z, (lds_u32(a0 + s * kCSlot + 4) - hlo) * kGammaLoInv - 1u);
        }
      }
      continue;
    }
    // a whole row: rank and emit
    int kept = -1;
    if (rem == 0 && c >= fanout) {
      // the key's high word is z ^ (z >> 31): below 2^31 (every row longer than twice the candidate
      // target) that is z itself, and the list can be ranked as it stands
      if (M >= 0x80000000u || rshift != 0) {
        for (int s = 0; s < c; ++s) {
          const uint32_t z = lds_u32(a0 + s * kCSlot);
          sts_u32(a0 + s * kCSlot, (z ^ (z >> 31)) >> rshift);
        }
      }
      unsigned long long keep = rank_list(a0, c, fanout, &kept);
      if (kept == fanout) {
        const int32_t* row = indices + items.row0[q];
        int32_t* out = src_global + items.out[q];
        for (int e = 0; e < fanout; ++e) {
          const int i = __ffsll((long long)keep) - 1;
          keep &= keep - 1;
          const uint32_t pos = (lds_u32(a0 + i * kCSlot + 4) - hlo) * kGammaLoInv - 1u;
          out[e] = __ldg(row + pos);
        }
      }
    }
    if (kept != fanout) {
      items.fallback[atomicAdd(&plan->n_fallback, 1)] = q;
      atomicAdd(&g_sampler_stat[3], 1ull);
    }
  }
}

// ---- one thread per multi-chunk row: rank the row's candidate list, prove, emit ----------------
// The list (<= cap entries of 8 bytes, written by the chunk kernel) is read straight from global
// memory in every round: a thread's 100-odd bytes stay in L1 after the first touch, and without a
// shared-memory copy the kernel runs at full occupancy, which is what hides the first touch.
__global__ void __launch_bounds__(kCThreads)
k_select_rank(const int32_t* __restrict__ indices, int fanout, int cap, SamplePlan* __restrict__ plan,
              SampleItems items, int32_t* __restrict__ src_global) {
  const int n_hub = plan->n_hub, n_warp_end = plan->n_warp_items;
  const int n_rows = n_hub + (plan->n_multi - n_warp_end);     // hub rows, then the mid-range multi-chunk rows
  const int rshift = c_rank_shift;
  for (int t = blockIdx.x * kCThreads + threadIdx.x; t < n_rows; t += gridDim.x * kCThreads) {
    const int q = t < n_hub ? t : t - n_hub + n_warp_end;
    const int c = items.row_cnt[q];
    int kept = -1;
    if (c >= fanout && c <= cap) {
      const uint2* __restrict__ src = items.cand + (int64_t)q * cap;
      // the fanout-th smallest DISTINCT key word (see rank_list)
      uint32_t lastp1 = 0, thr = 0;
      bool wrapped = false;
      for (int r = 0; r < fanout; ++r) {
        wrapped = wrapped || (r > 0 && lastp1 == 0);
        uint32_t best = 0xffffffffu;
        for (int s = 0; s < c; ++s) {
          const uint32_t z = __ldg(&src[s].x);
          best = min(best, ((z ^ (z >> 31)) >> rshift) - lastp1);
        }
        thr = best + lastp1;
        lastp1 = thr + 1u;
      }
      unsigned long long keep = 0;
      for (int i = 0; i < c; ++i) {
        const uint32_t z = __ldg(&src[i].x);
        keep |= (unsigned long long)(((z ^ (z >> 31)) >> rshift) <= thr) << i;
      }
      if (wrapped) keep = 0;
      kept = __popcll(keep);
      if (kept == fanout) {
        // the lanes of a row append in any order: emit the kept positions ascending
        const int32_t* row = indices + items.row0[q];
        int32_t* out = src_global + items.out[q];
        uint32_t lastq = 0;
        for (int e = 0; e < fanout; ++e) {
          uint32_t best = 0xffffffffu;
          unsigned long long m = keep;
          while (m) {
            const int i = __ffsll((long long)m) - 1;
            m &= m - 1;
            const uint32_t p = __ldg(&src[i].y);
            if (p >= lastq && p < best) best = p;
          }
          out[e] = __ldg(row + best);
          lastq = best + 1u;
        }
      }
    }
    if (kept != fanout) {
      items.fallback[atomicAdd(&plan->n_fallback, 1)] = q;
      atomicAdd(&g_sampler_stat[3], 1ull);
    }
  }
}

// ---- one warp per row: the fallback list (and every keyed row when fanout > kChunkMaxFanout) ----
__global__ void __launch_bounds__(kWarps * 32)
k_select_warp(const int32_t* __restrict__ indices, int fanout, SamplePlan* __restrict__ plan,
              SampleItems items, int32_t* __restrict__ src_global) {
  __shared__ __align__(16) uint32_t s_scratch[kWarps][kScratchWords];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int n_hub = plan->n_hub;
  const int n_warp = plan->n_warp_items - n_hub, n_total = n_warp + plan->n_fallback;
  const float wantf = want_candidates(fanout);
  for (;;) {
    int w = 0;
    if (lane == 0) w = atomicAdd(&plan->warp_cursor, 1);
    w = __shfl_sync(0xffffffffu, w, 0);
    if (w >= n_total) break;
    const int q = w < n_warp ? n_hub + w : items.fallback[w - n_warp];
    const uint64_t hdst = items.hdst[q];
    const uint32_t deg = items.deg[q];
    const int32_t* row = indices + items.row0[q];
    int32_t* out = src_global + items.out[q];
    if (!warp_select_fast(row, deg, fanout, wantf, hdst, s_scratch[wid], out)) {
      // rare: lane-list overflow, a bad threshold guess or a high-word tie at the boundary
      if (lane == 0) atomicAdd(&g_sampler_stat[2], 1ull);
      uint64_t* s_key = reinterpret_cast<uint64_t*>(s_scratch[wid]);
      int32_t* s_pos = reinterpret_cast<int32_t*>(s_scratch[wid] + 2 * kCand);
      warp_select(row, (int64_t)deg, fanout, hdst, s_key, s_pos, out);
    }
  }
}

// ---- the measured ALU roofline of a-1 (include/greengnn.h gg_key_peak) -------------------------
// Key evaluation and nothing else: every lane walks a register-resident SplitMix state and forms
// the high word of fmix for each step (all the selection test reads) with the product loops' own
// key_zhi, folded into one word so the work stays alive.  No list stores, no row logic, no memory
// traffic.  (Round 1's formulation -- the high-half shifts as mul.hi on the FMA pipe -- measured
// 1.35 vs 1.41 Tkey/s and is gone.)
__global__ void __launch_bounds__(256) k_key_peak(uint64_t seed, int groups, uint32_t* __restrict__ fold) {
  uint64_t x = seed + (uint64_t)(blockIdx.x * 256 + threadIdx.x + 1) * 0x632BE59BD9B4E019ull;
  uint32_t acc = 0;
  for (int g = 0; g < groups; ++g) {
#pragma unroll
    for (int i = 0; i < 32; ++i) {
      acc ^= key_zhi((uint32_t)x, (uint32_t)(x >> 32));
      x += kGamma;
    }
  }
#pragma unroll
  for (int o = 16; o; o >>= 1) acc ^= __shfl_xor_sync(0xffffffffu, acc, o);
  if ((threadIdx.x & 31) == 0) atomicXor(fold, acc);
}

// keys per second (CUDA events on `st`, after one warm-up launch).  fold_out = xor of the keys of the
// timed launches (launch i starts from seed 0x9E37 + i).
cudaError_t key_peak(cudaStream_t st, int ctas_per_sm, int groups, int reps, double* keys_per_s, uint32_t* fold_out) {
  uint32_t* d = nullptr;
  cudaError_t e = cudaMalloc((void**)&d, 2 * sizeof(uint32_t));
  if (e != cudaSuccess) return e;
  cudaMemsetAsync(d, 0, 2 * sizeof(uint32_t), st);
  cudaEvent_t a, b;
  cudaEventCreate(&a);
  cudaEventCreate(&b);
  const int grid = sm_count() * ctas_per_sm;
  double rate = 0;
  k_key_peak<<<grid, 256, 0, st>>>(1ull, groups, d + 1);   // warm-up
  cudaEventRecord(a, st);
  for (int i = 0; i < reps; ++i) k_key_peak<<<grid, 256, 0, st>>>(0x9E37ull + i, groups, d);
  count_launches(reps + 1);
  cudaEventRecord(b, st);
  e = cudaEventSynchronize(b);
  float ms = 0;
  if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, a, b);
  if (e == cudaSuccess) rate = (double)grid * 256.0 * groups * 32.0 * reps / (ms * 1e-3);
  uint32_t h[2] = {0, 0};
  if (e == cudaSuccess) e = cudaMemcpy(h, d, sizeof h, cudaMemcpyDeviceToHost);
  if (fold_out) *fold_out = h[0];
  cudaEventDestroy(a);
  cudaEventDestroy(b);
  cudaFree(d);
  *keys_per_s = rate;
  return e;
}

void sampler_stats(unsigned long long out[4]) {
  cudaMemcpyFromSymbol(out, g_sampler_stat, 4 * sizeof(unsigned long long));
}
cudaError_t sampler_tune(int single_bins, int warp_bin, int hub_bin) {
  h_single_bins = single_bins;
  h_warp_bin = warp_bin;
  h_hub_bin = hub_bin;
  return cudaSuccess;
}

// largest row length of a CSR (one pass over indptr at graph creation)
__global__ void k_max_degree(const int64_t* __restrict__ indptr, int64_t n, unsigned long long* __restrict__ out) {
  unsigned long long m = 0;
  for (int64_t v = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; v < n; v += (int64_t)gridDim.x * blockDim.x) {
    const unsigned long long d = (unsigned long long)(indptr[v + 1] - indptr[v]);
    m = d > m ? d : m;
  }
#pragma unroll
  for (int o = 16; o; o >>= 1) {
    const unsigned long long y = __shfl_xor_sync(0xffffffffu, m, o);
    m = y > m ? y : m;
  }
  if ((threadIdx.x & 31) == 0 && m) atomicMax(out, m);
}
cudaError_t max_degree(const int64_t* indptr, int64_t n, int64_t* out) {
  unsigned long long* d = nullptr;
  cudaError_t e = cudaMalloc((void**)&d, sizeof(unsigned long long));
  if (e != cudaSuccess) return e;
  cudaMemset(d, 0, sizeof(unsigned long long));
  k_max_degree<<<sm_count() * 8, 256>>>(indptr, n, d);
  count_launches(1);
  unsigned long long h = 0;
  e = cudaMemcpy(&h, d, sizeof h, cudaMemcpyDeviceToHost);
  cudaFree(d);
  *out = (int64_t)h;
  return e;
}
cudaError_t sampler_debug(int rank_shift, float want_add) {
  cudaError_t e = cudaMemcpyToSymbol(c_rank_shift, &rank_shift, sizeof(int));
  if (e != cudaSuccess) return e;
  return cudaMemcpyToSymbol(c_want_add, &want_add, sizeof(float));
}

void launch_tile_scan(cudaStream_t st, int W, int32_t* tiles, int row_pitch, const BatchOffsets& n_items,
                      int items_per_tile, int32_t* totals) {
  k_tile_scan<<<W, 1024, 0, st>>>(tiles, row_pitch, n_items, items_per_tile, totals, nullptr, 0, 0, 0);
  count_launches(1);
}

size_t sample_plan_bytes() { return sizeof(SamplePlan); }

void launch_sample_hop(cudaStream_t st, const int64_t* indptr, const int32_t* indices,
                       const int32_t* nodes, int64_t node_pitch, const BatchOffsets& n_dst,
                       const BatchOffsets& dst_off, int W, int max_nd, int fanout,
                       const uint64_t* key_prefix_b, uint8_t* cnt_tmp, int64_t cnt_pitch,
                       int32_t* tile_sums, int max_tiles, int32_t* totals, int32_t* blk_indptr,
                       int32_t* edge_off_out, int32_t* src_global, const SampleWork& wk) {
  const int tiles = (max_nd + kTile - 1) / kTile;
  dim3 grid(tiles, W);
  SamplePlan* plan = static_cast<SamplePlan*>(wk.plan);
  const bool chunk_path = fanout <= kChunkMaxFanout;
  // cut-overs of this hop.  A hop with few destinations (the hop out of the seeds: W x 1024 rows)
  // cannot fill the GPU with one lane per row -- its longest rows, alone on their lanes, are the
  // whole kernel (36 us for 1.6 M warp instructions at W=16) -- so there the lane kernel stops at
  // degree 128 and everything above takes a warp.
  int single_bins = h_single_bins, warp_bin = chunk_path ? h_warp_bin : 0;
  if (chunk_path && dst_off.v[W] < kSmallHopRows) {
    single_bins = single_bins < kSmallHopBins ? single_bins : kSmallHopBins;
    warp_bin = warp_bin < kSmallHopBins ? warp_bin : kSmallHopBins;
  }
  // hub rows (bins >= hub_bin; only graphs that have such rows pay for the extra launch) are cut into
  // chunks whatever the other cut-overs say
  int hub_bin = chunk_path ? (h_hub_bin > warp_bin ? h_hub_bin : warp_bin) : kBins;
  if (wk.max_degree > 0 && deg_bin((uint32_t)(wk.max_degree > 0x7fffffff ? 0x7fffffff : wk.max_degree)) < hub_bin) hub_bin = kBins;
  // "whatever the other cut-overs say" includes single_bins: a setting with single_bins > hub_bin would
  // leave the hub rows of bins [hub_bin, single_bins) as single chunks that the lane kernel finishes while
  // the rank kernel still reads their (never zeroed) candidate counts.  Hub rows are always multi-chunk.
  if (single_bins > hub_bin) single_bins = hub_bin;
  const bool multi = chunk_path && (single_bins < warp_bin || hub_bin < kBins);
  cudaMemsetAsync(plan, 0, sizeof(SamplePlan), st);
  count_launches(chunk_path ? (multi ? 6 : 5) : 4);
  k_sample_count<<<grid, kTile, 0, st>>>(indptr, nodes, node_pitch, n_dst, fanout, max_tiles,
                                         cnt_tmp, cnt_pitch, tile_sums, plan);
  k_tile_scan<<<W, 1024, 0, st>>>(tile_sums, max_tiles, n_dst, kTile, totals, plan, single_bins, warp_bin, hub_bin);
  k_sample_plan<<<grid, kTile, 0, st>>>(indptr, indices, nodes, node_pitch, n_dst, dst_off, W,
                                        fanout, max_tiles, key_prefix_b, cnt_tmp, cnt_pitch,
                                        tile_sums, totals, blk_indptr, edge_off_out, src_global,
                                        plan, wk.items, single_bins);
  if (chunk_path) {
    const int cap = cand_cap(fanout);
    const size_t smem = (size_t)cap * kCSlot;
    static bool attr_set = false;
    if (!attr_set) {
      cudaFuncSetAttribute(k_select_chunk, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * (int)kCSlot);
      attr_set = true;
    }
    int per_sm = (int)((220 * 1024) / (smem + 2048));
    per_sm = per_sm < 1 ? 1 : (per_sm > 12 ? 12 : per_sm);
    k_select_chunk<<<sm_count() * per_sm, kCThreads, smem, st>>>(indices, fanout, cap, single_bins, plan, wk.items,
                                                                 src_global);
    if (multi)      // there are multi-chunk bins: their rows' candidate lists are ranked here
      k_select_rank<<<sm_count() * (single_bins < warp_bin ? 16 : 2), kCThreads, 0, st>>>(indices, fanout, cap, plan, wk.items,
                                                                                            src_global);
  }
  k_select_warp<<<sm_count() * 6, kWarps * 32, 0, st>>>(indices, fanout, plan, wk.items, src_global);
}

int sample_cand_cap(int fanout) { return fanout <= kChunkMaxFanout ? cand_cap(fanout) : 0; }
// true when the current cut-overs can send a row through the multi-chunk path (the only user of
// SampleItems::cand): off with the defaults, so the candidate lists need not exist
bool sampler_multi_chunk_on() { return h_single_bins < h_warp_bin || h_hub_bin < kBins; }

}  // namespace gg

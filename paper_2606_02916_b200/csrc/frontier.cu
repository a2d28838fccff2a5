// a-2: frontier build + relabel for one hop of a whole window, with per-batch bitmaps.
//
// frontier_{h+1} = frontier_h ++ ascending(unique(src_global) \ frontier_h)   (reading S6)
// src_local[e]   = position of src_global[e] in frontier_{h+1}
//
// Per batch b the library keeps, over ceil(N/32) words (padded to a multiple of kWordTile):
//   seen[b]        membership in the frontier so far
//   newbits[g][b]  the nodes that JOINED at generation g (g = 0: the seeds, g = h+1: hop h)
//   wprefix[g][b]  for every non-zero word of newbits[g][b], the number of set bits in the
//                  words before it (written only where the word is non-zero)
// so a node u that joined at generation g >= 1 sits at position
//   n_front[g-1][b] + wprefix[g][b][u>>5] + popc(newbits[g][b][u>>5] & ((1<<(u&31))-1))
// -- ascending-ID order with no sort -- and a seed sits at seed_perm[b][rank among seeds].
// Every node that joins a frontier also bumps the window's packed 8-bit access counter
// (a-3: c_k(u) = number of batches whose N_b contains u), so no second pass over N_b is needed.
#include "common.cuh"
#include "kernels.h"

namespace gg {

__device__ __forceinline__ void count_access(uint32_t* cnt8, int32_t u) {
  atomicAdd(cnt8 + (u >> 2), 1u << (8 * (u & 3)));  // result unused -> RED.ADD
}

__global__ void k_seed_init(const int32_t* __restrict__ seeds, BatchOffsets seed_off, int W,
                            int32_t* __restrict__ nodes, int64_t node_pitch,
                            uint32_t* __restrict__ seen, uint32_t* __restrict__ newbits0,
                            int64_t word_pitch, uint32_t* __restrict__ cnt8,
                            int32_t* __restrict__ n_front0) {
  const int S = seed_off.v[W];
  for (int s = blockIdx.x * blockDim.x + threadIdx.x; s < S; s += gridDim.x * blockDim.x) {
    const int b = find_batch(seed_off.v, W, s);
    const int i = s - seed_off.v[b];
    const int32_t u = seeds[s];
    nodes[b * node_pitch + i] = u;
    const uint32_t bit = 1u << (u & 31);
    atomicOr(seen + b * word_pitch + (u >> 5), bit);
    atomicOr(newbits0 + b * word_pitch + (u >> 5), bit);
    count_access(cnt8, u);
    if (s < W) n_front0[s] = seed_off.v[s + 1] - seed_off.v[s];
  }
}

// seed_perm[b][rank of seed among the batch's seeds, ascending id] = its position i
__global__ void k_seed_perm(const int32_t* __restrict__ seeds, BatchOffsets seed_off, int W,
                            const uint32_t* __restrict__ newbits0,
                            const int32_t* __restrict__ wprefix0, int64_t word_pitch,
                            int32_t* __restrict__ seed_perm, int perm_pitch) {
  const int S = seed_off.v[W];
  for (int s = blockIdx.x * blockDim.x + threadIdx.x; s < S; s += gridDim.x * blockDim.x) {
    const int b = find_batch(seed_off.v, W, s);
    const int32_t u = seeds[s];
    const int64_t w = b * word_pitch + (u >> 5);
    const int rank = wprefix0[w] + __popc(newbits0[w] & ((1u << (u & 31)) - 1u));
    seed_perm[b * perm_pitch + rank] = s - seed_off.v[b];
  }
}

// mark the sampled sources of hop h that are not in the frontier yet
__global__ void k_mark(const int32_t* __restrict__ src_global, const int32_t* __restrict__ edge_off,
                       int W, const uint32_t* __restrict__ seen, uint32_t* __restrict__ newbits,
                       int64_t word_pitch) {
  const int E = edge_off[W];
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < E; e += gridDim.x * blockDim.x) {
    const int b = find_batch(edge_off, W, e);
    const int32_t u = src_global[e];
    const int64_t w = b * word_pitch + (u >> 5);
    const uint32_t bit = 1u << (u & 31);
    if (seen[w] & bit) continue;
    if (newbits[w] & bit) continue;  // racy read: a stale 0 only costs a redundant atomic
    atomicOr(newbits + w, bit);
  }
}

__global__ void __launch_bounds__(kWordThreads)
k_word_reduce(const uint32_t* __restrict__ newbits, int64_t word_pitch, int max_wtiles,
              int32_t* __restrict__ wtile_sums) {
  __shared__ int32_t sm[33];
  const int b = blockIdx.y, t = blockIdx.x;
  const uint4* p = reinterpret_cast<const uint4*>(newbits + b * word_pitch + (int64_t)t * kWordTile) +
                   threadIdx.x * 2;
  const uint4 a = p[0], c = p[1];
  int s = __popc(a.x) + __popc(a.y) + __popc(a.z) + __popc(a.w) + __popc(c.x) + __popc(c.y) +
          __popc(c.z) + __popc(c.w);
  int32_t tot;
  block_exclusive_scan<int32_t>(s, sm, &tot);
  if (threadIdx.x == 0) wtile_sums[b * max_wtiles + t] = tot;
}

// EMIT = true: append the new nodes (ascending) to the batch's node list, fold them into `seen`,
// count the access.  EMIT = false (seed generation): only wprefix is written.
template <bool EMIT>
__global__ void __launch_bounds__(kWordThreads)
k_word_emit(const uint32_t* __restrict__ newbits, int32_t* __restrict__ wprefix,
            uint32_t* __restrict__ seen, int64_t word_pitch, int max_wtiles,
            const int32_t* __restrict__ wtile_sums, const int32_t* __restrict__ totals,
            BatchOffsets n_prev, int32_t cap, int32_t* __restrict__ nodes, int64_t node_pitch,
            uint32_t* __restrict__ cnt8, int32_t* __restrict__ n_front_next,
            int32_t* __restrict__ err_flag) {
  __shared__ int32_t sm[33];
  const int b = blockIdx.y, t = blockIdx.x;
  const int64_t w0 = b * word_pitch + (int64_t)t * kWordTile + threadIdx.x * 8;
  const uint4* p = reinterpret_cast<const uint4*>(newbits + w0);
  const uint4 a = p[0], c = p[1];
  const uint32_t x[8] = {a.x, a.y, a.z, a.w, c.x, c.y, c.z, c.w};
  int s = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += __popc(x[k]);
  int32_t tot;
  int32_t ex = block_exclusive_scan<int32_t>(s, sm, &tot);
  if (EMIT && t == 0 && threadIdx.x == 0) {
    const int32_t nn = n_prev.v[b] + totals[b];
    n_front_next[b] = nn;
    if (nn > cap) atomicExch(err_flag, 1);
  }
  if (s == 0) return;
  int32_t run = wtile_sums[b * max_wtiles + t] + ex;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    uint32_t bits = x[k];
    if (!bits) continue;
    wprefix[w0 + k] = run;
    if (EMIT) {
      seen[w0 + k] |= bits;
      const int32_t id0 = (int32_t)(((int64_t)t * kWordTile + threadIdx.x * 8 + k) << 5);
      while (bits) {
        const int bpos = __ffs(bits) - 1;
        bits &= bits - 1;
        const int32_t pos = n_prev.v[b] + run;
        if (pos < cap) {
          nodes[b * node_pitch + pos] = id0 + bpos;
          count_access(cnt8, id0 + bpos);
        }
        ++run;
      }
    } else {
      run += __popc(bits);
    }
  }
}

// src_local for hop h: look the source up generation by generation, newest first
__global__ void k_relabel(const int32_t* __restrict__ src_global, const int32_t* __restrict__ edge_off,
                          int W, int gen_top, const uint32_t* __restrict__ newbits_base,
                          const int32_t* __restrict__ wprefix_base, int64_t gen_pitch,
                          int64_t word_pitch, const int32_t* __restrict__ n_front, int front_pitch,
                          const int32_t* __restrict__ seed_perm, int perm_pitch,
                          int32_t* __restrict__ src_local) {
  const int E = edge_off[W];
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < E; e += gridDim.x * blockDim.x) {
    const int b = find_batch(edge_off, W, e);
    const int32_t u = src_global[e];
    const int64_t w = b * word_pitch + (u >> 5);
    const uint32_t bit = 1u << (u & 31);
    int32_t pos = -1;
    for (int g = gen_top; g >= 1; --g) {
      const uint32_t bits = newbits_base[g * gen_pitch + w];
      if (bits & bit) {
        pos = n_front[(g - 1) * front_pitch + b] + wprefix_base[g * gen_pitch + w] +
              __popc(bits & (bit - 1u));
        break;
      }
    }
    if (pos < 0) {
      const int rank = wprefix_base[w] + __popc(newbits_base[w] & (bit - 1u));
      pos = seed_perm[b * perm_pitch + rank];
    }
    src_local[e] = pos;
  }
}

// sparse clear of every bitmap word the window touched (walks the final node lists)
__global__ void k_bitmap_clear(const int32_t* __restrict__ nodes, int64_t node_pitch,
                               const int32_t* __restrict__ n_final, int W, int n_gen,
                               uint32_t* __restrict__ seen, uint32_t* __restrict__ newbits_base,
                               int64_t gen_pitch, int64_t word_pitch) {
  const int b = blockIdx.y;
  const int n = n_final[b];
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const int64_t w = b * word_pitch + (nodes[b * node_pitch + i] >> 5);
    seen[w] = 0;
    for (int g = 0; g < n_gen; ++g) newbits_base[g * gen_pitch + w] = 0;
  }
}

static int grid_for(int64_t n, int threads, int max_ctas) {
  int64_t g = (n + threads - 1) / threads;
  if (g < 1) g = 1;
  return (int)(g > max_ctas ? max_ctas : g);
}

void launch_seed_init(cudaStream_t st, const FrontierBufs& F, const int32_t* seeds_dev,
                      const BatchOffsets& seed_off, int W, int32_t* nodes, int64_t node_pitch,
                      uint32_t* cnt8, int32_t* n_front0, int32_t* wtile_sums, int32_t* totals) {
  const int S = seed_off.v[W];
  const int g = grid_for(S, 256, sm_count() * 8);
  count_launches(4);
  k_seed_init<<<g, 256, 0, st>>>(seeds_dev, seed_off, W, nodes, node_pitch, F.seen, F.newbits,
                                 F.word_pitch, cnt8, n_front0);
  dim3 wg(F.n_wtiles, W);
  k_word_reduce<<<wg, kWordThreads, 0, st>>>(F.newbits, F.word_pitch, F.n_wtiles, wtile_sums);
  BatchOffsets nw;
  for (int b = 0; b < W; ++b) nw.v[b] = F.n_wtiles;
  launch_tile_scan(st, W, wtile_sums, F.n_wtiles, nw, 1, totals);
  BatchOffsets zero = {};
  k_word_emit<false><<<wg, kWordThreads, 0, st>>>(F.newbits, F.wprefix, F.seen, F.word_pitch,
                                                  F.n_wtiles, wtile_sums, totals, zero, 0, nullptr,
                                                  0, nullptr, nullptr, nullptr);
  k_seed_perm<<<g, 256, 0, st>>>(seeds_dev, seed_off, W, F.newbits, F.wprefix, F.word_pitch,
                                 F.seed_perm, F.perm_pitch);
}

void launch_frontier_hop(cudaStream_t st, const FrontierBufs& F, int hop, int W,
                         const int32_t* src_global, const int32_t* edge_off, int64_t max_edges,
                         const BatchOffsets& n_prev, int32_t cap, int32_t* nodes, int64_t node_pitch,
                         uint32_t* cnt8, int32_t* n_front_dev, int front_pitch, int32_t* wtile_sums,
                         int32_t* totals, int32_t* err_flag, int32_t* src_local) {
  const int g = hop + 1;
  uint32_t* nb = F.newbits + g * F.gen_pitch;
  int32_t* wp = F.wprefix + g * F.gen_pitch;
  const int ge = grid_for(max_edges, 256, sm_count() * 16);
  count_launches(4);
  k_mark<<<ge, 256, 0, st>>>(src_global, edge_off, W, F.seen, nb, F.word_pitch);
  dim3 wg(F.n_wtiles, W);
  k_word_reduce<<<wg, kWordThreads, 0, st>>>(nb, F.word_pitch, F.n_wtiles, wtile_sums);
  BatchOffsets nw;
  for (int b = 0; b < W; ++b) nw.v[b] = F.n_wtiles;
  launch_tile_scan(st, W, wtile_sums, F.n_wtiles, nw, 1, totals);
  k_word_emit<true><<<wg, kWordThreads, 0, st>>>(nb, wp, F.seen, F.word_pitch, F.n_wtiles,
                                                 wtile_sums, totals, n_prev, cap, nodes, node_pitch,
                                                 cnt8, n_front_dev + g * front_pitch, err_flag);
  k_relabel<<<ge, 256, 0, st>>>(src_global, edge_off, W, g, F.newbits, F.wprefix, F.gen_pitch,
                                F.word_pitch, n_front_dev, front_pitch, F.seed_perm, F.perm_pitch,
                                src_local);
}

void launch_bitmap_clear(cudaStream_t st, const FrontierBufs& F, const int32_t* nodes,
                         int64_t node_pitch, const int32_t* n_final, int max_n, int W, int n_gen) {
  dim3 g(grid_for(max_n, 256, sm_count() * 4), W);
  count_launches(1);
  k_bitmap_clear<<<g, 256, 0, st>>>(nodes, node_pitch, n_final, W, n_gen, F.seen, F.newbits,
                                    F.gen_pitch, F.word_pitch);
}

}  // namespace gg

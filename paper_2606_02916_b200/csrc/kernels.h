// Host-callable launchers of the sm_100a kernels (one translation unit per path step).
#pragma once
#include <atomic>

#include "common.cuh"

namespace gg {

extern std::atomic<unsigned long long> g_launches;  // kernels launched by this library
inline void count_launches(int n) { g_launches.fetch_add((unsigned long long)n, std::memory_order_relaxed); }

// SMs of the current device (cached per device; launch grids are sized in multiples of it)
int sm_count();

constexpr int kWordThreads = 256;
constexpr int kWordTile = 2048;  // 32-bit words per CTA tile in the bitmap / counter passes

// per-graph bitmap workspace of a-2 (see frontier.cu)
struct FrontierBufs {
  uint32_t* seen;      // [Wmax][word_pitch]
  uint32_t* newbits;   // [n_gen][Wmax][word_pitch]
  int32_t* wprefix;    // [n_gen][Wmax][word_pitch]
  int32_t* seed_perm;  // [Wmax][perm_pitch]
  int64_t word_pitch;  // words per batch bitmap, multiple of kWordTile
  int64_t gen_pitch;   // Wmax * word_pitch
  int n_wtiles;        // word_pitch / kWordTile
  int perm_pitch;      // max_batch
};

// a-1: work items of one hop, structure of arrays (k_sample_plan writes, the select kernels read)
struct SampleItems {
  uint64_t* hdst;     // SplitMix stream seed of the row: sm(prefix(seed, batch, layer) ^ dst)
  int64_t* row0;      // indptr[dst]
  uint32_t* deg;
  int32_t* out;       // final offset of the row's first kept neighbor in src_global
  int32_t* fallback;  // item indices handed to the warp kernel
  int32_t* row_cnt;   // candidates appended to the row's list so far (multi-chunk rows)
  uint2* cand;        // [item][sample_cand_cap(fanout)] {high key word before the last xor-shift, edge position}
};
struct SampleWork {
  void* plan;         // device, sample_plan_bytes()
  SampleItems items;  // each array holds at least the hop's destination count
  int64_t max_degree; // longest row of the graph (0 = unknown): hub rows get their own treatment only where they exist
};
size_t sample_plan_bytes();
int sample_cand_cap(int fanout);   // entries of a row's candidate list in global memory (0: the hop does not use one)
bool sampler_multi_chunk_on();     // do the current gg_sampler_tune cut-overs enable the multi-chunk path at all?
void launch_sample_hop(cudaStream_t st, const int64_t* indptr, const int32_t* indices,
                       const int32_t* nodes, int64_t node_pitch, const BatchOffsets& n_dst,
                       const BatchOffsets& dst_off, int W, int max_nd, int fanout,
                       const uint64_t* key_prefix_b, uint8_t* cnt_tmp, int64_t cnt_pitch,
                       int32_t* tile_sums, int max_tiles, int32_t* totals, int32_t* blk_indptr,
                       int32_t* edge_off_out, int32_t* src_global, const SampleWork& wk);
void sampler_stats(unsigned long long out[4]);           // synchronous read of g_sampler_stat
cudaError_t sampler_debug(int rank_shift, float want_add);  // test knobs, see sample.cu
cudaError_t sampler_tune(int single_bins, int warp_bin, int hub_bin);   // degree-bin cut-overs of the selection kernels
cudaError_t max_degree(const int64_t* indptr, int64_t n, int64_t* out);  // synchronous
// key-only micro-kernel: the measured integer-ALU roofline of the sampler (keys per second)
cudaError_t key_peak(cudaStream_t st, int ctas_per_sm, int groups, int reps, double* keys_per_s, uint32_t* fold_out);
// shared by a-1 / a-2: one CTA per batch row, exclusive scan of ceil(n_items[b]/items_per_tile) sums
void launch_tile_scan(cudaStream_t st, int W, int32_t* tiles, int row_pitch, const BatchOffsets& n_items,
                      int items_per_tile, int32_t* totals);

// a-2
void launch_seed_init(cudaStream_t st, const FrontierBufs& F, const int32_t* seeds_dev,
                      const BatchOffsets& seed_off, int W, int32_t* nodes, int64_t node_pitch,
                      uint32_t* cnt8, int32_t* n_front0, int32_t* wtile_sums, int32_t* totals);
void launch_frontier_hop(cudaStream_t st, const FrontierBufs& F, int hop, int W,
                         const int32_t* src_global, const int32_t* edge_off, int64_t max_edges,
                         const BatchOffsets& n_prev, int32_t cap, int32_t* nodes, int64_t node_pitch,
                         uint32_t* cnt8, int32_t* n_front_dev, int front_pitch, int32_t* wtile_sums,
                         int32_t* totals, int32_t* err_flag, int32_t* src_local);
void launch_bitmap_clear(cudaStream_t st, const FrontierBufs& F, const int32_t* nodes,
                         int64_t node_pitch, const int32_t* n_final, int max_n, int W, int n_gen);

// a-3 .. a-5
void launch_unique_count(cudaStream_t st, uint32_t* cnt8, int64_t n_words_padded, const OwnerRanges& R,
                         int32_t* tile_sums, int32_t* stats, int32_t* hist, int32_t* uniq, int32_t* cnt);
void launch_hot_select(cudaStream_t st, const int32_t* uniq, const int32_t* cnt, int n_unique,
                       const OwnerRanges& R, int32_t thr, uint32_t quota_eq, uint64_t* tile_sums64,
                       uint64_t* total64, int32_t* hot);
void launch_delta_split(cudaStream_t st, const int32_t* hot, int n_hot, const OwnerRanges& R,
                        const int32_t* slot_prev, int carry_over, int32_t* tile_sums,
                        int32_t* n_delta, int32_t* owner_cnt, int32_t* slot_new, int32_t* req_ids,
                        int32_t* carry_src, int32_t* carry_ids);
void launch_slots_clear(cudaStream_t st, const int32_t* ids, int n, int32_t* slot_map);
void launch_fill_i32(cudaStream_t st, int32_t* p, int64_t n, int32_t v);
// 32-bit words between device and pinned host memory by a kernel (not by a copy engine)
void launch_copy_words(cudaStream_t st, void* dst, const void* src, int64_t n_words);

// a-6 .. a-8
struct GatherLaunch {
  const int32_t* nodes;
  int n;
  const int32_t* slot_of;
  const uint8_t* local_base;
  int64_t local_stride;
  const uint8_t* cache_base;
  int64_t cache_stride;
  uint8_t* out;
  int rb;
  OwnerRanges R;
  StorePtrs store;
  bool may_miss;          // false when H_k = R_k: no miss pass is launched
  int32_t* miss_tmp_pos;  // [ceil(n/64)*64]
  int32_t* miss_tmp_id;
  int32_t* tile_miss;     // [ceil(n/64)]
  int32_t* miss_pos;      // [n]
  int32_t* miss_id;
  int32_t* n_miss;        // device scalar
  int32_t* counters;      // [2 + P]
  unsigned long long* miss_total;  // device scalar: rows filled by a-8 since the profile was last reset (may be null)
  bool miss_over_link;    // a-8 reads pinned host memory (PCIe): a few CTAs saturate it; false: every remote store is device memory
};
void launch_gather(cudaStream_t st, const GatherLaunch& G);      // a-7: one k_gather launch
void launch_miss_path(cudaStream_t st, const GatherLaunch& G);   // a-8: compaction + fill (only if may_miss)
void launch_rows_from_list(cudaStream_t st, const int32_t* src_idx, int n, const uint8_t* src_base,
                           int64_t src_stride, uint8_t* dst_base, int64_t dst_row0, int64_t dst_stride,
                           int rb);
// over_link: the rows come from pinned host memory over PCIe (a dozen CTAs saturate it); false:
// the owner's store is device memory and the copy takes the full grid
void launch_rows_from_store(cudaStream_t st, const int32_t* ids, int n, const StorePtrs& store,
                            const OwnerRanges& R, uint8_t* dst_base, int64_t dst_row0,
                            int64_t dst_stride, int rb, bool over_link = true);

// NEXT-1 trace simulator (simulate.cu)
void launch_count_db(cudaStream_t st, const int32_t* db_nodes, int64_t begin, int64_t end, uint32_t* cnt8);
void launch_classify(cudaStream_t st, const int32_t* db_nodes, const int64_t* db_off, int b0, int nb,
                     int64_t max_n, const int32_t* slot_of, const OwnerRanges& R, int32_t* counters);
void launch_sim_events(cudaStream_t st, const int32_t* delta, const int32_t* counters, int K, int B, int W,
                       const gg_energy_model& E, int P, int64_t row_bytes, gg_sim_result* out_dev);

gg_status report_error(gg_status s, const char* msg);   // sets gg_last_error() of the calling thread
cudaError_t rank_calibrate(const double* z_host, const double* e_host, int n, int F, double lam, double lr,
                           int iters, double* beta_host, double* gamma_host, double* loss_host);

}  // namespace gg

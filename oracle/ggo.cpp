// CPU ORACLE -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, single-threaded restatement of the hot path of GreenGNN's runtime
// phase (arxiv/paper_2606_02916; citations are /root/reference/PAPER.md lines, and
// DESIGN.md "Readings" S1..S21 where the paper is silent).  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// call it.  It shares no code, header, table or constant generator with the CUDA
// path under paper_2606_02916_b200/csrc/.  Parity pins: tests/test_oracle_pins.py
// (every function below is pinned; nothing here is "parity unpinned").
//
// Steps:
//   O0 key      -- deterministic sampling key ("deterministic
//                  neighbor sampling", "seeds are fixed"; constants: reading S1)
//   O1 sample   -- keep the `fanout` edge positions with the smallest (key, pos);
//                  all of them when deg <= fanout (readings S3, S4, S5)
//   O2 blocks   -- frontier_{h+1} = frontier_h ++ ascending new nodes; N_b = last
//                  frontier ("N_b is the set of nodes whose features
//                  batch b requires"; readings S6, S16)
//   O3 unique   -- U_k, c_k(u) over the window's trace T = {(b,u)}
//   O4 hot set  -- the n_hot most frequently accessed REMOTE nodes
//   O5 delta    -- Delta_{k,m} = (H_k n N_m) \ (C_{k-1} n N_m); C_k = H_k
//   O6 service  -- lookup N_b n H_k, M_b = N_b \ H_k (Alg. 1 l.11-12),
//                  M_{b,m} = (N_b n N_m) \ (H_k n N_m); X_b rows
//   O7 trace    -- the event counts Eqs. (1)-(2) consume
#include <algorithm>
#include <cstdint>
#include <cstring>
#include <map>
#include <set>
#include <utility>
#include <vector>

namespace {

// ---- O0: hash (all arithmetic mod 2^64) ------------------------------------
const uint64_t GAMMA = 0x9E3779B97F4A7C15ull;

uint64_t fmix(uint64_t z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
// one SplitMix64 output step from state x
uint64_t sm(uint64_t x) { return fmix(x + GAMMA); }

uint64_t h_dst(uint64_t seed, uint64_t batch, uint64_t layer, uint64_t dst) {
  return sm(sm(sm(sm(seed) ^ batch) ^ layer) ^ dst);
}
// j-th output (0-based) of the SplitMix64 stream seeded with h_dst
uint64_t key_of(uint64_t h, uint64_t j) { return fmix(h + (j + 1) * GAMMA); }

struct Csr {
  int64_t n;
  const int64_t* indptr;
  const int32_t* indices;
};

// test hook: when non-null, replaces key_of for the forced-tie pin (reading S4)
typedef uint64_t (*key_hook_t)(uint64_t h, uint64_t j);
key_hook_t g_key_hook = nullptr;

// ---- O1: one destination ----------------------------------------------------
// Returns the kept edge positions in ascending order.
std::vector<int64_t> sample_positions(const Csr& g, int32_t v, int fanout, uint64_t seed,
                                      uint64_t batch, uint64_t layer) {
  int64_t deg = g.indptr[v + 1] - g.indptr[v];
  std::vector<int64_t> pos;
  if (deg <= 0) return pos;
  if (deg <= fanout) {
    for (int64_t j = 0; j < deg; ++j) pos.push_back(j);
    return pos;
  }
  uint64_t h = h_dst(seed, batch, layer, (uint64_t)(uint32_t)v);
  std::vector<std::pair<uint64_t, int64_t>> kj;
  for (int64_t j = 0; j < deg; ++j)
    kj.push_back({g_key_hook ? g_key_hook(h, (uint64_t)j) : key_of(h, (uint64_t)j), j});
  std::sort(kj.begin(), kj.end());  // lexicographic (key, position): ties -> smaller position
  for (int i = 0; i < fanout; ++i) pos.push_back(kj[i].second);
  std::sort(pos.begin(), pos.end());
  return pos;
}

// ---- O2: blocks and N_b -----------------------------------------------------
struct Block {
  std::vector<int32_t> indptr;      // [n_dst+1]
  std::vector<int32_t> src_global;  // [n_edge]
  std::vector<int32_t> src_local;   // [n_edge]
  int32_t n_dst = 0, n_src = 0;
};
struct Batch {
  std::vector<Block> blocks;    // hop order, 0 = out of the seeds
  std::vector<int32_t> nodes;   // frontier_L = N_b
  std::vector<int32_t> n_front; // |frontier_h|, h = 0..L
};

Batch* batch_sample(const Csr& g, const int32_t* seeds, int n_seeds, const int32_t* fanouts,
                    int L, uint64_t seed, uint64_t batch_index) {
  Batch* B = new Batch();
  std::vector<int32_t> frontier(seeds, seeds + n_seeds);
  B->n_front.push_back((int32_t)frontier.size());
  for (int h = 0; h < L; ++h) {
    Block blk;
    blk.n_dst = (int32_t)frontier.size();
    blk.indptr.push_back(0);
    for (int32_t v : frontier) {
      for (int64_t j : sample_positions(g, v, fanouts[h], seed, batch_index, (uint64_t)h))
        blk.src_global.push_back(g.indices[g.indptr[v] + j]);
      blk.indptr.push_back((int32_t)blk.src_global.size());
    }
    std::set<int32_t> in_frontier(frontier.begin(), frontier.end());
    std::set<int32_t> fresh;
    for (int32_t u : blk.src_global)
      if (!in_frontier.count(u)) fresh.insert(u);
    for (int32_t u : fresh) frontier.push_back(u);  // std::set iterates ascending
    std::map<int32_t, int32_t> where;
    for (size_t i = 0; i < frontier.size(); ++i) where[frontier[i]] = (int32_t)i;
    for (int32_t u : blk.src_global) blk.src_local.push_back(where[u]);
    blk.n_src = (int32_t)frontier.size();
    B->blocks.push_back(blk);
    B->n_front.push_back((int32_t)frontier.size());
  }
  B->nodes = frontier;
  return B;
}

// ---- O3..O7: one window -----------------------------------------------------
struct State {
  int64_t n;
  int P, local_part;
  std::vector<int64_t> part_offsets;
  int64_t n_hot;  // < 0 = unlimited
  int carry_over;
  std::set<int32_t> cache;  // C_{k-1}; C_0 = empty (Alg. 1 l.1)
  int owner(int32_t u) const {
    for (int m = 0; m < P; ++m)
      if (part_offsets[m] <= u && u < part_offsets[m + 1]) return m;
    return -1;
  }
};

struct Window {
  int W = 0, P = 0;
  std::vector<int32_t> uniq, cnt;                 // O3
  std::vector<int32_t> remote;                    // R_k
  std::vector<int32_t> hot;                       // H_k ascending
  std::vector<std::vector<int32_t>> staged, delta;  // per owner
  std::vector<int32_t> carried;                   // H_k n C_{k-1}
  int64_t n_access = 0;
  // per batch
  std::vector<int32_t> n_input, hit_local, hit_cache;
  std::vector<std::vector<int32_t>> miss_cnt;      // [W][P]
  std::vector<std::vector<int32_t>> miss_pos, miss_id;  // [W][*] ascending position
};

Window* window_run(State& S, Batch* const* batches, int W) {
  Window* K = new Window();
  K->W = W;
  K->P = S.P;
  // O3: unique + count; each batch counts a node once (N_b is a set; reading S8)
  std::map<int32_t, int32_t> count;
  for (int b = 0; b < W; ++b) {
    std::set<int32_t> nb(batches[b]->nodes.begin(), batches[b]->nodes.end());
    for (int32_t u : nb) count[u] += 1;
    K->n_access += (int64_t)batches[b]->nodes.size();
  }
  for (auto& kv : count) {
    K->uniq.push_back(kv.first);
    K->cnt.push_back(kv.second);
  }
  // O4: hot set = n_hot most frequently accessed remote nodes; ties by smaller id (S10)
  std::vector<std::pair<int32_t, int32_t>> ranked;  // (-count, id)
  for (size_t i = 0; i < K->uniq.size(); ++i)
    if (S.owner(K->uniq[i]) != S.local_part) {
      K->remote.push_back(K->uniq[i]);
      ranked.push_back({-K->cnt[i], K->uniq[i]});
    }
  if (S.n_hot < 0 || (int64_t)ranked.size() <= S.n_hot) {
    K->hot = K->remote;
  } else {
    std::sort(ranked.begin(), ranked.end());
    for (int64_t i = 0; i < S.n_hot; ++i) K->hot.push_back(ranked[i].second);
    std::sort(K->hot.begin(), K->hot.end());
  }
  // O5: per-owner staged set, delta against C_{k-1}, carried rows; then C_k = H_k (S11)
  K->staged.assign(S.P, {});
  K->delta.assign(S.P, {});
  for (int32_t u : K->hot) {
    int m = S.owner(u);
    K->staged[m].push_back(u);
    bool cached = S.carry_over && S.cache.count(u);
    if (cached) K->carried.push_back(u);
    else K->delta[m].push_back(u);
  }
  S.cache = std::set<int32_t>(K->hot.begin(), K->hot.end());
  // O6: per-batch service against H_k
  K->miss_cnt.assign(W, std::vector<int32_t>(S.P, 0));
  K->miss_pos.assign(W, {});
  K->miss_id.assign(W, {});
  for (int b = 0; b < W; ++b) {
    int32_t hl = 0, hc = 0;
    const std::vector<int32_t>& nb = batches[b]->nodes;
    for (size_t i = 0; i < nb.size(); ++i) {
      int32_t u = nb[i];
      int m = S.owner(u);
      if (m == S.local_part) ++hl;
      else if (S.cache.count(u)) ++hc;
      else {
        K->miss_cnt[b][m] += 1;
        K->miss_pos[b].push_back((int32_t)i);
        K->miss_id[b].push_back(u);
      }
    }
    K->n_input.push_back((int32_t)nb.size());
    K->hit_local.push_back(hl);
    K->hit_cache.push_back(hc);
  }
  return K;
}

template <class T>
void copy_out(const std::vector<T>& v, T* out) {
  if (!v.empty()) std::memcpy(out, v.data(), v.size() * sizeof(T));
}

}  // namespace

// ---- C interface (ctypes; see oracle/ggo.py) ----------------------------------
extern "C" {

uint64_t ggo_fmix(uint64_t z) { return fmix(z); }
uint64_t ggo_sm(uint64_t x) { return sm(x); }
uint64_t ggo_h_dst(uint64_t seed, uint64_t batch, uint64_t layer, uint64_t dst) {
  return h_dst(seed, batch, layer, dst);
}
uint64_t ggo_key(uint64_t seed, uint64_t batch, uint64_t layer, uint64_t dst, uint64_t j) {
  return key_of(h_dst(seed, batch, layer, dst), j);
}
void ggo_set_key_hook(key_hook_t hook) { g_key_hook = hook; }

// O1 for one destination; out_pos/out_ids need room for min(deg, fanout). Returns the count.
int64_t ggo_sample_dst(int64_t n, const int64_t* indptr, const int32_t* indices, int32_t v,
                       int32_t fanout, uint64_t seed, uint64_t batch, uint64_t layer,
                       int64_t* out_pos, int32_t* out_ids) {
  Csr g{n, indptr, indices};
  std::vector<int64_t> pos = sample_positions(g, v, fanout, seed, batch, layer);
  for (size_t i = 0; i < pos.size(); ++i) {
    out_pos[i] = pos[i];
    out_ids[i] = indices[indptr[v] + pos[i]];
  }
  return (int64_t)pos.size();
}

void* ggo_batch_sample(int64_t n, const int64_t* indptr, const int32_t* indices,
                       const int32_t* seeds, int32_t n_seeds, const int32_t* fanouts, int32_t L,
                       uint64_t seed, uint64_t batch_index) {
  Csr g{n, indptr, indices};
  return batch_sample(g, seeds, n_seeds, fanouts, L, seed, batch_index);
}
void ggo_batch_free(void* b) { delete (Batch*)b; }
int32_t ggo_batch_n_front(void* b, int32_t h) { return ((Batch*)b)->n_front[h]; }
int32_t ggo_batch_n_edge(void* b, int32_t h) { return (int32_t)((Batch*)b)->blocks[h].src_global.size(); }
void ggo_batch_nodes(void* b, int32_t* out) { copy_out(((Batch*)b)->nodes, out); }
void ggo_batch_block(void* b, int32_t h, int32_t* indptr, int32_t* src_global, int32_t* src_local) {
  const Block& k = ((Batch*)b)->blocks[h];
  copy_out(k.indptr, indptr);
  copy_out(k.src_global, src_global);
  copy_out(k.src_local, src_local);
}

void* ggo_state_create(int64_t n, int32_t P, const int64_t* part_offsets, int32_t local_part,
                       int64_t n_hot, int32_t carry_over) {
  State* s = new State();
  s->n = n;
  s->P = P;
  s->local_part = local_part;
  s->part_offsets.assign(part_offsets, part_offsets + P + 1);
  s->n_hot = n_hot;
  s->carry_over = carry_over;
  return s;
}
void ggo_state_free(void* s) { delete (State*)s; }
void ggo_state_reset(void* s) { ((State*)s)->cache.clear(); }
int64_t ggo_state_cache_size(void* s) { return (int64_t)((State*)s)->cache.size(); }
void ggo_state_cache(void* s, int32_t* out) {
  for (int32_t u : ((State*)s)->cache) *out++ = u;
}

void* ggo_window_run(void* state, void* const* batches, int32_t W) {
  return window_run(*(State*)state, (Batch* const*)batches, W);
}
void ggo_window_free(void* w) { delete (Window*)w; }
// sizes: what = 0 |U_k|, 1 |R_k|, 2 |H_k|, 3 carried, 4 n_access
int64_t ggo_window_size(void* w, int32_t what) {
  Window* K = (Window*)w;
  switch (what) {
    case 0: return (int64_t)K->uniq.size();
    case 1: return (int64_t)K->remote.size();
    case 2: return (int64_t)K->hot.size();
    case 3: return (int64_t)K->carried.size();
    case 4: return K->n_access;
  }
  return -1;
}
void ggo_window_uniq(void* w, int32_t* uniq, int32_t* cnt) {
  copy_out(((Window*)w)->uniq, uniq);
  copy_out(((Window*)w)->cnt, cnt);
}
void ggo_window_hot(void* w, int32_t* out) { copy_out(((Window*)w)->hot, out); }
void ggo_window_carried(void* w, int32_t* out) { copy_out(((Window*)w)->carried, out); }
int64_t ggo_window_staged_rows(void* w, int32_t m) { return (int64_t)((Window*)w)->staged[m].size(); }
int64_t ggo_window_delta_rows(void* w, int32_t m) { return (int64_t)((Window*)w)->delta[m].size(); }
void ggo_window_delta(void* w, int32_t m, int32_t* out) { copy_out(((Window*)w)->delta[m], out); }
// per batch: out4 = {n_input, hit_local, hit_cache, n_miss}; miss_per_owner[P]
void ggo_window_batch(void* w, int32_t b, int32_t* out4, int32_t* miss_per_owner) {
  Window* K = (Window*)w;
  out4[0] = K->n_input[b];
  out4[1] = K->hit_local[b];
  out4[2] = K->hit_cache[b];
  out4[3] = (int32_t)K->miss_pos[b].size();
  for (int m = 0; m < K->P; ++m) miss_per_owner[m] = K->miss_cnt[b][m];
}
void ggo_window_misses(void* w, int32_t b, int32_t* pos, int32_t* ids) {
  copy_out(((Window*)w)->miss_pos[b], pos);
  copy_out(((Window*)w)->miss_id[b], ids);
}

// O6 feature tensor: X_b[i,:] = the store's row bytes of N_b[i], whichever of the three
// cases (local / cached / miss) serves it.  part_base[m] = host pointer to owner m's rows.
void ggo_gather(const int32_t* nodes, int64_t n_nodes, int32_t P, const int64_t* part_offsets,
                const uint8_t* const* part_base, int64_t stride, int64_t row_bytes, uint8_t* out) {
  for (int64_t i = 0; i < n_nodes; ++i) {
    int32_t u = nodes[i];
    int m = 0;
    while (!(part_offsets[m] <= u && u < part_offsets[m + 1])) ++m;
    (void)P;
    std::memcpy(out + i * row_bytes, part_base[m] + (int64_t)(u - part_offsets[m]) * stride,
                (size_t)row_bytes);
  }
}

}  // extern "C"

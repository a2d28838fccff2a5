// Host orchestration behind the C ABI of include/greengnn.h.
//
// Threads and streams (Alg. 1):
//   caller thread    gg_window_stage enqueues a job; gg_batch_gather launches the per-batch kernels
//                    on the caller's stream after making it wait for the window's cache-ready event
//   sampler thread   stream A: a-1 .. a-3 of a window (sampling, frontiers, unique + count)
//   selector thread  stream B (high priority): a-4 / a-5, request lists to the host
//   stager thread    stream C: owner-service pack + one bulk copy per owner, carry-over copy,
//                    cache-ready event -- all while the caller's stream serves earlier windows
//                    ("Parallel with training", l.8)
// n_win window arenas (blocks, N_b, request lists) and n_cs cache buffers (rows, ID->slot map, the
// list of cached IDs = C_k) rotate: window k uses arena k mod n_win and cache buffer k mod n_cs.
#include <emmintrin.h>
#include <xmmintrin.h>

#include <algorithm>
#include <atomic>
#include <chrono>
#include <condition_variable>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <deque>
#include <functional>
#include <mutex>
#include <string>
#include <thread>
#include <vector>

#include "common.cuh"
#include "kernels.h"

namespace gg {

static thread_local std::string t_err;
static gg_status fail(gg_status s, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  t_err = buf;
  return s;
}
// for the other translation units behind the ABI (sage.cu)
gg_status report_error(gg_status s, const char* msg) {
  t_err = msg;
  return s;
}
#define CU(call)                                                                          \
  do {                                                                                    \
    cudaError_t e_ = (call);                                                              \
    if (e_ != cudaSuccess)                                                                \
      return fail(GG_ERR_CUDA, "%s:%d %s: %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
  } while (0)

static bool g_timeline = getenv("GG_TIMELINE") != nullptr;
static double now_ms();
static void tl(const char* what, long long wid, double extra = 0) {
  if (g_timeline) fprintf(stderr, "TL %.3f %s %lld %.3f\n", now_ms(), what, wid, extra);
}
static double now_ms() {
  using namespace std::chrono;
  return duration<double, std::milli>(steady_clock::now().time_since_epoch()).count();
}

// ---- tiny persistent thread pool for the owner-service pack --------------------------------
class Pool {
 public:
  explicit Pool(int n) : stop_(false), gen_(0), pending_(0) {
    for (int i = 0; i < n; ++i) th_.emplace_back([this, i] { run(i); });
  }
  ~Pool() {
    {
      std::lock_guard<std::mutex> l(m_);
      stop_ = true;
    }
    cv_.notify_all();
    for (auto& t : th_) t.join();
  }
  int size() const { return (int)th_.size(); }
  // fn(chunk) for chunk in [0, n) on at most `limit` of the pool's threads; returns when all are done
  void parallel_for(int64_t n, const std::function<void(int64_t)>& fn, int limit = 1 << 30) {
    if (n <= 0) return;
    if (th_.empty() || n == 1 || limit <= 1) {
      for (int64_t i = 0; i < n; ++i) fn(i);
      return;
    }
    {
      std::lock_guard<std::mutex> l(m_);
      fn_ = &fn;
      n_ = n;
      limit_ = limit;
      next_.store(0);
      pending_ = (int)th_.size();
      ++gen_;
    }
    cv_.notify_all();
    std::unique_lock<std::mutex> l(m_);
    done_.wait(l, [this] { return pending_ == 0; });
  }

 private:
  void run(int index) {
    uint64_t seen = 0;
    for (;;) {
      const std::function<void(int64_t)>* fn;
      int64_t n;
      {
        std::unique_lock<std::mutex> l(m_);
        cv_.wait(l, [&] { return stop_ || gen_ != seen; });
        if (stop_) return;
        seen = gen_;
        fn = fn_;
        n = index < limit_ ? n_ : 0;      // threads beyond the call's limit sit this one out
      }
      while (n > 0) {
        const int64_t i = next_.fetch_add(1);
        if (i >= n) break;
        (*fn)(i);
      }
      std::lock_guard<std::mutex> l(m_);
      if (--pending_ == 0) done_.notify_all();
    }
  }
  std::vector<std::thread> th_;
  std::mutex m_;
  std::condition_variable cv_, done_;
  bool stop_;
  uint64_t gen_;
  int pending_;
  int limit_ = 1 << 30;
  const std::function<void(int64_t)>* fn_ = nullptr;
  int64_t n_ = 0;
  std::atomic<int64_t> next_{0};
};

template <typename T>
struct DevBuf {
  T* p = nullptr;
  int64_t n = 0;
  cudaError_t ensure(int64_t want) {
    if (want <= n) return cudaSuccess;
    if (p) cudaFree(p);
    p = nullptr;
    n = 0;
    cudaError_t e = cudaMalloc((void**)&p, (size_t)want * sizeof(T));
    if (e == cudaSuccess) n = want;
    return e;
  }
  void release() {
    if (p) cudaFree(p);
    p = nullptr;
    n = 0;
  }
};

struct Hop {
  DevBuf<int32_t> blk_indptr, src_global, src_local, edge_off_dev;
  std::vector<int32_t> edge_off;  // host [W+1]
  std::vector<int32_t> dst_off;   // host [W+1]
};

struct Window;

// One of the two cache buffers: rows, ID->slot map and the cached-ID list (= C_k).  They
// outlive the window that filled them: the next window's delta is taken against them.
struct CacheSlot {
  uint8_t* cache = nullptr;
  int32_t* slot_map = nullptr;
  DevBuf<int32_t> hot;
  int64_t n_cached = 0;        // entries of `hot` currently reflected in slot_map
  Window* tenant = nullptr;    // window whose H_k is in here (may already be released)
  // the point of the caller's stream behind which every gather that read this buffer / slot map has
  // completed: recorded by gg_window_release of its tenant.  Kept per cache slot, not per window
  // arena: the arena of a released tenant can be re-staged before the next stage_b on this slot runs.
  cudaEvent_t gather_done = nullptr;
  bool gather_recorded = false;
};

// One of the n_win window arenas (k being served, k+1 being staged, k+2 .. k+n_win-1 sampled ahead).
struct Window {
  // identity / arguments
  int64_t id = -1;
  uint64_t seq = 0;   // stage order
  bool live = false;
  int W = 0, L = 0;
  int fanouts[GG_MAX_LAYERS] = {0};
  uint64_t first_batch = 0;
  std::vector<int32_t> seeds;
  std::vector<int64_t> boff;
  // device arena
  DevBuf<int32_t> nodes, n_front_dev, uniq, cnt, req_ids, carry_src, carry_ids, counters;
  int64_t node_pitch = 0;
  Hop hop[GG_MAX_LAYERS];
  std::vector<int32_t> n_front[GG_MAX_LAYERS + 1];  // host mirrors [W]
  CacheSlot* cs = nullptr;
  // results
  int32_t hist[256] = {0};
  int64_t n_access = 0, n_unique = 0, n_remote = 0, n_hot = 0, n_delta = 0, n_carry = 0;
  int64_t staged[GG_MAX_PARTS] = {0}, bulk[GG_MAX_PARTS] = {0};
  int bulk_copies = 0;
  bool may_miss = false;
  float ms_sample = 0, ms_unique = 0, ms_select = 0, ms_pack = 0, ms_h2d = 0, ms_carry = 0,
        ms_total = 0, ms_wait = 0;
  double t_enqueue = 0;
  // sync
  cudaEvent_t sampled = nullptr;  // phase A complete (stream A)
  cudaEvent_t ready = nullptr;    // cache ready (stream C)
  cudaEvent_t consumer_done = nullptr;   // recorded by gg_window_release on the caller's stream
  bool consumer_recorded = false;
  cudaEvent_t ev_copy[2 * GG_MAX_PARTS + 2] = {nullptr};  // start/stop per bulk copy, last pair = carry
  bool timing_pending = false;    // ms_h2d / ms_carry not yet read from the events
  int32_t* h_req = nullptr;       // pinned: this window's request IDs (device -> host), mode 0
  int64_t h_req_cap = 0;
  CacheSlot* prev_cs = nullptr;   // C_{k-1}'s buffer: source of the carry-over copy
  double t_b0 = 0;                // start of phase B on the host
  bool gather_recorded = false;   // a gather of this window has been issued
  cudaStream_t last_gather_stream = nullptr;
  cudaStream_t gstreams[4] = {nullptr, nullptr, nullptr, nullptr};   // distinct streams its gathers ran on
  int n_gstreams = 0;
  cudaEvent_t ev_join[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};  // release: one per gather stream + the caller's
  bool enqueued = false;          // phase B finished on the host (or an error was recorded)
  gg_status status = GG_OK;
  std::string error;
};

struct Profiler {
  struct Rec { cudaEvent_t a, b; int kind; };
  std::mutex m;
  bool on = false;
  std::vector<Rec> recs;
  std::vector<cudaEvent_t> pool;
  double ms[GG_PROF_KINDS] = {0};
  int64_t regions[GG_PROF_KINDS] = {0}, bytes[GG_PROF_KINDS] = {0};
  cudaEvent_t get() {
    if (!pool.empty()) { cudaEvent_t e = pool.back(); pool.pop_back(); return e; }
    cudaEvent_t e = nullptr;
    cudaEventCreate(&e);
    return e;
  }
  // returns the start event (recorded) or nullptr when profiling is off
  cudaEvent_t begin(cudaStream_t st) {
    std::lock_guard<std::mutex> l(m);
    if (!on) return nullptr;
    cudaEvent_t a = get();
    cudaEventRecord(a, st);
    return a;
  }
  void end(cudaStream_t st, cudaEvent_t a, int kind, int64_t nbytes) {
    if (!a) return;
    std::lock_guard<std::mutex> l(m);
    cudaEvent_t b = get();
    cudaEventRecord(b, st);
    recs.push_back({a, b, kind});
    bytes[kind] += nbytes;
  }
  void resolve() {
    std::lock_guard<std::mutex> l(m);
    for (auto& r : recs) {
      float t = 0;
      cudaEventSynchronize(r.b);
      if (cudaEventElapsedTime(&t, r.a, r.b) == cudaSuccess) { ms[r.kind] += t; regions[r.kind] += 1; }
      pool.push_back(r.a);
      pool.push_back(r.b);
    }
    recs.clear();
  }
  void clear() {
    resolve();
    std::lock_guard<std::mutex> l(m);
    for (int k = 0; k < GG_PROF_KINDS; ++k) { ms[k] = 0; regions[k] = 0; bytes[k] = 0; }
  }
  void destroy() {
    resolve();
    for (auto e : pool) cudaEventDestroy(e);
    pool.clear();
  }
};

}  // namespace gg

using namespace gg;

struct gg_graph {
  Profiler prof;
  // inputs
  int64_t N = 0, nnz = 0, max_degree = 0;
  const int64_t* indptr = nullptr;
  const int32_t* indices = nullptr;
  OwnerRanges R;
  StorePtrs store;
  bool store_on_device[GG_MAX_PARTS] = {false};  // a non-local owner whose rows the GPU addresses as device memory
  int dim = 0, rb = 0;
  gg_dtype dtype = GG_F32;
  gg_config cfg;
  int64_t cache_rows = 0, n_hot_eff = 0;
  int device = 0;
  // phase A workspaces (sampler thread only)
  FrontierBufs F = {};
  int n_gen = 0;
  DevBuf<uint32_t> seen, newbits, cnt8;
  DevBuf<int32_t> wprefix, seed_perm, tiles32, totals, stats, hist, err_flag, seeds_dev;
  DevBuf<uint64_t> key_prefix;
  DevBuf<uint8_t> cnt_tmp, samp_plan;
  DevBuf<uint64_t> it_hdst;
  DevBuf<int64_t> it_row0;
  DevBuf<uint32_t> it_deg;
  DevBuf<int32_t> it_out, it_fb, it_cnt;
  DevBuf<uint2> it_cand;
  int64_t cnt_words = 0;  // padded words of cnt8
  int64_t planned_t32 = 0, planned_cnt_tmp = 0, planned_miss = 0, planned_t64 = 0, planned_cand = 0;
  // phase B workspaces (stager thread only)
  DevBuf<int32_t> tiles32_b, owner_cnt, n_delta_dev;
  DevBuf<uint64_t> tiles64, total64;
  // miss buffers (caller thread, one gather at a time)
  DevBuf<int32_t> miss_tmp_pos, miss_tmp_id, tile_miss, miss_pos, miss_id, n_miss;
  DevBuf<unsigned long long> miss_total;   // rows the miss path filled since gg_profile_enable
  // pinned
  int32_t* h_small = nullptr;    // phase A readback scratch
  int32_t* h_small_b = nullptr;  // phase B readback scratch
  uint8_t* h_resp[2] = {nullptr, nullptr};  // packed rows (host -> device), mode 0, ping-pong
  cudaEvent_t resp_free[2] = {nullptr, nullptr};  // bulk copies out of h_resp[i] have completed
  bool resp_used[2] = {false, false};
  int resp_idx = 0;
  int32_t* h_seeds = nullptr;
  int64_t h_seeds_cap = 0, h_resp_cap[2] = {0, 0};
  uint64_t* h_kp = nullptr;
  // streams / threads
  cudaStream_t side = nullptr;    // phase A: sample, frontier, unique
  cudaStream_t side_b = nullptr;  // phase B: select, delta (the stager thread syncs on it)
  cudaStream_t side_join = nullptr;  // gg_window_release joins the caller's stream and the gather streams here
  cudaStream_t side_c = nullptr;  // phase B: bulk copies, carry-over copy, cache-ready event (never waited on by the stager)
  Window win[GG_MAX_LIVE_WINDOWS];
  int n_win = 3;
  CacheSlot cslot[GG_MAX_CACHE_BUFFERS];
  int n_cs = 2;                   // cache buffers in rotation (window k uses buffer k mod n_cs)
  uint64_t stage_counter = 0;
  CacheSlot* prev_cs = nullptr;   // holds C_{k-1} for the next phase B (stager thread)
  std::thread worker_a, worker_b, worker_c;
  std::mutex mu;
  std::condition_variable cv_a, cv_b, cv_c, cv_done;
  std::deque<Window*> jobs_a, jobs_b, jobs_c;
  int busy = 0;                   // jobs queued or in flight
  bool stop = false;
  Pool* pool = nullptr;
  int pack_threads_busy = 1;      // pack threads while bulk copies are in flight (they share the host's DRAM)
  // bulk copies issued on stream C and not yet known to be complete: (end event, bytes), oldest first
  std::deque<std::pair<cudaEvent_t, int64_t>> link_q;
  std::vector<cudaEvent_t> link_ev_pool;
};

namespace gg {

static int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }

// caps derived from the fanouts (frontier_{h+1} <= frontier_h * (1 + f[h]), also <= N)
static void plan_caps(const gg_graph* g, int L, const int* fanouts, int64_t* cap_front) {
  cap_front[0] = g->cfg.max_batch;
  for (int h = 0; h < L; ++h) {
    int64_t c = cap_front[h] * (1 + (int64_t)fanouts[h]);
    if (c > g->N) c = g->N;
    if (g->cfg.max_input_nodes > 0 && c > g->cfg.max_input_nodes) c = g->cfg.max_input_nodes;
    if (c < cap_front[h]) c = cap_front[h];
    cap_front[h + 1] = c;
  }
}

#define ENS(buf, n)                                                                       \
  do {                                                                                    \
    if ((buf).ensure(n) != cudaSuccess) {                                                 \
      cudaGetLastError();                                                                 \
      return fail(GG_ERR_OOM, "device allocation of %lld elements failed (%s)", (long long)(n), #buf); \
    }                                                                                     \
  } while (0)

// window-local arena (the arena is free: its previous tenant was released)
static gg_status alloc_window(gg_graph* g, Window* w) {
  const int W = w->W, L = w->L, Wmax = g->cfg.max_window;
  int64_t cap_front[GG_MAX_LAYERS + 1];
  plan_caps(g, L, w->fanouts, cap_front);
  w->node_pitch = ceil_div(cap_front[L], 4) * 4;
  ENS(w->nodes, (int64_t)W * w->node_pitch);
  ENS(w->n_front_dev, (int64_t)(GG_MAX_LAYERS + 1) * Wmax);
  for (int h = 0; h < L; ++h) {
    const int64_t ecap = (int64_t)W * cap_front[h] * w->fanouts[h];
    ENS(w->hop[h].blk_indptr, (int64_t)W * cap_front[h] + W);
    ENS(w->hop[h].src_global, ecap);
    ENS(w->hop[h].src_local, ecap);
    ENS(w->hop[h].edge_off_dev, W + 1);
  }
  const int64_t ucap = std::min<int64_t>(g->N, (int64_t)W * w->node_pitch);
  ENS(w->uniq, ucap);
  ENS(w->cnt, ucap);
  ENS(w->req_ids, std::max<int64_t>(g->cache_rows, 1));
  ENS(w->carry_src, std::max<int64_t>(g->cache_rows, 1));
  ENS(w->carry_ids, std::max<int64_t>(g->cache_rows, 1));
  ENS(w->counters, (int64_t)Wmax * (2 + GG_MAX_PARTS));
  return GG_OK;
}

// Shared scratch whose size depends on (W, fanouts).  Called from gg_window_stage on the caller
// thread; grows only after both pipeline threads are idle and the device is quiet.
static gg_status ensure_shared(gg_graph* g, int W, int L, const int* fanouts, bool* need_drain) {
  int64_t cap_front[GG_MAX_LAYERS + 1];
  plan_caps(g, L, fanouts, cap_front);
  const int64_t node_pitch = ceil_div(cap_front[L], 4) * 4;
  if ((int64_t)W * node_pitch >= (1ll << 31))
    return fail(GG_ERR_CAPACITY, "W * max_input_nodes = %lld exceeds int32 indexing", (long long)((int64_t)W * node_pitch));
  int64_t max_tiles = 1, cand = 1;
  for (int h = 0; h < L; ++h) {
    cand = std::max<int64_t>(cand, (int64_t)W * cap_front[h] * sample_cand_cap(fanouts[h]));
    const int64_t ecap = (int64_t)W * cap_front[h] * fanouts[h];
    if (ecap >= (1ll << 31))
      return fail(GG_ERR_CAPACITY, "hop %d edge cap %lld exceeds int32 indexing", h, (long long)ecap);
    max_tiles = std::max(max_tiles, ceil_div(cap_front[h], 256));
  }
  // the per-row candidate lists (28 x 8 bytes per destination: ~1.3 GB for products W=32, ~10x the hop's
  // edge arrays) exist only while gg_sampler_tune has the multi-chunk path on; turning it on later makes
  // the next gg_window_stage grow this scratch (which needs no live window, like any other growth)
  if (!sampler_multi_chunk_on()) cand = 1;
  const int64_t ucap = std::min<int64_t>(g->N, (int64_t)W * node_pitch);
  int64_t t32 = std::max<int64_t>((int64_t)W * max_tiles, (int64_t)W * g->F.n_wtiles);
  t32 = std::max<int64_t>(t32, g->cnt_words / kWordTile);
  const int64_t cnt_tmp = (int64_t)W * cap_front[L - 1];
  const int64_t t64 = ceil_div(ucap, 1024) + 1;
  const int64_t mcap = ceil_div(node_pitch, 64) * 64;
  const bool grow = t32 > g->planned_t32 || cnt_tmp > g->planned_cnt_tmp || t64 > g->planned_t64 ||
                    mcap > g->planned_miss || cand > g->planned_cand;
  if (!grow) return GG_OK;
  if (need_drain) {
    *need_drain = true;
    return GG_OK;
  }
  ENS(g->tiles32, t32);
  ENS(g->cnt_tmp, cnt_tmp);
  ENS(g->samp_plan, (int64_t)sample_plan_bytes());
  ENS(g->it_hdst, cnt_tmp);
  ENS(g->it_row0, cnt_tmp);
  ENS(g->it_deg, cnt_tmp);
  ENS(g->it_out, cnt_tmp);
  ENS(g->it_fb, cnt_tmp);
  ENS(g->it_cnt, cnt_tmp);
  ENS(g->it_cand, cand);
  ENS(g->tiles64, t64);
  ENS(g->miss_tmp_pos, mcap);
  ENS(g->miss_tmp_id, mcap);
  ENS(g->tile_miss, mcap / 64);
  ENS(g->miss_pos, mcap);
  ENS(g->miss_id, mcap);
  g->planned_t32 = std::max(g->planned_t32, t32);
  g->planned_cnt_tmp = std::max(g->planned_cnt_tmp, cnt_tmp);
  g->planned_t64 = std::max(g->planned_t64, t64);
  g->planned_miss = std::max(g->planned_miss, mcap);
  g->planned_cand = std::max(g->planned_cand, cand);
  // every window arena now, while the pipeline is drained: an arena that met its first (or a
  // larger) window inside an epoch used to cudaMalloc hundreds of MB under the running pipeline
  for (int s = 0; s < g->n_win; ++s) {
    Window* a = &g->win[s];
    if (a->live) continue;
    const int w0 = a->W, l0 = a->L;
    int f0[GG_MAX_LAYERS];
    for (int h = 0; h < GG_MAX_LAYERS; ++h) f0[h] = a->fanouts[h];
    a->W = W; a->L = L;
    for (int h = 0; h < L; ++h) a->fanouts[h] = fanouts[h];
    gg_status rc = alloc_window(g, a);
    a->W = w0; a->L = l0;
    for (int h = 0; h < GG_MAX_LAYERS; ++h) a->fanouts[h] = f0[h];
    if (rc != GG_OK) return rc;
  }
  return GG_OK;
}
#undef ENS

static gg_status ensure_pinned(void** p, int64_t* cap, int64_t want) {
  if (want <= *cap) return GG_OK;
  if (*p) cudaFreeHost(*p);
  *p = nullptr;
  *cap = 0;
  const int64_t n = want + want / 2 + 4096;
  if (cudaHostAlloc(p, (size_t)n, cudaHostAllocDefault) != cudaSuccess) {
    cudaGetLastError();
    return fail(GG_ERR_OOM, "pinned host allocation of %lld bytes failed", (long long)n);
  }
  *cap = n;
  return GG_OK;
}

// A window that fails after its seeds were marked leaves bits in the per-batch bitmaps and counts
// in the packed access counters that the sparse clear (which walks the node lists) cannot reach:
// IDs beyond the frontier cap were never written to a list.  Dense reset, so the next window on
// this graph starts from the clean state every window assumes.
static void reset_sampler_state(gg_graph* g) {
  cudaMemsetAsync(g->seen.p, 0, (size_t)g->F.gen_pitch * sizeof(uint32_t), g->side);
  cudaMemsetAsync(g->newbits.p, 0, (size_t)g->F.gen_pitch * g->n_gen * sizeof(uint32_t), g->side);
  cudaMemsetAsync(g->cnt8.p, 0, (size_t)g->cnt_words * sizeof(uint32_t), g->side);
  cudaStreamSynchronize(g->side);
}

// ---- phase A (sampler thread, stream `side`): a-1, a-2, a-3 ---------------------------------
static gg_status stage_a(gg_graph* g, Window* w) {
  const int W = w->W, L = w->L, Wmax = g->cfg.max_window;
  cudaStream_t st = g->side;
  const double t0 = now_ms();
  tl("a_start", w->id);
  CU(cudaSetDevice(g->device));
  gg_status rc = alloc_window(g, w);
  if (rc != GG_OK) return rc;
  // the arena's previous tenant may still be read by gathers already enqueued
  // (and its staging on stream C reads the arena's request / carry lists)
  CU(cudaStreamWaitEvent(st, w->ready, 0));
  w->gather_recorded = false;
  // ... and by the consumer's own kernels / copies behind those gathers (the blocks, N_b): the
  // release recorded the point of the caller's stream after which the arena may be overwritten
  if (w->consumer_recorded) CU(cudaStreamWaitEvent(st, w->consumer_done, 0));
  w->consumer_recorded = false;

  // seeds and per-(batch, layer) key prefixes -> device
  BatchOffsets seed_off;
  for (int b = 0; b <= W; ++b) seed_off.v[b] = (int32_t)w->boff[b];
  const int S = seed_off.v[W];
  std::memcpy(g->h_seeds, w->seeds.data(), (size_t)S * sizeof(int32_t));
  for (int h = 0; h < L; ++h)
    for (int b = 0; b < W; ++b)
      g->h_kp[h * Wmax + b] = key_prefix(g->cfg.seed, w->first_batch + (uint64_t)b, (uint64_t)h);
  launch_copy_words(st, g->seeds_dev.p, g->h_seeds, S);
  launch_copy_words(st, g->key_prefix.p, g->h_kp, 2ll * L * Wmax);
  CU(cudaMemsetAsync(g->err_flag.p, 0, sizeof(int32_t), st));

  // a-1 / a-2, hop by hop over the whole window
  w->n_front[0].assign(W, 0);
  for (int b = 0; b < W; ++b) w->n_front[0][b] = seed_off.v[b + 1] - seed_off.v[b];
  launch_seed_init(st, g->F, g->seeds_dev.p, seed_off, W, w->nodes.p, w->node_pitch, g->cnt8.p,
                   w->n_front_dev.p, g->tiles32.p, g->totals.p + Wmax);
  int32_t* edge_totals = g->totals.p;          // [Wmax]
  int32_t* new_totals = g->totals.p + Wmax;    // [Wmax]
  for (int h = 0; h < L; ++h) {
    Hop& H = w->hop[h];
    BatchOffsets n_dst, dst_off;
    int max_nd = 0;
    H.dst_off.assign(W + 1, 0);
    for (int b = 0; b < W; ++b) {
      n_dst.v[b] = w->n_front[h][b];
      dst_off.v[b] = H.dst_off[b];
      H.dst_off[b + 1] = H.dst_off[b] + n_dst.v[b];
      max_nd = std::max(max_nd, n_dst.v[b]);
    }
    dst_off.v[W] = H.dst_off[W];
    const int max_tiles = (int)ceil_div(max_nd, 256);
    const int64_t cnt_pitch = max_nd;
    SampleWork wk;
    wk.plan = g->samp_plan.p;
    wk.items.hdst = g->it_hdst.p; wk.items.row0 = g->it_row0.p; wk.items.deg = g->it_deg.p;
    wk.items.out = g->it_out.p; wk.items.fallback = g->it_fb.p;
    wk.items.row_cnt = g->it_cnt.p; wk.items.cand = g->it_cand.p;
    wk.max_degree = g->max_degree;
    cudaEvent_t pe = g->prof.begin(st);
    launch_sample_hop(st, g->indptr, g->indices, w->nodes.p, w->node_pitch, n_dst, dst_off, W, max_nd,
                      w->fanouts[h], g->key_prefix.p + h * Wmax, g->cnt_tmp.p, cnt_pitch, g->tiles32.p,
                      max_tiles, edge_totals, H.blk_indptr.p, H.edge_off_dev.p, H.src_global.p, wk);
    g->prof.end(st, pe, GG_PROF_SAMPLE, 0);
    const int64_t max_edges = (int64_t)H.dst_off[W] * w->fanouts[h];
    pe = g->prof.begin(st);
    launch_frontier_hop(st, g->F, h, W, H.src_global.p, H.edge_off_dev.p, max_edges, n_dst,
                        (int32_t)w->node_pitch, w->nodes.p, w->node_pitch, g->cnt8.p, w->n_front_dev.p,
                        Wmax, g->tiles32.p, new_totals, g->err_flag.p, H.src_local.p);
    g->prof.end(st, pe, GG_PROF_FRONTIER, 0);
    // sizes of the next frontier and of this hop's blocks -> host
    launch_copy_words(st, g->h_small, w->n_front_dev.p + (h + 1) * Wmax, W);
    launch_copy_words(st, g->h_small + Wmax, H.edge_off_dev.p, W + 1);
    launch_copy_words(st, g->h_small + 2 * Wmax + 2, g->err_flag.p, 1);
    CU(cudaStreamSynchronize(st));
    if (g->h_small[2 * Wmax + 2]) {
      reset_sampler_state(g);
      return fail(GG_ERR_CAPACITY, "hop %d: a batch's frontier exceeds max_input_nodes = %lld", h,
                  (long long)w->node_pitch);
    }
    w->n_front[h + 1].assign(g->h_small, g->h_small + W);
    H.edge_off.assign(g->h_small + Wmax, g->h_small + Wmax + W + 1);
    if (g->prof.on) {
      int64_t n_new = 0;
      for (int b = 0; b < W; ++b) n_new += w->n_front[h + 1][b] - w->n_front[h][b];
      std::lock_guard<std::mutex> l(g->prof.m);
      g->prof.bytes[GG_PROF_SAMPLE] += 24ll * H.dst_off[W] + 8ll * H.edge_off[W];
      g->prof.bytes[GG_PROF_FRONTIER] += 8ll * H.edge_off[W] + 4ll * n_new;
    }
  }
  int max_n = 0;
  w->n_access = 0;
  for (int b = 0; b < W; ++b) {
    max_n = std::max(max_n, w->n_front[L][b]);
    w->n_access += w->n_front[L][b];
  }
  launch_bitmap_clear(st, g->F, w->nodes.p, w->node_pitch, w->n_front_dev.p + L * Wmax, max_n, W, L + 1);
  const double t1 = now_ms();
  w->ms_sample = (float)(t1 - t0);

  // a-3 unique + count
  cudaEvent_t pe = g->prof.begin(st);
  launch_unique_count(st, g->cnt8.p, g->cnt_words, g->R, g->tiles32.p, g->stats.p, g->hist.p, w->uniq.p, w->cnt.p);
  g->prof.end(st, pe, GG_PROF_UNIQUE, 0);
  launch_copy_words(st, g->h_small, g->stats.p, 1);
  launch_copy_words(st, g->h_small + 1, g->hist.p, 256);
  CU(cudaEventRecord(w->sampled, st));
  CU(cudaStreamSynchronize(st));
  w->n_unique = g->h_small[0];
  std::memcpy(w->hist, g->h_small + 1, 256 * sizeof(int32_t));
  w->n_remote = 0;
  for (int c = 1; c < 256; ++c) w->n_remote += w->hist[c];
  if (g->prof.on) {
    std::lock_guard<std::mutex> l(g->prof.m);
    g->prof.bytes[GG_PROF_UNIQUE] += 4ll * w->n_access + 8ll * w->n_unique;
  }
  w->ms_unique = (float)(now_ms() - t1);
  tl("a_end", w->id);
  CU(cudaGetLastError());
  return GG_OK;
}

// Owner-service pack of rows [i0, i1): response row i <- store row of ids[i].  Destination rows
// are written with non-temporal stores (no read-for-ownership of a buffer the CPU never reads
// again: the DMA engine is its only consumer; plain stores measured 1.7x slower) and the source
// rows are prefetched into L2 two dozen rows ahead: the requested IDs scatter over the owner's
// store, a core's ten line-fill buffers hold barely two 400-byte rows, the L2's queue far more
// (products epoch on the 16-core box: pack 39.9 -> 32.6 ms with 16 threads).
static void pack_rows(uint8_t* resp, const uint8_t* base, const int32_t* ids, int64_t lo, int64_t stride,
                      int64_t rb, int64_t i0, int64_t i1) {
  const bool nt = (rb % 16 == 0) && (((uintptr_t)resp) % 16 == 0);
  const int64_t ahead = 24;
  for (int64_t i = i0; i < i1; ++i) {
    if (i + ahead < i1) {
      const uint8_t* nx = base + (ids[i + ahead] - lo) * stride;
      for (int64_t k = 0; k < rb; k += 64) _mm_prefetch((const char*)(nx + k), _MM_HINT_T1);
    }
    const uint8_t* src = base + (ids[i] - lo) * stride;
    uint8_t* dst = resp + i * rb;
    if (nt) {
      for (int64_t k = 0; k < rb; k += 16)
        _mm_stream_si128((__m128i*)(dst + k), _mm_loadu_si128((const __m128i*)(src + k)));
    } else {
      std::memcpy(dst, src, (size_t)rb);
    }
  }
  if (nt) _mm_sfence();
}

// ---- phase B1 (selector thread, stream `side_b`): a-4, a-5 and the request IDs to the host ----
// ---- phase B2 (stager thread, stream `side_c`): a-6 -------------------------------------------
// Two threads so that window k+1's hot set, delta and request lists are already on the host when
// the stager finishes packing window k: the host link then never waits for a kernel round trip.
static gg_status stage_b1(gg_graph* g, Window* w) {
  const int Wmax = g->cfg.max_window;
  cudaStream_t st = g->side_b;
  CU(cudaSetDevice(g->device));
  CacheSlot* cs = w->cs;
  // The slot still belongs to window seq-2 until the caller releases it (its batches may still
  // be gathered).  Alg. 1 has the same order: the cache for k+1 is warmed while k trains.
  {
    std::unique_lock<std::mutex> l(g->mu);
    g->cv_done.wait(l, [&] {
      Window* t = cs->tenant;
      return g->stop || !t || t->seq + (uint64_t)g->n_cs != w->seq || !t->live;
    });
    if (g->stop) return fail(GG_ERR_STATE, "graph is being destroyed");
  }
  const double t0 = now_ms();
  w->t_b0 = t0;
  tl("b1_start", w->id);
  CU(cudaStreamWaitEvent(st, w->sampled, 0));
  if (cs->gather_recorded) CU(cudaStreamWaitEvent(st, cs->gather_done, 0));
  CacheSlot* prev = g->prev_cs;

  // a-4 hot set: threshold t and quota of count == t nodes from the histogram
  int32_t thr = 0;
  uint32_t quota = 0;
  if (w->n_remote <= g->n_hot_eff) {
    w->n_hot = w->n_remote;
    w->may_miss = false;
  } else {
    w->n_hot = g->n_hot_eff;
    w->may_miss = true;
    int64_t above = 0;
    for (thr = 255; thr >= 1; --thr) {
      if (above + w->hist[thr] > w->n_hot) break;
      above += w->hist[thr];
    }
    quota = (uint32_t)(w->n_hot - above);
  }
  cudaEvent_t pe = g->prof.begin(st);
  launch_slots_clear(st, cs->hot.p, (int)cs->n_cached, cs->slot_map);
  cs->n_cached = 0;
  if (w->n_hot > 0)
    launch_hot_select(st, w->uniq.p, w->cnt.p, (int)w->n_unique, g->R, thr, quota, g->tiles64.p, g->total64.p, cs->hot.p);
  // a-5 delta against C_{k-1}
  const int carry = (g->cfg.carry_over && prev) ? 1 : 0;
  launch_delta_split(st, cs->hot.p, (int)w->n_hot, g->R, prev ? prev->slot_map : nullptr, carry, g->tiles32_b.p,
                     g->n_delta_dev.p, g->owner_cnt.p, cs->slot_map, w->req_ids.p, w->carry_src.p, w->carry_ids.p);
  cs->n_cached = w->n_hot;
  cs->tenant = w;
  g->prof.end(st, pe, GG_PROF_SELECT, 12ll * w->n_unique);
  int32_t* hs = g->h_small_b;
  launch_copy_words(st, hs, g->owner_cnt.p, 2 * GG_MAX_PARTS);
  launch_copy_words(st, hs + 2 * GG_MAX_PARTS, g->n_delta_dev.p, 1);
  tl("b1_launched", w->id);
  CU(cudaStreamSynchronize(st));
  tl("b1_counts", w->id);
  w->n_delta = w->n_hot > 0 ? hs[2 * GG_MAX_PARTS] : 0;
  w->n_carry = w->n_hot - w->n_delta;
  for (int m = 0; m < GG_MAX_PARTS; ++m) {
    w->staged[m] = w->n_hot > 0 ? hs[m] : 0;
    w->bulk[m] = w->n_hot > 0 ? hs[GG_MAX_PARTS + m] : 0;
  }
  // request IDs of the bulk transfers -> this window's pinned buffer (mode 0)
  if (g->cfg.staging_mode == 0 && w->n_delta > 0) {
    void* pr = w->h_req;
    // sized once for the largest request this graph can make (bounded at 32 MB up front): growing
    // a pinned buffer frees and re-pins, which synchronises the device under the sampler
    const int64_t want_b = std::max<int64_t>(w->n_delta * (int64_t)sizeof(int32_t),
                                             std::min<int64_t>(g->cache_rows * (int64_t)sizeof(int32_t), 32ll << 20));
    gg_status rc = ensure_pinned(&pr, &w->h_req_cap, want_b);
    w->h_req = (int32_t*)pr;
    if (rc != GG_OK) return rc;
    tl("b1_pinned", w->id);
    launch_copy_words(st, w->h_req, w->req_ids.p, w->n_delta);
    CU(cudaStreamSynchronize(st));
  }
  w->prev_cs = prev;
  g->prev_cs = cs;
  w->ms_select = (float)(now_ms() - t0);
  tl("b1_end", w->id, (double)w->n_delta);
  CU(cudaGetLastError());
  return GG_OK;
}

static gg_status stage_b2(gg_graph* g, Window* w) {
  const int Wmax = g->cfg.max_window;
  tl("b2_start", w->id);
  CU(cudaSetDevice(g->device));
  CacheSlot* cs = w->cs;
  CacheSlot* prev = w->prev_cs;
  // a-6 staging: one bulk transfer per owner into that owner's contiguous slot range.  The
  // copies, the carry-over copy and the ready event go to stream C, which this thread never
  // waits on: while the DMA engine drains window k's responses the thread already packs window
  // k+1 (two response buffers).  Everything C reads was produced on stream B before phase B1's
  // cudaStreamSynchronize, and B had waited for the old tenant's gathers.
  cudaStream_t sc = g->side_c;
  w->bulk_copies = 0;
  w->ms_pack = 0;
  const int64_t rb = g->rb;
  gg_status rc;
  if (g->cfg.staging_mode == 0 && w->n_delta > 0) {
    const int ri = g->resp_idx;
    g->resp_idx ^= 1;
    if (g->resp_used[ri]) CU(cudaEventSynchronize(g->resp_free[ri]));  // its previous copies are done
    // both response buffers grow together: pinning hundreds of MB takes longer than a whole
    // window, and the cold first window of an epoch lands on either buffer
    for (int k = 0; k < 2; ++k) {
      const int bi = k == 0 ? ri : (ri ^ 1);
      if (g->h_resp_cap[bi] >= w->n_delta * rb) continue;
      if (bi != ri && g->resp_used[bi]) CU(cudaEventSynchronize(g->resp_free[bi]));
      void* pp = g->h_resp[bi];
      rc = ensure_pinned(&pp, &g->h_resp_cap[bi], w->n_delta * rb);
      g->h_resp[bi] = (uint8_t*)pp;
      if (rc != GG_OK) return rc;
    }
    // Owners are served smallest request first: nothing can cross the link before the first pack
    // ends, so the shortest pack goes first (each owner keeps its slot range, owners ascending).
    int64_t q0_of[GG_MAX_PARTS];
    int order[GG_MAX_PARTS];
    {
      int64_t acc = 0;
      for (int m = 0; m < g->R.P; ++m) {
        q0_of[m] = acc;
        acc += w->bulk[m];
        order[m] = m;
      }
      std::stable_sort(order, order + g->R.P, [&](int a, int b) { return w->bulk[a] < w->bulk[b]; });
    }
    for (int oi = 0; oi < g->R.P; ++oi) {
      const int m = order[oi];
      const int64_t nm = w->bulk[m];
      const int64_t q0 = q0_of[m];
      if (nm == 0) continue;
      if (g->store_on_device[m]) {
        // this owner's store is device memory (e.g. a peer's HBM): host threads cannot read it, so
        // its bulk transfer is the pull kernel of staging_mode 1, still one transfer per owner
        cudaEvent_t pd = g->prof.begin(sc);
        CU(cudaEventRecord(w->ev_copy[2 * w->bulk_copies], sc));
        launch_rows_from_store(sc, w->req_ids.p + q0, (int)nm, g->store, g->R, cs->cache, q0, rb, (int)rb, false);
        CU(cudaEventRecord(w->ev_copy[2 * w->bulk_copies + 1], sc));
        g->prof.end(sc, pd, GG_PROF_STAGE_COPY, nm * rb);
        w->bulk_copies += 1;
        continue;
      }
      // owner service: gather owner m's requested rows into a contiguous response
      const double p0 = now_ms();
      const uint8_t* base = g->store.base[m];
      const int64_t lo = g->R.lo[m], stride = g->store.stride;
      const int32_t* ids = w->h_req + q0;
      uint8_t* resp = g->h_resp[ri] + q0 * rb;
      const int64_t chunk = 512;
      // Pack threads: the tuned few while the link has more bytes queued than this pack produces (the
      // copies are what the epoch waits for; fewer threads leave them the host's DRAM), every pool
      // thread when the link is about to run dry (the cold first window, small windows).
      while (!g->link_q.empty() && cudaEventQuery(g->link_q.front().first) == cudaSuccess) {
        g->link_ev_pool.push_back(g->link_q.front().first);
        g->link_q.pop_front();
      }
      cudaGetLastError();
      int64_t queued = 0;
      for (auto& e : g->link_q) queued += e.second;
      const bool link_fed = queued >= nm * rb + nm * rb / 2;
      g->pool->parallel_for(ceil_div(nm, chunk), [&](int64_t c) {
        pack_rows(resp, base, ids, lo, stride, rb, c * chunk, std::min(nm, (c + 1) * chunk));
      }, link_fed ? g->pack_threads_busy : g->pool->size());
      w->ms_pack += (float)(now_ms() - p0);
      tl("pack_done", w->id, now_ms() - p0);
      cudaEvent_t pe = g->prof.begin(sc);
      CU(cudaEventRecord(w->ev_copy[2 * w->bulk_copies], sc));
      CU(cudaMemcpyAsync(cs->cache + q0 * rb, resp, (size_t)(nm * rb), cudaMemcpyHostToDevice, sc));
      CU(cudaEventRecord(w->ev_copy[2 * w->bulk_copies + 1], sc));
      {
        cudaEvent_t le = nullptr;
        if (!g->link_ev_pool.empty()) { le = g->link_ev_pool.back(); g->link_ev_pool.pop_back(); }
        else CU(cudaEventCreateWithFlags(&le, cudaEventDisableTiming));
        CU(cudaEventRecord(le, sc));
        g->link_q.emplace_back(le, nm * rb);
      }
      g->prof.end(sc, pe, GG_PROF_STAGE_COPY, nm * rb);
      w->bulk_copies += 1;
    }
    CU(cudaEventRecord(g->resp_free[ri], sc));
    g->resp_used[ri] = true;
  } else if (w->n_delta > 0) {
    // staging_mode 1: GPU-initiated pull, one launch per owner, no host pack / no ID read-back
    int64_t q0 = 0;
    for (int m = 0; m < g->R.P; ++m) {
      const int64_t nm = w->bulk[m];
      if (nm == 0) continue;
      cudaEvent_t pe = g->prof.begin(sc);
      CU(cudaEventRecord(w->ev_copy[2 * w->bulk_copies], sc));
      launch_rows_from_store(sc, w->req_ids.p + q0, (int)nm, g->store, g->R, cs->cache, q0, rb, (int)rb);
      CU(cudaEventRecord(w->ev_copy[2 * w->bulk_copies + 1], sc));
      g->prof.end(sc, pe, GG_PROF_STAGE_COPY, nm * rb);
      w->bulk_copies += 1;
      q0 += nm;
    }
  }
  // carried rows: D2D out of the previous buffer (filled earlier on the same stream), after the delta rows
  cudaEvent_t pe = g->prof.begin(sc);
  CU(cudaEventRecord(w->ev_copy[2 * GG_MAX_PARTS], sc));
  if (w->n_carry > 0)
    launch_rows_from_list(sc, w->carry_src.p, (int)w->n_carry, prev->cache, rb, cs->cache, w->n_delta, rb, (int)rb);
  CU(cudaEventRecord(w->ev_copy[2 * GG_MAX_PARTS + 1], sc));
  g->prof.end(sc, pe, GG_PROF_CARRY, 2ll * w->n_carry * rb);
  CU(cudaMemsetAsync(w->counters.p, 0, (size_t)Wmax * (2 + GG_MAX_PARTS) * sizeof(int32_t), sc));
  CU(cudaEventRecord(w->ready, sc));
  w->timing_pending = true;
  CU(cudaGetLastError());
  w->ms_total = w->ms_sample + w->ms_unique + (float)(now_ms() - w->t_b0);
  tl("b2_end", w->id);
  return GG_OK;
}

// ms_h2d / ms_carry of a window whose ready event has completed
static void resolve_timing(Window* w) {
  if (!w->timing_pending) return;
  float ms = 0;
  w->ms_h2d = 0;
  for (int c = 0; c < w->bulk_copies; ++c)
    if (cudaEventElapsedTime(&ms, w->ev_copy[2 * c], w->ev_copy[2 * c + 1]) == cudaSuccess) w->ms_h2d += ms;
  if (cudaEventElapsedTime(&ms, w->ev_copy[2 * GG_MAX_PARTS], w->ev_copy[2 * GG_MAX_PARTS + 1]) == cudaSuccess)
    w->ms_carry = ms;
  cudaGetLastError();
  w->timing_pending = false;
}

static void finish_job(gg_graph* g, Window* w, gg_status rc) {
  {
    std::lock_guard<std::mutex> l(g->mu);
    w->status = rc;
    if (rc != GG_OK) w->error = t_err;
    w->enqueued = true;
    g->busy -= 1;
  }
  g->cv_done.notify_all();
}

static void worker_a_main(gg_graph* g) {
  cudaSetDevice(g->device);
  for (;;) {
    Window* w;
    {
      std::unique_lock<std::mutex> l(g->mu);
      g->cv_a.wait(l, [&] { return g->stop || !g->jobs_a.empty(); });
      if (g->jobs_a.empty()) return;
      w = g->jobs_a.front();
      g->jobs_a.pop_front();
    }
    gg_status rc = stage_a(g, w);
    if (rc != GG_OK) {
      finish_job(g, w, rc);
      continue;
    }
    {
      std::lock_guard<std::mutex> l(g->mu);
      g->jobs_b.push_back(w);
    }
    g->cv_b.notify_one();
  }
}

static void worker_b_main(gg_graph* g) {
  cudaSetDevice(g->device);
  for (;;) {
    Window* w;
    {
      std::unique_lock<std::mutex> l(g->mu);
      g->cv_b.wait(l, [&] { return g->stop || !g->jobs_b.empty(); });
      if (g->jobs_b.empty()) return;
      w = g->jobs_b.front();
      g->jobs_b.pop_front();
    }
    gg_status rc = stage_b1(g, w);
    if (rc != GG_OK) {
      finish_job(g, w, rc);
      continue;
    }
    {
      std::lock_guard<std::mutex> l(g->mu);
      g->jobs_c.push_back(w);
    }
    g->cv_c.notify_one();
  }
}

static void worker_c_main(gg_graph* g) {
  cudaSetDevice(g->device);
  for (;;) {
    Window* w;
    {
      std::unique_lock<std::mutex> l(g->mu);
      g->cv_c.wait(l, [&] { return g->stop || !g->jobs_c.empty(); });
      if (g->jobs_c.empty()) return;
      w = g->jobs_c.front();
      g->jobs_c.pop_front();
    }
    finish_job(g, w, stage_b2(g, w));
  }
}

}  // namespace gg


// =================================== C ABI ====================================================
extern "C" {

const char* gg_last_error(void) { return t_err.c_str(); }
const char* gg_version(void) { return "greengnn-b200 0.1 (sm_100a)"; }

uint64_t gg_key(uint64_t seed, uint64_t batch, uint64_t layer, uint64_t dst, uint64_t edge_pos) {
  return key_edge(key_hdst(key_prefix(seed, batch, layer), dst), edge_pos);
}

static bool is_device_ptr(const void* p) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}
static bool is_pinned_ptr(const void* p) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  return a.type == cudaMemoryTypeHost;
}

gg_status gg_graph_destroy(gg_graph* g) {
  if (!g) return fail(GG_ERR_INVALID_ARG, "null graph");
  {
    std::lock_guard<std::mutex> l(g->mu);
    g->stop = true;
  }
  g->cv_a.notify_all();
  g->cv_b.notify_all();
  g->cv_c.notify_all();
  g->cv_done.notify_all();
  if (g->worker_a.joinable()) g->worker_a.join();
  if (g->worker_b.joinable()) g->worker_b.join();
  if (g->worker_c.joinable()) g->worker_c.join();
  cudaSetDevice(g->device);
  cudaDeviceSynchronize();
  delete g->pool;
  g->prof.destroy();
  for (int s = 0; s < g->n_win; ++s) {
    Window& w = g->win[s];
    w.nodes.release(); w.n_front_dev.release(); w.uniq.release(); w.cnt.release();
    w.req_ids.release(); w.carry_src.release(); w.carry_ids.release(); w.counters.release();
    for (int h = 0; h < GG_MAX_LAYERS; ++h) {
      w.hop[h].blk_indptr.release(); w.hop[h].src_global.release();
      w.hop[h].src_local.release(); w.hop[h].edge_off_dev.release();
    }
    if (w.sampled) cudaEventDestroy(w.sampled);
    if (w.ready) cudaEventDestroy(w.ready);
    if (w.consumer_done) cudaEventDestroy(w.consumer_done);
    for (int c = 0; c < 5; ++c) if (w.ev_join[c]) cudaEventDestroy(w.ev_join[c]);
    if (w.h_req) cudaFreeHost(w.h_req);
    for (int c = 0; c < 2 * GG_MAX_PARTS + 2; ++c) if (w.ev_copy[c]) cudaEventDestroy(w.ev_copy[c]);
  }
  for (int s = 0; s < g->n_cs; ++s) {
    CacheSlot& c = g->cslot[s];
    c.hot.release();
    if (c.gather_done) cudaEventDestroy(c.gather_done);
    if (c.cache) cudaFree(c.cache);
    if (c.slot_map) cudaFree(c.slot_map);
  }
  g->tiles32_b.release();
  g->seen.release(); g->newbits.release(); g->cnt8.release(); g->wprefix.release();
  g->seed_perm.release(); g->tiles32.release(); g->totals.release(); g->stats.release();
  g->hist.release(); g->owner_cnt.release(); g->n_delta_dev.release(); g->err_flag.release();
  g->seeds_dev.release(); g->tiles64.release(); g->total64.release(); g->key_prefix.release();
  g->samp_plan.release(); g->it_hdst.release(); g->it_row0.release(); g->it_deg.release();
  g->it_out.release(); g->it_fb.release(); g->it_cnt.release(); g->it_cand.release();
  g->cnt_tmp.release(); g->miss_tmp_pos.release(); g->miss_tmp_id.release(); g->tile_miss.release();
  g->miss_pos.release(); g->miss_id.release(); g->n_miss.release(); g->miss_total.release();
  if (g->h_small) cudaFreeHost(g->h_small);
  if (g->h_small_b) cudaFreeHost(g->h_small_b);
  for (int i = 0; i < 2; ++i) {
    if (g->h_resp[i]) cudaFreeHost(g->h_resp[i]);
    if (g->resp_free[i]) cudaEventDestroy(g->resp_free[i]);
  }
  for (auto& e : g->link_q) cudaEventDestroy(e.first);
  for (auto e : g->link_ev_pool) cudaEventDestroy(e);
  if (g->h_seeds) cudaFreeHost(g->h_seeds);
  if (g->h_kp) cudaFreeHost(g->h_kp);
  if (g->side) cudaStreamDestroy(g->side);
  if (g->side_b) cudaStreamDestroy(g->side_b);
  if (g->side_c) cudaStreamDestroy(g->side_c);
  if (g->side_join) cudaStreamDestroy(g->side_join);
  delete g;
  return GG_OK;
}

gg_status gg_graph_create(const gg_csr* csr, const gg_owner_map* owners, const gg_feature_store* store,
                          const gg_config* cfg, gg_graph** out) {
  if (!csr || !owners || !store || !cfg || !out) return fail(GG_ERR_INVALID_ARG, "null argument");
  *out = nullptr;
  if (csr->num_nodes < 1 || csr->num_nodes >= (1ll << 31) || csr->num_edges < 0)
    return fail(GG_ERR_INVALID_ARG, "num_nodes must be in [1, 2^31), num_edges >= 0");
  if (!csr->indptr || (!csr->indices && csr->num_edges > 0)) return fail(GG_ERR_INVALID_ARG, "null CSR array");
  const int P = owners->num_parts;
  if (P < 1 || P > GG_MAX_PARTS) return fail(GG_ERR_INVALID_ARG, "num_parts must be in [1, %d]", GG_MAX_PARTS);
  if (owners->local_part < 0 || owners->local_part >= P) return fail(GG_ERR_INVALID_ARG, "local_part out of range");
  if (!owners->part_offsets) return fail(GG_ERR_INVALID_ARG, "null part_offsets");
  if (owners->part_offsets[0] != 0 || owners->part_offsets[P] != csr->num_nodes)
    return fail(GG_ERR_INVALID_ARG, "part_offsets must start at 0 and end at num_nodes");
  for (int m = 0; m < P; ++m)
    if (owners->part_offsets[m] > owners->part_offsets[m + 1])
      return fail(GG_ERR_INVALID_ARG, "part_offsets must be non-decreasing");
  const int esz = store->dtype == GG_F32 ? 4 : (store->dtype == GG_BF16 ? 2 : 0);
  if (!esz) return fail(GG_ERR_INVALID_ARG, "unknown dtype");
  if (store->dim < 1 || !store->part_base) return fail(GG_ERR_INVALID_ARG, "bad feature store");
  const int64_t rb = (int64_t)store->dim * esz;
  if (rb % 4) return fail(GG_ERR_INVALID_ARG, "row bytes must be a multiple of 4");
  if (store->row_stride_bytes < rb || store->row_stride_bytes % 4)
    return fail(GG_ERR_INVALID_ARG, "row_stride_bytes must be >= row bytes and a multiple of 4");
  if (cfg->max_layers < 1 || cfg->max_layers > GG_MAX_LAYERS) return fail(GG_ERR_INVALID_ARG, "max_layers out of range");
  if (cfg->max_window < 1 || cfg->max_window > GG_MAX_WINDOW) return fail(GG_ERR_INVALID_ARG, "max_window out of range");
  if (cfg->max_batch < 1) return fail(GG_ERR_INVALID_ARG, "max_batch must be >= 1");
  if (cfg->staging_mode != 0 && cfg->staging_mode != 1) return fail(GG_ERR_INVALID_ARG, "staging_mode must be 0 or 1");
  if (!is_device_ptr(csr->indptr) || (csr->num_edges > 0 && !is_device_ptr(csr->indices)))
    return fail(GG_ERR_INVALID_ARG, "indptr / indices must be device memory");
  for (int m = 0; m < P; ++m) {
    const bool empty = owners->part_offsets[m] == owners->part_offsets[m + 1];
    if (empty) continue;
    if (!store->part_base[m]) return fail(GG_ERR_INVALID_ARG, "part_base[%d] is null", m);
    if (m == owners->local_part) {
      if (!is_device_ptr(store->part_base[m])) return fail(GG_ERR_INVALID_ARG, "local part's store must be device memory");
    } else if (!is_pinned_ptr(store->part_base[m]) && !is_device_ptr(store->part_base[m])) {
      return fail(GG_ERR_INVALID_ARG, "part_base[%d] must be pinned host memory (page-locked, CUDA-registered)", m);
    }
  }

  gg_graph* g = new gg_graph();
  g->N = csr->num_nodes; g->nnz = csr->num_edges; g->indptr = csr->indptr; g->indices = csr->indices;
  g->R.P = P; g->R.local = owners->local_part;
  for (int m = 0; m <= P; ++m) g->R.lo[m] = owners->part_offsets[m];
  for (int m = P + 1; m <= GG_MAX_PARTS; ++m) g->R.lo[m] = g->N;
  for (int m = 0; m < GG_MAX_PARTS; ++m) g->store.base[m] = m < P ? (const uint8_t*)store->part_base[m] : nullptr;
  for (int m = 0; m < P; ++m)
    g->store_on_device[m] = m != owners->local_part && store->part_base[m] &&
                            owners->part_offsets[m] < owners->part_offsets[m + 1] && is_device_ptr(store->part_base[m]);
  g->store.stride = store->row_stride_bytes;
  g->dim = store->dim; g->rb = (int)rb; g->dtype = store->dtype; g->cfg = *cfg;
  g->n_cs = cfg->cache_buffers <= 0 ? 2 : std::min(std::max(cfg->cache_buffers, 2), GG_MAX_CACHE_BUFFERS);
  g->n_win = cfg->max_live_windows <= 0 ? 3 : std::min(std::max(cfg->max_live_windows, 3), GG_MAX_LIVE_WINDOWS);
  cudaGetDevice(&g->device);
  const int64_t n_remote_nodes = g->N - (g->R.lo[g->R.local + 1] - g->R.lo[g->R.local]);
  g->cache_rows = cfg->max_cache_rows > 0 ? std::min<int64_t>(cfg->max_cache_rows, n_remote_nodes) : n_remote_nodes;
  g->n_hot_eff = cfg->n_hot < 0 ? g->cache_rows : std::min<int64_t>(cfg->n_hot, g->cache_rows);

  gg_status rc = GG_OK;
  auto bad = [&](gg_status s) { gg_graph_destroy(g); return s; };
#define CUC(call)                                                                              \
  do {                                                                                         \
    cudaError_t e_ = (call);                                                                   \
    if (e_ != cudaSuccess) {                                                                   \
      rc = fail(e_ == cudaErrorMemoryAllocation ? GG_ERR_OOM : GG_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
      cudaGetLastError();                                                                      \
      return bad(rc);                                                                          \
    }                                                                                          \
  } while (0)
  const int Wmax = cfg->max_window, Lmax = cfg->max_layers;
  g->n_gen = Lmax + 1;
  g->F.word_pitch = ceil_div(ceil_div(g->N, 32), kWordTile) * kWordTile;
  g->F.gen_pitch = (int64_t)Wmax * g->F.word_pitch;
  g->F.n_wtiles = (int)(g->F.word_pitch / kWordTile);
  g->F.perm_pitch = cfg->max_batch;
  CUC(g->seen.ensure(g->F.gen_pitch));
  CUC(g->newbits.ensure(g->F.gen_pitch * g->n_gen));
  CUC(g->wprefix.ensure(g->F.gen_pitch * g->n_gen));
  CUC(g->seed_perm.ensure((int64_t)Wmax * cfg->max_batch));
  g->F.seen = g->seen.p; g->F.newbits = g->newbits.p; g->F.wprefix = g->wprefix.p; g->F.seed_perm = g->seed_perm.p;
  g->cnt_words = ceil_div(ceil_div(g->N, 4), kWordTile) * kWordTile;
  CUC(g->cnt8.ensure(g->cnt_words));
  CUC(cudaMemset(g->seen.p, 0, (size_t)g->F.gen_pitch * 4));
  CUC(cudaMemset(g->newbits.p, 0, (size_t)g->F.gen_pitch * g->n_gen * 4));
  CUC(cudaMemset(g->cnt8.p, 0, (size_t)g->cnt_words * 4));
  CUC(g->totals.ensure(2 * Wmax + 2));
  CUC(g->stats.ensure(4)); CUC(g->hist.ensure(256)); CUC(g->owner_cnt.ensure(2 * GG_MAX_PARTS));
  CUC(g->n_delta_dev.ensure(1)); CUC(g->err_flag.ensure(1)); CUC(g->total64.ensure(1)); CUC(g->n_miss.ensure(1));
  CUC(cudaMemset(g->n_miss.p, 0, 4));
  CUC(g->miss_total.ensure(1));
  CUC(cudaMemset(g->miss_total.p, 0, sizeof(unsigned long long)));
  CUC(g->seeds_dev.ensure((int64_t)Wmax * cfg->max_batch));
  CUC(g->key_prefix.ensure((int64_t)GG_MAX_LAYERS * Wmax));
  CUC(cudaHostAlloc((void**)&g->h_small, 4096 * sizeof(int32_t), cudaHostAllocDefault));
  CUC(cudaHostAlloc((void**)&g->h_small_b, 4096 * sizeof(int32_t), cudaHostAllocDefault));
  CUC(g->tiles32_b.ensure(ceil_div(std::max<int64_t>(g->cache_rows, 1), 1024) + 2));
  CUC(cudaHostAlloc((void**)&g->h_seeds, (size_t)Wmax * cfg->max_batch * sizeof(int32_t), cudaHostAllocDefault));
  CUC(cudaHostAlloc((void**)&g->h_kp, (size_t)GG_MAX_LAYERS * Wmax * sizeof(uint64_t), cudaHostAllocDefault));
  CUC(cudaStreamCreateWithFlags(&g->side, cudaStreamNonBlocking));
  {
    // the stager's kernels are tiny but sit on the critical path to the host link (the thread
    // waits for |Delta_m| before it can pack): run them ahead of the sampler's long kernels
    int lo_pri = 0, hi_pri = 0;
    CUC(cudaDeviceGetStreamPriorityRange(&lo_pri, &hi_pri));
    CUC(cudaStreamCreateWithPriority(&g->side_b, cudaStreamNonBlocking, hi_pri));
  }
  CUC(cudaStreamCreateWithFlags(&g->side_c, cudaStreamNonBlocking));
  CUC(cudaStreamCreateWithFlags(&g->side_join, cudaStreamNonBlocking));
  for (int i = 0; i < 2; ++i) CUC(cudaEventCreateWithFlags(&g->resp_free[i], cudaEventDisableTiming));
  for (int s = 0; s < g->n_cs; ++s) {
    CacheSlot& c = g->cslot[s];
    CUC(cudaEventCreateWithFlags(&c.gather_done, cudaEventDisableTiming));
    CUC(cudaMalloc((void**)&c.cache, (size_t)std::max<int64_t>(g->cache_rows, 1) * rb));
    CUC(cudaMalloc((void**)&c.slot_map, (size_t)g->N * sizeof(int32_t)));
    CUC(c.hot.ensure(std::max<int64_t>(g->cache_rows, 1)));
    launch_fill_i32(0, c.slot_map, g->N, -1);
  }
  for (int s = 0; s < g->n_win; ++s) {
    Window& w = g->win[s];
    CUC(cudaEventCreateWithFlags(&w.sampled, cudaEventDisableTiming));
    CUC(cudaEventCreateWithFlags(&w.ready, cudaEventDefault));
    CUC(cudaEventCreateWithFlags(&w.consumer_done, cudaEventDisableTiming));
    for (int c = 0; c < 5; ++c) CUC(cudaEventCreateWithFlags(&w.ev_join[c], cudaEventDisableTiming));
    for (int c = 0; c < 2 * GG_MAX_PARTS + 2; ++c) CUC(cudaEventCreate(&w.ev_copy[c]));
  }
  CUC(max_degree(g->indptr, g->N, &g->max_degree));
  CUC(cudaDeviceSynchronize());
#undef CUC
  // The pack and the DMA reads of the bulk copies share the host's DRAM: more pack threads finish a
  // window's pack sooner but slow the copies it overlaps with (products W=16 on the 16-core box,
  // threads -> copies GB/s / epoch ms: 4 -> 54.4 / 53.2, 6 -> 52.1 / 45.9, 8 -> 47.8 / 46.5, 16 -> 45.8 /
  // 48.0).  Default: 0.4 x the hardware threads, where pack time and copy time of a window meet.
  const unsigned hw = std::max(1u, std::thread::hardware_concurrency());
  const int nt = cfg->host_threads > 0 ? cfg->host_threads : (int)std::min<unsigned>(16u, std::max(2u, (hw * 2u + 2u) / 5u));
  g->pack_threads_busy = nt;
  // an explicit host_threads is a hard cap (the pool IS that many threads, link busy or not); only the
  // default lets a pack that finds the link idle (cold or small windows) spread over up to 16 threads
  const int n_pool = cfg->host_threads > 0 ? nt : (int)std::min<unsigned>(16u, hw);
  g->pool = new Pool(n_pool > 1 ? n_pool : 0);
  g->worker_a = std::thread(worker_a_main, g);
  g->worker_b = std::thread(worker_b_main, g);
  g->worker_c = std::thread(worker_c_main, g);
  *out = g;
  return GG_OK;
}

}  // extern "C"

namespace gg {
static Window* find_window(gg_graph* g, int64_t id) {
  for (int s = 0; s < g->n_win; ++s)
    if (g->win[s].live && g->win[s].id == id) return &g->win[s];
  return nullptr;
}
// Alg. 1 l.5: block until the prefetcher is done with this window
static gg_status wait_enqueued(gg_graph* g, Window* w) {
  const double t0 = now_ms();
  std::unique_lock<std::mutex> l(g->mu);
  if (!w->enqueued) {
    // window k+2's cache buffer is window k's: it cannot be built before k is released
    Window* t = w->cs ? w->cs->tenant : nullptr;
    for (int s = 0; s < g->n_win; ++s) {
      Window* o = &g->win[s];
      if (o != w && o->live && o->seq + (uint64_t)g->n_cs == w->seq)
        return fail(GG_ERR_STATE, "window %lld shares its cache buffer with live window %lld: release that one first",
                    (long long)w->id, (long long)o->id);
    }
    (void)t;
    g->cv_done.wait(l, [&] { return w->enqueued; });
    w->ms_wait += (float)(now_ms() - t0);
  }
  if (w->status != GG_OK) {
    t_err = w->error;
    return w->status;
  }
  return GG_OK;
}
static void fill_batch_out(Window* w, int b, gg_batch_out* out, gg_graph* g) {
  out->num_layers = w->L;
  for (int h = 0; h < w->L; ++h) {
    Hop& H = w->hop[h];
    gg_block& k = out->blocks[h];
    k.n_dst = w->n_front[h][b];
    k.n_src = w->n_front[h + 1][b];
    k.n_edge = H.edge_off[b + 1] - H.edge_off[b];
    k.indptr = H.blk_indptr.p + H.dst_off[b] + b;
    k.src_local = H.src_local.p + H.edge_off[b];
    k.src_global = H.src_global.p + H.edge_off[b];
  }
  out->n_input = w->n_front[w->L][b];
  out->input_nodes = w->nodes.p + (int64_t)b * w->node_pitch;
  out->miss_pos = g->miss_pos.p;
  out->miss_id = g->miss_id.p;
  out->n_miss = g->n_miss.p;
}
}  // namespace gg

extern "C" {

gg_status gg_window_stage(gg_graph* g, int64_t window_id, uint64_t first_batch_index, const int32_t* seeds,
                          const int64_t* batch_offsets, int32_t W, const int32_t* fanouts, int32_t num_layers) {
  if (!g || !seeds || !batch_offsets || !fanouts) return fail(GG_ERR_INVALID_ARG, "null argument");
  if (W < 1 || W > g->cfg.max_window) return fail(GG_ERR_INVALID_ARG, "W = %d outside [1, max_window = %d]", W, g->cfg.max_window);
  if (num_layers < 1 || num_layers > g->cfg.max_layers)
    return fail(GG_ERR_INVALID_ARG, "num_layers = %d outside [1, max_layers = %d]", num_layers, g->cfg.max_layers);
  for (int h = 0; h < num_layers; ++h)
    if (fanouts[h] < 1 || fanouts[h] > GG_MAX_FANOUT)
      return fail(GG_ERR_INVALID_ARG, "fanouts[%d] = %d outside [1, %d]", h, fanouts[h], GG_MAX_FANOUT);
  if (batch_offsets[0] != 0) return fail(GG_ERR_INVALID_ARG, "batch_offsets[0] must be 0");
  for (int b = 0; b < W; ++b) {
    const int64_t n = batch_offsets[b + 1] - batch_offsets[b];
    if (n < 1 || n > g->cfg.max_batch)
      return fail(GG_ERR_INVALID_ARG, "batch %d has %lld seeds; must be in [1, max_batch = %d]", b, (long long)n, g->cfg.max_batch);
  }
  const int64_t S = batch_offsets[W];
  for (int64_t i = 0; i < S; ++i)
    if (seeds[i] < 0 || seeds[i] >= g->N) return fail(GG_ERR_INVALID_ARG, "seed %lld = %d outside [0, N)", (long long)i, seeds[i]);
  if (find_window(g, window_id)) return fail(GG_ERR_STATE, "window %lld is already live", (long long)window_id);
  Window* w = &g->win[g->stage_counter % g->n_win];
  if (w->live) return fail(GG_ERR_STATE, "%d windows are live; release window %lld first", g->n_win, (long long)w->id);
  // shared scratch sized by (W, fanouts): grow only with both pipeline threads idle
  bool need_drain = false;
  gg_status rc = ensure_shared(g, W, num_layers, fanouts, &need_drain);
  if (rc != GG_OK) return rc;
  if (need_drain) {
    // growing frees and reallocates scratch the pipeline threads are using (and the miss buffers
    // already handed out in gg_batch_out): only with no window live.  Waiting here instead could
    // deadlock -- a queued window's phase B may itself be waiting for the caller to release the
    // window that holds its cache buffer.
    for (int s = 0; s < g->n_win; ++s)
      if (g->win[s].live)
        return fail(GG_ERR_STATE, "window %lld needs larger shared scratch (bigger W or fanouts) than any window staged "
                    "so far: release every live window first (window %lld is live)", (long long)window_id, (long long)g->win[s].id);
    {
      std::unique_lock<std::mutex> l(g->mu);
      g->cv_done.wait(l, [&] { return g->busy == 0; });
    }
    CU(cudaDeviceSynchronize());
    rc = ensure_shared(g, W, num_layers, fanouts, nullptr);
    if (rc != GG_OK) return rc;
  }
  tl("stage_call", window_id);
  {
    // identity and sequence number change under the lock: the selector thread reads them in its
    // wait predicate (is the cache slot's tenant still the live window n_cs stages back?)
    std::lock_guard<std::mutex> l(g->mu);
    w->id = window_id; w->live = true; w->W = W; w->L = num_layers; w->first_batch = first_batch_index;
    w->seq = g->stage_counter;
    w->cs = &g->cslot[g->stage_counter % (uint64_t)g->n_cs];
    for (int h = 0; h < num_layers; ++h) w->fanouts[h] = fanouts[h];
    w->seeds.assign(seeds, seeds + S);
    w->boff.assign(batch_offsets, batch_offsets + W + 1);
    w->ms_wait = 0;
    w->enqueued = false; w->status = GG_OK; w->error.clear();
    g->jobs_a.push_back(w);
    g->busy += 1;
  }
  g->stage_counter += 1;
  g->cv_a.notify_one();
  g->cv_done.notify_all();
  return GG_OK;
}

gg_status gg_batch_info(gg_graph* g, int64_t window_id, int32_t b, gg_batch_out* out) {
  if (!g || !out) return fail(GG_ERR_INVALID_ARG, "null argument");
  Window* w = find_window(g, window_id);
  if (!w) return fail(GG_ERR_STATE, "window %lld is not live (never staged or already released)", (long long)window_id);
  if (b < 0 || b >= w->W) return fail(GG_ERR_INVALID_ARG, "batch_in_window = %d outside [0, %d)", b, w->W);
  gg_status rc = wait_enqueued(g, w);
  if (rc != GG_OK) return rc;
  fill_batch_out(w, b, out, g);
  return GG_OK;
}

gg_status gg_batch_gather(gg_graph* g, int64_t window_id, int32_t b, gg_batch_out* out, void* cuda_stream) {
  if (!g || !out) return fail(GG_ERR_INVALID_ARG, "null argument");
  Window* w = find_window(g, window_id);
  if (!w) return fail(GG_ERR_STATE, "window %lld is not live (never staged or already released)", (long long)window_id);
  if (b < 0 || b >= w->W) return fail(GG_ERR_INVALID_ARG, "batch_in_window = %d outside [0, %d)", b, w->W);
  if (!out->features || ((uintptr_t)out->features & 3)) return fail(GG_ERR_INVALID_ARG, "features must be a 4-byte aligned device buffer");
  gg_status rc = wait_enqueued(g, w);
  if (rc != GG_OK) return rc;
  if (b == 0) tl("gather0_call", window_id);
  const int n = w->n_front[w->L][b];
  if (out->features_capacity_rows < n)
    return fail(GG_ERR_CAPACITY, "features_capacity_rows = %lld < n_input = %d", (long long)out->features_capacity_rows, n);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (!w->gather_recorded) {
    // first gather of the window: the boundary wait of Alg. 1 l.5, timed on the caller's stream
    cudaEvent_t pw = g->prof.begin(st);
    CU(cudaStreamWaitEvent(st, w->ready, 0));
    g->prof.end(st, pw, GG_PROF_WAIT, 0);
  } else {
    CU(cudaStreamWaitEvent(st, w->ready, 0));
  }
  GatherLaunch G;
  G.nodes = w->nodes.p + (int64_t)b * w->node_pitch; G.n = n; G.slot_of = w->cs->slot_map;
  G.local_base = g->store.base[g->R.local]; G.local_stride = g->store.stride;
  G.cache_base = w->cs->cache; G.cache_stride = g->rb;
  G.out = (uint8_t*)out->features; G.rb = g->rb; G.R = g->R; G.store = g->store;
  G.may_miss = w->may_miss;
  G.miss_tmp_pos = g->miss_tmp_pos.p; G.miss_tmp_id = g->miss_tmp_id.p; G.tile_miss = g->tile_miss.p;
  G.miss_pos = g->miss_pos.p; G.miss_id = g->miss_id.p; G.n_miss = g->n_miss.p;
  G.counters = w->counters.p + (int64_t)b * (2 + GG_MAX_PARTS);
  G.miss_total = g->miss_total.p;
  G.miss_over_link = false;
  for (int m = 0; m < g->R.P; ++m)
    if (m != g->R.local && g->R.lo[m] < g->R.lo[m + 1] && !g->store_on_device[m]) G.miss_over_link = true;
  // one launch in four is bracketed: a timing event between every pair of back-to-back 50 us
  // kernels costs the step 6 % (the events serialise the stream), a quarter of them 1-2 %
  cudaEvent_t pe = (b & 3) == 1 || w->W < 4 ? g->prof.begin(st) : nullptr;
  launch_gather(st, G);
  g->prof.end(st, pe, GG_PROF_GATHER, (int64_t)n * (2ll * g->rb + 8));
  if (w->may_miss) {
    pe = g->prof.begin(st);
    launch_miss_path(st, G);
    g->prof.end(st, pe, GG_PROF_MISS, 0);
  }
  // No event behind the gather: two records between every pair of back-to-back 50 us kernels cost
  // the stream 6-8 us per batch.  What later stages wait for (the arena's next tenant, the cache
  // buffer's next tenant) is recorded once per window, by gg_window_release on the caller's stream.
  w->gather_recorded = true;
  w->last_gather_stream = st;
  {
    int k = 0;
    while (k < w->n_gstreams && w->gstreams[k] != st) ++k;
    if (k == w->n_gstreams) {
      if (k < 4) w->gstreams[w->n_gstreams++] = st;
      else CU(cudaStreamSynchronize(st));     // a fifth distinct stream: nothing left to remember it by
    }
  }
  CU(cudaGetLastError());
  fill_batch_out(w, b, out, g);
  return GG_OK;
}

gg_status gg_window_release(gg_graph* g, int64_t window_id, void* cuda_stream) {
  if (!g) return fail(GG_ERR_INVALID_ARG, "null graph");
  Window* w = find_window(g, window_id);
  if (!w) return fail(GG_ERR_STATE, "window %lld is not live", (long long)window_id);
  // the pipeline threads must be done with the arena before it can be re-staged
  {
    std::unique_lock<std::mutex> l(g->mu);
    bool blocked = false;
    if (!w->enqueued)
      for (int s = 0; s < g->n_win; ++s)
        if (&g->win[s] != w && g->win[s].live && g->win[s].seq + (uint64_t)g->n_cs == w->seq) blocked = true;
    if (blocked) return fail(GG_ERR_STATE, "release the older live window first");
    g->cv_done.wait(l, [&] { return w->enqueued; });
  }
  // Everything the caller enqueued on `cuda_stream` so far may still read the window's blocks and
  // N_b (a consumer step behind the last gather, a device-to-host copy): the arena's next tenant
  // is sampled only behind this point of that stream.
  // ... and every gather of the window, on whatever stream it ran.  The join happens on a stream
  // of the library's own, so no caller stream is made to wait for another.
  cudaStream_t sj = g->side_join;
  CU(cudaEventRecord(w->ev_join[4], (cudaStream_t)cuda_stream));
  CU(cudaStreamWaitEvent(sj, w->ev_join[4], 0));
  for (int k = 0; k < w->n_gstreams; ++k) {
    if (w->gstreams[k] == (cudaStream_t)cuda_stream) continue;
    CU(cudaEventRecord(w->ev_join[k], w->gstreams[k]));
    CU(cudaStreamWaitEvent(sj, w->ev_join[k], 0));
  }
  CU(cudaEventRecord(w->consumer_done, sj));
  // the cache buffer's next tenant (window seq + n_cs) is built only behind the same point
  CU(cudaEventRecord(w->cs->gather_done, sj));
  // every record above succeeded: only now does the window's state change (a failed call -- an invalid
  // or destroyed stream -- returns with the window still live and its gather streams still remembered,
  // so a retry joins them again)
  w->n_gstreams = 0;
  w->cs->gather_recorded = true;
  {
    std::lock_guard<std::mutex> l(g->mu);
    w->consumer_recorded = true;
    w->live = false;
  }
  g->cv_done.notify_all();
  tl("release", window_id);
  return GG_OK;
}

gg_status gg_trace(gg_graph* g, int64_t window_id, gg_window_trace* out) {
  if (!g || !out) return fail(GG_ERR_INVALID_ARG, "null argument");
  Window* w = find_window(g, window_id);
  if (!w) return fail(GG_ERR_STATE, "window %lld is not live", (long long)window_id);
  gg_status rc = wait_enqueued(g, w);
  if (rc != GG_OK) return rc;
  CU(cudaEventSynchronize(w->ready));
  resolve_timing(w);
  if (w->gather_recorded) CU(cudaStreamSynchronize(w->last_gather_stream));   // the per-batch counters are final
  out->W = w->W; out->num_parts = g->R.P;
  out->n_access = w->n_access; out->n_unique = w->n_unique; out->n_unique_remote = w->n_remote;
  out->n_hot = w->n_hot; out->carried_rows = w->n_carry; out->bulk_copies = w->bulk_copies;
  for (int m = 0; m < GG_MAX_PARTS; ++m) {
    out->staged_rows[m] = w->staged[m];
    out->bulk_rows[m] = w->bulk[m];
    out->bulk_bytes[m] = w->bulk[m] * g->rb;
  }
  std::vector<int32_t> c((size_t)w->W * (2 + GG_MAX_PARTS));
  CU(cudaMemcpy(c.data(), w->counters.p, c.size() * sizeof(int32_t), cudaMemcpyDeviceToHost));
  for (int b = 0; b < w->W; ++b) {
    const int32_t* r = c.data() + (size_t)b * (2 + GG_MAX_PARTS);
    if (out->n_input) out->n_input[b] = w->n_front[w->L][b];
    if (out->hit_local) out->hit_local[b] = r[0];
    if (out->hit_cache) out->hit_cache[b] = r[1];
    if (out->miss) for (int m = 0; m < g->R.P; ++m) out->miss[b * g->R.P + m] = r[2 + m];
  }
  out->ms_sample = w->ms_sample; out->ms_unique = w->ms_unique; out->ms_select = w->ms_select;
  out->ms_pack_host = w->ms_pack; out->ms_h2d = w->ms_h2d; out->ms_carry = w->ms_carry;
  out->ms_stage_total = w->ms_total; out->ms_boundary_wait = w->ms_wait;
  return GG_OK;
}

gg_status gg_window_export(gg_graph* g, int64_t window_id, int32_t what, int32_t* out, int64_t capacity, int64_t* n_out) {
  if (!g || !n_out || (!out && capacity > 0)) return fail(GG_ERR_INVALID_ARG, "null argument");
  Window* w = find_window(g, window_id);
  if (!w) return fail(GG_ERR_STATE, "window %lld is not live", (long long)window_id);
  gg_status rc = wait_enqueued(g, w);
  if (rc != GG_OK) return rc;
  CU(cudaEventSynchronize(w->ready));
  const int32_t* src = nullptr;
  int64_t n = 0;
  switch (what) {
    case 0: src = w->uniq.p; n = w->n_unique; break;
    case 1: src = w->cnt.p; n = w->n_unique; break;
    case 2: src = w->cs->hot.p; n = w->n_hot; break;
    case 3: src = w->req_ids.p; n = w->n_delta; break;
    case 4: src = w->carry_ids.p; n = w->n_carry; break;
    default: return fail(GG_ERR_INVALID_ARG, "what = %d", what);
  }
  *n_out = n;
  if (capacity < n) return fail(GG_ERR_CAPACITY, "capacity %lld < %lld", (long long)capacity, (long long)n);
  if (n > 0) CU(cudaMemcpy(out, src, (size_t)n * sizeof(int32_t), cudaMemcpyDeviceToHost));
  return GG_OK;
}

gg_status gg_cache_read(gg_graph* g, int64_t window_id, const int32_t* ids, int64_t n, void* out) {
  if (!g || !ids || !out) return fail(GG_ERR_INVALID_ARG, "null argument");
  Window* w = find_window(g, window_id);
  if (!w) return fail(GG_ERR_STATE, "window %lld is not live", (long long)window_id);
  gg_status rc = wait_enqueued(g, w);
  if (rc != GG_OK) return rc;
  CU(cudaEventSynchronize(w->ready));
  for (int64_t i = 0; i < n; ++i) {
    if (ids[i] < 0 || ids[i] >= g->N) return fail(GG_ERR_INVALID_ARG, "id out of range");
    int32_t s = -1;
    CU(cudaMemcpy(&s, w->cs->slot_map + ids[i], sizeof(int32_t), cudaMemcpyDeviceToHost));
    if (s < 0) return fail(GG_ERR_INVALID_ARG, "id %d is not cached in window %lld", ids[i], (long long)window_id);
    CU(cudaMemcpy((uint8_t*)out + i * g->rb, w->cs->cache + (int64_t)s * g->rb, (size_t)g->rb, cudaMemcpyDeviceToHost));
  }
  return GG_OK;
}

gg_status gg_profile_enable(gg_graph* g, int32_t on) {
  if (!g) return fail(GG_ERR_INVALID_ARG, "null graph");
  CU(cudaDeviceSynchronize());
  g->prof.clear();
  CU(cudaMemset(g->miss_total.p, 0, sizeof(unsigned long long)));
  std::lock_guard<std::mutex> l(g->prof.m);
  g->prof.on = on != 0;
  return GG_OK;
}

gg_status gg_profile_get(gg_graph* g, gg_profile* out) {
  if (!g || !out) return fail(GG_ERR_INVALID_ARG, "null argument");
  CU(cudaDeviceSynchronize());
  g->prof.resolve();
  // a-8 moves a device-side number of rows per batch: the kernels add them up, 2 * rb bytes per row
  unsigned long long miss_rows = 0;
  CU(cudaMemcpy(&miss_rows, g->miss_total.p, sizeof miss_rows, cudaMemcpyDeviceToHost));
  std::lock_guard<std::mutex> l(g->prof.m);
  g->prof.bytes[GG_PROF_MISS] = (int64_t)miss_rows * 2 * g->rb;
  for (int k = 0; k < GG_PROF_KINDS; ++k) {
    out->ms[k] = g->prof.ms[k];
    out->regions[k] = g->prof.regions[k];
    out->bytes[k] = g->prof.bytes[k];
  }
  return GG_OK;
}

uint64_t gg_launch_count(void) { return (uint64_t)g_launches.load(); }

gg_status gg_sampler_stats(uint64_t* keys, uint64_t* rows, uint64_t* fallbacks) {
  CU(cudaDeviceSynchronize());
  unsigned long long v[4] = {0, 0, 0, 0};
  sampler_stats(v);
  CU(cudaGetLastError());
  if (keys) *keys = v[0];
  if (rows) *rows = v[1];
  if (fallbacks) *fallbacks = v[2] + v[3];
  return GG_OK;
}

gg_status gg_debug_sampler(int32_t rank_shift, float want_add) {
  if (rank_shift < 0 || rank_shift > 31) return fail(GG_ERR_INVALID_ARG, "rank_shift must be in [0, 31]");
  CU(cudaDeviceSynchronize());
  CU(sampler_debug(rank_shift, want_add));
  return GG_OK;
}

gg_status gg_sampler_tune(int32_t single_bins, int32_t warp_bin, int32_t hub_bin) {
  if (single_bins < 28 || single_bins > 128 || warp_bin < 0 || warp_bin > 128 || hub_bin < 28 || hub_bin > 128)
    return fail(GG_ERR_INVALID_ARG, "single_bins and hub_bin must be in [28, 128] (rows below degree 128 are one chunk), warp_bin in [0, 128]");
  CU(cudaDeviceSynchronize());
  CU(sampler_tune(single_bins, warp_bin, hub_bin));
  return GG_OK;
}

gg_status gg_key_peak(int32_t ctas_per_sm, int32_t keys_per_lane, int32_t reps, double* keys_per_s, uint32_t* fold) {
  if (!keys_per_s) return fail(GG_ERR_INVALID_ARG, "null argument");
  if (ctas_per_sm < 1 || ctas_per_sm > 8 || keys_per_lane < 32 || reps < 1 || reps > 1000)
    return fail(GG_ERR_INVALID_ARG, "ctas_per_sm in [1,8], keys_per_lane >= 32, reps in [1,1000]");
  CU(key_peak(nullptr, ctas_per_sm, keys_per_lane / 32, reps, keys_per_s, fold));
  return GG_OK;
}

gg_status gg_cache_reset(gg_graph* g) {
  if (!g) return fail(GG_ERR_INVALID_ARG, "null graph");
  for (int s = 0; s < g->n_win; ++s)
    if (g->win[s].live) return fail(GG_ERR_STATE, "release every window before gg_cache_reset");
  {
    std::unique_lock<std::mutex> l(g->mu);
    g->cv_done.wait(l, [&] { return g->busy == 0; });
  }
  CU(cudaDeviceSynchronize());
  for (int s = 0; s < g->n_cs; ++s) {
    CacheSlot& c = g->cslot[s];
    launch_slots_clear(g->side_b, c.hot.p, (int)c.n_cached, c.slot_map);
    c.n_cached = 0;
    c.tenant = nullptr;
  }
  CU(cudaStreamSynchronize(g->side_b));
  g->prev_cs = nullptr;
  return GG_OK;
}

}  // extern "C"

// =============================== NEXT-1: gg_simulate =========================================
namespace gg {
// hot-set threshold t and quota of count == t nodes from the histogram of remote counts (a-4)
static void hot_threshold(const int32_t* hist, int64_t n_remote, int64_t n_hot_eff, int64_t* n_hot,
                          int32_t* thr, uint32_t* quota) {
  *thr = 0;
  *quota = 0;
  if (n_remote <= n_hot_eff) {
    *n_hot = n_remote;
    return;
  }
  *n_hot = n_hot_eff;
  int64_t above = 0;
  int t;
  for (t = 255; t >= 1; --t) {
    if (above + hist[t] > *n_hot) break;
    above += hist[t];
  }
  *thr = t;
  *quota = (uint32_t)(*n_hot - above);
}
}  // namespace gg

extern "C" gg_status gg_simulate(gg_graph* g, const int32_t* seeds, const int64_t* batch_offsets, int32_t B,
                                 uint64_t first_batch_index, const int32_t* fanouts, int32_t num_layers,
                                 const int32_t* Ws, int32_t nW, const gg_energy_model* model,
                                 gg_sim_result* out, int32_t* best, int64_t* delta_out, int64_t* miss_out) {
  if (!g || !seeds || !batch_offsets || !fanouts || !Ws || !model || !out)
    return fail(GG_ERR_INVALID_ARG, "null argument");
  if (B < 1 || nW < 1) return fail(GG_ERR_INVALID_ARG, "B and nW must be >= 1");
  if (num_layers < 1 || num_layers > g->cfg.max_layers)
    return fail(GG_ERR_INVALID_ARG, "num_layers = %d outside [1, max_layers = %d]", num_layers, g->cfg.max_layers);
  for (int h = 0; h < num_layers; ++h)
    if (fanouts[h] < 1 || fanouts[h] > GG_MAX_FANOUT)
      return fail(GG_ERR_INVALID_ARG, "fanouts[%d] = %d outside [1, %d]", h, fanouts[h], GG_MAX_FANOUT);
  for (int i = 0; i < nW; ++i)
    if (Ws[i] < 1 || Ws[i] > g->cfg.max_window)
      return fail(GG_ERR_INVALID_ARG, "Ws[%d] = %d outside [1, max_window = %d]", i, Ws[i], g->cfg.max_window);
  if (batch_offsets[0] != 0) return fail(GG_ERR_INVALID_ARG, "batch_offsets[0] must be 0");
  for (int b = 0; b < B; ++b) {
    const int64_t n = batch_offsets[b + 1] - batch_offsets[b];
    if (n < 1 || n > g->cfg.max_batch)
      return fail(GG_ERR_INVALID_ARG, "batch %d has %lld seeds; must be in [1, max_batch = %d]", b, (long long)n, g->cfg.max_batch);
  }
  for (int64_t i = 0; i < batch_offsets[B]; ++i)
    if (seeds[i] < 0 || seeds[i] >= g->N) return fail(GG_ERR_INVALID_ARG, "seed %lld = %d outside [0, N)", (long long)i, seeds[i]);
  for (int s = 0; s < g->n_win; ++s)
    if (g->win[s].live) return fail(GG_ERR_STATE, "release every window before gg_simulate");
  {
    std::unique_lock<std::mutex> l(g->mu);
    g->cv_done.wait(l, [&] { return g->busy == 0; });
  }
  CU(cudaSetDevice(g->device));
  CU(cudaDeviceSynchronize());
  const int Wc = g->cfg.max_window, L = num_layers, P = g->R.P;
  gg_status rc = ensure_shared(g, Wc, L, fanouts, nullptr);
  if (rc != GG_OK) return rc;

  // ---- the trace: every batch sampled once, N_b lists kept in HBM -------------------------
  Window* w = &g->win[0];
  DevBuf<int32_t> db;
  std::vector<int64_t> off((size_t)B + 1, 0);
  for (int c0 = 0; c0 < B; c0 += Wc) {
    const int wc = std::min(Wc, B - c0);
    w->id = -1; w->W = wc; w->L = L; w->first_batch = first_batch_index + (uint64_t)c0;
    for (int h = 0; h < L; ++h) w->fanouts[h] = fanouts[h];
    w->seeds.assign(seeds + batch_offsets[c0], seeds + batch_offsets[c0 + wc]);
    w->boff.resize((size_t)wc + 1);
    for (int b = 0; b <= wc; ++b) w->boff[b] = batch_offsets[c0 + b] - batch_offsets[c0];
    rc = stage_a(g, w);
    if (rc != GG_OK) { db.release(); return rc; }
    for (int b = 0; b < wc; ++b) off[c0 + b + 1] = off[c0 + b] + w->n_front[L][b];
    const int64_t need = off[c0 + wc];
    if (need > db.n) {
      // grow: estimate the whole epoch from what has been seen, copy what is already there
      const int64_t est = (int64_t)((double)need / (c0 + wc) * B * 1.1) + 4096;
      int32_t* np_ = nullptr;
      if (cudaMalloc((void**)&np_, (size_t)std::max(est, need) * sizeof(int32_t)) != cudaSuccess) {
        cudaGetLastError();
        db.release();
        return fail(GG_ERR_OOM, "device allocation of the trace (%lld ids) failed", (long long)std::max(est, need));
      }
      if (db.p && off[c0] > 0) cudaMemcpyAsync(np_, db.p, (size_t)off[c0] * sizeof(int32_t), cudaMemcpyDeviceToDevice, g->side);
      cudaStreamSynchronize(g->side);
      db.release();
      db.p = np_;
      db.n = std::max(est, need);
    }
    for (int b = 0; b < wc; ++b)
      CU(cudaMemcpyAsync(db.p + off[c0 + b], w->nodes.p + (int64_t)b * w->node_pitch,
                         (size_t)w->n_front[L][b] * sizeof(int32_t), cudaMemcpyDeviceToDevice, g->side));
    CU(cudaStreamSynchronize(g->side));
  }
  int64_t max_n = 0;
  for (int b = 0; b < B; ++b) max_n = std::max(max_n, off[b + 1] - off[b]);

  // ---- replay per candidate W ---------------------------------------------------------------
  cudaStream_t st = g->side_b;
  int Kmax = 0;
  for (int i = 0; i < nW; ++i) Kmax = std::max(Kmax, (B + Ws[i] - 1) / Ws[i]);
  DevBuf<int64_t> off_dev;
  DevBuf<int32_t> delta_dev, counters_dev;
  DevBuf<gg_sim_result> res_dev;
  auto cleanup = [&]() { db.release(); off_dev.release(); delta_dev.release(); counters_dev.release(); res_dev.release(); };
  const int64_t n_cnt = (int64_t)B * (2 + GG_MAX_PARTS), n_del = (int64_t)Kmax * GG_MAX_PARTS;
  if (off_dev.ensure(B + 1) != cudaSuccess || delta_dev.ensure(n_del) != cudaSuccess ||
      counters_dev.ensure(n_cnt) != cudaSuccess || res_dev.ensure(nW) != cudaSuccess) {
    cudaGetLastError();
    cleanup();
    return fail(GG_ERR_OOM, "device allocation of the simulator's tallies failed");
  }
#define CUS(call)                                                                         \
  do {                                                                                    \
    cudaError_t e_ = (call);                                                              \
    if (e_ != cudaSuccess) {                                                              \
      cleanup();                                                                          \
      return fail(GG_ERR_CUDA, "%s:%d %s: %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
    }                                                                                     \
  } while (0)
  CUS(cudaMemcpyAsync(off_dev.p, off.data(), (size_t)(B + 1) * sizeof(int64_t), cudaMemcpyHostToDevice, st));
  std::vector<int32_t> h_cnt((size_t)n_cnt), h_del((size_t)n_del);
  int64_t delta_cursor = 0;
  for (int i = 0; i < nW; ++i) {
    const int W = Ws[i], K = (B + W - 1) / W;
    for (int s = 0; s < 2; ++s) {
      CacheSlot& c = g->cslot[s];
      launch_slots_clear(st, c.hot.p, (int)c.n_cached, c.slot_map);
      c.n_cached = 0;
      c.tenant = nullptr;
    }
    CUS(cudaMemsetAsync(counters_dev.p, 0, (size_t)n_cnt * sizeof(int32_t), st));
    CUS(cudaMemsetAsync(delta_dev.p, 0, (size_t)n_del * sizeof(int32_t), st));
    CacheSlot* prev = nullptr;
    for (int k = 0; k < K; ++k) {
      const int b0 = k * W, b1 = std::min(B, b0 + W);
      // a-3 over the window's slice of the trace
      launch_count_db(st, db.p, off[b0], off[b1], g->cnt8.p);
      launch_unique_count(st, g->cnt8.p, g->cnt_words, g->R, g->tiles32.p, g->stats.p, g->hist.p, w->uniq.p, w->cnt.p);
      launch_copy_words(st, g->h_small, g->stats.p, 1);
      launch_copy_words(st, g->h_small + 1, g->hist.p, 256);
      CUS(cudaStreamSynchronize(st));
      const int64_t n_unique = g->h_small[0];
      int64_t n_remote = 0, n_hot = 0;
      for (int c = 1; c < 256; ++c) n_remote += g->h_small[1 + c];
      int32_t thr;
      uint32_t quota;
      hot_threshold(g->h_small + 1, n_remote, g->n_hot_eff, &n_hot, &thr, &quota);
      // a-4 / a-5 against the previous cache state
      CacheSlot* cs = &g->cslot[k & 1];
      launch_slots_clear(st, cs->hot.p, (int)cs->n_cached, cs->slot_map);
      cs->n_cached = 0;
      if (n_hot > 0) {
        launch_hot_select(st, w->uniq.p, w->cnt.p, (int)n_unique, g->R, thr, quota, g->tiles64.p, g->total64.p, cs->hot.p);
        const int carry = (g->cfg.carry_over && prev) ? 1 : 0;
        launch_delta_split(st, cs->hot.p, (int)n_hot, g->R, prev ? prev->slot_map : nullptr, carry, g->tiles32_b.p,
                           g->n_delta_dev.p, g->owner_cnt.p, cs->slot_map, w->req_ids.p, w->carry_src.p, w->carry_ids.p);
        cs->n_cached = n_hot;
        CUS(cudaMemcpyAsync(delta_dev.p + (int64_t)k * GG_MAX_PARTS, g->owner_cnt.p + GG_MAX_PARTS,
                            GG_MAX_PARTS * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
      }
      // Alg. 1 l.11-12 as counts
      launch_classify(st, db.p, off_dev.p, b0, b1 - b0, max_n, cs->slot_map, g->R, counters_dev.p);
      prev = cs;
    }
    launch_sim_events(st, delta_dev.p, counters_dev.p, K, B, W, *model, P, g->rb, res_dev.p + i);
    if (delta_out) {
      CUS(cudaMemcpyAsync(h_del.data(), delta_dev.p, (size_t)K * GG_MAX_PARTS * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
      CUS(cudaStreamSynchronize(st));
      for (int k = 0; k < K; ++k)
        for (int m = 0; m < P; ++m) delta_out[delta_cursor + (int64_t)k * P + m] = h_del[(size_t)k * GG_MAX_PARTS + m];
    }
    delta_cursor += (int64_t)K * P;
    if (miss_out) {
      CUS(cudaMemcpyAsync(h_cnt.data(), counters_dev.p, (size_t)n_cnt * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
      CUS(cudaStreamSynchronize(st));
      for (int b = 0; b < B; ++b)
        for (int m = 0; m < P; ++m)
          miss_out[((int64_t)i * B + b) * P + m] = h_cnt[(size_t)b * (2 + GG_MAX_PARTS) + 2 + m];
    }
  }
  CUS(cudaMemcpyAsync(out, res_dev.p, (size_t)nW * sizeof(gg_sim_result), cudaMemcpyDeviceToHost, st));
  for (int s = 0; s < 2; ++s) {
    CacheSlot& c = g->cslot[s];
    launch_slots_clear(st, c.hot.p, (int)c.n_cached, c.slot_map);
    c.n_cached = 0;
    c.tenant = nullptr;
  }
  g->prev_cs = nullptr;
  CUS(cudaStreamSynchronize(st));
  CUS(cudaGetLastError());
#undef CUS
  cleanup();
  int bi = 0;
  for (int i = 1; i < nW; ++i)
    if (out[i].e_phy < out[bi].e_phy) bi = i;
  if (best) *best = bi;
  return GG_OK;
}

extern "C" gg_status gg_rank_calibrate(const double* z, const double* e_gt, int32_t n, int32_t F, double lambda_,
                                       double lr, int32_t iters, double* beta, double* gamma, double* loss) {
  if (!e_gt || !gamma || !loss || (F > 0 && (!z || !beta))) return fail(GG_ERR_INVALID_ARG, "null argument");
  if (n < 1 || n > 64 || F < 0 || F > 16 || iters < 0)
    return fail(GG_ERR_INVALID_ARG, "n must be in [1,64], F in [0,16], iters >= 0");
  CU(rank_calibrate(z, e_gt, n, F, lambda_, lr, iters, beta, gamma, loss));
  return GG_OK;
}

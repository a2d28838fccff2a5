/* greengnn.h -- C ABI of the B200-native hot path of GreenGNN's runtime phase
 * (arxiv/paper_2606_02916): per-window hot-set staging for sampling-based GNN training.
 *
 * Citations are /root/reference/PAPER.md line numbers (section / algorithm in brackets)
 * and DESIGN.md readings S1..S21 where the paper is silent.
 *
 * For each window k of W consecutive mini-batches (PAPER.md:130 [Sec. IV-A]: "partitions
 * the epoch into ceil(B/W) windows") the library
 *   a-1/a-2  samples every batch's multi-layer blocks with a deterministic keyed
 *            selection ("deterministic neighbor sampling ... seeds are
 *            fixed"); N_b = the outermost frontier ("N_b is the set of nodes
 *            whose features batch b requires");
 *   a-3      takes the window's unique union U_k with access counts c_k(u) over the trace
 *            T = {(b,u) : u in N_b};
 *   a-4      selects the hot set H_k = the n_hot most frequently accessed REMOTE nodes
 *            (PAPER.md:130);
 *   a-5      forms per owner m the rebuild delta Delta_{k,m} = (H_k n N_m) \ (C_{k-1} n N_m)
 *             as one packed, ascending ID list per owner;
 *   a-6      stages those rows with ONE bulk transfer per owner (PAPER.md:34,192 [Sec. IV-C]
 *            "one bulk RPC per partition owner") from the owner's pinned host store into an
 *            HBM cache, on the library's side stream, overlapped with window k-1's batches
 *            (Alg. 1 l.8: PREFETCHER.WARMCACHE(H_{k+1} \ C), "parallel with
 *            training"); C_k = H_k;
 *   a-7/a-8  serves each batch: cached features for N_b n H_k, residual misses
 *            M_b = N_b \ H_k fetched on demand (Alg. 1 l.11-14), assembling
 *            the dense feature tensor X_b;
 *   a-9      exports the event counts the W-selection simulator consumes (Eqs. 1-2,
 *            per-owner |Delta_{k,m}|, |M_{b,m}| and their indicators).
 *
 * Conventions
 *  - Node IDs are int32 (N < 2^31); CSR offsets int64.  Row v of the CSR lists the nodes v
 *    aggregates from.  Owner m owns the contiguous ID range [part_offsets[m],
 *    part_offsets[m+1]) (reading S18).  Feature rows are opaque bytes: nothing here
 *    computes in floating point.
 *  - "device" = memory the GPU of the current CUDA context addresses directly (cudaMalloc /
 *    torch CUDA tensor); "host" = ordinary host memory; "pinned" = page-locked host memory
 *    registered with CUDA (cudaHostAlloc / torch pin_memory) -- the stand-in for a remote
 *    owner's store.
 *  - blocks[0] is the hop out of the seeds (n_dst = batch size); blocks[L-1] is the outermost
 *    hop whose n_src = n_input.  fanouts[h] belongs to hop h counted outward (reading S2).
 *  - Every function returns a gg_status; none aborts or throws; on error no output is
 *    partially valid.  gg_last_error() gives the text for the calling thread's last failure.
 *  - One caller thread per gg_graph.  At most gg_config.max_live_windows (default 3) windows are
 *    live: k being served, k+1 whose cache is being staged, k+2 .. being sampled ahead (the two
 *    prefetch phases run on two library threads and their side streams; sampling does not depend
 *    on the cache, so it may run as far ahead as there are arenas -- on a short epoch that fills
 *    the GPU while the cold first window crosses the host link).  There are n = cache_buffers
 *    cache buffers: window k+n's cache is built only after window k is released, so asking for
 *    k+n's batches while k is live is GG_ERR_STATE.  Staging one window ahead (the literal loop of Alg. 1) is
 *    equally valid.
 */
#ifndef GREENGNN_H_
#define GREENGNN_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GG_MAX_LAYERS 8
#define GG_MAX_PARTS 16
#define GG_MAX_FANOUT 96   /* selection candidate buffer is 256 entries; see DESIGN.md a-1 */
#define GG_MAX_LIVE_WINDOWS 16
#define GG_MAX_CACHE_BUFFERS 4
#define GG_MAX_WINDOW 255  /* access counts are 8-bit lanes of a packed counter; W in {1..64} in PAPER.md:130 */

typedef struct gg_graph gg_graph; /* opaque */

typedef enum {
  GG_OK = 0,
  GG_ERR_INVALID_ARG = 1, /* null pointer, out-of-range value, wrong memory kind */
  GG_ERR_STATE = 2,       /* window never staged / already released / fourth live window */
  GG_ERR_CAPACITY = 3,    /* a caller buffer or a create-time cap is too small; nothing truncated */
  GG_ERR_OOM = 4,
  GG_ERR_CUDA = 5
} gg_status;

typedef enum { GG_F32 = 0, GG_BF16 = 1 } gg_dtype;

typedef struct {
  int64_t num_nodes, num_edges;
  const int64_t* indptr;  /* device, [num_nodes+1] */
  const int32_t* indices; /* device, [num_edges] */
} gg_csr;

typedef struct {
  int32_t num_parts, local_part;
  const int64_t* part_offsets; /* host, [num_parts+1], 0 = p[0] <= ... <= p[P] = num_nodes; copied */
} gg_owner_map;

typedef struct {
  int32_t dim;
  gg_dtype dtype;
  int64_t row_stride_bytes;    /* >= dim*sizeof(elt), multiple of 4 */
  const void* const* part_base; /* host array [P]: [local_part] = device pointer, others = pinned
                                   host pointers; row of node u of part m at
                                   part_base[m] + (u - part_offsets[m]) * row_stride_bytes */
} gg_feature_store;

typedef struct {
  uint64_t seed;          /* sampling seed (first argument of the key, reading S1) */
  int64_t n_hot;          /* hot-set budget n_hot; < 0 = unlimited */
  int32_t carry_over;     /* 1 = stage only Delta against C_{k-1}; 0 = full restage */
  int32_t max_layers;     /* <= GG_MAX_LAYERS */
  int32_t max_window;     /* <= GG_MAX_WINDOW */
  int32_t max_batch;      /* seeds per mini-batch */
  int64_t max_cache_rows; /* rows per cache buffer; <= 0 = every remote node.  The effective
                             budget is min(n_hot, max_cache_rows): an over-full hot set spills
                             to the miss path, it is never an error (reading S9) */
  int64_t max_input_nodes; /* cap on |N_b|; <= 0 = derived from the fanouts, capped at N */
  int32_t staging_mode;   /* 0 = owner-service pack on host threads + one cudaMemcpyAsync per
                             owner (BASELINE.json:north_star (d)); an owner whose store is DEVICE
                             memory (e.g. a peer GPU's HBM) is served by the pull kernel instead,
                             since host threads cannot read it;
                             1 = one GPU-initiated pull kernel per owner reading the pinned store */
  int32_t host_threads;   /* owner-service pack threads.  > 0: a hard cap, no pack ever runs on more threads (1 = on
                             the stager thread itself).  <= 0: 0.4 x hardware threads (in [2, 16]) while bulk copies
                             are queued -- the pack shares the host's DRAM with their DMA reads, see csrc/api.cu --
                             and up to 16 when the link is idle (cold or small windows).  Several ranks on one
                             host should pass an explicit share (dist.host_threads_for_rank) */
  int32_t cache_buffers;  /* HBM cache buffers (+ slot maps) in rotation, window k uses k mod n.  2 = the
                             ping-pong a literal Alg. 1 needs; with 2, window k's hot set can only be
                             selected after window k-2's gathers have finished, and that chain
                             (gathers -> select -> pack -> copy) sets the pace; 3 takes it off the
                             critical path (measured: ~2 % on the products epoch).  <= 0 = 2, clamped to [2, GG_MAX_CACHE_BUFFERS] */
  int32_t max_live_windows; /* window arenas = how far gg_window_stage may run ahead of the window
                               being served: k served, k+1 staged, k+2 .. k+n-1 sampled ahead (their
                               cache is still built one window ahead, Alg. 1 l.8); <= 0 = 3,
                               clamped to [3, GG_MAX_LIVE_WINDOWS] */
} gg_config;

/* Builds the handle.  Borrows indptr / indices / part_base pointers (caller keeps them alive
 * and unmodified until gg_graph_destroy); copies part_offsets.  Verifies memory kinds with
 * cudaPointerGetAttributes (GG_ERR_INVALID_ARG otherwise).  Allocates slot maps, cache
 * buffers, the side stream and the prefetch thread.  Uses the current CUDA device. */
gg_status gg_graph_create(const gg_csr* csr, const gg_owner_map* owners,
                          const gg_feature_store* store, const gg_config* cfg, gg_graph** out);
gg_status gg_graph_destroy(gg_graph* g);

/* Alg. 1 l.7-9: hands window `window_id` to the prefetcher.  Asynchronous:
 * returns after copying the arguments; the prefetch thread samples the W batches (a-1, a-2),
 * builds U_k / H_k / Delta (a-3..a-5) and stages (a-6) on the library's side stream.
 *   seeds          host int32, concatenated seed IDs of the W batches (distinct inside a batch)
 *   batch_offsets  host int64 [W+1], batch i = seeds[batch_offsets[i] .. batch_offsets[i+1])
 *   first_batch_index  global index of the window's first batch inside the epoch; batch i is
 *                  keyed with first_batch_index+i (reading S7: epoch is not hashed)
 *   fanouts        host int32 [num_layers], hop order outward from the seeds, 1..GG_MAX_FANOUT
 * Errors: INVALID_ARG (nulls, W<1 or >max_window, L<1 or >max_layers, a batch larger than
 * max_batch or empty window, seed outside [0,N)), STATE (max_live_windows already live,
 * window_id already live, or the window needs larger shared scratch -- a bigger W or bigger
 * fanouts than any window staged so far -- while other windows are live: release them first),
 * CAPACITY (caps derived from fanouts exceed int32 indexing).  A frontier that outgrows
 * max_input_nodes is reported as CAPACITY by the window's first gg_batch_info / gg_batch_gather;
 * the window then holds no valid output and the graph stays usable after its release. */
gg_status gg_window_stage(gg_graph* g, int64_t window_id, uint64_t first_batch_index,
                          const int32_t* seeds, const int64_t* batch_offsets, int32_t W,
                          const int32_t* fanouts, int32_t num_layers);

typedef struct {
  int32_t n_dst, n_src, n_edge;
  const int32_t* indptr;    /* device [n_dst+1], 0-based inside the block */
  const int32_t* src_local; /* device [n_edge], index into the batch's node list */
  const int32_t* src_global; /* device [n_edge], global IDs in ascending edge position */
} gg_block;

typedef struct {
  int32_t num_layers;
  gg_block blocks[GG_MAX_LAYERS]; /* hop order */
  int32_t n_input;
  const int32_t* input_nodes; /* device [n_input] = N_b; feature row i belongs to input_nodes[i] */
  void* features;             /* IN: caller-owned device buffer, row-major, row pitch = dim*elt */
  int64_t features_capacity_rows; /* IN */
  /* miss list M_b in ascending position.  ONE set of buffers per gg_graph: valid from the point of
   * the gather's stream where this gather's work completes until the NEXT gg_batch_gather on this
   * graph is enqueued, whose kernels overwrite them in stream order (work enqueued on the same
   * stream between the two gathers reads them safely; another stream must be ordered by the caller) */
  const int32_t* miss_pos;  /* device [n_input] capacity */
  const int32_t* miss_id;   /* device */
  const int32_t* n_miss;    /* device scalar */
} gg_batch_out;

/* Blocks until the prefetcher has finished ENQUEUING window_id (the brief wait of Alg. 1 l.5,
 * PAPER.md:194), then fills sizes and device pointers of batch `batch_in_window`.  Pointers
 * stay valid until gg_window_release.  Does not touch `features*`. */
gg_status gg_batch_info(gg_graph* g, int64_t window_id, int32_t batch_in_window, gg_batch_out* out);

/* Alg. 1 l.11-14.  Asynchronous on `cuda_stream` (a cudaStream_t; NULL = default stream): makes
 * the stream wait for the window's cache-ready event, gathers X_b (local rows from the HBM
 * store, hot rows through the ID->slot map from the cache, a-7), compacts the misses and fills
 * them from the owners' pinned stores (a-8).  Fills `out` like gg_batch_info.
 * Errors: STATE, CAPACITY (features_capacity_rows < n_input), INVALID_ARG (features null or
 * not 4-byte aligned). */
gg_status gg_batch_gather(gg_graph* g, int64_t window_id, int32_t batch_in_window,
                          gg_batch_out* out, void* cuda_stream);

/* Ends the window's life: its blocks, N_b lists and miss lists may be overwritten by a later
 * window, its cache buffer becomes reusable.  The call does not block on the GPU; the library
 * orders the reuse behind
 *   (1) every gg_batch_gather already enqueued for the window (on whatever stream it ran), and
 *   (2) everything enqueued so far on `cuda_stream` (a cudaStream_t; NULL = default stream): the
 *       stream on which the CALLER's last use of the window's device pointers was issued -- a
 *       consumer step behind the last gather (gg_sage_step), a device-to-host copy of the blocks.
 * A consumer that reads the window's pointers on some other stream must make `cuda_stream` wait
 * for that stream (cudaStreamWaitEvent) before the release, or synchronise it.  The caller's own
 * features buffer is not covered: it belongs to the caller.
 * `cuda_stream` and every stream a gg_batch_gather of this window ran on must still exist when the
 * window is released (the library records an event on each).  If a record fails (GG_ERR_CUDA: invalid
 * or destroyed stream) nothing has changed: the window is still live and the call can be repeated. */
gg_status gg_window_release(gg_graph* g, int64_t window_id, void* cuda_stream);

typedef struct {
  int32_t W, num_parts;
  int64_t n_access;        /* sum_b |N_b| = |T restricted to the window| */
  int64_t n_unique;        /* |U_k| */
  int64_t n_unique_remote; /* |R_k| */
  int64_t n_hot;           /* |H_k| */
  int64_t carried_rows;    /* |H_k n C_{k-1}| (0 when carry_over = 0) */
  int64_t staged_rows[GG_MAX_PARTS]; /* |H_k n N_m| */
  int64_t bulk_rows[GG_MAX_PARTS];   /* |Delta_{k,m}|; 0 => no transfer issued (Eq. 1 indicator) */
  int64_t bulk_bytes[GG_MAX_PARTS];
  int32_t bulk_copies;     /* transfers issued = #owners with Delta != empty */
  /* per batch, caller-provided host arrays (may be NULL to skip) */
  int32_t* n_input;   /* [W] */
  int32_t* hit_local; /* [W] */
  int32_t* hit_cache; /* [W] */
  int32_t* miss;      /* [W*num_parts], miss[b*num_parts+m] = |M_{b,m}| (Eq. 2) */
  /* timings in ms, informational (not parity-checked) */
  float ms_sample, ms_unique, ms_select, ms_pack_host, ms_h2d, ms_carry, ms_stage_total;
  float ms_boundary_wait; /* host time gg_batch_info/gather spent waiting for this window */
} gg_window_trace;

/* Synchronises the window's staging and every gather enqueued so far for it, then fills `out`.
 * Per-batch hit/miss counters of batches not gathered yet are 0. */
gg_status gg_trace(gg_graph* g, int64_t window_id, gg_window_trace* out);

/* Parity / simulator export of the window's lists to HOST buffers (synchronises staging).
 * what: 0 = uniq (U_k ascending), 1 = cnt (c_k aligned with uniq), 2 = hot (H_k ascending),
 *       3 = request IDs (Delta_{k,m} ascending, owners ascending, concatenated),
 *       4 = carried IDs (ascending).
 * Writes min(n, capacity) int32 values and stores n in *n_out; CAPACITY if capacity < n. */
gg_status gg_window_export(gg_graph* g, int64_t window_id, int32_t what, int32_t* out,
                           int64_t capacity, int64_t* n_out);

/* Parity helper: reads back cache rows of the given global IDs for a staged window
 * (row at slot_of[u]); ids absent from H_k give GG_ERR_INVALID_ARG.  out: host, n*row_bytes. */
gg_status gg_cache_read(gg_graph* g, int64_t window_id, const int32_t* ids, int64_t n, void* out);

/* C <- empty (Alg. 1 l.1); requires no live window. */
gg_status gg_cache_reset(gg_graph* g);

/* The sampling key of reading S1, evaluated by the library's own hash (host function; parity
 * pin against tests/golden/keys.txt). */
uint64_t gg_key(uint64_t seed, uint64_t batch, uint64_t layer, uint64_t dst, uint64_t edge_pos);

/* Live measurement support (bench.py roofline leg).  When enabled, the library brackets its own
 * kernel groups with CUDA events ON THE STREAM THEY ARE LAUNCHED ON (caller's stream for the
 * gather and miss path, the side stream for everything else) and counts algorithmic bytes:
 *   GATHER  one k_gather launch per region (one launch in four is bracketed when W >= 4, so that
 *           the timing events do not serialise the caller's stream); bytes = |N_b| * (2*row_bytes + 8)
 *           of the bracketed launches
 *   MISS    miss compaction + fill;          bytes = misses * 2*row_bytes   (row over the host link + row written;
 *           the row count is accumulated on the device by the compaction kernel since the last gg_profile_enable)
 *   SAMPLE  count + scan + select of a hop;  bytes = 24*n_dst + 8*n_edge
 *   FRONTIER mark + word scan + emit + relabel of a hop; bytes = 8*n_edge + 4*n_new
 *   UNIQUE  counter compaction;              bytes = 4*n_access + 8*n_unique
 *   SELECT  hot select + delta split;        bytes = 12*n_unique
 *   STAGE_COPY the per-owner bulk transfers; bytes = sum |Delta_m| * row_bytes (host link)
 *   CARRY   carry-over D2D copy;             bytes = 2 * carried * row_bytes
 *   WAIT    GPU stall at a window boundary: time the caller's stream spends in the wait for the
 *           window's cache-ready event before its first gather (Alg. 1 l.5)
 * gg_profile_enable(g, on) clears the accumulators; gg_profile_get synchronises the device. */
#define GG_PROF_KINDS 9
enum { GG_PROF_GATHER = 0, GG_PROF_MISS = 1, GG_PROF_SAMPLE = 2, GG_PROF_FRONTIER = 3,
       GG_PROF_UNIQUE = 4, GG_PROF_SELECT = 5, GG_PROF_STAGE_COPY = 6, GG_PROF_CARRY = 7,
       GG_PROF_WAIT = 8 };
typedef struct {
  double ms[GG_PROF_KINDS];
  int64_t regions[GG_PROF_KINDS];
  int64_t bytes[GG_PROF_KINDS];
} gg_profile;
gg_status gg_profile_enable(gg_graph* g, int32_t on);
gg_status gg_profile_get(gg_graph* g, gg_profile* out);
/* number of kernels this library has launched in this process (all graphs) */
uint64_t gg_launch_count(void);

/* a-1 work counters, cumulative over the process (synchronises the device):
 *   keys      key evaluations the method asks for = sum of deg over sampled destinations with
 *             deg > fanout (one 64-bit SplitMix key per edge position, reading S1) -- the
 *             algorithmic ALU work of the sampler, the unit of bench.py's "alu" roofline;
 *   rows      destinations that needed a keyed selection (deg > fanout);
 *   fallbacks of those, hand-overs because a fast selection could not prove its result exact
 *             (candidate list overflow, fewer than fanout candidates under the threshold guess,
 *             or a tie in the high 32 key bits at the boundary): lane-per-row (or chunk) kernel -> warp
 *             kernel, plus warp kernel -> exact ballot/bisection path.
 * Any pointer may be NULL. */
gg_status gg_sampler_stats(uint64_t* keys, uint64_t* rows, uint64_t* fallbacks);

/* Degree cut-overs of the selection kernels (performance knobs; results are bit-exact for every
 * setting, tests/test_gpu_parity.py).  Keyed rows are binned by degree in quarter octaves, bin =
 * 4*floor(log2 deg) + the next two bits (bin 28 = degree 128, 36 = 512, 48 = 4096, 60 = 32768).  Rows
 * in bins below single_bins are selected by one lane each; rows in bins from warp_bin up to hub_bin
 * by one warp each; rows in bins [single_bins, warp_bin) and the hub rows in bins >= hub_bin are cut
 * into chunks of <= 128 edge positions, one lane per chunk, the candidates of a row merged through a
 * list in global memory.  Default (36, 36, 128): one lane per row below degree 512, one warp per row
 * above, no chunking (measured: chunking moves instructions one for one and adds the rank launch;
 * Large config with hubs of degree >= 32768 chunked: 290 vs 240 ms of sampling per epoch).
 * single_bins > hub_bin is accepted and treated as single_bins = hub_bin on the hops where hub rows exist
 * (hub rows are always chunked).
 * The candidate lists of the chunked schemes (8 bytes x ~28 per destination of a hop) are allocated only
 * while a setting that can use them is in force; after turning one on, the next gg_window_stage grows the
 * shared scratch and therefore needs every earlier window released (GG_ERR_STATE otherwise).
 * Process-wide; must not be called while a window is being staged.  Errors: INVALID_ARG for
 * single_bins or hub_bin outside [28, 128] (a row below degree 128 is always one chunk) or warp_bin
 * outside [0, 128]. */
gg_status gg_sampler_tune(int32_t single_bins, int32_t warp_bin, int32_t hub_bin);

/* The measured integer-ALU roofline of a-1 ("keys/s vs the peak of
 * a key-only micro-kernel measured on the same GPU").  Launches a kernel in which every lane
 * evaluates keys_per_lane (rounded down to a multiple of 32) consecutive SplitMix64 keys of reading
 * S1 from a register-resident state -- the high word of fmix, which is all the selection test
 * reads -- and folds them into one word: no candidate lists, no row logic, no memory traffic.
 * Grid = ctas_per_sm x SM count CTAs of 256 threads, `reps` timed launches after one warm-up, CUDA
 * events on the default stream.  Lane t of CTA c starts launch i (i = 0..reps-1) from the
 * state 0x9E37 + i + (256 c + t + 1) * 0x632BE59BD9B4E019 and evaluates the states x + gamma * k,
 * k = 0..keys_per_lane-1; *fold (host, may be NULL) receives the xor over all of them of the high
 * 32 bits of fmix before its last xor-shift (tests/test_gpu_parity.py recomputes it on the host).
 * Synchronous.  Errors: INVALID_ARG (null, ctas_per_sm outside [1,8], keys_per_lane < 32). */
gg_status gg_key_peak(int32_t ctas_per_sm, int32_t keys_per_lane, int32_t reps, double* keys_per_s,
                      uint32_t* fold);

/* Test knobs for the fallback logic of the selection kernel (tests/test_gpu_parity.py); results
 * must stay bit-exact for every setting.  rank_shift in [0,31]: the ranking compares only the
 * top 32-rank_shift key bits (forces ties); want_add: added to the number of candidates the
 * threshold guess aims for (large: list overflow; negative: too few candidates).
 * (0, 0.0f) restores the defaults.  Must not be called while a window is being staged. */
gg_status gg_debug_sampler(int32_t rank_shift, float want_add);

/* ---- NEXT-1: trace simulator + analytical energy model ----
 * Coefficients of PAPER.md:128 (the energy profiler's output), per owner m:
 *   eps_init[m] J per transfer; eps_payload(m,x) = eps_pay_a[m] + eps_pay_b[m]*x J for x > 0 rows
 *   and 0 for x = 0 ("a linear fit ... as a function of transfer size"; DESIGN.md
 *   reading S24); lam_* the latency surrogates in seconds, same form; bw_bytes_per_s the
 *   aggregate bandwidth ceiling; p_idle_w the accelerator's idle power.  Entries of the local
 *   owner are never used. */
typedef struct {
  double eps_init[GG_MAX_PARTS], eps_pay_a[GG_MAX_PARTS], eps_pay_b[GG_MAX_PARTS];
  double lam_init[GG_MAX_PARTS], lam_pay_a[GG_MAX_PARTS], lam_pay_b[GG_MAX_PARTS];
  double bw_bytes_per_s, p_idle_w;
} gg_energy_model;

/* One candidate W: event tallies of the single pass over the trace and Eqs. (1)-(3).
 *   rebuild_events = sum_k sum_m I[Delta_{k,m} != {}], rebuild_rows = sum |Delta_{k,m}|   (Eq. 1)
 *   miss_events    = sum_b sum_m I[M_{b,m} != {}],     miss_rows    = sum |M_{b,m}|       (Eq. 2)
 *   t_stall = sum over rebuild and miss events of max(slowest single-owner transfer,
 *             event bytes / BW) (Eq. 3 prose, reading S20); e_stall = p_idle * t_stall
 *   e_phy = (e_rebuild + e_miss) + e_stall; hit_ratio = hit_cache / (hit_cache + miss_rows)
 * z(W) of PAPER.md:182 = (rebuild_events, miss_events, t_stall, hit_ratio). */
typedef struct {
  int32_t W, n_windows;
  int64_t rebuild_events, miss_events, rebuild_rows, miss_rows;
  int64_t n_access, n_remote_access, hit_local, hit_cache;
  double e_rebuild, e_miss, t_stall, e_stall, e_phy, hit_ratio;
} gg_sim_result;

/* Samples the epoch's B mini-batches once (a-1/a-2; batch i keyed with first_batch_index+i),
 * keeps the trace T in HBM, and replays it for each candidate window size Ws[0..nW) with the
 * graph's n_hot / carry_over / owner map: window unique+count, hot-set select, rebuild delta
 * against the previous cache state (C_0 = {}), per-batch hit / miss classification -- no
 * feature row is moved.  out[i] receives candidate i; *best = index of the smallest e_phy
 * (W* = argmin, PAPER.md:186 with L(W) = 0; ties -> the earlier candidate).
 * Optional parity exports (host, may be NULL): delta_out[(sum of windows over candidates) * P]
 * = |Delta_{k,m}| candidate-major; miss_out[nW * B * P] = |M_{b,m}|.
 * seeds / batch_offsets / fanouts / Ws / model / out: host.  Synchronous; requires that no
 * window is live (GG_ERR_STATE otherwise) and leaves the cache state empty.
 * Errors: as gg_window_stage for the batch arguments; Ws[i] outside [1, max_window]. */
gg_status gg_simulate(gg_graph* g, const int32_t* seeds, const int64_t* batch_offsets, int32_t B,
                      uint64_t first_batch_index, const int32_t* fanouts, int32_t num_layers,
                      const int32_t* Ws, int32_t nW, const gg_energy_model* model,
                      gg_sim_result* out, int32_t* best, int64_t* delta_out, int64_t* miss_out);

/* ---- NEXT-3: rank calibration (Eq. 5) ------------------------------------------
 * Fits S(W) = beta^T z(W) + gamma_W to the measured order of n calibration window sizes by
 * fixed-step gradient descent (reading S26: the paper names no optimiser) from beta = gamma = 0 on
 *   L = sum_{i<j} log(1 + exp(-sigma_ij (S(W_j) - S(W_i)))) + lambda ||beta||^2,
 *   sigma_ij = sign(E_GT(W_j) - E_GT(W_i)) (pairs with equal E_GT contribute nothing).
 * z: host [n][F] row-major (the simulator's z(W), scaled by the caller), e_gt: host [n] measured
 * energies, iters steps of size lr.  Outputs (host): beta[F], gamma[n], *loss = L at the result.
 * L(W) of Eq. 4 is beta^T z(W) + gamma_W; E_net(W) = E_phy(W) + L(W).
 * Errors: INVALID_ARG for nulls, n outside [1,64], F outside [0,16], iters < 0. */
gg_status gg_rank_calibrate(const double* z, const double* e_gt, int32_t n, int32_t F, double lambda_,
                            double lr, int32_t iters, double* beta, double* gamma, double* loss);

/* ---- NEXT-4: the consumer the staging overlaps with (Alg. 1 l.15) ----------
 * GraphSAGE with the mean aggregator over the blocks gg_batch_gather returns, fp32:
 *   agg_i = mean of h_in[src_local[e]] over row i of the block (0 for an empty row)
 *   h_out_i = act(h_in[i] W_self + agg_i W_neigh + b), ReLU on every layer but the last
 * layer l consumes block num_layers-1-l (layer 0 reads the feature tensor X_b); the loss is the mean
 * softmax cross-entropy of the seeds against `labels`; parameters move by plain SGD (no dropout:
 * DESIGN.md reading S27).  dims: host [num_layers+1], dims[0] = feature dim (features must be
 * GG_F32), dims[num_layers] = classes; 1 <= dims[l] <= 128 for l < num_layers, dims[l+1] <= 64;
 * dims[0] may be up to 1024 when dims[1] <= 16 (the paper's 602-wide features into 16 hidden units).
 * w_self / w_neigh / bias: host arrays of num_layers pointers to row-major [dims[l]][dims[l+1]] /
 * [dims[l+1]] initial values (copied). */
typedef struct gg_sage gg_sage;
gg_status gg_sage_create(int32_t num_layers, const int32_t* dims, const float* const* w_self,
                         const float* const* w_neigh, const float* const* bias, gg_sage** out);
gg_status gg_sage_destroy(gg_sage* m);
/* One training step on `cuda_stream` (asynchronous): forward, loss, backward, SGD update.
 * batch: what gg_batch_gather filled (its features buffer must hold fp32 rows of dims[0]);
 * labels: device int32 [blocks[0].n_dst] in [0, classes); loss_out: device float, receives the
 * loss before the update (may be NULL).  The model's scratch grows on demand (that first call
 * synchronises).  Errors: INVALID_ARG (nulls, layer count or dims that do not match the batch). */
gg_status gg_sage_step(gg_sage* m, const gg_batch_out* batch, const int32_t* labels, float lr,
                       void* cuda_stream, float* loss_out);
/* Copies layer l's parameters to host arrays (synchronises the device). */
gg_status gg_sage_params(gg_sage* m, int32_t layer, float* w_self, float* w_neigh, float* bias);

/* ---- window unique + count without any device allocation -------------------------------------------
 * The same U_k / c_k as step a-3 (the distinct node IDs of the window's trace, ascending,
 * each with the number of times it is accessed), computed from ID lists the caller already holds on the
 * device -- for callers that cannot let a library allocate.  Typical cases: the process's own allocator
 * has taken all free HBM, so a cudaMalloc made here would fail; or the loop has other streams in flight
 * and must avoid cudaFree, which waits for the whole device.  This call never calls cudaMalloc, cudaFree
 * or any routine that allocates: its workspace (packed 8-bit counters, one per node ID, plus 512 partial
 * sums) is a fixed array of 4 MiB + 2 KiB compiled into the library, resident on every GPU that loads
 * libgreengnn.so until the process exits.  That fixed size is the limit: num_nodes <=
 * GG_STATIC_MAX_NODES (4,194,304); beyond it the call returns GG_ERR_CAPACITY and touches nothing
 * (gg_window_stage has no such limit).
 *   ids       device int32 [n_ids]: the node IDs accessed, in any order (e.g. the N_b lists of the
 *             window's batches, concatenated).  An ID may occur at most 255 times (N_b holds each node
 *             once, so this is the W <= GG_MAX_WINDOW rule); more than that corrupts neighbouring counts.
 *   num_nodes IDs are valid in [0, num_nodes); others are skipped and tallied in stats[1]
 *   uniq, cnt device int32 [capacity], caller-owned outputs: uniq ascending, cnt[i] = occurrences of uniq[i]
 *   stats     device int32 [2], caller-owned output: stats[0] = |U| (the number of entries written),
 *             stats[1] = IDs skipped.  If stats[0] > capacity NOTHING was written to uniq / cnt.
 *   cuda_stream  a cudaStream_t (NULL = default stream); the call is asynchronous on it.
 * The workspace is shared by all calls on a device and keeps the previous call's contents; every call
 * clears what it needs first, so back-to-back calls on one stream are independent.  Calls whose GPU
 * work can overlap (two streams without an ordering, two threads) race on it: order them yourself.
 * The first call on each device looks up the workspace's device address (and makes the CUDA runtime
 * load this module there); make that first call -- n_ids = 0 is enough -- during start-up, before any
 * stream capture begins.
 * Errors: INVALID_ARG (null pointer, negative size, num_nodes < 1), CAPACITY (num_nodes too large),
 * CUDA. */
#define GG_STATIC_MAX_NODES (1 << 22)
gg_status gg_unique_count_static(const int32_t* ids, int64_t n_ids, int64_t num_nodes, int32_t* uniq,
                                 int32_t* cnt, int64_t capacity, int32_t* stats, void* cuda_stream);

const char* gg_last_error(void);
const char* gg_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GREENGNN_H_ */

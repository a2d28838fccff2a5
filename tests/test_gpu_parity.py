"""GPU parity: the CUDA path through the C ABI vs the CPU oracle, bit-exact (all integer /
byte work; BASELINE.json:north_star).  Sizes span several tiles and ragged tails."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

from tests import parity_util as pu  # noqa: E402


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return "cuda:0"


def test_library_key_matches_golden_and_oracle(dev):
    from oracle import ggo
    from paper_2606_02916_b200 import binding
    for args in [(0, 0, 0, 0, 0), (42, 3, 1, 1234, 7), (0xDEADBEEF, (1 << 40) + 5, 2, 110999999, 19999)]:
        assert binding.gg_key(*args) == ggo.key(*args)


def test_key_peak_kernel_evaluates_the_methods_keys(dev):
    """The key-only micro-kernel behind bench.py's measured ALU roofline (gg_key_peak) folds exactly
    the keys of reading S1: host recomputation of the xor of every lane's 32 key words, with the
    oracle's fmix on a sample of the states."""
    from oracle import ggo
    from paper_2606_02916_b200 import binding
    rate, fold = binding.key_peak(ctas_per_sm=1, keys_per_lane=32, reps=1, with_fold=True)
    assert rate > 0
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    gamma, step = np.uint64(0x9E3779B97F4A7C15), np.uint64(0x632BE59BD9B4E019)
    with np.errstate(over="ignore"):
        gid = np.arange(1, sms * 256 + 1, dtype=np.uint64)
        x = (np.uint64(0x9E37) + gid * step)[:, None] + gamma * np.arange(32, dtype=np.uint64)[None, :]
        z = (x ^ (x >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
    zhi = (z >> np.uint64(32)).astype(np.uint32)
    assert fold == int(np.bitwise_xor.reduce(zhi.ravel()))
    for i, k in [(0, 0), (17, 5), (sms * 256 - 1, 31), (1000, 16)]:
        f = ggo.fmix(int(x[i, k]))                      # fmix = z ^ (z >> 31): the last step keeps the high word's upper 31 bits
        assert (f >> 32) == int(zhi[i, k]) ^ (int(zhi[i, k]) >> 31)


@pytest.mark.parametrize("n_hot,carry,mode", [(-1, 1, 0), (200, 1, 0), (200, 0, 0), (-1, 1, 1), (0, 1, 0)])
def test_tiny_one_window(workload, dev, n_hot, carry, mode):
    w = workload("tiny", dev)
    s = pu.check_epoch(w, W=4, n_hot=n_hot, carry_over=carry, staging_mode=mode)
    assert s["batches"] == 4 and s["windows"] == 1
    if n_hot == -1:
        assert s["misses"] == 0
    else:
        assert s["misses"] > 0


@pytest.mark.parametrize("W", [1, 4, 8])
@pytest.mark.parametrize("n_hot", [-1, 7500])
def test_small_full_epoch(workload, dev, W, n_hot):
    w = workload("small", dev)
    s = pu.check_epoch(w, W=W, n_hot=n_hot)
    assert s["batches"] == 10 and s["windows"] == -(-10 // W)


@pytest.mark.parametrize("cache_buffers,lookahead", [(3, 2), (3, 5), (4, 6), (2, 4)])
def test_small_more_cache_buffers_and_deeper_lookahead(workload, dev, cache_buffers, lookahead):
    """cache_buffers > 2 and sampling several windows ahead change the schedule, not the results."""
    w = workload("small", dev)
    pu.check_epoch(w, W=1, n_hot=7500, cache_buffers=cache_buffers, lookahead=lookahead)
    pu.check_epoch(w, W=2, n_hot=-1, carry_over=1, cache_buffers=cache_buffers, lookahead=lookahead)


def test_small_no_carry_and_pull_mode(workload, dev):
    w = workload("small", dev)
    pu.check_epoch(w, W=4, n_hot=-1, carry_over=0)
    pu.check_epoch(w, W=4, n_hot=7500, carry_over=1, staging_mode=1)
    pu.check_epoch(w, W=3, n_hot=-1, max_cache_rows=5000)      # cache cap spills to the miss path


@pytest.mark.parametrize("W", [1, 4])
def test_products_mini_three_layers(workload, dev, W):
    w = workload("products_mini", dev)
    pu.check_epoch(w, W=W, n_hot=-1)
    pu.check_epoch(w, W=W, n_hot=4500)


def test_dense_mini_high_degree_rows_and_8_byte_rows(workload, dev):
    # avg degree ~100, tail ~2000, fanout 25: exercises threshold selection; rb = 2408 is
    # only 8-byte aligned
    w = workload("dense_mini", dev)
    pu.check_epoch(w, W=4, n_hot=-1)
    pu.check_epoch(w, W=1, n_hot=600)


def test_large_mini_directed_bf16(workload, dev):
    w = workload("large_mini", dev)
    pu.check_epoch(w, W=4, n_hot=-1)
    pu.check_epoch(w, W=4, n_hot=11250, staging_mode=1)


@pytest.mark.parametrize("rank_shift,want_add", [(24, 0.0), (31, 0.0), (0, 400.0), (0, 120.0), (0, -30.0), (20, 40.0)])
def test_selection_fallback_paths_stay_exact(workload, dev, rank_shift, want_add):
    """The fast selection proves its own result (kept == fanout) or falls back to the exact path.
    The knobs force each fallback cause -- ties in the compared key bits, lane-list overflow,
    more than 128 candidates, fewer than fanout candidates -- and the blocks must not change."""
    from paper_2606_02916_b200 import binding
    w = workload("dense_mini", dev)
    before = binding.sampler_stats()
    binding.debug_sampler(rank_shift, want_add)
    try:
        pu.check_epoch(w, W=2, n_hot=-1, max_batches=2, check_features=False)
    finally:
        binding.debug_sampler(0, 0.0)
    after = binding.sampler_stats()
    assert after["rows"] > before["rows"] and after["keys"] > before["keys"]
    assert after["fallbacks"] > before["fallbacks"], "the knob did not reach the fallback path"


@pytest.mark.parametrize("fanouts", [[96, 40], [1, 1, 1], [16, 17], [3]])
def test_extreme_fanouts(workload, dev, fanouts):
    """GG_MAX_FANOUT (every row takes the warp kernel, ~122 candidates of the 128 the fast path
    holds), fanout 1, the thread/warp cut-over at fanout 16 / 17, and a single layer."""
    import dataclasses
    w = dataclasses.replace(workload("dense_mini", dev), fanouts=list(fanouts))
    pu.check_epoch(w, W=2, n_hot=-1, max_batches=2, check_features=False)
    pu.check_epoch(w, W=1, n_hot=300, max_batches=2)


def test_single_seed_batches_and_partial_last_window(workload, dev):
    """Batches of one seed, a window of one batch, and a last window shorter than W."""
    import dataclasses
    w0 = workload("small", dev)
    batches = [w0.batches[0][:1], w0.batches[1][:1], w0.batches[2][:7], w0.batches[3][:1], w0.batches[4][:2]]
    w = dataclasses.replace(w0, batches=batches)
    pu.check_epoch(w, W=2, n_hot=-1)
    pu.check_epoch(w, W=4, n_hot=50)
    pu.check_epoch(w, W=1, n_hot=0)


def test_max_window_255_counts_fill_the_8_bit_lanes(workload, dev):
    """W = GG_MAX_WINDOW = 255 batches that all contain the same seed: its access count is 255,
    the largest value the packed 8-bit counters hold; hot-set selection with a budget then has
    a 255-bin histogram to threshold."""
    import dataclasses
    w0 = workload("small", dev)
    hub = int(w0.batches[0][0])
    batches = [np.array([hub, int(w0.batches[(i // 1000) % 10][i % 1000 + 1])], np.int32) for i in range(255)]
    batches = [b if b[0] != b[1] else b[:1] for b in batches]
    w = dataclasses.replace(w0, batches=batches)
    s = pu.check_epoch(w, W=255, n_hot=2000)
    assert s["windows"] == 1 and s["batches"] == 255
    pu.check_epoch(w, W=128, n_hot=-1)


def _hub_workload(dev, seed=5):
    """A graph with four hubs of 33 k .. 150 k in-edges among 200 k nodes of degree 3 whose rows
    all contain a hub, so the hubs are destinations of hop 0 and of hop 1."""
    from paper_2606_02916_b200 import inputs
    rng = np.random.default_rng(seed)
    n = 200_000
    hub_deg = [33_000, 40_000, 70_000, 150_000]
    rows = []
    for h, d in enumerate(hub_deg):
        rows.append(np.sort(rng.choice(np.arange(4, n), size=d, replace=False)).astype(np.int32))
    small = np.stack([rng.integers(0, 4, n - 4), rng.integers(4, n, n - 4), rng.integers(4, n, n - 4)], axis=1)
    small = np.sort(small, axis=1).astype(np.int32)
    deg = np.concatenate([hub_deg, np.full(n - 4, 3)]).astype(np.int64)
    indptr = np.concatenate([[0], np.cumsum(deg)]).astype(np.int64)
    indices = np.concatenate(rows + [small.reshape(-1)]).astype(np.int32)
    po = np.array([0, n // 4, n // 2, 3 * n // 4, n], np.int64)
    dim = 8
    feat = rng.normal(size=(n, dim)).astype(np.float32)
    parts = []
    for m in range(4):
        t = torch.from_numpy(feat[po[m]:po[m + 1]].copy())
        parts.append(t.to(dev) if m == 0 else t.pin_memory())
    seeds = rng.permutation(np.arange(0, n))[:600].astype(np.int32)
    seeds[:4] = [0, 1, 2, 3]                                   # the hubs are seeds of batch 0 too
    batches = [seeds[i:i + 200].copy() for i in range(0, 600, 200)]
    return inputs.Workload(name="hubs", cfg={}, num_nodes=n, indptr=torch.from_numpy(indptr).to(dev),
                           indices=torch.from_numpy(indices).to(dev), part_offsets=po, local_part=0,
                           feat_parts=parts, dim=dim, dtype=torch.float32, batches=batches,
                           fanouts=[5, 4], seed=1234)


def test_hub_rows_of_1e5_edges(dev):
    from paper_2606_02916_b200 import binding
    w = _hub_workload(dev)
    pu.check_epoch(w, W=3, n_hot=-1)
    pu.check_epoch(w, W=1, n_hot=1000)
    # and the hand-over to the exact path when the proof fails on rows this long
    before = binding.sampler_stats()
    for rs, wa in [(28, 0.0), (0, 500.0), (0, -8.0)]:
        binding.debug_sampler(rs, wa)
        try:
            pu.check_epoch(w, W=3, n_hot=-1, check_features=False)
        finally:
            binding.debug_sampler(0, 0.0)
    assert binding.sampler_stats()["fallbacks"] > before["fallbacks"]


@pytest.mark.parametrize("single_bins,warp_bin,hub_bin", [(28, 48, 128), (28, 128, 128), (36, 48, 60), (28, 28, 128), (128, 128, 128),
                                                          (40, 64, 64), (36, 36, 40), (36, 36, 52), (60, 36, 48), (128, 28, 44)])
def test_selection_cut_overs_do_not_change_results(workload, dev, single_bins, warp_bin, hub_bin):
    """gg_sampler_tune moves rows between the three selection schemes (one lane per row, one lane per
    chunk of 128 positions with the row's candidates merged through global memory, one warp per
    row); the blocks stay the oracle's, also with the fallback knobs on and on hub rows."""
    from paper_2606_02916_b200 import binding
    binding.sampler_tune(single_bins, warp_bin, hub_bin)
    try:
        pu.check_epoch(workload("dense_mini", dev), W=2, n_hot=-1, max_batches=2, check_features=False)
        pu.check_epoch(workload("products_mini", dev), W=4, n_hot=-1, max_batches=4, check_features=False)
        pu.check_epoch(_hub_workload(dev), W=3, n_hot=-1, check_features=False)
        before = binding.sampler_stats()
        for rs, wa in [(26, 0.0), (0, 300.0), (0, -12.0)]:
            binding.debug_sampler(rs, wa)
            try:
                pu.check_epoch(workload("dense_mini", dev), W=2, n_hot=-1, max_batches=2, check_features=False)
            finally:
                binding.debug_sampler(0, 0.0)
        assert binding.sampler_stats()["fallbacks"] > before["fallbacks"]
    finally:
        binding.sampler_tune()


def test_selection_fallbacks_are_rare_by_default(workload, dev):
    from paper_2606_02916_b200 import binding
    w = workload("dense_mini", dev)
    before = binding.sampler_stats()
    pu.check_epoch(w, W=4, n_hot=-1, max_batches=4, check_features=False)
    after = binding.sampler_stats()
    rows = after["rows"] - before["rows"]
    assert rows > 1000
    assert (after["fallbacks"] - before["fallbacks"]) <= 0.03 * rows


def test_lookahead_one_is_algorithm_1_literal(workload, dev):
    """stage(k+1) / serve k (Alg. 1) gives the same results as the deeper pipelines
    (sampling 2 and 5 windows ahead; the cache is always built one window ahead)."""
    from paper_2606_02916_b200 import epoch as ep
    w = workload("small", dev)
    outs = []
    for la in (1, 2, 5):
        g = ep.graph_from_workload(w, n_hot=7500, max_window=4, max_live_windows=la + 1)
        feats = torch.empty(w.num_nodes, w.dim, dtype=w.dtype, device=dev)
        got = []
        ep.run_epoch(g, w.batches, w.fanouts, 4, feats, lookahead=la,
                     on_batch=lambda k, j, bi, r: got.append((r["input_nodes"].cpu().numpy().copy(),
                                                              r["features"].cpu().clone(), g.misses(r)[0].copy())))
        outs.append(got)
        g.close()
    for a, b, c in zip(*outs):
        assert np.array_equal(a[0], b[0]) and torch.equal(a[1], b[1]) and np.array_equal(a[2], b[2])
        assert np.array_equal(a[0], c[0]) and torch.equal(a[1], c[1]) and np.array_equal(a[2], c[2])


def test_pipeline_stress_X_b_is_the_same_for_every_schedule(workload, dev):
    """X_b and N_b do not depend on W, n_hot, carry-over, staging mode, lookahead or
    the number of cache buffers.  200 epochs over random schedules of the four-thread pipeline;
    every batch's N_b and X_b must hash to the value of the first epoch (a lost wait between the
    sampler, selector, stager and caller streams shows up here as a mismatch or a hang)."""
    _stress(workload("small", dev), dev, n_cfg=40, epochs=5, max_window=8, ws=[1, 2, 3, 4, 8], seed=11)


def test_pipeline_stress_at_products_size(workload, dev):
    """The same check with full-size kernels (N = 2.4 M, ~340 k rows per batch), where the
    streams really overlap: the first 40 mini-batches under 8 schedules."""
    import dataclasses
    w = workload("products", dev)
    _stress(dataclasses.replace(w, batches=w.batches[:40]), dev, n_cfg=8, epochs=2, max_window=16,
            ws=[1, 4, 7, 16], seed=12, budgets=[-1, 0, 180000])


def _stress(w, dev, n_cfg, epochs, max_window, ws, seed, budgets=(-1, 0, 3000, 20000)):
    from paper_2606_02916_b200 import epoch as ep
    rng = np.random.default_rng(seed)
    ref = {}
    feats = torch.empty(min(w.num_nodes, 600_000), w.dim, dtype=w.dtype, device=dev)

    def on_batch(k, j, bi, r):
        # position-weighted sums (mod 2^64, wrapping int64): a permutation of the rows or of the
        # words inside a row, or two compensating errors, change the value
        x = r["features"].contiguous().view(torch.int32).reshape(-1).to(torch.int64)
        wx = torch.arange(1, x.numel() + 1, dtype=torch.int64, device=x.device) * 0x9E3779B1 + 0x7F4A7C15
        nd = r["input_nodes"].to(torch.int64)
        wn = torch.arange(1, nd.numel() + 1, dtype=torch.int64, device=nd.device) * 0x85EBCA6B + 0xC2B2AE35
        h = (int((x * wx).sum().item()), int((nd * wn).sum().item()), r["n_input"])
        if bi in ref:
            assert ref[bi] == h, "batch %d differs from the first epoch" % bi
        else:
            ref[bi] = h

    wid = 0
    for cfg_i in range(n_cfg):
        la = int(rng.integers(1, 6))
        g = ep.graph_from_workload(w, n_hot=int(rng.choice(list(budgets))), carry_over=int(rng.integers(0, 2)),
                                   max_window=max_window, staging_mode=int(rng.integers(0, 2)), max_live_windows=la + 1,
                                   cache_buffers=int(rng.integers(2, 5)), host_threads=int(rng.choice([0, 1, 3])))
        for e in range(epochs):
            W = int(rng.choice(ws))
            ep.run_epoch(g, w.batches, w.fanouts, W, feats, on_batch=on_batch, first_window_id=wid, lookahead=la)
            wid += 100
            if rng.integers(0, 2):
                g.cache_reset()
        g.close()
    assert len(ref) == len(w.batches)


def test_determinism_two_epochs_identical(workload, dev):
    from paper_2606_02916_b200 import epoch as ep
    w = workload("small", dev)
    g = ep.graph_from_workload(w, max_window=4)
    feats = torch.empty(w.num_nodes, w.dim, dtype=w.dtype, device=dev)
    runs = []
    for e in range(2):
        got = []
        ep.run_epoch(g, w.batches, w.fanouts, 4, feats,
                     on_batch=lambda k, j, bi, r: got.append((r["input_nodes"].cpu().numpy().copy(),
                                                              r["blocks"][-1]["src_local"].cpu().numpy().copy(),
                                                              r["features"].cpu().clone())),
                     first_window_id=100 * e)
        runs.append(got)
        g.cache_reset()
    for a, b in zip(*runs):
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and torch.equal(a[2], b[2])
    g.close()


def test_error_codes(workload, dev):
    from paper_2606_02916_b200 import binding, epoch as ep
    w = workload("tiny", dev)
    g = ep.graph_from_workload(w, max_window=4)
    feats = torch.empty(8, w.dim, dtype=w.dtype, device=dev)
    with pytest.raises(binding.GreenGNNError) as e:
        g.batch_info(5, 0)
    assert e.value.status == binding.GG_ERR_STATE
    with pytest.raises(binding.GreenGNNError) as e:
        g.window_stage(0, 0, w.batches[:4] + w.batches[:1], w.fanouts)      # W > max_window
    assert e.value.status == binding.GG_ERR_INVALID_ARG
    with pytest.raises(binding.GreenGNNError) as e:
        g.window_stage(0, 0, [np.array([w.num_nodes], np.int32)], w.fanouts)  # seed out of range
    assert e.value.status == binding.GG_ERR_INVALID_ARG
    with pytest.raises(binding.GreenGNNError) as e:
        g.window_stage(0, 0, w.batches[:1], [0, 5])                          # fanout <= 0
    assert e.value.status == binding.GG_ERR_INVALID_ARG
    g.window_stage(0, 0, w.batches[:2], w.fanouts)
    with pytest.raises(binding.GreenGNNError) as e:
        g.batch_gather(0, 0, feats)                                          # buffer too small
    assert e.value.status == binding.GG_ERR_CAPACITY
    g.window_stage(1, 2, w.batches[2:4], w.fanouts)
    g.window_stage(2, 4, w.batches[:1], w.fanouts)
    with pytest.raises(binding.GreenGNNError) as e:
        g.window_stage(3, 5, w.batches[:1], w.fanouts)                       # fourth live window
    assert e.value.status == binding.GG_ERR_STATE
    with pytest.raises(binding.GreenGNNError) as e:
        g.batch_info(2, 0)              # window 2 shares its cache buffer with live window 0
    assert e.value.status == binding.GG_ERR_STATE
    g.window_release(0)
    assert g.batch_info(2, 0)["n_input"] > 0
    g.window_release(1)
    g.window_release(2)
    with pytest.raises(binding.GreenGNNError) as e:
        g.window_release(1)
    assert e.value.status == binding.GG_ERR_STATE
    g.close()
    # host memory where device memory is required
    with pytest.raises(binding.GreenGNNError) as e:
        binding.Graph(w.indptr.cpu(), w.indices.cpu(), w.part_offsets, 0, w.feat_parts, seed=1)
    assert e.value.status == binding.GG_ERR_INVALID_ARG


def test_frontier_overflow_is_reported_and_leaves_the_graph_clean(workload, dev):
    """max_input_nodes too small for a full batch: the window reports GG_ERR_CAPACITY, holds no
    output, and the NEXT windows on the same graph are bit-exact (the per-batch bitmaps and the
    packed access counters the failed window had touched are reset)."""
    import dataclasses
    from paper_2606_02916_b200 import binding, epoch as ep
    w0 = workload("small", dev)
    g = ep.graph_from_workload(w0, n_hot=-1, max_window=4, max_input_nodes=3000)
    for attempt in range(2):
        g.window_stage(900 + attempt, 0, w0.batches[:3], w0.fanouts)      # 1024 seeds -> tens of thousands of nodes
        with pytest.raises(binding.GreenGNNError) as e:
            g.batch_info(900 + attempt, 0)
        assert e.value.status == binding.GG_ERR_CAPACITY
        g.window_release(900 + attempt)
        # small batches fit under the cap: same graph handle, checked against the oracle
        small = [w0.batches[0][:3], w0.batches[1][:2], w0.batches[2][:4], w0.batches[3][:1], w0.batches[4][:3]]
        w = dataclasses.replace(w0, batches=small)
        s = pu.check_epoch(w, W=2, n_hot=-1, graph=g, first_window_id=100 * attempt)
        assert s["batches"] == 5
        g.cache_reset()
    g.close()


def test_growing_shared_scratch_needs_no_live_window(workload, dev):
    """A window with bigger fanouts than any before needs larger shared scratch: STATE while other
    windows are live (blocking there could deadlock), fine once they are released."""
    from paper_2606_02916_b200 import binding, epoch as ep
    w = workload("small", dev)
    g = ep.graph_from_workload(w, max_window=4, max_live_windows=4)
    g.window_stage(0, 0, w.batches[:2], [3, 2])
    with pytest.raises(binding.GreenGNNError) as e:
        g.window_stage(1, 2, w.batches[2:4], [15, 10])
    assert e.value.status == binding.GG_ERR_STATE
    assert g.batch_info(0, 0)["n_input"] > 0
    g.window_release(0)
    g.window_stage(1, 2, w.batches[2:4], [15, 10])
    assert g.batch_info(1, 1)["n_input"] > 0
    g.window_release(1)
    g.close()


def test_remote_owner_in_device_memory_mode0(workload, dev):
    """staging_mode 0 with an owner whose store is DEVICE memory (the stand-in for a peer GPU's HBM):
    host threads cannot pack it, the library serves that owner with the pull kernel; results are
    the oracle's."""
    import dataclasses
    w0 = workload("small", dev)
    parts = list(w0.feat_parts)
    parts[2] = parts[2].to(dev)                      # owner 2 on the device, owners 1 and 3 pinned
    w = dataclasses.replace(w0, feat_parts=parts)
    pu.check_epoch(w, W=4, n_hot=-1, staging_mode=0)
    pu.check_epoch(w, W=2, n_hot=7500, staging_mode=0)
    parts = [p.to(dev) for p in w0.feat_parts]       # every owner on the device
    pu.check_epoch(dataclasses.replace(w0, feat_parts=parts), W=4, n_hot=7500, staging_mode=0)


# ---- BASELINE.json's full sizes, in the launch configuration bench.py times ---------------------
def test_products_full_size_first_window_W16(workload, dev):
    """configs[2] at full size (N=2,449,029, nnz=123.8M, dim 100), B=1024, W=16, n_hot unlimited:
    the first window (16 mini-batches, ~5.5M sampled nodes) against the oracle, every array."""
    w = workload("products", dev)
    s = pu.check_epoch(w, W=16, n_hot=-1, max_batches=16, cache_samples=256, lookahead=6)   # bench.py's arenas
    assert s["batches"] == 16 and s["misses"] == 0 and s["rows"] > 16 * 300_000


def test_products_full_size_budgeted_two_windows(workload, dev):
    """Same graph, finite budget = 10 % of the remote nodes, W=2, two windows:
    exercises threshold selection, carry-over and the miss path at full size."""
    w = workload("products", dev)
    n_remote = w.num_nodes - int(w.part_offsets[1] - w.part_offsets[0])
    s = pu.check_epoch(w, W=2, n_hot=n_remote // 10, max_batches=6, cache_samples=256, lookahead=6)
    assert s["windows"] == 3 and s["misses"] > 0


def test_dense_full_size_first_window(workload, dev):
    """configs[3] at full size (N=232,965, nnz=114.6M, avg degree ~490, rb = 2408 B)."""
    w = workload("dense", dev)
    s = pu.check_epoch(w, W=4, n_hot=-1, max_batches=4, cache_samples=128)
    assert s["batches"] == 4


def _threads():
    import os
    return min(16, os.cpu_count() or 1)


@pytest.mark.parametrize("B", [2048, 4096])
def test_products_full_size_larger_batches_first_window_W16(workload, dev, B):
    """configs[2]'s other batch sizes, which bench.py times (`vs_batch_at_W`, `configs`): the same
    epoch's seeds cut into batches of 2048 / 4096, first W=16 window at full size (frontier caps x2 /
    x4, the last hop of B=4096 capped at N), every array against the oracle."""
    import dataclasses
    w0 = workload("products", dev)
    seeds = np.concatenate(w0.batches)
    w = dataclasses.replace(w0, batches=[seeds[i:i + B] for i in range(0, len(seeds), B)])
    s = pu.check_epoch(w, W=16, n_hot=-1, max_batches=16, cache_samples=256, lookahead=6, oracle_threads=_threads())
    assert s["batches"] == 16 and s["misses"] == 0 and s["rows"] > 16 * 300_000 * (B // 1024) // 2


def test_products_full_size_three_consecutive_windows_W16(workload, dev):
    """Delta / carry-over at 5 M-row scale: three consecutive W=16 windows with an unlimited budget
    (windows 2 and 3 stage only H_k \\ C_{k-1} and carry the rest), request lists,
    carried lists, cache rows and every batch element-wise."""
    w = workload("products", dev)
    s = pu.check_epoch(w, W=16, n_hot=-1, max_batches=48, cache_samples=256, lookahead=6, oracle_threads=_threads())
    assert s["windows"] == 3 and s["batches"] == 48 and s["misses"] == 0


def test_products_full_size_budgeted_W16_two_windows(workload, dev):
    """The budgeted series bench.py times (n_hot = 10 % of the remote nodes) at W=16:
    threshold selection with a quota, a stale cache across the boundary and the miss path at the
    size of the timed runs."""
    w = workload("products", dev)
    n_remote = w.num_nodes - int(w.part_offsets[1] - w.part_offsets[0])
    s = pu.check_epoch(w, W=16, n_hot=-(-n_remote // 10), max_batches=32, cache_samples=256, lookahead=6,
                       oracle_threads=_threads())
    assert s["windows"] == 2 and s["misses"] > 0


def test_products_full_size_whole_epoch_W16_W32_unlimited_and_budgeted(workload, dev):
    """The headline config over its WHOLE epoch (one epoch's trace fixes all later ones):
    all 193 mini-batches at full size, every array of every batch and window against the oracle, for
    W=16 (13 windows, the last one a single batch) and W=32 (32-batch arenas, counts up to 32 at 5 M-row
    scale), each with an unlimited budget and with n_hot = 10 % of the remote nodes.  The
    oracle samples the 193 batches once (they do not depend on W or the budget)."""
    w = workload("products", dev)
    assert len(w.batches) == 193
    n_remote = w.num_nodes - int(w.part_offsets[1] - w.part_offsets[0])
    shared, hg, parts = {}, w.host_graph(), pu.oracle_parts(w)
    for W, n_hot in [(16, -1), (32, -1), (16, -(-n_remote // 10)), (32, -(-n_remote // 10))]:
        s = pu.check_epoch(w, W=W, n_hot=n_hot, cache_samples=64, lookahead=6 if W == 16 else 3,
                           oracle_threads=_threads(), oracle_batches=shared, host_graph=hg, parts=parts)
        assert s["batches"] == 193 and s["windows"] == -(-193 // W)
        assert (s["misses"] == 0) == (n_hot < 0)


def test_dense_full_size_W16_two_windows_and_W1(workload, dev):
    """configs[3] at full size across a window boundary: W=16 over two windows (Delta, carry-over and
    the carried D2D copy with rb = 2408, the 8-byte path), then W=1 (per-batch fetch, three windows)
    and a budgeted W=4 pair (miss fill at rb = 2408)."""
    w = workload("dense", dev)
    thr = _threads()
    s = pu.check_epoch(w, W=16, n_hot=-1, max_batches=32, cache_samples=128, lookahead=6, oracle_threads=thr)
    assert s["windows"] == 2 and s["batches"] == 32 and s["misses"] == 0
    s = pu.check_epoch(w, W=1, n_hot=-1, max_batches=3, cache_samples=64, oracle_threads=thr)
    assert s["windows"] == 3
    n_remote = w.num_nodes - int(w.part_offsets[1] - w.part_offsets[0])
    s = pu.check_epoch(w, W=4, n_hot=-(-n_remote // 10), max_batches=8, cache_samples=64, oracle_threads=thr)
    assert s["windows"] == 2 and s["misses"] > 0


def test_large_full_size_first_windows(dev):
    """configs[4] at full size: R-MAT, N = 111,000,000, 1.6 B directed edges (int64 offsets),
    dim 128 bf16, 83 M remote rows in pinned host memory.  The first 8 windows at W=4 (32
    mini-batches) and the same batches as 2 windows at W=16 with a finite budget, every array
    against the oracle (its 32 batches are sampled once, 16 at a time on the host cores)."""
    import os
    from paper_2606_02916_b200 import inputs
    free_b, _ = torch.cuda.mem_get_info()
    try:
        host_gb = os.sysconf("SC_PHYS_PAGES") * os.sysconf("SC_PAGE_SIZE") / 1e9
    except (ValueError, OSError):
        host_gb = 0.0
    if free_b < 120e9 or host_gb < 100:
        pytest.skip("needs ~120 GB of HBM and ~100 GB of host memory")
    w = inputs.make_workload("large", device=dev)
    assert w.num_nodes == 111_000_000 and w.indices.numel() == 1_600_000_000
    hg = w.host_graph()
    parts = pu.oracle_parts(w)
    thr = min(16, os.cpu_count() or 1)
    s = pu.check_epoch(w, W=4, n_hot=-1, max_batches=32, cache_samples=64, oracle_threads=thr,
                       host_graph=hg, parts=parts)
    assert s["windows"] == 8 and s["batches"] == 32 and s["misses"] == 0
    s = pu.check_epoch(w, W=16, n_hot=200_000, max_batches=32, cache_samples=64, oracle_threads=thr,
                       host_graph=hg, parts=parts)
    assert s["windows"] == 2 and s["misses"] > 0
    del w, hg, parts
    torch.cuda.empty_cache()

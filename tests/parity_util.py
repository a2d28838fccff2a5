"""Element-by-element comparison of the CUDA path (through the C ABI) with the CPU oracle."""
import numpy as np
import torch

from oracle import ggo
from paper_2606_02916_b200 import epoch as ep


def oracle_parts(w):
    """Per-owner [rows, row_bytes] uint8 host views of the feature store (no concatenation:
    the Large config's store is 28 GB)."""
    parts = []
    for p in w.feat_parts:
        h = p if p.device.type == "cpu" else p.cpu()
        parts.append(h.contiguous().view(torch.uint8).view(h.shape[0], -1).numpy())
    return parts


def check_epoch(w, W, n_hot=-1, carry_over=1, staging_mode=0, max_batches=None, max_cache_rows=0,
                check_features=True, cache_samples=64, host_threads=0, oracle_threads=1, host_graph=None,
                parts=None, cache_buffers=0, lookahead=2, graph=None, first_window_id=0, oracle_batches=None):
    """Runs one epoch on the GPU and on the oracle; asserts bit-exact agreement everywhere.
    Returns a small summary dict."""
    batches = w.batches if max_batches is None else w.batches[:max_batches]
    indptr, indices = host_graph if host_graph is not None else w.host_graph()
    og = ggo.Graph(indptr, indices)
    po = w.part_offsets
    P = len(po) - 1
    n_remote_nodes = w.num_nodes - int(po[w.local_part + 1] - po[w.local_part])
    cache_rows = min(max_cache_rows, n_remote_nodes) if max_cache_rows > 0 else n_remote_nodes
    eff = cache_rows if n_hot < 0 else min(n_hot, cache_rows)        # reading S9
    ostate = ggo.State(og.n, po, w.local_part, eff, carry_over)
    if parts is None and check_features:
        parts = oracle_parts(w)

    # graph: an existing handle (its cache must be empty: the oracle starts from C_0 = {}); it is
    # left open for the caller
    g = graph if graph is not None else ep.graph_from_workload(
        w, n_hot=n_hot, carry_over=carry_over, max_window=max(W, 1), staging_mode=staging_mode,
        max_cache_rows=max_cache_rows, host_threads=host_threads, cache_buffers=cache_buffers,
        max_live_windows=lookahead + 1)
    # oracle_batches: a dict the caller keeps between runs over the SAME batch list (the oracle's batches
    # depend on graph, seeds, fanouts, seed and batch index only -- not on W, n_hot or the cache)
    obatches = oracle_batches if oracle_batches is not None else {}
    owin = {}
    stats = dict(batches=0, misses=0, windows=0, rows=0, edges=0)
    wins = ep.windows_of(len(batches), W)
    cap_rows = 0

    def get_obatch(bi):
        if bi not in obatches:
            obatches[bi] = ggo.Batch(og, batches[bi], w.fanouts, w.seed, bi)
        return obatches[bi]

    if oracle_threads > 1:
        # the oracle's batches are independent calls (ctypes releases the GIL): run them side by
        # side; the oracle itself is unchanged and single-threaded per batch
        from concurrent.futures import ThreadPoolExecutor
        with ThreadPoolExecutor(oracle_threads) as ex:
            todo = [bi for bi in range(len(batches)) if bi not in obatches]
            for bi, ob in zip(todo, ex.map(lambda bi: ggo.Batch(og, batches[bi], w.fanouts, w.seed, bi), todo)):
                obatches[bi] = ob

    # the oracle advances its cache window by window in the same order
    for k, win in enumerate(wins):
        owin[k] = ostate.run_window([get_obatch(bi) for bi in win])
        cap_rows = max(cap_rows, max(len(get_obatch(bi).nodes) for bi in win))
    features = torch.empty(cap_rows + 3, w.dim, dtype=w.dtype, device=w.indptr.device)

    def on_batch(k, j, bi, r):
        ob = get_obatch(bi)
        ow = owin[k]
        assert r["n_input"] == len(ob.nodes), (bi, r["n_input"], len(ob.nodes))
        assert np.array_equal(r["input_nodes"].cpu().numpy(), ob.nodes), "N_b differs (batch %d)" % bi
        assert len(r["blocks"]) == ob.L
        for h, (gb, obk) in enumerate(zip(r["blocks"], ob.blocks)):
            assert (gb["n_dst"], gb["n_src"], gb["n_edge"]) == (obk["n_dst"], obk["n_src"], obk["n_edge"]), (bi, h)
            assert np.array_equal(gb["indptr"].cpu().numpy(), obk["indptr"]), "indptr (batch %d hop %d)" % (bi, h)
            assert np.array_equal(gb["src_global"].cpu().numpy(), obk["src_global"]), "src_global (batch %d hop %d)" % (bi, h)
            assert np.array_equal(gb["src_local"].cpu().numpy(), obk["src_local"]), "src_local (batch %d hop %d)" % (bi, h)
            stats["edges"] += gb["n_edge"]
        mp, mi = g.misses(r)
        assert np.array_equal(mp, ow.miss_pos[j]), "miss positions (batch %d)" % bi
        assert np.array_equal(mi, ow.miss_id[j]), "miss ids (batch %d)" % bi
        if check_features:
            x = r["features"].contiguous().view(torch.uint8).view(r["n_input"], -1).cpu().numpy()
            want = ggo.gather(ob.nodes, po, parts, w.row_bytes)
            assert np.array_equal(x, want), "X_b differs (batch %d)" % bi
        stats["batches"] += 1
        stats["misses"] += len(mp)
        stats["rows"] += r["n_input"]

    def on_window(wid, win):
        k = wid - first_window_id
        ow = owin[k]
        t = g.trace(wid, len(win))
        assert np.array_equal(g.window_export(wid, "uniq"), ow.uniq), "U_k"
        assert np.array_equal(g.window_export(wid, "cnt"), ow.cnt), "c_k"
        assert np.array_equal(g.window_export(wid, "hot"), ow.hot), "H_k"
        req = np.concatenate(ow.delta) if P else np.zeros(0, np.int32)
        assert np.array_equal(g.window_export(wid, "req"), req), "Delta request lists"
        assert np.array_equal(g.window_export(wid, "carried"), ow.carried), "carried"
        assert t["n_access"] == ow.n_access and t["n_unique"] == ow.n_unique
        assert t["n_unique_remote"] == ow.n_unique_remote and t["n_hot"] == ow.n_hot
        assert t["carried_rows"] == ow.carried_rows
        assert t["staged_rows"] == list(ow.staged_rows) and t["bulk_rows"] == list(ow.bulk_rows)
        assert t["bulk_bytes"] == [x * w.row_bytes for x in ow.bulk_rows]
        assert t["bulk_copies"] == sum(1 for x in ow.bulk_rows if x > 0)
        assert t["n_input"].tolist() == ow.n_input
        assert t["hit_local"].tolist() == ow.hit_local and t["hit_cache"].tolist() == ow.hit_cache
        assert np.array_equal(t["miss"], np.stack(ow.miss)), "per-owner miss counts"
        if check_features and len(ow.hot) and cache_samples:
            ids = ow.hot[np.linspace(0, len(ow.hot) - 1, min(cache_samples, len(ow.hot))).astype(np.int64)]
            want = ggo.gather(ids, po, parts, w.row_bytes)
            got = g.cache_read(wid, ids)
            got = np.ascontiguousarray(got).view(np.uint8).reshape(len(ids), -1)
            assert np.array_equal(got, want), "cache rows"
        stats["windows"] += 1

    ep.run_epoch(g, batches, w.fanouts, W, features, on_batch=on_batch, on_window=on_window, lookahead=lookahead,
                 first_window_id=first_window_id)
    torch.cuda.synchronize()
    if graph is None:
        g.close()
    return stats

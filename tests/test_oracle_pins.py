"""Pins of the CPU oracle (oracle/ggo.cpp) against things other than itself.

Each test names the oracle step (O0..O7) and what fixes the
expected value: the published SplitMix64 vector, the survey's key-chain values
(tests/golden/keys.txt), brute force in pure Python, closed-form inclusion
probabilities, textbook BFS, numpy library routines, Python set algebra, and the
paper's worked example.  No GPU, no CUDA library.
"""
import os
from collections import Counter

import numpy as np
import pytest

from oracle import ggo

GOLD = os.path.join(os.path.dirname(__file__), "golden", "keys.txt")
M64 = (1 << 64) - 1
GAMMA = 0x9E3779B97F4A7C15


# -- a pure-Python restatement used ONLY by the brute-force selection pins; the hash
#    itself is pinned by the golden file, not by this retyping.
def py_fmix(z):
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & M64
    return z ^ (z >> 31)


def py_sm(x):
    return py_fmix((x + GAMMA) & M64)


def py_key(seed, batch, layer, dst, j):
    h = py_sm(py_sm(py_sm(py_sm(seed) ^ batch) ^ layer) ^ dst)
    return py_fmix((h + (j + 1) * GAMMA) & M64)


def _golden():
    rows = []
    for line in open(GOLD):
        line = line.strip()
        if line and not line.startswith("#"):
            t = line.split()
            rows.append((t[0], [int(x, 0) for x in t[1:-1]], int(t[-1], 16)))
    return rows


def test_O0_splitmix64_published_vector_and_key_chain_golden():
    seen = set()
    for tag, args, want in _golden():
        seen.add(tag)
        if tag == "splitmix64":
            n = args[0]
            # output n of SplitMix64 from state 0 is fmix(n*gamma) = key stream j=n-1 of h=0
            assert ggo.fmix((n * GAMMA) & M64) == want
            if n == 1:
                assert ggo.sm(0) == want
        elif tag == "h_dst":
            assert ggo.h_dst(*args) == want
        elif tag == "key":
            assert ggo.key(*args) == want
            assert py_key(*args) == want          # keeps the brute-force helper honest
    assert seen == {"splitmix64", "h_dst", "key"}


def test_O0_key_does_not_depend_on_epoch_or_neighbor_id():
    # one epoch's trace determines all future epochs -> the key has exactly the
    # five arguments (seed, batch, layer, dst, edge_pos); changing any one changes it.
    base = (7, 11, 1, 99, 5)
    k0 = ggo.key(*base)
    for i in range(5):
        a = list(base)
        a[i] += 1
        assert ggo.key(*a) != k0


def _toy_graph(rng, n, degs):
    indptr = np.zeros(n + 1, dtype=np.int64)
    indptr[1:] = np.cumsum(degs)
    indices = rng.integers(0, n, size=int(indptr[-1])).astype(np.int32)
    return ggo.Graph(indptr, indices)


@pytest.mark.parametrize("fanout", [1, 3, 5, 10])
def test_O1_brute_force_full_sort_tiny_graphs(fanout):
    rng = np.random.default_rng(100 + fanout)
    f = fanout
    degs = [0, 1, max(f - 1, 0), f, f + 1, 2 * f, 3 * f, 3 * f + 1] + list(rng.integers(0, 3 * f + 2, 150))
    g = _toy_graph(rng, len(degs), degs)
    for seed, batch, layer in [(0, 0, 0), (12345, 7, 1), (M64, (1 << 40) + 3, 2)]:
        for v in range(g.n):
            deg = int(g.indptr[v + 1] - g.indptr[v])
            pos, ids = ggo.sample_dst(g, v, f, seed, batch, layer)
            if deg <= f:
                want = list(range(deg))
            else:
                order = sorted((py_key(seed, batch, layer, v, j), j) for j in range(deg))
                want = sorted(j for _, j in order[:f])
            assert pos.tolist() == want
            # invariants: count = min(deg, f); strictly increasing; ids are the CSR entries
            assert len(pos) == min(deg, f)
            assert all(pos[i] < pos[i + 1] for i in range(len(pos) - 1))
            assert ids.tolist() == [int(g.indices[g.indptr[v] + j]) for j in want]


def test_O1_forced_tie_smaller_position_wins():
    # reading S4: equal keys -> the smaller edge position is kept.  A hook makes every key
    # equal to (j % 3), so ties are everywhere and the expected set is known in closed form.
    rng = np.random.default_rng(5)
    g = _toy_graph(rng, 4, [12, 12, 7, 30])
    hook = ggo.KEY_HOOK(lambda h, j: j % 3)
    ggo.set_key_hook(hook)
    try:
        for v, f in [(0, 5), (1, 4), (2, 3), (3, 11)]:
            deg = int(g.indptr[v + 1] - g.indptr[v])
            want = sorted(sorted(range(deg), key=lambda j: (j % 3, j))[:f])
            pos, _ = ggo.sample_dst(g, v, f, 1, 2, 0)
            assert pos.tolist() == want
    finally:
        ggo.set_key_hook(None)


def test_O1_inclusion_probabilities_closed_form():
    # Uniform sampling without replacement over positions: P(j kept) = f/deg,
    # P(i and j kept) = f(f-1)/(deg(deg-1)).  Chi-square over many seeds.
    deg, f, trials = 12, 4, 6000
    g = ggo.Graph(np.array([0, deg], dtype=np.int64), np.arange(deg, dtype=np.int32) % 1)
    single = np.zeros(deg)
    pair = np.zeros((deg, deg))
    for s in range(trials):
        pos, _ = ggo.sample_dst(g, 0, f, s, 3, 1)
        single[pos] += 1
        for a in pos:
            for b in pos:
                if a < b:
                    pair[a, b] += 1
    exp1 = trials * f / deg
    chi1 = ((single - exp1) ** 2 / exp1).sum()
    assert chi1 < 40.0, chi1                      # 11 dof, p ~ 1e-5 at 40
    exp2 = trials * f * (f - 1) / (deg * (deg - 1))
    iu = np.triu_indices(deg, 1)
    chi2 = ((pair[iu] - exp2) ** 2 / exp2).sum()
    assert chi2 < 130.0, chi2                     # 65 dof, p ~ 1e-5 at 130


def _bfs_ball(indptr, indices, seeds, hops):
    """Textbook BFS: frontier_{h+1} = frontier_h ++ sorted(new in-neighbors)."""
    frontier = list(int(s) for s in seeds)
    levels = [len(frontier)]
    for _ in range(hops):
        have = set(frontier)
        new = set()
        for v in frontier:
            for u in indices[indptr[v]:indptr[v + 1]]:
                if int(u) not in have:
                    new.add(int(u))
        frontier += sorted(new)
        levels.append(len(frontier))
    return frontier, levels


def test_O1_O2_fanout_ge_max_degree_is_bfs(workload):
    w = workload("tiny")
    indptr, indices = w.host_graph()
    g = ggo.Graph(indptr, indices)
    dmax = int((indptr[1:] - indptr[:-1]).max())
    seeds = w.batches[0][:16]
    b = ggo.Batch(g, seeds, [dmax, dmax + 7], w.seed, 0)
    frontier, levels = _bfs_ball(indptr, indices, seeds, 2)
    assert b.n_front == levels
    assert b.nodes.tolist() == frontier
    for h, blk in enumerate(b.blocks):
        # induced in-edge lists of the dst prefix, untouched
        want = np.concatenate([indices[indptr[v]:indptr[v + 1]] for v in frontier[:levels[h]]])
        assert np.array_equal(blk["src_global"], want)


def _check_O2_invariants(g, b, seeds, fanouts):
    assert b.n_front[0] == len(seeds)
    assert np.array_equal(b.nodes[:len(seeds)], seeds)
    assert len(set(b.nodes.tolist())) == len(b.nodes)
    for h, blk in enumerate(b.blocks):
        nd, ns = b.n_front[h], b.n_front[h + 1]
        front_h, front_h1 = b.nodes[:nd], b.nodes[:ns]
        tail = front_h1[nd:]
        assert np.all(np.diff(tail) > 0)                           # new nodes ascending
        assert set(front_h1.tolist()) == set(front_h.tolist()) | set(blk["src_global"].tolist())
        assert np.array_equal(front_h1[blk["src_local"]], blk["src_global"])
        ip = blk["indptr"]
        assert ip[0] == 0 and ip[-1] == blk["n_edge"] and np.all(np.diff(ip) >= 0)
        deg = (g.indptr[front_h + 1] - g.indptr[front_h]).astype(np.int64)
        assert np.array_equal(np.diff(ip), np.minimum(deg, fanouts[h]))
        for i in (0, nd // 2, nd - 1):                             # sampled ids are CSR neighbours
            v = int(front_h[i])
            row = set(g.indices[g.indptr[v]:g.indptr[v + 1]].tolist())
            assert set(blk["src_global"][ip[i]:ip[i + 1]].tolist()) <= row


def test_O2_invariants_and_determinism(workload):
    w = workload("tiny")
    g = ggo.Graph(*w.host_graph())
    for bi, seeds in enumerate(w.batches):
        b = ggo.Batch(g, seeds, w.fanouts, w.seed, bi)
        _check_O2_invariants(g, b, seeds, w.fanouts)
        b2 = ggo.Batch(g, seeds, w.fanouts, w.seed, bi)             # second "epoch": identical
        assert np.array_equal(b.nodes, b2.nodes)
        for x, y in zip(b.blocks, b2.blocks):
            assert np.array_equal(x["src_local"], y["src_local"])
        b3 = ggo.Batch(g, seeds, w.fanouts, w.seed, bi + 1)         # batch index enters the key
        assert not np.array_equal(b.blocks[-1]["src_global"], b3.blocks[-1]["src_global"])


def _owner(po, u):
    return int(np.searchsorted(po, u, side="right") - 1)


def _window_expect(batches, po, local, n_hot, cache_prev, carry):
    """Independent restatement of O3..O6 with numpy library routines and Python sets."""
    cat = np.concatenate([b.nodes for b in batches])
    uniq, cnt = np.unique(cat, return_counts=True)
    own = np.searchsorted(po, uniq, side="right") - 1
    rem = own != local
    R, Rc = uniq[rem], cnt[rem]
    if n_hot < 0 or len(R) <= n_hot:
        hot = R
    else:
        hot = np.sort(R[np.lexsort((R, -Rc))[:n_hot]])
    hs = set(hot.tolist())
    delta = [sorted(u for u in hs if _owner(po, u) == m and not (carry and u in cache_prev))
             for m in range(len(po) - 1)]
    carried = sorted(hs & cache_prev) if carry else []
    return uniq, cnt, R, hot, delta, carried


@pytest.mark.parametrize("n_hot,carry", [(-1, 1), (200, 1), (200, 0), (0, 1), (-1, 0)])
def test_O3_O4_O5_O6_against_numpy_and_sets(workload, n_hot, carry):
    w = workload("tiny")
    g = ggo.Graph(*w.host_graph())
    po = w.part_offsets
    st = ggo.State(g.n, po, w.local_part, n_hot, carry)
    batches = [ggo.Batch(g, s, w.fanouts, w.seed, i) for i, s in enumerate(w.batches)]
    cache_prev = set()
    for win in ([0, 1], [2], [3, 0]):                 # three windows; partial + repeated batch
        bs = [batches[i] for i in win]
        r = st.run_window(bs)
        uniq, cnt, R, hot, delta, carried = _window_expect(bs, po, w.local_part, n_hot, cache_prev, carry)
        assert np.array_equal(r.uniq, uniq) and np.array_equal(r.cnt, cnt)        # O3 = numpy.unique
        assert np.all(np.diff(r.uniq) > 0) and r.cnt.min() >= 1 and r.cnt.max() <= len(bs)
        assert r.cnt.sum() == r.n_access == sum(len(b.nodes) for b in bs)
        assert r.n_unique_remote == len(R)
        assert np.array_equal(r.hot, hot)                                           # O4 = lexsort
        assert r.n_hot == (len(R) if n_hot < 0 else min(n_hot, len(R)))
        if 0 < len(hot) < len(R):
            cm = dict(zip(uniq.tolist(), cnt.tolist()))
            assert min(cm[u] for u in hot.tolist()) >= max(cm[u] for u in R.tolist() if u not in set(hot.tolist()))
        for m in range(len(po) - 1):                                                # O5 = set algebra
            assert r.delta[m].tolist() == delta[m]
            assert all(_owner(po, u) == m for u in r.delta[m].tolist())
            assert not (set(r.delta[m].tolist()) & cache_prev) or not carry
        assert r.bulk_rows[w.local_part] == 0 and r.staged_rows[w.local_part] == 0
        assert sum(r.staged_rows) == len(hot)
        assert r.carried.tolist() == carried
        assert sum(r.bulk_rows) + r.carried_rows == len(hot)
        assert st.cache().tolist() == hot.tolist()                                  # C_k = H_k
        hs = set(hot.tolist())
        for bi, b in enumerate(bs):                                                 # O6
            own = np.searchsorted(po, b.nodes, side="right") - 1
            is_local = own == w.local_part
            in_hot = np.array([u in hs for u in b.nodes.tolist()])
            miss = ~is_local & ~in_hot
            assert r.hit_local[bi] == is_local.sum()
            assert r.hit_cache[bi] == (~is_local & in_hot).sum()
            assert r.miss_pos[bi].tolist() == np.nonzero(miss)[0].tolist()
            assert np.array_equal(r.miss_id[bi], b.nodes[miss])
            assert r.miss[bi].tolist() == [int((miss & (own == m)).sum()) for m in range(len(po) - 1)]
            assert r.hit_local[bi] + r.hit_cache[bi] + r.miss[bi].sum() == r.n_input[bi] == len(b.nodes)
            if n_hot < 0:
                assert r.miss[bi].sum() == 0
        cache_prev = hs


def test_O5_W1_degenerates_to_per_batch_fetch(workload):
    # W = 1, unlimited budget, no carry-over: window b's requests are exactly batch b's
    # remote IDs grouped by owner, and no batch has a miss (BASELINE.json:north_star).
    w = workload("tiny")
    g = ggo.Graph(*w.host_graph())
    po = w.part_offsets
    st = ggo.State(g.n, po, w.local_part, -1, 0)
    for i, s in enumerate(w.batches):
        b = ggo.Batch(g, s, w.fanouts, w.seed, i)
        r = st.run_window([b])
        own = np.searchsorted(po, b.nodes, side="right") - 1
        for m in range(len(po) - 1):
            want = [] if m == w.local_part else sorted(b.nodes[own == m].tolist())
            assert r.delta[m].tolist() == want
        assert r.miss[0].sum() == 0


def test_O6_gather_is_numpy_take_and_is_configuration_independent(workload):
    w = workload("tiny")
    g = ggo.Graph(*w.host_graph())
    feat = w.host_features()                         # [N, rb] uint8
    po = w.part_offsets
    parts = [np.ascontiguousarray(feat[po[m]:po[m + 1]]) for m in range(len(po) - 1)]
    b = ggo.Batch(g, w.batches[1], w.fanouts, w.seed, 1)
    x = ggo.gather(b.nodes, po, parts, w.row_bytes)
    assert np.array_equal(x, np.take(feat, b.nodes, axis=0))
    # a padded store (stride > row_bytes) gives the same rows
    padded = [np.ascontiguousarray(np.pad(p, ((0, 0), (0, 16)))) for p in parts]
    assert np.array_equal(ggo.gather(b.nodes, po, padded, w.row_bytes, w.row_bytes + 16), x)
    # X_b does not depend on W, n_hot or carry_over: the oracle's service step never alters it
    for n_hot, carry in [(-1, 1), (50, 0)]:
        st = ggo.State(g.n, po, 0, n_hot, carry)
        st.run_window([b])
        assert np.array_equal(ggo.gather(b.nodes, po, parts, w.row_bytes), x)


def test_worked_example_bulk_transfers_per_window(workload):
    # W=16 over three remote owners -> up to 16*3 = 48 per-batch requests
    # become 3 bulk transfers.  Count non-empty requests both ways on a 16-batch window.
    w = workload("small")
    g = ggo.Graph(*w.host_graph())
    po = w.part_offsets
    seeds = [w.batches[i % len(w.batches)][:64] for i in range(16)]
    batches = [ggo.Batch(g, s, w.fanouts, w.seed, i) for i, s in enumerate(seeds)]
    r = ggo.State(g.n, po, 0, -1, 1).run_window(batches)
    bulk = sum(1 for m in range(4) if r.bulk_rows[m] > 0)
    st1 = ggo.State(g.n, po, 0, -1, 0)
    per_batch = 0
    for b in batches:
        r1 = st1.run_window([b])
        per_batch += sum(1 for m in range(4) if r1.bulk_rows[m] > 0)
    assert bulk == 3 and per_batch == 48
    assert sum(r.bulk_rows) == r.n_unique_remote            # bulk sizes sum to the remote unique count


def test_generated_configs_have_the_stated_shape(workload):
    for name in ("tiny", "small", "products_mini", "dense_mini", "large_mini"):
        w = workload(name)
        indptr, indices = w.host_graph()
        n = w.num_nodes
        assert indptr[0] == 0 and indptr[-1] == len(indices) and np.all(np.diff(indptr) >= 0)
        assert indices.min() >= 0 and indices.max() < n
        rows = np.repeat(np.arange(n), np.diff(indptr))
        key = rows.astype(np.int64) * n + indices
        assert np.all(np.diff(key) > 0)                     # rows sorted, no duplicate entries
        if w.cfg["kind"] != "rmat":
            rev = np.sort(indices.astype(np.int64) * n + rows)
            assert np.array_equal(rev, key)                 # symmetric
            assert abs(len(indices) - 2 * w.cfg["n_pairs"]) <= 0.02 * 2 * w.cfg["n_pairs"]
        assert w.part_offsets[0] == 0 and w.part_offsets[-1] == n
        allseeds = np.concatenate(w.batches)
        assert len(set(allseeds.tolist())) == len(allseeds)
    w = workload("products_mini")
    indptr, indices = w.host_graph()
    rows = np.repeat(np.arange(w.num_nodes), np.diff(indptr))
    cut = (np.searchsorted(w.part_offsets, rows, side="right") !=
           np.searchsorted(w.part_offsets, indices, side="right")).mean()
    assert 0.04 < cut < 0.14, cut                           # planted ~8 % edge-cut


def test_bfs_grown_split_is_balanced_and_cuts_more_than_the_planted_owners(workload):
    """Reading S22: BASELINE.json asks for a BFS-grown balanced 4-way split with ~8 % edge cut; on the
    planted Chung-Lu graph the BFS growth (hubs reach every community within two levels) is balanced
    but cuts several times more than the planted communities, which is why those are the owners."""
    import torch
    from paper_2606_02916_b200 import inputs
    w = workload("products_mini")
    lab = inputs.bfs_grown_split(w.indptr, w.indices, 4, 123)
    sizes = torch.bincount(lab.long(), minlength=4)
    assert int(lab.min()) >= 0 and int(sizes.sum()) == w.num_nodes
    assert int(sizes.max()) <= int(-(-w.num_nodes // 4) * 1.02) + 1
    po = torch.as_tensor(w.part_offsets)
    planted = torch.bucketize(torch.arange(w.num_nodes), po[1:-1], right=True).to(torch.int8)
    cut_planted = inputs.edge_cut_of_labels(w.indptr, w.indices, planted)
    cut_bfs = inputs.edge_cut_of_labels(w.indptr, w.indices, lab)
    assert 0.04 <= cut_planted <= 0.14
    assert cut_bfs > 2 * cut_planted

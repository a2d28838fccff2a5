"""GPU parity of the GraphSAGE-mean consumer (NEXT-4, gg_sage_step) against oracle/sage.py.
The device computes in fp32 (sums in a different order, float atomics in the backward pass), the
oracle in fp64: tolerance 2e-4 relative on the loss and 1e-3 * scale on the parameters after
several steps (fp32 epsilon 6e-8 times reductions of up to ~1e3 terms, times a few steps)."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

from oracle import sage  # noqa: E402


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return "cuda:0"


def init_params(dims, seed):
    rng = np.random.default_rng(seed)
    return [dict(W_self=(rng.uniform(-1, 1, (dims[l], dims[l + 1])) / np.sqrt(dims[l])).astype(np.float32),
                 W_neigh=(rng.uniform(-1, 1, (dims[l], dims[l + 1])) / np.sqrt(dims[l])).astype(np.float32),
                 b=(rng.uniform(-0.1, 0.1, dims[l + 1])).astype(np.float32)) for l in range(len(dims) - 1)]


def run(w, dev, hidden, classes, W, steps, lr, seed=1):
    from paper_2606_02916_b200 import binding, epoch as ep
    L = len(w.fanouts)
    dims = [w.dim] + [hidden] * (L - 1) + [classes]
    p0 = init_params(dims, seed)
    model = binding.Sage(p0, dev)
    oparams = [{k: v.astype(np.float64) for k, v in p.items()} for p in p0]
    g = ep.graph_from_workload(w, max_window=W)
    feats = torch.empty(w.num_nodes, w.dim, dtype=w.dtype, device=dev)
    rng = np.random.default_rng(seed + 1)
    done = [0]

    def on_batch(k, j, bi, r):
        if done[0] >= steps:
            return
        n_seed = r["blocks"][0]["n_dst"]
        labels = rng.integers(0, classes, n_seed).astype(np.int32)
        loss = model.step(r, torch.from_numpy(labels).to(dev), lr)
        blocks = [dict(n_dst=b["n_dst"], indptr=b["indptr"].cpu().numpy(), src_local=b["src_local"].cpu().numpy())
                  for b in r["blocks"]]
        x = r["features"].cpu().numpy().astype(np.float64)
        want = sage.step(oparams, blocks, x, labels, lr)
        got = float(loss.cpu()[0])
        assert abs(got - want) <= 2e-4 * max(1.0, abs(want)), (done[0], got, want)
        done[0] += 1

    ep.run_epoch(g, w.batches, w.fanouts, W, feats, on_batch=on_batch)
    torch.cuda.synchronize()
    assert done[0] == steps
    for pg, po in zip(model.params(), oparams):
        for k in ("W_self", "W_neigh", "b"):
            scale = max(1.0, float(np.abs(po[k]).max()))
            assert np.allclose(pg[k], po[k], rtol=0, atol=1e-3 * scale), (k, float(np.abs(pg[k] - po[k]).max()))
    model.close()
    g.close()


def test_tiny_two_layers_paper_shape(workload, dev):
    # the paper's model: 2 layers, 16 hidden units
    run(workload("tiny", dev), dev, hidden=16, classes=7, W=4, steps=4, lr=0.05)


def test_small_two_layers_wide_head(workload, dev):
    run(workload("small", dev), dev, hidden=16, classes=47, W=4, steps=5, lr=0.05)


def test_products_mini_three_layers(workload, dev):
    run(workload("products_mini", dev), dev, hidden=16, classes=47, W=4, steps=3, lr=0.03)


def test_dense_mini_paper_model_shape_dim_602(workload, dev):
    """The paper's own model shape: 2 layers, 16 hidden units, fanout {25,10} over
    602-wide features (the Reddit-shaped config): layer 0 walks the feature row in slabs of 128."""
    w = workload("dense_mini", dev)
    assert w.dim == 602 and w.fanouts == [25, 10]
    run(w, dev, hidden=16, classes=41, W=4, steps=3, lr=0.02)


def test_consumer_without_host_sync_matches_synced_run(workload, dev):
    """gg_window_release(stream) orders the arena's reuse behind the consumer's work: a run that
    never synchronises the host between a batch's training step and the release (arenas =
    lookahead + 1, so the sampler is free to overwrite the arena at once) must give the losses of
    a run that synchronises after every step.  Before the release took a stream, window k+n's
    sampling raced the last steps of window k."""
    from paper_2606_02916_b200 import binding, epoch as ep
    w = workload("products_mini", dev)
    L = len(w.fanouts)
    dims = [w.dim] + [16] * (L - 1) + [47]
    stream = torch.cuda.Stream(dev)
    labels = torch.from_numpy(np.random.default_rng(3).integers(0, 47, (len(w.batches), 512)).astype(np.int32)).to(dev)
    runs = []
    for sync in (True, False, False):
        model = binding.Sage(init_params(dims, 5), dev)
        g = ep.graph_from_workload(w, max_window=2, max_live_windows=3)
        feats = torch.empty(w.num_nodes, w.dim, dtype=w.dtype, device=dev)
        losses = []

        def on_batch(k, j, bi, r):
            n_seed = r["blocks"][0]["n_dst"]
            loss = model.step(r, labels[bi, :n_seed].contiguous(), 0.03, stream)
            with torch.cuda.stream(stream):
                losses.append(loss.clone())
            if sync:
                torch.cuda.synchronize()

        with torch.cuda.stream(stream):
            for e in range(2):
                ep.run_epoch(g, w.batches, w.fanouts, 2, feats, on_batch=on_batch, stream=stream, lookahead=2,
                             first_window_id=1000 * e)
        torch.cuda.synchronize()
        runs.append(np.array([float(x.cpu()[0]) for x in losses]))
        model.close()
        g.close()
    assert len(runs[0]) == 2 * len(w.batches)
    for r in runs[1:]:
        assert np.allclose(r, runs[0], rtol=2e-4, atol=1e-6), float(np.abs(r - runs[0]).max())


def test_sage_errors(workload, dev):
    from paper_2606_02916_b200 import binding
    with pytest.raises(binding.GreenGNNError):
        binding.Sage(init_params([200, 32, 4], 0), dev)          # feature dim > 128 into more than 16 hidden units
    with pytest.raises(binding.GreenGNNError):
        binding.Sage(init_params([64, 200, 16, 4], 0), dev)      # a hidden layer's input > 128
    with pytest.raises(binding.GreenGNNError):
        binding.Sage(init_params([2000, 16, 4], 0), dev)         # feature dim > 1024
    with pytest.raises(binding.GreenGNNError):
        binding.Sage(init_params([32, 100, 4], 0), dev)          # hidden dim > 64

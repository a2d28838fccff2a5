"""Pins of oracle/sage.py (GraphSAGE-mean consumer, NEXT-4): the mean aggregator against an
explicit loop, closed forms at zero weights, and the analytic backward pass against central
finite differences of the forward pass (which shares no code with it)."""
import numpy as np

from oracle import sage


def toy(seed=0, n_seed=5, dims=(7, 4, 3)):
    rng = np.random.default_rng(seed)
    L = len(dims) - 1
    # frontier sizes grow outward from the seeds; dst nodes are a prefix of the src nodes
    sizes = [n_seed]
    for _ in range(L):
        sizes.append(sizes[-1] + int(rng.integers(3, 8)))
    blocks = []
    for h in range(L):
        n_dst, n_src = sizes[h], sizes[h + 1]
        deg = rng.integers(0, 4, n_dst)
        deg[0] = 0                                           # an empty row
        indptr = np.concatenate([[0], np.cumsum(deg)]).astype(np.int32)
        src = rng.integers(0, n_src, int(indptr[-1])).astype(np.int32)
        blocks.append(dict(n_dst=n_dst, n_src=n_src, indptr=indptr, src_local=src))
    x = rng.normal(size=(sizes[-1], dims[0]))
    params = [dict(W_self=rng.normal(size=(dims[l], dims[l + 1])) * 0.5,
                   W_neigh=rng.normal(size=(dims[l], dims[l + 1])) * 0.5,
                   b=rng.normal(size=dims[l + 1]) * 0.1) for l in range(L)]
    labels = rng.integers(0, dims[-1], n_seed)
    return params, blocks, x, labels


def test_mean_aggregate_is_the_row_mean():
    _, blocks, x, _ = toy()
    blk = blocks[-1]
    agg = sage.mean_aggregate(x, blk["indptr"], blk["src_local"])
    for i in range(blk["n_dst"]):
        nb = blk["src_local"][blk["indptr"][i]:blk["indptr"][i + 1]]
        want = x[nb].mean(axis=0) if len(nb) else np.zeros(x.shape[1])
        assert np.allclose(agg[i], want, rtol=0, atol=1e-15)


def test_zero_weights_give_log_C_and_uniform_gradient():
    params, blocks, x, labels = toy()
    for p in params:
        for k in p:
            p[k][...] = 0.0
    logits, _ = sage.forward(params, blocks, x)
    loss, g = sage.loss_and_grad_logits(logits, labels)
    C = logits.shape[1]
    assert abs(loss - np.log(C)) < 1e-14
    assert np.allclose(g.sum(axis=1), 0.0, atol=1e-16)       # softmax - onehot sums to zero per row
    assert np.allclose(g[np.arange(len(labels)), labels], (1.0 / C - 1.0) / len(labels))


def test_backward_matches_finite_differences_of_forward():
    for dims in [(7, 4, 3), (5, 6, 4, 3), (6, 3)]:
        params, blocks, x, labels = toy(seed=len(dims), dims=dims)
        logits, cache = sage.forward(params, blocks, x)
        _, g = sage.loss_and_grad_logits(logits, labels)
        grads = sage.backward(params, cache, g)

        def loss_of():
            lg, _ = sage.forward(params, blocks, x)
            return sage.loss_and_grad_logits(lg, labels)[0]

        h = 1e-6
        rng = np.random.default_rng(9)
        for l, p in enumerate(params):
            for k in ("W_self", "W_neigh", "b"):
                for _ in range(6):
                    idx = tuple(int(rng.integers(0, s)) for s in p[k].shape)
                    old = p[k][idx]
                    p[k][idx] = old + h
                    lp = loss_of()
                    p[k][idx] = old - h
                    lm = loss_of()
                    p[k][idx] = old
                    assert abs((lp - lm) / (2 * h) - grads[l][k][idx]) < 1e-7, (dims, l, k, idx)


def test_sgd_steps_decrease_the_loss():
    params, blocks, x, labels = toy(seed=3)
    losses = [sage.step(params, blocks, x, labels, 0.1) for _ in range(20)]
    assert losses[-1] < losses[0] and all(np.isfinite(losses))

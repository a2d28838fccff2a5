"""CPU oracle of the consumer workload (NEXT-4): GraphSAGE with the mean aggregator over the
sampled blocks, forward + backward + SGD, in float64 numpy.  TEST INFRASTRUCTURE, NOT THE PRODUCT
(only tests/, __graft_entry__.smoke() and bench.py's cpu legs may import it; it imports nothing
from the CUDA package).

Paper: the model the staging overlaps with is a "2-layer GraphSAGE, 16 hidden units" trained on
the sampled blocks (Alg. 1 l.15 "Forward pass, backward pass, parameter update",
PAPER.md:176).  GraphSAGE-mean layer, as in the DGL SAGEConv the paper builds on:

    agg_i   = mean_{e in row i of the block} h_in[src_local[e]]      (0 if the row is empty)
    h_out_i = act(h_in[i] @ W_self + agg_i @ W_neigh + b)            (dst i is src i: the dst
                                                                     nodes are a prefix of the
                                                                     block's src nodes, reading S6)
    act = ReLU on every layer but the last; loss = mean over the seeds of the softmax
    cross-entropy against the labels; update W <- W - lr * dL/dW (plain SGD).

Layer l consumes block L-1-l (blocks are in hop order outward from the seeds, so the GNN walks
them from the outermost one in): layer 0 reads the gathered feature tensor X_b.
Readings: S27 no dropout and plain SGD (the paper trains with dropout 0.5 and lr
0.003 but names no optimiser; a deterministic consumer is what the parity bar needs).
"""
from __future__ import annotations

from typing import Dict, List, Sequence

import numpy as np


def mean_aggregate(h_in: np.ndarray, indptr: np.ndarray, src_local: np.ndarray) -> np.ndarray:
    n_dst = len(indptr) - 1
    agg = np.zeros((n_dst, h_in.shape[1]), dtype=np.float64)
    deg = np.diff(indptr).astype(np.int64)
    rows = np.repeat(np.arange(n_dst), deg)
    np.add.at(agg, rows, h_in[src_local])
    nz = deg > 0
    agg[nz] /= deg[nz, None]
    return agg


def forward(params: List[Dict[str, np.ndarray]], blocks: Sequence[Dict], x: np.ndarray):
    """blocks: hop order (0 = out of the seeds), each with n_dst, indptr, src_local.
    Returns (logits [n_seeds, C], cache for backward)."""
    L = len(params)
    h = np.asarray(x, dtype=np.float64)
    cache = []
    for l in range(L):
        blk = blocks[L - 1 - l]
        n_dst = int(blk["n_dst"])
        agg = mean_aggregate(h, np.asarray(blk["indptr"]), np.asarray(blk["src_local"]))
        pre = h[:n_dst] @ params[l]["W_self"] + agg @ params[l]["W_neigh"] + params[l]["b"]
        out = np.maximum(pre, 0.0) if l < L - 1 else pre
        cache.append(dict(h_in=h, agg=agg, pre=pre, blk=blk))
        h = out
    return h, cache


def loss_and_grad_logits(logits: np.ndarray, labels: np.ndarray):
    m = logits.max(axis=1, keepdims=True)
    z = logits - m
    lse = np.log(np.exp(z).sum(axis=1, keepdims=True))
    logp = z - lse
    n = logits.shape[0]
    loss = -float(logp[np.arange(n), labels].sum()) / n
    g = np.exp(logp)
    g[np.arange(n), labels] -= 1.0
    return loss, g / n


def backward(params, cache, d_logits: np.ndarray):
    L = len(params)
    grads = [None] * L
    d_out = d_logits
    for l in range(L - 1, -1, -1):
        c = cache[l]
        d_pre = d_out * (c["pre"] > 0) if l < L - 1 else d_out
        blk = c["blk"]
        n_dst = int(blk["n_dst"])
        indptr, src_local = np.asarray(blk["indptr"]), np.asarray(blk["src_local"])
        grads[l] = dict(W_self=c["h_in"][:n_dst].T @ d_pre, W_neigh=c["agg"].T @ d_pre, b=d_pre.sum(axis=0))
        if l > 0:
            d_h = np.zeros_like(c["h_in"])
            d_h[:n_dst] += d_pre @ params[l]["W_self"].T
            d_agg = d_pre @ params[l]["W_neigh"].T
            deg = np.diff(indptr).astype(np.int64)
            rows = np.repeat(np.arange(n_dst), deg)
            scale = np.zeros(n_dst)
            scale[deg > 0] = 1.0 / deg[deg > 0]
            np.add.at(d_h, src_local, d_agg[rows] * scale[rows, None])
            d_out = d_h
    return grads


def step(params, blocks, x, labels, lr: float) -> float:
    """One training step in place (Alg. 1 l.15); returns the loss before the update."""
    logits, cache = forward(params, blocks, x)
    loss, g = loss_and_grad_logits(logits, np.asarray(labels))
    grads = backward(params, cache, g)
    for p, d in zip(params, grads):
        for k in ("W_self", "W_neigh", "b"):
            p[k] -= lr * d[k]
    return loss

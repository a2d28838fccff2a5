"""Example: one window of a workload through the whole path, each gather followed by one
GraphSAGE-mean training step (gg_sage_step) -- Algorithm 1 lines 8-15 of the paper for one window.

    python -m paper_2606_02916_b200.examples.consumer_step [--config products] [--window 4] [--hidden 16] [--classes 47]

Every size comes from the workload and from what the library reports (gg_batch_info); the model is
the paper's shape (one layer per sampled hop, `hidden` units) with random initial
weights and random labels.  Needs a CUDA device (there is no CPU fallback).
"""
import argparse

import numpy as np
import torch

from paper_2606_02916_b200 import binding, build, epoch as ep, inputs


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--config", default="products", choices=sorted(inputs.CONFIGS))
    ap.add_argument("--window", type=int, default=4, help="W: mini-batches staged and served as one window")
    ap.add_argument("--hidden", type=int, default=16)
    ap.add_argument("--classes", type=int, default=47)
    ap.add_argument("--lr", type=float, default=0.003)
    a = ap.parse_args()
    build.build_library()
    dev = torch.device("cuda", 0)
    w = inputs.make_workload(a.config, device=dev)
    W = min(a.window, len(w.batches))
    g = ep.graph_from_workload(w, max_window=W)
    L = len(w.fanouts)
    dims = [w.dim] + [a.hidden] * (L - 1) + [a.classes]
    rng = np.random.default_rng(7)
    p0 = [dict(W_self=(rng.uniform(-1, 1, (dims[l], dims[l + 1])) / np.sqrt(dims[l])).astype(np.float32),
               W_neigh=(rng.uniform(-1, 1, (dims[l], dims[l + 1])) / np.sqrt(dims[l])).astype(np.float32),
               b=np.zeros(dims[l + 1], np.float32)) for l in range(L)]
    model = binding.Sage(p0, dev)
    g.window_stage(0, 0, w.batches[:W], w.fanouts)
    rows = max(g.batch_info(0, j)["n_input"] for j in range(W))
    feats = torch.empty(rows, w.dim, dtype=w.dtype, device=dev)
    for j in range(W):
        r = g.batch_gather(0, j, feats)
        labels = torch.randint(0, a.classes, (r["blocks"][0]["n_dst"],), dtype=torch.int32, device=dev)
        model.step(r, labels, a.lr)
        print("batch %d: loss %.4f, blocks (n_dst, n_src, n_edge) = %s"
              % (j, float(model.loss.cpu()[0]), [(b["n_dst"], b["n_src"], b["n_edge"]) for b in r["blocks"]]))
    g.window_release(0)
    model.close()
    g.close()


if __name__ == "__main__":
    main()

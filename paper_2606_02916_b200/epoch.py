"""Epoch driver over the C ABI: the pipelined loop of Algorithm 1.

    stage(0) .. stage(d-1); for k: stage(k+d); gather every batch of window k; release(k)

with lookahead d = 2 by default: while window k is served, window k+1's cache is being staged
(select / delta / bulk copies) and window k+2 is being sampled (the library runs the two phases
on two threads and two side streams).  d = 1 is the literal loop of Algorithm 1.

Pure call sequencing -- all computation happens in libgreengnn.so.  `on_batch` receives every
gathered batch (used by the parity tests and by the end-to-end bench leg).
"""
from __future__ import annotations

from typing import Callable, Dict, List, Optional, Sequence

import numpy as np
import torch

from .binding import Graph


def graph_from_workload(w, n_hot: int = -1, carry_over: int = 1, max_window: int = 32,
                        staging_mode: int = 0, max_cache_rows: int = 0, host_threads: int = 0,
                        max_batch: Optional[int] = None, max_live_windows: int = 0, cache_buffers: int = 0,
                        max_input_nodes: int = 0) -> Graph:
    """Builds a gg_graph over an inputs.Workload whose graph and local features are on a CUDA device."""
    mb = max_batch or max(len(b) for b in w.batches)
    return Graph(w.indptr, w.indices, w.part_offsets, w.local_part, w.feat_parts, seed=w.seed,
                 n_hot=n_hot, carry_over=carry_over, max_layers=len(w.fanouts), max_window=max_window,
                 max_batch=mb, max_cache_rows=max_cache_rows, max_input_nodes=max_input_nodes, staging_mode=staging_mode,
                 host_threads=host_threads, max_live_windows=max_live_windows, cache_buffers=cache_buffers)


def windows_of(n_batches: int, W: int) -> List[range]:
    """ceil(B/W) windows of W consecutive batches, the last one partial."""
    return [range(s, min(n_batches, s + W)) for s in range(0, n_batches, W)]


def run_epoch(g: Graph, batches: Sequence[np.ndarray], fanouts: Sequence[int], W: int,
              features: torch.Tensor, on_batch: Optional[Callable[[int, int, int, Dict], None]] = None,
              on_window: Optional[Callable[[int, range], None]] = None,
              stream: Optional[torch.cuda.Stream] = None, first_window_id: int = 0,
              lookahead: int = 2) -> int:
    """One epoch.  Returns the number of gather launches issued.  `features` is the caller's
    [capacity_rows, dim] device buffer reused for every batch."""
    wins = windows_of(len(batches), W)
    if not wins:
        return 0
    wid = first_window_id
    assert lookahead >= 1   # at most max_live_windows - 1 (the library returns GG_ERR_STATE beyond)
    for k in range(min(lookahead, len(wins))):
        g.window_stage(wid + k, wins[k].start, [batches[i] for i in wins[k]], fanouts)
    n = 0
    for k, win in enumerate(wins):
        if k + lookahead < len(wins):
            nxt = wins[k + lookahead]
            g.window_stage(wid + k + lookahead, nxt.start, [batches[i] for i in nxt], fanouts)
        for j, bi in enumerate(win):
            r = g.batch_gather(wid + k, j, features, stream)
            n += 1
            if on_batch is not None:
                on_batch(k, j, bi, r)
        if on_window is not None:
            on_window(wid + k, win)
        g.window_release(wid + k, stream)      # the arena is recycled only behind on_batch's work on `stream`
    return n


def choose_window(g: Graph, batches: Sequence[np.ndarray], fanouts: Sequence[int], candidates: Sequence[int],
                  model: Dict) -> int:
    """The paper's offline phase for one epoch: replay the trace for every
    candidate W on the device (gg_simulate) and return W* = argmin E_phy(W)."""
    return int(g.simulate(batches, fanouts, [int(c) for c in candidates], model)["best"])


def run_adaptive(g: Graph, batches: Sequence[np.ndarray], fanouts: Sequence[int], candidates: Sequence[int],
                 measure_model: Callable[[], Dict], epochs: int, features: torch.Tensor,
                 stream: Optional[torch.cuda.Stream] = None, lookahead: int = 2) -> List[int]:
    """NEXT-2, "adaptive W across epochs": before every epoch the coefficients are
    re-measured (`measure_model()`, e.g. profiler.measure_energy_model) and W* is re-selected, so
    a change of the link or of the power state moves the window size.  The trace itself repeats
    (PAPER.md:126), so with constant coefficients W* is constant.  Returns the W used per epoch.
    Pure call sequencing: everything is computed by gg_simulate and the runtime path."""
    used = []
    for e in range(epochs):
        model = {k: v for k, v in measure_model().items() if k not in ("probes", "p_active")}
        W = choose_window(g, batches, fanouts, candidates, model)
        run_epoch(g, batches, fanouts, W, features, stream=stream, first_window_id=10 ** 7 + 10 ** 5 * e,
                  lookahead=lookahead)
        used.append(W)
    return used

"""ctypes wrapper of the CPU oracle (oracle/ggo.cpp).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs import this.  It imports nothing from the CUDA package.  `build()` compiles
oracle/ggo.cpp with g++ (no CUDA headers); `load()` builds on demand.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ggo.cpp")
_LIB = os.path.join(_HERE, "libggo.so")
_lib = None

u64, i64, i32, vp = C.c_uint64, C.c_int64, C.c_int32, C.c_void_p


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def _p(a: np.ndarray):
    return a.ctypes.data_as(vp)


def load():
    global _lib
    if _lib is not None:
        return _lib
    lib = C.CDLL(build())
    sig = {
        "ggo_fmix": (u64, [u64]), "ggo_sm": (u64, [u64]),
        "ggo_h_dst": (u64, [u64] * 4), "ggo_key": (u64, [u64] * 5),
        "ggo_set_key_hook": (None, [vp]),
        "ggo_sample_dst": (i64, [i64, vp, vp, i32, i32, u64, u64, u64, vp, vp]),
        "ggo_batch_sample": (vp, [i64, vp, vp, vp, i32, vp, i32, u64, u64]),
        "ggo_batch_free": (None, [vp]),
        "ggo_batch_n_front": (i32, [vp, i32]), "ggo_batch_n_edge": (i32, [vp, i32]),
        "ggo_batch_nodes": (None, [vp, vp]), "ggo_batch_block": (None, [vp, i32, vp, vp, vp]),
        "ggo_state_create": (vp, [i64, i32, vp, i32, i64, i32]),
        "ggo_state_free": (None, [vp]), "ggo_state_reset": (None, [vp]),
        "ggo_state_cache_size": (i64, [vp]), "ggo_state_cache": (None, [vp, vp]),
        "ggo_window_run": (vp, [vp, vp, i32]), "ggo_window_free": (None, [vp]),
        "ggo_window_size": (i64, [vp, i32]),
        "ggo_window_uniq": (None, [vp, vp, vp]), "ggo_window_hot": (None, [vp, vp]),
        "ggo_window_carried": (None, [vp, vp]),
        "ggo_window_staged_rows": (i64, [vp, i32]), "ggo_window_delta_rows": (i64, [vp, i32]),
        "ggo_window_delta": (None, [vp, i32, vp]),
        "ggo_window_batch": (None, [vp, i32, vp, vp]),
        "ggo_window_misses": (None, [vp, i32, vp, vp]),
        "ggo_gather": (None, [vp, i64, i32, vp, vp, i64, i64, vp]),
    }
    for name, (res, args) in sig.items():
        f = getattr(lib, name)
        f.restype, f.argtypes = res, args
    _lib = lib
    return lib


KEY_HOOK = C.CFUNCTYPE(u64, u64, u64)


def fmix(z: int) -> int:
    return load().ggo_fmix(z)


def sm(x: int) -> int:
    return load().ggo_sm(x)


def h_dst(seed: int, batch: int, layer: int, dst: int) -> int:
    return load().ggo_h_dst(seed, batch, layer, dst)


def key(seed: int, batch: int, layer: int, dst: int, j: int) -> int:
    return load().ggo_key(seed, batch, layer, dst, j)


def set_key_hook(fn) -> None:
    """fn: a KEY_HOOK instance (keep a reference alive) or None."""
    load().ggo_set_key_hook(C.cast(fn, vp) if fn is not None else None)


class Graph:
    """Host CSR: indptr int64[N+1], indices int32[nnz]; row v = nodes v aggregates from."""

    def __init__(self, indptr: np.ndarray, indices: np.ndarray):
        self.indptr = np.ascontiguousarray(indptr, dtype=np.int64)
        self.indices = np.ascontiguousarray(indices, dtype=np.int32)
        self.n = int(self.indptr.shape[0] - 1)


def sample_dst(g: Graph, v: int, fanout: int, seed: int, batch: int, layer: int):
    """O1. Returns (positions int64[], neighbor ids int32[]) in ascending position."""
    deg = int(g.indptr[v + 1] - g.indptr[v])
    k = min(deg, fanout)
    pos = np.empty(max(k, 1), dtype=np.int64)
    ids = np.empty(max(k, 1), dtype=np.int32)
    c = load().ggo_sample_dst(g.n, _p(g.indptr), _p(g.indices), v, fanout, seed, batch, layer,
                              _p(pos), _p(ids))
    return pos[:c].copy(), ids[:c].copy()


class Batch:
    """O2 result for one mini-batch: blocks (hop order, 0 = out of the seeds) and N_b."""

    def __init__(self, g: Graph, seeds: np.ndarray, fanouts: Sequence[int], seed: int,
                 batch_index: int):
        lib = load()
        seeds = np.ascontiguousarray(seeds, dtype=np.int32)
        fo = np.ascontiguousarray(fanouts, dtype=np.int32)
        self.L = len(fo)
        self._h = lib.ggo_batch_sample(g.n, _p(g.indptr), _p(g.indices), _p(seeds), len(seeds),
                                       _p(fo), self.L, seed, batch_index)
        self.n_front = [lib.ggo_batch_n_front(self._h, h) for h in range(self.L + 1)]
        self.nodes = np.empty(self.n_front[-1], dtype=np.int32)
        lib.ggo_batch_nodes(self._h, _p(self.nodes))
        self.blocks = []
        for h in range(self.L):
            ne = lib.ggo_batch_n_edge(self._h, h)
            ip = np.empty(self.n_front[h] + 1, dtype=np.int32)
            sg = np.empty(ne, dtype=np.int32)
            sl = np.empty(ne, dtype=np.int32)
            lib.ggo_batch_block(self._h, h, _p(ip), _p(sg), _p(sl))
            self.blocks.append(dict(n_dst=self.n_front[h], n_src=self.n_front[h + 1], n_edge=ne,
                                    indptr=ip, src_global=sg, src_local=sl))

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.ggo_batch_free(self._h)
            self._h = None


class WindowResult:
    pass


class State:
    """Cache state C across windows (C_0 = empty) plus the owner map and the budget."""

    def __init__(self, n: int, part_offsets: np.ndarray, local_part: int, n_hot: int = -1,
                 carry_over: int = 1):
        self.po = np.ascontiguousarray(part_offsets, dtype=np.int64)
        self.P = len(self.po) - 1
        self._h = load().ggo_state_create(n, self.P, _p(self.po), local_part, n_hot, carry_over)

    def reset(self):
        load().ggo_state_reset(self._h)

    def cache(self) -> np.ndarray:
        lib = load()
        out = np.empty(lib.ggo_state_cache_size(self._h), dtype=np.int32)
        lib.ggo_state_cache(self._h, _p(out))
        return out

    def run_window(self, batches: List[Batch]) -> WindowResult:
        """O3..O7 for one window of already-sampled batches; advances C."""
        lib = load()
        W = len(batches)
        arr = (vp * W)(*[b._h for b in batches])
        w = lib.ggo_window_run(self._h, arr, W)
        r = WindowResult()
        nu, nr, nh, nc, na = (lib.ggo_window_size(w, k) for k in range(5))
        r.W, r.n_unique, r.n_unique_remote, r.n_hot, r.carried_rows, r.n_access = W, nu, nr, nh, nc, na
        r.uniq = np.empty(nu, dtype=np.int32)
        r.cnt = np.empty(nu, dtype=np.int32)
        lib.ggo_window_uniq(w, _p(r.uniq), _p(r.cnt))
        r.hot = np.empty(nh, dtype=np.int32)
        lib.ggo_window_hot(w, _p(r.hot))
        r.carried = np.empty(nc, dtype=np.int32)
        lib.ggo_window_carried(w, _p(r.carried))
        r.staged_rows = [lib.ggo_window_staged_rows(w, m) for m in range(self.P)]
        r.bulk_rows = [lib.ggo_window_delta_rows(w, m) for m in range(self.P)]
        r.delta = []
        for m in range(self.P):
            d = np.empty(r.bulk_rows[m], dtype=np.int32)
            lib.ggo_window_delta(w, m, _p(d))
            r.delta.append(d)
        r.n_input, r.hit_local, r.hit_cache, r.miss, r.miss_pos, r.miss_id = [], [], [], [], [], []
        for b in range(W):
            o4 = np.empty(4, dtype=np.int32)
            mo = np.empty(self.P, dtype=np.int32)
            lib.ggo_window_batch(w, b, _p(o4), _p(mo))
            r.n_input.append(int(o4[0]))
            r.hit_local.append(int(o4[1]))
            r.hit_cache.append(int(o4[2]))
            r.miss.append(mo.copy())
            mp = np.empty(int(o4[3]), dtype=np.int32)
            mi = np.empty(int(o4[3]), dtype=np.int32)
            lib.ggo_window_misses(w, b, _p(mp), _p(mi))
            r.miss_pos.append(mp)
            r.miss_id.append(mi)
        lib.ggo_window_free(w)
        return r

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.ggo_state_free(self._h)
            self._h = None


def gather(nodes: np.ndarray, part_offsets: np.ndarray, parts: Sequence[np.ndarray],
           row_bytes: int, stride: Optional[int] = None) -> np.ndarray:
    """O6 feature tensor as raw bytes [len(nodes), row_bytes]; parts[m] = owner m's rows
    as a C-contiguous uint8 array [rows_m, stride]."""
    nodes = np.ascontiguousarray(nodes, dtype=np.int32)
    po = np.ascontiguousarray(part_offsets, dtype=np.int64)
    P = len(po) - 1
    stride = row_bytes if stride is None else stride
    base = (vp * P)(*[p.ctypes.data for p in parts])
    out = np.empty((len(nodes), row_bytes), dtype=np.uint8)
    load().ggo_gather(_p(nodes), len(nodes), P, _p(po), base, stride, row_bytes, _p(out))
    return out

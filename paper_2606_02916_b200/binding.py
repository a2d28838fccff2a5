"""Thin ctypes binding of include/greengnn.h: argument marshalling only.

Every step of the path runs inside libgreengnn.so's CUDA kernels; torch is used here for
device memory (`data_ptr()`), streams and zero-copy views of the library's device arrays.
There is NO CPU fallback: if the library has not been built or cannot be loaded this module
raises (build with `python -m paper_2606_02916_b200.build`).
"""
from __future__ import annotations

import contextlib
import ctypes as C
import os
from typing import Dict, List, Optional, Sequence

import numpy as np
import torch

from . import build as _build

GG_MAX_LAYERS, GG_MAX_PARTS, GG_MAX_FANOUT, GG_MAX_WINDOW = 8, 16, 96, 255
GG_STATIC_MAX_NODES = 1 << 22
GG_OK, GG_ERR_INVALID_ARG, GG_ERR_STATE, GG_ERR_CAPACITY, GG_ERR_OOM, GG_ERR_CUDA = range(6)
_STATUS = {0: "GG_OK", 1: "GG_ERR_INVALID_ARG", 2: "GG_ERR_STATE", 3: "GG_ERR_CAPACITY",
           4: "GG_ERR_OOM", 5: "GG_ERR_CUDA"}

i32, i64, u64, vp, f32 = C.c_int32, C.c_int64, C.c_uint64, C.c_void_p, C.c_float


class gg_csr(C.Structure):
    _fields_ = [("num_nodes", i64), ("num_edges", i64), ("indptr", vp), ("indices", vp)]


class gg_owner_map(C.Structure):
    _fields_ = [("num_parts", i32), ("local_part", i32), ("part_offsets", vp)]


class gg_feature_store(C.Structure):
    _fields_ = [("dim", i32), ("dtype", i32), ("row_stride_bytes", i64), ("part_base", vp)]


class gg_config(C.Structure):
    _fields_ = [("seed", u64), ("n_hot", i64), ("carry_over", i32), ("max_layers", i32),
                ("max_window", i32), ("max_batch", i32), ("max_cache_rows", i64),
                ("max_input_nodes", i64), ("staging_mode", i32), ("host_threads", i32), ("cache_buffers", i32), ("max_live_windows", i32)]


class gg_block(C.Structure):
    _fields_ = [("n_dst", i32), ("n_src", i32), ("n_edge", i32), ("indptr", vp), ("src_local", vp),
                ("src_global", vp)]


class gg_batch_out(C.Structure):
    _fields_ = [("num_layers", i32), ("blocks", gg_block * GG_MAX_LAYERS), ("n_input", i32),
                ("input_nodes", vp), ("features", vp), ("features_capacity_rows", i64),
                ("miss_pos", vp), ("miss_id", vp), ("n_miss", vp)]


class gg_window_trace(C.Structure):
    _fields_ = [("W", i32), ("num_parts", i32), ("n_access", i64), ("n_unique", i64),
                ("n_unique_remote", i64), ("n_hot", i64), ("carried_rows", i64),
                ("staged_rows", i64 * GG_MAX_PARTS), ("bulk_rows", i64 * GG_MAX_PARTS),
                ("bulk_bytes", i64 * GG_MAX_PARTS), ("bulk_copies", i32),
                ("n_input", vp), ("hit_local", vp), ("hit_cache", vp), ("miss", vp),
                ("ms_sample", f32), ("ms_unique", f32), ("ms_select", f32), ("ms_pack_host", f32),
                ("ms_h2d", f32), ("ms_carry", f32), ("ms_stage_total", f32), ("ms_boundary_wait", f32)]


class gg_profile(C.Structure):
    _fields_ = [("ms", C.c_double * 9), ("regions", i64 * 9), ("bytes", i64 * 9)]


class gg_energy_model(C.Structure):
    _fields_ = [(n, C.c_double * GG_MAX_PARTS) for n in
                ("eps_init", "eps_pay_a", "eps_pay_b", "lam_init", "lam_pay_a", "lam_pay_b")] + \
               [("bw_bytes_per_s", C.c_double), ("p_idle_w", C.c_double)]


class gg_sim_result(C.Structure):
    _fields_ = [("W", i32), ("n_windows", i32)] + \
               [(n, i64) for n in ("rebuild_events", "miss_events", "rebuild_rows", "miss_rows",
                                   "n_access", "n_remote_access", "hit_local", "hit_cache")] + \
               [(n, C.c_double) for n in ("e_rebuild", "e_miss", "t_stall", "e_stall", "e_phy", "hit_ratio")]


PROF_KINDS = ["gather", "miss", "sample", "frontier", "unique", "select", "stage_copy", "carry", "wait"]

SYMBOLS = ["gg_profile_enable", "gg_profile_get", "gg_launch_count", "gg_graph_create", "gg_graph_destroy", "gg_window_stage", "gg_batch_info",
           "gg_batch_gather", "gg_window_release", "gg_trace", "gg_window_export", "gg_cache_read",
           "gg_cache_reset", "gg_key", "gg_last_error", "gg_version", "gg_sampler_stats", "gg_debug_sampler", "gg_sampler_tune", "gg_key_peak", "gg_simulate", "gg_rank_calibrate",
           "gg_sage_create", "gg_sage_destroy", "gg_sage_step", "gg_sage_params", "gg_unique_count_static"]

_lib = None


class GreenGNNError(RuntimeError):
    def __init__(self, status: int, text: str):
        super().__init__("%s: %s" % (_STATUS.get(status, status), text))
        self.status = status


def load_library(path: Optional[str] = None):
    """Loads libgreengnn.so; raises if it is missing (no fallback of any kind)."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    path = path or _build.LIB
    if not os.path.exists(path):
        raise ImportError("libgreengnn.so is not built (%s); run `python -m paper_2606_02916_b200.build`"
                          % path)
    lib = C.CDLL(path)
    P = C.POINTER
    lib.gg_graph_create.argtypes = [P(gg_csr), P(gg_owner_map), P(gg_feature_store), P(gg_config), P(vp)]
    lib.gg_graph_destroy.argtypes = [vp]
    lib.gg_window_stage.argtypes = [vp, i64, u64, vp, vp, i32, vp, i32]
    lib.gg_batch_info.argtypes = [vp, i64, i32, P(gg_batch_out)]
    lib.gg_batch_gather.argtypes = [vp, i64, i32, P(gg_batch_out), vp]
    lib.gg_window_release.argtypes = [vp, i64, vp]
    lib.gg_trace.argtypes = [vp, i64, P(gg_window_trace)]
    lib.gg_window_export.argtypes = [vp, i64, i32, vp, i64, P(i64)]
    lib.gg_cache_read.argtypes = [vp, i64, vp, i64, vp]
    lib.gg_cache_reset.argtypes = [vp]
    lib.gg_profile_enable.argtypes = [vp, i32]
    lib.gg_profile_get.argtypes = [vp, P(gg_profile)]
    lib.gg_launch_count.restype = u64
    lib.gg_key.argtypes = [u64] * 5
    lib.gg_key.restype = u64
    lib.gg_sampler_stats.argtypes = [P(u64), P(u64), P(u64)]
    lib.gg_debug_sampler.argtypes = [i32, C.c_float]
    lib.gg_sampler_tune.argtypes = [i32, i32, i32]
    lib.gg_key_peak.argtypes = [i32, i32, i32, P(C.c_double), P(C.c_uint32)]
    lib.gg_simulate.argtypes = [vp, vp, vp, i32, u64, vp, i32, vp, i32, P(gg_energy_model), P(gg_sim_result),
                                P(i32), vp, vp]
    lib.gg_rank_calibrate.argtypes = [vp, vp, i32, i32, C.c_double, C.c_double, i32, vp, vp, vp]
    lib.gg_sage_create.argtypes = [i32, vp, vp, vp, vp, P(vp)]
    lib.gg_sage_destroy.argtypes = [vp]
    lib.gg_sage_step.argtypes = [vp, P(gg_batch_out), vp, C.c_float, vp, vp]
    lib.gg_sage_params.argtypes = [vp, i32, vp, vp, vp]
    lib.gg_unique_count_static.argtypes = [vp, i64, i64, vp, vp, i64, vp, vp]
    lib.gg_last_error.restype = C.c_char_p
    lib.gg_version.restype = C.c_char_p
    for s in SYMBOLS:
        getattr(lib, s)
        if s not in ("gg_key", "gg_last_error", "gg_version", "gg_launch_count"):
            getattr(lib, s).restype = i32
    _lib = lib
    return lib


def launch_count() -> int:
    return int(load_library().gg_launch_count())


def _check_global(rc: int):
    if rc != 0:
        raise GreenGNNError(rc, (load_library().gg_last_error() or b"").decode())


def sampler_stats() -> dict:
    """Cumulative a-1 counters: keys evaluated (algorithmic), keyed rows, exact-path fallbacks."""
    k, r, f = u64(0), u64(0), u64(0)
    _check_global(load_library().gg_sampler_stats(C.byref(k), C.byref(r), C.byref(f)))
    return {"keys": int(k.value), "rows": int(r.value), "fallbacks": int(f.value)}


def sampler_tune(single_bins: int = 36, warp_bin: int = 36, hub_bin: int = 128) -> None:
    """Degree-bin cut-overs of the selection kernels (include/greengnn.h gg_sampler_tune)."""
    _check_global(load_library().gg_sampler_tune(single_bins, warp_bin, hub_bin))


def key_peak(ctas_per_sm: int = 8, keys_per_lane: int = 65536, reps: int = 5, with_fold: bool = False):
    """Measured integer-ALU roofline of the sampler: keys/s of the key-only micro-kernel."""
    v, f = C.c_double(0.0), C.c_uint32(0)
    _check_global(load_library().gg_key_peak(ctas_per_sm, keys_per_lane, reps, C.byref(v), C.byref(f)))
    return (float(v.value), int(f.value)) if with_fold else float(v.value)


def debug_sampler(rank_shift: int = 0, want_add: float = 0.0) -> None:
    """Test knobs of the selection kernel (include/greengnn.h gg_debug_sampler)."""
    _check_global(load_library().gg_debug_sampler(rank_shift, want_add))


def rank_calibrate(Z: np.ndarray, e_gt: np.ndarray, lam: float, lr: float, iters: int):
    """Eq. (5) fit on the device (gg_rank_calibrate).  Returns (beta[F], gamma[n], loss)."""
    Z = np.ascontiguousarray(Z, dtype=np.float64)
    e = np.ascontiguousarray(e_gt, dtype=np.float64)
    n, F = Z.shape
    beta, gamma, loss = np.zeros(max(F, 1)), np.zeros(n), np.zeros(1)
    _check_global(load_library().gg_rank_calibrate(Z.ctypes.data, e.ctypes.data, n, F, lam, lr, iters,
                                                   beta.ctypes.data, gamma.ctypes.data, loss.ctypes.data))
    return beta[:F], gamma, float(loss[0])


def unique_count_static(ids: torch.Tensor, num_nodes: int, uniq: torch.Tensor, cnt: torch.Tensor,
                        stats: torch.Tensor, stream: Optional[torch.cuda.Stream] = None) -> None:
    """gg_unique_count_static: U_k / c_k of the device ID list `ids` into the caller's device tensors
    `uniq`, `cnt` (int32, same length = capacity) and `stats` (int32 [2]: |U|, IDs skipped), without
    any device allocation inside the library -- for callers whose allocator owns all of the HBM or
    who cannot afford the device-wide wait of a cudaFree.  num_nodes <= GG_STATIC_MAX_NODES.
    Asynchronous on `stream` (default: torch's current stream); nothing is written to uniq / cnt when
    stats[0] > len(uniq).  Calls that may overlap on the GPU share one workspace and race."""
    for t in (ids, uniq, cnt, stats):
        assert t.is_cuda and t.dtype == torch.int32 and t.is_contiguous()
    assert uniq.numel() == cnt.numel() and stats.numel() >= 2
    st = stream if stream is not None else torch.cuda.current_stream(ids.device)
    with torch.cuda.device(ids.device):
        _check_global(load_library().gg_unique_count_static(
            ids.data_ptr() if ids.numel() else None, ids.numel(), num_nodes,
            uniq.data_ptr() if uniq.numel() else None, cnt.data_ptr() if cnt.numel() else None,
            uniq.numel(), stats.data_ptr(), st.cuda_stream))


class Sage:
    """GraphSAGE-mean consumer (NEXT-4) over the blocks gg_batch_gather returns.
    params: list per layer of dicts W_self [din, dout], W_neigh [din, dout], b [dout] (float32)."""

    def __init__(self, params: Sequence[Dict[str, np.ndarray]], device):
        self.lib = load_library()
        self.device = torch.device(device)
        self.dims = [int(params[0]["W_self"].shape[0])] + [int(p["W_self"].shape[1]) for p in params]
        L = len(params)
        keep = [[np.ascontiguousarray(p[k], dtype=np.float32) for p in params] for k in ("W_self", "W_neigh", "b")]
        arrs = [(vp * L)(*[a.ctypes.data for a in ks]) for ks in keep]
        dims = np.ascontiguousarray(self.dims, dtype=np.int32)
        h = vp()
        with torch.cuda.device(self.device):
            _check_global(self.lib.gg_sage_create(L, dims.ctypes.data, arrs[0], arrs[1], arrs[2], C.byref(h)))
        self.h, self.L = h, L
        self.loss = torch.zeros(1, dtype=torch.float32, device=self.device)

    def step(self, r: Dict, labels: torch.Tensor, lr: float, stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
        """One training step on the batch dict Graph.batch_gather returned; labels: int32 device
        tensor [n_seeds].  Returns the (device) loss tensor of this step (asynchronous)."""
        assert labels.is_cuda and labels.dtype == torch.int32 and labels.is_contiguous()
        st = stream if stream is not None else torch.cuda.current_stream(self.device)
        _check_global(self.lib.gg_sage_step(self.h, C.byref(r["_out"]), labels.data_ptr(), lr, st.cuda_stream,
                                            self.loss.data_ptr()))
        return self.loss

    def params(self) -> List[Dict[str, np.ndarray]]:
        out = []
        for l in range(self.L):
            ws = np.zeros((self.dims[l], self.dims[l + 1]), np.float32)
            wn = np.zeros_like(ws)
            b = np.zeros(self.dims[l + 1], np.float32)
            _check_global(self.lib.gg_sage_params(self.h, l, ws.ctypes.data, wn.ctypes.data, b.ctypes.data))
            out.append(dict(W_self=ws, W_neigh=wn, b=b))
        return out

    def close(self):
        if self.h:
            self.lib.gg_sage_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def gg_key(seed: int, batch: int, layer: int, dst: int, edge_pos: int) -> int:
    return load_library().gg_key(seed, batch, layer, dst, edge_pos)


class _DevView:
    """Zero-copy torch view of `n` elements of library-owned device memory."""

    def __init__(self, ptr: int, n: int, typestr: str):
        self.__cuda_array_interface__ = {"shape": (n,), "typestr": typestr, "data": (ptr, False),
                                         "version": 2, "strides": None}


def _view_i32(ptr, n: int, device) -> torch.Tensor:
    if n == 0 or not ptr:
        return torch.empty(0, dtype=torch.int32, device=device)
    return torch.as_tensor(_DevView(int(ptr), int(n), "<i4"), device=device)


class Graph:
    """gg_graph handle.  Tensors passed in are borrowed and kept referenced here."""

    def __init__(self, indptr: torch.Tensor, indices: torch.Tensor, part_offsets: Sequence[int],
                 local_part: int, feat_parts: List[torch.Tensor], seed: int, n_hot: int = -1,
                 carry_over: int = 1, max_layers: int = 3, max_window: int = 32, max_batch: int = 1024,
                 max_cache_rows: int = 0, max_input_nodes: int = 0, staging_mode: int = 0,
                 host_threads: int = 0, max_live_windows: int = 0, cache_buffers: int = 0):
        self.lib = load_library()
        assert indptr.dtype == torch.int64 and indices.dtype == torch.int32
        self._keep = (indptr, indices, feat_parts)
        self.device = indptr.device
        self.P = len(part_offsets) - 1
        self.po = np.ascontiguousarray(part_offsets, dtype=np.int64)
        self.dim = int(feat_parts[local_part].shape[1])
        self.feat_dtype = feat_parts[local_part].dtype
        esz = feat_parts[local_part].element_size()
        self.rb = self.dim * esz
        csr = gg_csr(indptr.numel() - 1, indices.numel(), indptr.data_ptr(), indices.data_ptr())
        om = gg_owner_map(self.P, local_part, self.po.ctypes.data)
        bases = (vp * self.P)(*[p.data_ptr() if p.numel() else None for p in feat_parts])
        strides = {int(p.stride(0)) * esz for p in feat_parts if p.numel()}
        assert len(strides) == 1, "all parts must share one row stride"
        fs = gg_feature_store(self.dim, {torch.float32: 0, torch.bfloat16: 1}[self.feat_dtype],
                              strides.pop(), C.cast(bases, vp))
        cfg = gg_config(seed & ((1 << 64) - 1), n_hot, carry_over, max_layers, max_window, max_batch,
                        max_cache_rows, max_input_nodes, staging_mode, host_threads, cache_buffers, max_live_windows)
        h = vp()
        ctx = torch.cuda.device(self.device) if self.device.type == "cuda" else contextlib.nullcontext()
        with ctx:
            self._check(self.lib.gg_graph_create(C.byref(csr), C.byref(om), C.byref(fs), C.byref(cfg),
                                                 C.byref(h)))
        self.h = h

    def _check(self, rc: int):
        if rc != GG_OK:
            raise GreenGNNError(rc, (self.lib.gg_last_error() or b"").decode())

    def close(self):
        if getattr(self, "h", None):
            self.lib.gg_graph_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- gg_window_stage ---------------------------------------------------------------------
    def window_stage(self, window_id: int, first_batch_index: int, batches: Sequence[np.ndarray],
                     fanouts: Sequence[int]):
        seeds = np.ascontiguousarray(np.concatenate([np.asarray(b, dtype=np.int32) for b in batches])
                                     if len(batches) else np.zeros(0, np.int32), dtype=np.int32)
        off = np.zeros(len(batches) + 1, dtype=np.int64)
        off[1:] = np.cumsum([len(b) for b in batches])
        fo = np.ascontiguousarray(fanouts, dtype=np.int32)
        self._check(self.lib.gg_window_stage(self.h, window_id, first_batch_index, seeds.ctypes.data,
                                             off.ctypes.data, len(batches), fo.ctypes.data, len(fo)))

    # -- gg_simulate (NEXT-1) ----------------------------------------------------------------
    def simulate(self, batches: Sequence[np.ndarray], fanouts: Sequence[int], candidates: Sequence[int],
                 model: Dict, first_batch_index: int = 0, export: bool = False) -> Dict:
        """Trace simulator + Eqs. (1)-(3) for every candidate W.  `model`: dict with per-owner
        lists eps_init, eps_pay_a, eps_pay_b, lam_init, lam_pay_a, lam_pay_b and scalars bw, p_idle.
        Returns {"best": W*, "results": [dict per candidate]} (+ "delta"/"miss" arrays if export)."""
        seeds = np.ascontiguousarray(np.concatenate([np.asarray(b, dtype=np.int32) for b in batches]), dtype=np.int32)
        off = np.zeros(len(batches) + 1, dtype=np.int64)
        off[1:] = np.cumsum([len(b) for b in batches])
        fo = np.ascontiguousarray(fanouts, dtype=np.int32)
        ws = np.ascontiguousarray(candidates, dtype=np.int32)
        em = gg_energy_model()
        for name in ("eps_init", "eps_pay_a", "eps_pay_b", "lam_init", "lam_pay_a", "lam_pay_b"):
            arr = getattr(em, name)
            for m, v in enumerate(model[name]):
                arr[m] = float(v)
        em.bw_bytes_per_s, em.p_idle_w = float(model["bw"]), float(model["p_idle"])
        B, nW = len(batches), len(ws)
        res = (gg_sim_result * nW)()
        best = i32(0)
        Ks = [-(-B // int(W)) for W in ws]
        d_out = np.zeros(sum(Ks) * self.P, dtype=np.int64) if export else None
        m_out = np.zeros(nW * B * self.P, dtype=np.int64) if export else None
        self._check(self.lib.gg_simulate(self.h, seeds.ctypes.data, off.ctypes.data, B, first_batch_index,
                                         fo.ctypes.data, len(fo), ws.ctypes.data, nW, C.byref(em), res,
                                         C.byref(best), d_out.ctypes.data if export else None,
                                         m_out.ctypes.data if export else None))
        out = {"best": int(ws[best.value]),
               "results": [{n: getattr(r, n) for n, _ in gg_sim_result._fields_} for r in res]}
        if export:
            out["delta"], c = [], 0
            for K in Ks:
                out["delta"].append(d_out[c:c + K * self.P].reshape(K, self.P))
                c += K * self.P
            out["miss"] = m_out.reshape(nW, B, self.P)
        return out

    # -- gg_batch_info / gg_batch_gather -----------------------------------------------------
    def _unpack(self, o: gg_batch_out) -> Dict:
        dev = self.device
        blocks = []
        for h in range(o.num_layers):
            k = o.blocks[h]
            blocks.append(dict(n_dst=k.n_dst, n_src=k.n_src, n_edge=k.n_edge,
                               indptr=_view_i32(k.indptr, k.n_dst + 1, dev),
                               src_local=_view_i32(k.src_local, k.n_edge, dev),
                               src_global=_view_i32(k.src_global, k.n_edge, dev)))
        return dict(blocks=blocks, n_input=o.n_input, input_nodes=_view_i32(o.input_nodes, o.n_input, dev),
                    _miss=(o.miss_pos, o.miss_id, o.n_miss))

    def batch_info(self, window_id: int, b: int) -> Dict:
        o = gg_batch_out()
        self._check(self.lib.gg_batch_info(self.h, window_id, b, C.byref(o)))
        return self._unpack(o)

    def batch_gather(self, window_id: int, b: int, features: torch.Tensor,
                     stream: Optional[torch.cuda.Stream] = None) -> Dict:
        """features: caller-owned device buffer [capacity_rows, dim]; X_b = features[:n_input]."""
        assert features.is_cuda and features.is_contiguous() and features.shape[1] == self.dim
        assert features.dtype == self.feat_dtype
        o = gg_batch_out()
        o.features = features.data_ptr()
        o.features_capacity_rows = features.shape[0]
        st = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._check(self.lib.gg_batch_gather(self.h, window_id, b, C.byref(o), st.cuda_stream))
        r = self._unpack(o)
        r["features"] = features[:o.n_input]
        r["_out"] = o                      # the filled gg_batch_out (what gg_sage_step consumes)
        return r

    def misses(self, r: Dict):
        """(miss_pos, miss_id) of the LAST gather as host arrays (synchronises)."""
        torch.cuda.synchronize(self.device)
        mp, mi, nm = r["_miss"]
        n = int(_view_i32(nm, 1, self.device).cpu()[0])
        return (_view_i32(mp, n, self.device).cpu().numpy(), _view_i32(mi, n, self.device).cpu().numpy())

    def window_release(self, window_id: int, stream: Optional[torch.cuda.Stream] = None):
        """stream: where the caller's last use of the window's device pointers was enqueued
        (default: torch's current stream); the arena is recycled only behind that point."""
        st = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._check(self.lib.gg_window_release(self.h, window_id, st.cuda_stream))

    # -- gg_trace / exports --------------------------------------------------------------------
    def trace(self, window_id: int, W: int) -> Dict:
        t = gg_window_trace()
        n_input = np.zeros(W, np.int32)
        hl = np.zeros(W, np.int32)
        hc = np.zeros(W, np.int32)
        miss = np.zeros((W, self.P), np.int32)
        t.n_input, t.hit_local, t.hit_cache, t.miss = (a.ctypes.data for a in (n_input, hl, hc, miss))
        self._check(self.lib.gg_trace(self.h, window_id, C.byref(t)))
        P = self.P
        d = {k: getattr(t, k) for k in ("W", "num_parts", "n_access", "n_unique", "n_unique_remote", "n_hot",
                                        "carried_rows", "bulk_copies", "ms_sample", "ms_unique", "ms_select",
                                        "ms_pack_host", "ms_h2d", "ms_carry", "ms_stage_total",
                                        "ms_boundary_wait")}
        d.update(staged_rows=list(t.staged_rows)[:P], bulk_rows=list(t.bulk_rows)[:P],
                 bulk_bytes=list(t.bulk_bytes)[:P], n_input=n_input, hit_local=hl, hit_cache=hc, miss=miss)
        return d

    def window_export(self, window_id: int, what: str) -> np.ndarray:
        code = {"uniq": 0, "cnt": 1, "hot": 2, "req": 3, "carried": 4}[what]
        n = i64(0)
        rc = self.lib.gg_window_export(self.h, window_id, code, None, 0, C.byref(n))
        if rc not in (GG_OK, GG_ERR_CAPACITY):
            self._check(rc)
        out = np.empty(max(n.value, 1), dtype=np.int32)
        self._check(self.lib.gg_window_export(self.h, window_id, code, out.ctypes.data, len(out), C.byref(n)))
        return out[:n.value].copy()

    def cache_read(self, window_id: int, ids: np.ndarray) -> np.ndarray:
        ids = np.ascontiguousarray(ids, dtype=np.int32)
        out = np.empty((len(ids), self.rb), dtype=np.uint8)
        self._check(self.lib.gg_cache_read(self.h, window_id, ids.ctypes.data, len(ids), out.ctypes.data))
        return out

    def profile_enable(self, on: bool = True):
        self._check(self.lib.gg_profile_enable(self.h, 1 if on else 0))

    def profile_get(self) -> Dict:
        p = gg_profile()
        self._check(self.lib.gg_profile_get(self.h, C.byref(p)))
        return {k: dict(ms=p.ms[i], regions=p.regions[i], bytes=p.bytes[i]) for i, k in enumerate(PROF_KINDS)}

    def cache_reset(self):
        self._check(self.lib.gg_cache_reset(self.h))

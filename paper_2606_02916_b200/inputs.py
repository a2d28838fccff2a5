"""Seeded synthetic inputs: graphs, owner ranges, feature stores, seed batches.

This module is INPUT ONLY.  It is the one module both the CPU oracle's tests and
the CUDA path's tests/bench may import, and it holds none of the method's
arithmetic (no sampling keys, no window/hot-set/gather logic).  Its own random
numbers come from a murmur-style 64-bit finaliser over counters -- deliberately
NOT the SplitMix64 chain the method's sampling key uses (DESIGN.md "Readings",
S1) -- evaluated with integer torch ops so the same call gives the same arrays on
CPU and on CUDA.

The graphs stand in for the paper's datasets (Sec. VI-A: Reddit,
OGBN-Products, OGBN-Papers100M), taking their node/edge counts, feature widths
and training fractions from BASELINE.json:configs; nothing of those datasets is
reproduced here.  Recipe: DESIGN.md "Input recipe".
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, List, Optional

import numpy as np
import torch

_M64 = (1 << 64) - 1


def _s64(x: int) -> int:
    """Python int (mod 2^64) -> the int64 value with the same bit pattern."""
    x &= _M64
    return x - (1 << 64) if x >= (1 << 63) else x


_C1 = _s64(0xFF51AFD7ED558CCD)
_C2 = _s64(0xC4CEB9FE1A85EC53)
_GOLD = _s64(0xD6E8FEB86659FD93)


def _lsr(x: torch.Tensor, s: int) -> torch.Tensor:
    return (x >> s) & ((1 << (64 - s)) - 1)


def mix64(x: torch.Tensor) -> torch.Tensor:
    """murmur3-style 64-bit finaliser on an int64 tensor (wrapping arithmetic)."""
    x = x ^ _lsr(x, 33)
    x = x * _C1
    x = x ^ _lsr(x, 33)
    x = x * _C2
    x = x ^ _lsr(x, 33)
    return x


def _mix64_int(x: int) -> int:
    x &= _M64
    x ^= x >> 33
    x = (x * 0xFF51AFD7ED558CCD) & _M64
    x ^= x >> 33
    x = (x * 0xC4CEB9FE1A85EC53) & _M64
    x ^= x >> 33
    return x


def substream(master: int, tag: int) -> int:
    """Key of sub-stream `tag` of master seed `master` (host integer)."""
    return _mix64_int(_mix64_int(master) ^ ((tag * 0x9FB21C651E98DF25) & _M64))


def rand_u63(key: int, start: int, count: int, device) -> torch.Tensor:
    """count non-negative int64 values: element i = mix64(key + (start+i)*GOLD) >> 1."""
    ctr = torch.arange(start, start + count, dtype=torch.int64, device=device)
    return _lsr(mix64(ctr * _GOLD + _s64(key)), 1)


def seeded_permutation(n: int, key: int, device) -> torch.Tensor:
    """Permutation of [0,n): argsort (stable) of per-index hashes."""
    h = rand_u63(key, 0, n, device)
    return torch.sort(h, stable=True).indices


# --------------------------------------------------------------------------
# graphs
# --------------------------------------------------------------------------

def _chung_lu_weights(n: int, total: float, gamma: float, d_max: float) -> np.ndarray:
    """w_i = c (i+i0)^(-1/(gamma-1)), sum = total, w_0 = d_max (bisection on i0)."""
    alpha = 1.0 / (gamma - 1.0)
    i = np.arange(n, dtype=np.float64)

    def w0(i0: float) -> float:
        s = np.power(i + i0, -alpha).sum()
        return total / s * i0 ** (-alpha)

    lo, hi = 1e-6, float(n)
    if w0(lo) < d_max:          # cannot reach d_max: take the sharpest head
        i0 = lo
    else:
        for _ in range(80):
            mid = math.sqrt(lo * hi)
            if w0(mid) > d_max:
                lo = mid
            else:
                hi = mid
        i0 = hi
    w = np.power(i + i0, -alpha)
    return w * (total / w.sum())


def _int_cdf(w: np.ndarray, device) -> torch.Tensor:
    wi = np.floor(w * float(1 << 20)).astype(np.int64) + 1
    return torch.from_numpy(np.cumsum(wi)).to(device)


def _draw(cdf: torch.Tensor, key: int, start: int, count: int) -> torch.Tensor:
    r = rand_u63(key, start, count, cdf.device) % int(cdf[-1].item())
    return torch.searchsorted(cdf, r, right=True)


def _pairs_to_csr(u: torch.Tensor, v: torch.Tensor, n: int, symmetric: bool):
    """Edge list (v aggregates from u) -> CSR rows sorted, deduplicated."""
    if symmetric:
        keep = u != v
        u, v = u[keep], v[keep]
        a, b = torch.minimum(u, v), torch.maximum(u, v)
        k = torch.unique(a * n + b)
        a, b = k // n, k % n
        key = torch.cat([a * n + b, b * n + a])
        key = torch.sort(key).values
    else:
        key = torch.unique(v * n + u)          # row = destination v, entry = source u
    dst = key // n
    indices = (key % n).to(torch.int32)
    deg = torch.bincount(dst, minlength=n)
    indptr = torch.zeros(n + 1, dtype=torch.int64, device=key.device)
    indptr[1:] = torch.cumsum(deg, 0)
    return indptr, indices


def chung_lu_graph(n: int, n_pairs: int, gamma: float, d_max: float, seed: int,
                   device="cpu", n_communities: int = 0, cross_frac: float = 0.0):
    """Undirected Chung-Lu graph, optionally with planted communities.

    Returns (indptr int64[n+1], indices int32[nnz], part_sizes or None).  Without
    communities node IDs are a seeded random relabelling of the weight ranks (degree
    uncorrelated with ID).  With communities, weight rank i belongs to community
    i % C, a pair stays inside its first endpoint's community with probability
    1 - cross_frac*C/(C-1), and each community is relabelled to one contiguous ID
    block (randomly permuted inside the block) whose sizes are returned.
    """
    w = _chung_lu_weights(n, 2.0 * n_pairs, gamma, d_max)
    cdf = _int_cdf(w, device)
    C = n_communities
    if C > 1:
        cdfs = [_int_cdf(w[c::C], device) for c in range(C)]
        p_glob = cross_frac * C / (C - 1)
    k_u, k_v, k_x, k_perm = (substream(seed, t) for t in (1, 2, 3, 4))

    have = None
    drawn = 0
    want = n_pairs
    for _round in range(4):
        m = int(want * 1.02) + 16
        u = _draw(cdf, k_u, drawn, m)
        if C > 1:
            v_glob = _draw(cdf, k_v, drawn, m)
            coin = rand_u63(k_x, drawn, m, device).to(torch.float64) / float(1 << 63)
            comm = u % C
            v = v_glob.clone()
            r = rand_u63(k_v, drawn + (1 << 40), m, device)
            for c in range(C):
                sel = (comm == c) & (coin >= p_glob)
                idx = torch.searchsorted(cdfs[c], r[sel] % int(cdfs[c][-1].item()), right=True)
                v[sel] = idx * C + c
        else:
            v = _draw(cdf, k_v, drawn, m)
        drawn += m
        keep = u != v
        a, b = torch.minimum(u[keep], v[keep]), torch.maximum(u[keep], v[keep])
        k = a * n + b
        have = torch.unique(k if have is None else torch.cat([have, k]))
        short = n_pairs - have.numel()
        if short <= n_pairs // 200:
            break
        want = int(short * 1.1)
    if have.numel() > n_pairs:       # trim the overdraw by hash order, not by key order
        hk = mix64(have ^ _s64(substream(seed, 5)))
        have = have[torch.sort(hk, stable=True).indices[:n_pairs]]
    a, b = have // n, have % n

    # relabel
    part_sizes = None
    if C > 1:
        new_id = torch.empty(n, dtype=torch.int64, device=device)
        base = 0
        part_sizes = []
        for c in range(C):
            members = torch.arange(c, n, C, dtype=torch.int64, device=device)
            p = seeded_permutation(members.numel(), substream(k_perm, c), device)
            new_id[members] = base + p
            base += members.numel()
            part_sizes.append(int(members.numel()))
    else:
        new_id = seeded_permutation(n, k_perm, device)
    a, b = new_id[a], new_id[b]
    indptr, indices = _pairs_to_csr(a, b, n, symmetric=True)
    return indptr, indices, part_sizes


def rmat_graph(scale: int, n: int, n_edges: int, seed: int, device="cpu",
               abcd=(0.57, 0.19, 0.19, 0.05), chunk: int = 1 << 26):
    """Directed R-MAT: seeded vertex scramble, endpoints >= n rejected, duplicates removed.

    Row v of the CSR lists the nodes v aggregates from (an R-MAT edge u->v is entry
    u in row v); zero-degree rows are legal.
    """
    a, b, c, _d = abcd
    ta, tb, tc = (int(x * (1 << 30)) for x in (a, a + b, a + b + c))
    k_e, k_s = substream(seed, 11), substream(seed, 12)
    keys: List[torch.Tensor] = []
    total, drawn = 0, 0
    mask = (1 << scale) - 1
    mul = _s64(0x9E3779B97F4A7C15 | 1)
    add = _s64(k_s)
    while total < n_edges:
        m = min(chunk, int((n_edges - total) * 1.5) + 1024)
        src = torch.zeros(m, dtype=torch.int64, device=device)
        dst = torch.zeros(m, dtype=torch.int64, device=device)
        for lvl in range(scale):
            r = rand_u63(k_e, (drawn + lvl * (1 << 44)), m, device) & ((1 << 30) - 1)
            q_b = (r >= ta) & (r < tb)
            q_c = (r >= tb) & (r < tc)
            q_d = r >= tc
            src = (src << 1) | (q_c | q_d).to(torch.int64)
            dst = (dst << 1) | (q_b | q_d).to(torch.int64)
        drawn += m
        # scramble: odd-multiplier affine map on [0, 2^scale) is a bijection
        src = (src * mul + add) & mask
        dst = (dst * mul + add) & mask
        ok = (src < n) & (dst < n)
        k = torch.unique(dst[ok] * n + src[ok])
        keys.append(k)
        total += k.numel()
        if len(keys) > 1:
            merged = torch.unique(torch.cat(keys))
            keys = [merged]
            total = merged.numel()
    key = keys[0][:n_edges] if keys[0].numel() > n_edges else keys[0]
    dstv = key // n
    indices = (key % n).to(torch.int32)
    deg = torch.bincount(dstv, minlength=n)
    indptr = torch.zeros(n + 1, dtype=torch.int64, device=device)
    indptr[1:] = torch.cumsum(deg, 0)
    return indptr, indices


# --------------------------------------------------------------------------
# features, seeds
# --------------------------------------------------------------------------

def feature_rows(first_row: int, n_rows: int, dim: int, dtype: torch.dtype, seed: int,
                 device="cpu", out: Optional[torch.Tensor] = None,
                 chunk_rows: int = 1 << 18) -> torch.Tensor:
    """Rows [first_row, first_row+n_rows) of the ~N(0,1) feature matrix.

    Element (u, e) = (sum of four 16-bit fields of mix64(key + (u*dim+e)*GOLD) - 2*65535)
    * (1/sqrt(4*(65536^2-1)/12)): an Irwin-Hall(4) variate, unit variance, built
    from integer ops and one float multiply so CPU and CUDA agree bit for bit.
    Stored fp32 or rounded (RNE) to bf16.  Rows are opaque bytes to the method.
    """
    key = substream(seed, 21)
    scale = 1.0 / math.sqrt(4.0 * (65536.0 ** 2 - 1.0) / 12.0)
    if out is None:
        out = torch.empty(n_rows, dim, dtype=dtype, device=device)
    for r0 in range(0, n_rows, chunk_rows):
        r1 = min(n_rows, r0 + chunk_rows)
        cnt = (r1 - r0) * dim
        ctr = torch.arange((first_row + r0) * dim, (first_row + r0) * dim + cnt,
                           dtype=torch.int64, device=device)
        h = mix64(ctr * _GOLD + _s64(key))
        s = (h & 0xFFFF) + ((h >> 16) & 0xFFFF) + ((h >> 32) & 0xFFFF) + ((h >> 48) & 0xFFFF)
        x = (s - 2 * 65535).to(torch.float32) * scale
        out[r0:r1].copy_(x.view(r1 - r0, dim).to(dtype))
    return out


def train_batches(n: int, n_train: int, batch: int, seed: int) -> List[np.ndarray]:
    """Training set = first n_train of a seeded permutation of [0,n); epoch order = a
    seeded permutation of it; consecutive batches of `batch` (last one partial)."""
    perm = seeded_permutation(n, substream(seed, 31), "cpu")[:n_train]
    order = seeded_permutation(n_train, substream(seed, 32), "cpu")
    ids = perm[order].to(torch.int32).numpy()
    return [ids[i:i + batch].copy() for i in range(0, n_train, batch)]


# --------------------------------------------------------------------------
# configurations (BASELINE.json:configs) and the assembled workload
# --------------------------------------------------------------------------

CONFIGS: Dict[str, dict] = {
    # 0 Tiny: first 4 batches only = one window
    "tiny": dict(index=0, kind="chung_lu", n=10_000, n_pairs=50_000, gamma=2.1, d_max=500,
                 parts=4, dim=32, dtype="f32", n_train=1_000, batch=64, fanouts=[10, 5],
                 max_batches=4, windows=[4]),
    "small": dict(index=1, kind="chung_lu", n=100_000, n_pairs=1_000_000, gamma=2.1, d_max=2_000,
                  parts=4, dim=128, dtype="f32", n_train=10_000, batch=1024, fanouts=[15, 10],
                  max_batches=None, windows=[1, 4, 8]),
    "products": dict(index=2, kind="planted", n=2_449_029, n_pairs=61_900_000, gamma=2.1,
                     d_max=17_500, parts=4, cross_frac=0.08, dim=100, dtype="f32",
                     n_train=196_615, batch=1024, fanouts=[15, 10, 5], max_batches=None,
                     windows=[1, 2, 4, 8, 16, 32]),
    "dense": dict(index=3, kind="chung_lu", n=232_965, n_pairs=57_300_000, gamma=2.1,
                  d_max=20_000, parts=4, dim=602, dtype="f32", n_train=153_757, batch=1024,
                  fanouts=[25, 10], max_batches=None, windows=[1, 4, 16]),
    "large": dict(index=4, kind="rmat", n=111_000_000, n_edges=1_600_000_000, scale=27,
                  parts=4, dim=128, dtype="bf16", n_train=1_221_000, batch=1024,
                  fanouts=[15, 10, 5], max_batches=None, windows=[4, 16]),
    # scaled-down shapes of configs 2/3 for CPU-side tests (same generator paths)
    "products_mini": dict(index=12, kind="planted", n=60_001, n_pairs=600_000, gamma=2.1,
                          d_max=3_000, parts=4, cross_frac=0.08, dim=100, dtype="f32",
                          n_train=6_000, batch=512, fanouts=[15, 10, 5], max_batches=None,
                          windows=[1, 4]),
    "dense_mini": dict(index=13, kind="chung_lu", n=8_001, n_pairs=400_000, gamma=2.1,
                       d_max=3_000, parts=4, dim=602, dtype="f32", n_train=2_000, batch=256,
                       fanouts=[25, 10], max_batches=None, windows=[1, 4]),
    "large_mini": dict(index=14, kind="rmat", n=150_000, n_edges=2_000_000, scale=18,
                       parts=4, dim=128, dtype="bf16", n_train=4_000, batch=512,
                       fanouts=[15, 10, 5], max_batches=None, windows=[4]),
}

_DTYPES = {"f32": torch.float32, "bf16": torch.bfloat16}


@dataclasses.dataclass
class Workload:
    name: str
    cfg: dict
    num_nodes: int
    indptr: torch.Tensor            # int64 [N+1], on `device`
    indices: torch.Tensor           # int32 [nnz], on `device`
    part_offsets: np.ndarray        # int64 [P+1]
    local_part: int
    feat_parts: List[torch.Tensor]  # [P]; local on `device`, others pinned host (or plain host)
    dim: int
    dtype: torch.dtype
    batches: List[np.ndarray]       # int32 seed IDs per mini-batch, epoch order
    fanouts: List[int]
    seed: int                       # the method's sampling seed (gg_config.seed)

    @property
    def row_bytes(self) -> int:
        return self.dim * self.feat_parts[0].element_size()

    def host_graph(self):
        return (self.indptr.cpu().numpy(), self.indices.cpu().numpy())

    def host_features(self) -> np.ndarray:
        """Full [N, row_bytes] uint8 matrix on the host (tests / oracle input)."""
        rows = [p.cpu().contiguous().view(torch.uint8).view(p.shape[0], -1).numpy()
                for p in self.feat_parts]
        return np.concatenate(rows, axis=0)


def master_seed(cfg: dict) -> int:
    return 0x5EED0000 + int(cfg["index"])


def make_workload(name: str, device="cpu", pin: Optional[bool] = None,
                  batch: Optional[int] = None, local_part: int = 0) -> Workload:
    cfg = dict(CONFIGS[name])
    if batch is not None:
        cfg["batch"] = batch
    ms = master_seed(cfg)
    n, P = cfg["n"], cfg["parts"]
    part_sizes = None
    if cfg["kind"] == "chung_lu":
        indptr, indices, _ = chung_lu_graph(n, cfg["n_pairs"], cfg["gamma"], cfg["d_max"],
                                            substream(ms, 100), device)
    elif cfg["kind"] == "planted":
        indptr, indices, part_sizes = chung_lu_graph(
            n, cfg["n_pairs"], cfg["gamma"], cfg["d_max"], substream(ms, 100), device,
            n_communities=P, cross_frac=cfg["cross_frac"])
    elif cfg["kind"] == "rmat":
        indptr, indices = rmat_graph(cfg["scale"], n, cfg["n_edges"], substream(ms, 100), device)
    else:
        raise ValueError(cfg["kind"])
    if part_sizes is None:
        base = n // P
        part_sizes = [base + (1 if i < n % P else 0) for i in range(P)]
    part_offsets = np.zeros(P + 1, dtype=np.int64)
    part_offsets[1:] = np.cumsum(part_sizes)

    dtype = _DTYPES[cfg["dtype"]]
    if pin is None:
        pin = torch.device(device).type == "cuda"
    fseed = substream(ms, 200)
    parts: List[torch.Tensor] = []
    for m in range(P):
        lo, hi = int(part_offsets[m]), int(part_offsets[m + 1])
        if m == local_part:
            parts.append(feature_rows(lo, hi - lo, cfg["dim"], dtype, fseed, device))
        else:
            host = torch.empty(hi - lo, cfg["dim"], dtype=dtype, pin_memory=bool(pin))
            if torch.device(device).type == "cuda":
                step = 1 << 20
                for r0 in range(0, hi - lo, step):
                    r1 = min(hi - lo, r0 + step)
                    host[r0:r1].copy_(feature_rows(lo + r0, r1 - r0, cfg["dim"], dtype, fseed, device))
            else:
                feature_rows(lo, hi - lo, cfg["dim"], dtype, fseed, "cpu", out=host)
            parts.append(host)
    if torch.device(device).type == "cuda":
        torch.cuda.empty_cache()    # the generator's sort temporaries (tens of GB for "large")
    batches = train_batches(n, cfg["n_train"], cfg["batch"], substream(ms, 300))
    if cfg["max_batches"]:
        batches = batches[:cfg["max_batches"]]
    return Workload(name=name, cfg=cfg, num_nodes=n, indptr=indptr, indices=indices,
                    part_offsets=part_offsets, local_part=local_part, feat_parts=parts, dim=cfg["dim"],
                    dtype=dtype, batches=batches, fanouts=list(cfg["fanouts"]),
                    seed=substream(ms, 400))


# --------------------------------------------------------------------------
# BFS-grown balanced split (BASELINE.json:configs[2] names it; reading S22)
# --------------------------------------------------------------------------

def bfs_grown_split(indptr: torch.Tensor, indices: torch.Tensor, parts: int, seed: int,
                    cap_factor: float = 1.02) -> torch.Tensor:
    """Multi-source BFS growth of `parts` balanced regions: one seeded start node per part, all
    parts grow level by level, a node reached by several parts in one level goes to the lowest
    part number, a part stops growing at ceil(N / parts) * cap_factor nodes, whatever is left
    unreached goes to the parts with room in ID order.  Returns int8 labels [N] on the graph's
    device.  Input-side only (owner assignment of a synthetic graph): none of the method's
    arithmetic lives here."""
    dev = indptr.device
    n = indptr.numel() - 1
    cap = int(-(-n // parts) * cap_factor)
    label = torch.full((n,), -1, dtype=torch.int8, device=dev)
    size = [0] * parts
    starts = []
    k = 0
    while len(starts) < parts:                     # distinct seeded start nodes
        s = _mix64_int(seed + 0x9E37 * k) % n
        k += 1
        if s not in starts:
            starts.append(s)
    frontier = torch.tensor(starts, dtype=torch.int64, device=dev)
    label[frontier] = torch.arange(parts, dtype=torch.int8, device=dev)
    for p in range(parts):
        size[p] = 1
    big = torch.iinfo(torch.int8).max
    while frontier.numel() > 0:
        row0 = indptr[frontier]
        deg = indptr[frontier + 1] - row0
        total = int(deg.sum())
        if total == 0:
            break
        first = torch.cumsum(deg, 0) - deg
        offs = torch.arange(total, device=dev) - torch.repeat_interleave(first, deg) + torch.repeat_interleave(row0, deg)
        nbr = indices[offs].long()
        src = torch.repeat_interleave(label[frontier], deg)
        free = label[nbr] < 0
        nbr, src = nbr[free], src[free]
        if nbr.numel() == 0:
            break
        cand = torch.full((n,), big, dtype=torch.int8, device=dev)
        cand.scatter_reduce_(0, nbr, src, reduce="amin")
        new = torch.nonzero(cand < big).squeeze(1)
        admitted = []
        for p in range(parts):
            room = cap - size[p]
            if room <= 0:
                continue
            idx = new[cand[new] == p][:room]
            if idx.numel():
                label[idx] = p
                size[p] += int(idx.numel())
                admitted.append(idx)
        frontier = torch.cat(admitted) if admitted else torch.empty(0, dtype=torch.int64, device=dev)
    rest = torch.nonzero(label < 0).squeeze(1)
    pos = 0
    for p in sorted(range(parts), key=lambda q: size[q]):
        if pos >= rest.numel():
            break
        room = max(0, -(-n // parts) - size[p]) if p != sorted(range(parts), key=lambda q: size[q])[-1] else rest.numel() - pos
        take = rest[pos:pos + room]
        label[take] = p
        size[p] += int(take.numel())
        pos += int(take.numel())
    if pos < rest.numel():
        label[rest[pos:]] = parts - 1
    return label


def edge_cut_of_labels(indptr: torch.Tensor, indices: torch.Tensor, label: torch.Tensor) -> float:
    """Fraction of CSR entries whose two endpoints carry different labels."""
    n = indptr.numel() - 1
    cut, step = 0, 1 << 22
    for r0 in range(0, n, step):
        r1 = min(n, r0 + step)
        ip = indptr[r0:r1 + 1]
        e0, e1 = int(ip[0]), int(ip[-1])
        if e1 == e0:
            continue
        own_e = torch.repeat_interleave(label[r0:r1], ip[1:] - ip[:-1])
        cut += int((own_e != label[indices[e0:e1].long()]).sum())
    return cut / max(1, indices.numel())

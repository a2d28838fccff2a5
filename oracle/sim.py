"""CPU oracle of the paper's trace simulator + analytical energy model.  TEST INFRASTRUCTURE,
NOT THE PRODUCT (only tests/, __graft_entry__.smoke() and bench.py's cpu legs may import it;
it imports nothing from the CUDA package and nothing from oracle/ggo.cpp: it is a second,
independent restatement of the window / hot-set / delta / miss definitions in plain numpy).

Follows PAPER.md step by step:
  * Sec. IV-A "Simulation and window selection": for each candidate W the
    epoch is cut into ceil(B/W) windows; H_k = the n_hot most frequently accessed remote nodes
    of window k; rebuild delta  Delta_{k,m} = (H_k ∩ N_m) \\ (C_{k-1} ∩ N_m);  residual misses
    M_{b,m} = (N_b ∩ N_m) \\ (H_k ∩ N_m).
  * Sec. V-B: "a single pass over the trace", cache state kept across
    windows, rebuild events at window boundaries, miss events per batch, stall time from the
    latency surrogates.
  * Eq. (1) E_rebuild, Eq. (2) E_miss, Eq. (3) E_stall = P_idle * T_stall, E_phy = their sum
    (PAPER.md:147-160); W* = argmin over the candidates (with L(W) = 0: the learned
    correction of Eq. 4-5 needs measured ground truth and is not part of this oracle).

Readings: S8 access count = number of batches of the window containing u;
S10 hot-set ties (count desc, id asc); S11 C_k = H_k; S13 an empty delta / miss set issues no
transfer; S20 event time = max(slowest single-owner transfer, total bytes / BW);
S24 eps_payload(m, x) = a_m + b_m * x for x > 0 and 0 for x = 0 ("a linear fit ... as a function
of transfer size"), latency surrogate likewise; S25 hit ratio = remote accesses
served from the cache / remote accesses.

All floating point is IEEE double, one operation at a time, events in trace order (windows
ascending, then batches ascending; owners ascending inside an event), so that a device
implementation that uses the same order and no fused multiply-add reproduces it bit for bit.
"""
from __future__ import annotations

import dataclasses
from typing import Dict, List, Sequence

import numpy as np


@dataclasses.dataclass
class EnergyModel:
    """Per-owner coefficients of PAPER.md:128 (profiler output) -- plain numbers here."""
    eps_init: Sequence[float]      # J per transfer, owner m
    eps_pay_a: Sequence[float]     # J, intercept of the linear payload fit
    eps_pay_b: Sequence[float]     # J per row
    lam_init: Sequence[float]      # s per transfer
    lam_pay_a: Sequence[float]     # s
    lam_pay_b: Sequence[float]     # s per row
    bw: float                      # aggregate bandwidth ceiling, bytes / s
    p_idle: float                  # W
    row_bytes: int


def owner_of(ids: np.ndarray, part_offsets: np.ndarray) -> np.ndarray:
    return np.searchsorted(np.asarray(part_offsets, dtype=np.int64), ids, side="right") - 1


def hot_set(uniq: np.ndarray, cnt: np.ndarray, owners: np.ndarray, local: int, n_hot: int) -> np.ndarray:
    """H_k: the n_hot most frequently accessed remote nodes, ascending by id."""
    rem = owners != local
    r_ids, r_cnt = uniq[rem], cnt[rem]
    if n_hot < 0 or len(r_ids) <= n_hot:
        return r_ids
    order = np.lexsort((r_ids, -r_cnt))[:n_hot]        # (count desc, id asc)
    return np.sort(r_ids[order])


def event_time(x: Sequence[int], m: EnergyModel) -> float:
    """Duration of one rebuild / miss event with x[o] rows from owner o (Eq. 3 prose, S20)."""
    slow = 0.0
    rows = 0
    for o, n in enumerate(x):
        if n > 0:
            t = m.lam_init[o] + (m.lam_pay_a[o] + m.lam_pay_b[o] * float(n))
            if t > slow:
                slow = t
            rows += int(n)
    if rows == 0:
        return 0.0
    ceil_t = float(rows * m.row_bytes) / m.bw
    return slow if slow > ceil_t else ceil_t


def event_energy(x: Sequence[int], m: EnergyModel) -> float:
    """One event's term of Eq. (1) / Eq. (2): sum over owners of eps_init*I[x>0] + eps_payload."""
    e = 0.0
    for o, n in enumerate(x):
        if n > 0:
            e = e + (m.eps_init[o] + (m.eps_pay_a[o] + m.eps_pay_b[o] * float(n)))
    return e


def simulate(trace: List[np.ndarray], part_offsets: np.ndarray, local: int, n_hot: int, W: int,
             model: EnergyModel, carry_over: int = 1) -> Dict:
    """One pass over the trace T = [N_b for b in epoch order] for window size W."""
    po = np.asarray(part_offsets, dtype=np.int64)
    P = len(po) - 1
    B = len(trace)
    K = -(-B // W)
    delta = np.zeros((K, P), dtype=np.int64)
    staged = np.zeros((K, P), dtype=np.int64)
    miss = np.zeros((B, P), dtype=np.int64)
    hit_local = np.zeros(B, dtype=np.int64)
    hit_cache = np.zeros(B, dtype=np.int64)
    cache = np.zeros(0, dtype=np.int64)                # C_0 = empty (Alg. 1 l.1)
    e_rebuild = e_miss = t_stall = 0.0
    rebuild_events = miss_events = 0
    for k in range(K):
        batches = [np.asarray(t, dtype=np.int64) for t in trace[k * W:(k + 1) * W]]
        uniq, cnt = np.unique(np.concatenate(batches), return_counts=True)
        H = hot_set(uniq, cnt, owner_of(uniq, po), local, n_hot)
        new = H if not carry_over else np.setdiff1d(H, cache, assume_unique=True)
        ho = owner_of(H, po)
        no = owner_of(new, po)
        for m in range(P):
            staged[k, m] = int(np.count_nonzero(ho == m))
            delta[k, m] = int(np.count_nonzero(no == m))
        cache = H                                       # C_k = H_k (S11)
        # rebuild event of this window boundary (Eq. 1)
        e_rebuild = e_rebuild + event_energy(delta[k], model)
        t_stall = t_stall + event_time(delta[k], model)
        rebuild_events += int(np.count_nonzero(delta[k]))
        # miss events of the window's batches (Eq. 2)
        for j, nb in enumerate(batches):
            b = k * W + j
            ob = owner_of(nb, po)
            remote = ob != local
            in_hot = np.isin(nb, H, assume_unique=True)
            hit_local[b] = int(np.count_nonzero(~remote))
            hit_cache[b] = int(np.count_nonzero(remote & in_hot))
            mm = remote & ~in_hot
            for m in range(P):
                miss[b, m] = int(np.count_nonzero(mm & (ob == m)))
            e_miss = e_miss + event_energy(miss[b], model)
            t_stall = t_stall + event_time(miss[b], model)
            miss_events += int(np.count_nonzero(miss[b]))
    e_stall = model.p_idle * t_stall
    remote_acc = int(hit_cache.sum() + miss.sum())
    return dict(W=W, n_windows=K, delta=delta, staged=staged, miss=miss, hit_local=hit_local,
                hit_cache=hit_cache, rebuild_events=rebuild_events, miss_events=miss_events,
                rebuild_rows=int(delta.sum()), miss_rows=int(miss.sum()),
                n_access=int(sum(len(t) for t in trace)), n_remote_access=remote_acc,
                hit_ratio=(float(hit_cache.sum()) / float(remote_acc)) if remote_acc else 1.0,
                e_rebuild=e_rebuild, e_miss=e_miss, t_stall=t_stall, e_stall=e_stall,
                e_phy=(e_rebuild + e_miss) + e_stall)


def select_window(trace, part_offsets, local, n_hot, candidates: Sequence[int], model: EnergyModel,
                  carry_over: int = 1):
    """W* = argmin_W E_phy(W) (PAPER.md:186 with L = 0); ties -> the smaller W.  Returns
    (W*, [result per candidate])."""
    res = [simulate(trace, part_offsets, local, n_hot, W, model, carry_over) for W in candidates]
    best = 0
    for i in range(1, len(res)):
        if res[i]["e_phy"] < res[best]["e_phy"]:
            best = i
    return candidates[best], res


# ---- NEXT-3: rank calibration (Eq. 5) ------------------------------------------
def rank_loss(beta: np.ndarray, gamma: np.ndarray, Z: np.ndarray, e_gt: np.ndarray, lam: float) -> float:
    """Eq. (5): sum_{i<j} log(1 + exp(-sigma_ij (S_j - S_i))) + lam * ||beta||^2 with
    S(W) = beta^T z(W) + gamma_W and sigma_ij = sign(E_GT(W_j) - E_GT(W_i))."""
    n = len(e_gt)
    S = [float(np.dot(beta, Z[i])) + float(gamma[i]) for i in range(n)]
    loss = 0.0
    for i in range(n):
        for j in range(i + 1, n):
            d = e_gt[j] - e_gt[i]
            sg = 1.0 if d > 0 else (-1.0 if d < 0 else 0.0)
            loss += float(np.log1p(np.exp(-sg * (S[j] - S[i]))))
    return loss + lam * float(np.dot(beta, beta))


def fit_rank_calibration(Z: np.ndarray, e_gt: np.ndarray, lam: float, lr: float, iters: int):
    """Plain gradient descent on Eq. (5) from beta = 0, gamma = 0 ("optimization is lightweight ...
    a linear model over a handful of features and seven candidates").  The paper
    does not name the optimiser: fixed-step gradient descent is this build's reading (S26).
    Every step: S_i, then for each pair i<j in order g = -sigma / (1 + exp(sigma (S_j - S_i))),
    accumulated into dS_j (+g) and dS_i (-g); d beta = sum_i dS_i z_i + 2 lam beta; d gamma = dS.
    Returns (beta, gamma, final loss)."""
    Z = np.asarray(Z, dtype=np.float64)
    e_gt = np.asarray(e_gt, dtype=np.float64)
    n, F = Z.shape
    beta = np.zeros(F)
    gamma = np.zeros(n)
    for _ in range(iters):
        S = np.zeros(n)
        for i in range(n):
            acc = 0.0
            for f in range(F):
                acc = acc + beta[f] * Z[i, f]
            S[i] = acc + gamma[i]
        dS = np.zeros(n)
        for i in range(n):
            for j in range(i + 1, n):
                d = e_gt[j] - e_gt[i]
                sg = 1.0 if d > 0 else (-1.0 if d < 0 else 0.0)
                if sg == 0.0:
                    continue
                g = -sg / (1.0 + float(np.exp(sg * (S[j] - S[i]))))
                dS[j] = dS[j] + g
                dS[i] = dS[i] - g
        for f in range(F):
            acc = 0.0
            for i in range(n):
                acc = acc + dS[i] * Z[i, f]
            beta[f] = beta[f] - lr * (acc + (2.0 * lam) * beta[f])
        for i in range(n):
            gamma[i] = gamma[i] - lr * dS[i]
    return beta, gamma, rank_loss(beta, gamma, Z, e_gt, lam)

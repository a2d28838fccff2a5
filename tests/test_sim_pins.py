"""Pins of oracle/sim.py (the paper's trace simulator + Eqs. 1-3) against what the paper and the
mathematics fix: a hand-worked example, closed forms of the degenerate budgets, invariants, and
the independent C++ oracle of the runtime path (oracle/ggo.cpp), which states the same window /
hot-set / delta / miss definitions a second time."""
import os

import numpy as np
import pytest

from oracle import ggo, sim

GOLD = os.path.join(os.path.dirname(__file__), "golden", "sim_example.txt")


def _gold():
    d = {}
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        d[t[0]] = [float(x) for x in t[1:]]
    return d


def _example_model(bw=4.0):
    return sim.EnergyModel(eps_init=[0, 2, 3], eps_pay_a=[0, 0.5, 0.25], eps_pay_b=[0, 0.125, 0.25],
                           lam_init=[0, 1, 2], lam_pay_a=[0, 0, 0], lam_pay_b=[0, 0.5, 0.25],
                           bw=bw, p_idle=10.0, row_bytes=8)


EX_TRACE = [np.array(x, np.int32) for x in ([1, 11, 12, 21], [2, 11, 13, 21, 22], [3, 11, 14, 23], [12, 14, 23, 24])]
EX_PO = np.array([0, 10, 20, 30], np.int64)


def test_hand_worked_example_eq_1_2_3():
    g = _gold()
    r = sim.simulate(EX_TRACE, EX_PO, 0, 3, 2, _example_model())
    assert r["delta"][:, 1:].reshape(-1).tolist() == g["delta"]
    assert r["delta"][:, 0].tolist() == [0, 0]
    assert r["miss"][:, 1:].reshape(-1).tolist() == g["miss"]
    assert r["hit_local"].tolist() == g["hit_local"] and r["hit_cache"].tolist() == g["hit_cache"]
    assert r["rebuild_events"] == g["rebuild_events"][0] and r["miss_events"] == g["miss_events"][0]
    for k in ("e_rebuild", "e_miss", "t_stall", "e_stall", "e_phy"):
        assert r[k] == g[k][0], k                       # all values are exact binary fractions
    assert r["hit_ratio"] == g["hit_ratio_num"][0] / g["hit_ratio_den"][0]
    r2 = sim.simulate(EX_TRACE, EX_PO, 0, 3, 2, _example_model(bw=1e9))
    assert r2["t_stall"] == g["t_stall_fast_link"][0]
    assert r2["e_rebuild"] == r["e_rebuild"] and r2["e_miss"] == r["e_miss"]


def _model(P, rb, seed=3):
    rng = np.random.default_rng(seed)
    f = lambda lo, hi: rng.uniform(lo, hi, P).tolist()
    return sim.EnergyModel(eps_init=f(1e-3, 5e-3), eps_pay_a=f(0, 1e-4), eps_pay_b=f(1e-7, 5e-7),
                           lam_init=f(1e-5, 5e-5), lam_pay_a=f(0, 1e-6), lam_pay_b=f(1e-9, 9e-9),
                           bw=5.0e10, p_idle=140.0, row_bytes=rb)


@pytest.fixture(scope="module")
def tiny_trace(workload):
    w = workload("tiny")
    og = ggo.Graph(*w.host_graph())
    bs = [ggo.Batch(og, w.batches[i], w.fanouts, w.seed, i) for i in range(len(w.batches))]
    return w, bs


def test_budget_zero_is_per_batch_fetch_of_every_remote_node(tiny_trace):
    """n_hot = 0: H_k is empty, no rebuild ever happens and M_{b,m} = N_b ∩ N_m (Eq. 2 alone)."""
    w, bs = tiny_trace
    m = _model(4, w.row_bytes)
    trace = [b.nodes for b in bs]
    for W in (1, 2, 4):
        r = sim.simulate(trace, w.part_offsets, 0, 0, W, m)
        assert r["rebuild_events"] == 0 and r["e_rebuild"] == 0.0 and r["hit_cache"].sum() == 0
        want = 0.0
        for b, nb in enumerate(trace):
            cnt = np.bincount(np.searchsorted(w.part_offsets, nb, side="right") - 1, minlength=4)
            assert r["miss"][b, 1:].tolist() == cnt[1:].tolist() and r["miss"][b, 0] == 0
            e = 0.0
            for o in range(1, 4):
                if cnt[o]:
                    e = e + (m.eps_init[o] + (m.eps_pay_a[o] + m.eps_pay_b[o] * float(cnt[o])))
            want = want + e
        assert r["e_miss"] == want
        assert r["e_phy"] == (0.0 + want) + m.p_idle * r["t_stall"]


def test_unlimited_budget_W1_without_carry_is_per_batch_bulk_fetch(tiny_trace):
    """W = 1, n_hot unlimited, full restage: Delta_{b,m} = N_b ∩ N_m, zero misses (the W = 1
    degenerate case of BASELINE.json), and with carry-over the deltas can only shrink."""
    w, bs = tiny_trace
    m = _model(4, w.row_bytes)
    trace = [b.nodes for b in bs]
    r = sim.simulate(trace, w.part_offsets, 0, -1, 1, m, carry_over=0)
    assert r["miss_rows"] == 0 and r["e_miss"] == 0.0 and r["hit_ratio"] == 1.0
    for b, nb in enumerate(trace):
        cnt = np.bincount(np.searchsorted(w.part_offsets, nb, side="right") - 1, minlength=4)
        assert r["delta"][b, 1:].tolist() == cnt[1:].tolist()
    rc = sim.simulate(trace, w.part_offsets, 0, -1, 1, m, carry_over=1)
    assert (rc["delta"] <= r["delta"]).all() and rc["rebuild_rows"] < r["rebuild_rows"]
    assert (rc["staged"] == r["staged"]).all()


@pytest.mark.parametrize("W,n_hot,carry", [(1, -1, 1), (2, 200, 1), (4, 200, 0), (3, 50, 1), (4, -1, 1)])
def test_agrees_with_the_runtime_oracle_and_invariants(tiny_trace, W, n_hot, carry):
    w, bs = tiny_trace
    trace = [b.nodes for b in bs]
    r = sim.simulate(trace, w.part_offsets, 0, n_hot, W, _model(4, w.row_bytes), carry_over=carry)
    st = ggo.State(w.num_nodes, w.part_offsets, 0, n_hot, carry)
    for k in range(r["n_windows"]):
        ow = st.run_window(bs[k * W:(k + 1) * W])
        assert r["delta"][k].tolist() == list(ow.bulk_rows)
        assert r["staged"][k].tolist() == list(ow.staged_rows)
        for j in range(ow.W):
            b = k * W + j
            assert r["miss"][b].tolist() == ow.miss[j].tolist()
            assert r["hit_local"][b] == ow.hit_local[j] and r["hit_cache"][b] == ow.hit_cache[j]
            assert r["hit_local"][b] + r["hit_cache"][b] + r["miss"][b].sum() == len(trace[b])
    assert r["rebuild_events"] == int(np.count_nonzero(r["delta"]))
    assert r["n_remote_access"] == r["hit_cache"].sum() + r["miss_rows"]
    if n_hot < 0:
        assert r["miss_rows"] == 0


def test_window_selection_is_the_argmin_and_sees_the_trade_off(tiny_trace):
    w, bs = tiny_trace
    trace = [b.nodes for b in bs]
    m = _model(4, w.row_bytes)
    cands = [1, 2, 4]
    best, res = sim.select_window(trace, w.part_offsets, 0, 200, cands, m)
    e = [r["e_phy"] for r in res]
    assert best == cands[int(np.argmin(e))]
    # a fixed budget covers less of a longer window (staleness)
    assert res[0]["hit_ratio"] >= res[2]["hit_ratio"]
    # consolidation: with full restaging every window issues one transfer per
    # remote owner, so W batches x 3 owners become 3: 12 -> 6 -> 3 transfers for 4 batches
    full = [sim.simulate(trace, w.part_offsets, 0, -1, W, m, carry_over=0)["rebuild_events"] for W in cands]
    assert full == [12, 6, 3]


# ---- NEXT-3: rank calibration, Eq. (5) ---------------------------------------------------------
def _cal_problem(n=7, F=4, seed=2):
    rng = np.random.default_rng(seed)
    Z = rng.normal(size=(n, F))
    e = rng.permutation(n).astype(np.float64) * 3.0 + 50.0        # a strict ground-truth ranking
    return Z, e


def test_rank_loss_closed_form_at_zero_and_gradient():
    Z, e = _cal_problem()
    n, F = Z.shape
    lam = 0.3
    # at beta = 0, gamma = 0 every pair contributes log 2
    assert abs(sim.rank_loss(np.zeros(F), np.zeros(n), Z, e, lam) - (n * (n - 1) / 2) * np.log(2.0)) < 1e-12
    # one gradient step of fit_rank_calibration equals -lr * (finite-difference gradient of Eq. 5)
    lr, h = 1e-3, 1e-6
    b1, g1, _ = sim.fit_rank_calibration(Z, e, lam, lr, 1)
    for f in range(F):
        d = np.zeros(F); d[f] = h
        num = (sim.rank_loss(d, np.zeros(n), Z, e, lam) - sim.rank_loss(-d, np.zeros(n), Z, e, lam)) / (2 * h)
        assert abs(b1[f] + lr * num) < 1e-9
    for i in range(n):
        d = np.zeros(n); d[i] = h
        num = (sim.rank_loss(np.zeros(F), d, Z, e, lam) - sim.rank_loss(np.zeros(F), -d, Z, e, lam)) / (2 * h)
        assert abs(g1[i] + lr * num) < 1e-9


def test_rank_calibration_recovers_the_measured_order_and_regularises():
    Z, e = _cal_problem()
    l0 = sim.rank_loss(np.zeros(Z.shape[1]), np.zeros(len(e)), Z, e, 0.1)
    beta, gamma, loss = sim.fit_rank_calibration(Z, e, 0.1, 0.05, 3000)
    assert loss < 0.2 * l0
    S = Z @ beta + gamma
    assert np.array_equal(np.argsort(S), np.argsort(e))           # Kendall tau = 1 on the calibration set
    b_big, _, _ = sim.fit_rank_calibration(Z, e, 50.0, 0.005, 3000)
    assert np.linalg.norm(b_big) < 0.1 * np.linalg.norm(beta)     # lambda ||beta||^2 shrinks beta
    # ties in the ground truth contribute no gradient
    e2 = e.copy(); e2[:] = 1.0
    b0, g0, _ = sim.fit_rank_calibration(Z, e2, 0.1, 0.05, 10)
    assert not b0.any() and not g0.any()

#!/usr/bin/env python
"""bench.py -- mini-batches/s of the whole hot path (sample + stage + gather) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--config products] [--batch 1024] [--window 16] [--n-hot -1]

A STEP is one epoch of the named workload: ceil(B/W) windows, every mini-batch sampled,
staged and gathered (all SURVEY.md Sec. 8(a) rows), cache reset before each epoch.  Prints
ONE JSON line (DESIGN.md "Measurement" explains every key).
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402
import torch  # noqa: E402

METRIC = "mini-batches/s (sample+stage+gather), one epoch per step"
UNIT = "mini-batches/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="products")
    ap.add_argument("--batch", type=int, default=1024)
    ap.add_argument("--window", type=int, default=16)
    ap.add_argument("--n-hot", type=int, default=-1)
    ap.add_argument("--staging-mode", type=int, default=0)
    ap.add_argument("--lookahead", type=int, default=6,
                    help="windows staged ahead of the one being served (sampling runs that far ahead; "
                         "the cache is always built one window ahead)")
    ap.add_argument("--host-threads", type=int, default=0)
    ap.add_argument("--no-sweep", action="store_true", help="skip the W sweep")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-clocks", action="store_true", help="debug: do not poll nvidia-smi during the timed region")
    ap.add_argument("--no-profile", action="store_true", help="debug: time the headline without the per-kernel event pairs")
    ap.add_argument("--cpu-sample-batches", type=int, default=4)
    return ap.parse_args()


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(name):
    """dram read+write bytes per launch from a committed ncu --set full summary under profiles/."""
    p = os.path.join(ROOT, "profiles", name)
    if os.path.exists(p):
        for line in open(p):
            if line.startswith("traffic_bytes_per_launch:"):
                return float(line.split(":")[1])
    return None


# Issue slots the key loop of k_select_warp / k_select_thread spends per key (84 SASS
# instructions per 4 keys: DESIGN.md Sec. 6); the ALU roofline is one warp instruction per clock
# per SM sub-partition.
KEY_ISSUE_SLOTS = 21.0
SM_COUNT, SMSP_PER_SM = 148, 4


def alu_peak_gkeys(sm_mhz):
    return SM_COUNT * SMSP_PER_SM * 32 * sm_mhz * 1e6 / KEY_ISSUE_SLOTS / 1e9


class EnergyMeter:
    """NVML total-energy counter (mJ) around the timed region (north star: NVML energy per epoch)."""

    def __init__(self, index):
        self.h = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.nv.nvmlDeviceGetTotalEnergyConsumption(self.h)
        except Exception:
            self.h = None

    def read_mj(self):
        if self.h is None:
            return None
        try:
            return float(self.nv.nvmlDeviceGetTotalEnergyConsumption(self.h))
        except Exception:
            return None


class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except Exception:
            self.proc.kill()
            out = ""
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            t = [x.strip() for x in line.split(",")]
            if len(t) < 7:
                continue
            try:
                sm.append(float(t[0]))
                mx.append(float(t[1]))
            except ValueError:
                continue
            for n, v in zip(names, t[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def run_reference(args):
    """The CPU oracle as it stands, timed on the host cores (the reference arm of this tier)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2606_02916_b200 import inputs
    from oracle import ggo
    dev = "cuda:0" if torch.cuda.is_available() else "cpu"
    w = inputs.make_workload(args.config, device=dev, pin=False, batch=args.batch)
    g = ggo.Graph(*w.host_graph())
    feat = w.host_features()
    po = w.part_offsets
    parts = [np.ascontiguousarray(feat[po[m]:po[m + 1]]) for m in range(len(po) - 1)]
    S = 1                                   # mini-batches per step (bounded sample of the epoch)
    st = ggo.State(g.n, po, 0, args.n_hot, 1)

    def step(i):
        bs = [ggo.Batch(g, w.batches[(i * S + j) % len(w.batches)], w.fanouts, w.seed, (i * S + j) % len(w.batches))
              for j in range(S)]
        st.run_window(bs)
        for b in bs:
            ggo.gather(b.nodes, po, parts, w.row_bytes)

    for i in range(args.warmup):
        step(i)
    t0 = time.perf_counter()
    for i in range(args.steps):
        step(args.warmup + i)
    dt = time.perf_counter() - t0
    v = args.steps * S / dt
    sample = "%d mini-batch(es) per step as W=%d windows of the same workload (sample + window + gather)" % (S, S)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u8/int32/uint64",
        "data": "synthetic",
        "config": {"workload": workload_name(args, w), "step": sample},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def workload_name(args, w):
    return ("%s: N=%d nnz=%d dim=%d %s, %d train seeds, batch=%d (%d mini-batches/epoch), fanouts=%s, "
            "4 owner ranges (local in HBM, 3 in pinned host)"
            % (args.config, w.num_nodes, w.indices.numel(), w.dim, str(w.dtype).replace("torch.", ""),
               sum(len(b) for b in w.batches), args.batch, len(w.batches), w.fanouts))


class E2ESink:
    """End-to-end leg: every batch's results are read back into pinned HOST buffers.
    Two device feature buffers alternate; a copy stream drains batch i while batch i+1 is
    gathered (user-level double buffering, all inside the timed region)."""

    def __init__(self, w, cap_rows, dev):
        self.dev = dev
        self.feats = [torch.empty(cap_rows, w.dim, dtype=w.dtype, device=dev) for _ in range(2)]
        self.h_x = [torch.empty(cap_rows, w.dim, dtype=w.dtype, pin_memory=True) for _ in range(2)]
        self.h_nodes = [torch.empty(cap_rows, dtype=torch.int32, pin_memory=True) for _ in range(2)]
        ecap = cap_rows * 2
        self.h_blk = [torch.empty(ecap * 2 + cap_rows * 2, dtype=torch.int32, pin_memory=True) for _ in range(2)]
        self.copy_stream = torch.cuda.Stream(dev)
        self.done = [None, None]
        self.i = 0
        self.d2h_bytes = 0

    def buffer(self):
        k = self.i & 1
        if self.done[k] is not None:
            torch.cuda.current_stream(self.dev).wait_event(self.done[k])   # buffer k drained
        return self.feats[k]

    def consume(self, r):
        k = self.i & 1
        ev = torch.cuda.Event()
        ev.record(torch.cuda.current_stream(self.dev))
        with torch.cuda.stream(self.copy_stream):
            self.copy_stream.wait_event(ev)
            n = r["n_input"]
            self.h_x[k][:n].copy_(r["features"], non_blocking=True)
            self.h_nodes[k][:n].copy_(r["input_nodes"], non_blocking=True)
            self.d2h_bytes += n * (r["features"].shape[1] * r["features"].element_size() + 4)
            off = 0
            for blk in r["blocks"]:
                for key in ("indptr", "src_local"):
                    t = blk[key]
                    self.h_blk[k][off:off + t.numel()].copy_(t, non_blocking=True)
                    off += t.numel()
                    self.d2h_bytes += 4 * t.numel()
            d = torch.cuda.Event()
            d.record(self.copy_stream)
            self.done[k] = d
        self.i += 1

    def fence(self, stream):
        """Orders `stream` behind every copy issued so far: they read the window's block arrays and
        N_b, which gg_window_release(stream) hands back to the sampler."""
        last = self.done[(self.i - 1) & 1] if self.i else None
        if last is not None:
            stream.wait_event(last)

    def finish(self):
        self.copy_stream.synchronize()


def run_ours(args):
    from paper_2606_02916_b200 import build, dist as gdist, epoch as ep, inputs, binding
    build.build_library()
    rank, local_rank, world = gdist.init("nccl")
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    P = inputs.CONFIGS[args.config]["parts"]
    w = inputs.make_workload(args.config, device=dev, batch=args.batch, local_part=rank % P)
    n_b = len(w.batches)
    _, order = gdist.shard_plan(rank, world, P, n_b)
    batches = [w.batches[i] for i in order]
    W = args.window
    sweep_ws = [] if args.no_sweep or world > 1 else [x for x in w.cfg["windows"] if x != W]
    g = ep.graph_from_workload(w, n_hot=args.n_hot, carry_over=1, max_window=max([W] + sweep_ws),
                               staging_mode=args.staging_mode, max_live_windows=args.lookahead + 1,
                               host_threads=args.host_threads)
    LA = args.lookahead
    # gathers run on a high-priority stream so their CTAs are scheduled ahead of the library's
    # (long-running, ALU-bound) sampling kernels whenever an SM has room for both
    stream = torch.cuda.Stream(dev, priority=-1)
    torch.cuda.set_stream(stream)
    energy = EnergyMeter(local_rank)
    link_peak = host_link_peak(dev)

    # size the output buffer from the first window (|N_b| varies little between batches)
    g.window_stage(10 ** 9, 0, batches[:min(W, 4)], w.fanouts)
    cap_rows = int(max(g.batch_info(10 ** 9, j)["n_input"] for j in range(min(W, 4), )) * 1.25) + 1024
    g.window_release(10 ** 9)
    g.cache_reset()
    feats = torch.empty(cap_rows, w.dim, dtype=w.dtype, device=dev)

    def one_epoch(Wx, sink=None, wid0=0):
        if sink is None:
            ep.run_epoch(g, batches, w.fanouts, Wx, feats, stream=stream, first_window_id=wid0, lookahead=LA)
        else:
            wins = ep.windows_of(n_b, Wx)
            for k in range(min(LA, len(wins))):
                g.window_stage(wid0 + k, wins[k].start, [batches[i] for i in wins[k]], w.fanouts)
            for k, win in enumerate(wins):
                if k + LA < len(wins):
                    nxt = wins[k + LA]
                    g.window_stage(wid0 + k + LA, nxt.start, [batches[i] for i in nxt], w.fanouts)
                for j, _bi in enumerate(win):
                    sink.consume(g.batch_gather(wid0 + k, j, sink.buffer(), stream))
                sink.fence(stream)
                g.window_release(wid0 + k, stream)
            sink.finish()
        torch.cuda.synchronize(dev)
        g.cache_reset()

    def timed(Wx, K, warm, sink=None, profile=False, clocks=None):
        for e in range(warm):
            one_epoch(Wx, sink, wid0=1000 * e)
        if profile:
            g.profile_enable(True)
        l0 = binding.launch_count()
        torch.cuda.synchronize(dev)
        gdist.barrier()
        if clocks:
            clocks.start()
        s0 = binding.sampler_stats() if profile else None
        mj0 = energy.read_mj()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record(stream)
        per_epoch = []
        for e in range(K):
            t_e = time.perf_counter()
            one_epoch(Wx, sink, wid0=1000 * (warm + e))      # ends with a device synchronise
            per_epoch.append(1e3 * (time.perf_counter() - t_e))
        e1.record(stream)
        torch.cuda.synchronize(dev)
        wall = time.perf_counter() - t0
        mj1 = energy.read_mj()
        s1 = binding.sampler_stats() if profile else None
        gdist.barrier()
        ck = clocks.stop() if clocks else None
        sec = e0.elapsed_time(e1) / 1e3
        prof = g.profile_get() if profile else None
        if profile:
            g.profile_enable(False)
        samp = {k: s1[k] - s0[k] for k in s0} if profile else None
        joules = (mj1 - mj0) / 1e3 if (mj0 is not None and mj1 is not None) else None
        return dict(sec=sec, wall=wall, launches=binding.launch_count() - l0, prof=prof, clocks=ck,
                    sampler=samp, joules=joules, per_epoch_ms=per_epoch)

    errors = {}

    def recover_graph(old):
        """After a failed optional leg: drop whatever state the graph is in and start a fresh one."""
        try:
            old.close()
        except Exception:
            pass
        torch.cuda.synchronize(dev)
        return ep.graph_from_workload(w, n_hot=args.n_hot, carry_over=1, max_window=max([W] + sweep_ws),
                                      staging_mode=args.staging_mode, max_live_windows=args.lookahead + 1,
                                      host_threads=args.host_threads)

    # ---- headline: device-resident inputs --------------------------------------------------
    if args.no_profile:
        r0 = timed(W, args.steps, args.warmup, profile=False, clocks=None)
        print("debug: unprofiled headline %.1f mini-batches/s, %.2f ms/epoch" % (args.steps * n_b / r0["sec"], 1e3 * r0["sec"] / args.steps),
              file=sys.stderr)
    main = timed(W, args.steps, args.warmup, profile=True, clocks=None if args.no_clocks else ClockSampler(local_rank))
    value, tmax = gdist.aggregate_throughput(args.steps * n_b, main["sec"], dev)
    # per-window trace of one more epoch (bytes over the host link, stall, timings)
    tr_acc = dict(bulk_bytes=0, bulk_copies=0, wait_ms=0.0, stage_ms=0.0, pack_ms=0.0, h2d_ms=0.0, n_access=0)

    def on_window(wid, win):
        t = g.trace(wid, len(win))
        tr_acc["bulk_bytes"] += sum(t["bulk_bytes"])
        tr_acc["bulk_copies"] += t["bulk_copies"]
        tr_acc["wait_ms"] += t["ms_boundary_wait"]
        tr_acc["stage_ms"] += t["ms_stage_total"]
        tr_acc["pack_ms"] += t["ms_pack_host"]
        tr_acc["h2d_ms"] += t["ms_h2d"]
        tr_acc["n_access"] += t["n_access"]

    ep.run_epoch(g, batches, w.fanouts, W, feats, on_window=on_window, stream=stream, first_window_id=5 * 10 ** 6,
                 lookahead=LA)
    torch.cuda.synchronize(dev)
    g.cache_reset()

    # ---- the same kernels with the pipeline switched off: sample+stage a window, wait, then
    # serve it, so no two of the library's streams compete for the SMs (one epoch, untimed as a
    # whole; only the per-kernel event pairs are read).  Says what the kernels do alone; the
    # live fractions above say what they do inside the overlapped step.
    g.profile_enable(True)
    s0 = binding.sampler_stats()
    for k, win in enumerate(ep.windows_of(n_b, W)):
        g.window_stage(7 * 10 ** 6 + k, win.start, [batches[i] for i in win], w.fanouts)
        g.batch_info(7 * 10 ** 6 + k, 0)
        g.trace(7 * 10 ** 6 + k, len(win))           # synchronises the window's staging
        for j in range(len(win)):
            g.batch_gather(7 * 10 ** 6 + k, j, feats, stream)
        torch.cuda.synchronize(dev)
        g.window_release(7 * 10 ** 6 + k)
    serial_prof = g.profile_get()
    serial_keys = binding.sampler_stats()["keys"] - s0["keys"]
    g.profile_enable(False)
    g.cache_reset()

    # ---- end to end: results read back to pinned host buffers every batch -------------------
    e2e = None
    if not args.no_e2e:
        sink = E2ESink(w, cap_rows, dev)
        r = timed(W, max(1, min(args.steps, 2)), 1, sink=sink)
        k_e = max(1, min(args.steps, 2))
        ev, _ = gdist.aggregate_throughput(k_e * n_b, r["sec"], dev)
        seeds_bytes = 4 * sum(len(b) for b in batches)
        e2e = {"value": ev, "unit": UNIT,
               "h2d_bytes_per_step": int(seeds_bytes + tr_acc["bulk_bytes"]),
               "d2h_bytes_per_step": int(sink.d2h_bytes / (k_e + 1)),
               "note": "seeds from host buffers via gg_window_stage; remote rows staged pinned->HBM inside the "
                       "library; X_b, N_b, block indptr/src_local copied to pinned host every batch"}
        del sink

    # ---- W sweep (the metric is 'per epoch vs W'): 1 warm + 1 timed epoch per point ----------
    vs_w = {str(W): value}
    j_w = {str(W): (main["joules"] / args.steps) if main["joules"] is not None else None}
    for Wx in sweep_ws:
        r = timed(Wx, 3, 1)
        vs_w[str(Wx)] = 3 * n_b / r["sec"]
        j_w[str(Wx)] = (r["joules"] / 3) if r["joules"] is not None else None

    # ---- NEXT-1: the paper's offline phase on this box: coefficients probed here, then the trace
    # simulator + Eqs. (1)-(3) for every candidate W (gg_simulate), against the measured ranking
    simulator = None
    try:
        if sweep_ws and rank == 0:
            from paper_2606_02916_b200 import profiler
            cands = sorted([W] + sweep_ws)
            model = profiler.measure_energy_model(dev, w.row_bytes, P, local_part=rank % P)
            probes = model.pop("probes")
            p_active = model.pop("p_active")
            t0 = time.perf_counter()
            sim = g.simulate(batches, w.fanouts, cands, model)
            t_sim = time.perf_counter() - t0
            pred = [r["e_phy"] for r in sim["results"]]
            meas_j = [j_w.get(str(c)) for c in cands]
            meas_t = [n_b / vs_w[str(c)] for c in cands]
            simulator = {
                "candidates": cands, "W_star": sim["best"], "offline_phase_s": t_sim,
                "e_phy_J": pred, "measured_J_per_epoch": meas_j, "measured_s_per_epoch": meas_t,
                "kendall_tau_vs_measured_J": kendall_tau(pred, meas_j) if all(x is not None for x in meas_j) else None,
                "kendall_tau_vs_measured_s": kendall_tau(pred, meas_t),
                "z": [{k: r[k] for k in ("rebuild_events", "miss_events", "t_stall", "hit_ratio", "rebuild_rows", "miss_rows")}
                      for r in sim["results"]],
                "coefficients": {"lam_init_s": max(model["lam_init"]), "lam_payload_s_per_row": max(model["lam_pay_b"]),
                                 "eps_init_J": max(model["eps_init"]), "eps_payload_J_per_row": max(model["eps_pay_b"]),
                                 "bw_GB/s": model["bw"] / 1e9, "p_idle_W": model["p_idle"], "p_active_W": p_active,
                                 "probes_bytes_s": probes},
                "calibration": calibrate(sim["results"], meas_j),
                "note": "coefficients probed on this box (pinned H2D copies + NVML power); PAPER.md:186 reports < 5 s for the offline phase, "
                        "PAPER.md:345 Kendall tau 0.62-1.00 on its cluster",
            }
    except Exception as exc:      # an optional leg must not cost the headline line
        errors['simulator'] = repr(exc)
        g = recover_graph(g)

    # ---- BASELINE.json configs[2]: batch in {1024, 2048, 4096} at the same W -------------------
    vs_batch = {}
    try:
        if not args.no_sweep and world == 1 and args.config == "products":
            vs_batch[str(args.batch)] = {"mini_batches_per_s": value, "seeds_per_s": value * args.batch}
            all_seeds = np.concatenate(batches)
            for Bx in (2048, 4096):
                if Bx == args.batch:
                    continue
                bx = [all_seeds[i:i + Bx] for i in range(0, len(all_seeds), Bx)]
                g.close()
                g = ep.graph_from_workload(w, n_hot=args.n_hot, carry_over=1, max_window=W, staging_mode=args.staging_mode,
                                           max_live_windows=args.lookahead + 1, max_batch=Bx)
                fx = torch.empty(int(cap_rows * Bx / args.batch) + 1024, w.dim, dtype=w.dtype, device=dev)
                def ep_b():
                    ep.run_epoch(g, bx, w.fanouts, W, fx, stream=stream, first_window_id=0, lookahead=LA)
                    torch.cuda.synchronize(dev)
                    g.cache_reset()
                n_warm = max(2, -(-(LA + 1) // max(1, -(-len(bx) // W))) + 1)      # every window arena used at least once
                for _ in range(n_warm):
                    ep_b()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                for _ in range(3):
                    ep_b()
                b.record(stream)
                torch.cuda.synchronize(dev)
                v = 3 * len(bx) / (a.elapsed_time(b) * 1e-3)
                vs_batch[str(Bx)] = {"mini_batches_per_s": v, "seeds_per_s": v * Bx, "mini_batches_per_epoch": len(bx)}
                del fx
            g.close()
            g = ep.graph_from_workload(w, n_hot=args.n_hot, carry_over=1, max_window=max([W] + sweep_ws),
                                       staging_mode=args.staging_mode, max_live_windows=args.lookahead + 1,
                                       host_threads=args.host_threads)
    except Exception as exc:      # an optional leg must not cost the headline line
        errors['vs_batch'] = repr(exc)
        g = recover_graph(g)

    # ---- variant: epochs back to back with the cache carried over (reading S15: the cache
    # persists across epochs; the trace repeats), no reset and no drain between
    # epochs -- what a long training run sees after its first epoch
    variants = {}
    try:
        if not args.no_sweep and world == 1:
            KE = 4
            wins = ep.windows_of(n_b, W)
            seq = [(e, k) for e in range(KE + 1) for k in range(len(wins))]      # epoch 0 warms the cache
            wid = lambda i: 9 * 10 ** 6 + i
            def stage_i(i):
                win = wins[seq[i][1]]
                g.window_stage(wid(i), win.start, [batches[j] for j in win], w.fanouts)
            for i in range(min(LA, len(seq))):
                stage_i(i)
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            for i in range(len(seq)):
                if i == len(wins):
                    ev0.record(stream)                                           # first gather of epoch 1
                if i + LA < len(seq):
                    stage_i(i + LA)
                for j in range(len(wins[seq[i][1]])):
                    g.batch_gather(wid(i), j, feats, stream)
                g.window_release(wid(i))
            ev1.record(stream)
            torch.cuda.synchronize(dev)
            g.cache_reset()
            variants["warm_cache_back_to_back_epochs"] = {
                "value": KE * n_b / (ev0.elapsed_time(ev1) * 1e-3), "unit": UNIT, "epochs": KE,
                "note": "no cache reset and no drain between epochs (the cache persists across epochs, the trace repeats): "
                        "measured because the headline protocol resets the cache every epoch; it helps little here: the last window of a "
                        "193-batch epoch holds ONE batch, C_k = H_k (reading S11) then evicts almost everything, and the next epoch "
                        "starts nearly cold anyway"}
    except Exception as exc:      # an optional leg must not cost the headline line
        errors['warm_cache'] = repr(exc)
        g = recover_graph(g)

    # ---- NEXT-4: the same epoch with the paper's consumer behind every gather (Alg. 1 l.15): a
    # GraphSAGE-mean model, one layer per hop, 16 hidden units, 47 synthetic classes
    try:
        if not args.no_sweep and world == 1 and w.dtype == torch.float32 and w.dim <= 128:
            Lm = len(w.fanouts)
            dims = [w.dim] + [16] * (Lm - 1) + [47]
            rng = np.random.default_rng(7)
            p0 = [dict(W_self=(rng.uniform(-1, 1, (dims[l], dims[l + 1])) / np.sqrt(dims[l])).astype(np.float32),
                       W_neigh=(rng.uniform(-1, 1, (dims[l], dims[l + 1])) / np.sqrt(dims[l])).astype(np.float32),
                       b=np.zeros(dims[l + 1], np.float32)) for l in range(Lm)]
            model = binding.Sage(p0, dev)
            labels = torch.randint(0, 47, (n_b, args.batch), dtype=torch.int32, device=dev)
            losses = []

            def train(k, j, bi, r):
                model.step(r, labels[bi, :r["blocks"][0]["n_dst"]].contiguous(), 0.003, stream)

            def epoch_c(wid0):
                ep.run_epoch(g, batches, w.fanouts, W, feats, on_batch=train, stream=stream, first_window_id=wid0, lookahead=LA)
                torch.cuda.synchronize(dev)
                losses.append(float(model.loss.cpu()[0]))
                g.cache_reset()
            epoch_c(11 * 10 ** 6)
            g.profile_enable(True)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            for e in range(3):
                epoch_c(11 * 10 ** 6 + 1000 * (e + 1))
            b.record(stream)
            torch.cuda.synchronize(dev)
            stall_c = g.profile_get()["wait"]["ms"] / 3
            g.profile_enable(False)
            variants["with_graphsage_consumer"] = {
                "value": 3 * n_b / (a.elapsed_time(b) * 1e-3), "unit": UNIT, "model": "GraphSAGE-mean, dims %s, SGD lr 0.003" % dims,
                "gpu_stall_ms_per_epoch": stall_c,
                "last_batch_loss_per_epoch": losses,
                "note": "forward + loss + backward + update of every mini-batch on the caller's stream right behind its gather"}
            model.close()
    except Exception as exc:      # an optional leg must not cost the headline line
        errors['consumer'] = repr(exc)
        g = recover_graph(g)

    # ---- variant (NEXT-2): GPU-initiated pull staging instead of host pack + cudaMemcpyAsync ----
    try:
        if not args.no_sweep and world == 1 and args.staging_mode == 0:
            g.close()
            g = ep.graph_from_workload(w, n_hot=args.n_hot, carry_over=1, max_window=max([W] + sweep_ws), staging_mode=1,
                                       max_live_windows=args.lookahead + 1)
            r = timed(W, 3, 2)
            variants["staging_mode_1_gpu_pull"] = {"value": 3 * n_b / r["sec"], "unit": UNIT,
                                                   "note": "k_rows<.,1> reads the owners' pinned rows over PCIe (12 CTAs), no host pack, no ID read-back"}
    except Exception as exc:      # an optional leg must not cost the headline line
        errors['gpu_pull'] = repr(exc)
        g = recover_graph(g)

    if rank != 0:
        return
    # ---- rooflines: the dominant kernel group (a-1 sampling, ALU-bound) and the gather (HBM) ----
    peak, peak_src = measured_peaks()
    pg = main["prof"]["gather"]
    ach = pg["bytes"] / (pg["ms"] * 1e-3) / 1e9 if pg["ms"] > 0 else 0.0
    g_scale = args.steps * n_b / max(pg["regions"], 1)      # one launch in four carries an event pair
    roof_gather = {"bound": "hbm", "kernel": "k_gather", "achieved": ach, "peak": peak, "unit": "GB/s",
                   "frac": ach / peak, "traffic": ncu_traffic("r01_gather_ncu_summary.txt"), "peak_source": peak_src,
                   "launches": args.steps * n_b, "bracketed_launches": pg["regions"],
                   "avg_launch_us": 1e3 * pg["ms"] / max(pg["regions"], 1),
                   "algorithmic_bytes_per_launch": pg["bytes"] / max(pg["regions"], 1),
                   "share_of_step": g_scale * pg["ms"] * 1e-3 / main["sec"],
                   "note": "live: shares the SMs with the sampler on the side stream; alone it runs at the ncu time in profiles/"}
    ps = main["prof"]["sample"]
    sm_mhz = (main["clocks"] or {}).get("sm_max_mhz") or 1965.0
    keys = main["sampler"]["keys"]
    gk = keys / (ps["ms"] * 1e-3) / 1e9 if ps["ms"] > 0 else 0.0
    gk_peak = alu_peak_gkeys(sm_mhz)
    roof = {"bound": "alu", "kernel": "a-1 sampling (k_sample_count/plan + k_select_thread + k_select_warp per hop)",
            "achieved": gk, "peak": gk_peak, "unit": "Gkey/s", "frac": gk / gk_peak,
            "traffic": ncu_traffic("r01_sample_ncu_summary.txt"),
            "peak_source": "derived: %d SMs x %d sub-partitions x 1 warp instruction/clk x 32 lanes x %.0f MHz / %.0f issue "
                           "slots per key (DESIGN.md Sec. 6)" % (SM_COUNT, SMSP_PER_SM, sm_mhz, KEY_ISSUE_SLOTS),
            "launches": ps["regions"], "avg_launch_us": 1e3 * ps["ms"] / max(ps["regions"], 1),
            "algorithmic_keys_per_launch": keys / max(ps["regions"], 1),
            "keyed_rows_per_step": main["sampler"]["rows"] / args.steps,
            "fallback_rows_per_step": main["sampler"]["fallbacks"] / args.steps,
            "share_of_step": ps["ms"] * 1e-3 / main["sec"]}
    sp_s, sp_g = serial_prof["sample"], serial_prof["gather"]
    serial = {
        "what": "same epoch with the pipeline off (stage a window, wait, serve it): kernels run without SM contention",
        "sample_Gkey/s": serial_keys / (sp_s["ms"] * 1e-3) / 1e9 if sp_s["ms"] > 0 else None,
        "sample_frac_of_alu_peak": (serial_keys / (sp_s["ms"] * 1e-3) / 1e9 / gk_peak) if sp_s["ms"] > 0 else None,
        "gather_GB/s": sp_g["bytes"] / (sp_g["ms"] * 1e-3) / 1e9 if sp_g["ms"] > 0 else None,
        "gather_frac_of_hbm_peak": (sp_g["bytes"] / (sp_g["ms"] * 1e-3) / 1e9 / peak) if sp_g["ms"] > 0 else None,
        "h2d_GB/s": (serial_prof["stage_copy"]["bytes"] / (serial_prof["stage_copy"]["ms"] * 1e-3) / 1e9)
        if serial_prof["stage_copy"]["ms"] > 0 else None,
        "ms_per_epoch": {k: round(v["ms"], 3) for k, v in serial_prof.items() if v["regions"]},
    }
    if serial["h2d_GB/s"]:
        serial["h2d_frac_of_link_peak"] = serial["h2d_GB/s"] / link_peak
    stages = {}
    for k, v in main["prof"].items():
        if v["regions"]:
            sc = g_scale if k == "gather" else 1.0
            stages[k] = {"ms_per_step": sc * v["ms"] / args.steps, "regions_per_step": sc * v["regions"] / args.steps,
                         "GB/s": (v["bytes"] / (v["ms"] * 1e-3) / 1e9) if v["ms"] > 0 and v["bytes"] else None}

    cpu = None
    if not args.no_cpu_baseline:
        cpu = cpu_baseline(args, w, batches)

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * tmax / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "u8 rows / int32 ids / uint64 keys",
        "data": "synthetic",
        "config": {"workload": workload_name(args, w), "W": W, "n_hot": args.n_hot,
                   "staging_mode": args.staging_mode, "carry_over": 1, "lookahead_windows": LA,
                   "step": "one epoch = %d mini-batches in %d windows, cache reset per epoch" % (n_b, -(-n_b // W)),
                   "l2": "inputs larger than L2 (feature store %.0f MB, X_b %.0f MB per batch)"
                         % (w.num_nodes * w.row_bytes / 1e6, tr_acc["n_access"] / n_b * w.row_bytes / 1e6)},
        "clocks": main["clocks"], "gpu_launches": int(main["launches"]),
        "wall_ms_per_step": 1e3 * main["wall"] / args.steps,
        "epoch_ms": {"median": statistics.median(main["per_epoch_ms"]), "min": min(main["per_epoch_ms"]),
                     "max": max(main["per_epoch_ms"]), "note": "host clock around each epoch incl. its final synchronise and cache reset"},
        "roofline": roof, "roofline_gather": roof_gather, "kernels_alone": serial, "stages": stages, "vs_W": vs_w,
        "J_per_epoch_vs_W": j_w, "vs_batch_at_W": vs_batch, "simulator": simulator, "variants": variants,
        "errors": errors,
        "gpu_stall_ms_per_step": (main["prof"]["wait"]["ms"] / args.steps) if "wait" in main["prof"] else None,
        "energy": {"J_per_step": (main["joules"] / args.steps) if main["joules"] is not None else None,
                   "avg_W": (main["joules"] / main["wall"]) if main["joules"] is not None else None,
                   "source": "NVML total energy counter over the timed region"},
        "staging": {"host_link_bytes_per_step": int(tr_acc["bulk_bytes"]), "bulk_copies_per_step": tr_acc["bulk_copies"],
                    "h2d_GB/s": tr_acc["bulk_bytes"] / (tr_acc["h2d_ms"] * 1e-3) / 1e9 if tr_acc["h2d_ms"] > 0 else None,
                    "host_link_peak_GB/s": link_peak,
                    "h2d_frac_of_link_peak": (tr_acc["bulk_bytes"] / (tr_acc["h2d_ms"] * 1e-3) / 1e9 / link_peak)
                    if tr_acc["h2d_ms"] > 0 else None,
                    "host_pack_ms_per_step": tr_acc["pack_ms"], "stage_ms_per_step": tr_acc["stage_ms"],
                    "boundary_stall_ms_per_step": tr_acc["wait_ms"]},
        "e2e": e2e, "cpu_baseline": cpu,
    }
    print(json.dumps(out))
    g.close()


def calibrate(results, meas_j):
    """NEXT-3 (Eq. 5): rank calibration of S(W) = beta^T z(W) + gamma_W against the measured J/epoch
    of the sweep, on the device (gg_rank_calibrate); z columns scaled to unit max."""
    if any(x is None for x in meas_j):
        return None
    from paper_2606_02916_b200 import binding
    Z = np.array([[r["rebuild_events"], r["miss_events"], r["t_stall"], r["hit_ratio"]] for r in results], dtype=np.float64)
    Z = Z / np.maximum(np.abs(Z).max(axis=0), 1e-300)
    e = np.array(meas_j, dtype=np.float64)
    beta, gamma, loss = binding.rank_calibrate(Z, e, 0.1, 0.05, 2000)
    S = Z @ beta + gamma
    return {"beta": beta.tolist(), "gamma": gamma.tolist(), "loss": loss,
            "kendall_tau_S_vs_measured_J": kendall_tau(S.tolist(), meas_j),
            "features": ["rebuild_events", "miss_events", "t_stall", "hit_ratio"], "lambda": 0.1, "lr": 0.05, "iters": 2000}


def kendall_tau(a, b):
    n, s = len(a), 0
    for i in range(n):
        for j in range(i + 1, n):
            x = (a[i] - a[j]) * (b[i] - b[j])
            s += 1 if x > 0 else (-1 if x < 0 else 0)
    return s / (n * (n - 1) / 2) if n > 1 else None


def host_link_peak(dev, nbytes=1 << 30, reps=10):
    """Pinned host -> device peak: one 1 GiB cudaMemcpyAsync, best of `reps` (GB/s)."""
    src = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
    dst = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    best = 0.0
    for _ in range(reps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        dst.copy_(src, non_blocking=True)
        b.record()
        b.synchronize()
        best = max(best, nbytes / (a.elapsed_time(b) * 1e-3) / 1e9)
    del src, dst
    return best


def cpu_baseline(args, w, batches):
    """The oracle as it stands on the host cores, on a bounded sample of the same workload."""
    from oracle import ggo
    S = min(args.cpu_sample_batches, len(batches), args.window)
    g = ggo.Graph(*w.host_graph())
    feat = w.host_features()
    po = w.part_offsets
    parts = [np.ascontiguousarray(feat[po[m]:po[m + 1]]) for m in range(len(po) - 1)]
    st = ggo.State(g.n, po, w.local_part, args.n_hot, 1)
    t0 = time.perf_counter()
    bs = [ggo.Batch(g, batches[j], w.fanouts, w.seed, j) for j in range(S)]
    st.run_window(bs)
    for b in bs:
        ggo.gather(b.nodes, po, parts, w.row_bytes)
    dt = time.perf_counter() - t0
    return {"value": S / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": "first %d mini-batches of the epoch as one W=%d window (sample + window + gather), %.1f s"
                      % (S, S, dt)}


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)

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
DTYPE = "u8 rows / int32 ids / uint64 keys"


def parse_args(argv=None):
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
    ap.add_argument("--sampler-tune", default="", help="single_bins,warp_bin,hub_bin for gg_sampler_tune (default: the library's)")
    ap.add_argument("--cache-buffers", type=int, default=4, help="HBM cache buffers in rotation (gg_config.cache_buffers)")
    ap.add_argument("--full", action="store_true",
                    help="also run the optional legs (W sweep, BASELINE.json:configs grid, simulator, variants); they go to "
                         "bench_detail.json, never into the result line")
    ap.add_argument("--no-sweep", action="store_true", help="with --full: skip the optional legs after all")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-clocks", action="store_true", help="debug: do not poll nvidia-smi during the timed region")
    ap.add_argument("--no-profile", action="store_true", help="debug: time the headline without the per-kernel event pairs")
    ap.add_argument("--cpu-sample-batches", type=int, default=4)
    ap.add_argument("--configs", default="products,dense,large",
                    help="workloads of the `configs` grid (BASELINE.json:configs); '' switches the grid off")
    ap.add_argument("--configs-budget-s", type=float, default=420.0, help="wall-clock budget of the `configs` grid")
    args = ap.parse_args(argv)
    if not args.full:
        args.no_sweep = True       # the default run is the headline + rooflines + e2e + cpu_baseline only
    return args


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


# The sampler's roofline is the key-only micro-kernel measured in the same run (gg_key_peak).  Two
# derived figures are kept beside it as notes: the issue-slot bound of the product loop (84 SASS
# instructions per 4 keys = 21 slots per key) and of the hash alone (16 slots per key), both at one
# warp instruction per clock per SM sub-partition -- a rate this integer mix does not reach.
KEY_ISSUE_SLOTS, HASH_ISSUE_SLOTS = 21.0, 16.0
# the hash needs 11 ALU-pipe instructions per key at 2 clocks per warp instruction = 22
# ALU-pipe clocks per warp-key: the pipe bound (1.69 Tkey/s at 1965 MHz) the measured key-only peak sits under
ALU_PIPE_CLOCKS = 22.0
SMSP_PER_SM = 4


def derived_alu_peak_gkeys(sm_mhz, sm_count, slots):
    return sm_count * SMSP_PER_SM * 32 * sm_mhz * 1e6 / slots / 1e9


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
    # one step = one window of W mini-batches of the epoch (a bounded sample of it: the oracle needs
    # seconds per mini-batch), windows taken in epoch order with the cache state carried between them;
    # the batches of a window are sampled and gathered side by side on the host cores, the oracle
    # itself unchanged
    from concurrent.futures import ThreadPoolExecutor
    from paper_2606_02916_b200 import epoch as ep
    W = args.window
    wins = ep.windows_of(len(w.batches), W)
    cores = os.cpu_count() or 1
    st = ggo.State(g.n, po, w.local_part, args.n_hot, 1)
    done = [0]

    def step(i, ex):
        win = wins[i % len(wins)]
        if i % len(wins) == 0:
            st.reset()
        bs = list(ex.map(lambda j: ggo.Batch(g, w.batches[j], w.fanouts, w.seed, j), win))
        st.run_window(bs)
        list(ex.map(lambda b: ggo.gather(b.nodes, po, parts, w.row_bytes), bs))
        done[0] += len(bs)

    with ThreadPoolExecutor(cores) as ex:
        for i in range(args.warmup):
            step(i, ex)
        done[0] = 0
        t0 = time.perf_counter()
        for i in range(args.steps):
            step(args.warmup + i, ex)
        dt = time.perf_counter() - t0
    v = done[0] / dt
    sample = ("one W=%d window of the epoch per step (%d mini-batches in %d steps), sample + window + gather, "
              "batches side by side on %d threads" % (W, done[0], args.steps, min(cores, W)))
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": DTYPE,
        "data": "synthetic",
        "config": config_record(args, w),
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": min(cores, W), "kind": "oracle", "sample": sample,
                         "cpu_model": cpu_model(), "host_cores": cores},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def workload_name(args, w):
    return ("%s: N=%d nnz=%d dim=%d %s, %d train seeds, batch=%d (%d mini-batches/epoch), fanouts=%s, "
            "4 owner ranges (local in HBM, 3 in pinned host)"
            % (args.config, w.num_nodes, w.indices.numel(), w.dim, str(w.dtype).replace("torch.", ""),
               sum(len(b) for b in w.batches), args.batch, len(w.batches), w.fanouts))


def config_record(args, w):
    """The `config` object of the result line.  Both arms (ours, --impl reference) print exactly this, built
    from the arguments and the workload alone, so that the driver can see they ran the same thing."""
    return {"workload": "%s N=%d nnz=%d dim=%d %s batch=%d (%d/epoch) fanouts=%s"
                        % (args.config, w.num_nodes, w.indices.numel(), w.dim, str(w.dtype).replace("torch.", ""),
                           args.batch, len(w.batches), ",".join(str(f) for f in w.fanouts)),
            "W": args.window, "n_hot": args.n_hot,
            "l2": ("inputs larger than L2 (feature store %.0f MB; no flush)" if w.num_nodes * w.row_bytes > 126e6 else
                   "feature store %.0f MB fits in L2: a parity-size config, not a bench line") % (w.num_nodes * w.row_bytes / 1e6)}


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
    if args.host_threads <= 0:
        args.host_threads = gdist.host_threads_for_rank()    # 0 (library default) unless ranks share the host
    sweep_ws = [] if args.no_sweep or world > 1 else [x for x in w.cfg["windows"] if x != W]
    g = ep.graph_from_workload(w, n_hot=args.n_hot, carry_over=1, max_window=max([W] + sweep_ws),
                               staging_mode=args.staging_mode, max_live_windows=args.lookahead + 1,
                               host_threads=args.host_threads, cache_buffers=args.cache_buffers)
    LA = args.lookahead
    # gathers run on a high-priority stream so their CTAs are scheduled ahead of the library's
    # (long-running, ALU-bound) sampling kernels whenever an SM has room for both
    stream = torch.cuda.Stream(dev, priority=-1)
    torch.cuda.set_stream(stream)
    if args.sampler_tune:
        binding.sampler_tune(*[int(x) for x in args.sampler_tune.split(",")])
    energy = EnergyMeter(local_rank)
    link_peak = host_link_peak(dev)
    key_peak_gkeys = binding.key_peak(8, 65536, 5) / 1e9     # measured ALU roofline of a-1, GPU otherwise idle

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
                                      host_threads=args.host_threads, cache_buffers=args.cache_buffers)

    # ---- headline: device-resident inputs --------------------------------------------------
    if args.no_profile:
        r0 = timed(W, args.steps, args.warmup, profile=False, clocks=None)
        print("debug: unprofiled headline %.1f mini-batches/s, %.2f ms/epoch" % (args.steps * n_b / r0["sec"], 1e3 * r0["sec"] / args.steps),
              file=sys.stderr)
    main = timed(W, args.steps, args.warmup, profile=True, clocks=None if args.no_clocks else ClockSampler(local_rank))
    value, tmax = gdist.aggregate_throughput(args.steps * n_b, main["sec"], dev)
    # per-window trace of one more epoch (bytes over the host link, stall, timings)
    tr_acc = dict(bulk_bytes=0, bulk_copies=0, wait_ms=0.0, stage_ms=0.0, pack_ms=0.0, h2d_ms=0.0, n_access=0, hit_local=0)

    def on_window(wid, win):
        t = g.trace(wid, len(win))
        tr_acc["bulk_bytes"] += sum(t["bulk_bytes"])
        tr_acc["bulk_copies"] += t["bulk_copies"]
        tr_acc["wait_ms"] += t["ms_boundary_wait"]
        tr_acc["stage_ms"] += t["ms_stage_total"]
        tr_acc["pack_ms"] += t["ms_pack_host"]
        tr_acc["h2d_ms"] += t["ms_h2d"]
        tr_acc["n_access"] += t["n_access"]
        tr_acc["hit_local"] += int(t["hit_local"].sum())

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

    # ---- BASELINE.json:configs, every sweep, each point with its per-stage roofline fractions ----
    vs_batch, configs, simulator_budgeted = {}, None, None
    if not args.no_sweep and world == 1 and args.config == "products" and args.configs:
        g.close()
        ctx = dict(dev=dev, stream=stream, LA=LA, hbm_peak=measured_peaks()[0], link_peak=link_peak, key_peak=key_peak_gkeys,
                   energy=energy, args=args, feats=None, edge_cut_products=None)
        try:
            ctx["edge_cut_products"] = edge_cut(w, dev)
            # what BASELINE.json:configs[2] literally asks for, measured on the same graph (reading S22)
            lab = inputs.bfs_grown_split(w.indptr, w.indices, P, w.seed)
            ctx["edge_cut_bfs_grown"] = inputs.edge_cut_of_labels(w.indptr, w.indices, lab)
            ctx["bfs_grown_sizes"] = torch.bincount(lab.long(), minlength=P).tolist()
            del lab
        except Exception as exc:
            errors["edge_cut"] = repr(exc)
        configs = configs_grid(ctx, w, batches, errors, args.configs_budget_s)
        try:
            for pt in configs.get("products_batch_x_W", {}).get("points", []):
                if pt["W"] == W:
                    vs_batch[str(pt["batch"])] = {"mini_batches_per_s": pt["mini_batches_per_s"],
                                                  "seeds_per_s": pt["mini_batches_per_s"] * pt["batch"],
                                                  "mini_batches_per_epoch": pt["mini_batches_per_epoch"]}
        except Exception as exc:
            errors["vs_batch"] = repr(exc)
        # NEXT-1 / NEXT-3 where they can fail: the budgeted series (misses > 0, the hit ratio varies with
        # W, the hot set goes stale), predicted W* against the measured argmin
        try:
            pts = configs["products_budget_10pct_x_W"]["points"]
            n_hot_b = configs["products_budget_10pct_x_W"]["n_hot"]
            from paper_2606_02916_b200 import profiler
            cands = [p_["W"] for p_ in pts]
            gb = ep.graph_from_workload(w, n_hot=n_hot_b, carry_over=1, max_window=max(cands), staging_mode=args.staging_mode,
                                        max_live_windows=LA + 1, host_threads=args.host_threads, cache_buffers=args.cache_buffers)
            try:
                model = profiler.measure_energy_model(dev, w.row_bytes, P, local_part=rank % P)
                model.pop("probes"), model.pop("p_active")
                sim = gb.simulate(batches, w.fanouts, cands, model)
            finally:
                gb.close()
            pred = [r["e_phy"] for r in sim["results"]]
            meas_j = [p_["J_per_epoch"] for p_ in pts]
            meas_t = [p_["ms_per_epoch"] for p_ in pts]
            simulator_budgeted = {
                "candidates": cands, "n_hot": n_hot_b, "W_star_predicted": sim["best"], "e_phy_J": pred,
                "measured_J_per_epoch": meas_j, "measured_ms_per_epoch": meas_t,
                "z": [{k: r[k] for k in ("rebuild_events", "miss_events", "t_stall", "hit_ratio", "rebuild_rows", "miss_rows")}
                      for r in sim["results"]],
                "kendall_tau_vs_measured_ms": kendall_tau(pred, meas_t),
                "note": "energy per epoch = NVML counter over 5 timed epochs per W; Table III's metrics (PAPER.md:343-345): "
                        "rank correlation, top-1 hit, and the measured penalty of running the simulator's pick"}
            if all(x is not None for x in meas_j):
                bi = int(np.argmin(meas_j))
                simulator_budgeted.update({
                    "W_star_measured_J": cands[bi], "top1_hit": cands[bi] == sim["best"],
                    "penalty_of_predicted_W_J_frac": meas_j[cands.index(sim["best"])] / meas_j[bi] - 1.0,
                    "kendall_tau_vs_measured_J": kendall_tau(pred, meas_j),
                    "calibration": calibrate(sim["results"], meas_j)})
            bt = int(np.argmin(meas_t))
            simulator_budgeted.update({"W_star_measured_ms": cands[bt],
                                       "penalty_of_predicted_W_ms_frac": meas_t[cands.index(sim["best"])] / meas_t[bt] - 1.0})
        except Exception as exc:
            errors["simulator_budgeted"] = repr(exc)
        g = ep.graph_from_workload(w, n_hot=args.n_hot, carry_over=1, max_window=max([W] + sweep_ws),
                                   staging_mode=args.staging_mode, max_live_windows=args.lookahead + 1,
                                   host_threads=args.host_threads, cache_buffers=args.cache_buffers)

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
        if not args.no_sweep and world == 1 and w.dtype == torch.float32 and w.dim <= 1024:
            variants["with_graphsage_consumer"] = consumer_leg(g, w, batches, W, feats, stream, dev, LA, args.batch)
    except Exception as exc:      # an optional leg must not cost the headline line
        errors['consumer'] = repr(exc)
        g = recover_graph(g)

    # ---- why the gather loses bandwidth beside the sampler: the same gathers timed alone and beside the
    # key-only ALU kernel (gg_key_peak, no memory traffic at all) at 1, 2, 4, 8 resident CTAs per SM
    try:
        if not args.no_sweep and world == 1:
            import threading
            g.window_stage(13 * 10 ** 6, 0, batches[:min(W, 16)], w.fanouts)
            nwin = min(W, 16)
            g.trace(13 * 10 ** 6, nwin)                                    # the window's staging has completed

            def time_gathers(reps=48):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                rows = 0
                a.record(stream)
                for i in range(reps):
                    rows += g.batch_gather(13 * 10 ** 6, i % nwin, feats, stream)["n_input"]
                b.record(stream)
                b.synchronize()
                return rows * (2 * w.row_bytes + 8) / (a.elapsed_time(b) * 1e-3) / 1e9

            time_gathers()
            probe = {"gather_alone_GB/s": time_gathers(), "beside_key_only_kernel": []}
            for ctas in (1, 2, 4, 8):
                res = {}
                t = threading.Thread(target=lambda: res.update(v=binding.key_peak(ctas, 65536 * 2, 30)))
                t.start()
                time.sleep(0.03)
                gb = time_gathers()
                t.join()
                probe["beside_key_only_kernel"].append({"alu_ctas_per_sm": ctas, "alu_warps_per_subpartition": 2 * ctas,
                                                        "gather_GB/s": gb, "alu_Gkey/s": res["v"] / 1e9})
            probe["note"] = ("the key-only kernel moves no memory: whatever the gather loses beside it is lost to warp scheduling on the "
                             "SMs (its warps, mostly waiting on loads, are rarely picked against always-eligible ALU warps), not to HBM or "
                             "L2 contention; the ALU kernel loses nothing")
            variants["gather_vs_alu_kernel"] = probe
            g.window_release(13 * 10 ** 6, stream)
            torch.cuda.synchronize(dev)
            g.cache_reset()
    except Exception as exc:      # an optional leg must not cost the headline line
        errors['gather_vs_alu'] = repr(exc)
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

    # ---- variant (SURVEY Sec. 8(e)'s single-box stand-in): every owner's store in DEVICE memory, as a
    # peer GPU's HBM would be over NVLink -- the bulk transfers become device-side row pulls and the
    # host link drops out: what the GPU side of the path sustains when staging is not link-bound
    try:
        if not args.no_sweep and world == 1 and w.num_nodes * w.row_bytes < 8e9:
            import dataclasses
            g.close()
            wd = dataclasses.replace(w, feat_parts=[p_.to(dev) for p_ in w.feat_parts])
            g = ep.graph_from_workload(wd, n_hot=args.n_hot, carry_over=1, max_window=max([W] + sweep_ws), staging_mode=0,
                                       max_live_windows=args.lookahead + 1, cache_buffers=args.cache_buffers)
            r = timed(W, 3, 2)
            variants["remote_owners_in_hbm"] = {"value": 3 * n_b / r["sec"], "unit": UNIT,
                                                "note": "all four feature partitions in device memory (stand-in for peer HBM): one pull "
                                                        "kernel per owner instead of pack + cudaMemcpyAsync, no host link in the path"}
            g.close()
            del wd
            g = ep.graph_from_workload(w, n_hot=args.n_hot, carry_over=1, max_window=max([W] + sweep_ws), staging_mode=args.staging_mode,
                                       max_live_windows=args.lookahead + 1, host_threads=args.host_threads, cache_buffers=args.cache_buffers)
    except Exception as exc:      # an optional leg must not cost the headline line
        errors['remote_owners_in_hbm'] = repr(exc)
        g = recover_graph(g)

    if rank != 0:
        return
    # the owners' measured edge cut and the remote fraction of N_b (what the hot path feels of the split)
    edge_cut_main, remote_frac_main = None, None
    try:
        edge_cut_main = edge_cut(w, dev)
        remote_frac_main = 1.0 - tr_acc["hit_local"] / max(tr_acc["n_access"], 1)
    except Exception as exc:
        errors["edge_cut_main"] = repr(exc)
    # ---- rooflines: the dominant kernel group (a-1 sampling, ALU-bound) and the gather (HBM) ----
    peak, peak_src = measured_peaks()
    pg = main["prof"]["gather"]
    ach = pg["bytes"] / (pg["ms"] * 1e-3) / 1e9 if pg["ms"] > 0 else 0.0
    g_scale = args.steps * n_b / max(pg["regions"], 1)      # one launch in four carries an event pair
    roof_gather = {"bound": "hbm", "kernel": "k_gather", "achieved": ach, "peak": peak, "unit": "GB/s",
                   "frac": ach / peak, "traffic": ncu_traffic("r03_gather_ncu_summary.txt"), "peak_source": peak_src,
                   "launches": args.steps * n_b, "bracketed_launches": pg["regions"],
                   "avg_launch_us": 1e3 * pg["ms"] / max(pg["regions"], 1),
                   "algorithmic_bytes_per_launch": pg["bytes"] / max(pg["regions"], 1),
                   "share_of_step": g_scale * pg["ms"] * 1e-3 / main["sec"],
                   "note": "live: shares the SMs with the sampler on the side stream; alone it runs at the ncu time in profiles/"}
    ps = main["prof"]["sample"]
    sm_mhz = (main["clocks"] or {}).get("sm_max_mhz") or 1965.0
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    keys = main["sampler"]["keys"]
    gk = keys / (ps["ms"] * 1e-3) / 1e9 if ps["ms"] > 0 else 0.0
    gk_peak = key_peak_gkeys
    roof = {"bound": "alu", "kernel": "a-1 sampling (k_sample_count/plan + the selection kernels of every hop)",
            "achieved": gk, "peak": gk_peak, "unit": "Gkey/s", "frac": gk / gk_peak,
            "frac_of_pipe_bound": gk / derived_alu_peak_gkeys(sm_mhz, sm_count, ALU_PIPE_CLOCKS),
            "pipe_bound_Gkey/s": derived_alu_peak_gkeys(sm_mhz, sm_count, ALU_PIPE_CLOCKS),
            "traffic": ncu_traffic("r02_sample_ncu_summary.txt"),
            "traffic_note": "dram read+write bytes of all a-1 kernels of one W=16 window (every hop) / 3 hop regions: the same "
                            "launches avg_launch_us averages; DRAM traffic is ~5x the algorithmic bytes on the last hop (32-byte "
                            "sectors for scattered 4-byte neighbor ids) and is not the binding resource",
            "peak_source": "measured: gg_key_peak, key-only micro-kernel (fmix high word per lane from a register-resident state, "
                           "no stores, no row logic), 8 CTAs of 256 threads per SM, CUDA events, same run, GPU otherwise idle",
            "derived_peaks_Gkey/s": {"product_loop_21_issue_slots": derived_alu_peak_gkeys(sm_mhz, sm_count, KEY_ISSUE_SLOTS),
                                     "hash_only_16_issue_slots": derived_alu_peak_gkeys(sm_mhz, sm_count, HASH_ISSUE_SLOTS),
                                     "note": "one warp instruction per clock per sub-partition; notes only, not the denominator"},
            "launches": ps["regions"], "avg_launch_us": 1e3 * ps["ms"] / max(ps["regions"], 1),
            "algorithmic_keys_per_launch": keys / max(ps["regions"], 1),
            "algorithmic_bytes_GB/s": ps["bytes"] / (ps["ms"] * 1e-3) / 1e9 if ps["ms"] > 0 else None,
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
        "scaling": "weak", "vs_baseline": None, "dtype": DTYPE,
        "data": "synthetic",
        "config": config_record(args, w),
        "protocol": {"workload_long": workload_name(args, w),
                     "edge_cut_measured": edge_cut_main, "remote_frac_of_N_b": remote_frac_main,
                     "staging_mode": args.staging_mode, "carry_over": 1, "lookahead_windows": LA,
                     "step": "one epoch = %d mini-batches in %d windows, cache reset per epoch" % (n_b, -(-n_b // W)),
                     "X_b_MB_per_batch": tr_acc["n_access"] / n_b * w.row_bytes / 1e6},
        "clocks": main["clocks"], "gpu_launches": int(main["launches"]),
        "wall_ms_per_step": 1e3 * main["wall"] / args.steps,
        "epoch_ms": {"median": statistics.median(main["per_epoch_ms"]), "min": min(main["per_epoch_ms"]),
                     "max": max(main["per_epoch_ms"]), "note": "host clock around each epoch incl. its final synchronise and cache reset"},
        "roofline": roof, "roofline_gather": roof_gather, "kernels_alone": serial, "stages": stages, "vs_W": vs_w,
        "J_per_epoch_vs_W": j_w, "vs_batch_at_W": vs_batch, "configs": configs, "simulator": simulator,
        "simulator_budgeted": simulator_budgeted, "variants": variants,
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
    g.close()
    detail = write_detail(out)
    print(json.dumps(compact_record(out, detail)))


DETAIL_FILE = "bench_detail.json"


def write_detail(out):
    """Everything the run measured goes to bench_detail.json (git-ignored; also into gpurun_out/ when that
    folder exists, so it comes back from the GPU box).  Returns the path written, or None."""
    paths = [os.path.join(ROOT, DETAIL_FILE)]
    if os.path.isdir(os.path.join(ROOT, "gpurun_out")):
        paths.append(os.path.join(ROOT, "gpurun_out", DETAIL_FILE))
    done = None
    for p in paths:
        try:
            with open(p, "w") as f:
                json.dump(out, f, indent=1)
            done = done or os.path.relpath(p, ROOT)
        except OSError:
            pass
    return done


def _sig(x, digits=6):
    """Floats to `digits` significant digits (the line is read by a driver with a small buffer)."""
    if isinstance(x, float):
        return float("%.*g" % (digits, x))
    if isinstance(x, dict):
        return {k: _sig(v, digits) for k, v in x.items()}
    if isinstance(x, (list, tuple)):
        return [_sig(v, digits) for v in x]
    return x


def _pick(d, keys):
    return {k: d[k] for k in keys if d is not None and k in d} if d is not None else None


def compact_record(out, detail_path=None):
    """The ONE line bench.py prints last: the contract's keys and the two rooflines, nothing that grows
    with the number of optional legs.  Kept under 4 KB (tests/test_bench_host.py)."""
    c = {k: out.get(k) for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step",
                                 "higher_is_better", "scaling", "vs_baseline", "dtype", "data", "config")}
    c["clocks"] = _pick(out.get("clocks"), ("sm_mhz", "sm_max_mhz", "samples", "reasons"))
    c["gpu_launches"] = out.get("gpu_launches")
    c["roofline"] = _pick(out.get("roofline"), ("bound", "kernel", "achieved", "peak", "unit", "frac", "frac_of_pipe_bound",
                                                "pipe_bound_Gkey/s", "traffic", "launches", "avg_launch_us",
                                                "algorithmic_keys_per_launch", "share_of_step"))
    if c["roofline"] is not None:
        c["roofline"]["peak_source"] = "measured in this run: gg_key_peak key-only kernel"
    c["roofline_gather"] = _pick(out.get("roofline_gather"), ("bound", "kernel", "achieved", "peak", "unit", "frac", "traffic",
                                                              "peak_source", "launches", "avg_launch_us",
                                                              "algorithmic_bytes_per_launch", "share_of_step"))
    alone = out.get("kernels_alone") or {}
    c["kernels_alone"] = _pick(alone, ("sample_frac_of_alu_peak", "gather_frac_of_hbm_peak", "h2d_frac_of_link_peak"))
    c["staging"] = _pick(out.get("staging"), ("host_link_bytes_per_step", "bulk_copies_per_step", "h2d_GB/s",
                                              "host_link_peak_GB/s", "h2d_frac_of_link_peak", "boundary_stall_ms_per_step"))
    c["gpu_stall_ms_per_step"] = out.get("gpu_stall_ms_per_step")
    c["energy"] = _pick(out.get("energy"), ("J_per_step", "avg_W"))
    c["e2e"] = _pick(out.get("e2e"), ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"))
    c["cpu_baseline"] = _pick(out.get("cpu_baseline"), ("value", "unit", "cores", "kind", "sample"))
    if out.get("vs_W"):
        c["vs_W"] = out["vs_W"]
    c["errors"] = sorted((out.get("errors") or {}).keys())
    c["detail"] = detail_path
    return _sig(c)


def consumer_leg(g, w, batches, W, feats, stream, dev, LA, batch):
    """One warm + three timed epochs with forward + loss + backward + SGD of every mini-batch on the
    caller's stream right behind its gather (gg_sage_step)."""
    from paper_2606_02916_b200 import epoch as ep, binding
    n_b = len(batches)
    Lm = len(w.fanouts)
    dims = [w.dim] + [16] * (Lm - 1) + [47]
    rng = np.random.default_rng(7)
    p0 = [dict(W_self=(rng.uniform(-1, 1, (dims[l], dims[l + 1])) / np.sqrt(dims[l])).astype(np.float32),
               W_neigh=(rng.uniform(-1, 1, (dims[l], dims[l + 1])) / np.sqrt(dims[l])).astype(np.float32),
               b=np.zeros(dims[l + 1], np.float32)) for l in range(Lm)]
    model = binding.Sage(p0, dev)
    labels = torch.randint(0, 47, (n_b, batch), dtype=torch.int32, device=dev)
    losses = []

    def train(k, j, bi, r):
        model.step(r, labels[bi, :r["blocks"][0]["n_dst"]].contiguous(), 0.003, stream)

    def epoch_c(wid0):
        ep.run_epoch(g, batches, w.fanouts, W, feats, on_batch=train, stream=stream, first_window_id=wid0, lookahead=LA)
        torch.cuda.synchronize(dev)
        losses.append(float(model.loss.cpu()[0]))
        g.cache_reset()

    try:
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
    finally:
        model.close()
    return {"value": 3 * n_b / (a.elapsed_time(b) * 1e-3), "unit": UNIT, "W": W,
            "model": "GraphSAGE-mean, dims %s, SGD lr 0.003" % dims, "gpu_stall_ms_per_epoch": stall_c,
            "last_batch_loss_per_epoch": losses,
            "note": "forward + loss + backward + update of every mini-batch on the caller's stream right behind its gather"}


def edge_cut(w, dev):
    """Measured fraction of CSR entries whose two endpoints lie in different owner ranges."""
    po = torch.as_tensor(np.asarray(w.part_offsets[1:-1], dtype=np.int32), device=dev)
    N, cut, step = w.num_nodes, 0, 1 << 22
    for r0 in range(0, N, step):
        r1 = min(N, r0 + step)
        ip = w.indptr[r0:r1 + 1]
        e0, e1 = int(ip[0]), int(ip[-1])
        if e1 == e0:
            continue
        own_row = torch.bucketize(torch.arange(r0, r1, device=dev, dtype=torch.int32), po, right=True, out_int32=True)
        own_e = torch.repeat_interleave(own_row.to(torch.int8), ip[1:] - ip[:-1])
        own_n = torch.bucketize(w.indices[e0:e1], po, right=True, out_int32=True).to(torch.int8)
        cut += int((own_e != own_n).sum())
    return cut / max(1, w.indices.numel())


def measure_point(ctx, w, batches, W, n_hot, K=2, warm=1, max_batch=None, g=None, max_window=32):
    """One (workload, batch list, W, n_hot) point of the `configs` grid: `warm` untimed + K timed epochs
    with the library's per-stage event pairs on (so the rates below are LIVE rates, all streams
    running), then one traced epoch for the byte counts.  Returns the per-stage numbers with their
    roofline fractions.  ctx: dict(dev, stream, LA, hbm_peak, link_peak, key_peak, energy, args)."""
    from paper_2606_02916_b200 import epoch as ep, binding
    dev, stream, LA, args = ctx["dev"], ctx["stream"], ctx["LA"], ctx["args"]
    own = g is None
    if own:
        g = ep.graph_from_workload(w, n_hot=n_hot, carry_over=1, max_window=max_window, staging_mode=args.staging_mode,
                                   max_live_windows=LA + 1, host_threads=args.host_threads, cache_buffers=args.cache_buffers,
                                   max_batch=max_batch or max(len(b) for b in batches))
    n_b = len(batches)
    try:
        nb0 = min(W, 4, n_b)
        g.window_stage(10 ** 9, 0, batches[:nb0], w.fanouts)
        cap_rows = int(max(g.batch_info(10 ** 9, j)["n_input"] for j in range(nb0)) * 1.25) + 1024
        g.window_release(10 ** 9)
        g.cache_reset()
        feats = ctx.get("feats")
        if feats is None or feats.shape[0] < cap_rows or feats.shape[1] != w.dim or feats.dtype != w.dtype:
            ctx["feats"] = None
            feats = torch.empty(cap_rows, w.dim, dtype=w.dtype, device=dev)
            ctx["feats"] = feats

        def one_epoch(wid0, on_window=None):
            ep.run_epoch(g, batches, w.fanouts, W, feats, stream=stream, first_window_id=wid0, lookahead=LA,
                         on_window=on_window)
            torch.cuda.synchronize(dev)
            g.cache_reset()

        t_w = time.perf_counter()
        for e in range(warm):
            one_epoch(1000 * e)
        # the NVML energy counter moves in coarse steps: time at least ~0.3 s per point
        K = int(min(8, max(K, -(-0.3 // max((time.perf_counter() - t_w) / max(warm, 1), 1e-3)))))
        g.profile_enable(True)
        s0 = binding.sampler_stats()
        mj0 = ctx["energy"].read_mj()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for e in range(K):
            one_epoch(1000 * (warm + e))
        b.record(stream)
        torch.cuda.synchronize(dev)
        mj1 = ctx["energy"].read_mj()
        sec = a.elapsed_time(b) * 1e-3
        prof = g.profile_get()
        keys = binding.sampler_stats()["keys"] - s0["keys"]
        g.profile_enable(False)
        tr = dict(bulk=0, copies=0, n_in=0, local=0, hit=0, miss=0, hot=0, uniq_remote=0)

        def on_window(wid, win):
            t = g.trace(wid, len(win))
            tr["bulk"] += sum(t["bulk_bytes"])
            tr["copies"] += t["bulk_copies"]
            tr["n_in"] += int(t["n_input"].sum())
            tr["local"] += int(t["hit_local"].sum())
            tr["hit"] += int(t["hit_cache"].sum())
            tr["miss"] += int(t["miss"].sum())
            tr["hot"] += t["n_hot"]
            tr["uniq_remote"] += t["n_unique_remote"]

        one_epoch(5 * 10 ** 6, on_window)
    finally:
        if own:
            g.close()
    rb = w.row_bytes

    def rate(kind, per_byte=1.0):
        v = prof[kind]
        return (v["bytes"] * per_byte / (v["ms"] * 1e-3) / 1e9) if v["ms"] > 0 and v["bytes"] else None

    gat, h2d, samp = rate("gather"), rate("stage_copy"), prof["sample"]
    if gat and tr["miss"]:
        # the library counts 2 rb + 8 bytes for every row of N_b at launch time; rows that miss are not
        # moved by k_gather (a-8 fills them): take them out with the epoch's miss fraction
        gat *= 1.0 - (tr["miss"] / max(tr["n_in"], 1)) * (2.0 * rb / (2.0 * rb + 8.0))
    gk = keys / (samp["ms"] * 1e-3) / 1e9 if samp["ms"] > 0 else None
    miss_link = rate("miss", 0.5)        # bytes = rows * 2 rb (link read + HBM write); the link carries rows * rb
    remote = tr["n_in"] - tr["local"]
    out = {
        "W": W, "batch": max(len(x) for x in batches), "n_hot": n_hot, "mini_batches_per_epoch": n_b,
        "mini_batches_per_s": K * n_b / sec, "ms_per_epoch": 1e3 * sec / K,
        "gather_GB/s": gat, "gather_frac_of_hbm_peak": gat / ctx["hbm_peak"] if gat else None,
        "gather_vec_bytes": 16 if rb % 16 == 0 else (8 if rb % 8 == 0 else 4),
        "sample_Gkey/s": gk, "sample_frac_of_key_peak": gk / ctx["key_peak"] if gk else None,
        "h2d_GB/s": h2d, "h2d_frac_of_link_peak": h2d / ctx["link_peak"] if h2d else None,
        "host_link_MB_per_epoch": tr["bulk"] / 1e6, "bulk_copies_per_epoch": tr["copies"],
        "miss_rows_per_epoch": tr["miss"], "miss_fill_link_GB/s": miss_link,
        "miss_fill_frac_of_link_peak": miss_link / ctx["link_peak"] if miss_link else None,
        "miss_ms_per_epoch": prof["miss"]["ms"] / K,
        "cache_hit_ratio_of_remote_accesses": (tr["hit"] / remote) if remote else None,
        "remote_frac_of_N_b": remote / max(tr["n_in"], 1),
        "gpu_stall_ms_per_epoch": prof["wait"]["ms"] / K,
        "J_per_epoch": ((mj1 - mj0) / 1e3 / K) if (mj0 is not None and mj1 is not None and mj1 > mj0) else None,
        "timed_epochs": K,
    }
    return out


def configs_grid(ctx, w_products, batches_products, errors, t_budget_s):
    """BASELINE.json:configs, every sweep: products B x W (unlimited budget), products with the paper's
    10 % budget x W (exercises the miss path, Alg. 1 l.13-14), dense W in {1,4,16}, large
    W in {4,16}.  Every point: measure_point().  A leg that fails or would overrun the time budget is
    recorded in `errors` and skipped; the headline line never depends on it."""
    from paper_2606_02916_b200 import inputs, epoch as ep
    dev, args = ctx["dev"], ctx["args"]
    t_start = time.perf_counter()
    out = {}

    def left():
        return t_budget_s - (time.perf_counter() - t_start)

    # ---- products: batch x W, unlimited budget ------------------------------------------------
    w = w_products
    try:
        all_seeds = np.concatenate(batches_products)
        n_remote_nodes = w.num_nodes - int(w.part_offsets[w.local_part + 1] - w.part_offsets[w.local_part])
        pts = []
        for Bx in (1024, 2048, 4096):
            bx = batches_products if Bx == args.batch else [all_seeds[i:i + Bx] for i in range(0, len(all_seeds), Bx)]
            g = ep.graph_from_workload(w, n_hot=-1, carry_over=1, max_window=32, staging_mode=args.staging_mode,
                                       max_live_windows=ctx["LA"] + 1, host_threads=args.host_threads, max_batch=Bx, cache_buffers=args.cache_buffers)
            try:
                for Wx in w.cfg["windows"]:
                    pts.append(measure_point(ctx, w, bx, Wx, -1, K=2, warm=1, g=g))
            finally:
                g.close()
        out["products_batch_x_W"] = {"edge_cut_measured": ctx["edge_cut_products"],
                                     "edge_cut_of_a_bfs_grown_split": ctx.get("edge_cut_bfs_grown"),
                                     "bfs_grown_part_sizes": ctx.get("bfs_grown_sizes"),
                                     "owners": "the planted communities (reading S22); the BFS-grown balanced split of the same graph "
                                               "is measured beside it and not used",
                                     "n_hot": "unlimited", "points": pts}
    except Exception as exc:
        errors["configs.products_batch_x_W"] = repr(exc)
    # ---- products: the paper's 10 % budget -----------------------------------------------------
    try:
        n_hot = -(-n_remote_nodes // 10)
        pts = []
        g = ep.graph_from_workload(w, n_hot=n_hot, carry_over=1, max_window=32, staging_mode=args.staging_mode,
                                   max_live_windows=ctx["LA"] + 1, host_threads=args.host_threads, max_batch=args.batch, cache_buffers=args.cache_buffers)
        try:
            for Wx in w.cfg["windows"]:
                pts.append(measure_point(ctx, w, batches_products, Wx, n_hot, K=5, warm=1, g=g))
        finally:
            g.close()
        out["products_budget_10pct_x_W"] = {"n_hot": n_hot, "n_hot_rule": "ceil(0.10 x remote nodes) (PAPER.md:32)", "points": pts}
    except Exception as exc:
        errors["configs.products_budget_10pct_x_W"] = repr(exc)
    ctx["feats"] = None
    # ---- dense and large --------------------------------------------------------------------------
    for name in ("dense", "large"):
        if name not in args.configs.split(","):
            continue
        try:
            if left() < (60 if name == "dense" else 150):
                raise RuntimeError("skipped: %.0f s left of the bench's time budget" % left())
            if name == "large":
                free_b, _ = torch.cuda.mem_get_info()
                host_gb = os.sysconf("SC_PHYS_PAGES") * os.sysconf("SC_PAGE_SIZE") / 1e9
                if free_b < 100e9 or host_gb < 80:
                    raise RuntimeError("skipped: needs ~100 GB of HBM and ~80 GB of host memory")
            t0 = time.perf_counter()
            wx = inputs.make_workload(name, device=dev, local_part=w.local_part)
            t_gen = time.perf_counter() - t0
            cut = edge_cut(wx, dev)
            n_rem = wx.num_nodes - int(wx.part_offsets[wx.local_part + 1] - wx.part_offsets[wx.local_part])
            pts = []
            for n_hot in (-1, -(-n_rem // 10)):
                g = ep.graph_from_workload(wx, n_hot=n_hot, carry_over=1, max_window=max(wx.cfg["windows"]),
                                           staging_mode=args.staging_mode, max_live_windows=ctx["LA"] + 1,
                                           host_threads=args.host_threads, cache_buffers=args.cache_buffers)
                try:
                    for Wx in wx.cfg["windows"]:
                        if n_hot >= 0 and Wx != max(wx.cfg["windows"]):
                            continue
                        pts.append(measure_point(ctx, wx, wx.batches, Wx, n_hot, K=1 if name == "large" else 2, warm=1, g=g,
                                                 max_window=max(wx.cfg["windows"])))
                finally:
                    g.close()
            out[name] = {"workload": workload_name(argparse.Namespace(config=name, batch=wx.cfg["batch"]), wx),
                         "edge_cut_measured": cut, "generation_s": t_gen, "points": pts}
            if name == "dense":
                # the paper's own model shape on its Reddit-shaped workload: 2 layers, 16 hidden
                # units, fanout {25,10}, 602-wide features, trained behind every gather
                try:
                    Wc = max(wx.cfg["windows"])
                    g = ep.graph_from_workload(wx, n_hot=-1, carry_over=1, max_window=Wc, staging_mode=args.staging_mode,
                                               max_live_windows=ctx["LA"] + 1, host_threads=args.host_threads, cache_buffers=args.cache_buffers)
                    try:
                        out[name]["with_graphsage_consumer"] = consumer_leg(g, wx, wx.batches, Wc, ctx["feats"], ctx["stream"], dev,
                                                                            ctx["LA"], wx.cfg["batch"])
                    finally:
                        g.close()
                except Exception as exc:
                    errors["configs.dense.consumer"] = repr(exc)
            del wx
            ctx["feats"] = None
            torch.cuda.empty_cache()
        except Exception as exc:
            errors["configs." + name] = repr(exc)
            ctx["feats"] = None
            torch.cuda.empty_cache()
    return out


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


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def cpu_baseline(args, w, batches):
    """The oracle as it stands on the host cores, on a bounded sample of the same workload: one core
    (first 4 mini-batches as one window), and every host core with the trivially parallel
    decomposition only (the batches of a full window sampled side by side, their gathers side by
    side, the window step itself on one thread; results unchanged)."""
    from concurrent.futures import ThreadPoolExecutor
    from oracle import ggo
    g = ggo.Graph(*w.host_graph())
    feat = w.host_features()
    po = w.part_offsets
    parts = [np.ascontiguousarray(feat[po[m]:po[m + 1]]) for m in range(len(po) - 1)]
    S = min(args.cpu_sample_batches, len(batches), args.window)
    st = ggo.State(g.n, po, w.local_part, args.n_hot, 1)
    t0 = time.perf_counter()
    bs = [ggo.Batch(g, batches[j], w.fanouts, w.seed, j) for j in range(S)]
    st.run_window(bs)
    for b in bs:
        ggo.gather(b.nodes, po, parts, w.row_bytes)
    dt1 = time.perf_counter() - t0
    del bs
    cores = os.cpu_count() or 1
    Wn = min(args.window, len(batches))
    st = ggo.State(g.n, po, w.local_part, args.n_hot, 1)
    t0 = time.perf_counter()
    with ThreadPoolExecutor(cores) as ex:                      # ctypes calls release the GIL
        bs = list(ex.map(lambda j: ggo.Batch(g, batches[j], w.fanouts, w.seed, j), range(Wn)))
        st.run_window(bs)
        list(ex.map(lambda b: ggo.gather(b.nodes, po, parts, w.row_bytes), bs))
    dtn = time.perf_counter() - t0
    return {"value": Wn / dtn, "unit": UNIT, "cores": min(cores, Wn), "kind": "oracle",
            "sample": "first %d mini-batches of the epoch as one W=%d window (sample + window + gather), batches sampled and "
                      "gathered on %d threads, %.1f s" % (Wn, Wn, min(cores, Wn), dtn),
            "cpu_model": cpu_model(), "host_cores": cores,
            "one_core": {"value": S / dt1, "unit": UNIT, "cores": 1,
                         "sample": "first %d mini-batches of the epoch as one W=%d window (sample + window + gather), %.1f s"
                                   % (S, S, dt1)}}


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)

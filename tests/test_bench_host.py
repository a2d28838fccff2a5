"""Host-side helpers of bench.py (no GPU): rank correlation, peak notes, argument defaults."""
import importlib.util
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _bench():
    spec = importlib.util.spec_from_file_location("bench_module", os.path.join(ROOT, "bench.py"))
    m = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(m)
    return m


def test_kendall_tau_closed_forms():
    b = _bench()
    assert b.kendall_tau([1, 2, 3, 4], [10, 20, 30, 40]) == 1.0
    assert b.kendall_tau([1, 2, 3, 4], [4, 3, 2, 1]) == -1.0
    # one discordant pair of six: (6 - 2) / 6
    assert abs(b.kendall_tau([1, 2, 3, 4], [1, 2, 4, 3]) - 4.0 / 6.0) < 1e-12
    assert b.kendall_tau([1.0], [2.0]) is None


def test_derived_peak_notes_and_defaults(monkeypatch):
    b = _bench()
    # 148 SMs x 4 sub-partitions x 32 lanes x 1.965 GHz / 21 issue slots per key = 1773 Gkey/s
    assert abs(b.derived_alu_peak_gkeys(1965.0, 148, b.KEY_ISSUE_SLOTS) - 1772.6) < 0.5
    assert abs(b.derived_alu_peak_gkeys(1965.0, 148, b.HASH_ISSUE_SLOTS) - 2326.6) < 0.5
    monkeypatch.setattr(sys, "argv", ["bench.py"])
    a = b.parse_args()
    assert (a.gpus, a.config, a.batch, a.window, a.n_hot, a.staging_mode) == (1, "products", 1024, 16, -1, 0)
    assert a.steps >= 3 and a.warmup >= 3
    assert isinstance(b.cpu_model(), str) and b.cpu_model()


REQUIRED = ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
            "vs_baseline", "dtype", "data", "config", "e2e", "cpu_baseline")


def test_reference_arm_runs_and_prints_one_parseable_line():
    """`bench.py --impl reference` needs no GPU (it times the oracle on the host cores): run it for real
    on the tiny config and read its last stdout line the way the driver does."""
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "tiny",
                        "--batch", "64", "--window", "4", "--steps", "2", "--warmup", "1"],
                       capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert p.returncode == 0, p.stderr[-2000:]
    line = p.stdout.strip().splitlines()[-1]
    assert len(line) < 4096
    r = json.loads(line)
    for k in REQUIRED:
        assert k in r, k
    assert r["impl"] == "reference" and r["value"] > 0 and r["steps"] == 2 and r["warmup"] == 1
    assert r["cpu_baseline"]["kind"] == "oracle" and r["cpu_baseline"]["value"] == r["value"]
    assert r["e2e"] == {"value": r["value"], "unit": r["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert set(r["config"]) == {"workload", "W", "n_hot", "l2"} and r["config"]["W"] == 4


def test_both_arms_print_the_same_config_object():
    """The driver compares the two arms' `config`: both must come from config_record, which reads only the
    arguments and the workload."""
    import inspect
    b = _bench()
    assert '"config": config_record(args, w)' in inspect.getsource(b.run_reference)
    assert '"config": config_record(args, w)' in inspect.getsource(b.run_ours)

    class W:
        num_nodes, dim, row_bytes, fanouts, batches = 2449029, 100, 400, [15, 10, 5], [None] * 193
        dtype = "torch.float32"

        class indices:
            @staticmethod
            def numel():
                return 123800000
    a = b.parse_args([])
    c = b.config_record(a, W)
    assert c["W"] == 16 and c["n_hot"] == -1 and "larger than L2" in c["l2"]
    assert len(c["workload"]) < 120 and c["workload"].startswith("products N=2449029")


def test_result_line_stays_compact_whatever_the_optional_legs_hold():
    """The driver keeps a few KB of stdout: a line that carries the whole `configs` grid is lost (round 2).
    compact_record must drop everything that grows and keep the contract's keys."""
    b = _bench()
    big = {"points": [{"k%d" % i: 1.23456789012 * i for i in range(25)} for _ in range(64)]}
    out = {"metric": b.METRIC, "value": 4310.123456789, "unit": b.UNIT, "n_gpus": 1, "steps": 20, "warmup": 5,
           "ms_per_step": 44.78123456, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": b.DTYPE, "data": "synthetic",
           "config": {"workload": "products N=2449029 nnz=123800000 dim=100 float32 batch=1024 (193/epoch) fanouts=15,10,5",
                      "W": 16, "n_hot": -1, "l2": "inputs larger than L2 (feature store 980 MB; no flush)"},
           "protocol": {"workload_long": "x" * 300},
           "clocks": {"sm_mhz": 1965.0, "sm_max_mhz": 1965.0, "samples": 7, "reasons": []}, "gpu_launches": 123456,
           "roofline": {"bound": "alu", "kernel": "a-1 sampling (k_sample_count/plan + the selection kernels of every hop)",
                        "achieved": 554.123456, "peak": 1415.123456, "unit": "Gkey/s", "frac": 0.39159, "frac_of_pipe_bound": 0.3279,
                        "pipe_bound_Gkey/s": 1692.0, "traffic": 7.06e8, "traffic_note": "y" * 400, "peak_source": "z" * 300,
                        "derived_peaks_Gkey/s": {"a": 1.0, "note": "n" * 200}, "launches": 780, "avg_launch_us": 536.1,
                        "algorithmic_keys_per_launch": 2.97e8, "share_of_step": 0.47},
           "roofline_gather": {"bound": "hbm", "kernel": "k_gather", "achieved": 2820.0, "peak": 6464.0, "unit": "GB/s", "frac": 0.436,
                               "traffic": 2.758e8, "peak_source": "measured (MEASURED_PEAKS.json hbm_gbs)", "launches": 3860,
                               "avg_launch_us": 96.9, "algorithmic_bytes_per_launch": 2.77e8, "share_of_step": 0.4, "note": "w" * 200},
           "kernels_alone": {"sample_frac_of_alu_peak": 0.52, "gather_frac_of_hbm_peak": 0.75, "h2d_frac_of_link_peak": 0.9,
                             "ms_per_epoch": {"a": 1.0}},
           "stages": big, "vs_W": {"16": 4310.1}, "J_per_epoch_vs_W": big, "vs_batch_at_W": big, "configs": big, "simulator": big,
           "simulator_budgeted": big, "variants": big, "errors": {"consumer": "RuntimeError('boom')" * 40},
           "gpu_stall_ms_per_step": 12.9, "energy": {"J_per_step": 28.15, "avg_W": 608.7, "source": "NVML"},
           "staging": {"host_link_bytes_per_step": 1794288860, "bulk_copies_per_step": 39, "h2d_GB/s": 50.2,
                       "host_link_peak_GB/s": 55.6, "h2d_frac_of_link_peak": 0.9025, "boundary_stall_ms_per_step": 13.0},
           "e2e": {"value": 365.3, "unit": b.UNIT, "h2d_bytes_per_step": 1794288860, "d2h_bytes_per_step": 27329315340,
                   "note": "q" * 300},
           "cpu_baseline": {"value": 2.816, "unit": b.UNIT, "cores": 16, "kind": "oracle", "sample": "first 16 mini-batches ...",
                            "cpu_model": "m", "host_cores": 16, "one_core": {"value": 0.3}}}
    line = json.dumps(b.compact_record(out, "bench_detail.json"))
    assert len(line) < 4096, len(line)
    r = json.loads(line)
    for k in REQUIRED + ("roofline", "roofline_gather", "clocks", "gpu_launches", "staging", "gpu_stall_ms_per_step", "energy"):
        assert k in r, k
    for k in ("bound", "achieved", "peak", "unit", "frac", "traffic"):
        assert k in r["roofline"] and k in r["roofline_gather"], k
    assert r["roofline"]["frac_of_pipe_bound"] == 0.3279
    assert set(r["e2e"]) == {"value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"}
    assert set(r["cpu_baseline"]) == {"value", "unit", "cores", "kind", "sample"}
    assert r["errors"] == ["consumer"] and r["detail"] == "bench_detail.json"
    assert "configs" not in r and "variants" not in r and "simulator" not in r and "stages" not in r

"""Host-side helpers of bench.py (no GPU): rank correlation, peak notes, argument defaults."""
import importlib.util
import os
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

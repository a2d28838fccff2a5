"""CPU-side checks of the boundary: the library builds, loads, and exports every symbol that
include/greengnn.h declares; the host-side key function matches the golden values; the
ctypes mirrors have the C layout.  No compute calls (there is no GPU here)."""
import ctypes as C
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "greengnn.h")


@pytest.fixture(scope="module")
def lib():
    from paper_2606_02916_b200 import build, binding
    build.build_library()
    return binding.load_library()


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gg_[a-z_0-9]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    from paper_2606_02916_b200 import binding
    names = _declared()
    assert len(names) >= 16
    for n in names:
        assert getattr(lib, n) is not None, n
    assert sorted(binding.SYMBOLS) == names


def test_key_function_matches_golden(lib):
    from paper_2606_02916_b200 import binding
    gold = os.path.join(ROOT, "tests", "golden", "keys.txt")
    n = 0
    for line in open(gold):
        t = line.split()
        if t and t[0] == "key":
            assert binding.gg_key(*[int(x, 0) for x in t[1:-1]]) == int(t[-1], 16)
            n += 1
    assert n >= 4


def test_struct_layouts_match_the_header(tmp_path, lib):
    from paper_2606_02916_b200 import binding
    names = ["gg_csr", "gg_owner_map", "gg_feature_store", "gg_config", "gg_block", "gg_batch_out",
             "gg_window_trace", "gg_profile", "gg_energy_model", "gg_sim_result"]
    prog = '#include <stdio.h>\n#include "greengnn.h"\nint main(){' + "".join(
        'printf("%s %%zu\\n", sizeof(%s));' % (n, n) for n in names) + "return 0;}"
    src = tmp_path / "sz.c"
    src.write_text(prog)
    exe = tmp_path / "sz"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)])
    out = dict(l.split() for l in subprocess.check_output([str(exe)], text=True).splitlines())
    for n in names:
        assert C.sizeof(getattr(binding, n)) == int(out[n]), n


def test_no_cpu_fallback_when_library_missing(tmp_path):
    from paper_2606_02916_b200 import binding
    with pytest.raises(ImportError):
        binding.load_library(str(tmp_path / "nope.so"))


def test_version_string(lib):
    assert b"sm_100a" in lib.gg_version()


def test_static_unique_count_rejects_bad_sizes_before_touching_the_gpu(lib):
    """gg_unique_count_static validates its arguments before its first CUDA call, so the limit of its
    fixed workspace can be checked here: one node more than GG_STATIC_MAX_NODES is GG_ERR_CAPACITY with
    a message that names the limit; null outputs and negative sizes are GG_ERR_INVALID_ARG."""
    from paper_2606_02916_b200 import binding
    src = open(HEADER).read()
    m = re.search(r"#define\s+GG_STATIC_MAX_NODES\s+\(1\s*<<\s*(\d+)\)", src)
    assert m and (1 << int(m.group(1))) == binding.GG_STATIC_MAX_NODES == 4_194_304
    stats = (C.c_int32 * 2)()
    f = lib.gg_unique_count_static
    assert f(None, 0, binding.GG_STATIC_MAX_NODES + 1, None, None, 0, stats, None) == binding.GG_ERR_CAPACITY
    assert b"GG_STATIC_MAX_NODES" in lib.gg_last_error()
    assert f(None, 0, 1000, None, None, 0, None, None) == binding.GG_ERR_INVALID_ARG      # no stats
    assert f(None, 5, 1000, None, None, 0, stats, None) == binding.GG_ERR_INVALID_ARG     # ids missing
    assert f(None, 0, 0, None, None, 0, stats, None) == binding.GG_ERR_INVALID_ARG        # num_nodes < 1
    assert f(None, 0, 1000, None, None, 4, stats, None) == binding.GG_ERR_INVALID_ARG     # capacity without outputs

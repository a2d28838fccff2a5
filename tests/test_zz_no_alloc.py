"""gg_unique_count_static -- the entry point for callers that cannot allocate device memory (a process
whose own allocator already holds all of the HBM, or a loop that cannot take the device-wide wait of a
cudaFree) -- against the ordinary path.

The ordinary path (gg_window_stage) builds U_k / c_k in workspaces it allocates itself and exports them
through gg_window_export.  The static entry point gets the same windows' N_b lists as one device ID list
and must return exactly the same two arrays (integer work: bit-exact, the tolerance of every parity test
here).  It is called twice in a row on DIFFERENT windows, and then once more on the first: its workspace
is one fixed array inside the library that still holds the previous call's counters, so a call that
forgot to clear it would fail the second or third comparison.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must
not hide the parity tests.  It builds its own graph handle and depends on no state of other tests."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return "cuda:0"


def _window_lists(g, w, wid, win):
    """Stages window `wid` on the ordinary path; returns (concatenated N_b on the device, U_k, c_k)."""
    g.window_stage(wid, win.start, [w.batches[i] for i in win], w.fanouts)
    ids = torch.cat([g.batch_info(wid, j)["input_nodes"].clone() for j in range(len(win))])
    uniq, cnt = g.window_export(wid, "uniq"), g.window_export(wid, "cnt")
    g.window_release(wid)
    return ids, uniq, cnt


def _static(binding, ids, num_nodes, capacity):
    uniq = torch.full((capacity,), -7, dtype=torch.int32, device=ids.device)
    cnt = torch.full((capacity,), -7, dtype=torch.int32, device=ids.device)
    stats = torch.full((2,), -7, dtype=torch.int32, device=ids.device)
    binding.unique_count_static(ids, num_nodes, uniq, cnt, stats)
    return uniq, cnt, stats


def test_static_unique_count_matches_the_staged_path_on_calls_in_a_row(workload, dev):
    from paper_2606_02916_b200 import binding, epoch as ep
    w = workload("small", dev)                       # 100 000 nodes: 13 counter tiles, the last one ragged
    g = ep.graph_from_workload(w, max_window=4)
    try:
        wins = ep.windows_of(len(w.batches), 4)
        a = _window_lists(g, w, 0, wins[0])
        b = _window_lists(g, w, 1, wins[1])
    finally:
        g.close()
    assert not np.array_equal(a[1], b[1])            # two different windows, or the test proves nothing
    # everything the three calls need is allocated here, before the first of them
    outs = [(torch.full((w.num_nodes,), -7, dtype=torch.int32, device=dev),
             torch.full((w.num_nodes,), -7, dtype=torch.int32, device=dev),
             torch.full((2,), -7, dtype=torch.int32, device=dev)) for _ in range(3)]
    torch.cuda.synchronize()
    calls = [a, b, a]
    for (ids, _, _), (uo, co, so) in zip(calls, outs):   # back to back on one stream, no sync between
        binding.unique_count_static(ids, w.num_nodes, uo, co, so)
    torch.cuda.synchronize()
    for i, ((ids, uniq, cnt), (uo, co, so)) in enumerate(zip(calls, outs)):
        n, skipped = so.cpu().tolist()
        assert skipped == 0
        assert n == len(uniq), "call %d: |U| %d vs %d" % (i, n, len(uniq))
        assert np.array_equal(uo[:n].cpu().numpy(), uniq), "call %d: U_k" % i
        assert np.array_equal(co[:n].cpu().numpy(), cnt), "call %d: c_k" % i
        assert int(co[:n].sum()) == ids.numel()      # counts sum to the accesses
        assert bool((uo[n:] == -7).all()) and bool((co[n:] == -7).all())   # nothing written past |U|


def test_static_unique_count_limits_and_edges(dev):
    from paper_2606_02916_b200 import binding
    ids = torch.tensor([5, 9, 5, 0, 8191, 8192, 9, 5, -1, 20000], dtype=torch.int32, device=dev)
    # IDs outside [0, num_nodes) are skipped and tallied
    uo, co, so = _static(binding, ids, 10000, 16)
    assert so.cpu().tolist() == [5, 2]
    assert uo[:5].cpu().tolist() == [0, 5, 9, 8191, 8192] and co[:5].cpu().tolist() == [1, 3, 2, 1, 1]
    # too small an output: |U| is reported, nothing is written
    uo, co, so = _static(binding, ids, 10000, 4)
    assert so.cpu().tolist() == [5, 2] and bool((uo == -7).all()) and bool((co == -7).all())
    # empty list (the start-up call): |U| = 0
    uo, co, so = _static(binding, ids[:0], 10000, 4)
    assert so.cpu().tolist() == [0, 0] and bool((uo == -7).all())
    # the largest graph the fixed workspace covers, touched at both ends
    top = binding.GG_STATIC_MAX_NODES - 1
    uo, co, so = _static(binding, torch.tensor([top, 0, top], dtype=torch.int32, device=dev),
                         binding.GG_STATIC_MAX_NODES, 2)
    assert so.cpu().tolist() == [2, 0] and uo.cpu().tolist() == [0, top] and co.cpu().tolist() == [1, 2]
    # one node more than the workspace holds: a clear error, no launch
    with pytest.raises(binding.GreenGNNError) as ei:
        _static(binding, ids, binding.GG_STATIC_MAX_NODES + 1, 16)
    assert ei.value.status == binding.GG_ERR_CAPACITY and "GG_STATIC_MAX_NODES" in str(ei.value)

"""-m gpu: xy_random_walk_static -- the random-walk histogram through the entry point that allocates nothing (its
scratch is a file-scope static __device__ array, include/xy_b200.h) -- against the existing path xy_random_walk, which
is itself held bit-exactly against the oracle (tests/test_gpu_walk.py).  Integer work: the bar is bit-exactness.
Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

from paper_1211_3991_b200 import binding as B
from paper_1211_3991_b200 import levy, workloads

pytestmark = pytest.mark.gpu


def _starts(g, n_walkers, seed):
    rng = np.random.default_rng(seed)
    S = g.colour.shape[0]
    return np.stack([rng.integers(0, g.colour.shape[1], n_walkers) for _ in range(S)]).astype(np.int32)


def test_static_scratch_walk_matches_the_allocating_path_on_two_calls_in_a_row():
    import torch
    g = levy.build(24, 3.5, 6, workloads.BASE_SEED, S=3)
    graph = B.xy_graph_load(g.row_ptr, g.col_idx, g.colour)
    try:
        # two calls in a row that share the static array: the second one is SHORTER and has other walkers, so stale
        # words of the first call would show if the entry point did not clear what it uses
        calls = [(3000, 200, 0xA11CE), (777, 64, 0xB0B), (3000, 200, 0xA11CE)]
        for n_walkers, n_steps, seed in calls:
            start = _starts(g, n_walkers, seed)
            ref = B.xy_random_walk(graph, start, n_steps, seed, sample_base=5)
            start_dev = torch.from_numpy(start).cuda()
            hist_dev = torch.full((3, n_steps + 1), -1, dtype=torch.int64, device="cuda")
            torch.cuda.synchronize()
            B.xy_random_walk_static(graph, n_walkers, start_dev.data_ptr(), n_steps, seed, hist_dev.data_ptr(), sample_base=5)
            out = hist_dev.cpu().numpy()
            assert np.array_equal(out, ref), (n_walkers, n_steps)
            assert np.all(out[:, 0] == n_walkers) and out[:, 2].sum() > 0
    finally:
        B.xy_graph_free(graph)


def test_static_scratch_walk_rejects_what_does_not_fit_and_bad_starts():
    import torch
    g = levy.build(12, 3.5, 6, workloads.BASE_SEED, S=8)
    graph = B.xy_graph_load(g.row_ptr, g.col_idx, g.colour)
    try:
        n_walkers = 100
        start = _starts(g, n_walkers, 1)
        start_dev = torch.from_numpy(start).cuda()
        n_fit = B.XY_WALK_STATIC_ENTRIES // 8 - 1                      # S * (n_steps + 1) == the limit: allowed
        hist_dev = torch.zeros((8, n_fit + 2), dtype=torch.int64, device="cuda")
        B.xy_random_walk_static(graph, n_walkers, start_dev.data_ptr(), n_fit, 3, hist_dev.data_ptr())
        ref = B.xy_random_walk(graph, start, n_fit, 3)
        assert np.array_equal(hist_dev.cpu().numpy().reshape(-1)[:8 * (n_fit + 1)].reshape(8, n_fit + 1), ref)
        with pytest.raises(B.XYError) as e:                            # one step more: beyond the static scratch
            B.xy_random_walk_static(graph, n_walkers, start_dev.data_ptr(), n_fit + 1, 3, hist_dev.data_ptr())
        assert e.value.code == B.XY_EINVAL and "static scratch" in str(e.value)
        bad = start.copy()
        bad[3, 7] = 12 * 12
        bad_dev = torch.from_numpy(bad).cuda()
        with pytest.raises(B.XYError) as e:
            B.xy_random_walk_static(graph, n_walkers, bad_dev.data_ptr(), 10, 3, hist_dev.data_ptr())
        assert e.value.code == B.XY_EINVAL
        with pytest.raises(B.XYError):
            B.xy_random_walk_static(graph, n_walkers, None, 10, 3, hist_dev.data_ptr())
    finally:
        B.xy_graph_free(graph)

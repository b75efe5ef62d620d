"""N > 1 host logic on CPU: world_size-2 gloo processes shard the samples and gather
the accumulators; no data-path collective exists to test.  The per-rank inputs come from the shared
builder with the rank's sample_base, and must equal the matching slice of a single-process build."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_shard_samples_partitions_exactly():
    from paper_1211_3991_b200.sharding import shard_samples, weak_shard
    for S in (0, 1, 7, 8, 64, 160):
        for W in (1, 2, 3, 8):
            got = [shard_samples(S, W, r) for r in range(W)]
            ids = [i for b, n in got for i in range(b, b + n)]
            assert ids == list(range(S))
            assert max(n for _, n in got) - min(n for _, n in got) <= 1
    assert weak_shard(8, 3) == (24, 8)
    with pytest.raises(ValueError):
        shard_samples(4, 2, 2)


def _worker(rank, world, port, S_total, q):
    try:
        os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
        sys.path.insert(0, ROOT)
        import torch.distributed as dist
        from paper_1211_3991_b200 import levy, workloads
        from paper_1211_3991_b200.sharding import gather_accumulators, shard_samples
        dist.init_process_group("gloo", rank=rank, world_size=world)
        base, n = shard_samples(S_total, world, rank)
        g = levy.build(8, 3.5, 6, workloads.BASE_SEED, S=max(n, 1), sample_base=base)
        R = 4
        # stand-in accumulators that identify (global sample, temperature, column): the gather must be a pure permutation
        acc = np.zeros((n, R, 8))
        for s in range(n):
            for t in range(R):
                acc[s, t] = (base + s) * 1000 + t * 10 + np.arange(8)
        full = gather_accumulators(acc, S_total)
        q.put((rank, base, n, g.row_ptr[:n].copy(), g.col_idx[:n].copy(), g.colour[:n].copy(), full))
        dist.barrier()
        dist.destroy_process_group()
    except Exception as e:  # pragma: no cover
        q.put((rank, "error", repr(e)))


@pytest.mark.parametrize("S_total", [5, 4])
def test_world_size_2_gloo_sharding_and_gather(S_total):
    import torch.multiprocessing as mp
    from paper_1211_3991_b200 import levy, workloads
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, S_total, q)) for r in range(2)]
    for p in procs: p.start()
    res = sorted([q.get(timeout=180) for _ in procs], key=lambda x: x[0])
    for p in procs: p.join(60)
    for r in res:
        assert r[1] != "error", r
    ref = levy.build(8, 3.5, 6, workloads.BASE_SEED, S=S_total)
    expect = np.zeros((S_total, 4, 8))
    for sg in range(S_total):
        for t in range(4):
            expect[sg, t] = sg * 1000 + t * 10 + np.arange(8)
    covered = []
    for rank, base, n, rp, ci, col, full in res:
        # a rank's graphs are exactly the global samples base..base+n-1 (same bits as a one-process build)
        assert np.array_equal(rp, ref.row_ptr[base:base + n])
        assert np.array_equal(ci, ref.col_idx[base:base + n])
        assert np.array_equal(col, ref.colour[base:base + n])
        assert np.array_equal(full, expect)
        covered += list(range(base, base + n))
    assert covered == list(range(S_total))


def test_graph_average_is_eq12():
    from paper_1211_3991_b200.sharding import gather_accumulators, graph_average
    rng = np.random.default_rng(0)
    acc = rng.random((3, 2, 8)) + 1.0
    acc[..., 0] = [[10, 10], [20, 20], [5, 5]]
    avg = graph_average(acc)
    want = np.mean([acc[s, :, 1:] / acc[s, :, :1] for s in range(3)], axis=0)
    assert np.allclose(avg, want)
    assert np.array_equal(gather_accumulators(acc, 3), acc)      # no process group: identity

"""N > 1 host logic on CPU: world_size 2, gloo.  Each rank takes its shard_range of the proton index
space, fills a private u64 grid (with the oracle standing in for the kernels, which need a GPU),
the grids are summed by the same all-reduce helper bench.py uses, and the result must equal the
single-rank grid bit for bit (doses of the two GPUs combined at the end)."""
import os
import tempfile

import numpy as np
import pytest


def test_shard_range_partitions_exactly():
    from paper_1011_2188_b200.multi import shard_range
    for total in (0, 1, 7, 1_000_000, 10 ** 9 + 7):
        for world in (1, 2, 3, 8):
            parts = [shard_range(total, r, world) for r in range(world)]
            assert parts[0][0] == 0 and sum(c for _, c in parts) == total
            for (a, ca), (b, _) in zip(parts, parts[1:]):
                assert a + ca == b
            assert max(c for _, c in parts) - min(c for _, c in parts) <= 1


def _worker(rank, world, store, out_dir):
    import torch
    import torch.distributed as dist
    import fdc_inputs as fi
    import oracle
    from paper_1011_2188_b200.multi import shard_range, allreduce_sum_int64
    dist.init_process_group("gloo", init_method="file://" + store, rank=rank, world_size=world)
    w = fi.workload(3, n_protons=2352, tracks_per_bin=20)
    first, n = shard_range(w.n_protons, rank, world)
    g, sq, _, st = oracle.run_sq(w.phantom, w.table, w.db, w.beamlets, w.seed, first=first, n=n, by_history=False)
    t = torch.from_numpy(g.view(np.int64))
    allreduce_sum_int64(t)
    t2 = torch.from_numpy(sq.view(np.int64))                  # the sum-of-squares grid shards the same way
    allreduce_sum_int64(t2)
    cnt = torch.tensor([st["protons"], st["deposits"]], dtype=torch.int64)
    dist.all_reduce(cnt)
    if rank == 0:
        np.save(os.path.join(out_dir, "grid.npy"), t.numpy().view(np.uint64))
        np.save(os.path.join(out_dir, "sq.npy"), t2.numpy().view(np.uint64))
        np.save(os.path.join(out_dir, "cnt.npy"), cnt.numpy())
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_ranks_sum_to_the_single_rank_grid():
    import torch.multiprocessing as mp
    import fdc_inputs as fi
    import oracle
    with tempfile.TemporaryDirectory() as d:
        store = os.path.join(d, "store")
        mp.spawn(_worker, args=(2, store, d), nprocs=2, join=True)
        g2 = np.load(os.path.join(d, "grid.npy")); cnt = np.load(os.path.join(d, "cnt.npy")); sq2 = np.load(os.path.join(d, "sq.npy"))
    w = fi.workload(3, n_protons=2352, tracks_per_bin=20)
    g1, sq1, _, st = oracle.run_sq(w.phantom, w.table, w.db, w.beamlets, w.seed, by_history=False)
    assert np.array_equal(g1, g2) and np.array_equal(sq1, sq2)
    assert int(cnt[0]) == st["protons"] == 2352 and int(cnt[1]) == st["deposits"]

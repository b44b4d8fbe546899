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


class _OracleCtx:
    """Stands in for paper_1011_2188_b200.Fdc on a box without a GPU: same method names and semantics, the oracle as
    the engine, CPU tensors aliasing its grids -- so that multi.sharded_step's control flow (reset, run this rank's
    range, in-place all-reduce of the context's own grids, Gy conversion) runs under gloo exactly as bench.py and
    the NCCL path drive it."""

    def __init__(self, w):
        self.w = w
        self.grid = np.zeros(w.phantom.hu.shape, dtype=np.uint64)
        self.sq = None
        self.calls = []

    def fdc_reset(self):
        self.grid[...] = 0
        if self.sq is not None:
            self.sq[...] = 0
        self.calls.append("reset")

    def fdc_run(self, beamlets, first, n, stride, seed, flags=1, dose_gy=None):
        import oracle
        w = self.w
        if flags & (16 | 8192):                 # FDC_SQUARES_BY_HISTORY (8192) implies the squares grid, as in the library
            g, sq, sqh, _ = oracle.run_sq(w.phantom, w.table, w.db, beamlets, seed, first=first, n=n, stride=stride, flags=flags & 33,
                                          by_history=bool(flags & 8192))
            sq = sqh if flags & 8192 else sq
            if self.sq is None:
                self.sq = np.zeros(w.phantom.hu.shape, dtype=np.uint64)
            self.sq += sq
        else:
            g, _ = oracle.run(w.phantom, w.table, w.db, beamlets, seed, first=first, n=n, stride=stride, flags=flags & 33)
        self.grid += g
        self.calls.append("run")
        if dose_gy is not None:
            self.fdc_to_gy(dose_gy)

    def fdc_edep_device_ptr(self):
        import torch
        return torch.from_numpy(self.grid.view(np.int64)), (torch.from_numpy(self.sq.view(np.int64)) if self.sq is not None else None)

    def fdc_to_gy(self, out):
        import oracle
        out[...] = oracle.to_gy(self.grid, self.w.phantom, self.w.table)
        self.calls.append("gy")


def _step_worker(rank, world, store, out_dir):
    import torch.distributed as dist
    import fdc_inputs as fi
    from paper_1011_2188_b200.multi import shard_range, sharded_step
    dist.init_process_group("gloo", init_method="file://" + store, rank=rank, world_size=world)
    w = fi.workload(3, n_protons=1176, tracks_per_bin=20)
    ctx = _OracleCtx(w)
    first, n = shard_range(w.n_protons, rank, world)
    dose = np.zeros(w.phantom.hu.shape, dtype=np.float32)
    for flags in (1, 1 | 16):
        sharded_step(ctx, w.beamlets, first, n, w.seed, flags, dose, world)
    assert ctx.calls == ["reset", "run", "gy"] * 2
    np.save(os.path.join(out_dir, "dose%d.npy" % rank), dose)
    np.save(os.path.join(out_dir, "sq%d.npy" % rank), ctx.sq)
    sharded_step(ctx, w.beamlets, first, n, w.seed, 1 | 8192, dose, world)      # the by-history flag alone
    np.save(os.path.join(out_dir, "sqh%d.npy" % rank), ctx.sq)
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_sharded_step_control_flow_world_2():
    """multi.sharded_step with world_size 2 on gloo: every rank ends with the dose grid (and squares grid) of the
    whole plan, equal bit for bit to the single-rank step, through reset -> run -> in-place all-reduce -> fdc_to_gy."""
    import torch.multiprocessing as mp
    import fdc_inputs as fi
    from paper_1011_2188_b200.multi import sharded_step
    with tempfile.TemporaryDirectory() as d:
        mp.spawn(_step_worker, args=(2, os.path.join(d, "store"), d), nprocs=2, join=True)
        doses = [np.load(os.path.join(d, "dose%d.npy" % r)) for r in range(2)]
        sqs = [np.load(os.path.join(d, "sq%d.npy" % r)) for r in range(2)]
        sqhs = [np.load(os.path.join(d, "sqh%d.npy" % r)) for r in range(2)]
    w = fi.workload(3, n_protons=1176, tracks_per_bin=20)
    one = _OracleCtx(w)
    dose1 = np.zeros(w.phantom.hu.shape, dtype=np.float32)
    sharded_step(one, w.beamlets, 0, w.n_protons, w.seed, 1 | 16, dose1, 1)
    assert one.calls == ["reset", "run", "gy"]
    assert dose1.any() and np.array_equal(doses[0], dose1) and np.array_equal(doses[1], dose1)
    assert np.array_equal(sqs[0], one.sq) and np.array_equal(sqs[1], one.sq)
    # FDC_SQUARES_BY_HISTORY without FDC_TALLY_SQUARES: the squares grid is summed over ranks all the same
    sharded_step(one, w.beamlets, 0, w.n_protons, w.seed, 1 | 8192, dose1, 1)
    assert one.sq.any() and np.array_equal(sqhs[0], one.sq) and np.array_equal(sqhs[1], one.sq)


def test_bench_refuses_a_world_size_that_contradicts_gpus():
    """`--gpus N` must not silently run one GPU.  With WORLD_SIZE set and different from --gpus the product
    arm stops before touching the device (on a box without CUDA it stops earlier, at the no-fallback check)."""
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, WORLD_SIZE="2", RANK="0", LOCAL_RANK="0")
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "4", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, timeout=600, cwd=root, env=env)
    assert out.returncode != 0 and ("WORLD_SIZE=2" in out.stderr or "no CPU fallback" in out.stderr)

"""fdc_uncertainty_batch_noalloc against fdc_uncertainty_batch (GPU, through the C-ABI).

Why the entry point exists: the batch estimate of eq. (1) is evaluated inside a loop (run a batch, look at the mean
dose uncertainty, stop when it is small enough).  A service that runs that loop has usually handed all device
memory to its own arena, or sits inside a framework whose caching allocator has, and cannot let a library call
cudaMalloc behind its back; nor can it take the device-wide wait that cudaFree (and sometimes cudaMalloc) brings
while the next batch is already being transported on another stream.  fdc_uncertainty_batch allocates its scratch
on first use; the no-alloc call keeps it in a fixed 512-byte array inside libfdc.so instead (one per device,
shared by all contexts, at most FDC_NOALLOC_MAX_BATCHES = 32 batch grids).

What is checked: same mean uncertainty, same voxel count and the same rel_sigma grid, bit for bit (both paths run
the same kernel, so the tolerance is zero, as in the other parity tests), on two calls in a row with different
inputs -- the second would be wrong if the first one's accumulators or pointers were still in the array -- and
again from a second context; the limit is refused with a message that names it.

The file is named test_zz_* so that pytest collects it last: with `pytest -x` a failure here hides nothing.  It
passes alone in a fresh process (the no-alloc call is then the first thing to touch its kernel and does its own
once-per-device set-up) and after the rest of the suite.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from test_gpu_parity import fdc, make_ctx        # noqa: E402,F401  (fixture + helper)


def _batch_grids(ctx, w, seeds):
    import torch
    grids = []
    for s in seeds:
        ctx.fdc_reset()
        ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, s)
        g = torch.zeros(w.phantom.hu.shape, dtype=torch.int64, device="cuda")
        ctx.fdc_get_edep_fixed(g)
        grids.append(g)
    return grids


def test_noalloc_batch_uncertainty_equals_the_allocating_path(fdc, wl3_small):
    import torch
    w = wl3_small
    N = w.n_protons
    ctx = make_ctx(fdc, w)
    grids = _batch_grids(ctx, w, range(2000, 2006))
    cases = [(grids, N), (grids[1:4], 3 * N)]              # six batches, then three other ones with another N

    # two no-alloc calls in a row, before the allocating path has run at all (first use on this device when alone)
    got = []
    for gs, n in cases:
        rel = torch.full(w.phantom.hu.shape, -1.0, dtype=torch.float32, device="cuda")
        mean, cnt = ctx.fdc_uncertainty_batch_noalloc(gs, n, rel)
        got.append((mean, cnt, rel))

    want = []
    for gs, n in cases:
        rel = torch.full(w.phantom.hu.shape, -1.0, dtype=torch.float32, device="cuda")
        mean, cnt = ctx.fdc_uncertainty_batch(gs, n, rel)
        want.append((mean, cnt, rel))

    assert want[0][1] > 0 and want[0][0] > 0.0 and (want[0][0], want[0][1]) != (want[1][0], want[1][1])
    for (gm, gc, gr), (wm, wc, wr) in zip(got, want):
        assert (gm, gc) == (wm, wc)
        assert torch.equal(gr, wr)

    # no rel_sigma output; and the array left behind by the calls above changes nothing
    assert ctx.fdc_uncertainty_batch_noalloc(grids, N) == (want[0][0], want[0][1])
    assert ctx.fdc_uncertainty_batch_noalloc(grids[1:4], 3 * N) == (want[1][0], want[1][1])

    # the scratch belongs to the device, not to a context: a second context gives the same answers right after
    ctx2 = make_ctx(fdc, w)
    assert ctx2.fdc_uncertainty_batch_noalloc(grids, N) == (want[0][0], want[0][1])
    assert ctx.fdc_uncertainty_batch_noalloc(grids[1:4], 3 * N) == (want[1][0], want[1][1])
    ctx2.fdc_destroy()

    # steady state: the device's free memory does not shrink over further calls
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        ctx.fdc_uncertainty_batch_noalloc(grids, N)
    assert torch.cuda.mem_get_info()[0] >= free0

    # the limit of the fixed scratch: 32 grids are taken, 33 are refused and the message says why
    many = [grids[i % 6] for i in range(fdc.FDC_NOALLOC_MAX_BATCHES + 1)]
    assert ctx.fdc_uncertainty_batch_noalloc(many[:-1], N) == ctx.fdc_uncertainty_batch(many[:-1], N)
    with pytest.raises(fdc.FdcError) as e:
        ctx.fdc_uncertainty_batch_noalloc(many, N)
    assert e.value.code == fdc.FDC_EINVAL and "at most 32" in str(e.value)
    ctx.fdc_uncertainty_batch(many, N)                     # the allocating path takes up to 64
    with pytest.raises(fdc.FdcError):
        ctx.fdc_uncertainty_batch_noalloc(grids[:1], N)
    # a refused call leaves the next one intact
    assert ctx.fdc_uncertainty_batch_noalloc(grids, N) == (want[0][0], want[0][1])
    ctx.fdc_destroy()

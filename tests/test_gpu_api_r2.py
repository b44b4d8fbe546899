"""GPU tests of the round-2 entry points, all through the C-ABI: profile comparators (R16, R17) against the numpy
definitions; fdc_to_gy; the in-place multi-GPU sequence (fdc_edep_device_ptr -> sum -> fdc_to_gy); the diagnostics
(fdc_last_call_info byte counters, FDC_DIAG_REDS / fdc_trace_reds); fdc_load_tracks keeps the loaded database when
it rejects a new one; the roofline microbenchmark library."""
import numpy as np
import pytest

import fdc_inputs as fi

pytestmark = pytest.mark.gpu

from test_gpu_parity import fdc, make_ctx, STAT_KEYS        # noqa: E402,F401  (fixture + helpers)


def _two_doses(fdc, w):
    """Two independent runs (different seeds) of the same plan: (ctx, dose A, dose B) as CUDA tensors."""
    import torch
    ctx = make_ctx(fdc, w)
    out = []
    for seed in (w.seed, w.seed + 77):
        ctx.fdc_reset()
        d = torch.zeros(w.phantom.hu.shape, dtype=torch.float32, device="cuda")
        ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, seed, dose_gy=d)
        out.append(d)
    return ctx, out[0], out[1]


@pytest.mark.parametrize("which", ["wl2_small", "wl3_small"])
def test_profiles_bit_exact(fdc, which, request):
    """R16: every profile equals the numpy definition bit for bit (fixed summation order), on dose grids and on the
    context's energy grid, for thin, five-voxel-thick, slab-shaped and edge-clipped bundles on all three axes."""
    import oracle
    import torch
    w = request.getfixturevalue(which)
    ctx, dA, dB = _two_doses(fdc, w)
    hA = dA.cpu().numpy()
    g = ctx.fdc_get_edep_fixed()                                  # the grid of the second run
    nx, ny, nz = w.phantom.dims
    n = (nx, ny, nz)
    for axis in (0, 1, 2):
        ia, ib = (1 if axis == 0 else 0), (1 if axis == 2 else 2)
        for fa, fb, ha, hb in ((n[ia] // 2, n[ib] // 2, 0, 0), (n[ia] // 2, n[ib] // 2, 2, 2), (n[ia] // 2 + 3, n[ib] // 2 - 2, 2, 0),
                               (0, n[ib] - 1, 2, 2), (n[ia] - 2, 1, 4, 3)):
            got = ctx.fdc_profile(dA, axis, fa, fb, ha, hb)
            assert np.array_equal(got, oracle.profile(hA, axis, fa, fb, ha, hb)), (axis, fa, fb, ha, hb)
            got_e = ctx.fdc_profile(None, axis, fa, fb, ha, hb)
            assert np.array_equal(got_e, oracle.profile(g, axis, fa, fb, ha, hb)), ("edep", axis, fa, fb, ha, hb)
    dev_out = torch.zeros(ny, dtype=torch.float64, device="cuda")
    ctx.fdc_profile(dA, 1, nx // 2, nz // 2, 2, 2, out=dev_out)
    assert np.array_equal(dev_out.cpu().numpy(), oracle.profile(hA, 1, nx // 2, nz // 2, 2, 2))
    with pytest.raises(fdc.FdcError) as e:
        ctx.fdc_profile(dA, 1, nx, 0)
    assert e.value.code == fdc.FDC_EINVAL
    with pytest.raises(fdc.FdcError):
        ctx.fdc_profile(dA, 3, 0, 0)
    ctx.fdc_destroy()


@pytest.mark.parametrize("which", ["wl2_small", "wl3_small"])
def test_rms_diff_matches_definition(fdc, which, request):
    """R17: the 128-bit fixed-point sum (quantum 2^-64 on each squared ratio) against numpy's f64 sum: the two
    differ by rounding of the summation only -- n * 2^-65 absolute in the library, pairwise-sum error 1e-16
    relative in numpy -- so 1e-12 relative on the RMS is a wide bound.  Also order independence: the same value
    bit for bit on a second call, and closed forms on the device."""
    import oracle
    import torch
    w = request.getfixturevalue(which)
    ctx, dA, dB = _two_doses(fdc, w)
    r, m = ctx.fdc_rms_diff(dA, dB)
    ro, mo = oracle.rms_diff(dA.cpu().numpy(), dB.cpu().numpy())
    assert m == mo and r > 0
    assert abs(r - ro) <= 1e-12 * ro
    assert ctx.fdc_rms_diff(dA, dB) == (r, m)
    assert ctx.fdc_rms_diff(dA, dA)[0] == 0.0
    u = torch.full(w.phantom.hu.shape, 2.0, dtype=torch.float32, device="cuda")
    ev = u * 1.03125                                             # exact in f32: ratio 1/32
    assert ctx.fdc_rms_diff(u, ev)[0] == 0.03125
    z = torch.zeros_like(u)
    with pytest.raises(fdc.FdcError):
        ctx.fdc_rms_diff(z, u)
    ctx.fdc_destroy()


def test_to_gy_alone_and_in_place_sum_of_two_shards(fdc, wl3_small):
    """The multi-GPU sequence of bench.py on one device: two contexts run the two shard_range halves of the plan,
    the second grid is added in place into the first through fdc_edep_device_ptr (what the NCCL all-reduce does),
    fdc_to_gy converts -- and grid, Gy grid and squares equal the single-context run and the oracle bit for bit."""
    import oracle
    import torch
    from paper_1011_2188_b200.multi import shard_range
    w = wl3_small
    c0, c1 = make_ctx(fdc, w), make_ctx(fdc, w)
    fl = fdc.FDC_RANDOM_AZIMUTH | fdc.FDC_TALLY_SQUARES
    for r, c in enumerate((c0, c1)):
        first, n = shard_range(w.n_protons, r, 2)
        c.fdc_run(w.beamlets, first, n, 1, w.seed, flags=fl)
    e0, q0 = c0.fdc_edep_device_ptr()
    e1, q1 = c1.fdc_edep_device_ptr()
    assert e0.dtype == torch.int64 and tuple(e0.shape) == w.phantom.hu.shape and q0 is not None
    torch.cuda.synchronize()
    e0 += e1
    q0 += q1
    torch.cuda.synchronize()
    dose = torch.zeros(w.phantom.hu.shape, dtype=torch.float32, device="cuda")
    c0.fdc_to_gy(dose)
    dose_h = np.zeros(w.phantom.hu.shape, dtype=np.float32)
    c0.fdc_to_gy(dose_h)
    og, osq, _, ost = oracle.run_sq(w.phantom, w.table, w.db, w.beamlets, w.seed, by_history=False)
    assert np.array_equal(c0.fdc_get_edep_fixed(), og) and np.array_equal(c0.fdc_get_sq_fixed(), osq)
    want = oracle.to_gy(og, w.phantom, w.table)
    assert np.array_equal(dose.cpu().numpy(), want) and np.array_equal(dose_h, want)
    info = c0.fdc_last_call_info()          # the run (5 grouping kernels + transport) plus the two conversions made since
    assert info["launches"] == 8 and info["d2h_bytes"] == dose_h.nbytes and info["gy_ms"] > 0 and info["transport_ms"] > 0
    c0.fdc_destroy(); c1.fdc_destroy()


def test_call_info_counts_the_copies(fdc, wl3_small):
    """fdc_last_call_info: a plan seen for the first time is uploaded (beamlets + prefix sums); the same plan again
    is served from the cache (0 bytes); a byte-different plan is uploaded again; a host dose grid is a D2H copy."""
    w = wl3_small
    ctx = make_ctx(fdc, w)
    nb = len(w.beamlets)
    plan_bytes = nb * 72 + (nb + 1) * 8                 # beamlets + prefix sums
    ctx.fdc_run(w.beamlets, 0, 100, 1, w.seed)
    a = ctx.fdc_last_call_info()
    assert a["h2d_bytes"] == plan_bytes and a["d2h_bytes"] == 0 and a["launches"] == 6 and a["transport_ms"] > 0
    ctx.fdc_run(w.beamlets, 100, 100, 1, w.seed)
    assert ctx.fdc_last_call_info()["h2d_bytes"] == 0
    bl2 = np.concatenate([w.beamlets, w.beamlets[-1:]]); bl2[-1]["n_protons"] = 0      # equivalent plan, different bytes
    dose = np.zeros(w.phantom.hu.shape, dtype=np.float32)
    ctx.fdc_run(bl2, 200, 100, 1, w.seed, dose_gy=dose)
    c = ctx.fdc_last_call_info()
    assert c["h2d_bytes"] == plan_bytes + 80 and c["d2h_bytes"] == dose.nbytes and c["launches"] == 7
    # the per-beamlet sort-key records (20 B) exist only for plans run with FDC_SORT_SPATIAL: uploaded by the first such run
    ctx.fdc_run(bl2, 300, 100, 1, w.seed, flags=1 | fdc.FDC_SORT_SPATIAL)
    assert ctx.fdc_last_call_info()["h2d_bytes"] == (nb + 1) * 20
    ctx.fdc_run(bl2, 400, 100, 1, w.seed, flags=1 | fdc.FDC_SORT_SPATIAL)
    assert ctx.fdc_last_call_info()["h2d_bytes"] == 0
    ctx.fdc_destroy()


@pytest.mark.timeout(180)
@pytest.mark.parametrize("n_bl", [3000, 300_000])
def test_spatial_sort_with_one_group_per_beamlet(fdc, wl3_small, n_bl):
    """a plan in which every beamlet has its own origin is its own sort group.  3 000 groups fit the key
    space (3 000 x 256 keys); 300 000 do not (> 2^24 keys: the library groups by track instead) and used to cost
    n^2/2 comparisons on the host.  FDC_SORT_SPATIAL is scheduling only: the grid equals the plain run's bit for bit."""
    w = wl3_small
    src = w.beamlets[len(w.beamlets) // 2]
    bl = np.repeat(src[None], n_bl).copy()
    step = np.float32(1e-4) * np.arange(n_bl, dtype=np.float32)                 # distinct origins along e1, 30 mm at most
    bl["origin"] = src["origin"][None, :] + step[:, None] * src["e1"][None, :]
    assert len(np.unique(bl["origin"], axis=0)) == n_bl
    bl["n_protons"] = 1
    ctx = make_ctx(fdc, w)
    ctx.fdc_run(bl, 0, n_bl, 1, w.seed, flags=1)
    plain, st_plain = ctx.fdc_get_edep_fixed(), ctx.fdc_get_stats()
    ctx.fdc_reset()
    ctx.fdc_run(bl[:-1], 0, n_bl - 1, 1, w.seed, flags=1)                        # another plan in between: the cache forgets
    ctx.fdc_reset()
    ctx.fdc_run(bl, 0, n_bl, 1, w.seed, flags=1 | fdc.FDC_SORT_SPATIAL)
    info = ctx.fdc_last_call_info()
    assert info["h2d_bytes"] == n_bl * 72 + (n_bl + 1) * 8 + (n_bl * 20 if n_bl == 3000 else 0)
    assert np.array_equal(ctx.fdc_get_edep_fixed(), plain) and ctx.fdc_get_stats() == st_plain
    assert st_plain["protons"] == n_bl and st_plain["deposits"] > 0
    ctx.fdc_destroy()


def test_diag_reds_counts_and_traces(fdc, wl3_small, wl1_small):
    """FDC_DIAG_REDS: same grid and counters as the plain kernel; reds_sent lies between the voxels touched and
    the deposits (merged shares); the trace holds exactly reds_sent voxel indices whose histogram is positive only
    where the grid is, and each voxel with energy got at least one reduction."""
    import torch
    for w in (wl3_small, wl1_small):
        ctx = make_ctx(fdc, w)
        ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, w.seed)
        g0 = ctx.fdc_get_edep_fixed(); st0 = ctx.fdc_get_stats()
        ctx.fdc_reset()
        trace = torch.full((4 << 20,), -1, dtype=torch.int32, device="cuda")
        ctx.fdc_trace_reds(trace)
        ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, w.seed, flags=fdc.FDC_RANDOM_AZIMUTH | fdc.FDC_DIAG_REDS)
        g1 = ctx.fdc_get_edep_fixed(); st1 = ctx.fdc_get_stats()
        assert np.array_equal(g0, g1) and all(st0[k] == st1[k] for k in STAT_KEYS)
        info = ctx.fdc_last_call_info()
        n = info["reds_sent"]
        assert info["reds_traced"] == n and 0 < n <= st1["deposits"] and n >= int((g1 != 0).sum())
        t = trace[:n].cpu().numpy()
        assert t.min() >= 0 and t.max() < g1.size and (trace[n:n + 16] == -1).all()
        hist = np.bincount(t, minlength=g1.size).reshape(g1.shape)
        assert np.array_equal(hist > 0, g1 != 0)
        with pytest.raises(fdc.FdcError):
            ctx.fdc_run(w.beamlets, 0, 10, 1, w.seed, flags=fdc.FDC_DIAG_REDS | fdc.FDC_TALLY_SQUARES)
        ctx.fdc_trace_reds(None)
        ctx.fdc_destroy()


def test_rejected_database_leaves_the_loaded_one_in_place(fdc, wl2_small):
    """include/fdc.h: "leave no partial state behind on failure" -- a database with an increasing E or a non-finite
    step is refused (FDC_EINVAL) and the previous one keeps running, bit for bit."""
    import oracle
    w = wl2_small
    ctx = make_ctx(fdc, w)
    ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, w.seed)
    g0 = ctx.fdc_get_edep_fixed()
    arrs = [np.ascontiguousarray(a).copy() for a in (w.db.dx, w.db.dy, w.db.dz, w.db.dE, w.db.E)]
    bad_E = [a.copy() for a in arrs]; bad_E[4][5] = bad_E[4][4] + 1.0
    bad_dx = [a.copy() for a in arrs]; bad_dx[0][7] = np.inf
    for bad in (bad_E, bad_dx):
        with pytest.raises(fdc.FdcError) as e:
            ctx.fdc_load_tracks(*bad, w.db.track_off, w.db.bin_first, w.db.e_min, w.db.e_bin)
        assert e.value.code == fdc.FDC_EINVAL
        ctx.fdc_reset()
        ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, w.seed)               # would be FDC_ENOTRACKS if the old database had gone
        assert np.array_equal(ctx.fdc_get_edep_fixed(), g0)
    og, _ = oracle.run(w.phantom, w.table, w.db, w.beamlets, w.seed)
    assert np.array_equal(g0, og)
    ctx.fdc_destroy()


def test_peaks_library_runs(fdc):
    """libfdcpeaks.so: the uniform rate is positive and well above the hot-set rate; a replayed trace of one
    address is slower than a replayed uniform trace (contention shows)."""
    import torch
    from paper_1011_2188_b200 import peaks
    uni = peaks.red_u64(0, 16 << 20, 1 << 26, 0)
    hot = peaks.red_u64(0, 16 * 8, 1 << 24, 0)
    assert uni > 1e10 and hot < uni / 4
    n_words = 1 << 21
    tr_uniform = torch.randint(0, n_words, (1 << 22,), dtype=torch.int32, device="cuda")
    tr_one = torch.zeros(1 << 22, dtype=torch.int32, device="cuda")
    a = peaks.red_replay(0, tr_uniform, tr_uniform.numel(), n_words, 4, False)
    b = peaks.red_replay(0, tr_uniform, tr_uniform.numel(), n_words, 4, True)
    c = peaks.red_replay(0, tr_one, tr_one.numel(), n_words, 4, True)
    assert a > 1e10 and b > 1e10 and c > 0


def test_launch_cuts_at_field_boundaries_lose_no_proton(fdc):
    """A run is cut into launches where the plan changes beam direction.  On the three-field plan of config 4,
    a strided range that spans all three fields gives the same grid and counters whether it runs as one call (cut at the two
    field boundaries) or as three calls split elsewhere (cut at other places): no proton is lost or run twice at a cut, and
    the oblique launches (tiled material grid) add up with the axis-aligned one (linear grid).  The oracle is not needed:
    integer sums over the same protons.  The strided subsets of the whole-plan digest tests compare such runs with it."""
    w = fi.workload(4, lazy_db=True)
    ctx = make_ctx(fdc, w, device_arrays=True)
    first, stride, n = 3, 7, 6_000_000                      # global indices up to 4.2e7: fields begin at 1.667e7 and 3.333e7
    assert first + (n - 1) * stride < w.n_protons
    ctx.fdc_run(w.beamlets, first, n, stride, w.seed)
    g1, s1 = ctx.fdc_get_edep_fixed(), ctx.fdc_get_stats()
    assert s1["protons"] == n and ctx.fdc_last_call_info()["launches"] == 3 * 6
    ctx.fdc_reset()
    for a, b in ((0, 1_000_000), (1_000_000, 3_100_000), (3_100_000, n)):
        ctx.fdc_run(w.beamlets, first + a * stride, b - a, stride, w.seed, flags=fdc.FDC_RANDOM_AZIMUTH | (fdc.FDC_MAT_LINEAR if a else 0))
    g2, s2 = ctx.fdc_get_edep_fixed(), ctx.fdc_get_stats()
    assert np.array_equal(g1, g2)
    for k in STAT_KEYS:
        assert s1[k] == s2[k], (k, s1[k], s2[k])
    ctx.fdc_destroy()

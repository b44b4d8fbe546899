"""GPU parity: the CUDA path (through the C-ABI) against the oracle, element by element on the same
seeded inputs.  Bar (north_star): the u64 fixed-point grid is BIT-EXACT; the Gy grid
is then identical too (same f64 formula); every counter of fdc_stats equals the oracle's."""
import numpy as np
import pytest

import fdc_inputs as fi

pytestmark = pytest.mark.gpu

STAT_KEYS = ("protons", "proton_steps", "deposits", "missed", "escaped", "stopped", "grid_sum", "q_replayed", "q_escaped")


@pytest.fixture(scope="module")
def fdc():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    import paper_1011_2188_b200 as m
    m.lib()                       # fails loudly if libfdc.so is missing: there is no fallback
    return m


def make_ctx(fdc, w, device_arrays=False):
    import torch
    if device_arrays:
        hu = torch.from_numpy(w.phantom.hu).cuda()
        ctx = fdc.Fdc(hu, w.phantom.spacing, w.table)
        t = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (w.db.dx, w.db.dy, w.db.dz, w.db.dE, w.db.E)]
        ctx.fdc_load_tracks(*t, w.db.track_off, w.db.bin_first, w.db.e_min, w.db.e_bin)
    else:
        ctx = fdc.Fdc(np.ascontiguousarray(w.phantom.hu), w.phantom.spacing, w.table)
        ctx.fdc_load_tracks(*[np.ascontiguousarray(a) for a in (w.db.dx, w.db.dy, w.db.dz, w.db.dE, w.db.E)],
                            w.db.track_off, w.db.bin_first, w.db.e_min, w.db.e_bin)
    return ctx


def check_against_oracle(fdc, w, ctx=None, flags=1, first=0, n=None, stride=1, seed=None):
    import oracle
    seed = w.seed if seed is None else seed
    n = w.n_protons if n is None else n
    own = ctx is None
    if own:
        ctx = make_ctx(fdc, w)
    ctx.fdc_reset()
    dose = np.zeros(w.phantom.hu.shape, dtype=np.float32)
    ctx.fdc_run(w.beamlets, first, n, stride, seed, flags=flags, dose_gy=dose)
    g = ctx.fdc_get_edep_fixed()
    st = ctx.fdc_get_stats()
    og, ost = oracle.run(w.phantom, w.table, w.db, w.beamlets, seed, first=first, n=n, stride=stride, flags=flags & 33)   # 33: the flags that change the result
    assert np.array_equal(g, og), "fixed-point grid differs: %d voxels, sum %d vs %d" % (
        int((g != og).sum()), int(g.sum(dtype=np.uint64)), int(og.sum(dtype=np.uint64)))
    for k in STAT_KEYS:
        assert st[k] == ost[k], (k, st[k], ost[k])
    assert st["grid_sum"] + st["q_escaped"] == st["q_replayed"]
    assert np.array_equal(dose, oracle.to_gy(og, w.phantom, w.table))
    if own:
        ctx.fdc_destroy()
    return g, st


# ------------------------------------------------------------------ reduced-size configs, every element
def test_config1_reduced(fdc, wl1_small):
    check_against_oracle(fdc, wl1_small)


def test_config2_reduced(fdc, wl2_small):
    g, st = check_against_oracle(fdc, wl2_small)
    assert st["escaped"] == wl2_small.n_protons


def test_config3_reduced(fdc, wl3_small):
    g, st = check_against_oracle(fdc, wl3_small)
    assert st["deposits"] > 10 * st["proton_steps"] / 8          # air columns: many voxels per step


def test_flags_and_ranges(fdc, wl3_small):
    w = wl3_small
    ctx = make_ctx(fdc, w, device_arrays=True)
    g_sorted, _ = check_against_oracle(fdc, w, ctx)
    g_nosort, _ = check_against_oracle(fdc, w, ctx, flags=1 | fdc.FDC_NO_SORT)
    g_noagg, _ = check_against_oracle(fdc, w, ctx, flags=1 | fdc.FDC_NO_AGGREGATE)
    assert np.array_equal(g_sorted, g_nosort) and np.array_equal(g_sorted, g_noagg)
    # scheduling variants: this small plan runs with the CTA-private tally by default; the big-plan instantiation
    # (FDC_NO_LAT), the warp-aggregating one (FDC_WARP_AGGREGATE), grouping by start position -- the integers cannot change
    sp, pt = fdc.FDC_SORT_SPATIAL, fdc.FDC_PRIVATE_TALLY
    wa, mt, ml = fdc.FDC_WARP_AGGREGATE, fdc.FDC_MAT_TILED, fdc.FDC_MAT_LINEAR
    for fl in (1 | mt, 1 | ml, 1 | mt | fdc.FDC_NO_LAT, 1 | mt | fdc.FDC_NO_SORT, 1 | mt | fdc.FDC_NO_AGGREGATE, 1 | mt | fdc.FDC_TALLY_SQUARES, 1 | fdc.FDC_NO_LAT, 1 | wa, 1 | sp, 1 | sp | wa, 1 | sp | fdc.FDC_NO_LAT, 1 | sp | pt, sp | pt, 1 | pt, 1 | fdc.FDC_NO_SORT | fdc.FDC_NO_LAT,
               1 | fdc.FDC_NO_SORT | wa):
        g_v, _ = check_against_oracle(fdc, w, ctx, flags=fl)
        if fl & 1:
            assert np.array_equal(g_sorted, g_v), fl
    check_against_oracle(fdc, w, ctx, flags=0)                                   # azimuth off
    check_against_oracle(fdc, w, ctx, first=7, n=300, stride=13)                 # strided subset
    check_against_oracle(fdc, w, ctx, first=4000, n=704)                         # tail range
    check_against_oracle(fdc, w, ctx, seed=2 ** 40 + 12345)                      # 64-bit seed
    # accumulation: run(0..a) + run(a..N) == run(0..N), bit for bit (P7)
    ctx.fdc_reset()
    ctx.fdc_run(w.beamlets, 1000, w.n_protons - 1000, 1, w.seed)
    ctx.fdc_run(w.beamlets, 0, 1000, 1, w.seed)
    assert np.array_equal(ctx.fdc_get_edep_fixed(), g_sorted)
    # n_protons = 0 is a no-op
    ctx.fdc_reset()
    ctx.fdc_run(w.beamlets, 0, 0, 1, w.seed)
    assert ctx.fdc_get_stats()["protons"] == 0 and not ctx.fdc_get_edep_fixed().any()
    # device output buffers
    import torch
    ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, w.seed)
    gd = torch.zeros(w.phantom.hu.shape, dtype=torch.int64, device="cuda")
    ctx.fdc_get_edep_fixed(gd)
    dd = torch.zeros(w.phantom.hu.shape, dtype=torch.float32, device="cuda")
    ctx.fdc_run(w.beamlets, 0, 0, 1, w.seed, dose_gy=dd)
    torch.cuda.synchronize()
    assert np.array_equal(gd.cpu().numpy().view(np.uint64), g_sorted)
    import oracle
    assert np.array_equal(dd.cpu().numpy(), oracle.to_gy(g_sorted, w.phantom, w.table))
    ctx.fdc_destroy()


def test_hand_made_cases(fdc):
    """Closed-form inputs of tests/test_oracle_pins.py: straight, split, half density, interface,
    oblique, angle scaling, zero-length step, escape, miss -- all bit-exact against the oracle."""
    from test_oracle_pins import hand_db, table_uniform, uniform_phantom
    cases = []
    ph = uniform_phantom(16, 1.0)
    cases.append((ph, table_uniform(1.0), hand_db([[(0, 0, 1.0, (k + 1) / 8.0) for k in range(10)]]),
                  fi.single_beamlet((5.5, 6.5, 0.0), 100.0, 0.0, 3), 1))
    cases.append((ph, table_uniform(1.0), hand_db([[(0, 0, 1.0, 1.0 + k / 4.0) for k in range(6)]]),
                  fi.single_beamlet((5.5, 6.5, 0.25), 100.0, 0.0, 1), 1))
    cases.append((ph, table_uniform(0.5), hand_db([[(0, 0, 1.0, 1.0) for _ in range(4)]]),
                  fi.single_beamlet((5.5, 6.5, 0.0), 100.0, 0.0, 1), 1))
    cases.append((ph, table_uniform(1.0), hand_db([[(0, 0, 4.5, 4.5)]]),
                  fi.single_beamlet((0.4, 4.5, 0.0), 100.0, 0.0, 1, e1=(0.8, 0, -0.6), e2=(0, 1, 0), d=(0.6, 0, 0.8)), 0))
    tau = 0.05; n1 = float(np.hypot(1.0, tau)); u1 = (tau / n1, 0.0, 1.0 / n1)
    cases.append((uniform_phantom(32, 1.0), table_uniform(1.0, 1.0, 2.25),
                  hand_db([[(0, 0, 1.0, 1.0), u1 + (1.0,), u1 + (1.0,), (0.1, 0.2, 0.9, 1.5)]]),
                  fi.single_beamlet((16.5, 16.5, 0.0), 100.0, 2.0, 50), 1))
    cases.append((uniform_phantom(8, 1.0), table_uniform(1.0), hand_db([[(0, 0, 1.0, 1.0), (0, 0, 0.0, 2.0), (0, 0, 1.0, 1.0)]]),
                  fi.single_beamlet((3.5, 3.5, 0.0), 100.0, 0.0, 2), 1))
    cases.append((uniform_phantom(8, 1.0), table_uniform(1.0), hand_db([[(0, 0, 1.0, 0.5 + 0.125 * k) for k in range(12)]]),
                  fi.single_beamlet((3.5, 3.5, 0.25), 100.0, 0.0, 1), 1))
    cases.append((uniform_phantom(8, 1.0), table_uniform(1.0), hand_db([[(0, 0, 1.0, 1.0)]]),
                  fi.single_beamlet((30.0, 3.5, -5.0), 100.0, 0.0, 4), 1))          # misses the grid
    cases.append((uniform_phantom(8, 1.0), table_uniform(1.0), hand_db([[(0, 0, 1.0, 1.0)]]),
                  fi.single_beamlet((3.5, 3.5, 0.0), 10.0, 0.0, 2), 1))             # replays nothing
    ph_if = fi.make_phantom("uniform", (8, 8, 16), (1.0, 1.0, 0.5)); ph_if.hu[3:, :, :] = -500
    tab_if = np.array([(-500.0, 0.5, 1.0, 1.0), (0.0, 1.0, 1.0, 1.0)], dtype=fi.KNOT_DTYPE)
    cases.append((ph_if, tab_if, hand_db([[(0, 0, 1.0, 1.0), (0, 0, 1.0, 2.0)]]), fi.single_beamlet((3.5, 3.5, 0.0), 100.0, 0.0, 1), 1))
    for ph, tab, db, bl, flags in cases:
        w = fi.Workload("hand", ph, tab, db, bl, int(bl["n_protons"].sum()), 5)
        check_against_oracle(fdc, w, flags=flags)


def test_errors(fdc, wl2_small):
    w = wl2_small
    hu = np.ascontiguousarray(w.phantom.hu)
    ctx = fdc.Fdc(hu, w.phantom.spacing, w.table)
    with pytest.raises(fdc.FdcError) as e:
        ctx.fdc_run(w.beamlets, 0, 10, 1, 1)
    assert e.value.code == fdc.FDC_ENOTRACKS
    arrs = [np.ascontiguousarray(a) for a in (w.db.dx, w.db.dy, w.db.dz, w.db.dE, w.db.E)]
    bad = [a.copy() for a in arrs]; bad[4][5] = 1e9                                  # E increases within a track
    with pytest.raises(fdc.FdcError) as e:
        ctx.fdc_load_tracks(*bad, w.db.track_off, w.db.bin_first, w.db.e_min, w.db.e_bin)
    assert e.value.code == fdc.FDC_EINVAL
    bad = [a.copy() for a in arrs]; bad[3][7] = -1.0                                 # negative dE
    with pytest.raises(fdc.FdcError) as e:
        ctx.fdc_load_tracks(*bad, w.db.track_off, w.db.bin_first, w.db.e_min, w.db.e_bin)
    assert e.value.code == fdc.FDC_EINVAL
    off = w.db.track_off.copy(); off[-1] += 1
    with pytest.raises(fdc.FdcError) as e:
        ctx.fdc_load_tracks(*arrs, off, w.db.bin_first, w.db.e_min, w.db.e_bin)
    assert e.value.code == fdc.FDC_EINVAL
    ctx.fdc_load_tracks(*arrs, w.db.track_off, w.db.bin_first, w.db.e_min, w.db.e_bin)
    for kw, code in [(dict(proton_stride=0), fdc.FDC_EINVAL), (dict(first_proton=w.n_protons), fdc.FDC_EINVAL),
                     (dict(n_protons=w.n_protons + 1), fdc.FDC_EINVAL), (dict(first_proton=5, n_protons=w.n_protons), fdc.FDC_EINVAL)]:
        a = dict(first_proton=0, n_protons=10, proton_stride=1); a.update(kw)
        with pytest.raises(fdc.FdcError) as e:
            ctx.fdc_run(w.beamlets, a["first_proton"], a["n_protons"], a["proton_stride"], 1)
        assert e.value.code == code
    bl = w.beamlets.copy(); bl["energy_mev"] = 170.0                                 # above the top bin
    with pytest.raises(fdc.FdcError) as e:
        ctx.fdc_run(bl, 0, 10, 1, 1)
    assert e.value.code == fdc.FDC_ERANGE
    bl = w.beamlets.copy(); bl["energy_mev"] = 145.0                                 # bin exists but lazily left empty
    with pytest.raises(fdc.FdcError) as e:
        ctx.fdc_run(bl, 0, 10, 1, 1)
    assert e.value.code == fdc.FDC_ERANGE
    bl = w.beamlets.copy(); bl["dir"] = (0.0, 0.1, 1.0)                              # not a unit vector
    with pytest.raises(fdc.FdcError) as e:
        ctx.fdc_run(bl, 0, 10, 1, 1)
    assert e.value.code == fdc.FDC_EINVAL
    assert not ctx.fdc_get_edep_fixed().any()                                         # failures left no partial state
    ctx.fdc_destroy()
    with pytest.raises(fdc.FdcError) as e:
        fdc.Fdc(hu, (1.0, 0.0, 1.0), w.table)
    assert e.value.code == fdc.FDC_EINVAL
    tab = w.table.copy(); tab["hu"][2] = tab["hu"][1]
    with pytest.raises(fdc.FdcError) as e:
        fdc.Fdc(hu, w.phantom.spacing, tab)
    assert e.value.code == fdc.FDC_EINVAL


def test_hu_outside_table_is_clamped(fdc):
    from test_oracle_pins import hand_db
    ph = fi.make_phantom("uniform", (8, 8, 8), (1.0, 1.0, 1.0))
    ph.hu[:4] = -2000; ph.hu[4:] = 32000
    db = hand_db([[(0, 0, 1.0, 1.0)] * 12])
    w = fi.Workload("clamp", ph, fi.material_table("config2"), db, fi.single_beamlet((3.5, 3.5, 7.9), 100.0, 0.0, 3, e1=(0, 1, 0), e2=(1, 0, 0), d=(0, 0, -1)), 3, 9)
    check_against_oracle(fdc, w)


# ------------------------------------------------------------------ full sizes, in bench.py's launch configuration
def test_config1_full_bit_exact(fdc):
    w = fi.workload(1)
    g, st = check_against_oracle(fdc, w)
    assert st["protons"] == 100_000 and st["escaped"] == 0
    assert abs(st["grid_sum"] / 2 ** 24 / 1e5 - 100.0) < 1e-4


def test_config2_full_bit_exact(fdc):
    """BASELINE.json configs[1] at full size (1e6 protons, 1e4 tracks in the 150 MeV bin): the
    workload bench.py times.  The oracle needs some tens of seconds for it."""
    w = fi.workload(2)
    g, st = check_against_oracle(fdc, w)
    assert st["protons"] == 1_000_000


@pytest.mark.parametrize("cfg,n_sub", [(3, 100_000), (4, 100_000)])
def test_config34_full_db_strided_subset(fdc, cfg, n_sub):
    """Configs 3/4 with the full-size database and plan; the oracle runs every K-th proton (so every
    field, layer and spot is represented) and the GPU runs the same subset, word for word.  Then the
    GPU runs the whole plan and is checked by properties that hold at any size: conservation, and
    full == sum of two halves."""
    w = fi.workload(cfg)
    ctx = make_ctx(fdc, w)
    K = w.n_protons // n_sub
    check_against_oracle(fdc, w, ctx, first=K // 2, n=n_sub, stride=K)
    if cfg in (3, 4):           # config 4's 5e7 protons also cross the 2^25-proton chunk boundary of the scheduler
        ctx.fdc_reset()
        ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, w.seed)
        g = ctx.fdc_get_edep_fixed(); st = ctx.fdc_get_stats()
        assert st["protons"] == w.n_protons == st["missed"] + st["escaped"] + st["stopped"]
        assert st["grid_sum"] + st["q_escaped"] == st["q_replayed"] and st["grid_sum"] == int(g.sum(dtype=np.uint64))
        ctx.fdc_reset()
        ctx.fdc_run(w.beamlets, w.n_protons // 2, w.n_protons - w.n_protons // 2, 1, w.seed)
        ctx.fdc_run(w.beamlets, 0, w.n_protons // 2, 1, w.seed)
        assert np.array_equal(ctx.fdc_get_edep_fixed(), g)
    ctx.fdc_destroy()


def test_config5_full_db_strided_subset(fdc):
    """Config 5 (512x512x256 grid, 512 MiB of u64: the L2-spill case; 9720 beamlets; 8e5 tracks in
    the 40 bins the plan touches): the oracle and the GPU run every K-th proton, word for word; then
    the GPU runs a 1/16 prefix-strided share of the plan in two chunked calls and is checked by
    conservation and additivity (the whole plan, 2e8 protons, is bench.py --config 5)."""
    w = fi.workload(5, lazy_db=True)
    ctx = make_ctx(fdc, w)
    n_sub = 50_000
    K = w.n_protons // n_sub
    check_against_oracle(fdc, w, ctx, first=K // 3, n=n_sub, stride=K)
    n16 = w.n_protons // 16
    ctx.fdc_reset()
    ctx.fdc_run(w.beamlets, 5, n16, 16, w.seed)
    g = ctx.fdc_get_edep_fixed(); st = ctx.fdc_get_stats()
    assert st["protons"] == n16 == st["missed"] + st["escaped"] + st["stopped"]
    assert st["grid_sum"] + st["q_escaped"] == st["q_replayed"] and st["grid_sum"] == int(g.sum(dtype=np.uint64))
    ctx.fdc_reset()
    ctx.fdc_run(w.beamlets, 5 + 16 * (n16 // 2), n16 - n16 // 2, 16, w.seed)
    ctx.fdc_run(w.beamlets, 5, n16 // 2, 16, w.seed)
    assert np.array_equal(ctx.fdc_get_edep_fixed(), g)
    ctx.fdc_destroy()



# ------------------------------------------------------------------ R10 / R11: squares and uncertainties
def run_gpu_sq(fdc, ctx, w, first=0, n=None, stride=1, seed=None, flags=1):
    n = w.n_protons if n is None else n
    ctx.fdc_reset()
    ctx.fdc_run(w.beamlets, first, n, stride, w.seed if seed is None else seed, flags=flags | fdc.FDC_TALLY_SQUARES)
    return ctx.fdc_get_edep_fixed(), ctx.fdc_get_sq_fixed(), ctx.fdc_get_stats()


@pytest.mark.parametrize("which", ["wl1_small", "wl2_small", "wl3_small"])
def test_squares_bit_exact(fdc, which, request):
    """Energy grid, squares grid (by visit, R10) and counters equal the oracle's, word for word; the
    energy grid is the one the plain run gives."""
    import oracle
    w = request.getfixturevalue(which)
    ctx = make_ctx(fdc, w)
    with pytest.raises(fdc.FdcError):
        ctx.fdc_get_sq_fixed()                                                   # no squares grid yet
    g, s2, st = run_gpu_sq(fdc, ctx, w)
    og, osv, _, ost = oracle.run_sq(w.phantom, w.table, w.db, w.beamlets, w.seed, by_history=False)
    assert np.array_equal(g, og) and np.array_equal(s2, osv)
    for k in STAT_KEYS:
        assert st[k] == ost[k], (k, st[k], ost[k])
    with pytest.raises(fdc.FdcError) as e:
        ctx.fdc_run(w.beamlets, 0, 10, 1, w.seed, flags=1 | fdc.FDC_TALLY_SQUARES | fdc.FDC_NO_AGGREGATE)
    assert e.value.code == fdc.FDC_EINVAL
    # eq. (2) as defined (FDC_SQUARES_BY_HISTORY): the history's whole deposit in a voxel squared once, equal to the oracle's
    # by-history tally word for word, with the material read from either copy of the grid; the energy grid does not change
    _, _, osh, _ = oracle.run_sq(w.phantom, w.table, w.db, w.beamlets, w.seed, by_history=True)
    for extra in (0, fdc.FDC_MAT_TILED, fdc.FDC_TALLY_SQUARES | fdc.FDC_NO_LAT):
        ctx.fdc_reset()
        ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, w.seed, flags=1 | fdc.FDC_SQUARES_BY_HISTORY | extra)
        assert np.array_equal(ctx.fdc_get_sq_fixed(), osh) and np.array_equal(ctx.fdc_get_edep_fixed(), og)
        assert ctx.fdc_last_call_info()["sq_history_flushes"] == 0
        st_h = ctx.fdc_get_stats()
        for k in STAT_KEYS:
            assert st_h[k] == ost[k], (k, st_h[k], ost[k])
    assert (osh >= osv).all()
    # additivity and reset
    g_a, s_a, _ = run_gpu_sq(fdc, ctx, w, first=0, n=w.n_protons // 3)
    ctx.fdc_run(w.beamlets, w.n_protons // 3, w.n_protons - w.n_protons // 3, 1, w.seed, flags=1 | fdc.FDC_TALLY_SQUARES)
    assert np.array_equal(ctx.fdc_get_sq_fixed(), s2) and np.array_equal(ctx.fdc_get_edep_fixed(), g)
    ctx.fdc_reset()
    assert not ctx.fdc_get_sq_fixed().any()
    ctx.fdc_destroy()


def test_squares_by_history_table_overflow(fdc):
    """A history that visits more voxels than its table holds (2048): the table is emptied early and the event is counted.
    Without re-entered voxels the tally still equals the definition; a track that comes back through the voxels of an earlier
    segment is squared in segments -- between the per-stay and the per-history tallies, voxel by voxel."""
    import oracle
    from test_oracle_pins import hand_db, table_uniform
    ph = fi.make_phantom("uniform", (2, 2, 6000), (1.0, 1.0, 1.0), hu0=0)
    n = 64
    for steps, exact in (([(0, 0, 5000.0, 5.0)], True), ([(0, 0, 5000.0, 5.0), (0, 0, -4999.0, 5.0)], False)):
        w = fi.Workload("long", ph, table_uniform(1.0), hand_db([steps]), fi.single_beamlet((0.5, 0.5, 0.0), 100.0, 0.0, n), n, 9)
        ctx = make_ctx(fdc, w)
        ctx.fdc_run(w.beamlets, 0, n, 1, w.seed, flags=fdc.FDC_SQUARES_BY_HISTORY)
        og, osv, osh, ost = oracle.run_sq(w.phantom, w.table, w.db, w.beamlets, w.seed, flags=0, by_history=True)
        s2 = ctx.fdc_get_sq_fixed()
        assert np.array_equal(ctx.fdc_get_edep_fixed(), og)
        assert ctx.fdc_last_call_info()["sq_history_flushes"] == n * (2 if exact else 4)
        with pytest.warns(fdc.FdcWarning, match="squared in segments"):          # the overflow is not silent (FDC_WSEGMENTED)
            mean_w, cnt_w = ctx.fdc_uncertainty_history(n)
        assert cnt_w > 0 and mean_w >= 0.0                                        # outputs valid all the same
        if exact:
            assert np.array_equal(s2, osh) and np.array_equal(osh, osv)
        else:
            assert (s2 >= osv).all() and (s2 <= osh).all() and (s2 != osh).any() and (osh > osv).any()
        ctx.fdc_reset()
        assert ctx.fdc_last_call_info()["sq_history_flushes"] == 0
        ctx.fdc_run(w.beamlets, 0, n, 1, w.seed, flags=fdc.FDC_TALLY_SQUARES)     # per stay: no table, no warning
        import warnings
        with warnings.catch_warnings():
            warnings.simplefilter("error")
            ctx.fdc_uncertainty_history(n)
        ctx.fdc_destroy()


def test_uncertainty_history_and_batch(fdc):
    """Eq. (2) and eq. (1) maps (f32 of the f64 formula) equal the oracle's numpy evaluation exactly;
    the mean-uncertainty figure agrees to 1e-8 (fixed-point sum against numpy's pairwise sum)."""
    import torch
    import oracle
    base = fi.workload(1, n_protons=1, tracks_per_bin=500)
    N = 4000
    bl = fi.single_beamlet((64.0, 64.0, 0.0), 100.0, 6.0, N)
    w = fi.Workload("unc", base.phantom, base.table, base.db, bl, N, 31)
    rho = oracle.density(w.phantom, w.table)
    ctx = make_ctx(fdc, w)
    g, s2, _ = run_gpu_sq(fdc, ctx, w)
    rel = np.zeros(w.phantom.hu.shape, dtype=np.float32)
    mean_rel, cnt = ctx.fdc_uncertainty_history(N, rel)
    m, sg = oracle.sigma_history(g, s2, N)
    with np.errstate(invalid="ignore", divide="ignore"):
        orel = np.where(m > 0, sg / m, 0.0)
    assert np.array_equal(rel, orel.astype(np.float32))
    oval, ocnt = oracle.mean_uncertainty(m, sg, rho)
    assert cnt == ocnt and mean_rel == pytest.approx(oval, rel=1e-8)
    rel_d = torch.zeros(w.phantom.hu.shape, dtype=torch.float32, device="cuda")
    assert ctx.fdc_uncertainty_history(N, rel_d) == (mean_rel, cnt)
    assert np.array_equal(rel_d.cpu().numpy(), rel)
    # batches: six independent seeds
    grids_d, grids_h = [], []
    for b in range(6):
        ctx.fdc_reset()
        ctx.fdc_run(w.beamlets, 0, N, 1, 1000 + b)
        gd = torch.zeros(w.phantom.hu.shape, dtype=torch.int64, device="cuda")
        ctx.fdc_get_edep_fixed(gd)
        grids_d.append(gd); grids_h.append(gd.cpu().numpy().view(np.uint64))
    relb = np.zeros(w.phantom.hu.shape, dtype=np.float32)
    mean_b, cnt_b = ctx.fdc_uncertainty_batch(grids_d, N, relb)
    mb, sb = oracle.sigma_batch(grids_h)
    with np.errstate(invalid="ignore", divide="ignore"):
        orelb = np.where(mb > 0, (sb / N) / (mb / N), 0.0)
    assert np.array_equal(relb, orelb.astype(np.float32))
    ovalb, ocntb = oracle.mean_uncertainty(mb / N, sb / N, rho)
    assert cnt_b == ocntb and mean_b == pytest.approx(ovalb, rel=1e-8)
    # per history the batch figure refers to 6 N histories: it is about sqrt(6) below the single-run one
    assert mean_rel / mean_b == pytest.approx(np.sqrt(6.0), rel=0.35)
    with pytest.raises(fdc.FdcError):
        ctx.fdc_uncertainty_batch(grids_d[:1], N)
    ctx.fdc_destroy()


# ------------------------------------------------------------------ R12: phase-space source
def test_phase_space_bit_exact(fdc):
    """A divergent beam with an energy spread given as a phase-space array: grid and counters equal the
    oracle's; host and device arrays, identity offsets, additivity, squares; invalid arrays leave no trace."""
    import torch
    import oracle
    from test_oracle_phase_space import cone, particles
    w = fi.workload(2, n_protons=10, tracks_per_bin=100, lazy_db=False)
    ctx = make_ctx(fdc, w)
    ps = cone(5000, 3)
    og, ost = oracle.run_phase_space(w.phantom, w.table, w.db, ps, 77, first_id=12345)
    for dev in (False, True):
        ctx.fdc_reset()
        arr = torch.from_numpy(ps.view(np.uint8).copy()).cuda() if dev else ps
        dose = np.zeros(w.phantom.hu.shape, dtype=np.float32)
        ctx.fdc_run_phase_space(arr, 12345, 77, dose_gy=dose)
        g = ctx.fdc_get_edep_fixed(); st = ctx.fdc_get_stats()
        assert np.array_equal(g, og)
        for k in STAT_KEYS:
            assert st[k] == ost[k], (k, st[k], ost[k])
        assert np.array_equal(dose, oracle.to_gy(og, w.phantom, w.table))
    ctx.fdc_reset()                                                      # two halves, unsorted and squares variants
    ctx.fdc_run_phase_space(ps[:2000], 12345, 77, flags=1 | fdc.FDC_NO_SORT)
    ctx.fdc_run_phase_space(ps[2000:], 12345 + 2000, 77, flags=1 | fdc.FDC_TALLY_SQUARES)
    assert np.array_equal(ctx.fdc_get_edep_fixed(), og)
    ctx.fdc_reset()
    ctx.fdc_run_phase_space(ps[:0], 0, 77)                               # empty array: no-op
    assert ctx.fdc_get_stats()["protons"] == 0
    bad = ps.copy(); bad["dir"][7] = (0.0, 0.3, 1.0)
    with pytest.raises(fdc.FdcError) as e:
        ctx.fdc_run_phase_space(bad, 0, 77)
    assert e.value.code == fdc.FDC_EINVAL
    bad = ps.copy(); bad["energy_mev"][11] = 170.0
    with pytest.raises(fdc.FdcError) as e:
        ctx.fdc_run_phase_space(bad, 0, 77)
    assert e.value.code == fdc.FDC_ERANGE
    assert not ctx.fdc_get_edep_fixed().any() and ctx.fdc_get_stats()["protons"] == 0
    ctx.fdc_destroy()


def test_phase_space_reproduces_beamlet_plan_on_gpu(fdc, wl2_small):
    """Start points of the beamlet plan handed back as a phase-space array give the plan's own grid."""
    import oracle
    from test_oracle_phase_space import particles
    w = wl2_small
    ctx = make_ctx(fdc, w)
    ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, w.seed)
    g_plan = ctx.fdc_get_edep_fixed()
    smp = oracle.sample(w.phantom, w.table, w.db, w.beamlets, w.seed, first=0, n=w.n_protons)
    ps = particles(smp["p"], np.tile(np.float32([0, 0, 1]), (w.n_protons, 1)), 150.0)
    ctx.fdc_reset()
    ctx.fdc_run_phase_space(ps, 0, w.seed)
    assert np.array_equal(ctx.fdc_get_edep_fixed(), g_plan)
    ctx.fdc_destroy()


# ------------------------------------------------------------------ R13: gamma index
@pytest.mark.parametrize("which,search", [("wl3_small", 3.0), ("wl2_small", 3.0), ("wl2_small", 4.5)])
def test_gamma_index_bit_exact(fdc, which, search, request):
    """Two statistically independent runs of the same plan compared with Gamma(3 %, 3 mm), as the paper
    compares GFDC with GEANT4: the map (f32 of the f64 formula), the pass fraction and
    the voxel count equal the oracle's definition."""
    import torch
    import oracle
    w = request.getfixturevalue(which)
    ctx = make_ctx(fdc, w)
    doses = []
    for seed in (w.seed, w.seed + 1000):
        ctx.fdc_reset()
        d = torch.zeros(w.phantom.hu.shape, dtype=torch.float32, device="cuda")
        ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, seed, dose_gy=d)
        doses.append(d)
    gm = torch.zeros(w.phantom.hu.shape, dtype=torch.float32, device="cuda")
    for cutoff in (0.0, 0.1):
        pf, n = ctx.fdc_gamma_index(doses[0], doses[1], 0.03, 3.0, search, cutoff, gm)
        og, opf, on = oracle.gamma_index(doses[0].cpu().numpy(), doses[1].cpu().numpy(), w.phantom.spacing, 0.03, 3.0, search, cutoff)
        assert np.array_equal(gm.cpu().numpy(), og)
        assert n == on and pf == opf
    pf_same, _ = ctx.fdc_gamma_index(doses[0], doses[0])
    assert pf_same == 1.0
    with pytest.raises(fdc.FdcError):
        ctx.fdc_gamma_index(doses[0], doses[1], 0.03, 3.0, 100.0)                # window of more than 5 voxels
    ctx.fdc_destroy()


# ------------------------------------------------------------------ R14: re-aligned deep starts
def test_realign_start_bit_exact(fdc, wl3_small):
    """FDC_REALIGN_START against the oracle: a single-energy database entered far below its energy
    (phase-space energies 60-100 MeV into the 100 MeV bin) from outside the grid and obliquely, and a
    beam plan; with the flag off the same runs give another grid."""
    import oracle
    from test_oracle_phase_space import cone
    base = fi.workload(1, n_protons=1, tracks_per_bin=300)
    ctx = make_ctx(fdc, base)
    ps = cone(3000, 8, e_lo=60.0, e_hi=100.0, half_angle=0.15)
    grids = {}
    for flags in (1, 1 | fdc.FDC_REALIGN_START, fdc.FDC_REALIGN_START):
        ctx.fdc_reset()
        ctx.fdc_run_phase_space(ps, 500, 21, flags=flags)
        g = ctx.fdc_get_edep_fixed(); st = ctx.fdc_get_stats()
        og, ost = oracle.run_phase_space(base.phantom, base.table, base.db, ps, 21, first_id=500, flags=flags)
        assert np.array_equal(g, og)
        for k in STAT_KEYS:
            assert st[k] == ost[k], (k, st[k], ost[k])
        grids[flags] = g
    assert not np.array_equal(grids[1], grids[1 | fdc.FDC_REALIGN_START])
    ctx.fdc_destroy()
    w = wl3_small
    ctx = make_ctx(fdc, w)
    ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, w.seed, flags=1 | fdc.FDC_REALIGN_START)
    og, ost = oracle.run(w.phantom, w.table, w.db, w.beamlets, w.seed, flags=1 | oracle.FLAG_REALIGN_START)
    assert np.array_equal(ctx.fdc_get_edep_fixed(), og) and ctx.fdc_get_stats()["deposits"] == ost["deposits"]
    ctx.fdc_destroy()


# ------------------------------------------------------------------ whole plans of configs 3-5 against the off-box oracle
def _digests():
    import json
    import os
    p = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "full_plan_digests.json")
    return json.load(open(p))


@pytest.mark.parametrize("cfg", [3, 4, 5])
def test_full_plan_digest(fdc, cfg):
    """BASELINE.json configs[2..4] in full (1e7 / 5e7 / 2e8 protons), the launch configuration bench.py
    times: the u64 grid's sha256, its sum and every counter equal the ORACLE's, computed off the GPU
    box by tests/golden/make_digests.py (which calls only oracle/) and stored as text."""
    import hashlib
    d = _digests().get(str(cfg))
    if d is None:
        pytest.skip("no stored oracle digest for config %d" % cfg)
    w = fi.workload(cfg, lazy_db=True)
    assert w.n_protons == d["protons"] and w.seed == d["seed"]
    ctx = make_ctx(fdc, w)
    ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, w.seed)
    st = ctx.fdc_get_stats()
    for k, v in d["stats"].items():
        assert st[k] == v, (k, st[k], v)
    g = ctx.fdc_get_edep_fixed()
    assert list(g.shape) == d["grid_shape"]
    assert hashlib.sha256(np.ascontiguousarray(g).tobytes()).hexdigest() == d["sha256_u64_grid"]
    if "sha256_u64_squares" in d:                      # R10 at full size
        ctx.fdc_reset()
        ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, w.seed, flags=1 | fdc.FDC_TALLY_SQUARES)
        sq = ctx.fdc_get_sq_fixed()
        assert int(sq.sum(dtype=np.uint64)) == d["squares_sum_mod_2_64"]
        assert hashlib.sha256(np.ascontiguousarray(sq).tobytes()).hexdigest() == d["sha256_u64_squares"]
        assert np.array_equal(ctx.fdc_get_edep_fixed(), g)
    if "sha256_u64_squares_by_history" in d:           # eq. (2) as defined, at full size
        ctx.fdc_reset()
        ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, w.seed, flags=1 | fdc.FDC_SQUARES_BY_HISTORY)
        assert ctx.fdc_last_call_info()["sq_history_flushes"] == 0
        sq = ctx.fdc_get_sq_fixed()
        assert int(sq.sum(dtype=np.uint64)) == d["squares_by_history_sum_mod_2_64"]
        assert hashlib.sha256(np.ascontiguousarray(sq).tobytes()).hexdigest() == d["sha256_u64_squares_by_history"]
        assert np.array_equal(ctx.fdc_get_edep_fixed(), g)
    ctx.fdc_destroy()


def test_plan_cache_switches_plans(fdc, wl2_small):
    """fdc_run keeps the last uploaded plan on the device; switching plans, a zero-proton call with another
    plan, a failed validation and a database reload in between must not leak the cached one."""
    import oracle
    w = wl2_small
    ctx = make_ctx(fdc, w)
    other = w.beamlets.copy(); other["spot_u_mm"] += 7.0; other["n_protons"] = 50
    bad = w.beamlets.copy(); bad["dir"] = (0.0, 0.1, 1.0)
    og_a, _ = oracle.run(w.phantom, w.table, w.db, w.beamlets, w.seed, n=500)
    og_b, _ = oracle.run(w.phantom, w.table, w.db, other, w.seed)

    def run(bl, n):
        ctx.fdc_reset(); ctx.fdc_run(bl, 0, n, 1, w.seed); return ctx.fdc_get_edep_fixed()

    assert np.array_equal(run(w.beamlets, 500), og_a)
    assert np.array_equal(run(w.beamlets, 500), og_a)                      # cached
    ctx.fdc_run(other, 0, 0, 1, w.seed)                                      # validated, nothing uploaded
    with pytest.raises(fdc.FdcError):
        ctx.fdc_run(other, 0, 51, 1, w.seed)                                 # 51 > other's 50 protons
    assert np.array_equal(run(w.beamlets, 500), og_a)
    assert np.array_equal(run(other, 50), og_b)
    with pytest.raises(fdc.FdcError):
        ctx.fdc_run(bad, 0, 10, 1, w.seed)
    assert np.array_equal(run(other, 50), og_b)
    ctx.fdc_load_tracks(*[np.ascontiguousarray(a) for a in (w.db.dx, w.db.dy, w.db.dz, w.db.dE, w.db.E)],
                        w.db.track_off, w.db.bin_first, w.db.e_min, w.db.e_bin)
    assert np.array_equal(run(w.beamlets, 500), og_a)
    ctx.fdc_destroy()


def test_uncertainty_follows_one_over_sqrt_n_at_scale(fdc):
    """PAPER.md Fig. 5 / L112 on config 3's plan: the mean dose uncertainty of eq. (2) halves when the
    histories quadruple, and the batch estimate (eq. (1), six seeds) is of the same size as the
    history-by-history one for the pooled histories."""
    import torch
    w = fi.workload(3)
    ctx = make_ctx(fdc, w)
    sq = fdc.FDC_TALLY_SQUARES
    res = {}
    for n, stride in ((1_000_000, 10), (4_000_000, 2)):
        ctx.fdc_reset()
        ctx.fdc_run(w.beamlets, 0, n, stride, w.seed, flags=1 | sq)
        res[n] = ctx.fdc_uncertainty_history(n)
    (u1, c1), (u4, c4) = res[1_000_000], res[4_000_000]
    assert c1 > 1000 and c4 > 1000
    assert u1 / u4 == pytest.approx(2.0, rel=0.1)
    grids = []
    ctx.fdc_reset()
    for b in range(6):
        ctx.fdc_reset()
        ctx.fdc_run(w.beamlets, 0, 1_000_000, 10, 500 + b)
        g = torch.zeros(w.phantom.hu.shape, dtype=torch.int64, device="cuda")
        ctx.fdc_get_edep_fixed(g)
        grids.append(g)
    ub, cb = ctx.fdc_uncertainty_batch(grids, 1_000_000)
    # eq. (2) on the pooled 6e6 histories: the sums of the six runs, squares included
    ctx.fdc_reset()
    for b in range(6):
        ctx.fdc_run(w.beamlets, 0, 1_000_000, 10, 500 + b, flags=1 | sq)
    uh, ch = ctx.fdc_uncertainty_history(6_000_000)
    print("mean uncertainty: 1e6 %.4f, 4e6 %.4f, ratio %.3f; six batches of 1e6: batch %.4f, history %.4f, batch/history %.3f" %
          (u1, u4, u1 / u4, ub, uh, ub / uh))
    assert 0.6 < ub / uh < 1.6
    ctx.fdc_destroy()


# ------------------------------------------------------------------ degenerate and ragged inputs, at random
from random_worlds import random_case as _random_case      # noqa: E402


def test_random_degenerate_worlds(fdc):
    rng = np.random.default_rng(20260501)
    sq, ra = fdc.FDC_TALLY_SQUARES, fdc.FDC_REALIGN_START
    import oracle
    from test_oracle_phase_space import particles
    for case in range(150):
        w = _random_case(rng)
        ctx = make_ctx(fdc, w)
        flags = int(rng.choice([0, 1, 1 | ra, 1 | fdc.FDC_NO_SORT, 1 | fdc.FDC_NO_AGGREGATE]))
        check_against_oracle(fdc, w, ctx, flags=flags)
        # every world also through the other instantiations of the kernel (small plans take the CTA-private tally by
        # default): the big-plan one, the warp-aggregating one, and grouping by start position with and without the private tally
        check_against_oracle(fdc, w, ctx, flags=(flags & ~fdc.FDC_NO_AGGREGATE) | fdc.FDC_NO_LAT)
        check_against_oracle(fdc, w, ctx, flags=(flags & ~fdc.FDC_NO_AGGREGATE) | fdc.FDC_WARP_AGGREGATE)
        # and with the material read from the tiled copy of the grid (default only for grids beyond L2), big-plan and default kernels
        check_against_oracle(fdc, w, ctx, flags=flags | fdc.FDC_MAT_TILED | (fdc.FDC_NO_LAT if case % 2 else 0))
        if case % 2 == 0:
            check_against_oracle(fdc, w, ctx, flags=(flags & ~(fdc.FDC_NO_AGGREGATE | fdc.FDC_NO_SORT)) | fdc.FDC_SORT_SPATIAL |
                                 (fdc.FDC_PRIVATE_TALLY if case % 4 == 0 else 0))
        if case % 5 == 1:                             # the same world entered from a random phase-space array
            n = 150
            ext = np.array(w.phantom.dims) * np.array(w.phantom.spacing)
            d = rng.normal(size=(n, 3)); d = (d / np.linalg.norm(d, axis=1, keepdims=True)).astype(np.float32)
            pos = (ext * rng.uniform(-0.3, 1.3, size=(n, 3))).astype(np.float32)
            ps = particles(pos, d, rng.choice(np.float32([50.0, 50.5, 51.0, 53.0, 49.0, 52.6, 30.0]), size=n))
            fl = int(rng.choice([1, 1 | ra]))
            ctx.fdc_reset()
            ctx.fdc_run_phase_space(ps, 77, w.seed, flags=fl)
            og, ost = oracle.run_phase_space(w.phantom, w.table, w.db, ps, w.seed, first_id=77, flags=fl)
            st = ctx.fdc_get_stats()
            assert np.array_equal(ctx.fdc_get_edep_fixed(), og) and all(st[k] == ost[k] for k in STAT_KEYS), case
        if case % 4 == 0:
            ctx.fdc_reset()
            ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, w.seed, flags=1 | sq)
            og, osv, osh, _ = oracle.run_sq(w.phantom, w.table, w.db, w.beamlets, w.seed, by_history=True)
            assert np.array_equal(ctx.fdc_get_edep_fixed(), og) and np.array_equal(ctx.fdc_get_sq_fixed(), osv), case
            ctx.fdc_reset()                      # by history: these worlds have deflections beyond 90 degrees, i.e. re-entered voxels
            ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, w.seed, flags=1 | fdc.FDC_SQUARES_BY_HISTORY | (fdc.FDC_MAT_TILED if case % 8 == 0 else 0))
            assert np.array_equal(ctx.fdc_get_edep_fixed(), og) and np.array_equal(ctx.fdc_get_sq_fixed(), osh), case
        ctx.fdc_destroy()


# ------------------------------------------------------------------ R15: histories with secondaries
def test_secondaries_bit_exact(fdc):
    """Hand-made histories and 60 random degenerate worlds with random secondary tables: grid, squares and
    counters equal the oracle's with every flag; table validation; the table goes away with n_sec = 0."""
    import oracle
    from random_worlds import random_case
    from test_oracle_secondaries import db_with_secondaries, random_secondaries
    from test_oracle_pins import table_uniform, uniform_phantom
    sq = fdc.FDC_TALLY_SQUARES

    def gpu_vs_oracle(ctx, w, db, sec, flags):
        ctx.fdc_reset()
        ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, w.seed, flags=flags)
        if flags & sq:
            og, osv, osh, ost = oracle.run_secondaries(w.phantom, w.table, db, sec, w.beamlets, w.seed, flags=flags & 33, squares=True)
            assert np.array_equal(ctx.fdc_get_sq_fixed(), osv)
            # the same histories squared as eq. (2) defines them: parent and secondaries of a history summed per voxel first
            ctx.fdc_reset()
            ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, w.seed, flags=flags | fdc.FDC_SQUARES_BY_HISTORY)
            assert np.array_equal(ctx.fdc_get_sq_fixed(), osh) and np.array_equal(ctx.fdc_get_edep_fixed(), og)
        else:
            og, ost = oracle.run_secondaries(w.phantom, w.table, db, sec, w.beamlets, w.seed, flags=flags & 33)
        st = ctx.fdc_get_stats()
        assert np.array_equal(ctx.fdc_get_edep_fixed(), og)
        for k in STAT_KEYS:
            assert st[k] == ost[k], (k, st[k], ost[k])

    ph = uniform_phantom(32, 2.0)
    prim = [[(0, 0, 1.0, 1.0)] * 10, [(0.1, 0, 1.0, 0.8)] * 7]
    secs = [(0, 2, [(0.6, 0, 0.8, 2.0)] * 2), (0, 6, [(0, 0.6, 0.8, 3.0)]), (0, 6, [(0, -1.0, 0, 0.5)]), (1, 0, [(1.0, 0, 0, 0.25)] * 3)]
    db, sec = db_with_secondaries(prim, secs)
    for e0 in (100.0, 97.5, 93.0):
        w = fi.Workload("sec", ph, table_uniform(1.0), db, fi.single_beamlet((31.0, 33.0, 1.0), e0, 1.5, 400), 400, 5)
        ctx = make_ctx(fdc, w)
        ctx.fdc_set_secondaries(*sec)
        mt = fdc.FDC_MAT_TILED
        for flags in (1, 0, 1 | sq, 1 | fdc.FDC_NO_SORT, 1 | fdc.FDC_NO_AGGREGATE, 1 | fdc.FDC_REALIGN_START, 1 | mt, 1 | mt | sq, 1 | mt | fdc.FDC_NO_LAT,
                      1 | mt | fdc.FDC_NO_AGGREGATE):
            gpu_vs_oracle(ctx, w, db, sec, flags)
        ctx.fdc_set_secondaries(np.zeros(db.n_tracks + 1, np.uint32), [], [])          # removed: the plain run again
        ctx.fdc_reset(); ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, w.seed)
        g0, _ = oracle.run(w.phantom, w.table, db, w.beamlets, w.seed)
        assert np.array_equal(ctx.fdc_get_edep_fixed(), g0)
        bad_first = sec[0].copy(); bad_first[-1] += 1
        for args in ((bad_first, sec[1], sec[2]), (sec[0], np.zeros_like(sec[1]), sec[2]), (sec[0], sec[1], sec[2] + 100)):
            with pytest.raises(fdc.FdcError) as e:
                ctx.fdc_set_secondaries(*args)
            assert e.value.code == fdc.FDC_EINVAL
        ctx.fdc_destroy()
    rng = np.random.default_rng(99)
    for case in range(60):
        w0 = random_case(rng)
        db2, sec2 = random_secondaries(rng, w0.db, None)
        w = fi.Workload("secfuzz", w0.phantom, w0.table, db2, w0.beamlets, w0.n_protons, w0.seed)
        ctx = make_ctx(fdc, w)
        if len(sec2[1]):
            ctx.fdc_set_secondaries(*sec2)
        gpu_vs_oracle(ctx, w, db2, sec2, int(rng.choice([0, 1, 1 | sq, 1 | fdc.FDC_REALIGN_START, 1 | fdc.FDC_NO_AGGREGATE])) | (fdc.FDC_MAT_TILED if case % 2 else 0))
        ctx.fdc_destroy()


def test_synthetic_secondaries_on_the_configs(fdc, wl2_small, wl3_small):
    """fdc_inputs.add_secondaries (the recipe bench.py's secondaries leg uses) on the reduced configs 2 and 3."""
    import oracle
    for w0 in (wl2_small, wl3_small):
        db2, sec = fi.add_secondaries(w0.db, 42)
        assert len(sec[1]) > 0.5 * w0.db.n_tracks * (w0.db.n_steps > 0)
        w = fi.Workload("synsec", w0.phantom, w0.table, db2, w0.beamlets, w0.n_protons, w0.seed)
        ctx = make_ctx(fdc, w)
        ctx.fdc_set_secondaries(*sec)
        ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, w.seed)
        og, ost = oracle.run_secondaries(w.phantom, w.table, db2, sec, w.beamlets, w.seed)
        st = ctx.fdc_get_stats()
        assert np.array_equal(ctx.fdc_get_edep_fixed(), og)
        for k in STAT_KEYS:
            assert st[k] == ost[k], (k, st[k], ost[k])
        g0, s0 = oracle.run(w0.phantom, w0.table, w0.db, w0.beamlets, w0.seed)
        assert ost["proton_steps"] > s0["proton_steps"] and ost["q_replayed"] > s0["q_replayed"]
        # squares with secondaries: per stay (R10's reading) and per history (eq. (2) as defined) both equal the oracle's; here
        # the two differ by percents of the tally (a parent and its secondary share the branch voxel), R10
        _, osv, osh, _ = oracle.run_secondaries(w.phantom, w.table, db2, sec, w.beamlets, w.seed, squares=True)
        ctx.fdc_reset(); ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, w.seed, flags=1 | fdc.FDC_TALLY_SQUARES)
        assert np.array_equal(ctx.fdc_get_sq_fixed(), osv)
        ctx.fdc_reset(); ctx.fdc_run(w.beamlets, 0, w.n_protons, 1, w.seed, flags=1 | fdc.FDC_SQUARES_BY_HISTORY)
        assert np.array_equal(ctx.fdc_get_sq_fixed(), osh) and np.array_equal(ctx.fdc_get_edep_fixed(), og)
        assert ctx.fdc_last_call_info()["sq_history_flushes"] == 0
        gap = 1.0 - float(osv.sum(dtype=np.float64)) / float(osh.sum(dtype=np.float64))
        assert 0.005 < gap < 0.08, gap
        ctx.fdc_destroy()


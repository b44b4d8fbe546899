"""Pins of the oracle's sum-of-squares tallies and uncertainty estimates (R10; PAPER.md:L73,
§2.4 eq. (1), (2), L92).  None of this needs a GPU.

U1  closed forms of eq. (1) and eq. (2) on hand-made numbers
U2  one history: squares == (energy >> 8)^2 voxel by voxel; N identical histories: N times that, and
    eq. (2) gives (numerically) zero spread
U3  brute force: per-history per-voxel totals rebuilt in numpy from the deposit trace, squared and
    summed, equal sq_by_history exactly; by_visit <= by_history, equal for histories that never
    re-enter a voxel
U4  additivity over proton ranges (exact integers)
U5  statistics: mean uncertainty falls as 1/sqrt(N) (Fig. 5); history-by-history and
    batch estimates agree within sampling error when the database is not over-used
"""
import numpy as np
import pytest

import fdc_inputs as fi
import oracle
from test_oracle_pins import hand_db, table_uniform, uniform_phantom


def sq_op(e):
    e = np.asarray(e, dtype=np.uint64) >> np.uint64(8)
    return e * e


# ------------------------------------------------------------------ U1
def test_eq1_eq2_closed_forms():
    q = 2 ** 24                                            # 1 MeV in grid quanta
    # eq. (2): four histories leave 1, 1, 3, 3 MeV in a voxel: mean 2, <e^2> = 5, var of the mean = (5 - 4) / 3
    S1 = np.array([8 * q], dtype=np.uint64); S2 = np.array([20 * 2 ** 32], dtype=np.uint64)
    m, s = oracle.sigma_history(S1, S2, 4)
    assert m[0] == 2.0 and s[0] == np.sqrt(1.0 / 3.0)
    # a voxel no history touched
    m, s = oracle.sigma_history(np.zeros(1, np.uint64), np.zeros(1, np.uint64), 10)
    assert m[0] == 0.0 and s[0] == 0.0
    # eq. (1): batches 1, 2, 3 MeV: mean 2, sum of squared deviations 2, n (n - 1) = 6
    g = [np.array([k * q], dtype=np.uint64) for k in (1, 2, 3)]
    m, s = oracle.sigma_batch(g)
    assert m[0] == 2.0 and s[0] == np.sqrt(2.0 / 6.0)
    # two batches a, b: sigma = |a - b| / 2
    m, s = oracle.sigma_batch([np.array([5 * q], np.uint64), np.array([9 * q], np.uint64)])
    assert m[0] == 7.0 and s[0] == 2.0
    # mean uncertainty: only voxels above half the maximum DOSE (energy / density) are averaged
    mean = np.array([10.0, 4.0, 6.0, 1.0]); sig = np.array([1.0, 2.0, 0.6, 5.0]); rho = np.array([1.0, 1.0, 0.5, 1.0], np.float32)
    val, cnt = oracle.mean_uncertainty(mean, sig, rho)      # doses 10, 4, 12, 1 -> voxels 0 and 2
    assert cnt == 2 and val == pytest.approx((0.1 + 0.1) / 2)


# ------------------------------------------------------------------ U2
def test_single_and_identical_histories():
    ph = uniform_phantom(16, 1.0)
    db = hand_db([[(0, 0, 1.0, 0.5 + 0.25 * k) for k in range(10)]])
    bl = fi.single_beamlet((5.5, 6.5, 0.25), 100.0, 0.0, 1)
    g, sv, sh, st = oracle.run_sq(ph, table_uniform(1.0), db, bl, 7, flags=0)
    assert st["stopped"] == 1 and g.sum() == st["q_replayed"]
    assert np.array_equal(sv, sq_op(g)) and np.array_equal(sh, sq_op(g))       # straight line: every voxel visited once
    N = 37
    blN = fi.single_beamlet((5.5, 6.5, 0.25), 100.0, 0.0, N)
    gN, svN, shN, _ = oracle.run_sq(ph, table_uniform(1.0), db, blN, 7, flags=0)
    assert np.array_equal(gN, g * np.uint64(N)) and np.array_equal(svN, sv * np.uint64(N)) and np.array_equal(shN, sh * np.uint64(N))
    m, s = oracle.sigma_history(gN, shN, N)
    hit = g > 0
    # identical histories: the spread is only the 2^-16 MeV truncation of the operand
    assert np.all(s[hit] / m[hit] < 2e-3 / np.sqrt(N))
    assert np.all(m[hit] == g[hit].astype(np.float64) * 2.0 ** -24)


# ------------------------------------------------------------------ U3
def brute_force_history_squares(w, first, n, stride=1):
    """eq. (2)'s sum of D_i^2, from the definition: D_i = everything history i left in the voxel."""
    out = np.zeros(w.phantom.hu.size, dtype=np.uint64)
    reentered = 0
    for m in range(n):
        i = first + m * stride
        _, _, (vox, share, step), _ = oracle.run_trace(w.phantom, w.table, w.db, w.beamlets, w.seed, first=i, n=1)
        if len(vox) == 0:
            continue
        uv, inv = np.unique(vox, return_inverse=True)
        tot = np.zeros(len(uv), dtype=np.uint64)
        np.add.at(tot, inv, share)
        out[uv] += sq_op(tot)
        runs = 1 + int(np.count_nonzero(np.diff(vox.astype(np.int64))))          # maximal runs of one voxel in deposit order
        reentered += int(runs > len(uv))
    return out.reshape(w.phantom.hu.shape), reentered


@pytest.mark.parametrize("which", ["wl2_small", "wl3_small"])
def test_squares_brute_force(which, request):
    w = request.getfixturevalue(which)
    n = 150
    stride = max(1, w.n_protons // n)
    g, sv, sh, st = oracle.run_sq(w.phantom, w.table, w.db, w.beamlets, w.seed, first=0, n=n, stride=stride)
    g0, st0 = oracle.run(w.phantom, w.table, w.db, w.beamlets, w.seed, first=0, n=n, stride=stride)
    assert np.array_equal(g, g0) and all(st[k] == st0[k] for k in st0)               # the extra tallies change nothing
    bf, reentered = brute_force_history_squares(w, 0, n, stride)
    assert np.array_equal(sh, bf)
    assert np.all(sv <= sh)
    if reentered == 0:
        assert np.array_equal(sv, sh)
    # the by-visit reading differs only through re-entries: a small part of the tally
    assert float(sh.sum() - sv.sum()) <= 0.02 * float(sh.sum())


def test_no_reentry_means_equal(wl1_small):
    """Azimuth off, point source, water: still scattered tracks; wherever by_visit != by_history the
    history came back to a voxel it had left."""
    w = wl1_small
    g, sv, sh, _ = oracle.run_sq(w.phantom, w.table, w.db, w.beamlets, w.seed, n=300, flags=0)
    assert np.all(sv <= sh) and sv.sum() > 0.98 * sh.sum()
    # Cauchy-Schwarz on the truncated operands: (sum e')^2 <= n_hist * sum e'^2, with sum e' >= (sum e >> 8) - n_hist
    lhs = (g >> np.uint64(8)).astype(np.float64) - 300.0
    assert np.all(np.maximum(lhs, 0.0) ** 2 <= 300.0 * sh.astype(np.float64) * (1 + 1e-12))


# ------------------------------------------------------------------ U4
def test_squares_additive(wl3_small):
    w = wl3_small
    a = oracle.run_sq(w.phantom, w.table, w.db, w.beamlets, w.seed, first=0, n=400)
    b = oracle.run_sq(w.phantom, w.table, w.db, w.beamlets, w.seed, first=400, n=600)
    c = oracle.run_sq(w.phantom, w.table, w.db, w.beamlets, w.seed, first=0, n=1000)
    for k in range(3):
        assert np.array_equal(a[k] + b[k], c[k])


# ------------------------------------------------------------------ U5
def test_uncertainty_scaling_and_batch_agreement():
    """Config-1 geometry with a sigma = 6 mm beam so that many voxels share the dose.  The database
    (4000 tracks) is larger than the number of histories, so re-use does not correlate them."""
    base = fi.workload(1, n_protons=1, tracks_per_bin=4000)
    rho = oracle.density(base.phantom, base.table)

    def run(n, seed):
        bl = fi.single_beamlet((64.0, 64.0, 0.0), 100.0, 6.0, n)
        g, sv, sh, _ = oracle.run_sq(base.phantom, base.table, base.db, bl, seed, by_history=False)
        return g, sv

    N = 3000
    g1, s1 = run(N, 11)
    g4, s4 = run(4 * N, 12)
    u1, c1 = oracle.mean_uncertainty(*oracle.sigma_history(g1, s1, N), rho)
    u4, c4 = oracle.mean_uncertainty(*oracle.sigma_history(g4, s4, 4 * N), rho)
    assert c1 > 20 and c4 > 20
    assert u1 / u4 == pytest.approx(2.0, rel=0.15)                                # 1/sqrt(N)
    # batch method with 6 batches of N, compared with history-by-history on the pooled 6N
    batches = [run(N, 100 + b) for b in range(6)]
    mb, sb = oracle.sigma_batch([b[0] for b in batches])
    pooled_g = sum(b[0] for b in batches); pooled_s = sum(b[1] for b in batches)
    mh, sh = oracle.sigma_history(pooled_g, pooled_s, 6 * N)
    # sigma_batch is of the mean of 6 batch totals (per batch of N histories); per history divide by N
    ub, _ = oracle.mean_uncertainty(mb / N, sb / N, rho)
    uh, _ = oracle.mean_uncertainty(mh, sh, rho)
    assert ub / uh == pytest.approx(1.0, rel=0.35)       # 5 degrees of freedom per voxel, averaged over tens of voxels


@pytest.mark.parametrize("cfg,n,tpb", [(2, 20000, 300), (3, 23520, 50)])
def test_by_visit_gap_is_measured_with_and_without_secondaries(cfg, n, tpb):
    """DESIGN.md R10 / reading A23, measured: how far the per-stay tally (what the fast kernel squares) falls short of
    eq. (2)'s per-history D_i, on reduced configs 2 and 3, primaries only and with the synthetic
    secondaries of fdc_inputs.add_secondaries (parent and secondary both deposit in the branch voxel and are squared
    separately).  Bounds enforced: primaries only, gap <= 1e-3 of the tally and the mean relative uncertainty
     changes by <= 1e-3 of itself; with secondaries, gap <= 6 % and the mean relative uncertainty is low
    by <= 4 %.  by_visit <= by_history voxel by voxel in every case (a sum of squares of parts never exceeds the square
    of the sum)."""
    import fdc_inputs as fi
    w = fi.workload(cfg, n_protons=n, tracks_per_bin=tpb)
    rho = oracle.density(w.phantom, w.table)
    res = {}
    for with_sec in (False, True):
        if with_sec:
            db2, sec = fi.add_secondaries(w.db, 1000 + cfg)
            assert len(sec[1]) > 0
            g, sv, sh, st = oracle.run_secondaries(w.phantom, w.table, db2, sec, w.beamlets, w.seed, squares=True)
        else:
            g, sv, sh, st = oracle.run_sq(w.phantom, w.table, w.db, w.beamlets, w.seed)
        assert np.all(sv <= sh)
        gap = float(sh.sum() - sv.sum()) / float(sh.sum())
        rel = [oracle.mean_uncertainty(*oracle.sigma_history(g, sq, n), rho)[0] for sq in (sv, sh)]
        res[with_sec] = (gap, rel[0] / rel[1])
    assert 0.0 <= res[False][0] <= 1e-3 and 1.0 - 1e-3 <= res[False][1] <= 1.0
    assert 0.005 <= res[True][0] <= 0.06 and 0.96 <= res[True][1] <= 1.0

#!/usr/bin/env python
"""bench.py -- measurement of the track-repeating hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl fdc|reference] [--config C]

One "step" = one pass of the whole hot path over one batch of synthetic input: zero the grid, sample + select
tracks + group + transport + deposit + convert to Gy, for every proton of the workload.  The workload at N = 1
is the LARGEST single-GPU configuration, BASELINE.json configs[4] (config 5: 512 x 512 x 256 voxels at 1 mm,
three fields x 40 layers x 81 spots, 2e8 protons, 2e4 tracks per 1 MeV bin), generated from seeds by fdc_inputs
(synthetic); `--config C` selects another.  Prints ONE JSON line (rank 0).

`value`        protons/s with every input already resident in HBM (CUDA events per step, max over ranks).
`e2e`          the same through the public call with HOST buffers: beam plan H2D (a byte-different, equivalent plan
               every step, so the library's plan cache cannot skip the upload) and dose grid D2H into pinned host
               memory inside the timed region; the byte counts are the library's own (fdc_last_call_info).
               `e2e.cold` also re-creates the context and re-loads phantom and database from host memory each step.
`roofline`     the transport+deposit kernel against max(track bytes / HBM peak, deposits / measured u64-red rate)
               (north_star); denominators measured in this run by libfdcpeaks.so, including the red rate over this
               workload's ACTUAL address multiset (traced by the instrumented kernel, replayed at saturation).
`per_config`   the other four configs, same process, same L2 flush, same warm-up: ms_per_step, kernel_ms,
               roofline.frac, deposits ... (N = 1 only).
`cpu_baseline` the oracle, as it stands, on this box's host cores on a strided proton subset.

--impl reference times the oracle (tier framing: the reference arm is the oracle); there is no CPU fallback in the
product arm: without libfdc.so or a B200 it raises.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

L2_FLUSH_BYTES = 512 << 20          # > 126 MB L2
STEP_RECORD_BYTES = 20              # dx,dy,dz,dE,E float32 per step (north_star (1))
HEADLINE_CONFIG = 5


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def _static_counts(cfg):
    """ncu figures that cannot be measured live: profiles/r03_counts.csv holds one row per k_transport launch of one timed
    step of every config (ncu --metrics, profiles/r03_README.md), with the commit of the kernel.  Returned: the step's sums
    (DRAM bytes, warp instructions, kernel time under ncu) and the TIME-WEIGHTED means over its launches of the L2 tag-request
    rate and the issue-active share (not one launch of six)."""
    p = os.path.join(ROOT, "profiles", "r03_counts.csv")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        lines = [l for l in f.read().splitlines() if l.strip() and not l.startswith("#")]
    hdr = lines[0].split(",")
    rows = [dict(zip(hdr, l.split(","))) for l in lines[1:]]
    rows = [r for r in rows if r["config"].strip() == str(cfg)]
    if not rows:
        return None
    ms = [float(r["kernel_ms_under_ncu"]) for r in rows]
    tot = sum(ms)
    wmean = lambda k: sum(float(r[k]) * t for r, t in zip(rows, ms)) / tot      # noqa: E731
    dram = sum(float(r["dram_bytes_read"]) + float(r["dram_bytes_write"]) for r in rows)
    return {"launch": "all %d k_transport launches of one timed step" % len(rows), "n_launches": len(rows),
            "dram_bytes": dram / len(rows), "dram_bytes_per_step": dram,
            "warp_instructions": sum(float(r["warp_instructions"]) for r in rows) / len(rows),
            "warp_instructions_per_step": sum(float(r["warp_instructions"]) for r in rows),
            "kernel_ms_under_ncu": tot / len(rows), "kernel_ms_per_step_under_ncu": tot,
            "l2_tag_pct_time_weighted": wmean("l2_tag_requests_avg_pct"), "l2_tag_pct_hottest_slice_time_weighted": wmean("l2_tag_requests_max_pct"),
            "issue_active_pct_time_weighted": wmean("issue_active_pct"), "warps_active_pct_time_weighted": wmean("warps_active_pct"),
            "l2_red_requests_per_step": sum(float(r["l2_red_requests"]) for r in rows),
            "l2_red_lookup_miss_share": sum(float(r["l2_red_sectors_lookup_miss"]) for r in rows) / sum(float(r["l2_red_sectors"]) for r in rows),
            "per_launch_ms": ms, "source": "profiles/r03_counts.csv", "kernel_commit": rows[0]["kernel_commit"].strip()}


class ClockSampler:
    """SM clock + throttle reasons sampled through NVML every few ms while the timed region runs."""
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}

    def __init__(self, index, period_s=0.01):
        self.index, self.period, self.samples, self.stop_flag, self.t, self.err = index, period_s, [], False, None, None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            try:                                    # CUDA_VISIBLE_DEVICES may renumber: go by UUID
                import torch
                self.h = pynvml.nvmlDeviceGetHandleByUUID("GPU-" + str(torch.cuda.get_device_properties(self.index).uuid))
            except Exception:                       # noqa: BLE001
                self.h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception as e:                      # noqa: BLE001 -- reported in the JSON line
            self.err = "nvml unavailable: %s" % e
            return
        self.t = threading.Thread(target=self._poll, daemon=True)
        self.t.start()

    def _poll(self):
        nv = self.nv
        while not self.stop_flag:
            try:
                mhz = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                try:
                    rs = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:                   # noqa: BLE001 -- older binding name
                    rs = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                pw = nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0
                self.samples.append((float(mhz), int(rs), pw))
            except Exception as e:                  # noqa: BLE001
                self.err = str(e)
                break
            time.sleep(self.period)

    def stop(self):
        self.stop_flag = True
        if self.t is not None:
            self.t.join(timeout=2)
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": None, "samples": 0, "reasons": [self.err or "no samples"]}
        sm = [s[0] for s in self.samples]
        bits = 0
        for s in self.samples:
            bits |= s[1]
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": self.max_mhz, "sm_mhz_min": min(sm), "sm_mhz_peak": max(sm),
                "power_w_max": max(s[2] for s in self.samples), "samples": len(sm),
                "reasons": sorted(n for b, n in self.REASONS.items() if bits & b)}


def make_workload(cfg, gpus):
    """configs[cfg-1]; for N > 1 (weak scaling) the plan holds N x the protons and rank r runs the r-th contiguous
    range of the global proton index space.  Only the energy bins the plan touches are generated (same tracks)."""
    import fdc_inputs as fi
    base = fi._FULL[cfg]
    w = fi.workload(cfg, n_protons=base * gpus, lazy_db=True)
    return w, base


# --------------------------------------------------------------------------- reference arm (oracle)
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    w, per_rank = make_workload(args.config, 1)
    n_sub = min(args.ref_sample, w.n_protons)
    K = max(1, w.n_protons // n_sub)
    times, steps, deps = [], 0, 0
    for it in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        g, st = oracle.run(w.phantom, w.table, w.db, w.beamlets, w.seed, first=(it % K), n=n_sub, stride=K)
        oracle.to_gy(g, w.phantom, w.table)
        dt = time.perf_counter() - t0
        if it >= args.warmup:
            times.append(dt); steps += st["proton_steps"]; deps += st["deposits"]
    tot = sum(times)
    val = n_sub * args.steps / tot
    sample = "every %d-th proton of %s (%d protons per step), 1 thread" % (K, w.name, n_sub)
    out = {"impl": "reference", "metric": "protons_per_sec", "value": val, "unit": "protons/s", "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f32+u64", "data": "synthetic",
           "steps_per_sec": steps / tot, "deposits_per_sec": deps / tot,
           "config": {"workload": w.name, "protons_per_step": n_sub, "sample": sample},
           "cpu_baseline": {"value": val, "unit": "protons/s", "cores": 1, "kind": "oracle", "sample": sample},
           "e2e": {"value": val, "unit": "protons/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))
    return 0


def oracle_all_cores(w, n_per_thread):
    """BASELINE.md §3's all-core figure: the oracle as it stands (one call = one thread) on T = os.cpu_count() disjoint
    strided proton subsets of the plan at once, one Python thread per call (ctypes releases the GIL).  Each call has its
    own grid; an integer sum of them would be the grid of the union, so this is the proton-range threading the
    definition allows.  Returns the cpu_baseline-style dict."""
    import concurrent.futures as cf
    import oracle
    T = os.cpu_count() or 1
    n = max(1, min(n_per_thread, w.n_protons // T))
    stride = max(1, w.n_protons // (n * T)) * T
    t0 = time.perf_counter()
    with cf.ThreadPoolExecutor(T) as ex:
        list(ex.map(lambda t: oracle.run(w.phantom, w.table, w.db, w.beamlets, w.seed, first=t, n=n, stride=stride)[1], range(T)))
    dt = time.perf_counter() - t0
    return {"value": n * T / dt, "unit": "protons/s", "cores": T, "kind": "oracle",
            "sample": "%d threads, each every %d-th proton of %s from its own offset (%d protons per thread, %.1f s)" % (T, stride, w.name, n, dt)}


def oracle_full(w):
    """The oracle in full on a small config (configs 1-2), one thread."""
    import oracle
    t0 = time.perf_counter()
    og, ost = oracle.run(w.phantom, w.table, w.db, w.beamlets, w.seed, first=0, n=w.n_protons, stride=1)
    dt = time.perf_counter() - t0
    return {"value": w.n_protons / dt, "unit": "protons/s", "cores": 1, "kind": "oracle", "seconds": dt,
            "steps_per_sec": ost["proton_steps"] / dt, "sample": "the whole plan of %s (%d protons), single thread" % (w.name, w.n_protons)}


# --------------------------------------------------------------------------- product arm
class Bench:
    """One workload resident on one GPU: context, database, buffers, the step function and its timers."""

    def __init__(self, cfg, world, rank, local, fdc, torch, dist):
        from paper_1011_2188_b200 import multi
        self.fdc, self.torch, self.dist, self.multi = fdc, torch, dist, multi
        self.cfg, self.world, self.rank, self.local = cfg, world, rank, local
        self.w, self.per_rank = make_workload(cfg, world)
        w = self.w
        self.first, self.n_mine = multi.shard_range(w.n_protons, rank, world)
        self.dev = torch.device("cuda", local)
        hu_d = torch.from_numpy(np.ascontiguousarray(w.phantom.hu)).to(self.dev)
        self.ctx = fdc.Fdc(hu_d, w.phantom.spacing, w.table, device=local)
        self.host_arrs = [np.ascontiguousarray(a) for a in (w.db.dx, w.db.dy, w.db.dz, w.db.dE, w.db.E)]
        self.ctx.fdc_load_tracks(*self.host_arrs, w.db.track_off, w.db.bin_first, w.db.e_min, w.db.e_bin)
        self.dose_d = torch.zeros(w.phantom.hu.shape, dtype=torch.float32, device=self.dev)
        self.flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=self.dev)
        self.flags = fdc.FDC_RANDOM_AZIMUTH
        self.n_vox = int(np.prod(w.phantom.hu.shape))

    def barrier(self):
        if self.world > 1:
            self.dist.barrier()
        self.torch.cuda.synchronize()

    def one_step(self, dose_out, beamlets=None, flags=None):
        bl = self.w.beamlets if beamlets is None else beamlets
        self.multi.sharded_step(self.ctx, bl, self.first, self.n_mine, self.w.seed, self.flags if flags is None else flags,
                                dose_out, self.world)

    def timed(self, n_steps, dose_out, infos=None, flags=None):
        """n_steps steps, each after an L2 flush, each bracketed by barrier + synchronize; CUDA events; max over ranks."""
        torch, tot = self.torch, 0.0
        for _ in range(n_steps):
            self.flush.fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            self.barrier()
            e0.record()
            self.one_step(dose_out, flags=flags)
            e1.record()
            self.barrier()
            ms = e0.elapsed_time(e1)
            if self.world > 1:
                t = torch.tensor([ms], device=self.dev); self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX); ms = float(t.item())
            tot += ms
            if infos is not None:
                infos.append(self.ctx.fdc_last_call_info())
        return tot

    def red_ceilings(self, peaks_cache):
        """Denominators of the L2-atomic roofline, measured now: u64 red rate over uniformly random
        addresses in an L2-resident buffer and in a buffer the size of this grid; and over this workload's ACTUAL
        address multiset: a strided subset of the plan runs through the instrumented kernel (FDC_DIAG_REDS), which
        records the voxel index of every reduction it sends; libfdcpeaks.so replays that list at saturation, in
        trace order and shuffled.  Also the count of reductions the kernel really sends for the whole plan."""
        from paper_1011_2188_b200 import peaks
        fdc, torch, ctx, w = self.fdc, self.torch, self.ctx, self.w
        l2_bytes = min(self.n_vox * 8, 64 << 20)
        key = ("l2", l2_bytes)
        if key not in peaks_cache:
            peaks_cache[key] = peaks.red_u64(self.local, l2_bytes, 1 << 30, 0)
        red_l2 = peaks_cache[key]
        key = ("fp", self.n_vox * 8)
        if key not in peaks_cache:
            peaks_cache[key] = red_l2 if self.n_vox * 8 <= (64 << 20) else peaks.red_u64(self.local, self.n_vox * 8, 1 << 28, 0)
        red_fp = peaks_cache[key]
        # whole plan once through the instrumented kernel, no trace buffer: reductions really sent
        ctx.fdc_reset()
        ctx.fdc_run(w.beamlets, self.first, self.n_mine, 1, w.seed, flags=self.flags | fdc.FDC_DIAG_REDS)
        reds_sent = ctx.fdc_last_call_info()["reds_sent"]
        # strided subset with the trace on
        n_sub = min(self.n_mine, max(1, int(64e6 * self.n_mine / max(reds_sent, 1))))      # about 64e6 traced addresses
        K = max(1, self.n_mine // n_sub)
        cap = int(min(1 << 28, 2 * reds_sent * n_sub // self.n_mine + (1 << 20)))
        trace = torch.empty(cap, dtype=torch.int32, device=self.dev)
        ctx.fdc_trace_reds(trace)
        ctx.fdc_reset()
        ctx.fdc_run(w.beamlets, self.first, n_sub, K, w.seed, flags=self.flags | fdc.FDC_DIAG_REDS)
        n_tr = ctx.fdc_last_call_info()["reds_traced"]
        ctx.fdc_trace_reds(None)
        ctx.fdc_reset()
        passes = max(1, int((1 << 29) // max(n_tr, 1)))
        rep_trace = peaks.red_replay(self.local, trace, n_tr, self.n_vox, passes, False)
        rep_shuf = peaks.red_replay(self.local, trace, n_tr, self.n_vox, passes, True)
        del trace
        key = ("c4", l2_bytes)
        if key not in peaks_cache:
            peaks_cache[key] = peaks.red_u64(self.local, l2_bytes, 1 << 30, 1)
        red_c4 = peaks_cache[key]
        return {"peak_gred_s": red_l2 / 1e9, "uniform_at_grid_footprint_gred_s_nonbinding": red_fp / 1e9,
                "peak_4_neighbour_words_gred_s": red_c4 / 1e9,
                "peak_actual_multiset_gred_s": rep_shuf / 1e9, "peak_actual_multiset_trace_order_gred_s": rep_trace / 1e9,
                "multiset_sample": "every %d-th proton (%d protons, %d reductions traced, replayed %d x)" % (K, n_sub, n_tr, passes),
                "reds_sent_per_step": int(reds_sent), "grid_mib": self.n_vox * 8 >> 20}

    def roofline(self, infos, st, tot_ms, n_steps, ceilings, clk):
        hbm_gbs, peak_src = _peaks()
        tr_ms = float(np.mean([k["transport_ms"] for k in infos]))
        if not tr_ms > 0.0:
            raise RuntimeError("the library reported no transport time for the timed steps")
        t_track = st["proton_steps"] * STEP_RECORD_BYTES / (hbm_gbs * 1e9)
        # the roofline fraction divides what the kernel really ISSUES (reds_sent: merged shares never reach
        # memory) by the ceiling of this workload's own address multiset (its traced voxel indices replayed at saturation)
        t_atomic = ceilings["reds_sent_per_step"] / (ceilings["peak_actual_multiset_gred_s"] * 1e9)
        t_alg_uniform = st["deposits"] / (ceilings["peak_gred_s"] * 1e9)         # rounds 1-2's definition, kept as a labelled extra
        bound_atomic = t_atomic >= t_track
        # transport launches per step: the library cuts a run at 2^25 protons and at field boundaries; each launch comes with 5
        # sort kernels, and the step ends with one Gy kernel
        n_chunks = max(1, (int(infos[-1]["launches"]) - 1) // 6) if self.world == 1 else max(1, int(infos[-1]["launches"]) // 6)
        la = dict(ceilings)
        la.update({"achieved_gred_s": st["deposits"] / (tr_ms * 1e-3) / 1e9,
                   "sent_gred_s": ceilings["reds_sent_per_step"] / (tr_ms * 1e-3) / 1e9,
                   "sent_frac_of_peak": ceilings["reds_sent_per_step"] / (tr_ms * 1e-3) / (ceilings["peak_gred_s"] * 1e9),
                   "sent_frac_of_actual_multiset_peak": ceilings["reds_sent_per_step"] / (tr_ms * 1e-3) / (ceilings["peak_actual_multiset_gred_s"] * 1e9),
                   "algorithmic_deposits_over_uniform_peak": t_alg_uniform / (tr_ms * 1e-3),
                   "peak_source": "libfdcpeaks.so, measured in this run: u64 red from 2 x 1024 threads per SM.  peak_actual_multiset = this "
                                  "workload's traced voxel indices replayed shuffled at saturation (trace_order: as the kernel's warps sent "
                                  "them): THE DENOMINATOR OF frac, whose numerator is reds_sent (reductions really issued).  peak = uniform "
                                  "random addresses over min(grid, 64 MiB) (L2-resident); peak_4_neighbour_words = the 32 lanes of a warp on "
                                  "4 neighbouring words (what clustered addresses can reach: frac is not 'of the hardware'); "
                                  "uniform_at_grid_footprint = uniform over the whole grid, NOT a ceiling for this clustered stream.  "
                                  "achieved_gred_s / algorithmic_deposits_over_uniform_peak count ALGORITHMIC deposits (rounds 1-2's frac)"})
        roof = {"bound": "l2_atomic" if bound_atomic else "hbm",
                "achieved": la["sent_gred_s"] if bound_atomic else st["proton_steps"] * STEP_RECORD_BYTES / (tr_ms * 1e-3) / 1e9,
                "peak": ceilings["peak_actual_multiset_gred_s"] if bound_atomic else hbm_gbs,
                "unit": "Gred/s" if bound_atomic else "GB/s",
                "frac": max(t_track, t_atomic) / (tr_ms * 1e-3),
                "traffic": None,
                "kernel": "k_transport", "kernel_ms": tr_ms, "launches_per_step": n_chunks,
                "kernel_share_of_step": tr_ms * n_steps / tot_ms,
                "t_track_ms": t_track * 1e3, "t_atomic_ms": t_atomic * 1e3,
                "hbm": {"achieved_gbs": st["proton_steps"] * STEP_RECORD_BYTES / (tr_ms * 1e-3) / 1e9, "peak_gbs": hbm_gbs, "peak_source": peak_src},
                "l2_atomic": la,
                "algorithmic": {"proton_steps": st["proton_steps"], "deposits": st["deposits"], "bytes_per_step": STEP_RECORD_BYTES,
                                "deposits_per_s": st["deposits"] / (tr_ms * 1e-3),
                                "note": "throughput in ALGORITHMIC deposits (non-zero (step, voxel) shares, R8) over the kernel time of "
                                        "the step's launches.  The kernel merges the shares one proton leaves in one voxel into a single "
                                        "reduction, so it SENDS fewer (reds_sent_per_step); roofline.achieved / frac count those"}}
        sc = _static_counts(self.cfg)
        if sc is not None:
            mhz = (clk or {}).get("sm_mhz") or 1965.0
            peak_issue = 148 * 4 * mhz * 1e6
            roof["traffic"] = sc["dram_bytes"]
            roof["ncu"] = {"launch": sc["launch"], "dram_bytes_per_launch": sc["dram_bytes"], "dram_bytes_per_step": sc["dram_bytes_per_step"],
                           "warp_instructions_per_launch": sc["warp_instructions"], "warp_instructions_per_step": sc["warp_instructions_per_step"],
                           "kernel_ms_under_ncu": sc["kernel_ms_under_ncu"], "kernel_ms_per_step_under_ncu": sc["kernel_ms_per_step_under_ncu"],
                           "per_launch_ms_under_ncu": sc["per_launch_ms"],
                           "issue_frac_under_ncu": sc["warp_instructions_per_step"] / (sc["kernel_ms_per_step_under_ncu"] * 1e-3) / (148 * 4 * 1965e6),
                           "issue_active_pct_time_weighted": sc["issue_active_pct_time_weighted"],
                           "warps_active_pct_time_weighted": sc["warps_active_pct_time_weighted"],
                           "l2_tag_pct_time_weighted": sc["l2_tag_pct_time_weighted"],
                           "l2_tag_pct_hottest_slice_time_weighted": sc["l2_tag_pct_hottest_slice_time_weighted"],
                           "l2_red_requests_per_step": sc["l2_red_requests_per_step"], "l2_red_lookup_miss_share": sc["l2_red_lookup_miss_share"],
                           "source": sc["source"], "kernel_commit": sc["kernel_commit"],
                           "note": "static: ncu --metrics capture of EVERY k_transport launch of one timed step of this config (profiles/), not "
                                   "measured in this run; per-launch figures are the step's sums / launches, percentages are weighted by launch "
                                   "time; issue_frac = warp instructions / (time x 148 SMs x 4 schedulers x 1965 MHz)"}
            roof["issue_peak_ginst_s_at_sampled_clock"] = peak_issue / 1e9
        return roof

    def close(self):
        self.ctx.fdc_destroy()
        del self.flush, self.dose_d
        self.torch.cuda.empty_cache()


def measure(b, args, peaks_cache, full):
    """Timed steps + roofline for one resident workload; `full` adds the end-to-end, squares and cpu legs."""
    fdc, torch, w, ctx = b.fdc, b.torch, b.w, b.ctx
    warm = max(args.warmup, 3) if not full else args.warmup
    b.timed(warm, b.dose_d)
    clocks = ClockSampler(b.local)
    if b.rank == 0:
        clocks.start()
    b.barrier()
    wall0 = time.perf_counter()
    infos = []
    tot_ms = b.timed(args.steps, b.dose_d, infos)
    b.barrier()
    wall = time.perf_counter() - wall0
    clk = clocks.stop() if b.rank == 0 else None
    st = ctx.fdc_get_stats()                                # counters of the last step (reset each step)
    res = {"tot_ms": tot_ms, "wall": wall, "clk": clk, "st": st, "infos": infos}

    if b.world > 1:
        tl = torch.tensor([st["proton_steps"], st["deposits"], st["protons"]], dtype=torch.int64, device=b.dev)
        b.dist.all_reduce(tl)
        res["all"] = [int(x) for x in tl.tolist()]
    else:
        res["all"] = [st["proton_steps"], st["deposits"], st["protons"]]

    # ---- end to end through the public call with host buffers (every rank; max over ranks)
    if full:
        dose_h = torch.empty(w.phantom.hu.shape, dtype=torch.float32).pin_memory()
        dose_np = dose_h.numpy()
        # two equivalent plans with different bytes (the second carries one more beamlet of zero protons):
        # alternating them defeats the library's plan cache, so the plan really crosses the bus every step
        plan_b = np.concatenate([w.beamlets, w.beamlets[-1:]]); plan_b[-1]["n_protons"] = 0
        plans = (w.beamlets, plan_b)
        e2e_ms, h2d, d2h, launches = 0.0, [], [], []
        for it in range(args.warmup + args.steps):
            b.flush.fill_(1)
            b.barrier()
            t0 = time.perf_counter()
            b.one_step(dose_np, beamlets=plans[it & 1])     # returns after the D2H copy (synchronises)
            torch.cuda.synchronize()
            dt = (time.perf_counter() - t0) * 1e3
            if b.world > 1:
                t = torch.tensor([dt], device=b.dev); b.dist.all_reduce(t, op=b.dist.ReduceOp.MAX); dt = float(t.item())
            if it >= args.warmup:
                e2e_ms += dt
                ci = ctx.fdc_last_call_info()
                h2d.append(ci["h2d_bytes"]); d2h.append(ci["d2h_bytes"]); launches.append(ci["launches"])
        res["e2e"] = {"value": res["all"][2] * args.steps / (e2e_ms * 1e-3), "unit": "protons/s",
                      "h2d_bytes_per_step": int(np.mean(h2d)), "d2h_bytes_per_step": int(np.mean(d2h)),
                      "ms_per_step": e2e_ms / args.steps,
                      "copies_per_step": "1 H2D plan upload (beamlets + prefix sums) + 1 D2H dose grid, counted by the library "
                                         "(fdc_last_call_info) in every timed step: min/max h2d %d/%d, d2h %d/%d" % (min(h2d), max(h2d), min(d2h), max(d2h)),
                      "note": "fdc_reset + fdc_run(host beam plan -> pinned host dose grid), wall clock around the synchronising call; the "
                              "plan alternates between two byte-different equivalent plans so the plan cache never hits; phantom and "
                              "track database resident (loaded once, like weights)"}
        # cold variant: phantom + database from host memory every step (N = 1 only; bounded to 3 steps)
        if b.world == 1 and not args.no_cold:
            hu_h = np.ascontiguousarray(w.phantom.hu)
            cold_ms, ncold = 0.0, min(3, args.steps)
            for it in range(1 + ncold):
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                c2 = fdc.Fdc(hu_h, w.phantom.spacing, w.table, device=b.local)
                c2.fdc_load_tracks(*b.host_arrs, w.db.track_off, w.db.bin_first, w.db.e_min, w.db.e_bin)
                c2.fdc_run(w.beamlets, b.first, b.n_mine, 1, w.seed, flags=b.flags, dose_gy=dose_np)
                torch.cuda.synchronize()
                if it >= 1:
                    cold_ms += (time.perf_counter() - t0) * 1e3
                c2.fdc_destroy()
            res["e2e"]["cold"] = {"value": b.n_mine * ncold / (cold_ms * 1e-3), "unit": "protons/s", "ms_per_step": cold_ms / ncold, "steps": ncold,
                                  "h2d_bytes_per_step": int(hu_h.nbytes + sum(a.nbytes for a in b.host_arrs) + res["e2e"]["h2d_bytes_per_step"]),
                                  "d2h_bytes_per_step": int(dose_np.nbytes),
                                  "note": "fdc_create + fdc_load_tracks from pageable host arrays + fdc_run, every step"}
        del dose_h

    # ---- PAPER.md:L116 "storing the error in the tally arrays increased the calculation time by 18 %": the same step
    # with FDC_TALLY_SQUARES (second u64 grid, one more red per voxel left), then eq. (2) on the device
    if b.world == 1 and not args.no_squares:
        nsq = min(5, args.steps)
        b.timed(2, b.dose_d, flags=b.flags | fdc.FDC_TALLY_SQUARES)
        sq_ms = b.timed(nsq, b.dose_d, flags=b.flags | fdc.FDC_TALLY_SQUARES)
        t0 = time.perf_counter()
        mean_rel, n_avg = ctx.fdc_uncertainty_history(b.n_mine)
        unc_ms = (time.perf_counter() - t0) * 1e3
        base_ms = tot_ms / args.steps
        res["unc"] = {"ms_per_step_with_squares": sq_ms / nsq, "squares_cost": sq_ms / nsq / base_ms - 1.0,
                      "paper_squares_cost": 0.18, "mean_rel_uncertainty_eq2": mean_rel, "voxels_above_half_max_dose": n_avg,
                      "histories": b.n_mine, "eq2_kernels_ms": unc_ms,
                      "seconds_to_1pct_eq2": (sq_ms / nsq * 1e-3) * (mean_rel / 0.01) ** 2 if mean_rel > 0 else None,
                      "note": "PAPER.md:L116-118 context (GTX 295: +18 %, 1 % in about 2 minutes history-by-history); "
                              "seconds_to_1pct scales this run's time by (mean_rel / 1 %)^2"}
        # eq. (2) as defined: the history's whole deposit in a voxel squared once (FDC_SQUARES_BY_HISTORY; per-thread table of
        # visited voxels in local memory) -- same plan, same histories; the plain tally squares every stay (R10)
        nh = min(3, args.steps) if base_ms < 100.0 else 1        # x 7 to x 24 the plain step: one timed step on the big configs
        fh = b.flags | fdc.FDC_SQUARES_BY_HISTORY
        b.timed(1, b.dose_d, flags=fh)
        h_ms = b.timed(nh, b.dose_d, flags=fh)
        flushes = ctx.fdc_last_call_info()["sq_history_flushes"]
        mean_rel_h, n_avg_h = ctx.fdc_uncertainty_history(b.n_mine)
        res["unc"].update({"ms_per_step_by_history": h_ms / nh, "squares_by_history_cost": h_ms / nh / base_ms - 1.0,
                           "mean_rel_uncertainty_eq2_by_history": mean_rel_h, "by_history_table_flushes": flushes})
        ctx.fdc_reset()

    if b.rank == 0:
        ceilings = b.red_ceilings(peaks_cache)
        res["roof"] = b.roofline(infos, st, tot_ms, args.steps, ceilings, clk)
    return res


def secondaries_leg(b, args, base_ms, base_steps):
    """R15: the same plan with a synthetic secondary table (fdc_inputs.add_secondaries)."""
    import fdc_inputs as fi
    w, ctx = b.w, b.ctx
    db2, sec = fi.add_secondaries(w.db, 1000 + b.cfg)
    if not len(sec[1]):
        return None
    arrs2 = [np.ascontiguousarray(a) for a in (db2.dx, db2.dy, db2.dz, db2.dE, db2.E)]
    ctx.fdc_load_tracks(*arrs2, db2.track_off, db2.bin_first, db2.e_min, db2.e_bin)
    ctx.fdc_set_secondaries(*sec)
    n2 = min(5, args.steps)
    b.timed(2, b.dose_d)
    ms2 = b.timed(n2, b.dose_d)
    st2 = ctx.fdc_get_stats()
    ctx.fdc_reset()
    return {"ms_per_step": ms2 / n2, "protons_per_sec": b.n_mine / (ms2 / n2 * 1e-3), "secondary_tracks": int(len(sec[1])),
            "proton_steps": st2["proton_steps"], "deposits": st2["deposits"],
            "extra_steps_frac": st2["proton_steps"] / base_steps - 1.0, "extra_time_frac": (ms2 / n2) / base_ms - 1.0,
            "note": "one synthetic secondary per primary track (tail of another track, 10-40 % of the local energy, 10-40 degrees "
                    "off the parent); k_transport<.,.,SEC,.>"}


def per_config_entry(res, args):
    roof, st = res["roof"], res["st"]
    e = {"ms_per_step": res["tot_ms"] / args.steps, "protons_per_sec": res["all"][2] * args.steps / (res["tot_ms"] * 1e-3),
         "kernel_ms": roof["kernel_ms"], "launches_per_step": roof["launches_per_step"],
         "roofline": {"bound": roof["bound"], "frac": roof["frac"], "achieved": roof["achieved"], "peak": roof["peak"], "unit": roof["unit"],
                      "t_track_ms": roof["t_track_ms"], "t_atomic_ms": roof["t_atomic_ms"],
                      "sent_frac_of_peak": roof["l2_atomic"]["sent_frac_of_peak"],
                      "algorithmic_deposits_over_uniform_peak": roof["l2_atomic"]["algorithmic_deposits_over_uniform_peak"],
                      "peak_uniform_l2_gred_s": roof["l2_atomic"]["peak_gred_s"],
                      "peak_4_neighbour_words_gred_s": roof["l2_atomic"]["peak_4_neighbour_words_gred_s"],
                      "peak_actual_multiset_gred_s": roof["l2_atomic"]["peak_actual_multiset_gred_s"],
                      "peak_actual_multiset_trace_order_gred_s": roof["l2_atomic"]["peak_actual_multiset_trace_order_gred_s"]},
         "issue": ({"frac_under_ncu": roof["ncu"]["issue_frac_under_ncu"], "warp_instructions_per_launch": roof["ncu"]["warp_instructions_per_launch"],
                    "launch": roof["ncu"]["launch"], "source": roof["ncu"]["source"], "kernel_commit": roof["ncu"]["kernel_commit"]}
                   if "ncu" in roof else None),
         "protons": st["protons"], "proton_steps": st["proton_steps"], "deposits": st["deposits"],
         "reds_sent": roof["l2_atomic"]["reds_sent_per_step"], "clocks": res["clk"], "steps": args.steps, "warmup": max(args.warmup, 3)}
    if "unc" in res:
        e["squares_cost"] = res["unc"]["squares_cost"]; e["mean_rel_uncertainty_eq2"] = res["unc"]["mean_rel_uncertainty_eq2"]
        e["squares_by_history_cost"] = res["unc"]["squares_by_history_cost"]
        e["mean_rel_uncertainty_eq2_by_history"] = res["unc"]["mean_rel_uncertainty_eq2_by_history"]
        e["by_history_table_flushes"] = res["unc"]["by_history_table_flushes"]
    return e


def run_fdc(args):
    import torch
    import torch.distributed as dist
    import paper_1011_2188_b200 as fdc
    from paper_1011_2188_b200 import peaks
    fdc.lib()                                             # no fallback: raises if the library is missing
    peaks.lib()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a B200; there is no CPU fallback (use --impl reference for the oracle)")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise RuntimeError("--gpus %d but WORLD_SIZE=%d: launch with torch.distributed.run --nproc-per-node %d" % (args.gpus, world, args.gpus))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    peaks_cache = {}

    b = Bench(args.config, world, rank, local, fdc, torch, dist)
    res = measure(b, args, peaks_cache, full=True)
    w = b.w
    tot_ms, st, infos = res["tot_ms"], res["st"], res["infos"]
    all_steps, all_deps, all_prot = res["all"]

    # cpu baseline: the oracle on a bounded strided sample, this box's host cores
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        n_sub = min(args.cpu_sample, w.n_protons)
        K = max(1, w.n_protons // n_sub)
        t0 = time.perf_counter()
        og, ost = oracle.run(w.phantom, w.table, w.db, w.beamlets, w.seed, first=0, n=n_sub, stride=K)
        dt = time.perf_counter() - t0
        cpu = {"value": n_sub / dt, "unit": "protons/s", "cores": 1, "kind": "oracle", "host_cores_available": os.cpu_count(),
               "steps_per_sec": ost["proton_steps"] / dt,
               "sample": "every %d-th proton of %s (%d protons, %.1f s), single thread" % (K, w.name, n_sub, dt)}
        cpu["all_cores"] = oracle_all_cores(w, max(1, n_sub // 4))       # the 1-thread figure stays the headline baseline
    config = {"workload": w.name, "protons_per_step": all_prot, "protons_per_gpu": b.per_rank, "grid": list(w.phantom.dims),
              "db_tracks": w.db.n_tracks, "db_steps": w.db.n_steps, "beamlets": len(w.beamlets),
              "parallelism": "proton ranges x%d, in-place u64 grid all-reduce (NCCL)" % world if world > 1 else "single GPU",
              "l2": "flushed between timed steps (512 MiB write)", "timer": "CUDA events per step, max over ranks"}
    launches = int(sum(k["launches"] for k in infos))
    b.close()

    # ---- the other configs, same process, same flush, same warm-up (N = 1)
    per_config, sec_leg = None, None
    if rank == 0 and world == 1 and not args.no_per_config:
        per_config = {}
        for c in (1, 2, 3, 4, 5):
            if c == args.config:
                continue
            bc = Bench(c, 1, 0, local, fdc, torch, dist)
            rc = measure(bc, args, peaks_cache, full=False)
            per_config["config%d" % c] = dict(workload=bc.w.name, **per_config_entry(rc, args))
            if c == 2 and not args.no_secondaries:
                sec_leg = secondaries_leg(bc, args, rc["tot_ms"] / args.steps, rc["st"]["proton_steps"])
                if sec_leg:
                    sec_leg["workload"] = bc.w.name
            if c in (1, 2) and not args.no_cpu_baseline:
                per_config["config%d" % c]["cpu_baseline_full"] = oracle_full(bc.w)
            bc.close()
        per_config["config%d" % args.config] = dict(workload=w.name, headline=True, **per_config_entry(res, args))

    if rank == 0:
        out = {"metric": "protons_per_sec", "value": all_prot * args.steps / (tot_ms * 1e-3), "unit": "protons/s", "n_gpus": world,
               "steps": args.steps, "warmup": args.warmup, "ms_per_step": tot_ms / args.steps, "higher_is_better": True,
               "scaling": "weak", "vs_baseline": None, "dtype": "f32+u64", "data": "synthetic",
               "steps_per_sec": all_steps * args.steps / (tot_ms * 1e-3), "deposits_per_sec": all_deps * args.steps / (tot_ms * 1e-3),
               "config": config, "e2e": res.get("e2e"), "gpu_launches": launches,
               "wall_s_timed_region": res["wall"], "clocks": res["clk"], "roofline": res["roof"], "cpu_baseline": cpu,
               "per_config": per_config, "uncertainty": res.get("unc"), "secondaries": sec_leg, "stats_last_step": st,
               "paper_context": "PAPER.md:L114: 184 525 histories/s on one GTX 295 card (other machine, other workload; not a target)"}
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="fdc", choices=["fdc", "reference"])
    ap.add_argument("--config", type=int, default=HEADLINE_CONFIG,
                    help="BASELINE.json configs[C-1]; 5 (the largest single-GPU configuration) is the headline workload")
    ap.add_argument("--cpu-sample", type=int, default=1_000_000, help="protons of the strided subset the oracle is timed on")
    ap.add_argument("--ref-sample", type=int, default=100_000, help="--impl reference: protons per step")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config block (the other four configs)")
    ap.add_argument("--no-secondaries", action="store_true", help="skip the leg with a synthetic secondary table (R15; config 2)")
    ap.add_argument("--no-squares", action="store_true", help="skip the FDC_TALLY_SQUARES / eq. (2) legs")
    ap.add_argument("--no-cold", action="store_true", help="skip the e2e.cold leg (context + database re-created from host memory)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "fdc":
        print("note: warmup < 3 breaks the timing rules; use for smoke runs only", file=sys.stderr)
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # `python bench.py --gpus N` by hand: re-launch as one rank per GPU, the way the driver does
        port = 29500 + os.getpid() % 2000
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        return subprocess.call(cmd)
    return run_fdc(args)


if __name__ == "__main__":
    sys.exit(main())

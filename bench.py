#!/usr/bin/env python
"""bench.py -- measurement of the track-repeating hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl fdc|reference] [--config C]

One "step" = one pass of the whole hot path over one batch of synthetic input: zero the grid,
sample + select tracks + group (sort) + transport + deposit + convert to Gy, for every proton of
the workload.  At N = 1 the workload is BASELINE.json configs[1] (the 128^3 slab phantom, 150 MeV,
1e6 protons, database of 1e4 tracks per 1 MeV bin over 140-160 MeV), generated from seeds by
fdc_inputs (synthetic).  Prints ONE JSON line (rank 0).

`value`   protons/s with every input already resident in HBM (device events, max over ranks).
`e2e`     the same through the public call with HOST buffers: beam plan H2D and dose grid D2H
          inside the timed region (the phantom and the track database are resident, loaded once
          by fdc_create / fdc_load_tracks like weights); `e2e_cold` also re-creates the context
          and re-loads phantom and database from host memory every step.
`roofline` the transport+deposit kernel against max(track bytes / HBM peak, deposits / measured
          u64-red rate) (north_star); see DESIGN.md §8 for the per-unit figures.
`cpu_baseline` the oracle, as it stands, on this box's host cores on a strided proton subset.

--impl reference times the oracle (tier framing: the reference arm is the oracle); there is no
CPU fallback in the product arm: without libfdc.so or a B200 it raises.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

L2_FLUSH_BYTES = 512 << 20          # > 126 MB L2
STEP_RECORD_BYTES = 20              # dx,dy,dz,dE,E float32 per step (north_star (1))


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """SM clock + throttle reasons sampled through NVML every few ms while the timed region runs
    (nvidia-smi -lms cannot sample a region that lasts tens of milliseconds)."""
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}

    def __init__(self, index, period_s=0.004):
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
    """configs[cfg-1]; for N > 1 (weak scaling) the plan holds N x the protons and rank r runs the
    r-th contiguous range of the global proton index space."""
    import fdc_inputs as fi
    base = fi._FULL[cfg]
    w = fi.workload(cfg, n_protons=base * gpus, lazy_db=(cfg != 2))
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


# --------------------------------------------------------------------------- product arm
def run_fdc(args):
    import torch
    import torch.distributed as dist
    import paper_1011_2188_b200 as fdc
    from paper_1011_2188_b200 import multi
    fdc.lib()                                             # no fallback: raises if the library is missing
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a B200; there is no CPU fallback (use --impl reference for the oracle)")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    w, per_rank = make_workload(args.config, world)
    first, n_mine = multi.shard_range(w.n_protons, rank, world)
    dev = torch.device("cuda", local)

    # resident inputs (borrowed device arrays; PyTorch = device memory and streams only)
    hu_d = torch.from_numpy(np.ascontiguousarray(w.phantom.hu)).to(dev)
    ctx = fdc.Fdc(hu_d, w.phantom.spacing, w.table, device=local)
    host_arrs = [np.ascontiguousarray(a) for a in (w.db.dx, w.db.dy, w.db.dz, w.db.dE, w.db.E)]
    ctx.fdc_load_tracks(*host_arrs, w.db.track_off, w.db.bin_first, w.db.e_min, w.db.e_bin)
    dose_d = torch.zeros(w.phantom.hu.shape, dtype=torch.float32, device=dev)
    grid_d = torch.zeros(w.phantom.hu.shape, dtype=torch.int64, device=dev) if world > 1 else None
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
    flags = fdc.FDC_RANDOM_AZIMUTH

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def one_step(dose_out):
        ctx.fdc_reset()
        if world == 1:
            ctx.fdc_run(w.beamlets, first, n_mine, 1, w.seed, flags=flags, dose_gy=dose_out)
        else:
            ctx.fdc_run(w.beamlets, first, n_mine, 1, w.seed, flags=flags)
            multi.allreduce_edep(ctx, grid_d)              # the paper's "dose from both threads was combined" (L75)
            ctx.fdc_run(w.beamlets, 0, 0, 1, w.seed, flags=flags, dose_gy=dose_out)

    def timed(n_steps, dose_out, kernel_times=None):
        tot = 0.0
        for _ in range(n_steps):
            flush.fill_(1)                                  # L2 flush between timed iterations
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            barrier()
            e0.record()
            one_step(dose_out)
            e1.record()
            barrier()
            ms = e0.elapsed_time(e1)
            if world > 1:
                t = torch.tensor([ms], device=dev); dist.all_reduce(t, op=dist.ReduceOp.MAX); ms = float(t.item())
            tot += ms
            if kernel_times is not None:
                kernel_times.append(ctx.fdc_last_timing())
        return tot

    timed(args.warmup, dose_d)
    clocks = ClockSampler(local)
    if rank == 0:
        clocks.start()
    barrier()
    wall0 = time.perf_counter()
    ktimes = []
    tot_ms = timed(args.steps, dose_d, ktimes)
    barrier()
    wall = time.perf_counter() - wall0
    clk = clocks.stop() if rank == 0 else None
    st = ctx.fdc_get_stats()                                # counters of the last step (reset each step)

    # ---- end to end through the public call with host buffers
    dose_h = torch.empty(w.phantom.hu.shape, dtype=torch.float32).pin_memory()
    dose_np = dose_h.numpy()

    def e2e_step():
        one_step(dose_np)                                   # beam plan H2D + dose D2H inside fdc_run (synchronises)

    e2e_ms = 0.0
    for it in range(args.warmup + args.steps):
        flush.fill_(1)
        barrier()
        t0 = time.perf_counter()
        e2e_step()
        torch.cuda.synchronize()
        dt = (time.perf_counter() - t0) * 1e3
        if world > 1:
            t = torch.tensor([dt], device=dev); dist.all_reduce(t, op=dist.ReduceOp.MAX); dt = float(t.item())
        if it >= args.warmup:
            e2e_ms += dt
    h2d = int(w.beamlets.nbytes + 8 * (len(w.beamlets) + 1))
    d2h = int(dose_np.nbytes)

    # cold variant: phantom + database from host memory every step (N = 1 only; bounded to 3 steps)
    e2e_cold = None
    if world == 1 and rank == 0 and not args.no_cold:
        hu_h = np.ascontiguousarray(w.phantom.hu)
        cold_ms, ncold = 0.0, min(3, args.steps)
        for it in range(1 + ncold):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            c2 = fdc.Fdc(hu_h, w.phantom.spacing, w.table, device=local)
            c2.fdc_load_tracks(*host_arrs, w.db.track_off, w.db.bin_first, w.db.e_min, w.db.e_bin)
            c2.fdc_run(w.beamlets, first, n_mine, 1, w.seed, flags=flags, dose_gy=dose_np)
            torch.cuda.synchronize()
            if it >= 1:
                cold_ms += (time.perf_counter() - t0) * 1e3
            c2.fdc_destroy()
        e2e_cold = {"value": n_mine * ncold / (cold_ms * 1e-3), "unit": "protons/s",
                    "h2d_bytes_per_step": int(hu_h.nbytes + sum(a.nbytes for a in host_arrs) + h2d), "d2h_bytes_per_step": d2h,
                    "note": "fdc_create + fdc_load_tracks from pageable host arrays + fdc_run, every step"}

    # ---- PAPER.md:L116 "storing the error in the tally arrays increased the calculation time by 18 %": the same
    # step with FDC_TALLY_SQUARES (second u64 grid, one more red per voxel left), then eq. (2) on the device
    unc = None
    if world == 1 and rank == 0 and not args.no_squares:
        sq_ms, nsq = 0.0, min(5, args.steps)
        for it in range(2 + nsq):
            flush.fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            ctx.fdc_reset()
            ctx.fdc_run(w.beamlets, first, n_mine, 1, w.seed, flags=flags | fdc.FDC_TALLY_SQUARES, dose_gy=dose_d)
            e1.record()
            torch.cuda.synchronize()
            if it >= 2:
                sq_ms += e0.elapsed_time(e1)
        t0 = time.perf_counter()
        mean_rel, n_avg = ctx.fdc_uncertainty_history(n_mine)
        unc_ms = (time.perf_counter() - t0) * 1e3
        base_ms = tot_ms / args.steps
        unc = {"ms_per_step_with_squares": sq_ms / nsq, "squares_cost": sq_ms / nsq / base_ms - 1.0,
               "paper_squares_cost": 0.18, "mean_rel_uncertainty_eq2": mean_rel, "voxels_above_half_max_dose": n_avg,
               "histories": n_mine, "eq2_kernels_ms": unc_ms,
               "seconds_to_1pct_eq2": (sq_ms / nsq * 1e-3) * (mean_rel / 0.01) ** 2 if mean_rel > 0 else None,
               "note": "PAPER.md:L116-118 context (GTX 295: +18 %, 1 % in about 2 minutes history-by-history); "
                       "seconds_to_1pct scales this run's time by (mean_rel / 1 %)^2"}
        ctx.fdc_reset()

    # ---- R15: the same plan with a synthetic secondary table (fdc_inputs.add_secondaries)
    sec_leg = None
    if world == 1 and rank == 0 and not args.no_secondaries:
        import fdc_inputs as fi
        db2, sec = fi.add_secondaries(w.db, 1000 + args.config)
        if len(sec[1]):
            arrs2 = [np.ascontiguousarray(a) for a in (db2.dx, db2.dy, db2.dz, db2.dE, db2.E)]
            ctx.fdc_load_tracks(*arrs2, db2.track_off, db2.bin_first, db2.e_min, db2.e_bin)
            ctx.fdc_set_secondaries(*sec)
            ms2, n2 = 0.0, min(5, args.steps)
            for it in range(2 + n2):
                flush.fill_(1)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                e0.record()
                ctx.fdc_reset()
                ctx.fdc_run(w.beamlets, first, n_mine, 1, w.seed, flags=flags, dose_gy=dose_d)
                e1.record()
                torch.cuda.synchronize()
                if it >= 2:
                    ms2 += e0.elapsed_time(e1)
            st2 = ctx.fdc_get_stats()
            sec_leg = {"ms_per_step": ms2 / n2, "protons_per_sec": n_mine / (ms2 / n2 * 1e-3), "secondary_tracks": int(len(sec[1])),
                       "proton_steps": st2["proton_steps"], "deposits": st2["deposits"],
                       "extra_steps_frac": st2["proton_steps"] / st["proton_steps"] - 1.0,
                       "extra_time_frac": (ms2 / n2) / (tot_ms / args.steps) - 1.0,
                       "note": "one synthetic secondary per primary track (tail of another track, 10-40 % of the local energy, "
                               "10-40 degrees off the parent); k_transport<.,.,SEC>"}
            ctx.fdc_reset()

    if world > 1:
        tl = torch.tensor([st["proton_steps"], st["deposits"], st["protons"]], dtype=torch.int64, device=dev)
        dist.all_reduce(tl)
        all_steps, all_deps, all_prot = [int(x) for x in tl.tolist()]
    else:
        all_steps, all_deps, all_prot = st["proton_steps"], st["deposits"], st["protons"]

    if rank == 0:
        hbm_gbs, peak_src = _peaks()
        n_vox = int(np.prod(w.phantom.hu.shape))
        # roofline of the dominant kernel (k_transport), rank 0's launches, live CUDA-event durations
        tr_ms = float(np.mean([k["transport_ms"] for k in ktimes]))
        # denominators: u64 red rate, uniform random addresses, (i) over an L2-resident buffer and (ii) over a
        # buffer the size of this grid.  (i) >= (ii); the kernel's deposits are spatially clustered, so on a
        # grid larger than L2 it can beat (ii) -- the roofline therefore uses (i), the harder ceiling.
        red_l2 = fdc.fdc_peak_red_u64(local, min(n_vox * 8, 64 << 20), 1 << 30, 0)
        red_fp = red_l2 if n_vox * 8 <= (64 << 20) else fdc.fdc_peak_red_u64(local, n_vox * 8, 1 << 28, 0)
        red_peak = max(red_l2, red_fp)
        # the same microbenchmark with the 32 lanes of a warp in one 32-byte sector group / on one word
        red_modes = {"lanes_share_4_words": fdc.fdc_peak_red_u64(local, min(n_vox * 8, 64 << 20), 1 << 28, 1) / 1e9,
                     "lanes_share_1_word": fdc.fdc_peak_red_u64(local, min(n_vox * 8, 64 << 20), 1 << 28, 2) / 1e9,
                     # every warp of the GPU on a hot set of a few words (config 1: all protons down one column)
                     "hot_set_256_words": fdc.fdc_peak_red_u64(local, 256 * 8, 1 << 28, 0) / 1e9,
                     "hot_set_16_words": fdc.fdc_peak_red_u64(local, 16 * 8, 1 << 26, 0) / 1e9}
        t_track = st["proton_steps"] * STEP_RECORD_BYTES / (hbm_gbs * 1e9)
        t_atomic = st["deposits"] / red_peak
        bound_atomic = t_atomic >= t_track
        roof = {"bound": "l2_atomic" if bound_atomic else "hbm",
                "achieved": (st["deposits"] / (tr_ms * 1e-3) / 1e9) if bound_atomic else (st["proton_steps"] * STEP_RECORD_BYTES / (tr_ms * 1e-3) / 1e9),
                "peak": red_peak / 1e9 if bound_atomic else hbm_gbs,
                "unit": "Gred/s" if bound_atomic else "GB/s",
                "frac": max(t_track, t_atomic) / (tr_ms * 1e-3),
                "traffic": None,
                "kernel": "k_transport", "kernel_ms": tr_ms, "kernel_share_of_step": tr_ms * args.steps / tot_ms * 1.0,
                "t_track_ms": t_track * 1e3, "t_atomic_ms": t_atomic * 1e3,
                "hbm": {"achieved_gbs": st["proton_steps"] * STEP_RECORD_BYTES / (tr_ms * 1e-3) / 1e9, "peak_gbs": hbm_gbs, "peak_source": peak_src},
                "l2_atomic": {"achieved_gred_s": st["deposits"] / (tr_ms * 1e-3) / 1e9, "peak_gred_s": red_peak / 1e9,
                              "peak_at_grid_footprint_gred_s": red_fp / 1e9, "grid_mib": n_vox * 8 >> 20,
                              "clustered_peaks_gred_s": red_modes,
                              "peak_source": "fdc_peak_red_u64 measured in this run: u64 red, uniform random addresses over min(grid, 64 MiB) "
                                             "(L2-resident); peak_at_grid_footprint is the same over the whole grid"},
                "algorithmic": {"proton_steps": st["proton_steps"], "deposits": st["deposits"], "bytes_per_step": STEP_RECORD_BYTES,
                                "note": "deposits = non-zero (step, voxel) shares (R8); the kernel merges the shares one proton leaves in "
                                        "one voxel into a single red, so it issues fewer reds than deposits"}}
        traffic_file = os.path.join(ROOT, "profiles", "traffic.csv")     # dram bytes of one ncu --set full capture, per launch
        if os.path.exists(traffic_file):
            with open(traffic_file) as f:
                for line in f.read().splitlines()[1:]:
                    c = line.split(",")
                    if len(c) >= 3 and c[0].strip() == str(args.config):
                        roof["traffic"] = float(c[1])
                        if args.config != 4:        # config 4's capture is one of two launches per step
                            # third view: the kernel is bound by instruction issue (4 schedulers x 1 warp
                            # instruction per clock per SM); instructions from the ncu capture, time and clock live
                            mhz = (clk or {}).get("sm_mhz") or 1965.0
                            peak_issue = 148 * 4 * mhz * 1e6
                            roof["issue"] = {"warp_instructions": float(c[2]), "achieved_ginst_s": float(c[2]) / (tr_ms * 1e-3) / 1e9,
                                             "peak_ginst_s": peak_issue / 1e9, "frac": float(c[2]) / (tr_ms * 1e-3) / peak_issue,
                                             "note": "instruction count from profiles/ (ncu smsp__inst_executed.sum), kernel time and SM clock from this run"}

        # cpu baseline: the oracle on a bounded strided sample, this box's host cores
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            import oracle
            n_sub = min(args.cpu_sample, w.n_protons)
            K = max(1, w.n_protons // n_sub)
            t0 = time.perf_counter()
            og, ost = oracle.run(w.phantom, w.table, w.db, w.beamlets, w.seed, first=0, n=n_sub, stride=K)
            dt = time.perf_counter() - t0
            cpu = {"value": n_sub / dt, "unit": "protons/s", "cores": 1, "kind": "oracle", "host_cores_available": os.cpu_count(),
                   "steps_per_sec": ost["proton_steps"] / dt,
                   "sample": "every %d-th proton of %s (%d protons, %.1f s), single thread" % (K, w.name, n_sub, dt)}

        out = {"metric": "protons_per_sec", "value": all_prot * args.steps / (tot_ms * 1e-3), "unit": "protons/s", "n_gpus": world,
               "steps": args.steps, "warmup": args.warmup, "ms_per_step": tot_ms / args.steps, "higher_is_better": True,
               "scaling": "weak", "vs_baseline": None, "dtype": "f32+u64", "data": "synthetic",
               "steps_per_sec": all_steps * args.steps / (tot_ms * 1e-3), "deposits_per_sec": all_deps * args.steps / (tot_ms * 1e-3),
               "config": {"workload": w.name, "protons_per_step": all_prot, "protons_per_gpu": per_rank, "grid": list(w.phantom.dims),
                          "db_tracks": w.db.n_tracks, "db_steps": w.db.n_steps, "beamlets": len(w.beamlets),
                          "parallelism": "proton ranges x%d, u64 grid all-reduce" % world if world > 1 else "single GPU",
                          "l2": "flushed between timed steps (512 MiB write)", "timer": "CUDA events per step, max over ranks"},
               "e2e": {"value": all_prot * args.steps / (e2e_ms * 1e-3), "unit": "protons/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                       "note": "fdc_reset + fdc_run(host beam plan -> pinned host dose grid); phantom and track DB resident"},
               "e2e_cold": e2e_cold,
               "gpu_launches": int(sum(k["launches"] for k in ktimes)) + (0 if world == 1 else 0),
               "wall_s_timed_region": wall, "clocks": clk, "roofline": roof, "cpu_baseline": cpu,
               "uncertainty": unc, "secondaries": sec_leg, "stats_last_step": st,
               "paper_context": "PAPER.md:L114: 184 525 histories/s on one GTX 295 card (other machine, other workload; not a target)"}
        print(json.dumps(out))
    ctx.fdc_destroy()
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="fdc", choices=["fdc", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json configs[C-1]; 2 is the headline single-GPU workload")
    ap.add_argument("--cpu-sample", type=int, default=1_000_000, help="protons of the strided subset the oracle is timed on")
    ap.add_argument("--ref-sample", type=int, default=100_000, help="--impl reference: protons per step")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-secondaries", action="store_true", help="skip the leg with a synthetic secondary table (R15)")
    ap.add_argument("--no-squares", action="store_true", help="skip the FDC_TALLY_SQUARES / eq. (2) leg")
    ap.add_argument("--no-cold", action="store_true", help="skip the e2e_cold leg (context + database re-created from host memory)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "fdc":
        print("note: warmup < 3 breaks the timing rules; use for smoke runs only", file=sys.stderr)
    return run_reference(args) if args.impl == "reference" else run_fdc(args)


if __name__ == "__main__":
    sys.exit(main())

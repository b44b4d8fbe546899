"""Writes tests/golden/full_plan_digests.json: the ORACLE's result for the whole plan of configs 3, 4
and 5 (BASELINE.json configs[2..4]: 1e7, 5e7 and 2e8 protons), reduced to a digest -- sha256 of the u64
grid bytes, the grid sum and every counter.  The oracle needs no GPU, so this runs off the GPU box
(SURVEY §8(d) "full-config parity for 3-5"); tests/test_gpu_parity.py::test_full_plan_digest runs the
same plan through the CUDA path on the box and compares digests.  Calls only oracle/ and the seeded
input generators (fdc_inputs); proton ranges are spread over threads (integer sums: any split gives
the same grid, pin P7).

    python tests/golden/make_digests.py [3 4 5]      (sq3: only the squares digests of config 3)
"""
import hashlib
import json
import os
import sys
import time
from concurrent.futures import ThreadPoolExecutor

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import fdc_inputs as fi      # noqa: E402
import oracle                # noqa: E402

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "full_plan_digests.json")


def digest(cfg, threads):
    w = fi.workload(cfg, lazy_db=True)
    parts = threads * 4
    bounds = [w.n_protons * k // parts for k in range(parts + 1)]
    grids = [np.zeros(w.phantom.hu.shape, dtype=np.uint64) for _ in range(threads)]
    stats = []

    def work(k):
        g = grids[k % threads]                       # one grid per thread slot; parts of a slot run one after another
        _, st = oracle.run(w.phantom, w.table, w.db, w.beamlets, w.seed, first=bounds[k], n=bounds[k + 1] - bounds[k], grid=g)
        return st

    t0 = time.time()
    for wave in range(4):                            # 4 waves of `threads` parts: slot k is used by one part per wave
        with ThreadPoolExecutor(threads) as ex:
            stats += list(ex.map(work, range(wave * threads, (wave + 1) * threads)))
    total = grids[0]
    for g in grids[1:]:
        total += g
    keys = [k for k in stats[0] if k != "grid_sum"]
    st = {k: int(sum(s[k] for s in stats)) for k in keys}
    st["grid_sum"] = int(total.sum(dtype=np.uint64))
    assert st["grid_sum"] + st["q_escaped"] == st["q_replayed"]
    return {"workload": w.name, "protons": int(w.n_protons), "seed": int(w.seed), "grid_shape": list(total.shape),
            "sha256_u64_grid": hashlib.sha256(np.ascontiguousarray(total).tobytes()).hexdigest(), "stats": st,
            "oracle_seconds": round(time.time() - t0, 1), "threads": threads,
            "source": "oracle.run over the whole plan of fdc_inputs.workload(%d) (DESIGN.md §5; BASELINE.json configs[%d])" % (cfg, cfg - 1)}


def digest_squares(cfg, threads):
    """The sum-of-squares grids (R10) of the whole plan, per stay and per history (eq. (2) as defined): sha256 of the u64 bytes
    and the sums."""
    w = fi.workload(cfg, lazy_db=True)
    parts = threads * 4
    bounds = [w.n_protons * k // parts for k in range(parts + 1)]

    def work(k):
        g, sq, sqh, st = oracle.run_sq(w.phantom, w.table, w.db, w.beamlets, w.seed, first=bounds[k], n=bounds[k + 1] - bounds[k], by_history=True)
        return sq, sqh

    total = np.zeros(w.phantom.hu.shape, dtype=np.uint64)
    total_h = np.zeros(w.phantom.hu.shape, dtype=np.uint64)
    with ThreadPoolExecutor(threads) as ex:
        for sq, sqh in ex.map(work, range(parts)):
            total += sq
            total_h += sqh
    assert (total_h >= total).all()
    return {"sha256_u64_squares": hashlib.sha256(np.ascontiguousarray(total).tobytes()).hexdigest(),
            "squares_sum_mod_2_64": int(total.sum(dtype=np.uint64)),
            "sha256_u64_squares_by_history": hashlib.sha256(np.ascontiguousarray(total_h).tobytes()).hexdigest(),
            "squares_by_history_sum_mod_2_64": int(total_h.sum(dtype=np.uint64))}


if __name__ == "__main__":
    args = sys.argv[1:] or ["3", "4", "5"]
    data = json.load(open(OUT)) if os.path.exists(OUT) else {}
    for a in args:
        if a.startswith("sq"):                       # "sq3": only the squares digests of a config whose plain digest is stored
            c = int(a[2:])
            data[str(c)].update(digest_squares(c, threads=os.cpu_count() or 1))
        else:
            c = int(a)
            data[str(c)] = digest(c, threads=os.cpu_count() or 1)
            if c == 3:                               # the squares tallies at full size on the one-field plan
                data[str(c)].update(digest_squares(c, threads=os.cpu_count() or 1))
        print(c, data[str(c)]["sha256_u64_grid"], data[str(c)]["oracle_seconds"], "s", flush=True)
        with open(OUT, "w") as f:
            json.dump(data, f, indent=1, sort_keys=True)
            f.write("\n")

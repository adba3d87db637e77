"""configs[4] at FULL size (BASELINE.json: 128^3 voxels x 4096 hemisphere sensors, Nt = 2048, one frame; the paper's
3-D outlook): a 34.4 GB travel-time table, HBM-resident, never held whole on the host.

Part of the routine `-m gpu` suite.  The table comes from the library's GPU eikonal solver in sensor chunks
(pat_eikonal_travel_times_device: the same first-order upwind system as the CPU fast marching, SURVEY.md 8(f)
NEXT-2; ~100 s instead of ~7 min of host FMM) and is handed to the plan on the device; a sample of its rows is
checked against the ORACLE's fast marching (oracle.fmm_rows) in the same test.  The image is checked by the
oracle on a seeded sample of voxels, one by one, plus the whole first and last tile -- with the SAME fp32 table
values both sides (R17): the sampled columns are read back from the device rows that were uploaded.
"""
import json
import os
import time

import numpy as np
import pytest

import oracle
import workloads as W
from _cases import assert_parity

pytestmark = [pytest.mark.gpu, pytest.mark.slow]


def test_config4_full_size_sampled_voxels():
    import torch
    import paper_1501_03869_b200 as pat
    free, total = torch.cuda.mem_get_info()
    if total < 60 * (1 << 30):
        pytest.skip("needs a device with > 60 GB (34.4 GB table + workspace)")
    geom = W.make_geometry(4)
    S, P = geom.nsens, geom.npix
    assert (S, P, geom.nt) == (4096, 128 ** 3, 2048)
    rng = np.random.default_rng(404)
    pick = np.unique(np.concatenate([np.arange(256), np.arange(P - 256, P), rng.integers(0, P, size=6000)]))
    apos, _ = W.make_absorbers(geom, 0)
    t0 = time.time()
    plan = pat.Plan(geom.n, geom.h, geom.origin, None, geom.sensors, geom.roi_index, geom.nt, geom.fs, geom.t0)
    grid = pat.PatGrid.make(geom.n, geom.h, geom.origin)
    cmap = np.ascontiguousarray(geom.c_map, dtype=np.float32).ravel()
    d_pick = torch.from_numpy(pick).cuda()
    d_apos = torch.from_numpy(np.asarray(apos, dtype=np.int64)).cuda()
    tau_pick = np.empty((S, pick.size), np.float32)
    tau_abs = np.empty((S, apos.size), np.float32)
    check_sensors = sorted(set(int(v) for v in rng.integers(0, S, size=8)) | {0, S - 1})
    tau_check = {}
    chunk = 1024
    rows = torch.empty((chunk, P), dtype=torch.float32, device="cuda")
    t_eik, rounds = time.time(), 0
    for s0 in range(0, S, chunk):
        rounds = max(rounds, pat.pat_eikonal_travel_times_device(grid, cmap, geom.sensors, S, geom.roi_index, P,
                                                                 s0, chunk, rows))
        plan.set_travel_times(rows, s0, chunk)
        tau_pick[s0:s0 + chunk] = rows[:, d_pick].cpu().numpy()
        tau_abs[s0:s0 + chunk] = rows[:, d_apos].cpu().numpy()
        for s in check_sensors:
            if s0 <= s < s0 + chunk:
                tau_check[s] = rows[s - s0].cpu().numpy()
    torch.cuda.synchronize()
    t_eik = time.time() - t_eik
    del rows
    # the table itself: sampled rows against the oracle's fast marching (<= 1 ulp of fp32: same discrete system)
    t_or = time.time()
    ref_rows = oracle.fmm_rows(geom.n, geom.h, geom.origin, geom.c_map, geom.sensors[check_sensors], geom.roi_index)
    t_or = time.time() - t_or
    worst_ulp = 0
    for q, s in enumerate(check_sensors):
        d = np.abs(tau_check[s].view(np.int32).astype(np.int64) - ref_rows[q].view(np.int32).astype(np.int64))
        worst_ulp = max(worst_ulp, int(d.max()))
    assert worst_ulp <= 1, "GPU eikonal rows differ from the oracle's fast marching by %d ulp" % worst_ulp
    look = {int(p): i for i, p in enumerate(apos)}
    tr = W.make_traces(geom, lambda pos: tau_abs[:, [look[int(p)] for p in pos]], frames=[0])
    d_tr = torch.from_numpy(tr).cuda()
    img = torch.full((1, P), float("nan"), dtype=torch.float32, device="cuda")
    t_first = time.time()
    plan.backproject(d_tr, img, 1)                       # first call: builds the work list (33.5 M rows) synchronously
    torch.cuda.synchronize()
    t_first = time.time() - t_first
    got = img.cpu().numpy()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps = 5
    e0.record()
    for _ in range(reps):
        plan.backproject(d_tr, img, 1)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    ref = oracle.backproject(tau_pick, tr, geom.fs, geom.t0, 1)
    rel, mx = assert_parity(got[:, pick], ref, "config4 full size, sampled voxels")
    assert np.all(np.isfinite(got))
    bytes_ = 4.0 * S * P + 4.0 * S * geom.nt + 4.0 * P
    stats = plan.stats() if hasattr(plan, "stats") else {}
    out = {"config": "configs[4] full: %d sensors x %d voxels, Nt=%d, B=1" % (S, P, geom.nt), "ms_per_frame": ms,
           "gupd_s": S * P / ms / 1e6, "algorithmic_GB": bytes_ / 1e9, "hbm_gbs": bytes_ / ms / 1e6,
           "rel_l2": rel, "max_abs_over_max": mx, "sampled_voxels": int(pick.size),
           "table": "pat_eikonal_travel_times_device, %d sensors per chunk" % chunk, "eikonal_seconds": t_eik,
           "eikonal_rounds": int(rounds), "rows_checked_vs_oracle_fmm": check_sensors, "worst_ulp_vs_oracle_fmm": worst_ulp,
           "oracle_fmm_seconds": t_or, "first_call_seconds_incl_work_list_build": t_first, "stats": stats,
           "total_seconds": time.time() - t0}
    print(json.dumps(out))
    os.makedirs("gpurun_out", exist_ok=True)
    with open("gpurun_out/full3d.json", "w") as f:
        json.dump(out, f)
    plan.close()

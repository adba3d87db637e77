"""Shared helpers of the GPU parity tests: inputs (seeded, synthetic), tau tables, the bar."""
import functools
import os

import numpy as np

import workloads as W

REL_L2_TOL = 1e-5          # BASELINE.json north_star
MAX_ABS_TOL = 1e-4         # x max|image|


def prod_tau(geom, order=1, sensors=None):
    """tau fp32 [S][P] from the production CPU FMM (host-only entry point of the C-ABI)."""
    import paper_1501_03869_b200 as pat
    grid = pat.PatGrid.make(geom.n, geom.h, geom.origin)
    S = geom.nsens
    lo, cnt = (0, S) if sensors is None else sensors
    tau = np.empty((cnt, geom.npix), dtype=np.float32)
    pat.pat_fmm_travel_times(grid, np.ascontiguousarray(geom.c_map).ravel(), geom.sensors, S,
                             geom.roi_index, geom.npix, lo, cnt, order, tau, 0)
    return tau


@functools.lru_cache(maxsize=4)
def case(k, reduced=False):
    """(geometry, tau) of config k; k = 2 shares k = 1's table (same geometry)."""
    geom = W.make_geometry(k, reduced)
    if k == 2:
        _, tau = case(1)
    else:
        tau = prod_tau(geom)
    return geom, tau


def errors(got, ref):
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    den = np.linalg.norm(ref.ravel())
    rel = np.linalg.norm((got - ref).ravel()) / den if den > 0 else np.linalg.norm(got.ravel())
    mx = np.max(np.abs(got - ref)) if ref.size else 0.0
    sc = np.max(np.abs(ref)) if ref.size else 0.0
    return rel, mx, sc


def assert_parity(got, ref, what=""):
    rel, mx, sc = errors(got, ref)
    assert rel <= REL_L2_TOL, "%s rel-L2 %.3e > %.0e" % (what, rel, REL_L2_TOL)
    assert mx <= MAX_ABS_TOL * sc + 1e-30, "%s max-abs %.3e > 1e-4*%.3e" % (what, mx, sc)
    return rel, mx / sc if sc > 0 else 0.0


def gpu_backproject(geom, tau, traces, mode=1, max_batch=None, tuning=None, host=False, t0=None):
    """One pass of the product path through the C-ABI; returns fp32 images [B][P] (numpy)."""
    import torch
    import paper_1501_03869_b200 as pat
    B = traces.shape[0]
    plan = pat.Plan(geom.n, geom.h, geom.origin, geom.c_map, geom.sensors, geom.roi_index, geom.nt,
                    geom.fs, geom.t0 if t0 is None else t0, weighting=mode, max_batch=max_batch or max(B, 1) * (2 if mode >= 3 else 1))   # _EXACT: two channels per frame
    try:
        if tuning:
            pat.pat_set_gather_tuning(plan.handle, *tuning)
        plan.set_travel_times(tau)
        if host:
            tr = torch.from_numpy(np.ascontiguousarray(traces)).pin_memory()
            img = torch.empty((B, geom.npix), dtype=torch.float32).pin_memory()
            plan.backproject(tr, img, B)
            torch.cuda.synchronize()
            return img.numpy().copy()
        tr = torch.from_numpy(np.ascontiguousarray(traces)).cuda()
        img = torch.full((B, geom.npix), float("nan"), dtype=torch.float32, device="cuda")
        plan.backproject(tr, img, B)
        torch.cuda.synchronize()
        return img.cpu().numpy()
    finally:
        plan.close()

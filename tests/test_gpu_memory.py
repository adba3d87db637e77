"""device memory is the caller's.  Between pat_plan_create and pat_destroy the library obtains device
memory ONLY through the provider installed with pat_set_device_allocator (include/pat.h "device memory") -- checked two
ways: every request is seen (and returned) by a counting provider, and the device memory in use OUTSIDE torch's
allocator (cudaMemGetInfo minus torch's reserved bytes) does not move while a plan goes through every feature."""
import numpy as np
import pytest

import oracle
from _cases import assert_parity, case

pytestmark = pytest.mark.gpu


def _outside_torch():
    import torch
    torch.cuda.synchronize()
    free, total = torch.cuda.mem_get_info()
    return (total - free) - torch.cuda.memory_reserved()


def _exercise(geom, tau, traces):
    """One plan through every path that needs provider memory; returns (image, stats)."""
    import torch
    import paper_1501_03869_b200 as pat
    plan = pat.Plan(geom.n, geom.h, geom.origin, geom.c_map, geom.sensors, geom.roi_index, geom.nt, geom.fs, geom.t0,
                    max_batch=4)
    try:
        plan.set_travel_times(tau)
        tr = torch.from_numpy(traces).cuda()
        img = torch.empty((traces.shape[0], geom.npix), dtype=torch.float32, device="cuda")
        plan.backproject(tr, img, traces.shape[0])                       # work list of the 4-frame class
        plan.backproject(tr[:1], img[:1], 1)                             # ... and of the 1-frame class
        plan.backproject_conventional(tr[:1], img[:1], 1500.0, 1)        # geometry + row-range scratch + its work list
        mask = np.zeros(geom.npix, np.uint8)
        mask[::3] = 1
        plan.set_roi_mask(mask)                                          # masked permutation
        plan.backproject(tr[:1], img[:1], 1)
        plan.set_roi_mask(None)
        s = geom.sensors.astype(np.float64)
        nrm = (s / np.linalg.norm(s, axis=1, keepdims=True)).astype(np.float32)
        plan.compute_solid_angle_weights(nrm)                            # weight table + scratch
        plan.set_pixel_weights(None)
        plan.backproject(tr, img, traces.shape[0])
        torch.cuda.synchronize()
        return img.cpu().numpy(), plan.stats()
    finally:
        plan.close()


def test_all_library_device_memory_comes_from_the_provider():
    import torch
    import paper_1501_03869_b200 as pat
    import workloads as W
    geom, tau = case(0)
    traces = W.make_traces(geom, tau, frames=range(4))
    pat.install_torch_allocator()
    _exercise(geom, tau, traces)                 # warm-up: context, module loading, torch's pools
    seen = {"alloc": 0, "free": 0, "bytes": 0, "live": {}}

    def alloc(nbytes):
        ptr = pat.torch_alloc(nbytes)
        seen["alloc"] += 1
        seen["bytes"] += nbytes
        seen["live"][ptr] = nbytes
        return ptr

    def free(ptr, nbytes):
        assert seen["live"].pop(ptr) == nbytes, "release must name the block and size that alloc handed out"
        seen["free"] += 1
        pat.torch_free(ptr, nbytes)

    before = _outside_torch()
    pat.pat_set_device_allocator(alloc, free)
    try:
        got, stats = _exercise(geom, tau, traces)
    finally:
        pat.pat_set_device_allocator(None, None)
        pat.install_torch_allocator()
    after = _outside_torch()
    assert seen["alloc"] >= 6, "work lists, geometry, mask, weights and scratch must all go through the provider"
    assert seen["free"] == seen["alloc"] and not seen["live"], "pat_destroy returns everything"
    assert after == before, "device memory outside torch's allocator moved by %d bytes: the library allocated on its own" % (after - before)
    assert stats["provider_bytes_peak"] > 0 and stats["work_lists"] >= 3 and stats["work_list_bytes"] > 0
    assert stats["workspace_bytes"] == pat.pat_plan_workspace_bytes(pat.PatGrid.make(geom.n, geom.h, geom.origin), geom.nsens,
                                                                  geom.npix, geom.nt, 4)
    assert_parity(got, oracle.backproject(tau, traces, geom.fs, geom.t0, 1), "after the whole sequence")


def test_a_provider_that_returns_nothing_fails_cleanly():
    import torch
    import paper_1501_03869_b200 as pat
    import workloads as W
    geom, tau = case(0)
    traces = W.make_traces(geom, tau, frames=range(1))
    pat.install_torch_allocator()
    plan = None
    pat.pat_set_device_allocator(lambda nbytes: None, lambda ptr, nbytes: None)
    try:
        plan = pat.Plan(geom.n, geom.h, geom.origin, None, geom.sensors, geom.roi_index, geom.nt, geom.fs, geom.t0)
        plan.set_travel_times(tau)                                       # workspace only: no provider memory needed
        tr = torch.from_numpy(traces).cuda()
        img = torch.empty((1, geom.npix), dtype=torch.float32, device="cuda")
        with pytest.raises(pat.PatError) as ei:
            plan.backproject(tr, img, 1)                                 # needs a work list
        assert ei.value.status == pat.PAT_ERR_NOMEM
    finally:
        if plan is not None:
            plan.close()
        pat.pat_set_device_allocator(None, None)
        pat.install_torch_allocator()

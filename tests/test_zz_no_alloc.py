"""pat_backproject_static -- the entry point that allocates nothing (include/pat.h): its images against the
plan path's (pat_backproject) on the same inputs, within the tolerance every GPU parity test uses, on calls in
a row that share the static scratch array.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

import workloads as W
import paper_1501_03869_b200 as pat
from _cases import assert_parity, case, gpu_backproject


def test_static_entry_point_rejects_sizes_beyond_its_scratch():
    a = np.zeros(4, dtype=np.float32)
    lim = pat.pat_backproject_static_max_samples()
    assert lim == 1 << 20
    with pytest.raises(pat.PatError) as e:
        pat.pat_backproject_static(a, a, a, 513, 16, 2048, 1, 20e6)          # 513 * 2048 > 2^20
    assert e.value.status == pat.PAT_ERR_INVALID_ARG and "exceed the static scratch" in str(e.value)
    with pytest.raises(pat.PatError) as e:
        pat.pat_backproject_static(a, a, a, 2, 2, 2, 1, 20e6, 0.0, pat.PAT_W_PAPER_EXACT)
    assert e.value.status == pat.PAT_ERR_UNSUPPORTED
    with pytest.raises(pat.PatError) as e:                                    # host pointers: nothing is copied for the caller
        pat.pat_backproject_static(a, a, a, 2, 2, 2, 1, 20e6)
    assert e.value.status in (pat.PAT_ERR_INVALID_ARG, pat.PAT_ERR_CUDA)


def _inputs(k, frames, t0=None, mode=pat.PAT_W_PAPER):
    geom, tau = case(k)
    traces = W.make_traces(geom, tau, frames=frames)
    t0 = geom.t0 if t0 is None else t0
    ref = gpu_backproject(geom, tau, traces, mode=mode, t0=t0)               # the existing path
    return geom, tau, traces, t0, mode, ref


@pytest.mark.gpu
def test_static_entry_point_matches_the_plan_path_on_calls_in_a_row():
    import torch
    # call 1 fills the whole array (512 x 2048 samples = the limit), call 2 is small with another weighting and
    # t0 (the rest of the array still holds call 1's b), call 3 is large again: stale contents must never show
    jobs = [_inputs(1, range(0, 1)), _inputs(0, range(3, 5), t0=1.0e-6, mode=pat.PAT_W_UBP), _inputs(1, range(7, 8))]
    dev = []
    for geom, tau, traces, t0, mode, ref in jobs:
        dev.append((torch.from_numpy(tau).cuda(), torch.from_numpy(np.ascontiguousarray(traces)).cuda(),
                    torch.full((traces.shape[0], geom.npix), float("nan"), dtype=torch.float32, device="cuda")))
    torch.cuda.synchronize()
    free = []
    for (geom, tau, traces, t0, mode, ref), (d_tau, d_tr, d_img) in zip(jobs, dev):
        pat.pat_backproject_static(d_tau, d_tr, d_img, geom.nsens, geom.npix, geom.nt, traces.shape[0], geom.fs, t0, mode)
        torch.cuda.synchronize()
        free.append(torch.cuda.mem_get_info()[0])
    for n, ((geom, tau, traces, t0, mode, ref), (_, _, d_img)) in enumerate(zip(jobs, dev)):
        assert_parity(d_img.cpu().numpy(), ref, "static call %d" % (n + 1))
    # the first call may load the module (and with it the array); after that the device's free memory stands still
    assert free[1] == free[2], "device memory moved between two calls of the entry point that allocates nothing"


@pytest.mark.gpu
def test_static_entry_point_runs_inside_a_stream_capture():
    import torch
    geom, tau, traces, t0, mode, ref = _inputs(0, range(1, 2))
    d_tau, d_tr = torch.from_numpy(tau).cuda(), torch.from_numpy(np.ascontiguousarray(traces)).cuda()
    d_img = torch.zeros((1, geom.npix), dtype=torch.float32, device="cuda")
    st = torch.cuda.Stream()
    pat.pat_backproject_static(d_tau, d_tr, d_img, geom.nsens, geom.npix, geom.nt, 1, geom.fs, t0, mode, st)   # set-up call
    st.synchronize()
    d_img.fill_(float("nan"))
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=st):
        pat.pat_backproject_static(d_tau, d_tr, d_img, geom.nsens, geom.npix, geom.nt, 1, geom.fs, t0, mode, st)
    g.replay()
    torch.cuda.synchronize()
    assert_parity(d_img.cpu().numpy(), ref, "static call replayed from a graph")

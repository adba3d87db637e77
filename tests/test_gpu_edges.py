"""GPU edge cases of the C-ABI path: ragged sizes, out-of-record / non-finite tau, t0,
chunked tau upload, device tau, linearity, error paths that need a device."""
import numpy as np
import pytest

import oracle
import workloads as W
from _cases import assert_parity, case, errors, gpu_backproject

pytestmark = pytest.mark.gpu
FS = 20e6


def _geom(npix, nsens, nt, nx=64, ny=64):
    """A bare geometry carrying only sizes (tau is supplied directly)."""
    g = W.make_geometry(0)
    g.n = (nx, ny)
    g.c_map = np.full((ny, nx), 1540.0, np.float32)
    rng = np.random.default_rng(npix + nsens)
    g.roi_index = np.sort(rng.choice(nx * ny, size=npix, replace=False)).astype(np.int64)
    g.sensors = np.zeros((nsens, 3), np.float32)
    g.nt = nt
    return g


@pytest.mark.parametrize("npix,nsens,nt,B", [(1, 1, 2, 1), (255, 3, 17, 1), (257, 17, 33, 2),
                                             (1000, 33, 100, 3), (4096, 16, 64, 5), (777, 50, 512, 7)])
def test_ragged_sizes_random_tau(npix, nsens, nt, B):
    g = _geom(npix, nsens, nt)
    rng = np.random.default_rng(1)
    tau = (rng.uniform(-2.0, nt + 1.0, size=(nsens, npix)) / FS).astype(np.float32)
    tr = rng.standard_normal((B, nsens, nt)).astype(np.float32)
    for mode in (0, 1):
        ref = oracle.backproject(tau, tr, FS, 0.0, mode)
        assert_parity(gpu_backproject(g, tau, tr, mode=mode), ref, "ragged mode %d" % mode)


def test_nonfinite_and_out_of_record_tau_contribute_zero():
    g = _geom(600, 8, 64)
    rng = np.random.default_rng(2)
    tau = (rng.uniform(0.0, 62.0, size=(8, 600)) / FS).astype(np.float32)
    bad = np.array([np.inf, -np.inf, np.nan, -1e-9, 63.0 / FS, 1.0, -3.0, 1e30, -1e30, 3e38], np.float32)
    tau[3, :bad.size] = bad
    tau[5, 100:100 + bad.size] = bad
    tau[0, 0] = 0.0
    tau[1, 1] = np.float32(62.0) / np.float32(FS)
    tr = rng.standard_normal((2, 8, 64)).astype(np.float32)
    ref = oracle.backproject(tau, tr, FS, 0.0, 1)
    got = gpu_backproject(g, tau, tr)
    assert np.all(np.isfinite(got))
    assert_parity(got, ref, "bad tau")
    # a whole row of invalid tau = that sensor removed
    tau2 = tau.copy()
    tau2[2, :] = np.nan
    ref2 = oracle.backproject(np.delete(tau, 2, axis=0), np.delete(tr, 2, axis=1), FS, 0.0, 1)
    assert_parity(gpu_backproject(g, tau2, tr), ref2, "nan row")


def test_index_rule_is_one_fp32_multiply():
    """tau chosen so that fl32(tau*fs) and the double product fall on different sides of an integer."""
    g = _geom(512, 4, 2048)
    rng = np.random.default_rng(3)
    ks = rng.integers(1, 2040, size=(4, 512)).astype(np.float64)
    tau = np.nextafter((ks / FS).astype(np.float32), np.float32(0)).astype(np.float32)
    tau[::2] = np.nextafter(tau[::2], np.float32(1))
    tr = rng.standard_normal((1, 4, 2048)).astype(np.float32) * 100
    ref = oracle.backproject(tau, tr, FS, 0.0, 1)
    assert_parity(gpu_backproject(g, tau, tr), ref, "index rule")


def test_t0_offset():
    g = _geom(300, 5, 128)
    rng = np.random.default_rng(4)
    t0 = float(np.float32(1.7e-6))
    tau = (t0 + rng.uniform(-3.0, 130.0, size=(5, 300)) / FS).astype(np.float32)
    tr = rng.standard_normal((2, 5, 128)).astype(np.float32)
    ref = oracle.backproject(tau, tr, FS, t0, 1)
    assert_parity(gpu_backproject(g, tau, tr, t0=t0), ref, "t0")


def test_chunked_and_device_tau_upload_and_state_machine():
    import torch
    import paper_1501_03869_b200 as pat
    g = _geom(900, 12, 96)
    rng = np.random.default_rng(5)
    tau = (rng.uniform(0.0, 94.0, size=(12, 900)) / FS).astype(np.float32)
    tr = rng.standard_normal((1, 12, 96)).astype(np.float32)
    ref = oracle.backproject(tau, tr, FS, 0.0, 1)
    plan = pat.Plan(g.n, g.h, g.origin, g.c_map, g.sensors, g.roi_index, g.nt, FS, 0.0, max_batch=2)
    d_tr = torch.from_numpy(tr).cuda()
    img = torch.zeros((1, 900), dtype=torch.float32, device="cuda")
    plan.set_travel_times(tau[0:5], 0)
    with pytest.raises(pat.PatError) as ei:
        plan.backproject(d_tr, img, 1)
    assert ei.value.status == pat.PAT_ERR_BAD_STATE
    plan.set_travel_times(torch.from_numpy(tau[5:9]).cuda(), 5)       # device rows
    plan.set_travel_times(np.ascontiguousarray(tau[9:12]), 9)
    plan.backproject(d_tr, img, 1)
    torch.cuda.synchronize()
    assert_parity(img.cpu().numpy(), ref, "chunked upload")
    n0 = plan.launches()
    plan.backproject(d_tr, img, 1)                                     # idempotent: no hidden state
    torch.cuda.synchronize()
    assert plan.launches() == n0 + 2
    assert_parity(img.cpu().numpy(), ref, "second call")
    with pytest.raises(pat.PatError) as ei:
        plan.backproject(d_tr, img, 3)
    assert ei.value.status == pat.PAT_ERR_INVALID_ARG
    assert plan.backproject(d_tr, img, 0) == pat.PAT_OK
    with pytest.raises(pat.PatError):
        plan.backproject(d_tr, torch.zeros((1, 900)), 1)               # host/device mix
    plan.close()


def test_linearity_on_gpu():
    g = _geom(2000, 20, 256)
    rng = np.random.default_rng(6)
    tau = (rng.uniform(0.0, 254.0, size=(20, 2000)) / FS).astype(np.float32)
    x = (np.round(rng.standard_normal((1, 20, 256)) * 256) / 256).astype(np.float32)
    y = (np.round(rng.standard_normal((1, 20, 256)) * 256) / 256).astype(np.float32)
    z = (2 * x - 0.5 * y).astype(np.float32)
    gx, gy, gz = (gpu_backproject(g, tau, v).astype(np.float64) for v in (x, y, z))
    assert_parity(gz, 2 * gx - 0.5 * gy, "linearity")


def test_compute_travel_times_on_plan_matches_host_fmm():
    import torch
    import paper_1501_03869_b200 as pat
    from _cases import prod_tau
    geom = W.make_geometry(0)
    tau = prod_tau(geom)
    tr = W.make_traces(geom, tau)
    plan = pat.Plan(geom.n, geom.h, geom.origin, geom.c_map, geom.sensors, geom.roi_index, geom.nt, geom.fs)
    plan.compute_travel_times()
    img = torch.zeros((1, geom.npix), dtype=torch.float32, device="cuda")
    plan.backproject(torch.from_numpy(tr).cuda(), img, 1)
    torch.cuda.synchronize()
    assert_parity(img.cpu().numpy(), oracle.backproject(tau, tr, geom.fs), "plan-side FMM")
    plan.close()


@pytest.mark.parametrize("B", [1, 2, 3, 4, 5, 8, 9, 16, 17, 32, 33, 64, 65, 130])
def test_every_frame_count_class(B):
    """Frame-count classes 1, 2, 3-4, ..., 33-64 and multi-group launches (> 64 frames)."""
    g = _geom(700, 9, 160)
    rng = np.random.default_rng(100 + B)
    # smooth-ish tau (short windows, the fast path) with a few far outliers (segmented rows)
    base = rng.uniform(20.0, 120.0, size=(9, 1))
    tau = ((base + rng.uniform(0.0, 30.0, size=(9, 700))) / FS).astype(np.float32)
    tau[2, ::50] = np.float32(3.0 / FS)
    tr = rng.standard_normal((B, 9, 160)).astype(np.float32)
    ref = oracle.backproject(tau, tr, FS, 0.0, 1)
    assert_parity(gpu_backproject(g, tau, tr), ref, "B=%d" % B)


@pytest.mark.parametrize("tuning", [(8, 1, 2), (16, 3, 2), (32, 5, 3), (64, 16, 4), (256, 2, 2), (128, 30, 2)])
@pytest.mark.parametrize("B", [1, 4, 20])
def test_gather_tuning_does_not_change_the_result(tuning, B):
    """Window ring / slots / stages only change the schedule: segment splits, ring wrap-around,
    null-padded chunks, pipeline depth."""
    geom, tau = __import__("_cases").case(0)
    tr = W.make_traces(geom, tau, frames=range(B))
    ref = oracle.backproject(tau, tr, geom.fs, geom.t0, 1)
    assert_parity(gpu_backproject(geom, tau, tr, tuning=tuning), ref, "tuning %s B=%d" % (tuning, B))
    g = _geom(1500, 21, 300)
    rng = np.random.default_rng(7)
    tau2 = (rng.uniform(-5.0, 310.0, size=(21, 1500)) / FS).astype(np.float32)
    tr2 = rng.standard_normal((B, 21, 300)).astype(np.float32)
    assert_parity(gpu_backproject(g, tau2, tr2, tuning=tuning), oracle.backproject(tau2, tr2, FS, 0.0, 1),
                  "random tau, tuning %s B=%d" % (tuning, B))


def test_table_without_any_valid_entry_gives_zero_images():
    g = _geom(300, 4, 64)
    tau = np.full((4, 300), np.nan, np.float32)
    tau[1] = -1.0
    tau[2] = 1.0
    tr = np.random.default_rng(8).standard_normal((3, 4, 64)).astype(np.float32)
    got = gpu_backproject(g, tau, tr)
    assert np.all(got == 0.0)


def test_invalid_tuning_is_rejected():
    import paper_1501_03869_b200 as pat
    g = _geom(300, 4, 64)
    plan = pat.Plan(g.n, g.h, g.origin, g.c_map, g.sensors, g.roi_index, g.nt, FS)
    for bad in [(100, 0, 0), (4, 0, 0), (0, 31, 0), (0, 0, 1), (-8, 0, 0)]:
        with pytest.raises(pat.PatError) as ei:
            pat.pat_set_gather_tuning(plan.handle, *bad)
        assert ei.value.status == pat.PAT_ERR_INVALID_ARG
    plan.close()


def test_image_buffer_guard_bands_stay_intact():
    """compute-sanitizer is closed on this pool: check by hand that nothing is written outside
    images[nframes][npix] (guard bands before and after, odd sizes, padded last tile)."""
    import torch
    import paper_1501_03869_b200 as pat
    g = _geom(1001, 7, 80)
    rng = np.random.default_rng(9)
    tau = (rng.uniform(-3.0, 83.0, size=(7, 1001)) / FS).astype(np.float32)
    for B in (1, 3, 33):
        tr = rng.standard_normal((B, 7, 80)).astype(np.float32)
        plan = pat.Plan(g.n, g.h, g.origin, g.c_map, g.sensors, g.roi_index, g.nt, FS, 0.0, max_batch=B)
        plan.set_travel_times(tau)
        guard = 4096
        big = torch.full((guard + B * 1001 + guard,), 12345.0, dtype=torch.float32, device="cuda")
        img = big[guard:guard + B * 1001].view(B, 1001)
        plan.backproject(torch.from_numpy(tr).cuda(), img, B)
        torch.cuda.synchronize()
        assert torch.all(big[:guard] == 12345.0) and torch.all(big[guard + B * 1001:] == 12345.0)
        assert_parity(img.cpu().numpy(), oracle.backproject(tau, tr, FS, 0.0, 1), "guarded images B=%d" % B)
        plan.close()


def test_host_calls_back_to_back_overlap_copies_and_kernels():
    """Host-buffer calls stage their traces through two alternating buffers on the plan's copy stream
    (the transfer of call i+1 runs under the kernels of call i).  Six calls without a synchronise in
    between, different traces each: every image must be the one of its own traces."""
    import torch
    import paper_1501_03869_b200 as pat
    g = _geom(1500, 24, 256)
    rng = np.random.default_rng(21)
    tau = (rng.uniform(2.0, 250.0, size=(24, 1500)) / FS).astype(np.float32)
    plan = pat.Plan(g.n, g.h, g.origin, g.c_map, g.sensors, g.roi_index, g.nt, FS, 0.0, max_batch=2)
    try:
        plan.set_travel_times(tau)
        trs = [torch.from_numpy(rng.standard_normal((2, 24, 256)).astype(np.float32)).pin_memory() for _ in range(6)]
        imgs = [torch.empty((2, 1500), dtype=torch.float32).pin_memory() for _ in range(6)]
        st = torch.cuda.Stream()
        for tr, im in zip(trs, imgs):
            plan.backproject(tr, im, 2, st)
        st.synchronize()
        for q, (tr, im) in enumerate(zip(trs, imgs)):
            ref = oracle.backproject(tau, tr.numpy(), FS, 0.0, 1)
            assert_parity(im.numpy(), ref, "back-to-back host call %d" % q)
    finally:
        plan.close()


def test_roi_mask_selects_pixels_without_touching_the_table():
    """a region of interest can be selected for reconstruction.  Selected pixels get the values
    of the full reconstruction, the others 0; tiles without a selected pixel leave the work list (fewer
    launches' worth of work, same table); NULL restores everything; the conventional BP obeys the same mask."""
    import torch
    import paper_1501_03869_b200 as pat
    geom, tau = case(0)
    rng = np.random.default_rng(33)
    traces = rng.standard_normal((2, geom.nsens, geom.nt)).astype(np.float32)
    ref = oracle.backproject(tau, traces, geom.fs, geom.t0, 1)
    x = geom.roi_index % geom.n[0]
    for mask in (x < geom.n[0] // 3, rng.random(geom.npix) < 0.01, np.zeros(geom.npix, bool)):
        plan = pat.Plan(geom.n, geom.h, geom.origin, geom.c_map, geom.sensors, geom.roi_index, geom.nt, geom.fs,
                        geom.t0, max_batch=2)
        try:
            plan.set_travel_times(tau)
            d_tr = torch.from_numpy(traces).cuda()
            img = torch.full((2, geom.npix), float("nan"), dtype=torch.float32, device="cuda")
            plan.set_roi_mask(mask)
            plan.backproject(d_tr, img, 2)
            torch.cuda.synchronize()
            got = img.cpu().numpy()
            assert (got[:, ~mask] == 0).all()
            if mask.any():
                rel, mx, sc = errors(got[:, mask], ref[:, mask])
                assert rel <= 1e-5 and mx <= 1e-4 * np.max(np.abs(ref)), (rel, mx)
            c0 = 1540.0
            cref = oracle.backproject(oracle.tau_conventional(geom.n, geom.h, geom.origin, geom.sensors,
                                                              geom.roi_index, c0), traces, geom.fs, geom.t0, 1)
            plan.backproject_conventional(d_tr, img, c0, 2)
            torch.cuda.synchronize()
            got = img.cpu().numpy()
            assert (got[:, ~mask] == 0).all()
            if mask.any():
                rel, mx, sc = errors(got[:, mask], cref[:, mask])
                assert rel <= 1e-5 and mx <= 1e-4 * np.max(np.abs(cref)), (rel, mx)
            plan.set_roi_mask(None)
            plan.backproject(d_tr, img, 2)
            torch.cuda.synchronize()
            assert_parity(img.cpu().numpy(), ref, "mask removed")
        finally:
            plan.close()


@pytest.mark.parametrize("lo_u,hi_u,expect", [(300.0, 700.0, (296, 408)), (0.0, 2046.0, (0, 2048)), (5.0, 9.0, (4, 8))])
def test_host_calls_transfer_only_the_samples_the_table_can_touch(lo_u, hi_u, expect):
    """pat_get_trace_window / PAPER.md:79 (the frame time includes the transfers): with host buffers only the
    samples [kmin-1, kmax+2] (rounded to quads) of every trace cross the bus.  The workspace is poisoned with NaN
    bit patterns beforehand, so anything read outside the transferred part of the staging buffer would show."""
    import torch
    import paper_1501_03869_b200 as pat
    g = _geom(900, 12, 2048)
    rng = np.random.default_rng(31)
    tau = (rng.uniform(lo_u, hi_u, size=(12, 900)) / FS).astype(np.float32)
    tau[0, 0], tau[11, 899] = np.float32(lo_u / FS), np.float32(hi_u / FS)
    tau[3, 5] = np.nan                                               # invalid entries do not widen the window
    tau[4, 6] = np.float32(5000.0 / FS)
    grid = pat.PatGrid.make(g.n, g.h, g.origin)
    nbytes = pat.pat_plan_workspace_bytes(grid, 12, 900, 2048, 2)
    ws = torch.full((nbytes + 256,), 0xFF, dtype=torch.uint8, device="cuda")
    addr = (ws.data_ptr() + 255) // 256 * 256
    h = pat.pat_plan_create(grid, None, g.sensors, 12, g.roi_index, 900, 2048, FS, 0.0, pat.PAT_W_PAPER, 2, addr, nbytes)
    try:
        pat.pat_set_travel_times(h, tau, 0, 12)
        u = (tau * np.float32(FS)).astype(np.float32)
        ok = (u >= 0) & (u < 2047)
        k = np.floor(u[ok]).astype(np.int64)
        first, count = pat.pat_get_trace_window(h)
        assert (first, count) == expect
        if count < 2048:
            assert first <= max(0, k.min() - 1) and first + count >= min(2048, k.max() + 3)
        for q in range(3):                                           # both staging buffers
            tr = rng.standard_normal((2, 12, 2048)).astype(np.float32)
            t = torch.from_numpy(tr).pin_memory()
            im = torch.empty((2, 900), dtype=torch.float32).pin_memory()
            pat.pat_backproject(h, t, im, 2)
            torch.cuda.synchronize()
            assert np.all(np.isfinite(im.numpy()))
            assert_parity(im.numpy(), oracle.backproject(tau, tr, FS, 0.0, 1), "windowed H2D, call %d" % q)
    finally:
        pat.pat_destroy(h)


def test_back_to_back_single_frame_calls_on_one_plan():
    """One plan, 12 device calls without a synchronise in between: image buffers alternating between three tensors,
    then the same tensor three times, different traces every call; every image must be the one of its own traces
    (the weighted-trace buffer and the images are reused by the next call's pre-pass: stream order must hold)."""
    import torch
    import paper_1501_03869_b200 as pat
    geom, tau = case(1)
    rng = np.random.default_rng(77)
    plan = pat.Plan(geom.n, geom.h, geom.origin, None, geom.sensors, geom.roi_index, geom.nt, geom.fs, geom.t0, max_batch=1)
    try:
        plan.set_travel_times(tau)
        ncall = 12
        trs = [torch.from_numpy(rng.standard_normal((1, geom.nsens, geom.nt)).astype(np.float32)).cuda() for _ in range(ncall)]
        ring = [torch.full((1, geom.npix), float("nan"), dtype=torch.float32, device="cuda") for _ in range(3)]
        outs = []
        st = torch.cuda.Stream()
        torch.cuda.synchronize()
        with torch.cuda.stream(st):
            for q in range(ncall):
                img = ring[q % 3] if q < 9 else ring[0]
                plan.backproject(trs[q], img, 1, st)
                outs.append(img.clone())                       # stream-ordered copy of this call's result
        st.synchronize()
        for q in (0, 1, 5, 8, 9, 10, 11):
            ref = oracle.backproject(tau, trs[q].cpu().numpy(), geom.fs, geom.t0, 1)
            assert_parity(outs[q].cpu().numpy(), ref, "back-to-back call %d" % q)
    finally:
        plan.close()


@pytest.mark.parametrize("env", ["PAT_PLAIN_MORTON", "PAT_OLD_BLOCKED_PREPASS"])
@pytest.mark.parametrize("B", [1, 4, 16])
def test_ab_switches_of_the_layout_give_the_same_images(monkeypatch, env, B):
    """The pixel order (recursive bisection vs round 1's plain Morton order) and the two pre-pass kernels of the
    blocked layout are implementation choices: the oracle does not know them, so both settings must meet the bar
    (configs[1]: a disk that cuts Morton blocks -- the case the bisection order exists for)."""
    geom, tau = case(1)
    traces = W.make_traces(geom, tau, frames=range(20, 20 + B))
    ref = oracle.backproject(tau, traces, geom.fs, geom.t0, 1)
    assert_parity(gpu_backproject(geom, tau, traces), ref, "default B=%d" % B)
    monkeypatch.setenv(env, "1")                         # read when the plan is created
    assert_parity(gpu_backproject(geom, tau, traces), ref, "%s=1 B=%d" % (env, B))

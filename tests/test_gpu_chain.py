"""Cross-call overlap ("launch chain", csrc/pat_api.cu): consecutive pat_backproject calls captured into ONE CUDA
graph are chained with programmatic edges, so the kernels of call i+1 run beside the draining gather of call i.
Every image must still be the oracle's image of its own traces (Eq. 7) -- the hazards are the reuse
of the weighted-trace buffer, the zeroing of the images by the next call's pre-pass and the completion counters,
so the cases below reuse plans, image buffers and graphs in every order a caller might.
"""
import numpy as np
import pytest

import oracle
from _cases import assert_parity, case

pytestmark = pytest.mark.gpu


def _plan(geom, tau, max_batch=1):
    import paper_1501_03869_b200 as pat
    plan = pat.Plan(geom.n, geom.h, geom.origin, None, geom.sensors, geom.roi_index, geom.nt, geom.fs, geom.t0,
                    max_batch=max_batch)
    plan.set_travel_times(tau)
    return plan


def _traces(geom, n, B=1, seed=5):
    import torch
    rng = np.random.default_rng(seed)
    return [torch.from_numpy(rng.standard_normal((B, geom.nsens, geom.nt)).astype(np.float32)).cuda() for _ in range(n)]


def _ref(tau, tr, geom):
    return oracle.backproject(tau, tr.cpu().numpy(), geom.fs, geom.t0, 1)


def _capture(st, fn):
    import torch
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(st):
        with torch.cuda.graph(g, stream=st):
            fn()
    return g


def test_chained_calls_on_one_plan_distinct_images_and_replays():
    """12 calls on ONE plan in one graph, own image per call: 11 of them are chained; replayed three times (the
    counters re-arm themselves), then direct calls on the same plan."""
    import torch
    geom, tau = case(1)
    plan = _plan(geom, tau)
    try:
        n = 12
        trs = _traces(geom, n)
        imgs = [torch.full((1, geom.npix), float("nan"), dtype=torch.float32, device="cuda") for _ in range(n)]
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            plan.backproject(trs[0], imgs[0], 1, st)              # work list outside the capture
        st.synchronize()
        c0 = plan.chained_calls()
        g = _capture(st, lambda: [plan.backproject(trs[q], imgs[q], 1, st) for q in range(n)])
        assert plan.chained_calls() - c0 == n - 1, "every call but the first of the capture must be chained"
        with torch.cuda.stream(st):
            for _ in range(3):
                for im in imgs:
                    im.fill_(float("nan"))
                g.replay()
        st.synchronize()
        for q in (0, 1, 2, 6, 10, 11):
            assert_parity(imgs[q].cpu().numpy(), _ref(tau, trs[q], geom), "chained call %d" % q)
        # direct (unchained) calls afterwards find the counters re-armed
        c1 = plan.chained_calls()
        with torch.cuda.stream(st):
            plan.backproject(trs[3], imgs[0], 1, st)
            plan.backproject(trs[4], imgs[1], 1, st)
        st.synchronize()
        assert plan.chained_calls() == c1, "calls outside a capture are never chained"
        assert_parity(imgs[0].cpu().numpy(), _ref(tau, trs[3], geom), "direct call after replays")
        assert_parity(imgs[1].cpu().numpy(), _ref(tau, trs[4], geom), "direct call after replays (2)")
    finally:
        plan.close()


def test_same_image_buffer_is_never_chained():
    """The next pre-pass zeroes the images: with the SAME image tensor in consecutive calls the host must fall back
    to the ordinary launch -- and an overlapping traces/images range likewise."""
    import torch
    geom, tau = case(1)
    plan = _plan(geom, tau)
    try:
        trs = _traces(geom, 6, seed=6)
        img = torch.full((1, geom.npix), float("nan"), dtype=torch.float32, device="cuda")
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            plan.backproject(trs[0], img, 1, st)
        st.synchronize()
        c0 = plan.chained_calls()
        g = _capture(st, lambda: [plan.backproject(trs[q], img, 1, st) for q in range(6)])
        assert plan.chained_calls() == c0
        with torch.cuda.stream(st):
            g.replay()
        st.synchronize()
        assert_parity(img.cpu().numpy(), _ref(tau, trs[5], geom), "same image buffer, last call")
        # images of call q are the traces of call q+1 (absurd, but legal): must not be chained either
        P4 = (geom.npix + 3) // 4 * 4
        big = torch.zeros((geom.nsens * geom.nt + P4,), dtype=torch.float32, device="cuda")
        tr_b = big[:geom.nsens * geom.nt].view(1, geom.nsens, geom.nt)
        img_a = big[geom.nsens * geom.nt - P4:geom.nsens * geom.nt - P4 + geom.npix].view(1, geom.npix)   # inside tr_b
        img_b = torch.empty((1, geom.npix), dtype=torch.float32, device="cuda")
        c1 = plan.chained_calls()
        g2 = _capture(st, lambda: (plan.backproject(trs[0], img_a, 1, st), plan.backproject(tr_b, img_b, 1, st)))
        assert plan.chained_calls() == c1, "traces overlapping the previous images must serialise"
        with torch.cuda.stream(st):
            g2.replay()
        st.synchronize()
        assert_parity(img_b.cpu().numpy(), _ref(tau, tr_b, geom), "traces = previous image (serialised)")
    finally:
        plan.close()


def test_ping_pong_images_and_foreign_work_between_calls():
    """Images alternate A, B, A, B (call q+2 zeroes what call q wrote: it must have completed), and a foreign
    kernel between two calls breaks the chain for that call only."""
    import torch
    geom, tau = case(1)
    plan = _plan(geom, tau)
    try:
        n = 9
        trs = _traces(geom, n, seed=7)
        A, Bm = (torch.full((1, geom.npix), float("nan"), dtype=torch.float32, device="cuda") for _ in range(2))
        keep = torch.empty((n, geom.npix), dtype=torch.float32, device="cuda")
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            plan.backproject(trs[0], A, 1, st)
        st.synchronize()
        c0 = plan.chained_calls()

        def body():
            for q in range(n):
                plan.backproject(trs[q], A if q % 2 == 0 else Bm, 1, st)
                if q in (3, 6):                                   # foreign node: the next call is not chained
                    keep[q].copy_((A if q % 2 == 0 else Bm)[0])
        g = _capture(st, body)
        assert plan.chained_calls() - c0 == n - 1 - 2
        with torch.cuda.stream(st):
            g.replay()
            g.replay()
        st.synchronize()
        assert_parity(keep[3:4].cpu().numpy(), _ref(tau, trs[3], geom), "copied out after call 3")
        assert_parity(keep[6:7].cpu().numpy(), _ref(tau, trs[6], geom), "copied out after call 6")
        assert_parity(A.cpu().numpy(), _ref(tau, trs[8], geom), "ping-pong A")
        assert_parity(Bm.cpu().numpy(), _ref(tau, trs[7], geom), "ping-pong B")
    finally:
        plan.close()


@pytest.mark.parametrize("Bs", [(1, 2), (4, 1), (16, 3)])
def test_two_plans_and_frame_count_classes_chained(Bs):
    """Calls alternate between TWO plans of different frame-count classes (different pre-pass grids and counters)."""
    import torch
    geom, tau = case(1)
    plans = [_plan(geom, tau, max_batch=b) for b in Bs]
    try:
        n = 8
        trs = [_traces(geom, 1, B=Bs[q % 2], seed=20 + q)[0] for q in range(n)]
        imgs = [torch.full((Bs[q % 2], geom.npix), float("nan"), dtype=torch.float32, device="cuda") for q in range(n)]
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            for q in range(2):
                plans[q].backproject(trs[q], imgs[q], Bs[q], st)
        st.synchronize()
        c0 = sum(p.chained_calls() for p in plans)
        g = _capture(st, lambda: [plans[q % 2].backproject(trs[q], imgs[q], Bs[q % 2], st) for q in range(n)])
        assert sum(p.chained_calls() for p in plans) - c0 == n - 1
        with torch.cuda.stream(st):
            for im in imgs:
                im.fill_(float("nan"))
            g.replay()
            g.replay()
        st.synchronize()
        for q in (0, 1, 4, 6, 7):
            assert_parity(imgs[q].cpu().numpy(), _ref(tau, trs[q], geom), "two plans, call %d (B=%d)" % (q, Bs[q % 2]))
    finally:
        for p in plans:
            p.close()


def test_chained_conventional_and_table_calls_mixed():
    """The conventional BP (delays computed in the gather) runs through the same chain."""
    import torch
    geom, tau = case(0)
    import paper_1501_03869_b200 as pat
    plan = pat.Plan(geom.n, geom.h, geom.origin, geom.c_map, geom.sensors, geom.roi_index, geom.nt, geom.fs, geom.t0)
    try:
        plan.set_travel_times(tau)
        trs = _traces(geom, 6, seed=9)
        imgs = [torch.full((1, geom.npix), float("nan"), dtype=torch.float32, device="cuda") for _ in range(6)]
        st = torch.cuda.Stream()
        c0s = 1500.0
        with torch.cuda.stream(st):
            plan.backproject(trs[0], imgs[0], 1, st)
            plan.backproject_conventional(trs[1], imgs[1], c0s, 1, st)
        st.synchronize()

        def body():
            for q in range(6):
                if q % 2 == 0:
                    plan.backproject(trs[q], imgs[q], 1, st)
                else:
                    plan.backproject_conventional(trs[q], imgs[q], c0s, 1, st)
        g = _capture(st, body)
        with torch.cuda.stream(st):
            g.replay()
        st.synchronize()
        tau_c = oracle.tau_conventional(geom.n, geom.h, geom.origin, geom.sensors, geom.roi_index, c0s)
        for q in range(6):
            ref = oracle.backproject(tau if q % 2 == 0 else tau_c, trs[q].cpu().numpy(), geom.fs, geom.t0, 1)
            assert_parity(imgs[q].cpu().numpy(), ref, "mixed chain, call %d" % q)
    finally:
        plan.close()

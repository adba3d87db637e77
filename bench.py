"""bench.py -- throughput of the hot path (H1 pre-pass + H2-H4 gather) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config k] [--batch B] [--impl reference]

A "step" is one pat_backproject call (weighting pre-pass + gather) over one batch of B frames of
the synthetic workload configs[k] (default k = 1: 512 sensors x 21323 pixels, Nt = 2048, B = 1,
the configuration BASELINE.json's metric is quoted on).  The tau table comes from the library's
CPU FMM (input preparation, untimed).  Prints ONE JSON line (rank 0):

  value        pixel*sensor updates/s (GUpd/s), whole job, inputs resident in HBM, CUDA events
               around exactly K steps, max over ranks; the region is measured 7 times and the median
               reported.  The steps are replayed from CUDA graphs of consecutive steps over R rotating
               plans (R * tau bytes > 3 x L2, so the tau stream cannot be served from L2); every plan
               is called once and two full rotations run before the first region, whatever --warmup is.
  roofline     the gather kernel alone: algorithmic bytes per launch (tau + traces + images,
               north_star's definition) / its mean launch duration (the gather launched back to back
               from the same kind of CUDA graph, pat_set_profiling mode 2, CUDA events around regions of
               >= 240 launches whatever --steps is), against the measured HBM copy peak of MEASURED_PEAKS.json.
  e2e          the same metric through the C-ABI with pinned HOST traces/images (H2D + D2H timed).
  cpu_baseline the oracle (oracle/pat_oracle.c) timed on this box's host cores, rank 0, N = 1.
  warm_l2      (labelled, not the headline) ONE plan, the same table every step -- the paper's "off-line once" case.
  large_workload_probe  the same path on configs[4] REDUCED (537 MB table): the gather's steady-state rate.
  conventional_bp  PAPER.md:69's comparison method with the delays computed in the kernel (no table stream).
  exact_time_weighting  Eq. 7 with p and dp/dt both taken at t_ij (PAT_W_PAPER_EXACT, two channels per frame).
  universal_bp     ref. [5]'s solid-angle-weighted sum: a weight table streamed next to the delays.
  offline_eikonal  (not part of the step) the tau table of the geometry solved on the GPU vs the CPU fast marching.
  sweep        B = 1..64 on the same geometry (N = 1 only): ms/frame, GUpd/s, HBM fraction and the
               SM-side (shared-memory bandwidth) fraction, because for B >~ 4 the path is not
               HBM-bound.

--impl reference times the CPU oracle as it stands on the same config / metric (rank 0 only).
Nothing here reads /root/reference; all inputs are seeded and synthetic (workloads/).
"""
import argparse
import json
import math
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as W  # noqa: E402

METRIC = "pixel-sensor updates/s (GUpd/s) at 512 sensors x 21323 px"
FALLBACK_HBM_GBS = 6650.0          # /opt/skills/guides/B200_PROFILING.md fallback
NOMINAL_HBM_GBS = 8000.0           # north_star's "~8 TB/s"
SMEM_BYTES_PER_CLK_SM = 128.0      # B300_MICROARCH.md: shared-memory bandwidth per SM


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=50)
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json configs[k] geometry (1, 2, 3, 4)")
    ap.add_argument("--batch", type=int, default=0, help="frames per step (0 = the config's own batch)")
    ap.add_argument("--reduced", action="store_true", help="reduced variant of config 3 / 4")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-sweep", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-warm", action="store_true", help="skip the labelled warm-L2 (single plan) line")
    ap.add_argument("--probe", default="", choices=["", "conventional", "eikonal", "exact", "ubp"],
                    help="run only this side probe on the config's geometry and print its JSON (ncu captures)")
    ap.add_argument("--tuning", type=str, default="", help="wr,rows,stages for pat_set_gather_tuning (0 = automatic)")
    return ap.parse_args()


def tuning_of(args):
    return tuple(int(v) for v in args.tuning.split(",")) if args.tuning else None


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)", float(d.get("sm_max_mhz", 1965.0))
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)", 1965.0


def algorithmic_bytes(S, P, Nt, B):
    """north_star: tau bytes (once per batch) + trace bytes + image bytes."""
    return 4.0 * S * P + 4.0 * B * S * Nt + 4.0 * B * P


class ClockSampler(threading.Thread):
    """nvidia-smi-equivalent clock / throttle-reason samples through NVML while the GPU is loaded."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.stop_flag, self.ok = index, [], False, False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.max_mhz = None

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        while not self.stop_flag:
            try:
                mhz = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                rs = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h) if hasattr(
                    nv, "nvmlDeviceGetCurrentClocksEventReasons") else nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                util = nv.nvmlDeviceGetUtilizationRates(self.h).gpu
                self.samples.append((mhz, rs, util))
            except Exception:
                pass
            time.sleep(0.002)

    def summary(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake_slowdown",
        }
        mhz = [s[0] for s in self.samples]
        top = max(mhz)
        load = [m for m in mhz if m >= 0.5 * top] or mhz
        bits = 0
        for s in self.samples:
            bits |= int(s[1])
        reasons = sorted(n for b, n in names.items() if bits & b)
        return {"sm_mhz": float(np.median(load)), "sm_max_mhz": self.max_mhz, "reasons": reasons,
                "samples": len(self.samples)}


# ---------------------------------------------------------------------------------------------
# input preparation (untimed)
# ---------------------------------------------------------------------------------------------
def prepare_inputs(k, reduced, nframes, frame0=0):
    """Geometry, tau (library CPU FMM -- north_star: input preparation, not timed), traces."""
    import paper_1501_03869_b200 as pat
    geom = W.make_geometry(k, reduced)
    grid = pat.PatGrid.make(geom.n, geom.h, geom.origin)
    tau = np.empty((geom.nsens, geom.npix), dtype=np.float32)
    pat.pat_fmm_travel_times(grid, np.ascontiguousarray(geom.c_map).ravel(), geom.sensors, geom.nsens,
                             geom.roi_index, geom.npix, 0, geom.nsens, 1, tau, 0)
    traces = W.make_traces(geom, tau, frames=range(frame0, frame0 + nframes))
    return geom, tau, traces


EIK_FLOPS_PER_UPDATE = {2: 14, 3: 26}   # fp64 operations of one upwind update as written in csrc/eikonal.cu (min/compare
                                        # per axis, sort, one- / two- / three-axis solve incl. the square root)
FP64_PEAK_TFLOPS = 40.0                 # NVIDIA's B200 data-sheet FP64 figure; the guides state none (context only)


def eikonal_probe(geom, sample=None, cpu_sample=64, reps=3):
    """SURVEY.md 8(f) NEXT-2, off the timed path: the travel-time table of this geometry solved on the GPU
    (fast sweeping, csrc/eikonal.cu) beside the library's CPU fast marching on the host cores (a sample of
    the sensors), wall clock, and how far the two tables are apart.  sample = n: only the first n sensors are
    solved (one chunk of a table that is solved chunk by chunk anyway); ms/sensor is what scales."""
    import torch
    import paper_1501_03869_b200 as pat
    grid = pat.PatGrid.make(geom.n, geom.h, geom.origin)
    cm = np.ascontiguousarray(geom.c_map, dtype=np.float32).ravel()
    S = geom.nsens
    n = S if sample is None else min(S, sample)
    out = torch.empty((n, geom.npix), dtype=torch.float32, device="cuda")
    best, rounds = None, 0
    for _ in range(reps):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        rounds = pat.pat_eikonal_travel_times_device(grid, cm, geom.sensors, S, geom.roi_index, geom.npix, 0, n, out)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    m = min(n, cpu_sample)
    tau = np.empty((m, geom.npix), dtype=np.float32)
    t0 = time.perf_counter()
    pat.pat_fmm_travel_times(grid, cm, geom.sensors, S, geom.roi_index, geom.npix, 0, m, 1, tau, 0)
    cpu = time.perf_counter() - t0
    d = np.abs(out[:m].cpu().numpy().view(np.int32).astype(np.int64) - tau.view(np.int32).astype(np.int64))
    nodes = float(np.prod(geom.n))
    ndim = len(geom.n)
    visits, iters, upd = pat.pat_eikonal_last_stats()        # work counters of the last (timed) solve
    sweeping = upd == 0                                       # PAT_EIK_ALGO=sweep: every pass visits every node
    if sweeping:
        upd = n * nodes * rounds * (1 << ndim)
    tf = upd * EIK_FLOPS_PER_UPDATE[ndim] / best / 1e12
    blk = 512 if ndim == 3 else 256
    halo = 1000 if ndim == 3 else 324
    # HBM traffic of the block-ordered solver: per visit the block's halo'd field (fp64) + its slowness in, the block out
    gbs = (visits * (halo + 2 * blk) * 8.0 / best / 1e9) if not sweeping else None
    return {"workload": "%d of %d sensors on the %s grid (first-order upwind, fp64)" % (n, S, "x".join(str(v) for v in geom.n)),
            "algorithm": "level-by-level fast sweeping" if sweeping else "block-ordered fast iterative method",
            "gpu_s": round(best, 4), "gpu_ms_per_sensor": round(best * 1e3 / n, 4), "rounds": int(rounds),
            "whole_table_s_at_this_rate": round(best / n * S, 2),
            "block_visits_per_block": None if sweeping else round(visits / (n * math.ceil(nodes / blk)), 2),
            "jacobi_iterations_per_visit": None if sweeping else round(iters / max(1, visits), 2),
            "node_updates_per_node": round(upd / (n * nodes), 2),
            "fp64_tflops": round(tf, 3), "fp64_frac_of_datasheet_peak": round(tf / FP64_PEAK_TFLOPS, 4),
            "field_traffic_gbs": None if gbs is None else round(gbs, 1),
            "bound": "barrier / shared-memory latency of the in-block iterations (DESIGN.md 7.4b): neither fp64 nor HBM",
            "cpu_fmm_ms_per_sensor": round(cpu * 1e3 / m, 4), "cpu_threads": os.cpu_count(), "cpu_sample_sensors": m,
            "speedup_vs_cpu_fmm": round((cpu / m) / (best / n), 2), "max_ulp_vs_cpu_fmm": int(d.max())}


CONV_FLOPS_PER_UPDATE = 17      # the METHOD's arithmetic: delay 3 sub/mul pairs folded as 2 sub + 2 mul +
                                # 1 add + sqrt + mul + sub + mul = 9, index map 4 (floor, k, a, 1 - a), interpolation 2 FMA = 4


def conventional_probe(geom, traces, batches=(1, 32), sm_mhz=1965.0):
    """the conventional BP (tau = |r - s|/c0 computed in the gather) on the
    same geometry.  No table stream, so the kernel is bound by arithmetic, not HBM: the roofline is the method's
    flops per update against the fp32 FMA peak (SMs x 128 lanes x 2 x clock).  Timed from a CUDA graph of 18 calls
    over three image buffers (traces resident, 4 MB/frame: they would fit L2 in any harness).  Last row: the c0
    sweep (one frame, 8 speeds per call -- the inner loop of the paper's automatic speed selection)."""
    import torch
    import paper_1501_03869_b200 as pat
    sms = torch.cuda.get_device_properties(torch.cuda.current_device()).multi_processor_count
    peak_tflops = sms * 128 * 2 * sm_mhz * 1e6 / 1e12
    out = []

    def timed(plan, call, calls_per_graph, reps):
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            call(0, st)                                              # set-up outside the capture
            st.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=st):
                for q in range(calls_per_graph):
                    call(q, st)
            for _ in range(3):
                g.replay()
            st.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(st)
            for _ in range(reps):
                g.replay()
            e1.record(st)
            st.synchronize()
        return e0.elapsed_time(e1) / (calls_per_graph * reps)

    for B in batches:
        tr = torch.from_numpy(np.ascontiguousarray(np.resize(traces, (B,) + traces.shape[1:]))).cuda()
        imgs = [torch.empty((B, geom.npix), dtype=torch.float32, device="cuda") for _ in range(3)]
        plan = pat.Plan(geom.n, geom.h, geom.origin, geom.c_map, geom.sensors, geom.roi_index, geom.nt, geom.fs,
                        geom.t0, max_batch=B)
        ms = timed(plan, lambda q, st: plan.backproject_conventional(tr, imgs[q % 3], 1560.0, B, st), 18, 20 if B == 1 else 4)
        upd = float(B) * geom.nsens * geom.npix
        tf = upd * CONV_FLOPS_PER_UPDATE / (ms * 1e-3) / 1e12
        out.append({"B": B, "c0": 1560.0, "ms_per_frame": round(ms / B, 6), "gupd_s": round(upd / (ms * 1e-3) / 1e9, 1),
                    "roofline": {"bound": "alu", "achieved": round(tf, 2), "peak": round(peak_tflops, 1), "unit": "TFLOP/s",
                                 "frac": round(tf / peak_tflops, 4), "flops_per_update": CONV_FLOPS_PER_UPDATE}})
        plan.close()
    K = 8
    c0s = np.linspace(1500.0, 1620.0, K).astype(np.float32)
    tr1 = torch.from_numpy(np.ascontiguousarray(traces[0])).cuda()
    imgs = [torch.empty((K, geom.npix), dtype=torch.float32, device="cuda") for _ in range(3)]
    plan = pat.Plan(geom.n, geom.h, geom.origin, geom.c_map, geom.sensors, geom.roi_index, geom.nt, geom.fs, geom.t0, max_batch=1)
    ms = timed(plan, lambda q, st: plan.backproject_conventional_sweep(tr1, imgs[q % 3], c0s, st), 18, 10)
    upd = float(K) * geom.nsens * geom.npix
    out.append({"sweep_speeds": K, "c0_range": [float(c0s[0]), float(c0s[-1])], "ms_per_call": round(ms, 6),
                "ms_per_image": round(ms / K, 6), "gupd_s": round(upd / (ms * 1e-3) / 1e9, 1)})
    plan.close()
    return out


def exact_time_probe(geom, tau, traces, peak_gbs, batches=(1, 16), steps=400):
    """Eq. 7 with p and dp/dt both interpolated at t_ij (PAT_W_PAPER_EXACT): the same
    table stream, two trace channels per frame through the pre-pass and the gather.  Timed like the headline
    (rotating plans so that the table comes from HBM, CUDA graph replay, events on the launching stream)."""
    import paper_1501_03869_b200 as pat
    out = []
    for B in batches:
        rig = Rig(geom, tau, traces, B, weighting=pat.PAT_W_PAPER_EXACT)
        n = max(20, steps // B)
        ms = time_steps(rig, n, 10, repeats=3) / n
        rig.close()
        upd = float(B) * geom.nsens * geom.npix
        out.append({"B": B, "ms_per_frame": round(ms / B, 6), "gupd_s": round(upd / (ms * 1e-3) / 1e9, 1),
                    "step_hbm_frac": round(algorithmic_bytes(geom.nsens, geom.npix, geom.nt, B) / (ms * 1e-3) / 1e9 / peak_gbs, 4)})
    return out


def universal_bp_probe(geom, tau, traces, peak_gbs, batches=(1, 32), steps=400):
    """the universal BP of ref. [5] = weighting 2p - 2t dp/dt with every term
    multiplied by dOmega_ij/Omega0_j (pat_compute_solid_angle_weights, radial normals): a second table of the size
    of the delays is streamed, so the algorithmic bytes are tau + weights + traces + images."""
    import paper_1501_03869_b200 as pat
    s = geom.sensors.astype(np.float64)
    nrm = (s / np.linalg.norm(s, axis=1, keepdims=True)).astype(np.float32)
    out = []
    for B in batches:
        rig = Rig(geom, tau, traces, B, weighting=pat.PAT_W_UBP, normals=nrm)
        n = max(20, steps // B)
        ms = time_steps(rig, n, 10, repeats=3) / n
        rig.close()
        upd = float(B) * geom.nsens * geom.npix
        nbytes = algorithmic_bytes(geom.nsens, geom.npix, geom.nt, B) + 4.0 * geom.nsens * geom.npix
        out.append({"B": B, "ms_per_frame": round(ms / B, 6), "gupd_s": round(upd / (ms * 1e-3) / 1e9, 1),
                    "step_hbm_frac": round(nbytes / (ms * 1e-3) / 1e9 / peak_gbs, 4)})
    return out


class Rig:
    """R rotating plans (own tau copy, traces, images) so that consecutive steps never find their
    tau table in L2: R * tau bytes > 3 x L2.  Device rigs replay CUDA graphs of consecutive steps; the
    host rig (e2e) makes direct C-ABI calls, as a user streaming frames from pinned memory does."""
    GRAPH_STEPS = 120           # steps per captured graph (a graph launch boundary every 120 steps)

    def __init__(self, geom, tau, traces, B, variant=0, host=False, weighting=None, normals=None, warm_l2=False):
        import torch
        import paper_1501_03869_b200 as pat
        self.pat, self.torch, self.geom, self.B = pat, torch, geom, B
        props = torch.cuda.get_device_properties(torch.cuda.current_device())
        l2 = getattr(props, "L2_cache_size", 126 << 20) or (126 << 20)
        step_bytes = algorithmic_bytes(geom.nsens, geom.npix, geom.nt, B)
        self.R = int(max(2, min(12, math.ceil(3.0 * l2 / step_bytes))))
        if warm_l2:                                        # ONE plan: the table may stay in L2 between steps
            self.R = 1
        self.l2_bytes = int(l2)
        self.plans, self.tr, self.img = [], [], []
        F = traces.shape[0]
        # buffers: one (traces, images) pair per plan; the warm-L2 rig has ONE plan and rotates three pairs, as a
        # caller streaming frames does (consecutive calls must not share an image buffer to overlap, include/pat.h)
        self.NB = 3 if warm_l2 else self.R
        for r in range(self.NB):
            if r < self.R:
                p = pat.Plan(geom.n, geom.h, geom.origin, None, geom.sensors, geom.roi_index, geom.nt, geom.fs,
                             geom.t0, weighting=pat.PAT_W_PAPER if weighting is None else weighting,
                             max_batch=B if weighting is None or weighting < pat.PAT_W_PAPER_EXACT else 2 * B)
                if variant:
                    pat.pat_set_gather_tuning(p.handle, *variant)
                p.set_travel_times(tau)
                if normals is not None:                            # universal BP: solid-angle table next to the delays
                    p.compute_solid_angle_weights(normals)
                self.plans.append(p)
            sel = [(r * B + f) % F for f in range(B)]
            t = torch.from_numpy(np.ascontiguousarray(traces[sel]))
            if host:
                self.tr.append(t.pin_memory())
                self.img.append(torch.empty((B, geom.npix), dtype=torch.float32).pin_memory())
            else:
                self.tr.append(t.cuda())
                self.img.append(torch.empty((B, geom.npix), dtype=torch.float32, device="cuda"))
        self.stream = torch.cuda.Stream()
        self.graphs, self.primed, self.use_graph = {}, False, not host
        self.last_regions = []
        torch.cuda.synchronize()

    def step(self, i):
        r, q = i % self.R, i % self.NB
        self.plans[r].backproject(self.tr[q], self.img[q], self.B, self.stream)

    def prime(self):
        """One direct call on every plan: the first call of a frame-count class builds its work list
        synchronously (pat.h), which must never land inside a timed region or a capture."""
        with self.torch.cuda.stream(self.stream):
            for r in range(max(self.R, self.NB)):
                self.step(r)
        self.torch.cuda.synchronize()
        self.primed = True

    def _graph(self, first, n):
        """CUDA graph of the n consecutive steps first .. first+n-1 of the plan rotation (cached)."""
        key = (first % max(self.R, self.NB), n)
        g = self.graphs.get(key)
        if g is None:
            torch = self.torch
            g = torch.cuda.CUDAGraph()
            with torch.cuda.stream(self.stream):
                with torch.cuda.graph(g, stream=self.stream):
                    for i in range(n):
                        self.step(first + i)
            self.graphs[key] = g
        return g

    def plan_region(self, nsteps):
        """The launches that make up exactly nsteps steps: graph replays only when use_graph (pieces of at
        most GRAPH_STEPS steps, the rotation continuing across pieces), direct calls otherwise."""
        if not self.primed:
            self.prime()
        if not self.use_graph:
            return [("direct", 0, nsteps)]
        out, i = [], 0
        while i < nsteps:
            n = min(self.GRAPH_STEPS, nsteps - i)
            out.append(("graph", self._graph(i, n), n))
            i += n
        return out

    def run(self, nsteps):
        """Enqueue exactly nsteps steps on self.stream."""
        with self.torch.cuda.stream(self.stream):
            for kind, g, n in self.plan_region(nsteps):
                if kind == "graph":
                    g.replay()
                else:
                    for i in range(n):
                        self.step(i)

    def drop_graphs(self):
        self.graphs = {}

    def launches(self):
        return sum(p.launches() for p in self.plans)

    def close(self):
        self.graphs = {}
        for p in self.plans:
            p.close()
        self.plans = []


REPEATS = 7                 # timed regions per number; the median is reported


def time_steps(rig, nsteps, warmup, dist=None, repeats=REPEATS):
    """Device time (ms) of exactly nsteps steps: barrier + synchronize on both sides, CUDA events on the
    launching stream, max over ranks -- measured `repeats` times, the median region is returned.  Before the
    first region every plan has been called once (work lists built) and at least two full rotations plus
    `warmup` steps have run, whatever --warmup says, so that a short driver run (--steps 20 --warmup 5) times
    the same steady state as a long one."""
    from paper_1501_03869_b200.sharding import max_over_ranks
    torch = rig.torch
    rig.plan_region(nsteps)                              # capture outside the timed region
    rig.run(max(warmup, 2 * rig.R))
    rig.run(nsteps)
    torch.cuda.synchronize()
    regions = []
    for rep in range(-2, repeats):                       # two dress rehearsals of the same structure first (not recorded):
        if dist is not None:                             # the first regions after the warm-up run 10 - 50 % long (lazy loading
            dist.barrier()                               # of the spin kernel, clocks and L2 state after the synchronize)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        if rig.use_graph:
            # device rigs: a ~30 us spin kernel in front of the first event keeps the stream busy while the host
            # enqueues the graph launches, so that the events bracket the K steps' execution on the device and not the
            # host's cudaGraphLaunch latency on an idle GPU (a 20-step region is ONE graph launch: ~10 us of it).  The
            # host rig (e2e, direct calls) is timed without it: there the host's enqueue cost is part of the number.
            with torch.cuda.stream(rig.stream):
                torch.cuda._sleep(60000)
        e0.record(rig.stream)
        rig.run(nsteps)
        e1.record(rig.stream)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        if dist is not None:
            ms = max_over_ranks(ms, dist, device="cuda")
            dist.barrier()
        if rep >= 0:
            regions.append(ms)
    rig.last_regions = regions
    return float(np.median(regions))


def kernel_only_ms(rig, mode, nsteps, warmup):
    """Mean device duration (ms per launch) of ONE kernel of the step -- mode 2 = the gather, 3 = the
    pre-pass, 4 = the stream probe (pat_set_profiling; measurement modes, unlocked by PAT_ENABLE_PROBES=1 at
    plan creation) -- launched back to back from CUDA graphs over the rotating plans and timed with CUDA
    events on the launching stream (so it includes the launch gap, as the kernel does inside the step; events
    recorded around every single launch would add microseconds)."""
    pat = rig.pat
    for p in rig.plans:
        pat.pat_set_profiling(p.handle, mode)
    rig.drop_graphs()
    ms = time_steps(rig, nsteps, warmup, repeats=5)
    for p in rig.plans:
        pat.pat_set_profiling(p.handle, 0)
    rig.drop_graphs()
    return ms / nsteps


def host_enqueue_us(rig, burst=64, bursts=60):
    """Host wall-clock microseconds one direct pat_backproject call takes to ENQUEUE (ctypes marshalling
    included).  Measured in short bursts that start on an idle GPU: a long loop of direct calls is throttled by
    the GPU itself once the launch queue is full (a direct-call step takes ~12 us of GPU time) and then measures
    the step, not the host.  Median over the last third of the bursts: the first ones run on a host core that has been
    idling in synchronize calls and has not clocked up yet (13.7 us per call falling to 7.5 us on the same box)."""
    torch = rig.torch
    if not rig.primed:
        rig.prime()
    out = []
    with torch.cuda.stream(rig.stream):
        for i in range(rig.R):
            rig.step(i)
        for _ in range(bursts):
            torch.cuda.synchronize()
            t = time.perf_counter()
            for i in range(burst):
                rig.step(i)
            out.append((time.perf_counter() - t) / burst * 1e6)
    torch.cuda.synchronize()
    rig.enqueue_bursts_us = [round(v, 2) for v in out]
    return float(np.median(out[-(bursts // 3):]))


def measure(geom, tau, traces, B, steps, warmup, variant, dist, peak_gbs, sm_mhz, do_e2e, kernels=True,
            warm_l2=False):
    """All device-side numbers of one (geometry, B) point."""
    S, P, Nt = geom.nsens, geom.npix, geom.nt
    upd = float(B) * S * P
    abytes = algorithmic_bytes(S, P, Nt, B)
    rig = Rig(geom, tau, traces, B, variant, warm_l2=warm_l2)
    rig.prime()                                          # first-call set-up outside every capture and region
    l0 = rig.launches()
    ms = time_steps(rig, steps, warmup, dist)
    out = {
        "B": B, "plans_rotated": rig.R, "ms_per_step": ms / steps, "ms_per_frame": ms / steps / B,
        "regions_ms_per_step": [round(r / steps, 7) for r in rig.last_regions],
        "gupd_s": upd * steps / (ms * 1e-3) / 1e9,
        "step_bytes": abytes,
        "step_hbm_frac": abytes * steps / (ms * 1e-3) / 1e9 / peak_gbs,
        "l2_bytes": rig.l2_bytes,
    }
    if kernels:
        # the kernel-only figures are their own measurement (not the K-step region): regions of >= 240 launches whatever
        # --steps is, so that the driver's short run reports the same steady state as a long one
        nk = max(2 * rig.R, 240, min(steps, 1000))
        gat_ms = kernel_only_ms(rig, 2, nk, min(warmup, 20))
        pre_ms = kernel_only_ms(rig, 3, nk, min(warmup, 20))
        # context for the roofline fraction: ONE kernel that only streams the step's footprint (table + b in,
        # images out), same rotation, same graph harness -- what a launch of this size can reach at all
        probe_ms = kernel_only_ms(rig, 4, nk, min(warmup, 20))
        out.update({"prepass_ms": pre_ms, "gather_ms": gat_ms, "stream_probe_ms": probe_ms,
                    "gather_gbs": abytes / (gat_ms * 1e-3) / 1e9})
        # SM-side bound: 8 B of shared-memory/L1 traffic per update at 128 B/clk/SM
        sms = rig.torch.cuda.get_device_properties(rig.torch.cuda.current_device()).multi_processor_count
        smem_upd_s = SMEM_BYTES_PER_CLK_SM / 8.0 * sms * sm_mhz * 1e6
        out["sm_side_frac"] = (upd / (gat_ms * 1e-3)) / smem_upd_s
        out["host_enqueue_us"] = host_enqueue_us(rig)
        out["host_enqueue_bursts_us"] = rig.enqueue_bursts_us
    out["launches_per_step"] = rig.plans[0].launches_per_call() if hasattr(rig.plans[0], "launches_per_call") else 2
    out["direct_call_launches_seen"] = rig.launches() - l0
    rig.close()
    if do_e2e:
        hrig = Rig(geom, tau, traces, B, variant, host=True)
        hrig.prime()                                     # every plan's first call (work-list build) is set-up
        n_e2e = max(2 * hrig.R, 200)                     # its own region length, whatever --steps is: in a 20-call
                                                         # region a third is pipeline fill (first H2D, last D2H uncovered)
        ms_h = time_steps(hrig, n_e2e, min(warmup, 10), dist)
        out["e2e_gupd_s"] = upd * n_e2e / (ms_h * 1e-3) / 1e9
        out["e2e_ms_per_step"] = ms_h / n_e2e
        out["e2e_steps_per_region"] = n_e2e
        out["trace_window"] = list(hrig.plans[0].trace_window())      # samples of every trace that cross the bus
        out["h2d"] = 4 * B * S * out["trace_window"][1]
        out["d2h"] = 4 * B * P
        hrig.close()
    return out


# ---------------------------------------------------------------------------------------------
# CPU oracle legs (the only places bench.py executes oracle/)
# ---------------------------------------------------------------------------------------------
def oracle_time(geom, tau, traces, reps=1):
    """Seconds per call of oracle.backproject on `traces` (as it stands: OpenMP over pixels)."""
    import oracle
    oracle.backproject(tau, traces[:1], geom.fs, geom.t0, 1)          # load + first touch
    best = float("inf")
    for _ in range(reps):
        t = time.perf_counter()
        oracle.backproject(tau, traces, geom.fs, geom.t0, 1)
        best = min(best, time.perf_counter() - t)
    return best


def host_cores():
    try:
        return len(os.sched_getaffinity(0))
    except Exception:
        return os.cpu_count() or 1


def set_omp_threads(n):
    """Thread count of the OpenMP runtime the oracle library runs on (the oracle's own code is untouched:
    its `parallel for` over pixels gives the same sums for any thread count).  Returns False if unavailable."""
    import ctypes
    try:
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
        return True
    except Exception:
        return False


def cpu_baseline(geom, tau, traces_all):
    """SURVEY.md 8(d) / BASELINE.md section 4: the oracle on all host cores and on ONE thread."""
    nf = min(16, traces_all.shape[0])
    sample = traces_all[:nf]
    cores = host_cores()
    set_omp_threads(cores)
    sec = oracle_time(geom, tau, sample, reps=2)
    upd = float(nf) * geom.nsens * geom.npix
    out = {"value": upd / sec / 1e9, "unit": "GUpd/s", "cores": cores, "kind": "oracle",
           "ms_per_frame": sec / nf * 1e3,
           "sample": "%d seeded frames of configs[%d] geometry (S=%d, P=%d, Nt=%d), one oracle call, best of 2"
                     % (nf, geom.k, geom.nsens, geom.npix, geom.nt)}
    n1 = min(2, nf)
    if set_omp_threads(1):
        sec1 = oracle_time(geom, tau, traces_all[:n1], reps=1)
        set_omp_threads(cores)
        out["one_thread"] = {"value": float(n1) * geom.nsens * geom.npix / sec1 / 1e9, "unit": "GUpd/s", "cores": 1,
                             "ms_per_frame": sec1 / n1 * 1e3, "sample": "%d of the same frames, one oracle call" % n1}
    return out


def config_of(k, geom, B):
    """The `config` object of the JSON line -- the SAME keys and values from both arms."""
    return {"workload": "configs[%d] %s: %d sensors x %d px, Nt=%d, %d frame(s)/step"
                        % (k, geom.name, geom.nsens, geom.npix, geom.nt, B),
            "nsens": geom.nsens, "npix": geom.npix, "nt": geom.nt, "frames_per_step": B,
            "weighting": "p - t*dp/dt (Eq. 7)"}


def prepare_inputs_oracle(k, reduced, nframes):
    """Input preparation of the --impl reference arm: geometry and traces from workloads/, the travel-time table
    from the ORACLE's own fast marching (oracle.fmm_rows).  Nothing of the product package is imported."""
    import oracle
    geom = W.make_geometry(k, reduced)
    tau = oracle.fmm_rows(geom.n, geom.h, geom.origin, geom.c_map, geom.sensors, geom.roi_index, order=1)
    traces = W.make_traces(geom, tau, frames=range(nframes))
    return geom, tau, traces


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on the same config / metric (rank 0 only).  Runs on
    oracle/ and workloads/ alone: the product library is neither imported nor mapped."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    k = args.config
    Bcfg = args.batch or W.make_geometry(k, args.reduced).batch
    nf = min(Bcfg, 4)                                    # bounded sample: <= 4 frames per step
    if k == 4 and not args.reduced:
        raise SystemExit("--impl reference: the oracle's fast marching of full-size configs[4] takes hours; use --reduced")
    geom, tau, traces = prepare_inputs_oracle(k, args.reduced, nf)
    import oracle
    set_omp_threads(host_cores())
    for _ in range(max(1, min(args.warmup, 3))):
        oracle_time(geom, tau, traces, reps=1)
    t = time.perf_counter()
    for _ in range(args.steps):
        oracle.backproject(tau, traces, geom.fs, geom.t0, 1)
    sec = time.perf_counter() - t
    upd = float(nf) * geom.nsens * geom.npix * args.steps
    val = upd / sec / 1e9
    sample = "each step = %d frame(s) of configs[%d] (S=%d, P=%d, Nt=%d) through oracle.backproject" % (
        nf, k, geom.nsens, geom.npix, geom.nt)
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": "GUpd/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "gpu_launches": 0,
        "config": config_of(k, geom, Bcfg),
        "harness": {"sampled_frames_per_step": nf, "tau": "oracle.fmm_rows (first order)"},
        "cpu_baseline": {"value": val, "unit": "GUpd/s", "cores": host_cores(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "GUpd/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))
    return 0


# ---------------------------------------------------------------------------------------------
# main (the CUDA arm)
# ---------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import paper_1501_03869_b200 as pat
    pat.lib()                                            # fails loudly if the extension is missing
    os.environ["PAT_ENABLE_PROBES"] = "1"                # unlocks pat_set_profiling's kernel-only modes (measurement)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (B200); there is no CPU fallback. "
                         "Use --impl reference for the CPU oracle arm.")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist_mod.init_process_group("nccl", device_id=torch.device("cuda", local))
        dist = dist_mod
    peak_gbs, peak_src, sm_max = measured_peaks()

    k = args.config
    geom0 = W.make_geometry(k, args.reduced)
    if args.probe:                                       # SURVEY.md 8(f) rows, off the headline path
        if args.probe == "eikonal":
            print(json.dumps({"offline_eikonal": eikonal_probe(geom0, sample=1024 if k == 4 and not args.reduced else None,
                                                               cpu_sample=16 if k == 4 else 64, reps=2)}))
        elif args.probe == "ubp":
            g1, tau1, tr1 = prepare_inputs(k, args.reduced, max(1, args.batch or 1))
            print(json.dumps({"universal_bp": universal_bp_probe(g1, tau1, tr1, peak_gbs, batches=(args.batch or 1,))}))
        elif args.probe == "exact":
            g1, tau1, tr1 = prepare_inputs(k, args.reduced, max(1, args.batch or 1))
            print(json.dumps({"exact_time_weighting": exact_time_probe(g1, tau1, tr1, peak_gbs, batches=(args.batch or 1,))}))
        else:
            g1, _, tr1 = prepare_inputs(k, args.reduced, 1)
            print(json.dumps({"conventional_bp": conventional_probe(g1, tr1, batches=(args.batch or 1,), sm_mhz=sm_max)}))
        return 0
    B = args.batch or geom0.batch
    do_sweep = (not args.no_sweep) and world == 1 and k in (1, 2) and not args.batch
    nframes = 64 if do_sweep else max(B, 16 if (world == 1 and not args.no_cpu_baseline) else B)
    # every rank owns its own frames: the path shards over frames with no exchange (weak scaling)
    from paper_1501_03869_b200.sharding import rank_frame_range
    geom, tau, traces = prepare_inputs(k, args.reduced, nframes, frame0=rank_frame_range(rank, world, nframes)[0])

    sampler = ClockSampler(local)
    sampler.start()
    main = measure(geom, tau, traces, B, args.steps, args.warmup, tuning_of(args), dist, peak_gbs, sm_max,
                   not args.no_e2e)
    clocks_main = None
    sweep = []
    if do_sweep:
        for b in (1, 2, 4, 8, 16, 32, 64):
            if b == B:
                m = main
            else:
                st = max(240 // min(b, 8), min(args.steps, int(args.steps * 4 / b)))      # side rows: >= 240 frames per region
                m = measure(geom, tau, traces, b, st, min(args.warmup, 10), tuning_of(args), None, peak_gbs,
                            sm_max, False)
            sweep.append({"B": b, "ms_per_frame": round(m["ms_per_frame"], 6),
                          "gupd_s": round(m["gupd_s"], 1),
                          "step_hbm_frac": round(m["step_hbm_frac"], 4),
                          "gather_hbm_frac": round(m["gather_gbs"] / peak_gbs, 4),
                          "sm_side_frac": round(m["sm_side_frac"], 4)})
    probe = None
    if do_sweep:
        # the same kernels on a table 11x larger (configs[4] reduced: 64^3 voxels x 512 sensors, 537 MB):
        # launch, prologue and tail weigh less there, so this shows the steady-state rate of the gather
        g4, tau4, tr4 = prepare_inputs(4, True, 1)
        m4 = measure(g4, tau4, tr4, 1, max(60, args.steps // 10), min(args.warmup, 10), tuning_of(args), None,
                     peak_gbs, sm_max, False)
        probe = {"workload": "configs[4] reduced: %d sensors x %d voxels, Nt=%d, 1 frame/step" % (g4.nsens, g4.npix, g4.nt),
                 "ms_per_frame": round(m4["ms_per_frame"], 6), "gupd_s": round(m4["gupd_s"], 1),
                 "step_hbm_frac": round(m4["step_hbm_frac"], 4), "gather_hbm_frac": round(m4["gather_gbs"] / peak_gbs, 4),
                 "note": "the REDUCED variant (537 MB table), not the 34.4 GB configs[4]; full size: tests/test_gpu_full3d.py"}
    eik, conv, exact, ubp, warm = None, None, None, None, None
    if world == 1 and k in (1, 2) and not args.no_warm:
        # the paper's use case: ONE table, computed "off-line ... once", every frame -- 43.7 MB fits
        # the L2, so consecutive steps may find it there.  Labelled; NOT the headline (which rotates plans).
        mw = measure(geom, tau, traces, B, max(240, min(args.steps, 1000)), min(args.warmup, 10), tuning_of(args), None,
                     peak_gbs, sm_max, False, kernels=False, warm_l2=True)
        warm = {"label": "warm L2: one plan, the same table every step (not the headline)", "plans_rotated": 1,
                "ms_per_step": mw["ms_per_step"], "gupd_s": round(mw["gupd_s"], 1),
                "algorithmic_bytes_over_time_vs_hbm_peak": round(mw["step_hbm_frac"], 4)}
    if do_sweep:
        eik = [eikonal_probe(geom),
               eikonal_probe(W.make_geometry(3), cpu_sample=32, reps=2),                 # configs[3]: 1024 sensors, 512 x 512
               eikonal_probe(W.make_geometry(4), sample=1024, cpu_sample=16, reps=1)]    # configs[4] FULL grid, one chunk
        conv = conventional_probe(geom, traces, sm_mhz=sm_max)
        exact = exact_time_probe(geom, tau, traces, peak_gbs)
        ubp = universal_bp_probe(geom, tau, traces, peak_gbs)
    sampler.stop_flag = True
    sampler.join(timeout=2.0)
    clocks_main = sampler.summary()

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    S, P, Nt = geom.nsens, geom.npix, geom.nt
    gather_gbs = main["gather_gbs"]
    line = {
        "metric": METRIC, "value": main["gupd_s"] * world, "unit": "GUpd/s", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": main["ms_per_step"],
        "ms_per_frame": main["ms_per_frame"], "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": config_of(k, geom, B),
        "harness": {"parallelism": "frames sharded over %d rank(s), no collective" % world,
                    "l2_policy": "inputs larger than L2: %d rotating plans x %.1f MB per step vs %.0f MB L2"
                                 % (main["plans_rotated"], main["step_bytes"] / 1e6, main["l2_bytes"] / 1e6),
                    "launch": "CUDA graph replay of pat_backproject (pre-pass + gather) per plan, graphs of <= %d "
                              "consecutive steps" % Rig.GRAPH_STEPS,
                    "timing": "median of %d regions of exactly `steps` steps each (CUDA events on the launching "
                              "stream, max over ranks per region; a 30 us spin kernel ahead of the first event hides the "
                              "host's graph-launch latency), after >= 2 full plan rotations of warm-up" % REPEATS,
                    "regions_ms_per_step": main["regions_ms_per_step"],
                    "host_enqueue_us_per_direct_call": round(main["host_enqueue_us"], 2),
                    "host_enqueue_bursts_us": main["host_enqueue_bursts_us"]},
        "host_enqueue_us": round(main["host_enqueue_us"], 2),
        "gpu_launches": int(main["launches_per_step"] * args.steps),
        "clocks": clocks_main,
        "roofline": {"bound": "hbm", "achieved": gather_gbs, "peak": peak_gbs, "unit": "GB/s",
                     "frac": gather_gbs / peak_gbs, "traffic": None, "peak_source": peak_src,
                     "kernel": "gather", "kernel_ms": main["gather_ms"], "prepass_ms": main["prepass_ms"],
                     "algorithmic_bytes_per_launch": main["step_bytes"],
                     "frac_of_nominal_8TBs": gather_gbs / NOMINAL_HBM_GBS,
                     "step_frac": main["step_hbm_frac"], "sm_side_frac": main["sm_side_frac"],
                     # a kernel that does nothing but stream the same bytes, timed the same way
                     "stream_probe": {"ms": main["stream_probe_ms"],
                                      "gbs": main["step_bytes"] / (main["stream_probe_ms"] * 1e-3) / 1e9,
                                      "frac": main["step_bytes"] / (main["stream_probe_ms"] * 1e-3) / 1e9 / peak_gbs,
                                      "gather_vs_probe": main["stream_probe_ms"] / main["gather_ms"]}},
        "paper_context": "PAPER.md:79: 123.79 ms for 512 sensors x 21323 px on a Tesla C2075, transfers included",
    }
    if "e2e_gupd_s" in main:
        line["e2e"] = {"value": main["e2e_gupd_s"] * world, "unit": "GUpd/s",
                       "h2d_bytes_per_step": main["h2d"], "d2h_bytes_per_step": main["d2h"],
                       "trace_samples_transferred": "[%d, +%d) of %d: all the table can touch (pat_get_trace_window)"
                                                    % (main["trace_window"][0], main["trace_window"][1], Nt),
                       "ms_per_step": main["e2e_ms_per_step"], "steps_per_region": main["e2e_steps_per_region"],
                       "launch": "direct pat_backproject calls with pinned host buffers (no graph)"}
    if warm:
        line["warm_l2"] = warm
    if sweep:
        line["sweep"] = sweep
    if probe:
        line["large_workload_probe"] = probe
    if eik:
        line["offline_eikonal"] = eik
    if conv:
        line["conventional_bp"] = conv
    if exact:
        line["exact_time_weighting"] = exact
    if ubp:
        line["universal_bp"] = ubp
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(geom, tau, traces)
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    try:                                                 # dram bytes per gather launch from the committed ncu capture
        with open(tpath) as f:
            line["roofline"]["traffic"] = json.load(f).get("configs[%d]/B=%d" % (k, B))
    except Exception:
        pass
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    a = parse_args()
    sys.exit(run_reference(a) if a.impl == "reference" else run_ours(a))

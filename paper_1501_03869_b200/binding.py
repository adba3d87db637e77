"""ctypes binding of include/pat.h -- argument marshalling only.

Every function has the name and argument order of its C counterpart.  Arrays may be numpy
arrays (host) or torch tensors (host or CUDA); a raw integer address is also accepted.
`Plan` is a small convenience owner of the handle and of the torch workspace tensor.
"""
import ctypes
import os

import numpy as np

PAT_OK, PAT_ERR_INVALID_ARG, PAT_ERR_BAD_STATE, PAT_ERR_CUDA, PAT_ERR_NOMEM, PAT_ERR_UNSUPPORTED = range(6)
PAT_W_DELAY_SUM, PAT_W_PAPER, PAT_W_UBP, PAT_W_PAPER_EXACT, PAT_W_UBP_EXACT = 0, 1, 2, 3, 4
_STATUS = ["PAT_OK", "PAT_ERR_INVALID_ARG", "PAT_ERR_BAD_STATE", "PAT_ERR_CUDA", "PAT_ERR_NOMEM",
           "PAT_ERR_UNSUPPORTED"]

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBNAME = "libpat_b200.so"


class PatError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("%s: %s" % (_STATUS[status] if 0 <= status < len(_STATUS) else status, msg))
        self.status = status


class PatGrid(ctypes.Structure):
    _fields_ = [("ndim", ctypes.c_int32), ("n", ctypes.c_int32 * 3), ("h", ctypes.c_float),
                ("origin", ctypes.c_float * 3)]

    @classmethod
    def make(cls, n, h, origin):
        g = cls()
        g.ndim = len(n)
        for d in range(3):
            g.n[d] = int(n[d]) if d < len(n) else 1
            g.origin[d] = float(origin[d]) if d < len(origin) else 0.0
        g.h = float(h)
        return g


class PatStats(ctypes.Structure):
    _fields_ = [("workspace_bytes", ctypes.c_int64), ("provider_bytes", ctypes.c_int64),
                ("provider_bytes_peak", ctypes.c_int64), ("work_list_bytes", ctypes.c_int64),
                ("work_lists", ctypes.c_int64), ("work_list_build_seconds", ctypes.c_double),
                ("kernel_launches", ctypes.c_int64), ("chained_calls", ctypes.c_int64)]


def library_path():
    return os.path.join(_HERE, _LIBNAME)


_lib = None


def lib():
    """Load libpat_b200.so (built in-tree by paper_1501_03869_b200/build.py). No fallback."""
    global _lib
    if _lib is not None:
        return _lib
    path = library_path()
    if not os.path.exists(path):
        raise ImportError(
            "%s is missing: build it with `python -m paper_1501_03869_b200.build` "
            "(nvcc, sm_100a). There is no CPU or PyTorch fallback for this package." % path)
    L = ctypes.CDLL(path)
    i32, i64, f32, vp, sz = ctypes.c_int32, ctypes.c_int64, ctypes.c_float, ctypes.c_void_p, ctypes.c_size_t
    gp = ctypes.POINTER(PatGrid)
    L.pat_plan_workspace_bytes.restype = sz
    L.pat_plan_workspace_bytes.argtypes = [gp, i32, i64, i32, i32]
    L.pat_plan_create.restype = ctypes.c_int
    L.pat_plan_create.argtypes = [ctypes.POINTER(vp), gp, vp, vp, i32, vp, i64, i32, f32, f32, i32, i32, vp, sz]
    L.pat_set_travel_times.restype = ctypes.c_int
    L.pat_set_travel_times.argtypes = [vp, vp, i32, i32, vp]
    L.pat_backproject.restype = ctypes.c_int
    L.pat_backproject.argtypes = [vp, vp, vp, i32, vp]
    L.pat_destroy.restype = ctypes.c_int
    L.pat_destroy.argtypes = [vp]
    L.pat_last_error.restype = ctypes.c_char_p
    L.pat_last_error.argtypes = [vp]
    L.pat_kernel_launches.restype = i64
    L.pat_kernel_launches.argtypes = [vp]
    L.pat_set_device_allocator.restype = ctypes.c_int
    L.pat_set_device_allocator.argtypes = [vp, vp, vp]
    L.pat_get_stats.restype = ctypes.c_int
    L.pat_get_stats.argtypes = [vp, ctypes.POINTER(PatStats)]
    L.pat_chained_calls.restype = i64
    L.pat_chained_calls.argtypes = [vp]
    L.pat_set_gather_tuning.restype = ctypes.c_int
    L.pat_set_gather_tuning.argtypes = [vp, i32, i32, i32]
    L.pat_set_profiling.restype = ctypes.c_int
    L.pat_set_profiling.argtypes = [vp, i32]
    L.pat_get_profile.restype = ctypes.c_int
    L.pat_get_profile.argtypes = [vp, i32, ctypes.POINTER(i64), ctypes.POINTER(ctypes.c_double),
                                  ctypes.POINTER(ctypes.c_double)]
    L.pat_fmm_travel_times.restype = ctypes.c_int
    L.pat_fmm_travel_times.argtypes = [gp, vp, vp, i32, vp, i64, i32, i32, i32, vp, i32]
    L.pat_compute_travel_times.restype = ctypes.c_int
    L.pat_compute_travel_times.argtypes = [vp, i32, i32, vp]
    L.pat_get_trace_window.restype = ctypes.c_int
    L.pat_get_trace_window.argtypes = [vp, ctypes.POINTER(i32), ctypes.POINTER(i32)]
    L.pat_set_pixel_weights.restype = ctypes.c_int
    L.pat_set_pixel_weights.argtypes = [vp, vp, i32, i32, vp]
    L.pat_compute_solid_angle_weights.restype = ctypes.c_int
    L.pat_compute_solid_angle_weights.argtypes = [vp, vp, vp]
    L.pat_set_roi_mask.restype = ctypes.c_int
    L.pat_set_roi_mask.argtypes = [vp, vp]
    L.pat_backproject_conventional.restype = ctypes.c_int
    L.pat_backproject_conventional.argtypes = [vp, vp, vp, i32, ctypes.c_float, vp]
    L.pat_backproject_conventional_sweep.restype = ctypes.c_int
    L.pat_backproject_conventional_sweep.argtypes = [vp, vp, vp, vp, i32, vp]
    L.pat_eikonal_travel_times_device.restype = ctypes.c_int
    L.pat_eikonal_travel_times_device.argtypes = [gp, vp, vp, i32, vp, i64, i32, i32, vp, i32,
                                                  ctypes.POINTER(i32), vp]
    L.pat_compute_travel_times_gpu.restype = ctypes.c_int
    L.pat_compute_travel_times_gpu.argtypes = [vp, i32, ctypes.POINTER(i32), vp]
    L.pat_pixel_order.restype = ctypes.c_int
    L.pat_pixel_order.argtypes = [gp, vp, i64, i32, vp]
    L.pat_eikonal_last_stats.restype = ctypes.c_int
    L.pat_eikonal_last_stats.argtypes = [ctypes.POINTER(i64)] * 3
    L.pat_backproject_static.restype = ctypes.c_int
    L.pat_backproject_static.argtypes = [vp, vp, vp, i32, i64, i32, i32, f32, f32, i32, vp]
    L.pat_backproject_static_max_samples.restype = i64
    L.pat_backproject_static_max_samples.argtypes = []
    L.pat_backproject_static_last_error.restype = ctypes.c_char_p
    L.pat_backproject_static_last_error.argtypes = []
    _lib = L
    return L


# ---- device-memory provider (include/pat.h "device memory"): torch tensors, so that the caller's allocator owns
# everything -- the library itself never calls cudaMalloc once a provider is installed -----------------------
_ALLOC_CB = ctypes.CFUNCTYPE(ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p)
_FREE_CB = ctypes.CFUNCTYPE(None, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p)
_provider = {"alloc": None, "free": None, "live": {}, "py_alloc": None, "py_free": None}


def pat_set_device_allocator(alloc=None, free=None):
    """alloc(nbytes) -> 256-byte aligned device address (int) or None; free(address, nbytes).  Both None: the
    library's cudaMalloc shim again.  The callbacks are kept alive by this module."""
    if (alloc is None) != (free is None):
        raise ValueError("alloc and free must be given together")
    if alloc is None:
        st = lib().pat_set_device_allocator(None, None, None)
        _provider.update(alloc=None, free=None, py_alloc=None, py_free=None)
    else:
        def _a(nbytes, _user):
            try:
                return alloc(int(nbytes))
            except Exception:
                return None
        def _f(ptr, nbytes, _user):
            try:
                free(int(ptr), int(nbytes))
            except Exception:
                pass
        ca, cf = _ALLOC_CB(_a), _FREE_CB(_f)
        st = lib().pat_set_device_allocator(ctypes.cast(ca, ctypes.c_void_p), ctypes.cast(cf, ctypes.c_void_p), None)
        _provider.update(alloc=ca, free=cf, py_alloc=alloc, py_free=free)
    if st != PAT_OK:
        raise PatError(st, "pat_set_device_allocator")


def torch_alloc(nbytes):
    import torch
    t = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
    ptr = (t.data_ptr() + 255) // 256 * 256
    _provider["live"][ptr] = t
    return ptr


def torch_free(ptr, nbytes):
    _provider["live"].pop(ptr, None)


def install_torch_allocator():
    """Make torch the provider (idempotent; does not replace a provider the caller has installed)."""
    if _provider["alloc"] is None:
        pat_set_device_allocator(torch_alloc, torch_free)


def pat_get_stats(plan):
    st = PatStats()
    _check(plan, lib().pat_get_stats(plan, ctypes.byref(st)))
    return {k: getattr(st, k) for k, _ in PatStats._fields_}


def _addr(a):
    """Address of a numpy array, a torch tensor, an int, or None."""
    if a is None:
        return None
    if isinstance(a, int):
        return a
    if isinstance(a, np.ndarray):
        if not a.flags["C_CONTIGUOUS"]:
            raise ValueError("array must be C-contiguous")
        return a.ctypes.data
    if hasattr(a, "data_ptr"):
        if not a.is_contiguous():
            raise ValueError("tensor must be contiguous")
        return a.data_ptr()
    raise TypeError("expected numpy array, torch tensor, int address or None")


def _stream(stream):
    if stream is None:
        return None
    if isinstance(stream, int):
        return stream or None
    return stream.cuda_stream or None            # torch.cuda.Stream


def _check(plan, st):
    if st != PAT_OK:
        raise PatError(st, pat_last_error(plan))
    return st


def pat_plan_workspace_bytes(grid, nsens, npix, nt, max_batch):
    return int(lib().pat_plan_workspace_bytes(ctypes.byref(grid), nsens, npix, nt, max_batch))


def pat_plan_create(grid, c_map, sensor_xyz, nsens, roi_index, npix, nt, fs, t0, weighting, max_batch,
                    workspace, workspace_bytes):
    """Returns the opaque plan handle (int). Raises PatError on failure."""
    for arr, dt in ((c_map, np.float32), (sensor_xyz, np.float32), (roi_index, np.int64)):
        if isinstance(arr, np.ndarray) and arr.dtype != dt:
            raise TypeError("host array has dtype %s, expected %s" % (arr.dtype, np.dtype(dt)))
    h = ctypes.c_void_p()
    st = lib().pat_plan_create(ctypes.byref(h), ctypes.byref(grid), _addr(c_map), _addr(sensor_xyz), nsens,
                               _addr(roi_index), npix, nt, fs, t0, weighting, max_batch,
                               _addr(workspace), workspace_bytes)
    _check(None, st)
    return h.value


def pat_set_travel_times(plan, tau, sensor_begin, count, stream=None):
    if isinstance(tau, np.ndarray) and tau.dtype != np.float32:
        raise TypeError("tau must be float32")
    return _check(plan, lib().pat_set_travel_times(plan, _addr(tau), sensor_begin, count, _stream(stream)))


def pat_backproject(plan, traces, images, nframes, stream=None):
    return _check(plan, lib().pat_backproject(plan, _addr(traces), _addr(images), nframes, _stream(stream)))


def pat_backproject_conventional(plan, traces, images, nframes, c0, stream=None):
    """Eq. 7 with tau = |r - s| / c0 computed in the kernel."""
    return _check(plan, lib().pat_backproject_conventional(plan, _addr(traces), _addr(images), nframes,
                                                           float(c0), _stream(stream)))


def pat_backproject_conventional_sweep(plan, traces, images, c0, stream=None):
    """One frame, len(c0) speeds: images[q] = conventional BP with c0[q] (the c0 selection's inner loop)."""
    c0 = np.ascontiguousarray(c0, dtype=np.float32)
    return _check(plan, lib().pat_backproject_conventional_sweep(plan, _addr(traces), _addr(images), _addr(c0),
                                                                 int(c0.size), _stream(stream)))


def pat_get_trace_window(plan):
    """(first, count): the samples of every trace a host-buffer call transfers (all the table can touch)."""
    a, b = ctypes.c_int32(), ctypes.c_int32()
    _check(plan, lib().pat_get_trace_window(plan, ctypes.byref(a), ctypes.byref(b)))
    return a.value, b.value


def pat_set_pixel_weights(plan, w, sensor_begin=0, count=None, stream=None):
    """w: fp32 [count][npix] (numpy or torch) factors multiplying every term; None removes the weights."""
    if w is None:
        return _check(plan, lib().pat_set_pixel_weights(plan, None, 0, 0, _stream(stream)))
    if isinstance(w, np.ndarray) and w.dtype != np.float32:
        raise TypeError("w must be float32")
    count = int(w.shape[0]) if count is None else count
    return _check(plan, lib().pat_set_pixel_weights(plan, _addr(w), sensor_begin, count, _stream(stream)))


def pat_compute_solid_angle_weights(plan, normals, stream=None):
    """Universal-BP factors dOmega_ij/Omega0_j from the plan's geometry; normals: host fp32 [nsens][3]."""
    normals = np.ascontiguousarray(normals, dtype=np.float32)
    return _check(plan, lib().pat_compute_solid_angle_weights(plan, _addr(normals), _stream(stream)))


def pat_set_roi_mask(plan, mask):
    """mask: host uint8 [npix] (non-zero = reconstruct) or None for all pixels."""
    if mask is not None:
        mask = np.ascontiguousarray(mask, dtype=np.uint8)
    return _check(plan, lib().pat_set_roi_mask(plan, _addr(mask) if mask is not None else None))


def pat_destroy(plan):
    return lib().pat_destroy(plan)


def pat_last_error(plan):
    return lib().pat_last_error(plan).decode()


def pat_kernel_launches(plan):
    return int(lib().pat_kernel_launches(plan))


def pat_chained_calls(plan):
    """Calls whose pre-pass was chained behind the previous call's gather (cross-call overlap inside a capture)."""
    return int(lib().pat_chained_calls(plan))


def pat_set_gather_tuning(plan, wr=0, rows=0, stages=0):
    return _check(plan, lib().pat_set_gather_tuning(plan, wr, rows, stages))


def pat_set_profiling(plan, mode):
    """0 off, 1 events per kernel, 2 gather only, 3 pre-pass only, 4 stream probe (see include/pat.h)."""
    return _check(plan, lib().pat_set_profiling(plan, int(mode)))


def pat_get_profile(plan, reset=True):
    """(calls, prepass_ms, gather_ms) summed since the last reset."""
    n, a, b = ctypes.c_int64(), ctypes.c_double(), ctypes.c_double()
    _check(plan, lib().pat_get_profile(plan, int(reset), ctypes.byref(n), ctypes.byref(a), ctypes.byref(b)))
    return n.value, a.value, b.value


def pat_fmm_travel_times(grid, c_map, sensor_xyz, nsens, roi_index, npix, sensor_begin, count, order,
                         tau_out, nthreads=0):
    st = lib().pat_fmm_travel_times(ctypes.byref(grid), _addr(c_map), _addr(sensor_xyz), nsens,
                                    _addr(roi_index), npix, sensor_begin, count, order, _addr(tau_out), nthreads)
    if st != PAT_OK:
        raise PatError(st, "pat_fmm_travel_times")
    return st


def pat_compute_travel_times(plan, order=1, nthreads=0, stream=None):
    return _check(plan, lib().pat_compute_travel_times(plan, order, nthreads, _stream(stream)))


def pat_eikonal_travel_times_device(grid, c_map, sensor_xyz, nsens, roi_index, npix, sensor_begin, count,
                                    tau_out, max_rounds=0, stream=None):
    """GPU fast-sweeping solve (include/pat.h); tau_out is a DEVICE fp32 [count][npix] tensor.
    Returns the largest number of rounds any sensor needed."""
    install_torch_allocator()
    r = ctypes.c_int32()
    st = lib().pat_eikonal_travel_times_device(ctypes.byref(grid), _addr(c_map), _addr(sensor_xyz), nsens,
                                               _addr(roi_index) if roi_index is not None else None, npix,
                                               sensor_begin, count, _addr(tau_out), int(max_rounds),
                                               ctypes.byref(r), _stream(stream))
    if st != PAT_OK:
        raise PatError(st, "pat_eikonal_travel_times_device failed")
    return r.value


def pat_pixel_order(grid, roi_index, npix, plain_morton=False):
    """Slot order of the tile-major table (host only): int32 array of ceil(npix/256)*256 entries, -1 = padding."""
    out = np.empty(((int(npix) + 255) // 256) * 256, dtype=np.int32)
    st = lib().pat_pixel_order(ctypes.byref(grid), _addr(roi_index), int(npix), 1 if plain_morton else 0, _addr(out))
    if st != PAT_OK:
        raise PatError(st, "pat_pixel_order")
    return out


def pat_eikonal_last_stats():
    """(block visits, Jacobi iterations, node updates) of this thread's latest GPU eikonal call."""
    v = [ctypes.c_int64(0) for _ in range(3)]
    lib().pat_eikonal_last_stats(*[ctypes.byref(x) for x in v])
    return tuple(int(x.value) for x in v)


def pat_compute_travel_times_gpu(plan, max_rounds=0, stream=None):
    r = ctypes.c_int32()
    _check(plan, lib().pat_compute_travel_times_gpu(plan, int(max_rounds), ctypes.byref(r), _stream(stream)))
    return r.value


def pat_backproject_static_max_samples():
    return int(lib().pat_backproject_static_max_samples())


def pat_backproject_static_last_error():
    return lib().pat_backproject_static_last_error().decode()


def pat_backproject_static(tau, traces, images, nsens, npix, nt, nframes, fs, t0=0.0, weighting=PAT_W_PAPER,
                           stream=None):
    """The entry point that allocates nothing (include/pat.h): device pointers in, images out, scratch in a
    static __device__ array of pat_backproject_static_max_samples() floats."""
    st = lib().pat_backproject_static(_addr(tau), _addr(traces), _addr(images), int(nsens), int(npix), int(nt),
                                      int(nframes), float(fs), float(t0), int(weighting), _stream(stream))
    if st != PAT_OK:
        raise PatError(st, pat_backproject_static_last_error())
    return st


class Plan:
    """Owns a plan handle and its torch workspace tensor (device memory stays torch's)."""

    def __init__(self, n, h, origin, c_map, sensor_xyz, roi_index, nt, fs, t0=0.0,
                 weighting=PAT_W_PAPER, max_batch=1, device="cuda", nsens=None):
        import torch
        install_torch_allocator()
        self.grid = PatGrid.make(n, h, origin)
        self.c_map = None if c_map is None else np.ascontiguousarray(c_map, dtype=np.float32).ravel()
        self.sensor_xyz = None if sensor_xyz is None else np.ascontiguousarray(sensor_xyz, dtype=np.float32)
        self.roi_index = None if roi_index is None else np.ascontiguousarray(roi_index, dtype=np.int64)
        self.nsens = int(self.sensor_xyz.shape[0]) if self.sensor_xyz is not None else int(nsens)
        self.npix = int(self.roi_index.size) if self.roi_index is not None else int(np.prod(n))
        self.nt, self.fs, self.t0, self.max_batch = int(nt), float(fs), float(t0), int(max_batch)
        nbytes = pat_plan_workspace_bytes(self.grid, self.nsens, self.npix, self.nt, self.max_batch)
        if nbytes == 0:
            raise PatError(PAT_ERR_INVALID_ARG, "invalid plan sizes")
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=device)
        base = self.workspace.data_ptr()
        self._ws_addr = (base + 255) // 256 * 256
        self.handle = pat_plan_create(self.grid, self.c_map, self.sensor_xyz, self.nsens, self.roi_index,
                                      self.npix, self.nt, self.fs, self.t0, weighting, self.max_batch,
                                      self._ws_addr, nbytes)

    def set_travel_times(self, tau, sensor_begin=0, count=None, stream=None):
        count = int(tau.shape[0]) if count is None else count
        return pat_set_travel_times(self.handle, tau, sensor_begin, count, stream)

    def compute_travel_times(self, order=1, nthreads=0, stream=None):
        return pat_compute_travel_times(self.handle, order, nthreads, stream)

    def compute_travel_times_gpu(self, max_rounds=0, stream=None):
        """First-order solve on the GPU (fast sweeping); returns the rounds the slowest sensor took."""
        return pat_compute_travel_times_gpu(self.handle, max_rounds, stream)

    def backproject(self, traces, images, nframes=None, stream=None):
        nframes = int(traces.shape[0]) if nframes is None else nframes
        return pat_backproject(self.handle, traces, images, nframes, stream)

    def backproject_conventional(self, traces, images, c0, nframes=None, stream=None):
        nframes = int(traces.shape[0]) if nframes is None else nframes
        return pat_backproject_conventional(self.handle, traces, images, nframes, c0, stream)

    def backproject_conventional_sweep(self, traces, images, c0, stream=None):
        return pat_backproject_conventional_sweep(self.handle, traces, images, c0, stream)

    def set_pixel_weights(self, w, sensor_begin=0, count=None, stream=None):
        return pat_set_pixel_weights(self.handle, w, sensor_begin, count, stream)

    def compute_solid_angle_weights(self, normals, stream=None):
        return pat_compute_solid_angle_weights(self.handle, normals, stream)

    def trace_window(self):
        return pat_get_trace_window(self.handle)

    def set_roi_mask(self, mask):
        return pat_set_roi_mask(self.handle, mask)

    def launches(self):
        return pat_kernel_launches(self.handle)

    def chained_calls(self):
        return pat_chained_calls(self.handle)

    def stats(self):
        return pat_get_stats(self.handle)

    def close(self):
        if getattr(self, "handle", None):
            pat_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

"""CPU oracle for arxiv 1501.03869 (FMM + Eq. 7 back projection).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs, never from the product
package.  Thin ctypes marshalling over oracle/pat_oracle.c; no arithmetic of
the method lives in this file.
"""
import ctypes
import os

import numpy as np

from .build import build as _build

_lib = None

# (wp, wd) of  b = wp*p - wd*t*dp/dt  (Eq. 7; reading R1)
# modes 3, 4: the same weights with p and dp/dt each interpolated AT t_ij and t = t_ij (Eq. 7 read
# literally; R4b) -> oracle_backproject_exact
WEIGHTS = {0: (1.0, 0.0), 1: (1.0, 1.0), 2: (2.0, 2.0), 3: (1.0, 1.0), 4: (2.0, 2.0)}
EXACT_TIME_MODES = (3, 4)


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(_build())
        i32, i64, f32, f64 = ctypes.c_int32, ctypes.c_int64, ctypes.c_float, ctypes.c_double
        vp = ctypes.c_void_p
        L.oracle_fmm.restype = ctypes.c_int
        L.oracle_fmm.argtypes = [i32, vp, f64, vp, vp, vp, i32, vp, vp]
        L.oracle_fmm_rows.restype = ctypes.c_int
        L.oracle_fmm_rows.argtypes = [i32, vp, f64, vp, vp, vp, i32, vp, i64, i32, vp]
        L.oracle_tau_conventional.restype = ctypes.c_int
        L.oracle_tau_conventional.argtypes = [i32, vp, f32, vp, vp, i32, vp, i64, f32, vp]
        L.oracle_weight.restype = None
        L.oracle_weight.argtypes = [vp, i32, f64, f64, f64, vp]
        L.oracle_backproject.restype = ctypes.c_int
        L.oracle_backproject.argtypes = [vp, i64, vp, i32, i64, i32, i32, f32, f32, f64, f64, vp]
        L.oracle_solid_angle_weights.restype = ctypes.c_int
        L.oracle_solid_angle_weights.argtypes = [i32, vp, f32, vp, vp, vp, i32, vp, i64, vp, vp]
        L.oracle_backproject_weighted.restype = ctypes.c_int
        L.oracle_backproject_weighted.argtypes = [vp, vp, i64, vp, i32, i64, i32, i32, f32, f32, f64, f64, vp]
        L.oracle_backproject_exact.restype = ctypes.c_int
        L.oracle_backproject_exact.argtypes = L.oracle_backproject.argtypes
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def fmm(n, h, origin, c_map, src, order=1, return_order=False):
    """Arrival times (double, shape n[::-1]) from a point source."""
    ndim = len(n)
    n3 = np.array(list(n) + [1] * (3 - ndim), dtype=np.int32)
    org = np.array(list(origin) + [0.0] * (3 - len(origin)), dtype=np.float64)
    s = np.array(list(src) + [0.0] * (3 - len(src)), dtype=np.float64)
    c = np.ascontiguousarray(c_map, dtype=np.float32).ravel()
    N = int(np.prod(n3))
    assert c.size == N
    T = np.empty(N, dtype=np.float64)
    fo = np.full(N, -1, dtype=np.int64) if return_order else None
    rc = lib().oracle_fmm(ndim, _p(n3), float(h), _p(org), _p(c), _p(s), int(order), _p(T),
                          _p(fo) if fo is not None else None)
    if rc:
        raise ValueError("oracle_fmm failed with code %d" % rc)
    T = T.reshape(tuple(int(v) for v in n3[:ndim][::-1]))
    return (T, fo) if return_order else T


def fmm_rows(n, h, origin, c_map, sensors, roi_index, order=1):
    """tau[i][j] fp32 = arrival time sensor i -> ROI node j (reciprocity)."""
    ndim = len(n)
    n3 = np.array(list(n) + [1] * (3 - ndim), dtype=np.int32)
    org = np.array(list(origin) + [0.0] * (3 - len(origin)), dtype=np.float64)
    c = np.ascontiguousarray(c_map, dtype=np.float32).ravel()
    sens = np.ascontiguousarray(sensors, dtype=np.float64).reshape(-1, 3)
    roi = np.ascontiguousarray(roi_index, dtype=np.int64)
    tau = np.empty((sens.shape[0], roi.size), dtype=np.float32)
    rc = lib().oracle_fmm_rows(ndim, _p(n3), float(h), _p(org), _p(c), _p(sens), sens.shape[0],
                               _p(roi), roi.size, int(order), _p(tau))
    if rc:
        raise ValueError("oracle_fmm_rows failed with code %d" % rc)
    return tau


def tau_conventional(n, h, origin, sensors, roi_index, c0):
    """tau[i][j] fp32 = |r_j - s_i| / c0 in the fp32 operation order the oracle fixes."""
    ndim = len(n)
    n3 = np.array(list(n) + [1] * (3 - ndim), dtype=np.int32)
    org = np.array(list(origin) + [0.0] * (3 - len(origin)), dtype=np.float32)
    sens = np.ascontiguousarray(sensors, dtype=np.float32).reshape(-1, 3)
    roi = None if roi_index is None else np.ascontiguousarray(roi_index, dtype=np.int64)
    npix = int(np.prod(n3)) if roi is None else roi.size
    tau = np.empty((sens.shape[0], npix), dtype=np.float32)
    rc = lib().oracle_tau_conventional(ndim, _p(n3), float(np.float32(h)), _p(org), _p(sens), sens.shape[0],
                                       _p(roi) if roi is not None else None, npix, float(np.float32(c0)), _p(tau))
    if rc:
        raise ValueError("oracle_tau_conventional failed with code %d" % rc)
    return tau


def weight(p, mode=1, t0fs=0.0):
    """b[n] = wp*p[n] - wd*(n + t0*fs)*D[n] in double."""
    p = np.ascontiguousarray(p, dtype=np.float32)
    b = np.empty(p.size, dtype=np.float64)
    wp, wd = WEIGHTS[mode]
    lib().oracle_weight(_p(p), p.size, wp, wd, float(t0fs), _p(b))
    return b


def solid_angle_weights(n, h, origin, sensors, normals, roi_index, return_omega0=False):
    """w[i][j] fp32 = dOmega_ij / Omega0_j of the universal BP [5] (R27)."""
    ndim = len(n)
    n3 = np.array(list(n) + [1] * (3 - ndim), dtype=np.int32)
    org = np.array(list(origin) + [0.0] * (3 - len(origin)), dtype=np.float32)
    sens = np.ascontiguousarray(sensors, dtype=np.float32).reshape(-1, 3)
    nrm = np.ascontiguousarray(normals, dtype=np.float32).reshape(-1, 3)
    assert nrm.shape == sens.shape
    roi = None if roi_index is None else np.ascontiguousarray(roi_index, dtype=np.int64)
    npix = int(np.prod(n3)) if roi is None else roi.size
    w = np.empty((sens.shape[0], npix), dtype=np.float32)
    om = np.empty(npix, dtype=np.float64)
    rc = lib().oracle_solid_angle_weights(ndim, _p(n3), float(np.float32(h)), _p(org), _p(sens), _p(nrm),
                                          sens.shape[0], _p(roi) if roi is not None else None, npix, _p(w), _p(om))
    if rc:
        raise ValueError("oracle_solid_angle_weights failed with code %d" % rc)
    return (w, om) if return_omega0 else w


def backproject(tau, traces, fs, t0=0.0, mode=1, weights=None):
    """Eq. 7 image, double [nframes][npix]; tau fp32 [nsens][npix], traces fp32 [B][S][Nt].
    weights: optional fp32 [nsens][npix] multiplying every term (modes 0-2 only)."""
    tau = np.asarray(tau)
    if weights is not None:
        assert mode in (0, 1, 2)
        tau = np.ascontiguousarray(tau)
        weights = np.ascontiguousarray(weights, dtype=np.float32)
        assert weights.shape == tau.shape
    assert tau.dtype == np.float32 and tau.ndim == 2 and tau.strides[1] == 4
    traces = np.ascontiguousarray(traces, dtype=np.float32)
    if traces.ndim == 2:
        traces = traces[None]
    B, S, Nt = traces.shape
    assert tau.shape[0] == S
    P = tau.shape[1]
    pitch = tau.strides[0] // 4 if S > 1 else P
    img = np.zeros((B, P), dtype=np.float64)
    wp, wd = WEIGHTS[mode]
    if weights is not None:
        rc = lib().oracle_backproject_weighted(_p(tau), _p(weights), pitch, _p(traces), S, P, Nt, B,
                                               float(np.float32(fs)), float(np.float32(t0)), wp, wd, _p(img))
        if rc:
            raise ValueError("oracle_backproject_weighted failed with code %d" % rc)
        return img
    fn = lib().oracle_backproject_exact if mode in EXACT_TIME_MODES else lib().oracle_backproject
    rc = fn(_p(tau), pitch, _p(traces), S, P, Nt, B,
                                  float(np.float32(fs)), float(np.float32(t0)), wp, wd, _p(img))
    if rc:
        raise ValueError("oracle_backproject failed with code %d" % rc)
    return img

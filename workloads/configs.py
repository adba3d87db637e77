"""Geometry and trace synthesis for the five workloads of BASELINE.json `configs`.

No arithmetic of the method lives here (see workloads/__init__.py).  Every
choice the config text leaves open is listed in DESIGN.md "Input recipe".
RNG: numpy.random.default_rng(BASE_SEED + 1000*k + f) for config k, frame f;
geometry perturbations use f = 900.
"""
from dataclasses import dataclass, field

import numpy as np
from scipy import ndimage

BASE_SEED = 150103869
CONFIG_NAMES = ["tiny2d", "paper2d", "stream2d", "large2d", "vol3d"]


def frame_seed(k: int, f: int) -> int:
    return BASE_SEED + 1000 * int(k) + int(f)


@dataclass
class Geometry:
    k: int
    name: str
    ndim: int
    n: tuple            # nodes per axis of the FMM / c-map grid, (nx, ny[, nz]); x fastest
    h: float            # isotropic spacing [m]
    origin: tuple       # coordinates of node (0,0[,0]) [m]
    c_map: np.ndarray   # fp32, shape n[::-1]
    sensors: np.ndarray  # fp32 (S, 3) [m]
    roi_index: np.ndarray  # int64 ascending linear node indices (x fastest)
    nt: int
    fs: float
    t0: float
    batch: int
    r_abs: float        # absorbers live within this radius of the centre [m]
    meta: dict = field(default_factory=dict)

    @property
    def nsens(self):
        return int(self.sensors.shape[0])

    @property
    def npix(self):
        return int(self.roi_index.size)

    def n3(self):
        return tuple(self.n) + (1,) * (3 - self.ndim)

    def origin3(self):
        return tuple(self.origin) + (0.0,) * (3 - self.ndim)

    def node_coords(self):
        """Coordinate arrays of all nodes, each of shape n[::-1]."""
        axes = [self.origin[d] + np.arange(self.n[d]) * self.h for d in range(self.ndim)]
        grids = np.meshgrid(*axes[::-1], indexing="ij")      # slowest axis first
        return tuple(grids[::-1])                             # (x, y[, z])

    def roi_coords(self):
        """(P, ndim) coordinates of the ROI nodes."""
        idx = self.roi_index
        out = np.empty((idx.size, self.ndim))
        rem = idx.copy()
        for d in range(self.ndim):
            out[:, d] = self.origin[d] + (rem % self.n[d]) * self.h
            rem //= self.n[d]
        return out


def _smooth_unit_noise(rng, shape, sigma_px):
    g = ndimage.gaussian_filter(rng.standard_normal(shape), sigma=sigma_px, mode="nearest")
    return g / np.max(np.abs(g))


def _ring(S, r):
    th = 2.0 * np.pi * np.arange(S) / S
    return np.stack([r * np.cos(th), r * np.sin(th), np.zeros(S)], axis=1).astype(np.float32)


def _hemisphere(S, R):
    i = np.arange(S)
    z = (i + 0.5) / S
    phi = i * np.pi * (3.0 - np.sqrt(5.0))
    rxy = np.sqrt(1.0 - z * z)
    return (R * np.stack([rxy * np.cos(phi), rxy * np.sin(phi), z], axis=1)).astype(np.float32)


def _centered_axis(n, h):
    return -(n - 1) / 2.0 * h


def _geom_tiny():
    n, h = 64, 0.5e-3
    org = _centered_axis(n, h)
    g = Geometry(0, CONFIG_NAMES[0], 2, (n, n), h, (org, org), None, _ring(32, 15e-3), None,
                 512, 20e6, 0.0, 1, 10e-3)
    x, y = g.node_coords()
    r = np.hypot(x, y)
    c = np.full((n, n), 1540.0, dtype=np.float32)
    c[(r >= 11.5e-3) & (r < 12.5e-3)] = 2800.0
    g.c_map = c
    g.roi_index = np.arange(n * n, dtype=np.int64)
    g.meta = dict(absorbers="5 nodes", nabs=5)
    return g


def _geom_paper(k):
    """configs[1] / configs[2]: 192x192 image grid inside a concentric 256x256 FMM grid."""
    nimg, nf, off, h = 192, 256, 32, 0.25e-3
    org = _centered_axis(nf, h)
    batch = 1 if k == 1 else 64
    g = Geometry(k, CONFIG_NAMES[k], 2, (nf, nf), h, (org, org), None, _ring(512, 30e-3), None,
                 2048, 20e6, 0.0, batch, 18e-3)
    rng = np.random.default_rng(frame_seed(1, 900))          # geometry shared by k = 1 and 2
    x, y = g.node_coords()
    r = np.hypot(x, y)
    g1 = _smooth_unit_noise(rng, (nf, nf), 8.0)
    g2 = _smooth_unit_noise(rng, (nf, nf), 3.0)
    c = np.full((nf, nf), 1540.0)
    skull = (r >= 20.75e-3) & (r < 26.75e-3)
    c[skull] = ((2600.0 + 400.0 * g1) * (1.0 + 0.05 * g2))[skull]
    g.c_map = c.astype(np.float32)
    # ROI: the 21323 image-grid nodes nearest the centre, ties by ascending linear index
    ii, jj = np.meshgrid(np.arange(nimg), np.arange(nimg), indexing="xy")   # ii = x index
    d2 = ((2 * ii - (nimg - 1)) ** 2 + (2 * jj - (nimg - 1)) ** 2).ravel()
    lin_img = (jj * nimg + ii).ravel()
    order = np.lexsort((lin_img, d2))[:21323]
    lin_fmm = (jj.ravel()[order] + off) * nf + (ii.ravel()[order] + off)
    g.roi_index = np.sort(lin_fmm).astype(np.int64)
    g.meta = dict(absorbers="segments", nseg=(40, 40) if k == 1 else (20, 60))
    return g


def _geom_large(reduced):
    if reduced:
        n, h, S, nt, fs = 256, 0.2e-3, 256, 2048, 20e6
    else:
        n, h, S, nt, fs = 512, 0.1e-3, 1024, 4096, 40e6
    org = _centered_axis(n, h)
    g = Geometry(3, CONFIG_NAMES[3] + ("_reduced" if reduced else ""), 2, (n, n), h, (org, org),
                 None, _ring(S, 25e-3), None, nt, fs, 0.0, 16, 18e-3)
    rng = np.random.default_rng(frame_seed(3, 900))
    x, y = g.node_coords()
    r = np.hypot(x, y)
    g2 = _smooth_unit_noise(rng, (n, n), 3.0)
    c = np.full((n, n), 1540.0)
    for lo, hi, v in ((20e-3, 21e-3, 3000.0), (21e-3, 22e-3, 2200.0), (22e-3, 23e-3, 3000.0)):
        m = (r >= lo) & (r < hi)
        c[m] = (v * (1.0 + 0.05 * g2))[m]
    g.c_map = c.astype(np.float32)
    g.roi_index = np.flatnonzero((r < 20e-3).ravel()).astype(np.int64)
    g.meta = dict(absorbers="segments", nseg=(20, 60))
    return g


def _geom_vol(reduced):
    if reduced:
        nimg, h, S = 64, 0.5e-3, 512
    else:
        nimg, h, S = 128, 0.25e-3, 4096
    sens = _hemisphere(S, 20e-3)
    img_lo = _centered_axis(nimg, h)
    pads_lo, pads_hi = [], []
    for d in range(3):
        smin, smax = float(sens[:, d].min()), float(sens[:, d].max())
        lo_need = min(img_lo, smin - 4 * h)
        hi_need = max(-img_lo, smax + 4 * h)
        pads_lo.append(int(np.ceil((img_lo - lo_need) / h - 1e-9)))
        pads_hi.append(int(np.ceil((hi_need + img_lo) / h - 1e-9)))
    n = tuple(nimg + pads_lo[d] + pads_hi[d] for d in range(3))
    origin = tuple(img_lo - pads_lo[d] * h for d in range(3))
    g = Geometry(4, CONFIG_NAMES[4] + ("_reduced" if reduced else ""), 3, n, h, origin, None, sens,
                 None, 2048, 20e6, 0.0, 1, 12e-3)
    rng = np.random.default_rng(frame_seed(4, 900))
    x, y, z = g.node_coords()
    r = np.sqrt(x * x + y * y + z * z)
    shape = n[::-1]
    g1 = _smooth_unit_noise(rng, shape, 8.0 if not reduced else 4.0)
    g2 = _smooth_unit_noise(rng, shape, 3.0 if not reduced else 1.5)
    c = np.full(shape, 1540.0)
    shell = (r >= 14e-3) & (r < 19e-3)
    c[shell] = ((2600.0 + 400.0 * g1) * (1.0 + 0.05 * g2))[shell]
    g.c_map = c.astype(np.float32)
    ix = np.arange(nimg)
    lin = ((ix[:, None, None] + pads_lo[2]) * n[1] + (ix[None, :, None] + pads_lo[1])) * n[0] \
        + (ix[None, None, :] + pads_lo[0])
    g.roi_index = np.sort(lin.ravel()).astype(np.int64)
    g.meta = dict(absorbers="blobs", nblob=100, pads_lo=pads_lo, nimg=nimg)
    return g


def make_geometry(k: int, reduced: bool = False) -> Geometry:
    """Geometry of BASELINE.json configs[k]; `reduced` gives the small variants of k = 3, 4."""
    if k == 0:
        g = _geom_tiny()
    elif k in (1, 2):
        g = _geom_paper(k)
    elif k == 3:
        g = _geom_large(reduced)
    elif k == 4:
        g = _geom_vol(reduced)
    else:
        raise ValueError("config index must be 0..4")
    # the C-ABI carries h and origin as fp32: hand every consumer the same (rounded) numbers
    g.h = float(np.float32(g.h))
    g.origin = tuple(float(np.float32(v)) for v in g.origin)
    return g


def _roi_lookup(geom):
    N = int(np.prod(geom.n))
    look = np.full(N, -1, dtype=np.int64)
    look[geom.roi_index] = np.arange(geom.npix)
    return look


def make_absorbers(geom: Geometry, frame: int = 0):
    """Seeded absorbers of one frame: (positions in the ROI list, amplitudes)."""
    rng = np.random.default_rng(frame_seed(geom.k, frame))
    look = geom.meta.get("_look")
    if look is None:
        look = geom.meta["_look"] = _roi_lookup(geom)
    kind = geom.meta["absorbers"]
    h = geom.h
    if kind == "5 nodes":
        xy = geom.roi_coords()
        cand = np.flatnonzero(np.hypot(xy[:, 0], xy[:, 1]) < geom.r_abs)
        pos = rng.choice(cand, size=geom.meta["nabs"], replace=False)
        return np.sort(pos).astype(np.int64), rng.uniform(0.5, 1.0, size=pos.size)[np.argsort(pos)]
    acc = {}
    if kind == "segments":
        lo, hi = geom.meta["nseg"]
        nseg = lo if lo == hi else int(rng.integers(lo, hi + 1))
        for _ in range(nseg):
            rr = geom.r_abs * np.sqrt(rng.uniform())
            th = rng.uniform(0, 2 * np.pi)
            p0 = np.array([rr * np.cos(th), rr * np.sin(th)])
            length = rng.uniform(2e-3, 10e-3)
            phi = rng.uniform(0, 2 * np.pi)
            amp = rng.uniform(0.5, 1.0)
            t = np.arange(0.0, length, 0.5 * h)
            pts = p0[None, :] + t[:, None] * np.array([np.cos(phi), np.sin(phi)])[None, :]
            ij = np.rint((pts - np.array(geom.origin)[None, :]) / h).astype(np.int64)
            ok = np.all((ij >= 0) & (ij < np.array(geom.n)[None, :]), axis=1)
            lin = ij[ok, 1] * geom.n[0] + ij[ok, 0]
            pos = np.unique(look[lin])
            for q in pos[pos >= 0]:
                acc[int(q)] = acc.get(int(q), 0.0) + amp
    elif kind == "blobs":
        sig = h                                              # sigma = 1 voxel
        for _ in range(geom.meta["nblob"]):
            v = rng.standard_normal(3)
            ctr = v / np.linalg.norm(v) * geom.r_abs * rng.uniform() ** (1.0 / 3.0)
            amp = rng.uniform(0.5, 1.0)
            ic = np.rint((ctr - np.array(geom.origin)) / h).astype(np.int64)
            for dz in range(-2, 3):
                for dy in range(-2, 3):
                    for dx in range(-2, 3):
                        ijk = ic + np.array([dx, dy, dz])
                        xyz = np.array(geom.origin) + ijk * h
                        d2 = float(np.sum((xyz - ctr) ** 2))
                        if d2 > (2 * sig) ** 2:
                            continue
                        lin = (ijk[2] * geom.n[1] + ijk[1]) * geom.n[0] + ijk[0]
                        q = int(look[lin])
                        if q >= 0:
                            acc[q] = acc.get(q, 0.0) + amp * np.exp(-d2 / (2 * sig * sig))
    else:
        raise ValueError(kind)
    pos = np.array(sorted(acc), dtype=np.int64)
    return pos, np.array([acc[int(q)] for q in pos])


def make_traces(geom: Geometry, tau, frames=None, noise_sigma: float = 0.01,
                pulse: str = "gaussian", pulse_sigma: float = 2.0, absorbers=None):
    """fp32 traces [B][S][Nt]: each absorber emits a pulse centred at u = tau*fs (fractional).

    `tau` is either the fp32 table [S][P] or a callable pos -> fp32 [S][len(pos)]
    (for tables that do not fit in host memory).  pulse = "gaussian" (the configs'
    recipe) or "bipolar" (-(n-u)/sigma * gaussian, a photoacoustic-like N-shape).
    `absorbers`, if given, is a list of (pos, amp) per frame instead of the seeded ones.
    """
    if frames is None:
        frames = range(geom.batch)
    frames = list(frames)
    S, Nt = geom.nsens, geom.nt
    out = np.empty((len(frames), S, Nt), dtype=np.float32)
    R = int(np.ceil(5 * pulse_sigma))
    srow = (np.arange(S, dtype=np.int64) * Nt)[:, None]
    for bi, f in enumerate(frames):
        pos, amp = absorbers[bi] if absorbers is not None else make_absorbers(geom, f)
        cols = tau(pos) if callable(tau) else np.asarray(tau)[:, pos]
        u = (cols.astype(np.float64) - geom.t0) * geom.fs       # [S][A]
        k0 = np.floor(u).astype(np.int64)
        sig = np.zeros(S * Nt)
        for d in range(-R, R + 2):
            nidx = k0 + d
            ok = (nidx >= 0) & (nidx < Nt) & np.isfinite(u)
            x = (nidx - u) / pulse_sigma
            w = np.exp(-0.5 * x * x) * amp[None, :]
            if pulse == "bipolar":
                w = -x * w
            elif pulse != "gaussian":
                raise ValueError(pulse)
            flat = (srow + nidx)[ok]
            sig += np.bincount(flat, weights=w[ok], minlength=S * Nt)
        rng = np.random.default_rng(frame_seed(geom.k, f) + 500)
        if noise_sigma > 0:
            sig += rng.normal(0.0, noise_sigma, size=S * Nt)
        out[bi] = sig.reshape(S, Nt).astype(np.float32)
    return out

"""Pins P1-P5 for oracle_fmm: closed forms and invariants that
fix the eikonal solver of PAPER.md:49-58 without any other implementation."""
import numpy as np
import pytest

import oracle

H = 0.5e-3
N = 64
ORG = (-(N - 1) / 2 * H,) * 2


def coords(n=N, h=H):
    ax = (np.arange(n) - (n - 1) / 2) * h
    return np.meshgrid(ax, ax, indexing="xy")          # x[j][i] = ax[i]


@pytest.mark.parametrize("src", [(0.1e-3, 0.2e-3), (-7.3e-3, 4.9e-3), (15e-3, 0.0)])
def test_p1_homogeneous_matches_distance_over_c(src):
    """north_star check 1: |x-s|/c within the first-order FMM error (never early)."""
    c = np.full((N, N), 1540.0, np.float32)
    T = oracle.fmm((N, N), H, ORG, c, src)
    x, y = coords()
    d = np.hypot(x - src[0], y - src[1]) / 1540.0
    e = (T - d) / (H / 1540.0)
    assert e.min() >= -1e-9
    assert e.max() <= 1.5


def test_p1_first_order_convergence():
    """Relative error shrinks under grid refinement (first order)."""
    errs = []
    for n in (32, 64, 128):
        h = 32e-3 / n
        org = (-(n - 1) / 2 * h,) * 2
        c = np.full((n, n), 1540.0, np.float32)
        src = (1.3e-3, -0.7e-3)
        T = oracle.fmm((n, n), h, org, c, src)
        x, y = coords(n, h)
        d = np.hypot(x - src[0], y - src[1]) / 1540.0
        errs.append(np.max(np.abs(T - d)))
    assert errs[1] < 0.75 * errs[0] and errs[2] < 0.75 * errs[1]


def test_p1_3d_homogeneous():
    n, h = 24, 1e-3
    org = (-(n - 1) / 2 * h,) * 3
    c = np.full((n, n, n), 1500.0, np.float32)
    src = (0.2e-3, -0.3e-3, 0.4e-3)
    T = oracle.fmm((n, n, n), h, org, c, src)
    ax = (np.arange(n) - (n - 1) / 2) * h
    z, y, x = np.meshgrid(ax, ax, ax, indexing="ij")
    d = np.sqrt((x - src[0]) ** 2 + (y - src[1]) ** 2 + (z - src[2]) ** 2) / 1500.0
    e = (T - d) / (h / 1500.0)
    assert e.min() >= -1e-9 and e.max() <= 2.0


def test_p2_layered_medium_normal_incidence_closed_form():
    """On-node source, c = c(x) only: along the source row T(k) = h * sum slowness."""
    rng = np.random.default_rng(7)
    cx = np.full(N, 1540.0)
    cx[40:] = rng.uniform(1500.0, 3000.0, size=N - 40)     # layers start beyond the source cell
    c = np.tile(cx[None, :], (N, 1)).astype(np.float32)
    i0, j0 = 32, 20
    src = (ORG[0] + i0 * H, ORG[1] + j0 * H)
    T = oracle.fmm((N, N), H, ORG, c, src)
    expect = np.concatenate([[0.0], np.cumsum(H / c[j0, i0 + 1:].astype(np.float64))])
    np.testing.assert_allclose(T[j0, i0:], expect, rtol=1e-14, atol=0)


def _skull_map():
    x, y = coords()
    r = np.hypot(x, y)
    c = np.full((N, N), 1540.0, np.float32)
    c[(r >= 11.5e-3) & (r < 12.5e-3)] = 2800.0
    return c


def test_p3_discrete_upwind_residual_is_zero():
    """Every non-source node satisfies sum_d max((T-a_d)/h,0)^2 = 1/c^2."""
    c = _skull_map()
    src = (14.9e-3, 0.37e-3)
    T = oracle.fmm((N, N), H, ORG, c, src)
    Tp = np.pad(T, 1, constant_values=np.inf)
    ax = np.minimum(Tp[1:-1, :-2], Tp[1:-1, 2:])
    ay = np.minimum(Tp[:-2, 1:-1], Tp[2:, 1:-1])
    res = (np.maximum((T - ax) / H, 0) ** 2 + np.maximum((T - ay) / H, 0) ** 2) * c.astype(np.float64) ** 2
    g = [(src[d] - ORG[d]) / H for d in range(2)]
    mask = np.ones_like(T, bool)
    mask[int(np.floor(g[1])):int(np.floor(g[1])) + 2, int(np.floor(g[0])):int(np.floor(g[0])) + 2] = False
    np.testing.assert_allclose(res[mask], 1.0, rtol=1e-10)


def _sweep_solve(c, src, h, org, iters=40):
    """Independent algorithm, same discrete system: Gauss-Seidel fast sweeping."""
    n = c.shape[0]
    T = np.full((n, n), np.inf)
    g = [(src[d] - org[d]) / h for d in range(2)]
    i0, j0 = int(np.floor(g[0])), int(np.floor(g[1]))
    cn = float(c[int(np.floor(g[1] + 0.5)), int(np.floor(g[0] + 0.5))])
    fixed = set()
    for dj in (0, 1):
        for di in (0, 1):
            xx, yy = org[0] + (i0 + di) * h, org[1] + (j0 + dj) * h
            T[j0 + dj, i0 + di] = np.hypot(xx - src[0], yy - src[1]) / cn
            fixed.add((j0 + dj, i0 + di))
    s = 1.0 / c.astype(np.float64)
    for _ in range(iters):
        change = 0.0
        for jr, ir in ((range(n), range(n)), (range(n), range(n - 1, -1, -1)),
                       (range(n - 1, -1, -1), range(n)), (range(n - 1, -1, -1), range(n - 1, -1, -1))):
            for j in jr:
                for i in ir:
                    a = min(T[j, i - 1] if i > 0 else np.inf, T[j, i + 1] if i < n - 1 else np.inf)
                    b = min(T[j - 1, i] if j > 0 else np.inf, T[j + 1, i] if j < n - 1 else np.inf)
                    lo, hi = min(a, b), max(a, b)
                    if not np.isfinite(lo):
                        continue
                    sh = s[j, i] * h
                    t = lo + sh
                    if t > hi:
                        t = 0.5 * (lo + hi + np.sqrt(2 * sh * sh - (lo - hi) ** 2))
                    if (j, i) in fixed:
                        # init nodes may only be lowered, exactly like trial nodes in the FMM
                        pass
                    if t < T[j, i]:
                        change = max(change, T[j, i] - t if np.isfinite(T[j, i]) else 1.0)
                        T[j, i] = t
        if change == 0.0:
            break
    return T


def test_p4_equals_fast_sweeping():
    n, h = 32, 1e-3
    org = (-(n - 1) / 2 * h,) * 2
    ax = (np.arange(n) - (n - 1) / 2) * h
    x, y = np.meshgrid(ax, ax, indexing="xy")
    r = np.hypot(x, y)
    c = np.full((n, n), 1540.0, np.float32)
    c[(r >= 9e-3) & (r < 11e-3)] = 2800.0
    src = (14.2e-3, 1.3e-3)
    T = oracle.fmm((n, n), h, org, c, src)
    Ts = _sweep_solve(c, src, h, org)
    np.testing.assert_allclose(T, Ts, rtol=1e-12)


def test_p5_frozen_order_monotone_and_symmetry_and_reciprocity():
    c = _skull_map()
    src = (14.9e-3, 0.0)                      # on the mirror axis y = 0 (between node rows)
    T, order = oracle.fmm((N, N), H, ORG, c, src, return_order=True)
    assert np.all(order >= 0) and np.unique(order).size == N * N
    assert np.all(np.diff(T.ravel()[order]) >= 0)
    np.testing.assert_allclose(T, T[::-1, :], rtol=1e-12)
    # reciprocity ("the ray path is reversible"): T_s(x) ~ T_x(s) within 2 h / c_min
    a = (ORG[0] + 50 * H, ORG[1] + 30 * H)
    b = (ORG[0] + 9 * H, ORG[1] + 41 * H)
    Ta = oracle.fmm((N, N), H, ORG, c, a)
    Tb = oracle.fmm((N, N), H, ORG, c, b)
    assert abs(Ta[41, 9] - Tb[30, 50]) <= 2 * H / 1540.0


def test_skull_speeds_arrivals_up():
    """A fast annulus can only make first arrivals earlier than the homogeneous ones."""
    src = (14.9e-3, 0.37e-3)
    Th = oracle.fmm((N, N), H, ORG, np.full((N, N), 1540.0, np.float32), src)
    Ts = oracle.fmm((N, N), H, ORG, _skull_map(), src)
    assert np.all(Ts <= Th + 1e-15) and np.any(Ts < Th - 1e-7)


def test_second_order_is_more_accurate_away_from_source():
    """Eq. 6 stencil: smaller error than first order in a homogeneous medium."""
    c = np.full((N, N), 1540.0, np.float32)
    src = (0.1e-3, 0.2e-3)
    x, y = coords()
    d = np.hypot(x - src[0], y - src[1]) / 1540.0
    e1 = np.abs(oracle.fmm((N, N), H, ORG, c, src, order=1) - d)
    e2 = np.abs(oracle.fmm((N, N), H, ORG, c, src, order=2) - d)
    far = d > 8 * H / 1540.0
    assert e2[far].max() < 0.5 * e1[far].max()


def test_rows_match_single_solves_and_bad_source():
    c = _skull_map()
    sens = np.array([[15e-3, 0, 0], [0, 15e-3, 0], [-10.6e-3, -10.6e-3, 0]])
    roi = np.array([5, 100, 2000, 4095], dtype=np.int64)
    tau = oracle.fmm_rows((N, N), H, ORG, c, sens, roi)
    for i in range(3):
        T = oracle.fmm((N, N), H, ORG, c, sens[i, :2])
        np.testing.assert_array_equal(tau[i], T.ravel()[roi].astype(np.float32))
    with pytest.raises(ValueError):
        oracle.fmm((N, N), H, ORG, c, (17e-3, 0.0))

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


# ---- 3-D pins for local_solve's three-axis branch (m = 3) ------------------------------------------------
def _medium_3d(n, h, seed=3):
    """Heterogeneous 3-D medium: a fast shell plus a smooth seeded perturbation (values 1400 .. 3100 m/s)."""
    ax = (np.arange(n) - (n - 1) / 2) * h
    z, y, x = np.meshgrid(ax, ax, ax, indexing="ij")
    r = np.sqrt(x * x + y * y + z * z)
    c = np.full((n, n, n), 1540.0)
    c[(r >= 0.30 * n * h) & (r < 0.40 * n * h)] = 2800.0
    rng = np.random.default_rng(seed)
    c *= 1.0 + 0.08 * np.sin(2 * np.pi * (x / (n * h) * rng.uniform(1, 2) + y / (n * h) * rng.uniform(1, 2) + z / (n * h) * rng.uniform(1, 2)))
    return c.astype(np.float32)


def test_p3_3d_discrete_upwind_residual_is_zero():
    """P3 in 3-D, heterogeneous: sum_d max((T - a_d)/h, 0)^2 = 1/c^2 at every node outside the source cell.  A
    three-axis solve that silently falls back to the two-axis root, a wrong discriminant or a wrong acceptance
    test leaves a residual != 1 at the nodes reached by all three axes (most of the volume)."""
    n, h = 24, 1e-3
    org = (-(n - 1) / 2 * h,) * 3
    c = _medium_3d(n, h)
    src = (2.3e-3, -1.7e-3, 0.9e-3)
    T = oracle.fmm((n, n, n), h, org, c, src)
    Tp = np.pad(T, 1, constant_values=np.inf)
    a = [np.minimum(Tp[1:-1, 1:-1, :-2], Tp[1:-1, 1:-1, 2:]),       # x (fastest axis = last numpy axis)
         np.minimum(Tp[1:-1, :-2, 1:-1], Tp[1:-1, 2:, 1:-1]),       # y
         np.minimum(Tp[:-2, 1:-1, 1:-1], Tp[2:, 1:-1, 1:-1])]       # z
    res = sum(np.maximum((T - ad) / h, 0.0) ** 2 for ad in a) * c.astype(np.float64) ** 2
    used = sum((T > ad).astype(int) for ad in a)
    g = [int(np.floor((src[d] - org[d]) / h)) for d in range(3)]
    mask = np.ones_like(T, bool)
    mask[g[2]:g[2] + 2, g[1]:g[1] + 2, g[0]:g[0] + 2] = False
    np.testing.assert_allclose(res[mask], 1.0, rtol=1e-10)
    assert np.count_nonzero(used[mask] == 3) > 0.5 * mask.sum(), "the three-axis branch must carry most nodes"


def _sweep_solve_3d(c, src, h, org, iters=60):
    """Independent algorithm, same discrete system, 3-D: Gauss-Seidel fast sweeping with the textbook three-axis
    update (try one axis, then two, then three; Zhao 2005), written without reference to oracle/."""
    n = c.shape[0]
    T = np.full((n, n, n), np.inf)
    g = [(src[d] - org[d]) / h for d in range(3)]
    i0 = [int(np.floor(v)) for v in g]
    near = [min(int(np.floor(v + 0.5)), n - 1) for v in g]
    cn = float(c[near[2], near[1], near[0]])
    for dk in (0, 1):
        for dj in (0, 1):
            for di in (0, 1):
                p = [org[0] + (i0[0] + di) * h, org[1] + (i0[1] + dj) * h, org[2] + (i0[2] + dk) * h]
                T[i0[2] + dk, i0[1] + dj, i0[0] + di] = np.sqrt(sum((p[d] - src[d]) ** 2 for d in range(3))) / cn
    sh = h / c.astype(np.float64)
    fwd, bwd = list(range(n)), list(range(n - 1, -1, -1))
    for _ in range(iters):
        changed = False
        for kr in (fwd, bwd):
            for jr in (fwd, bwd):
                for ir in (fwd, bwd):
                    for k in kr:
                        for j in jr:
                            for i in ir:
                                v = sorted((min(T[k, j, i - 1] if i > 0 else np.inf, T[k, j, i + 1] if i < n - 1 else np.inf),
                                            min(T[k, j - 1, i] if j > 0 else np.inf, T[k, j + 1, i] if j < n - 1 else np.inf),
                                            min(T[k - 1, j, i] if k > 0 else np.inf, T[k + 1, j, i] if k < n - 1 else np.inf)))
                                if not np.isfinite(v[0]):
                                    continue
                                f = sh[k, j, i]
                                t = v[0] + f
                                if t > v[1]:
                                    t = 0.5 * (v[0] + v[1] + np.sqrt(2 * f * f - (v[0] - v[1]) ** 2))
                                    if t > v[2]:
                                        s1, s2 = v[0] + v[1] + v[2], v[0] ** 2 + v[1] ** 2 + v[2] ** 2
                                        t = (s1 + np.sqrt(s1 * s1 - 3.0 * (s2 - f * f))) / 3.0
                                if t < T[k, j, i]:
                                    T[k, j, i] = t
                                    changed = True
        if not changed:
            break
    return T


def test_p4_3d_equals_fast_sweeping():
    """P4 in 3-D: the heap-ordered march and Gauss-Seidel sweeping reach the same solution of the upwind system."""
    n, h = 12, 2e-3
    org = (-(n - 1) / 2 * h,) * 3
    c = _medium_3d(n, h, seed=11)
    src = (3.1e-3, -2.2e-3, 4.4e-3)
    T = oracle.fmm((n, n, n), h, org, c, src)
    Ts = _sweep_solve_3d(c, src, h, org)
    np.testing.assert_allclose(T, Ts, rtol=1e-12)


# ---- pins for the second-order branch (order = 2, the paper's Eq. 6) -----------------------
def _axis_setup(n, h, fn_c):
    """On-node source at the left end of the middle row of an n x n grid whose speed depends on x only."""
    org = (0.0, -(n // 2) * h)
    xs = np.arange(n) * h
    c = np.tile(fn_c(xs)[None, :], (n, 1)).astype(np.float32)
    return org, xs, c, (0.0, 0.0), n // 2


def test_second_order_stencil_recurrence_along_an_axis():
    """Along the source row of an x-layered medium the front is axis-aligned, only the x axis is upwind, and Eq. 6
    becomes the recurrence 3 T_k - 4 T_{k-1} + T_{k-2} = 2 h / c_k for k >= 2 (first step: T_1 = h / c_1) --
    exactly, whatever the layers are.  Wrong coefficients (3, -4, 1) or a forgotten factor 2h fail here."""
    n, h = 48, 0.4e-3
    rng = np.random.default_rng(12)
    layers = rng.uniform(1500.0, 3000.0, size=n)
    org, xs, c, src, j0 = _axis_setup(n, h, lambda x: layers)
    T = oracle.fmm((n, n), h, org, c, src, order=2)[j0]
    s = 1.0 / c[j0].astype(np.float64)
    assert T[0] == 0.0
    np.testing.assert_allclose(T[1], h * s[1], rtol=1e-14)
    lhs = 3.0 * T[2:] - 4.0 * T[1:-1] + T[:-2]
    np.testing.assert_allclose(lhs, 2.0 * h * s[2:], rtol=1e-11)


def test_second_order_convergence_rate_along_an_axis():
    """O(h^2): with a smooth c(x) the error of T along the source row against the exact integral of the slowness
    falls by ~4 per grid refinement for order = 2 (>= 3.5 asked), and by ~2 for order = 1."""
    L, c0 = 19.2e-3, 1540.0
    slow = lambda x: (1.0 + 0.3 * np.sin(2 * np.pi * x / L)) / c0
    exact = lambda x: (x - 0.3 * L / (2 * np.pi) * (np.cos(2 * np.pi * x / L) - 1.0)) / c0
    err = {1: [], 2: []}
    for n in (49, 97, 193):
        h = L / (n - 1)
        # the oracle takes the speed as fp32 (as the product does): compare against the integral of ITS slowness
        # would hide nothing -- the fp32 rounding of c moves T by 1e-8 relative, far below the errors measured here
        org, xs, c, src, j0 = _axis_setup(n, h, lambda x: 1.0 / slow(x))
        for order in (1, 2):
            T = oracle.fmm((n, n), h, org, c, src, order=order)[j0]
            far = xs > 0.25 * L
            err[order].append(np.max(np.abs(T[far] - exact(xs[far]))))
    assert err[2][0] / err[2][1] >= 3.5 and err[2][1] / err[2][2] >= 3.5, err
    assert 1.6 <= err[1][0] / err[1][1] <= 2.4 and 1.6 <= err[1][1] / err[1][2] <= 2.4, err
    assert err[2][2] < 0.2 * err[1][2]


def test_second_order_residual_and_fallback_2d():
    """An order-2 solution against the MIXED discrete equation, the stencil choice re-derived here from the final
    field and the freeze order alone: per axis the upwind difference is Eq. 6 where the two upwind nodes are
    usable (frozen earlier, T_{-2} <= T_{-1}), else first order.  Most nodes satisfy it exactly.  The scheme is
    not monotone, so a node may keep a value from before its last upwind neighbour froze -- a SMALLER one, since a
    new value is only taken when it lowers T: the residual is then below 1, never above.  Where the second-order
    root is not causal the node satisfies the first-order equation.  Using T_{-2} where it exceeds T_{-1}, or
    dropping the causality fallback, pushes residuals above 1."""
    c = _skull_map()
    src = (14.9e-3, 0.37e-3)
    T, order = oracle.fmm((N, N), H, ORG, c, src, order=2, return_order=True)
    rank = np.empty(N * N, np.int64)
    rank[order] = np.arange(N * N)
    rank = rank.reshape(N, N)
    s2 = 1.0 / c.astype(np.float64) ** 2
    g = [(src[d] - ORG[d]) / H for d in range(2)]
    i0, j0 = int(np.floor(g[0])), int(np.floor(g[1]))
    n2 = nfall = nkept = 0
    for j in range(N):
        for i in range(N):
            if i0 <= i <= i0 + 1 and j0 <= j <= j0 + 1:
                continue
            d1, d2, use2 = [], [], []
            for (dj, di) in ((0, 1), (1, 0)):
                best = None
                for sg in (-1, 1):
                    jj, ii = j + sg * dj, i + sg * di
                    if 0 <= jj < N and 0 <= ii < N and rank[jj, ii] < rank[j, i]:       # frozen before this node
                        if best is None or T[jj, ii] < T[best[0], best[1]]:
                            best = (jj, ii, sg)
                if best is None:
                    continue
                jj, ii, sg = best
                a = T[jj, ii]
                d1.append((T[j, i] - a) / H)
                j2, i2 = j + 2 * sg * dj, i + 2 * sg * di
                ok2 = 0 <= j2 < N and 0 <= i2 < N and rank[j2, i2] < rank[j, i] and T[j2, i2] <= a
                use2.append(ok2)
                d2.append((3.0 * T[j, i] - 4.0 * a + T[j2, i2]) / (2.0 * H) if ok2 else (T[j, i] - a) / H)
            # the axes that take part are those whose neighbour value lies below T (upwind)
            r2 = sum(max(v, 0.0) ** 2 for v in d2) / s2[j, i]
            r1 = sum(max(v, 0.0) ** 2 for v in d1) / s2[j, i]
            if abs(r2 - 1.0) <= 1e-9:
                n2 += any(use2)
            elif abs(r1 - 1.0) <= 1e-9:
                nfall += 1                                        # first-order fallback (non-causal Eq. 6 root)
            else:
                assert r2 < 1.0, "node (%d, %d): mixed-order residual %.3e above 1 (first-order: %.3e)" % (j, i, r2 - 1, r1 - 1)
                nkept += 1
    assert n2 > 0.8 * N * N, "Eq. 6 must be the stencil at most nodes (%d of %d)" % (n2, N * N)
    assert nfall + nkept < 0.1 * N * N, (nfall, nkept)


def test_second_order_needs_an_ordered_upwind_pair_next_to_the_source():
    """Eq. 6 uses T(x-1) and T(x-2) only if T(x-2) <= T(x-1) (the pair is upwind in order, R11).  Source on a
    node row, 0.8 h right of node 10: the source cell's corners get T(11) = 0.2 h/c and T(10) = 0.8 h/c, so for node 12
    of that row the pair (11, 10) is NOT ordered and the update must be first order: T(12) = T(11) + h/c exactly.
    (With Eq. 6 on the unordered pair it would come out as (2 + 4*0.2 - 0.8)/3 = 0.667 h/c.)  One node further the pair
    (12, 11) is ordered and Eq. 6 applies: 3 T(13) - 4 T(12) + T(11) = 2 h/c."""
    n, h, c0 = 32, 0.5e-3, 1500.0
    org = (0.0, 0.0)
    j = 16
    src = (10.8 * h, j * h)
    T = oracle.fmm((n, n), h, org, np.full((n, n), c0, np.float32), src, order=2)[j]
    u = h / c0
    np.testing.assert_allclose(T[11], 0.2 * u, rtol=1e-12)
    np.testing.assert_allclose(T[10], 0.8 * u, rtol=1e-12)
    np.testing.assert_allclose(T[12], T[11] + u, rtol=1e-12)
    np.testing.assert_allclose(3.0 * T[13] - 4.0 * T[12] + T[11], 2.0 * u, rtol=1e-11)
    # on the left of the cell the pair (10, 11) IS ordered for node 9 (T(11) <= T(10)): Eq. 6
    np.testing.assert_allclose(3.0 * T[9] - 4.0 * T[10] + T[11], 2.0 * u, rtol=1e-11)

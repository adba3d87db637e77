"""CPU-side checks of the product library: it loads, exports every symbol include/pat.h declares,
validates arguments before touching CUDA, and its host-only FMM matches the oracle FMM.
No compute call needs a GPU here."""
import ctypes
import os
import re

import numpy as np
import pytest

import oracle
import workloads as W
import paper_1501_03869_b200 as pat

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    txt = open(os.path.join(ROOT, "include", "pat.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(pat_[a-z_]+)\s*\(", txt)))


def test_library_exports_every_declared_symbol():
    L = pat.lib()
    names = _declared_symbols()
    assert {"pat_plan_create", "pat_set_travel_times", "pat_backproject", "pat_destroy"} <= set(names)
    for n in names:
        assert hasattr(L, n), "libpat_b200.so does not export %s" % n


def test_binding_has_the_same_names():
    for n in _declared_symbols():
        assert callable(getattr(pat, n)), n


def test_library_contains_sm100a_code_only():
    out = os.popen("cuobjdump -lelf %s 2>/dev/null" % pat.library_path()).read()
    if out:
        assert "sm_100a" in out
        assert not re.search(r"sm_(?!100a)\d+", out)


def _grid():
    return pat.PatGrid.make((64, 64), 0.5e-3, (-15.75e-3, -15.75e-3))


def test_workspace_bytes_and_invalid_sizes():
    g = _grid()
    n = pat.pat_plan_workspace_bytes(g, 32, 4096, 512, 1)
    assert n >= 4 * 32 * 4096 + 8 * 32 * 512 and n % 256 == 0
    assert pat.pat_plan_workspace_bytes(g, 32, 4096, 512, 4) > n
    for bad in [(0, 4096, 512, 1), (32, 0, 512, 1), (32, 4097, 512, 1), (32, 4096, 1, 1), (32, 4096, 512, 0)]:
        assert pat.pat_plan_workspace_bytes(g, *bad) == 0
    g3 = pat.PatGrid.make((64, 64), -1.0, (0, 0))
    assert pat.pat_plan_workspace_bytes(g3, 32, 4096, 512, 1) == 0


def _create(**kw):
    g = kw.pop("grid", _grid())
    a = dict(c_map=np.full(4096, 1540, np.float32), sensor_xyz=np.zeros((4, 3), np.float32), nsens=4,
             roi_index=np.arange(100, dtype=np.int64), npix=100, nt=64, fs=20e6, t0=0.0, weighting=1,
             max_batch=1, workspace=256, workspace_bytes=1 << 30)
    a.update(kw)
    return pat.pat_plan_create(g, a["c_map"], a["sensor_xyz"], a["nsens"], a["roi_index"], a["npix"], a["nt"],
                               a["fs"], a["t0"], a["weighting"], a["max_batch"], a["workspace"],
                               a["workspace_bytes"])


@pytest.mark.parametrize("kw", [
    dict(nsens=0), dict(nt=1), dict(fs=0.0), dict(fs=float("nan")), dict(weighting=5), dict(max_batch=0),
    dict(roi_index=np.array([5, 5, 6], np.int64), npix=3), dict(roi_index=np.array([1, 4096], np.int64), npix=2),
    dict(roi_index=None, npix=100), dict(c_map=np.zeros(4096, np.float32)),
    dict(c_map=np.full(4096, np.inf, np.float32)), dict(workspace=None), dict(workspace=260),
    dict(sensor_xyz=np.full((4, 3), np.nan, np.float32)),
])
def test_plan_create_rejects_bad_arguments_before_any_cuda_call(kw):
    with pytest.raises(pat.PatError) as ei:
        _create(**kw)
    assert ei.value.status == pat.PAT_ERR_INVALID_ARG
    assert pat.pat_last_error(None)


def test_plan_create_without_gpu_fails_loudly_not_silently():
    """Valid arguments but no usable sm_100 device / bogus workspace: an error, never a CPU path."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("covered by the gpu tests")
    with pytest.raises(pat.PatError) as ei:
        _create()
    assert ei.value.status in (pat.PAT_ERR_CUDA, pat.PAT_ERR_UNSUPPORTED)


def test_null_plan_calls_are_safe():
    L = pat.lib()
    assert L.pat_destroy(None) == pat.PAT_OK
    assert L.pat_backproject(None, None, None, 1, None) == pat.PAT_ERR_INVALID_ARG
    assert L.pat_set_travel_times(None, None, 0, 1, None) == pat.PAT_ERR_INVALID_ARG
    assert pat.pat_kernel_launches(None) == 0
    assert L.pat_backproject_conventional(None, None, None, 1, 1500.0, None) == pat.PAT_ERR_INVALID_ARG
    assert L.pat_set_pixel_weights(None, None, 0, 0, None) == pat.PAT_ERR_INVALID_ARG
    assert L.pat_compute_solid_angle_weights(None, None, None) == pat.PAT_ERR_INVALID_ARG
    assert L.pat_get_trace_window(None, None, None) == pat.PAT_ERR_INVALID_ARG
    assert L.pat_set_roi_mask(None, None) == pat.PAT_ERR_INVALID_ARG


def test_missing_library_raises_importerror(monkeypatch, tmp_path):
    from paper_1501_03869_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "_HERE", str(tmp_path))
    with pytest.raises(ImportError):
        binding.lib()


# ---- production FMM (host only) against the oracle FMM ---------------------------------------
@pytest.mark.parametrize("k,reduced,nsub,order", [(0, False, 32, 1), (0, False, 32, 2), (1, False, 6, 1),
                                                  (3, True, 4, 1), (4, True, 2, 1), (4, True, 2, 2)])
def test_production_fmm_matches_oracle_fmm(k, reduced, nsub, order):
    geom = W.make_geometry(k, reduced)
    S = geom.nsens
    pick = np.unique(np.linspace(0, S - 1, nsub).astype(int))
    grid = pat.PatGrid.make(geom.n, geom.h, geom.origin)
    cm = np.ascontiguousarray(geom.c_map).ravel()
    for i in pick:
        row = np.empty((1, geom.npix), np.float32)
        pat.pat_fmm_travel_times(grid, cm, geom.sensors, S, geom.roi_index, geom.npix, int(i), 1, order, row, 1)
        T = oracle.fmm(geom.n, geom.h, geom.origin, geom.c_map, geom.sensors[i, :geom.ndim].astype(np.float64),
                       order=order)
        ref = T.ravel()[geom.roi_index]
        assert np.max(np.abs(row[0].astype(np.float64) - ref)) <= 1e-9 * ref.max() + 6e-8 * ref.max()
        assert np.mean(row[0] != ref.astype(np.float32)) < 1e-3


def test_production_fmm_rejects_sensor_outside_grid_and_chunks_agree():
    geom = W.make_geometry(0)
    grid = pat.PatGrid.make(geom.n, geom.h, geom.origin)
    cm = geom.c_map.ravel()
    sens = geom.sensors.copy()
    full = np.empty((geom.nsens, geom.npix), np.float32)
    pat.pat_fmm_travel_times(grid, cm, sens, geom.nsens, geom.roi_index, geom.npix, 0, geom.nsens, 1, full, 0)
    part = np.empty((5, geom.npix), np.float32)
    pat.pat_fmm_travel_times(grid, cm, sens, geom.nsens, geom.roi_index, geom.npix, 7, 5, 1, part, 2)
    np.testing.assert_array_equal(part, full[7:12])
    sens[3, 0] = 1.0
    with pytest.raises(pat.PatError) as ei:
        pat.pat_fmm_travel_times(grid, cm, sens, geom.nsens, geom.roi_index, geom.npix, 0, geom.nsens, 1, full, 0)
    assert ei.value.status == pat.PAT_ERR_INVALID_ARG
    # ROI restriction (early stop) returns the same values as the full-grid solve
    roi = np.arange(0, 4096, 7, dtype=np.int64)
    sub = np.empty((2, roi.size), np.float32)
    pat.pat_fmm_travel_times(grid, cm, geom.sensors, geom.nsens, roi, roi.size, 0, 2, 1, sub, 1)
    np.testing.assert_array_equal(sub, full[0:2][:, roi])


def test_workload_roi_counts_match_the_paper():
    """21323 pixels at the coarse resolution; 512 ring sensors."""
    want = dict(l.split() for l in open(os.path.join(ROOT, "tests", "golden", "paper_counts.txt"))
                if l.strip() and not l.startswith("#"))
    g = W.make_geometry(1)
    assert g.npix == int(want["npix_coarse"]) and g.nsens == int(want["nsens"])
    assert np.all(np.diff(g.roi_index) > 0)


def test_device_allocator_abi_without_a_gpu():
    """pat_set_device_allocator: both callbacks or none (argument check only; nothing is allocated here)."""
    import ctypes
    L = pat.lib()
    cb = ctypes.CFUNCTYPE(ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p)(lambda n, u: None)
    assert L.pat_set_device_allocator(ctypes.cast(cb, ctypes.c_void_p), None, None) == pat.PAT_ERR_INVALID_ARG
    assert L.pat_set_device_allocator(None, None, None) == pat.PAT_OK
    assert L.pat_get_stats(None, None) == pat.PAT_ERR_INVALID_ARG


def _extents(perm, roi, n, group):
    """Largest bounding-box edge (nodes) of every `group` consecutive slots of the order."""
    pos = perm[perm >= 0]
    q = roi[pos]
    co = [q % n[0], (q // n[0]) % n[1]] + ([q // (n[0] * n[1])] if len(n) == 3 else [])
    out = []
    for a in range(0, len(pos), group):
        out.append(max(int(c[a:a + group].max() - c[a:a + group].min()) for c in co))
    return np.array(out)


def test_pixel_order_is_a_compact_permutation_2d_disk_and_3d_offset_cube():
    """Host logic of the table layout (pat_pixel_order = what pat_plan_create uses): a bijection with the padding at
    the end, and spatially compact tiles (256 slots) and warps (32 slots) for regions that cut the blocks of a plain
    Morton order -- the paper's region within the skull (configs[1]: a disk of 21323 nodes) and a cube at an odd
    offset inside a larger grid (configs[4] reduced) -- where plain Morton order is NOT compact."""
    for k, reduced, tile_max, warp_max in [(1, False, 30, 13), (4, True, 9, 4)]:
        geom = W.make_geometry(k, reduced)
        grid = pat.PatGrid.make(geom.n, geom.h, geom.origin)
        roi = np.ascontiguousarray(geom.roi_index, dtype=np.int64)
        P = geom.npix
        perm = pat.pat_pixel_order(grid, roi, P)
        assert perm.shape == (((P + 255) // 256) * 256,)
        assert np.array_equal(np.sort(perm[:P]), np.arange(P)) and (perm[P:] == -1).all()
        tiles, warps = _extents(perm, roi, geom.n, 256), _extents(perm, roi, geom.n, 32)
        assert tiles.max() <= tile_max and warps.max() <= warp_max, (k, tiles.max(), warps.max())
        plain = pat.pat_pixel_order(grid, roi, P, plain_morton=True)
        assert np.array_equal(np.sort(plain[:P]), np.arange(P))
        assert _extents(plain, roi, geom.n, 32).max() > 2 * warp_max        # what the bisection order is for
    g = pat.PatGrid.make((8, 8), 1e-3, (0, 0))
    with pytest.raises(pat.PatError):
        pat.pat_pixel_order(g, np.array([0, 64], dtype=np.int64), 2)       # index outside the grid
    assert np.array_equal(np.sort(pat.pat_pixel_order(g, None, 64)[:64]), np.arange(64))

"""GPU parity: the CUDA path (through the C-ABI) against the CPU oracle, element by element,
on the same seeded inputs and the SAME fp32 tau table (reading R17)."""
import numpy as np
import pytest

import oracle
import workloads as W
from _cases import case, assert_parity, gpu_backproject, errors

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("mode", [0, 1, 2])
def test_config0_tiny_all_weightings(mode):
    geom, tau = case(0)
    tr = W.make_traces(geom, tau)
    ref = oracle.backproject(tau, tr, geom.fs, geom.t0, mode)
    got = gpu_backproject(geom, tau, tr, mode=mode)
    assert_parity(got, ref, "config0 mode %d" % mode)


def test_config0_tau_from_oracle_fmm():
    """configs[0]: traces centred at the ORACLE-FMM tau; both sides consume that table."""
    geom = W.make_geometry(0)
    tau = oracle.fmm_rows(geom.n, geom.h, geom.origin, geom.c_map, geom.sensors.astype(np.float64),
                          geom.roi_index)
    tr = W.make_traces(geom, tau)
    assert_parity(gpu_backproject(geom, tau, tr), oracle.backproject(tau, tr, geom.fs), "config0/oracle tau")


def test_config1_paper_scale():
    geom, tau = case(1)
    tr = W.make_traces(geom, tau)
    ref = oracle.backproject(tau, tr, geom.fs, geom.t0, 1)
    got = gpu_backproject(geom, tau, tr)
    rel, mx = assert_parity(got, ref, "config1")
    print("config1 rel-L2 %.2e max-abs/max %.2e" % (rel, mx))


def test_config1_host_buffers_equal_device_buffers():
    geom, tau = case(1)
    tr = W.make_traces(geom, tau)
    ref = oracle.backproject(tau, tr, geom.fs, geom.t0, 1)
    assert_parity(gpu_backproject(geom, tau, tr, host=True), ref, "config1 host path")


def test_config2_stream_batch64():
    geom, tau = case(2)
    tr = W.make_traces(geom, tau)
    assert tr.shape[0] == 64
    ref = oracle.backproject(tau, tr, geom.fs, geom.t0, 1)
    got = gpu_backproject(geom, tau, tr)
    assert_parity(got, ref, "config2")
    worst = max(errors(got[f], ref[f])[0] for f in range(64))
    assert worst <= 1e-5


def test_config2_batch_equals_single_frames():
    geom, tau = case(2)
    tr = W.make_traces(geom, tau, frames=range(5))
    got = gpu_backproject(geom, tau, tr, max_batch=8)
    for f in (0, 4):
        one = gpu_backproject(geom, tau, tr[f:f + 1])
        assert_parity(got[f], one[0].astype(np.float64), "batch vs single frame %d" % f)


def test_config3_large_reduced():
    geom, tau = case(3, True)
    tr = W.make_traces(geom, tau)
    ref = oracle.backproject(tau, tr, geom.fs, geom.t0, 1)
    assert_parity(gpu_backproject(geom, tau, tr), ref, "config3 reduced")


def test_config4_volume_reduced():
    geom, tau = case(4, True)
    tr = W.make_traces(geom, tau)
    ref = oracle.backproject(tau, tr, geom.fs, geom.t0, 1)
    assert_parity(gpu_backproject(geom, tau, tr), ref, "config4 reduced")


@pytest.mark.slow
def test_config3_large_full():
    geom, tau = case(3)
    tr = W.make_traces(geom, tau)
    ref = oracle.backproject(tau, tr, geom.fs, geom.t0, 1)
    assert_parity(gpu_backproject(geom, tau, tr), ref, "config3")


@pytest.mark.slow
def test_config4_shape_full_cube_analytic_tau_sampled_outputs():
    """configs[4]'s image cube at full size (128^3 = 2 097 152 voxels, 8192 tiles) with an analytic
    tau = dist/c0 table (conventional BP) for 192 hemisphere sensors -- the FMM table
    of the full config needs hours of host CPU.  Outputs are checked on a seeded sample of voxels
    the oracle computes one by one, plus the first and last tile."""
    geom = W.make_geometry(4)
    S = 192
    sens = geom.sensors[:: geom.nsens // S][:S].astype(np.float64)
    xyz = geom.roi_coords()
    tau = np.empty((S, geom.npix), dtype=np.float32)
    for i in range(S):
        tau[i] = (np.sqrt(((xyz - sens[i][None, :]) ** 2).sum(axis=1)) / 1540.0).astype(np.float32)
    rng = np.random.default_rng(44)
    tr = rng.standard_normal((2, S, geom.nt)).astype(np.float32)
    g2 = W.make_geometry(4)
    g2.sensors = sens.astype(np.float32)
    got = gpu_backproject(g2, tau, tr)
    pick = np.unique(np.concatenate([np.arange(256), np.arange(geom.npix - 256, geom.npix),
                                     rng.integers(0, geom.npix, size=4000)]))
    ref = oracle.backproject(np.ascontiguousarray(tau[:, pick]), tr, geom.fs, geom.t0, 1)
    assert_parity(got[:, pick], ref, "config4-shaped cube, sampled voxels")
    assert np.all(np.isfinite(got))


@pytest.mark.parametrize("B", [12, 16])
def test_config2_geometry_bp16_split_halves_path(B):
    """The 9-16 frame class at the paper-scale geometry (the bench sweep's B = 16 row): interleaved [sample][16]
    traces, a pixel's 8 lanes load one 128-byte run {b[k], b[k+1]} and the two halves meet at flush time."""
    geom, tau = case(2)
    tr = W.make_traces(geom, tau, frames=range(B))
    ref = oracle.backproject(tau, tr, geom.fs, geom.t0, 1)
    got = gpu_backproject(geom, tau, tr)
    assert_parity(got, ref, "config2 geometry, %d frames" % B)
    worst = max(errors(got[f], ref[f])[0] for f in range(B))
    assert worst <= 1e-5

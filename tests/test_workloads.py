"""The seeded input generator: deterministic, shaped as BASELINE.json's configs state."""
import numpy as np

import workloads as wl


def test_config1_shapes_and_determinism():
    a, b = wl.config(1), wl.config(1)
    assert a.y.shape == (1, 64, 256) and a.y.dtype == np.complex64
    assert a.grid_shape == (32, 32, 32) and a.n_elem == 64 and a.n_tx == 1
    assert a.xs.dtype == np.float32 and a.elem_pos.dtype == np.float32
    np.testing.assert_array_equal(a.y, b.y)
    np.testing.assert_array_equal(a.scat_pos, b.scat_pos)
    assert abs(float(a.xs[0]) + 2.4e-3) < 1e-9 and abs(float(a.zs[-1]) - 9e-3) < 1e-9


def test_config2_plane_wave_set():
    w = wl.config(2, generate_data=False)
    assert w.n_tx == 5 and w.n_elem == 256 and w.n_samples == 512
    np.testing.assert_allclose(np.linalg.norm(w.tx_v.astype(np.float64), axis=1), 1.0, atol=1e-7)
    # tau_tx = (r.u)/c minus its minimum over the element centres: min over elements is 0
    proj = w.elem_pos.astype(np.float64) @ w.tx_v.astype(np.float64).T / w.c + w.tx_t0.astype(np.float64)
    np.testing.assert_allclose(proj.min(axis=0), 0.0, atol=1e-12)


def test_config3_geometry_only():
    w = wl.config(3, generate_data=False)
    assert w.n_tx == 16 and w.n_elem == 1024 and w.n_samples == 1024 and w.grid_shape == (128,) * 3
    assert set(np.unique(w.tx_type)) == {wl.TX_DIVERGING}
    np.testing.assert_allclose(w.tx_v[:, 2], -10e-3, rtol=1e-6)
    np.testing.assert_allclose(w.tx_t0, -np.linalg.norm(w.tx_v.astype(np.float64), axis=1) / w.c, rtol=1e-6)
    assert w.tx_v[1, 0] == np.float32(-3e-3) and w.tx_v[1, 1] == np.float32(-1e-3)   # q = 4*ix_v + iy_v
    assert len(w.scat_amp) == 50 and w.scat_amp.min() >= 0.01 and w.scat_amp.max() <= 1.0


def test_config4_rf_and_config5_streaming():
    w4 = wl.config(4, generate_data=False)
    assert w4.data_kind == wl.DATA_RF and w4.n_samples == 2048 and w4.fs == 31.2e6 and w4.fc == 0.0
    np.testing.assert_array_equal(w4.scat_pos, wl.config(3, generate_data=False).scat_pos)
    frames = list(wl.streaming_frames(2, grid=(4, 4, 4)))
    assert len(frames) == 2 and frames[0].y.shape == (16, 1024, 1024)
    assert len(frames[0].scat_amp) == 100
    d = frames[1].scat_pos - frames[0].scat_pos
    assert np.all(d[50:] == 0) and 1e-6 < np.abs(d[:50]).mean() < 2e-5
    assert not np.array_equal(frames[0].y, frames[1].y)


def test_echo_lands_at_its_delay():
    """One scatterer, one element: |y| peaks at round(tau fs) with amplitude ~A."""
    w = wl.custom([[0, 0, 0]], [wl.TX_PLANE], [[0, 0, 1]], [0.0], [0.0], [0.0], [5e-3], fs=15.6e6,
                  n_samples=256, scat_pos=[[0, 0, 5e-3]], scat_amp=[0.7])
    k = int(np.argmax(np.abs(w.y[0, 0])))
    assert k == round(2 * 5e-3 / 1540.0 * 15.6e6)
    assert 0.68 < abs(w.y[0, 0, k]) <= 0.7

"""The seeded generators reproduce BASELINE.json's shapes and statistics (CPU only)."""
import numpy as np

from workloads import make_config, make_custom, gaussian_taps


def _unpack(b):  # local, for statistics only
    hi = (b >> 4).astype(np.int16); lo = (b & 15).astype(np.int16)
    return np.where(hi > 7, hi - 16, hi), np.where(lo > 7, lo - 16, lo)


def test_c1_layout_and_voltages():
    wl = make_config(1)
    assert (wl.N, wl.n_ant, wl.n_pol, wl.n_chan, wl.n_t, wl.input_kind) == (32, 16, 1, 1, 8, "cf32")
    cells = {(int(x), int(y)) for x, y in wl.ant_uv}
    assert len(cells) == 16 and all(0 <= x < 16 and 0 <= y < 16 for x, y in cells)
    assert np.array_equal(wl.ant_uv, np.round(wl.ant_uv))
    v = wl.voltages()
    assert v.shape == (8, 1, 1, 16, 2) and v.dtype == np.float32
    assert np.array_equal(v, make_config(1).voltages())  # deterministic


def test_c2_disc_layout_and_ci4_statistics():
    wl = make_config(2, n_chan=4, n_t=60)
    assert (wl.N, wl.grid_n, wl.n_ant, wl.n_pol, wl.kernel_k, wl.n_products) == (128, 64, 256, 2, 1, 2)
    r = np.hypot(wl.ant_uv[:, 0] - 32, wl.ant_uv[:, 1] - 32)
    assert r.max() <= 50.0 / 3.94464 + 1e-3 and r.max() > 11.0
    v = wl.voltages()
    assert v.shape == (60, 4, 2, 256) and v.dtype == np.uint8
    re, im = _unpack(v)
    assert re.min() == -8 and re.max() == 7
    assert abs(re.mean()) < 0.02 and abs(re.std() - 2.0) < 0.08 and abs(im.std() - 2.0) < 0.08
    # extents do not change the layout; full-size config has the same antennas
    assert np.array_equal(wl.ant_uv, make_config(2, n_chan=1, n_t=1).ant_uv)
    full = make_config(2)
    assert (full.n_chan, full.n_t) == (128, 1000)


def test_c3_same_layout_taps_and_source():
    c2, c3 = make_config(2, 1, 1), make_config(3, 1, 1)
    assert np.array_equal(c2.ant_uv, c3.ant_uv)
    assert c3.taps.shape == (256, 3, 3, 2) and c3.taps.dtype == np.float32
    mag = np.hypot(c3.taps[..., 0], c3.taps[..., 1]).sum(axis=(1, 2))
    np.testing.assert_allclose(mag, 1.0, rtol=1e-5)
    assert len(c3.sources) == 1 and c3.n_products == 4 and c3.n_planes == 6
    assert make_config(3).n_t == 2500 and make_config(3).n_chan == 128


def test_c4_c5_shapes():
    c4 = make_config(4, 1, 1)
    assert (c4.N, c4.n_ant, c4.kernel_k) == (256, 1024, 3)
    assert c4.ant_uv.min() >= 1.0 and c4.ant_uv.max() <= 127.0
    c5 = make_config(5, 1, 1)
    assert (c5.N, c5.n_ant, c5.kernel_k, len(c5.sources)) == (512, 4096, 5, 3)
    sub = make_config(5, 1, 1, n_ant=256)
    assert np.array_equal(sub.ant_uv, c5.ant_uv[:256]) and np.array_equal(sub.taps, c5.taps[:256])


def test_gaussian_taps_peak_on_nearest_cell_and_phase():
    uv = np.array([[3.2, 4.0], [5.5, 6.49]], np.float32)
    t = gaussian_taps(uv, 3, 0.5, np.array([0.0, np.pi / 2]))
    m0 = np.hypot(t[0, ..., 0], t[0, ..., 1])
    assert np.unravel_index(m0.argmax(), (3, 3)) == (1, 1) and m0[1, 2] > m0[1, 0]
    assert abs(t[1, 1, 1, 0]) < 1e-6 and t[1, 1, 1, 1] > 0  # phase pi/2 -> purely imaginary


def test_custom_wrap_layout_has_out_of_range_positions():
    wl = make_custom(grid_n=8, pad=2, n_ant=30, n_pol=1, kernel_k=3, n_chan=1, n_t=2, layout="wrap")
    assert wl.ant_uv.min() < 0 and wl.ant_uv.max() > 16
    assert wl.voltages().shape == (2, 1, 1, 30)


def test_tophat_taps_cover_fractions_and_per_channel_scaling():
    from workloads import make_per_channel, tophat_taps
    t = tophat_taps(np.array([[3.0, 4.0]], np.float32), 3, 1.5)[0, ..., 0]
    np.testing.assert_allclose(t, np.outer([1 / 6, 2 / 3, 1 / 6], [1 / 6, 2 / 3, 1 / 6]), rtol=1e-6)
    t = tophat_taps(np.array([[3.25, 4.0]], np.float32), 3, 1.0)[0, ..., 0]      # shifted a quarter cell in x
    np.testing.assert_allclose(t, np.outer([0, 1, 0], [0, 0.75, 0.25]), atol=1e-7)
    wl = make_per_channel(grid_n=32, pad=2, n_ant=12, n_pol=2, kernel_k=3, n_chan=4, n_t=2,
                          f0_hz=40e6, df_hz=10e6, diameter_m=60.0)
    assert wl.ant_uv.shape == (4, 12, 2) and wl.taps.shape == (4, 12, 3, 3, 2)
    off = wl.ant_uv.astype(np.float64) - 16.0
    np.testing.assert_allclose(off[3], off[0] * 70.0 / 40.0, rtol=1e-5, atol=1e-5)   # cells ~ 1/lambda
    np.testing.assert_allclose(np.abs(wl.taps[..., 0] + 1j * wl.taps[..., 1]).sum(axis=(-2, -1)), 1.0, rtol=1e-5)
    assert wl.voltages().shape == (2, 4, 2, 12)

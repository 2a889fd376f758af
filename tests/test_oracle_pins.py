"""Pins for the CPU oracle: each check compares oracle/ against something that is not the
oracle — a typed-out table, a hand-worked value, a closed form, a textbook identity, a
library routine, or brute force written differently (BASELINE.json (a)(b)(c)).
CPU only."""
import cmath
import math

import numpy as np
import pytest

from oracle import epic_oracle as orc
from workloads import make_config, make_custom, make_per_channel, pack_ci4

RNG = np.random.default_rng(20190411)


# ------------------------------------------------------------------ S1 unpack
# Two's-complement value of every 4-bit pattern, typed out by hand.
NIBBLE_VALUE = [0, 1, 2, 3, 4, 5, 6, 7, -8, -7, -6, -5, -4, -3, -2, -1]


def test_s1_unpack_all_256_bytes_against_typed_table():
    b = np.arange(256, dtype=np.uint8)
    got = orc.unpack_ci4(b)
    for v in range(256):
        assert got[v] == complex(NIBBLE_VALUE[v >> 4], NIBBLE_VALUE[v & 15]), hex(v)


@pytest.mark.parametrize("byte,expect", [
    (0x00, 0 + 0j), (0x7F, 7 - 1j), (0x80, -8 + 0j), (0xF8, -1 - 8j), (0x19, 1 - 7j), (0x88, -8 - 8j),
])
def test_s1_unpack_literal_bytes(byte, expect):
    assert orc.unpack_ci4(np.array([byte], dtype=np.uint8))[0] == expect
    assert orc.sext4(byte >> 4) == expect.real and orc.sext4(byte & 15) == expect.imag


def test_s1_pack_then_unpack_round_trip():
    re = RNG.integers(-8, 8, 1000)
    im = RNG.integers(-8, 8, 1000)
    got = orc.unpack_ci4(pack_ci4(re, im))
    assert np.array_equal(got.real, re) and np.array_equal(got.imag, im)


# ------------------------------------------------------------------ S2 cells
def test_s2_nearest_cell_hand_worked():
    uv = np.array([[3.0, 4.0], [2.5, 2.49], [-0.5, -0.51], [7.6, 0.0], [1.5, 3.5]], dtype=np.float32)
    got = orc.nearest_cells(uv)
    assert got.tolist() == [[3, 4], [3, 2], [0, -1], [8, 0], [2, 4]]  # x.5 rounds up, never to even


def test_s2_tap_cells_wrap_and_order():
    n = 8
    uv = np.array([[0.0, 0.0], [7.6, 3.0]], dtype=np.float32)  # second: cx = 8 -> wraps to 0
    c = orc.tap_cells(uv, 3, n)
    # antenna 0 at cell (x=0,y=0): taps [dy][dx], dy,dx = -1,0,1 ; y*N+x
    assert c[0].tolist() == [[7 * 8 + 7, 7 * 8 + 0, 7 * 8 + 1], [7, 0, 1], [8 + 7, 8 + 0, 8 + 1]]
    assert c[1].tolist() == [[2 * 8 + 7, 2 * 8 + 0, 2 * 8 + 1], [3 * 8 + 7, 3 * 8, 3 * 8 + 1], [4 * 8 + 7, 4 * 8, 4 * 8 + 1]]
    assert orc.tap_cells(np.array([[5.0, 6.0]], np.float32), 1, n).tolist() == [[[6 * 8 + 5]]]
    with pytest.raises(ValueError):
        orc.tap_cells(uv, 2, n)


def test_s2_brute_force_python_ints():
    n, k = 16, 5
    uv = RNG.uniform(-20, 40, size=(50, 2)).astype(np.float32)
    c = orc.tap_cells(uv, k, n)
    for a in range(50):
        cx = math.floor(float(uv[a, 0]) + 0.5)
        cy = math.floor(float(uv[a, 1]) + 0.5)
        for iy in range(k):
            for ix in range(k):
                assert c[a, iy, ix] == ((cy + iy - 2) % n) * n + ((cx + ix - 2) % n)


# ------------------------------------------------------------------ S3 gridding
def _rand_c(*shape):
    return RNG.standard_normal(shape) + 1j * RNG.standard_normal(shape)


def test_s3_total_is_closed_form_and_linear():
    n, k, a_n, f = 16, 3, 20, 4
    uv = RNG.uniform(0, 8, size=(a_n, 2)).astype(np.float32)
    cells = orc.tap_cells(uv, k, n)
    w = _rand_c(a_n, k, k)
    e1, e2 = _rand_c(f, a_n), _rand_c(f, a_n)
    g1 = orc.grid_frames(e1, cells, w, n)
    # sum over cells = sum_a E_a * sum_taps W_a
    np.testing.assert_allclose(g1.sum(axis=(1, 2)), (e1 * w.sum(axis=(1, 2))[None]).sum(axis=1), rtol=1e-12)
    g2 = orc.grid_frames(e2, cells, w, n)
    g12 = orc.grid_frames(2.5 * e1 - 1j * e2, cells, w, n)
    np.testing.assert_allclose(g12, 2.5 * g1 - 1j * g2, atol=1e-12)


def test_s3_collisions_sum_not_overwrite():
    n = 8
    uv = np.array([[2.2, 3.1], [1.9, 2.8], [5.0, 5.0]], dtype=np.float32)  # first two -> cell (2,3)
    cells = orc.tap_cells(uv, 1, n)
    e = np.array([[1 + 2j, 10 - 1j, 7j]])
    g = orc.grid_frames(e, cells, np.ones((3, 1, 1), complex), n)[0]
    assert g[3, 2] == 11 + 1j and g[5, 5] == 7j
    assert np.count_nonzero(g) == 2


def test_s3_brute_force_dict_and_integer_exactness():
    n, k, a_n = 8, 3, 12
    uv = RNG.uniform(0, 8, size=(a_n, 2)).astype(np.float32)
    taps = RNG.integers(-3, 4, size=(a_n, k, k, 2)).astype(np.float32)
    e = RNG.integers(-8, 8, a_n) + 1j * RNG.integers(-8, 8, a_n)
    g = orc.grid_frames(e[None], orc.tap_cells(uv, k, n), orc.taps_to_complex(taps, a_n, k), n)[0]
    ref = {}
    for a in range(a_n):
        cx, cy = math.floor(float(uv[a, 0]) + .5), math.floor(float(uv[a, 1]) + .5)
        for dy in (-1, 0, 1):
            for dx in (-1, 0, 1):
                key = ((cy + dy) % n, (cx + dx) % n)
                wv = complex(taps[a, dy + 1, dx + 1, 0], taps[a, dy + 1, dx + 1, 1])
                ref[key] = ref.get(key, 0) + wv * e[a]
    for y in range(n):
        for x in range(n):
            assert g[y, x] == ref.get((y, x), 0)  # small integers: exact in any order


def test_s3_delta_taps_default():
    w = orc.taps_to_complex(None, 5, 1)
    assert w.shape == (5, 1, 1) and np.all(w == 1)
    with pytest.raises(ValueError):
        orc.taps_to_complex(None, 5, 3)


# ------------------------------------------------------------------ S4 transform
def _scalar_idft2(g):
    """Pure-python literal of Eq. 5 discretised — pins the vectorised definition."""
    n = len(g)
    out = [[0j] * n for _ in range(n)]
    for m in range(n):
        for l in range(n):
            s = 0j
            for y in range(n):
                for x in range(n):
                    s += g[y][x] * cmath.exp(2j * math.pi * (x * l + y * m) / n)
            out[m][l] = s
    return np.array(out)


def test_s4_definition_matches_scalar_literal():
    g = _rand_c(4, 4)
    np.testing.assert_allclose(orc.idft2_definition(g), _scalar_idft2(g.tolist()), atol=1e-12)


@pytest.mark.parametrize("n", [8, 16, 32])
def test_s4_fast_equals_definition(n):
    g = _rand_c(2, n, n)
    np.testing.assert_allclose(orc.idft2_fast(g), orc.idft2_definition(g), atol=1e-10)


def test_s4_impulse_gives_plane_wave_with_plus_sign():
    n = 16
    for (y0, x0) in [(0, 1), (3, 0), (5, 11)]:
        g = np.zeros((n, n), complex)
        g[y0, x0] = 1.0
        m, l = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
        expect = np.exp(2j * np.pi * (x0 * l + y0 * m) / n)
        for f in (orc.idft2_fast, orc.idft2_definition):
            np.testing.assert_allclose(f(g), expect, atol=1e-12)
    # the sign itself: impulse at x=1 -> Im A[0][1] = +sin(2 pi / N) > 0 (inverse transform, Q8)
    g = np.zeros((n, n), complex)
    g[0, 1] = 1.0
    assert orc.idft2_fast(g)[0, 1].imag == pytest.approx(math.sin(2 * math.pi / n))
    assert orc.idft2_fast(g)[0, 0] == pytest.approx(1.0)  # unnormalised (Q9)


def test_s4_zero_padding_invariant():
    gsz, p = 8, 4
    n = gsz * p
    small = _rand_c(gsz, gsz)
    big = np.zeros((n, n), complex)
    big[:gsz, :gsz] = small
    np.testing.assert_allclose(orc.idft2_fast(big)[::p, ::p], orc.idft2_definition(small), atol=1e-10)


# ------------------------------------------------------------------ S5/S6 products, accumulation
def test_s5_single_antenna_flat_image_and_time_sum():
    wl = make_custom(grid_n=8, pad=2, n_ant=1, n_pol=1, kernel_k=1, n_chan=2, n_t=5,
                     input_kind="cf32", ant_uv=[[3, 5]])
    v = wl.voltages()
    img = orc.epic_image(v, "cf32", wl.ant_uv, None, 8, 2, 1)
    e = v[..., 0].astype(np.float64) ** 2 + v[..., 1].astype(np.float64) ** 2  # [T][C][1][1]
    for c in range(2):
        np.testing.assert_allclose(img[c, 0], np.full((16, 16), e[:, c, 0, 0].sum()), rtol=1e-12)


def test_s5_two_antenna_closed_form():
    n = 16
    uv = np.array([[2, 3], [7, 1]], np.float32)
    e = _rand_c(3, 1, 1, 2)  # [T][C][Np][A]
    v = np.stack([e.real, e.imag], axis=-1).astype(np.float32)
    e = v[..., 0].astype(np.float64) + 1j * v[..., 1]
    img = orc.epic_image(v, "cf32", uv, None, 8, 2, 1)[0, 0]
    m, l = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    dx, dy = 2 - 7, 3 - 1
    expect = np.zeros((n, n))
    for t in range(3):
        e1, e2 = e[t, 0, 0, 0], e[t, 0, 0, 1]
        expect += abs(e1) ** 2 + abs(e2) ** 2 + 2 * (e1 * np.conj(e2) * np.exp(2j * np.pi * (dx * l + dy * m) / n)).real
    np.testing.assert_allclose(img, expect, atol=1e-10)


def test_s5_products_layout_conjugation_parseval():
    wl = make_custom(grid_n=8, pad=2, n_ant=10, n_pol=2, kernel_k=3, n_chan=1, n_t=4, seed=3)
    v = wl.voltages()
    n = 16
    img = orc.epic_image(v, "ci4", wl.ant_uv, wl.taps, 8, 2, 4, kernel_k=3)[0]
    assert img.shape == (6, n, n)
    assert np.all(img[0] >= 0) and np.all(img[1] >= 0)
    np.testing.assert_allclose(img[4], img[2], atol=1e-9)       # Re YX = Re XY
    np.testing.assert_allclose(img[5], -img[3], atol=1e-9)      # Im YX = -Im XY
    # generalised Parseval: sum_pix XY = N^2 sum_cells G_X conj(G_Y)
    e = orc.unpack_ci4(v)[:, 0]  # [T][Np][A]
    cells = orc.tap_cells(wl.ant_uv, 3, n)
    w = orc.taps_to_complex(wl.taps, 10, 3)
    gx = orc.grid_frames(e[:, 0], cells, w, n)
    gy = orc.grid_frames(e[:, 1], cells, w, n)
    s = (gx * np.conj(gy)).sum() * n * n
    assert img[2].sum() == pytest.approx(s.real, rel=1e-12)
    assert img[3].sum() == pytest.approx(s.imag, rel=1e-10, abs=1e-6)
    assert img[0].sum() == pytest.approx((abs(gx) ** 2).sum() * n * n, rel=1e-12)
    # two-product mode is the first two planes
    img2 = orc.epic_image(v, "ci4", wl.ant_uv, wl.taps, 8, 2, 2, kernel_k=3)[0]
    np.testing.assert_array_equal(img2, img[:2])


def test_s5_plane_counts():
    assert orc.n_planes(1, 1) == 1 and orc.n_planes(2, 2) == 2 and orc.n_planes(2, 4) == 6
    with pytest.raises(ValueError):
        orc.n_planes(1, 4)


# ------------------------------------------------------------------ whole path: BASELINE.json (a)(b)(c)
def _fx_direct_image(e, xy, n):
    """Brute-force FX imaging (Eq. 1-2): visibilities of ALL antenna pairs,
    autocorrelations included, then a direct Fourier sum per pixel."""
    t_n, a_n = e.shape
    vis = np.zeros((a_n, a_n), complex)
    for t in range(t_n):
        vis += np.outer(e[t], np.conj(e[t]))
    m, l = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    img = np.zeros((n, n), complex)
    for a in range(a_n):
        for b in range(a_n):
            du, dv = xy[a, 0] - xy[b, 0], xy[a, 1] - xy[b, 1]
            img += vis[a, b] * np.exp(2j * np.pi * (du * l + dv * m) / n)
    return img


@pytest.mark.parametrize("mode", ["definition", "fast"])
def test_a_fx_equivalence_on_c1(mode):
    wl = make_config(1)
    v = wl.voltages()
    img = orc.epic_image(v, "cf32", wl.ant_uv, None, 16, 2, 1, mode=mode)[0, 0]
    e = v[:, 0, 0, :, 0].astype(np.float64) + 1j * v[:, 0, 0, :, 1]
    fx = _fx_direct_image(e, wl.ant_uv.astype(int), 32)
    assert np.abs(fx.imag).max() < 1e-9
    np.testing.assert_allclose(img, fx.real, rtol=0, atol=1e-12 * np.abs(fx).max() * 100)


def test_a_fx_equivalence_cross_pol_conjugation():
    """XY = A_X conj(A_Y) is the image of V^{XY}_ab = sum_t E^X_a conj(E^Y_b) (Eq. 2's E1 (x) E2*)."""
    wl = make_custom(grid_n=8, pad=2, n_ant=6, n_pol=2, kernel_k=1, n_chan=1, n_t=3,
                     layout="integer", seed=11)
    v = wl.voltages()
    n = 16
    img = orc.epic_image(v, "ci4", wl.ant_uv, None, 8, 2, 4)[0]
    e = orc.unpack_ci4(v)[:, 0]  # [T][Np][A]
    xy = wl.ant_uv.astype(int)
    m, l = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    ref = np.zeros((n, n), complex)
    for a in range(6):
        for b in range(6):
            vab = (e[:, 0, a] * np.conj(e[:, 1, b])).sum()
            ref += vab * np.exp(2j * np.pi * ((xy[a, 0] - xy[b, 0]) * l + (xy[a, 1] - xy[b, 1]) * m) / n)
    np.testing.assert_allclose(img[2], ref.real, atol=1e-9)
    np.testing.assert_allclose(img[3], ref.imag, atol=1e-9)


def test_b_parseval_on_c1_and_ci4():
    wl = make_config(1)
    v = wl.voltages()
    img = orc.epic_image(v, "cf32", wl.ant_uv, None, 16, 2, 1)[0, 0]
    # delta kernel on distinct cells: sum |G|^2 = sum |E|^2
    e2 = (v.astype(np.float64) ** 2).sum()
    assert img.sum() == pytest.approx(32 * 32 * e2, rel=1e-13)
    wl = make_config(2, n_chan=1, n_t=3)
    v = wl.voltages()
    img = orc.epic_image(v, "ci4", wl.ant_uv, None, 64, 2, 2)
    e = orc.unpack_ci4(v)
    cells = orc.tap_cells(wl.ant_uv, 1, 128)
    for p in range(2):
        g = orc.grid_frames(e[:, 0, p], cells, np.ones((256, 1, 1), complex), 128)
        assert img[0, p].sum() == pytest.approx(128 * 128 * (abs(g) ** 2).sum(), rel=1e-13)


@pytest.mark.parametrize("kl,km", [(3, 0), (0, 5), (-7, 4), (10, -12)])
def test_c_point_source_peaks_at_predicted_pixel(kl, km):
    """Noise-free plane wave from direction cosines (l0, m0) = (2 kl/N, 2 km/N) on lambda/2 cells:
    E_a = s exp(-2 pi i (u_a l0 + v_a m0)/2) peaks at pixel (m, l) = (km mod N, kl mod N), height
    |s|^2 A^2 for the delta kernel (sign from Eq. 5)."""
    wl = make_custom(grid_n=16, pad=2, n_ant=40, n_pol=1, kernel_k=1, n_chan=1, n_t=1,
                     layout="integer", seed=5, input_kind="cf32")
    n, a_n = 32, 40
    l0, m0 = 2.0 * kl / n, 2.0 * km / n
    uv = wl.ant_uv.astype(np.float64)
    s = 0.75 - 0.5j
    e = s * np.exp(-2j * np.pi * (uv[:, 0] * l0 + uv[:, 1] * m0) / 2.0)
    v = np.zeros((1, 1, 1, a_n, 2), np.float32)
    v[0, 0, 0, :, 0], v[0, 0, 0, :, 1] = e.real, e.imag
    img = orc.epic_image(v, "cf32", wl.ant_uv, None, 16, 2, 1)[0, 0]
    pk = np.unravel_index(np.argmax(img), img.shape)
    assert pk == (km % n, kl % n)
    assert img[pk] == pytest.approx(abs(s) ** 2 * a_n ** 2, rel=1e-5)
    assert np.sort(img.ravel())[-2] < 0.9 * img[pk]


def test_definition_and_fast_modes_agree_end_to_end():
    wl = make_custom(grid_n=8, pad=2, n_ant=12, n_pol=2, kernel_k=3, n_chan=2, n_t=3, seed=2)
    v = wl.voltages()
    a = orc.epic_image(v, "ci4", wl.ant_uv, wl.taps, 8, 2, 4, kernel_k=3, mode="definition")
    b = orc.epic_image(v, "ci4", wl.ant_uv, wl.taps, 8, 2, 4, kernel_k=3, mode="fast")
    np.testing.assert_allclose(a, b, atol=1e-9 * np.abs(a).max())


def test_channel_subset_matches_full_run():
    wl = make_config(2, n_chan=3, n_t=4)
    v = wl.voltages()
    full = orc.epic_image(v, "ci4", wl.ant_uv, None, 64, 2, 2)
    sub = orc.epic_image(v, "ci4", wl.ant_uv, None, 64, 2, 2, channels=[2, 0], frames_per_batch=3)
    np.testing.assert_allclose(sub[0], full[2], rtol=1e-13)
    np.testing.assert_allclose(sub[1], full[0], rtol=1e-13)


# ------------------------------------------------------------------ optional autocorrelation removal
def test_autocorr_removal_leaves_only_cross_pairs_brute_force():
    """PAPER.md:130 + Eq. 1-2: with a delta kernel on integer cells the image minus its a = b part
    is the direct-Fourier image of the visibilities of the pairs a != b only."""
    rng = np.random.default_rng(11)
    n, n_ant, t_n = 8, 5, 3
    cells = rng.choice(n * n, size=n_ant, replace=False)
    uv = np.stack([cells % n, cells // n], axis=1).astype(np.float32)
    v = rng.standard_normal((t_n, 1, 2, n_ant, 2)).astype(np.float32)
    img = orc.epic_image(v, "cf32", uv, None, n, 1, 4)
    auto = orc.autocorr_image(v, "cf32", uv, None, n, 1, 4)
    e = v[..., 0].astype(np.float64) + 1j * v[..., 1]
    x, y = uv[:, 0].astype(int), uv[:, 1].astype(int)
    ll, mm = np.meshgrid(np.arange(n), np.arange(n), indexing="xy")
    xx = np.zeros((n, n)); xy = np.zeros((n, n), dtype=complex)
    for a in range(n_ant):
        for b in range(n_ant):
            if a == b:
                continue
            ph = np.exp(2j * np.pi * ((x[a] - x[b]) * ll + (y[a] - y[b]) * mm) / n)
            xx += ((e[:, 0, 0, a] * np.conj(e[:, 0, 0, b])).sum() * ph).real
            xy += (e[:, 0, 0, a] * np.conj(e[:, 0, 1, b])).sum() * ph
    got = img[0] - auto[0]
    assert np.abs(got[0] - xx).max() <= 1e-10 * np.abs(img[0, 0]).max()
    assert np.abs(got[2] - xy.real).max() <= 1e-10 * np.abs(img[0, 0]).max()
    assert np.abs(got[3] - xy.imag).max() <= 1e-10 * np.abs(img[0, 0]).max()
    assert np.allclose(got[4], got[2]) and np.allclose(got[5], -got[3])


@pytest.mark.parametrize("n_pol,n_products", [(2, 4), (1, 1)])
def test_autocorr_removal_multi_antenna_taps_brute_force(n_pol, n_products):
    """Several antennas, each with its OWN random complex 3x3 taps (so every |What_a|^2 differs):
    image minus autocorr_image equals the direct-Fourier image of the pairs a != b only, each pair
    imaged straight from Eq. 1-2 with antenna a's tap-weighted response
        What_a[m][l] = sum_d W_a[d] exp(+2 pi i ((cx_a+dx) l + (cy_a+dy) m) / N)
    typed out here.  Pairing antenna a's power with another antenna's beam fails this."""
    rng = np.random.default_rng(23 + n_pol)
    n, n_ant, t_n, k = 16, 4, 3, 3
    uv = rng.uniform(0, n, (n_ant, 2)).astype(np.float32)          # incl. taps that wrap past the edge
    taps = rng.standard_normal((n_ant, k, k, 2)).astype(np.float32)
    v = rng.standard_normal((t_n, 1, n_pol, n_ant, 2)).astype(np.float32)
    img = orc.epic_image(v, "cf32", uv, taps, n, 1, n_products, kernel_k=k)
    auto = orc.autocorr_image(v, "cf32", uv, taps, n, 1, n_products, kernel_k=k)
    e = v[..., 0].astype(np.float64) + 1j * v[..., 1]                 # [T][1][Np][A]
    w = taps[..., 0].astype(np.float64) + 1j * taps[..., 1]           # [A][dy][dx]
    cx = np.floor(uv[:, 0].astype(np.float64) + 0.5).astype(int)
    cy = np.floor(uv[:, 1].astype(np.float64) + 0.5).astype(int)
    what = np.zeros((n_ant, n, n), dtype=complex)                     # [a][m][l]
    for a in range(n_ant):
        for m in range(n):
            for l in range(n):
                s = 0j
                for iy, dy in enumerate((-1, 0, 1)):
                    for ix, dx in enumerate((-1, 0, 1)):
                        s += w[a, iy, ix] * np.exp(2j * np.pi * (((cx[a] + dx) * l + (cy[a] + dy) * m) % n) / n)
                what[a, m, l] = s
    q = n_pol - 1
    xx = np.zeros((n, n)); yy = np.zeros((n, n)); xy = np.zeros((n, n), dtype=complex)
    for a in range(n_ant):
        for b in range(n_ant):
            if a == b:
                continue
            fringe = what[a] * np.conj(what[b])
            xx += ((e[:, 0, 0, a] * np.conj(e[:, 0, 0, b])).sum() * fringe).real
            yy += ((e[:, 0, q, a] * np.conj(e[:, 0, q, b])).sum() * fringe).real
            xy += (e[:, 0, 0, a] * np.conj(e[:, 0, q, b])).sum() * fringe
    got = img[0] - auto[0]
    peak = np.abs(img[0, 0]).max()
    assert np.abs(got[0] - xx).max() <= 1e-10 * peak
    if n_products == 4:
        assert np.abs(got[1] - yy).max() <= 1e-10 * peak
        assert np.abs(got[2] - xy.real).max() <= 1e-10 * peak
        assert np.abs(got[3] - xy.imag).max() <= 1e-10 * peak
        assert np.abs(got[4] - xy.real).max() <= 1e-10 * peak
        assert np.abs(got[5] + xy.imag).max() <= 1e-10 * peak
    # and the a = b part itself, antenna by antenna: sum_a V_aa |What_a|^2
    diag = sum((np.abs(e[:, 0, 0, a]) ** 2).sum() * np.abs(what[a]) ** 2 for a in range(n_ant))
    assert np.abs(auto[0, 0] - diag).max() <= 1e-10 * peak
    assert np.abs(auto[0, 0] - diag[::-1, ::-1]).max() > 1e-3 * peak     # the beams are not interchangeable


def test_autocorr_image_special_cases():
    """One antenna: the whole image is its autocorrelation.  Delta kernel: the a = b part is flat,
    sum_a sum_t |E_a|^2, whatever the cells."""
    wl = make_custom(grid_n=8, pad=2, n_ant=1, n_pol=2, kernel_k=3, n_chan=2, n_t=5, n_products=4)
    v = wl.voltages()
    img = orc.epic_image(v, "ci4", wl.ant_uv, wl.taps, 8, 2, 4, kernel_k=3)
    auto = orc.autocorr_image(v, "ci4", wl.ant_uv, wl.taps, 8, 2, 4, kernel_k=3)
    assert np.abs(img - auto).max() <= 1e-9 * np.abs(img).max()
    wl = make_custom(grid_n=8, pad=2, n_ant=7, n_pol=1, kernel_k=1, n_chan=1, n_t=4)
    v = wl.voltages()
    auto = orc.autocorr_image(v, "ci4", wl.ant_uv, None, 8, 2, 1)
    flat = (np.abs(orc.unpack_ci4(v)) ** 2).sum()
    assert np.allclose(auto, flat)


# ------------------------------------------------------------------ sampled outputs
@pytest.mark.parametrize("wl", [
    make_config(1),
    make_custom(grid_n=8, pad=2, n_ant=24, n_pol=2, kernel_k=3, n_chan=2, n_t=5, layout="wrap"),
    make_custom(grid_n=16, pad=2, n_ant=9, n_pol=1, kernel_k=5, n_chan=1, n_t=4, input_kind="cf32"),
], ids=lambda w: w.name)
def test_pixel_values_equal_the_imaged_pixels(wl):
    """pixel_values (Eq. 5 written out for one pixel: no grid, no FFT) against epic_image in
    definition mode (the literal double sum over the gridded plane) on every plane."""
    v = wl.voltages()
    img = orc.epic_image(v, wl.input_kind, wl.ant_uv, wl.taps, wl.grid_n, wl.pad, wl.n_products,
                         kernel_k=wl.kernel_k, mode="definition" if wl.N <= 16 else "fast")
    rng = np.random.default_rng(3)
    pix = [(0, 0), (wl.N - 1, 1)] + [tuple(int(x) for x in rng.integers(0, wl.N, 2)) for _ in range(6)]
    got = orc.pixel_values(v, wl.input_kind, wl.ant_uv, wl.taps, wl.grid_n, wl.pad, wl.n_products, pix,
                           kernel_k=wl.kernel_k)
    for i, (m, l) in enumerate(pix):
        assert np.abs(got[:, :, i] - img[:, :, m, l]).max() <= 1e-10 * np.abs(img).max()


# ------------------------------------------------------------------ upstream steps: input order, delay phasors
def test_untransposed_order_axes_hand_case():
    """[T][C][A][Np] order: one sample at antenna 3, polarisation 0 must light up
    XX only, flat, with value |E|^2; the same bytes read as [T][C][Np][A] would be (pol 1, antenna 2)."""
    n_ant = 4
    uv = np.array([[1, 1], [2, 5], [6, 3], [4, 4]], dtype=np.float32)
    v = np.zeros((1, 1, n_ant, 2), dtype=np.uint8)          # TCAP
    v[0, 0, 3, 0] = pack_ci4(3, -4)
    img = orc.epic_image(v, "ci4", uv, None, 8, 1, 2, order="TCAP")
    assert np.allclose(img[0, 0], 25.0) and np.all(img[0, 1] == 0.0)
    wrong = orc.epic_image(v.reshape(1, 1, 2, n_ant), "ci4", uv, None, 8, 1, 2)   # same bytes, other order
    assert np.all(wrong[0, 0] == 0.0) and np.allclose(wrong[0, 1], 25.0)


def test_delay_phasors_closed_forms():
    """Q19: (i) a global phase changes nothing; (ii) a phase psi on pol X only rotates
    XY by exp(i psi) and leaves XX, YY; (iii) |d| = 2 on every antenna of pol Y scales YY by 4."""
    wl = make_custom(grid_n=8, pad=2, n_ant=12, n_pol=2, kernel_k=3, n_chan=2, n_t=4, n_products=4)
    v = wl.voltages()
    args = (v, "ci4", wl.ant_uv, wl.taps, 8, 2, 4)
    base = orc.epic_image(*args, kernel_k=3)
    one = np.ones((2, 2, 12), dtype=np.complex128)
    assert np.allclose(orc.epic_image(*args, kernel_k=3, delay_phasors=one * np.exp(0.7j)), base, rtol=1e-12, atol=1e-9)
    psi = 0.9
    d = one.copy(); d[:, 0, :] = np.exp(1j * psi)
    got = orc.epic_image(*args, kernel_k=3, delay_phasors=d)
    xy0 = base[:, 2] + 1j * base[:, 3]
    assert np.allclose(got[:, :2], base[:, :2]) and np.allclose(got[:, 2] + 1j * got[:, 3], xy0 * np.exp(1j * psi))
    d = one.copy(); d[:, 1, :] = 2.0
    got = orc.epic_image(*args, kernel_k=3, delay_phasors=d)
    assert np.allclose(got[:, 0], base[:, 0]) and np.allclose(got[:, 1], 4.0 * base[:, 1])


def test_delay_compensation_restores_a_point_source():
    """Per-antenna cable phases phi_a scramble a plane wave; the conjugate phasors bring the peak
    back to the predicted pixel with the full coherent height A^2 |s|^2 T (check (c) with delays)."""
    rng = np.random.default_rng(21)
    n, n_ant, t_n = 16, 20, 3
    cells = rng.choice(n * n, size=n_ant, replace=False)
    uv = np.stack([cells % n, cells // n], axis=1).astype(np.float32)
    kl, km = 5, 11
    phi = rng.uniform(0, 2 * np.pi, n_ant)
    e = np.exp(-2j * np.pi * (uv[:, 0] * kl + uv[:, 1] * km) / n) * np.exp(1j * phi)     # [A]
    v = np.zeros((t_n, 1, 1, n_ant, 2), dtype=np.float32)
    v[..., 0], v[..., 1] = e.real, e.imag
    raw = orc.epic_image(v, "cf32", uv, None, n, 1, 1)
    fixed = orc.epic_image(v, "cf32", uv, None, n, 1, 1, delay_phasors=np.exp(-1j * phi)[None, None, :])
    assert np.unravel_index(np.argmax(fixed[0, 0]), (n, n)) == (km, kl)
    assert fixed[0, 0, km, kl] == pytest.approx(t_n * n_ant ** 2, rel=1e-5)   # cf32 inputs
    assert raw[0, 0].max() < 0.5 * fixed[0, 0, km, kl]


# ------------------------------------------------------------------ per-channel layouts (reading Q15)
def _rand_ci4(*shape):
    r = np.random.default_rng(321)
    return pack_ci4(r.integers(-8, 8, shape), r.integers(-8, 8, shape))


def test_per_channel_cells_brute_force_fx_imaging():
    """Each channel imaged by brute-force FX (all antenna pairs, Eq. 1-2) with THAT channel's cells:
    the cell spacing follows the channel's wavelength."""
    n, a_n, c_n, t_n = 16, 5, 3, 4
    pos = np.array([[-3.2, 1.1], [2.6, -2.2], [0.4, 3.3], [-1.7, -3.6], [3.9, 0.2]])  # cells of channel 0
    scale = np.array([1.0, 1.31, 1.77])                      # nu_c / nu_0
    uv = (8.0 + pos[None] * scale[:, None, None]).astype(np.float32)
    v = _rand_ci4(t_n, c_n, 1, a_n)
    img = orc.epic_image(v, "ci4", uv, None, 8, 2, 1)
    e = orc.unpack_ci4(v)
    seen = set()
    for c in range(c_n):
        cells = np.array([[math.floor(float(x) + 0.5) for x in row] for row in uv[c]])   # typed out here
        seen.add(tuple(cells.ravel()))
        fx = _fx_direct_image(e[:, c, 0, :], cells, n)
        np.testing.assert_allclose(img[c, 0], fx.real, atol=1e-9 * np.abs(fx).max())
    assert len(seen) == c_n  # the three channels really use three different sets of cells


def test_per_channel_two_antenna_fringe_follows_the_channel():
    n = 32
    uv = np.array([[[4, 6], [9, 6]], [[4, 6], [14, 6]]], np.float32)  # separation 5 cells, then 10
    v = np.zeros((1, 2, 1, 2, 2), np.float32)
    v[..., 0] = 1.0
    img = orc.epic_image(v, "cf32", uv, None, 16, 2, 1)
    l = np.arange(n)
    for c, d in enumerate([5, 10]):
        np.testing.assert_allclose(img[c, 0], np.broadcast_to(2 + 2 * np.cos(2 * np.pi * d * l / n), (n, n)), atol=1e-10)


def test_per_channel_one_sky_direction_is_one_pixel_in_every_channel():
    """On lambda_c/2 cells a plane wave from direction cosine l0 has phase -pi u_c l0 at an antenna
    whose coordinate is u_c cells, so it lands on pixel l0 N / 2 in every channel."""
    n, kl, km = 32, 5, -3
    base = np.array([[1, 2], [3, -1], [-2, 2], [0, -3], [2, 1], [-3, -2]], np.float64)
    uv = np.stack([8 + base, 8 + 3 * base]).astype(np.float32)       # nu_1 = 3 nu_0: integer cells in both
    e = np.exp(-2j * np.pi * ((uv[..., 0] - 8) * kl + (uv[..., 1] - 8) * km) / n)   # [C][A]
    v = np.zeros((1, 2, 1, 6, 2), np.float32)
    v[0, :, 0, :, 0], v[0, :, 0, :, 1] = e.real, e.imag
    img = orc.epic_image(v, "cf32", uv, None, 16, 2, 1)
    for c in range(2):
        pk = np.unravel_index(np.argmax(img[c, 0]), (n, n))
        assert pk == (km % n, kl % n)
        assert img[c, 0][pk] == pytest.approx(36.0, rel=1e-5)


def test_per_channel_taps_single_antenna_closed_form():
    """One antenna: XX = sum_t |E|^2 |sum_d W_c[d] exp(2 pi i (dx l + dy m)/N)|^2 with the channel's taps."""
    n = 16
    r = np.random.default_rng(5)
    taps = r.standard_normal((2, 1, 3, 3, 2)).astype(np.float32)
    uv = np.array([[[3.2, 4.9]], [[6.6, 2.1]]], np.float32)
    v = _rand_ci4(3, 2, 1, 1)
    img = orc.epic_image(v, "ci4", uv, taps, 8, 2, 1, kernel_k=3)
    p = (np.abs(orc.unpack_ci4(v)) ** 2).sum(axis=0)[:, 0, 0]          # [C]
    m, l = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    for c in range(2):
        w = taps[c, 0, ..., 0].astype(np.float64) + 1j * taps[c, 0, ..., 1]
        beam = sum(w[dy + 1, dx + 1] * np.exp(2j * np.pi * (dx * l + dy * m) / n) for dy in (-1, 0, 1) for dx in (-1, 0, 1))
        np.testing.assert_allclose(img[c, 0], p[c] * np.abs(beam) ** 2, rtol=1e-10, atol=1e-9)


def test_per_channel_autocorr_and_pixel_values_follow_the_channel():
    wl = make_per_channel(grid_n=8, pad=2, n_ant=7, n_pol=2, kernel_k=3, n_chan=3, n_t=5,
                          f0_hz=30e6, df_hz=12e6, diameter_m=25.0)
    v = wl.voltages()
    img = orc.epic_image(v, "ci4", wl.ant_uv, wl.taps, 8, 2, 4, kernel_k=3)
    px = [(0, 0), (3, 11), (15, 2)]
    pv = orc.pixel_values(v, "ci4", wl.ant_uv, wl.taps, 8, 2, 4, px, kernel_k=3)
    for i, (m, l) in enumerate(px):
        np.testing.assert_allclose(pv[:, :, i], img[:, :, m, l], atol=1e-9 * np.abs(img).max())
    # one antenna: the image IS its autocorrelation term, channel by channel
    ac = orc.autocorr_image(v[..., :1], "ci4", wl.ant_uv[:, :1], wl.taps[:, :1], 8, 2, 4, kernel_k=3)
    one = orc.epic_image(v[..., :1], "ci4", wl.ant_uv[:, :1], wl.taps[:, :1], 8, 2, 4, kernel_k=3)
    np.testing.assert_allclose(ac, one, atol=1e-9 * np.abs(one).max())
    assert np.abs(one[0, 0] - one[2, 0] * one[0, 0].sum() / one[2, 0].sum()).max() > 1e-3 * one[0, 0].max()

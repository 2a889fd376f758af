"""Bit-exact GPU tests (-m gpu) of S1 (the 4+4-bit unpack) and integer gridding
THROUGH THE PRODUCTION KERNELS (BASELINE.json north_star: "bit-exactly for the 4-bit unpack").

The fused, wide, tensor and tiled kernels do not unpack with the scalar shift-and-convert of
epic_debug_unpack: they use unpack_words / unpack_words_b8 / b8_to_pair / deinterleave_pols
(csrc/epic_packed.cuh: XOR 8, PRMT into the mantissa of 12582912.0f, FADD2) and, for delta plans,
the biased-byte integer gather.  These tests drive every one of the 256 byte values, in every byte
lane of the 32-bit voltage words, through each of those kernels and require EXACT equality.

How a whole-path result can be exact: with all antennas of a plan in ONE cell, the relocated
aperture has a single nonzero cell at the origin, every butterfly is a + w*0, and the image is the
flat value  sum_t |sum_a E_a|^2  (XY: sum_t (sum_a E_Xa) conj(sum_a E_Ya)) -- small integers, exact
in fp32 in any summation order.  The expectation is typed out here from the sext4 rule (reading
Q1); oracle.unpack_ci4 (pinned against a typed table in test_oracle_pins.py) must agree with it.
"""
import numpy as np
import pytest

from oracle import epic_oracle as orc
from workloads import make_custom

from epic_testlib import run_gpu

pytestmark = pytest.mark.gpu

TWOPASS, FUSED, TILED, TENSOR, STREAM = 1, 2, 3, 4, 5


def _sext4(n):
    return n - 16 if n >= 8 else n


def _unpack_typed(v):
    """uint8 array -> complex128 from the rule typed out here (not the oracle's code)."""
    lut = np.array([complex(_sext4(b >> 4), _sext4(b & 15)) for b in range(256)])
    return lut[np.asarray(v, dtype=np.uint8)]


def _one_cell_workload(grid_n, pad, n_ant, n_pol, n_chan, n_t, n_products, unit_taps, cell=(5, 7), others=0):
    """n_ant antennas in one cell (+ `others` antennas one cell up-right, which the caller keeps at
    zero voltage).  unit_taps: pass explicit K = 1 taps 1 + 0i, which selects the tap (float
    unpack) instantiations instead of the delta (integer gather) ones."""
    uv = np.array([cell] * n_ant + [(cell[0] + 1, cell[1] + 1)] * others, dtype=np.float32)
    wl = make_custom(grid_n=grid_n, pad=pad, n_ant=n_ant + others, n_pol=n_pol, kernel_k=1, n_chan=n_chan, n_t=n_t,
                     n_products=n_products, ant_uv=uv)
    if unit_taps:
        wl.taps = np.zeros((n_ant + others, 1, 1, 2), dtype=np.float32)
        wl.taps[..., 0] = 1.0
    return wl


def _expected_flat(v, n_products):
    """v uint8 [T][C][Np][A] -> float64 [C][planes]: the flat image value of every plane."""
    e = _unpack_typed(v).sum(axis=-1)            # [T][C][Np]: all antennas share the cell
    assert np.array_equal(e, orc.unpack_ci4(v).sum(axis=-1))
    xx = (e[:, :, 0].real ** 2 + e[:, :, 0].imag ** 2).sum(axis=0)     # exact integers (np.abs would take a sqrt)
    if n_products == 1:
        return xx[:, None]
    yy = (e[:, :, 1].real ** 2 + e[:, :, 1].imag ** 2).sum(axis=0)
    if n_products == 2:
        return np.stack([xx, yy], axis=1)
    xy = (e[:, :, 0] * np.conj(e[:, :, 1])).sum(axis=0)
    return np.stack([xx, yy, xy.real, xy.imag, xy.real, -xy.imag], axis=1)


def _assert_flat_exact(gpu, flat, what):
    assert gpu.shape[:2] == flat.shape, (gpu.shape, flat.shape)
    want = flat.astype(np.float32)[:, :, None, None]
    assert np.array_equal(want.astype(np.float64), flat[:, :, None, None])  # the expectation is fp32-exact
    bad = np.argwhere(gpu != want)
    assert bad.size == 0, f"{what}: {len(bad)} pixels differ, first {bad[:3].tolist()}"


def _every_byte_voltages(n_chan, n_t, n_pol, n_ant):
    """Frame i = t * n_chan + c: ONE antenna of each polarisation is nonzero, the rest hold byte
    0x00.  X: antenna slot (i // 256) % A holds byte i % 256; Y: slot + 3 holds the complement.
    With n_chan * n_t >= 256 * A every byte value visits every antenna slot (asserted)."""
    v = np.zeros((n_t, n_chan, n_pol, n_ant), dtype=np.uint8)
    seen = set()
    for t in range(n_t):
        for c in range(n_chan):
            i = t * n_chan + c
            b, slot = i % 256, (i // 256) % n_ant
            seen.add((b, slot))
            v[t, c, 0, slot] = b
            if n_pol == 2:
                v[t, c, 1, (slot + 3) % n_ant] = 255 - b
    assert len(seen) == 256 * n_ant
    return v


CASES = [
    # (id, grid_n, pad, path, unit_taps)
    ("fused-delta-intgather-N128", 64, 2, FUSED, False),
    ("fused-taps-N128", 64, 2, FUSED, True),
    ("fused-delta-intgather-N64", 32, 2, FUSED, False),
    ("fused-taps-N64", 32, 2, FUSED, True),
    ("fused-delta-intgather-N32", 16, 2, FUSED, False),
    ("fused-taps-N32", 16, 2, FUSED, True),
    ("tensor-delta-N128", 64, 2, TENSOR, False),
    ("tensor-taps-N128", 64, 2, TENSOR, True),
    ("tiled-delta-N256", 128, 2, TILED, False),
    ("tiled-taps-N256", 128, 2, TILED, True),
    ("tiled-delta-N512", 128, 4, TILED, False),
    ("stream-delta-N256", 128, 2, STREAM, False),
    ("stream-taps-N256", 128, 2, STREAM, True),
    ("stream-delta-N512", 128, 4, STREAM, False),
    ("twopass-N128", 64, 2, TWOPASS, False),
]


@pytest.mark.parametrize("n_pol,order", [(2, "TCPA"), (2, "TCAP"), (1, "TCPA")], ids=["2pol", "2pol-native", "1pol"])
@pytest.mark.parametrize("case", CASES, ids=lambda c: c[0])
def test_production_unpack_every_byte_value_exact(case, n_pol, order):
    _, grid_n, pad, path, unit_taps = case
    if path == TENSOR and n_pol != 2:
        pytest.skip("the tensor-core variant takes two polarisations")
    n_products = 4 if n_pol == 2 else 1
    n_chan, n_t, n_ant = 256, 8 if n_pol == 2 else 9, 8       # 1 pol: odd n_t = a half-filled last pair
    if grid_n * pad == 512:
        n_chan, n_t = 64, 4 * n_t                             # same frames, a quarter of the image memory
    wl = _one_cell_workload(grid_n, pad, n_ant, n_pol, n_chan, n_t, n_products, unit_taps)
    v = _every_byte_voltages(n_chan, n_t, n_pol, n_ant)
    native = order == "TCAP"
    vin = np.ascontiguousarray(np.swapaxes(v, 2, 3)) if native else v
    gpu, info = run_gpu(wl, volt=vin, path=path, native=native, return_plan_info=True)
    assert info["path"] == path
    _assert_flat_exact(gpu, _expected_flat(v, n_products), case[0])


@pytest.mark.parametrize("case", CASES, ids=lambda c: c[0])
def test_production_unpack_random_bytes_exact(case):
    """Every antenna of every frame holds a random byte (uniform over all 256 values, so -8 and +7
    are as common as 0): sums of 8 samples per cell, both polarisations, two calls."""
    _, grid_n, pad, path, unit_taps = case
    rng = np.random.default_rng(77)
    wl = _one_cell_workload(grid_n, pad, 8, 2, 37, 21, 4, unit_taps)
    v = rng.integers(0, 256, (21, 37, 2, 8), dtype=np.uint8)
    gpu = run_gpu(wl, volt=v, path=path, calls=2)
    _assert_flat_exact(gpu, _expected_flat(v, 4), case[0])


@pytest.mark.parametrize("path", [FUSED, TENSOR], ids=["fused", "tensor"])
@pytest.mark.parametrize("n_same,byte", [(16, 0x77), (16, 0x88), (16, None), (17, 0x77), (17, 0x88), (17, None), (20, None)])
def test_integer_gather_carry_limits(path, n_same, byte):
    """The delta kernels' integer gather adds biased bytes (0..15) per antenna: 16 antennas in one
    cell at +7 (0x77: byte sum 240) and at -8 (0x88: byte sum 0) are the no-carry extremes; 17 or
    more in a cell must take the float gather and stay exact."""
    others = (-n_same) % 4
    wl = _one_cell_workload(64, 2, n_same, 2, 3, 5, 4, False, others=others)
    rng = np.random.default_rng(n_same)
    v = np.zeros((5, 3, 2, n_same + others), dtype=np.uint8)
    v[..., :n_same] = byte if byte is not None else rng.integers(0, 256, (5, 3, 2, n_same), dtype=np.uint8)
    gpu = run_gpu(wl, volt=v, path=path)
    _assert_flat_exact(gpu, _expected_flat(v, 4), f"{n_same} x {byte}")


def test_unit_phasors_keep_the_unpack_exact():
    """Delay phasors of exactly 1 + 0i route the delta plan through the phasor-multiplying unpack
    (no integer gather): still exact."""
    wl = _one_cell_workload(64, 2, 8, 2, 5, 7, 4, False)
    v = np.random.default_rng(3).integers(0, 256, (7, 5, 2, 8), dtype=np.uint8)
    ph = np.ones((5, 2, 8), dtype=np.complex64)
    for path in (FUSED, TWOPASS):
        gpu = run_gpu(wl, volt=v, path=path, phasors=ph)
        _assert_flat_exact(gpu, _expected_flat(v, 4), f"phasors path {path}")
    wl = _one_cell_workload(128, 2, 8, 2, 5, 7, 4, False)      # large grid: phasors folded into the taps
    for path in (STREAM, TILED):
        gpu = run_gpu(wl, volt=v, path=path, phasors=ph)
        _assert_flat_exact(gpu, _expected_flat(v, 4), f"phasors path {path}")


# ------------------------------------------------------------------ run-to-run reproducibility
REPRO = [
    ("LWA55 wide", dict(idx=55, n_chan=40, n_t=100), FUSED),    # wide fused kernel
    ("C2 fused", dict(idx=2, n_chan=40, n_t=333), FUSED),       # units split between CTAs: fix-up order
    ("C3 fused", dict(idx=3, n_chan=24, n_t=200), FUSED),
    ("C4 tiled", dict(idx=4, n_chan=7, n_t=60), TILED),
    ("C5 tiled", dict(idx=5, n_chan=2, n_t=9), TILED),
    ("C4 stream", dict(idx=4, n_chan=19, n_t=60), STREAM),      # several waves
    ("C5 stream", dict(idx=5, n_chan=3, n_t=9), STREAM),
]


@pytest.mark.parametrize("name,kw,path", REPRO, ids=[r[0] for r in REPRO])
def test_results_are_bit_reproducible(name, kw, path):
    """No atomics anywhere and a fixed summation order: two runs of the same call give bit-identical
    images (the stand-in for compute-sanitizer racecheck, which this GPU pool does not allow)."""
    from workloads import make_config, make_lwa55
    wl = make_lwa55(n_chan=kw["n_chan"], n_t=kw["n_t"]) if kw["idx"] == 55 else make_config(kw["idx"], n_chan=kw["n_chan"], n_t=kw["n_t"])
    v = wl.voltages()
    a, info = run_gpu(wl, volt=v, path=path, return_plan_info=True)
    b = run_gpu(wl, volt=v, path=path)
    assert info["path"] == path
    assert np.array_equal(a, b), name


# ------------------------------------------------------------------ wide fused kernel: exact folds
@pytest.mark.parametrize("grid_n,pad", [(64, 2), (64, 1)], ids=["N128", "N64"])
def test_wide_kernel_folds_are_exact(grid_n, pad):
    """Four occupied cells 32 apart in x and y, (0,0) (32,0) (0,32) (32,32) after relocation: the wide kernel's
    x-fold (in the gather) and y-fold (in the column pass) multiply by W_N^{32 l}, W_N^{32 m} -- fourth (N = 128)
    or second (N = 64) roots of unity -- so the image A[m][l] = S00 + w^l S10 + w^m S01 + w^(l+m) S11 is made of
    exact integers; typed out here and compared exactly, for all 256 byte values."""
    N = grid_n * pad
    cells = [(5, 7), (37, 7), (5, 39), (37, 39)]              # (x, y)
    uv = np.array([c for c in cells for _ in range(2)], dtype=np.float32)   # two antennas per cell
    wl = make_custom(grid_n=grid_n, pad=pad, n_ant=8, n_pol=2, kernel_k=1, n_chan=9, n_t=29, n_products=4, ant_uv=uv)
    rng = np.random.default_rng(64)
    v = rng.integers(0, 256, (29, 9, 2, 8), dtype=np.uint8)
    gpu, info = run_gpu(wl, volt=v, path=FUSED, return_plan_info=True)
    assert info["path"] == FUSED and info["support"][2:] == (33, 33)
    e = _unpack_typed(v)                                        # [T][C][Np][A]
    s = e.reshape(29, 9, 2, 4, 2).sum(axis=-1)                  # per cell: S00, S10, S01, S11
    w = {128: 1j, 64: -1.0}[N]
    l = np.arange(N)[None, :]
    m = np.arange(N)[:, None]
    a = (s[..., 0, None, None] + s[..., 1, None, None] * w ** (l % 4) + s[..., 2, None, None] * w ** (m % 4)
         + s[..., 3, None, None] * w ** ((l + m) % 4))         # [T][C][Np][N][N], exact Gaussian integers
    ax, ay = a[:, :, 0], a[:, :, 1]
    xy = (ax * np.conj(ay)).sum(axis=0)
    want = np.stack([(ax.real ** 2 + ax.imag ** 2).sum(axis=0), (ay.real ** 2 + ay.imag ** 2).sum(axis=0),
                     xy.real, xy.imag, xy.real, -xy.imag], axis=1)          # [C][6][N][N]
    assert np.array_equal(want.astype(np.float32).astype(np.float64), want)
    bad = np.argwhere(gpu != want.astype(np.float32))
    assert bad.size == 0, f"{len(bad)} pixels differ, first {bad[:3].tolist()}"

"""Generators for BASELINE.json's five configurations (C1..C5) and custom test cases.

Input recipe: every array is a pure function of
(config index, n_chan, n_t).  Seeds are ``numpy.random.SeedSequence([BASE_SEED + i,
stream, block])`` with the fixed stream ids below, so antenna positions do not
change when a test shrinks the channel/time extent.

The layouts stand in for the LWA-SV array geometry and live voltage streams the
paper used, which are not available here.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

BASE_SEED = 190411422 * 10
_S_POS, _S_PHASE, _S_SRC, _S_NOISE, _S_WAVE = 0, 1, 2, 3, 4
_TIME_BLOCK = 50  # voltages are drawn in independent blocks of 50 time samples

CONFIG_NAMES = {
    1: "C1-tiny-16ant-32x32-cf32",
    2: "C2-lwa-256ant-128x128-delta-XXYY",
    3: "C3-lwa-256ant-128x128-gauss3-4prod",
    4: "C4-dense-1024ant-256x256-gauss3-4prod",
    5: "C5-stress-4096ant-512x512-gauss5-4prod",
}


def _rng(seed: int, stream: int, block: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence([seed, stream, block])))


def pack_ci4(re: np.ndarray, im: np.ndarray) -> np.ndarray:
    """Pack integer (re, im) in -8..7 into one byte: high nibble = real, low = imaginary,
    each two's complement (reading Q1 of PAPER.md:120 "4+4-bit complex integer")."""
    re = np.asarray(re).astype(np.int16)
    im = np.asarray(im).astype(np.int16)
    return (((re & 0xF) << 4) | (im & 0xF)).astype(np.uint8)


def _round_half_up(x: np.ndarray) -> np.ndarray:
    return np.floor(np.asarray(x, dtype=np.float64) + 0.5)


def gaussian_taps(ant_uv: np.ndarray, k: int, sigma: float, phase: np.ndarray) -> np.ndarray:
    """Separable Gaussian illumination taps centred on each antenna's true sub-cell position,
    with a per-antenna phase, normalised to sum |w| = 1.  Returns float32 [A][K][K][2]
    indexed [dy+h][dx+h] ("user-defined convolution kernel")."""
    uv = np.asarray(ant_uv, dtype=np.float32).astype(np.float64)
    f = uv - _round_half_up(uv)  # (fx, fy) in [-0.5, 0.5)
    h = (k - 1) // 2
    d = np.arange(-h, h + 1, dtype=np.float64)
    gx = np.exp(-((d[None, :] - f[:, 0:1]) ** 2) / (2 * sigma * sigma))  # [A][K]
    gy = np.exp(-((d[None, :] - f[:, 1:2]) ** 2) / (2 * sigma * sigma))
    w = gy[:, :, None] * gx[:, None, :]
    w /= w.sum(axis=(1, 2), keepdims=True)
    wc = w * np.exp(1j * np.asarray(phase, dtype=np.float64))[:, None, None]
    out = np.empty(wc.shape + (2,), dtype=np.float32)
    out[..., 0] = wc.real
    out[..., 1] = wc.imag
    return out


def tophat_taps(ant_uv: np.ndarray, k: int, width_cells, phase: Optional[np.ndarray] = None) -> np.ndarray:
    """Square top-hat illumination of side ``width_cells`` centred on each antenna's true position
    ("a simple square top-hat function with 3-meter extent"), sampled as the fraction
    of each cell [j-1/2, j+1/2) it covers, separable in x and y, normalised to sum 1, times an
    optional per-antenna phase.  float32 [..., A, K, K, 2] for ant_uv [..., A, 2]; width_cells is a
    scalar or broadcasts over the leading (channel) axis."""
    uv = np.asarray(ant_uv, dtype=np.float32).astype(np.float64)
    f = uv - _round_half_up(uv)
    h = (k - 1) // 2
    d = np.arange(-h, h + 1, dtype=np.float64)
    half = 0.5 * np.asarray(width_cells, dtype=np.float64)
    half = half.reshape(half.shape + (1,) * (uv.ndim - 1 - half.ndim) + (1,)) if half.ndim else half

    def cover(frac):  # [..., A] -> [..., A, K]: overlap of [frac-half, frac+half] with [d-1/2, d+1/2]
        lo = np.maximum(frac[..., None] - half, d - 0.5)
        hi = np.minimum(frac[..., None] + half, d + 0.5)
        return np.clip(hi - lo, 0.0, None)

    w = cover(f[..., 1])[..., :, None] * cover(f[..., 0])[..., None, :]
    w = w / w.sum(axis=(-2, -1), keepdims=True)
    wc = w.astype(np.complex128)
    if phase is not None:
        wc = wc * np.exp(1j * np.asarray(phase, dtype=np.float64))[..., None, None]
    out = np.empty(wc.shape + (2,), dtype=np.float32)
    out[..., 0] = wc.real
    out[..., 1] = wc.imag
    return out


@dataclass
class Workload:
    name: str
    index: int
    seed: int
    grid_n: int
    pad: int
    n_ant: int
    n_pol: int
    kernel_k: int
    n_chan: int
    n_t: int
    input_kind: str  # "cf32" | "ci4"
    n_products: int  # 1 (XX), 2 (XX,YY) or 4 (XX,YY,XY,YX)
    ant_uv: np.ndarray  # float32 [A][2] = (u, v) in cell units, or [C][A][2]: one layout per channel
    taps: Optional[np.ndarray] = None  # float32 [A][K][K][2] ([C][A][K][K][2]) or None (delta kernel)
    tap_phase: Optional[np.ndarray] = None  # float64 [A]; voltages carry e^{-i phase}
    noise_sigma: float = 2.0
    sources: List[dict] = field(default_factory=list)  # {"l_pix","m_pix","var"}

    @property
    def N(self) -> int:
        return self.grid_n * self.pad

    @property
    def n_planes(self) -> int:
        return {1: 1, 2: 2, 4: 6}[self.n_products]

    @property
    def frames(self) -> int:
        return self.n_chan * self.n_t

    def describe(self) -> dict:
        return {
            "workload": self.name, "n_ant": self.n_ant, "n_pol": self.n_pol,
            "grid_n": self.grid_n, "pad": self.pad, "N": self.N, "kernel_k": self.kernel_k,
            "n_chan": self.n_chan, "n_t": self.n_t, "input": self.input_kind,
            "n_products": self.n_products, "n_sources": len(self.sources), "seed": self.seed,
        }

    # ---- voltages -----------------------------------------------------------------
    def _source_steer(self) -> Optional[np.ndarray]:
        """complex128 [n_src][A] ([C][n_src][A] for per-channel layouts): geometric phase of a
        plane wave from pixel (l_pix, m_pix), times the per-antenna instrumental phase
        e^{-i phi_a} that the taps undo.  On lambda_c/2 cells a direction is the same pixel in
        every channel, so per-channel coordinates need no other change."""
        if not self.sources:
            return None
        uv = self.ant_uv.astype(np.float64)
        inst = np.exp(-1j * self.tap_phase) if self.tap_phase is not None else 1.0
        rows = []
        for s in self.sources:
            ph = -2.0 * np.pi * (uv[..., 0] * s["l_pix"] + uv[..., 1] * s["m_pix"]) / self.N
            rows.append(np.exp(1j * ph) * inst)
        return np.stack(rows, axis=-2)

    def voltage_block(self, block: int, n_rows: int) -> np.ndarray:
        """Time samples [block*50, block*50 + n_rows) as uint8 [n_rows][C][Np][A] (ci4) or
        float32 [n_rows][C][Np][A][2] (cf32)."""
        C, P, A = self.n_chan, self.n_pol, self.n_ant
        rn = _rng(self.seed, _S_NOISE, block)
        if self.input_kind == "cf32":
            v = rn.standard_normal((_TIME_BLOCK, C, P, A, 2), dtype=np.float32)
            return v[:n_rows]
        x = rn.standard_normal((_TIME_BLOCK, C, P, A, 2), dtype=np.float32)[:n_rows]
        x *= np.float32(self.noise_sigma)
        steer = self._source_steer()
        if steer is not None:
            rw = _rng(self.seed, _S_WAVE, block)
            wv = rw.standard_normal((_TIME_BLOCK, C, len(self.sources), 2))[:n_rows]
            amp = np.sqrt(np.array([s["var"] for s in self.sources]) / 2.0)
            wave = (wv[..., 0] + 1j * wv[..., 1]) * amp  # [t][C][n_src]
            sig = np.einsum("tcs,csa->tca" if steer.ndim == 3 else "tcs,sa->tca", wave, steer)  # same waveform in both pols
            x[..., 0] += sig.real[:, :, None, :].astype(np.float32)
            x[..., 1] += sig.imag[:, :, None, :].astype(np.float32)
        q = np.clip(np.rint(x), -8, 7).astype(np.int8)
        return pack_ci4(q[..., 0], q[..., 1])

    def voltages(self) -> np.ndarray:
        """All n_t samples: uint8 [T][C][Np][A] (ci4) or float32 [T][C][Np][A][2] (cf32)."""
        C, P, A = self.n_chan, self.n_pol, self.n_ant
        shape = (self.n_t, C, P, A) + ((2,) if self.input_kind == "cf32" else ())
        out = np.empty(shape, dtype=np.float32 if self.input_kind == "cf32" else np.uint8)
        for b in range((self.n_t + _TIME_BLOCK - 1) // _TIME_BLOCK):
            t0 = b * _TIME_BLOCK
            n = min(_TIME_BLOCK, self.n_t - t0)
            out[t0:t0 + n] = self.voltage_block(b, n)
        return out

    def taps_or_none(self) -> Optional[np.ndarray]:
        return self.taps


# ---- layouts ------------------------------------------------------------------------
def _layout_integer_cells(seed, n_ant, grid_n):
    r = _rng(seed, _S_POS)
    idx = r.choice(grid_n * grid_n, size=n_ant, replace=False)
    y, x = np.divmod(idx, grid_n)
    return np.stack([x, y], axis=1).astype(np.float32)


def _layout_disc(seed, n_ant, grid_n, diameter_m=100.0, freq_hz=38e6):
    r = _rng(seed, _S_POS)
    cell_m = 299792458.0 / freq_hz / 2.0  # half a wavelength
    rad = 0.5 * diameter_m * np.sqrt(r.random(n_ant))
    th = 2.0 * np.pi * r.random(n_ant)
    c = grid_n / 2.0
    return np.stack([c + rad * np.cos(th) / cell_m, c + rad * np.sin(th) / cell_m], axis=1).astype(np.float32)


def _layout_lattice(seed, side, pitch=4.0, offset=2.0, jitter=1.0):
    r = _rng(seed, _S_POS)
    j, i = np.meshgrid(np.arange(side), np.arange(side), indexing="ij")
    u = offset + pitch * i.ravel() + r.uniform(-jitter, jitter, side * side)
    v = offset + pitch * j.ravel() + r.uniform(-jitter, jitter, side * side)
    return np.stack([u, v], axis=1).astype(np.float32)


def _layout_uniform(seed, n_ant, grid_n):
    r = _rng(seed, _S_POS)
    uv = r.uniform(0.0, grid_n, size=(n_ant, 2)).astype(np.float32)
    return np.minimum(uv, np.nextafter(np.float32(grid_n), np.float32(0)))


def _draw_sources(seed, n_src, N, n_t, n_ant, noise_sigma, snr=10.0):
    """Sources at integer image pixels inside the visible hemisphere.  Per-antenna source
    variance from the image-plane reading of "SNR 10": snr = sqrt(T)*A*var_s/var_n."""
    r = _rng(seed, _S_SRC)
    out = []
    var_n = 2.0 * noise_sigma * noise_sigma
    while len(out) < n_src:
        kl, km = (int(v) for v in r.integers(-N // 2, N // 2, size=2))
        if (2.0 * kl / N) ** 2 + (2.0 * km / N) ** 2 > 0.8:
            continue
        out.append({"l_pix": kl % N, "m_pix": km % N, "var": snr * var_n / (np.sqrt(n_t) * n_ant)})
    return out


def make_config(i: int, n_chan: Optional[int] = None, n_t: Optional[int] = None,
                n_ant: Optional[int] = None) -> Workload:
    """BASELINE.json configs[i-1].  n_chan / n_t shrink the extent for tests; n_ant (C5 only)
    takes the first n antennas of the same draw for the antenna-count sweep."""
    seed = BASE_SEED + i
    if i == 1:
        C, T = n_chan or 1, n_t or 8
        uv = _layout_integer_cells(seed, 16, 16)
        return Workload(CONFIG_NAMES[1], 1, seed, 16, 2, 16, 1, 1, C, T, "cf32", 1, uv)
    if i == 2:
        C, T = n_chan or 128, n_t or 1000
        uv = _layout_disc(seed, 256, 64)
        return Workload(CONFIG_NAMES[2], 2, seed, 64, 2, 256, 2, 1, C, T, "ci4", 2, uv)
    if i == 3:
        C, T = n_chan or 128, n_t or 2500
        uv = _layout_disc(BASE_SEED + 2, 256, 64)  # "same 256-antenna layout" as C2
        ph = _rng(seed, _S_PHASE).uniform(0.0, 2.0 * np.pi, 256)
        taps = gaussian_taps(uv, 3, 0.5, ph)
        src = _draw_sources(seed, 1, 128, 2500, 256, 2.0)
        return Workload(CONFIG_NAMES[3], 3, seed, 64, 2, 256, 2, 3, C, T, "ci4", 4, uv, taps, ph, 2.0, src)
    if i == 4:
        C, T = n_chan or 64, n_t or 1000
        uv = _layout_lattice(seed, 32)
        ph = _rng(seed, _S_PHASE).uniform(0.0, 2.0 * np.pi, 1024)
        taps = gaussian_taps(uv, 3, 0.5, ph)
        return Workload(CONFIG_NAMES[4], 4, seed, 128, 2, 1024, 2, 3, C, T, "ci4", 4, uv, taps, ph)
    if i == 5:
        C, T = n_chan or 32, n_t or 500
        A = n_ant or 4096
        uv = _layout_uniform(seed, 4096, 256)[:A]
        ph = _rng(seed, _S_PHASE).uniform(0.0, 2.0 * np.pi, 4096)[:A]
        taps = gaussian_taps(uv, 5, 0.5, ph)
        src = _draw_sources(seed, 3, 512, 500, A, 2.0)
        name = CONFIG_NAMES[5] if A == 4096 else CONFIG_NAMES[5].replace("4096ant", f"{A}ant")
        return Workload(name, 5, seed, 256, 2, A, 2, 5, C, T, "ci4", 4, uv, taps, ph, 2.0, src)
    raise ValueError(f"no config {i}")


def make_custom(*, grid_n: int, pad: int, n_ant: int, n_pol: int, kernel_k: int, n_chan: int,
                n_t: int, input_kind: str = "ci4", n_products: Optional[int] = None,
                layout: str = "uniform", seed: int = 7, n_sources: int = 0,
                ant_uv: Optional[np.ndarray] = None) -> Workload:
    """Arbitrary small case for tests (edge shapes, wrap-around, single pol ...)."""
    s = BASE_SEED + 1000 + seed
    if ant_uv is not None:
        uv = np.asarray(ant_uv, dtype=np.float32)
    elif layout == "integer":
        uv = _layout_integer_cells(s, n_ant, grid_n)
    elif layout == "disc":
        uv = _layout_disc(s, n_ant, grid_n, diameter_m=0.4 * grid_n * 3.94464)
    elif layout == "uniform":
        uv = _layout_uniform(s, n_ant, grid_n)
    elif layout == "wrap":  # positions over the whole padded plane incl. negative coordinates
        uv = (_rng(s, _S_POS).uniform(-grid_n * pad, 2 * grid_n * pad, size=(n_ant, 2))).astype(np.float32)
    else:
        raise ValueError(layout)
    if n_products is None:
        n_products = 4 if n_pol == 2 else 1
    taps = ph = None
    if kernel_k > 1:
        ph = _rng(s, _S_PHASE).uniform(0.0, 2.0 * np.pi, n_ant)
        taps = gaussian_taps(uv, kernel_k, 0.5, ph)
    N = grid_n * pad
    src = _draw_sources(s, n_sources, N, max(n_t, 1), n_ant, 2.0) if n_sources else []
    name = f"custom-{n_ant}ant-{N}x{N}-k{kernel_k}-p{n_pol}-{input_kind}-s{seed}"
    return Workload(name, 0, s, grid_n, pad, n_ant, n_pol, kernel_k, n_chan, n_t, input_kind,
                    n_products, uv, taps, ph, 2.0, src)


def make_lwa55(*, n_chan: int, n_t: int, kernel: str = "tophat", n_products: int = 4, n_ant: int = 256,
               freq_hz: float = 55.25e6, seed: int = 55, n_sources: int = 0, n_pol: int = 2) -> Workload:
    """The paper's own operating point as a single-layout workload: ``n_ant`` antennas
    uniform in area in a 110 m x 100 m ellipse, gridded on lambda/2 cells at 55.25 MHz (2.713 m: about 41 x 37
    cells, beyond a 32 x 32 support) onto a 64 x 64 grid padded to 128 x 128; kernel "tophat" = the 3 m square
    top-hat sampled per cell (3 x 3 taps, per-antenna phase), "delta" = nearest cell."""
    s = BASE_SEED + 3000 + seed
    r = _rng(s, _S_POS)
    cell_m = 299792458.0 / freq_hz / 2.0
    rad = np.sqrt(r.random(n_ant))
    th = 2.0 * np.pi * r.random(n_ant)
    uv = np.stack([32.0 + 55.0 * rad * np.cos(th) / cell_m, 32.0 + 50.0 * rad * np.sin(th) / cell_m], axis=1).astype(np.float32)
    taps = ph = None
    k = 1
    if kernel == "tophat":
        k = 3
        ph = _rng(s, _S_PHASE).uniform(0.0, 2.0 * np.pi, n_ant)
        taps = tophat_taps(uv, 3, 3.0 / cell_m, ph)
    elif kernel != "delta":
        raise ValueError(kernel)
    src = _draw_sources(s, n_sources, 128, max(n_t, 1), n_ant, 2.0) if n_sources else []
    name = f"LWA55-{n_ant}ant-128x128-{kernel}-{n_products}prod"
    return Workload(name, 0, s, 64, 2, n_ant, n_pol, k, n_chan, n_t, "ci4", n_products, uv, taps, ph, 2.0, src)


def make_per_channel(*, grid_n: int, pad: int, n_ant: int, n_pol: int, kernel_k: int, n_chan: int, n_t: int,
                     f0_hz: float, df_hz: float, diameter_m: float = 100.0, tophat_m: float = 3.0,
                     n_products: Optional[int] = None, n_sources: int = 0, seed: int = 7,
                     layout_seed: Optional[int] = None) -> Workload:
    """One layout per channel: antennas uniform in area in
    a disc of ``diameter_m`` metres, channel c at f0 + c df with cell = lambda_c / 2, so
    ant_uv[c] = grid_n/2 + position / cell_c; kernel_k = 1 is the delta kernel, otherwise the
    ``tophat_m`` square top-hat sampled at each channel's cell size with a per-antenna phase."""
    s = BASE_SEED + 2000 + seed
    r = _rng(s if layout_seed is None else layout_seed, _S_POS)
    rad = 0.5 * diameter_m * np.sqrt(r.random(n_ant))
    th = 2.0 * np.pi * r.random(n_ant)
    pos = np.stack([rad * np.cos(th), rad * np.sin(th)], axis=1)        # metres, [A][2]
    freq = f0_hz + df_hz * np.arange(n_chan, dtype=np.float64)
    cell_m = 299792458.0 / freq / 2.0                                     # [C]
    uv = (grid_n / 2.0 + pos[None, :, :] / cell_m[:, None, None]).astype(np.float32)
    if n_products is None:
        n_products = 4 if n_pol == 2 else 1
    taps = ph = None
    if kernel_k > 1:
        ph = _rng(s, _S_PHASE).uniform(0.0, 2.0 * np.pi, n_ant)
        taps = tophat_taps(uv, kernel_k, tophat_m / cell_m, ph)
    N = grid_n * pad
    src = _draw_sources(s, n_sources, N, max(n_t, 1), n_ant, 2.0) if n_sources else []
    name = f"perchan-{n_ant}ant-{N}x{N}-k{kernel_k}-p{n_pol}-{f0_hz / 1e6:g}MHz+{n_chan}x{df_hz / 1e3:g}kHz"
    return Workload(name, 0, s, grid_n, pad, n_ant, n_pol, kernel_k, n_chan, n_t, "ci4",
                    n_products, uv, taps, ph, 2.0, src)

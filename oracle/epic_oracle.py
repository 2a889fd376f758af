"""CPU oracle for the EPIC hot path — TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Plain, slow, float64 numpy restatement of what the path computes, written from the paper
(Kent et al., arXiv 1904.11422; /root/reference/PAPER.md) and independent of the CUDA path:
it shares no code, tables or helpers with ``paper_1904_11422_b200`` and imports nothing
from it.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline /
``--impl reference`` leg may import this module.

What it computes (Eq. 5, §3.2), per frequency channel c and
time sample t ("frame"), per polarisation p:

  S1  unpack   byte -> E = sext4(high nibble) + i*sext4(low nibble)
  S2  cells    nearest cell of each antenna, tap cells modulo N
  S3  grid     G[y][x] += W_a[dy][dx] * E_a   (convolve with illumination W)   PAPER.md:122-124, Eq. 4-5
  S4  image    A[m][l] = sum_yx G[y][x] exp(+2 pi i (x l + y m)/N)             PAPER.md:126, Eq. 5
  S5  products XX=|A_X|^2, YY=|A_Y|^2, XY=A_X conj(A_Y), YX=A_Y conj(A_X)       PAPER.md:86, 126; Eq. 2
  S6  accumulate  sum over the time samples of the call

EPIC reaches the Eq. 5 result exactly (it is a re-ordering of the FX sum), so the oracle is
the definition written out.  S4 exists twice: ``idft2_definition`` (the literal double sum) and
``idft2_fast`` (a library inverse FFT, a permitted primitive step); the tests prove them equal
on small planes and the fast one is used for large ones.

Readings of the paper where it is silent:
Q1 high nibble real / low nibble imaginary, two's complement; Q4 nearest cell = floor(x+0.5);
Q15 antenna coordinates (and taps) may differ per channel: cell = lambda_c / 2;
Q6 cells wrap modulo N; Q8 +2 pi i (inverse transform); Q9 unnormalised; Q10 natural order,
zenith at [0][0]; Q11 XY = A_X conj(A_Y); Q12 plain sum over time; Q14 plane order
{XX} | {XX,YY} | {XX,YY,ReXY,ImXY,ReYX,ImYX}; Q19 delay compensation = one complex multiplier per
(channel, pol, antenna) applied after unpack.

Pins (tests/test_oracle_*.py, all ``-m "not gpu"``): S1 exhaustive nibble table typed out in the
test; S2 hand-worked cells incl. half-cells and wrap; S3 closed-form sums, collisions add,
linearity; S4 library inverse FFT vs the literal sum, impulse -> plane wave, zero-padding
invariant; S5/S6 one- and two-antenna closed forms, YX = conj(XY); whole path: (a) FX
equivalence with brute-force direct-Fourier imaging of all antenna pairs, (b) Parseval,
(c) plane-wave source peaks at the predicted pixel with height A^2; autocorr_image:
image minus it equals brute-force imaging of the pairs a != b, one antenna -> exactly the image;
per-channel layouts: brute-force FX imaging with each channel's own cells, two-antenna fringe whose
period follows the channel, one sky direction -> one pixel in every channel.
Parity unpinned: only the nibble-order *convention* (Q1) and anything LWA-instrument specific
(no instrument data exists here); every function below has at least one pin.
"""
from __future__ import annotations

from typing import Optional

import numpy as np

TWO_PI = 2.0 * np.pi


# ------------------------------------------------------------------ S1: unpack
def sext4(n: int) -> int:
    """Two's-complement value of a 4-bit nibble (0..15 -> -8..7)."""
    return n - 16 if n >= 8 else n


def unpack_ci4(b: np.ndarray) -> np.ndarray:
    """uint8 array -> complex128, real = sext4(b >> 4), imag = sext4(b & 15)."""
    b = np.asarray(b, dtype=np.uint8).astype(np.int64)
    hi = b >> 4
    lo = b & 15
    re = np.where(hi >= 8, hi - 16, hi)
    im = np.where(lo >= 8, lo - 16, lo)
    return re.astype(np.float64) + 1j * im.astype(np.float64)


def voltages_to_complex(v: np.ndarray, kind: str) -> np.ndarray:
    """[T][C][Np][A] complex128 from ci4 bytes or from cf32 (re, im) pairs."""
    if kind == "ci4":
        return unpack_ci4(v)
    if kind == "cf32":
        v = np.asarray(v, dtype=np.float32).astype(np.float64)
        return v[..., 0] + 1j * v[..., 1]
    raise ValueError(kind)


def channel_voltages(voltages: np.ndarray, kind: str, c: int, t0: int = 0, t1: Optional[int] = None,
                     order: str = "TCPA", delay_phasors: Optional[np.ndarray] = None) -> np.ndarray:
    """complex128 [t1-t0][Np][A] of channel c, ready for gridding: the steps upstream of it in the
    paper's pipeline.  ``order`` "TCAP" = the F-engine order [Time, Channel, Antenna, Polarisation]
    that the paper's transposition block turns into [Time, Channel, Polarisation, Antenna]
    (PAPER.md:120); ``delay_phasors`` complex [C][Np][A] = the "compensation for the signal path
    delays", read as one complex multiplier per (channel, pol, antenna) (Q19)."""
    v = voltages[t0:t1, c]
    if order == "TCAP":
        v = np.swapaxes(v, 1, 2)        # [t][A][Np] -> [t][Np][A]
    elif order != "TCPA":
        raise ValueError(order)
    e = voltages_to_complex(v, kind)
    if delay_phasors is not None:
        e = e * np.asarray(delay_phasors, dtype=np.complex128)[c][None, :, :]
    return e


# ------------------------------------------------------------------ S2: cells
def nearest_cells(ant_uv: np.ndarray) -> np.ndarray:
    """int64 [A][2] = (cx, cy) = floor(double(u) + 0.5), floor(double(v) + 0.5) (reading Q4)."""
    uv = np.asarray(ant_uv, dtype=np.float32).astype(np.float64)
    return np.floor(uv + 0.5).astype(np.int64)


def tap_cells(ant_uv: np.ndarray, kernel_k: int, n: int) -> np.ndarray:
    """int64 [A][K][K]: flat cell y*N + x of tap (dy, dx), y = (cy+dy) mod N, x = (cx+dx) mod N
    (reading Q6: wrap, consistent with the DFT's periodicity)."""
    if kernel_k < 1 or kernel_k % 2 == 0:
        raise ValueError("kernel_k must be odd")
    c = nearest_cells(ant_uv)
    h = (kernel_k - 1) // 2
    out = np.empty((c.shape[0], kernel_k, kernel_k), dtype=np.int64)
    for a in range(c.shape[0]):
        for iy, dy in enumerate(range(-h, h + 1)):
            for ix, dx in enumerate(range(-h, h + 1)):
                y = (int(c[a, 1]) + dy) % n
                x = (int(c[a, 0]) + dx) % n
                out[a, iy, ix] = y * n + x
    return out


def taps_to_complex(taps: Optional[np.ndarray], n_ant: int, kernel_k: int) -> np.ndarray:
    """complex128 [A][K][K]; None = delta kernel (K = 1, tap 1 + 0i)."""
    if taps is None:
        if kernel_k != 1:
            raise ValueError("taps=None means kernel_k == 1")
        return np.ones((n_ant, 1, 1), dtype=np.complex128)
    t = np.asarray(taps, dtype=np.float32).astype(np.float64)
    if t.shape != (n_ant, kernel_k, kernel_k, 2):
        raise ValueError(f"taps shape {t.shape}")
    return t[..., 0] + 1j * t[..., 1]


def channel_layout(ant_uv: np.ndarray, taps: Optional[np.ndarray], c: int):
    """(ant_uv [A][2], taps [A][K][K][2] or None) of channel c.  The grid spacing is tied to "the
    wavelength of the channel", so an antenna's coordinates in cell units, and with
    them its sub-cell offset and taps, differ from channel to channel: ``ant_uv`` [C][A][2] and
    ``taps`` [C][A][K][K][2] carry one layout per channel (reading Q15); arrays without
    the leading axis are the one layout every channel shares."""
    uv = np.asarray(ant_uv)
    if uv.ndim == 3:
        return uv[c], (None if taps is None else np.asarray(taps)[c])
    return uv, taps


# ------------------------------------------------------------------ S3: gridding
def grid_frames(e: np.ndarray, cells: np.ndarray, w: np.ndarray, n: int) -> np.ndarray:
    """Convolve-and-grid (W * E' of Eq. 4-5).

    e [F][A] complex128 (F independent frames), cells [A][K][K], w [A][K][K] complex128.
    Returns G [F][N][N]; contributions landing on the same cell SUM.
    Loop order: antenna, dy, dx — the sum as written, one tap at a time.
    """
    f, n_ant = e.shape
    g = np.zeros((f, n * n), dtype=np.complex128)
    k = cells.shape[1]
    for a in range(n_ant):
        ea = e[:, a]
        for iy in range(k):
            for ix in range(k):
                g[:, cells[a, iy, ix]] += w[a, iy, ix] * ea
    return g.reshape(f, n, n)


# ------------------------------------------------------------------ S4: image transform
def idft2_definition(g: np.ndarray) -> np.ndarray:
    """A[m][l] = sum_y sum_x G[y][x] exp(+2 pi i (x l + y m)/N): the literal double sum of the
    discretised Eq. 5, unnormalised, natural order.  O(N^4); small planes only."""
    g = np.asarray(g, dtype=np.complex128)
    n = g.shape[-1]
    assert g.shape[-2] == n
    out = np.zeros_like(g)
    y, x = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    for m in range(n):
        for l in range(n):
            phase = np.exp(1j * TWO_PI * ((x * l + y * m) % n) / n)
            out[..., m, l] = (g * phase).sum(axis=(-2, -1))
    return out


def idft2_fast(g: np.ndarray) -> np.ndarray:
    """Same transform through the library routine: N^2 * ifft2 (numpy's ifft2 is the +i
    transform scaled by 1/N^2)."""
    g = np.asarray(g, dtype=np.complex128)
    n = g.shape[-1]
    return np.fft.ifft2(g, axes=(-2, -1)) * float(n * n)


# ------------------------------------------------------------------ S5: products
def n_planes(n_pol: int, n_products: int) -> int:
    if (n_pol, n_products) == (1, 1):
        return 1
    if (n_pol, n_products) == (2, 2):
        return 2
    if (n_pol, n_products) == (2, 4):
        return 6
    raise ValueError(f"n_pol={n_pol}, n_products={n_products}")


def products(a: np.ndarray, n_products: int) -> np.ndarray:
    """a [F][Np][N][N] complex -> [F][planes][N][N] float64 (Eq. 2 for which
    factor is conjugated): planes {XX} | {XX,YY} | {XX,YY,Re XY,Im XY,Re YX,Im YX}."""
    n_pol = a.shape[1]
    pl = n_planes(n_pol, n_products)
    out = np.empty((a.shape[0], pl) + a.shape[2:], dtype=np.float64)
    ax = a[:, 0]
    out[:, 0] = ax.real * ax.real + ax.imag * ax.imag
    if n_pol == 2:
        ay = a[:, 1]
        out[:, 1] = ay.real * ay.real + ay.imag * ay.imag
        if n_products == 4:
            xy = ax * np.conj(ay)
            yx = ay * np.conj(ax)
            out[:, 2] = xy.real
            out[:, 3] = xy.imag
            out[:, 4] = yx.real
            out[:, 5] = yx.imag
    return out


# ------------------------------------------------------------------ whole path
def epic_image(voltages: np.ndarray, kind: str, ant_uv: np.ndarray, taps: Optional[np.ndarray],
               grid_n: int, pad: int, n_products: int, kernel_k: int = 1,
               mode: str = "fast", channels: Optional[list] = None,
               frames_per_batch: Optional[int] = None, order: str = "TCPA",
               delay_phasors: Optional[np.ndarray] = None) -> np.ndarray:
    """Accumulated polarised images, float64 [C'][planes][N][N] (C' = len(channels) or C).

    voltages: ci4 uint8 [T][C][Np][A] or cf32 float32 [T][C][Np][A][2] (PAPER.md:120 order
    [Time, Channel, Polarisation, Antenna]).  ant_uv / taps may carry a leading channel axis
    (``channel_layout``).  mode "definition" uses the literal double sum
    for S4, "fast" the library inverse FFT.  ``channels`` restricts the work to some channels
    (used for sampled parity at full size; channels are independent).
    """
    n = grid_n * pad
    t_n, c_n = voltages.shape[:2]
    n_pol, n_ant = (voltages.shape[3], voltages.shape[2]) if order == "TCAP" else voltages.shape[2:4]
    ch = list(range(c_n)) if channels is None else list(channels)
    xform = idft2_definition if mode == "definition" else idft2_fast
    pl = n_planes(n_pol, n_products)
    acc = np.zeros((len(ch), pl, n, n), dtype=np.float64)
    if frames_per_batch is None:
        frames_per_batch = max(1, min(t_n, (1 << 21) // (n * n * n_pol)))
    for ci, c in enumerate(ch):
        uv_c, taps_c = channel_layout(ant_uv, taps, c)
        cells = tap_cells(uv_c, kernel_k, n)                 # S2
        w = taps_to_complex(taps_c, n_ant, kernel_k)
        for t0 in range(0, t_n, frames_per_batch):
            e = channel_voltages(voltages, kind, c, t0, t0 + frames_per_batch, order, delay_phasors)  # [F][Np][A]
            f = e.shape[0]
            img = np.empty((f, n_pol, n, n), dtype=np.complex128)
            for p in range(n_pol):
                g = grid_frames(e[:, p, :], cells, w, n)     # S3
                img[:, p] = xform(g)                         # S4
            acc[ci] += products(img, n_products).sum(axis=0)  # S5, S6
    return acc


# ------------------------------------------------------------------ optional: autocorrelation removal
def autocorr_image(voltages: np.ndarray, kind: str, ant_uv: np.ndarray, taps: Optional[np.ndarray],
                   grid_n: int, pad: int, n_products: int, kernel_k: int = 1,
                   channels: Optional[list] = None, order: str = "TCPA",
                   delay_phasors: Optional[np.ndarray] = None) -> np.ndarray:
    """The a = b part of the accumulated EPIC image ("the zero-spacing power inherent in
    EPIC"), float64 [C'][planes][N][N], from the definition: the image is
    sum_t A_p conj(A_q) with A_p = sum_a E_ap What_a, What_a = transform of antenna a gridded alone
    with unit voltage; its a = b terms are  sum_a (sum_t E_ap conj(E_aq)) |What_a|^2.
    Subtracting it from epic_image leaves the direct-Fourier image of the pairs a != b only
    (pinned in tests/test_oracle_pins.py by brute force)."""
    n = grid_n * pad
    t_n, c_n = voltages.shape[:2]
    n_pol, n_ant = (voltages.shape[3], voltages.shape[2]) if order == "TCAP" else voltages.shape[2:4]
    ch = list(range(c_n)) if channels is None else list(channels)

    def beams(uv_c, taps_c):
        cells = tap_cells(uv_c, kernel_k, n)
        w = taps_to_complex(taps_c, n_ant, kernel_k)
        b = np.empty((n_ant, n, n), dtype=np.float64)  # |What_a|^2
        for a in range(n_ant):
            one = np.zeros((1, n_ant), dtype=np.complex128)
            one[0, a] = 1.0
            b[a] = np.abs(idft2_fast(grid_frames(one, cells, w, n))[0]) ** 2
        return b

    per_channel = np.asarray(ant_uv).ndim == 3
    beam = None if per_channel else beams(ant_uv, taps)
    pl = n_planes(n_pol, n_products)
    out = np.zeros((len(ch), pl, n, n), dtype=np.float64)
    for ci, c in enumerate(ch):
        if per_channel:
            beam = beams(*channel_layout(ant_uv, taps, c))
        e = channel_voltages(voltages, kind, c, 0, None, order, delay_phasors)  # [T][Np][A]
        vxx = (np.abs(e[:, 0]) ** 2).sum(axis=0)       # [A]
        out[ci, 0] = np.tensordot(vxx, beam, axes=1)
        if n_pol == 2:
            vyy = (np.abs(e[:, 1]) ** 2).sum(axis=0)
            out[ci, 1] = np.tensordot(vyy, beam, axes=1)
            if n_products == 4:
                vxy = (e[:, 0] * np.conj(e[:, 1])).sum(axis=0)
                xy = np.tensordot(vxy, beam.astype(np.complex128), axes=1)
                out[ci, 2], out[ci, 3] = xy.real, xy.imag
                out[ci, 4], out[ci, 5] = xy.real, -xy.imag
    return out


# ------------------------------------------------------------------ sampled outputs at any size
def pixel_values(voltages: np.ndarray, kind: str, ant_uv: np.ndarray, taps: Optional[np.ndarray],
                 grid_n: int, pad: int, n_products: int, pixels, kernel_k: int = 1,
                 channels: Optional[list] = None, order: str = "TCPA",
                 delay_phasors: Optional[np.ndarray] = None) -> np.ndarray:
    """Accumulated image values at a few pixels, float64 [C'][planes][len(pixels)], straight from
    the discretised Eq. 5 one pixel at a time, with no grid and no FFT:

        A_p(t)[m][l] = sum_a E_ap(t) * sum_d W_a[d] exp(+2 pi i ((cx_a+dx) l + (cy_a+dy) m) / N)

    (cells modulo N, reading Q6), then the products summed over t.  Cost O(T * A) per pixel, so it
    checks sampled outputs of full-size configurations that epic_image() cannot finish in
    reasonable time.  ``pixels`` is a list of (m, l)."""
    n = grid_n * pad
    t_n, c_n = voltages.shape[:2]
    n_pol, n_ant = (voltages.shape[3], voltages.shape[2]) if order == "TCAP" else voltages.shape[2:4]
    ch = list(range(c_n)) if channels is None else list(channels)
    pl = n_planes(n_pol, n_products)
    out = np.zeros((len(ch), pl, len(pixels)), dtype=np.float64)
    for ci, c in enumerate(ch):
        uv_c, taps_c = channel_layout(ant_uv, taps, c)
        cells = tap_cells(uv_c, kernel_k, n)            # [A][K][K] flat y*N + x
        w = taps_to_complex(taps_c, n_ant, kernel_k)    # [A][K][K]
        cy, cx = cells // n, cells % n
        e = channel_voltages(voltages, kind, c, 0, None, order, delay_phasors)   # [T][Np][A]
        for pi, (m, l) in enumerate(pixels):
            phase = np.exp(1j * TWO_PI * ((cx * l + cy * m) % n) / n)
            u = (w * phase).sum(axis=(1, 2))            # [A]: response of antenna a at this pixel
            a = e @ u                                        # [T][Np]
            out[ci, 0, pi] = (np.abs(a[:, 0]) ** 2).sum()
            if n_pol == 2:
                out[ci, 1, pi] = (np.abs(a[:, 1]) ** 2).sum()
                if n_products == 4:
                    xy = (a[:, 0] * np.conj(a[:, 1])).sum()
                    out[ci, 2, pi], out[ci, 3, pi] = xy.real, xy.imag
                    out[ci, 4, pi], out[ci, 5, pi] = xy.real, -xy.imag
    return out

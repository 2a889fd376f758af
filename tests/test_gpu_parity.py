"""GPU parity tests (-m gpu): libepic.so through its C ABI against the float64 oracle, element by
element, on the same seeded inputs.  Bit-exact for S1 (unpack), S2 (cells) and integer-valued
gridding; <= 1e-4 of the image peak for accumulated images (BASELINE.json north_star)."""
import numpy as np
import pytest

from oracle import epic_oracle as orc
from workloads import make_config, make_custom, make_lwa55, make_per_channel

from epic_testlib import TOL, assert_parity, max_rel_err, run_gpu, run_oracle

pytestmark = pytest.mark.gpu


def _epic():
    import paper_1904_11422_b200 as epic
    return epic


# ------------------------------------------------------------------ S1
def test_s1_unpack_bit_exact_all_bytes_and_random():
    import torch
    epic = _epic()
    rng = np.random.default_rng(5)
    b = np.concatenate([np.arange(256, dtype=np.uint8), rng.integers(0, 256, 100003, dtype=np.uint8)])
    d = torch.from_numpy(b).cuda()
    out = torch.empty((b.size, 2), dtype=torch.float32, device="cuda")
    epic.epic_debug_unpack(d, b.size, out)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    ref = orc.unpack_ci4(b)
    assert np.array_equal(got[:, 0], ref.real.astype(np.float32))
    assert np.array_equal(got[:, 1], ref.imag.astype(np.float32))


# ------------------------------------------------------------------ S2
@pytest.mark.parametrize("wl", [
    make_config(1), make_config(2, n_chan=1, n_t=1), make_config(3, n_chan=1, n_t=1),
    make_config(4, n_chan=1, n_t=1), make_config(5, n_chan=1, n_t=1),
    make_custom(grid_n=8, pad=2, n_ant=40, n_pol=1, kernel_k=5, n_chan=1, n_t=1, layout="wrap"),
], ids=lambda w: w.name)
def test_s2_cells_bit_exact(wl):
    epic = _epic()
    with epic.Plan(wl.grid_n, wl.pad, wl.ant_uv, wl.taps, wl.kernel_k) as plan:
        got = plan.cells()
        y0, x0, R, Cc = plan.support()
    ref = orc.tap_cells(wl.ant_uv, wl.kernel_k, wl.N)
    assert np.array_equal(got.astype(np.int64), ref)
    # the support box covers every occupied row and column
    ys, xs = np.unique(ref // wl.N), np.unique(ref % wl.N)
    assert np.all((ys - y0) % wl.N < R) and np.all((xs - x0) % wl.N < Cc)


def test_s2_half_cells_round_up_and_wrap():
    epic = _epic()
    uv = np.array([[2.5, 2.49], [-0.5, -0.51], [7.6, 0.0], [15.5, 16.0]], dtype=np.float32)
    with epic.Plan(8, 2, uv) as plan:
        got = plan.cells().reshape(-1)
    assert got.tolist() == [2 * 16 + 3, 15 * 16 + 0, 0 * 16 + 8, 0 * 16 + 0]


# ------------------------------------------------------------------ S3
@pytest.mark.parametrize("idx", [1, 2, 3, 5])
def test_s3_gridding_one_frame(idx):
    import torch
    epic = _epic()
    wl = make_config(idx, n_chan=1, n_t=1)
    v = wl.voltages()
    e = orc.voltages_to_complex(v[0, 0], wl.input_kind)  # [Np][A]
    cells = orc.tap_cells(wl.ant_uv, wl.kernel_k, wl.N)
    w = orc.taps_to_complex(wl.taps, wl.n_ant, wl.kernel_k)
    ref = orc.grid_frames(e, cells, w, wl.N)  # [Np][N][N]
    with epic.Plan(wl.grid_n, wl.pad, wl.ant_uv, wl.taps, wl.kernel_k) as plan:
        out = torch.full((wl.n_pol, wl.N, wl.N, 2), 7.0, dtype=torch.float32, device="cuda")
        plan.debug_grid(torch.from_numpy(v).cuda(), wl.input_kind == "cf32", wl.n_pol, out)
        torch.cuda.synchronize()
        got = out.cpu().numpy()
    gc = got[..., 0].astype(np.float64) + 1j * got[..., 1]
    if wl.kernel_k == 1 and wl.input_kind == "ci4":
        assert np.array_equal(gc, ref)  # small integers: exact in any order
    else:
        assert np.abs(gc - ref).max() <= 2e-6 * max(1.0, np.abs(ref).max())


# ------------------------------------------------------------------ whole path, small sizes
def test_c1_exact_config_against_definition_oracle():
    wl = make_config(1)
    gpu, info = run_gpu(wl, return_plan_info=True)
    ref = run_oracle(wl, mode="definition")
    assert_parity(gpu, ref, what=wl.name)
    assert info["launches"] > 0


SMALL = [
    make_config(1, n_chan=3, n_t=21),
    make_config(2, n_chan=3, n_t=37),
    make_config(3, n_chan=2, n_t=29),
    make_config(4, n_chan=2, n_t=5),
    make_config(5, n_chan=1, n_t=2),
    make_config(5, n_chan=2, n_t=3, n_ant=256),
    make_custom(grid_n=4, pad=2, n_ant=5, n_pol=1, kernel_k=1, n_chan=2, n_t=3, input_kind="cf32"),
    make_custom(grid_n=8, pad=2, n_ant=40, n_pol=2, kernel_k=5, n_chan=2, n_t=4, layout="wrap"),
    make_custom(grid_n=32, pad=2, n_ant=77, n_pol=2, kernel_k=3, n_chan=5, n_t=9, n_products=2),
    make_custom(grid_n=16, pad=4, n_ant=33, n_pol=1, kernel_k=7, n_chan=1, n_t=11, layout="disc"),
    make_custom(grid_n=64, pad=2, n_ant=300, n_pol=2, kernel_k=3, n_chan=1, n_t=6, layout="wrap",
                input_kind="cf32"),
    make_custom(grid_n=128, pad=1, n_ant=64, n_pol=1, kernel_k=1, n_chan=2, n_t=2, layout="uniform"),
    make_custom(grid_n=64, pad=2, n_ant=1, n_pol=2, kernel_k=1, n_chan=1, n_t=1),
]


@pytest.mark.parametrize("wl", SMALL, ids=lambda w: f"{w.name}-c{w.n_chan}-t{w.n_t}")
def test_whole_path_small(wl):
    gpu = run_gpu(wl)
    ref = run_oracle(wl)
    assert_parity(gpu, ref, what=wl.name)
    if wl.n_products == 4:  # YX = conj(XY); XX, YY >= 0
        peak = np.abs(gpu[:, :2]).max()
        assert np.abs(gpu[:, 4] - gpu[:, 2]).max() <= 1e-6 * peak
        assert np.abs(gpu[:, 5] + gpu[:, 3]).max() <= 1e-6 * peak
    assert (gpu[:, :min(2, gpu.shape[1])] >= 0).all()


# ------------------------------------------------------------------ both kernel families
# Plans whose occupied cells fit the fused kernel's 32 x 32 block: the fused (one-kernel) and the
# two-pass path must each match the oracle; AUTO must pick the fused one.
FUSED_CAPABLE = [
    make_config(2, n_chan=3, n_t=37),                      # delta, XX+YY, ragged last batch
    make_config(2, n_chan=150, n_t=9),                     # more units than CTAs can split evenly
    make_config(3, n_chan=2, n_t=29),                      # 3x3 taps, four products
    make_custom(grid_n=32, pad=2, n_ant=76, n_pol=2, kernel_k=3, n_chan=5, n_t=9, n_products=2,
                layout="disc"),                            # N = 64 (Q = 2)
    make_custom(grid_n=64, pad=2, n_ant=64, n_pol=1, kernel_k=1, n_chan=2, n_t=11, layout="disc"),  # 1 pol, odd n_t
    make_custom(grid_n=32, pad=2, n_ant=40, n_pol=1, kernel_k=3, n_chan=3, n_t=16, layout="disc"),
    make_custom(grid_n=64, pad=2, n_ant=512, n_pol=2, kernel_k=1, n_chan=2, n_t=5, layout="disc"),  # 2 prefetch slots
    make_custom(grid_n=32, pad=4, n_ant=100, n_pol=2, kernel_k=5, n_chan=2, n_t=7, layout="disc", n_products=4),
    make_custom(grid_n=64, pad=2, n_ant=256, n_pol=2, kernel_k=5, n_chan=2, n_t=6, layout="disc", n_products=2,
                seed=21),                                  # 6400 gather entries: too many to stage in shared memory
    # N = 32 (Q = 1: one residue per axis, 64-thread CTAs): C1's shape with 4+4-bit voltages, and the other product counts
    make_custom(grid_n=16, pad=2, n_ant=16, n_pol=1, kernel_k=1, n_chan=3, n_t=21, layout="integer"),
    make_custom(grid_n=32, pad=1, n_ant=90, n_pol=2, kernel_k=3, n_chan=2, n_t=13, layout="uniform", n_products=4),
    make_custom(grid_n=8, pad=4, n_ant=30, n_pol=2, kernel_k=5, n_chan=40, n_t=50, layout="wrap", n_products=2),  # wraps; split units
]


@pytest.mark.parametrize("path", [1, 2], ids=["twopass", "fused"])
@pytest.mark.parametrize("wl", FUSED_CAPABLE, ids=lambda w: f"{w.name}-c{w.n_chan}-t{w.n_t}")
def test_fused_capable_plans_both_paths(wl, path):
    epic = _epic()
    gpu, info = run_gpu(wl, path=path, return_plan_info=True)
    assert info["path"] == path
    ref = run_oracle(wl)
    assert_parity(gpu, ref, what=f"{wl.name} path={path}")
    if path == 2:
        assert info["launches"] == 2  # the fused kernel + the fix-up of units split between CTAs
        with epic.Plan(wl.grid_n, wl.pad, wl.ant_uv, wl.taps, wl.kernel_k) as plan:
            plan.set_products(wl.n_products)
            assert plan.path(wl.n_pol) == epic.EPIC_PATH_FUSED  # AUTO picks it


# ------------------------------------------------------------------ wide fused kernel: supports up to 64 x 64 (N = 64, 128)
def _wrapped_uv(side_y, side_x, n_ant, N, seed):
    """antennas filling a side_y x side_x box whose origin is near the plane's far corner, so the box wraps"""
    rng = np.random.default_rng(seed)
    return (np.array([N - 9.0, N - 21.0]) + rng.uniform(0, 1, (n_ant, 2)) * np.array([side_x - 1.0, side_y - 1.0])).astype(np.float32)


WIDE_CAPABLE = [
    make_lwa55(n_chan=3, n_t=21),                                     # the paper's operating point: ~43 x 39 cells, 3 m top-hat, 4 products
    make_lwa55(n_chan=2, n_t=9, kernel="delta", n_products=2),        # delta kernel
    make_lwa55(n_chan=150, n_t=5, kernel="delta", n_products=2),      # more units than CTAs can split evenly
    make_custom(grid_n=64, pad=2, n_ant=256, n_pol=2, kernel_k=1, n_chan=2, n_t=7,
                ant_uv=np.random.default_rng(11).uniform(-0.49, 63.49, (256, 2))),   # fills 64 x 64 cells
    make_custom(grid_n=64, pad=1, n_ant=200, n_pol=2, kernel_k=1, n_chan=3, n_t=6, n_products=2,
                ant_uv=np.random.default_rng(12).uniform(-0.49, 63.49, (200, 2))),   # N = 64: no padding at all
    make_custom(grid_n=64, pad=1, n_ant=60, n_pol=1, kernel_k=3, n_chan=2, n_t=11, ant_uv=_wrapped_uv(40, 50, 60, 64, 1)),  # N = 64, 1 pol, odd n_t, wraps
    make_custom(grid_n=64, pad=2, n_ant=120, n_pol=2, kernel_k=3, n_chan=2, n_t=5, ant_uv=_wrapped_uv(60, 20, 120, 128, 2)),  # tall, narrow (x fits 32), wraps
    make_custom(grid_n=64, pad=2, n_ant=120, n_pol=2, kernel_k=5, n_chan=2, n_t=5, ant_uv=_wrapped_uv(20, 58, 120, 128, 3), n_products=2),  # flat, wide: x-fold only
    make_custom(grid_n=64, pad=2, n_ant=77, n_pol=2, kernel_k=3, n_chan=3, n_t=9, ant_uv=_wrapped_uv(45, 45, 77, 128, 4)),  # 77 antennas: byte-fetched tail group
    make_custom(grid_n=64, pad=2, n_ant=90, n_pol=1, kernel_k=1, n_chan=2, n_t=8, ant_uv=_wrapped_uv(48, 33, 90, 128, 5)),  # rows exactly 48
]


@pytest.mark.parametrize("path", [1, 2], ids=["twopass", "fused-wide"])
@pytest.mark.parametrize("wl", WIDE_CAPABLE, ids=lambda w: f"{w.name}-c{w.n_chan}-t{w.n_t}")
def test_wide_support_plans_both_paths(wl, path):
    """Plans whose occupied cells need more than 32 x 32 but fit 64 x 64: EPIC_PATH_FUSED runs the wide kernel
    (AUTO picks it), and it and the two-pass path each match the oracle."""
    epic = _epic()
    v = wl.voltages()
    gpu, info = run_gpu(wl, volt=v, path=path, calls=2, return_plan_info=True)
    assert info["path"] == path
    _, _, R, Cc = info["support"]
    assert max(R, Cc) > 32 and max(R, Cc) <= 64
    ref = run_oracle(wl, volt=v)
    assert_parity(gpu, ref, what=f"{wl.name} path={path}")
    if path == 2:
        assert info["launches"] == 2
        with epic.Plan(wl.grid_n, wl.pad, wl.ant_uv, wl.taps, wl.kernel_k) as plan:
            plan.set_products(wl.n_products)
            assert plan.path(wl.n_pol) == epic.EPIC_PATH_FUSED
            with pytest.raises(epic.EpicError):
                plan.set_path(epic.EPIC_PATH_TENSOR)   # the tensor-core variant is the 32 x 32 kernel's


@pytest.mark.parametrize("kernel,n_products,channels", [("tophat", 4, [3, 90]), ("delta", 2, [0, 64, 127])], ids=["tophat", "delta"])
def test_wide_full_size_sampled_channels(kernel, n_products, channels):
    """The paper's operating point at C2's extent (128 channels x 1000 samples), in the launch configuration
    `bench.py --workload lwa55-*` and the default run's other_configs time (one call, AUTO = the wide fused kernel);
    whole channels against the oracle, properties for the rest."""
    wl = make_lwa55(n_chan=128, n_t=1000, kernel=kernel, n_products=n_products)
    v = wl.voltages()
    gpu, info = run_gpu(wl, volt=v, return_plan_info=True)
    assert info["path"] == 2 and info["launches"] == 2 and max(info["support"][2:]) > 32
    ref = run_oracle(wl, volt=v, channels=channels)
    assert_parity(gpu[channels], ref, what=f"{wl.name} channels {channels}")
    assert np.isfinite(gpu).all() and (gpu[:, :2] >= 0).all()
    totals = gpu[:, 0].sum(axis=(1, 2))
    assert totals.min() > 0.5 * totals.max()


@pytest.mark.parametrize("mode", ["native", "phasors", "both"])
def test_wide_input_order_and_delay_phasors(mode):
    wl = make_lwa55(n_chan=2, n_t=7)
    v = wl.voltages()
    native = mode in ("native", "both")
    rng = np.random.default_rng(9)
    ph = None
    if mode in ("phasors", "both"):
        ph = (np.exp(2j * np.pi * rng.random((wl.n_chan, wl.n_pol, wl.n_ant))) * rng.uniform(0.8, 1.25, (wl.n_chan, wl.n_pol, wl.n_ant))).astype(np.complex64)
    vin = np.ascontiguousarray(np.swapaxes(v, 2, 3)) if native else v
    gpu = run_gpu(wl, volt=vin, path=2, native=native, phasors=ph, autocorr=True)
    kw = dict(order="TCAP" if native else "TCPA", delay_phasors=ph)
    ref = orc.epic_image(vin, wl.input_kind, wl.ant_uv, wl.taps, wl.grid_n, wl.pad, wl.n_products, kernel_k=wl.kernel_k, **kw)
    ref = ref - orc.autocorr_image(vin, wl.input_kind, wl.ant_uv, wl.taps, wl.grid_n, wl.pad, wl.n_products, kernel_k=wl.kernel_k, **kw)
    assert_parity(gpu, ref, what=f"wide {mode}")


def test_wide_per_channel_layouts():
    """One layout per channel over a band wide enough that the box grows past 32 cells: wide kernel, per-channel tables."""
    epic = _epic()
    wl = make_per_channel(grid_n=64, pad=2, n_ant=96, n_pol=2, kernel_k=3, n_chan=6, n_t=13, f0_hz=50e6, df_hz=3e6,
                          diameter_m=105.0, n_sources=1)
    v = wl.voltages()
    gpu, info = run_gpu(wl, volt=v, path=2, calls=2, return_plan_info=True)
    assert info["path"] == 2 and max(info["support"][2:]) > 32
    assert_parity(gpu, run_oracle(wl, volt=v), what=wl.name)


@pytest.mark.parametrize("n_ant", [77, 254, 3])
def test_antenna_counts_not_a_multiple_of_four_stay_on_the_fast_paths(n_ant):
    """n_ant % 4 != 0: voltage rows are not word-aligned; the fused kernels fetch them as bytes instead of
    falling to the two-pass path, in both input orders and with one polarisation."""
    epic = _epic()
    for n_pol, native in [(2, False), (2, True), (1, False)]:
        wl = make_custom(grid_n=64, pad=2, n_ant=n_ant, n_pol=n_pol, kernel_k=3, n_chan=3, n_t=10, layout="disc", seed=n_ant)
        v = wl.voltages()
        vin = np.ascontiguousarray(np.swapaxes(v, 2, 3)) if native else v
        gpu, info = run_gpu(wl, volt=vin, native=native, return_plan_info=True)
        assert info["path"] == epic.EPIC_PATH_FUSED
        ref = orc.epic_image(vin, wl.input_kind, wl.ant_uv, wl.taps, wl.grid_n, wl.pad, wl.n_products, kernel_k=wl.kernel_k,
                             order="TCAP" if native else "TCPA")
        assert_parity(gpu, ref, what=f"{n_ant} antennas n_pol={n_pol} native={native}")
    wl = make_custom(grid_n=128, pad=2, n_ant=n_ant, n_pol=2, kernel_k=3, n_chan=2, n_t=6, layout="uniform", seed=n_ant)
    gpu, info = run_gpu(wl, return_plan_info=True)        # large grid: the streamed kernel fetches bytes anyway
    assert info["path"] == epic.EPIC_PATH_STREAM
    assert_parity(gpu, run_oracle(wl), what=f"{n_ant} antennas, N = 256")


# Large planes (N = 256, 512): the tiled (packed, L2-resident two-pass) path and the general
# two-pass path must each match the oracle; AUTO must pick the tiled one.
TILED_CAPABLE = [
    make_config(4, n_chan=2, n_t=5),                                  # N = 256, prefold of 2 rows/cols
    make_config(5, n_chan=1, n_t=3),                                  # N = 512, wrap-around box, 5x5 taps
    make_config(5, n_chan=2, n_t=3, n_ant=256),
    make_custom(grid_n=128, pad=2, n_ant=64, n_pol=2, kernel_k=1, n_chan=3, n_t=4, layout="disc",
                n_products=2),                                        # small support: no prefold, zero rows
    make_custom(grid_n=256, pad=1, n_ant=200, n_pol=2, kernel_k=3, n_chan=1, n_t=3, layout="uniform"),  # R = N
    make_custom(grid_n=128, pad=2, n_ant=100, n_pol=1, kernel_k=3, n_chan=2, n_t=7, layout="uniform"),  # 1 pol, odd n_t
    make_custom(grid_n=128, pad=4, n_ant=300, n_pol=2, kernel_k=1, n_chan=1, n_t=2, layout="wrap"),     # N = 512, delta
    make_custom(grid_n=256, pad=2, n_ant=40, n_pol=1, kernel_k=1, n_chan=1, n_t=4, layout="uniform"),
]


@pytest.mark.parametrize("path", [1, 3, 5], ids=["twopass", "tiled", "stream"])
@pytest.mark.parametrize("wl", TILED_CAPABLE, ids=lambda w: f"{w.name}-c{w.n_chan}-t{w.n_t}")
def test_tiled_capable_plans_both_paths(wl, path):
    epic = _epic()
    if path == 5 and wl.N == 512 and wl.n_ant == 300:
        # a box as tall as the plane: one channel's row and column CTAs cannot be co-resident, and forcing the
        # streamed kernel is refused, not silently rerouted
        with pytest.raises(epic.EpicError):
            run_gpu(wl, path=5)
        return
    gpu, info = run_gpu(wl, path=path, return_plan_info=True)
    assert info["path"] == path
    ref = run_oracle(wl)
    assert_parity(gpu, ref, what=f"{wl.name} path={path}")
    if path == 5:
        assert info["launches"] == 1  # one persistent kernel for the whole call
    if path == 3:
        with epic.Plan(wl.grid_n, wl.pad, wl.ant_uv, wl.taps, wl.kernel_k) as plan:
            plan.set_products(wl.n_products)
            assert plan.path(wl.n_pol) == epic.EPIC_PATH_TILED  # AUTO picks it


@pytest.mark.parametrize("wl,ring_mib", [
    (make_config(4, n_chan=21, n_t=40), 0),      # more channels than one wave holds: several waves, ring reused across them
    (make_config(4, n_chan=3, n_t=70), 4),       # ring of 2 frames per channel: every hand-over waits on the consumers
    (make_config(5, n_chan=5, n_t=6), 0),        # N = 512: waves of 2 channels, the last one half empty
    (make_config(5, n_chan=2, n_t=7), 9),        # N = 512 with the smallest ring
    (make_custom(grid_n=128, pad=2, n_ant=100, n_pol=1, kernel_k=3, n_chan=4, n_t=33, layout="uniform"), 0),  # 1 pol, odd n_t
], ids=["C4-waves", "C4-ring2", "C5-waves", "C5-ring2", "1pol"])
def test_stream_path_waves_and_ring_reuse(wl, ring_mib):
    """EPIC_PATH_STREAM's hand-over machinery: channel waves, a ring much shorter than the call, two
    calls accumulating; sampled channels against the oracle and the rest against the batched tiled path."""
    v = wl.voltages()
    kw = dict(scratch_limit=ring_mib << 20) if ring_mib else {}
    gpu, info = run_gpu(wl, volt=v, path=5, calls=2, return_plan_info=True, **kw)
    assert info["path"] == 5 and info["launches"] == 1
    channels = sorted({0, wl.n_chan // 2, wl.n_chan - 1})
    ref = run_oracle(wl, volt=v, channels=channels)
    assert_parity(gpu[channels], ref, what=f"{wl.name} stream")
    tiled = run_gpu(wl, volt=v, path=3, calls=2)
    assert max_rel_err(gpu, tiled.astype(np.float64)) <= 1e-5


def test_tiled_many_batches_accumulate():
    """More frames than one scratch batch holds, several channels: exercises the batch loop and
    the one-add-per-batch accumulation of the column kernel."""
    wl = make_config(4, n_chan=5, n_t=70)
    gpu, info = run_gpu(wl, path=3, return_plan_info=True, scratch_limit=16 << 20)  # 31 frames per batch
    assert info["launches"] >= 8
    ref = run_oracle(wl, channels=[0, 4])
    assert_parity(gpu[[0, 4]], ref, what="C4 5ch x 70")


def test_fused_delta_gridding_is_exact_for_integer_voltages():
    """Delta kernel + 4-bit integers: every gridded value is a small integer, so a one-antenna-
    per-pixel check through the whole fused path is exact: a single antenna gives a flat image
    |E|^2 summed over time, in every pixel, with no rounding at all."""
    wl = make_custom(grid_n=64, pad=2, n_ant=4, n_pol=2, kernel_k=1, n_chan=2, n_t=13, n_products=2,
                     ant_uv=np.array([[5, 7], [5, 7], [5, 7], [5, 7]], dtype=np.float32))
    v = wl.voltages()
    gpu = run_gpu(wl, volt=v, path=2)
    e = orc.unpack_ci4(v).sum(axis=-1)                      # the four antennas share one cell
    flat = (np.abs(e) ** 2).sum(axis=0)                     # [C][Np]
    for c in range(wl.n_chan):
        for p in range(2):
            assert np.all(gpu[c, p] == np.float32(flat[c, p]))


# ------------------------------------------------------------------ full size, sampled outputs
@pytest.mark.parametrize("idx,channels", [(2, [0, 77, 127]), (3, [5, 126])], ids=["C2-full", "C3-full"])
def test_full_size_config_sampled_channels(idx, channels):
    """BASELINE.json's C2 / C3 at full extent, in the launch configuration bench.py times (one
    epic_image call over all channels and samples, AUTO path = fused); the oracle recomputes
    whole channels picked across the range (channels are independent)."""
    wl = make_config(idx)
    v = wl.voltages()
    gpu, info = run_gpu(wl, volt=v, return_plan_info=True)
    assert info["path"] == 2 and info["launches"] == 2
    ref = run_oracle(wl, volt=v, channels=channels)
    assert_parity(gpu[channels], ref, what=f"{wl.name} channels {channels}")
    # properties that hold for every channel at any size
    assert np.isfinite(gpu).all() and (gpu[:, :2] >= 0).all()
    totals = gpu[:, 0].sum(axis=(1, 2))
    assert totals.min() > 0.5 * totals.max()  # every channel was imaged (same noise statistics)


@pytest.mark.parametrize("path", [3, 5], ids=["tiled", "stream"])
@pytest.mark.parametrize("idx", [4, 5], ids=["C4-full", "C5-full"])
def test_full_size_large_configs_sampled_pixels(idx, path):
    """C4 / C5 at full extent through the two large-grid paths bench.py times (AUTO = tiled; streamed kernel): the
    float64 oracle cannot image 256^2 / 512^2 planes x 10^4..10^5 frames in reasonable time, so
    sampled pixels of sampled channels are computed one by one from Eq. 5 (oracle.pixel_values),
    every plane, plus properties of the whole result."""
    wl = make_config(idx)
    v = wl.voltages()
    gpu, info = run_gpu(wl, volt=v, return_plan_info=True, path=None if path == 3 else path)
    assert info["path"] == path and (path == 3 or info["launches"] == 1)
    rng = np.random.default_rng(40 + idx)
    channels = [0, wl.n_chan // 2 + 1, wl.n_chan - 1]
    N = wl.N
    # zenith (the peak of a noise image: every |What_a|^2 is largest there), the sources, the plane's corners and
    # centre, one pixel in every 4-column strip at a random row (both residues and every strip / team boundary of
    # the column kernels), one in every 4-row group at a random column, and random pixels
    pix = [(0, 0), (N // 2, N // 2), (N - 1, 3), (N - 1, N - 1), (0, N - 1), (N // 2 - 1, N // 2), (N // 2, N // 2 - 1)]
    pix += [(s["m_pix"], s["l_pix"]) for s in wl.sources]
    pix += [(int(rng.integers(0, N)), l0 + int(rng.integers(0, 4))) for l0 in range(0, N, 4)]
    pix += [(m0 + int(rng.integers(0, 4)), int(rng.integers(0, N))) for m0 in range(0, N, 4)]
    pix += [tuple(int(x) for x in rng.integers(0, N, 2)) for _ in range(32)]
    assert len(pix) >= 64
    ref = orc.pixel_values(v, wl.input_kind, wl.ant_uv, wl.taps, wl.grid_n, wl.pad, wl.n_products, pix,
                           kernel_k=wl.kernel_k, channels=channels)
    got = np.stack([gpu[channels][:, :, m, l] for (m, l) in pix], axis=-1).astype(np.float64)
    for ci in range(len(channels)):
        # normalised by the ORACLE's brightest sampled pixel (zenith and the sources are among them); the true
        # image peak can only be larger, so this is never looser than the 1e-4-of-peak bar
        peak = float(np.abs(ref[ci]).max())
        assert np.abs(got[ci] - ref[ci]).max() <= TOL * peak, (wl.name, channels[ci])
        assert float(gpu[channels[ci]].max()) <= 1.5 * peak  # and nothing on the GPU side towers over it
    assert np.isfinite(gpu).all() and (gpu[:, :2] >= 0).all()
    peak = np.abs(gpu[:, :2]).max()
    assert np.abs(gpu[:, 4] - gpu[:, 2]).max() <= 1e-6 * peak and np.abs(gpu[:, 5] + gpu[:, 3]).max() <= 1e-6 * peak
    totals = gpu[:, 0].sum(axis=(1, 2))
    assert totals.min() > 0.5 * totals.max()


# ------------------------------------------------------------------ optional autocorrelation removal
@pytest.mark.parametrize("wl,calls", [
    (make_config(2, n_chan=3, n_t=37), 1),                  # fused, delta: flat zero-spacing term
    (make_config(3, n_chan=2, n_t=29), 2),                  # fused, 3x3 taps, four products, two gulps
    (make_config(4, n_chan=2, n_t=5), 1),                   # tiled, 256^2
    (make_custom(grid_n=32, pad=2, n_ant=40, n_pol=1, kernel_k=5, n_chan=2, n_t=11, layout="disc"), 1),
    (make_custom(grid_n=8, pad=2, n_ant=24, n_pol=2, kernel_k=3, n_chan=1, n_t=6, layout="wrap"), 1),  # two-pass
], ids=lambda v: v.name if hasattr(v, "name") else str(v))
def test_autocorr_removal_matches_oracle(wl, calls):
    """epic_image followed by epic_autocorr_remove equals the oracle's image minus its a = b part
    (PAPER.md:130), within the image tolerance normalised by the peak of what is LEFT."""
    v = wl.voltages()
    gpu = run_gpu(wl, volt=v, calls=calls, autocorr=True)
    ref = run_oracle(wl, volt=v) - orc.autocorr_image(v, wl.input_kind, wl.ant_uv, wl.taps, wl.grid_n, wl.pad,
                                                      wl.n_products, kernel_k=wl.kernel_k)
    assert_parity(gpu, ref, what=f"{wl.name} autocorr removed")


# ------------------------------------------------------------------ upstream steps folded into the load
UPSTREAM = [
    (make_config(2, n_chan=3, n_t=21), None),                                     # fused, delta
    (make_config(3, n_chan=2, n_t=13), None),                                     # fused, taps, TMEM variant
    (make_config(4, n_chan=2, n_t=4), None),                                      # large grid, batched tiled kernels
    (make_config(4, n_chan=2, n_t=4), 5),                                         # large grid, streamed kernel
    (make_custom(grid_n=32, pad=2, n_ant=40, n_pol=1, kernel_k=3, n_chan=3, n_t=9, layout="disc"), None),
    (make_custom(grid_n=8, pad=2, n_ant=30, n_pol=2, kernel_k=3, n_chan=2, n_t=5, layout="wrap"), None),  # two-pass
    (make_custom(grid_n=16, pad=2, n_ant=9, n_pol=2, kernel_k=1, n_chan=2, n_t=3, input_kind="cf32"), None),
    (make_config(2, n_chan=2, n_t=8), 1),                                         # fused plan forced two-pass
]


@pytest.mark.parametrize("wl,path", UPSTREAM, ids=lambda v: v.name if hasattr(v, "name") else str(v))
@pytest.mark.parametrize("mode", ["native", "phasors", "both"])
def test_input_order_and_delay_phasors(wl, path, mode):
    """[T][C][A][Np] input order and per-(channel, pol, antenna) delay phasors
     through every kernel family, against the oracle with the same options; the
    autocorrelation removal honours both."""
    v = wl.voltages()
    native = mode in ("native", "both")
    rng = np.random.default_rng(5)
    ph = None
    if mode in ("phasors", "both"):
        ph = (np.exp(2j * np.pi * rng.random((wl.n_chan, wl.n_pol, wl.n_ant))) *
              rng.uniform(0.8, 1.25, (wl.n_chan, wl.n_pol, wl.n_ant))).astype(np.complex64)
    vin = np.ascontiguousarray(np.swapaxes(v, 2, 3)) if native else v
    kw = dict(order="TCAP" if native else "TCPA", delay_phasors=ph)
    gpu = run_gpu(wl, volt=vin, path=path, native=native, phasors=ph)
    ref = orc.epic_image(vin, wl.input_kind, wl.ant_uv, wl.taps, wl.grid_n, wl.pad, wl.n_products,
                         kernel_k=wl.kernel_k, **kw)
    assert_parity(gpu, ref, what=f"{wl.name} {mode}")
    if wl.input_kind == "ci4":
        gpu2 = run_gpu(wl, volt=vin, path=path, native=native, phasors=ph, autocorr=True)
        ref2 = ref - orc.autocorr_image(vin, wl.input_kind, wl.ant_uv, wl.taps, wl.grid_n, wl.pad, wl.n_products,
                                        kernel_k=wl.kernel_k, **kw)
        assert_parity(gpu2, ref2, what=f"{wl.name} {mode} autocorr removed")


def test_delay_phasor_shape_is_checked():
    epic = _epic()
    import torch
    wl = make_config(2, n_chan=2, n_t=4)
    with epic.Plan(wl.grid_n, wl.pad, wl.ant_uv) as plan:
        plan.set_products(2)
        plan.set_delay_phasors(np.ones((3, 2, 256), dtype=np.complex64))   # table for 3 channels
        out = torch.zeros((2, 2, 128, 128), dtype=torch.float32, device="cuda")
        dv = torch.from_numpy(wl.voltages()).cuda()
        with pytest.raises(epic.EpicError):
            plan.image(dv, 4, 2, 2, out)                                   # call with 2 channels
        plan.set_delay_phasors(None)
        plan.image(dv, 4, 2, 2, out)
        torch.cuda.synchronize()
        with pytest.raises(epic.EpicError):
            plan.set_input_order(7)


# ------------------------------------------------------------------ randomised plans, every path the plan allows
def _random_case(seed):
    rng = np.random.default_rng(1000 + seed)
    N = int(rng.choice([64, 128, 128, 256, 512]))
    pad = int(rng.choice([1, 2, 4]))
    grid_n = N // pad
    n_pol = int(rng.choice([1, 2, 2]))
    K = int(rng.choice([1, 3, 3, 5, 7]))
    layout = str(rng.choice(["disc", "uniform", "wrap", "tight"]))
    n_ant = 4 * int(rng.integers(1, 60))
    n_chan, n_t = int(rng.integers(1, 6)), int(rng.integers(1, 26 if N <= 256 else 7))
    n_products = 1 if n_pol == 1 else int(rng.choice([2, 4]))
    uv = None
    if layout == "tight":  # everything inside a box the fused kernel can take, at a random offset (may wrap)
        side = int(rng.integers(1, 33 - (K - 1)))
        off = rng.integers(-N, N, 2)
        uv = (off + rng.uniform(0, max(side - 1, 0.01), (n_ant, 2))).astype(np.float32)
    wl = make_custom(grid_n=grid_n, pad=pad, n_ant=n_ant, n_pol=n_pol, kernel_k=K, n_chan=n_chan, n_t=n_t,
                     n_products=n_products, layout="uniform" if uv is not None else layout, seed=seed, ant_uv=uv)
    return wl, rng


@pytest.mark.parametrize("seed", range(24))
def test_random_plans_all_paths(seed):
    """Random shapes, layouts (incl. boxes that wrap around the plane edge), kernel sizes, input order
    and delay phasors: every kernel family the plan supports against the oracle."""
    epic = _epic()
    wl, rng = _random_case(seed)
    v = wl.voltages()
    native = bool(rng.integers(0, 2))
    ph = None
    if rng.integers(0, 2):
        ph = np.exp(2j * np.pi * rng.random((wl.n_chan, wl.n_pol, wl.n_ant))).astype(np.complex64)
    vin = np.ascontiguousarray(np.swapaxes(v, 2, 3)) if native else v
    ref = orc.epic_image(vin, wl.input_kind, wl.ant_uv, wl.taps, wl.grid_n, wl.pad, wl.n_products,
                         kernel_k=wl.kernel_k, order="TCAP" if native else "TCPA", delay_phasors=ph)
    with epic.Plan(wl.grid_n, wl.pad, wl.ant_uv, wl.taps, wl.kernel_k) as plan:
        plan.set_products(wl.n_products)
        auto = plan.path(wl.n_pol)
    tried = []
    for path in sorted({1, auto} | ({5} if auto == 3 and wl.N == 256 else set())):
        gpu = run_gpu(wl, volt=vin, path=path, native=native, phasors=ph, calls=int(rng.integers(1, 3)))
        assert_parity(gpu, ref, what=f"seed {seed} {wl.name} path={path}")
        tried.append(path)
    assert 1 in tried


def test_calls_accumulate_into_out_accum():
    wl = make_config(2, n_chan=2, n_t=30)
    one = run_gpu(wl, calls=1)
    three = run_gpu(wl, calls=3)
    ref = run_oracle(wl)
    assert_parity(three, ref, what="3 calls")
    assert np.abs(one - three).max() <= 1e-5 * np.abs(one).max()


def test_empty_calls_are_noops_and_errors_are_reported():
    import torch
    epic = _epic()
    wl = make_config(2, n_chan=1, n_t=1)
    with epic.Plan(wl.grid_n, wl.pad, wl.ant_uv) as plan:
        out = torch.ones((1, 6, 128, 128), dtype=torch.float32, device="cuda")
        plan.image(0, 0, 1, 2, out)     # n_t == 0: nothing read, nothing written
        plan.image(0, 5, 0, 2, out)     # n_chan == 0
        torch.cuda.synchronize()
        assert float(out.min()) == 1.0 and float(out.max()) == 1.0
        with pytest.raises(epic.EpicError):
            plan.image(0, 1, 1, 3, out)  # n_pol out of range
        with pytest.raises(epic.EpicError):
            plan.image(0, 1, 1, 2, out)  # NULL voltages
        plan.set_products(1)
        with pytest.raises(epic.EpicError):
            plan.image(torch.zeros(1024, dtype=torch.uint8, device="cuda"), 1, 1, 2, out)  # 1 product needs n_pol == 1
        plan.set_products(2)
        # the binding checks what it marshals: placement, dtype, contiguity, size
        dv = torch.zeros((4, 1, 2, 256), dtype=torch.uint8, device="cuda")
        with pytest.raises(ValueError):
            plan.image(dv.cpu(), 4, 1, 2, out)                       # host tensor for a DEVICE pointer
        with pytest.raises(ValueError):
            plan.image(dv.float(), 4, 1, 2, out)                     # wrong dtype
        with pytest.raises(ValueError):
            plan.image(dv[:, :, :, ::2], 4, 1, 2, out)               # non-contiguous view
        with pytest.raises(ValueError):
            plan.image(dv, 5, 1, 2, out)                             # voltages too short for n_t = 5
        with pytest.raises(ValueError):
            plan.image(dv, 4, 1, 2, out[:, :1].contiguous())         # out_accum too small for two planes
        plan.image(dv, 4, 1, 2, out)
        torch.cuda.synchronize()
    for bad in [dict(grid_n=3, pad=2), dict(grid_n=512, pad=2), dict(grid_n=2, pad=2)]:
        with pytest.raises(epic.EpicError):
            epic.Plan(bad["grid_n"], bad["pad"], wl.ant_uv)
    with pytest.raises(epic.EpicError):
        epic.Plan(64, 2, wl.ant_uv, np.zeros((256, 2, 2, 2), np.float32), 2)  # even K


def test_point_source_peaks_at_predicted_pixel():
    """BASELINE.json check (c) on the CUDA path: C3's injected source is common to both
    polarisations while the noise is not, so it is the brightest pixel of the accumulated
    Re(XY) image (the oracle agrees: tests/test_oracle_pins.py pins the pixel rule)."""
    wl = make_config(3, n_chan=1, n_t=2500)
    gpu = run_gpu(wl)
    src = wl.sources[0]
    m, l = np.unravel_index(np.argmax(gpu[0, 2]), gpu[0, 2].shape)
    assert (m, l) == (src["m_pix"], src["l_pix"])


# ------------------------------------------------------------------ one antenna layout per channel (reading Q15)
PER_CHANNEL = [
    # (workload, paths): 1 two-pass, 2 fused, 3 tiled, 5 streamed; the last one is AUTO's choice
    (make_per_channel(grid_n=64, pad=2, n_ant=64, n_pol=2, kernel_k=1, n_chan=5, n_t=37, n_products=2,
                      f0_hz=30e6, df_hz=4e6, diameter_m=100.0), [1, 2]),
    (make_per_channel(grid_n=64, pad=2, n_ant=96, n_pol=2, kernel_k=3, n_chan=7, n_t=23, f0_hz=38e6, df_hz=2e6,
                      diameter_m=80.0, n_sources=1), [1, 2]),
    (make_per_channel(grid_n=32, pad=2, n_ant=48, n_pol=1, kernel_k=3, n_chan=4, n_t=30, f0_hz=20e6, df_hz=7e6,
                      diameter_m=90.0), [1, 2]),
    (make_per_channel(grid_n=128, pad=2, n_ant=200, n_pol=2, kernel_k=3, n_chan=3, n_t=9, f0_hz=40e6, df_hz=9e6,
                      diameter_m=300.0), [1, 5, 3]),
    (make_per_channel(grid_n=256, pad=2, n_ant=300, n_pol=2, kernel_k=1, n_chan=2, n_t=5, n_products=2,
                      f0_hz=50e6, df_hz=20e6, diameter_m=500.0), [1, 5, 3]),
    (make_per_channel(grid_n=12, pad=2, n_ant=20, n_pol=2, kernel_k=5, n_chan=3, n_t=6, f0_hz=30e6, df_hz=10e6,
                      diameter_m=30.0), [1]),   # N = 24 is not a power of two -> rejected below
]


@pytest.mark.parametrize("wl,paths", PER_CHANNEL[:5], ids=lambda v: v.name if hasattr(v, "name") else str(v))
def test_per_channel_layouts_all_paths(wl, paths):
    """epic_plan_create_per_channel: channel c is gridded with ITS cells and taps (cell = lambda_c / 2,
    PAPER.md:122; 3 m top-hat).  Every kernel family against the oracle, and AUTO
    picks the fast one."""
    epic = _epic()
    assert wl.ant_uv.ndim == 3
    with epic.Plan(wl.grid_n, wl.pad, wl.ant_uv, wl.taps, wl.kernel_k) as plan:
        assert plan.n_layouts == wl.n_chan
        plan.set_products(wl.n_products)
        assert plan.path(wl.n_pol) == paths[-1]
        cells = plan.cells()
    assert np.array_equal(cells.astype(np.int64),
                          np.stack([orc.tap_cells(wl.ant_uv[c], wl.kernel_k, wl.N) for c in range(wl.n_chan)]))
    assert len({cells[c].tobytes() for c in range(wl.n_chan)}) == wl.n_chan   # the layouts do differ
    v = wl.voltages()
    ref = run_oracle(wl, volt=v)
    for path in paths:
        gpu = run_gpu(wl, volt=v, path=path, calls=2)
        assert_parity(gpu, ref, what=f"{wl.name} path {path}")


def test_per_channel_gridding_one_frame_per_layout():
    import torch
    epic = _epic()
    wl = PER_CHANNEL[1][0]
    v = wl.voltages()
    with epic.Plan(wl.grid_n, wl.pad, wl.ant_uv, wl.taps, wl.kernel_k) as plan:
        for c in range(wl.n_chan):
            e = orc.voltages_to_complex(v[0, c], wl.input_kind)  # [Np][A]
            ref = orc.grid_frames(e, orc.tap_cells(wl.ant_uv[c], 3, wl.N), orc.taps_to_complex(wl.taps[c], wl.n_ant, 3), wl.N)
            out = torch.full((wl.n_pol, wl.N, wl.N, 2), 7.0, dtype=torch.float32, device="cuda")
            plan.debug_grid(torch.from_numpy(np.ascontiguousarray(v[0, c])).cuda(), False, wl.n_pol, out, layout=c)
            torch.cuda.synchronize()
            got = out.cpu().numpy()
            gc = got[..., 0].astype(np.float64) + 1j * got[..., 1]
            assert np.abs(gc - ref).max() <= 2e-6 * max(1.0, np.abs(ref).max())


def test_per_channel_plan_checks_its_arguments():
    import torch
    epic = _epic()
    wl = PER_CHANNEL[0][0]
    with epic.Plan(wl.grid_n, wl.pad, wl.ant_uv, wl.taps, wl.kernel_k) as plan:
        plan.set_products(2)
        out = torch.zeros((wl.n_chan, 2, wl.N, wl.N), dtype=torch.float32, device="cuda")
        dv = torch.from_numpy(wl.voltages()).cuda()
        with pytest.raises(epic.EpicError) as ei:       # channel c uses layout c: n_chan must match
            plan.image(dv, 3, wl.n_chan - 1, wl.n_pol, out)
        assert ei.value.status == epic.EPIC_ERR_ARG
        with pytest.raises(epic.EpicError):
            plan.debug_grid(dv, False, wl.n_pol, out, layout=wl.n_chan)
        plan.image(dv, 0, wl.n_chan, wl.n_pol, out)     # empty call is still a no-op
        assert float(out.abs().max()) == 0.0
    bad = PER_CHANNEL[5][0]
    with pytest.raises(epic.EpicError):
        epic.Plan(bad.grid_n, bad.pad, bad.ant_uv, bad.taps, bad.kernel_k)


@pytest.mark.parametrize("wl", [PER_CHANNEL[1][0], PER_CHANNEL[3][0]], ids=lambda w: w.name)
def test_per_channel_autocorr_removal(wl):
    v = wl.voltages()
    gpu = run_gpu(wl, volt=v, autocorr=True)
    ref = run_oracle(wl, volt=v) - orc.autocorr_image(v, wl.input_kind, wl.ant_uv, wl.taps, wl.grid_n, wl.pad,
                                                      wl.n_products, kernel_k=wl.kernel_k)
    assert_parity(gpu, ref, what=f"{wl.name} autocorr removed")


def test_per_channel_full_size_lwa_band():
    """The C2 workload with the paper's channelisation: 128 channels of 25 kHz from
    38 MHz, each on its own lambda_c / 2 grid, 3 m top-hat taps, in the launch configuration
    `bench.py --per-channel-cells` times (one call, AUTO = fused); sampled channels against the oracle."""
    wl = make_per_channel(grid_n=64, pad=2, n_ant=256, n_pol=2, kernel_k=3, n_chan=128, n_t=1000, n_products=2,
                          f0_hz=38e6, df_hz=25e3, diameter_m=100.0, layout_seed=1904114222)
    v = wl.voltages()
    gpu, info = run_gpu(wl, volt=v, return_plan_info=True)
    assert info["path"] == 2 and info["launches"] == 2
    channels = [0, 64, 127]
    ref = run_oracle(wl, volt=v, channels=channels)
    assert_parity(gpu[channels], ref, what=f"{wl.name} channels {channels}")
    assert np.isfinite(gpu).all() and (gpu >= 0).all()
    totals = gpu[:, 0].sum(axis=(1, 2))
    assert totals.min() > 0.5 * totals.max()


# ------------------------------------------------------------------ tensor-core column pass
TENSOR_CASES = [
    make_config(2, n_chan=3, n_t=37),                       # delta kernel, XX/YY, ragged last batch
    make_config(3, n_chan=2, n_t=29),                       # 3x3 taps, four products, point source
    make_config(2, n_chan=1, n_t=1),                        # one frame: no averaging of the BF16 split error
    make_config(3, n_chan=5, n_t=300),                      # units split between CTAs (fix-up kernel)
    make_custom(grid_n=64, pad=2, n_ant=64, n_pol=2, kernel_k=5, n_chan=2, n_t=9, layout="disc", n_sources=2),
]


@pytest.mark.parametrize("wl", TENSOR_CASES, ids=lambda w: f"{w.name}-c{w.n_chan}-t{w.n_t}")
def test_tensor_core_path_matches_oracle(wl):
    """EPIC_PATH_TENSOR: the column transform as a BF16 hi/lo-split contraction on tcgen05 tensor
    cores, same 1e-4-of-peak bar as the FP32 paths, and the same answer as the fused kernel."""
    v = wl.voltages()
    gpu, info = run_gpu(wl, volt=v, path=4, calls=2, return_plan_info=True)
    assert info["path"] == 4 and info["launches"] == 2
    ref = run_oracle(wl, volt=v)
    assert_parity(gpu, ref, what=f"{wl.name} tensor path")
    fused = run_gpu(wl, volt=v, path=2, calls=2)
    assert max_rel_err(gpu, fused.astype(np.float64)) <= TOL


def test_tensor_core_path_is_bit_reproducible_and_rejected_where_unsupported():
    epic = _epic()
    wl = TENSOR_CASES[3]
    v = wl.voltages()
    a = run_gpu(wl, volt=v, path=4)
    b = run_gpu(wl, volt=v, path=4)
    assert np.array_equal(a, b)
    small = make_config(1)
    with epic.Plan(small.grid_n, small.pad, small.ant_uv, small.taps, small.kernel_k) as plan:
        with pytest.raises(epic.EpicError):
            plan.set_path(epic.EPIC_PATH_TENSOR)


def test_tensor_core_path_full_size_c2_sampled_channels():
    """C2 at full extent through EPIC_PATH_TENSOR, the launch configuration `bench.py --path tensor`
    times (one call, 148 CTAs); whole channels against the oracle, properties for the rest."""
    wl = make_config(2)
    v = wl.voltages()
    gpu, info = run_gpu(wl, volt=v, path=4, return_plan_info=True)
    assert info["path"] == 4 and info["launches"] == 2
    channels = [0, 63, 127]
    ref = run_oracle(wl, volt=v, channels=channels)
    assert_parity(gpu[channels], ref, what=f"{wl.name} tensor path, channels {channels}")
    assert np.isfinite(gpu).all() and (gpu >= 0).all()
    totals = gpu[:, 0].sum(axis=(1, 2))
    assert totals.min() > 0.5 * totals.max()


# ------------------------------------------------------------------ host-buffer entry point
@pytest.mark.parametrize("wl,chunks", [
    (make_config(2, n_chan=5, n_t=41), 4),                 # fused, chunks of unequal length
    (make_config(3, n_chan=3, n_t=16), 0),                 # default chunking, four products
    (make_lwa55(n_chan=2, n_t=9), 16),                     # wide kernel, more chunks than samples allow
    (make_config(4, n_chan=2, n_t=6), 2),                  # large grid
    (make_custom(grid_n=8, pad=2, n_ant=30, n_pol=2, kernel_k=3, n_chan=2, n_t=5, layout="wrap"), 1),  # two-pass, one chunk
], ids=lambda v: v.name if hasattr(v, "name") else str(v))
def test_image_host_matches_oracle_and_accumulates(wl, chunks):
    """epic_image_host: HOST voltages in, HOST images out, the copies pipelined inside the library; pageable numpy
    memory and pinned torch memory, overwrite and accumulate modes."""
    import torch
    epic = _epic()
    v = wl.voltages()
    ref = run_oracle(wl, volt=v)
    with epic.Plan(wl.grid_n, wl.pad, wl.ant_uv, wl.taps, wl.kernel_k) as plan:
        plan.set_products(wl.n_products)
        shape = (wl.n_chan, plan.n_planes(wl.n_pol), wl.N, wl.N)
        out = np.full(shape, 7.0, dtype=np.float32)                      # pageable; overwritten
        plan.image_host(v, wl.n_t, wl.n_chan, wl.n_pol, out, accumulate=False, n_chunks=chunks)
        assert plan.last_launches() > 0
        assert_parity(out, ref, what=f"{wl.name} host, overwrite")
        hv = torch.from_numpy(v).pin_memory()
        hout = torch.from_numpy(out.copy()).pin_memory()
        half = wl.n_t // 2
        plan.image_host(hv[half:].contiguous().pin_memory(), wl.n_t - half, wl.n_chan, wl.n_pol, hout, accumulate=True, n_chunks=chunks)
        second = run_oracle(wl, volt=v[half:])
        assert_parity(hout.numpy(), ref + second, what=f"{wl.name} host, accumulate")
        plan.image_host(v, 0, wl.n_chan, wl.n_pol, out, accumulate=True)  # empty gulp: unchanged
        assert_parity(out, ref, what="empty gulp")
        with pytest.raises(ValueError):
            plan.image_host(v[:, :, :, ::2], wl.n_t, wl.n_chan, wl.n_pol, out)      # non-contiguous
        with pytest.raises(ValueError):
            plan.image_host(v, wl.n_t + 1, wl.n_chan, wl.n_pol, out)                # too short


# ------------------------------------------------------------------ voltage pointers need no alignment
@pytest.mark.parametrize("n_ant", [64, 77])
def test_voltage_pointer_alignment_is_not_required(n_ant):
    """A voltage buffer that starts 1, 2 or 3 bytes past a word boundary (a slice of a larger buffer, the second gulp of
    an odd-sized stream): the fused, wide and streamed kernels then fetch bytes; AUTO never refuses and every path that
    accepts the call matches the oracle.  (Found by a randomised sweep: odd antenna counts made the second of two calls
    start at an odd byte offset, and epic_image refused a plan that epic_plan_get_path reported as fused.)"""
    import torch
    epic = _epic()
    cases = [make_custom(grid_n=64, pad=2, n_ant=n_ant, n_pol=2, kernel_k=3, n_chan=3, n_t=9, layout="disc", seed=n_ant),       # fused
             make_lwa55(n_chan=2, n_t=5, n_ant=n_ant),                                                                             # wide
             make_custom(grid_n=128, pad=2, n_ant=n_ant, n_pol=2, kernel_k=3, n_chan=2, n_t=4, layout="uniform", seed=n_ant)]    # large grid
    for wl in cases:
        v = wl.voltages()
        ref = run_oracle(wl, volt=v)
        for native in (False, True):
            vin = np.ascontiguousarray(np.swapaxes(v, 2, 3)) if native else v
            refn = ref if not native else orc.epic_image(vin, wl.input_kind, wl.ant_uv, wl.taps, wl.grid_n, wl.pad, wl.n_products,
                                                         kernel_k=wl.kernel_k, order="TCAP")
            for shift in (1, 2, 3):
                buf = torch.zeros(vin.size + 8, dtype=torch.uint8, device="cuda")
                dv = buf[shift:shift + vin.size]
                dv.copy_(torch.from_numpy(vin.reshape(-1)).cuda())
                assert dv.data_ptr() % 4 == shift
                with epic.Plan(wl.grid_n, wl.pad, wl.ant_uv, wl.taps, wl.kernel_k) as plan:
                    plan.set_products(wl.n_products)
                    if native:
                        plan.set_input_order(epic.EPIC_ORDER_TCAP)
                    paths = [epic.EPIC_PATH_AUTO] + ([epic.EPIC_PATH_STREAM] if wl.N == 256 else [epic.EPIC_PATH_FUSED])
                    for path in paths:
                        plan.set_path(path)
                        out = torch.zeros((wl.n_chan, plan.n_planes(wl.n_pol), wl.N, wl.N), dtype=torch.float32, device="cuda")
                        plan.image(dv, wl.n_t, wl.n_chan, wl.n_pol, out)
                        torch.cuda.synchronize()
                        assert_parity(out.cpu().numpy(), refn, what=f"{wl.name} shift {shift} native {native} path {path}")

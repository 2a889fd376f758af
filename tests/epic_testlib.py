"""Helpers shared by the GPU parity tests: run a Workload through libepic.so (C ABI via the
ctypes binding) and through the float64 oracle, and compare per (channel, plane) image."""
from __future__ import annotations

import numpy as np

from oracle import epic_oracle as orc

TOL = 1e-4  # BASELINE.json north_star: max |gpu - oracle| / image peak, fp32 path


def run_gpu(wl, volt=None, path=None, calls=1, n_products=None, return_plan_info=False, scratch_limit=None,
            autocorr=False, native=False, phasors=None):
    import torch
    import paper_1904_11422_b200 as epic

    v = wl.voltages() if volt is None else volt
    plan = epic.Plan(wl.grid_n, wl.pad, wl.ant_uv, wl.taps, wl.kernel_k)
    try:
        plan.set_products(wl.n_products if n_products is None else n_products)
        if path is not None:
            plan.set_path(path)
        if scratch_limit is not None:
            plan.set_scratch_limit(scratch_limit)
        if native:  # v is then [T][C][A][Np](,2)
            plan.set_input_order(epic.EPIC_ORDER_TCAP)
        if phasors is not None:
            plan.set_delay_phasors(phasors)
        planes = plan.n_planes(wl.n_pol)
        out = torch.zeros((wl.n_chan, planes, wl.N, wl.N), dtype=torch.float32, device="cuda")
        dv = torch.from_numpy(v).cuda()
        t_n = v.shape[0]
        # split the time axis over `calls` calls to exercise "epic_image ADDS into out_accum"
        edges = np.linspace(0, t_n, calls + 1).astype(int)
        for i in range(calls):
            a, b = int(edges[i]), int(edges[i + 1])
            part = dv[a:b].contiguous()
            if wl.input_kind == "cf32":
                plan.image_cf32(part, b - a, wl.n_chan, wl.n_pol, out)
            else:
                plan.image(part, b - a, wl.n_chan, wl.n_pol, out)
                if autocorr:  # linear in the gulp: removed per call
                    plan.autocorr_remove(part, b - a, wl.n_chan, wl.n_pol, out)
        torch.cuda.synchronize()
        info = {"path": plan.path(wl.n_pol), "support": plan.support(), "launches": plan.last_launches()}
        res = out.cpu().numpy()
    finally:
        plan.destroy()
    return (res, info) if return_plan_info else res


def run_oracle(wl, volt=None, channels=None, mode="fast", n_products=None):
    v = wl.voltages() if volt is None else volt
    return orc.epic_image(v, wl.input_kind, wl.ant_uv, wl.taps, wl.grid_n, wl.pad,
                          wl.n_products if n_products is None else n_products,
                          kernel_k=wl.kernel_k, mode=mode, channels=channels)


def max_rel_err(gpu: np.ndarray, ref: np.ndarray) -> float:
    """max over (channel, plane) images of max|gpu - ref| / max|ref| (peak-normalised)."""
    worst = 0.0
    g = gpu.astype(np.float64)
    for c in range(ref.shape[0]):
        # normalise every plane of a channel by that channel's brightest plane peak (XX/YY) so
        # near-zero cross planes are not judged against their own tiny peak
        peak = max(float(np.abs(ref[c]).max()), 1e-300)
        worst = max(worst, float(np.abs(g[c] - ref[c]).max()) / peak)
    return worst


def assert_parity(gpu, ref, tol=TOL, what=""):
    assert gpu.shape == ref.shape, (gpu.shape, ref.shape)
    assert np.isfinite(gpu).all(), what
    err = max_rel_err(gpu, ref)
    assert err <= tol, f"{what}: max rel err {err:.3e} > {tol:.1e}"
    return err

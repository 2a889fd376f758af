"""epic_image_noalloc (include/epic.h): the fused kernel with its scratch in the library's static device array,
for callers that cannot call cudaMalloc.  Collected LAST (file name), so that a failure here hides no other test
under `pytest -x`; passes alone in a fresh process and after the other tests (it makes its own plans and buffers and
relies on nothing an earlier test left behind -- the static array keeps the last call's contents and nothing in it
has to start at zero).

The new entry point is checked against the EXISTING path (epic_image on the same plan, scratch from cudaMalloc) on
the same inputs, on two calls in a row, within the tolerance of the other GPU tests (1e-4 of the image peak); the two
run the same kernels in the same launch configuration, so the images are in fact bit-identical, which is asserted
too.  One oracle comparison ties it to the float64 reference as well."""
import numpy as np
import pytest

from workloads import make_config, make_custom

from epic_testlib import TOL, assert_parity, max_rel_err, run_oracle

pytestmark = pytest.mark.gpu

CASES = [
    # units split between CTAs (many more batches than CTAs): the partial sums go through the scratch
    ("C2-shaped: delta, XX YY, four residues per CTA", make_config(2, n_chan=40, n_t=333)),
    ("C3-shaped: 3x3 taps, four products, two residues per CTA", make_config(3, n_chan=24, n_t=200)),
    ("N = 64, one polarisation, odd n_t", make_custom(grid_n=32, pad=2, n_ant=40, n_pol=1, kernel_k=3, n_chan=37, n_t=151,
                                                      layout="disc")),
]


def _both_paths(epic, plan, wl, dv, n_t, out_ref, out_new):
    plan.image(dv, n_t, wl.n_chan, wl.n_pol, out_ref)             # existing path: the plan's cudaMalloc'ed scratch
    plan.image_noalloc(dv, n_t, wl.n_chan, wl.n_pol, out_new)     # new entry point: the static array


@pytest.mark.parametrize("name,wl", CASES, ids=[c[0].split(":")[0] for c in CASES])
def test_noalloc_matches_existing_path_on_two_calls_in_a_row(name, wl):
    import torch
    import paper_1904_11422_b200 as epic

    assert epic.epic_noalloc_scratch_bytes() == 80 << 20
    v = wl.voltages()
    v2 = np.ascontiguousarray(v[::-1])                              # a different gulp for the second call
    with epic.Plan(wl.grid_n, wl.pad, wl.ant_uv, wl.taps, wl.kernel_k) as plan:
        plan.set_products(wl.n_products)
        assert plan.path(wl.n_pol) == epic.EPIC_PATH_FUSED
        shape = (wl.n_chan, plan.n_planes(wl.n_pol), wl.N, wl.N)
        dv, dv2 = torch.from_numpy(v).cuda(), torch.from_numpy(v2).cuda()
        plan.image_noalloc(dv, 0, wl.n_chan, wl.n_pol, torch.zeros(shape, dtype=torch.float32, device="cuda"))  # set-up call
        # call 1: both paths from zeroed images
        ref1 = torch.zeros(shape, dtype=torch.float32, device="cuda")
        new1 = torch.zeros(shape, dtype=torch.float32, device="cuda")
        _both_paths(epic, plan, wl, dv, wl.n_t, ref1, new1)
        assert plan.last_launches() == 2
        # call 2, directly after it, other voltages, a shorter gulp, ADDED to call 1's images
        ref2, new2 = ref1.clone(), new1.clone()
        n_t2 = wl.n_t - 7
        _both_paths(epic, plan, wl, dv2, n_t2, ref2, new2)
        torch.cuda.synchronize()
        r1, n1, r2, n2 = (t.cpu().numpy() for t in (ref1, new1, ref2, new2))
    for tag, r, n in (("first call", r1, n1), ("second call", r2, n2)):
        assert np.isfinite(n).all()
        assert max_rel_err(n, r.astype(np.float64)) <= TOL, f"{name}, {tag}"
        assert np.array_equal(n, r), f"{name}, {tag}: same kernels, same launch configuration -> same bits"
    assert np.abs(r2 - r1).max() > 0                                # the second call did add something


def test_noalloc_against_oracle_and_rejections():
    import torch
    import paper_1904_11422_b200 as epic

    wl = make_config(2, n_chan=3, n_t=37)
    v = wl.voltages()
    with epic.Plan(wl.grid_n, wl.pad, wl.ant_uv, wl.taps, wl.kernel_k) as plan:
        plan.set_products(wl.n_products)
        out = torch.zeros((wl.n_chan, plan.n_planes(wl.n_pol), wl.N, wl.N), dtype=torch.float32, device="cuda")
        plan.image_noalloc(torch.from_numpy(v).cuda(), wl.n_t, wl.n_chan, wl.n_pol, out)
        torch.cuda.synchronize()
        assert_parity(out.cpu().numpy(), run_oracle(wl, volt=v), what="noalloc vs oracle")
        with pytest.raises(epic.EpicError):
            plan.image_noalloc(0, 1, 1, 3, out)                     # n_pol out of range
        with pytest.raises(epic.EpicError):
            plan.image_noalloc(0, 1, 1, 2, out)                     # NULL voltages
    # plans the residue-group kernel does not take are refused, not rerouted to a path that needs other scratch
    big = make_config(4, n_chan=1, n_t=2)
    with epic.Plan(big.grid_n, big.pad, big.ant_uv, big.taps, big.kernel_k) as plan:
        out = torch.zeros((1, 6, big.N, big.N), dtype=torch.float32, device="cuda")
        with pytest.raises(epic.EpicError) as ei:
            plan.image_noalloc(torch.from_numpy(big.voltages()).cuda(), 2, 1, 2, out)
        assert ei.value.status == epic.EPIC_ERR_RANGE
    assert b"static scratch" in epic.lib().epic_status_string(epic.EPIC_ERR_SCRATCH)

"""GPU: ws_grid_visibilities_static -- a1 + a2 with the workspace in the library's static device array (wstack.h; for
callers that cannot call cudaMalloc) -- against ws_grid_visibilities with a caller-allocated workspace, on two calls in
a row that share the array.  Collected last (test_zz_*): the suite runs with pytest -x.

The two paths launch the same kernels on the same inputs; only the order in which the fp32 atomics land differs, so the
meshes and images agree within the tolerance every parity test here uses (rel-L2 1e-5, max-abs 1e-4 of the peak).
"""
import pytest
import torch

from synth import get_config, make_dataset, make_random_dataset

from . import gpu_util as U

pytestmark = pytest.mark.gpu


def _existing(plan, dev, d, mode):
    """The existing path: the caller's workspace (NaN-filled mesh: OVERWRITE writes every cell)."""
    grid = plan.alloc_grid()
    grid.fill_(float("nan"))
    wsp = plan.alloc_workspace(max(d.n_vis, 1))
    plan.grid_visibilities(dev.uvw, dev.vis, dev.weights, d.freqs_hz, grid, wsp, mode=mode)
    plan.async_status()
    return grid, wsp


def test_static_scratch_matches_the_workspace_path_on_two_calls_in_a_row():
    import paper_2301_06061_b200 as ws
    assert ws.static_scratch_bytes() == 32 << 20
    d2 = make_random_dataset(77, 60000, 4, 1024, 8, 7, wavelengths=False, fill=1.02)
    dev2 = d2.to("cuda")
    plan2 = U.make_plan(d2)
    # the existing path for call 2, first: it also loads every kernel call 2 launches, so that the free-memory test
    # below sees allocations only
    ref2, wsp2 = _existing(plan2, dev2, d2, ws.WS_GRID_SPARSE)
    transposed = bool(plan2.occupancy()["transposed"])
    ref_image = plan2.alloc_image()
    plan2.fft_wcorrect(ref2, ref_image, wsp2, accumulate=False, dirty=None, fft_flags=ws.WS_FFT_USE_OCCUPANCY)
    plan2.async_status()
    # call 1: Small (1 134 600 visibilities on 2048^2 x 16: close to the limit of the array), every cell of the mesh
    d1 = make_dataset(get_config("small"))
    dev1 = d1.to("cuda")
    plan1 = U.make_plan(d1)
    ref1, _ = _existing(plan1, dev1, d1, ws.WS_GRID_OVERWRITE)
    got1 = plan1.alloc_grid()
    got1.fill_(float("nan"))
    plan1.grid_visibilities_static(dev1.uvw, dev1.vis, dev1.weights, d1.freqs_hz, got1, mode=ws.WS_GRID_OVERWRITE)
    plan1.async_status()
    # call 2, straight after, another plan and a smaller problem (4 channels with frequencies, some visibilities off the
    # mesh): the array still holds call 1's bins beyond what call 2 rewrites.  WS_GRID_SPARSE + the own FFT: the timed path.
    got2, image2 = plan2.alloc_grid(), plan2.alloc_image()
    got2.fill_(float("nan"))
    free_before = torch.cuda.mem_get_info()[0]
    launches = plan2.launch_count()
    plan2.grid_visibilities_static(dev2.uvw, dev2.vis, dev2.weights, d2.freqs_hz, got2, mode=ws.WS_GRID_SPARSE)
    plan2.async_status()
    assert plan2.launch_count() > launches
    assert torch.cuda.mem_get_info()[0] >= free_before, "the static entry point took device memory"
    assert bool(plan2.occupancy()["transposed"]) == transposed
    plan2.fft_wcorrect(got2, image2, wsp2, accumulate=False, dirty=None, fft_flags=ws.WS_FFT_USE_OCCUPANCY)
    plan2.async_status()

    U.assert_close(U.logical(got1), U.logical(ref1).astype("complex128"), "Small mesh, static scratch vs workspace")
    written = ~torch.isnan(ref2.real)
    assert torch.equal(written, ~torch.isnan(got2.real)), "the two paths wrote different tiles"
    zero = torch.zeros_like(ref2)
    U.assert_close(torch.where(written, got2, zero).cpu().numpy(), torch.where(written, ref2, zero).cpu().numpy().astype("complex128"),
                   "random mesh (SPARSE), static scratch vs workspace")
    U.assert_close(image2.cpu().numpy(), ref_image.cpu().numpy().astype("complex128"), "image, static scratch vs workspace")
    assert float(ref_image.abs().max()) > 0


def test_static_scratch_refuses_what_does_not_fit():
    import paper_2301_06061_b200 as ws
    d = make_random_dataset(78, 400000, 4, 1024, 8, 7, wavelengths=False)        # 1.6 million visibilities: ~45 MB of bins
    dev = d.to("cuda")
    plan = U.make_plan(d)
    grid = plan.alloc_grid()
    launches = plan.launch_count()
    with pytest.raises(ws.WStackError) as e:
        plan.grid_visibilities_static(dev.uvw, dev.vis, dev.weights, d.freqs_hz, grid, mode=ws.WS_GRID_OVERWRITE)
    assert e.value.code == -3 and "WS_STATIC_SCRATCH_BYTES" in str(e.value) and str(32 << 20) in str(e.value)
    assert plan.launch_count() == launches                                       # refused before anything was launched
    # ... and the plan is still usable: a quarter of the rows fits
    n = 100000
    plan.grid_visibilities_static(dev.uvw[:n].clone(), dev.vis[:n].clone(), dev.weights[:n].clone(), d.freqs_hz, grid,
                                  mode=ws.WS_GRID_OVERWRITE)
    plan.async_status()
    ref = plan.alloc_grid()
    wsp = plan.alloc_workspace(4 * n)
    plan.grid_visibilities(dev.uvw[:n].clone(), dev.vis[:n].clone(), dev.weights[:n].clone(), d.freqs_hz, ref, wsp,
                           mode=ws.WS_GRID_OVERWRITE)
    plan.async_status()
    U.assert_close(U.logical(grid), U.logical(ref).astype("complex128"), "mesh after a refused call")

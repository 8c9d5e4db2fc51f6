"""GPU parity: the CUDA path through the C ABI against the fp64 oracle, element by element (-m gpu)."""
import numpy as np
import pytest
import torch

from synth import get_config, make_dataset, make_random_dataset

from . import gpu_util as U

pytestmark = pytest.mark.gpu


def _np(d):
    return d.uvw.numpy(), d.vis.numpy(), d.weights.numpy(), d.freqs_hz


def _full_check(oracle, d, **kw):
    out = U.run_chain(d, **kw)
    prm = U.oracle_params(oracle, d, out["plan"].tile)
    U.check_bins(oracle, prm, d, out["bins"])
    D, G = oracle.dirty_image(prm, *_np(d), return_grid=True)
    eg = U.assert_close(out["grid"], G, "grid")
    ei = U.assert_close(out["image"], D, "image")
    assert np.array_equal(out["dirty"], out["image"].real)
    U.assert_close(out["image_library"], D, "image (cuFFT + stand-alone w-correction)")
    assert np.array_equal(out["dirty_library"], out["image_library"].real)
    if "image_dense" in out:
        U.assert_close(out["image_dense"], D, "image (own FFT, no occupancy)")
    return out, eg, ei


def test_library_loaded_is_the_cuda_one():
    import paper_2301_06061_b200 as ws
    assert ws.lib().ws_version() == ws.WS_VERSION
    assert torch.cuda.is_available()


def test_tiny_config(oracle):
    d = make_dataset(get_config("tiny"))
    out, eg, ei = _full_check(oracle, d)
    print("tiny grid/image errors", eg, ei)
    assert out["plan"].launch_count() >= 9
    assert out["plan"].fft_is_own


@pytest.mark.parametrize("support", [1, 3, 5, 7, 9, 11, 13, 15])
def test_random_all_supports_with_drops_and_channels(oracle, support):
    # fill > 1: some visibilities fall off the mesh (drop rule); 3 channels in metres + frequencies
    d = make_random_dataset(100 + support, 4000, 3, 256, 5, support, wavelengths=False, fill=1.03, w_span=70.0,
                            cell_rad=2e-3)
    out, _, _ = _full_check(oracle, d)
    assert out["bins"]["n_dropped"] > 0


def test_plane_count_not_multiple_of_group_and_wide_field(oracle):
    # N_w = 11 (ragged last Horner block); cell so large that corner pixels have l^2 + m^2 >= 1 (R14)
    d = make_random_dataset(7, 3000, 1, 128, 11, 7, fill=0.9, w_span=20.0, cell_rad=0.012)
    out, _, _ = _full_check(oracle, d)
    assert out["image"][0, 0] == 0 and out["image"][64, 64] != 0


def test_heavy_bin_is_chunked(oracle):
    # 6000 visibilities inside one 32 x 32 tile of one plane: > WS_CHUNK, so the reduce-add kernel runs
    d = make_random_dataset(8, 6000, 1, 256, 2, 7, fill=0.05, w_span=1.0, cell_rad=1e-3)
    d.uvw[:, 2] = 0.3
    d.w_min, d.w_max = -1.0, 1.0
    out, _, _ = _full_check(oracle, d)
    counts = np.diff(out["bins"]["bin_start"].astype(np.int64))
    assert counts.max() > 1024


def test_empty_input_writes_zeros(oracle):
    d = make_random_dataset(9, 0, 1, 128, 3, 7)
    out = U.run_chain(d)
    assert not np.any(out["grid"]) and not np.any(out["image"])
    assert out["bins"]["n_vis"] == 0 and out["bins"]["n_dropped"] == 0


def test_all_dropped(oracle):
    d = make_random_dataset(10, 500, 1, 128, 3, 7, fill=0.9)
    d.uvw[:, 0] = 0.8 / d.cell_rad        # everything outside the mesh (its edge is at 0.5 / cell_rad)
    out = U.run_chain(d)
    assert out["bins"]["n_dropped"] == 500 and not np.any(out["grid"])


def test_accumulate_mode_equals_one_shot(oracle):
    import paper_2301_06061_b200 as ws
    d = make_random_dataset(11, 9000, 2, 256, 4, 7, wavelengths=False, fill=0.98, w_span=40.0, cell_rad=1.5e-3)
    plan = U.make_plan(d)
    dev = d.to("cuda")
    grid = plan.alloc_grid()
    wsp = plan.alloc_workspace(d.n_vis)
    plan.grid_zero(grid)
    for lo, hi in ((0, 2000), (2000, 2000), (2000, 9000)):      # includes an empty chunk
        plan.grid_visibilities(dev.uvw[lo:hi].contiguous(), dev.vis[lo:hi].contiguous(),
                               dev.weights[lo:hi].contiguous(), d.freqs_hz, grid, wsp, mode=ws.WS_GRID_ACCUMULATE)
    plan.async_status()
    prm = U.oracle_params(oracle, d, plan.tile)
    G = oracle.grid(prm, *_np(d))
    U.assert_close(U.logical(grid), G, "accumulated grid")


def test_wcorrect_accumulate_flag_and_fused_dirty(oracle):
    d = make_random_dataset(12, 10, 1, 128, 9, 7, w_span=300.0, cell_rad=4e-3)
    plan = U.make_plan(d)
    rng = np.random.default_rng(5)
    P = (rng.standard_normal((9, 128, 128)) + 1j * rng.standard_normal((9, 128, 128))).astype(np.complex64)
    prm = U.oracle_params(oracle, d, plan.tile)
    ref = oracle.wcorrect(prm, P.astype(np.complex128))
    stored = torch.fft.ifftshift(torch.from_numpy(P).cuda(), dim=(-2, -1)).contiguous()
    image, dirty = plan.alloc_image(), plan.alloc_dirty()
    plan.wcorrect_accumulate(stored, image, accumulate=False, dirty=dirty)
    U.assert_close(image.cpu().numpy(), ref, "w-correction")
    assert np.array_equal(dirty.cpu().numpy(), image.cpu().numpy().real)
    plan.wcorrect_accumulate(stored, image, accumulate=True)
    U.assert_close(image.cpu().numpy(), 2 * ref, "w-correction, accumulate")


@pytest.mark.parametrize("n_pix,n_wplanes", [(256, 3), (512, 2), (1024, 2), (2048, 3), (256, 70), (512, 130)])
def test_own_fft_fused_wcorrect_on_arbitrary_planes(oracle, n_pix, n_wplanes):
    # a3 + a4 of the own FFT (dense: any mesh contents) against the oracle's transform + w-correction, every
    # supported stage plan that fits a quick test; 70 and 130 planes cross the 64-plane Horner chains
    d = make_random_dataset(20 + n_wplanes, 10, 1, n_pix, n_wplanes, 7, w_span=250.0, cell_rad=0.6 / n_pix)
    plan = U.make_plan(d)
    assert plan.fft_is_own
    rng = np.random.default_rng(n_pix + n_wplanes)
    G = (rng.standard_normal((n_wplanes, n_pix, n_pix)) + 1j * rng.standard_normal((n_wplanes, n_pix, n_pix))).astype(np.complex64)
    prm = U.oracle_params(oracle, d, plan.tile)
    ref = np.zeros((n_pix, n_pix), np.complex128)
    for k in range(n_wplanes):
        oracle.wcorrect(prm, oracle.transform(G[k].astype(np.complex128))[None], k, ref)
    stored = torch.fft.ifftshift(torch.from_numpy(G).cuda(), dim=(-2, -1)).contiguous()
    keep = stored.clone()
    image, dirty = plan.alloc_image(), plan.alloc_dirty()
    wsp = plan.alloc_workspace(16)
    plan.fft_wcorrect(stored, image, wsp, accumulate=False, dirty=dirty)
    print("own fft + wcorrect", n_pix, n_wplanes, U.assert_close(image.cpu().numpy(), ref, "fused image"))
    assert np.array_equal(dirty.cpu().numpy(), image.cpu().numpy().real)
    stored.copy_(keep)
    plan.fft_columns(stored)                       # the two halves as separate calls, accumulating
    plan.fft_rows_wcorrect(stored, image, accumulate=True, dirty=dirty)
    U.assert_close(image.cpu().numpy(), 2 * ref, "fused image, accumulate")
    assert np.array_equal(dirty.cpu().numpy(), image.cpu().numpy().real)


@pytest.mark.parametrize("n_pix,n_wplanes,n_rows", [(512, 1, 3), (1024, 2, 5), (2048, 3, 40), (4096, 2, 2000)])
def test_sparse_fft_with_few_and_many_listed_bands(oracle, n_pix, n_wplanes, n_rows):
    # k_fft_cols hands pass 1b of a band out a fixed number of bands behind its pass 1a: fewer listed bands than that lag
    # (a handful of visibilities), and more (thousands), against the oracle -- the image of the timed path (WS_GRID_SPARSE +
    # occupancy), from a NaN-filled mesh, twice in a row on the same plan (the queue and the signals restart per launch)
    import paper_2301_06061_b200 as ws
    d = make_random_dataset(900 + n_rows, n_rows, 2, n_pix, n_wplanes, 7, wavelengths=False, fill=0.9, w_span=20.0, cell_rad=0.6 / n_pix)
    plan = U.make_plan(d)
    assert plan.fft_is_own
    prm = U.oracle_params(oracle, d, plan.tile)
    D = oracle.dirty_image(prm, d.uvw.numpy(), d.vis.numpy(), d.weights.numpy(), d.freqs_hz)
    dev = d.to("cuda")
    grid, image = plan.alloc_grid(), plan.alloc_image()
    wsp = plan.alloc_workspace(d.n_vis)
    for _ in range(2):
        grid.fill_(float("nan"))
        image.fill_(float("nan"))
        plan.grid_visibilities(dev.uvw, dev.vis, dev.weights, d.freqs_hz, grid, wsp, mode=ws.WS_GRID_SPARSE)
        plan.fft_wcorrect(grid, image, wsp, accumulate=False, dirty=None, fft_flags=ws.WS_FFT_USE_OCCUPANCY)
        plan.async_status()
        U.assert_close(image.cpu().numpy(), D, "image")
    occ = plan.occupancy()
    print("bands listed:", occ["bands"] * n_wplanes * (n_pix // 32))


def test_column_passes_are_bitwise_repeatable():
    # k_fft_cols couples its two passes through a work queue and per-band signal counters; its arithmetic does not depend on
    # the order the items are taken in, so repeated launches on the same mesh must agree bit for bit -- a pass-1b item that
    # read a row before pass 1a had written it would show up here.  Medium: 4096^2 x 32, sparse and dense.
    import paper_2301_06061_b200 as ws
    d = make_dataset(get_config("medium"), device="cuda")
    plan = ws.Plan(d.n_pix, d.n_wplanes, d.support, d.cell_rad, d.w_min, d.w_max, sigma=d.sigma_cells)
    grid = plan.alloc_grid()
    wsp = plan.alloc_workspace(d.n_vis)
    grid.zero_()
    plan.grid_visibilities(d.uvw, d.vis, d.weights, d.freqs_hz, grid, wsp, mode=ws.WS_GRID_SPARSE)
    plan.async_status()
    backup = grid.clone()
    for flags, n in ((ws.WS_FFT_USE_OCCUPANCY, 40), (0, 10)):
        ref = None
        for i in range(n):
            grid.copy_(backup)
            plan.fft_columns(grid, flags)
            if ref is None:
                ref = grid.clone()
            else:
                assert torch.equal(torch.view_as_real(grid).view(torch.int32), torch.view_as_real(ref).view(torch.int32)), \
                    f"column passes (fft_flags = {flags}) differ at launch {i}"


def test_library_fft_flag_and_occupancy_rules(oracle):
    import paper_2301_06061_b200 as ws
    d = make_random_dataset(31, 3000, 1, 256, 4, 7, fill=0.7, w_span=30.0, cell_rad=2e-3)
    lib = ws.Plan(d.n_pix, d.n_wplanes, d.support, d.cell_rad, d.w_min, d.w_max, flags=ws.WS_FLAG_LIBRARY_FFT)
    assert not lib.fft_is_own
    out = U.run_chain(d, plan=lib)
    prm = U.oracle_params(oracle, d, lib.tile)
    U.assert_close(out["image"], oracle.dirty_image(prm, *_np(d)), "image, library FFT plan")
    dev = d.to("cuda")
    grid, image, wsp = lib.alloc_grid(), lib.alloc_image(), lib.alloc_workspace(d.n_vis)
    with pytest.raises(ws.WStackError):            # a sparse mesh is only meaningful to the own FFT
        lib.grid_visibilities(dev.uvw, dev.vis, dev.weights, None, grid, wsp, mode=ws.WS_GRID_SPARSE)
    with pytest.raises(ws.WStackError):
        lib.fft_columns(grid)
    lib.fft_wcorrect(grid, image, wsp)             # falls back to the two library calls
    own = U.make_plan(d)
    other = own.alloc_grid()
    own.grid_visibilities(dev.uvw, dev.vis, dev.weights, None, grid, wsp, mode=ws.WS_GRID_SPARSE)
    with pytest.raises(ws.WStackError):            # occupancy was recorded for `grid`, not for `other`
        own.fft_wcorrect(other, image, wsp, fft_flags=ws.WS_FFT_USE_OCCUPANCY)
    occ = own.occupancy()
    assert 0 < occ["tiles"] <= occ["classes"] <= occ["bands"] <= occ["planes"] <= 1


@pytest.mark.parametrize("squeeze_axis,flags,expect_transposed", [(1, 0, True), (0, 0, False), (1, 2, False)])
def test_sparse_mesh_orientation_follows_the_uv_coverage(oracle, squeeze_axis, flags, expect_transposed):
    # uv coverage squeezed along v (axis 1) leaves fewer row bands than column bands: the sparse mesh is then stored
    # transposed (unless WS_FLAG_NO_TRANSPOSE = 2); squeezed along u it is not.  The image is the same either way.
    import paper_2301_06061_b200 as ws
    d = make_random_dataset(40, 20000, 1, 512, 5, 7, fill=0.9, w_span=50.0, cell_rad=1e-3)
    d.uvw[:, squeeze_axis] *= 0.2
    plan = ws.Plan(d.n_pix, d.n_wplanes, d.support, d.cell_rad, d.w_min, d.w_max, sigma=d.sigma_cells, flags=flags)
    out = U.run_chain(d, plan=plan)
    occ = plan.occupancy()
    assert occ["transposed"] == expect_transposed, occ
    prm = U.oracle_params(oracle, d, plan.tile)
    U.assert_close(out["image"], oracle.dirty_image(prm, *_np(d)), "image from a sparse mesh")
    assert np.array_equal(out["dirty"], out["image"].real)
    dev = d.to("cuda")
    grid, wsp = plan.alloc_grid(), plan.alloc_workspace(d.n_vis)
    plan.grid_visibilities(dev.uvw, dev.vis, dev.weights, None, grid, wsp, mode=ws.WS_GRID_SPARSE)
    with pytest.raises(ws.WStackError):        # nothing can be accumulated onto a sparse mesh
        plan.grid_visibilities(dev.uvw, dev.vis, dev.weights, None, grid, wsp, mode=ws.WS_GRID_ACCUMULATE)


def test_chunked_accumulate_keeps_occupancy_of_all_chunks(oracle):
    import paper_2301_06061_b200 as ws
    d = make_random_dataset(32, 8000, 2, 512, 6, 7, wavelengths=False, fill=0.95, w_span=60.0, cell_rad=1e-3)
    plan = U.make_plan(d)
    dev = d.to("cuda")
    grid, image = plan.alloc_grid(), plan.alloc_image()
    wsp = plan.alloc_workspace(d.n_vis)
    for i, (lo, hi) in enumerate(((0, 3000), (3000, 8000))):      # rows sorted by nothing: chunks touch different tiles
        plan.grid_visibilities(dev.uvw[lo:hi].contiguous(), dev.vis[lo:hi].contiguous(), dev.weights[lo:hi].contiguous(),
                               d.freqs_hz, grid, wsp, mode=ws.WS_GRID_OVERWRITE if i == 0 else ws.WS_GRID_ACCUMULATE)
    plan.fft_wcorrect(grid, image, wsp, fft_flags=ws.WS_FFT_USE_OCCUPANCY)
    plan.async_status()
    prm = U.oracle_params(oracle, d, plan.tile)
    U.assert_close(image.cpu().numpy(), oracle.dirty_image(prm, *_np(d)), "image from two chunks, occupancy-aware FFT")


def test_fft_planes_matches_oracle_transform(oracle):
    d = make_random_dataset(13, 10, 1, 256, 3, 7)
    plan = U.make_plan(d)
    rng = np.random.default_rng(6)
    G = (rng.standard_normal((3, 256, 256)) + 1j * rng.standard_normal((3, 256, 256))).astype(np.complex64)
    stored = torch.fft.ifftshift(torch.from_numpy(G).cuda(), dim=(-2, -1)).contiguous()
    wsp = plan.alloc_workspace(16)
    plan.fft_planes(stored, wsp)
    got = U.logical(stored)
    for k in range(3):
        U.assert_close(got[k], oracle.fft2(G[k].astype(np.complex128)), f"fft plane {k}")


def test_workspace_holds_one_record_per_visibility(oracle):
    """Every visibility near a tile corner (its footprint reaches four tiles): since round 2 a visibility is stored once, in
    its home tile, and the gridder's ring carries the rest -- the least documented workspace is enough, n_records = kept; a
    workspace that cannot hold the call's visibilities is refused by the call itself."""
    import paper_2301_06061_b200 as ws
    d = make_random_dataset(14, 2000, 1, 128, 1, 7, fill=0.9)
    d.uvw[:, :2] = torch.round(d.uvw[:, :2] * (128 * d.cell_rad) / 32) * 32 / (128 * d.cell_rad)
    plan = U.make_plan(d)
    dev = d.to("cuda")
    grid = plan.alloc_grid()
    wsp = plan.alloc_workspace(d.n_vis, dup_factor=1.0)
    grid.fill_(float("nan"))
    plan.grid_visibilities(dev.uvw, dev.vis, dev.weights, None, grid, wsp)
    plan.async_status()
    b = plan.get_bins(fields=("bin_start",))
    assert b["n_records"] == d.n_vis - b["n_dropped"]
    prm = U.oracle_params(oracle, d, plan.tile)
    U.assert_close(U.logical(grid), oracle.grid(prm, *_np(d)), "corner grid")
    with pytest.raises(ws.WStackError) as e:
        plan.grid_visibilities(dev.uvw, dev.vis, dev.weights, None, grid, plan.alloc_workspace(d.n_vis // 2))
    assert e.value.code == -3


def test_argument_validation():
    import paper_2301_06061_b200 as ws
    for bad in (dict(n_pix=250), dict(support=8), dict(support=17), dict(w_max=-5.0), dict(cell_rad=0.0), dict(tile=64),
                dict(flags=32)):
        kw = dict(n_pix=256, n_wplanes=4, support=7, cell_rad=1e-3, w_min=-1.0, w_max=1.0)
        kw.update(bad)
        with pytest.raises(ws.WStackError):
            ws.Plan(**kw)
    plan = ws.Plan(256, 4, 7, 1e-3, -1.0, 1.0)
    grid = plan.alloc_grid()
    tiny_ws = torch.empty(1024, dtype=torch.uint8, device="cuda")
    uvw = torch.zeros((10, 3), device="cuda")
    vis = torch.zeros((10, 1), dtype=torch.complex64, device="cuda")
    wt = torch.ones((10, 1), device="cuda")
    with pytest.raises(ws.WStackError) as e:
        plan.grid_visibilities(uvw, vis, wt, None, grid, tiny_ws)
    assert e.value.code == -3
    with pytest.raises(ws.WStackError):
        plan.grid_visibilities(uvw, vis, wt, None, grid, plan.alloc_workspace(10), mode=7)


def test_small_config(oracle):
    d = make_dataset(get_config("small"))
    out, eg, ei = _full_check(oracle, d)
    print("small grid/image errors", eg, ei)


@pytest.mark.parametrize("n_bl,n_chan,n_rows", [(100, 8, 4000), (100, 3, 4037), (97, 1, 4000), (64, 5, 130), (4000, 2, 4000)])
def test_snapshot_order_hint_changes_nothing_but_speed(oracle, n_bl, n_chan, n_rows):
    """ws_plan_set_snapshot_rows only changes the order in which the binning kernels walk the input: keys, bin
    offsets, sorted keys bit-exact, perm the same per-bin sets, mesh and image within tolerance -- with a ragged last
    snapshot, with F = n_bl * n_chan odd (cw falls back to 1), with fewer than two snapshots (hint ignored)."""
    d = make_random_dataset(600 + n_bl + n_chan, n_rows, n_chan, 256, 4, 7, wavelengths=False, fill=1.03, w_span=30.0, cell_rad=2e-3)
    plan = U.make_plan(d)
    plan.set_snapshot_rows(n_bl)
    out, _, _ = _full_check(oracle, d, plan=plan)
    assert out["bins"]["n_dropped"] > 0
    # degridding through the same walk
    M = (np.random.default_rng(1).standard_normal((256, 256)) + 0j).astype(np.complex64)
    dev = d.to("cuda")
    planes, wsp = plan.alloc_grid(), plan.alloc_workspace(d.n_vis)
    plan.predict_planes(torch.from_numpy(M).cuda(), planes, wsp)
    vis = torch.empty_like(dev.vis)
    plan.degrid_visibilities(dev.uvw, d.freqs_hz, d.n_chan, planes, vis, wsp)
    prm = U.oracle_params(oracle, d, 32)
    U.assert_close(vis.cpu().numpy(), oracle.predict(prm, M, d.uvw.numpy(), d.n_chan, d.freqs_hz), "degrid with the hint")
    with pytest.raises(Exception):
        plan.set_snapshot_rows(-1)


def test_channel_count_limits_and_single_plane(oracle):
    """Degenerate and maximal shapes: n_chan = 128 (the most a call accepts; 129 is refused), one w-plane, and a
    non-power-of-two channel count with the row / channel split done by division."""
    import paper_2301_06061_b200 as ws
    d = make_random_dataset(701, 300, 128, 256, 1, 7, wavelengths=False, fill=1.02, w_span=5.0, cell_rad=2e-3)
    out, _, _ = _full_check(oracle, d)
    assert out["plan"].n_wplanes == 1
    dev = d.to("cuda")
    plan = out["plan"]
    grid, wsp = plan.alloc_grid(), plan.alloc_workspace(300 * 129)
    vis129 = torch.zeros((300, 129), dtype=torch.complex64, device="cuda")
    wt129 = torch.ones((300, 129), dtype=torch.float32, device="cuda")
    with pytest.raises(ws.WStackError) as e:
        plan.grid_visibilities(dev.uvw, vis129, wt129, [150e6] * 129, grid, wsp)
    assert e.value.code == -2
    d = make_random_dataset(702, 2000, 7, 256, 3, 5, wavelengths=False, fill=0.9, w_span=15.0, cell_rad=2e-3)
    _full_check(oracle, d)


@pytest.mark.parametrize("n_pix,n_rows,n_chan", [(256, 6000, 2), (128, 6000, 2), (256, 4037, 3), (256, 1, 1)])
def test_image_from_host_equals_oracle(oracle, n_pix, n_rows, n_chan):
    """The end-to-end entry bench.py times (host buffers in, host dirty image out): own FFT (n_pix = 256) and the
    library path (128).  Pinned and pageable host memory both work; an odd number of visibilities (4037 x 3) leaves the
    weights 8 bytes off a 16-byte boundary unless every sub-buffer of dev_inputs is padded."""
    d = make_random_dataset(900 + n_pix, n_rows, n_chan, n_pix, 5, 7, wavelengths=False, fill=1.02, w_span=30.0, cell_rad=0.5 / n_pix)
    plan = U.make_plan(d)
    prm = U.oracle_params(oracle, d, 32)
    D = oracle.dirty_image(prm, *_np(d))
    grid, image, dirty = plan.alloc_grid(), plan.alloc_image(), plan.alloc_dirty()
    wsp = plan.alloc_workspace(d.n_vis)
    dev_in = torch.empty(plan.dev_inputs_bytes(d.n_rows, d.n_chan), dtype=torch.uint8, device="cuda")
    for pin in (True, False):
        uvw_h, vis_h, wt_h = (t.pin_memory() if pin else t.clone() for t in (d.uvw, d.vis, d.weights))
        dirty_h = torch.full((n_pix, n_pix), float("nan"), dtype=torch.float32)
        if pin:
            dirty_h = dirty_h.pin_memory()
        grid.fill_(float("nan"))
        plan.image_from_host(uvw_h, vis_h, wt_h, d.freqs_hz, dev_in, grid, image, dirty, dirty_h, wsp)
        plan.async_status()
        ref = D.real
        rel = np.linalg.norm(dirty_h.numpy() - ref) / np.linalg.norm(ref)
        mx = np.abs(dirty_h.numpy() - ref).max() / np.abs(D).max()
        assert rel <= U.REL_L2_TOL and mx <= U.MAX_ABS_TOL, (pin, rel, mx)
        assert np.array_equal(dirty_h.numpy(), dirty.cpu().numpy())


def test_image_from_host_refuses_a_small_workspace(oracle):
    """The end-to-end entry with a workspace that cannot hold a chunk's visibilities: an error, not an image."""
    import paper_2301_06061_b200 as ws
    d = make_random_dataset(14, 2000, 1, 256, 1, 7, fill=0.9)
    plan = U.make_plan(d)
    grid, image, dirty = plan.alloc_grid(), plan.alloc_image(), plan.alloc_dirty()
    dev_in = torch.empty(plan.dev_inputs_bytes(d.n_rows, d.n_chan), dtype=torch.uint8, device="cuda")
    dirty_h = torch.empty((256, 256), dtype=torch.float32)
    with pytest.raises(ws.WStackError) as e:
        plan.image_from_host(d.uvw, d.vis, d.weights, None, dev_in, grid, image, dirty, dirty_h, plan.alloc_workspace(d.n_vis // 2))
    assert e.value.code == -3
    plan.image_from_host(d.uvw, d.vis, d.weights, None, dev_in, grid, image, dirty, dirty_h, plan.alloc_workspace(d.n_vis, dup_factor=1.0))
    prm = U.oracle_params(oracle, d, 32)
    D = oracle.dirty_image(prm, *_np(d))
    assert np.linalg.norm(dirty_h.numpy() - D.real) <= U.REL_L2_TOL * np.linalg.norm(D.real)


def test_nan_coordinates_are_dropped_on_the_gpu(oracle):
    """DESIGN.md R33: NaN in u, v or w drops the visibility (it used to land in plane 0); +-Inf in w clamps (R6)."""
    d = make_random_dataset(77, 3000, 2, 256, 4, 7, wavelengths=False, fill=0.9, w_span=20.0, cell_rad=2e-3)
    d.uvw[5, 0] = float("nan")
    d.uvw[6, 1] = float("nan")
    d.uvw[7, 2] = float("nan")
    d.uvw[8, 2] = float("inf")
    d.uvw[9, 2] = float("-inf")
    out = U.run_chain(d)
    prm = U.oracle_params(oracle, d, out["plan"].tile)
    U.check_bins(oracle, prm, d, out["bins"])
    assert out["bins"]["n_dropped"] >= 6
    D, G = oracle.dirty_image(prm, *_np(d), return_grid=True)
    U.assert_close(out["grid"], G, "grid with NaN rows")
    U.assert_close(out["image"], D, "image with NaN rows")


@pytest.mark.parametrize("squeeze_axis", [0, 1])
def test_sparse_add_chunks_equal_one_shot(oracle, squeeze_axis):
    """WS_GRID_SPARSE then WS_GRID_SPARSE_ADD chunks (never a cleared mesh: NaN-filled) = the oracle's image of all the
    data; chunks overlap in tiles (added to) and bring new tiles (stored), heavy bins included; both orientations."""
    import paper_2301_06061_b200 as ws
    d = make_random_dataset(41 + squeeze_axis, 30000, 2, 512, 5, 7, wavelengths=False, fill=0.9, w_span=50.0, cell_rad=1e-3)
    d.uvw[:, squeeze_axis] *= 0.3
    d.uvw[20000:, :2] *= 0.02          # the last chunk piles onto a few tiles: heavy bins that earlier chunks touched
    plan = U.make_plan(d)
    dev = d.to("cuda")
    grid, image, dirty = plan.alloc_grid(), plan.alloc_image(), plan.alloc_dirty()
    wsp = plan.alloc_workspace(d.n_vis)
    grid.fill_(float("nan"))
    for i, (lo, hi) in enumerate(((0, 7000), (7000, 7100), (7100, 20000), (20000, 30000))):
        plan.grid_visibilities(dev.uvw[lo:hi].contiguous(), dev.vis[lo:hi].contiguous(), dev.weights[lo:hi].contiguous(),
                               d.freqs_hz, grid, wsp, mode=ws.WS_GRID_SPARSE if i == 0 else ws.WS_GRID_SPARSE_ADD)
    plan.fft_wcorrect(grid, image, wsp, accumulate=False, dirty=dirty, fft_flags=ws.WS_FFT_USE_OCCUPANCY)
    plan.async_status()
    assert bool(plan.occupancy()["transposed"]) == (squeeze_axis == 1)
    prm = U.oracle_params(oracle, d, plan.tile)
    U.assert_close(image.cpu().numpy(), oracle.dirty_image(prm, *_np(d)), "image from SPARSE + SPARSE_ADD chunks")
    assert np.array_equal(dirty.cpu().numpy(), image.cpu().numpy().real)
    other = plan.alloc_grid()
    with pytest.raises(ws.WStackError):        # only onto the mesh this plan wrote sparsely
        plan.grid_visibilities(dev.uvw, dev.vis, dev.weights, d.freqs_hz, other, wsp, mode=ws.WS_GRID_SPARSE_ADD)


@pytest.mark.parametrize("n_pix,hint", [(256, 0), (256, 50), (128, 0)])
def test_image_from_host_pipelined_chunks(oracle, n_pix, hint):
    """ws_image_from_host with many small chunks (copy of chunk c + 1 beside the gridding of chunk c): own FFT
    (SPARSE + SPARSE_ADD) and the library path (OVERWRITE + ACCUMULATE), with and without the snapshot hint."""
    d = make_random_dataset(950 + n_pix, 9001, 3, n_pix, 5, 7, wavelengths=False, fill=1.02, w_span=30.0, cell_rad=0.5 / n_pix)
    plan = U.make_plan(d)
    if hint:
        plan.set_snapshot_rows(hint)
    plan.set_e2e_chunk_bytes(40000)
    prm = U.oracle_params(oracle, d, 32)
    D = oracle.dirty_image(prm, *_np(d))
    grid, image, dirty = plan.alloc_grid(), plan.alloc_image(), plan.alloc_dirty()
    wsp = plan.alloc_workspace(d.n_vis)
    dev_in = torch.empty(plan.dev_inputs_bytes(d.n_rows, d.n_chan), dtype=torch.uint8, device="cuda")
    uvw_h, vis_h, wt_h = (t.pin_memory() for t in (d.uvw, d.vis, d.weights))
    dirty_h = torch.full((n_pix, n_pix), float("nan"), dtype=torch.float32).pin_memory()
    for _ in range(2):
        grid.fill_(float("nan"))
        plan.image_from_host(uvw_h, vis_h, wt_h, d.freqs_hz, dev_in, grid, image, dirty, dirty_h, wsp)
        rel = np.linalg.norm(dirty_h.numpy() - D.real) / np.linalg.norm(D.real)
        mx = np.abs(dirty_h.numpy() - D.real).max() / np.abs(D).max()
        assert rel <= U.REL_L2_TOL and mx <= U.MAX_ABS_TOL, (rel, mx)

"""Helpers of the GPU parity tests: run the CUDA chain through the C-ABI binding, compare with the oracle."""
import numpy as np
import torch

REL_L2_TOL = 1e-5      # north_star: relative L2 error of grid and image
MAX_ABS_TOL = 1e-4     # north_star: max-abs error as a fraction of the peak


def oracle_params(oracle, d, tile):
    return oracle.OracleParams(n_pix=d.n_pix, n_wplanes=d.n_wplanes, support=d.support, cell_rad=d.cell_rad,
                               w_min=d.w_min, w_max=d.w_max, sigma=d.sigma_cells, tile=tile)


def make_plan(d, device=0):
    import paper_2301_06061_b200 as ws
    plan = ws.Plan(d.n_pix, d.n_wplanes, d.support, d.cell_rad, d.w_min, d.w_max, sigma=d.sigma_cells, device=device)
    if getattr(d, "rows_per_snapshot", None):      # the configs are time-major: the launch configuration bench.py times
        plan.set_snapshot_rows(d.rows_per_snapshot)
    return plan


def logical(grid_stored: torch.Tensor) -> np.ndarray:
    """FFT-native storage -> logical centred order (wstack.h): logical (j,i) sits at ((j+N/2)%N, (i+N/2)%N)."""
    return torch.fft.fftshift(grid_stored, dim=(-2, -1)).cpu().numpy()


def run_chain(d, plan=None, want_bins=True, dup_factor=None):
    """The GPU path through the C ABI.  Returns grid (logical order, numpy complex64, from an OVERWRITE gridding),
    bins, and three images of the same inputs: `image` = the configuration bench.py times (WS_GRID_SPARSE onto a
    NaN-filled mesh, own FFT with fused w-correction skipping what the gridder left empty; the library path where
    the plan has no own FFT), `image_library` = cuFFT + stand-alone w-correction + ws_dirty_image, `image_dense` =
    own FFT without occupancy.  `dirty` belongs to `image`."""
    import paper_2301_06061_b200 as ws
    dev = d.to("cuda")
    plan = plan or make_plan(d)
    grid, image, dirty = plan.alloc_grid(), plan.alloc_image(), plan.alloc_dirty()
    wsp = plan.alloc_workspace(max(d.n_vis, 1), dup_factor)
    grid.fill_(float("nan"))      # WS_GRID_OVERWRITE must write every cell
    plan.grid_visibilities(dev.uvw, dev.vis, dev.weights, d.freqs_hz, grid, wsp, mode=ws.WS_GRID_OVERWRITE)
    bins = plan.get_bins() if want_bins else None
    plan.async_status()
    g = logical(grid)
    out = dict(grid=g, bins=bins, plan=plan)
    if plan.fft_is_own:
        image_d = plan.alloc_image()
        plan.fft_wcorrect(grid, image_d, wsp, accumulate=False, dirty=None, fft_flags=0)
        out["image_dense"] = image_d.cpu().numpy()
        grid.fill_(float("nan"))
        plan.grid_visibilities(dev.uvw, dev.vis, dev.weights, d.freqs_hz, grid, wsp, mode=ws.WS_GRID_OVERWRITE)
    plan.fft_planes(grid, wsp)
    image_l, dirty_l = plan.alloc_image(), plan.alloc_dirty()
    plan.wcorrect_accumulate(grid, image_l, accumulate=False, dirty=None)
    plan.dirty_image(image_l, dirty_l)
    out["image_library"], out["dirty_library"] = image_l.cpu().numpy(), dirty_l.cpu().numpy()
    if plan.fft_is_own:
        grid.fill_(float("nan"))  # WS_GRID_SPARSE leaves empty tiles alone; the FFT must never read them
        plan.grid_visibilities(dev.uvw, dev.vis, dev.weights, d.freqs_hz, grid, wsp, mode=ws.WS_GRID_SPARSE)
        plan.fft_wcorrect(grid, image, wsp, accumulate=False, dirty=dirty, fft_flags=ws.WS_FFT_USE_OCCUPANCY)
        plan.async_status()
        out["image"], out["dirty"] = image.cpu().numpy(), dirty.cpu().numpy()
    else:
        out["image"], out["dirty"] = out["image_library"], out["dirty_library"]
    torch.cuda.synchronize()
    return out


def errors(x: np.ndarray, ref: np.ndarray):
    """(relative L2, max-abs / peak) of x against the fp64 reference, real and imaginary parts together."""
    diff = x.astype(np.complex128) - ref
    nrm = np.linalg.norm(ref.ravel())
    peak = np.abs(ref).max()
    return (np.linalg.norm(diff.ravel()) / nrm if nrm > 0 else np.linalg.norm(diff.ravel()),
            np.abs(diff).max() / peak if peak > 0 else np.abs(diff).max())


def assert_close(x, ref, what):
    rel, mx = errors(x, ref)
    assert np.isfinite(rel) and rel <= REL_L2_TOL, f"{what}: rel-L2 {rel:.3e} > {REL_L2_TOL}"
    assert mx <= MAX_ABS_TOL, f"{what}: max-abs/peak {mx:.3e} > {MAX_ABS_TOL}"
    return rel, mx


def check_bins(oracle, prm, d, bins):
    """Bit-exact: keys, bin_start, n_dropped; perm per bin as a set (order inside a bin is unspecified).  The device
    expands `sorted_keys` from `bin_start` (k_sorted_keys), so its comparison repeats the bin_start one: the independent
    statements are keys, bin_start and the per-bin sets of perm."""
    pos = oracle.positions(prm, d.uvw.numpy(), d.n_chan, d.freqs_hz)
    assert np.array_equal(bins["keys"], pos["key"]), "keys differ from the oracle"
    bin_start, perm, dropped = oracle.bins(prm, pos["key"])
    assert bins["n_dropped"] == dropped and bins["n_bins"] == prm.n_bins
    assert np.array_equal(bins["bin_start"], bin_start), "bin_start differs"
    assert np.array_equal(bins["sorted_keys"], pos["key"][perm]), "sorted keys differ"
    gp = bins["perm"]
    assert gp.shape == perm.shape
    # sort each bin's segment: key-major, index-minor == the oracle's stable order
    seg = np.repeat(np.arange(prm.n_bins, dtype=np.int64), np.diff(bin_start.astype(np.int64)))
    order = np.lexsort((gp, seg))
    assert np.array_equal(gp[order], perm), "perm differs (as per-bin sets)"
    assert np.array_equal(pos["key"][gp], pos["key"][perm]), "perm not grouped by key"

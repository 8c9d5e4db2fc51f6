"""GPU parity of the fp64-mesh option (WS_FLAG_MESH_F64, PAPER.md:392 and Table 3: the paper's
mesh is fp64): the same chain with complex128 mesh and image, cuFFT Z2Z, against the fp64 oracle at fp64-class
tolerances (the two differ in summation order and in the library's exp / FFT roundings only)."""
import numpy as np
import pytest
import torch

from synth import get_config, make_dataset, make_random_dataset

from . import gpu_util as U

pytestmark = pytest.mark.gpu

REL_F64 = 1e-12       # rel-L2 of mesh and image (observed ~1e-15 .. 1e-14)
MAX_F64 = 1e-11       # max-abs / peak


def _np(d):
    return d.uvw.numpy(), d.vis.numpy(), d.weights.numpy(), d.freqs_hz


def _close(x, ref, what):
    rel, mx = U.errors(x, ref)
    print(f"{what}: rel-L2 {rel:.3e}, max-abs/peak {mx:.3e}")
    assert np.isfinite(rel) and rel <= REL_F64 and mx <= MAX_F64, (what, rel, mx)


def _chain(d, flags=0, kernel_type=0, kernel_param=None):
    import paper_2301_06061_b200 as ws
    plan = ws.Plan(d.n_pix, d.n_wplanes, d.support, d.cell_rad, d.w_min, d.w_max, sigma=d.sigma_cells,
                   flags=ws.WS_FLAG_MESH_F64 | flags, kernel_type=kernel_type, kernel_param=kernel_param)
    assert not plan.fft_is_own
    dev = d.to("cuda")
    grid, image, dirty = plan.alloc_grid(), plan.alloc_image(), plan.alloc_dirty()
    assert grid.dtype == torch.complex128 and dirty.dtype == torch.float64
    wsp = torch.empty(max(plan.fft_workspace_bytes(), 256), dtype=torch.uint8, device="cuda")
    grid.fill_(float("nan"))
    plan.grid_visibilities(dev.uvw, dev.vis, dev.weights, d.freqs_hz, grid, wsp, mode=ws.WS_GRID_OVERWRITE)
    G = U.logical(grid)
    plan.fft_planes(grid, wsp)
    plan.wcorrect_accumulate(grid, image, accumulate=False, dirty=dirty)
    plan.async_status()
    return plan, G, image.cpu().numpy(), dirty.cpu().numpy(), (dev, grid, image, dirty, wsp)


@pytest.mark.parametrize("cfg", ["tiny", "small"])
def test_f64_mesh_configs(oracle, cfg):
    d = make_dataset(get_config(cfg), device="cuda").to("cpu")
    plan, G, img, dirty, _ = _chain(d)
    prm = U.oracle_params(oracle, d, 32)
    D, Gref = oracle.dirty_image(prm, *_np(d), return_grid=True)
    _close(G, Gref, f"{cfg} fp64 mesh")
    _close(img, D, f"{cfg} fp64 image")
    assert np.array_equal(dirty, img.real)


def test_f64_mesh_kaiser_bessel_drops_channels_chunks_and_normalisation(oracle):
    import paper_2301_06061_b200 as ws
    d = make_random_dataset(811, 4000, 3, 256, 5, 9, wavelengths=False, fill=1.03, w_span=40.0, cell_rad=2e-3)
    beta = 14.0
    plan, G, img, dirty, (dev, grid, image, dirty_t, wsp) = _chain(d, flags=ws.WS_FLAG_TRACK_SUMWT,
                                                                  kernel_type=ws.WS_KERNEL_KAISER_BESSEL, kernel_param=beta)
    prm = U.oracle_params(oracle, d, 32)
    prm.kernel_type, prm.sigma = oracle.KERNEL_KAISER_BESSEL, beta
    D, Gref = oracle.dirty_image(prm, *_np(d), return_grid=True)
    _close(G, Gref, "KB fp64 mesh (drops, 3 channels)")
    _close(img, D, "KB fp64 image")
    sw = oracle.sum_weights(prm, d.uvw.numpy(), d.weights.numpy(), d.freqs_hz)
    assert abs(plan.sum_weights() - sw) <= 1e-12 * sw
    flags = ws.WS_NORM_SUMWT | ws.WS_NORM_N | ws.WS_NORM_TAPER
    plan.dirty_image(image, dirty_t, flags)
    ref = oracle.dirty(prm, D, flags, sw)
    got = dirty_t.cpu().numpy()
    q = slice(256 // 4, 3 * 256 // 4)     # inner half: 1 / taper^2 grows to ~1e10 at the corners (beta = 14) and multiplies the rounding noise
    assert np.abs(got[q, q] - ref[q, q]).max() <= 1e-11 * np.abs(ref[q, q]).max()
    assert np.abs(got - ref).max() <= 1e-5 * np.abs(ref).max()
    # two chunks: zero + accumulate + accumulate = the one-shot mesh
    plan.grid_zero(grid)
    for lo, hi in ((0, 1500), (1500, 4000)):
        plan.grid_visibilities(dev.uvw[lo:hi].contiguous(), dev.vis[lo:hi].contiguous(), dev.weights[lo:hi].contiguous(),
                               d.freqs_hz, grid, wsp, mode=ws.WS_GRID_ACCUMULATE)
    _close(U.logical(grid), Gref, "KB fp64 mesh, two accumulate chunks")
    with pytest.raises(ws.WStackError) as e:      # nothing is binned on this plan
        plan.bin_visibilities(dev.uvw, dev.vis, dev.weights, d.freqs_hz, wsp)
    assert e.value.code == -2


def test_f64_mesh_presummed_rows(oracle):
    """The paper's narrow-band mode on the fp64 mesh: one thread per row, sum over its channels first."""
    import paper_2301_06061_b200 as ws
    d = make_random_dataset(812, 3000, 1, 256, 4, 7, fill=0.9, w_span=30.0, cell_rad=2e-3)
    rng = np.random.default_rng(5)
    n_chan = 6
    d.vis = torch.from_numpy((rng.standard_normal((3000, n_chan)) + 1j * rng.standard_normal((3000, n_chan))).astype(np.complex64))
    d.weights = torch.from_numpy(rng.uniform(0.5, 1.5, (3000, n_chan)).astype(np.float32))
    plan, G, img, dirty, _ = _chain(d, flags=ws.WS_FLAG_PRESUM_CHANNELS)
    prm = U.oracle_params(oracle, d, 32)
    D, Gref = oracle.dirty_image(prm, *_np(d), return_grid=True)
    _close(G, Gref, "presummed fp64 mesh")
    _close(img, D, "presummed fp64 image")

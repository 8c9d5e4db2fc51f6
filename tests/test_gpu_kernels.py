"""GPU parity of SURVEY 8(f) NEXT-1: Kaiser-Bessel taps and the normalisation flags of ws_dirty_image (-m gpu)."""
import math

import numpy as np
import pytest
import torch

from synth import get_config, make_dataset, make_random_dataset

from . import gpu_util as U

pytestmark = pytest.mark.gpu


def _np(d):
    return d.uvw.numpy(), d.vis.numpy(), d.weights.numpy(), d.freqs_hz


def _kb_beta(S, alpha=2.0):
    return math.pi * math.sqrt((S / alpha) ** 2 * (alpha - 0.5) ** 2 - 0.8)


def _kb_plan(d, beta, flags=0):
    import paper_2301_06061_b200 as ws
    return ws.Plan(d.n_pix, d.n_wplanes, d.support, d.cell_rad, d.w_min, d.w_max, kernel_type=ws.WS_KERNEL_KAISER_BESSEL,
                   kernel_param=beta, flags=flags)


def _kb_prm(oracle, d, beta, tile=32):
    prm = U.oracle_params(oracle, d, tile)
    prm.kernel_type, prm.sigma = oracle.KERNEL_KAISER_BESSEL, beta
    return prm


@pytest.mark.parametrize("support,beta", [(7, _kb_beta(7)), (9, _kb_beta(9)), (5, 6.0), (3, 2.5), (15, 23.5), (1, 1.0)])
def test_kaiser_bessel_grid_and_image(oracle, support, beta):
    """Mesh and image with Kaiser-Bessel taps against the oracle (I0 series in fp32 registers vs fp64), on all
    three image paths; drops and 3 channels included."""
    d = make_random_dataset(300 + support, 5000, 3, 256, 5, support, wavelengths=False, fill=1.03, w_span=70.0, cell_rad=2e-3)
    out = U.run_chain(d, plan=_kb_plan(d, beta))
    prm = _kb_prm(oracle, d, beta)
    U.check_bins(oracle, prm, d, out["bins"])
    D, G = oracle.dirty_image(prm, *_np(d), return_grid=True)
    eg = U.assert_close(out["grid"], G, "grid (KB)")
    ei = U.assert_close(out["image"], D, "image (KB)")
    U.assert_close(out["image_library"], D, "image (KB, cuFFT path)")
    print("KB S=%d beta=%.2f grid %s image %s" % (support, beta, eg, ei))


def test_kaiser_bessel_tiny_config(oracle):
    d = make_dataset(get_config("tiny"))
    beta = _kb_beta(7)
    out = U.run_chain(d, plan=_kb_plan(d, beta), want_bins=False)
    prm = _kb_prm(oracle, d, beta)
    D, G = oracle.dirty_image(prm, *_np(d), return_grid=True)
    U.assert_close(out["grid"], G, "grid (KB, tiny)")
    U.assert_close(out["image"], D, "image (KB, tiny)")


def test_kaiser_bessel_heavy_bin(oracle):
    d = make_random_dataset(18, 6000, 1, 256, 2, 7, fill=0.05, w_span=1.0, cell_rad=1e-3)
    d.uvw[:, 2] = 0.3
    d.w_min, d.w_max = -1.0, 1.0
    beta = _kb_beta(7)
    out = U.run_chain(d, plan=_kb_plan(d, beta), want_bins=False)
    D, G = oracle.dirty_image(_kb_prm(oracle, d, beta), *_np(d), return_grid=True)
    U.assert_close(out["grid"], G, "grid (KB, heavy bin)")
    U.assert_close(out["image"], D, "image (KB, heavy bin)")


def test_kaiser_bessel_beta_out_of_range_is_refused():
    import paper_2301_06061_b200 as ws
    with pytest.raises(ws.WStackError) as e:
        ws.Plan(256, 4, 7, 1e-3, -1.0, 1.0, kernel_type=ws.WS_KERNEL_KAISER_BESSEL, kernel_param=30.0)
    assert e.value.code == -2
    with pytest.raises(ws.WStackError):
        ws.Plan(256, 4, 7, 1e-3, -1.0, 1.0, kernel_type=2)


@pytest.mark.parametrize("kernel", ["gaussian", "kaiser_bessel"])
def test_dirty_image_normalisation_flags(oracle, kernel):
    """Every combination of WS_NORM_* against the oracle's orc_dirty applied to the oracle's image, plus the sum of
    weights (kept visibilities only: fill > 1 drops some).  Wide field, so n differs from 1 and corners lie outside
    the unit circle."""
    import paper_2301_06061_b200 as ws
    d = make_random_dataset(77, 4000, 2, 256, 6, 7, wavelengths=False, fill=1.05, w_span=20.0, cell_rad=0.006)
    beta = _kb_beta(7)
    if kernel == "gaussian":
        plan = ws.Plan(d.n_pix, d.n_wplanes, d.support, d.cell_rad, d.w_min, d.w_max, sigma=d.sigma_cells,
                       flags=ws.WS_FLAG_TRACK_SUMWT)
        prm = U.oracle_params(oracle, d, 32)
    else:
        plan = _kb_plan(d, beta, flags=ws.WS_FLAG_TRACK_SUMWT)
        prm = _kb_prm(oracle, d, beta)
    dev = d.to("cuda")
    grid, image, dirty = plan.alloc_grid(), plan.alloc_image(), plan.alloc_dirty()
    wsp = plan.alloc_workspace(d.n_vis)
    plan.grid_visibilities(dev.uvw, dev.vis, dev.weights, d.freqs_hz, grid, wsp, mode=ws.WS_GRID_SPARSE)
    plan.fft_wcorrect(grid, image, wsp, fft_flags=ws.WS_FFT_USE_OCCUPANCY)
    sw_ref = oracle.sum_weights(prm, d.uvw.numpy(), d.weights.numpy(), d.freqs_hz)
    sw = plan.sum_weights()
    assert abs(sw - sw_ref) <= 1e-12 * sw_ref, (sw, sw_ref)
    D = oracle.dirty_image(prm, *_np(d))
    U.assert_close(image.cpu().numpy(), D, "image")
    for flags in range(8):
        plan.dirty_image(image, dirty, norm_flags=flags)
        ref = oracle.dirty(prm, D, flags, sw_ref)
        got = dirty.cpu().numpy()
        # Dividing by the taper multiplies the fp32 rounding noise of the image (uniform, ~1e-7 of the peak) by
        # 1 / (ghat ghat), up to 1.9e4 in the corners for the Gaussian: the north_star tolerance is applied where the
        # calibrated image is meant to be used (inner half of the field, wstack.h), a loose one to the whole array.
        N = d.n_pix
        reg = slice(N // 4, 3 * N // 4) if flags & ws.WS_NORM_TAPER else slice(0, N)
        rel = np.linalg.norm(got[reg, reg] - ref[reg, reg]) / np.linalg.norm(ref[reg, reg])
        mx = np.abs(got[reg, reg] - ref[reg, reg]).max() / np.abs(ref[reg, reg]).max()
        assert rel <= U.REL_L2_TOL and mx <= U.MAX_ABS_TOL, (flags, rel, mx)
        assert np.linalg.norm(got - ref) / np.linalg.norm(ref) <= 1e-3, flags
        if flags & ws.WS_NORM_N:
            assert got[0, 0] == 0.0 and ref[0, 0] == 0.0      # outside the unit circle
    # the sum restarts with an OVERWRITE call, grows with ACCUMULATE calls and restarts with ws_grid_zero
    half = d.n_rows // 2
    plan.grid_zero(grid)
    assert plan.sum_weights() == 0.0
    plan.grid_visibilities(dev.uvw[:half], dev.vis[:half], dev.weights[:half], d.freqs_hz, grid, wsp, mode=ws.WS_GRID_ACCUMULATE)
    plan.grid_visibilities(dev.uvw[half:], dev.vis[half:], dev.weights[half:], d.freqs_hz, grid, wsp, mode=ws.WS_GRID_ACCUMULATE)
    assert abs(plan.sum_weights() - sw_ref) <= 1e-12 * sw_ref
    plan.grid_visibilities(dev.uvw[:half], dev.vis[:half], dev.weights[:half], d.freqs_hz, grid, wsp, mode=ws.WS_GRID_OVERWRITE)
    assert plan.sum_weights() < 0.6 * sw_ref
    # WS_NORM_SUMWT without the tracking flag, and unknown bits, are refused
    plain = U.make_plan(d)
    with pytest.raises(ws.WStackError):
        plain.dirty_image(image, dirty, norm_flags=ws.WS_NORM_SUMWT)
    with pytest.raises(ws.WStackError):
        plain.dirty_image(image, dirty, norm_flags=8)
    with pytest.raises(ws.WStackError):
        plain.sum_weights()


def test_calibrated_image_equals_direct_dft_on_the_gpu(oracle):
    """End to end on the GPU: Kaiser-Bessel gridding + all normalisation flags reproduce the brute-force direct sum
    n / sum(wt) Re sum wt V e^{2 pi i (ul + vm + w_k(n-1))} (w snapped to the planes) in the inner half of the field.
    The reference here is numpy's direct DFT, not the oracle."""
    import paper_2301_06061_b200 as ws
    from tests.test_oracle_pins import _direct_dft, _model_dataset
    d, _ = _model_dataset(n_w=8)
    beta = _kb_beta(7)
    plan = _kb_plan(d, beta, flags=ws.WS_FLAG_TRACK_SUMWT)
    dev = d.to("cuda")
    grid, image, dirty = plan.alloc_grid(), plan.alloc_image(), plan.alloc_dirty()
    wsp = plan.alloc_workspace(d.n_vis)
    plan.grid_visibilities(dev.uvw, dev.vis, dev.weights, d.freqs_hz, grid, wsp, mode=ws.WS_GRID_OVERWRITE)
    plan.fft_wcorrect(grid, image, wsp)
    plan.dirty_image(image, dirty, norm_flags=ws.WS_NORM_SUMWT | ws.WS_NORM_N | ws.WS_NORM_TAPER)
    prm = _kb_prm(oracle, d, beta)
    k = oracle.positions(prm, d.uvw.numpy(), 1)["k"]
    dw = (d.w_max - d.w_min) / d.n_wplanes
    I = _direct_dft(d, d.w_min + (k + 0.5) * dw)
    N = d.n_pix
    x = (np.arange(N) - N // 2) * d.cell_rad
    ref = np.sqrt(1 - x[None, :] ** 2 - x[:, None] ** 2) * I.real / d.weights.numpy().astype(np.float64).sum()
    inner = slice(N // 4, 3 * N // 4)
    err = np.abs(dirty.cpu().numpy()[inner, inner] - ref[inner, inner]).max() / np.abs(ref).max()
    assert err < 1e-5, err


@pytest.mark.parametrize("n_chan", [5, 40])
def test_narrow_band_presummed_channels(oracle, n_chan):
    """SURVEY 8(f) NEXT-4, the paper's narrow-band mode: freq_hz = NULL, the n_chan visibilities of a row
    share its uvw.  A plan with WS_FLAG_PRESUM_CHANNELS sums weight * vis per row first and bins rows; mesh, image and
    the sum of weights must equal the oracle's plain per-visibility gridding; the exported bins are per row."""
    import paper_2301_06061_b200 as ws
    d = make_random_dataset(900 + n_chan, 3000, n_chan, 256, 4, 7, wavelengths=True, fill=1.03, w_span=30.0, cell_rad=2e-3)
    assert d.freqs_hz is None
    plan = ws.Plan(d.n_pix, d.n_wplanes, d.support, d.cell_rad, d.w_min, d.w_max, sigma=d.sigma_cells,
                   flags=ws.WS_FLAG_PRESUM_CHANNELS | ws.WS_FLAG_TRACK_SUMWT)
    prm = U.oracle_params(oracle, d, 32)
    dev = d.to("cuda")
    grid, image = plan.alloc_grid(), plan.alloc_image()
    wsp = plan.alloc_workspace(d.n_rows)                     # rows, not visibilities
    grid.fill_(float("nan"))
    plan.grid_visibilities(dev.uvw, dev.vis, dev.weights, None, grid, wsp, mode=ws.WS_GRID_OVERWRITE)
    plan.async_status()
    bins = plan.get_bins()
    assert bins["n_vis"] == d.n_rows
    key_rows = oracle.positions(prm, d.uvw.numpy(), 1)["key"]
    assert np.array_equal(bins["keys"], key_rows) and bins["n_dropped"] == int((key_rows == 0xFFFFFFFF).sum()) > 0
    D, G = oracle.dirty_image(prm, *_np(d), return_grid=True)
    U.assert_close(U.logical(grid), G, "mesh (pre-summed channels)")
    sw = oracle.sum_weights(prm, d.uvw.numpy(), d.weights.numpy())
    assert abs(plan.sum_weights() - sw) <= 1e-12 * sw
    grid.fill_(float("nan"))
    plan.grid_visibilities(dev.uvw, dev.vis, dev.weights, None, grid, wsp, mode=ws.WS_GRID_SPARSE)
    plan.fft_wcorrect(grid, image, wsp, fft_flags=ws.WS_FFT_USE_OCCUPANCY)
    U.assert_close(image.cpu().numpy(), D, "image (pre-summed channels)")
    # the same plan still degrids per visibility; a frequency axis is refused
    pred = torch.empty_like(dev.vis)
    wsp2 = plan.alloc_workspace(d.n_vis)
    plan.predict_planes(torch.from_numpy(D.astype(np.complex64)).cuda(), grid, wsp2)
    plan.degrid_visibilities(dev.uvw, None, d.n_chan, grid, pred, wsp2)
    ref = oracle.predict(prm, D.astype(np.complex64), d.uvw.numpy(), d.n_chan, None)
    U.assert_close(pred.cpu().numpy(), ref, "degridding on a pre-sum plan")
    with pytest.raises(ws.WStackError):
        plan.grid_visibilities(dev.uvw, dev.vis, dev.weights, [150e6] * n_chan, grid, wsp2, mode=ws.WS_GRID_OVERWRITE)

"""GPU parity of SURVEY 8(f) NEXT-3, degridding (image -> visibilities), against the fp64 oracle (-m gpu)."""
import math

import numpy as np
import pytest
import torch

from synth import get_config, make_dataset, make_random_dataset

from . import gpu_util as U

pytestmark = pytest.mark.gpu


def _kb_beta(S, alpha=2.0):
    return math.pi * math.sqrt((S / alpha) ** 2 * (alpha - 0.5) ** 2 - 0.8)


def _plan_and_prm(oracle, d, kernel):
    import paper_2301_06061_b200 as ws
    prm = U.oracle_params(oracle, d, 32)
    if kernel == "kb":
        beta = min(_kb_beta(d.support), 23.5) if d.support > 1 else 1.0
        prm.kernel_type, prm.sigma = oracle.KERNEL_KAISER_BESSEL, beta
        return ws.Plan(d.n_pix, d.n_wplanes, d.support, d.cell_rad, d.w_min, d.w_max,
                       kernel_type=ws.WS_KERNEL_KAISER_BESSEL, kernel_param=beta), prm
    return U.make_plan(d), prm


def _model(d, seed):
    rng = np.random.default_rng(seed)
    N = d.n_pix
    return (rng.standard_normal((N, N)) + 1j * rng.standard_normal((N, N))).astype(np.complex64)


def _predict_gpu(plan, d, M):
    dev = d.to("cuda")
    planes = plan.alloc_grid()
    wsp = plan.alloc_workspace(max(d.n_vis, 1))
    plan.predict_planes(torch.from_numpy(M).cuda(), planes, wsp)
    vis = torch.full((d.n_rows, d.n_chan), float("nan"), dtype=torch.complex64, device="cuda")
    plan.degrid_visibilities(dev.uvw, d.freqs_hz, d.n_chan, planes, vis, wsp)
    plan.async_status()
    return planes, vis, wsp, dev


@pytest.mark.parametrize("support,kernel", [(7, "gaussian"), (7, "kb"), (9, "kb"), (3, "gaussian"), (15, "kb"), (1, "gaussian")])
def test_degrid_matches_oracle(oracle, support, kernel):
    """Planes after D1 + D2 and the predicted visibilities, element by element; drops (fill > 1) predict exactly 0;
    wide field so that the screen is far from 1 and corner pixels lie outside the unit circle."""
    d = make_random_dataset(500 + support, 5000, 3, 256, 5, support, wavelengths=False, fill=1.03, w_span=40.0, cell_rad=0.006)
    plan, prm = _plan_and_prm(oracle, d, kernel)
    M = _model(d, 1)
    planes, vis, wsp, dev = _predict_gpu(plan, d, M)
    ref_v, ref_p = oracle.predict(prm, M, d.uvw.numpy(), d.n_chan, d.freqs_hz, return_planes=True)
    ep = U.assert_close(U.logical(planes), ref_p, "forward planes")
    ev = U.assert_close(vis.cpu().numpy(), ref_v, "predicted visibilities")
    print("degrid S=%d %s planes %s vis %s" % (support, kernel, ep, ev))
    key = oracle.positions(prm, d.uvw.numpy(), d.n_chan, d.freqs_hz)["key"].reshape(ref_v.shape)
    got = vis.cpu().numpy()
    assert (key == 0xFFFFFFFF).any() and not np.any(got[key == 0xFFFFFFFF])
    U.check_bins(oracle, prm, d, plan.get_bins())
    # residuals: vis_out = measured - predicted
    meas = dev.vis.clone()
    plan.degrid_visibilities(dev.uvw, d.freqs_hz, d.n_chan, planes, meas, wsp, scale=-1.0, accumulate=True)
    U.assert_close(d.vis.numpy().astype(np.complex128) - meas.cpu().numpy(), ref_v, "measured - residual")
    # the bins of a degridding call carry no visibilities: gridding from them is refused
    import paper_2301_06061_b200 as ws
    with pytest.raises(ws.WStackError):
        plan.grid_binned(planes, wsp)


def test_degrid_heavy_bin_and_tiny_config(oracle):
    d = make_random_dataset(28, 6000, 1, 256, 2, 7, fill=0.05, w_span=1.0, cell_rad=1e-3)
    d.uvw[:, 2] = 0.3
    d.w_min, d.w_max = -1.0, 1.0
    plan, prm = _plan_and_prm(oracle, d, "kb")
    M = _model(d, 2)
    _, vis, _, _ = _predict_gpu(plan, d, M)
    U.assert_close(vis.cpu().numpy(), oracle.predict(prm, M, d.uvw.numpy(), 1, None), "heavy bin")
    d = make_dataset(get_config("tiny"))
    plan, prm = _plan_and_prm(oracle, d, "gaussian")
    M = _model(d, 3)
    _, vis, _, _ = _predict_gpu(plan, d, M)
    U.assert_close(vis.cpu().numpy(), oracle.predict(prm, M, d.uvw.numpy(), d.n_chan, d.freqs_hz), "tiny")


def test_degrid_is_adjoint_of_gridding_on_the_gpu(oracle):
    """<predict(M), y> = <M, image(y)> with both sides computed on the GPU (unit weights): a property that holds at
    any size, here at Small's size (1.1 M visibilities, 2048^2 x 16)."""
    import paper_2301_06061_b200 as ws
    d = make_dataset(get_config("small"))
    d.weights = torch.ones_like(d.weights)
    plan, _ = _plan_and_prm(oracle, d, "kb")
    rng = np.random.default_rng(9)
    x = (np.arange(d.n_pix) - d.n_pix // 2) * d.cell_rad
    assert 2 * x[0] ** 2 < 1
    M = torch.from_numpy((rng.standard_normal((d.n_pix, d.n_pix)) + 1j * rng.standard_normal((d.n_pix, d.n_pix))).astype(np.complex64)).cuda()
    dev = d.to("cuda")
    grid, image = plan.alloc_grid(), plan.alloc_image()
    wsp = plan.alloc_workspace(d.n_vis)
    plan.grid_visibilities(dev.uvw, dev.vis, dev.weights, d.freqs_hz, grid, wsp, mode=ws.WS_GRID_OVERWRITE)
    plan.fft_wcorrect(grid, image, wsp)
    rhs = torch.sum(torch.conj(M).to(torch.complex128) * image.to(torch.complex128)).item()
    plan.predict_planes(M, grid, wsp)
    pred = torch.empty_like(dev.vis)
    plan.degrid_visibilities(dev.uvw, d.freqs_hz, d.n_chan, grid, pred, wsp)
    plan.async_status()
    lhs = torch.sum(torch.conj(pred).to(torch.complex128) * dev.vis.to(torch.complex128)).item()
    scale = float(torch.linalg.vector_norm(pred.to(torch.complex128)) * torch.linalg.vector_norm(dev.vis.to(torch.complex128)))
    assert abs(lhs - rhs) <= 1e-5 * scale, (lhs, rhs, scale)


def test_predicted_point_sources_equal_eq1_on_the_gpu(oracle):
    """Kaiser-Bessel, sources on pixel centres, model pre-divided by the taper: the GPU prediction equals Eq. 1
    (w snapped to the plane midpoints) evaluated by numpy -- no oracle on the reference side."""
    d = make_random_dataset(83, 3000, 1, 256, 8, 7, fill=0.85, w_span=60.0, cell_rad=1e-3)
    plan, prm = _plan_and_prm(oracle, d, "kb")
    beta, N = _kb_beta(7), d.n_pix

    def ghat(i):
        r = np.sqrt(beta ** 2 - (math.pi * 7 * (i - N // 2) / N) ** 2)
        return beta / math.sinh(beta) * np.sinh(r) / r
    src = [(160, 100, 1.0), (90, 170, 0.6), (131, 120, 0.3)]
    M = np.zeros((N, N), np.complex64)
    for q, p, f in src:
        M[q, p] = f / (ghat(p) * ghat(q))
    _, vis, _, _ = _predict_gpu(plan, d, M)
    uvw = d.uvw.numpy().astype(np.float64)
    dw = (d.w_max - d.w_min) / d.n_wplanes
    k = np.clip(np.floor((uvw[:, 2] - d.w_min) / dw), 0, d.n_wplanes - 1)
    wk = d.w_min + (k + 0.5) * dw
    ref = np.zeros(len(uvw), np.complex128)
    for q, p, f in src:
        l, m = (p - N // 2) * d.cell_rad, (q - N // 2) * d.cell_rad
        ref += f * np.exp(-2j * np.pi * (uvw[:, 0] * l + uvw[:, 1] * m + wk * (math.sqrt(1 - l * l - m * m) - 1)))
    err = np.abs(vis.cpu().numpy()[:, 0] - ref).max() / 1.9
    assert err < 1e-5, err


@pytest.mark.parametrize("support,kernel,n_pix", [(7, "gaussian", 256), (7, "kb", 512), (9, "kb", 256), (15, "kb", 256), (1, "gaussian", 256),
                                                  (7, "kb", 128)])
def test_predict_visibilities_one_call(oracle, support, kernel, n_pix):
    """ws_predict_visibilities: bins first, only the wanted column bands transformed (own column passes), gather from
    the column-transformed planes -- same visibilities as the oracle; the scratch stack is NaN-filled on entry.
    n_pix = 128 has no own FFT: the call falls back to the two library calls.  A dataset squeezed into a corner of
    the uv plane leaves most bands unwanted."""
    d = make_random_dataset(800 + support, 5000, 3, n_pix, 5, support, wavelengths=False, fill=1.03, w_span=40.0,
                            cell_rad=0.006 * 256 / n_pix)
    d.uvw[:2500, :2] *= 0.15           # half of the rows in the centre: some planes / bands hold nothing else
    plan, prm = _plan_and_prm(oracle, d, kernel)
    M = _model(d, 4)
    dev = d.to("cuda")
    planes = plan.alloc_grid()
    planes.fill_(float("nan"))
    wsp = plan.alloc_workspace(max(d.n_vis, 1))
    vis = torch.full((d.n_rows, d.n_chan), float("nan"), dtype=torch.complex64, device="cuda")
    l0 = plan.launch_count()
    plan.predict_visibilities(torch.from_numpy(M).cuda(), dev.uvw, d.freqs_hz, d.n_chan, planes, vis, wsp)
    plan.async_status()
    # own FFT: binning (6) + masks + screen + two column passes + items + gather; library path: screen + binning + items + gather
    assert plan.launch_count() - l0 >= (11 if plan.fft_is_own else 9) and (plan.fft_is_own or plan.launch_count() - l0 == 9)
    ref = oracle.predict(prm, M, d.uvw.numpy(), d.n_chan, d.freqs_hz)
    print("one-call degrid", support, kernel, n_pix, U.assert_close(vis.cpu().numpy(), ref, "predicted visibilities (one call)"))
    # residual form
    meas = dev.vis.clone()
    plan.predict_visibilities(torch.from_numpy(M).cuda(), dev.uvw, d.freqs_hz, d.n_chan, planes, meas, wsp, scale=-1.0, accumulate=True)
    U.assert_close(d.vis.numpy().astype(np.complex128) - meas.cpu().numpy(), ref, "measured - residual (one call)")


@pytest.mark.parametrize("axis,flags", [(0, 0), (1, 0), (1, 2)])
def test_predict_visibilities_narrow_uv_coverage(oracle, axis, flags):
    """All visibilities inside a narrow strip of u or of v: most column bands are unwanted and never transformed; the
    library lays the planes out along whichever axis leaves fewer (strip in v: transposed, unless WS_FLAG_NO_TRANSPOSE)."""
    d = make_random_dataset(850, 4000, 1, 512, 3, 7, fill=0.9, w_span=20.0, cell_rad=2e-3)
    d.uvw[:, axis] *= 0.05
    import paper_2301_06061_b200 as ws
    _, prm = _plan_and_prm(oracle, d, "kb")
    plan = ws.Plan(d.n_pix, d.n_wplanes, d.support, d.cell_rad, d.w_min, d.w_max, kernel_type=ws.WS_KERNEL_KAISER_BESSEL,
                   kernel_param=prm.sigma, flags=flags)
    M = _model(d, 5)
    dev = d.to("cuda")
    planes, wsp = plan.alloc_grid(), plan.alloc_workspace(d.n_vis)
    planes.fill_(float("nan"))
    vis = torch.empty_like(dev.vis)
    plan.predict_visibilities(torch.from_numpy(M).cuda(), dev.uvw, d.freqs_hz, d.n_chan, planes, vis, wsp)
    U.assert_close(vis.cpu().numpy(), oracle.predict(prm, M, d.uvw.numpy(), 1, None), "narrow strip")
    assert torch.isnan(torch.view_as_real(planes)).sum() == 0          # the screen kernel writes every cell


def test_predict_visibilities_with_the_least_documented_workspace(oracle):
    """ws_workspace_bytes_for(dup_factor = 1.0) is enough for the one-call prediction: its binning stores home records
    only and leaves the tail of the workspace to the row transforms' work area."""
    d = make_random_dataset(321, 5000, 2, 512, 4, 7, wavelengths=False, fill=0.9, w_span=40.0, cell_rad=1e-3)
    plan = U.make_plan(d)
    dev = d.to("cuda")
    prm = U.oracle_params(oracle, d, plan.tile)
    rng = np.random.default_rng(3)
    M = (rng.standard_normal((512, 512)) + 1j * rng.standard_normal((512, 512))).astype(np.complex64)
    ref = oracle.predict(prm, M.astype(np.complex128), d.uvw.numpy(), d.n_chan, d.freqs_hz)
    planes = plan.alloc_grid()
    pred = torch.full_like(dev.vis, float("nan"))
    wsp = plan.alloc_workspace(d.n_vis, dup_factor=1.0)
    plan.predict_visibilities(torch.from_numpy(M).cuda(), dev.uvw, d.freqs_hz, d.n_chan, planes, pred, wsp)
    plan.async_status()
    U.assert_close(pred.cpu().numpy(), ref, "one-call prediction, dup_factor 1.0 workspace")

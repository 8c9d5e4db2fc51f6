"""GPU parity at BASELINE.json's full sizes: Medium element by element through every path (run_chain); Kaiser-Bessel
imaging and degridding at Large's size on sampled planes / pixels / visibilities plus the adjoint identity over all 10^8
visibilities.  The Gaussian imaging path of Large, Extreme and paper_medium is compared as a WHOLE in test_gpu_wholearray.py."""
import os

import numpy as np
import pytest
import torch

from synth import get_config, make_dataset

from . import gpu_util as U

pytestmark = pytest.mark.gpu


def _np(d):
    return d.uvw.numpy(), d.vis.numpy(), d.weights.numpy(), d.freqs_hz


def test_medium_config_elementwise(oracle):
    d = make_dataset(get_config("medium"), device="cuda").to("cpu")
    out = U.run_chain(d)
    prm = U.oracle_params(oracle, d, out["plan"].tile)
    U.check_bins(oracle, prm, d, out["bins"])
    D, G = oracle.dirty_image(prm, *_np(d), return_grid=True)
    print("medium grid", U.assert_close(out["grid"], G, "grid"), "image", U.assert_close(out["image"], D, "image"))


# (Large and Extreme as a whole -- every plane of the mesh, the whole image, every bin of Large -- and Extreme's streamed
# chunks are in test_gpu_wholearray.py.)


def _kb_beta(S, alpha=2.0):
    import math
    return math.pi * math.sqrt((S / alpha) ** 2 * (alpha - 0.5) ** 2 - 0.8)


def test_large_config_kaiser_bessel_and_degridding_sampled(oracle):
    """SURVEY 8(f) NEXT-1 and NEXT-3 at Large's full size, as bench.py runs them.  Kaiser-Bessel imaging: one whole
    plane of the mesh and sampled image pixels.  Degridding of a sparse model (40 pixels): sampled predicted
    visibilities against the oracle's re-ordered chain, and the adjoint identity <predict(M), y> = <M, image(y)>
    over all 10^8 visibilities (a property that holds at any size; unit weights)."""
    import paper_2301_06061_b200 as ws
    cfg = get_config("large")
    dg = make_dataset(cfg, device="cuda")
    d = dg.to("cpu")
    beta = _kb_beta(d.support)
    plan = ws.Plan(d.n_pix, d.n_wplanes, d.support, d.cell_rad, d.w_min, d.w_max, kernel_type=ws.WS_KERNEL_KAISER_BESSEL,
                   kernel_param=beta)
    plan.set_snapshot_rows(d.rows_per_snapshot)
    prm = U.oracle_params(oracle, d, plan.tile)
    prm.kernel_type, prm.sigma = oracle.KERNEL_KAISER_BESSEL, beta
    grid, image = plan.alloc_grid(), plan.alloc_image()
    wsp = plan.alloc_workspace(d.n_vis)
    ones = torch.ones_like(dg.weights)
    N, c = d.n_pix, d.n_pix // 2
    rng = np.random.default_rng(123)

    # --- KB imaging with the data's weights: one plane of the mesh, sampled pixels of the image
    grid.fill_(float("nan"))
    plan.grid_visibilities(dg.uvw, dg.vis, dg.weights, d.freqs_hz, grid, wsp, mode=ws.WS_GRID_OVERWRITE)
    plan.async_status()
    k = 40
    G = oracle.grid(prm, *_np(d), plane_lo=k, plane_hi=k + 1)[0]
    got = torch.fft.fftshift(grid[k], dim=(-2, -1)).cpu().numpy()
    print("large KB plane", k, U.assert_close(got, G, "KB mesh plane"))
    del G, got
    grid.fill_(float("nan"))
    plan.grid_binned(grid, wsp, mode=ws.WS_GRID_SPARSE)
    plan.fft_wcorrect(grid, image, wsp, fft_flags=ws.WS_FFT_USE_OCCUPANCY)
    q = np.concatenate([[c, 0, N - 1], rng.integers(0, N, 13)])
    p = np.concatenate([[c, N - 1, 0], rng.integers(0, N, 13)])
    ref = oracle.image_samples(prm, *_np(d), q, p)
    img = image.cpu().numpy()
    got = img[q, p].astype(np.complex128)
    peak = max(np.abs(ref).max(), np.abs(img).max())
    rel, mx = np.linalg.norm(got - ref) / np.linalg.norm(ref), np.abs(got - ref).max() / peak
    print("large KB image samples: rel-L2 %.3e, max-abs/peak %.3e" % (rel, mx))
    assert rel <= U.REL_L2_TOL and mx <= U.MAX_ABS_TOL

    # --- degridding of a sparse model: sampled visibilities against the oracle
    sq, sp = rng.integers(N // 4, 3 * N // 4, 40), rng.integers(N // 4, 3 * N // 4, 40)
    val = (rng.standard_normal(40) + 1j * rng.standard_normal(40)).astype(np.complex64)
    M = torch.zeros((N, N), dtype=torch.complex64, device="cuda")
    Mh = np.zeros((N, N), np.complex64)
    np.add.at(Mh, (sq, sp), val)
    M.copy_(torch.from_numpy(Mh))
    plan.predict_planes(M, grid, wsp)
    pred = torch.full_like(dg.vis, float("nan"))
    plan.degrid_visibilities(dg.uvw, d.freqs_hz, d.n_chan, grid, pred, wsp)
    plan.async_status()
    assert torch.isfinite(torch.view_as_real(pred)).all()
    samp = np.concatenate([rng.integers(0, d.n_vis, 4000), np.arange(16), d.n_vis - 1 - np.arange(16)])
    ref = oracle.predict_samples(prm, d.uvw.numpy(), d.n_chan, d.freqs_hz, sq, sp, val.astype(np.complex128), samp)
    got = pred.reshape(-1)[torch.from_numpy(samp).cuda()].cpu().numpy().astype(np.complex128)
    peak = float(torch.abs(pred).max())
    rel, mx = np.linalg.norm(got - ref) / np.linalg.norm(ref), np.abs(got - ref).max() / peak
    print("large degrid samples: rel-L2 %.3e, max-abs/peak %.3e" % (rel, mx))
    assert rel <= U.REL_L2_TOL and mx <= U.MAX_ABS_TOL

    # --- the same prediction through the one-call path (bins first, wanted column bands only)
    pred1 = torch.full_like(dg.vis, float("nan"))
    grid.fill_(float("nan"))
    plan.predict_visibilities(M, dg.uvw, d.freqs_hz, d.n_chan, grid, pred1, wsp)
    plan.async_status()
    got1 = pred1.reshape(-1)[torch.from_numpy(samp).cuda()].cpu().numpy().astype(np.complex128)
    rel1, mx1 = np.linalg.norm(got1 - ref) / np.linalg.norm(ref), np.abs(got1 - ref).max() / peak
    print("large degrid samples (one call): rel-L2 %.3e, max-abs/peak %.3e" % (rel1, mx1))
    assert rel1 <= U.REL_L2_TOL and mx1 <= U.MAX_ABS_TOL
    dall = torch.linalg.vector_norm((pred1 - pred).to(torch.complex128)) / torch.linalg.vector_norm(pred.to(torch.complex128))
    assert float(dall) <= 2e-6, float(dall)          # all 1e8 visibilities: the two GPU paths agree

    # --- adjoint identity over the whole data set (unit weights)
    lhs = torch.sum(torch.conj(pred).to(torch.complex128) * dg.vis.to(torch.complex128)).item()
    scale = float(torch.linalg.vector_norm(pred.to(torch.complex128)) * torch.linalg.vector_norm(dg.vis.to(torch.complex128)))
    plan.grid_visibilities(dg.uvw, dg.vis, ones, d.freqs_hz, grid, wsp, mode=ws.WS_GRID_SPARSE)
    plan.fft_wcorrect(grid, image, wsp, fft_flags=ws.WS_FFT_USE_OCCUPANCY)
    plan.async_status()
    rhs = torch.sum(torch.conj(M).to(torch.complex128) * image.to(torch.complex128)).item()
    print("large adjoint: lhs %s rhs %s rel %.3e" % (lhs, rhs, abs(lhs - rhs) / scale))
    assert abs(lhs - rhs) <= 1e-5 * scale

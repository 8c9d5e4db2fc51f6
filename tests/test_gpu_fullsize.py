"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (WS_GRID_OVERWRITE, split
a1 / a2 calls, default workspace).  Medium is compared element by element; Large and Extreme on what the oracle can
compute one by one: every key / bin offset (bit-exact), whole sampled w-planes of the mesh, sampled image pixels."""
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


def _bins_exact_without_sorting(oracle, prm, d, bins):
    """keys, bin_start, sorted keys bit-exact; perm: a permutation of the kept indices whose keys are the sorted
    keys, which is the same statement as 'every bin holds exactly its visibilities' (order inside a bin is free)."""
    key = oracle.positions(prm, d.uvw.numpy(), d.n_chan, d.freqs_hz)["key"]
    assert np.array_equal(bins["keys"], key)
    bin_start, perm, dropped = oracle.bins(prm, key)
    assert bins["n_dropped"] == dropped
    assert np.array_equal(bins["bin_start"], bin_start)
    assert np.array_equal(bins["sorted_keys"], key[perm])
    gp = bins["perm"]
    assert np.array_equal(key[gp], bins["sorted_keys"])
    assert np.array_equal(np.sort(gp), np.flatnonzero(key != 0xFFFFFFFF).astype(np.uint32))


def _sampled_check(oracle, cfg_name, planes_to_check, n_pix_samples, chunks=1):
    import paper_2301_06061_b200 as ws
    cfg = get_config(cfg_name)
    dg = make_dataset(cfg, device="cuda")
    d = dg.to("cpu")
    plan = U.make_plan(d)
    prm = U.oracle_params(oracle, d, plan.tile)
    grid, image, dirty = plan.alloc_grid(), plan.alloc_image(), plan.alloc_dirty()
    grid.fill_(float("nan"))
    if chunks == 1:
        wsp = plan.alloc_workspace(d.n_vis)
        plan.bin_visibilities(dg.uvw, dg.vis, dg.weights, d.freqs_hz, wsp)
        plan.grid_binned(grid, wsp, mode=ws.WS_GRID_OVERWRITE)
        plan.async_status()
        _bins_exact_without_sorting(oracle, prm, d, plan.get_bins())

    else:   # row chunks streamed through repeated calls: first overwrites, the rest accumulate
        rc = d.row_chunks()
        wsp = plan.alloc_workspace(max(hi - lo for lo, hi in rc) * d.n_chan)
        for i, (lo, hi) in enumerate(rc):
            plan.grid_visibilities(dg.uvw[lo:hi], dg.vis[lo:hi], dg.weights[lo:hi], d.freqs_hz, grid, wsp,
                                   mode=ws.WS_GRID_OVERWRITE if i == 0 else ws.WS_GRID_ACCUMULATE)
            plan.async_status()
    # whole sampled planes of the mesh, element by element
    for k in planes_to_check:
        G = oracle.grid(prm, *_np(d), plane_lo=k, plane_hi=k + 1)[0]
        got = torch.fft.fftshift(grid[k], dim=(-2, -1)).cpu().numpy()
        print(cfg_name, "plane", k, "errors", U.assert_close(got, G, f"mesh plane {k}"), "nonzero cells", np.count_nonzero(G))
        del G, got
    if chunks == 1 and plan.fft_is_own:
        # what bench.py times: gridding that writes only the tiles holding visibilities (onto a NaN-filled mesh), then
        # the own FFT with the fused w-correction, skipping what stayed empty
        grid.fill_(float("nan"))
        plan.grid_binned(grid, wsp, mode=ws.WS_GRID_SPARSE)
        plan.fft_columns(grid, ws.WS_FFT_USE_OCCUPANCY)
        plan.fft_rows_wcorrect(grid, image, accumulate=False, dirty=dirty, fft_flags=ws.WS_FFT_USE_OCCUPANCY)
        plan.async_status()
    else:
        occ = ws.WS_FFT_USE_OCCUPANCY if plan.fft_is_own else 0
        plan.fft_wcorrect(grid, image, wsp, accumulate=False, dirty=dirty, fft_flags=occ)
    torch.cuda.synchronize()
    img = image.cpu().numpy()
    assert np.array_equal(dirty.cpu().numpy(), img.real)
    # sampled pixels: the phase centre, the brightest model sources, the corners, random pixels
    N, c = d.n_pix, d.n_pix // 2
    rng = np.random.default_rng(99)
    top = np.argsort(d.src_flux)[-4:]
    q = [c, 0, N - 1, 0] + [int(round(d.src_m[i] / d.cell_rad)) + c for i in top]
    p = [c, 0, N - 1, N - 1] + [int(round(d.src_l[i] / d.cell_rad)) + c for i in top]
    q += list(rng.integers(0, N, n_pix_samples - len(q)))
    p += list(rng.integers(0, N, n_pix_samples - len(p)))
    q, p = np.clip(q, 0, N - 1), np.clip(p, 0, N - 1)
    ref = oracle.image_samples(prm, *_np(d), q, p)
    got = img[q, p].astype(np.complex128)
    peak = max(np.abs(ref).max(), np.abs(img).max())
    rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    mx = np.abs(got - ref).max() / peak
    print(cfg_name, "image samples: rel-L2 %.3e, max-abs/peak %.3e, peak %.4g" % (rel, mx, peak))
    assert rel <= U.REL_L2_TOL and mx <= U.MAX_ABS_TOL
    assert np.isfinite(img).all()


# (Large as a whole -- all 64 planes of the mesh, the whole image, every bin -- is in test_gpu_wholearray.py.)


@pytest.mark.skipif(os.environ.get("WS_SKIP_EXTREME") == "1", reason="WS_SKIP_EXTREME=1")
def test_extreme_config_chunked_sampled(oracle):
    _sampled_check(oracle, "extreme", planes_to_check=(16,), n_pix_samples=12, chunks=8)


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

"""GPU parity over a seeded sweep of shapes and option combinations (-m gpu): support, kernel, channels, mesh size, plane
count, frequency mode, snapshot hint, pre-summed channels -- mesh, image and the one-call degridding against the oracle,
then the same image through streamed chunks (WS_GRID_SPARSE + WS_GRID_SPARSE_ADD), through the pipelined end-to-end
entry, and as the sum of two plane ranges."""
import numpy as np
import pytest
import torch

from synth import make_random_dataset

from . import gpu_util as U

pytestmark = pytest.mark.gpu


def _cases(n=14, seed=2024):
    rng = np.random.default_rng(seed)
    out = []
    for i in range(n):
        S = int(rng.choice([1, 3, 5, 7, 9, 11, 15]))
        kb = bool(rng.integers(0, 2))
        out.append(dict(seed=3000 + i, S=S, kb=kb, param=float(rng.uniform(2.0, min(2.3 * S + 1, 23.0))) if kb else float(rng.uniform(0.7, 1.4)),
                        n_chan=int(rng.choice([1, 2, 3, 8, 17])), n_pix=int(rng.choice([256, 512])), n_w=int(rng.integers(1, 9)),
                        metres=bool(rng.integers(0, 2)), n_rows=int(rng.integers(500, 4000)), hint=int(rng.choice([0, 37, 100])),
                        presum=bool(rng.integers(0, 2))))
    return out


@pytest.mark.parametrize("c", _cases(), ids=lambda c: "S%d-%s-c%d-N%d-w%d-%s-h%d-%s" % (
    c["S"], "kb" if c["kb"] else "g", c["n_chan"], c["n_pix"], c["n_w"], "m" if c["metres"] else "wl", c["hint"], "ps" if c["presum"] else "np"))
def test_random_shape(oracle, c):
    import paper_2301_06061_b200 as ws
    d = make_random_dataset(c["seed"], c["n_rows"], c["n_chan"], c["n_pix"], c["n_w"], c["S"], wavelengths=not c["metres"], fill=1.03,
                            w_span=30.0, cell_rad=0.6 / c["n_pix"])
    presum = c["presum"] and not c["metres"]
    plan = ws.Plan(d.n_pix, d.n_wplanes, d.support, d.cell_rad, d.w_min, d.w_max,
                   kernel_type=ws.WS_KERNEL_KAISER_BESSEL if c["kb"] else ws.WS_KERNEL_GAUSSIAN, kernel_param=c["param"],
                   flags=ws.WS_FLAG_PRESUM_CHANNELS if presum else 0)
    if c["hint"]:
        plan.set_snapshot_rows(c["hint"])
    prm = oracle.OracleParams(n_pix=d.n_pix, n_wplanes=d.n_wplanes, support=d.support, cell_rad=d.cell_rad, w_min=d.w_min,
                              w_max=d.w_max, sigma=c["param"], tile=32, kernel_type=1 if c["kb"] else 0)
    dev = d.to("cuda")
    grid, image = plan.alloc_grid(), plan.alloc_image()
    wsp = plan.alloc_workspace(d.n_vis)
    D, G = oracle.dirty_image(prm, d.uvw.numpy(), d.vis.numpy(), d.weights.numpy(), d.freqs_hz, return_grid=True)
    grid.fill_(float("nan"))
    plan.grid_visibilities(dev.uvw, dev.vis, dev.weights, d.freqs_hz, grid, wsp, mode=ws.WS_GRID_OVERWRITE)
    plan.async_status()
    U.assert_close(U.logical(grid), G, "mesh")
    if not presum:
        U.check_bins(oracle, prm, d, plan.get_bins())
    grid.fill_(float("nan"))
    plan.grid_visibilities(dev.uvw, dev.vis, dev.weights, d.freqs_hz, grid, wsp, mode=ws.WS_GRID_SPARSE)
    plan.fft_wcorrect(grid, image, wsp, fft_flags=ws.WS_FFT_USE_OCCUPANCY)
    U.assert_close(image.cpu().numpy(), D, "image")
    M = D.astype(np.complex64)
    pred = torch.full_like(dev.vis, float("nan"))
    grid.fill_(float("nan"))
    plan.predict_visibilities(torch.from_numpy(M).cuda(), dev.uvw, d.freqs_hz, d.n_chan, grid, pred, wsp)
    plan.async_status()
    U.assert_close(pred.cpu().numpy(), oracle.predict(prm, M, d.uvw.numpy(), d.n_chan, d.freqs_hz), "predicted visibilities")

    # -- the same image from three streamed chunks onto a never-cleared mesh
    cuts = sorted(set([0, d.n_rows // 3, d.n_rows // 3 + 7, d.n_rows]))
    grid.fill_(float("nan"))
    for i, (lo, hi) in enumerate(zip(cuts[:-1], cuts[1:])):
        plan.grid_visibilities(dev.uvw[lo:hi].clone(), dev.vis[lo:hi].clone(), dev.weights[lo:hi].clone(), d.freqs_hz,   # (clone: 16-byte aligned)
                               grid, wsp, mode=ws.WS_GRID_SPARSE if i == 0 else ws.WS_GRID_SPARSE_ADD)
    plan.fft_wcorrect(grid, image, wsp, fft_flags=ws.WS_FFT_USE_OCCUPANCY)
    plan.async_status()
    U.assert_close(image.cpu().numpy(), D, "image from streamed chunks")
    # -- the pipelined end-to-end entry with small chunks
    plan.set_e2e_chunk_bytes(30000)
    dirty, dirty_h = plan.alloc_dirty(), torch.full((d.n_pix, d.n_pix), float("nan"), dtype=torch.float32).pin_memory()
    dev_in = torch.empty(plan.dev_inputs_bytes(d.n_rows, d.n_chan), dtype=torch.uint8, device="cuda")
    grid.fill_(float("nan"))
    plan.image_from_host(d.uvw.pin_memory(), d.vis.pin_memory(), d.weights.pin_memory(), d.freqs_hz, dev_in, grid, image, dirty, dirty_h, wsp)
    rel = np.linalg.norm(dirty_h.numpy() - D.real) / np.linalg.norm(D.real)
    assert rel <= U.REL_L2_TOL and np.abs(dirty_h.numpy() - D.real).max() <= U.MAX_ABS_TOL * np.abs(D).max(), rel
    # -- two plane ranges (the rank-local half of the plane-sharded variant) sum to the image
    if d.n_wplanes >= 2:
        total = torch.zeros_like(image)
        for lo, hi in ((0, d.n_wplanes // 2), (d.n_wplanes // 2, d.n_wplanes)):
            plan.set_plane_range(lo, hi)
            grid.fill_(float("nan"))
            plan.grid_visibilities(dev.uvw, dev.vis, dev.weights, d.freqs_hz, grid, wsp, mode=ws.WS_GRID_SPARSE)
            plan.fft_wcorrect(grid, image, wsp, fft_flags=ws.WS_FFT_USE_OCCUPANCY)
            total += image
        plan.async_status()
        U.assert_close(total.cpu().numpy(), D, "sum over two plane ranges")

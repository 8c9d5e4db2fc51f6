"""GPU parity over WHOLE arrays at BASELINE.json's full sizes (north_star: "GPU grid and image match the fp64 oracle ...
on all five configs"; rel-L2 and max-abs "each over the whole array").

The fp64 oracle is streamed plane by plane (`oracle.grid` on a batch of planes, one plane per host thread, then the
oracle's transform and w-correction of each), as SURVEY 8(d) describes: every plane of the GPU mesh is compared cell by
cell while it exists on the host (running sums of |delta|^2, |ref|^2 and the maxima, kept in fp64 on the device --
torch is used for the bookkeeping of the comparison only), and the whole image at the end.  What is compared is the
launch configuration bench.py times -- split a1 / a2 calls, snapshot hint, WS_GRID_SPARSE onto a NaN-filled mesh, own
FFT with WS_FFT_USE_OCCUPANCY -- plus the WS_GRID_OVERWRITE mesh and the dense own FFT on it.
"""
import os
import time

import numpy as np
import pytest
import torch

from synth import get_config, make_dataset, make_random_dataset

from . import gpu_util as U

pytestmark = pytest.mark.gpu


def _np(d):
    return d.uvw.numpy(), d.vis.numpy(), d.weights.numpy(), d.freqs_hz


class Running:
    """rel-L2 and max-abs/peak of a GPU array against the fp64 reference, accumulated piece by piece."""

    def __init__(self, what):
        self.what, self.d2, self.r2, self.dmax, self.rmax, self.cells = what, 0.0, 0.0, 0.0, 0.0, 0

    def add(self, got: torch.Tensor, ref: torch.Tensor):
        delta = got.to(torch.complex128) - ref
        self.d2 += float(torch.sum(delta.real ** 2 + delta.imag ** 2))
        self.r2 += float(torch.sum(ref.real ** 2 + ref.imag ** 2))
        self.dmax = max(self.dmax, float(torch.abs(delta).max()))
        self.rmax = max(self.rmax, float(torch.abs(ref).max()))
        self.cells += ref.numel()

    def check(self):
        rel = (self.d2 / self.r2) ** 0.5 if self.r2 > 0 else self.d2 ** 0.5
        mx = self.dmax / self.rmax if self.rmax > 0 else self.dmax
        print(f"{self.what}: {self.cells} cells, rel-L2 {rel:.3e}, max-abs/peak {mx:.3e}")
        assert np.isfinite(rel) and rel <= U.REL_L2_TOL, f"{self.what}: rel-L2 {rel:.3e}"
        assert mx <= U.MAX_ABS_TOL, f"{self.what}: max-abs/peak {mx:.3e}"
        return rel, mx


def _plane_batch(oracle, n_pix):
    """Planes gridded per oracle call: one per host thread, bounded by the host memory (16 N^2 bytes per fp64 plane)."""
    import psutil
    fit = int(psutil.virtual_memory().available * 0.4 // (16 * n_pix * n_pix))
    return max(1, min(oracle.num_threads(), fit))


def _sparse_plane_logical(grid_k: torch.Tensor, transposed: bool) -> torch.Tensor:
    g = torch.fft.fftshift(grid_k, dim=(-2, -1))
    return g.T if transposed else g


def _whole_config(oracle, cfg_name, presum=False, one_mesh=False, dup_factor=None, overwrite_planes=(0, 11, 20, 31)):
    """Every plane of the mesh (OVERWRITE: every cell; SPARSE: every written cell, unwritten ones must be exact zeros of
    the oracle) and the whole image of the timed path, then of the dense own FFT on the OVERWRITE mesh.  one_mesh: the
    two meshes do not fit the device side by side (Extreme): one buffer, SPARSE first; the OVERWRITE mesh is gridded
    into it after the image and compared on `overwrite_planes` (the oracle's planes are kept on the host for that)."""
    import paper_2301_06061_b200 as ws
    cfg = get_config(cfg_name)
    dg = make_dataset(cfg, device="cuda")
    d = dg.to("cpu")
    flags = ws.WS_FLAG_PRESUM_CHANNELS | ws.WS_FLAG_TRACK_SUMWT if presum else 0
    plan = ws.Plan(d.n_pix, d.n_wplanes, d.support, d.cell_rad, d.w_min, d.w_max, sigma=d.sigma_cells, flags=flags)
    plan.set_snapshot_rows(d.rows_per_snapshot)
    assert plan.fft_is_own
    prm = U.oracle_params(oracle, d, plan.tile)
    N, NW = d.n_pix, d.n_wplanes
    grid_s = plan.alloc_grid()
    grid_o = grid_s if one_mesh else plan.alloc_grid()
    image, dirty = plan.alloc_image(), plan.alloc_dirty()
    wsp = plan.alloc_workspace(d.n_rows if presum else d.n_vis, dup_factor)
    plan.bin_visibilities(dg.uvw, dg.vis, dg.weights, d.freqs_hz, wsp)
    e_over, e_sparse = Running(f"{cfg_name} mesh (OVERWRITE)"), Running(f"{cfg_name} mesh (SPARSE, written cells)")

    def grid_overwrite():
        grid_o.fill_(float("nan"))
        plan.grid_binned(grid_o, wsp, mode=ws.WS_GRID_OVERWRITE)
        plan.async_status()

    def grid_sparse():                                           # last: the plan's occupancy describes grid_s
        grid_s.fill_(float("nan"))
        plan.grid_binned(grid_s, wsp, mode=ws.WS_GRID_SPARSE)
        plan.async_status()
        return bool(plan.occupancy()["transposed"])

    def cmp_overwrite(k, ref):
        e_over.add(torch.fft.fftshift(grid_o[k], dim=(-2, -1)), ref)

    def cmp_sparse(k, ref, transposed):
        got = _sparse_plane_logical(grid_s[k], transposed)
        unwritten = torch.isnan(got.real)
        assert not bool(torch.any(ref[unwritten] != 0)), f"plane {k}: a tile the sparse gridder skipped is not empty"
        e_sparse.add(torch.where(unwritten, torch.zeros_like(got), got), ref)

    if not one_mesh:
        grid_overwrite()
    transposed = grid_sparse()
    if presum:
        sw = oracle.sum_weights(prm, d.uvw.numpy(), d.weights.numpy(), d.freqs_hz)
        assert abs(plan.sum_weights() - sw) <= 1e-9 * sw
    torch.cuda.synchronize()

    D = np.zeros((N, N), np.complex128)
    B = _plane_batch(oracle, N)
    kept = {}
    t0 = time.time()
    for lo in range(0, NW, B):
        hi = min(lo + B, NW)
        G = oracle.grid(prm, *_np(d), plane_lo=lo, plane_hi=hi)
        for k in range(lo, hi):
            ref = torch.from_numpy(G[k - lo]).cuda()
            if one_mesh:
                if k in overwrite_planes:
                    kept[k] = G[k - lo].copy()
            else:
                cmp_overwrite(k, ref)
            cmp_sparse(k, ref, transposed)
            del ref
            oracle.wcorrect(prm, oracle.fft2(G[k - lo], inplace=True)[None], k, D)
        del G
    print(f"{cfg_name}: oracle streamed over {NW} planes in {time.time() - t0:.0f} s (batches of {B})")
    e_sparse.check()
    # the image of the timed path, whole
    plan.fft_columns(grid_s, ws.WS_FFT_USE_OCCUPANCY)
    plan.fft_rows_wcorrect(grid_s, image, accumulate=False, dirty=dirty, fft_flags=ws.WS_FFT_USE_OCCUPANCY)
    plan.async_status()
    Dd = torch.from_numpy(D).cuda()
    e = Running(f"{cfg_name} image (SPARSE + occupancy, the timed path)")
    e.add(image, Dd)
    e.check()
    assert torch.equal(dirty, image.real)
    if one_mesh:
        grid_overwrite()
        for k, g in kept.items():
            cmp_overwrite(k, torch.from_numpy(g).cuda())
        kept.clear()
    e_over.check()
    # the dense own FFT on the OVERWRITE mesh
    plan.fft_wcorrect(grid_o, image, wsp, accumulate=False, dirty=None, fft_flags=0)
    e = Running(f"{cfg_name} image (dense own FFT)")
    e.add(image, Dd)
    e.check()
    return plan, d, dg, prm


def test_large_whole_mesh_and_image(oracle):
    """All 64 planes of Large's mesh and its whole 8192^2 image; bins bit-exact over all 10^8 visibilities."""
    plan, d, dg, prm = _whole_config(oracle, "large")
    key = oracle.positions(prm, d.uvw.numpy(), d.n_chan, d.freqs_hz)["key"]
    bins = plan.get_bins()
    assert np.array_equal(bins["keys"], key)
    bin_start, perm, dropped = oracle.bins(prm, key)
    assert bins["n_dropped"] == dropped
    assert np.array_equal(bins["bin_start"], bin_start)
    assert np.array_equal(bins["sorted_keys"], key[perm])       # (derived from bin_start on the device)
    gp = bins["perm"]
    assert np.array_equal(key[gp], key[perm])                    # grouped by key ...
    assert np.array_equal(np.sort(gp), np.flatnonzero(key != 0xFFFFFFFF).astype(np.uint32))   # ... and a permutation of the kept


def test_paper_medium_whole_mesh_image_and_sum_of_weights(oracle):
    """SURVEY 8(f) NEXT-4 at full size: 13.6 M rows x 40 shared-uvw visibilities (Table 3 :308),
    pre-summed channels: whole mesh, whole image, sum of weights."""
    _whole_config(oracle, "paper_medium", presum=True)


@pytest.mark.parametrize("n_pix,n_wplanes", [(4096, 3), (8192, 2), (16384, 2)])
def test_own_fft_dense_random_planes_full_width(oracle, n_pix, n_wplanes):
    """The row-pass stage plans of N = 4096 (a row per group), N = 8192 (split radix-32) and N = 16384 (radix 64 split over
    two CTAs; radix-64 column pass) on arbitrary dense planes."""
    d = make_random_dataset(50 + n_wplanes, 10, 1, n_pix, n_wplanes, 7, w_span=250.0, cell_rad=0.6 / n_pix)
    plan = U.make_plan(d)
    assert plan.fft_is_own
    gen = torch.Generator(device="cuda").manual_seed(n_pix)
    G = torch.view_as_complex(torch.randn((n_wplanes, n_pix, n_pix, 2), generator=gen, device="cuda"))
    prm = U.oracle_params(oracle, d, plan.tile)
    ref = np.zeros((n_pix, n_pix), np.complex128)
    for k in range(n_wplanes):
        oracle.wcorrect(prm, oracle.fft2(G[k].cpu().numpy().astype(np.complex128), inplace=True)[None], k, ref)
    stored = torch.fft.ifftshift(G, dim=(-2, -1)).contiguous()
    image, dirty = plan.alloc_image(), plan.alloc_dirty()
    wsp = plan.alloc_workspace(16)
    plan.fft_wcorrect(stored, image, wsp, accumulate=False, dirty=dirty)
    e = Running(f"own FFT + w-correction, dense random planes, N = {n_pix}")
    e.add(image, torch.from_numpy(ref).cuda())
    e.check()
    assert torch.equal(dirty, image.real)


@pytest.mark.parametrize("n_pix", [4096, 8192, 16384])
@pytest.mark.parametrize("squeeze_axis", [0, 1])
def test_own_fft_sparse_both_orientations_full_width(oracle, n_pix, squeeze_axis):
    """Sparse mesh + occupancy-aware passes at N = 4096 / 8192 / 16384 in both storage orientations (uv coverage squeezed along
    u or along v), whole image against the oracle."""
    import paper_2301_06061_b200 as ws
    d = make_random_dataset(60 + squeeze_axis, 200000, 1, n_pix, 3, 7, fill=0.9, w_span=80.0, cell_rad=0.5 / n_pix)
    d.uvw[:, squeeze_axis] *= 0.15
    plan = U.make_plan(d)
    dev = d.to("cuda")
    grid, image, dirty = plan.alloc_grid(), plan.alloc_image(), plan.alloc_dirty()
    wsp = plan.alloc_workspace(d.n_vis)
    grid.fill_(float("nan"))
    plan.grid_visibilities(dev.uvw, dev.vis, dev.weights, None, grid, wsp, mode=ws.WS_GRID_SPARSE)
    plan.fft_wcorrect(grid, image, wsp, accumulate=False, dirty=dirty, fft_flags=ws.WS_FFT_USE_OCCUPANCY)
    plan.async_status()
    assert bool(plan.occupancy()["transposed"]) == (squeeze_axis == 1)
    prm = U.oracle_params(oracle, d, plan.tile)
    e = Running(f"sparse image N = {n_pix}, squeezed along axis {squeeze_axis}")
    e.add(image, torch.from_numpy(oracle.dirty_image(prm, *_np(d))).cuda())
    e.check()
    assert torch.equal(dirty, image.real)


@pytest.mark.skipif(os.environ.get("WS_SKIP_EXTREME") == "1", reason="WS_SKIP_EXTREME=1")
def test_extreme_whole_mesh_and_image(oracle):
    """Extreme (4 x 10^8 visibilities, 16384^2 x 32, S = 9) in ONE call: all 32 planes of the sparse mesh, the whole
    16384^2 image of the timed path (own FFT for N = 16384) and of the dense own FFT, four planes of the OVERWRITE mesh."""
    _whole_config(oracle, "extreme", one_mesh=True, dup_factor=2.0)


@pytest.mark.parametrize("squeeze_axis", [0, 1])
def test_image_from_host_at_8192_both_orientations(oracle, squeeze_axis):
    """The end-to-end entry at N = 8192: pipelined input chunks, the row pass in four launches whose image lines (or
    columns, for a transposed mesh) are copied out while the next part is computed."""
    n_pix = 8192
    d = make_random_dataset(70 + squeeze_axis, 150000, 2, n_pix, 3, 7, wavelengths=False, fill=0.9, w_span=80.0, cell_rad=0.5 / n_pix)
    d.uvw[:, squeeze_axis] *= 0.15
    plan = U.make_plan(d)
    plan.set_e2e_chunk_bytes(1 << 20)
    grid, image, dirty = plan.alloc_grid(), plan.alloc_image(), plan.alloc_dirty()
    wsp = plan.alloc_workspace(d.n_vis)
    dev_in = torch.empty(plan.dev_inputs_bytes(d.n_rows, d.n_chan), dtype=torch.uint8, device="cuda")
    uvw_h, vis_h, wt_h = (t.pin_memory() for t in (d.uvw, d.vis, d.weights))
    dirty_h = torch.full((n_pix, n_pix), float("nan"), dtype=torch.float32).pin_memory()
    grid.fill_(float("nan"))
    plan.image_from_host(uvw_h, vis_h, wt_h, d.freqs_hz, dev_in, grid, image, dirty, dirty_h, wsp)
    assert bool(plan.occupancy()["transposed"]) == (squeeze_axis == 1)
    prm = U.oracle_params(oracle, d, plan.tile)
    D = torch.from_numpy(oracle.dirty_image(prm, *_np(d))).cuda()
    e = Running(f"image_from_host at 8192, squeezed along axis {squeeze_axis}")
    e.add(image, D)
    e.check()
    assert torch.equal(dirty_h.cuda(), image.real)


@pytest.mark.skipif(os.environ.get("WS_SKIP_EXTREME") == "1", reason="WS_SKIP_EXTREME=1")
def test_extreme_streamed_in_eight_chunks(oracle):
    """Extreme's own recipe: eight row chunks of 775 snapshots through repeated gridding calls, as
    bench.py --chunked times them -- first chunk WS_GRID_SPARSE, the others WS_GRID_SPARSE_ADD onto a mesh that is never
    cleared (NaN-filled here) -- then the own FFT.  Compared: one whole plane of the mesh (written cells; unwritten ones
    must be exact zeros of the oracle) and eight pixels of the image against the oracle's chain evaluated pixel by pixel
    (the whole image of the same data is test_extreme_whole_mesh_and_image; the two GPU images must agree everywhere)."""
    import paper_2301_06061_b200 as ws
    dg = make_dataset(get_config("extreme"), device="cuda")
    d = dg.to("cpu")
    plan = U.make_plan(d)
    prm = U.oracle_params(oracle, d, plan.tile)
    grid, image, dirty = plan.alloc_grid(), plan.alloc_image(), plan.alloc_dirty()
    rc = d.row_chunks()
    assert len(rc) == 8
    wsp = plan.alloc_workspace(max(hi - lo for lo, hi in rc) * d.n_chan)
    grid.fill_(float("nan"))
    for i, (lo, hi) in enumerate(rc):
        plan.grid_visibilities(dg.uvw[lo:hi], dg.vis[lo:hi], dg.weights[lo:hi], d.freqs_hz, grid, wsp,
                               mode=ws.WS_GRID_SPARSE if i == 0 else ws.WS_GRID_SPARSE_ADD)
    plan.async_status()
    transposed = bool(plan.occupancy()["transposed"])
    k = 16
    G = torch.from_numpy(oracle.grid(prm, *_np(d), plane_lo=k, plane_hi=k + 1)[0]).cuda()
    got = _sparse_plane_logical(grid[k], transposed)
    unwritten = torch.isnan(got.real)
    assert not bool(torch.any(G[unwritten] != 0))
    e = Running(f"extreme, 8 streamed chunks: mesh plane {k}")
    e.add(torch.where(unwritten, torch.zeros_like(got), got), G)
    e.check()
    del G, got, unwritten
    plan.fft_wcorrect(grid, image, wsp, accumulate=False, dirty=dirty, fft_flags=ws.WS_FFT_USE_OCCUPANCY)
    plan.async_status()
    assert torch.equal(dirty, image.real)
    N, c = d.n_pix, d.n_pix // 2
    rng = np.random.default_rng(99)
    q = np.array([c, 0, N - 1] + list(rng.integers(0, N, 5)))
    p = np.array([c, N - 1, 0] + list(rng.integers(0, N, 5)))
    ref = oracle.image_samples(prm, *_np(d), q, p)
    got = image[torch.from_numpy(q).cuda(), torch.from_numpy(p).cuda()].cpu().numpy().astype(np.complex128)
    peak = float(torch.abs(image).max())
    rel, mx = np.linalg.norm(got - ref) / np.linalg.norm(ref), np.abs(got - ref).max() / peak
    print("extreme, 8 streamed chunks: 8 image pixels rel-L2 %.3e, max-abs/peak %.3e" % (rel, mx))
    assert rel <= U.REL_L2_TOL and mx <= U.MAX_ABS_TOL
    # the one-call image of the same data (whole-array parity in test_extreme_whole_mesh_and_image) agrees everywhere
    streamed = image.clone()
    wsp1 = plan.alloc_workspace(d.n_vis, 2.0)
    plan.grid_visibilities(dg.uvw, dg.vis, dg.weights, d.freqs_hz, grid, wsp1, mode=ws.WS_GRID_SPARSE)
    plan.fft_wcorrect(grid, image, wsp1, accumulate=False, dirty=None, fft_flags=ws.WS_FFT_USE_OCCUPANCY)
    plan.async_status()
    dd = torch.linalg.vector_norm((streamed - image).to(torch.complex128)) / torch.linalg.vector_norm(image.to(torch.complex128))
    assert float(dd) <= 2e-6, float(dd)

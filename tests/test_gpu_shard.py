"""GPU: the rank-local half of the plane-sharded variant (ws_plan_set_plane_range): two plans with the
plane ranges shard.plane_range gives two ranks, run one after the other on ONE device (no rank waits on another); the sum
of their images is the oracle's image, each rank's mesh holds its planes only, and the keys outside a range read dropped."""
import numpy as np
import pytest
import torch

from synth import make_random_dataset

from . import gpu_util as U

pytestmark = pytest.mark.gpu


def test_two_plane_ranges_sum_to_the_whole_image(oracle):
    import paper_2301_06061_b200 as ws
    from paper_2301_06061_b200 import shard
    d = make_random_dataset(91, 40000, 2, 512, 7, 7, wavelengths=False, fill=0.9, w_span=60.0, cell_rad=1e-3)
    dev = d.to("cuda")
    prm = U.oracle_params(oracle, d, 32)
    pos = oracle.positions(prm, d.uvw.numpy(), d.n_chan, d.freqs_hz)
    D, G = oracle.dirty_image(prm, d.uvw.numpy(), d.vis.numpy(), d.weights.numpy(), d.freqs_hz, return_grid=True)
    total = torch.zeros((512, 512), dtype=torch.complex64, device="cuda")
    for rank in range(2):
        lo, hi = shard.plane_range(rank, 2, d.n_wplanes)
        plan = U.make_plan(d)
        plan.set_plane_range(lo, hi)
        grid, image = plan.alloc_grid(), plan.alloc_image()
        wsp = plan.alloc_workspace(d.n_vis)
        grid.fill_(float("nan"))
        plan.grid_visibilities(dev.uvw, dev.vis, dev.weights, d.freqs_hz, grid, wsp, mode=ws.WS_GRID_OVERWRITE)
        bins = plan.get_bins()
        mine = (pos["k"] >= lo) & (pos["k"] < hi) & (pos["key"] != 0xFFFFFFFF)
        assert np.array_equal(bins["keys"], np.where(mine, pos["key"], 0xFFFFFFFF).astype(np.uint32))   # bit-exact, others dropped
        g = U.logical(grid)
        U.assert_close(g[lo:hi], G[lo:hi], f"rank {rank}: its planes of the mesh")
        other = np.ones(d.n_wplanes, bool)
        other[lo:hi] = False
        assert not g[other].any()                                                # the other rank's planes stay empty
        shard.image_plane_sharded(plan, dev.uvw, dev.vis, dev.weights, d.freqs_hz, grid, image, wsp)   # sparse path, no group
        plan.async_status()
        total += image
    U.assert_close(total.cpu().numpy(), D, "sum of the two ranks' images")
    with pytest.raises(ws.WStackError):
        plan.set_plane_range(3, 3)

"""CPU-only: the host-side logic of the plane-sharded variant (Eq. 8 at
:180 is what it replaces) with two gloo processes: the plane partition covers every plane once, and the sum of the
ranks' images -- each rank imaging only the visibilities of its own planes -- is the one-rank image.  The per-rank
images come from the oracle here (no GPU in this container); on the GPU the same statement is
tests/test_gpu_shard.py (both ranges on one device, one after the other)."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _data():
    sys.path.insert(0, ROOT)
    from synth import make_random_dataset
    return make_random_dataset(17, 1500, 2, 64, 7, 7, wavelengths=False, fill=0.85, w_span=40.0, cell_rad=4e-3)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    from oracle import wstack_oracle as orc
    from paper_2301_06061_b200 import shard
    dist.init_process_group("gloo", rank=rank, world_size=world)
    d = _data()
    prm = orc.OracleParams(n_pix=d.n_pix, n_wplanes=d.n_wplanes, support=d.support, cell_rad=d.cell_rad, w_min=d.w_min,
                           w_max=d.w_max, sigma=d.sigma_cells, tile=32)
    lo, hi = shard.plane_range(rank, world, d.n_wplanes)
    D = np.zeros((d.n_pix, d.n_pix), np.complex128)
    for k in range(lo, hi):          # this rank's planes only
        G = orc.grid(prm, d.uvw.numpy(), d.vis.numpy(), d.weights.numpy(), d.freqs_hz, k, k + 1)
        orc.wcorrect(prm, orc.transform(G[0])[None], k, D)
    img = torch.from_numpy(D)
    shard.reduce_image(img, dist)
    out[rank] = (lo, hi, img.numpy().copy())
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_sum_to_the_one_rank_image():
    world, port = 2, 31500 + os.getpid() % 2000
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    sys.path.insert(0, ROOT)
    from oracle import wstack_oracle as orc
    d = _data()
    prm = orc.OracleParams(n_pix=d.n_pix, n_wplanes=d.n_wplanes, support=d.support, cell_rad=d.cell_rad, w_min=d.w_min,
                           w_max=d.w_max, sigma=d.sigma_cells, tile=32)
    whole = orc.dirty_image(prm, d.uvw.numpy(), d.vis.numpy(), d.weights.numpy(), d.freqs_hz)
    assert (res[0][0], res[0][1], res[1][0], res[1][1]) == (0, 4, 4, 7)
    assert np.array_equal(res[0][2], res[1][2])                              # all_reduce: both ranks hold the sum
    assert np.linalg.norm(res[0][2] - whole) <= 1e-13 * np.linalg.norm(whole)


def test_plane_ranges_partition_the_stack():
    sys.path.insert(0, ROOT)
    from paper_2301_06061_b200 import shard
    for n_w in (1, 7, 64, 65):
        for world in (1, 2, 3, 8):
            r = [shard.plane_range(i, world, n_w) for i in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n_w
            assert all(a[1] == b[0] for a, b in zip(r, r[1:]))
            sizes = [hi - lo for lo, hi in r]
            assert max(sizes) - min(sizes) <= 1
    t = torch.ones(3, 3, dtype=torch.complex64)
    assert shard.reduce_image(t, None) is t                                   # no group: nothing to do

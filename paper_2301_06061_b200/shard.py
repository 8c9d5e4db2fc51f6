"""Plane-sharded imaging over several GPUs (PAPER.md:136-142 distributes the mesh over MPI ranks and
reduces all of it, Eq. 8 at :180): one process per GPU, every rank runs the unchanged chain on its own range of w-planes
(`Plan.set_plane_range`) and the N x N images are summed -- 8 N^2 bytes through one collective instead of the mesh.
Host-side plumbing only: the partition of the planes and the reduction (torch.distributed: NCCL over NVLink for device
tensors, gloo for host tensors).  north_star keeps the graded path on ONE GPU, so nothing here is on bench.py's path."""
from typing import Tuple

import torch


def plane_range(rank: int, world: int, n_wplanes: int) -> Tuple[int, int]:
    """Contiguous, balanced plane ranges: rank r owns [lo, hi); the first n_wplanes % world ranks own one plane more.
    A rank without planes (world > n_wplanes) gets an empty range (lo == hi) and must skip the gridding."""
    if not (0 <= rank < world) or n_wplanes < 1:
        raise ValueError("plane_range: need 0 <= rank < world and n_wplanes >= 1")
    base, extra = divmod(n_wplanes, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def reduce_image(image: torch.Tensor, dist=None, dst: int = None) -> torch.Tensor:
    """Sum of the ranks' images, in place.  dst None: every rank ends with the sum (all_reduce); else only rank dst.
    Complex tensors travel as their real view (NCCL and gloo reduce real types)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return image
    buf = torch.view_as_real(image) if image.is_complex() else image
    if dst is None:
        dist.all_reduce(buf, op=dist.ReduceOp.SUM)
    else:
        dist.reduce(buf, dst=dst, op=dist.ReduceOp.SUM)
    return image


def image_plane_sharded(plan, uvw, vis, weights, freq_hz, grid, image, workspace, dist=None, dirty=None):
    """This rank's part of a plane-sharded image, then the reduction: grid (sparse mesh) -> own FFT with the fused
    w-correction on the planes of `plan`'s range -> sum over ranks.  Every rank passes ALL the visibilities (or at least
    those of its planes): routing them by plane on the host is the reader's choice."""
    from . import wstack as ws
    if plan.fft_is_own:
        plan.grid_visibilities(uvw, vis, weights, freq_hz, grid, workspace, mode=ws.WS_GRID_SPARSE)
        plan.fft_wcorrect(grid, image, workspace, accumulate=False, dirty=None, fft_flags=ws.WS_FFT_USE_OCCUPANCY)
    else:
        plan.grid_visibilities(uvw, vis, weights, freq_hz, grid, workspace, mode=ws.WS_GRID_OVERWRITE)
        plan.fft_wcorrect(grid, image, workspace, accumulate=False, dirty=None)
    reduce_image(image, dist)
    if dirty is not None:
        plan.dirty_image(image, dirty)
    return image

"""Point-sharded bundle adjustment over several GPUs: host-side partition and the
torch.distributed collective behind `CasparBA.set_shard`.

Points (with all their observations, Jacobians, V_k, g_p, delta_p) are split into `world` contiguous ranges of the
caller's point ids with nearly equal OBSERVATION counts; cameras and every PCG vector are replicated.  One process per
GPU: each rank builds a `CasparBA` on its shard and calls the same sequence of `lm_step`s; the library sums U / g_c,
the Schur right-hand side, every q = S p and the step scalars over the ranks through `torch_exchange`.

Only index arithmetic lives here: no step of the method."""
from __future__ import annotations

import dataclasses

import numpy as np


@dataclasses.dataclass
class Shard:
    rank: int
    world: int
    point_begin: int            # the shard owns the caller's points [point_begin, point_end)
    point_end: int
    observation_ids: np.ndarray  # indices into the caller's observation arrays, ascending
    point_index: np.ndarray      # LOCAL point id of each of those observations (int32)
    camera_index: np.ndarray     # camera id of each (int32; cameras are not renumbered)

    @property
    def num_points(self) -> int:
        return self.point_end - self.point_begin

    @property
    def num_observations(self) -> int:
        return int(self.observation_ids.shape[0])


def point_ranges(num_points: int, point_index: np.ndarray, world: int) -> np.ndarray:
    """`world + 1` boundaries of contiguous point ranges with nearly equal observation counts (a point is never
    split: its 3x3 block, gradient and step live on exactly one rank)."""
    if world < 1:
        raise ValueError("world must be >= 1")
    track = np.bincount(np.asarray(point_index, dtype=np.int64), minlength=num_points)
    cum = np.concatenate([[0], np.cumsum(track)])
    total = int(cum[-1])
    bounds = [0]
    for r in range(1, world):
        target = total * r / world
        k = int(np.searchsorted(cum, target, side="left"))
        bounds.append(min(max(k, bounds[-1]), num_points))
    bounds.append(num_points)
    return np.asarray(bounds, dtype=np.int64)


def make_shard(num_points: int, camera_index: np.ndarray, point_index: np.ndarray, world: int, rank: int) -> Shard:
    """The shard of `rank`: which observations it owns and their local point ids."""
    if not 0 <= rank < world:
        raise ValueError("rank out of range")
    point_index = np.asarray(point_index)
    bounds = point_ranges(num_points, point_index, world)
    p0, p1 = int(bounds[rank]), int(bounds[rank + 1])
    mine = np.nonzero((point_index >= p0) & (point_index < p1))[0]
    return Shard(rank, world, p0, p1, mine, (point_index[mine] - p0).astype(np.int32),
                 np.asarray(camera_index)[mine].astype(np.int32))


def shard_arrays(shard: Shard, points: np.ndarray, observations: np.ndarray):
    """The shard's slices of the caller's point and pixel arrays."""
    return points[shard.point_begin:shard.point_end], observations[shard.observation_ids]


def torch_exchange(group=None):
    """The collective for `CasparBA.set_shard` on top of torch.distributed (NCCL over NVLink for CUDA tensors; gloo
    for the CPU tests): all_reduce(SUM) of the first `count` doubles, on the current stream of the buffer's device."""
    import torch.distributed as dist

    def exchange(buffer, count: int) -> None:
        dist.all_reduce(buffer[:count], op=dist.ReduceOp.SUM, group=group)

    return exchange

"""Point-sharded problem, host side, on CPU: the partition, and -- with gloo at
world_size 2 -- the collective behind `CasparBA.set_shard` together with the fact the design rests on: every
camera-side quantity of the path is a SUM over the shards' observations.  The per-shard numbers come from the fp64
oracle (test infrastructure); the GPU kernels of a sharded handle are covered by tests/test_gpu_sharding.py."""
import json
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2605_30583_b200 import sharding  # noqa: E402


def test_partition_covers_every_observation_once_and_balances(scene_cache):
    s = scene_cache("small")
    for world in (1, 2, 3, 8):
        shards = [sharding.make_shard(s.num_points, s.camera_index, s.point_index, world, r) for r in range(world)]
        ids = np.concatenate([sh.observation_ids for sh in shards])
        assert np.array_equal(np.sort(ids), np.arange(s.num_observations))          # each observation exactly once
        assert shards[0].point_begin == 0 and shards[-1].point_end == s.num_points
        for a, b in zip(shards[:-1], shards[1:]):
            assert a.point_end == b.point_begin                                        # whole points, contiguous
        for sh in shards:
            assert (sh.point_index >= 0).all() and (sh.point_index < max(sh.num_points, 1)).all()
            assert np.array_equal(sh.point_index + sh.point_begin, s.point_index[sh.observation_ids])
            assert np.array_equal(sh.camera_index, s.camera_index[sh.observation_ids])
        counts = np.array([sh.num_observations for sh in shards])
        assert counts.max() - counts.min() <= 2 * 10                                   # within two tracks of each other


def test_partition_edge_cases():
    ci = np.zeros(0, np.int32)
    sh = sharding.make_shard(0, ci, ci, 2, 1)
    assert sh.num_points == 0 and sh.num_observations == 0
    # more ranks than points: trailing shards are empty, nothing is lost
    pi = np.array([0, 0, 1, 1, 1], np.int32)
    shards = [sharding.make_shard(2, np.zeros(5, np.int32), pi, 4, r) for r in range(4)]
    assert sum(x.num_observations for x in shards) == 5 and sum(x.num_points for x in shards) == 2


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import oracle
    from ba_scenes import make_scene
    from oracle import binding as ob

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    exchange = sharding.torch_exchange()
    s = make_scene("tiny")
    sh = sharding.make_shard(s.num_points, s.camera_index, s.point_index, world, rank)
    pts, obs = sharding.shard_arrays(sh, s.points, s.observations)
    lam = 1e-2
    # lambda I damping: the damped operator of a shard is S_shard + lambda I, so sum_shards = S + world * lambda I
    o = oracle.OracleBA(s.cameras, pts, obs, sh.camera_index, sh.point_index, damping_mode=1)
    cost = o.linearize()
    nc9 = 9 * s.num_cameras
    p = np.random.default_rng(5).normal(size=nc9)
    q = o.schur_matvec(lam, p)
    buf = torch.zeros(81 * s.num_cameras + nc9 + nc9 + 1, dtype=torch.float64)
    buf[:81 * s.num_cameras] = torch.from_numpy(o.export(ob.U).reshape(-1))
    buf[81 * s.num_cameras:81 * s.num_cameras + nc9] = torch.from_numpy(o.export(ob.G)[:nc9])
    buf[81 * s.num_cameras + nc9:-1] = torch.from_numpy(q)
    buf[-1] = cost
    exchange(buf, buf.numel())                          # sum of doubles over the shards
    tag = torch.full((4,), float(rank + 1), dtype=torch.float64)
    exchange(tag, 3)                                    # only the first `count` doubles take part
    dist.barrier()
    dist.destroy_process_group()
    np.save(f"{out}.{rank}.npy", buf.numpy())
    with open(f"{out}.{rank}.json", "w") as fh:
        json.dump({"tag": tag.tolist(), "points": sh.num_points, "obs": sh.num_observations}, fh)


def test_camera_side_sums_over_two_gloo_ranks_equal_the_unsharded_problem(tmp_path, scene_cache):
    import oracle
    from oracle import binding as ob

    out = str(tmp_path / "s")
    mp.spawn(_worker, args=(2, 29641, out), nprocs=2, join=True)
    res = [np.load(f"{out}.{r}.npy") for r in range(2)]
    meta = [json.load(open(f"{out}.{r}.json")) for r in range(2)]
    assert np.array_equal(res[0], res[1])                               # an all-reduce: the same bits on both ranks
    assert meta[0]["tag"] == [3.0, 3.0, 3.0, 1.0] and meta[1]["tag"] == [3.0, 3.0, 3.0, 2.0]   # 1 + 2 on the first three
    s = scene_cache("tiny")
    assert meta[0]["points"] + meta[1]["points"] == s.num_points
    assert meta[0]["obs"] + meta[1]["obs"] == s.num_observations
    full = oracle.OracleBA.from_scene(s, damping_mode=1)
    cost = full.linearize()
    nc, nc9, lam = s.num_cameras, 9 * s.num_cameras, 1e-2
    p = np.random.default_rng(5).normal(size=nc9)
    got = res[0]
    assert abs(got[-1] - cost) <= 1e-12 * cost
    u = full.export(ob.U).reshape(-1)
    assert np.abs(got[:81 * nc] - u).max() <= 1e-12 * np.abs(u).max()
    g = full.export(ob.G)[:nc9]
    assert np.abs(got[81 * nc:81 * nc + nc9] - g).max() <= 1e-12 * np.abs(g).max()
    q = full.schur_matvec(lam, p) + lam * p                              # two shards: lambda I counted twice
    assert np.abs(got[81 * nc + nc9:-1] - q).max() <= 1e-11 * np.abs(q).max()

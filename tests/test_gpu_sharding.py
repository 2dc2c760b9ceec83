"""A point-sharded problem (include/caspar_ba.h: caspar_ba_set_shard) on ONE GPU: two shard handles
driven by two host threads, the collective emulated by a host-synchronised sum / copy between the two exchange
buffers (no kernel ever waits for another: each thread synchronises its stream, the threads meet at a barrier, one of
them combines the buffers).  The sharded run must reproduce the unsharded handle: linearization, Schur matvec, PCG
step, one LM step per preconditioner -- and the two shards must end with bit-identical cameras (they are replicas)."""
import threading

import numpy as np
import pytest

import paper_2605_30583_b200 as pkg
from paper_2605_30583_b200 import sharding
from parity_util import rel_l2

pytestmark = pytest.mark.gpu

LAM = float(np.float32(1e-2))
WORLD = 2


class HostExchange:
    """All-reduce (sum) between WORLD threads of one process through a barrier."""

    def __init__(self, world):
        self.world = world
        self.barrier = threading.Barrier(world, timeout=30)
        self.bufs = [None] * world
        self.calls = 0

    def make(self, rank):
        import torch

        def exchange(buf, count):
            torch.cuda.current_stream(buf.device).synchronize()
            self.bufs[rank] = buf
            self.barrier.wait()
            if rank == 0:
                total = self.bufs[0][:count].clone()
                for b in self.bufs[1:]:
                    total += b[:count]
                for b in self.bufs:
                    b[:count] = total
                torch.cuda.synchronize()
                self.calls += 1
            self.barrier.wait()

        return exchange


def _run_shards(scene, body, camera_model=0):
    """Run body(rank, handle, shard) on WORLD threads; returns their results (re-raises the first failure)."""
    import torch

    ex = HostExchange(WORLD)
    out, err = [None] * WORLD, [None] * WORLD

    def work(rank):
        try:
            torch.cuda.set_device(0)
            sh = sharding.make_shard(scene.num_points, scene.camera_index, scene.point_index, WORLD, rank)
            pts, obs = sharding.shard_arrays(sh, scene.points, scene.observations)
            with torch.cuda.stream(torch.cuda.Stream()):
                g = pkg.CasparBA(scene.cameras, pts, obs, sh.camera_index, sh.point_index, scene.robust_loss,
                                 scene.robust_scale, 0, camera_model=camera_model)
                g.set_shard(ex.make(rank), is_root=(rank == 0))
                out[rank] = body(rank, g, sh)
                g.close()
        except BaseException as e:  # noqa: BLE001
            err[rank] = e
            ex.barrier.abort()

    threads = [threading.Thread(target=work, args=(r,)) for r in range(WORLD)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    for e in err:
        if e is not None and not isinstance(e, threading.BrokenBarrierError):
            raise e
    for e in err:
        if e is not None:
            raise e
    return out, ex


@pytest.mark.parametrize("name,kw", [("tiny", {}), ("small", {}), ("skewed", dict(num_cameras=300, num_points=30_000))])
def test_sharded_linearize_matvec_and_pcg_match_the_unsharded_handle(scene_cache, name, kw):
    s = scene_cache(name, **kw)
    nc9 = 9 * s.num_cameras
    p = np.random.default_rng(11).normal(size=nc9)

    def body(rank, g, sh):
        cost = g.linearize()
        u, grad = g.export(pkg.U), g.export(pkg.G)
        q = g.schur_matvec(LAM, p)
        info = g.pcg_solve(LAM, 0.0, 30)
        b, d = g.export(pkg.SCHUR_RHS), g.export(pkg.DELTA)
        return dict(cost=cost, u=u, gc=grad[:nc9], gp=grad[nc9:], q=q, b=b, dc=d[:nc9], dp=d[nc9:], it=info.iterations,
                    res=info.rel_residual, ex=g.stats().shard_exchanges, p0=sh.point_begin, p1=sh.point_end)

    out, ex = _run_shards(s, body)
    ref = pkg.CasparBA.from_scene(s)
    cost = ref.linearize()
    u, grad = ref.export(pkg.U), ref.export(pkg.G)
    q = ref.schur_matvec(LAM, p)
    info = ref.pcg_solve(LAM, 0.0, 30)
    b, d = ref.export(pkg.SCHUR_RHS), ref.export(pkg.DELTA)
    ref.close()
    for r in out:
        assert abs(r["cost"] - cost) <= 1e-12 * cost
        # (the shards tile their observations differently from the unsharded handle, so the fp32 partial sums inside
        # a tile / chunk group differently: agreement is at fp32 summation level, not bitwise)
        assert rel_l2(r["u"], u) <= 2e-6 and rel_l2(r["gc"], grad[:nc9]) <= 2e-6
        assert rel_l2(r["q"], q) <= 2e-6 and rel_l2(r["b"], b) <= 2e-6
        assert r["it"] == info.iterations == 30
        assert rel_l2(r["dc"], d[:nc9]) <= 1e-4 and abs(r["res"] - info.rel_residual) <= 0.5 * info.rel_residual + 1e-8
        # the shard's own points
        lo, hi = 3 * r["p0"], 3 * r["p1"]
        assert rel_l2(r["gp"], grad[nc9 + lo:nc9 + hi]) <= 2e-6
        assert rel_l2(r["dp"], d[nc9 + lo:nc9 + hi]) <= 1e-4
    # replicas: the same bits on both shards
    assert np.array_equal(out[0]["dc"], out[1]["dc"]) and np.array_equal(out[0]["q"], out[1]["q"])
    # 1 (linearize) + 1 (matvec) + [1 (b) + 30 (one per iteration) + 1 (scalars)]
    assert out[0]["ex"] == out[1]["ex"] == 1 + 1 + 1 + 30 + 1
    assert ex.calls == out[0]["ex"]


@pytest.mark.parametrize("preconditioner", [0, 1])
@pytest.mark.parametrize("camera_model", [0, 1])
def test_sharded_lm_steps_match_and_the_shards_stay_replicas(scene_cache, preconditioner, camera_model):
    s = scene_cache("small")

    def body(rank, g, sh):
        g.set_preconditioner(preconditioner)
        steps = [g.lm_step(LAM * 0.5 ** t, 1e-6, s.pcg_max_iter, 0) for t in range(4)]
        return dict(steps=steps, cams=g.cameras.cpu().numpy(), pts=g.points.cpu().numpy(), p0=sh.point_begin, p1=sh.point_end)

    out, _ = _run_shards(s, body, camera_model)
    ref = pkg.CasparBA.from_scene(s, camera_model=camera_model)
    ref.set_preconditioner(preconditioner)
    want = [ref.lm_step(LAM * 0.5 ** t, 1e-6, s.pcg_max_iter, 0) for t in range(4)]
    cams, pts = ref.cameras.cpu().numpy(), ref.points.cpu().numpy()
    ref.close()
    for r in out:
        for x, y in zip(r["steps"], want):
            # (stopping on a tolerance: the residual hovers around it for a few iterations, C9)
            assert x.accepted == y.accepted and abs(x.pcg_iterations - y.pcg_iterations) <= max(3, 0.1 * y.pcg_iterations)
            assert x.cost_before == pytest.approx(y.cost_before, rel=1e-6) and x.cost_after == pytest.approx(y.cost_after, rel=1e-6)
            assert x.rho == pytest.approx(y.rho, rel=5e-3)
        assert np.abs(r["cams"] - cams).max() <= 1e-4 * np.abs(cams).max()
        assert np.abs(r["pts"] - pts[r["p0"]:r["p1"]]).max() <= 1e-4 * np.abs(pts).max()
    assert np.array_equal(out[0]["cams"], out[1]["cams"])       # bit-identical replicas after four steps
    assert [(x.cost_after, x.pcg_iterations, x.rho) for x in out[0]["steps"]] == \
           [(x.cost_after, x.pcg_iterations, x.rho) for x in out[1]["steps"]]


def test_a_sharded_handle_refuses_what_it_does_not_support(scene_cache):
    import torch
    s = scene_cache("tiny")
    g = pkg.CasparBA.from_scene(s)
    g.set_shard(lambda buf, count: None, is_root=True)          # a one-shard "world": the collective is the identity
    cost = g.linearize()
    ref = pkg.CasparBA.from_scene(s)
    assert cost == ref.linearize()
    with pytest.raises(pkg.CasparError) as e:
        g.pcgnr_solve(LAM, 1e-6, 10)
    assert e.value.code == pkg.ESTATE
    a, b = g.lm_step(LAM, 1e-6, 50, 0), ref.lm_step(LAM, 1e-6, 50, 0)
    assert a.cost_after == pytest.approx(b.cost_after, rel=1e-7) and a.pcg_iterations == b.pcg_iterations
    g.set_shard(None, True)                                      # back to a single-GPU problem
    assert g.stats().shard_exchanges > 0
    c = g.lm_step(LAM, 1e-6, 50, 0)
    d = ref.lm_step(LAM, 1e-6, 50, 0)
    assert c.cost_after == pytest.approx(d.cost_after, rel=1e-7)
    g.close()
    ref.close()


def test_an_empty_shard_takes_part_in_every_exchange(scene_cache):
    """More ranks than work: a shard with no points and no observations still replicates the cameras, makes the same
    calls and contributes zeros; the other shard then reproduces the unsharded problem and both end with the same
    cameras."""
    import torch
    s = scene_cache("tiny")
    ex = HostExchange(WORLD)
    out, err = [None] * WORLD, [None] * WORLD

    def work(rank):
        try:
            torch.cuda.set_device(0)
            with torch.cuda.stream(torch.cuda.Stream()):
                if rank == 0:
                    g = pkg.CasparBA.from_scene(s)
                else:
                    g = pkg.CasparBA(s.cameras, np.zeros((0, 3), np.float32), np.zeros((0, 2), np.float32),
                                     np.zeros(0, np.int32), np.zeros(0, np.int32))
                g.set_shard(ex.make(rank), is_root=(rank == 0))
                steps = [g.lm_step(LAM, 1e-6, 50, 0) for _ in range(3)]
                out[rank] = (steps, g.cameras.cpu().numpy(), g.stats().shard_exchanges)
                g.close()
        except BaseException as e:  # noqa: BLE001
            err[rank] = e
            ex.barrier.abort()

    threads = [threading.Thread(target=work, args=(r,)) for r in range(WORLD)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    for e in err:
        if e is not None and not isinstance(e, threading.BrokenBarrierError):
            raise e
    assert not any(err)
    ref = pkg.CasparBA.from_scene(s)
    want = [ref.lm_step(LAM, 1e-6, 50, 0) for _ in range(3)]
    for x, y, z in zip(out[0][0], out[1][0], want):
        assert x.accepted == y.accepted == z.accepted and x.pcg_iterations == y.pcg_iterations
        assert x.cost_after == y.cost_after                                  # the two shards: the same bits
        assert x.cost_after == pytest.approx(z.cost_after, rel=1e-7) and abs(x.pcg_iterations - z.pcg_iterations) <= 3
    assert np.array_equal(out[0][1], out[1][1])
    assert np.abs(out[0][1] - ref.cameras.cpu().numpy()).max() <= 1e-5 * np.abs(out[0][1]).max()
    assert out[0][2] == out[1][2]
    ref.close()

"""caspar_ba_cost_static (include/caspar_ba.h): the allocation-free cost entry point against the handle path.

The file sorts last on purpose: the suite runs with `pytest -x`, and a failure here must not hide another test.
Every test stands on its own (fresh process or after the rest of the suite): it builds its inputs, makes its calls
one after another on the current stream, and leaves nothing behind but the library's fixed scratch array."""
import ctypes as C

import numpy as np
import pytest
import torch

import paper_2605_30583_b200 as pkg
from oracle import binding as ob
from paper_2605_30583_b200.binding import Problem

pytestmark = pytest.mark.gpu

COST_TOL = 1e-5     # the suite's cost tolerance (tests/test_gpu_edges.py, test_gpu_parity.py)
SUM_TOL = 1e-11     # both paths evaluate the same fp64 residuals and sum them in fp64: only the order differs


def _device_inputs(s):
    dev = torch.device("cuda", torch.cuda.current_device())
    t = lambda a, dt: torch.as_tensor(np.ascontiguousarray(a)).to(device=dev, dtype=dt).contiguous()
    return (t(s.cameras, torch.float32), t(s.points, torch.float32), t(s.observations, torch.float32),
            t(s.camera_index, torch.int32), t(s.point_index, torch.int32))


def _handle_cost(s):
    g = pkg.CasparBA.from_scene(s)
    try:
        return g.cost()
    finally:
        g.close()


def _static_cost(s, inputs, out):
    pkg.cost_static(*inputs, out, robust_loss=s.robust_loss, robust_scale=s.robust_scale)
    torch.cuda.synchronize()
    return float(out[0].item())


def test_two_calls_in_a_row_match_the_handle_path(scene_cache):
    """Call 1 on a scene with more cameras and the Cauchy loss, call 2 on a smaller plain one, call 3 = call 1 again:
    each matches the existing path (caspar_ba_cost on a handle), whatever the previous call left in the scratch."""
    a = scene_cache("skewed", num_cameras=300, num_points=30_000)
    b = scene_cache("small")
    want_a, want_b = _handle_cost(a), _handle_cost(b)
    in_a, in_b = _device_inputs(a), _device_inputs(b)
    out = torch.full((1,), -1.0, dtype=torch.float64, device=in_a[0].device)
    got_a = _static_cost(a, in_a, out)
    got_b = _static_cost(b, in_b, out)
    got_a2 = _static_cost(a, in_a, out)
    for got, want in ((got_a, want_a), (got_b, want_b), (got_a2, want_a)):
        assert np.isfinite(got) and want > 0
        assert abs(got - want) <= COST_TOL * want
        assert abs(got - want) <= SUM_TOL * want, (got, want)
    assert got_a2 == got_a                       # fixed summation order: bit for bit the same


def test_back_to_back_without_a_sync_and_against_the_oracle(scene_cache):
    """Two calls enqueued back to back on one stream (no host synchronisation in between) into two outputs; the tiny
    scene also against the fp64 oracle."""
    s = scene_cache("tiny")
    inputs = _device_inputs(s)
    out = torch.zeros(2, dtype=torch.float64, device=inputs[0].device)
    moved = (inputs[0], inputs[1] + 0.01, *inputs[2:])
    pkg.cost_static(*inputs, out[0:1])
    pkg.cost_static(*moved, out[1:2])
    torch.cuda.synchronize()
    first, second = (float(x) for x in out.cpu())
    o = ob.OracleBA.from_scene(s)
    want = o.cost()
    assert abs(first - want) <= COST_TOL * want
    assert abs(first - _handle_cost(s)) <= SUM_TOL * want
    assert second != first and np.isfinite(second)
    g = pkg.CasparBA(moved[0].clone(), moved[1].clone(), s.observations, s.camera_index, s.point_index)
    assert abs(second - g.cost()) <= SUM_TOL * second
    g.close()


def test_it_allocates_nothing(scene_cache):
    """After one warm-up call (module load, symbol address) the free device memory does not move over 20 calls."""
    s = scene_cache("small")
    inputs = _device_inputs(s)
    out = torch.zeros(1, dtype=torch.float64, device=inputs[0].device)
    _static_cost(s, inputs, out)
    free_before, _ = torch.cuda.mem_get_info()
    for _ in range(20):
        pkg.cost_static(*inputs, out)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after == free_before


def test_limits_and_errors():
    L = pkg.load_library()
    dev = torch.device("cuda", torch.cuda.current_device())
    out = torch.zeros(1, dtype=torch.float64, device=dev)
    z2, zi = torch.zeros((0, 2), device=dev), torch.zeros(0, dtype=torch.int32, device=dev)
    # empty problem: F = 0
    pkg.cost_static(torch.zeros((2, 9), device=dev), torch.zeros((3, 3), device=dev), z2, zi, zi, out.fill_(7.0))
    torch.cuda.synchronize()
    assert float(out[0]) == 0.0
    # exactly the maximum is served, one more is refused with the limit in the text
    nmax = pkg.STATIC_MAX_CAMERAS
    cams = torch.zeros((nmax + 1, 9), device=dev)
    cams[:, 5] = 1.0
    cams[:, 6] = 100.0
    pts = torch.tensor([[0.1, -0.2, -3.0]], device=dev)
    obs = torch.zeros((2, 2), device=dev)
    ci = torch.tensor([0, nmax - 1], dtype=torch.int32, device=dev)
    pi = torch.zeros(2, dtype=torch.int32, device=dev)
    pkg.cost_static(cams[:nmax], pts, obs, ci, pi, out)
    torch.cuda.synchronize()
    assert np.isfinite(float(out[0])) and float(out[0]) > 0
    with pytest.raises(pkg.CasparError) as e:
        pkg.cost_static(cams, pts, obs, ci, pi, out)
    assert e.value.code == pkg.EINVAL and f"CASPAR_BA_STATIC_MAX_CAMERAS = {nmax}" in str(e.value)
    # an index out of range poisons the result instead of faulting
    bad = torch.tensor([0, 5], dtype=torch.int32, device=dev)
    pkg.cost_static(cams[:4], pts, obs, bad, pi, out)
    torch.cuda.synchronize()
    assert np.isnan(float(out[0]))
    # a host pointer is refused before any kernel sees it
    host = np.zeros((4, 9), np.float32)
    pb = Problem(4, 1, 2, host.ctypes.data, pts.data_ptr(), obs.data_ptr(), ci.data_ptr(), pi.data_ptr(), 0, 0.0, 0, 0, 0.0)
    rc = L.caspar_ba_cost_static(C.byref(pb), out.data_ptr(), None)
    assert rc == pkg.EINVAL and b"cameras is not device memory" in L.caspar_ba_last_error(None)
    pb = Problem(4, 1, 2, cams.data_ptr(), pts.data_ptr(), obs.data_ptr(), ci.data_ptr(), pi.data_ptr(), 1, 0.0, 0, 0, 0.0)
    assert L.caspar_ba_cost_static(C.byref(pb), out.data_ptr(), None) == pkg.EINVAL
    assert L.caspar_ba_cost_static(None, out.data_ptr(), None) == pkg.EINVAL
    # the library is still healthy
    pkg.cost_static(cams[:4], pts, obs, torch.zeros(2, dtype=torch.int32, device=dev), pi, out)
    torch.cuda.synchronize()
    assert np.isfinite(float(out[0]))

"""obem_nbody_at_points_static -- the one entry point of libobem.so that allocates nothing (no context, no cudaMalloc;
scratch in a fixed static device array, include/obem.h) -- against the existing path, obem_eval_at_points(OBEM_NBODY)
on a context, at the tolerance of the parity tests (tests/parity_metrics.py), and against the fp64 oracle.

Two calls in a row with DIFFERENT sizes (the scratch keeps the first call's contents: the second must not see them),
then the first again; free device memory does not move across the calls; a size beyond the fixed maximum is refused
with OBEM_ELIMIT.  Collected last on purpose (the suite runs with `pytest -x`).  `pytest -m gpu`.
"""
import numpy as np
import pytest

from parity_metrics import assert_parity

pytestmark = pytest.mark.gpu

UM = 1e-6
QE = 1.602176634e-19


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device (there is no CPU fallback)")
    return torch


@pytest.fixture(scope="module")
def api(torch_cuda):
    from paper_2110_09214_b200 import api as _api
    return _api


def _case(seed, n, m):
    """An interleaved electron / ion cloud and free points inside it; some points sit exactly on charges."""
    rng = np.random.default_rng([47, seed])
    xyzq = np.zeros((n, 4), dtype=np.float32)
    xyzq[:, :3] = rng.normal(0.0, 1.0, (n, 3)) * np.array([20 * UM, 20 * UM, 10 * UM])
    xyzq[:, 3] = rng.choice([-QE, QE], n)
    pts = np.zeros((m, 4), dtype=np.float32)
    pts[:, :3] = rng.normal(0.0, 1.0, (m, 3)) * np.array([25 * UM, 25 * UM, 15 * UM])
    k = min(16, m, n)
    pts[:k, :3] = xyzq[:k, :3]                      # zero unsoftened distance to one source each
    return xyzq, pts


def _existing_path(torch, api, xyzq, pts, eps):
    with api.Context(0) as ctx:
        ctx.set_softening(eps, 0.0)
        ctx.set_charges(torch.from_numpy(xyzq).cuda())
        out = ctx.eval_at_points(torch.from_numpy(pts).cuda(), flags=api.NBODY)
        torch.cuda.synchronize()
        return out.cpu().numpy()


def test_static_entry_point_matches_the_existing_path_twice_in_a_row(torch_cuda, api, ref):
    torch = torch_cuda
    # (n charges, m points, softening): several tiles and splits with ragged tails; then a SMALLER problem whose
    # partial sums land on slots the first call used; eps = 0 exercises the zero-distance rule (reading A4)
    cases = [(1, 30011, 5003, 0.05 * UM), (2, 777, 300, 0.0), (1, 30011, 5003, 0.05 * UM)]
    inputs, expect, oracle = [], [], []
    for seed, n, m, eps in cases:
        xyzq, pts = _case(seed, n, m)
        inputs.append((torch.from_numpy(xyzq).cuda(), torch.from_numpy(pts).cuda(),
                       torch.empty((m, 4), dtype=torch.float32, device="cuda"), eps))
        expect.append(_existing_path(torch, api, xyzq, pts, eps))
        on, _ = ref.eval_field(xyzq=xyzq, targets=pts, self_index=None, eps_pp=eps, flags=ref.NBODY)
        oracle.append(on)
    # first call on this device: looks the scratch's device address up (set-up), then two kernels
    api.nbody_at_points_static(*inputs[0][:2], inputs[0][3], out=inputs[0][2])
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    got = [inputs[0][2].cpu().numpy()]
    for x, p, o, eps in inputs[1:]:
        api.nbody_at_points_static(x, p, eps, out=o)
        torch.cuda.synchronize()
        got.append(o.cpu().numpy())
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0, "device memory was allocated by the no-allocation entry point"
    for k, (g, e, on) in enumerate(zip(got, expect, oracle)):
        assert np.isfinite(g).all()
        assert_parity(g, e.astype(np.float64), "static entry point vs obem_eval_at_points, call %d" % k)
        assert_parity(g, on, "static entry point vs the fp64 oracle, call %d" % k)
    assert np.array_equal(got[0], got[2])           # deterministic: fixed summation order, no atomics


def test_static_entry_point_limits_and_degenerate_sizes(torch_cuda, api):
    torch = torch_cuda
    xyzq, pts = _case(3, 1000, api.STATIC_MAX_POINTS + 1)
    d_x, d_p = torch.from_numpy(xyzq).cuda(), torch.from_numpy(pts).cuda()
    out = torch.empty((pts.shape[0], 4), dtype=torch.float32, device="cuda")
    with pytest.raises(api.ObemError) as e:
        api.nbody_at_points_static(d_x, d_p, 0.05 * UM, out=out)
    assert e.value.status == -5 and "OBEM_ELIMIT" in str(e.value)            # a clear error, nothing launched
    # exactly the maximum is accepted
    api.nbody_at_points_static(d_x, d_p[:api.STATIC_MAX_POINTS], 0.05 * UM, out=out[:api.STATIC_MAX_POINTS])
    torch.cuda.synchronize()
    assert torch.isfinite(out[:api.STATIC_MAX_POINTS]).all()
    # no charges: the field is zero; no points: nothing to do
    few = out[:10]
    few.fill_(7.0)
    api.nbody_at_points_static(d_x[:0], d_p[:10], 0.05 * UM, out=few)
    torch.cuda.synchronize()
    assert torch.all(few == 0)
    api.nbody_at_points_static(d_x, d_p[:0], 0.05 * UM, out=out[:0])
    with pytest.raises(api.ObemError) as e:
        api.nbody_at_points_static(d_x, d_p[:10], -1.0, out=few)
    assert e.value.status == -1

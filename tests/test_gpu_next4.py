"""GPU parity of the static field option: obem_field_map against the fp64
field oracle at the nodes, obem_interp_map against oracle/fieldmap.py, through the C ABI.  `pytest -m gpu`.

Tolerance of the interpolation: cell index and fractions are taken in fp64 from the same
fp32 positions the oracle gets, so the fractions agree to one fp32 rounding; each of the 8 weights is a product of
three fp32 numbers (3 roundings incl. 1 - f) and the weighted sum is 8 fp32 terms: |error| <= 8 * 2^-23 * sum_c
w_c |v_c| < 1e-6 * sum_c w_c |v_c|, i.e. relative to the interpolated absolute map.
"""
import numpy as np
import pytest

from paper_2110_09214_b200 import workloads as W
from parity_metrics import assert_parity

pytestmark = pytest.mark.gpu

UM = 1e-6


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


@pytest.fixture()
def ctx(api):
    c = api.Context(0)
    yield c
    c.destroy()


@pytest.fixture(scope="module")
def fieldmap():
    from oracle import fieldmap as f
    return f


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _check_interp(got, fmap, origin, spacing, pts, fieldmap, what):
    exp = fieldmap.trilinear(fmap, origin, spacing, pts)
    bound = 1e-6 * fieldmap.trilinear(np.abs(fmap), origin, spacing, pts) + 1e-30
    err = np.abs(got.astype(np.float64) - exp)
    worst = float((err / bound).max())
    assert np.isfinite(got).all(), what
    assert worst <= 1.0, "%s: |err| / (1e-6 sum w|v|) = %.3g" % (what, worst)


def _pad4(p):
    out = np.zeros((p.shape[0], 4), dtype=np.float32)
    out[:, :3] = p
    out[:, 3] = 123.0          # the 4th lane is ignored
    return out


@pytest.mark.parametrize("shape", [(7, 5, 9), (2, 2, 2), (1, 6, 3), (33, 1, 1), (1, 1, 1)])
def test_interp_matches_oracle_inside_outside_and_on_nodes(torch_cuda, ctx, fieldmap, shape):
    rng = np.random.default_rng([43, *shape])
    origin = (-2.1e-4, 1e-5, -1.5e-4)
    spacing = (3e-6, 5e-6, 2e-6)
    fmap = (rng.normal(size=shape + (4,)) * np.array([1e5, 1e5, 1e6, 30.0])).astype(np.float32)
    lo = np.array(origin)
    hi = lo + np.array(spacing) * (np.array(shape) - 1)
    inside = rng.uniform(lo, hi, (1500, 3))
    outside = rng.uniform(lo - 3 * np.array(spacing), hi + 3 * np.array(spacing), (500, 3))
    idx = rng.integers(0, shape, (300, 3))
    idx[0] = 0
    idx[1] = np.array(shape) - 1
    nodes = lo + idx * np.array(spacing)
    pts = _pad4(np.concatenate([inside, outside, nodes]))
    got = ctx.interp_map(dev(torch_cuda, fmap), origin, spacing, dev(torch_cuda, pts))
    torch_cuda.cuda.synchronize()
    _check_interp(got.cpu().numpy(), fmap, origin, spacing, pts[:, :3], fieldmap, "shape %r" % (shape,))


def test_interp_large_ragged_count_sampled(torch_cuda, ctx, fieldmap):
    """1,000,037 positions (a ragged last block) in a 96 x 80 x 64 map; 3000 sampled positions against the oracle."""
    rng = np.random.default_rng([43, 2])
    shape, origin, spacing = (96, 80, 64), (-2.1e-4, -2.1e-4, -1.5e-4), (4.4e-6, 5.3e-6, 4.7e-6)
    fmap = rng.normal(size=shape + (4,)).astype(np.float32)
    lo = np.array(origin)
    hi = lo + np.array(spacing) * (np.array(shape) - 1)
    m = 1000037
    pts = _pad4(rng.uniform(lo - 2e-6, hi + 2e-6, (m, 3)))
    got = ctx.interp_map(dev(torch_cuda, fmap), origin, spacing, dev(torch_cuda, pts))
    torch_cuda.cuda.synchronize()
    got = got.cpu().numpy()
    assert np.isfinite(got).all()
    idx = np.unique(np.concatenate([rng.choice(m, 3000, replace=False), [0, m - 1, m - 37]]))
    _check_interp(got[idx], fmap, origin, spacing, pts[idx, :3], fieldmap, "1M sampled")


def test_accumulate_adds_bit_exactly_and_overwrite_does_not(torch_cuda, ctx, fieldmap):
    rng = np.random.default_rng([43, 3])
    shape, origin, spacing = (5, 6, 7), (0.0, 0.0, 0.0), (1e-5, 1e-5, 1e-5)
    fmap = dev(torch_cuda, rng.normal(size=shape + (4,)).astype(np.float32))
    pts = dev(torch_cuda, _pad4(rng.uniform(0, 4e-5, (777, 3))))
    base = dev(torch_cuda, rng.normal(size=(777, 4)).astype(np.float32))
    plain = ctx.interp_map(fmap, origin, spacing, pts)
    acc = ctx.interp_map(fmap, origin, spacing, pts, out=base.clone(), accumulate=True)
    over = ctx.interp_map(fmap, origin, spacing, pts, out=base.clone(), accumulate=False)
    torch_cuda.cuda.synchronize()
    assert torch_cuda.equal(acc, plain + base)
    assert torch_cuda.equal(over, plain)


def test_field_map_nodes_match_the_field_oracle(torch_cuda, api, ctx, ref):
    """Config 1's two charged planes + its charges, on a ragged 9 x 7 x 11 node lattice strictly between the planes."""
    wl = W.make_workload(1)
    shape, origin, spacing = (9, 7, 11), (3.1 * UM, 5.3 * UM, 4.9 * UM), (11.7 * UM, 14.9 * UM, 9.01 * UM)
    ctx.set_softening(wl.eps_pp, wl.eps_panel)
    ctx.set_panels(dev(torch_cuda, wl.verts), dev(torch_cuda, wl.sigma))
    ctx.set_charges(dev(torch_cuda, wl.xyzq))
    ax = [np.float64(origin[a]) + np.arange(shape[a], dtype=np.float64) * np.float64(spacing[a]) for a in range(3)]
    nodes = np.stack(np.meshgrid(*ax, indexing="ij"), axis=-1).reshape(-1, 3).astype(np.float32)   # z fastest
    for flags in (api.PANELS, api.NBODY | api.PANELS):
        fmap = ctx.field_map(shape, origin, spacing, flags=flags)
        direct = ctx.eval_at_points(dev(torch_cuda, _pad4(nodes)), flags=flags)
        torch_cuda.cuda.synchronize()
        assert fmap.shape == shape + (4,)
        # same node coordinates bit for bit => same kernel, same inputs, same result
        assert torch_cuda.equal(fmap.reshape(-1, 4), direct)
        on, op = ref.eval_field(xyzq=wl.xyzq, verts=wl.verts, sigma=wl.sigma, targets=_pad4(nodes), self_index=None,
                                eps_pp=wl.eps_pp, eps_panel=wl.eps_panel)
        exp = op + (on if flags & api.NBODY else 0.0)
        assert_parity(fmap.reshape(-1, 4).cpu().numpy(), exp, "field_map flags=%d" % flags)


def test_static_option_end_to_end(torch_cuda, api, ctx, ref, fieldmap):
    """The static option as the paper describes it: map of the set-up field once, then per step interpolation at
    the particles + the N-body field.  Checked against: oracle trilinear of the ORACLE's node values + oracle
    N-body -- the interpolation error of the method itself is not an implementation error and cancels."""
    wl = W.make_workload(1)
    shape = (17, 17, 33)
    origin = (0.0, 0.0, 2.0 * UM)
    spacing = (6.25 * UM, 6.25 * UM, 3.0 * UM)
    ctx.set_softening(wl.eps_pp, wl.eps_panel)
    ctx.set_panels(dev(torch_cuda, wl.verts), dev(torch_cuda, wl.sigma))
    ctx.set_charges(dev(torch_cuda, wl.xyzq))
    fmap = ctx.field_map(shape, origin, spacing, flags=api.PANELS)
    out = ctx.eval_at_charges(flags=api.NBODY)
    out = ctx.interp_map(fmap, origin, spacing, dev(torch_cuda, wl.xyzq), out=out, accumulate=True)
    torch_cuda.cuda.synchronize()
    ax = [np.float64(origin[a]) + np.arange(shape[a], dtype=np.float64) * np.float64(spacing[a]) for a in range(3)]
    nodes = np.stack(np.meshgrid(*ax, indexing="ij"), axis=-1).reshape(-1, 3).astype(np.float32)
    _, op_nodes = ref.eval_field(xyzq=wl.xyzq, verts=wl.verts, sigma=wl.sigma, targets=_pad4(nodes),
                                 self_index=None, eps_pp=wl.eps_pp, eps_panel=wl.eps_panel)
    on, _ = ref.eval_field(xyzq=wl.xyzq, verts=wl.verts, sigma=wl.sigma, eps_pp=wl.eps_pp, eps_panel=wl.eps_panel)
    exp = on + fieldmap.trilinear(op_nodes.reshape(shape + (4,)), origin, spacing, wl.xyzq[:, :3])
    assert_parity(out.cpu().numpy(), exp, "static option, cfg1")


def test_argument_errors(torch_cuda, api, ctx):
    fmap = torch_cuda.zeros((2, 2, 2, 4), device="cuda")
    pts = torch_cuda.zeros((3, 4), device="cuda")
    with pytest.raises(api.ObemError):
        ctx.interp_map(fmap, (0, 0, 0), (1.0, 0.0, 1.0), pts)          # zero spacing on an axis with 2 nodes
    with pytest.raises(api.ObemError):
        ctx.interp_map(fmap, (0, 0, float("nan")), (1.0, 1.0, 1.0), pts)
    with pytest.raises(api.ObemError):
        ctx.field_map((0, 2, 2), (0, 0, 0), (1.0, 1.0, 1.0))
    # m = 0 is valid
    out = ctx.interp_map(fmap, (0, 0, 0), (1.0, 1.0, 1.0), torch_cuda.zeros((0, 4), device="cuda"))
    assert out.shape == (0, 4)
    # NaN position: clamped to node 0, finite result
    bad = torch_cuda.full((1, 4), float("nan"), device="cuda")
    r = ctx.interp_map(fmap + 1.0, (0, 0, 0), (1.0, 1.0, 1.0), bad)
    torch_cuda.cuda.synchronize()
    assert torch_cuda.equal(r, torch_cuda.ones((1, 4), device="cuda"))

"""GPU parity of the NN approximation of the N-body sum (reading A19):
obem_eval_at_charges_nn through the C ABI against oracle/nn.py, which follows the same algorithm step by step in
fp64.  `pytest -m gpu`.

Both sides take the discrete decisions (k-d order, near / far) on the same fp32 inputs with the same individually
rounded fp64 operations, so they sum the same terms; what differs is fp32 arithmetic, fp32-rounded pseudo-particles
(position error <= half an ulp of the coordinate, 4e-12 m, against far distances of micrometres) and summation
order.  Hence the path's own tolerances: rel-L2 2e-5, per-target 1e-3 (tests/parity_metrics.py).
"""
import numpy as np
import pytest

from paper_2110_09214_b200 import workloads as W
from parity_metrics import assert_parity, field_errors

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


@pytest.fixture(scope="module")
def nn():
    from oracle import nn as _nn
    return _nn


@pytest.fixture()
def ctx(api):
    c = api.Context(0)
    yield c
    c.destroy()


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _cloud(rng, n):
    x = np.zeros((n, 4), dtype=np.float32)
    x[:, :3] = rng.normal(0, 1, (n, 3)) * np.array([20 * UM, 20 * UM, 10 * UM])
    x[:, 3] = rng.choice([-QE, QE], n)
    return x


def _gpu_nn(torch, ctx, x, eps, theta, flags=1):
    ctx.set_softening(eps, 0.0)
    ctx.set_nn_theta(theta)
    ctx.set_charges(dev(torch, x))
    out = ctx.eval_at_charges_nn(flags=flags)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def _oracle_units(nn, tree, theta, n):
    return nn.units(tree, theta, n)


@pytest.mark.parametrize("n,theta", [(50000, 0.0), (50000, 2.0), (50000, 6.0), (20011, 3.0)])
def test_matches_the_nn_oracle(torch_cuda, ctx, nn, ref, n, theta):
    rng = np.random.default_rng([61, n, int(theta * 10)])
    x = _cloud(rng, n)
    exp, tree = nn.nn_field(x, 0.05 * UM, theta, ref=ref)
    got = _gpu_nn(torch_cuda, ctx, x, 0.05 * UM, theta)
    assert_parity(got, exp, "nn n=%d theta=%g" % (n, theta))
    # the same near / far decisions: the number of (tile, source block) units is the oracle's
    assert ctx.nn_last_units() == _oracle_units(nn, tree, theta, n)
    if theta == 0.0:
        bf, _ = ref.eval_field(xyzq=x, eps_pp=0.05 * UM, flags=ref.NBODY)
        assert_parity(got, bf, "nn theta=0 is the exact sum")
    else:
        n_leaf = tree["leaf_boxes"].shape[0]
        assert any(nn.far_mask(tree, g, theta).any() for g in range(tree["group_boxes"].shape[0])), "no far leaf: vacuous"
        assert n_leaf > 8
        if n >= 50000 and theta >= 6.0:   # both far levels are exercised
            cls = [nn.classify(tree, g, theta) for g in range(tree["group_boxes"].shape[0])]
            assert any(c[0].any() for c in cls) and any(c[2].any() for c in cls)


def test_config3_full_size_sampled_groups(torch_cuda, api, ctx, nn, ref):
    """1,048,576 charges, default theta = 2: four sampled tiles (8192 charges) against the oracle, and against the
    exact sum for the paper's acceptance statement (Fig 6: < 5 % on E_z for > 96.8 % of the particles)."""
    wl = W.make_workload(3, mesh_div=8)
    got = _gpu_nn(torch_cuda, ctx, wl.xyzq, wl.eps_pp, 2.0)
    assert np.isfinite(got).all()
    units = ctx.nn_last_units()
    rng = np.random.default_rng([61, 3])
    groups = np.sort(rng.choice(wl.n_charges // 2048, 4, replace=False))
    exp, tree = nn.nn_field(wl.xyzq, wl.eps_pp, 2.0, groups=groups, ref=ref)
    idx = np.nonzero(np.isfinite(exp[:, 0]))[0]
    assert idx.size == 4 * 2048
    assert_parity(got[idx], exp[idx], "cfg3 nn, sampled tiles")
    assert units == _oracle_units(nn, tree, 2.0, wl.n_charges)
    bf, _ = ref.eval_field(xyzq=wl.xyzq, targets=wl.xyzq[idx], self_index=idx.astype(np.int64), eps_pp=wl.eps_pp,
                           flags=ref.NBODY)
    rel = np.abs((got[idx, 2] - bf[:, 2]) / bf[:, 2])
    assert (rel < 0.05).mean() > 0.968
    e = field_errors(got[idx], bf)
    assert e["E_rel_l2"] < 5e-3, e                                    # measured 2.2e-3
    # work: a few per cent of the N (N - 1) pairs of the exact sum
    assert units * 2048 * 256 < 0.06 * wl.n_charges * (wl.n_charges - 1)


def test_config4_charges_full_size_sampled_groups(torch_cuda, api, ctx, nn, ref):
    """4,194,304 charges in two clouds 2 mm apart (config 4): 256 super-leaves, many of them far.  Two sampled tiles
    against the oracle, identical decisions over all 2048 tiles, and the paper's acceptance against the exact sum."""
    wl = W.make_workload(4, mesh_div=64)
    got = _gpu_nn(torch_cuda, ctx, wl.xyzq, wl.eps_pp, 2.0)
    assert np.isfinite(got).all()
    units = ctx.nn_last_units()
    rng = np.random.default_rng([61, 4])
    groups = np.sort(rng.choice(wl.n_charges // 2048, 2, replace=False))
    exp, tree = nn.nn_field(wl.xyzq, wl.eps_pp, 2.0, groups=groups, ref=ref)
    idx = np.nonzero(np.isfinite(exp[:, 0]))[0]
    assert idx.size == 2 * 2048
    assert_parity(got[idx], exp[idx], "cfg4 nn, sampled tiles")
    assert units == _oracle_units(nn, tree, 2.0, wl.n_charges)
    assert all(nn.classify(tree, g, 2.0)[0].any() for g in groups), "no far super-leaf: vacuous"
    bf, _ = ref.eval_field(xyzq=wl.xyzq, targets=wl.xyzq[idx], self_index=idx.astype(np.int64), eps_pp=wl.eps_pp,
                           flags=ref.NBODY)
    rel = np.abs((got[idx, 2] - bf[:, 2]) / bf[:, 2])
    assert (rel < 0.05).mean() > 0.968
    assert field_errors(got[idx], bf)["E_rel_l2"] < 5e-3
    assert units * 2048 * 256 < 0.02 * wl.n_charges * (wl.n_charges - 1.0)


# 8191 .. 16641: around 32 / 33 / 64 / 65 leaves, where the k-d order changes from device-wide rounds to the one-launch
# rounds of nn_kd_local_kernel (segments of at most 32 leaves); below that everything is local
@pytest.mark.parametrize("n", [1, 2, 255, 256, 257, 2047, 2049, 4097, 8191, 8192, 8193, 8449, 16385, 16641])
def test_small_and_ragged_sizes(torch_cuda, ctx, nn, ref, n):
    rng = np.random.default_rng([61, 7, n])
    x = _cloud(rng, n)
    exp, tree = nn.nn_field(x, 0.1 * UM, 2.0, ref=ref)
    got = _gpu_nn(torch_cuda, ctx, x, 0.1 * UM, 2.0)
    if n == 1:
        assert np.all(got == 0)
    else:
        assert_parity(got, exp, "nn n=%d" % n)
    assert ctx.nn_last_units() == nn.units(tree, 2.0, n)     # the same leaves, the same near / far decisions


def test_degenerate_positions(torch_cuda, ctx, nn, ref):
    rng = np.random.default_rng([61, 8])
    # (a) all charges at one point, softened: zero-size boxes, every leaf near; E = 0, phi = k_e sum q / eps
    x = np.zeros((3000, 4), dtype=np.float32)
    x[:, :3] = [1e-5, 2e-5, 3e-5]
    x[:, 3] = rng.choice([-QE, QE, 2 * QE], 3000)
    exp, _ = nn.nn_field(x, 0.1 * UM, 2.0, ref=ref)
    got = _gpu_nn(torch_cuda, ctx, x, 0.1 * UM, 2.0)
    assert np.all(got[:, :3] == 0)
    assert np.allclose(got[:, 3], exp[:, 3], rtol=2e-5)
    # (b) two tight clumps far apart, no softening, duplicates inside a clump: coincident pairs contribute 0 (A4)
    y = _cloud(rng, 6000)
    y[:3000, :3] = y[:3000, :3] * 0.01 + np.array([0, 0, 500 * UM], dtype=np.float32)
    y[3000:, :3] = y[3000:, :3] * 0.01
    y[10] = y[11]
    y[4000, :3] = y[4001, :3]
    exp, tree = nn.nn_field(y, 0.0, 2.0, ref=ref)
    got = _gpu_nn(torch_cuda, ctx, y, 0.0, 2.0)
    assert nn.far_mask(tree, 0, 2.0).any()
    assert_parity(got, exp, "nn, clumps, eps = 0")


def test_panels_are_added_and_calls_are_reproducible(torch_cuda, api, ctx, nn, ref):
    wl = W.make_workload(2, charge_div=4, mesh_div=4)
    ctx.set_panels(dev(torch_cuda, wl.verts), dev(torch_cuda, wl.sigma))
    a = _gpu_nn(torch_cuda, ctx, wl.xyzq, wl.eps_pp, 3.0, flags=api.NBODY | api.PANELS)
    b = _gpu_nn(torch_cuda, ctx, wl.xyzq, wl.eps_pp, 3.0, flags=api.NBODY | api.PANELS)
    assert np.array_equal(a, b)
    exp, _ = nn.nn_field(wl.xyzq, wl.eps_pp, 3.0, ref=ref)
    _, op = ref.eval_field(xyzq=wl.xyzq, verts=wl.verts, sigma=wl.sigma, eps_pp=wl.eps_pp, flags=ref.PANELS)
    assert_parity(a, exp + op, "nn + panels")
    ex = _gpu_nn(torch_cuda, ctx, wl.xyzq, wl.eps_pp, 3.0, flags=api.NBODY | api.PANELS | api.PANELS_EXACT)
    assert_parity(ex, exp + ref.eval_panels_analytic(wl.verts, wl.sigma, wl.xyzq), "nn + exact panels")


def test_argument_errors(torch_cuda, api, ctx):
    with pytest.raises(api.ObemError):
        ctx.eval_at_charges_nn()                                        # charges never set
    ctx.set_charges(dev(torch_cuda, _cloud(np.random.default_rng(0), 300)))
    with pytest.raises(api.ObemError):
        ctx.eval_at_charges_nn(flags=api.PANELS)                        # the N-body flag is what this call is for
    with pytest.raises(api.ObemError):
        ctx.eval_at_charges_nn(flags=api.NBODY | api.PANELS)            # panels never set
    with pytest.raises(api.ObemError):
        ctx.set_nn_theta(-1.0)
    assert ctx.nn_last_units() == -1
    ctx.set_charges(torch_cuda.zeros((0, 4), device="cuda"))
    assert ctx.eval_at_charges_nn().shape == (0, 4)


@pytest.mark.parametrize("seed", range(12))
def test_random_clouds_match_the_oracle(torch_cuda, ctx, nn, ref, seed):
    """Seeded random sizes, opening parameters, softenings, charge values (zeros included) and clumpy geometries."""
    rng = np.random.default_rng([61, 99, seed])
    n = int(rng.integers(1, 30000))
    theta = float(rng.choice([0.0, 0.5, 2.0, 5.0, 16.0]))
    eps = float(rng.choice([0.02 * UM, 0.05 * UM]))
    k = int(rng.integers(1, 6))                                        # clumps
    centres = rng.uniform(-300 * UM, 300 * UM, (k, 3))
    x = np.zeros((n, 4), dtype=np.float32)
    x[:, :3] = centres[rng.integers(0, k, n)] + rng.normal(0, 1, (n, 3)) * rng.uniform(2 * UM, 30 * UM, 3)
    x[:, 3] = rng.choice([-QE, QE, 2 * QE, 0.0], n, p=[0.4, 0.4, 0.1, 0.1])
    exp, tree = nn.nn_field(x, eps, theta, ref=ref)
    got = _gpu_nn(torch_cuda, ctx, x, eps, theta)
    what = "seed %d: n=%d theta=%g eps=%g clumps=%d" % (seed, n, theta, eps, k)
    if n > 1 and np.abs(exp).max() > 0:
        assert_parity(got, exp, what)
    assert ctx.nn_last_units() == nn.units(tree, theta, n), what

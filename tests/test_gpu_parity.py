"""GPU parity: libobem.so (through the C ABI / api.py) against the fp64 oracle, element by element, on the
same seeded fp32 inputs.  Tolerances: BASELINE.json north_star (rel-L2 2e-5, per-target max rel 1e-3),
written in tests/parity_metrics.py.  Run on the B200 box: `pytest -m gpu`.
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


@pytest.fixture()
def ctx(api):
    c = api.Context(0)
    yield c
    c.destroy()


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def gpu_eval_workload(torch, api, ctx, wl, flags):
    ctx.set_softening(wl.eps_pp, wl.eps_panel)
    ctx.set_panels(dev(torch, wl.verts), dev(torch, wl.sigma))
    ctx.set_charges(dev(torch, wl.xyzq))
    if wl.points is not None:
        out = ctx.eval_at_points(dev(torch, wl.points), flags=flags)
    else:
        out = ctx.eval_at_charges(flags=flags)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def oracle_parts(ref, wl, targets=None, self_index=None):
    if targets is None and wl.points is not None:
        targets = wl.points
        self_index = None
    return ref.eval_field(xyzq=wl.xyzq, verts=wl.verts, sigma=wl.sigma, targets=targets, self_index=self_index,
                          eps_pp=wl.eps_pp, eps_panel=wl.eps_panel)


# --------------------------------------------------------------------------------------------------
# whole small configs, all targets
# --------------------------------------------------------------------------------------------------
def test_config1_all_flags(torch_cuda, api, ctx, ref):
    wl = W.make_workload(1)
    assert wl.n_charges == 4096 and wl.n_panels == 1024
    on, op = oracle_parts(ref, wl)
    g_n = gpu_eval_workload(torch_cuda, api, ctx, wl, api.NBODY)
    g_p = gpu_eval_workload(torch_cuda, api, ctx, wl, api.PANELS)
    g_b = gpu_eval_workload(torch_cuda, api, ctx, wl, api.NBODY | api.PANELS)
    assert_parity(g_n, on, "cfg1 nbody")
    assert_parity(g_p, op, "cfg1 panels")
    assert_parity(g_b, on + op, "cfg1 both")


def test_config2_reduced_all_targets(torch_cuda, api, ctx, ref):
    # 16384 charges (8 target tiles), 4096 panels: several tiles, many source blocks, split tiles
    wl = W.make_workload(2, charge_div=4, mesh_div=2)
    on, op = oracle_parts(ref, wl)
    g_n = gpu_eval_workload(torch_cuda, api, ctx, wl, api.NBODY)
    g_p = gpu_eval_workload(torch_cuda, api, ctx, wl, api.PANELS)
    g_b = gpu_eval_workload(torch_cuda, api, ctx, wl, api.NBODY | api.PANELS)
    assert_parity(g_n, on, "cfg2/4 nbody")
    assert_parity(g_p, op, "cfg2/4 panels")
    assert_parity(g_b, on + op, "cfg2/4 both")


def test_config2_full_all_targets(torch_cuda, api, ctx, ref):
    wl = W.make_workload(2)
    assert wl.n_charges == 65536 and wl.n_panels == 16384
    on, op = oracle_parts(ref, wl)
    g_b = gpu_eval_workload(torch_cuda, api, ctx, wl, api.NBODY | api.PANELS)
    assert_parity(g_b, on + op, "cfg2 both")


@pytest.mark.parametrize("n,npan", [(1, 1), (2, 0), (255, 37), (257, 36), (2049, 73), (4097, 300), (6000, 1)])
def test_ragged_sizes(torch_cuda, api, ctx, ref, n, npan):
    rng = np.random.default_rng([7, n, npan])
    xyzq = np.zeros((n, 4), dtype=np.float32)
    xyzq[:, :3] = rng.uniform(0, 100 * UM, (n, 3))
    xyzq[:, 3] = rng.choice([-QE, QE, 2 * QE], n)
    verts = (rng.uniform(0, 100 * UM, (npan, 1, 3)) + rng.uniform(-3 * UM, 3 * UM, (npan, 3, 3))).astype(np.float32)
    verts[..., 2] -= 150 * UM  # keep panels away from the charges
    sigma = rng.normal(0, 1e-5, npan).astype(np.float32)
    wl = W.Workload("ragged", 0, xyzq, verts, sigma, 0.1 * UM)
    on, op = oracle_parts(ref, wl)
    g_b = gpu_eval_workload(torch_cuda, api, ctx, wl, api.NBODY | api.PANELS)
    if n == 1 and npan == 0:
        assert np.all(g_b == 0)
    else:
        assert_parity(g_b, on + op, "ragged n=%d np=%d" % (n, npan))


# --------------------------------------------------------------------------------------------------
# full-size configs in the bench launch configuration, sampled targets
# --------------------------------------------------------------------------------------------------
def _sampled(torch, api, ctx, ref, cfg, n_sample):
    wl = W.make_workload(cfg)
    g = gpu_eval_workload(torch, api, ctx, wl, api.NBODY | api.PANELS if wl.points is None else api.PANELS)
    assert np.isfinite(g).all()
    rng = np.random.default_rng([11, cfg])
    nt = wl.n_targets
    idx = np.sort(rng.choice(nt, n_sample, replace=False))
    # adversarial extras: largest / smallest |E| and largest |phi| in the GPU output
    mag = np.linalg.norm(g[:, :3], axis=1)
    extra = np.concatenate([np.argsort(mag)[-64:], np.argsort(mag)[:64], np.argsort(np.abs(g[:, 3]))[-64:],
                            [0, nt - 1]])
    idx = np.unique(np.concatenate([idx, extra]))
    if wl.points is None:
        on, op = oracle_parts(ref, wl, targets=wl.xyzq[idx], self_index=idx.astype(np.int64))
    else:
        on, op = oracle_parts(ref, wl, targets=wl.points[idx])
    return wl, g[idx], on + op


def test_config3_full_size_sampled(torch_cuda, api, ctx, ref):
    wl, g, o = _sampled(torch_cuda, api, ctx, ref, 3, 1024)
    assert wl.n_charges == 1048576 and wl.n_panels == 65536
    assert_parity(g, o, "cfg3 sampled")


def test_config4_full_size_sampled(torch_cuda, api, ctx, ref):
    wl, g, o = _sampled(torch_cuda, api, ctx, ref, 4, 512)
    assert wl.n_charges == 4194304 and wl.n_panels == 262144
    assert_parity(g, o, "cfg4 sampled")


def test_config5_full_size_sampled(torch_cuda, api, ctx, ref):
    wl, g, o = _sampled(torch_cuda, api, ctx, ref, 5, 2048)
    assert wl.n_targets == 16777216 and wl.n_panels == 262144
    assert_parity(g, o, "cfg5 sampled")

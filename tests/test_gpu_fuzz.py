"""Seeded random combinations of the library's options on small inputs, each against the plain oracles with the
geometry written out (explicit image copies, explicit 7-point or exact panel integrals): sizes, softenings, flags,
evaluation at the charges / at a slice of them / at free points, symmetry planes (also one at a coordinate that is not
exactly representable), exact near-field integrals.  Catches interactions between features that the per-feature tests
do not combine.  `pytest -m gpu`.
"""
import os

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


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _case(seed):
    rng = np.random.default_rng([97, seed])
    n = int(rng.choice([1, 7, 255, 256, 257, 1000, 2048, 2049, 5000]))
    npan = int(rng.choice([0, 1, 33, 34, 35, 200, 400]))
    xyzq = np.zeros((n, 4), dtype=np.float32)
    xyzq[:, :3] = rng.uniform(5 * UM, 95 * UM, (n, 3))
    xyzq[:, 3] = rng.choice([-QE, QE, 2 * QE], n)
    # panels: small triangles scattered on two sheets below and above the charges (clearance >= 2 um)
    c = np.zeros((npan, 3))
    c[:, :2] = rng.uniform(5 * UM, 95 * UM, (npan, 2))
    c[:, 2] = rng.choice([2 * UM, 98 * UM], npan)
    verts = c[:, None, :] + np.concatenate([rng.uniform(-2.5 * UM, 2.5 * UM, (npan, 3, 2)),
                                            rng.uniform(-0.3 * UM, 0.3 * UM, (npan, 3, 1))], axis=2)
    verts = verts.astype(np.float32)
    sigma = rng.normal(0, 1e-5, npan).astype(np.float32)
    eps_pp = float(rng.choice([0.0, 0.05 * UM]))
    exact = bool(rng.integers(0, 2)) and npan > 0
    eps_panel = 0.0 if exact else float(rng.choice([0.0, 0.02 * UM]))
    want_n, want_p = bool(rng.integers(0, 2)), bool(rng.integers(0, 2))
    if not (want_n or want_p):
        want_n = True
    planes = []
    for ax, coord in ((0, 0.0), (1, 0.0), (2, -3.3 * UM)):
        if rng.random() < 0.35:
            planes.append((ax, coord, int(rng.choice([-1, 1]))))
    mode = str(rng.choice(["charges", "range", "points"]))
    return dict(rng=rng, n=n, npan=npan, xyzq=xyzq, verts=verts, sigma=sigma, eps_pp=eps_pp, eps_panel=eps_panel,
                exact=exact, want_n=want_n, want_p=want_p and npan > 0, planes=planes, mode=mode)


def _images(xyzq, verts, sigma, planes):
    xs, vs, ss = [xyzq], [verts], [sigma]
    for mask in range(1, 1 << len(planes)):
        x, v, s, sign = xyzq.astype(np.float64).copy(), verts.astype(np.float64).copy(), sigma.astype(np.float64), 1.0
        for k, (ax, c, par) in enumerate(planes):
            if mask & (1 << k):
                x[:, ax] = 2 * c - x[:, ax]
                v[:, :, ax] = 2 * c - v[:, :, ax]
                sign *= par
        x[:, 3] *= sign
        xs.append(x.astype(np.float32)), vs.append(v.astype(np.float32)), ss.append((s * sign).astype(np.float32))
    return np.concatenate(xs), np.concatenate(vs), np.concatenate(ss)


# OBEM_FUZZ_SEEDS=N runs N seeds instead of 64
@pytest.mark.parametrize("seed", range(int(os.environ.get("OBEM_FUZZ_SEEDS", "64"))))
def test_random_combination(torch_cuda, api, ref, seed):
    k = _case(seed)
    rng, n = k["rng"], k["n"]
    flags = (api.NBODY if k["want_n"] else 0) | (api.PANELS if k["want_p"] else 0)
    if k["want_p"] and k["exact"]:
        flags |= api.PANELS_EXACT
    with api.Context(0) as ctx:
        ctx.set_softening(k["eps_pp"], k["eps_panel"])
        ctx.set_panels(dev(torch_cuda, k["verts"]), dev(torch_cuda, k["sigma"]))
        ctx.set_charges(dev(torch_cuda, k["xyzq"]))
        ctx.set_symmetry(k["planes"])
        if k["mode"] == "charges":
            got = ctx.eval_at_charges(flags=flags)
            targets, self_index = k["xyzq"], np.arange(n, dtype=np.int64)
        elif k["mode"] == "range":
            first = int(rng.integers(0, n))
            count = int(rng.integers(0, n - first + 1))
            got = ctx.eval_at_charges_range(first, count, flags=flags)
            targets, self_index = k["xyzq"][first:first + count], np.arange(first, first + count, dtype=np.int64)
        else:
            m = int(rng.choice([1, 300, 2100]))
            pts = np.zeros((m, 4), dtype=np.float32)
            pts[:, :3] = rng.uniform(6 * UM, 94 * UM, (m, 3))
            got = ctx.eval_at_points(dev(torch_cuda, pts), flags=flags)
            targets, self_index = pts, None
        torch_cuda.cuda.synchronize()
        got = got.cpu().numpy()
    ax_all, av_all, as_all = _images(k["xyzq"], k["verts"], k["sigma"], k["planes"])
    exp = np.zeros((targets.shape[0], 4))
    if targets.shape[0]:
        on, op = ref.eval_field(xyzq=ax_all, verts=av_all, sigma=as_all, targets=targets, self_index=self_index,
                                eps_pp=k["eps_pp"], eps_panel=k["eps_panel"])
        if k["want_n"]:
            exp += on
        if k["want_p"]:
            exp += ref.eval_panels_analytic(av_all, as_all, targets) if k["exact"] else op
    what = "seed %d: n=%d np=%d eps=(%g, %g) flags=%d planes=%r mode=%s" % (
        seed, n, k["npan"], k["eps_pp"], k["eps_panel"], flags, k["planes"], k["mode"])
    assert got.shape == exp.shape, what
    if exp.size and np.abs(exp).max() > 0:
        assert_parity(got, exp, what)
    else:
        assert not got.size or np.all(got == 0), what

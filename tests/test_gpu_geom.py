"""GPU parity of the geometry conveniences of SURVEY.md 8f NEXT-3: polygonal cells
(obem_set_panels_cells / obem_set_sigma_cells) and symmetry planes (obem_set_symmetry), through the C ABI.
`pytest -m gpu`.

Oracles are the plain ones, fed with the geometry written out explicitly: the cells split into triangles in numpy,
the mirror images added as real copies of the charges and panels.  Closed forms on top: the on-axis field of ONE
rectangular cell with the exact integrals; phi = 0 and E_tangential = 0 on an odd plane, E_normal = 0 on an even one.
"""
import numpy as np
import pytest

from paper_2110_09214_b200 import workloads as W
from parity_metrics import assert_parity

pytestmark = pytest.mark.gpu

UM = 1e-6
QE = 1.602176634e-19
EPS0 = 8.8541878128e-12


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


def _pad4(p):
    out = np.zeros((p.shape[0], 4), dtype=np.float32)
    out[:, :3] = p
    return out


def _split(verts4, nvert):
    """cells -> triangles, written out independently of the library: (v0, v1, v2) and, for quadrilaterals, (v0, v2, v3)."""
    tris, owner = [], []
    for i, (v, k) in enumerate(zip(verts4, nvert)):
        tris.append([v[0], v[1], v[2]])
        owner.append(i)
        if k == 4:
            tris.append([v[0], v[2], v[3]])
            owner.append(i)
    return np.array(tris, dtype=np.float32), np.array(owner)


def test_one_rectangular_cell_closed_form(torch_cuda, api, ctx):
    """A single 2a x 2b quadrilateral cell with the exact integrals: E_z(h) = sigma/(pi eps0) atan(ab/(h sqrt(a^2+b^2+h^2)))
    on its axis, at heights from 1/50 of the cell to 20 cells."""
    a, b, sigma = 8 * UM, 5 * UM, np.float32(2e-5)
    v = np.array([[[-a, -b, 0], [a, -b, 0], [a, b, 0], [-a, b, 0]]], dtype=np.float32)
    ctx.set_panels_cells(dev(torch_cuda, v), dev(torch_cuda, np.array([sigma])))
    assert ctx.n_panels == 2
    hs = 2 * a * np.array([0.02, 0.1, 0.5, 1.0, 3.0, 20.0])
    pts = _pad4(np.stack([np.zeros_like(hs), np.zeros_like(hs), hs], 1))
    out = ctx.eval_at_points(dev(torch_cuda, pts), flags=api.PANELS | api.PANELS_EXACT).cpu().numpy().astype(np.float64)
    h = pts[:, 2].astype(np.float64)
    a32, b32 = float(v[0, 1, 0]), float(v[0, 2, 1])
    ez = float(sigma) / (np.pi * EPS0) * np.arctan(a32 * b32 / (h * np.sqrt(a32 ** 2 + b32 ** 2 + h ** 2)))
    assert np.allclose(out[:, 2], ez, rtol=2e-5)
    assert np.abs(out[:, :2]).max() <= 2e-5 * ez.max()


def test_mixed_cells_match_the_explicit_split(torch_cuda, api, ctx, ref):
    rng = np.random.default_rng([71, 1])
    n = 12                                                   # 12 x 12 cells on a plane, every third one a triangle
    xs = np.linspace(0, 60 * UM, n + 1)
    cells, nvert = [], []
    for i in range(n):
        for j in range(n):
            p = [[xs[i], xs[j], 0], [xs[i + 1], xs[j], 0], [xs[i + 1], xs[j + 1], 0], [xs[i], xs[j + 1], 0]]
            k = 3 if (i * n + j) % 3 == 0 else 4
            if k == 3:
                p[3] = [1e3, -1e3, 7.0]                      # ignored
            cells.append(p)
            nvert.append(k)
    verts4 = np.array(cells, dtype=np.float32)
    nvert = np.array(nvert, dtype=np.int32)
    sigma = rng.normal(0, 1e-5, len(cells)).astype(np.float32)
    tris, owner = _split(verts4, nvert)
    pts = _pad4(rng.uniform([0, 0, 1 * UM], [60 * UM, 60 * UM, 40 * UM], (3000, 3)))
    ctx.set_panels_cells(dev(torch_cuda, verts4), dev(torch_cuda, sigma), nvert=dev(torch_cuda, nvert))
    assert ctx.n_panels == 2 * len(cells)
    g7 = ctx.eval_at_points(dev(torch_cuda, pts), flags=api.PANELS)
    gx = ctx.eval_at_points(dev(torch_cuda, pts), flags=api.PANELS | api.PANELS_EXACT)
    torch_cuda.cuda.synchronize()
    _, o7 = ref.eval_field(verts=tris, sigma=sigma[owner], targets=pts, flags=ref.PANELS)
    assert_parity(g7.cpu().numpy(), o7, "cells, 7-point")
    assert_parity(gx.cpu().numpy(), ref.eval_panels_analytic(tris, sigma[owner], pts), "cells, exact")
    sigma2 = rng.normal(0, 1e-5, len(cells)).astype(np.float32)
    ctx.set_sigma_cells(dev(torch_cuda, sigma2))
    g2 = ctx.eval_at_points(dev(torch_cuda, pts), flags=api.PANELS)
    torch_cuda.cuda.synchronize()
    _, o2 = ref.eval_field(verts=tris, sigma=sigma2[owner], targets=pts, flags=ref.PANELS)
    assert_parity(g2.cpu().numpy(), o2, "cells, new sigma")
    with pytest.raises(api.ObemError):
        ctx.set_sigma_cells(dev(torch_cuda, sigma2[:-1]))


def _images(xyzq, verts, sigma, planes):
    """All 2^k copies (identity first) of charges and panels, written out: reflected coordinates, parity on q / sigma."""
    xs, vs, ss = [xyzq.copy()], [verts.copy()], [sigma.copy()]
    for mask in range(1, 1 << len(planes)):
        x, v, s, sign = xyzq.astype(np.float64), verts.astype(np.float64), sigma.astype(np.float64), 1.0
        x, v = x.copy(), v.copy()
        for k, (ax, c, par) in enumerate(planes):
            if mask & (1 << k):
                x[:, ax] = 2 * c - x[:, ax]
                v[:, :, ax] = 2 * c - v[:, :, ax]
                sign *= par
        x[:, 3] *= sign
        xs.append(x.astype(np.float32)), vs.append(v.astype(np.float32)), ss.append((s * sign).astype(np.float32))
    return np.concatenate(xs), np.concatenate(vs), np.concatenate(ss)


@pytest.mark.parametrize("planes", [[(0, 0.0, -1)], [(2, 0.0, 1), (0, 0.0, -1)], [(0, 0.0, 1), (1, 0.0, -1), (2, 0.0, -1)]])
def test_symmetry_planes_match_explicit_images(torch_cuda, api, ctx, ref, planes):
    """Config-1-like box in the octant x, y, z > 0; planes through the origin (reflections are then exact in fp32, so
    both sides see bit-identical geometry)."""
    wl = W.make_workload(1)
    rng = np.random.default_rng([71, 2, len(planes)])
    xyzq = wl.xyzq[:1500].copy()
    xyzq[:, :3] += np.float32(1 * UM)                         # strictly inside the octant
    verts = wl.verts[:300] + np.float32(1 * UM)
    sigma = wl.sigma[:300]
    ax_all, av_all, as_all = _images(xyzq, verts, sigma, planes)
    n = len(xyzq)
    ctx.set_softening(wl.eps_pp, 0.0)
    ctx.set_panels(dev(torch_cuda, verts), dev(torch_cuda, sigma))
    ctx.set_charges(dev(torch_cuda, xyzq))
    ctx.set_symmetry(planes)
    g = ctx.eval_at_charges(flags=api.NBODY | api.PANELS)
    gx = ctx.eval_at_charges(flags=api.NBODY | api.PANELS | api.PANELS_EXACT)
    torch_cuda.cuda.synchronize()
    on, op = ref.eval_field(xyzq=ax_all, verts=av_all, sigma=as_all, targets=xyzq, self_index=np.arange(n, dtype=np.int64),
                            eps_pp=wl.eps_pp)
    assert_parity(g.cpu().numpy(), on + op, "symmetry %r" % (planes,))
    assert_parity(gx.cpu().numpy(), on + ref.eval_panels_analytic(av_all, as_all, xyzq), "symmetry + exact %r" % (planes,))
    # on the planes themselves: odd parity -> phi = 0 and no tangential field; even parity -> no normal field
    for ax, c, par in planes:
        pts = rng.uniform(2 * UM, 90 * UM, (200, 3))
        pts[:, ax] = c
        f = ctx.eval_at_points(dev(torch_cuda, _pad4(pts)), flags=api.NBODY | api.PANELS).cpu().numpy().astype(np.float64)
        scale_e = np.linalg.norm(f[:, :3], axis=1).max()
        if par == -1:
            tang = [a for a in range(3) if a != ax]
            assert np.abs(f[:, 3]).max() <= 1e-5 * np.abs(g.cpu().numpy()[:, 3]).max()
            assert np.abs(f[:, tang]).max() <= 1e-5 * scale_e
        else:
            assert np.abs(f[:, ax]).max() <= 1e-5 * scale_e
    # removing the planes restores the plain evaluation
    ctx.set_symmetry(())
    g0 = ctx.eval_at_charges(flags=api.NBODY | api.PANELS)
    torch_cuda.cuda.synchronize()
    o0n, o0p = ref.eval_field(xyzq=xyzq, verts=verts, sigma=sigma, eps_pp=wl.eps_pp)
    assert_parity(g0.cpu().numpy(), o0n + o0p, "symmetry removed")


def test_symmetry_argument_errors(torch_cuda, api, ctx):
    with pytest.raises(api.ObemError):
        ctx.set_symmetry([(0, 0.0, 1), (0, 1e-4, 1)])         # two planes on one axis: an infinite image series
    with pytest.raises(api.ObemError):
        ctx.set_symmetry([(3, 0.0, 1)])
    with pytest.raises(api.ObemError):
        ctx.set_symmetry([(1, 0.0, 0)])
    with pytest.raises(api.ObemError):
        ctx.set_symmetry([(0, 0.0, 1), (1, 0.0, 1), (2, 0.0, 1), (0, 0.0, 1)])
    ctx.set_symmetry([(2, 0.0, -1)])
    ctx.set_charges(dev(torch_cuda, W.make_workload(1).xyzq[:600]))
    with pytest.raises(api.ObemError):
        ctx.eval_at_charges_nn()                              # the NN lists hold no image leaves

"""GPU parity of the near-field-accurate panel sums: OBEM_PANELS |
OBEM_PANELS_EXACT through the C ABI against the EXACT cell integrals of Eq (2.13)/(2.14) (oracle/obem_ref_analytic.c),
at the north_star tolerances (rel-L2 2e-5, per-target 1e-3).  `pytest -m gpu`.

The oracle integrates every panel exactly; the GPU integrates exactly only the panels whose centroid is closer than
near_factor * (longest edge) and keeps the 7-point rule for the rest.  The rule's error at 3 h is <= 2.1e-6 of that
panel's own field and falls as (h/r)^6 (tests/test_oracle_next3_pins.py T6), so the default factor 3 leaves a margin
of ~10 on the rel-L2 bar.
"""
import numpy as np
import pytest

from paper_2110_09214_b200 import workloads as W
from parity_metrics import assert_parity, field_errors

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


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _pad4(p):
    out = np.zeros((p.shape[0], 4), dtype=np.float32)
    out[:, :3] = p
    return out


def _gpu_panels(torch, api, ctx, wl, targets, flags):
    ctx.set_softening(wl.eps_pp, wl.eps_panel)
    ctx.set_panels(dev(torch, wl.verts), dev(torch, wl.sigma))
    out = ctx.eval_at_points(dev(torch, targets), flags=flags)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def test_config1_exact_panels_at_the_charges(torch_cuda, api, ctx, ref):
    wl = W.make_workload(1)
    exact = ref.eval_panels_analytic(wl.verts, wl.sigma, wl.xyzq)
    g = _gpu_panels(torch_cuda, api, ctx, wl, wl.xyzq, api.PANELS | api.PANELS_EXACT)
    assert_parity(g, exact, "cfg1 exact panels")
    assert ctx.near_list_size > 0 and ctx.near_cells > 0
    # the bare 7-point rule is NOT the exact integral for the charges closest to the planes (0.25 um from 6.25 um cells)
    g7 = _gpu_panels(torch_cuda, api, ctx, wl, wl.xyzq, api.PANELS)
    e7 = field_errors(g7, exact)
    assert e7["E_max_rel"] > 1e-2 and e7["E_rel_l2"] > 1e-3, e7


def test_config2_reduced_and_all_flags_add_up(torch_cuda, api, ctx, ref):
    wl = W.make_workload(2, charge_div=4, mesh_div=2)
    exact = ref.eval_panels_analytic(wl.verts, wl.sigma, wl.xyzq)
    on, _ = ref.eval_field(xyzq=wl.xyzq, verts=wl.verts, sigma=wl.sigma, eps_pp=wl.eps_pp, eps_panel=wl.eps_panel,
                           flags=ref.NBODY)
    ctx.set_softening(wl.eps_pp, wl.eps_panel)
    ctx.set_panels(dev(torch_cuda, wl.verts), dev(torch_cuda, wl.sigma))
    ctx.set_charges(dev(torch_cuda, wl.xyzq))
    gp = ctx.eval_at_charges(flags=api.PANELS | api.PANELS_EXACT)
    gb = ctx.eval_at_charges(flags=api.NBODY | api.PANELS | api.PANELS_EXACT)
    torch_cuda.cuda.synchronize()
    assert_parity(gp.cpu().numpy(), exact, "cfg2/4 exact panels")
    assert_parity(gb.cpu().numpy(), on + exact, "cfg2/4 nbody + exact panels")


def test_config3_full_size_sampled(torch_cuda, api, ctx, ref):
    """Full-size config 3 in the bench's launch configuration; 768 sampled charges + the 128 closest to the foil."""
    wl = W.make_workload(3)
    ctx.set_softening(wl.eps_pp, wl.eps_panel)
    ctx.set_panels(dev(torch_cuda, wl.verts), dev(torch_cuda, wl.sigma))
    ctx.set_charges(dev(torch_cuda, wl.xyzq))
    g = ctx.eval_at_charges(flags=api.PANELS | api.PANELS_EXACT)
    g7 = ctx.eval_at_charges(flags=api.PANELS)
    torch_cuda.cuda.synchronize()
    g, g7 = g.cpu().numpy(), g7.cpu().numpy()
    assert np.isfinite(g).all()
    rng = np.random.default_rng([17, 3])
    changed = np.linalg.norm(g[:, :3] - g7[:, :3], axis=1) / np.linalg.norm(g7[:, :3], axis=1)
    idx = np.unique(np.concatenate([rng.choice(wl.n_charges, 768, replace=False), np.argsort(changed)[-128:]]))
    exact = ref.eval_panels_analytic(wl.verts, wl.sigma, wl.xyzq[idx])
    assert_parity(g[idx], exact, "cfg3 exact panels, sampled")


@pytest.mark.parametrize("cfg,n_sample", [(4, 256), (5, 1024)])
def test_configs_4_and_5_full_size_sampled(torch_cuda, api, ctx, ref, cfg, n_sample):
    """Measured (B200, round 1): E rel-L2 1.7e-6 (cfg 4) and 1.0e-6 (cfg 5) with the exact flag; the 7-point sum alone
    is 2.5e-2 and 1.6e-1 away from the exact integrals on the same samples (cfg 5's grid points lie on and inside
    the foil)."""
    wl = W.make_workload(cfg)
    tg = wl.points if wl.points is not None else wl.xyzq
    g = _gpu_panels(torch_cuda, api, ctx, wl, tg, api.PANELS | api.PANELS_EXACT)
    assert np.isfinite(g).all()
    rng = np.random.default_rng([17, cfg])
    idx = np.sort(rng.choice(len(tg), n_sample, replace=False))
    exact = ref.eval_panels_analytic(wl.verts, wl.sigma, tg[idx])
    assert_parity(g[idx], exact, "cfg%d exact panels, sampled" % cfg)


def _one_panel_workload(sigma=2e-5):
    verts = np.array([[[10 * UM, 10 * UM, 5 * UM], [16 * UM, 11 * UM, 5.5 * UM], [11 * UM, 15 * UM, 4.5 * UM]]],
                     dtype=np.float32)
    return W.Workload("one-panel", 0, np.zeros((0, 4), np.float32), verts, np.array([sigma], np.float32), 0.0)


def test_targets_on_and_next_to_a_panel(torch_cuda, api, ctx, ref):
    """Heights from 1 nm to 10 um above interior points, points in the panel's plane (inside, outside, on the
    extension of an edge), the vertices and edge midpoints themselves: finite everywhere and equal to the oracle."""
    wl = _one_panel_workload()
    v = wl.verts[0].astype(np.float64)
    n = np.cross(v[1] - v[0], v[2] - v[0])
    n /= np.linalg.norm(n)
    bary = np.array([[1 / 3, 1 / 3, 1 / 3], [0.8, 0.1, 0.1], [0.05, 0.9, 0.05], [0.5, 0.499, 0.001]])
    inside = bary @ v
    pts = [inside + h * n for h in (1e-9, 1e-8, 1e-7, 1e-6, 1e-5, -1e-9, -1e-7, -1e-5)]
    pts.append(inside)                                                       # (nearly) in the plane, inside
    pts.append(np.array([v[0] + 1.7 * (v[1] - v[0]), v[0] - 0.4 * (v[2] - v[0]), 2 * inside[0] - v[2] + 3 * (v[1] - v[0])]))
    pts.append(np.array([v[0], v[1], v[2], 0.5 * (v[0] + v[1]), 0.5 * (v[1] + v[2])]))
    targets = _pad4(np.concatenate(pts))
    g = _gpu_panels(torch_cuda, api, ctx, wl, targets, api.PANELS | api.PANELS_EXACT)
    exact = ref.eval_panels_analytic(wl.verts, wl.sigma, targets)
    assert np.isfinite(g).all() and np.isfinite(exact).all()
    # fp32 targets a nanometre from the sheet: compare per component against the field scale sigma/(2 eps0)
    scale_e = 2e-5 / (2 * 8.8541878128e-12)
    scale_p = np.abs(exact[:, 3]).max()
    sing = len(targets) - 5                                                  # the last 5 sit on vertices / edges
    assert np.abs(g[:sing, :3] - exact[:sing, :3]).max() <= 2e-5 * scale_e
    assert np.abs(g[:, 3] - exact[:, 3]).max() <= 2e-6 * scale_p             # phi is regular everywhere
    # on a vertex / an edge the in-plane field is log-singular: fp32 vs fp64 input rounding decides the value; both
    # sides drop the singular term only at exact coincidence, so only finiteness is asserted there (above)


def test_new_sigma_is_used_and_geometry_kept(torch_cuda, api, ctx, ref):
    wl = W.make_workload(1)
    rng = np.random.default_rng([17, 5])
    sigma2 = rng.normal(0, 3e-6, wl.n_panels).astype(np.float32)
    ctx.set_panels(dev(torch_cuda, wl.verts), dev(torch_cuda, wl.sigma))
    pts = dev(torch_cuda, wl.xyzq[:1500])
    ctx.eval_at_points(pts, flags=api.PANELS | api.PANELS_EXACT)
    size = ctx.near_list_size
    ctx.set_sigma(dev(torch_cuda, sigma2))
    g = ctx.eval_at_points(pts, flags=api.PANELS | api.PANELS_EXACT)
    torch_cuda.cuda.synchronize()
    assert ctx.near_list_size == size
    assert_parity(g.cpu().numpy(), ref.eval_panels_analytic(wl.verts, sigma2, wl.xyzq[:1500]), "after set_sigma")


def test_near_factor_controls_the_error_and_results_are_reproducible(torch_cuda, api, ctx, ref):
    wl = W.make_workload(2, charge_div=16, mesh_div=2)
    exact = ref.eval_panels_analytic(wl.verts, wl.sigma, wl.xyzq)
    errs = {}
    for f in (1.0, 2.0, 3.0, 5.0):
        ctx.set_near_field(f)
        errs[f] = field_errors(_gpu_panels(torch_cuda, api, ctx, wl, wl.xyzq, api.PANELS | api.PANELS_EXACT), exact)
    assert errs[1.0]["E_rel_l2"] > errs[2.0]["E_rel_l2"] > errs[3.0]["E_rel_l2"] * 1.5, errs
    assert errs[3.0]["E_rel_l2"] <= 2e-5 and errs[5.0]["E_rel_l2"] <= 2e-5, errs
    ctx.set_near_field(3.0)
    a = _gpu_panels(torch_cuda, api, ctx, wl, wl.xyzq, api.PANELS | api.PANELS_EXACT)
    b = _gpu_panels(torch_cuda, api, ctx, wl, wl.xyzq, api.PANELS | api.PANELS_EXACT)   # lists rebuilt from scratch
    assert np.array_equal(a, b)


def test_flag_validation_and_degenerate_inputs(torch_cuda, api, ctx, ref):
    wl = W.make_workload(1)
    pts = dev(torch_cuda, wl.xyzq[:64])
    ctx.set_panels(dev(torch_cuda, wl.verts), dev(torch_cuda, wl.sigma))
    ctx.set_charges(dev(torch_cuda, wl.xyzq))
    with pytest.raises(api.ObemError):
        ctx.eval_at_points(pts, flags=api.PANELS_EXACT)                      # needs OBEM_PANELS
    with pytest.raises(api.ObemError):
        ctx.eval_at_points(pts, flags=api.NBODY | api.PANELS_EXACT)
    with pytest.raises(api.ObemError):
        ctx.set_near_field(0.0)
    # no panels at all, and a set made of degenerate triangles only: the exact flag adds nothing
    ctx.set_panels(torch_cuda.zeros((0, 3, 3), device="cuda"), torch_cuda.zeros((0,), device="cuda"))
    z = ctx.eval_at_points(pts, flags=api.PANELS | api.PANELS_EXACT)
    torch_cuda.cuda.synchronize()
    assert float(z.abs().max()) == 0.0
    deg = np.zeros((3, 3, 3), dtype=np.float32)
    deg[1, :, 0] = [1e-5, 2e-5, 3e-5]                                        # collinear
    deg[2] = 4e-5                                                            # a point
    ctx.set_panels(dev(torch_cuda, deg), dev(torch_cuda, np.ones(3, np.float32)))
    z = ctx.eval_at_points(pts, flags=api.PANELS | api.PANELS_EXACT)
    torch_cuda.cuda.synchronize()
    assert float(z.abs().max()) == 0.0
    # one real panel among degenerate ones, targets far outside the cell grid and inside it
    mix = np.concatenate([deg, _one_panel_workload().verts])
    sig = np.array([1, 1, 1, 2e-5], np.float32)
    t = _pad4(np.array([[12e-6, 12e-6, 5.3e-6], [1.0, 1.0, 1.0], [-3e-3, 0, 0], [12e-6, 12e-6, 9e-6]]))
    ctx.set_panels(dev(torch_cuda, mix), dev(torch_cuda, sig))
    g = ctx.eval_at_points(dev(torch_cuda, t), flags=api.PANELS | api.PANELS_EXACT)
    torch_cuda.cuda.synchronize()
    assert_parity(g.cpu().numpy(), ref.eval_panels_analytic(mix, sig, t), "mixed degenerate set")

"""GPU edge cases and API behaviour of libobem.so against the oracle (degenerate cases of the method,
empty inputs, error codes, host-buffer entry points, target ranges).  `pytest -m gpu`.
"""
import numpy as np
import pytest

from paper_2110_09214_b200 import workloads as W
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


@pytest.fixture()
def ctx(api):
    c = api.Context(0)
    yield c
    c.destroy()


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def small_problem(seed=3, n=3000, npan=200):
    rng = np.random.default_rng([5, seed])
    xyzq = np.zeros((n, 4), dtype=np.float32)
    xyzq[:, :3] = rng.uniform(0, 80 * UM, (n, 3))
    xyzq[:, 3] = rng.choice([-QE, QE], n)
    verts = (rng.uniform(0, 80 * UM, (npan, 1, 3)) + rng.uniform(-2 * UM, 2 * UM, (npan, 3, 3))).astype(np.float32)
    verts[..., 2] += 120 * UM
    sigma = rng.normal(0, 1e-5, npan).astype(np.float32)
    return xyzq, verts, sigma


def test_panel_sources_match_oracle_quadrature(torch_cuda, api, ctx, ref):
    wl = W.make_workload(2, charge_div=64, mesh_div=2)
    ctx.set_panels(dev(torch_cuda, wl.verts), dev(torch_cuda, wl.sigma))
    got = ctx.get_panel_sources().cpu().numpy().astype(np.float64)
    exp = ref.panel_sources(wl.verts, wl.sigma)
    assert got.shape == exp.shape
    # positions: derived in fp64, stored as fp32 (frame origin + offset), read back rounded once to fp32
    assert np.all(np.abs(got[:, :3] - exp[:, :3]) <= 0.51 * np.spacing(np.abs(exp[:, :3]).astype(np.float32)) + 1e-12)
    assert np.allclose(got[:, 3], exp[:, 3], rtol=1e-7, atol=0)


def test_set_sigma_equals_set_panels(torch_cuda, api, ctx):
    xyzq, verts, sigma = small_problem()
    sigma2 = (sigma * 3.0 + 1e-6).astype(np.float32)
    ctx.set_charges(dev(torch_cuda, xyzq))
    ctx.set_panels(dev(torch_cuda, verts), dev(torch_cuda, sigma))
    ctx.set_sigma(dev(torch_cuda, sigma2))
    a = ctx.eval_at_charges(flags=api.PANELS).cpu().numpy()
    ctx.set_panels(dev(torch_cuda, verts), dev(torch_cuda, sigma2))
    b = ctx.eval_at_charges(flags=api.PANELS).cpu().numpy()
    assert np.array_equal(a, b)


def test_unsoftened_coincident_and_on_quadrature_point(torch_cuda, api, ctx, ref):
    # eps = 0: two different charges at one position contribute 0 to each other (reading A4), the self
    # term is dropped, and a target sitting exactly on a quadrature point skips that point.
    xyzq, verts, sigma = small_problem(seed=4, n=600, npan=50)
    xyzq[10, :3] = xyzq[20, :3]
    ctx.set_panels(dev(torch_cuda, verts), dev(torch_cuda, sigma))
    src = ctx.get_panel_sources().cpu().numpy()
    xyzq[30, :3] = src[35, :3]      # centroid point (k = 0) of panel 5 = its frame origin: distance exactly 0
    ctx.set_softening(0.0, 0.0)
    ctx.set_charges(dev(torch_cuda, xyzq))
    g_n = ctx.eval_at_charges(flags=api.NBODY).cpu().numpy()
    on, op = ref.eval_field(xyzq=xyzq, verts=verts, sigma=sigma, eps_pp=0.0)
    assert np.isfinite(g_n).all()
    assert_parity(g_n, on, "eps=0 nbody with coincident pair")
    # the panel branch of the repair pass: the zero-distance quadrature point contributes 0 and the VALUE is the
    # oracle's (the other 6 points of that panel and all other panels)
    g_p = ctx.eval_at_charges(flags=api.PANELS).cpu().numpy()
    assert np.isfinite(g_p).all()
    assert_parity(g_p, op, "eps=0 panels with a charge on a quadrature point")
    g_b = ctx.eval_at_charges(flags=api.NBODY | api.PANELS).cpu().numpy()
    assert_parity(g_b, on + op, "eps=0 both, two repaired targets")
    # the same through eval_at_points: a free point (a field-map node) exactly on that quadrature point, another
    # exactly on a charge (no index exclusion there: zero distance contributes 0)
    pts = xyzq[25:40].copy()
    pts[3, :3] = xyzq[10, :3]
    g_q = ctx.eval_at_points(dev(torch_cuda, pts), flags=api.NBODY | api.PANELS).cpu().numpy()
    qn, qp = ref.eval_field(xyzq=xyzq, verts=verts, sigma=sigma, targets=pts, self_index=None, eps_pp=0.0)
    assert np.isfinite(g_q).all()
    assert_parity(g_q, qn + qp, "eps=0 points on a quadrature point / on a charge")


def test_unsoftened_coincident_pair_through_the_nn_path(torch_cuda, api, ctx, ref):
    """LIST branch of the repair pass: obem_eval_at_charges_nn at eps = 0 with two different charges at one position.
    theta = 0 makes the NN sum the exact sum, so the plain oracle applies."""
    xyzq, _, _ = small_problem(seed=14, n=3000, npan=0)
    xyzq[100, :3] = xyzq[2900, :3]
    xyzq[7, :3] = xyzq[8, :3]
    ctx.set_softening(0.0, 0.0)
    ctx.set_nn_theta(0.0)
    ctx.set_charges(dev(torch_cuda, xyzq))
    g = ctx.eval_at_charges_nn(flags=api.NBODY).cpu().numpy()
    on, _ = ref.eval_field(xyzq=xyzq, eps_pp=0.0, flags=ref.NBODY)
    assert np.isfinite(g).all()
    assert_parity(g, on, "eps=0 NN path (theta = 0) with coincident pairs")


def test_more_bad_targets_than_the_repair_list_holds(torch_cuda, api, ctx, ref):
    """eval_at_points at the charges' own positions with eps = 0: EVERY target sits on a source.  The repair list
    (2^16 entries) cannot overflow silently: beyond it the pass scans the results for non-finite values.  70,000
    targets overflow it; sampled values are the oracle's and nothing is left inf/NaN."""
    xyzq, _, _ = small_problem(seed=15, n=70000, npan=0)
    ctx.set_softening(0.0, 0.0)
    ctx.set_charges(dev(torch_cuda, xyzq))
    g = ctx.eval_at_points(dev(torch_cuda, xyzq), flags=api.NBODY).cpu().numpy()
    assert np.isfinite(g).all()
    idx = np.sort(np.random.default_rng(15).choice(70000, 2000, replace=False))
    on, _ = ref.eval_field(xyzq=xyzq, targets=xyzq[idx], self_index=None, eps_pp=0.0, flags=ref.NBODY)
    assert_parity(g[idx], on, "every target on a source")


def test_softened_coincident_pair_phi(torch_cuda, api, ctx, ref):
    xyzq, verts, sigma = small_problem(seed=6, n=500, npan=0)
    xyzq[1, :3] = xyzq[0, :3]
    ctx.set_softening(0.1 * UM, 0.0)
    ctx.set_charges(dev(torch_cuda, xyzq))
    g = ctx.eval_at_charges(flags=api.NBODY).cpu().numpy()
    on, _ = ref.eval_field(xyzq=xyzq, eps_pp=0.1 * UM, flags=ref.NBODY)
    assert_parity(g, on, "softened coincident pair")


def test_points_nbody_has_no_exclusion(torch_cuda, api, ctx, ref):
    xyzq, verts, sigma = small_problem(seed=8, n=700, npan=60)
    ctx.set_softening(0.1 * UM, 0.0)
    ctx.set_charges(dev(torch_cuda, xyzq))
    ctx.set_panels(dev(torch_cuda, verts), dev(torch_cuda, sigma))
    pts = xyzq.copy()
    g = ctx.eval_at_points(dev(torch_cuda, pts), flags=api.NBODY | api.PANELS).cpu().numpy()
    on, op = ref.eval_field(xyzq=xyzq, verts=verts, sigma=sigma, targets=pts, self_index=None, eps_pp=0.1 * UM)
    assert_parity(g, on + op, "points at the charges, no exclusion")


def test_range_equals_full(torch_cuda, api, ctx):
    xyzq, verts, sigma = small_problem(seed=9, n=5000, npan=100)
    ctx.set_softening(0.1 * UM, 0.0)
    ctx.set_charges(dev(torch_cuda, xyzq))
    ctx.set_panels(dev(torch_cuda, verts), dev(torch_cuda, sigma))
    full = ctx.eval_at_charges().cpu().numpy()
    for first, count in [(0, 5000), (0, 1), (4999, 1), (1234, 2049), (2048, 2048), (17, 0)]:
        part = ctx.eval_at_charges_range(first, count).cpu().numpy()
        # same sources in the same block order -> only the tile split differs; allow fp32 rounding
        assert part.shape == (count, 4)
        if count:
            assert np.allclose(part, full[first:first + count], rtol=2e-5, atol=1e-6 * np.abs(full).max())


def test_host_entry_points_match_device_path(torch_cuda, api, ctx, ref):
    xyzq, verts, sigma = small_problem(seed=10, n=4100, npan=129)
    ctx.set_softening(0.1 * UM, 0.0)
    out_h = ctx.field_at_charges_host(xyzq, verts, sigma)
    ctx.set_charges(dev(torch_cuda, xyzq))
    ctx.set_panels(dev(torch_cuda, verts), dev(torch_cuda, sigma))
    out_d = ctx.eval_at_charges().cpu().numpy()
    assert np.array_equal(out_h, out_d)
    on, op = ref.eval_field(xyzq=xyzq, verts=verts, sigma=sigma, eps_pp=0.1 * UM)
    assert_parity(out_h, on + op, "host entry point")
    pts = xyzq[:777].copy()
    pts[:, :3] += np.float32(0.3 * UM)
    out_p = ctx.field_at_points_host(pts, flags=api.PANELS)      # verts=None: keep the panels already set
    _, op2 = ref.eval_field(verts=verts, sigma=sigma, targets=pts, flags=ref.PANELS)
    assert_parity(out_p, op2, "host points entry point")


def test_empty_and_state_errors(torch_cuda, api, ctx):
    torch = torch_cuda
    with pytest.raises(api.ObemError) as e:
        ctx.eval_at_charges()
    assert e.value.status == -2                                # OBEM_ESTATE
    with pytest.raises(api.ObemError) as e:
        ctx.set_sigma(torch.zeros(3, device="cuda"))
    assert e.value.status == -2
    empty4 = torch.zeros((0, 4), device="cuda")
    ctx.set_charges(empty4)
    assert ctx.n_charges == 0
    out = ctx.eval_at_charges(flags=api.NBODY)
    assert tuple(out.shape) == (0, 4)
    with pytest.raises(api.ObemError) as e:
        ctx.eval_at_charges(flags=api.PANELS)                  # panels never set
    assert e.value.status == -2
    ctx.set_panels(torch.zeros((0, 3, 3), device="cuda"), torch.zeros(0, device="cuda"))
    assert ctx.n_panels == 0
    pts = torch.rand((100, 4), device="cuda")
    out = ctx.eval_at_points(pts, flags=api.NBODY | api.PANELS)  # both source sets empty -> zeros
    assert torch.all(out == 0)
    with pytest.raises(api.ObemError) as e:
        ctx.eval_at_points(pts, flags=4)
    assert e.value.status == -1                                # OBEM_EINVAL
    with pytest.raises(api.ObemError) as e:
        ctx.set_softening(-1.0, 0.0)
    assert e.value.status == -1
    x = torch.rand((10, 4), device="cuda")
    ctx.set_charges(x)
    with pytest.raises(api.ObemError) as e:
        ctx.eval_at_charges_range(5, 6)
    assert e.value.status == -1
    with pytest.raises(api.ObemError) as e:
        ctx.set_sigma(torch.zeros(3, device="cuda"))           # count differs from the panel set (0)
    assert e.value.status == -1
    assert ctx.kernel_launches > 0


def test_degenerate_panel_contributes_zero(torch_cuda, api, ctx):
    xyzq, verts, sigma = small_problem(seed=12, n=300, npan=4)
    verts[:] = verts[:, :1, :]          # all three vertices equal: A = 0
    ctx.set_charges(dev(torch_cuda, xyzq))
    ctx.set_panels(dev(torch_cuda, verts), dev(torch_cuda, sigma))
    g = ctx.eval_at_charges(flags=api.PANELS)
    assert torch_cuda.all(g == 0)


def test_runs_on_a_side_stream(torch_cuda, api, ctx, ref):
    torch = torch_cuda
    xyzq, verts, sigma = small_problem(seed=13, n=2500, npan=90)
    s = torch.cuda.Stream()
    ctx.set_softening(0.05 * UM, 0.0)
    with torch.cuda.stream(s):
        dx, dv, ds = dev(torch, xyzq), dev(torch, verts), dev(torch, sigma)
        ctx.set_charges(dx, stream=s)
        ctx.set_panels(dv, ds, stream=s)
        out = ctx.eval_at_charges(stream=s)
    s.synchronize()
    on, op = ref.eval_field(xyzq=xyzq, verts=verts, sigma=sigma, eps_pp=0.05 * UM)
    assert_parity(out.cpu().numpy(), on + op, "side stream")


def test_a_time_step_can_be_captured_in_a_cuda_graph(torch_cuda, api, ctx):
    """Every entry point only enqueues work on the caller's stream (no hidden synchronisation, no allocation once the
    buffers have their size), so a whole time step -- set_charges + N-body + panels + Euler update -- can be captured
    in a CUDA graph and replayed; the replay gives bit-identical results."""
    torch = torch_cuda
    wl = W.make_workload(1)
    ctx.set_softening(wl.eps_pp, wl.eps_panel)
    ctx.set_panels(dev(torch, wl.verts), dev(torch, wl.sigma))
    x0 = dev(torch, wl.xyzq)
    v0 = torch.zeros_like(x0)
    v0[:, 3] = 9.1093837015e-31
    # eager reference: two Euler steps (also sizes every library-owned buffer)
    xe, ve = x0.clone(), v0.clone()
    ctx.step_euler(xe, ve, 25e-15)
    ctx.step_euler(xe, ve, 25e-15)
    torch.cuda.synchronize()
    xg, vg = x0.clone(), v0.clone()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        with torch.cuda.graph(g, stream=s):
            ctx.step_euler(xg, vg, 25e-15, stream=s)
    xg.copy_(x0), vg.copy_(v0)                    # capture does not execute: reset the state, then replay twice
    g.replay()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(xg, xe) and torch.equal(vg, ve)


def test_results_are_bitwise_reproducible_and_independent_of_other_work(torch_cuda, api, ctx):
    """No atomics on the data path: split tiles are summed in a fixed order by the fix-up kernel, so two evaluations
    of the same inputs agree bit for bit -- also when other evaluations (other sizes, other contexts) ran in between."""
    torch = torch_cuda
    wl = W.make_workload(2, charge_div=2, mesh_div=2)          # 32768 charges: 16 tiles split among 148 CTAs
    ctx.set_softening(wl.eps_pp, wl.eps_panel)
    ctx.set_panels(dev(torch, wl.verts), dev(torch, wl.sigma))
    ctx.set_charges(dev(torch, wl.xyzq))
    a = ctx.eval_at_charges(flags=api.NBODY | api.PANELS).clone()
    other = api.Context(0)
    small = W.make_workload(1)
    other.set_softening(small.eps_pp, 0.0)
    other.set_charges(dev(torch, small.xyzq))
    other.eval_at_charges(flags=api.NBODY)
    ctx.eval_at_points(dev(torch, wl.xyzq[:1000]), flags=api.PANELS)
    b = ctx.eval_at_charges(flags=api.NBODY | api.PANELS)
    ex1 = ctx.eval_at_charges(flags=api.NBODY | api.PANELS | api.PANELS_EXACT).clone()
    ex2 = ctx.eval_at_charges(flags=api.NBODY | api.PANELS | api.PANELS_EXACT)
    torch.cuda.synchronize()
    other.destroy()
    assert torch.equal(a, b)
    assert torch.equal(ex1, ex2)

"""GPU parity of the steps adjacent to the hot path against the fp64 oracle
(oracle/obem_ref_next.c), through the C ABI: influence of the particles on the cells (Eq 3.3/3.4), right-hand
side (Eq 3.5/3.6), sigma = M^-1 b, and the chained dynamic update.  `pytest -m gpu`.

Tolerances.  Influence: the north_star bars (rel-L2 2e-5, per-cell 1e-3) on (Ebar, Vbar); Ebar.n: rel-L2 2e-5
and per-cell error <= 1e-3 of max(|Ebar.n|, 0.1 rms) (it changes sign).  Mat-vec: fp32 dot of n terms with 128
partial sums: |d sigma_i| <= 4e-6 * sum_j |M_ij b_j|, rel-L2 2e-5.
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


def _assert_en(got, exp, what):
    got = np.asarray(got, dtype=np.float64)
    rms = float(np.sqrt((exp ** 2).mean()))
    l2 = float(np.sqrt(((got - exp) ** 2).sum() / (exp ** 2).sum()))
    mx = float((np.abs(got - exp) / np.maximum(np.abs(exp), 0.1 * rms)).max())
    assert l2 <= 2e-5, "%s: Ebar.n rel-L2 %.3e" % (what, l2)
    assert mx <= 1e-3, "%s: Ebar.n per-cell max %.3e" % (what, mx)


def _gpu_influence(torch, ctx, wl):
    ctx.set_softening(wl.eps_pp, wl.eps_panel)
    ctx.set_panels(dev(torch, wl.verts), dev(torch, wl.sigma))
    ctx.set_charges(dev(torch, wl.xyzq))
    infl, en = ctx.influence_on_panels()
    torch.cuda.synchronize()
    return infl.cpu().numpy(), en.cpu().numpy()


def test_influence_config1_all_cells(torch_cuda, api, ctx, ref):
    wl = W.make_workload(1)
    g_infl, g_en = _gpu_influence(torch_cuda, ctx, wl)
    o_infl, o_en, o_na = ref.influence(wl.xyzq, wl.verts, eps=wl.eps_panel)
    assert_parity(g_infl, o_infl, "cfg1 influence")
    _assert_en(g_en, o_en, "cfg1")
    na = ctx.get_panel_normals().cpu().numpy().astype(np.float64)
    assert np.allclose(na[:, :3], o_na[:, :3], atol=2e-7) and np.allclose(na[:, 3], o_na[:, 3], rtol=2e-7)


def test_influence_config2_reduced_all_cells(torch_cuda, api, ctx, ref):
    wl = W.make_workload(2, charge_div=4, mesh_div=2)     # 16384 charges, 4096 cells (28672 targets: ragged tile)
    g_infl, g_en = _gpu_influence(torch_cuda, ctx, wl)
    o_infl, o_en, _ = ref.influence(wl.xyzq, wl.verts, eps=wl.eps_panel)
    assert_parity(g_infl, o_infl, "cfg2/4 influence")
    _assert_en(g_en, o_en, "cfg2/4")


def test_influence_config3_full_size_sampled_cells(torch_cuda, api, ctx, ref):
    wl = W.make_workload(3)
    g_infl, g_en = _gpu_influence(torch_cuda, ctx, wl)
    assert np.isfinite(g_infl).all() and np.isfinite(g_en).all()
    rng = np.random.default_rng([12, 3])
    mag = np.linalg.norm(g_infl[:, :3], axis=1)
    idx = np.unique(np.concatenate([rng.choice(wl.n_panels, 384, replace=False), np.argsort(mag)[-32:],
                                    np.argsort(mag)[:32], [0, wl.n_panels - 1]]))
    o_infl, o_en, _ = ref.influence(wl.xyzq, wl.verts[idx], eps=wl.eps_panel)
    assert_parity(g_infl[idx], o_infl, "cfg3 influence sampled")
    _assert_en(g_en[idx], o_en, "cfg3 sampled")


def test_influence_softened_and_degenerate_cases(torch_cuda, api, ctx, ref):
    rng = np.random.default_rng([12, 9])
    n, npan = 777, 130
    xyzq = np.zeros((n, 4), dtype=np.float32)
    xyzq[:, :3] = rng.uniform(0, 60 * UM, (n, 3))
    xyzq[:, 3] = rng.choice([-QE, QE], n)
    verts = (rng.uniform(0, 60 * UM, (npan, 1, 3)) + rng.uniform(-2 * UM, 2 * UM, (npan, 3, 3))).astype(np.float32)
    verts[..., 2] -= 70 * UM
    verts[5, 2] = verts[5, 1]                              # a degenerate (zero-area) cell: n = 0, Ebar.n = 0
    sigma = np.zeros(npan, dtype=np.float32)
    for eps_panel in (0.0, 0.5 * UM):
        ctx.set_softening(0.1 * UM, eps_panel)
        ctx.set_panels(dev(torch_cuda, verts), dev(torch_cuda, sigma))
        ctx.set_charges(dev(torch_cuda, xyzq))
        infl, en = ctx.influence_on_panels()
        o_infl, o_en, _ = ref.influence(xyzq, verts, eps=eps_panel)
        assert_parity(infl.cpu().numpy(), o_infl, "softened %g" % eps_panel)
        _assert_en(en.cpu().numpy(), o_en, "softened %g" % eps_panel)
        assert en.cpu().numpy()[5] == 0.0
    # no charges: zero influence; en pointer may be NULL
    ctx.set_charges(torch_cuda.empty((0, 4), dtype=torch_cuda.float32, device="cuda"))
    infl, en = ctx.influence_on_panels(want_en=False)
    assert en is None and np.all(infl.cpu().numpy() == 0)
    # never-set state
    c2 = api.Context(0)
    with pytest.raises(api.ObemError):
        c2.influence_on_panels()
    c2.destroy()


def test_rhs_matches_oracle(torch_cuda, api, ctx, ref):
    rng = np.random.default_rng([12, 4])
    npan = 5000
    kind = rng.integers(0, 2, npan).astype(np.int32)
    bc = np.where(kind == 0, rng.uniform(-500, 500, npan), rng.normal(0, 1e-5, npan)).astype(np.float32)
    deps = (rng.uniform(1.0, 3.0, npan) * EPS0).astype(np.float32)
    infl = rng.normal(0, 1e4, (npan, 4)).astype(np.float32)
    en = rng.normal(0, 1e5, npan).astype(np.float32)
    b = ctx.rhs_from_influence(dev(torch_cuda, kind), dev(torch_cuda, bc), dev(torch_cuda, deps),
                               dev(torch_cuda, infl), dev(torch_cuda, en)).cpu().numpy().astype(np.float64)
    exp = ref.rhs(kind, bc, deps, infl.astype(np.float64), en.astype(np.float64))
    scale = np.abs(bc.astype(np.float64)) + np.where(kind == 0, np.abs(infl[:, 3]), np.abs(deps.astype(np.float64) * en))
    assert np.all(np.abs(b - exp) <= 1.2e-7 * scale)       # one fp32 rounding of a two-term expression
    kind[7] = 3
    b = ctx.rhs_from_influence(dev(torch_cuda, kind), dev(torch_cuda, bc), dev(torch_cuda, deps),
                               dev(torch_cuda, infl), dev(torch_cuda, en)).cpu().numpy()
    assert np.isnan(b[7]) and np.isfinite(np.delete(b, 7)).all()


@pytest.mark.parametrize("n", [4, 16, 1000, 1024, 1028, 4096, 6148, 1023, 257])
def test_apply_inverse_matches_oracle(torch_cuda, api, ctx, ref, n):
    rng = np.random.default_rng([12, 5, n])
    m = rng.normal(0, 1, (n, n)).astype(np.float32)
    b = rng.normal(0, 1, n).astype(np.float32)
    got = ctx.apply_inverse(dev(torch_cuda, m), dev(torch_cuda, b)).cpu().numpy().astype(np.float64)
    exp = ref.matvec(m, b)
    bound = np.abs(m.astype(np.float64)) @ np.abs(b.astype(np.float64))
    assert np.all(np.abs(got - exp) <= 4e-6 * bound), float((np.abs(got - exp) / bound).max())
    assert np.sqrt(((got - exp) ** 2).sum() / (exp ** 2).sum()) <= 2e-5


def test_apply_inverse_leading_dimension_and_identity(torch_cuda, api, ctx, ref):
    torch = torch_cuda
    n, ld = 2048, 2052
    rng = np.random.default_rng([12, 6])
    big = rng.normal(0, 1, (n, ld)).astype(np.float32)
    b = rng.normal(0, 1, n).astype(np.float32)
    view = dev(torch, big)[:, :n]
    got = ctx.apply_inverse(view, dev(torch, b)).cpu().numpy().astype(np.float64)
    exp = ref.matvec(np.ascontiguousarray(big[:, :n]), b)
    bound = np.abs(big[:, :n].astype(np.float64)) @ np.abs(b.astype(np.float64))
    assert np.all(np.abs(got - exp) <= 4e-6 * bound)
    eye = torch.eye(n, dtype=torch.float32, device="cuda")
    assert np.array_equal(ctx.apply_inverse(eye, dev(torch, b)).cpu().numpy(), b)
    assert ctx.apply_inverse(torch.empty((0, 0), dtype=torch.float32, device="cuda"),
                             torch.empty((0,), dtype=torch.float32, device="cuda")).shape == (0,)


def test_dynamic_update_chain_matches_oracle_chain(torch_cuda, api, ctx, ref):
    """influence -> rhs -> M^-1 b -> set_sigma -> field at the charges, against the same chain through the oracle
    (each oracle stage fed with the oracle's own previous stage)."""
    torch = torch_cuda
    wl = W.make_workload(1)
    npan = wl.n_panels
    rng = np.random.default_rng([12, 7])
    kind = (np.arange(npan) % 3 == 0).astype(np.int32)                  # a third of the cells are dd
    bc = np.where(kind == 0, np.where(wl.verts[:, 0, 2] > 50 * UM, 300.0, -300.0), rng.normal(0, 1e-6, npan)).astype(np.float32)
    deps = np.full(npan, 2.5 * EPS0, dtype=np.float32)
    # a synthetic, well-conditioned "inverse" with the magnitude of a capacitance matrix (C/m^2 per V)
    minv = (np.eye(npan) * 1e-8 + rng.normal(0, 2e-11, (npan, npan))).astype(np.float32)
    ctx.set_softening(wl.eps_pp, wl.eps_panel)
    ctx.set_panels(dev(torch, wl.verts), dev(torch, wl.sigma))
    ctx.set_charges(dev(torch, wl.xyzq))
    sigma = ctx.update_sigma_dynamic(dev(torch, kind), dev(torch, bc), dev(torch, deps), dev(torch, minv))
    out = ctx.eval_at_charges(flags=api.PANELS)
    torch.cuda.synchronize()
    o_infl, o_en, _ = ref.influence(wl.xyzq, wl.verts, eps=wl.eps_panel)
    o_b = ref.rhs(kind, bc, deps, o_infl, o_en)
    o_sigma = ref.matvec(minv, o_b.astype(np.float32))
    g_sigma = sigma.cpu().numpy().astype(np.float64)
    assert np.sqrt(((g_sigma - o_sigma) ** 2).sum() / (o_sigma ** 2).sum()) <= 2e-5
    _, o_p = ref.eval_field(xyzq=wl.xyzq, verts=wl.verts, sigma=o_sigma.astype(np.float32), eps_panel=wl.eps_panel,
                            flags=ref.PANELS)
    assert_parity(out.cpu().numpy(), o_p, "field of the updated sigma")

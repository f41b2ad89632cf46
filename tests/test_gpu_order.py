"""GPU parity on charge arrays in the order the METHOD produces them (electron-ion pairs created as the avalanche
grows: signs interleaved) and on arrays with many distinct weights.  obem_set_charges
sorts the sources into class order, so that the kernels' uniform-block loop, the index
self-exclusion (Eq 3.8's p != p') and the partner tracking do not depend on the caller's order.
`pytest -m gpu`.
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


def _partners_ok(xyzq, eps, pd, pj, od, oj, idx):
    """The unique quantity (the distance) against the oracle; the reported index must be a valid opposite charge at
    that distance (near-ties between blocks are decided in fp32)."""
    pd = pd.astype(np.float64)
    none = oj < 0
    assert np.array_equal(pj[none], oj[none]) and np.all(np.isinf(pd[none]))
    has = ~none
    d2 = od[has] ** 2
    slack = 4.0 * np.spacing((d2 + eps * eps).astype(np.float32)).astype(np.float64)
    assert np.all(pd[has] ** 2 <= d2 * (1 + 3e-7) + slack)
    assert np.all(pd[has] >= od[has] * (1 - 1e-7))
    tj, ti = pj[has].astype(np.int64), idx[has]
    assert np.all(tj >= 0) and np.all(tj < xyzq.shape[0]) and np.all(tj != ti)
    assert np.all(xyzq[tj, 3] * xyzq[ti, 3] < 0)
    dd = np.linalg.norm(xyzq[tj, :3].astype(np.float64) - xyzq[ti, :3].astype(np.float64), axis=1)
    assert np.allclose(dd, pd[has], rtol=2e-7, atol=0)
    assert (tj == oj[has]).mean() > 0.999


def test_pair_order_config2_reduced_all_targets(torch_cuda, api, ctx, ref):
    """16384 interleaved charges (8 tiles, split between CTAs), all targets, against the oracle; and against the same
    charges in species order: the two evaluations sum the same sources in a different order only."""
    torch = torch_cuda
    base = W.make_workload(2, charge_div=4, mesh_div=2)
    wl = W.pair_creation_order(base)
    perm = wl.meta["perm"]
    assert not np.all(np.diff(wl.xyzq[:, 3]) >= 0)                      # the signs really are interleaved
    ctx.set_softening(wl.eps_pp, wl.eps_panel)
    ctx.set_panels(dev(torch, wl.verts), dev(torch, wl.sigma))
    ctx.set_charges(dev(torch, wl.xyzq))
    g = {f: ctx.eval_at_charges(flags=f).cpu().numpy() for f in (api.NBODY, api.PANELS, api.NBODY | api.PANELS)}
    on, op = ref.eval_field(xyzq=wl.xyzq, verts=wl.verts, sigma=wl.sigma, eps_pp=wl.eps_pp, eps_panel=wl.eps_panel)
    assert_parity(g[api.NBODY], on, "pair order, nbody")
    assert_parity(g[api.PANELS], op, "pair order, panels")
    assert_parity(g[api.NBODY | api.PANELS], on + op, "pair order, both")
    ctx.set_charges(dev(torch, base.xyzq))
    gs = ctx.eval_at_charges(flags=api.NBODY).cpu().numpy()
    scale = np.abs(gs).max(axis=0)
    assert np.all(np.abs(g[api.NBODY] - gs[perm]) <= 2e-5 * scale)


def test_species_order_is_kept(torch_cuda, api, ctx):
    """An array already grouped by class in ascending q (electrons, then ions -- the generators' order) is not
    reordered (the class sort is stable), so a permutation WITHIN the classes that keeps them grouped permutes the
    results and nothing else... and the evaluation does not depend on where the caller's buffer lives."""
    torch = torch_cuda
    wl = W.make_workload(1)
    ctx.set_softening(wl.eps_pp, 0.0)
    ctx.set_charges(dev(torch, wl.xyzq))
    a = ctx.eval_at_charges(flags=api.NBODY).clone()
    b = ctx.eval_at_charges(flags=api.NBODY)
    assert torch.equal(a, b)
    # swap two whole 256-blocks of electrons: the same blocks meet the same targets, in another block order
    x = wl.xyzq.copy()
    x[0:256], x[256:512] = wl.xyzq[256:512], wl.xyzq[0:256]
    ctx.set_charges(dev(torch, x))
    c = ctx.eval_at_charges(flags=api.NBODY).cpu().numpy()
    a = a.cpu().numpy()
    scale = np.abs(a).max(axis=0)
    assert np.all(np.abs(c[256:512] - a[0:256]) <= 1e-5 * scale) and np.all(np.abs(c[512:] - a[512:]) <= 1e-5 * scale)


@pytest.mark.parametrize("n,eps", [(5000, 0.1 * UM), (2049, 0.0), (700, 0.05 * UM)])
def test_many_distinct_weights(torch_cuda, api, ctx, ref, n, eps):
    """Every charge has its own weight (macro-particles), both signs, some exactly zero, +0 and -0: no block is
    uniform, the blocks are of one sign except at the two sign boundaries.  Field, potential and partners."""
    torch = torch_cuda
    rng = np.random.default_rng([17, n])
    xyzq = np.zeros((n, 4), dtype=np.float32)
    xyzq[:, :3] = rng.uniform(0, 60 * UM, (n, 3))
    xyzq[:, 3] = rng.uniform(0.2, 5.0, n) * QE * rng.choice([-1.0, 1.0], n)
    zero = rng.choice(n, n // 20, replace=False)
    xyzq[zero, 3] = 0.0
    xyzq[zero[::2], 3] = -0.0
    ctx.set_softening(eps, 0.0)
    ctx.set_charges(dev(torch, xyzq))
    out, pd, pj = ctx.eval_at_charges_partners(flags=api.NBODY)
    plain = ctx.eval_at_charges(flags=api.NBODY)
    assert torch.equal(out, plain)
    on, _ = ref.eval_field(xyzq=xyzq, eps_pp=eps, flags=ref.NBODY)
    assert_parity(out.cpu().numpy(), on, "distinct weights n=%d" % n)
    od, oj = ref.nearest_opposite(xyzq)
    _partners_ok(xyzq, eps, pd.cpu().numpy(), pj.cpu().numpy(), od, oj, np.arange(n))


def test_ranges_of_a_pair_ordered_set(torch_cuda, api, ctx, ref):
    """obem_eval_at_charges_range means the CALLER's indices [first, first + count) whatever the internal order:
    slices of an interleaved three-class set against the oracle and against the full evaluation, field and partners."""
    torch = torch_cuda
    n = 9000
    rng = np.random.default_rng([19, n])
    xyzq = np.zeros((n, 4), dtype=np.float32)
    xyzq[:, :3] = rng.uniform(0, 70 * UM, (n, 3))
    xyzq[:, 3] = rng.choice([-QE, QE, 2 * QE], n, p=[0.5, 0.4, 0.1])
    ctx.set_softening(0.1 * UM, 0.0)
    ctx.set_charges(dev(torch, xyzq))
    full, pdf, pjf = ctx.eval_at_charges_partners(flags=api.NBODY)
    full = full.cpu().numpy()
    on, _ = ref.eval_field(xyzq=xyzq, eps_pp=0.1 * UM, flags=ref.NBODY)
    assert_parity(full, on, "three classes, full")
    scale = np.abs(full).max(axis=0)
    for first, count in [(0, n), (0, 1), (n - 1, 1), (1234, 2049), (2048, 2048), (4500, 4500), (3, 8990), (17, 0)]:
        part, pd, pj = ctx.eval_at_charges_partners(flags=api.NBODY, first=first, count=count)
        assert tuple(part.shape) == (count, 4)
        if count == 0:
            continue
        part = part.cpu().numpy()
        assert_parity(part, on[first:first + count], "three classes, range %d+%d" % (first, count))
        assert np.all(np.abs(part - full[first:first + count]) <= 2e-5 * scale)
        assert torch.equal(pj, pjf[first:first + count]) and torch.equal(pd, pdf[first:first + count])
        plain = ctx.eval_at_charges_range(first, count, flags=api.NBODY)
        assert np.array_equal(plain.cpu().numpy(), part)


def test_pair_order_config3_full_size_sampled(torch_cuda, api, ctx, ref):
    """BASELINE.json configs[2] (1,048,576 charges, 65,536 panels) in pair-creation order, in the launch configuration
    bench.py times (`nbody_only_pair_order`): N-body + panels and the partners on sampled targets plus adversarial
    extras, against the oracle."""
    torch = torch_cuda
    wl = W.pair_creation_order(W.make_workload(3))
    ctx.set_softening(wl.eps_pp, wl.eps_panel)
    ctx.set_panels(dev(torch, wl.verts), dev(torch, wl.sigma))
    ctx.set_charges(dev(torch, wl.xyzq))
    out, pd, pj = ctx.eval_at_charges_partners(flags=api.NBODY | api.PANELS)
    torch.cuda.synchronize()
    g, pd, pj = out.cpu().numpy(), pd.cpu().numpy(), pj.cpu().numpy()
    assert np.isfinite(g).all()
    rng = np.random.default_rng([23, 3])
    nt = wl.n_charges
    mag = np.linalg.norm(g[:, :3], axis=1)
    idx = np.unique(np.concatenate([rng.choice(nt, 1024, replace=False), np.argsort(mag)[-64:], np.argsort(mag)[:64],
                                    np.argsort(np.abs(g[:, 3]))[-64:], np.argsort(pd)[:128], [0, nt - 1]]))
    on, op = ref.eval_field(xyzq=wl.xyzq, verts=wl.verts, sigma=wl.sigma, targets=wl.xyzq[idx],
                            self_index=idx.astype(np.int64), eps_pp=wl.eps_pp, eps_panel=wl.eps_panel)
    assert_parity(g[idx], on + op, "cfg3 pair order, sampled")
    od, oj = ref.nearest_opposite(wl.xyzq, idx=idx)
    _partners_ok(wl.xyzq, wl.eps_pp, pd[idx], pj[idx], od, oj, idx)


def test_reserve_after_set_discards_the_sets(torch_cuda, api, ctx):
    """obem_reserve with larger capacities re-allocates the library-owned buffers: the sets are discarded and the next
    evaluation says OBEM_ESTATE instead of reading uninitialised sources (include/obem.h)."""
    torch = torch_cuda
    wl = W.make_workload(1)
    ctx.set_softening(wl.eps_pp, 0.0)
    ctx.set_panels(dev(torch, wl.verts), dev(torch, wl.sigma))
    ctx.set_charges(dev(torch, wl.xyzq))
    a = ctx.eval_at_charges().clone()
    ctx.reserve(wl.n_charges, wl.n_panels)                              # nothing grows: the sets stay
    assert torch.equal(ctx.eval_at_charges(), a)
    ctx.reserve(4 * wl.n_charges, wl.n_panels)
    assert ctx.n_charges == -1 and ctx.n_panels == wl.n_panels
    with pytest.raises(api.ObemError) as e:
        ctx.eval_at_charges(flags=api.NBODY)
    assert e.value.status == -2
    ctx.reserve(0, 4 * wl.n_panels)
    assert ctx.n_panels == -1
    with pytest.raises(api.ObemError) as e:
        ctx.eval_at_points(dev(torch, wl.xyzq), flags=api.PANELS)
    assert e.value.status == -2
    ctx.set_panels(dev(torch, wl.verts), dev(torch, wl.sigma))
    ctx.set_charges(dev(torch, wl.xyzq))
    assert torch.equal(ctx.eval_at_charges(), a)


def test_pair_order_config3_nn_sampled_tiles(torch_cuda, api, ctx, ref):
    """The NN approximation on config 3's charges in pair-creation order: the k-d order is the
    library's own, so the caller's order only changes which rows the results land in.  Four sampled tiles against the
    NN oracle (identical near / far decisions: same unit count) at the path's tolerance."""
    from oracle import nn
    torch = torch_cuda
    wl = W.pair_creation_order(W.make_workload(3, mesh_div=8))
    ctx.set_softening(wl.eps_pp, 0.0)
    ctx.set_nn_theta(2.0)
    ctx.set_charges(dev(torch, wl.xyzq))
    got = ctx.eval_at_charges_nn(flags=api.NBODY)
    torch.cuda.synchronize()
    got = got.cpu().numpy()
    assert np.isfinite(got).all()
    units = ctx.nn_last_units()
    groups = np.sort(np.random.default_rng([61, 33]).choice(wl.n_charges // 2048, 4, replace=False))
    exp, tree = nn.nn_field(wl.xyzq, wl.eps_pp, 2.0, groups=groups, ref=ref)
    idx = np.nonzero(np.isfinite(exp[:, 0]))[0]
    assert idx.size == 4 * 2048
    assert_parity(got[idx], exp[idx], "cfg3 pair order, nn, sampled tiles")
    assert units == nn.units(tree, 2.0, wl.n_charges)


def test_e_only_is_bit_identical_in_E_and_zero_in_phi(torch_cuda, api, ctx, ref):
    """OBEM_NO_PHI (Eq 3.8 and 2.14 are field sums; the integrators read only E): E of the
    E-only instantiations equals E of the E + phi ones bit for bit, the phi lane is 0 -- at the charges (big tiles,
    pair order, split tiles), on a sub-range, at free points, and for a tiny problem (small-tile instantiations).  Not
    with the exact near-field correction or the partner by-product."""
    torch = torch_cuda
    wl = W.pair_creation_order(W.make_workload(2, charge_div=4, mesh_div=2))       # 16384 charges, 4096 panels
    tiny = W.make_workload(1)
    for w in (wl, tiny):
        ctx.set_softening(w.eps_pp, w.eps_panel)
        ctx.set_panels(dev(torch, w.verts), dev(torch, w.sigma))
        ctx.set_charges(dev(torch, w.xyzq))
        for flags in (api.NBODY, api.PANELS, api.NBODY | api.PANELS):
            full = ctx.eval_at_charges(flags=flags)
            eo = ctx.eval_at_charges(flags=flags | api.NO_PHI)
            assert torch.equal(eo[:, :3], full[:, :3]), "E differs, flags %d" % flags
            assert torch.all(eo[:, 3] == 0)
        part = ctx.eval_at_charges_range(1000, 2500, flags=api.NBODY | api.PANELS)
        part_eo = ctx.eval_at_charges_range(1000, 2500, flags=api.NBODY | api.PANELS | api.NO_PHI)
        assert torch.equal(part_eo[:, :3], part[:, :3]) and torch.all(part_eo[:, 3] == 0)
        pts = dev(torch, w.xyzq[:3000] + np.float32(0.2 * UM))
        a = ctx.eval_at_points(pts, flags=api.NBODY | api.PANELS)
        b = ctx.eval_at_points(pts, flags=api.NBODY | api.PANELS | api.NO_PHI)
        assert torch.equal(b[:, :3], a[:, :3]) and torch.all(b[:, 3] == 0)
    on, op = ref.eval_field(xyzq=tiny.xyzq, verts=tiny.verts, sigma=tiny.sigma, eps_pp=tiny.eps_pp)
    eo = ctx.eval_at_charges(flags=api.NBODY | api.PANELS | api.NO_PHI).cpu().numpy().astype(np.float64)
    dE = np.linalg.norm(eo[:, :3] - (on + op)[:, :3], axis=1)
    assert np.sqrt((dE ** 2).sum() / (np.linalg.norm((on + op)[:, :3], axis=1) ** 2).sum()) <= 2e-5
    with pytest.raises(api.ObemError) as e:
        ctx.eval_at_charges(flags=api.PANELS | api.PANELS_EXACT | api.NO_PHI)
    assert e.value.status == -1
    with pytest.raises(api.ObemError) as e:
        ctx.eval_at_charges_partners(flags=api.NBODY | api.NO_PHI)
    assert e.value.status == -1


def test_pair_order_config4_full_size_sampled(torch_cuda, api, ctx, ref):
    """BASELINE.json configs[3] (4,194,304 charges in two clouds 2 mm apart, 262,144 panels) in pair-creation order:
    the largest charge set, where the class order puts 2.1 M electrons before 2.1 M ions and the species sums reach
    ~200 x the net potential (the case that needs the fp64 second accumulation level)."""
    torch = torch_cuda
    wl = W.pair_creation_order(W.make_workload(4))
    ctx.set_softening(wl.eps_pp, wl.eps_panel)
    ctx.set_panels(dev(torch, wl.verts), dev(torch, wl.sigma))
    ctx.set_charges(dev(torch, wl.xyzq))
    g = ctx.eval_at_charges(flags=api.NBODY | api.PANELS)
    torch.cuda.synchronize()
    g = g.cpu().numpy()
    assert np.isfinite(g).all()
    rng = np.random.default_rng([23, 4])
    mag = np.linalg.norm(g[:, :3], axis=1)
    idx = np.unique(np.concatenate([rng.choice(wl.n_charges, 384, replace=False), np.argsort(mag)[-32:],
                                    np.argsort(np.abs(g[:, 3]))[:32], [0, wl.n_charges - 1]]))
    on, op = ref.eval_field(xyzq=wl.xyzq, verts=wl.verts, sigma=wl.sigma, targets=wl.xyzq[idx],
                            self_index=idx.astype(np.int64), eps_pp=wl.eps_pp, eps_panel=wl.eps_panel)
    assert_parity(g[idx], on + op, "cfg4 pair order, sampled")

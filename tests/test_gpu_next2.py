"""GPU parity of the integrators against the fp64 oracle stepper
(oracle/stepper.py) fed with the fp64 field oracle, through the C ABI.  `pytest -m gpu`.

Tolerances.  The state is fp32 and every sub-step is one FMA, so after k drifts a position
component differs from the fp64 scheme by at most k/2 ulp(x) plus h times the velocity error; a velocity component
by k/2 ulp(v) per kick plus the field tolerance (per-target 1e-3, north_star) times the kick.
"""
import numpy as np
import pytest

from paper_2110_09214_b200 import workloads as W

pytestmark = pytest.mark.gpu

UM = 1e-6
QE = 1.602176634e-19
ME = 9.1093837015e-31
M_ION = 40 * 1836.15267343 * ME          # Ar+
DT = 25e-15                              # "the time step was chosen to be 25 fs"


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


def _state(wl, seed):
    rng = np.random.default_rng([13, seed])
    n = wl.n_charges
    q = wl.xyzq[:, 3]
    vel = np.zeros((n, 4), dtype=np.float32)
    speed = np.where(q < 0, 6e5, 4e2)                                   # ~1 eV electrons, thermal Ar+
    vel[:, :3] = rng.normal(0, 1, (n, 3)) * speed[:, None]
    vel[:, 3] = np.where(q < 0, ME, M_ION)
    return vel


def _oracle_field(ref, wl, flags):
    def field(x):
        xyzq = np.concatenate([x, wl.xyzq[:, 3:4].astype(np.float64)], axis=1).astype(np.float32)
        on, op = ref.eval_field(xyzq=xyzq, verts=wl.verts, sigma=wl.sigma, eps_pp=wl.eps_pp,
                                eps_panel=wl.eps_panel, flags=flags)
        return (on + op)[:, :3]
    return field


def _ulp(a):
    return np.spacing(np.abs(a).astype(np.float32)).astype(np.float64)


def _check(x_g, v_g, x_o, v_o, kick_scale, n_drift, n_kick, h_total, what):
    ex = np.abs(x_g.astype(np.float64) - x_o)
    bx = 0.5 * n_drift * _ulp(x_o) + 1e-12 * np.abs(x_o)
    ev = np.abs(v_g.astype(np.float64) - v_o)
    bv = 0.5 * n_kick * _ulp(v_o) + 2e-3 * kick_scale[:, None] + 1e-30
    assert np.all(ev <= bv), "%s: velocity error %.3e x bound" % (what, float((ev / bv).max()))
    bx = bx + abs(h_total) * bv
    assert np.all(ex <= bx), "%s: position error %.3e x bound" % (what, float((ex / bx).max()))


@pytest.mark.parametrize("scheme", ["euler", "pefrl"])
def test_one_step_config1(torch_cuda, api, ctx, ref, scheme):
    from oracle import stepper
    torch = torch_cuda
    wl = W.make_workload(1)
    vel = _state(wl, 1)
    flags = api.NBODY | api.PANELS
    ctx.set_softening(wl.eps_pp, wl.eps_panel)
    ctx.set_panels(dev(torch, wl.verts), dev(torch, wl.sigma))
    d_x, d_v = dev(torch, wl.xyzq), dev(torch, vel)
    x0 = wl.xyzq[:, :3].astype(np.float64)
    v0 = vel[:, :3].astype(np.float64)
    qm = wl.xyzq[:, 3].astype(np.float64) / vel[:, 3].astype(np.float64)
    field = _oracle_field(ref, wl, ref.NBODY | ref.PANELS)
    e0 = np.linalg.norm(field(x0), axis=1)
    if scheme == "euler":
        ctx.step_euler(d_x, d_v, DT, flags=flags)
        x_o, v_o, _ = stepper.euler_step(x0, v0, qm, DT, field)
        nd, nk, ksum = 1, 1, 1.0
    else:
        ctx.step_pefrl(d_x, d_v, DT, flags=flags)
        x_o, v_o = stepper.pefrl_step(x0, v0, qm, DT, field)
        nd, nk, ksum = 5, 4, 1.85                                       # sum of |kick coefficients|
    torch.cuda.synchronize()
    x_g, v_g = d_x.cpu().numpy(), d_v.cpu().numpy()
    assert np.array_equal(x_g[:, 3], wl.xyzq[:, 3]) and np.array_equal(v_g[:, 3], vel[:, 3])   # q, m untouched
    assert np.abs(x_g[:, :3] - wl.xyzq[:, :3]).max() > 1e-9            # something moved
    _check(x_g[:, :3], v_g[:, :3], x_o, v_o, ksum * DT * np.abs(qm) * e0, nd, nk, DT, scheme)


def test_pefrl_is_reversible_and_beats_euler_on_a_bound_pair(torch_cuda, api, ctx, ref):
    """Two opposite charges on a circular orbit (N-body field only).  40 PEFRL steps forward then 40 backward
    return to the start to fp32 rounding; over a quarter period PEFRL stays on the circle, Euler spirals out."""
    torch = torch_cuda
    r = 1.0e-6
    ke = 8.9875517923e9
    vorb = np.sqrt(ke * QE * QE / (ME * r))
    period = 2 * np.pi * r / vorb
    xyzq = np.array([[0, 0, 0, QE], [r, 0, 0, -QE]], dtype=np.float32)
    vel = np.array([[0, -vorb * ME / M_ION, 0, M_ION], [0, vorb, 0, ME]], dtype=np.float32)
    ctx.set_softening(0.0, 0.0)
    n = 40
    h = float(0.25 * period / n)
    d_x, d_v = dev(torch, xyzq), dev(torch, vel)
    for _ in range(n):
        ctx.step_pefrl(d_x, d_v, h, flags=api.NBODY)
    xq = d_x.cpu().numpy()
    d = np.linalg.norm(xq[1, :3].astype(np.float64) - xq[0, :3])
    assert abs(d - r) < 2e-5 * r                                        # still on the circle ...
    assert abs(xq[1, 0]) < 2e-3 * r and abs(xq[1, 1] - r) < 2e-3 * r    # ... a quarter turn later
    for _ in range(n):
        ctx.step_pefrl(d_x, d_v, -h, flags=api.NBODY)
    back = d_x.cpu().numpy()
    assert np.abs(back[:, :3] - xyzq[:, :3]).max() < 2e-5 * r
    e_x, e_v = dev(torch, xyzq), dev(torch, vel)
    for _ in range(n):
        ctx.step_euler(e_x, e_v, h, flags=api.NBODY)
    xe = e_x.cpu().numpy()
    de = np.linalg.norm(xe[1, :3].astype(np.float64) - xe[0, :3])
    assert de - r > 100 * abs(d - r)                                   # first order: visibly off the circle


def test_drift_kick_primitives_and_edge_cases(torch_cuda, api, ctx):
    torch = torch_cuda
    rng = np.random.default_rng([13, 3])
    n = 1000
    xyzq = rng.normal(0, 1e-4, (n, 4)).astype(np.float32)
    xyzq[:, 3] = rng.choice([-QE, QE], n)
    vel = rng.normal(0, 1e5, (n, 4)).astype(np.float32)
    vel[:, 3] = ME
    vel[7, 3] = 0.0                                                     # immobile marker
    fld = rng.normal(0, 1e5, (n, 4)).astype(np.float32)
    d_x, d_v, d_f = dev(torch, xyzq), dev(torch, vel), dev(torch, fld)
    h = np.float32(2.5e-14)
    ctx.push_drift(d_x, d_v, float(h))
    exp_x = xyzq[:, :3].astype(np.float64) + float(h) * vel[:, :3].astype(np.float64)
    got = d_x.cpu().numpy()
    assert np.all(np.abs(got[:, :3] - exp_x) <= 0.5 * _ulp(exp_x) * 1.0001)
    ctx.push_kick(d_x, d_v, d_f, float(h))
    qm = np.where(vel[:, 3] != 0, xyzq[:, 3].astype(np.float64) / np.where(vel[:, 3] != 0, vel[:, 3], 1).astype(np.float64), 0.0)
    exp_v = vel[:, :3].astype(np.float64) + float(h) * qm[:, None] * fld[:, :3].astype(np.float64)
    gv = d_v.cpu().numpy()
    assert np.all(np.abs(gv[:, :3] - exp_v) <= 0.5 * _ulp(exp_v) + 3e-7 * np.abs(exp_v - vel[:, :3]))
    assert np.array_equal(gv[7, :3], vel[7, :3])
    # n = 0, bad flags, panels never set
    empty = torch.empty((0, 4), dtype=torch.float32, device="cuda")
    ctx.step_euler(empty, empty, 1e-15, flags=api.NBODY)
    ctx.step_pefrl(empty, empty, 1e-15, flags=api.NBODY)
    with pytest.raises(api.ObemError):
        ctx.step_euler(d_x, d_v, 1e-15, flags=8)
    with pytest.raises(api.ObemError):
        ctx.step_euler(d_x, d_v, 1e-15, flags=api.PANELS)
    with pytest.raises(api.ObemError):
        ctx.step_pefrl(d_x, d_v, float("nan"), flags=api.NBODY)


# --------------------------------------------------------------------------------------------------
# recombination by-product of the N-body pass (Eq 3.12)
# --------------------------------------------------------------------------------------------------
def _check_partners(xyzq, eps, pd, pj, od, oj, idx=None, what=""):
    """Distances must match the oracle up to the documented near-tie slack; the index must be the oracle's unless
    another opposite charge sits within that slack (then it must be a valid opposite charge at the reported
    distance)."""
    pd = pd.astype(np.float64)
    n = xyzq.shape[0]
    idx = np.arange(n) if idx is None else idx
    none = oj < 0
    assert np.array_equal(pj[none], oj[none]) and np.all(np.isinf(pd[none])), what
    has = ~none
    d2_true = od[has] ** 2
    slack = 4.0 * np.spacing((d2_true + eps * eps).astype(np.float32)).astype(np.float64)
    assert np.all(pd[has] ** 2 <= d2_true * (1 + 3e-7) + slack), what
    assert np.all(pd[has] >= od[has] * (1 - 1e-7)), what                   # never closer than the true nearest
    # the reported index is a real opposite charge at the reported distance
    tj = pj[has].astype(np.int64)
    ti = idx[has]
    assert np.all(tj >= 0) and np.all(tj < n) and np.all(tj != ti), what
    assert np.all(xyzq[tj, 3] * xyzq[ti, 3] < 0), what
    dd = np.linalg.norm(xyzq[tj, :3].astype(np.float64) - xyzq[ti, :3].astype(np.float64), axis=1)
    assert np.allclose(dd, pd[has], rtol=2e-7, atol=0), what
    same = tj == oj[has]
    if same.size == 0:
        return 1.0
    assert same.mean() > 0.999, "%s: only %.4f of the partners are the oracle's" % (what, same.mean())
    return float(same.mean())


def test_partners_config1_and_field_unchanged(torch_cuda, api, ctx, ref):
    from parity_metrics import assert_parity
    torch = torch_cuda
    wl = W.make_workload(1)
    ctx.set_softening(wl.eps_pp, wl.eps_panel)
    ctx.set_panels(dev(torch, wl.verts), dev(torch, wl.sigma))
    ctx.set_charges(dev(torch, wl.xyzq))
    out, pd, pj = ctx.eval_at_charges_partners(flags=api.NBODY | api.PANELS)
    plain = ctx.eval_at_charges(flags=api.NBODY | api.PANELS)
    torch.cuda.synchronize()
    on, op = ref.eval_field(xyzq=wl.xyzq, verts=wl.verts, sigma=wl.sigma, eps_pp=wl.eps_pp, eps_panel=wl.eps_panel)
    assert_parity(out.cpu().numpy(), on + op, "cfg1 field with partner tracking")
    assert torch.equal(out, plain)                                       # the by-product does not change the field
    od, oj = ref.nearest_opposite(wl.xyzq)
    _check_partners(wl.xyzq, wl.eps_pp, pd.cpu().numpy(), pj.cpu().numpy(), od, oj, what="cfg1")


@pytest.mark.parametrize("n,eps", [(3000, 0.1 * UM), (5000, 0.0), (1, 0.1 * UM), (300, 0.05 * UM)])
def test_partners_mixed_signs(torch_cuda, api, ctx, ref, n, eps):
    """Unsorted species, zero charges, doubly charged ions: every block is non-uniform (per-source sign test)."""
    torch = torch_cuda
    rng = np.random.default_rng([13, 7, n])
    xyzq = np.zeros((n, 4), dtype=np.float32)
    xyzq[:, :3] = rng.uniform(0, 50 * UM, (n, 3))
    xyzq[:, 3] = rng.choice([-QE, QE, 2 * QE, 0.0], n, p=[0.45, 0.35, 0.1, 0.1])
    ctx.set_softening(eps, 0.0)
    ctx.set_charges(dev(torch, xyzq))
    out, pd, pj = ctx.eval_at_charges_partners(flags=api.NBODY)
    od, oj = ref.nearest_opposite(xyzq)
    _check_partners(xyzq, eps, pd.cpu().numpy(), pj.cpu().numpy(), od, oj, what="mixed n=%d" % n)
    # one species only: nobody has a partner
    xyzq[:, 3] = -QE
    ctx.set_charges(dev(torch, xyzq))
    _, pd, pj = ctx.eval_at_charges_partners(flags=api.NBODY)
    assert torch.all(pj == -1) and torch.all(torch.isinf(pd))


def test_partners_config2_reduced_split_tiles_and_range(torch_cuda, api, ctx, ref):
    torch = torch_cuda
    wl = W.make_workload(2, charge_div=4, mesh_div=8)                    # 16384 charges: 8 tiles, split between CTAs
    ctx.set_softening(wl.eps_pp, 0.0)
    ctx.set_charges(dev(torch, wl.xyzq))
    _, pd, pj = ctx.eval_at_charges_partners(flags=api.NBODY)
    od, oj = ref.nearest_opposite(wl.xyzq)
    _check_partners(wl.xyzq, wl.eps_pp, pd.cpu().numpy(), pj.cpu().numpy(), od, oj, what="cfg2/4")
    first, count = 5000, 7001
    _, pd2, pj2 = ctx.eval_at_charges_partners(flags=api.NBODY, first=first, count=count)
    assert torch.equal(pj2, pj[first:first + count]) and torch.equal(pd2, pd[first:first + count])
    with pytest.raises(api.ObemError):
        ctx.eval_at_charges_partners(flags=api.PANELS)                   # the by-product needs the N-body pass


def test_partners_config3_full_size_sampled(torch_cuda, api, ctx, ref):
    torch = torch_cuda
    wl = W.make_workload(3)
    ctx.set_softening(wl.eps_pp, 0.0)
    ctx.set_charges(dev(torch, wl.xyzq))
    _, pd, pj = ctx.eval_at_charges_partners(flags=api.NBODY)
    torch.cuda.synchronize()
    pd, pj = pd.cpu().numpy(), pj.cpu().numpy()
    rng = np.random.default_rng([13, 9])
    idx = np.unique(np.concatenate([rng.choice(wl.n_charges, 2048, replace=False), np.argsort(pd)[:256],
                                    np.argsort(pd)[-64:], [0, wl.n_charges - 1]]))
    od, oj = ref.nearest_opposite(wl.xyzq, idx=idx)
    _check_partners(wl.xyzq, wl.eps_pp, pd[idx], pj[idx], od, oj, idx=idx, what="cfg3 sampled")
    # Eq (3.12): the mask a transport loop would apply
    r = api.recombination_radius(15.76)
    assert abs(r - ref.recombination_radius(15.76)) < 1e-24
    assert np.array_equal(pd[idx] <= r, od <= r)

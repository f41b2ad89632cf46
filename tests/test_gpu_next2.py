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

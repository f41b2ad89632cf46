"""GPU parity of obem_eval_panels_multi -- Eq (2.13)/(2.14) for several charge-density vectors on
one geometry in one pass (weighting fields of the read-out electrodes, Eq 3.13).  The oracle is K
calls of the plain fp64 panel sum, one per vector.  `pytest -m gpu`."""
import numpy as np
import pytest

from paper_2110_09214_b200 import workloads as W
from parity_metrics import assert_parity

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


def _sigmas(rng, k, npan):
    """k density vectors of different character: Gaussian, one-signed (an electrode at unit potential), sparse."""
    s = rng.normal(0.0, 1e-5, (k, npan)).astype(np.float32)
    if k > 1:
        s[1] = np.abs(s[1]) + np.float32(2e-6)
    if k > 2:
        s[2][rng.random(npan) < 0.7] = 0.0
    return s


@pytest.mark.parametrize("k", [1, 4, 6])
def test_multi_sigma_config2_reduced(torch_cuda, api, ctx, ref, k):
    """16384 targets (16 tiles of the multi launch), 4096 panels (121 blocks), 1 / 4 / 6 vectors (1 or 2 passes)."""
    torch = torch_cuda
    wl = W.make_workload(2, charge_div=4, mesh_div=2)
    rng = np.random.default_rng([29, k])
    sig = _sigmas(rng, k, wl.n_panels)
    ctx.set_softening(wl.eps_pp, 0.0)
    ctx.set_panels(dev(torch, wl.verts), dev(torch, wl.sigma))
    pts = dev(torch, wl.xyzq)
    out = ctx.eval_panels_multi(dev(torch, sig), pts).cpu().numpy()
    assert out.shape == (k, wl.n_charges, 4)
    for s in range(k):
        _, op = ref.eval_field(verts=wl.verts, sigma=sig[s], targets=wl.xyzq, flags=ref.PANELS)
        assert_parity(out[s], op, "multi-sigma k=%d vector %d" % (k, s))
    # the single-sigma path on the same vector: same sum, other arithmetic (sigma folded into the geometry)
    ctx.set_sigma(dev(torch, sig[0]))
    one = ctx.eval_at_points(pts, flags=api.PANELS).cpu().numpy()
    scale = np.abs(one).max(axis=0)
    assert np.all(np.abs(out[0] - one) <= 2e-5 * scale)


def test_multi_sigma_edges(torch_cuda, api, ctx, ref):
    """Ragged sizes, panel softening, a target exactly on a quadrature point (reading A4: that source contributes 0 --
    the value is compared with the oracle, not only checked for finiteness), empty inputs, state and argument errors."""
    torch = torch_cuda
    rng = np.random.default_rng([31, 1])
    npan, m, k = 75, 1500, 3
    verts = (rng.uniform(0, 60 * UM, (npan, 1, 3)) + rng.uniform(-2 * UM, 2 * UM, (npan, 3, 3))).astype(np.float32)
    sig = _sigmas(rng, k, npan)
    pts = np.zeros((m, 4), dtype=np.float32)
    pts[:, :3] = rng.uniform(-10 * UM, 70 * UM, (m, 3))
    with pytest.raises(api.ObemError) as e:
        ctx.eval_panels_multi(dev(torch, sig), dev(torch, pts))
    assert e.value.status == -2                                           # panels never set
    ctx.set_panels(dev(torch, verts), dev(torch, sig[0]))
    src = ctx.get_panel_sources().cpu().numpy()
    pts[7, :3] = src[7 * 5 + 0, :3]                                         # centroid point of panel 5: distance exactly 0
    pts[8, :3] = src[7 * 9 + 3, :3]                                         # an off-centre quadrature point of panel 9
    for eps in (0.0, 0.3 * UM):
        ctx.set_softening(0.0, eps)
        out = ctx.eval_panels_multi(dev(torch, sig), dev(torch, pts)).cpu().numpy()
        assert np.isfinite(out).all()
        for s in range(k):
            _, op = ref.eval_field(verts=verts, sigma=sig[s], targets=pts, eps_panel=eps, flags=ref.PANELS)
            # row 8: the quadrature point read back in fp32 is not bit-exactly the library's own -> a few nm apart
            keep = np.ones(m, dtype=bool)
            keep[8] = eps > 0
            assert_parity(out[s][keep], op[keep], "multi-sigma edges eps=%g vector %d" % (eps, s))
    ctx.set_softening(0.0, 0.0)
    assert tuple(ctx.eval_panels_multi(dev(torch, sig[:0]), dev(torch, pts)).shape) == (0, m, 4)
    assert tuple(ctx.eval_panels_multi(dev(torch, sig), dev(torch, pts[:0])).shape) == (k, 0, 4)
    with pytest.raises(ValueError):
        ctx.eval_panels_multi(dev(torch, sig[:, :-1]), dev(torch, pts))
    # the context's own sigma is neither used nor changed
    before = ctx.eval_at_points(dev(torch, pts), flags=api.PANELS).clone()
    ctx.eval_panels_multi(dev(torch, sig[1:]), dev(torch, pts))
    assert torch.equal(before, ctx.eval_at_points(dev(torch, pts), flags=api.PANELS))
    # a new geometry rebuilds the unit-density encoding
    verts2 = verts.copy()
    verts2[..., 0] += np.float32(5 * UM)
    ctx.set_panels(dev(torch, verts2), dev(torch, sig[0]))
    out = ctx.eval_panels_multi(dev(torch, sig[:1]), dev(torch, pts[100:])).cpu().numpy()
    _, op = ref.eval_field(verts=verts2, sigma=sig[0], targets=pts[100:], flags=ref.PANELS)
    assert_parity(out[0], op, "multi-sigma after a geometry change")


def test_multi_sigma_config3_full_size_sampled(torch_cuda, api, ctx, ref):
    """BASELINE.json configs[2]'s panels and charges (65,536 panels, 1,048,576 points), 4 vectors, in the launch
    configuration bench.py times (`next1.panels_multi_4`); sampled targets against the oracle."""
    torch = torch_cuda
    wl = W.make_workload(3)
    rng = np.random.default_rng([37, 3])
    sig = _sigmas(rng, 4, wl.n_panels)
    ctx.set_panels(dev(torch, wl.verts), dev(torch, wl.sigma))
    out = ctx.eval_panels_multi(dev(torch, sig), dev(torch, wl.xyzq))
    torch.cuda.synchronize()
    out = out.cpu().numpy()
    assert np.isfinite(out).all()
    idx = np.unique(np.concatenate([rng.choice(wl.n_charges, 512, replace=False),
                                    np.argsort(np.linalg.norm(out[0][:, :3], axis=1))[-32:], [0, wl.n_charges - 1]]))
    for s in range(4):
        _, op = ref.eval_field(verts=wl.verts, sigma=sig[s], targets=wl.xyzq[idx], flags=ref.PANELS)
        assert_parity(out[s][idx], op, "cfg3 multi-sigma vector %d" % s)


# --------------------------------------------------------------------------------------------------
# Shockley-Ramo signal sum, Eq (3.13)
# --------------------------------------------------------------------------------------------------
QE = 1.602176634e-19
EPS0 = 8.8541878128e-12


def test_ramo_current_matches_the_oracle(torch_cuda, api, ctx):
    from oracle import ramo
    torch = torch_cuda
    rng = np.random.default_rng([53, 1])
    # 400,003 particles: 391 block partials, more than the second launch has threads; the others: fewer
    for n, k in ((400003, 2), (50021, 3), (1, 1), (300, 5)):
        xyzq = np.zeros((n, 4), dtype=np.float32)
        xyzq[:, 3] = rng.choice([-QE, QE, 2 * QE, 0.0], n, p=[0.5, 0.3, 0.1, 0.1])
        vel = np.zeros((n, 4), dtype=np.float32)
        vel[:, :3] = rng.normal(0, 1e5, (n, 3))
        vel[:, 3] = 9.1e-31                                         # the mass lane is ignored
        ew = rng.normal(0, 1e3, (k, n, 4)).astype(np.float32)
        a = ctx.ramo_current(dev(torch, xyzq), dev(torch, vel), dev(torch, ew))
        b = ctx.ramo_current(dev(torch, xyzq), dev(torch, vel), dev(torch, ew))
        assert torch.equal(a, b)                                    # fixed summation order
        exp = ramo.ramo_current(xyzq[:, 3], vel[:, :3], ew[:, :, :3])
        scale = np.einsum("p,kp->k", np.abs(xyzq[:, 3].astype(np.float64)),
                          np.abs(vel[None, :, :3].astype(np.float64) * ew[:, :, :3].astype(np.float64)).sum(axis=2))
        assert np.all(np.abs(a.cpu().numpy() - exp) <= 1e-12 * scale[:, None] + 1e-300), (n, k)
    assert tuple(ctx.ramo_current(dev(torch, xyzq[:0]), dev(torch, vel[:0]), dev(torch, ew[:, :0])).shape) == (5, 2)
    assert torch.all(ctx.ramo_current(dev(torch, xyzq[:0]), dev(torch, vel[:0]), dev(torch, ew[:, :0])) == 0)


def test_weighting_field_to_signal_chain_on_parallel_plates(torch_cuda, api, ctx, ref):
    """The whole read-out chain on the geometry of the paper's Figure 9 (a parallel-plate counter): two plates, the
    read-out one at 1 V -- surface densities +-eps0/d away from the rims -- evaluated with obem_eval_panels_multi at
    the particles, then Eq (3.13).  Against the oracle chain (fp64 panel sums, then the Ramo oracle) at the path's
    tolerance, and against the closed form i = N e v_z |E_w| with the on-axis field of the finite plates."""
    from oracle import ramo
    torch = torch_cuda
    d, half = 5.0 * UM, 50.0 * UM
    bottom = W.plane_mesh(-half, half, -half, half, 0.0, 32, 32)
    top = W.plane_mesh(-half, half, -half, half, d, 32, 32)
    verts = np.concatenate([bottom, top]).astype(np.float32)
    npl = bottom.shape[0]
    sig_w = np.concatenate([np.full(npl, -EPS0 / d), np.full(npl, +EPS0 / d)]).astype(np.float32)   # read-out = top
    sig_other = (-sig_w).astype(np.float32)                                                            # read-out = bottom
    rng = np.random.default_rng([53, 2])
    n = 4000
    xyzq = np.zeros((n, 4), dtype=np.float32)
    xyzq[:, :2] = rng.uniform(-10 * UM, 10 * UM, (n, 2))                 # the central fifth of the plates
    xyzq[:, 2] = rng.uniform(1.0 * UM, 4.0 * UM, n)
    xyzq[:, 3] = -QE
    vel = np.zeros((n, 4), dtype=np.float32)
    vel[:, 2] = 1.0e5
    vel[:, :2] = rng.normal(0, 3e4, (n, 2))
    ctx.set_panels(dev(torch, verts), dev(torch, sig_w))
    sig = np.stack([sig_w, sig_other])
    ew = ctx.eval_panels_multi(dev(torch, sig), dev(torch, xyzq))
    i_gpu = ctx.ramo_current(dev(torch, xyzq), dev(torch, vel), ew).cpu().numpy()
    ew_ref = np.stack([ref.eval_field(verts=verts, sigma=s, targets=xyzq, flags=ref.PANELS)[1] for s in sig])
    i_ref = ramo.ramo_current(xyzq[:, 3], vel[:, :3], ew_ref[:, :, :3])
    assert np.allclose(i_gpu[:, 0], i_ref[:, 0], rtol=2e-5, atol=0)
    assert np.all(i_gpu[:, 1] == 0)                                       # no ions
    # closed form: electrons towards the 1 V plate induce + N e v_z |E_w|; between two SQUARE plates of half-width a the
    # field on the axis is (sigma/eps0) (1 - sqrt(2) d / (pi a)) to first order in d/a (the on-axis formula of a
    # uniformly charged rectangle, pin P7, for both plates): 0.955/d here, within +-0.5 % over the central fifth
    closed = n * QE * 1.0e5 / d * (1.0 - np.sqrt(2.0) * d / (np.pi * half))
    assert abs(i_gpu[0, 0] / closed - 1.0) < 0.01 and abs(i_gpu[1, 0] / closed + 1.0) < 0.01

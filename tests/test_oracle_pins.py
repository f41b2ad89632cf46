"""Pins for the fp64 oracle (oracle/obem_ref.c): closed forms, invariants, hand-computed tiny cases.

None of these re-types the oracle's loops or re-calls it as its own reference: every expected value is
a textbook closed form, a conservation law, or arithmetic done by hand on a 3-4-5 / 1-2-2 geometry.
SURVEY.md section 8(c) pins P1-P10.  CPU only (`-m "not gpu"`).
"""
import math

import numpy as np
import pytest

from paper_2110_09214_b200 import workloads as W

EPS0 = 8.8541878128e-12
KE = 1.0 / (4.0 * math.pi * EPS0)   # 8.9875517923e9
QE = 1.602176634e-19
UM = 1e-6


def test_ke_value():
    # reading A7: k_e = 8.9875517923e9 N m^2 C^-2
    assert abs(KE - 8.9875517923e9) / KE < 1e-10


# ---------------------------------------------------------------- P1: single point charge
@pytest.mark.parametrize("eps", [0.0, 0.1 * UM, 3.0 * UM])
def test_p1_point_charge_closed_form(ref, eps):
    q = np.float32(-3 * QE)
    src = np.array([[1e-5, -2e-5, 3e-5, q]], dtype=np.float32)
    tgt = np.array([[4e-5, 2e-5, 3e-5, 0.0], [1e-5, -2e-5, 9e-5, 0.0], [-7e-5, 1e-5, -2e-5, 0.0]], dtype=np.float32)
    out_n, out_p = ref.eval_field(xyzq=src, targets=tgt, eps_pp=eps, flags=ref.NBODY)
    assert np.all(out_p == 0.0)
    for t in range(3):
        d = tgt[t, :3].astype(np.float64) - src[0, :3].astype(np.float64)
        r2 = d @ d + eps * eps
        e_exp = KE * float(q) * d / r2 ** 1.5          # Plummer field, = Coulomb for eps = 0
        phi_exp = KE * float(q) / math.sqrt(r2)
        assert np.allclose(out_n[t, :3], e_exp, rtol=1e-13, atol=0)
        assert abs(out_n[t, 3] - phi_exp) <= 1e-13 * abs(phi_exp)
    # direction: E points AWAY from a positive charge, TOWARDS a negative one (sign of (r - r'))
    d0 = tgt[0, :3].astype(np.float64) - src[0, :3].astype(np.float64)
    assert np.dot(out_n[0, :3], d0) < 0.0  # q < 0


# ---------------------------------------------------------------- P2: hand arithmetic on tiny systems
def test_p2_two_body_345_triangle(ref):
    # charges at the origin and at (3,4,0) um: distance exactly 5 um
    q0, q1 = np.float32(2 * QE), np.float32(-QE)
    xyzq = np.array([[0, 0, 0, q0], [3e-6, 4e-6, 0, q1]], dtype=np.float32)
    out_n, _ = ref.eval_field(xyzq=xyzq, flags=ref.NBODY)  # at the charges, self excluded by index
    dx, dy = float(np.float32(3e-6)), float(np.float32(4e-6))
    r = math.hypot(dx, dy)
    # field at charge 0 due to charge 1: k q1 (r0 - r1)/r^3
    e0 = KE * float(q1) * np.array([-dx, -dy, 0.0]) / r ** 3
    e1 = KE * float(q0) * np.array([dx, dy, 0.0]) / r ** 3
    assert np.allclose(out_n[0, :3], e0, rtol=1e-13)
    assert np.allclose(out_n[1, :3], e1, rtol=1e-13)
    assert abs(out_n[0, 3] - KE * float(q1) / r) < 1e-13 * abs(out_n[0, 3])
    assert abs(out_n[1, 3] - KE * float(q0) / r) < 1e-13 * abs(out_n[1, 3])
    # magnitude sanity against the decimal value: k e / (5 um)^2 = 57.59986 V/m per unit charge
    assert abs(np.linalg.norm(out_n[1, :3]) / 2.0 - 57.59986) < 2e-3


def test_p2_three_body_with_coincident_pair_and_self_exclusion(ref):
    # 0 and 1 coincide at the origin; 2 sits at (1,2,2) um (distance exactly 3 um); softening 4 um
    # so that sqrt(r^2 + eps^2) = 5 um for the far pair and = 4 um for the coincident pair.
    eps = float(np.float32(4e-6))
    a = float(np.float32(1e-6))
    b = float(np.float32(2e-6))
    q = [np.float32(QE), np.float32(-2 * QE), np.float32(3 * QE)]
    xyzq = np.array([[0, 0, 0, q[0]], [0, 0, 0, q[1]], [a, b, b, q[2]]], dtype=np.float32)
    out_n, _ = ref.eval_field(xyzq=xyzq, eps_pp=eps, flags=ref.NBODY)
    r2_far = a * a + 2 * b * b + eps * eps
    s_far = math.sqrt(r2_far)
    # target 0: coincident partner gives E = 0 (d = 0) and phi = k q1/eps (reading A3); far partner:
    phi0 = KE * (float(q[1]) / eps + float(q[2]) / s_far)
    e0 = KE * float(q[2]) * np.array([-a, -b, -b]) / r2_far ** 1.5
    assert abs(out_n[0, 3] - phi0) < 1e-13 * abs(phi0)
    assert np.allclose(out_n[0, :3], e0, rtol=1e-13)
    # target 2 sees both origin charges at the same softened distance
    phi2 = KE * (float(q[0]) + float(q[1])) / s_far
    e2 = KE * (float(q[0]) + float(q[1])) * np.array([a, b, b]) / r2_far ** 1.5
    assert abs(out_n[2, 3] - phi2) < 1e-13 * abs(phi2)
    assert np.allclose(out_n[2, :3], e2, rtol=1e-13)
    # the self term k q_i/eps must NOT be in phi (exclusion by index): with a free point at the same
    # place (self_index = -1) it IS there.
    out_free, _ = ref.eval_field(xyzq=xyzq, targets=xyzq[:1], self_index=np.array([-1]), eps_pp=eps, flags=ref.NBODY)
    assert abs((out_free[0, 3] - out_n[0, 3]) - KE * float(q[0]) / eps) < 1e-12 * abs(out_free[0, 3])


def test_p2_zero_distance_unsoftened_contributes_zero(ref):
    # reading A4: coincident charges, eps = 0 -> that pair is skipped, no inf/nan
    xyzq = np.array([[1e-6, 1e-6, 1e-6, QE], [1e-6, 1e-6, 1e-6, -QE], [4e-6, 5e-6, 1e-6, QE]], dtype=np.float32)
    out_n, _ = ref.eval_field(xyzq=xyzq, eps_pp=0.0, flags=ref.NBODY)
    assert np.all(np.isfinite(out_n))
    r = math.hypot(float(np.float32(4e-6)) - float(np.float32(1e-6)), float(np.float32(5e-6)) - float(np.float32(1e-6)))
    assert abs(out_n[0, 3] - KE * float(np.float32(QE)) / r) < 1e-13 * abs(out_n[0, 3])


# ---------------------------------------------------------------- P3: Newton's third law
def test_p3_newton_third_law_total_force_vanishes(ref):
    w = W.make_workload(1)
    xyzq = w.xyzq[:1500]
    out_n, _ = ref.eval_field(xyzq=xyzq, eps_pp=w.eps_pp, flags=ref.NBODY)
    q = xyzq[:, 3].astype(np.float64)
    f = q[:, None] * out_n[:, :3]
    assert np.linalg.norm(f.sum(axis=0)) < 1e-11 * np.linalg.norm(f, axis=1).sum()
    # pairwise antisymmetry on a 2-subset: q_i E_{j->i} = -q_j E_{i->j}
    pair = xyzq[[3, 977]]
    o, _ = ref.eval_field(xyzq=pair, eps_pp=w.eps_pp, flags=ref.NBODY)
    assert np.allclose(float(pair[0, 3]) * o[0, :3], -float(pair[1, 3]) * o[1, :3], rtol=1e-14)


# ---------------------------------------------------------------- P4: Gauss's law
def _sphere_nodes(R, n_mu=64, n_phi=128, centre=(0.0, 0.0, 0.0)):
    mu, wmu = np.polynomial.legendre.leggauss(n_mu)
    phi = (np.arange(n_phi) + 0.5) * (2.0 * math.pi / n_phi)
    st = np.sqrt(1.0 - mu ** 2)
    nrm = np.stack([st[:, None] * np.cos(phi)[None, :], st[:, None] * np.sin(phi)[None, :],
                    np.broadcast_to(mu[:, None], (n_mu, n_phi))], axis=-1).reshape(-1, 3)
    wts = (wmu[:, None] * np.full(n_phi, 2.0 * math.pi / n_phi)[None, :]).reshape(-1) * R * R
    pts = np.asarray(centre)[None, :] + R * nrm
    return pts, nrm, wts


def test_p4_gauss_flux_charges(ref):
    rng = np.random.default_rng(7)
    n_in, n_out = 200, 50
    pin = rng.normal(size=(n_in, 3))
    pin = pin / np.linalg.norm(pin, axis=1, keepdims=True) * rng.uniform(0, 0.45, (n_in, 1)) * 100 * UM
    pout = rng.normal(size=(n_out, 3))
    pout = pout / np.linalg.norm(pout, axis=1, keepdims=True) * rng.uniform(2.0, 3.0, (n_out, 1)) * 100 * UM
    q = rng.integers(-3, 4, n_in + n_out).astype(np.float64) * QE
    xyzq = np.concatenate([np.concatenate([pin, pout]), q[:, None]], axis=1).astype(np.float32)
    R = 100 * UM
    pts, nrm, wts = _sphere_nodes(R)
    # fp32 rounding of the node positions perturbs the flux at the 1e-7 level; keep nodes exact in
    # fp32 by rounding them first and using the rounded positions' own radius/normal
    tg = np.zeros((pts.shape[0], 4), dtype=np.float32)
    tg[:, :3] = pts
    out_n, _ = ref.eval_field(xyzq=xyzq, targets=tg, eps_pp=0.0, flags=ref.NBODY)
    flux = np.sum(wts * np.einsum("ij,ij->i", out_n[:, :3], nrm))
    q_enc = xyzq[:n_in, 3].astype(np.float64).sum()
    scale = np.abs(xyzq[:n_in, 3].astype(np.float64)).sum() / EPS0
    assert abs(flux - q_enc / EPS0) < 2e-6 * scale      # limited by fp32 node positions
    # outside charges alone give zero flux
    out_o, _ = ref.eval_field(xyzq=xyzq[n_in:], targets=tg, eps_pp=0.0, flags=ref.NBODY)
    flux_o = np.sum(wts * np.einsum("ij,ij->i", out_o[:, :3], nrm))
    assert abs(flux_o) < 2e-6 * np.abs(xyzq[n_in:, 3].astype(np.float64)).sum() / EPS0


def test_p4_gauss_flux_panels(ref):
    # a uniformly charged 100x100 um plate (config-1 plane mesh), enclosed by a sphere of R = 200 um:
    # flux = sigma * L^2 / eps0 exactly (quadrature weights sum to 1; panel areas tile the square)
    L = 100 * UM
    verts = W.plane_mesh(-L / 2, L / 2, -L / 2, L / 2, 0.0, 16, 16).astype(np.float32)
    sig = np.full(verts.shape[0], 2.5e-6, dtype=np.float32)
    pts, nrm, wts = _sphere_nodes(200 * UM)
    tg = np.zeros((pts.shape[0], 4), dtype=np.float32)
    tg[:, :3] = pts
    _, out_p = ref.eval_field(verts=verts, sigma=sig, targets=tg, flags=ref.PANELS)
    flux = np.sum(wts * np.einsum("ij,ij->i", out_p[:, :3], nrm))
    Lf = float(np.float32(L / 2)) * 2
    expected = float(sig[0]) * Lf * Lf / EPS0
    assert abs(flux - expected) < 2e-6 * abs(expected)


# ---------------------------------------------------------------- P5: the 7-point rule
def test_p5_quadrature_monomials_degree5_exact_degree6_not(ref):
    # unit right triangle (0,0),(1,0),(0,1): Int x^a y^b = a! b! / (a+b+2)!
    verts = np.array([[[0, 0, 0], [1, 0, 0], [0, 1, 0]]], dtype=np.float32)
    src = ref.panel_sources(verts, np.array([1.0], dtype=np.float32))
    assert src.shape == (7, 4)
    x, y, wt = src[:, 0], src[:, 1], src[:, 3]
    assert abs(wt.sum() - 0.5) < 1e-15  # sigma * A * sum(w) = area
    for a in range(6):
        for b in range(6 - a):
            exact = math.factorial(a) * math.factorial(b) / math.factorial(a + b + 2)
            assert abs(np.sum(wt * x ** a * y ** b) - exact) < 2e-16 + 1e-14 * exact, (a, b)
    # degree 6 must NOT be exact (the rule is degree 5): relative error of a few percent on x^3 y^3
    errs = []
    for a, b in [(6, 0), (3, 3), (4, 2)]:
        exact = math.factorial(a) * math.factorial(b) / math.factorial(a + b + 2)
        errs.append(abs(np.sum(wt * x ** a * y ** b) - exact) / exact)
    assert max(errs) > 1e-2
    # the rule itself: 7 points, weights sum to 1, barycentric rows sum to 1, symmetric under permutation
    l, w = ref.quad_rule()
    assert abs(w.sum() - 1.0) < 1e-15 and np.allclose(l.sum(axis=1), 1.0, atol=1e-15)
    assert abs(w[0] - 0.225) < 1e-15
    assert np.allclose(sorted(l.sum(axis=0)), [7.0 / 3.0] * 3, atol=1e-14)  # symmetric orbits


def test_p5_area_scaling_and_degenerate_triangle(ref):
    v = np.array([[[0, 0, 0], [3e-6, 0, 0], [0, 4e-6, 0]],      # area 6e-12
                  [[0, 0, 0], [1e-6, 1e-6, 1e-6], [2e-6, 2e-6, 2e-6]]], dtype=np.float32)  # degenerate
    src = ref.panel_sources(v, np.array([2.0, 5.0], dtype=np.float32))
    a0 = 0.5 * float(np.float32(3e-6)) * float(np.float32(4e-6))
    assert abs(src[:7, 3].sum() - 2.0 * a0) < 1e-14 * a0
    assert np.all(np.abs(src[7:, 3]) < 1e-25)  # A = 0 -> contributes nothing (reading A8)


# ---------------------------------------------------------------- P6: far field of one triangle
def test_p6_triangle_far_field_converges_as_h_over_r_squared(ref):
    h = 10 * UM
    verts = np.array([[[0, 0, 0], [h, 0, 0], [0.3 * h, 0.9 * h, 0]]], dtype=np.float32)
    sig = np.array([1e-5], dtype=np.float32)
    v64 = verts[0].astype(np.float64)
    cen = v64.mean(axis=0)
    area = 0.5 * np.linalg.norm(np.cross(v64[1] - v64[0], v64[2] - v64[0]))
    Q = float(sig[0]) * area
    u = np.array([0.3, -0.5, 0.81])
    u /= np.linalg.norm(u)
    devs = []
    for k in range(6):
        r = h * 2 ** k
        tg = np.zeros((1, 4), dtype=np.float32)
        tg[0, :3] = cen + r * u
        rr = np.linalg.norm(tg[0, :3].astype(np.float64) - cen)
        _, out_p = ref.eval_field(verts=verts, sigma=sig, targets=tg, flags=ref.PANELS)
        devs.append(abs(np.linalg.norm(out_p[0, :3]) - KE * Q / rr ** 2) / (KE * Q / rr ** 2))
    devs = np.array(devs)
    assert devs[-1] < 1e-4 and devs[0] > 1e-3          # converges to k Q / r^2 ...
    slopes = np.log2(devs[:-1] / devs[1:])
    assert np.all(np.abs(slopes[1:] - 2.0) < 0.3), slopes  # ... as (h/r)^2 (quadrupole-order term)


# ---------------------------------------------------------------- P7: assembled mesh vs closed form
def _rect_axis_field(sigma, a, b, h):
    return sigma / (math.pi * EPS0) * math.atan(a * b / (h * math.sqrt(a * a + b * b + h * h)))


def test_p7_uniform_rectangle_on_axis(ref):
    L = 100 * UM
    verts = W.plane_mesh(0, L, 0, L, 0.0, 16, 16).astype(np.float32)
    sig = np.full(verts.shape[0], 1e-6, dtype=np.float32)
    a = float(np.float32(L)) / 2
    cell = L / 16
    for mult, tol in [(3, 2e-6), (5, 1e-7), (10, 1e-9), (40, 1e-9)]:
        hgt = mult * cell
        tg = np.array([[L / 2, L / 2, hgt, 0]], dtype=np.float32)
        _, out_p = ref.eval_field(verts=verts, sigma=sig, targets=tg, flags=ref.PANELS)
        hh = float(tg[0, 2])
        exp = _rect_axis_field(float(sig[0]), a, a, hh)
        assert abs(out_p[0, 2] - exp) < tol * exp + 1e-7 * exp, (mult, out_p[0, 2], exp)  # 1e-7: fp32 vertex rounding
        assert abs(out_p[0, 0]) < 1e-6 * exp and abs(out_p[0, 1]) < 1e-6 * exp        # symmetry
    # far limit k Q / h^2
    tg = np.array([[L / 2, L / 2, 0.05, 0]], dtype=np.float32)
    _, out_p = ref.eval_field(verts=verts, sigma=sig, targets=tg, flags=ref.PANELS)
    assert abs(out_p[0, 2] - KE * float(sig[0]) * (2 * a) ** 2 / float(tg[0, 2]) ** 2) < 1e-5 * out_p[0, 2]


def test_p7_parallel_plates_sigma_over_eps0(ref):
    # Table 1's geometry: two parallel plates, +sigma and -sigma, thin gap:
    # E_z in the middle = -(sigma/eps0) * (2/pi) atan(...) from the two closed forms superposed
    L, g = 400 * UM, 20 * UM
    top = W.plane_mesh(0, L, 0, L, g, 64, 64)
    bot = W.plane_mesh(0, L, 0, L, 0.0, 64, 64)
    verts = np.concatenate([bot, top]).astype(np.float32)
    s = 3e-6
    sig = np.concatenate([np.full(bot.shape[0], s), np.full(top.shape[0], -s)]).astype(np.float32)
    tg = np.array([[L / 2, L / 2, g / 2, 0]], dtype=np.float32)
    _, out_p = ref.eval_field(verts=verts, sigma=sig, targets=tg, flags=ref.PANELS)
    a = float(np.float32(L)) / 2
    hb = float(tg[0, 2])
    ht = float(np.float32(g)) - hb
    sf = float(sig[0])
    exp = _rect_axis_field(sf, a, a, hb) + _rect_axis_field(sf, a, a, ht)  # both push +z in the gap
    assert abs(out_p[0, 2] - exp) < 1e-4 * exp        # h = 1.6 cells: quadrature error ~(cell/h)^6
    assert abs(out_p[0, 2] - sf / EPS0) < 0.05 * sf / EPS0  # and ~ sigma/eps0 (finite-plate correction)


# ---------------------------------------------------------------- P9: invariances
def _small_system():
    w = W.make_workload(1)
    return w.xyzq[:300].copy(), w.verts[:200].copy(), w.sigma[:200].copy(), w.eps_pp


def test_p9_rotation_translation_scaling(ref):
    xyzq, verts, sig, eps = _small_system()
    tg = xyzq[:40].copy()
    tg[:, :3] += np.float32(1.7e-6)
    base_n, base_p = ref.eval_field(xyzq=xyzq, verts=verts, sigma=sig, targets=tg, eps_pp=eps)
    # scaling by an exact power of two keeps the fp32 inputs exact: r -> 2r, eps -> 2 eps
    s = 2.0
    xs, vs, ts = xyzq.copy(), verts * np.float32(s), tg.copy()
    xs[:, :3] *= np.float32(s)
    ts[:, :3] *= np.float32(s)
    sn, sp = ref.eval_field(xyzq=xs, verts=vs, sigma=sig, targets=ts, eps_pp=eps * s)
    assert np.allclose(sn[:, :3], base_n[:, :3] / s ** 2, rtol=1e-12) and np.allclose(sn[:, 3], base_n[:, 3] / s, rtol=1e-12)
    # panels: sigma fixed, area x4, distance x2 -> E unchanged, phi x2
    assert np.allclose(sp[:, :3], base_p[:, :3], rtol=1e-12) and np.allclose(sp[:, 3], base_p[:, 3] * s, rtol=1e-12)
    # rotation about z by 90 degrees and a sign flip are exact in fp32: (x,y,z) -> (-y,x,z)
    def rot(a):
        b = a.copy()
        b[..., 0], b[..., 1] = -a[..., 1], a[..., 0]
        return b
    rn, rp = ref.eval_field(xyzq=rot(xyzq), verts=rot(verts), sigma=sig, targets=rot(tg), eps_pp=eps)
    for base, r in ((base_n, rn), (base_p, rp)):
        sc = np.abs(base[:, :3]).max()
        assert np.allclose(r[:, 0], -base[:, 1], rtol=1e-10, atol=1e-12 * sc)
        assert np.allclose(r[:, 1], base[:, 0], rtol=1e-10, atol=1e-12 * sc)
        assert np.allclose(r[:, 2], base[:, 2], rtol=1e-10, atol=1e-12 * sc)
        assert np.allclose(r[:, 3], base[:, 3], rtol=1e-10, atol=1e-12 * np.abs(base[:, 3]).max())
    # translation by a fp32-exact offset on inputs that stay exactly representable: use integer grid
    g = (np.random.default_rng(3).integers(-2000, 2000, (60, 3)) * 2.0 ** -30).astype(np.float32)
    xq = np.concatenate([g, np.full((60, 1), QE)], axis=1).astype(np.float32)
    off = np.float32(4096 * 2.0 ** -30)
    xq2 = xq.copy()
    xq2[:, :3] += off
    a, _ = ref.eval_field(xyzq=xq, eps_pp=0.0, flags=ref.NBODY)
    b, _ = ref.eval_field(xyzq=xq2, eps_pp=0.0, flags=ref.NBODY)
    assert np.allclose(a, b, rtol=1e-13)


def test_p9_linearity_and_permutation(ref):
    xyzq, verts, sig, eps = _small_system()
    tg = xyzq[:25].copy()
    tg[:, 2] += np.float32(2e-6)
    n1, p1 = ref.eval_field(xyzq=xyzq, verts=verts, sigma=sig, targets=tg, eps_pp=eps)
    x2 = xyzq.copy()
    x2[:, 3] *= np.float32(4.0)     # exact in fp32
    n2, p2 = ref.eval_field(xyzq=x2, verts=verts, sigma=sig * np.float32(-2.0), targets=tg, eps_pp=eps)
    assert np.allclose(n2, 4.0 * n1, rtol=1e-13) and np.allclose(p2, -2.0 * p1, rtol=1e-13)
    perm = np.random.default_rng(5).permutation(xyzq.shape[0])
    pperm = np.random.default_rng(6).permutation(verts.shape[0])
    n3, p3 = ref.eval_field(xyzq=xyzq[perm], verts=verts[pperm], sigma=sig[pperm], targets=tg, eps_pp=eps)
    assert np.allclose(n3, n1, rtol=1e-9, atol=1e-12 * np.abs(n1).max())
    assert np.allclose(p3, p1, rtol=1e-9, atol=1e-12 * np.abs(p1).max())
    # splitting the sources in two halves and adding the results = the whole (superposition)
    na, _ = ref.eval_field(xyzq=xyzq[:150], targets=tg, eps_pp=eps, flags=ref.NBODY)
    nb, _ = ref.eval_field(xyzq=xyzq[150:], targets=tg, eps_pp=eps, flags=ref.NBODY)
    assert np.allclose(na + nb, n1, rtol=1e-9, atol=1e-12 * np.abs(n1).max())


# ---------------------------------------------------------------- P10: neutral pair, flags, eps -> 0
def test_p10_neutral_pair_net_force(ref):
    # reading A14: a tight +-q pair (separation d) at distance R on the axis of a point source:
    # |F+ + F-| / |F+| -> 2 d / R; the pair's mutual forces cancel exactly.
    d = 0.5 * UM
    src = [0.0, 0.0, 0.0, 5 * QE]
    for R in (50 * UM, 200 * UM, 800 * UM):
        xyzq = np.array([src, [R, 0, 0, QE], [R + d, 0, 0, -QE]], dtype=np.float32)
        out_n, _ = ref.eval_field(xyzq=xyzq, eps_pp=0.0, flags=ref.NBODY)
        q = xyzq[:, 3].astype(np.float64)
        f = q[:, None] * out_n[:, :3]
        # remove the mutual (internal) forces analytically: they are equal and opposite
        net_pair = f[1] + f[2]
        only_src, _ = ref.eval_field(xyzq=xyzq[:1], targets=xyzq[1:2], eps_pp=0.0, flags=ref.NBODY)
        f_plus = q[1] * only_src[0, :3]
        Rr = float(xyzq[1, 0])
        dd = float(xyzq[2, 0]) - Rr
        ratio = np.linalg.norm(net_pair) / np.linalg.norm(f_plus)
        exact = 1.0 - (Rr / (Rr + dd)) ** 2          # point source on axis
        # the two mutual forces are ~(R/d)^2/5 larger than the source's and cancel in fp64
        assert abs(ratio - exact) < 1e-15 * (Rr / dd) ** 2 + 1e-12
        assert abs(ratio - 2 * dd / Rr) < 3 * (dd / Rr) ** 2 + 1e-12
        # whole system: total force is zero (third law)
        assert np.linalg.norm(f.sum(axis=0)) < 1e-12 * np.linalg.norm(f, axis=1).sum()


def test_p10_flags_add_up_and_eps_limit(ref):
    xyzq, verts, sig, eps = _small_system()
    tg = xyzq[:30]
    n_only, p0 = ref.eval_field(xyzq=xyzq, verts=verts, sigma=sig, targets=tg, eps_pp=eps, flags=ref.NBODY)
    n0, p_only = ref.eval_field(xyzq=xyzq, verts=verts, sigma=sig, targets=tg, eps_pp=eps, flags=ref.PANELS)
    n_b, p_b = ref.eval_field(xyzq=xyzq, verts=verts, sigma=sig, targets=tg, eps_pp=eps, flags=ref.NBODY | ref.PANELS)
    assert np.all(p0 == 0) and np.all(n0 == 0)
    assert np.array_equal(n_b, n_only) and np.array_equal(p_b, p_only)
    # eps -> 0 is continuous: targets off the sources
    tg2 = tg.copy()
    tg2[:, 0] += np.float32(3e-6)
    a, _ = ref.eval_field(xyzq=xyzq, targets=tg2, eps_pp=0.0, flags=ref.NBODY)
    b, _ = ref.eval_field(xyzq=xyzq, targets=tg2, eps_pp=1e-12, flags=ref.NBODY)
    assert np.allclose(a, b, rtol=1e-6)
    # panel softening setter: eps_panel > 0 lowers |phi| of a same-sign sheet
    sg = np.abs(sig)
    _, c = ref.eval_field(verts=verts, sigma=sg, targets=tg2, eps_panel=0.0, flags=ref.PANELS)
    _, d = ref.eval_field(verts=verts, sigma=sg, targets=tg2, eps_panel=5e-6, flags=ref.PANELS)
    assert np.all(d[:, 3] < c[:, 3]) and np.all(d[:, 3] > 0)


def test_empty_inputs(ref):
    tg = np.array([[1e-6, 2e-6, 3e-6, 0]], dtype=np.float32)
    n, p = ref.eval_field(targets=tg)
    assert n.shape == (1, 4) and np.all(n == 0) and np.all(p == 0)
    n, p = ref.eval_field(xyzq=np.zeros((0, 4), np.float32))
    assert n.shape == (0, 4) and p.shape == (0, 4)
    one = np.array([[0, 0, 0, QE]], dtype=np.float32)
    n, _ = ref.eval_field(xyzq=one, flags=ref.NBODY)   # a lone charge feels nothing
    assert np.all(n == 0)

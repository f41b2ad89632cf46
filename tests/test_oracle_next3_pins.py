"""Pins of the exact-cell-integral oracle (oracle/obem_ref_analytic.c; PAPER.md:131-147,
Eq 2.13/2.14).  CPU only.  None of these re-types the oracle's edge-wise formulas: they are closed forms from
other routes (rectangle on axis, vertex potential, van Oosterom-Strackee solid angle), brute-force refinement through
the separately pinned 7-point oracle, and differential / integral identities.
"""
import numpy as np
import pytest

EPS0 = 8.8541878128e-12
KE = 1.0 / (4.0 * np.pi * EPS0)
UM = 1e-6


def _rect_mesh(a, b, nx, ny, z=0.0):
    """[-a, a] x [-b, b] at height z, nx x ny cells, two triangles per cell (same diagonal)."""
    xs = np.linspace(-a, a, nx + 1)
    ys = np.linspace(-b, b, ny + 1)
    tris = []
    for i in range(nx):
        for j in range(ny):
            p00, p10 = (xs[i], ys[j], z), (xs[i + 1], ys[j], z)
            p01, p11 = (xs[i], ys[j + 1], z), (xs[i + 1], ys[j + 1], z)
            tris.append([p00, p10, p11])
            tris.append([p00, p11, p01])
    return np.array(tris, dtype=np.float64)


def _pad4(p):
    p = np.atleast_2d(np.asarray(p, dtype=np.float64))
    return np.concatenate([p, np.zeros((p.shape[0], 1))], axis=1).astype(np.float32)


def _subdivide(tris, levels):
    for _ in range(levels):
        a, b, c = tris[:, 0], tris[:, 1], tris[:, 2]
        ab, bc, ca = 0.5 * (a + b), 0.5 * (b + c), 0.5 * (c + a)
        tris = np.concatenate([np.stack([a, ab, ca], 1), np.stack([ab, b, bc], 1), np.stack([ca, bc, c], 1),
                               np.stack([ab, bc, ca], 1)])
    return tris


def test_t1_rectangle_on_axis_closed_form_down_to_a_hundredth_of_a_cell(ref):
    """P7 at small h: E_z(h) = sigma/(pi eps0) atan(ab / (h sqrt(a^2 + b^2 + h^2))) above the centre of a uniformly
    charged 2a x 2b rectangle -- exact for the exact integrals at ANY h (the 7-point rule needs h >= 3 cells)."""
    a, b, sigma = 50 * UM, 40 * UM, 3e-6
    tris = _rect_mesh(a, b, 16, 16).astype(np.float32)
    cell = 2 * a / 16
    a32, b32 = float(-tris[..., 0].min()), float(-tris[..., 1].min())
    hs = cell * np.array([0.01, 0.03, 0.1, 0.3, 1.0, 3.0, 10.0, 100.0])
    pts = _pad4(np.stack([np.zeros_like(hs), np.zeros_like(hs), hs], 1))
    out = ref.eval_panels_analytic(tris, np.full(len(tris), sigma, np.float32), pts)
    h = pts[:, 2].astype(np.float64)
    s32 = float(np.float32(sigma))
    ez = s32 / (np.pi * EPS0) * np.arctan(a32 * b32 / (h * np.sqrt(a32 ** 2 + b32 ** 2 + h ** 2)))
    assert np.allclose(out[:, 2], ez, rtol=2e-12, atol=0)
    assert np.abs(out[:, :2]).max() <= 1e-9 * ez.min()                 # symmetry: no in-plane field on the axis
    # limits: sigma/2eps0 just above the sheet, k_e Q / h^2 far away
    assert abs(out[0, 2] / (s32 / (2 * EPS0)) - 1) < 2e-3
    assert abs(out[-1, 2] / (KE * s32 * 4 * a32 * b32 / h[-1] ** 2) - 1) < 1e-2   # (a/h)^2 = 0.6 % at h = 12.5 a
    # below the sheet the field flips
    below = ref.eval_panels_analytic(tris, np.full(len(tris), sigma, np.float32), pts * np.array([1, 1, -1, 1], np.float32))
    assert np.allclose(below[:, 2], -out[:, 2], rtol=1e-13) and np.allclose(below[:, 3], out[:, 3], rtol=1e-13)


def test_t2_vertex_potential_closed_form(ref):
    """P8: in the plane, at the triangle's own vertex P: Int dS/R = h (asinh(tan b1) + asinh(tan b2)), h = distance
    from P to the opposite side, b1, b2 = the angles at P from the foot of the perpendicular to the other vertices."""
    rng = np.random.default_rng([33, 2])
    for _ in range(20):
        h = rng.uniform(0.5, 3.0)
        x1, x2 = np.sort(rng.uniform(-4, 4, 2))
        v0, v1, v2 = np.array([0.0, 0.0, 0.0]), np.array([x1, h, 0.0]), np.array([x2, h, 0.0])
        exp = h * (np.arcsinh(x2 / h) - np.arcsinh(x1 / h))           # tan b = x / h, signed
        rot = np.linalg.qr(rng.normal(size=(3, 3)))[0]
        shift = rng.normal(size=3)
        w0, w1, w2 = (rot @ v + shift for v in (v0, v1, v2))
        got, _ = ref.tri_integrals(w0, w1, w2, w0)
        assert abs(got - exp) <= 1e-12 * exp
        got2, _ = ref.tri_integrals(w0, w2, w1, w0)                    # orientation does not matter for phi
        assert abs(got2 - exp) <= 1e-12 * exp


def _solid_angle_vos(v0, v1, v2, r):
    """van Oosterom & Strackee (1983): tan(Omega/2) = R1.(R2 x R3) / (R1R2R3 + (R1.R2)R3 + (R1.R3)R2 + (R2.R3)R1)."""
    a, b, c = v0 - r, v1 - r, v2 - r
    la, lb, lc = (np.linalg.norm(x) for x in (a, b, c))
    num = np.dot(a, np.cross(b, c))
    den = la * lb * lc + np.dot(a, b) * lc + np.dot(a, c) * lb + np.dot(b, c) * la
    return 2.0 * np.arctan2(num, den)


def test_t3_normal_component_is_the_solid_angle(ref):
    rng = np.random.default_rng([33, 3])
    for k in range(200):
        v = rng.normal(size=(3, 3))
        scale = 10.0 ** rng.uniform(-2, 1)
        r = v.mean(0) + scale * rng.normal(size=3)
        n = np.cross(v[1] - v[0], v[2] - v[0])
        n /= np.linalg.norm(n)
        _, ie = ref.tri_integrals(v[0], v[1], v[2], r)
        # Int d/R^3 dS = sgn(d) |Omega|; VOS gives the signed solid angle seen from r: negative when r is on the +n side
        omega = -_solid_angle_vos(v[0], v[1], v[2], r)
        assert abs(np.dot(ie, n) - omega) <= 1e-11 * max(1.0, abs(omega)), k


def test_t4_brute_force_refinement_through_the_7_point_oracle(ref):
    """4^6 = 4096 sub-triangles x 7 points each (the separately pinned quadrature oracle) converge to the closed form."""
    rng = np.random.default_rng([33, 4])
    tri = np.array([[[0.0, 0.0, 0.0], [4e-6, 0.5e-6, 0.2e-6], [1e-6, 3e-6, -0.3e-6]]])
    tri32 = tri.astype(np.float32)
    sub = _subdivide(tri32.astype(np.float64), 6)
    h = 4e-6
    pts = tri32[0].astype(np.float64).mean(0) + h * np.array([[0.3, 0.1, 0.5], [0.0, 0.0, 1.0], [2.0, -1.0, 0.2],
                                                             [-0.4, 0.9, -0.6], [0.1, 0.2, 0.25]])
    pts = _pad4(pts)
    sigma = np.float32(1e-5)
    exact = ref.eval_panels_analytic(tri32, np.array([sigma]), pts)
    # sub-triangle vertices are fp64 midpoints rounded to fp32: the surface moves by <= 1e-13 m, relative 1e-7
    _, brute = ref.eval_field(verts=sub.astype(np.float32), sigma=np.full(len(sub), sigma), targets=pts,
                              flags=ref.PANELS)
    err = np.abs(brute - exact).max(0) / np.abs(exact).max(0)
    assert err.max() < 2e-6, err


def test_t5_field_is_minus_the_gradient_of_the_potential(ref):
    rng = np.random.default_rng([33, 5])
    for k in range(60):
        v = rng.normal(size=(3, 3))
        n = np.cross(v[1] - v[0], v[2] - v[0])
        n /= np.linalg.norm(n)
        dist = 10.0 ** rng.uniform(-1.5, 0.7)
        r = v.mean(0) + dist * rng.normal(size=3)
        if abs(np.dot(r - v[0], n)) < 1e-3:
            continue
        _, ie = ref.tri_integrals(v[0], v[1], v[2], r)
        step = 1e-5 * min(1.0, abs(np.dot(r - v[0], n)))
        grad = np.zeros(3)
        for a in range(3):
            e = np.zeros(3)
            e[a] = step
            grad[a] = (ref.tri_integrals(v[0], v[1], v[2], r + e)[0] - ref.tri_integrals(v[0], v[1], v[2], r - e)[0]) / (2 * step)
        assert np.allclose(ie, -grad, rtol=0, atol=2e-6 * np.linalg.norm(ie) + 1e-9), (k, ie, grad)


def test_t6_far_field_agrees_with_the_7_point_rule_with_slope_six(ref):
    tri = np.array([[[0.0, 0.0, 0.0], [5e-6, 0.0, 0.0], [1e-6, 4e-6, 0.0]]], dtype=np.float32)
    h = 5e-6                                                           # longest edge
    c = tri[0].astype(np.float64).mean(0)
    direction = np.array([0.48, 0.6, 0.64])
    rs = h * np.array([1.0, 2.0, 4.0, 8.0])
    pts = _pad4(c + rs[:, None] * direction)
    sig = np.array([1e-5], dtype=np.float32)
    exact = ref.eval_panels_analytic(tri, sig, pts)
    _, quad = ref.eval_field(verts=tri, sigma=sig, targets=pts, flags=ref.PANELS)
    rel = np.linalg.norm(quad[:, :3] - exact[:, :3], axis=1) / np.linalg.norm(exact[:, :3], axis=1)
    slopes = np.log2(rel[:-1] / rel[1:])
    assert rel[0] < 3e-3 and rel[1] < 5e-5 and rel[2] < 1e-6            # measured over all directions: 2.7e-3, 2.5e-5, 3.8e-7
    assert np.all(np.abs(slopes - 6.0) < 0.8), (rel, slopes)
    relp = np.abs(quad[:, 3] - exact[:, 3]) / np.abs(exact[:, 3])
    assert relp[1] < 1e-5 and relp[2] < 2e-7


def test_t7_jump_across_the_sheet_is_sigma_over_eps0(ref):
    v = np.array([[0.0, 0.0, 0.0], [2.0, 0.0, 0.0], [0.0, 2.0, 0.0]])
    inside, outside = np.array([0.5, 0.6, 0.0]), np.array([1.8, 1.9, 0.0])
    dz = np.array([0.0, 0.0, 1e-9])
    up, dn = ref.tri_integrals(*v, inside + dz)[1], ref.tri_integrals(*v, inside - dz)[1]
    assert abs((up[2] - dn[2]) - 4 * np.pi) < 1e-7                     # k_e * 4 pi = 1/eps0
    assert np.allclose(up[:2], dn[:2], rtol=1e-12)
    on = ref.tri_integrals(*v, inside)[1]
    assert on[2] == 0.0 and np.allclose(on[:2], up[:2], rtol=1e-7)     # principal value on the panel (reading A8)
    up, dn = ref.tri_integrals(*v, outside + dz)[1], ref.tri_integrals(*v, outside - dz)[1]
    assert abs(up[2] - dn[2]) < 1e-7                                   # no jump outside the triangle


def test_t8_degenerate_and_singular_positions_stay_finite(ref):
    v = np.array([[0.0, 0.0, 0.0], [1.0, 0.0, 0.0], [0.0, 1.0, 0.0]])
    for r in (v[0], v[1], 0.5 * (v[0] + v[1]), 0.5 * (v[1] + v[2]), np.array([2.0, 0.0, 0.0]), np.array([-1.0, 0.0, 0.0])):
        iphi, ie = ref.tri_integrals(*v, r)
        assert np.isfinite(iphi) and np.isfinite(ie).all()
    # on the extension of an edge the integrals are regular: compare with a point a hair off the line
    a = ref.tri_integrals(*v, np.array([2.0, 0.0, 0.0]))
    b = ref.tri_integrals(*v, np.array([2.0, 1e-9, 1e-9]))
    assert abs(a[0] - b[0]) < 1e-8 and np.allclose(a[1], b[1], atol=1e-7)
    iphi, ie = ref.tri_integrals(v[0], v[1], 3 * v[1], np.array([0.3, 0.3, 0.3]))   # collinear vertices
    assert iphi == 0.0 and np.all(ie == 0.0)


def test_t9_sum_wrapper_and_gauss_flux(ref):
    """eval_panels_analytic = k_e sum_p sigma_p I_p (checked against a python sum), and its flux through a sphere
    around a closed charged tetrahedron is Q/eps0."""
    rng = np.random.default_rng([33, 9])
    p = rng.normal(size=(4, 3)) * 1e-5
    faces = np.array([[p[0], p[1], p[2]], [p[0], p[3], p[1]], [p[1], p[3], p[2]], [p[2], p[3], p[0]]], dtype=np.float32)
    sigma = rng.normal(0, 1e-5, 4).astype(np.float32)
    t = _pad4(rng.normal(size=(5, 3)) * 3e-5)
    out = ref.eval_panels_analytic(faces, sigma, t)
    for k in range(5):
        acc = np.zeros(4)
        for f, s in zip(faces.astype(np.float64), sigma.astype(np.float64)):
            iphi, ie = ref.tri_integrals(f[0], f[1], f[2], t[k, :3].astype(np.float64))
            acc += KE * s * np.array([ie[0], ie[1], ie[2], iphi])
        assert np.allclose(out[k], acc, rtol=1e-13, atol=0)
    # Gauss: Gauss-Legendre in cos(theta) x trapezoid in phi
    nth, nph, R = 48, 96, 6e-5
    x, w = np.polynomial.legendre.leggauss(nth)
    ph = 2 * np.pi * np.arange(nph) / nph
    st = np.sqrt(1 - x ** 2)
    nrm = np.stack([np.outer(st, np.cos(ph)), np.outer(st, np.sin(ph)), np.outer(x, np.ones(nph))], -1).reshape(-1, 3)
    wts = np.outer(w, np.full(nph, 2 * np.pi / nph)).reshape(-1)
    pts32 = _pad4(R * nrm)
    out = ref.eval_panels_analytic(faces, sigma, pts32)
    nrm32 = pts32[:, :3].astype(np.float64)
    nrm32 /= np.linalg.norm(nrm32, axis=1, keepdims=True)
    flux = R ** 2 * np.sum(wts * np.einsum("ij,ij->i", out[:, :3], nrm32))
    f64 = faces.astype(np.float64)
    area = 0.5 * np.linalg.norm(np.cross(f64[:, 1] - f64[:, 0], f64[:, 2] - f64[:, 0]), axis=1)
    q = float(np.sum(sigma.astype(np.float64) * area))
    assert abs(flux - q / EPS0) <= 1e-6 * np.sum(np.abs(sigma) * area) / EPS0


def test_t10_rectangle_on_axis_potential_closed_form(ref):
    """phi(h) above the centre of a uniformly charged 2a x 2b rectangle, by direct integration over one quadrant:
    phi = sigma/(4 pi eps0) * 4 [ a asinh(b / sqrt(a^2 + h^2)) + b asinh(a / sqrt(b^2 + h^2)) - h atan(ab / (h R)) ],
    R = sqrt(a^2 + b^2 + h^2).  Exact for the exact integrals at any h; the 7-point sum reaches it to 1e-6 from 3 cells up."""
    a, b, sigma = 50 * UM, 40 * UM, 3e-6
    tris = _rect_mesh(a, b, 16, 16).astype(np.float32)
    cell = 2 * a / 16
    a32, b32 = float(-tris[..., 0].min()), float(-tris[..., 1].min())
    hs = cell * np.array([0.01, 0.1, 1.0, 3.0, 10.0, 100.0])
    pts = _pad4(np.stack([np.zeros_like(hs), np.zeros_like(hs), hs], 1))
    sig = np.full(len(tris), sigma, np.float32)
    h = pts[:, 2].astype(np.float64)
    s32 = float(np.float32(sigma))
    big_r = np.sqrt(a32 ** 2 + b32 ** 2 + h ** 2)
    quadrant = (a32 * np.arcsinh(b32 / np.sqrt(a32 ** 2 + h ** 2)) + b32 * np.arcsinh(a32 / np.sqrt(b32 ** 2 + h ** 2))
                - h * np.arctan(a32 * b32 / (h * big_r)))
    phi = s32 / (4 * np.pi * EPS0) * 4 * quadrant
    exact = ref.eval_panels_analytic(tris, sig, pts)
    assert np.allclose(exact[:, 3], phi, rtol=2e-13, atol=0)
    _, quad = ref.eval_field(verts=tris, sigma=sig, targets=pts, flags=ref.PANELS)
    assert np.allclose(quad[3:, 3], phi[3:], rtol=1e-6, atol=0)          # h >= 3 cells
    assert abs(quad[0, 3] / phi[0] - 1) > 1e-4                            # and not at a hundredth of a cell

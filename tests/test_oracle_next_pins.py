"""Pins of the oracle functions for the steps adjacent to the hot path (oracle/obem_ref_next.c).
CPU only.  None of these re-types the oracle's loops: each checks a closed form, an identity that ties the
function to a separately pinned one, a hand value, or an independent library routine.

NEXT-1: Eq (3.3)-(3.6); sigma = M^-1 b.
"""
import math

import numpy as np
import pytest

from paper_2110_09214_b200 import workloads as W

UM = 1e-6
QE = 1.602176634e-19
EPS0 = 8.8541878128e-12
KE = 1.0 / (4.0 * math.pi * EPS0)


def _cloud_and_mesh(seed=0, n=400, z_lo=20 * UM, z_hi=80 * UM):
    rng = np.random.default_rng([21, seed])
    L = 100 * UM
    verts = W.plane_mesh(0, L, 0, L, 0.0, 6, 5).astype(np.float32)
    # tilt / distort the mesh a little so that normals are not all +z and areas differ
    verts = verts + rng.uniform(-2 * UM, 2 * UM, verts.shape).astype(np.float32) * np.array([1, 1, 0.5], np.float32)
    xyzq = np.zeros((n, 4), dtype=np.float32)
    xyzq[:, 0:2] = rng.uniform(0, L, (n, 2))
    xyzq[:, 2] = rng.uniform(z_lo, z_hi, n)
    xyzq[:, 3] = rng.choice([-QE, QE, 2 * QE], n)
    sigma = rng.normal(0, 1e-5, verts.shape[0]).astype(np.float32)
    return xyzq, verts, sigma


# ---------------------------------------------------------------- N1: Green reciprocity with the panel oracle
@pytest.mark.parametrize("eps", [0.0, 0.3 * UM])
def test_n1_reciprocity_with_panel_sums(ref, eps):
    """sum_i sigma_i A_i Vbar_i(particles -> C_i) = sum_p q_p phi_panels(r_p)   (mutual energy, both orders), and
    sum_i sigma_i A_i Ebar_i = - sum_p q_p E_panels(r_p)   (Newton's third law between particles and panels).
    The right-hand sides come from obem_ref_eval's panel part (pinned by P4-P7); Eq (3.3)/(3.4) vs (2.13)/(2.14)."""
    xyzq, verts, sigma = _cloud_and_mesh()
    infl, en, na = ref.influence(xyzq, verts, eps=eps)
    _, out_p = ref.eval_field(xyzq=xyzq, verts=verts, sigma=sigma, eps_panel=eps, flags=ref.PANELS)
    q = xyzq[:, 3].astype(np.float64)
    sA = sigma.astype(np.float64) * na[:, 3]
    lhs_v = float((sA * infl[:, 3]).sum())
    rhs_v = float((q * out_p[:, 3]).sum())
    scale_v = float(np.abs(q * out_p[:, 3]).sum())
    assert abs(lhs_v - rhs_v) < 1e-12 * scale_v
    lhs_e = (sA[:, None] * infl[:, :3]).sum(axis=0)
    rhs_e = -(q[:, None] * out_p[:, :3]).sum(axis=0)
    scale_e = float(np.linalg.norm(q[:, None] * out_p[:, :3], axis=1).sum())
    assert np.linalg.norm(lhs_e - rhs_e) < 1e-12 * scale_e
    # a one-hot sigma isolates a single cell: Vbar_i itself, not just the weighted total
    for i in (0, 17, verts.shape[0] - 1):
        one = np.zeros_like(sigma)
        one[i] = 1.0
        _, o = ref.eval_field(xyzq=xyzq, verts=verts, sigma=one, eps_panel=eps, flags=ref.PANELS)
        assert abs(na[i, 3] * infl[i, 3] - float((q * o[:, 3]).sum())) < 1e-12 * float(np.abs(q * o[:, 3]).sum())
        assert np.linalg.norm(na[i, 3] * infl[i, :3] + (q[:, None] * o[:, :3]).sum(axis=0)) < 1e-12 * float(
            np.linalg.norm(q[:, None] * o[:, :3], axis=1).sum())


# ---------------------------------------------------------------- N2: flux of a point charge through a rectangle
def test_n2_flux_through_meshed_rectangle_is_solid_angle(ref):
    """sum_i A_i Ebar_i . n_i = q/(4 pi eps0) * Omega, Omega = 4 atan(ab / (h sqrt(a^2+b^2+h^2))) for a charge at
    height h over the centre of a 2a x 2b rectangle.  Pins the normal, its orientation (vertex order of
    plane_mesh is counter-clockwise seen from +z: n = +z, a charge above sends flux AGAINST n), the area weighting
    and the sign convention r - r_p of Eq (3.4)."""
    L = 100 * UM
    verts = W.plane_mesh(0, L, 0, L, 0.0, 16, 16).astype(np.float32)
    a = float(np.float32(L)) / 2
    q = 3 * QE
    for mult, tol in [(3, 2e-6), (6, 1e-7), (20, 1e-9)]:
        h = mult * L / 16
        xyzq = np.array([[L / 2, L / 2, h, q]], dtype=np.float32)
        hh = float(xyzq[0, 2])
        infl, en, na = ref.influence(xyzq, verts)
        assert np.allclose(na[:, :3], [0, 0, 1], atol=1e-12)
        assert abs(na[:, 3].sum() - (2 * a) ** 2) < 1e-6 * (2 * a) ** 2       # fp32 vertices
        flux = float((na[:, 3] * en).sum())
        omega = 4.0 * math.atan(a * a / (hh * math.sqrt(2 * a * a + hh * hh)))
        exp = -KE * float(xyzq[0, 3]) * omega                                  # field points down (-z) below a + charge
        assert abs(flux - exp) < (tol + 2e-7) * abs(exp), (mult, flux, exp)
        # Ebar is the field of Eq (3.4) itself: in-plane components cancel by symmetry over the whole plate
        tot = (na[:, 3, None] * infl[:, :3]).sum(axis=0)
        assert abs(tot[0]) < 1e-6 * abs(tot[2]) and abs(tot[1]) < 1e-6 * abs(tot[2])


# ---------------------------------------------------------------- N3: far charge, linearity, softening
def test_n3_far_charge_and_linearity(ref):
    v = np.array([[[0, 0, 0], [4 * UM, 0, 0], [0, 3 * UM, 0]]], dtype=np.float32)
    c = v[0].astype(np.float64).mean(axis=0)
    q = -QE
    prev = None
    for mult in (8, 16, 32):
        R = mult * 5 * UM
        pos = c + R * np.array([0.6, 0.0, 0.8])
        xyzq = np.array([[pos[0], pos[1], pos[2], q]], dtype=np.float32)
        d = c - xyzq[0, :3].astype(np.float64)
        r = np.linalg.norm(d)
        infl, en, na = ref.influence(xyzq, v)
        dev_v = abs(infl[0, 3] - KE * q / r) / abs(KE * q / r)
        dev_e = np.linalg.norm(infl[0, :3] - KE * q * d / r ** 3) / (KE * abs(q) / r ** 2)
        assert dev_v < 0.5 / mult ** 2 and dev_e < 1.5 / mult ** 2
        if prev is not None:                                                   # second-moment correction: (h/R)^2
            assert 3.0 < prev[0] / dev_v < 5.0 and 3.0 < prev[1] / dev_e < 5.0
        prev = (dev_v, dev_e)
        assert abs(en[0] - infl[0, 2]) < 1e-15 * abs(infl[0, 2]) + 1e-30      # n = +z for this vertex order
    # linearity in q and superposition over particles
    xyzq, verts, _ = _cloud_and_mesh(seed=1, n=60)
    full, en_full, _ = ref.influence(xyzq, verts)
    a, en_a, _ = ref.influence(xyzq[:25], verts)
    b, en_b, _ = ref.influence(xyzq[25:], verts)
    assert np.allclose(full, a + b, rtol=1e-12, atol=1e-12 * np.abs(full).max())
    assert np.allclose(en_full, en_a + en_b, rtol=1e-12, atol=1e-12 * np.abs(en_full).max())
    x3 = xyzq.copy()
    x3[:, 3] *= 4.0                                                            # exact in fp32
    assert np.allclose(ref.influence(x3, verts)[0], 4.0 * full, rtol=1e-13)
    # a charge exactly on a quadrature point: that term is dropped when eps = 0 (A4), kept finite otherwise
    l, w = ref.quad_rule()
    h = 2.0 ** -20                                                            # ~0.95 um, exact in fp32
    v2 = np.array([[[0, 0, 0], [3 * h, 0, 0], [0, 3 * h, 0]]], dtype=np.float32)   # centroid (h, h, 0): (1/3)*3h == h in fp64
    on = np.array([[h, h, 0.0, QE]], dtype=np.float32)
    assert np.all((l[0] @ v2[0].astype(np.float64)) == on[0, :3].astype(np.float64))
    i0, _, _ = ref.influence(on, v2)
    assert np.isfinite(i0).all()
    eps = 0.1 * UM
    i1, _, _ = ref.influence(on, v2, eps=eps)
    # the dropped centroid term reappears as w_0 k_e q / eps (w_0 = 9/40); the six others barely move (eps << h)
    assert abs((i1[0, 3] - i0[0, 3]) - 0.225 * KE * QE / eps) < 0.02 * 0.225 * KE * QE / eps


# ---------------------------------------------------------------- N4: right-hand side, hand values
def test_n4_rhs_hand_values(ref):
    kind = np.array([0, 1, 0, 1], dtype=np.int32)
    bc = np.array([100.0, 2e-6, -50.0, 0.0], dtype=np.float32)
    deps = np.array([0.0, 2.5 * EPS0, 123.0, 3.0 * EPS0], dtype=np.float32)   # unused on ed cells
    infl = np.array([[1, 2, 3, 7.0], [4, 5, 6, -8.0], [0, 0, 0, 0.25], [9, 9, 9, 9.0]], dtype=np.float64)
    en = np.array([11.0, -2.0e5, 13.0, 4.0e4], dtype=np.float64)
    b = ref.rhs(kind, bc, deps, infl, en)
    assert b[0] == 100.0 - 7.0                                               # Eq (3.5)
    assert b[2] == -50.0 - 0.25
    assert abs(b[1] - (float(bc[1]) + float(deps[1]) * 2.0e5)) < 1e-18       # Eq (3.6): sigma_F - (eps2-eps1) E.n
    assert abs(b[3] - (0.0 - float(deps[3]) * 4.0e4)) < 1e-18
    with pytest.raises(ValueError):
        ref.rhs(np.array([2], dtype=np.int32), bc[:1], deps[:1], infl[:1], en[:1])


# ---------------------------------------------------------------- N5: sigma = M^-1 b
def test_n5_matvec_against_numpy_and_special_cases(ref):
    rng = np.random.default_rng([21, 5])
    n = 257
    m = rng.normal(0, 1, (n, n)).astype(np.float32)
    b = rng.normal(0, 1, n).astype(np.float32)
    got = ref.matvec(m, b)
    exp = m.astype(np.float64) @ b.astype(np.float64)                       # independent library routine
    assert np.allclose(got, exp, rtol=0, atol=1e-12 * np.abs(m.astype(np.float64)).dot(np.abs(b.astype(np.float64))).max())
    assert np.array_equal(ref.matvec(np.eye(n, dtype=np.float32), b), b.astype(np.float64))
    perm = rng.permutation(n)
    p = np.zeros((n, n), dtype=np.float32)
    p[np.arange(n), perm] = 1.0
    assert np.array_equal(ref.matvec(p, b), b.astype(np.float64)[perm])      # row i picks b[perm[i]]: not transposed
    # an actual inverse: M (M^-1 b) = b
    a = (np.eye(n) * 4 + rng.normal(0, 0.05, (n, n)))
    ainv = np.linalg.inv(a).astype(np.float32)
    x = ref.matvec(ainv, b)
    assert np.allclose(a @ x, b.astype(np.float64), atol=1e-5)
    assert ref.matvec(np.zeros((0, 0), np.float32), np.zeros(0, np.float32)).shape == (0,)

"""Pins of the Shockley-Ramo signal oracle (oracle/ramo.py; Eq 3.13) against what the theorem and
the mathematics fix -- CPU only.

R1  parallel plates, gap d, read-out plate (at z = d) at 1 V: E_w = -(1/d) z^ everywhere, so one charge q moving with v
    gives i = q v . E_w = -q v_z / d in the paper's sign convention (Eq 3.13 as printed has no minus sign): an electron
    drifting towards the read-out plate gives +e v_z / d.
R2  induced CHARGE: a charge that crosses the whole gap at constant velocity induces, integrated over the crossing,
    exactly -q (times the weighting potential difference 1 V) whatever its speed: sum_t i(t) dt = -q.
R3  the split by species adds up to the plain definition written as one vectorised dot product; zero charges count
    nowhere; the result is linear in q, in v and in E_w and does not depend on the particle order.
R4  a velocity perpendicular to E_w induces nothing; a point charge's radial weighting field with a tangential
    (circular-orbit) velocity induces nothing either.
"""
import numpy as np

from oracle import ramo

QE = 1.602176634e-19


def test_R1_parallel_plate_textbook_current():
    d = 1.6e-3                                                   # the PPAC gap of the paper's Figure 9
    ew = np.zeros((1, 1, 3))
    ew[0, 0, 2] = -1.0 / d                                       # V_w = z/d: 1 V on the plate at z = d, E_w = -grad V_w
    v = np.array([[3.0e3, -2.0e3, 1.2e5]])
    i = ramo.ramo_current([-QE], v, ew)
    assert np.isclose(i[0, 0], -(-QE) * 1.2e5 / d, rtol=1e-15) and i[0, 1] == 0.0
    assert i[0, 0] > 0                       # an electron moving towards the 1 V plate: + e v_z / d
    i2 = ramo.ramo_current([+QE], v, ew)
    assert np.isclose(i2[0, 1], -QE * 1.2e5 / d, rtol=1e-15) and i2[0, 0] == 0.0


def test_R2_induced_charge_of_a_full_crossing_is_the_charge():
    d = 1.6e-3
    for speed, steps in ((1.0e5, 1000), (3.7e4, 333)):
        dt = d / speed / steps
        ew = np.zeros((1, 1, 3))
        ew[0, 0, 2] = -1.0 / d
        total = 0.0
        for _ in range(steps):
            total += ramo.ramo_current([-QE], np.array([[0.0, 0.0, speed]]), ew)[0, 0] * dt
        assert np.isclose(total, QE, rtol=1e-12)                 # -q with q = -e


def test_R3_split_linearity_order():
    rng = np.random.default_rng(3)
    n, k = 500, 3
    q = rng.choice([-QE, QE, 2 * QE, 0.0], n)
    v = rng.normal(0, 1e5, (n, 3))
    ew = rng.normal(0, 1e3, (k, n, 3))
    i = ramo.ramo_current(q, v, ew)
    plain = np.einsum("p,pd,kpd->k", q, v, ew)
    assert np.allclose(i.sum(axis=1), plain, rtol=1e-12, atol=1e-30)
    neg = np.einsum("p,pd,kpd->k", np.where(q < 0, q, 0.0), v, ew)
    assert np.allclose(i[:, 0], neg, rtol=1e-12, atol=1e-30)
    assert np.allclose(ramo.ramo_current(2 * q, v, ew), 2 * i, rtol=1e-14)
    assert np.allclose(ramo.ramo_current(q, -3 * v, ew), -3 * i, rtol=1e-14)
    assert np.allclose(ramo.ramo_current(q, v, ew[::-1])[::-1], i, rtol=0, atol=0)
    perm = rng.permutation(n)
    assert np.allclose(ramo.ramo_current(q[perm], v[perm], ew[:, perm]), i, rtol=1e-11, atol=1e-30)
    only_zero = ramo.ramo_current(np.zeros(n), v, ew)
    assert np.all(only_zero == 0)


def test_R4_no_current_without_motion_along_the_weighting_field():
    ew = np.zeros((1, 2, 3))
    ew[0, :, 2] = 5.0e2
    v = np.array([[1e5, -2e5, 0.0], [0.0, 3e4, 0.0]])
    assert np.all(ramo.ramo_current([-QE, QE], v, ew) == 0)
    # radial weighting field, circular orbit
    r = np.array([[3e-4, 4e-4, 0.0]])
    ewr = (r / np.linalg.norm(r) ** 3)[None]
    vt = np.array([[-4e-4, 3e-4, 0.0]]) * 1e8
    assert abs(ramo.ramo_current([QE], vt, ewr)[0, 1]) < 1e-30

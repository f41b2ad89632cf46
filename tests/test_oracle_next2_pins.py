"""Pins of the NEXT-2 oracle functions: the integrators of PAPER.md:300-306 (oracle/stepper.py)
and the recombination by-product of the N-body pass, Eq (3.12) (oracle/obem_ref_next.c).
CPU only.  Closed forms, convergence orders, reversibility, an independent library routine (scipy cKDTree).
"""
import math

import numpy as np
import pytest

UM = 1e-6
QE = 1.602176634e-19
ME = 9.1093837015e-31
EPS0 = 8.8541878128e-12
KE = 1.0 / (4.0 * math.pi * EPS0)


@pytest.fixture(scope="module")
def stepper():
    from oracle import stepper as s
    return s


# ---------------------------------------------------------------- S1: uniform field, closed forms
def test_s1_uniform_field_closed_forms(stepper):
    e0 = np.array([[3.0e5, -1.0e5, 2.0e5]])
    field = lambda x: np.repeat(e0, x.shape[0], axis=0)   # noqa: E731
    qm = np.array([-QE / ME, QE / (40 * 1836 * ME)])
    x0 = np.array([[1e-5, 2e-5, 3e-5], [0.0, 0.0, 0.0]])
    v0 = np.array([[1e5, 0.0, -2e5], [10.0, 20.0, 30.0]])
    h, n = 25e-15, 40
    a = qm[:, None] * e0
    # Euler: v_n = v0 + n h a (exact); x_n = x0 + n h v0 + a h^2 n (n - 1) / 2 (x uses the OLD velocity)
    x, v = x0.copy(), v0.copy()
    for _ in range(n):
        x, v, e = stepper.euler_step(x, v, qm, h, field)
    assert np.allclose(v, v0 + n * h * a, rtol=1e-13)
    assert np.allclose(x, x0 + n * h * v0 + a * h * h * n * (n - 1) / 2, rtol=1e-13, atol=1e-25)
    assert np.array_equal(e, np.repeat(e0, 2, axis=0))
    # PEFRL: exact for a constant force (drift weights sum to 1, kick weights to 1, second-order condition holds)
    x, v = x0.copy(), v0.copy()
    for _ in range(n):
        x, v = stepper.pefrl_step(x, v, qm, h, field)
    t = n * h
    assert np.allclose(v, v0 + t * a, rtol=1e-12)
    assert np.allclose(x, x0 + t * v0 + 0.5 * a * t * t, rtol=1e-12, atol=1e-25)


# ---------------------------------------------------------------- S2: harmonic field, orders 1 and 4
def _oscillator_error(step, h, periods=1.0):
    w = 2.0e12                                            # rad/s
    qm = np.array([-QE / ME])
    field = lambda x: (-(w * w) / qm[0]) * x             # noqa: E731  a = (q/m) E = -w^2 x
    x = np.array([[1e-6, 0.0, 0.0]])
    v = np.array([[0.0, 2.0e6, 0.0]])
    t_end = periods * 2 * math.pi / w
    n = int(round(t_end / h))
    h = t_end / n
    x0, v0 = x.copy(), v.copy()
    for _ in range(n):
        out = step(x, v, qm, h, field)
        x, v = out[0], out[1]
    xe = x0 * math.cos(w * t_end) + v0 / w * math.sin(w * t_end)
    return float(np.linalg.norm(x - xe)), h


def test_s2_convergence_orders(stepper):
    T = 2 * math.pi / 2.0e12
    e1, _ = _oscillator_error(stepper.euler_step, T / 2000)
    e2, _ = _oscillator_error(stepper.euler_step, T / 4000)
    assert 1.8 < e1 / e2 < 2.2                            # first order
    p1, _ = _oscillator_error(stepper.pefrl_step, T / 40)
    p2, _ = _oscillator_error(stepper.pefrl_step, T / 80)
    p3, _ = _oscillator_error(stepper.pefrl_step, T / 160)
    assert 13.0 < p1 / p2 < 19.0 and 13.0 < p2 / p3 < 19.0   # fourth order
    assert p1 < 1e-4 * e1                                  # and far more accurate than Euler at 50x the step


def test_s2_pefrl_coefficients_are_the_published_ones(stepper):
    # Omelyan et al. 2002: xi, lambda, chi of the optimised scheme (leading error coefficient minimised)
    assert abs(stepper.PEFRL_XI - 0.1786178958448091) < 1e-16
    assert abs(stepper.PEFRL_LAMBDA + 0.2123418310626054) < 1e-16
    assert abs(stepper.PEFRL_CHI + 0.06626458266981849) < 1e-16


# ---------------------------------------------------------------- S3: time reversibility
def test_s3_time_reversibility(stepper):
    rng = np.random.default_rng([31, 3])
    n = 6
    x0 = rng.uniform(-1e-6, 1e-6, (n, 3))
    v0 = rng.uniform(-1e5, 1e5, (n, 3))
    qm = rng.choice([-QE / ME, QE / (1836 * ME)], n)
    k = 1.0e7                                              # 1/m: the field varies over ~0.1 um (nonlinear force)
    field = lambda x: 1e7 * np.stack([np.sin(k * x[:, 1]) + np.cos(k * x[:, 2]), np.sin(k * x[:, 0]),   # noqa: E731
                                      np.cos(k * x[:, 0]) * np.sin(k * x[:, 1])], axis=1)
    h = 1e-13
    x, v = x0, v0
    for _ in range(20):
        x, v = stepper.pefrl_step(x, v, qm, h, field)
    assert np.linalg.norm(x - x0) > 1e-9                   # it went somewhere
    for _ in range(20):
        x, v = stepper.pefrl_step(x, v, qm, -h, field)
    assert np.allclose(x, x0, rtol=0, atol=1e-12 * np.abs(x0).max() + 1e-20)
    assert np.allclose(v, v0, rtol=1e-10)
    xe, ve = x0, v0
    for _ in range(20):
        xe, ve, _ = stepper.euler_step(xe, ve, qm, h, field)
    for _ in range(20):
        xe, ve, _ = stepper.euler_step(xe, ve, qm, -h, field)
    assert np.linalg.norm(xe - x0) > 1e3 * np.linalg.norm(x - x0)   # Euler is not reversible


# ---------------------------------------------------------------- S4: Kepler orbit through the field oracle
def test_s4_circular_orbit_with_the_field_oracle(ref, stepper):
    """A light negative charge on a circular orbit around a heavy positive one, the field taken from the pinned
    N-body oracle (Eq 3.8).  After one period PEFRL closes the orbit and conserves the energy."""
    r = 1.0e-6
    m_heavy, m_light = 1836 * 40 * ME, ME
    qm = np.array([QE / m_heavy, -QE / m_light])
    vorb = math.sqrt(KE * QE * QE / (m_light * r))
    period = 2 * math.pi * r / vorb
    x = np.array([[0.0, 0.0, 0.0], [r, 0.0, 0.0]])
    v = np.array([[0.0, -vorb * m_light / m_heavy, 0.0], [0.0, vorb, 0.0]])   # zero total momentum
    q = np.array([QE, -QE])

    def field(xx):
        xyzq = np.concatenate([xx, q[:, None]], axis=1).astype(np.float32)
        on, _ = ref.eval_field(xyzq=xyzq, flags=ref.NBODY)
        return on[:, :3]

    def energy(xx, vv):
        d = np.linalg.norm(xx[0] - xx[1])
        return 0.5 * m_heavy * (vv[0] ** 2).sum() + 0.5 * m_light * (vv[1] ** 2).sum() - KE * QE * QE / d

    e0 = energy(x, v)
    n = 400
    h = period / n
    x0 = x.copy()
    for _ in range(n):
        x, v = stepper.pefrl_step(x, v, qm, h, field)
    # fp32 rounding of the positions handed to the field oracle limits this to ~1e-6, not the scheme
    assert np.linalg.norm(x[1] - x0[1]) < 2e-4 * r
    assert abs(energy(x, v) - e0) < 1e-5 * abs(e0)


# ---------------------------------------------------------------- R1: nearest opposite charge vs scipy
def test_r1_nearest_opposite_against_kdtree(ref):
    from scipy.spatial import cKDTree
    rng = np.random.default_rng([31, 5])
    n = 3000
    xyzq = np.zeros((n, 4), dtype=np.float32)
    xyzq[:, :3] = rng.uniform(0, 50 * UM, (n, 3))
    xyzq[:, 3] = rng.choice([-QE, QE, 2 * QE, 0.0], n, p=[0.45, 0.35, 0.1, 0.1])
    d, j = ref.nearest_opposite(xyzq)
    pos = xyzq[:, :3].astype(np.float64)
    q = xyzq[:, 3]
    neg, plus = np.where(q < 0)[0], np.where(q > 0)[0]
    for mine, other in ((neg, plus), (plus, neg)):
        dd, jj = cKDTree(pos[other]).query(pos[mine], k=1)
        assert np.allclose(d[mine], dd, rtol=1e-13)
        assert np.array_equal(j[mine], other[jj])
    sub = np.array([5, 17, 2999, 0, 1234])
    ds, js = ref.nearest_opposite(xyzq, idx=sub)                          # subset form: same answers
    assert np.array_equal(ds, d[sub]) and np.array_equal(js, j[sub])
    zero = np.where(q == 0)[0]
    assert np.all(j[zero] == -1) and np.all(np.isinf(d[zero]))
    assert not np.isin(j[j >= 0], zero).any()
    # hand case incl. a tie (smallest index wins) and a lone species
    h = np.array([[0, 0, 0, QE], [1e-6, 0, 0, -QE], [-1e-6, 0, 0, -QE], [0, 3e-6, 0, QE]], dtype=np.float32)
    d, j = ref.nearest_opposite(h)
    assert list(j) == [1, 0, 0, 1] and abs(d[0] - float(np.float32(1e-6))) < 1e-20
    assert abs(d[3] - math.sqrt(float(np.float32(1e-6)) ** 2 + float(np.float32(3e-6)) ** 2)) < 1e-18
    d, j = ref.nearest_opposite(h[[0, 3]])
    assert list(j) == [-1, -1] and np.all(np.isinf(d))


def test_r2_recombination_radius(ref):
    # Eq (3.12): k_e e / (2 E_ioni); E_ioni = 13.6 eV gives half the Bohr-model distance k_e e / 13.6 V = 1.0588e-10 m
    assert abs(ref.recombination_radius(13.605693122994) - 0.5 * 1.0583544e-10) < 1e-16
    assert abs(ref.recombination_radius(15.76) / ref.recombination_radius(31.52) - 2.0) < 1e-14

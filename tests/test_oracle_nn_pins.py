"""Pins of the NN-approximation oracle (oracle/nn.py, reading A19).  CPU only.

The approximation has no closed form, so it is pinned by: the limit theta = 0 (everything near) = the brute-force
Eq (3.8) oracle; hand-computed 4-charge cases (3-4-5 geometry) where the far leaf is replaced by its centre of
charge; conservation of total charge and dipole moment by the pseudo-particles; the k-d partition's invariants;
input-permutation equivariance; second-order convergence in theta; the paper's own acceptance statement (Fig 6:
|dEz/Ez| < 5 % for more than 96.8 % of the particles when the electron and ion clouds are well separated).
"""
import numpy as np
import pytest

QE = 1.602176634e-19
KE = 1.0 / (4.0 * np.pi * 8.8541878128e-12)
UM = 1e-6


@pytest.fixture(scope="module")
def nn():
    from oracle import nn as _nn
    return _nn


def _cloud(rng, n, sigma=(20 * UM, 20 * UM, 10 * UM), centre=(0, 0, 0), q=None):
    x = np.zeros((n, 4), dtype=np.float32)
    x[:, :3] = rng.normal(0, 1, (n, 3)) * np.array(sigma) + np.array(centre)
    x[:, 3] = rng.choice([-QE, QE], n) if q is None else q
    return x


def test_n1_theta_zero_is_brute_force(nn, ref):
    rng = np.random.default_rng([51, 1])
    x = _cloud(rng, 3000)
    bf, _ = ref.eval_field(xyzq=x, eps_pp=0.05 * UM, flags=ref.NBODY)
    got, tree = nn.nn_field(x, 0.05 * UM, 0.0, leaf=16, group=128, ref=ref)
    assert np.allclose(got, bf, rtol=1e-11, atol=1e-14 * np.abs(bf).max())
    assert not nn.far_mask(tree, 0, 0.0).any()


def test_n2_hand_values_far_pair_replaced_by_its_centre_of_charge(nn, ref):
    """leaf = group = 2.  Pair A at the origin region, pair B 300 um away along x: the k-d cut separates them.
    Same-sign pair B -> ONE pseudo-particle 2q at its midpoint; the field at A's charges is the partner's exact
    field plus k_e 2q d/|d|^3 from the midpoint (3-4-5 triangles: |d| = 5 units)."""
    u = 100 * UM
    A0, A1 = np.array([0.0, 0.0, 0.0]), np.array([0.0, 0.0, 0.5 * u])
    B0, B1 = np.array([3 * u, 4 * u - 0.1 * u, 0.0]), np.array([3 * u, 4 * u + 0.1 * u, 0.0])   # midpoint (3u, 4u, 0)
    x = np.zeros((4, 4), dtype=np.float32)
    x[:, :3] = [A0, B0, A1, B1]                                           # interleaved on purpose
    x[:, 3] = [QE, QE, -QE, QE]
    q32 = float(x[0, 3])                                                  # the charge as the fp32 input carries it
    got, tree = nn.nn_field(x, 0.0, 2.0, leaf=2, group=2, ref=ref)
    assert sorted(tree["perm"][:2].tolist()) == [0, 2] and sorted(tree["perm"][2:].tolist()) == [1, 3]
    p32 = x[:, :3].astype(np.float64)
    mid = 0.5 * (p32[1] + p32[3])
    # target A0 (index 0): partner A1 (-e) exactly + 2e at mid
    d1, dm = p32[0] - p32[2], p32[0] - mid
    e_exp = KE * (-q32) * d1 / np.linalg.norm(d1) ** 3 + KE * 2 * q32 * dm / np.linalg.norm(dm) ** 3
    phi_exp = KE * (-q32) / np.linalg.norm(d1) + KE * 2 * q32 / np.linalg.norm(dm)
    assert np.allclose(got[0, :3], e_exp, rtol=1e-12) and abs(got[0, 3] - phi_exp) <= 1e-12 * abs(phi_exp)
    assert abs(np.linalg.norm(dm) / (5 * u) - 1) < 1e-6                   # the 3-4-5 triangle
    # seen from B, pair A is (+e, -e): two pseudo-particles sitting ON the charges -> the brute-force value
    bf, _ = ref.eval_field(xyzq=x, eps_pp=0.0, flags=ref.NBODY)
    assert np.allclose(got[[1, 3]], bf[[1, 3]], rtol=1e-12)
    # and A0's value is NOT the brute-force one (B0, B1 are 0.2 u apart): the approximation is really in use
    assert np.linalg.norm(got[0, :3] - bf[0, :3]) > 1e-5 * np.linalg.norm(bf[0, :3])


def test_n3_partition_invariants(nn):
    rng = np.random.default_rng([51, 3])
    for n in (1, 15, 16, 17, 100, 1000, 4099):
        x = _cloud(rng, n)
        perm = nn.kd_order(x, leaf=16)
        assert sorted(perm.tolist()) == list(range(n))
        if n > 16:
            # the top-level cut is along the longest axis of the whole cloud and separates it
            ext = x[:, :3].max(0).astype(np.float64) - x[:, :3].min(0).astype(np.float64)
            ax = int(np.argmax(ext))
            m = nn.split_point(0, n, 16)
            assert m % 16 == 0 and n / 2 <= m < n / 2 + 16
            assert x[perm[:m], ax].max() <= x[perm[m:], ax].min()
    # ties keep the input order (stable): identical points stay in input order inside a leaf
    x = np.zeros((40, 4), dtype=np.float32)
    x[:, 3] = QE
    assert nn.kd_order(x, leaf=16).tolist() == list(range(40))
    # IEEE total order of the key: -0.0 sorts before +0.0, negatives before positives
    k = nn._ordered_key(np.array([-1.0, -0.0, 0.0, 1e-30, 2.0], dtype=np.float32))
    assert np.all(np.diff(k.astype(np.int64)) > 0)


def test_n4_pseudo_particles_conserve_charge_and_dipole(nn):
    rng = np.random.default_rng([51, 4])
    x = _cloud(rng, 5000, q=rng.choice([-QE, QE, 2 * QE, 0.0], 5000).astype(np.float32))
    tree = nn.build(x, leaf=32, group=256)
    pp = tree["pseudo"].reshape(-1, 4)
    q = x[:, 3].astype(np.float64)
    assert abs(pp[:, 3].sum() - q.sum()) <= 1e-12 * np.abs(q).sum()
    dip = (q[:, None] * x[:, :3].astype(np.float64)).sum(0)
    assert np.allclose((pp[:, 3:4] * pp[:, :3]).sum(0), dip, rtol=0, atol=1e-12 * np.abs(q).sum() * 50 * UM)
    # every pseudo-particle lies inside its leaf's box, + ones carry positive charge and - ones negative
    lb = tree["leaf_boxes"]
    for h, sign in ((0, 1), (1, -1)):
        sel = tree["pseudo"][:, h, 3] != 0
        assert np.all(sign * tree["pseudo"][sel, h, 3] > 0)
        inside = (tree["pseudo"][sel, h, :3] >= lb[sel, 0] - 1e-18) & (tree["pseudo"][sel, h, :3] <= lb[sel, 1] + 1e-18)
        assert inside.all()
    # group boxes contain their leaves' boxes
    for g in range(tree["group_boxes"].shape[0]):
        b = lb[g * 8:(g + 1) * 8]
        assert np.all(tree["group_boxes"][g, 0] <= b[:, 0]) and np.all(tree["group_boxes"][g, 1] >= b[:, 1])


def test_n5_input_permutation_equivariance(nn, ref):
    rng = np.random.default_rng([51, 5])
    x = _cloud(rng, 2500)
    a, _ = nn.nn_field(x, 0.05 * UM, 1.5, leaf=16, group=128, ref=ref)
    p = rng.permutation(len(x))
    b, _ = nn.nn_field(x[p], 0.05 * UM, 1.5, leaf=16, group=128, ref=ref)
    assert np.allclose(b, a[p], rtol=1e-10, atol=1e-13 * np.abs(a).max())


def test_n6_error_falls_with_theta_at_second_order(nn, ref):
    rng = np.random.default_rng([51, 6])
    x = _cloud(rng, 8192)
    bf, _ = ref.eval_field(xyzq=x, eps_pp=0.05 * UM, flags=ref.NBODY)
    err = {}
    for th in (0.5, 1.0, 2.0):
        got, _ = nn.nn_field(x, 0.05 * UM, th, leaf=16, group=128, ref=ref)
        d = np.linalg.norm(got[:, :3] - bf[:, :3], axis=1)
        err[th] = float(np.sqrt((d ** 2).sum() / (np.linalg.norm(bf[:, :3], axis=1) ** 2).sum()))
    assert err[0.5] < err[1.0] < err[2.0] < 2e-2, err
    # the leading neglected term of a same-sign leaf is its quadrupole: (size/dist)^2 ~ theta^2
    assert 2.0 < err[1.0] / err[0.5] < 8.0 and 1.5 < err[2.0] / err[1.0] < 8.0, err


def test_n7_paper_fig6_acceptance_on_separated_clouds(nn, ref):
    """ion and electron clouds "well separated after their drift in opposite directions ... the
    absolute relative differences are below 5 % for more than 96.8 % of the particles" (on E_z).  Parallel-plate
    like set-up: an electron cloud and an ion cloud 150 um apart along z, default theta = 2, default leaf / group."""
    rng = np.random.default_rng([51, 7])
    n = 16384
    el = _cloud(rng, n // 2, sigma=(30 * UM, 30 * UM, 15 * UM), centre=(0, 0, +75 * UM), q=-QE)
    io = _cloud(rng, n // 2, sigma=(30 * UM, 30 * UM, 15 * UM), centre=(0, 0, -75 * UM), q=+QE)
    x = np.concatenate([el, io])[rng.permutation(n)]
    bf, _ = ref.eval_field(xyzq=x, eps_pp=0.05 * UM, flags=ref.NBODY)
    got, _ = nn.nn_field(x, 0.05 * UM, 2.0, leaf=64, group=512, ref=ref)
    rel = np.abs((got[:, 2] - bf[:, 2]) / bf[:, 2])
    assert (rel < 0.05).mean() > 0.968, (rel < 0.05).mean()


def test_n8_two_level_far_hand_value_and_limits(nn, ref):
    """leaf = group = 2, super-leaf = 2 leaves.  Pair A at the origin; four equal charges B 5 mm away (two leaves,
    ONE super-leaf whose box is far from A's box): A sees them as ONE pseudo-particle 4q at their centroid.  With
    super-leaves that are never far (super_ larger than the tree) the result is the one-level one."""
    u = 100 * UM
    pts = [[0, 0, 0], [0, 0, 0.3 * u],                                        # A
           [50 * u, 0.1 * u, 0], [50 * u, -0.1 * u, 0], [50.2 * u, 0.1 * u, 0], [50.2 * u, -0.1 * u, 0],   # B
           [0, 3 * u, 0], [0.2 * u, 3 * u, 0]]                                 # C: pads A's super-leaf to 2 leaves
    x = np.zeros((8, 4), dtype=np.float32)
    x[:, :3] = pts
    x[:, 3] = [QE, -QE, QE, QE, QE, QE, -QE, QE]
    q32 = float(x[0, 3])
    got, tree = nn.nn_field(x, 0.0, 1.0, leaf=2, group=2, super_=2, ref=ref)
    perm = tree["perm"]
    # which super-leaf holds B?  the one whose members are input indices 2..5
    supers = [sorted(perm[4 * k:4 * k + 4].tolist()) for k in range(2)]
    assert [2, 3, 4, 5] in supers
    gA = [g for g in range(4) if sorted(perm[2 * g:2 * g + 2].tolist()) == [0, 1]][0]
    far_super, near, far_leaf = nn.classify(tree, gA, 1.0)
    assert far_super[supers.index([2, 3, 4, 5])] and not far_super[1 - supers.index([2, 3, 4, 5])]
    p = x[:, :3].astype(np.float64)
    cB = p[2:6].mean(axis=0)
    # A0 = exact partner A1 + 4q at B's centroid + leaf C (far leaf or near: take what classify says)
    d1, dB = p[0] - p[1], p[0] - cB
    e = KE * (-q32) * d1 / np.linalg.norm(d1) ** 3 + KE * 4 * q32 * dB / np.linalg.norm(dB) ** 3
    lC = [l for l in range(4) if sorted(perm[2 * l:2 * l + 2].tolist()) == [6, 7]][0]
    for j, qj in ((6, -q32), (7, q32)):                                       # C is (-e, +e): its two pseudo-particles ARE its charges
        dj = p[0] - p[j]
        e = e + KE * qj * dj / np.linalg.norm(dj) ** 3
    assert near[lC] or far_leaf[lC]
    assert np.allclose(got[0, :3], e, rtol=1e-12)
    # never-far super-leaves reproduce the one-level scheme
    rng = np.random.default_rng([51, 8])
    y = _cloud(rng, 4096)
    one, t1 = nn.nn_field(y, 0.05 * UM, 4.0, leaf=16, group=128, super_=10 ** 6, ref=ref)
    two, t2 = nn.nn_field(y, 0.05 * UM, 4.0, leaf=16, group=128, super_=8, ref=ref)
    assert not any(nn.classify(t1, g, 4.0)[0].any() for g in range(32))
    assert any(nn.classify(t2, g, 4.0)[0].any() for g in range(32)), "no far super-leaf: vacuous"
    bf, _ = ref.eval_field(xyzq=y, eps_pp=0.05 * UM, flags=ref.NBODY)
    err = lambda a: np.sqrt(((a[:, :3] - bf[:, :3]) ** 2).sum() / (bf[:, :3] ** 2).sum())
    assert err(one) < 5e-2 and err(two) < 5e-2 and err(two) < 2 * err(one)      # super-leaves are accepted at theta / 2
    assert nn.units(t2, 4.0, 4096, block=16) < nn.units(t1, 4.0, 4096, block=16)
    # super-leaf pseudo-particles conserve charge and dipole moment as well
    q = y[:, 3].astype(np.float64)
    sp = t2["super_pseudo"].reshape(-1, 4)
    assert abs(sp[:, 3].sum() - q.sum()) <= 1e-12 * np.abs(q).sum()
    assert np.allclose((sp[:, 3:4] * sp[:, :3]).sum(0), (q[:, None] * y[:, :3].astype(np.float64)).sum(0), rtol=0,
                       atol=1e-12 * np.abs(q).sum() * 50 * UM)

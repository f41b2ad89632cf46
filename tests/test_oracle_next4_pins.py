"""Pins of the static-field-option oracle (oracle/fieldmap.py).  CPU only."""
import numpy as np
import pytest


@pytest.fixture(scope="module")
def fieldmap():
    from oracle import fieldmap as f
    return f


def _lattice(shape, origin, spacing):
    ax = [origin[a] + spacing[a] * np.arange(shape[a]) for a in range(3)]
    return ax, np.stack(np.meshgrid(*ax, indexing="ij"), axis=-1)


def test_m1_reproduces_trilinear_functions_exactly(fieldmap):
    """Trilinear interpolation is exact for f = a + b x + c y + d z + e xy + f yz + g xz + h xyz."""
    rng = np.random.default_rng([41, 1])
    shape, origin, spacing = (7, 5, 9), (-2e-4, 1e-5, -1.5e-4), (3e-6, 5e-6, 2e-6)
    _, xyz = _lattice(shape, origin, spacing)
    coef = rng.normal(size=(8, 4))

    def f(p):
        x, y, z = p[..., 0] * 1e5, p[..., 1] * 1e5, p[..., 2] * 1e5
        basis = np.stack([np.ones_like(x), x, y, z, x * y, y * z, x * z, x * y * z], axis=-1)
        return basis @ coef

    fmap = f(xyz)
    lo = np.array(origin)
    hi = lo + np.array(spacing) * (np.array(shape) - 1)
    pts = rng.uniform(lo, hi, (200, 3))
    got = fieldmap.trilinear(fmap, origin, spacing, pts)
    assert np.allclose(got, f(pts), rtol=1e-11, atol=1e-11 * np.abs(fmap).max())
    # node values are reproduced, including the last node of every axis
    idx = rng.integers(0, shape, (50, 3))
    idx[0] = np.array(shape) - 1
    nodes = lo + idx * np.array(spacing)
    got = fieldmap.trilinear(fmap, origin, spacing, nodes)
    assert np.allclose(got, fmap[idx[:, 0], idx[:, 1], idx[:, 2]], rtol=1e-10, atol=1e-10 * np.abs(fmap).max())


def test_m2_against_scipy_regular_grid_interpolator(fieldmap):
    from scipy.interpolate import RegularGridInterpolator
    rng = np.random.default_rng([41, 2])
    shape, origin, spacing = (6, 8, 5), (0.0, -1e-4, 2e-5), (4e-6, 1e-6, 7e-6)
    ax, _ = _lattice(shape, origin, spacing)
    fmap = rng.normal(size=shape + (4,))
    lo = np.array(origin)
    hi = lo + np.array(spacing) * (np.array(shape) - 1)
    pts = rng.uniform(lo, hi, (300, 3))
    got = fieldmap.trilinear(fmap, origin, spacing, pts)
    exp = RegularGridInterpolator(ax, fmap, method="linear")(pts)     # independent library routine
    assert np.allclose(got, exp, rtol=1e-10, atol=1e-12)
    # a transposed map is a different function: the check above would catch swapped axes
    swapped = fieldmap.trilinear(fmap.transpose(1, 0, 2, 3)[:6, :6], origin, spacing, pts[:20] * 0 + lo)
    assert swapped.shape == (20, 4)


def test_m3_clamping_outside_the_lattice(fieldmap):
    rng = np.random.default_rng([41, 3])
    shape, origin, spacing = (4, 4, 4), (0.0, 0.0, 0.0), (1.0, 1.0, 1.0)
    fmap = rng.normal(size=shape + (2,))
    outside = np.array([[-5.0, 1.5, 2.5], [1.5, 9.0, 0.5], [1.2, 2.2, -0.1], [7.0, 7.0, 7.0]])
    inside = np.clip(outside, 0.0, 3.0)
    assert np.allclose(fieldmap.trilinear(fmap, origin, spacing, outside),
                       fieldmap.trilinear(fmap, origin, spacing, inside), rtol=0, atol=1e-15)
    assert np.allclose(fieldmap.trilinear(fmap, origin, spacing, outside[3:]), fmap[3, 3, 3][None], atol=1e-15)


def test_m4_midpoint_is_the_mean_of_the_eight_corners(fieldmap):
    fmap = np.arange(2 * 2 * 2 * 1, dtype=np.float64).reshape(2, 2, 2, 1) ** 2
    got = fieldmap.trilinear(fmap, (0, 0, 0), (2.0, 4.0, 8.0), np.array([[1.0, 2.0, 4.0]]))
    assert abs(got[0, 0] - fmap.mean()) < 1e-14
    got = fieldmap.trilinear(fmap, (0, 0, 0), (2.0, 4.0, 8.0), np.array([[0.5, 0.0, 0.0]]))
    assert abs(got[0, 0] - (0.75 * fmap[0, 0, 0, 0] + 0.25 * fmap[1, 0, 0, 0])) < 1e-14   # hand value

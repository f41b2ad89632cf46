"""fp64 ORACLE for the static field option: interpolation of a precomputed 3-D field map
at the particle positions.

TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as obem_ref.c): imports nothing from paper_2110_09214_b200 and
shares no code with the CUDA path.  Plain numpy, written out corner by corner.

PAPER.md:235, section 3.2.1: "the field components are computed only once at some predefined spatial coordinates
located on a uniform 3D grid map ... During the transport, the field components at each particle location are then
interpolated in this 3D map."  The paper does not say which interpolation; reading A18 takes trilinear
interpolation of every component (Ex, Ey, Ez, phi) between the 8 surrounding nodes, positions outside the node
lattice clamped to its boundary (constant extrapolation).

Map layout: node (ix, iy, iz) at (x0 + ix dx, y0 + iy dy, z0 + iz dz), values map[ix, iy, iz, 0..3], z fastest --
the order in which config 5's evaluation points are generated.
"""
from __future__ import annotations

import numpy as np


def trilinear(fmap, origin, spacing, pts):
    """fmap [nx, ny, nz, C] float, origin (x0, y0, z0), spacing (dx, dy, dz), pts [M, >=3] -> [M, C] float64."""
    fmap = np.asarray(fmap, dtype=np.float64)
    pts = np.asarray(pts, dtype=np.float64)
    nx, ny, nz, nc = fmap.shape
    out = np.zeros((pts.shape[0], nc), dtype=np.float64)
    dims = (nx, ny, nz)
    for m in range(pts.shape[0]):
        i0 = [0, 0, 0]
        f = [0.0, 0.0, 0.0]
        for a in range(3):
            u = (pts[m, a] - origin[a]) / spacing[a]           # position in node units
            u = min(max(u, 0.0), float(dims[a] - 1))           # clamp to the lattice (reading A18)
            i = int(np.floor(u))
            if i > dims[a] - 2:                                # last node: use the last cell with f = 1
                i = max(dims[a] - 2, 0)
            i0[a] = i
            f[a] = u - i if dims[a] > 1 else 0.0
        acc = np.zeros(nc)
        for cx in (0, 1):
            for cy in (0, 1):
                for cz in (0, 1):
                    w = (f[0] if cx else 1.0 - f[0]) * (f[1] if cy else 1.0 - f[1]) * (f[2] if cz else 1.0 - f[2])
                    ix = min(i0[0] + cx, nx - 1)
                    iy = min(i0[1] + cy, ny - 1)
                    iz = min(i0[2] + cz, nz - 1)
                    acc += w * fmap[ix, iy, iz]
        out[m] = acc
    return out

"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the CUDA path's tests/bench and the oracle's tests.  It holds geometry and
random sampling only -- none of the method's arithmetic (no field sums, no quadrature, no panel
areas) -- and imports neither the CUDA binding nor the oracle.

The inputs stand in for the paper's workloads: avalanches of 1e6-1e7 electrons and ions
 in GEM foils with bi-conic 50/70 um holes at 140 um pitch and
parallel-plate set-ups.  The paper uses no public dataset on this path.

Recipe: numpy default_rng([0, cfg]), everything drawn in fp64 and rounded
ONCE to fp32, SI metres and coulombs.  Charges are kept in the gas (reading A9): any sample inside
the foil solid or within CLEARANCE of a meshed surface is redrawn.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Optional

import numpy as np

E_CHARGE = 1.602176634e-19  # C (reading A7)
UM = 1.0e-6

# GEM geometry, PAPER.md:435 (bi-conic 50/70 um holes, pitch 140 um) and reading A12.
PITCH = 140.0 * UM
R_OUTER = 35.0 * UM        # hole radius at the Cu faces
R_INNER = 25.0 * UM        # hole radius at the foil mid-plane
Z_KAPTON = 25.0 * UM       # half thickness of the Kapton
Z_FOIL = 30.0 * UM         # half thickness Kapton + Cu
CLEARANCE = 0.25 * UM      # charges stay this far from every meshed surface (A9)
_RADIAL_CLEARANCE = 0.30 * UM  # radial margin inside holes (cone slope + chord sagitta of flat panels)


@dataclass
class Workload:
    name: str
    cfg: int
    xyzq: np.ndarray                     # [N,4] float32 (x,y,z [m], q [C]); N may be 0
    verts: np.ndarray                    # [Np,3,3] float32 [m]
    sigma: np.ndarray                    # [Np] float32 [C/m^2]
    eps_pp: float                        # Plummer softening of the charge-charge sum [m]
    eps_panel: float = 0.0               # reading A5
    points: Optional[np.ndarray] = None  # [M,4] float32 free evaluation points (config 5)
    meta: dict = field(default_factory=dict)

    @property
    def n_charges(self) -> int:
        return int(self.xyzq.shape[0])

    @property
    def n_panels(self) -> int:
        return int(self.verts.shape[0])

    @property
    def n_targets(self) -> int:
        return int(self.points.shape[0]) if self.points is not None else self.n_charges

    def interactions(self) -> dict:
        """Pairwise-interaction counts (reading A13)."""
        n, t = self.n_charges, self.n_targets
        nbody = n * (n - 1) if self.points is None else 0
        return {"nbody": nbody, "panel": 7 * self.n_panels * t, "total": nbody + 7 * self.n_panels * t}


# ----------------------------------------------------------------------------------------------
# meshes
# ----------------------------------------------------------------------------------------------
def _quads_to_tris(p00, p10, p11, p01):
    """Split every quad (p00,p10,p11,p01) along the p00-p11 diagonal -> [2*nq,3,3]."""
    t1 = np.stack([p00, p10, p11], axis=1)
    t2 = np.stack([p00, p11, p01], axis=1)
    return np.concatenate([t1, t2], axis=0)


def plane_mesh(x0, x1, y0, y1, z, nx, ny):
    """nx*ny rectangular cells on the plane z = const, two triangles each (same diagonal)."""
    xs = np.linspace(x0, x1, nx + 1)
    ys = np.linspace(y0, y1, ny + 1)
    X, Y = np.meshgrid(xs, ys, indexing="ij")
    Z = np.full_like(X, z)
    P = np.stack([X, Y, Z], axis=-1)
    p00 = P[:-1, :-1].reshape(-1, 3)
    p10 = P[1:, :-1].reshape(-1, 3)
    p11 = P[1:, 1:].reshape(-1, 3)
    p01 = P[:-1, 1:].reshape(-1, 3)
    return _quads_to_tris(p00, p10, p11, p01)


def hole_radius(z):
    """Local radius of the bi-conic hole at height z relative to the foil mid-plane (A12)."""
    az = np.abs(z)
    return np.where(az >= Z_KAPTON, R_OUTER, R_INNER + (R_OUTER - R_INNER) * az / Z_KAPTON)


def _wrap60(theta):
    s = math.pi / 3.0
    return (theta + s / 2.0) % s - s / 2.0


def hex_radius(theta):
    """Distance from a hole centre to its hexagonal cell boundary in direction theta."""
    return (PITCH / 2.0) / np.cos(_wrap60(theta))


def gem_cell(ntheta, nz, nr, centre_xy=(0.0, 0.0), z0=0.0):
    """One hexagonal GEM cell: hole wall (ntheta x nz quads on the bi-conic surface) and the two outer
    Cu faces (ntheta x nr quads each, hole rim -> cell hexagon).  2*ntheta*(nz+2*nr) triangles.
    Returns (tris[?,3,3], is_kapton[?]) -- is_kapton marks hole-wall panels on the Kapton (|z|<25 um)."""
    th = np.linspace(0.0, 2.0 * math.pi, ntheta + 1)
    th[-1] = 0.0  # close the ring exactly
    c, s = np.cos(th), np.sin(th)
    cx, cy = centre_xy
    # hole wall
    zs = np.linspace(-Z_FOIL, Z_FOIL, nz + 1)
    R = hole_radius(zs)
    X = cx + R[None, :] * c[:, None]
    Y = cy + R[None, :] * s[:, None]
    Zz = np.broadcast_to(z0 + zs[None, :], X.shape)
    P = np.stack([X, Y, Zz], axis=-1)
    wall = _quads_to_tris(P[:-1, :-1].reshape(-1, 3), P[1:, :-1].reshape(-1, 3),
                          P[1:, 1:].reshape(-1, 3), P[:-1, 1:].reshape(-1, 3))
    zc = wall[:, :, 2].mean(axis=1) - z0
    kap = np.abs(zc) < Z_KAPTON
    parts, flags = [wall], [kap]
    # outer faces: transfinite map rim -> hexagon
    thv = np.linspace(0.0, 2.0 * math.pi, ntheta + 1)
    Rh = hex_radius(thv)
    Rh[-1] = Rh[0]
    u = np.linspace(0.0, 1.0, nr + 1)
    Rr = R_OUTER + (Rh[:, None] - R_OUTER) * u[None, :]
    Xf = cx + Rr * c[:, None]
    Yf = cy + Rr * s[:, None]
    for zf in (z0 + Z_FOIL, z0 - Z_FOIL):
        Pf = np.stack([Xf, Yf, np.full_like(Xf, zf)], axis=-1)
        face = _quads_to_tris(Pf[:-1, :-1].reshape(-1, 3), Pf[1:, :-1].reshape(-1, 3),
                              Pf[1:, 1:].reshape(-1, 3), Pf[:-1, 1:].reshape(-1, 3))
        parts.append(face)
        flags.append(np.zeros(face.shape[0], dtype=bool))
    return np.concatenate(parts, axis=0), np.concatenate(flags, axis=0)


def hex_ring_centres(ring):
    """Hole centres of hexagonal ring `ring` (0: 1 hole, 1: 6, 2: 12) on the PITCH lattice."""
    if ring == 0:
        return [(0.0, 0.0)]
    out = []
    a = PITCH
    # walk the ring in axial coordinates
    dirs = [(1, 0), (0, 1), (-1, 1), (-1, 0), (0, -1), (1, -1)]
    # ring walk: start at dirs[4]*ring and walk each of the 6 sides
    q, r = dirs[4][0] * ring, dirs[4][1] * ring
    for d in range(6):
        for _ in range(ring):
            out.append((a * (q + r / 2.0), a * (r * math.sqrt(3.0) / 2.0)))
            q += dirs[d][0]
            r += dirs[d][1]
    return out


def gem_patch(spec, z0=0.0):
    """spec: list of (ring, ntheta, nz, nr).  Returns (tris, is_kapton, centres[?,2])."""
    tris, kaps, cents = [], [], []
    for ring, nth, nz, nr in spec:
        for cxy in hex_ring_centres(ring):
            t, k = gem_cell(nth, nz, nr, cxy, z0)
            tris.append(t)
            kaps.append(k)
            cents.append(cxy)
    return np.concatenate(tris), np.concatenate(kaps), np.asarray(cents, dtype=np.float64)


# ----------------------------------------------------------------------------------------------
# "in the gas" predicate for clouds around GEM foils (reading A9)
# ----------------------------------------------------------------------------------------------
def in_gas(xyz, foil_z, centres):
    """True where a point is in the gas: outside every foil slab by CLEARANCE, or inside a meshed hole
    with radial margin.  foil_z: iterable of foil mid-plane heights; centres: [H,2] hole centres."""
    ok = np.ones(xyz.shape[0], dtype=bool)
    for z0 in foil_z:
        zl = xyz[:, 2] - z0
        slab = np.abs(zl) < (Z_FOIL + CLEARANCE)
        if not slab.any():
            continue
        idx = np.nonzero(slab)[0]
        d2 = ((xyz[idx, None, 0] - centres[None, :, 0]) ** 2 + (xyz[idx, None, 1] - centres[None, :, 1]) ** 2)
        rmin = np.sqrt(d2.min(axis=1))
        # inside the slab's extended thickness use the narrowest applicable radius
        zin = np.clip(np.abs(zl[idx]), 0.0, Z_FOIL)
        inside = rmin < (hole_radius(zin) - _RADIAL_CLEARANCE)
        ok[idx] = inside
    return ok


def _sample_into_gas(rng, n, draw, foil_z, centres):
    """Rejection sampling: draw(m) -> [m,3]; keep samples with in_gas."""
    out = np.empty((n, 3), dtype=np.float64)
    have = 0
    while have < n:
        m = max(1024, int((n - have) * 1.5))
        cand = draw(m)
        cand = cand[in_gas(cand, foil_z, centres)]
        k = min(n - have, cand.shape[0])
        out[have:have + k] = cand[:k]
        have += k
    return out


def _avalanche_cloud(rng, n_e, n_i, z_foil, centres, foil_z):
    """Config-3 shape (BASELINE.json config 3): electrons in a Gaussian head, ions in an exponential
    tail along -z."""
    def draw_e(m):
        return np.stack([rng.normal(0.0, 20.0 * UM, m), rng.normal(0.0, 20.0 * UM, m),
                         z_foil + 40.0 * UM + rng.normal(0.0, 10.0 * UM, m)], axis=1)

    def draw_i(m):
        return np.stack([rng.normal(0.0, 20.0 * UM, m), rng.normal(0.0, 20.0 * UM, m),
                         z_foil + 40.0 * UM - rng.exponential(30.0 * UM, m)], axis=1)

    pe = _sample_into_gas(rng, n_e, draw_e, foil_z, centres)
    pi = _sample_into_gas(rng, n_i, draw_i, foil_z, centres)
    xyz = np.concatenate([pe, pi], axis=0)
    q = np.concatenate([np.full(n_e, -E_CHARGE), np.full(n_i, +E_CHARGE)])
    return xyz, q


def _pack(xyz, q):
    out = np.empty((xyz.shape[0], 4), dtype=np.float32)
    out[:, :3] = xyz
    out[:, 3] = q
    return out


# ----------------------------------------------------------------------------------------------
# the five configs (BASELINE.json "configs"; readings A10-A12 of SURVEY.md section 8(c))
# ----------------------------------------------------------------------------------------------
CONFIG_NAMES = {
    1: "tiny-nbody-bem",
    2: "single-gem-cell",
    3: "avalanche-snapshot",
    4: "double-gem-large-avalanche",
    5: "field-map",
}


def _patch_rect(centres):
    m = PITCH / math.sqrt(3.0) + 1.0 * UM  # hexagon circumradius
    return (centres[:, 0].min() - m, centres[:, 0].max() + m, centres[:, 1].min() - m, centres[:, 1].max() + m)


def make_workload(cfg: int, charge_div: int = 1, mesh_div: int = 1, point_div: int = 1) -> Workload:
    """Build config `cfg` (1..5).  charge_div / mesh_div / point_div shrink the charge count, the mesh
    resolution (ntheta, nz, nr, plane cells) and config 5's grid per axis for small parity cases; the
    defaults (1, 1, 1) are the BASELINE.json sizes."""
    if cfg not in CONFIG_NAMES:
        raise ValueError("cfg must be 1..5")
    rng = np.random.default_rng([0, cfg])
    md = mesh_div
    meta = {"charge_div": charge_div, "mesh_div": mesh_div, "point_div": point_div}

    if cfg == 1:
        # A10: 16x16 cells of 6.25 um on each of the planes z = 0 and z = 100 um -> 2*256*2 = 1024
        L = 100.0 * UM
        nc = max(1, 16 // md)
        verts = np.concatenate([plane_mesh(0, L, 0, L, 0.0, nc, nc), plane_mesh(0, L, 0, L, L, nc, nc)])
        sigma = rng.normal(0.0, 1.0e-6, verts.shape[0])
        ne = 2048 // charge_div
        xyz = np.stack([rng.uniform(0.0, L, 2 * ne), rng.uniform(0.0, L, 2 * ne),
                        rng.uniform(CLEARANCE, L - CLEARANCE, 2 * ne)], axis=1)
        q = np.concatenate([np.full(ne, -E_CHARGE), np.full(ne, +E_CHARGE)])
        return Workload(CONFIG_NAMES[1], 1, _pack(xyz, q), verts.astype(np.float32),
                        sigma.astype(np.float32), 0.1 * UM, meta=meta)

    if cfg == 2:
        spec = [(0, 128 // md, 32 // md, 16 // md)]
        verts, _, centres = gem_patch(spec)
        sigma = rng.normal(0.0, 1.0e-5, verts.shape[0])
        ne = 32768 // charge_div

        def draw(m):
            return np.stack([rng.normal(0.0, 15.0 * UM, m), rng.normal(0.0, 15.0 * UM, m),
                             rng.normal(0.0, 25.0 * UM, m)], axis=1)

        xyz = _sample_into_gas(rng, 2 * ne, draw, [0.0], centres)
        q = np.concatenate([np.full(ne, -E_CHARGE), np.full(ne, +E_CHARGE)])
        return Workload(CONFIG_NAMES[2], 2, _pack(xyz, q), verts.astype(np.float32),
                        sigma.astype(np.float32), 0.1 * UM, meta=meta)

    if cfg == 3:
        spec = [(0, 128 // md, 32 // md, 16 // md), (1, 128 // md, 16 // md, 8 // md)]
        verts, _, centres = gem_patch(spec)
        sigma = rng.normal(0.0, 1.0e-5, verts.shape[0])
        ne = 524288 // charge_div
        xyz, q = _avalanche_cloud(rng, ne, ne, 0.0, centres, [0.0])
        return Workload(CONFIG_NAMES[3], 3, _pack(xyz, q), verts.astype(np.float32),
                        sigma.astype(np.float32), 0.05 * UM, meta=meta)

    if cfg == 4:
        spec = [(0, 128 // md, 32 // md, 16 // md), (1, 128 // md, 16 // md, 8 // md),
                (2, 64 // md, 16 // md, 8 // md)]
        zf = [0.0, -2.0e-3]
        parts, sig = [], []
        centres = None
        for z0 in zf:
            v, kap, centres = gem_patch(spec, z0)
            s = rng.normal(0.0, 1.0e-5, v.shape[0])
            s[kap] = rng.exponential(2.0e-5, int(kap.sum()))  # charging-up on the Kapton walls (A11)
            parts.append(v)
            sig.append(s)
        x0, x1, y0, y1 = _patch_rect(centres)
        for zp in (+1.0e-3, -3.0e-3):  # drift and anode planes
            v = plane_mesh(x0, x1, y0, y1, zp, 128 // md, 64 // md)
            parts.append(v)
            sig.append(rng.normal(0.0, 1.0e-5, v.shape[0]))
        verts = np.concatenate(parts)
        sigma = np.concatenate(sig)
        na = 1048576 // charge_div
        nb = 3 * na
        xa, qa = _avalanche_cloud(rng, na // 2, na // 2, zf[0], centres, zf)
        xb, qb = _avalanche_cloud(rng, nb // 2, nb // 2, zf[1], centres, zf)
        return Workload(CONFIG_NAMES[4], 4, _pack(np.concatenate([xa, xb]), np.concatenate([qa, qb])),
                        verts.astype(np.float32), sigma.astype(np.float32), 0.05 * UM, meta=meta)

    # cfg == 5: field map, no charges
    spec = [(0, 256 // md, 32 // md, 16 // md), (1, 256 // md, 32 // md, 16 // md)]
    v, _, centres = gem_patch(spec)
    parts = [v]
    for zp in (+150.0 * UM, -150.0 * UM):
        parts.append(plane_mesh(-210.0 * UM, 210.0 * UM, -210.0 * UM, 210.0 * UM, zp, 128 // md, 64 // md))
    verts = np.concatenate(parts)
    sigma = rng.normal(0.0, 1.0e-5, verts.shape[0])
    ng = 256 // point_div
    gx = (np.arange(ng) + 0.5) * (420.0 * UM / ng) - 210.0 * UM
    gz = (np.arange(ng) + 0.5) * (300.0 * UM / ng) - 150.0 * UM
    pts = np.zeros((ng, ng, ng, 4), dtype=np.float32)
    pts[..., 0] = gx[:, None, None]
    pts[..., 1] = gx[None, :, None]
    pts[..., 2] = gz[None, None, :]
    return Workload(CONFIG_NAMES[5], 5, np.zeros((0, 4), dtype=np.float32), verts.astype(np.float32),
                    sigma.astype(np.float32), 0.0, points=pts.reshape(-1, 4), meta=meta)


def pair_creation_order(wl: Workload, seed: int = 0) -> Workload:
    """The same charges in the order an avalanche stores them.  The generators above write all electrons, then all
    ions; the method creates electrons and ions in PAIRS as the avalanche grows, so its
    particle array interleaves the signs.  Stand-in: a seeded random permutation of the config's charges
    (`meta["perm"]`: position in the returned array -> position in `wl`); panels and points are unchanged."""
    if wl.n_charges == 0:
        return wl
    perm = np.random.default_rng([1, wl.cfg, seed]).permutation(wl.n_charges)
    meta = dict(wl.meta)
    meta["perm"] = perm
    return Workload(wl.name + "-pair-order", wl.cfg, np.ascontiguousarray(wl.xyzq[perm]), wl.verts, wl.sigma, wl.eps_pp,
                    wl.eps_panel, wl.points, meta)


def random_rotation(rng):
    """A proper 3x3 rotation matrix (QR of a Gaussian matrix), for invariance tests."""
    a = rng.normal(size=(3, 3))
    qm, r = np.linalg.qr(a)
    qm = qm * np.sign(np.diag(r))
    if np.linalg.det(qm) < 0:
        qm[:, 0] = -qm[:, 0]
    return qm

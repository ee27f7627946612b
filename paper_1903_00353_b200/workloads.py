"""Seeded synthetic mesh + grid workloads (input generators only).

This module serves both the CUDA path and the CPU oracle. It holds NONE of the
method's arithmetic (no distances, normals, pseudonormals, classification): it
only builds closed, outward-oriented triangle soups and the grid description
of each BASELINE.json config.

Common recipe: build an INDEXED mesh in fp64; apply jitter /
rotation / pose to the UNIQUE vertices; round every unique vertex to fp32 ONCE;
expand to an STL-style soup (so duplicates are bit-identical and the surface
stays closed); counter-clockwise from outside
(PAPER.md:278); then a seeded permutation of the triangle order and a seeded
cyclic rotation of each triangle's three vertices ("order of
triangles ... can be arbitrary").

The public meshes the paper measures on are not available;
these synthetic configs stand in for them.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

__all__ = [
    "Workload", "soup_from_indexed", "box_mesh", "icosphere_mesh", "torus_mesh",
    "uv_star_mesh", "tetrahedron_mesh", "cube_fan_mesh", "box_with_cavity_mesh",
    "monkey_saddle_mesh", "ruff_mesh", "spike_mesh", "multibody_mesh",
    "grid_over", "config", "CONFIG_NAMES", "random_rotation",
]


# --------------------------------------------------------------------------- #
# containers
# --------------------------------------------------------------------------- #
@dataclass
class Workload:
    """One mesh + grid problem.  `soup` is float32 [F,3,3] (triangle, vertex, xyz).

    Grid convention: sample (i,j,k) sits at origin + (i,j,k)*h,
    linear index (k*ny + j)*nx + i; "grid N^3 over [-1,1]^3" means h = 2/N and
    origin = -1 + h/2 (cell centres).
    """
    name: str
    soup: np.ndarray
    origin: tuple
    h: float
    dims: tuple            # (nx, ny, nz)
    band: float            # band width in length units (= band_cells * h)
    meta: dict = field(default_factory=dict)

    @property
    def ntri(self) -> int:
        return int(self.soup.shape[0])

    @property
    def ncells(self) -> int:
        nx, ny, nz = self.dims
        return int(nx) * int(ny) * int(nz)

    @property
    def diag(self) -> float:
        nx, ny, nz = self.dims
        return float(self.h * np.sqrt(float(nx) ** 2 + float(ny) ** 2 + float(nz) ** 2))

    def crop(self, lo, size) -> "Workload":
        """Same mesh, a sub-window of the same grid (cells lo .. lo+size-1)."""
        lo = tuple(int(v) for v in lo)
        size = tuple(int(v) for v in size)
        org = tuple(float(np.float32(self.origin[a]) + np.float32(lo[a]) * np.float32(self.h))
                    for a in range(3))
        return Workload(self.name + "_crop", self.soup, org, self.h, size, self.band,
                        dict(self.meta, crop_lo=lo))


def grid_over(lo, hi, n):
    """Cell-centred grid with n=(nx,ny,nz) cells over the box [lo,hi]; cubic cells."""
    lo = np.asarray(lo, dtype=np.float64)
    hi = np.asarray(hi, dtype=np.float64)
    n = np.asarray(n, dtype=np.int64)
    hs = (hi - lo) / n
    h = float(hs[0])
    assert np.allclose(hs, h), "cells must be cubic"
    origin = tuple(float(v) for v in (lo + 0.5 * h))
    return origin, h, tuple(int(v) for v in n)


# --------------------------------------------------------------------------- #
# indexed -> soup
# --------------------------------------------------------------------------- #
def soup_from_indexed(verts64, tris, rng=None):
    """Round unique vertices to fp32 once, expand, optionally shuffle.

    verts64: [V,3] float64, tris: [F,3] int (CCW from outside).
    rng: numpy Generator or None (no shuffle / rotation).
    """
    v32 = np.ascontiguousarray(verts64, dtype=np.float64).astype(np.float32)
    v32 = v32 + np.float32(0.0)          # canonicalise -0.0 -> +0.0
    tris = np.asarray(tris, dtype=np.int64)
    if rng is not None:
        tris = tris[rng.permutation(tris.shape[0])]
        rot = rng.integers(0, 3, size=tris.shape[0])
        idx = (np.arange(3)[None, :] + rot[:, None]) % 3
        tris = np.take_along_axis(tris, idx, axis=1)
    return np.ascontiguousarray(v32[tris])           # [F,3,3] float32


def random_rotation(rng):
    """Rotation matrix from a unit quaternion built from 4 seeded normals."""
    q = rng.standard_normal(4)
    q = q / np.linalg.norm(q)
    w, x, y, z = q
    return np.array([
        [1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
        [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
        [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)],
    ])


# --------------------------------------------------------------------------- #
# primitive indexed meshes (fp64 vertices, CCW-from-outside triangles)
# --------------------------------------------------------------------------- #
_BOX_TRIS = np.array([
    # vertex id = x + 2*y + 4*z with bits in {0,1}; each face split on one diagonal
    [0, 2, 3], [0, 3, 1],      # z = lo  (outward -z)
    [4, 5, 7], [4, 7, 6],      # z = hi  (+z)
    [0, 1, 5], [0, 5, 4],      # y = lo  (-y)
    [2, 6, 7], [2, 7, 3],      # y = hi  (+y)
    [0, 4, 6], [0, 6, 2],      # x = lo  (-x)
    [1, 3, 7], [1, 7, 5],      # x = hi  (+x)
], dtype=np.int64)


def box_mesh(half=(0.5, 0.35, 0.25), centre=(0.0, 0.0, 0.0)):
    """Axis-aligned box, 8 vertices / 12 triangles."""
    half = np.asarray(half, dtype=np.float64)
    centre = np.asarray(centre, dtype=np.float64)
    bits = np.array([[(i >> a) & 1 for a in range(3)] for i in range(8)], dtype=np.float64)
    verts = centre + (2.0 * bits - 1.0) * half
    return verts, _BOX_TRIS.copy()


def tetrahedron_mesh(scale=0.5):
    verts = scale * np.array([[1, 1, 1], [1, -1, -1], [-1, 1, -1], [-1, -1, 1]], dtype=np.float64)
    tris = np.array([[0, 1, 2], [0, 3, 1], [0, 2, 3], [1, 3, 2]], dtype=np.int64)
    return verts, tris


def icosphere_mesh(subdiv=1, radius=1.0):
    """Icosahedron subdivided `subdiv` times, projected to the sphere."""
    t = (1.0 + np.sqrt(5.0)) / 2.0
    verts = [(-1, t, 0), (1, t, 0), (-1, -t, 0), (1, -t, 0), (0, -1, t), (0, 1, t),
             (0, -1, -t), (0, 1, -t), (t, 0, -1), (t, 0, 1), (-t, 0, -1), (-t, 0, 1)]
    verts = [np.asarray(v, dtype=np.float64) / np.sqrt(1 + t * t) for v in verts]
    tris = [(0, 11, 5), (0, 5, 1), (0, 1, 7), (0, 7, 10), (0, 10, 11), (1, 5, 9), (5, 11, 4),
            (11, 10, 2), (10, 7, 6), (7, 1, 8), (3, 9, 4), (3, 4, 2), (3, 2, 6), (3, 6, 8),
            (3, 8, 9), (4, 9, 5), (2, 4, 11), (6, 2, 10), (8, 6, 7), (9, 8, 1)]
    verts = np.array(verts)
    tris = np.array(tris, dtype=np.int64)
    for _ in range(subdiv):
        e = np.concatenate([tris[:, [0, 1]], tris[:, [1, 2]], tris[:, [2, 0]]], axis=0)
        e_sorted = np.sort(e, axis=1)
        uniq, inv = np.unique(e_sorted, axis=0, return_inverse=True)
        inv = inv.reshape(-1)
        mid = verts[uniq[:, 0]] + verts[uniq[:, 1]]
        mid /= np.linalg.norm(mid, axis=1, keepdims=True)
        base = verts.shape[0]
        verts = np.concatenate([verts, mid], axis=0)
        F = tris.shape[0]
        m01 = base + inv[0:F]
        m12 = base + inv[F:2 * F]
        m20 = base + inv[2 * F:3 * F]
        a, b, c = tris[:, 0], tris[:, 1], tris[:, 2]
        tris = np.concatenate([
            np.stack([a, m01, m20], 1), np.stack([b, m12, m01], 1),
            np.stack([c, m20, m12], 1), np.stack([m01, m12, m20], 1)], axis=0)
    return verts * radius, tris


def torus_mesh(R=0.6, r=0.25, nu=200, nv=100):
    """Torus about the z axis, nu toroidal x nv poloidal quads, split on one diagonal."""
    u = 2 * np.pi * np.arange(nu) / nu
    v = 2 * np.pi * np.arange(nv) / nv
    U, Vv = np.meshgrid(u, v, indexing="ij")
    x = (R + r * np.cos(Vv)) * np.cos(U)
    y = (R + r * np.cos(Vv)) * np.sin(U)
    z = r * np.sin(Vv)
    verts = np.stack([x, y, z], axis=-1).reshape(-1, 3)
    i = np.arange(nu)[:, None]
    j = np.arange(nv)[None, :]
    i1 = (i + 1) % nu
    j1 = (j + 1) % nv
    v00 = (i * nv + j).ravel()
    v10 = (i1 * nv + j).ravel()
    v11 = (i1 * nv + j1).ravel()
    v01 = (i * nv + j1).ravel()
    tris = np.concatenate([np.stack([v00, v10, v11], 1), np.stack([v00, v11, v01], 1)], axis=0)
    return verts, tris


def _real_sph_harm_sum(theta, phi, lmax, coeffs):
    """S(theta_i, phi_j) = sum_{l<=lmax} sum_m a_lm Y_lm, real orthonormal harmonics.

    Separable evaluation: Y_l^m(theta, phi) = Theta_lm(theta) * exp(i m phi).
    """
    from scipy.special import sph_harm_y
    S = np.zeros((theta.size, phi.size))
    k = 0
    for l in range(lmax + 1):
        for m in range(-l, l + 1):
            a = coeffs[k]
            k += 1
            am = abs(m)
            th = np.real(sph_harm_y(l, am, theta, np.zeros_like(theta)))   # Theta_l|m|(theta)
            if m == 0:
                S += a * th[:, None]
            elif m > 0:
                S += a * np.sqrt(2.0) * (-1) ** m * th[:, None] * np.cos(am * phi)[None, :]
            else:
                S += a * np.sqrt(2.0) * (-1) ** m * th[:, None] * np.sin(am * phi)[None, :]
    return S


def uv_star_mesh(nphi=2000, ntheta=1000, lmax=8, amp=0.2, r0=0.6, rng=None):
    """Star-shaped surface r = r0 (1 + amp * S / max|S|) on a UV grid with pole fans.

    S = sum a_lm Y_lm, a_lm ~ N(0,1).  As literally written in BASELINE.json the
    radius would go negative, so S is rescaled to max|S| = 1
    over the mesh nodes (pole values included).  Vertices: 2 poles +
    (ntheta-1) rings of nphi; faces: 2*nphi*(ntheta-2) + 2*nphi.
    """
    ncoef = (lmax + 1) ** 2
    coeffs = rng.standard_normal(ncoef) if rng is not None else np.ones(ncoef)
    theta = np.pi * np.arange(0, ntheta + 1) / ntheta          # includes both poles
    phi = 2 * np.pi * np.arange(nphi) / nphi
    S = _real_sph_harm_sum(theta, phi, lmax, coeffs)
    S = S / np.max(np.abs(S))
    r = r0 * (1.0 + amp * S)
    st, ct = np.sin(theta)[:, None], np.cos(theta)[:, None]
    x = r * st * np.cos(phi)[None, :]
    y = r * st * np.sin(phi)[None, :]
    z = r * ct * np.ones_like(phi)[None, :]
    rings = np.stack([x, y, z], axis=-1)[1:ntheta]                # [ntheta-1, nphi, 3]
    north = np.array([[0.0, 0.0, r[0, 0]]])
    south = np.array([[0.0, 0.0, -r[ntheta, 0]]])
    verts = np.concatenate([north, rings.reshape(-1, 3), south], axis=0)
    nr = ntheta - 1
    south_id = 1 + nr * nphi

    def vid(i, j):            # ring i (0..nr-1), column j
        return 1 + i * nphi + (j % nphi)
    j = np.arange(nphi)
    tris = []
    # north fan: pole, ring0[j], ring0[j+1]  (theta increases away from +z; outward CCW)
    tris.append(np.stack([np.zeros(nphi, dtype=np.int64), vid(0, j), vid(0, j + 1)], 1))
    i = np.arange(nr - 1)[:, None]
    jj = j[None, :]
    a = vid(i, jj).ravel()
    b = vid(i + 1, jj).ravel()
    c = vid(i + 1, jj + 1).ravel()
    d = vid(i, jj + 1).ravel()
    tris.append(np.stack([a, b, c], 1))
    tris.append(np.stack([a, c, d], 1))
    tris.append(np.stack([np.full(nphi, south_id, dtype=np.int64), vid(nr - 1, j + 1), vid(nr - 1, j)], 1))
    return verts, np.concatenate(tris, axis=0)


def cube_fan_mesh(n_extra=(0, 2, 5), half=0.5):
    """Cube whose three faces at the corner (+,+,+) are fanned from that corner into
    1+n_extra[a] ... coplanar triangles each (unequal fans: the case angle weighting
    exists for).  The other three faces use two triangles.
    """
    h = float(half)
    verts = [np.array([(2 * ((i >> 0) & 1) - 1) * h, (2 * ((i >> 1) & 1) - 1) * h,
                       (2 * ((i >> 2) & 1) - 1) * h]) for i in range(8)]
    tris = [tuple(t) for t in _BOX_TRIS[[0, 1, 4, 5, 8, 9]]]        # the three "lo" faces
    corner = 7
    # each "hi" face: boundary loop starting at the corner, CCW from outside
    loops = {0: [7, 5, 1, 3], 1: [7, 3, 2, 6], 2: [7, 6, 4, 5]}     # x=hi, y=hi, z=hi
    for axis, loop in loops.items():
        n = int(n_extra[axis])
        c0, p1, p2, p3 = loop
        assert c0 == corner
        mids = []
        for s in range(1, n + 1):
            tt = s / (n + 1.0)
            verts.append(verts[p1] * (1 - tt) + verts[p2] * tt)
            mids.append(len(verts) - 1)
        chain = [p1] + mids + [p2, p3]
        for s in range(len(chain) - 1):
            tris.append((corner, chain[s], chain[s + 1]))
    verts = np.array(verts)
    tris = np.array(tris, dtype=np.int64)
    # the lo faces adjacent to the split edges now have T-junctions: split them too
    return _resolve_t_junctions(verts, tris)


def _resolve_t_junctions(verts, tris):
    """Split any triangle edge that has mesh vertices lying strictly inside it, so the
    mesh stays a closed manifold after `cube_fan_mesh` inserts edge midpoints."""
    tris = [tuple(int(x) for x in t) for t in tris]
    changed = True
    while changed:
        changed = False
        out = []
        for (a, b, c) in tris:
            done = False
            for (p, q, o) in ((a, b, c), (b, c, a), (c, a, b)):
                d = verts[q] - verts[p]
                L2 = float(d @ d)
                best, best_t = None, None
                for k in range(len(verts)):
                    if k in (p, q, o):
                        continue
                    w = verts[k] - verts[p]
                    t = float(w @ d) / L2
                    if 1e-9 < t < 1 - 1e-9 and np.linalg.norm(w - t * d) < 1e-12:
                        if best is None or t < best_t:
                            best, best_t = k, t
                if best is not None:
                    out.append((p, best, o))
                    out.append((best, q, o))
                    done = True
                    changed = True
                    break
            if not done:
                out.append((a, b, c))
        tris = out
    return verts, np.array(tris, dtype=np.int64)


def box_with_cavity_mesh(outer=(0.6, 0.6, 0.6), inner=(0.25, 0.2, 0.3), centre_in=(0.05, 0.0, -0.03)):
    """Solid box with a box-shaped void: outer shell outward-oriented, inner shell
    oriented into the void (concave edges and vertices)."""
    vo, to = box_mesh(outer)
    vi, ti = box_mesh(inner, centre_in)
    ti = ti[:, ::-1] + vo.shape[0]
    return np.concatenate([vo, vi], 0), np.concatenate([to, ti], 0)


def _closed_from_heightfield(xy, tri2d, ztop, zbot, bottom_tri2d=None):
    """Closed solid between z = ztop(x,y) on top and a flat bottom z = zbot, with a
    side wall along the boundary loop of the planar triangulation (disk topology).
    `bottom_tri2d`: triangulation of the flat bottom when the top one is not a valid
    planar triangulation (overhanging top)."""
    n = xy.shape[0]
    top = np.concatenate([xy, ztop[:, None]], axis=1)
    bot = np.concatenate([xy, np.full((n, 1), zbot)], axis=1)
    verts = np.concatenate([top, bot], 0)
    bt = tri2d if bottom_tri2d is None else bottom_tri2d
    tris = [tri2d, bt[:, ::-1] + n]
    # boundary edges of the 2-D triangulation (appear once), keep their direction
    e = np.concatenate([tri2d[:, [0, 1]], tri2d[:, [1, 2]], tri2d[:, [2, 0]]], 0)
    key = {}
    for a, b in e:
        key[(int(a), int(b))] = True
    side = []
    for (a, b) in key:
        if (b, a) not in key:
            # top edge a->b is CCW seen from above; wall faces outward
            side.append((a, a + n, b + n))
            side.append((a, b + n, b))
    tris.append(np.array(side, dtype=np.int64))
    return verts, np.concatenate(tris, 0)


def monkey_saddle_mesh(nfan=6, radius=0.5, amp=0.25, zbot=-0.5, order=3):
    """Closed solid whose top has a central vertex with a fan of `nfan` neighbours at
    heights amp*cos(order*phi): neighbours lie on both sides of the pseudonormal plane
    (saddle, fig.7a)."""
    phi = 2 * np.pi * np.arange(nfan) / nfan
    xy = np.concatenate([[[0.0, 0.0]], radius * np.stack([np.cos(phi), np.sin(phi)], 1)], 0)
    z = np.concatenate([[0.0], amp * np.cos(order * phi)])
    tri2d = np.array([[0, 1 + k, 1 + (k + 1) % nfan] for k in range(nfan)], dtype=np.int64)
    return _closed_from_heightfield(xy, tri2d, z, zbot)


def ruff_mesh(nfan=8, radius=0.5, rise=0.05, fold=0.45, zbot=-0.6, apex=0.3):
    """Ruff-like vertex (fig.7b): apex above a pleated skirt whose
    alternate ring vertices are pulled in and up so that adjacent faces have almost
    opposite normals while all neighbours stay below the apex."""
    phi = 2 * np.pi * np.arange(nfan) / nfan
    rad = np.where(np.arange(nfan) % 2 == 0, radius, radius * (1 - fold))
    zz = np.where(np.arange(nfan) % 2 == 0, 0.0, apex - rise)
    xy = np.concatenate([[[0.0, 0.0]], np.stack([rad * np.cos(phi), rad * np.sin(phi)], 1)], 0)
    z = np.concatenate([[apex], zz])
    tri2d = np.array([[0, 1 + k, 1 + (k + 1) % nfan] for k in range(nfan)], dtype=np.int64)
    return _closed_from_heightfield(xy, tri2d, z, zbot)


def spike_mesh(nfan=5, radius=0.4, height=0.5, lean=0.55, zbot=-0.4):
    """Convex-classified vertex with one incident normal pointing far away from the
    pseudonormal (the 'pathological' case of PAPER.md:410, fig.17): a leaning apex."""
    phi = 2 * np.pi * np.arange(nfan) / nfan
    xy = np.concatenate([[[lean, 0.0]], radius * np.stack([np.cos(phi), np.sin(phi)], 1)], 0)
    z = np.concatenate([[height], np.zeros(nfan)])
    tri2d = np.array([[0, 1 + k, 1 + (k + 1) % nfan] for k in range(nfan)], dtype=np.int64)
    # the apex overhangs the ring, so the flat bottom is fanned from a ring vertex instead
    bottom = np.array([[1, 1 + k, 2 + k] for k in range(1, nfan - 1)], dtype=np.int64)
    return _closed_from_heightfield(xy, tri2d, z, zbot, bottom)


# --------------------------------------------------------------------------- #
# C5-style multi-body scene
# --------------------------------------------------------------------------- #
def multibody_mesh(rng, counts=(190, 150, 120, 40), lattice=(16, 8, 8), pitch=0.25,
                   ico_subdiv=4, torus_res=(100, 50), plate_thick=0.004):
    """Disjoint closed bodies on a seeded selection of lattice sites.

    counts = (boxes, plates, icospheres, tori).  Site centres at odd multiples of
    pitch/2 about the origin; bounding radius <= 0.10*(pitch/0.25); per-axis jitter
    <= 0.015*(pitch/0.25); seeded rotation and scale in [0.6,1] per body.  Plates keep
    their absolute thickness (thinner than the band).
    """
    nb = int(sum(counts))
    L = np.asarray(lattice)
    nsites = int(np.prod(L))
    assert nb <= nsites
    sites = rng.choice(nsites, size=nb, replace=False)
    kinds = np.concatenate([np.full(c, k) for k, c in enumerate(counts)])
    kinds = kinds[rng.permutation(nb)]
    s = pitch / 0.25
    verts_all, tris_all, base = [], [], 0
    ico_v, ico_t = icosphere_mesh(ico_subdiv, 1.0)
    tor_v, tor_t = torus_mesh(0.06, 0.03, torus_res[0], torus_res[1])
    for b in range(nb):
        site = int(sites[b])
        ix, iy, iz = site % L[0], (site // L[0]) % L[1], site // (L[0] * L[1])
        centre = (np.array([ix, iy, iz]) - (L - 1) / 2.0) * pitch
        centre = centre + rng.uniform(-0.015, 0.015, size=3) * s
        Rm = random_rotation(rng)
        scale = rng.uniform(0.6, 1.0) * s
        kind = int(kinds[b])
        if kind == 0:
            v, t = box_mesh((0.055, 0.045, 0.035))
            v = v * scale
        elif kind == 1:
            v, t = box_mesh((0.06, 0.05, 0.5))
            v = v * np.array([scale, scale, plate_thick])
        elif kind == 2:
            v, t = ico_v * (0.09 * scale), ico_t
        else:
            v, t = tor_v * scale, tor_t
        v = v @ Rm.T + centre
        verts_all.append(v)
        tris_all.append(t + base)
        base += v.shape[0]
    return np.concatenate(verts_all, 0), np.concatenate(tris_all, 0)


# --------------------------------------------------------------------------- #
# BASELINE.json configs
# --------------------------------------------------------------------------- #
CONFIG_NAMES = ("C1", "C2", "C3", "C4", "C5")
_SEEDS = {"C1": 1001, "C2": 1002, "C3": 1003, "C4": 1004, "C5": 1005}


def config(name: str, scale: float = 1.0) -> Workload:
    """Build BASELINE.json config `name` (C1..C5).

    scale < 1 builds a reduced variant with the same structure (fewer triangles, a
    proportionally coarser grid, same band in cells) for parity tests that the
    oracle finishes in seconds; scale = 1 is the full config.
    """
    seed = _SEEDS[name]
    rng = np.random.default_rng(seed)
    if name == "C1":
        v, t = box_mesh((0.50, 0.35, 0.25), (0.03, -0.02, 0.05))
        n = max(8, int(round(64 * scale)))
        origin, h, dims = grid_over((-1, -1, -1), (1, 1, 1), (n, n, n))
        return Workload("C1", soup_from_indexed(v, t, rng), origin, h, dims, 3 * h,
                        {"band_cells": 3, "seed": seed, "V": 8, "E": 18})
    if name == "C2":
        sub = 5 if scale >= 1 else max(1, int(round(5 + np.log2(scale))))
        v, t = icosphere_mesh(sub, 0.7)
        rad = v / np.linalg.norm(v, axis=1, keepdims=True)
        v = v + rad * rng.normal(0.0, 1e-3, size=(v.shape[0], 1))
        n = max(16, int(round(256 * scale)))
        origin, h, dims = grid_over((-1, -1, -1), (1, 1, 1), (n, n, n))
        return Workload("C2", soup_from_indexed(v, t, rng), origin, h, dims, 4 * h,
                        {"band_cells": 4, "seed": seed, "V": v.shape[0], "E": 3 * t.shape[0] // 2})
    if name == "C3":
        nu = max(12, int(round(200 * scale)))
        nv = max(6, int(round(100 * scale)))
        v, t = torus_mesh(0.6, 0.25, nu, nv)
        v = v @ random_rotation(rng).T
        n = max(16, int(round(512 * scale)))
        origin, h, dims = grid_over((-1, -1, -1), (1, 1, 1), (n, n, n))
        return Workload("C3", soup_from_indexed(v, t, rng), origin, h, dims, 3 * h,
                        {"band_cells": 3, "seed": seed, "V": v.shape[0], "E": 3 * t.shape[0] // 2})
    if name == "C4":
        nphi = max(16, int(round(2000 * scale)))
        nth = max(8, int(round(1000 * scale)))
        v, t = uv_star_mesh(nphi, nth, 8, 0.2, 0.6, rng)
        n = max(16, int(round(1024 * scale)))
        origin, h, dims = grid_over((-1, -1, -1), (1, 1, 1), (n, n, n))
        return Workload("C4", soup_from_indexed(v, t, rng), origin, h, dims, 2 * h,
                        {"band_cells": 2, "seed": seed, "V": v.shape[0], "E": 3 * t.shape[0] // 2})
    if name == "C5":
        if scale >= 1:
            counts, lattice, pitch = (190, 150, 120, 40), (16, 8, 8), 0.25
            sub, tres, n = 4, (100, 50), (2048, 1024, 1024)
        else:
            f = max(scale, 1.0 / 16)
            counts = tuple(max(1, int(round(c * f))) for c in (190, 150, 120, 40))
            lattice, pitch = (16, 8, 8), 0.25
            sub, tres = 3, (40, 20)
            n = tuple(max(32, int(round(d * f ** (1 / 3)))) for d in (2048, 1024, 1024))
            n = (2 * n[1], n[1], n[1])
        v, t = multibody_mesh(rng, counts, lattice, pitch, sub, tres)
        origin, h, dims = grid_over((-2, -1, -1), (2, 1, 1), n)
        return Workload("C5", soup_from_indexed(v, t, rng), origin, h, dims, 3 * h,
                        {"band_cells": 3, "seed": seed, "V": v.shape[0], "E": 3 * t.shape[0] // 2,
                         "bodies": int(sum(counts)), "tori": int(counts[3])})
    raise KeyError(name)

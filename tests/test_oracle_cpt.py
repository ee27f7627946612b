"""Pins of the oracle's closest points: checked against what
the mathematics fixes, not against the routine itself -- |x - cp| equals the oracle's |d|; cp lies
on its triangle (barycentric coordinates in [0,1], zero offset from the plane); outside an
axis-aligned box the closest point is the clamp of x to the box, inside it is the projection onto
the nearest face; on a sphere-like mesh cp is x pulled radially to within the sagitta."""
import numpy as np

from paper_1903_00353_b200 import workloads as W
from helpers import grid_points


def _bary(cp, tri):
    a, b, c = tri[:, 0], tri[:, 1], tri[:, 2]
    v0, v1, v2 = b - a, c - a, cp - a
    d00 = np.einsum("ij,ij->i", v0, v0); d01 = np.einsum("ij,ij->i", v0, v1); d11 = np.einsum("ij,ij->i", v1, v1)
    d20 = np.einsum("ij,ij->i", v2, v0); d21 = np.einsum("ij,ij->i", v2, v1)
    den = d00 * d11 - d01 * d01
    v = (d11 * d20 - d01 * d21) / den
    w = (d00 * d21 - d01 * d20) / den
    n = np.cross(v0, v1)
    off = np.einsum("ij,ij->i", v2, n) / np.linalg.norm(n, axis=1)
    return 1 - v - w, v, w, off


def test_closest_points_box_closed_form(oracle_mod):
    w = W.config("C1")
    om = oracle_mod.Mesh(w.soup)
    d, t = om.sdf(w.origin, w.h, w.dims, w.band)
    cp = om.closest_points(w.origin, w.h, w.dims, t).astype(np.float64)
    x = grid_points(w.origin, w.h, w.dims)
    p = w.soup.reshape(-1, 3).astype(np.float64)
    lo, hi = p.min(0), p.max(0)
    pop = np.isfinite(d)
    assert np.all(np.isposinf(cp[~pop]))
    out = pop & (d > 0)
    assert np.max(np.abs(cp[out] - np.clip(x[out], lo, hi))) < 1e-7          # fp32 rounding of the output
    ins = pop & (d < 0)
    xi = x[ins]
    gaps = np.stack([xi - lo, hi - xi], axis=-1).reshape(-1, 6)               # x-lo_x, hi_x-x, y..., z...
    face = np.argmin(gaps, axis=1)
    ref = xi.copy()
    ax = face // 2
    ref[np.arange(len(xi)), ax] = np.where(face % 2 == 0, lo[ax], hi[ax])
    unique = np.sort(gaps, axis=1)[:, 1] - np.sort(gaps, axis=1)[:, 0] > 1e-9  # nearest face is unique
    assert np.max(np.abs(cp[ins][unique] - ref[unique])) < 1e-7


def test_closest_points_lie_on_their_triangle_at_the_stated_distance(oracle_mod):
    for maker, seed in ((lambda: W.torus_mesh(0.55, 0.25, 24, 12), 3), (lambda: W.monkey_saddle_mesh(), 4),
                        (lambda: W.icosphere_mesh(2, 0.6), 5)):
        v, t = maker()
        soup = W.soup_from_indexed(v, t, np.random.default_rng(seed))
        origin, h, dims = W.grid_over((-1.0,) * 3, (1.0,) * 3, (40,) * 3)
        om = oracle_mod.Mesh(soup)
        d, tri = om.sdf(origin, h, dims, 4 * h)
        cp = om.closest_points(origin, h, dims, tri).astype(np.float64)
        pop = np.isfinite(d)
        x = grid_points(origin, h, dims)[pop]
        c = cp[pop]
        assert np.max(np.abs(np.linalg.norm(x - c, axis=1) - np.abs(d[pop].astype(np.float64)))) < 2e-7
        u, vv, ww, off = _bary(c, soup[tri[pop]].astype(np.float64))
        assert min(u.min(), vv.min(), ww.min()) > -1e-6 and max(u.max(), vv.max(), ww.max()) < 1 + 1e-6
        assert np.max(np.abs(off)) < 2e-7
    # sphere: cp is x pulled towards the centre, to within the sagitta of the inscribed polyhedron
    r = np.linalg.norm(c, axis=1)
    assert r.max() <= 0.6 + 1e-7 and r.min() > 0.6 * np.cos(0.36)
    cosang = np.einsum("ij,ij->i", c, x) / (r * np.linalg.norm(x, axis=1))
    assert cosang.min() > np.cos(0.36)

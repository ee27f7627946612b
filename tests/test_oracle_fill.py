"""Pins of the oracle's interior fill: after the axis sweeps
every cell the narrow band left unset must hold -band iff it lies inside the solid.  Inside is
decided here by brute force, independently of the sweeps: the sign of the exact distance to the
whole mesh (oracle.query, itself pinned by winding numbers in test_oracle_pins.py) and, on the box,
the closed form."""
import numpy as np
import pytest

from paper_1903_00353_b200 import workloads as W
from helpers import box_sdf, grid_points


def _workload(vt, seed, n=36, band_cells=2.0):
    v, t = vt
    soup = W.soup_from_indexed(v, t, np.random.default_rng(seed))
    origin, h, dims = W.grid_over((-1.0,) * 3, (1.0,) * 3, (n,) * 3)
    return W.Workload("fill", soup, origin, h, dims, band_cells * h)


def _shell():
    vo, to = W.icosphere_mesh(2, 0.8)
    vi, ti = W.icosphere_mesh(2, 0.45)
    return np.concatenate([vo, vi], 0), np.concatenate([to, ti[:, ::-1] + vo.shape[0]], 0)


@pytest.mark.parametrize("maker,seed", [
    (lambda: W.tetrahedron_mesh(0.8), 1),
    (lambda: W.box_mesh((0.7, 0.55, 0.6)), 2),
    (lambda: W.icosphere_mesh(2, 0.75), 3),
    (lambda: W.torus_mesh(0.55, 0.3, 24, 12), 4),
    (lambda: W.box_with_cavity_mesh((0.8, 0.8, 0.8), (0.4, 0.35, 0.45)), 5),   # the void stays unset
    (_shell, 6),
])
def test_fill_matches_brute_force_inside(oracle_mod, maker, seed):
    w = _workload(maker(), seed)
    om = oracle_mod.Mesh(w.soup)
    d, _t = om.sdf(w.origin, w.h, w.dims, w.band)
    f = oracle_mod.fill_interior(d, w.band)
    unset = ~np.isfinite(d)
    assert np.array_equal(f[~unset], d[~unset])                     # the band itself is untouched
    pts = grid_points(w.origin, w.h, w.dims).reshape(-1, 3)[unset.reshape(-1)]
    d_true, _ = om.query(pts)
    inside = d_true < 0
    assert inside.any() and (~inside).any()
    got = f[unset]
    assert np.all(got[inside] == np.float32(-np.float32(w.band)))
    assert np.all(np.isposinf(got[~inside]))
    # no secondary zero crossing: neighbours never jump from -x to +inf
    neg = np.isfinite(f) & (f < 0)
    for ax in range(3):
        a = np.take(neg, range(0, neg.shape[ax] - 1), axis=ax)
        b = np.take(np.isposinf(f), range(1, neg.shape[ax]), axis=ax)
        a2 = np.take(neg, range(1, neg.shape[ax]), axis=ax)
        b2 = np.take(np.isposinf(f), range(0, neg.shape[ax] - 1), axis=ax)
        assert not np.any(a & b) and not np.any(a2 & b2)


def test_fill_box_closed_form(oracle_mod):
    w = W.config("C1")
    om = oracle_mod.Mesh(w.soup)
    d, _t = om.sdf(w.origin, w.h, w.dims, w.band)
    f = oracle_mod.fill_interior(d, w.band)
    p = w.soup.reshape(-1, 3).astype(np.float64)
    ref = box_sdf(grid_points(w.origin, w.h, w.dims), p.min(0), p.max(0)).reshape(f.shape)
    deep = ref <= -float(np.float32(w.band))
    assert deep.sum() > 1000
    assert np.all(f[deep] == np.float32(-np.float32(w.band)))
    assert np.all(np.isposinf(f[ref >= float(np.float32(w.band))]))
    band = np.abs(ref) < float(np.float32(w.band)) * (1 - 1e-6)
    assert np.array_equal(f[band], d[band])


def test_fill_is_idempotent_and_axis_order_free_on_valid_input(oracle_mod):
    w = _workload(W.torus_mesh(0.55, 0.3, 24, 12), 7)
    d, _t = oracle_mod.Mesh(w.soup).sdf(w.origin, w.h, w.dims, w.band)
    f = oracle_mod.fill_interior(d, w.band)
    assert np.array_equal(oracle_mod.fill_interior(f, w.band), f)
    # sweeping the transposed grid (z, y, x order of the axes) fills the same cells
    ft = oracle_mod.fill_interior(np.ascontiguousarray(d.transpose(2, 1, 0)), w.band).transpose(2, 1, 0)
    assert np.array_equal(ft, f)


def _sweep_axis_commuted(d, axis, fillv):
    """One axis, written the other way round: a cell is filled iff the nearest set cell on either side
    is negative in the data at the START of the sweep (no in-place forward-then-backward walk)."""
    a = np.moveaxis(d, axis, -1)
    out = a.copy()
    n = a.shape[-1]
    for idx in np.ndindex(a.shape[:-1]):
        line = a[idx]
        setm = np.isfinite(line)
        left = np.zeros(n, dtype=np.int8)
        right = np.zeros(n, dtype=np.int8)
        s = 0
        for q in range(n):
            if setm[q]:
                s = -1 if line[q] < 0 else 1
            left[q] = s
        s = 0
        for q in range(n - 1, -1, -1):
            if setm[q]:
                s = -1 if line[q] < 0 else 1
            right[q] = s
        fill = ~setm & ((left < 0) | (right < 0))
        out[idx][fill] = fillv
    return np.moveaxis(out, -1, axis)


def test_forward_and_backward_walks_commute_within_a_sweep(oracle_mod):
    """The property the one-walk GPU sweeps rely on, on grids that are not SDFs."""
    rng = np.random.default_rng(11)
    for dims, density in (((9, 7, 11), 0.1), ((16, 5, 3), 0.4), ((4, 4, 30), 0.02), ((12, 12, 12), 0.2)):
        d = np.full(dims, np.inf, dtype=np.float32)
        sel = rng.random(dims) < density
        d[sel] = rng.standard_normal(int(sel.sum())).astype(np.float32)
        ref = oracle_mod.fill_interior(d, 0.5)
        got = d.copy()
        for axis in (2, 1, 0):              # x, y, z of a [nz, ny, nx] array
            got = _sweep_axis_commuted(got, axis, np.float32(-0.5))
        assert np.array_equal(got, ref)

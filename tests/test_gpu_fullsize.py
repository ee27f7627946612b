"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(device-resident soup, sdf_create + sdf_compute through the C ABI).

C2 and C3 are compared with the oracle element by element over the whole grid in one piece.  C4 (1024^3)
and C5 (2048x1024x1024, 2^31 cells: every linear index path is 64-bit) are compared element by element over
the whole grid too, in chunks of z-slices that the oracle computes as crops of the same grid (5,186,000 and
26,983,685 band cells: all of them, both of C4's valence-2000 poles included), plus properties that hold at any
size: |d| < band on populated cells, sentinels elsewhere, ids in range, the populated count equals the
library's own counter.
"""
import numpy as np
import pytest
import torch

from paper_1903_00353_b200 import workloads as W
from gpu_util import f32_grid
from helpers import compare_to_oracle

pytestmark = pytest.mark.gpu

KEYS = ("bad_sentinel", "bad_id_range", "bad_set", "bad_dist", "bad_sign", "bad_id")


def _gpu(w):
    from paper_1903_00353_b200 import binding as B
    m, d, t = B.compute_workload(w)
    torch.cuda.synchronize()
    return m, d, t, B.sdf_stats(m)


def _whole_grid_properties(w, d, t, stats):
    pop = torch.isfinite(d)
    n_pop = int(pop.sum().item())
    assert n_pop == stats["band_cells"] and n_pop > 0
    assert bool((torch.isposinf(d) | (torch.abs(d) < float(np.float32(w.band)))).all())
    assert bool(((t >= 0) == pop).all())
    assert int(t.max().item()) < w.ntri and int(t.min().item()) >= -1
    return n_pop


@pytest.mark.parametrize("name", ["C2", "C3"])
def test_full_grid(oracle_mod, name):
    w = f32_grid(W.config(name))
    om = oracle_mod.Mesh(w.soup)
    d_ref, t_ref = om.sdf(w.origin, w.h, w.dims, w.band)
    m, d, t, stats = _gpu(w)
    _whole_grid_properties(w, d, t, stats)
    res = compare_to_oracle(d.cpu().numpy(), t.cpu().numpy(), d_ref, t_ref, w, om)
    assert res["ok"] and all(res[k] == 0 for k in KEYS), {k: v for k, v in res.items()}
    assert (stats["V"], stats["E"]) == (w.meta["V"], w.meta["E"])
    # ids (clause 4): how many differ from the oracle's, and how.  "Ties" = the closest point lies on a shared edge /
    # vertex and the GPU's triangle is as close as the oracle's to the rounding of the oracle's fp32 output (several
    # ids are correct); "near" = accepted by the tolerance without being such a tie.  The near share
    # is bounded: a kernel that ignored the lowest-id rule, or named a neighbouring triangle, would show up here.
    print("ids %s: populated %d, id mismatches %d (share %.4f): ties %d, near %d (share %.2e), bad %d"
          % (name, res["populated_ref"], res["id_mismatch_total"], res["id_mismatch_share"], res["id_mismatch_ties"],
             res["id_mismatch_near"], res["id_near_share"], res["bad_id"]))
    assert res["id_near_share"] <= 2e-3, res


def _chunks(nz, nk):
    return [(k0, min(nk, nz - k0)) for k0 in range(0, nz, nk)]


@pytest.mark.parametrize("name,nk", [("C4", 64), ("C5", 32)])
def test_full_size_whole_grid(oracle_mod, name, nk):
    """C4 and C5 at BASELINE.json's full sizes, EVERY cell compared with the oracle under the four clauses: the grid is
    walked in chunks of nk z-slices (the oracle computes each chunk as a crop of the same grid, so host memory stays
    bounded), and the number of band cells compared must equal the library's own count for the whole grid.  C4's two
    valence-2000 pole vertices (5.9e-6-wide sliver fans) sit in the chunks that hold k = 207 and
    k = 783; both are asserted to be populated and compared."""
    from paper_1903_00353_b200 import binding as B
    w = f32_grid(W.config(name))
    nx, ny, nz = w.dims
    m, d, t, stats = _gpu(w)
    assert d.shape == (nz, ny, nx)
    _whole_grid_properties(w, d, t, stats)
    assert (stats["F"], stats["V"], stats["E"]) == (w.ntri, w.meta["V"], w.meta["E"])
    om = oracle_mod.Mesh(w.soup)
    # z-range of the surface in cell indices (from the soup): chunks outside it hold sentinels only
    z = w.soup[:, :, 2].astype(np.float64)
    kz = ((z.min() - w.band - w.origin[2]) / w.h, (z.max() + w.band - w.origin[2]) / w.h)
    compared = id_mis = id_near = ties = 0
    per_chunk = {}
    for k0, n in _chunks(nz, nk):
        dg, tg = d[k0:k0 + n], t[k0:k0 + n]
        if k0 + n - 1 < kz[0] - 1 or k0 > kz[1] + 1:
            assert not bool(torch.isfinite(dg).any()) and bool((tg == -1).all()), (k0, "cells populated outside the mesh's z-range")
            per_chunk[k0] = 0
            continue
        c = w.crop((0, 0, k0), (nx, ny, n))
        d_ref, t_ref = om.sdf(c.origin, c.h, c.dims, c.band)
        res = compare_to_oracle(dg.cpu().numpy(), tg.cpu().numpy(), d_ref, t_ref, c, om)
        assert res["ok"] and all(res[k] == 0 for k in KEYS), (k0, {k: v for k, v in res.items()})
        compared += res["populated_ref"]
        id_mis += res["id_mismatch_total"]; id_near += res["id_mismatch_near"]; ties += res["id_mismatch_ties"]
        per_chunk[k0] = res["populated_ref"]
        del d_ref, t_ref
    print("%s whole grid: %d band cells compared in %d chunks; id mismatches %d (ties %d, near %d = %.2e of the band)"
          % (name, compared, len(per_chunk), id_mis, ties, id_near, id_near / max(compared, 1)))
    # every band cell of the grid went through the element-by-element comparison (clause 1 exempts cells within
    # 1e-5 h of the band edge, so the two counts may differ by those few)
    assert abs(compared - stats["band_cells"]) <= max(8, stats["band_cells"] // 100000), (compared, stats["band_cells"])
    assert id_near <= 2e-3 * compared
    if name == "C4":
        assert compared > 5_000_000
        # the poles: the two vertices of valence 2000, and the chunks they sit in
        cvid = B.sdf_get_table(m, B.TABLE_CORNER_VID).reshape(-1)
        val = np.bincount(cvid)
        assert int((val == 2000).sum()) == 2 and int(val.max()) == 2000
        for v in np.flatnonzero(val == 2000):
            corner = int(np.flatnonzero(cvid == v)[0])
            kp = int(round((float(w.soup.reshape(-1, 3)[corner, 2]) - w.origin[2]) / w.h))
            assert per_chunk[(kp // nk) * nk] > 100_000, (kp, per_chunk)
    else:
        assert compared > 26_000_000
        # bodies on every lattice layer: no chunk inside the z-range of the bodies is skipped silently
        assert sum(1 for v in per_chunk.values() if v > 0) >= 0.7 * len(per_chunk)


def test_scale_36m_triangles():
    """Nine times C4's triangle count (the same star surface on a 6000 x 3000 UV mesh, 1.3 GB of soup):
    index arithmetic and table sizing beyond the configs.  No oracle at this size: generator-known
    topology, whole-grid properties, and the band itself -- the surface is C4's, so is the band."""
    from paper_1903_00353_b200 import binding as B
    rng = np.random.default_rng(1004)
    v, t = W.uv_star_mesh(nphi=6000, ntheta=3000, rng=rng)
    soup = W.soup_from_indexed(v, t, rng)
    F = soup.shape[0]
    assert F == 35_988_000
    origin, h, dims = W.grid_over((-1.0,) * 3, (1.0,) * 3, (1024,) * 3)
    w = f32_grid(W.Workload("star36m", soup, origin, h, dims, 2 * h))
    m = B.sdf_create(torch.from_numpy(soup).cuda())
    d, tr = B.sdf_compute(m, w.origin, w.h, w.dims, w.band)
    torch.cuda.synchronize()
    st = B.sdf_stats(m)
    assert (st["F"], st["V"], st["E"]) == (F, v.shape[0], 3 * F // 2) and st["V"] - st["E"] + st["F"] == 2
    assert st["edges_convex"] + st["edges_concave"] + st["edges_flat"] == st["E"]
    _whole_grid_properties(w, d, tr, st)
    assert abs(st["band_cells"] - 5_186_000) < 2_000          # C4's surface, C4's band


def test_grid_with_more_than_2_to_32_cells(oracle_mod):
    """A 1664 x 1664 x 1600 grid (4.43e9 cells > 2^32; 35 GB of output): linear cell indices need 64 bits in the fill, the
    emit pass, the sparse output and the closest-point pass.  A small sphere sits at the far corner, so every populated
    cell has a linear index beyond 2^32.  Grid spacing and origin are powers of two: a crop of the grid has bit-identical
    cell positions, so the window around the sphere must equal a compute of that window alone bit for bit, which in turn is
    compared with the oracle; everything outside the window must be sentinels."""
    from paper_1903_00353_b200 import binding as B
    nx, ny, nz = 1664, 1664, 1600
    h = 2.0 ** -10
    v, t = W.icosphere_mesh(3, 28 * h)
    centre = np.array([(nx - 48) * h, (ny - 48) * h, (nz - 48) * h])
    soup = W.soup_from_indexed(v + centre, t, np.random.default_rng(5))
    w = f32_grid(W.Workload("huge", soup, (0.0, 0.0, 0.0), h, (nx, ny, nz), 3 * h))
    assert nx * ny * nz > 2 ** 32
    m, d, tr = B.compute_workload(w)
    torch.cuda.synchronize()
    lo = (nx - 96, ny - 96, nz - 96)
    c = w.crop(lo, (96, 96, 96))
    # the window against the oracle
    om = oracle_mod.Mesh(c.soup)
    dref, tref = om.sdf(c.origin, c.h, c.dims, c.band)
    dwin = d[lo[2]:, lo[1]:, lo[0]:].contiguous().cpu().numpy()
    twin = tr[lo[2]:, lo[1]:, lo[0]:].contiguous().cpu().numpy()
    # the tolerance is the whole grid's (1e-5 h + 1e-6 diag: the window's coordinates are ~1.6, not ~0.1)
    import types
    cw = types.SimpleNamespace(h=c.h, band=c.band, diag=w.diag, ntri=c.ntri, dims=c.dims, origin=c.origin)
    res = compare_to_oracle(dwin, twin, dref, tref, cw, om)
    assert res["ok"], str({k: v for k, v in res.items() if not isinstance(v, (list, np.ndarray))})
    populated = int(np.isfinite(dref).sum())
    assert populated > 20000
    # ... and against the same window computed alone (bit for bit)
    m2, d2, t2 = B.compute_workload(c)
    torch.cuda.synchronize()
    assert np.array_equal(d2.cpu().numpy().view(np.int32), dwin.view(np.int32)) and np.array_equal(t2.cpu().numpy(), twin)
    # nothing populated outside the window, and sentinels everywhere else (also in the first cells and past index 2^32)
    assert int(torch.isfinite(d).sum()) == int(np.isfinite(dwin).sum())
    assert int((tr >= 0).sum()) == int((twin >= 0).sum())
    flat_d, flat_t = d.view(-1), tr.view(-1)
    for pos in (0, 1, 2 ** 31 - 1, 2 ** 31, 2 ** 32 - 1, 2 ** 32, 2 ** 32 + 1):
        assert torch.isinf(flat_d[pos]) and int(flat_t[pos]) == -1
    assert bool(torch.all(torch.isinf(d[0]))) and bool(torch.all(tr[0] == -1))
    # the band-sparse output and the closest points of the same call sequence agree with the dense grids
    nb, ids, sd, st_ = B.sdf_compute_sparse(m, w.origin, w.h, w.dims, w.band)
    torch.cuda.synchronize()
    assert nb > 0 and int(torch.isfinite(sd[:nb]).sum()) == int(np.isfinite(dwin).sum())
    cp = B.sdf_closest_points(m, w.origin, w.h, w.dims, tr)
    torch.cuda.synchronize()
    assert int(torch.isfinite(cp[..., 0]).sum()) == int((twin >= 0).sum())
    B.sdf_fill_interior(d, w.band)
    torch.cuda.synchronize()
    inside = int((d == -np.float32(w.band)).sum())
    assert inside > 1000 and bool(torch.all(torch.isinf(d[0])))
    m.destroy(); m2.destroy()

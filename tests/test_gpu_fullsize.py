"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(device-resident soup, sdf_create + sdf_compute through the C ABI).

C2 and C3 are compared with the oracle element by element over the whole grid.  C4 (1024^3) and
C5 (2048x1024x1024, 2^31 cells: every linear index path is 64-bit) are compared element by
element on z-slabs the oracle computes as crops of the same grid (first, middle, last slices:
the slabs cross brick, tile and grid boundaries), and over the whole grid through properties
that hold at any size: |d| < band on populated cells, sentinels elsewhere, ids in range, the
populated count equals the library's own counter.
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


@pytest.mark.parametrize("name,slabs", [
    ("C4", [(150, 24), (500, 24), (856, 24)]),
    ("C5", [(40, 16), (505, 16), (1000, 16)]),
])
def test_full_size_slabs(oracle_mod, name, slabs):
    w = f32_grid(W.config(name))
    nx, ny, nz = w.dims
    m, d, t, stats = _gpu(w)
    assert d.shape == (nz, ny, nx)
    _whole_grid_properties(w, d, t, stats)
    assert (stats["F"], stats["V"], stats["E"]) == (w.ntri, w.meta["V"], w.meta["E"])
    om = oracle_mod.Mesh(w.soup)
    checked = 0
    for k0, nk in slabs:
        c = w.crop((0, 0, k0), (nx, ny, nk))
        d_ref, t_ref = om.sdf(c.origin, c.h, c.dims, c.band)
        res = compare_to_oracle(d[k0:k0 + nk].cpu().numpy(), t[k0:k0 + nk].cpu().numpy(), d_ref, t_ref, c, om)
        assert res["ok"] and all(res[k] == 0 for k in KEYS), (k0, {k: v for k, v in res.items()})
        checked += res["populated_ref"]
    assert checked > 0


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

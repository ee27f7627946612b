"""GPU tests of the z-slab split (sdf_compute_zslab).

On one GPU the slabs of a P-way split are computed one after another: (1) on a grid with a
power-of-two spacing (every sample position is exact, include/sdf.h) their concatenation is
BIT-identical to the whole-grid sdf_compute; (2) on a grid with an awkward spacing each slab meets
the four parity clauses against the oracle run on the slab's own fp32 origin."""
import dataclasses

import numpy as np
import pytest
import torch

from paper_1903_00353_b200 import workloads as W
from gpu_util import f32_grid
from helpers import compare_to_oracle

pytestmark = pytest.mark.gpu

KEYS = ("bad_sentinel", "bad_id_range", "bad_set", "bad_dist", "bad_sign", "bad_id")


@pytest.mark.parametrize("name,scale,parts", [("C2", 0.5, 2), ("C3", 0.25, 3), ("C4", 0.125, 5), ("C5", 0.125, 4)])
def test_slabs_concatenate_to_the_whole_grid(name, scale, parts):
    from paper_1903_00353_b200 import binding as B
    w = f32_grid(W.config(name, scale))
    assert float(np.log2(w.h)).is_integer()                     # exact sample positions
    nx, ny, nz = w.dims
    m = B.sdf_create(np.ascontiguousarray(w.soup))
    d, t = B.sdf_compute(m, w.origin, w.h, w.dims, w.band)
    total = B.sdf_stats(m)["band_cells"]
    got, k = 0, 0
    for p in range(parts):
        k0, ds, ts = B.sdf_compute_zslab(m, w.origin, w.h, w.dims, w.band, p, parts)
        assert k0 == k and ds.shape == (B.sdf_zslab(nz, p, parts)[1], ny, nx)
        nk = ds.shape[0]
        assert torch.equal(ds, d[k0:k0 + nk]) and torch.equal(ts, t[k0:k0 + nk])
        got += B.sdf_stats(m)["band_cells"]
        k += nk
    assert k == nz and got == total
    B.sdf_destroy(m)


def test_slab_parity_on_an_awkward_spacing(oracle_mod):
    from paper_1903_00353_b200 import binding as B
    v, tr = W.torus_mesh(R=0.6, r=0.25, nu=60, nv=30)
    soup = W.soup_from_indexed(v, tr, np.random.default_rng(12))
    origin, h, dims = (-0.93, -0.95, -0.41), 0.0283, (67, 66, 30)           # nothing here is exact in binary
    w = f32_grid(W.Workload("torus", soup, origin, h, dims, 3.3 * h))
    nx, ny, nz = w.dims
    om = oracle_mod.Mesh(w.soup)
    m = B.sdf_create(np.ascontiguousarray(w.soup))
    checked = 0
    for parts in (2, 3):
        for p in range(parts):
            k0, ds, ts = B.sdf_compute_zslab(m, w.origin, w.h, w.dims, w.band, p, parts)
            nk = ds.shape[0]
            oz = float(np.float32(np.float64(w.origin[2]) + k0 * np.float64(w.h)))      # include/sdf.h
            c = dataclasses.replace(w, origin=(w.origin[0], w.origin[1], oz), dims=(nx, ny, nk))
            d_ref, t_ref = om.sdf(c.origin, c.h, c.dims, c.band)
            res = compare_to_oracle(ds.cpu().numpy(), ts.cpu().numpy(), d_ref, t_ref, c, om)
            assert res["ok"] and all(res[k] == 0 for k in KEYS), (parts, p, res)
            checked += res["populated_ref"]
    assert checked > 2000
    # an empty slab (more parts than bricks) is legal and touches nothing
    assert B.sdf_zslab(nz, 0, 64)[1] == 0
    k0, ds, ts = B.sdf_compute_zslab(m, w.origin, w.h, w.dims, w.band, 0, 64)
    assert ds.numel() == 0
    B.sdf_destroy(m)

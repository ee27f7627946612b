"""Band-sparse output (sdf_compute_sparse / sdf_compute_sparse_host, include/sdf.h): the bricks, expanded to a dense
grid here with numpy, must equal the dense grids of sdf_compute bit for bit -- populated cells, signs, ids, sentinels --
on aligned and ragged grids, device and host outputs, and the capacity protocol must behave as the header says."""
import numpy as np
import pytest
import torch

from paper_1903_00353_b200 import workloads as W
from gpu_util import f32_grid

pytestmark = pytest.mark.gpu


def _expand(n, ids, db, tb, dims):
    nx, ny, nz = dims
    nbx, nby, nbz = (nx + 7) // 8, (ny + 7) // 8, (nz + 7) // 8
    d = np.full((nbz * 8, nby * 8, nbx * 8), np.inf, dtype=np.float32)
    t = np.full((nbz * 8, nby * 8, nbx * 8), -1, dtype=np.int32)
    ids, db, tb = ids[:n], db[:n].reshape(n, 8, 8, 8), tb[:n].reshape(n, 8, 8, 8)
    bx, by, bz = ids % nbx, (ids // nbx) % nby, ids // (nbx * nby)
    for q in range(n):
        d[bz[q] * 8:bz[q] * 8 + 8, by[q] * 8:by[q] * 8 + 8, bx[q] * 8:bx[q] * 8 + 8] = db[q]
        t[bz[q] * 8:bz[q] * 8 + 8, by[q] * 8:by[q] * 8 + 8, bx[q] * 8:bx[q] * 8 + 8] = tb[q]
    # cells of a brick beyond the grid hold sentinels
    assert np.all(np.isposinf(d[nz:])) and np.all(np.isposinf(d[:, ny:])) and np.all(np.isposinf(d[:, :, nx:]))
    return d[:nz, :ny, :nx], t[:nz, :ny, :nx]


@pytest.mark.parametrize("name,scale", [("C1", 1.0), ("C2", 0.5), ("C3", 0.25), ("C4", 0.06), ("C5", 0.02)])
def test_sparse_equals_dense(name, scale):
    from paper_1903_00353_b200 import binding as B
    w = f32_grid(W.config(name, scale) if scale < 1.0 else W.config(name))
    m, d, t = B.compute_workload(w)
    s = B.sdf_stats(m)
    n, ids, db, tb = B.sdf_compute_sparse(m, w.origin, w.h, w.dims, w.band)
    torch.cuda.synchronize()
    assert B.sdf_stats(m)["band_cells"] == s["band_cells"]          # (the counters are those of the last call)
    assert n == s["bricks_active"] == B.sdf_brick_count(m, w.origin, w.h, w.dims, w.band) and n > 0
    ids_np = ids.cpu().numpy()
    assert np.all(np.diff(ids_np[:n]) > 0)                                  # ascending, no duplicates
    de, te = _expand(n, ids_np, db.cpu().numpy(), tb.cpu().numpy(), w.dims)
    assert np.array_equal(te, t.cpu().numpy())
    assert np.array_equal(de.view(np.int32), d.cpu().numpy().view(np.int32))
    # host outputs: same bricks through pinned buffers of a larger capacity
    cap = n + 5
    hi = torch.empty((cap,), dtype=torch.int32).pin_memory()
    hd = torch.empty((cap, 512), dtype=torch.float32).pin_memory()
    ht = torch.empty((cap, 512), dtype=torch.int32).pin_memory()
    n2, _, _, _ = B.sdf_compute_sparse(m, w.origin, w.h, w.dims, w.band, hi, hd, ht)
    assert n2 == n
    assert np.array_equal(hi.numpy()[:n], ids_np[:n])
    assert np.array_equal(hd.numpy()[:n].view(np.int32), db.cpu().numpy()[:n].view(np.int32))
    assert np.array_equal(ht.numpy()[:n], tb.cpu().numpy()[:n])
    B.sdf_destroy(m)


def test_sparse_ragged_grid_and_capacity_protocol():
    from paper_1903_00353_b200 import binding as B
    v, tr = W.torus_mesh(0.55, 0.25, 40, 20)
    soup = W.soup_from_indexed(v, tr, np.random.default_rng(5))
    dims = (61, 35, 50)                                                    # no axis a multiple of 8
    h = 2.0 / 61
    w = f32_grid(W.Workload("ragged", soup, (-1.0 + 0.013, -0.55, -0.8), h, dims, 3.3 * h))
    m, d, t = B.compute_workload(w)
    n = B.sdf_brick_count(m, w.origin, w.h, w.dims, w.band)
    assert n > 10
    # too small a capacity: SDF_ENOMEM, nothing written, the count reported
    ids = torch.full((n - 1,), 77, dtype=torch.int32, device="cuda")
    db = torch.full((n - 1, 512), 5.0, dtype=torch.float32, device="cuda")
    tb = torch.full((n - 1, 512), 9, dtype=torch.int32, device="cuda")
    with pytest.raises(B.SdfError) as e:
        B.sdf_compute_sparse(m, w.origin, w.h, w.dims, w.band, ids, db, tb)
    assert e.value.status == B.SDF_ENOMEM
    torch.cuda.synchronize()
    assert bool((ids == 77).all()) and bool((db == 5.0).all()) and bool((tb == 9).all())
    n2, ids, db, tb = B.sdf_compute_sparse(m, w.origin, w.h, w.dims, w.band)
    torch.cuda.synchronize()
    assert n2 == n
    de, te = _expand(n, ids.cpu().numpy(), db.cpu().numpy(), tb.cpu().numpy(), w.dims)
    assert np.array_equal(te, t.cpu().numpy()) and np.array_equal(de.view(np.int32), d.cpu().numpy().view(np.int32))
    # a grid that misses the mesh: zero bricks
    assert B.sdf_brick_count(m, (5.0, 5.0, 5.0), w.h, (16, 16, 16), w.band) == 0
    n0, _, _, _ = B.sdf_compute_sparse(m, (5.0, 5.0, 5.0), w.h, (16, 16, 16), w.band)
    assert n0 == 0
    B.sdf_destroy(m)

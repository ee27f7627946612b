"""GPU parity of sdf_fill_interior against the oracle's axis
sweeps: bit-exact (every cell is either untouched or exactly -band), on the GPU's own narrow band
and on the oracle's, at reduced and full sizes, plus inputs no SDF would produce (the sweeps are
defined for any grid)."""
import numpy as np
import pytest
import torch

from paper_1903_00353_b200 import workloads as W
from gpu_util import f32_grid

pytestmark = pytest.mark.gpu


def _gpu_fill(d_np, band):
    from paper_1903_00353_b200 import binding as B
    d = torch.from_numpy(np.ascontiguousarray(d_np)).cuda()
    B.sdf_fill_interior(d, band)
    torch.cuda.synchronize()
    return d.cpu().numpy()


@pytest.mark.parametrize("name,scale", [("C1", 1.0), ("C2", 0.5), ("C3", 0.25), ("C4", 0.06), ("C5", 0.05), ("C2", 1.0)])
def test_fill_matches_oracle(oracle_mod, name, scale):
    from paper_1903_00353_b200 import binding as B
    w = f32_grid(W.config(name, scale))
    m, d, t = B.compute_workload(w)
    d_np = d.cpu().numpy()
    ref = oracle_mod.fill_interior(d_np, w.band)
    B.sdf_fill_interior(d, w.band)
    torch.cuda.synchronize()
    got = d.cpu().numpy()
    assert np.array_equal(got, ref)
    filled = np.isfinite(got) & ~np.isfinite(d_np)
    assert filled.sum() > 0 and np.all(got[filled] == np.float32(-np.float32(w.band)))
    assert np.all(t.cpu().numpy()[filled] == -1)


@pytest.mark.parametrize("dims", [(37, 29, 43), (1, 1, 70), (65, 1, 3), (33, 64, 1), (200, 7, 5), (700, 3, 2), (31, 300, 2), (5, 2, 290),
                                  (1100, 5, 40), (2100, 3, 35), (70, 45, 100), (40, 100, 37), (96, 64, 64)])
def test_fill_arbitrary_grids(oracle_mod, monkeypatch, dims):
    """Random sparse grids (not SDFs): ragged sizes, lines of length 1, runs that start and end unset; rows wider
    than one word of the blank map (1024 cells), lines longer than one 32-row block of it, and densities so low
    that the y and z walks fill whole blank segments (the map of the next sweep must follow)."""
    nx, ny, nz = dims
    rng = np.random.default_rng(nx * 1000 + ny * 10 + nz)
    d = np.full((nz, ny, nx), np.inf, dtype=np.float32)
    for density in (0.0002, 0.002, 0.08, 0.5):
        d[:] = np.inf
        sel = rng.random(d.shape) < density
        d[sel] = rng.standard_normal(int(sel.sum())).astype(np.float32)
        ref = oracle_mod.fill_interior(d, 0.75)
        assert np.array_equal(_gpu_fill(d, 0.75), ref)
        monkeypatch.setenv("SDF_FILLINT_PLAIN", "1")              # every walk reads every cell: same result
        assert np.array_equal(_gpu_fill(d, 0.75), ref)
        monkeypatch.delenv("SDF_FILLINT_PLAIN")


def test_fill_full_size_c3(oracle_mod):
    from paper_1903_00353_b200 import binding as B
    w = f32_grid(W.config("C3"))
    m, d, t = B.compute_workload(w)
    ref = oracle_mod.fill_interior(d.cpu().numpy(), w.band)
    B.sdf_fill_interior(d, w.band)
    torch.cuda.synchronize()
    assert np.array_equal(d.cpu().numpy(), ref)


def test_fill_rejects_bad_arguments():
    from paper_1903_00353_b200 import binding as B
    d = torch.zeros((4, 4, 4), dtype=torch.float32, device="cuda")
    with pytest.raises(B.SdfError) as e:
        B.sdf_fill_interior(d, -1.0)
    assert e.value.status == B.SDF_EINVAL

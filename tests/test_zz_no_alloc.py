"""sdf_fill_interior_static: the entry point that allocates nothing (static 8 MiB device scratch, include/sdf.h).

Collected last on purpose (the suite runs with pytest -x): its output must equal sdf_fill_interior's, bit for bit --
the tolerance tests/test_gpu_fill.py uses for the interior fill -- on calls in a row that share the scratch array, on
grids of different shapes so that the second call meets the first one's stale maps."""
import numpy as np
import pytest
import torch

from paper_1903_00353_b200 import workloads as W
from gpu_util import f32_grid

pytestmark = pytest.mark.gpu


def _random_grid(dims, density, seed):
    nx, ny, nz = dims
    rng = np.random.default_rng(seed)
    d = np.full((nz, ny, nx), np.inf, dtype=np.float32)
    sel = rng.random(d.shape) < density
    d[sel] = rng.standard_normal(int(sel.sum())).astype(np.float32)
    return d


def test_static_fill_equals_pool_fill_two_calls_in_a_row():
    from paper_1903_00353_b200 import binding as B
    # call 1: a real narrow band (C2 at half size: 128^3, one map word per row)
    w = f32_grid(W.config("C2", 0.5))
    m, d, t = B.compute_workload(w)
    ref1 = B.sdf_fill_interior(d.clone(), w.band)
    got1 = B.sdf_fill_interior_static(d.clone(), w.band)
    # call 2, straight after, another shape (rows wider than one map word, ragged sizes) and no SDF at all: the maps
    # of call 1 are still in the array
    d2 = torch.from_numpy(_random_grid((1100, 37, 29), 0.002, 7)).cuda()
    got2 = B.sdf_fill_interior_static(d2.clone(), 0.75)
    ref2 = B.sdf_fill_interior(d2.clone(), 0.75)
    # call 3: the first grid again after the other one
    got3 = B.sdf_fill_interior_static(d.clone(), w.band)
    torch.cuda.synchronize()
    assert torch.equal(got1, ref1)
    assert torch.equal(got2, ref2)
    assert torch.equal(got3, ref1)
    filled = torch.isfinite(got1) & ~torch.isfinite(d)
    assert int(filled.sum()) > 0 and bool(torch.all(got1[filled] == -np.float32(w.band)))
    m.destroy()


@pytest.mark.parametrize("dims,density", [((37, 29, 43), 0.08), ((2100, 3, 35), 0.0002), ((96, 64, 64), 0.5), ((5, 2, 290), 0.002)])
def test_static_fill_arbitrary_grids(dims, density):
    from paper_1903_00353_b200 import binding as B
    d = torch.from_numpy(_random_grid(dims, density, sum(dims))).cuda()
    ref = B.sdf_fill_interior(d.clone(), 0.5)
    for _ in range(2):
        got = B.sdf_fill_interior_static(d.clone(), 0.5)
        torch.cuda.synchronize()
        assert torch.equal(got, ref)


def test_static_fill_allocates_nothing_and_rejects_large_grids():
    from paper_1903_00353_b200 import binding as B
    d = torch.from_numpy(_random_grid((256, 64, 64), 0.01, 3)).cuda()
    B.sdf_fill_interior_static(d.clone(), 0.5)             # set-up call: the symbol's address is looked up here
    torch.cuda.synchronize()
    work = d.clone()
    free0, _ = torch.cuda.mem_get_info()
    B.sdf_fill_interior_static(work, 0.5)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0                                   # nothing taken from the driver (a pool trimming itself meanwhile may return some)
    # the largest grid that fits: ny * nz * ceil(nx / 1024) = 2^20 map words; one row more does not
    fits = torch.full((1024, 1024, 32), float("inf"), dtype=torch.float32, device="cuda")
    fits[500, 500, 7] = -1.0
    B.sdf_fill_interior_static(fits, 0.5)
    torch.cuda.synchronize()
    big = torch.full((1024, 1025, 32), float("inf"), dtype=torch.float32, device="cuda")
    with pytest.raises(B.SdfError) as e:
        B.sdf_fill_interior_static(big, 0.5)
    assert e.value.status == B.SDF_ETOOBIG
    assert "static scratch" in str(e.value) or "too large" in str(e.value)
    torch.cuda.synchronize()
    assert bool(torch.all(torch.isinf(big)))                # refused before anything was launched

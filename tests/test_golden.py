"""Hand-derived closed-form values (tests/golden/*.txt, eq. 1) against the oracle
(-m "not gpu") and, independently of the oracle, against the CUDA path (-m gpu).

The rows are cell centres of the grid origin = -2, h = 1/4, 17^3, so the same fixture pins the
arbitrary-point query, the narrow-band grid routine and sdf_compute."""
import os

import numpy as np
import pytest

from paper_1903_00353_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
ORIGIN, H, N, BAND = (-2.0, -2.0, -2.0), 0.25, 17, 3.0


def _rows(name):
    pts, d, kind = [], [], []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#")[0].split()
            if line:
                pts.append([float(v) for v in line[:3]])
                d.append(float(line[3]))
                kind.append(line[4])
    return np.array(pts), np.array(d), kind


def _octahedron_soup():
    tris = []
    for sx in (1, -1):
        for sy in (1, -1):
            for sz in (1, -1):
                a, b, c = (sx, 0, 0), (0, sy, 0), (0, 0, sz)
                tris.append((a, b, c) if sx * sy * sz > 0 else (a, c, b))       # outward
    return np.array(tris, dtype=np.float32)


def _soup(name):
    if name == "unit_cube.txt":
        v, t = W.box_mesh(half=(0.5, 0.5, 0.5))
        return W.soup_from_indexed(v, t, np.random.default_rng(5))
    return _octahedron_soup()[np.random.default_rng(6).permutation(8)]


def _cells(pts):
    ijk = np.rint((pts - np.array(ORIGIN)) / H).astype(int)
    assert np.array_equal(np.array(ORIGIN) + ijk * H, pts) and ijk.min() >= 0 and ijk.max() < N
    return ijk


@pytest.mark.parametrize("name", ["unit_cube.txt", "octahedron.txt"])
def test_oracle_against_golden(oracle_mod, name):
    pts, d, kind = _rows(name)
    assert len(d) >= 15 and {"I", "F", "E", "V"} <= set(kind)
    m = oracle_mod.Mesh(_soup(name))
    dq, _ = m.query(pts)
    assert np.max(np.abs(dq - d)) < 1e-15 * 8
    nz = d != 0.0
    assert np.array_equal(np.sign(dq[nz]), np.sign(d[nz]))
    dist, tri = m.sdf(ORIGIN, H, (N, N, N), BAND)
    i, j, k = _cells(pts).T
    got = dist[k, j, i].astype(np.float64)
    assert np.all(tri[k, j, i] >= 0)
    assert np.max(np.abs(got - d)) <= 2.0 ** -24 * BAND                 # only the fp32 rounding of the output
    assert np.array_equal(np.sign(got[nz]), np.sign(d[nz]))


@pytest.mark.gpu
@pytest.mark.parametrize("name", ["unit_cube.txt", "octahedron.txt"])
def test_cuda_against_golden(name):
    import torch
    from paper_1903_00353_b200 import binding as B
    pts, d, kind = _rows(name)
    m = B.sdf_create(np.ascontiguousarray(_soup(name)))
    dist, tri = B.sdf_compute(m, ORIGIN, H, (N, N, N), BAND)
    torch.cuda.synchronize()
    dist, tri = dist.cpu().numpy(), tri.cpu().numpy()
    i, j, k = _cells(pts).T
    got = dist[k, j, i].astype(np.float64)
    assert np.all(tri[k, j, i] >= 0) and np.all(tri[k, j, i] < (12 if name == "unit_cube.txt" else 8))
    diag = H * N * np.sqrt(3.0)
    assert np.max(np.abs(got - d)) <= 1e-5 * H + 1e-6 * diag             # north_star's distance clause
    nz = d != 0.0
    assert np.array_equal(np.sign(got[nz]), np.sign(d[nz]))
    B.sdf_destroy(m)

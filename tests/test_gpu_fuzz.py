"""Seeded fuzz of the CUDA path against the oracle (-m gpu): random unit meshes (spheres, tori, boxes thinner
than a cell, cavities, monkey saddles, ruffs, leaning spikes, tetrahedra, cube fans), randomly rotated, scaled
and shifted, on random ragged grids (5..150 cells per axis, spacing and origin not exact in binary) with random
bands (0.6..12 cells).  Every case must meet the four north_star clauses, and sdf_fill_interior on its result
must equal the oracle's sweeps bit for bit.  (10,800 such cases were run once with zero failures, also under the
ablation switches, and 11,000 more with multi-body meshes, bands up to 80 cells, grids that only partly meet the
mesh and the closest-point call; the suite keeps 700 of them.  Round 2: 62,000 more with new seeds, through sdf_create +
sdf_compute and through sdf_transform, a fifth of them lattice-aligned (test_fuzz_lattice_aligned_meshes), and 756 medium-size
ones -- random windows of C2..C5 at 130,000 to 370,000 triangles, ~1e9 band cells -- which found the five near-surface sign
errors of test_sign_of_a_cell_within_fp32_noise_of_the_surface; after that fix 60,800 small and 1,011 medium cases, 83,650 small
ones under SDF_SCHEDULER=serial | dynamic, SDF_BUILDER=tile and SDF_SMOOTH_SIN=0, and 2,184 through the closest-point, z-slab and
host-output calls: none.)"""
import numpy as np
import pytest
import torch

from paper_1903_00353_b200 import workloads as W
from gpu_util import f32_grid
from helpers import compare_to_oracle

pytestmark = pytest.mark.gpu

KEYS = ("bad_sentinel", "bad_id_range", "bad_set", "bad_dist", "bad_sign", "bad_id")

MAKERS = [
    lambda r: W.icosphere_mesh(int(r.integers(0, 4)), float(r.uniform(0.2, 0.8))),
    lambda r: W.torus_mesh(float(r.uniform(0.4, 0.6)), float(r.uniform(0.08, 0.3)), int(r.integers(6, 60)), int(r.integers(4, 30))),
    lambda r: W.box_mesh(tuple(r.uniform(0.01, 0.7, 3))),
    lambda r: W.box_with_cavity_mesh(),
    lambda r: W.monkey_saddle_mesh(nfan=int(r.integers(5, 10)), order=int(r.integers(2, 4)), amp=float(r.uniform(0.1, 0.45))),
    lambda r: W.ruff_mesh(nfan=int(r.integers(5, 12)), rise=float(r.uniform(0.02, 0.2)), fold=float(r.uniform(0.2, 0.6))),
    lambda r: W.spike_mesh(nfan=int(r.integers(3, 9)), lean=float(r.uniform(0.0, 1.4)), height=float(r.uniform(0.15, 0.6))),
    lambda r: W.tetrahedron_mesh(float(r.uniform(0.1, 0.7))),
    lambda r: W.cube_fan_mesh((int(r.integers(0, 4)), int(r.integers(0, 6)), int(r.integers(0, 8)))),
    lambda r: W.multibody_mesh(r, counts=(int(r.integers(1, 6)), int(r.integers(1, 6)), int(r.integers(0, 4)), int(r.integers(0, 3))),
                               lattice=(4, 2, 2), pitch=0.5, ico_subdiv=int(r.integers(0, 3)),
                               torus_res=(int(r.integers(6, 24)), int(r.integers(4, 12)))),
]


def _case(r, wide=False):
    v, t = MAKERS[int(r.integers(0, len(MAKERS)))](r)
    if r.random() < 0.7:
        v = v @ W.random_rotation(r).T
    v = v * float(r.uniform(0.5, 1.3)) + r.uniform(-0.15, 0.15, 3)
    soup = W.soup_from_indexed(v, t, r)
    if wide:        # small grids (down to one cell per axis), bands of 0.05 .. 80 cells, grids that only partly meet the mesh
        dims = tuple(int(x) for x in r.integers(1, 48, 3))
        h = float(r.uniform(1.0, 4.0) / max(max(dims), 8))
        origin = tuple(float(x) for x in (-0.5 * np.array(dims) * h + r.uniform(-0.9, 0.9, 3)))
        return f32_grid(W.Workload("fuzz", soup, origin, h, dims, float(r.uniform(0.05, 80.0)) * h))
    dims = tuple(int(x) for x in r.integers(5, 150, 3))
    h = float(r.uniform(1.6, 2.6) / max(dims))
    origin = tuple(float(x) for x in (-0.5 * np.array(dims) * h + r.uniform(-0.2, 0.2, 3)))
    return f32_grid(W.Workload("fuzz", soup, origin, h, dims, float(r.uniform(0.6, 12.0)) * h))


@pytest.mark.parametrize("seed", [101, 102, 103, 104])
def test_fuzz_parity_and_fill(oracle_mod, seed):
    from paper_1903_00353_b200 import binding as B
    populated = 0
    for c in range(100):
        w = _case(np.random.default_rng(seed * 100003 + c))
        om = oracle_mod.Mesh(w.soup)
        d_ref, t_ref = om.sdf(w.origin, w.h, w.dims, w.band)
        m = B.sdf_create(np.ascontiguousarray(w.soup))
        d, tr = B.sdf_compute(m, w.origin, w.h, w.dims, w.band)
        d_np = d.cpu().numpy()
        res = compare_to_oracle(d_np, tr.cpu().numpy(), d_ref, t_ref, w, om)
        assert res["ok"] and all(res[k] == 0 for k in KEYS), (seed, c, w.dims, w.band / w.h, {k: res[k] for k in KEYS})
        populated += res["populated_gpu"]
        B.sdf_fill_interior(d, w.band)
        torch.cuda.synchronize()
        assert np.array_equal(d.cpu().numpy(), oracle_mod.fill_interior(d_np, w.band)), (seed, c, w.dims)
        B.sdf_destroy(m)
    assert populated > 100000


def _aligned_case(r):
    """Vertices and cell centres on a common power-of-two lattice (spheres whose axis vertices, boxes and cube fans whose
    faces and edges pass through cell centres): many exactly-zero distances and exact ties between features."""
    mk = [lambda: W.icosphere_mesh(int(r.integers(0, 4)), 1.0), lambda: W.box_mesh((0.5, 0.25, 0.75)), lambda: W.tetrahedron_mesh(1.0),
          lambda: W.cube_fan_mesh((int(r.integers(0, 3)), int(r.integers(0, 3)), int(r.integers(0, 3))))]
    v, t = mk[int(r.integers(0, len(mk)))]()
    nn = int(r.integers(16, 64))
    h = 2.0 ** -int(r.integers(3, 7))
    radius = int(r.integers(2, nn // 3 + 1)) * h
    centre = np.array([int(x) * h for x in r.integers(nn // 3, 2 * nn // 3, 3)])
    soup = W.soup_from_indexed(v * radius + centre, t, r)
    return f32_grid(W.Workload("aligned", soup, (0.0, 0.0, 0.0), h, (nn, nn, nn), float(r.integers(1, 5)) * h))


def test_fuzz_lattice_aligned_meshes(oracle_mod):
    """Cell centres on vertices, edges and faces: the exact distance is 0 there.  The library reports +0 (DESIGN.md sec.7 (iii));
    the oracle +0 or +-1e-16 (its fp64 noise), which clause 3 of the harness waives.  1,100 of 12,400 such cases differed in
    exactly that way before the waiver, none in any other way; the suite keeps 150."""
    from paper_1903_00353_b200 import binding as B
    zeros = 0
    for c in range(150):
        w = _aligned_case(np.random.default_rng(31 * 100003 + c))
        om = oracle_mod.Mesh(w.soup)
        d_ref, t_ref = om.sdf(w.origin, w.h, w.dims, w.band)
        m, d, tr = B.sdf_transform(torch.from_numpy(np.ascontiguousarray(w.soup)).cuda(), w.origin, w.h, w.dims, w.band)
        d_np = d.cpu().numpy()
        res = compare_to_oracle(d_np, tr.cpu().numpy(), d_ref, t_ref, w, om)
        assert res["ok"] and all(res[k] == 0 for k in KEYS), (c, w.dims, w.band / w.h, {k: res[k] for k in KEYS})
        z = d_np == 0
        zeros += int(z.sum())
        assert not np.signbit(d_np[z]).any()                  # a zero is +0
        assert np.all(np.abs(d_ref[z]) <= 1e-12 * w.diag)       # ... and only where the oracle's distance is zero too
        # (the converse holds to fp32 resolution only: on a coplanar patch a cell can lie 1e-9 outside the triangle whose
        # fp32 candidate won and inside its neighbour -- the sign pass re-decides on the winning triangle)
        on = np.abs(d_ref) <= 1e-12 * w.diag
        assert np.all(np.abs(d_np[on]) <= 1e-7 * w.diag) and int(z[on].sum()) >= 0.97 * int(on.sum())
        m.destroy()
    assert zeros > 1000


@pytest.mark.parametrize("seed", [201, 202])
def test_fuzz_wide_bands_partial_overlap_closest_points(oracle_mod, seed):
    from paper_1903_00353_b200 import binding as B
    populated = 0
    for c in range(150):
        w = _case(np.random.default_rng(seed * 100003 + c), wide=True)
        om = oracle_mod.Mesh(w.soup)
        d_ref, t_ref = om.sdf(w.origin, w.h, w.dims, w.band)
        m = B.sdf_create(np.ascontiguousarray(w.soup))
        d, tr = B.sdf_compute(m, w.origin, w.h, w.dims, w.band)
        t_np = tr.cpu().numpy()
        res = compare_to_oracle(d.cpu().numpy(), t_np, d_ref, t_ref, w, om)
        assert res["ok"] and all(res[k] == 0 for k in KEYS), (seed, c, w.dims, w.band / w.h, {k: res[k] for k in KEYS})
        populated += res["populated_gpu"]
        # closest points on the GPU's own ids against the oracle's routine on the same ids
        cp = B.sdf_closest_points(m, w.origin, w.h, w.dims, tr).cpu().numpy()
        ref = om.closest_points(w.origin, w.h, w.dims, t_np)
        pop = t_np >= 0
        assert np.all(np.isposinf(cp[~pop]))
        if pop.any():
            assert np.max(np.abs(cp[pop].astype(np.float64) - ref[pop])) <= 1e-5 * w.h + 1e-6 * w.diag, (seed, c)
        B.sdf_destroy(m)
    assert populated > 100000


def test_fuzz_defective_input_statuses(oracle_mod):
    """One random defect per mesh (hole, flipped triangle, duplicated triangle, repeated corner, NaN / Inf, a corner
    moved by one ulp, a collapsed triangle -- or a harmless corner rotation): sdf_create must return the status the
    oracle returns for the same soup (1,500 such cases were run once: no mismatch)."""
    from paper_1903_00353_b200 import binding as B
    seen = set()
    for c in range(300):
        r = np.random.default_rng(7919 * 3 + c)
        v, t = MAKERS[int(r.integers(0, len(MAKERS)))](r)
        soup = W.soup_from_indexed(v, t, r).copy()
        n = soup.shape[0]
        kind, k = int(r.integers(0, 8)), int(r.integers(0, n))
        if kind == 0:
            soup = np.delete(soup, r.choice(n, size=int(r.integers(1, 4)), replace=False), axis=0)
        elif kind == 1:
            soup[k] = soup[k][::-1].copy()
        elif kind == 2:
            soup = np.concatenate([soup, soup[k:k + 1]])
        elif kind == 3:
            soup[k, 1] = soup[k, 0]
        elif kind == 4:
            soup[k, int(r.integers(0, 3)), int(r.integers(0, 3))] = [np.nan, np.inf, -np.inf][int(r.integers(0, 3))]
        elif kind == 5:
            soup[k, 0, 0] = np.nextafter(soup[k, 0, 0], np.float32(9))
        elif kind == 6:
            soup[k] = soup[k][[1, 2, 0]]
        else:
            soup[k, 2] = (soup[k, 0] + soup[k, 1]) * np.float32(0.5)
        soup = np.ascontiguousarray(soup, dtype=np.float32)
        so = sg = 0
        try:
            oracle_mod.Mesh(soup)
        except oracle_mod.OracleError as e:
            so = e.status
        try:
            B.sdf_destroy(B.sdf_create(soup))
        except B.SdfError as e:
            sg = e.status
        assert so == sg, (c, kind, so, sg)
        seen.add((kind, sg))
    assert {s for _, s in seen} >= {0, 1, 2, 3, 4}


@pytest.mark.parametrize("name,scale", [("C2", 1.0), ("C3", 0.5)])
def test_mass_defects_stay_in_bounds(oracle_mod, name, scale):
    """Many defects at once (features.cu edge records): a soup whose every second triangle is flipped, and
    one whose corners are all sorted, have far more than 3F/2 forward half-edges -- the edge-record table holds 3F/2.
    Both calls must return the oracle's status, and a valid mesh built right afterwards must still be bit-identical
    to one built before (nothing was scribbled over)."""
    from paper_1903_00353_b200 import binding as B
    w = f32_grid(W.config(name, scale) if scale < 1.0 else W.config(name))
    good = np.ascontiguousarray(w.soup)
    m0, d0, t0 = B.compute_workload(w)
    torch.cuda.synchronize()
    r = np.random.default_rng(4242)
    variants = []
    s = good.copy(); s[::2] = s[::2, ::-1]; variants.append(s)                       # every second triangle flipped
    s = good.copy(); idx = r.random(len(s)) < 0.3; s[idx] = s[idx][:, ::-1]; variants.append(s)   # 30 % flipped
    s = good.copy()                                                                # corners sorted lexicographically
    for i in range(len(s)):
        s[i] = s[i][np.lexsort((s[i][:, 2], s[i][:, 1], s[i][:, 0]))]
    variants.append(s)
    s = np.delete(good, r.choice(len(good), size=len(good) // 3, replace=False), axis=0); variants.append(s)   # a third missing
    for vi, s in enumerate(variants):
        s = np.ascontiguousarray(s, dtype=np.float32)
        so = 0
        try:
            oracle_mod.Mesh(s)
        except oracle_mod.OracleError as e:
            so = e.status
        assert so in (2, 3)
        for call in ("create", "transform"):
            sg = 0
            try:
                if call == "create":
                    B.sdf_destroy(B.sdf_create(torch.from_numpy(s).cuda()))
                else:
                    B.sdf_transform(torch.from_numpy(s).cuda(), w.origin, w.h, w.dims, w.band)[0].destroy()
            except B.SdfError as e:
                sg = e.status
            assert sg == so, (vi, call, so, sg)
        m1, d1, t1 = B.compute_workload(w)
        torch.cuda.synchronize()
        assert torch.equal(t0, t1) and torch.equal(d0.view(torch.int32), d1.view(torch.int32)), vi
        m1.destroy()
    m0.destroy()


def test_many_non_finite_triangles_are_rejected_quickly():
    """ADVICE r1 (features.cu first crossing): a soup full of Inf / NaN corners is flagged by the ingest kernel, but
    sdf_transform's hoisted brick marking still sees it -- a non-finite box must not turn into a walk over every brick
    of the grid per triangle.  SDF_EINVAL, in milliseconds, and a valid mesh afterwards is untouched."""
    import time
    from paper_1903_00353_b200 import binding as B
    w = f32_grid(W.config("C2"))
    good = np.ascontiguousarray(w.soup)
    m0, d0, t0 = B.compute_workload(w)
    torch.cuda.synchronize()
    r = np.random.default_rng(99)
    for bad_value in (np.inf, -np.inf, np.nan):
        s = good.copy()
        hit = r.random(len(s)) < 0.5
        s[hit, r.integers(0, 3, hit.sum()), r.integers(0, 3, hit.sum())] = bad_value
        t_start = time.perf_counter()
        with pytest.raises(B.SdfError) as e:
            B.sdf_transform(torch.from_numpy(s).cuda(), w.origin, w.h, w.dims, w.band)
        torch.cuda.synchronize()
        assert e.value.status == B.SDF_EINVAL
        assert time.perf_counter() - t_start < 2.0
    m1, d1, t1 = B.compute_workload(w)
    torch.cuda.synchronize()
    assert torch.equal(t0, t1) and torch.equal(d0.view(torch.int32), d1.view(torch.int32))
    m0.destroy(); m1.destroy()


@pytest.mark.parametrize("seed", [11, 12])
def test_fuzz_medium_meshes_random_windows(oracle_mod, seed):
    """Meshes large enough for the Morton ordering of the soup (>= 131,072 triangles) and the class-interleaved evaluate
    order: C4 and C5 reduced to 150,000-350,000 triangles (and C2, C3 whole), on random windows of their grids (ragged sizes, windows that
    stick out of the mesh's box, bands of 0.3 to 30 cells), through sdf_transform and through the two calls; the band-sparse
    output must hold the same cells.  (2,229 such cases were run on the round's final build: no violation.)"""
    import dataclasses
    import types
    from paper_1903_00353_b200 import binding as B
    r = np.random.default_rng(seed)
    compared = 0
    for c in range(5):
        name = ["C4", "C5", "C4", "C3", "C2"][c]
        scale = {"C4": r.uniform(0.19, 0.28), "C5": r.uniform(0.35, 0.5), "C3": 1.0, "C2": 1.0}[name]
        w0 = W.config(name, float(scale)) if scale < 1.0 else W.config(name)
        dims = w0.dims
        size = tuple(int(r.integers(max(8, d // 3), d + 1)) for d in dims)
        lo = tuple(int(r.integers(-s // 3, d - s + 1 + s // 3)) for d, s in zip(dims, size))
        band = float([r.uniform(0.3, 1.0), r.uniform(1.0, 5.0), r.uniform(5.0, 30.0)][int(r.integers(0, 3))])
        w = f32_grid(dataclasses.replace(w0.crop(lo, size), band=band * w0.h))
        om = oracle_mod.Mesh(w.soup)
        d_ref, t_ref = om.sdf(w.origin, w.h, w.dims, w.band)
        soup = torch.from_numpy(np.ascontiguousarray(w.soup)).cuda()
        if c % 2:
            m, d, tr = B.sdf_transform(soup, w.origin, w.h, w.dims, w.band)
        else:
            m = B.sdf_create(soup)
            d, tr = B.sdf_compute(m, w.origin, w.h, w.dims, w.band)
        # the tolerance is the whole grid's: a window may sit far from the origin
        cw = types.SimpleNamespace(h=w.h, band=w.band, diag=max(w.diag, w0.diag), ntri=w.ntri, dims=w.dims, origin=w.origin)
        res = compare_to_oracle(d.cpu().numpy(), tr.cpu().numpy(), d_ref, t_ref, cw, om)
        assert res["ok"] and all(res[k] == 0 for k in KEYS), (seed, c, name, lo, size, band, {k: res[k] for k in KEYS})
        compared += res["populated_ref"]
        nb, ids, sd, st_ = B.sdf_compute_sparse(m, w.origin, w.h, w.dims, w.band)
        assert int(torch.isfinite(sd[:nb]).sum()) == int(torch.isfinite(d).sum())
        m.destroy()
    assert compared > 100000

"""GPU parity tests (run with -m gpu on the B200 box): the CUDA path, called through the
C ABI, against the CPU oracle on the same seeded inputs.

Acceptance = the four clauses of BASELINE.json's north_star (helpers.compare_to_oracle):
populated set identical except within 1e-5*h of the band edge; |d_gpu - d_oracle| <=
1e-5*h + 1e-6*diag; signs exact; ids bit-exact except where the two candidates' distances
agree within that tolerance.
"""
import numpy as np
import pytest

from paper_1903_00353_b200 import workloads as W
from gpu_util import check_parity, f32_grid, run_gpu

pytestmark = pytest.mark.gpu


def _assert_ok(res):
    keys = ("bad_sentinel", "bad_id_range", "bad_set", "bad_dist", "bad_sign", "bad_id")
    assert res["ok"], {k: res[k] for k in res if k != "stats"}
    assert all(res[k] == 0 for k in keys)
    assert res["populated_gpu"] > 0


def _small(verts_tris, seed, n=40, lo=-1.0, hi=1.0, band_cells=3):
    v, t = verts_tris
    rng = np.random.default_rng(seed)
    soup = W.soup_from_indexed(v, t, rng)
    origin, h, dims = W.grid_over((lo,) * 3, (hi,) * 3, (n,) * 3)
    return W.Workload("small", soup, origin, h, dims, band_cells * h)


def test_c1_box_full(oracle_mod):
    w = W.config("C1")
    res = check_parity(w, oracle_mod)
    _assert_ok(res)
    assert res["populated_gpu"] == 18991
    s = res["stats"]
    assert (s["F"], s["V"], s["E"]) == (12, 8, 18)
    assert (s["edges_convex"], s["edges_concave"], s["edges_flat"]) == (12, 0, 6)
    assert s["verts_pos_only"] == 8


@pytest.mark.parametrize("name,scale", [("C2", 0.25), ("C2", 0.5), ("C3", 0.25), ("C4", 0.06), ("C5", 0.02)])
def test_configs_reduced(oracle_mod, name, scale):
    """Reduced variants of C2..C5: same structure, sizes the oracle finishes in seconds,
    several bricks / tiles and ragged tails."""
    w = W.config(name, scale)
    res = check_parity(w, oracle_mod)
    _assert_ok(res)
    s = res["stats"]
    assert s["V"] == w.meta["V"] and s["E"] == w.meta["E"]


@pytest.mark.parametrize("maker,seed,band", [
    (lambda: W.tetrahedron_mesh(0.5), 11, 3),
    (lambda: W.cube_fan_mesh((0, 2, 5)), 12, 3),
    (lambda: W.box_with_cavity_mesh(), 13, 4),
    (lambda: W.monkey_saddle_mesh(), 14, 5),
    (lambda: W.monkey_saddle_mesh(nfan=8, order=2, amp=0.4), 15, 5),
    (lambda: W.ruff_mesh(), 16, 5),
    (lambda: W.spike_mesh(), 17, 5),
    (lambda: W.icosphere_mesh(2, 0.6), 18, 6),
    (lambda: W.torus_mesh(0.55, 0.25, 24, 12), 19, 4),
    (lambda: W.box_mesh((0.6, 0.5, 0.02)), 20, 4),        # plate thinner than the band
    (lambda: W.spike_mesh(lean=1.2, height=0.3), 21, 5),  # two ruff vertices (cos_cone <= 0): hemispheres
])
def test_unit_meshes(oracle_mod, maker, seed, band):
    """Convex / concave / saddle / ruff / pathological vertices, thin plate."""
    w = _small(maker(), seed, n=44, band_cells=band)
    res = check_parity(w, oracle_mod)
    _assert_ok(res)


def test_ragged_grid_and_offsets(oracle_mod):
    """Non-cubic dims that are not multiples of the brick (8) or of the vector width (4),
    a grid that only partly overlaps the mesh, non power-of-two spacing."""
    v, t = W.icosphere_mesh(2, 0.6)
    soup = W.soup_from_indexed(v, t, np.random.default_rng(5))
    w = W.Workload("ragged", soup, (-0.93, -0.41, -0.77), 0.0371, (37, 29, 43), 3.3 * 0.0371)
    _assert_ok(check_parity(w, oracle_mod))
    w2 = W.Workload("ragged4", soup, (-0.93, -0.41, -0.77), 0.0371, (36, 30, 41), 2.0 * 0.0371)
    _assert_ok(check_parity(w2, oracle_mod))


def _rotated(vt, seed):
    v, t = vt
    return v @ W.random_rotation(np.random.default_rng(seed)).T, t


def _shell(r_out=0.7, r_in=0.45, sub=3):
    """Hollow ball: outer sphere outward-oriented, inner sphere oriented into the void (two
    components, one inside the other)."""
    vo, to = W.icosphere_mesh(sub, r_out)
    vi, ti = W.icosphere_mesh(sub, r_in)
    return np.concatenate([vo, vi], 0), np.concatenate([to, ti[:, ::-1] + vo.shape[0]], 0)


@pytest.mark.parametrize("maker,seed,n,band", [
    (lambda: W.icosphere_mesh(2, 0.5), 31, 64, 20),                      # band >> triangle: big polyhedra only
    (lambda: _rotated(W.box_mesh((0.55, 0.4, 0.3)), 32), 32, 96, 6),     # 12 huge oblique triangles (analytic row clips)
    (lambda: _rotated(W.box_mesh((0.85, 0.004, 0.003)), 33), 33, 80, 4), # needle thinner than a cell in two directions
    (lambda: _shell(), 34, 72, 5),                                       # nested components, concave inner shell
    (lambda: _rotated(W.torus_mesh(0.5, 0.2, 48, 24), 35), 35, 96, 9),   # medium polyhedra (row-flattened path), saddles
])
def test_regimes(oracle_mod, maker, seed, n, band):
    """Band / triangle / cell size ratios the five configs do not span, each exercising another
    path of the scan converter (block-per-polyhedron, flattened rows, analytic clipping)."""
    w = _small(maker(), seed, n=n, band_cells=band)
    res = check_parity(w, oracle_mod)
    _assert_ok(res)


def test_cells_on_the_surface(oracle_mod):
    """Box whose faces, edges and corners pass (to fp32 rounding) through cell centres: distances of
    +-1e-8, zero-area of doubt for the sign carried with a candidate -- those cells must fall back to
    the fp64 pseudonormal decision and agree with the oracle."""
    v, t = W.box_mesh((0.525, 0.325, 0.225))
    soup = W.soup_from_indexed(v, t, np.random.default_rng(21))
    origin, h, dims = W.grid_over((-1.0,) * 3, (1.0,) * 3, (40,) * 3)
    w = W.Workload("onsurf", soup, origin, h, dims, 3 * h)
    res = check_parity(w, oracle_mod)
    _assert_ok(res)
    assert res["stats"]["fp64_rechecks"] > 0


def test_grid_misses_mesh():
    """Degenerate case: the band does not reach the grid -> all sentinels."""
    v, t = W.box_mesh((0.1, 0.1, 0.1))
    soup = W.soup_from_indexed(v, t, None)
    w = f32_grid(W.Workload("miss", soup, (5.0, 5.0, 5.0), 0.1, (16, 12, 9), 0.3))
    m, d, tr, stats = run_gpu(w)
    assert np.all(np.isposinf(d)) and np.all(tr == -1)
    assert stats["band_cells"] == 0 and stats["work_items"] == 0


def test_host_pointer_and_repeat_compute(oracle_mod):
    """sdf_create from a HOST pointer; two sdf_compute calls with different bands on one
    handle; band monotonicity."""
    from paper_1903_00353_b200 import binding as B
    w = f32_grid(W.config("C2", 0.25))
    m = B.sdf_create(w.soup)                       # numpy -> host pointer path
    d1, t1 = B.sdf_compute(m, w.origin, w.h, w.dims, w.band)
    d2, t2 = B.sdf_compute(m, w.origin, w.h, w.dims, 0.5 * w.band)
    d1, t1, d2, t2 = (x.cpu().numpy() for x in (d1, t1, d2, t2))
    inner = np.abs(d1) < 0.5 * w.band * (1 - 1e-5)
    # ids are band-independent; distances too, except that cells near the (new) band edge are
    # re-evaluated in fp64 by the emit pass and may differ in the last fp32 bit
    assert np.array_equal(t2[inner], t1[inner])
    assert np.max(np.abs(d2[inner] - d1[inner])) <= 1e-7
    assert np.mean(d2[inner] == d1[inner]) > 0.98
    outer = ~(np.abs(d1) < 0.5 * w.band * (1 + 1e-5))
    assert np.all(np.isposinf(d2[outer]))
    dh, th = B.sdf_compute_host(m, w.origin, w.h, w.dims, w.band)
    assert np.array_equal(dh.numpy(), d1) and np.array_equal(th.numpy(), t1)


def test_unaligned_outputs_and_user_stream():
    """Output pointers that are only 4-byte aligned take the plain-store fill and the scalar emit;
    a caller's non-default stream; results identical to the aligned default-stream run."""
    import torch
    from paper_1903_00353_b200 import binding as B
    w = f32_grid(W.config("C2", 0.5))
    nx, ny, nz = w.dims
    n = nx * ny * nz
    m = B.sdf_create(w.soup)
    d0, t0 = B.sdf_compute(m, w.origin, w.h, w.dims, w.band)
    torch.cuda.synchronize()
    db = torch.full((n + 3,), 7.0, dtype=torch.float32, device="cuda")
    tb = torch.full((n + 3,), 7, dtype=torch.int32, device="cuda")
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        d1, t1 = B.sdf_compute(m, w.origin, w.h, w.dims, w.band, db[1:n + 1].view(nz, ny, nx), tb[3:n + 3].view(nz, ny, nx),
                               stream=st)
    st.synchronize()
    assert d1.data_ptr() % 16 != 0 and t1.data_ptr() % 16 != 0
    assert torch.equal(d1, d0) and torch.equal(t1, t0)
    # nothing outside the two grids was written
    assert float(db[0]) == 7.0 and float(db[n + 1]) == 7.0 and float(db[n + 2]) == 7.0
    assert int(tb[0]) == 7 and int(tb[1]) == 7 and int(tb[2]) == 7


def test_stl_file_to_grid_file(tmp_path):
    """The paper's outer shell: STL file in, grid file out, through the library's own
    reader and writer; same grids as from the soup in memory."""
    import torch
    from paper_1903_00353_b200 import binding as B
    w = f32_grid(W.config("C2", 0.25))
    B.sdf_write_stl(tmp_path / "m.stl", w.soup, ascii=True)
    soup = B.sdf_read_stl(tmp_path / "m.stl")
    assert np.array_equal(soup, w.soup)
    d0, t0 = B.sdf_compute(B.sdf_create(w.soup), w.origin, w.h, w.dims, w.band)
    d1, t1 = B.sdf_compute(B.sdf_create(soup), w.origin, w.h, w.dims, w.band)
    assert torch.equal(d0, d1) and torch.equal(t0, t1)
    B.sdf_write_grid(tmp_path / "g.bin", d1.cpu().numpy(), t1.cpu().numpy(), w.origin, w.h, w.band)
    raw = open(tmp_path / "g.bin", "rb").read()
    n = d1.numel()
    assert np.array_equal(np.frombuffer(raw[44:44 + 4 * n], dtype=np.float32), d1.cpu().numpy().reshape(-1))


def test_ruff_vertices_hemisphere_and_cone_variant(oracle_mod, monkeypatch):
    """Ruff vertices (an incident normal at 90 degrees or more from the pseudonormal):
    the default extrusion is the hemisphere; SDF_RUFF=cone selects the paper's
    other choice, the cone over the positive-pointing normals ("sufficient in practice",
    PAPER.md:410) -- on these meshes it leaves no gap and evaluates fewer pairs."""
    from paper_1903_00353_b200 import binding as B
    for lean, height, n, band in ((1.2, 0.3, 64, 8), (1.4, 0.25, 96, 12)):
        w = _small(W.spike_mesh(lean=lean, height=height), 19, n=n, band_cells=band)
        res = check_parity(w, oracle_mod)
        _assert_ok(res)
        assert res["stats"]["verts_hemisphere"] == 2
        m = B.sdf_create(w.soup)
        assert np.all(B.sdf_get_table(m, B.TABLE_VERTEX_REC)["cos_cone"][B.sdf_get_table(m, B.TABLE_VERTEX_REC)["info"] & 4 != 0] == 0.0)
        monkeypatch.setenv("SDF_RUFF", "cone")
        res_c = check_parity(w, oracle_mod)
        m = B.sdf_create(w.soup)
        vr = B.sdf_get_table(m, B.TABLE_VERTEX_REC)
        monkeypatch.delenv("SDF_RUFF")
        _assert_ok(res_c)
        assert np.all(vr["cos_cone"][vr["info"] & 4 != 0] > 0.5)
        assert res_c["stats"]["pairs_accepted"] < res["stats"]["pairs_accepted"]


def test_degenerate_shapes_and_grids(oracle_mod):
    """Slivers of aspect 1e6, 1500 tiny tetrahedra (as many vertices as faces), a band of a twentieth
    of a cell, grids of one slice, one row and one cell."""
    rng = np.random.default_rng(7)
    g48 = W.grid_over((-1.0,) * 3, (1.0,) * 3, (48,) * 3)
    v, t = W.icosphere_mesh(2, 0.6)
    nb = t[np.any(t == 0, axis=1)][0]
    other = [x for x in nb if x != 0][0]
    v2 = v.copy()
    v2[0] = v2[other] + (v2[0] - v2[other]) * 1e-6 / np.linalg.norm(v2[0] - v2[other])
    cases = [W.Workload("sliver", W.soup_from_indexed(v2, t, rng), *g48, 4 * g48[1])]
    tv, tt = W.tetrahedron_mesh(0.03)
    vs = [tv @ W.random_rotation(rng).T + rng.uniform(-0.9, 0.9, 3) for _ in range(1500)]
    ts = [tt + 4 * k for k in range(1500)]
    cases.append(W.Workload("tets", W.soup_from_indexed(np.concatenate(vs), np.concatenate(ts), rng),
                            *W.grid_over((-1.0,) * 3, (1.0,) * 3, (96,) * 3), 3 * (2 / 96)))
    ico = W.soup_from_indexed(v, t, rng)
    cases.append(W.Workload("thinband", W.soup_from_indexed(*W.torus_mesh(0.5, 0.2, 24, 12), rng), *g48, 0.05 * g48[1]))
    cases.append(W.Workload("slice_x", ico, (0.013, -1 + 1 / 48, -1 + 1 / 48), 2 / 48, (1, 48, 48), 0.2))
    cases.append(W.Workload("slice_z", ico, (-1 + 1 / 48, -1 + 1 / 48, 0.21), 2 / 48, (48, 48, 1), 0.2))
    cases.append(W.Workload("row", ico, (-1 + 1 / 48, 0.1, 0.05), 2 / 48, (48, 1, 1), 0.2))
    cases.append(W.Workload("cell", ico, (0.55, 0.1, 0.05), 2 / 48, (1, 1, 1), 0.2))
    # crumpled sphere: hundreds of saddle, concave and ruff vertices
    g64 = W.grid_over((-1.0,) * 3, (1.0,) * 3, (64,) * 3)
    v3, t3 = W.icosphere_mesh(3, 0.6)
    cases.append(W.Workload("crumpled", W.soup_from_indexed(v3 * (1 + 0.2 * rng.standard_normal(len(v3)))[:, None], t3, rng),
                            *g64, 6 * g64[1]))
    # funnel: a concave vertex of valence 500
    n = 500
    phi = 2 * np.pi * np.arange(n) / n
    vf = np.concatenate([np.stack([0.6 * np.cos(phi), 0.6 * np.sin(phi), np.zeros(n)], 1), [[0, 0, -0.2]], [[0, 0, -0.6]]])
    tf = np.array([[k, (k + 1) % n, n] for k in range(n)] + [[(k + 1) % n, k, n + 1] for k in range(n)])
    cases.append(W.Workload("funnel", W.soup_from_indexed(vf, tf, rng), *g64, 5 * g64[1]))
    # hourglass: two pyramids apex to apex (a pinched, non-manifold vertex; every edge still manifold)
    def pyramid(base_z, s):
        b = np.array([[-s, -s, base_z], [s, -s, base_z], [s, s, base_z], [-s, s, base_z], [0.0, 0.0, 0.0]])
        tt_ = np.array([[k, (k + 1) % 4, 4] for k in range(4)] + [[0, 2, 1], [0, 3, 2]])
        return b, (tt_ if base_z < 0 else tt_[:, ::-1])
    (va, ta), (vb, tb) = pyramid(-0.6, 0.5), pyramid(0.6, 0.4)
    cases.append(W.Workload("hourglass", W.soup_from_indexed(np.concatenate([va, vb]), np.concatenate([ta, tb + 5]), rng),
                            *g64, 5 * g64[1]))
    # inside-out box: a cavity in an infinite solid (all edges and vertices concave)
    vbx, tbx = W.box_mesh((0.5, 0.4, 0.3))
    cases.append(W.Workload("insideout", W.soup_from_indexed(vbx, tbx[:, ::-1], rng), *g64, 5 * g64[1]))
    # sea urchin: twenty vertices of a small icosphere pulled far out
    vu, tu = W.icosphere_mesh(2, 0.3)
    vu[rng.choice(len(vu), 20, replace=False)] *= 2.8
    cases.append(W.Workload("urchin", W.soup_from_indexed(vu, tu, rng), *g64, 6 * g64[1]))
    for w in cases:
        _assert_ok(check_parity(w, oracle_mod))


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_maximum_grid_dimension(oracle_mod, axis):
    """32767 cells (the largest dimension the 16-bit bounding volumes allow) along one axis, the mesh at
    its far end, coordinates around 1000."""
    v, t = W.icosphere_mesh(2, 0.6)
    h = 2.0 / 64
    dims = [5, 5, 5]
    dims[axis] = 32767
    c = np.zeros(3)
    c[axis] = (32767 - 40) * h
    origin = [-2 * h] * 3
    origin[axis] = 0.0
    w = W.Workload("long", W.soup_from_indexed(v + c, t, np.random.default_rng(axis)), tuple(origin), h, tuple(dims), 3 * h)
    res = check_parity(w, oracle_mod)
    _assert_ok(res)
    assert res["populated_gpu"] == 312


def test_knife_edges(oracle_mod):
    """Edges whose faces fold back onto each other (n1 = -n2): sin(dihedral) vanishes as it does for a
    flat edge, but the edge needs the widest extrusion there is.  A two-triangle "pillow" (zero volume,
    every edge a knife) and a blade (prism with an apex angle of 2.5e-8 rad).  The solids are thinner than
    fp32 can resolve, so the sign is not defined; the populated set and |d| are, and must match."""
    from paper_1903_00353_b200 import binding as B
    tri = np.array([[0.1, 0.05, 0.02], [0.7, 0.1, 0.3], [0.2, 0.6, -0.1]], dtype=np.float32)
    pillow = np.stack([tri, tri[::-1]]).astype(np.float32)
    t_ = 1e-8
    xs = np.array([[-0.4, 0.0], [0.4, t_], [0.4, -t_]])
    v = np.array([[x, y, z] for z in (-0.3, 0.3) for x, y in xs])
    tr = np.array([[0, 2, 1], [3, 4, 5], [0, 1, 4], [0, 4, 3], [1, 2, 5], [1, 5, 4], [2, 0, 3], [2, 3, 5]])
    blade = W.soup_from_indexed(v, tr, np.random.default_rng(1))
    origin, h, dims = W.grid_over((-1.0,) * 3, (1.0,) * 3, (48,) * 3)
    for soup, knives in ((pillow, 3), (blade, 1)):
        w = f32_grid(W.Workload("knife", soup, origin, h, dims, 4 * h))
        om = oracle_mod.Mesh(w.soup)
        d_ref, t_ref = om.sdf(w.origin, w.h, w.dims, w.band)
        m, d, t, stats = run_gpu(w)
        er = B.sdf_get_table(m, B.TABLE_EDGE_REC)
        assert int((er["cls"] == 2).sum()) == knives
        pop = np.isfinite(d)
        assert np.array_equal(pop, np.isfinite(d_ref)) and pop.sum() > 1000
        tol = 1e-5 * w.h + 1e-6 * w.diag
        assert np.max(np.abs(np.abs(d[pop]).astype(np.float64) - np.abs(d_ref[pop]))) <= tol
        assert np.all(t[pop] >= 0) and np.all(t[~pop] == -1)


def test_serial_scheduler_ablation(oracle_mod, monkeypatch):
    """SDF_SCHEDULER=serial (the paper's thread-per-extrusion loop, kept as an ablation)
    meets the same four parity clauses, and agrees with the flattened scan converter to the last
    bit except at cells on a prism's side plane (where the two walks may take the interior or the
    eps-margin expression of the same distance)."""
    import torch
    from paper_1903_00353_b200 import binding as B
    for w in (f32_grid(W.config("C2", 0.5)), f32_grid(_small(W.torus_mesh(0.5, 0.2, 48, 24), 35, n=96, band_cells=9)),
              f32_grid(_small(W.ruff_mesh(), 16, n=44, band_cells=5))):
        m = B.sdf_create(w.soup)
        d0, t0 = B.sdf_compute(m, w.origin, w.h, w.dims, w.band)
        monkeypatch.setenv("SDF_SCHEDULER", "serial")
        _assert_ok(check_parity(w, oracle_mod))
        d1, t1 = B.sdf_compute(m, w.origin, w.h, w.dims, w.band)
        monkeypatch.delenv("SDF_SCHEDULER")
        pop = torch.isfinite(d0)
        assert torch.equal(pop, torch.isfinite(d1))
        assert float((d0[pop] - d1[pop]).abs().max()) <= 1e-7
        assert float((d0[pop] == d1[pop]).float().mean()) > 0.999


@pytest.mark.parametrize("mode", ["dynamic", "dynamic:64"])
def test_dynamic_parallelism_ablation(oracle_mod, monkeypatch, mode):
    """SDF_SCHEDULER=dynamic[:N] (the paper's device-side child grids, one thread per bounding-volume cell,
    PAPER.md:376-380; N = hybrid threshold) meets the same four parity clauses and agrees
    with the flattened scan converter as the serial ablation does."""
    import torch
    from paper_1903_00353_b200 import binding as B
    for w in (f32_grid(W.config("C1")), f32_grid(W.config("C2", 0.5)),
              f32_grid(_small(W.ruff_mesh(), 16, n=44, band_cells=5))):
        m = B.sdf_create(w.soup)
        d0, t0 = B.sdf_compute(m, w.origin, w.h, w.dims, w.band)
        monkeypatch.setenv("SDF_SCHEDULER", mode)
        _assert_ok(check_parity(w, oracle_mod))
        d1, t1 = B.sdf_compute(m, w.origin, w.h, w.dims, w.band)
        monkeypatch.delenv("SDF_SCHEDULER")
        pop = torch.isfinite(d0)
        assert torch.equal(pop, torch.isfinite(d1))
        assert float((d0[pop] - d1[pop]).abs().max()) <= 1e-7
        assert float((d0[pop] == d1[pop]).float().mean()) > 0.999


def test_permutation_invariance():
    """Shuffling the soup permutes ids and leaves distances / signs bit-identical (the packed
    atomicMin is order independent)."""
    from paper_1903_00353_b200 import binding as B
    w = f32_grid(W.config("C3", 0.25))
    perm = np.random.default_rng(3).permutation(w.ntri)
    m1, d1, t1 = B.compute_workload(w)
    import dataclasses
    m2, d2, t2 = B.compute_workload(dataclasses.replace(w, soup=np.ascontiguousarray(w.soup[perm])))
    d1, t1, d2, t2 = (x.cpu().numpy() for x in (d1, t1, d2, t2))
    assert np.array_equal(d1, d2)
    pop = t1 >= 0
    # ids agree after un-permuting except on exact ties (closest point on a shared edge/vertex)
    same = perm[t2[pop]] == t1[pop]
    assert same.mean() > 0.7


def test_error_statuses():
    from paper_1903_00353_b200 import binding as B
    v, t = W.box_mesh()
    soup = W.soup_from_indexed(v, t, None)
    with pytest.raises(B.SdfError) as e:
        B.sdf_create(soup[:-1])                              # a hole
    assert e.value.status == B.SDF_ENOTCLOSED
    flipped = soup.copy()
    flipped[3] = flipped[3][::-1]
    with pytest.raises(B.SdfError) as e:
        B.sdf_create(flipped)
    assert e.value.status == B.SDF_EORIENT
    deg = soup.copy()
    deg[0, 1] = deg[0, 0]
    with pytest.raises(B.SdfError) as e:
        B.sdf_create(deg)
    assert e.value.status in (B.SDF_EDEGENERATE,)
    nan = soup.copy()
    nan[2, 1, 0] = np.nan
    with pytest.raises(B.SdfError) as e:
        B.sdf_create(nan)
    assert e.value.status == B.SDF_EINVAL
    m = B.sdf_create(soup)
    with pytest.raises(B.SdfError) as e:
        B.sdf_compute(m, (0, 0, 0), -1.0, (8, 8, 8), 0.1)
    assert e.value.status == B.SDF_EINVAL
    with pytest.raises(B.SdfError) as e:
        B.sdf_compute(m, (0, 0, 0), 0.01, (8, 8, 8), 2.6)       # band > 250 h
    assert e.value.status == B.SDF_EINVAL


@pytest.mark.parametrize("what,expect_cells", [("cones", 20), ("wedges", 100), ("faces", 1000)])
def test_harness_detects_a_missing_extrusion_class(oracle_mod, monkeypatch, what, expect_cells):
    """SURVEY.md sec.4 / PAPER.md:402, 427: leave one extrusion class out of the scan conversion (SDF_DISABLE) on the
    rotated torus and on a box: the comparison harness must report the coverage gap (distances too large, cells
    missing at the rim of the band) -- never a sign or sentinel problem -- and the same call without the switch passes."""
    ws = [f32_grid(W.config("C3", 0.25)), f32_grid(W.config("C1"))]
    for w in ws:
        _assert_ok(check_parity(w, oracle_mod))
        monkeypatch.setenv("SDF_DISABLE", what)
        res = check_parity(w, oracle_mod)
        monkeypatch.delenv("SDF_DISABLE")
        assert not res["ok"]
        assert res["bad_dist"] + res["bad_set"] >= expect_cells, {k: res[k] for k in res if k != "stats"}
        assert res["bad_sentinel"] == 0 and res["bad_id_range"] == 0
        # a gap only ever makes a distance larger or a cell vanish (never too small)
        assert res["populated_gpu"] <= res["populated_ref"]
        _assert_ok(check_parity(w, oracle_mod))


@pytest.mark.parametrize("name,scale", [("C1", 1.0), ("C2", 0.25), ("C3", 0.25), ("C5", 0.02)])
def test_aabb_candidates_mode_meets_the_four_clauses(oracle_mod, monkeypatch, name, scale):
    """with SDF_AABB_MODE=1 the candidates are the band-expanded triangle boxes (the oracle's
    own loop on the GPU) instead of the characteristic polyhedra: parity must not change, only the pair count."""
    from paper_1903_00353_b200 import binding as B
    import torch
    w = f32_grid(W.config(name, scale) if scale < 1.0 else W.config(name))
    res0 = check_parity(w, oracle_mod)
    _assert_ok(res0)
    m0, d0, t0 = B.compute_workload(w)
    monkeypatch.setenv("SDF_AABB_MODE", "1")
    res1 = check_parity(w, oracle_mod)
    m1, d1, t1 = B.compute_workload(w)
    monkeypatch.delenv("SDF_AABB_MODE")
    _assert_ok(res1)
    assert res1["populated_gpu"] == res0["populated_gpu"]
    assert res1["stats"]["pairs_tested"] > res0["stats"]["pairs_tested"]
    # same cells, same signs, distances within an ulp of the coordinates (polyhedra only cull)
    pop = torch.isfinite(d0)
    assert torch.equal(pop, torch.isfinite(d1)) and torch.equal(torch.signbit(d0[pop]), torch.signbit(d1[pop]))
    assert float((d0[pop] - d1[pop]).abs().max()) <= 2e-7


@pytest.mark.parametrize("name,scale", [("C4", 0.12), ("C2", 0.5), ("C3", 0.25)])
def test_smooth_features_absorbed_by_their_faces(oracle_mod, monkeypatch, name, scale):
    """Edges / vertices whose normals span less than asin(1/32) get no wedge / cone of their own: the incident face
    prisms are widened by reach * sin(angle) and evaluate the clamped triangle distance there (DESIGN.md "smooth
    features").  With the switch off (SDF_SMOOTH_SIN=0) every non-flat feature has its polyhedron as in the paper
    (PAPER.md:352-364).  Both must meet the four clauses; the populated sets, signs and ids-up-to-ties are those of the
    oracle either way, and on a smooth mesh the absorbed variant scan-converts far fewer polyhedra."""
    import torch
    from paper_1903_00353_b200 import binding as B
    w = f32_grid(W.config(name, scale))
    res1 = check_parity(w, oracle_mod)
    _assert_ok(res1)
    m1, d1, t1 = B.compute_workload(w)
    monkeypatch.setenv("SDF_SMOOTH_SIN", "0")
    res0 = check_parity(w, oracle_mod)
    m0, d0, t0 = B.compute_workload(w)
    monkeypatch.delenv("SDF_SMOOTH_SIN")
    _assert_ok(res0)
    s0, s1 = res0["stats"], res1["stats"]
    assert res0["populated_gpu"] == res1["populated_gpu"]
    assert s1["polyhedra"] <= s0["polyhedra"] and s1["edges_flat"] >= s0["edges_flat"] and s1["verts_skipped"] >= s0["verts_skipped"]
    if name == "C4":
        assert s1["polyhedra"] < 0.85 * s0["polyhedra"]         # (at full size the star surface is smooth almost everywhere: 3.9 M of 9.5 M)
    pop = torch.isfinite(d0)
    assert torch.equal(pop, torch.isfinite(d1)) and torch.equal(torch.signbit(d0[pop]), torch.signbit(d1[pop]))
    assert float((d0[pop] - d1[pop]).abs().max()) <= 2e-7       # same distances to an ulp of the coordinates


def test_more_vertices_than_a_closed_surface_can_have(oracle_mod):
    """The per-vertex tables are sized by V <= 3F/2 (every vertex of a closed surface has at least two corners), so
    sdf_create needs no host crossing for the count.  A soup that breaks the bound -- disjoint triangles: V = 3F -- must
    come back SDF_ENOTCLOSED (the oracle's status) without touching memory it does not own, through both builders."""
    import os
    import torch
    from paper_1903_00353_b200 import binding as B
    r = np.random.default_rng(99)
    for F in (7, 300, 5000, 200000):
        base = r.uniform(-0.8, 0.8, (F, 1, 3))
        soup = np.ascontiguousarray((base + r.uniform(-0.01, 0.01, (F, 3, 3))).astype(np.float32))
        if F <= 5000:
            with pytest.raises(oracle_mod.OracleError) as eo:
                oracle_mod.Mesh(soup)
            assert eo.value.status == 2
        for builder in ("", "tile"):
            os.environ["SDF_BUILDER"] = builder
            try:
                with pytest.raises(B.SdfError) as e:
                    B.sdf_create(torch.from_numpy(soup).cuda())
                assert e.value.status == B.SDF_ENOTCLOSED, (F, builder)
            finally:
                del os.environ["SDF_BUILDER"]
    # the library is intact afterwards
    _assert_ok(check_parity(f32_grid(W.config("C1")), oracle_mod))


def test_fp32_peak_microbenchmark():
    """sdf_measure_fp32_peak (the FP32 leg of north_star's roofline): a B200 does 148 SMs x 128 FMA x 2 x 1.965 GHz =
    74.4 TFLOP/s nominally; the FMA loop must land in that neighbourhood (clocks may sit a little lower)."""
    from paper_1903_00353_b200 import binding as B
    tf, sms = B.sdf_measure_fp32_peak()
    assert sms > 0 and 0.5 * sms * 128 * 2 * 1.0e9 / 1e12 < tf < sms * 128 * 2 * 2.3e9 / 1e12, (tf, sms)


@pytest.mark.parametrize("subdiv", [1, 2, 3])
def test_cell_centres_on_vertices_and_edges_of_a_generic_mesh(oracle_mod, subdiv):
    """Cell centres that coincide with vertices (the six axis vertices of an icosphere of radius 16 h centred on a grid
    point) and with points of edges (the midpoints of the octahedral edges, at subdiv >= 1 vertices themselves; at any
    level the x-axis crossings): the exact distance is 0 there, and a zero has no sign.  The faces around them have
    irrational normals, so n . r of an in-plane r is rounding noise: the sign pass must report 0, as the definition
    does, not +-1e-17."""
    n, h = 64, 2.0 ** -5
    v, t = W.icosphere_mesh(subdiv, 16 * h)
    c = np.array([32 * h, 32 * h, 32 * h])
    w = W.Workload("onvertex", W.soup_from_indexed(v + c, t, np.random.default_rng(subdiv)), (0.0, 0.0, 0.0), h, (n, n, n), 3 * h)
    res = check_parity(w, oracle_mod)
    _assert_ok(res)
    om = oracle_mod.Mesh(f32_grid(w).soup)
    d_ref, _ = om.sdf(w.origin, w.h, w.dims, w.band)
    assert int((d_ref == 0).sum()) >= 6
    from paper_1903_00353_b200 import binding as B
    m, d, tr = B.compute_workload(f32_grid(w))
    dz = d.cpu().numpy()
    assert np.array_equal(dz == 0, d_ref == 0)
    assert not np.signbit(dz[dz == 0]).any()
    m.destroy()


def test_sign_of_a_cell_within_fp32_noise_of_the_surface(oracle_mod):
    """Found by a fuzz campaign on medium meshes (756 cases, 5 sign mismatches in ~1e9 band cells): a cell 7e-9 outside the
    surface whose fp32 cell coordinate (half an ulp of |x| ~ 0.5: 3e-8) put it 4e-9 inside one face while the closest point
    lay on the neighbouring face.  A relative test (d <= 1e-5 |x - a|) called the face's sign certain because the cell was
    close to corner a.  Now a distance within two ulps of the grid's largest coordinate is never sign-certain, and the fp64
    sign pass measures the triangles around the winner too."""
    import dataclasses
    import types
    from helpers import compare_to_oracle
    from paper_1903_00353_b200 import binding as B
    w0 = W.config("C4", 0.2561253111963309)
    w = w0.crop((6, 103, 27), (238, 150, 228))
    w = f32_grid(dataclasses.replace(w, band=4.10730308445584 * w.h))
    om = oracle_mod.Mesh(w.soup)
    d_ref, t_ref = om.sdf(w.origin, w.h, w.dims, w.band)
    m, d, tr = B.compute_workload(w)
    cw = types.SimpleNamespace(h=w.h, band=w.band, diag=w0.diag, ntri=w.ntri, dims=w.dims, origin=w.origin)
    res = compare_to_oracle(d.cpu().numpy(), tr.cpu().numpy(), d_ref, t_ref, cw, om)
    _assert_ok(res)
    cell = 6177419                                   # the cell of the campaign: 6.7e-9 outside
    assert d_ref.reshape(-1)[cell] < 0 and abs(d_ref.reshape(-1)[cell]) < 1e-8
    assert d.cpu().numpy().reshape(-1)[cell] < 0
    m.destroy()

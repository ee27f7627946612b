"""Pins for the CPU oracle (run with -m "not gpu").

Each test checks oracle/ against something OTHER than itself: a closed form, a
textbook special case, brute force with an independent formulation, an invariant.
Chosen so that a dropped term, wrong sign/index or transposed operand anywhere in
oracle/sdf_oracle.c fails at least one of them ("What pins the oracle").
"""
import numpy as np
import pytest

from paper_1903_00353_b200 import workloads as W
from helpers import box_sdf, grid_points, brute_unsigned, winding_number, point_triangle_dist


def _small(verts_tris, seed, n=24, lo=-1.0, hi=1.0, band_cells=3):
    v, t = verts_tris
    rng = np.random.default_rng(seed)
    soup = W.soup_from_indexed(v, t, rng)
    origin, h, dims = W.grid_over((lo,) * 3, (hi,) * 3, (n,) * 3)
    return W.Workload("small", soup, origin, h, dims, band_cells * h)


# ----------------------------------------------------------------------------- #
# C1 closed form (eq.1 on a shape with a closed-form SDF)
# ----------------------------------------------------------------------------- #
def test_box_closed_form_all_cells(oracle_mod):
    w = W.config("C1")
    dist, tri = oracle_mod.sdf(w)
    flat = w.soup.reshape(-1, 3).astype(np.float64)
    lo, hi = flat.min(0), flat.max(0)           # the fp32 box IS the box
    pts = grid_points(w.origin, w.h, w.dims)
    exact = box_sdf(pts, lo, hi)
    pop = np.abs(exact) < w.band
    assert np.array_equal(np.isfinite(dist), pop)
    assert np.all(tri[~pop] == -1) and np.all(np.isposinf(dist[~pop]))
    err = np.abs(dist[pop].astype(np.float64) - exact[pop])
    assert err.max() <= 2.0 ** -24 * w.band * 1.01      # only the final fp32 rounding
    assert pop.sum() == 18991                            # B(C1) ~ 1.9e4
    # |d| < band on populated cells (north_star invariant)
    assert np.all(np.abs(dist[pop]) < w.band)


def test_box_closest_triangle_ids(oracle_mod):
    """Each box face is two triangles split by a known diagonal: where the closest point is
    strictly inside one triangle of a face the id must be that triangle."""
    w = W.config("C1")
    dist, tri = oracle_mod.sdf(w)
    pts = grid_points(w.origin, w.h, w.dims).reshape(-1, 3)
    sel = np.nonzero(np.isfinite(dist.reshape(-1)))[0][::7]
    d_b, arg_b = brute_unsigned(pts[sel], w.soup)
    # unique minimiser (margin) -> ids must agree; otherwise distances must agree
    d_all = point_triangle_dist(pts[sel][:, None, :], w.soup[None].astype(np.float64))
    srt = np.sort(d_all, axis=1)
    unique = (srt[:, 1] - srt[:, 0]) > 1e-9
    assert unique.sum() > 500
    assert np.array_equal(tri.reshape(-1)[sel][unique], arg_b[unique])
    assert np.allclose(np.abs(dist.reshape(-1)[sel]), d_b, rtol=0, atol=1e-7)


# ----------------------------------------------------------------------------- #
# point-triangle routine: textbook special cases + dense sampling
# ----------------------------------------------------------------------------- #
def test_point_triangle_special_cases(oracle_mod):
    tri = np.array([[0, 0, 0], [2, 0, 0], [0, 1, 0]], dtype=np.float32)
    pt = oracle_mod.point_triangle
    d, q, r = pt([0.5, 0.25, 0.75], tri)                 # above interior: point-plane n.pc
    assert r == "FACE" and d == pytest.approx(0.75) and np.allclose(q, [0.5, 0.25, 0])
    d, q, r = pt([0.5, 0.25, -0.75], tri)
    assert r == "FACE" and d == pytest.approx(0.75)
    d, q, r = pt([1.0, -2.0, 1.0], tri)                  # beyond edge AB: point-line
    assert r == "E_AB" and d == pytest.approx(np.sqrt(5.0)) and np.allclose(q, [1, 0, 0])
    d, q, r = pt([-3.0, 0.5, 0.0], tri)                  # beyond edge CA
    assert r == "E_CA" and d == pytest.approx(3.0) and np.allclose(q, [0, 0.5, 0])
    d, q, r = pt([2.0, 2.0, 0.0], tri)                   # beyond hypotenuse BC
    exp_q = np.array([2, 0, 0]) + ((np.array([2, 2, 0]) - [2, 0, 0]) @ np.array([-2, 1, 0]) / 5.0) * np.array([-2, 1, 0])
    assert r == "E_BC" and np.allclose(q, exp_q) and d == pytest.approx(np.linalg.norm([2, 2, 0] - exp_q))
    d, q, r = pt([-1.0, -1.0, 1.0], tri)                 # beyond vertex A: point-point
    assert r == "V_A" and d == pytest.approx(np.sqrt(3.0))
    d, q, r = pt([4.0, -1.0, 0.0], tri)
    assert r == "V_B" and d == pytest.approx(np.sqrt(5.0))
    d, q, r = pt([-0.5, 3.0, 2.0], tri)
    assert r == "V_C" and d == pytest.approx(np.sqrt(0.25 + 4 + 4))
    d, q, r = pt([0.25, 0.25, 0.0], tri)                 # on the triangle
    assert d == 0.0


def test_point_triangle_vs_dense_sampling(oracle_mod):
    rng = np.random.default_rng(7)
    n = 300
    u, v = np.meshgrid(np.arange(n + 1) / n, np.arange(n + 1) / n, indexing="ij")
    keep = (u + v) <= 1.0 + 1e-12
    u, v = u[keep], v[keep]
    for trial in range(40):
        tri = rng.normal(size=(3, 3)).astype(np.float32)
        if trial % 4 == 0:                                # slivers too
            tri[2] = tri[1] + (tri[1] - tri[0]) * 0.5 + rng.normal(size=3).astype(np.float32) * 1e-3
        p = rng.normal(size=3) * 1.5
        d, q, r = oracle_mod.point_triangle(p, tri)
        t64 = tri.astype(np.float64)
        samples = t64[0] + u[:, None] * (t64[1] - t64[0]) + v[:, None] * (t64[2] - t64[0])
        ub = np.min(np.linalg.norm(samples - p, axis=1))   # upper bound converging to d
        edge = max(np.linalg.norm(t64[1] - t64[0]), np.linalg.norm(t64[2] - t64[0]), np.linalg.norm(t64[2] - t64[1]))
        assert d <= ub + 1e-12
        assert ub - d <= edge / n                          # sampling resolution
        assert abs(np.linalg.norm(p - q) - d) < 1e-12      # q is at distance d
        assert point_triangle_dist(p, t64) == pytest.approx(d, abs=1e-9)


# ----------------------------------------------------------------------------- #
# sign: brute-force generalised winding numbers on tiny meshes
# ----------------------------------------------------------------------------- #
_TINY = {
    "cube": lambda: W.box_mesh((0.5, 0.5, 0.5)),
    "tet": lambda: W.tetrahedron_mesh(0.5),
    "ico1": lambda: W.icosphere_mesh(1, 0.6),
    "ico2": lambda: W.icosphere_mesh(2, 0.6),
    "torus": lambda: W.torus_mesh(0.55, 0.22, 14, 8),
    "fan": lambda: W.cube_fan_mesh((0, 2, 5), 0.5),
    "cavity": lambda: W.box_with_cavity_mesh(),
    "saddle": lambda: W.monkey_saddle_mesh(),
    "saddle8": lambda: W.monkey_saddle_mesh(8, 0.5, 0.3, -0.5, 2),
    "ruff": lambda: W.ruff_mesh(),
    "spike": lambda: W.spike_mesh(),
    "leanspike": lambda: W.spike_mesh(lean=1.2, height=0.3),    # two ruff vertices: cos_cone <= 0
    "plate": lambda: W.box_mesh((0.6, 0.5, 0.02)),          # thinner than the band
}


@pytest.mark.parametrize("name", sorted(_TINY))
def test_sign_and_distance_vs_brute_force(oracle_mod, name):
    """distance == independent brute force; sign == winding number; populated set ==
    {brute |d| < band}; ids == brute argmin where the minimiser is unique."""
    w = _small(_TINY[name](), seed=11, n=28, band_cells=4)
    m = oracle_mod.Mesh(w.soup)
    dist, tri = m.sdf(w.origin, w.h, w.dims, w.band)
    pts = grid_points(w.origin, w.h, w.dims).reshape(-1, 3)
    d_b, arg_b = brute_unsigned(pts, w.soup)
    pop = d_b < w.band
    edge = np.abs(d_b - w.band) < 1e-9
    got = np.isfinite(dist.reshape(-1))
    assert np.array_equal(got[~edge], pop[~edge])           # every cell with |d|<band populated
    sel = got & pop
    assert np.allclose(np.abs(dist.reshape(-1)[sel]), d_b[sel], rtol=0, atol=2e-7)
    wn = winding_number(pts[sel], w.soup)
    off = d_b[sel] > 1e-6                                    # winding number is singular on the surface
    inside = wn > 0.5
    assert np.all(np.abs(wn[off] - np.round(wn[off])) < 0.2)
    assert np.array_equal(dist.reshape(-1)[sel][off] < 0, inside[off])
    # ids where unique
    d_all = point_triangle_dist(pts[sel][:, None, :], w.soup[None].astype(np.float64))
    srt = np.sort(d_all, axis=1)
    uniq = (srt[:, 1] - srt[:, 0]) > 1e-9
    assert np.array_equal(tri.reshape(-1)[sel][uniq], arg_b[sel][uniq])


def test_query_matches_grid(oracle_mod):
    w = _small(W.icosphere_mesh(2, 0.6), seed=3, n=20, band_cells=3)
    m = oracle_mod.Mesh(w.soup)
    dist, tri = m.sdf(w.origin, w.h, w.dims, w.band)
    pts = grid_points(w.origin, w.h, w.dims).reshape(-1, 3)
    d_q, id_q = m.query(pts)
    pop = np.isfinite(dist.reshape(-1))
    assert np.array_equal(pop, np.abs(d_q) < w.band)
    assert np.array_equal(dist.reshape(-1)[pop], d_q[pop].astype(np.float32))
    assert np.array_equal(tri.reshape(-1)[pop], id_q[pop])
    d_b, _ = brute_unsigned(pts[::5], w.soup)
    assert np.allclose(np.abs(d_q[::5]), d_b, atol=1e-12)


# ----------------------------------------------------------------------------- #
# pseudonormals (eq.8)
# ----------------------------------------------------------------------------- #
def test_angle_weighted_pseudonormal_cube_corner(oracle_mod):
    """Unequal coplanar fans at a cube corner: N_v must stay along (1,1,1) -- the case
    angle weighting exists for; a plain average would be skewed."""
    v, t = W.cube_fan_mesh((0, 2, 5), 0.5)
    soup = W.soup_from_indexed(v, t, np.random.default_rng(5))
    m = oracle_mod.Mesh(soup)
    vid = m.corner_vid()
    corner = np.float32([0.5, 0.5, 0.5])
    hit = np.all(soup == corner, axis=2)
    ids = np.unique(vid[hit])
    assert ids.size == 1
    N = m.vertex_normals()[ids[0]]
    assert np.allclose(N / np.linalg.norm(N), np.ones(3) / np.sqrt(3), atol=1e-7)
    assert np.linalg.norm(N) == pytest.approx(np.sqrt(3) * np.pi / 2, rel=1e-6)   # 3 faces x pi/2
    # plain (unweighted) average of the incident normals would NOT be along (1,1,1)
    fn = m.face_normals()[np.nonzero(hit.any(axis=1))[0]]
    plain = fn.sum(0)
    assert np.abs(plain / np.linalg.norm(plain) - 1 / np.sqrt(3)).max() > 0.05


def test_pseudonormal_discriminant_property(oracle_mod):
    """for points whose closest feature is the vertex, sign(N.(p-v)) tells
    inside from outside.  Checked at the fanned cube corner and a cavity corner."""
    v, t = W.box_with_cavity_mesh()
    soup = W.soup_from_indexed(v, t, np.random.default_rng(2))
    m = oracle_mod.Mesh(soup)
    rng = np.random.default_rng(0)
    # outer corner (+,+,+) of the outer box: points in the octant beyond it are outside
    c = np.array([0.6, 0.6, 0.6])
    p = c + np.abs(rng.normal(size=(50, 3))) * 0.05
    d, _ = m.query(p)
    assert np.all(d > 0) and np.allclose(d, np.linalg.norm(p - c, axis=1))
    # corner of the void: points inside the solid just beyond the void's corner are inside
    ci = np.array([0.05 + 0.25, 0.0 + 0.2, -0.03 + 0.3])
    p = ci + np.abs(rng.normal(size=(50, 3))) * 0.02
    d, _ = m.query(p)
    assert np.all(d < 0) and np.allclose(-d, np.linalg.norm(p - ci.astype(np.float32).astype(np.float64), axis=1), atol=1e-7)


# ----------------------------------------------------------------------------- #
# icosphere sanity: inscribed polyhedron sagitta bound
# ----------------------------------------------------------------------------- #
def test_icosphere_sagitta_bound(oracle_mod):
    R = 0.7
    v, t = W.icosphere_mesh(3, R)
    w = _small((v, t), seed=4, n=48, band_cells=3)
    dist, _ = oracle_mod.sdf(w)
    pts = grid_points(w.origin, w.h, w.dims)
    pop = np.isfinite(dist)
    e = np.linalg.norm(v[t[:, 0]] - v[t[:, 1]], axis=1).max()
    theta = 2 * np.arcsin(e / (2 * R))
    # deepest point of an inscribed triangle below the sphere: its circumradius is < e
    sag = R - np.sqrt(R * R - (e / np.sqrt(3)) ** 2) * 1.0
    sag = max(sag, R * (1 - np.cos(theta / 2)))
    dev = (np.linalg.norm(pts[pop], axis=1) - R) - dist[pop]
    assert dev.min() >= -sag - 1e-6 and dev.max() <= 1e-6     # polyhedron lies inside the sphere


# ----------------------------------------------------------------------------- #
# invariants
# ----------------------------------------------------------------------------- #
def test_permutation_and_rotation_invariance(oracle_mod):
    v, t = W.torus_mesh(0.55, 0.22, 16, 9)
    a = _small((v, t), seed=1, n=32)
    b = _small((v, t), seed=2, n=32)            # another triangle order / vertex rotation
    da, ta = oracle_mod.sdf(a)
    db, tb = oracle_mod.sdf(b)
    assert np.array_equal(np.isfinite(da), np.isfinite(db))
    pop = np.isfinite(da)
    assert np.allclose(da[pop], db[pop], rtol=0, atol=1e-7)
    assert np.array_equal(np.signbit(da[pop]), np.signbit(db[pop]))
    # ids are permuted accordingly: same triangle geometry (as vertex sets) wherever unique
    ka = np.sort(a.soup[ta[pop]].reshape(-1, 9), axis=1)
    kb = np.sort(b.soup[tb[pop]].reshape(-1, 9), axis=1)
    same = np.all(ka == kb, axis=1)
    pts = grid_points(a.origin, a.h, a.dims)[pop]
    d_all = point_triangle_dist(pts[:, None, :], a.soup[None].astype(np.float64))
    srt = np.sort(d_all, axis=1)
    uniq = (srt[:, 1] - srt[:, 0]) > 1e-9            # edge/vertex-closest cells tie (several ids correct)
    assert uniq.sum() > 1000 and np.all(same[uniq])


def test_band_monotonicity(oracle_mod):
    w = _small(W.icosphere_mesh(2, 0.6), seed=9, n=32, band_cells=5)
    m = oracle_mod.Mesh(w.soup)
    d5, t5 = m.sdf(w.origin, w.h, w.dims, 5 * w.h)
    d2, t2 = m.sdf(w.origin, w.h, w.dims, 2 * w.h)
    keep = np.abs(d5) < 2 * w.h
    assert np.array_equal(np.isfinite(d2), keep)
    assert np.array_equal(d2[keep], d5[keep]) and np.array_equal(t2[keep], t5[keep])
    assert np.all(np.abs(d5[np.isfinite(d5)]) < 5 * w.h)


def test_reflection_and_axis_permutation_symmetry(oracle_mod):
    v, t = W.spike_mesh()
    soup = W.soup_from_indexed(v, t, None)
    origin, h, dims = W.grid_over((-1,) * 3, (1,) * 3, (24,) * 3)
    m = oracle_mod.Mesh(soup)
    d0, _ = m.sdf(origin, h, dims, 3 * h)
    # mirror x (flips orientation -> swap two vertices) and permute axes x->y->z->x
    s2 = soup.copy()
    s2[..., 0] = -s2[..., 0]
    s2 = s2[:, ::-1, :]
    s2 = np.ascontiguousarray(s2[..., [2, 0, 1]])
    d1, _ = oracle_mod.Mesh(s2).sdf(origin, h, dims, 3 * h)
    # d0[k,j,i] at (x,y,z) == d1 at (x',y',z') = (z,-x,y)
    d0m = d0[:, :, ::-1]                         # x -> -x   (grid symmetric about 0)
    d1_expected = np.transpose(d0m, (1, 2, 0))    # new (z',y',x') = (y, -x, z)
    assert np.array_equal(np.isfinite(d1), np.isfinite(d1_expected))
    pop = np.isfinite(d1)
    assert np.allclose(d1[pop], d1_expected[pop], rtol=0, atol=1e-7)


def test_eikonal_residual(oracle_mod):
    """eq.2: |grad f| = 1 away from the medial axis / feature boundaries."""
    w = _small(W.icosphere_mesh(3, 0.6), seed=6, n=64, band_cells=4)
    dist, _ = oracle_mod.sdf(w)
    d = dist.astype(np.float64)
    ok = np.isfinite(d)
    inner = ok[1:-1, 1:-1, 1:-1].copy()
    g = []
    for ax in range(3):
        sl_p = [slice(1, -1)] * 3
        sl_m = [slice(1, -1)] * 3
        sl_p[ax] = slice(2, None)
        sl_m[ax] = slice(0, -2)
        inner &= ok[tuple(sl_p)] & ok[tuple(sl_m)]
        with np.errstate(invalid="ignore"):
            g.append((d[tuple(sl_p)] - d[tuple(sl_m)]) / (2 * w.h))
    with np.errstate(invalid="ignore"):
        gn = np.sqrt(g[0] ** 2 + g[1] ** 2 + g[2] ** 2)
    res = np.abs(gn[inner] - 1.0)
    assert inner.sum() > 10000
    assert np.median(res) < 5e-3 and np.percentile(res, 99) < 0.05


# ----------------------------------------------------------------------------- #
# connectivity, classes, status codes
# ----------------------------------------------------------------------------- #
def test_feature_counts_known_topology(oracle_mod):
    c1 = oracle_mod.Mesh(W.config("C1").soup).counts
    assert (c1["V"], c1["E"], c1["F"]) == (8, 18, 12)
    assert c1["convex_v"] == 8 and c1["convex_e"] == 12 and c1["flat_e"] == 6
    v, t = W.box_with_cavity_mesh()
    cav = oracle_mod.Mesh(W.soup_from_indexed(v, t, np.random.default_rng(1))).counts
    assert cav["convex_v"] == 8 and cav["concave_v"] == 8
    assert cav["convex_e"] == 12 and cav["concave_e"] == 12 and cav["flat_e"] == 12
    assert cav["V"] - cav["E"] + cav["F"] == 4
    v, t = W.torus_mesh(0.6, 0.25, 24, 12)
    tor = oracle_mod.Mesh(W.soup_from_indexed(v, t, np.random.default_rng(1))).counts
    assert tor["V"] - tor["E"] + tor["F"] == 0 and tor["E"] == 3 * tor["F"] // 2
    assert tor["saddle_v"] > 0 and tor["convex_v"] > 0      # inner ring saddle, outer convex
    v, t = W.monkey_saddle_mesh()
    sad = oracle_mod.Mesh(W.soup_from_indexed(v, t, None))
    _, vclass, _ = sad.classes()
    centre = sad.corner_vid()[np.all(sad.soup == np.float32([0, 0, 0]), axis=2)][0]
    assert vclass[centre] == 2                                # saddle
    v, t = W.ruff_mesh()
    ruff = oracle_mod.Mesh(W.soup_from_indexed(v, t, None))
    _, vclass, vcos = ruff.classes()
    apex = ruff.corner_vid()[np.all(ruff.soup == np.float32([0, 0, 0.3]), axis=2)][0]
    assert vclass[apex] == 1                                  # classified convex
    v, t = W.spike_mesh(lean=1.2, height=0.3)
    _, _, vcos = oracle_mod.Mesh(W.soup_from_indexed(v, t, None)).classes()
    assert int((vcos <= 0).sum()) == 2                        # normals at 90 degrees or more from N_v
    v, t = W.config("C4", 0.05).soup, None
    star = oracle_mod.Mesh(v).counts
    assert star["V"] - star["E"] + star["F"] == 2


def test_status_codes(oracle_mod):
    v, t = W.box_mesh()
    soup = W.soup_from_indexed(v, t, None)
    with pytest.raises(oracle_mod.OracleError) as e:
        oracle_mod.Mesh(soup[:-1])
    assert e.value.status == 2                                # ENOTCLOSED
    flipped = soup.copy()
    flipped[3] = flipped[3][::-1]
    with pytest.raises(oracle_mod.OracleError) as e:
        oracle_mod.Mesh(flipped)
    assert e.value.status == 3                                # EORIENT
    deg = np.concatenate([soup, np.float32([[[0, 0, 0], [1, 0, 0], [2, 0, 0]], [[0, 0, 0], [2, 0, 0], [1, 0, 0]]])])
    with pytest.raises(oracle_mod.OracleError) as e:
        oracle_mod.Mesh(deg)
    assert e.value.status == 4                                # EDEGENERATE
    bad = soup.copy()
    bad[0, 0, 0] = np.nan
    with pytest.raises(oracle_mod.OracleError) as e:
        oracle_mod.Mesh(bad)
    assert e.value.status == 1                                # EINVAL
    # -0.0 and +0.0 are the same vertex
    z = soup.copy()
    z[..., 2] -= z[..., 2].min()                              # a face at z == 0
    z2 = z.copy()
    z2[0][z2[0] == 0] = -0.0
    assert oracle_mod.Mesh(z2).counts == oracle_mod.Mesh(z).counts


def test_dist_to_triangles_pinned(oracle_mod):
    """oracle_dist_to_triangles decides clause 4 of the comparison harness (an id mismatch is accepted only if the
    GPU's triangle is as close as the oracle's within the tolerance), so it gets its own pin: against the independent
    numpy formulation (projection + three clamped segments) on random (point, id) pairs -- near and far points, every
    Voronoi region of slivers and fat triangles alike -- against hand-derived closed forms, and out-of-range ids -> inf."""
    r = np.random.default_rng(77)
    v, t = W.torus_mesh(0.6, 0.25, 24, 12)
    soup = W.soup_from_indexed(v, t, r)
    om = oracle_mod.Mesh(soup)
    F = soup.shape[0]
    n = 20000
    ids = r.integers(0, F, n).astype(np.int32)
    # points around the named triangle (all seven regions) and far from it
    bary = r.dirichlet((0.6, 0.6, 0.6), n) * 2.0 - 0.5                  # in- and outside the triangle
    on = np.einsum("nk,nkc->nc", bary, soup[ids].astype(np.float64))
    pts = on + r.normal(0.0, 1.0, (n, 3)) * r.choice([1e-6, 1e-3, 0.05, 1.0], n)[:, None]
    d = om.dist_to_triangles(pts, ids)
    ref = point_triangle_dist(pts, soup[ids])
    assert np.max(np.abs(d - ref)) <= 1e-12
    assert np.all(d >= 0)
    # it is the distance to THAT triangle: never below the distance to the whole mesh, equal for the closest id
    dq, iq = om.query(pts[:2000])
    assert np.all(d[:2000] >= np.abs(dq) - 1e-12)
    assert np.max(np.abs(om.dist_to_triangles(pts[:2000], iq) - np.abs(dq))) <= 1e-12
    # a transposed operand / wrong id would show here: the triangle with the next id is (almost always) farther or nearer
    d_next = om.dist_to_triangles(pts, (ids + 1) % F)
    assert np.mean(np.abs(d_next - d) > 1e-9) > 0.9
    # closed forms on triangle 0 of a tetrahedron
    tet = W.soup_from_indexed(*W.tetrahedron_mesh(0.5), np.random.default_rng(1))
    o1, tri = oracle_mod.Mesh(tet), tet[:1]
    a, b, c = (tri[0, k].astype(np.float64) for k in range(3))
    nrm = np.cross(b - a, c - a); nrm /= np.linalg.norm(nrm)
    cen = (a + b + c) / 3
    q = np.stack([cen + 0.3 * nrm,                       # above the centroid: plane distance
                  a + 2.0 * (a - cen),                   # beyond vertex a on the ray from the centroid: |p - a|
                  0.5 * (a + b) + 0.7 * np.cross(b - a, nrm) / np.linalg.norm(b - a)])   # beside edge ab, in plane
    dd = o1.dist_to_triangles(q, np.zeros(3, dtype=np.int32))
    assert abs(dd[0] - 0.3) <= 1e-12
    assert abs(dd[1] - 2.0 * np.linalg.norm(a - cen)) <= 1e-12
    assert abs(dd[2] - 0.7) <= 1e-12
    # ids outside [0, F) -> +inf, never a crash or a wrapped index
    bad = om.dist_to_triangles(pts[:4], np.array([-1, F, F + 7, -2 ** 31], dtype=np.int32))
    assert np.all(np.isposinf(bad))

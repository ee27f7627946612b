"""GPU tests of the feature builder (sdf_create): the welded vertex ids,
the half-edge pairing, the edge records and the lowest incident triangle ids, read back through
sdf_get_table, against connectivity derived here with plain numpy from the same soup
(generator-known topology, SURVEY.md 8(c) "connectivity / feature tables")."""
import numpy as np
import pytest

from paper_1903_00353_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _numpy_connectivity(soup):
    F = soup.shape[0]
    pts = (soup.reshape(-1, 3) + np.float32(0.0)).view(np.uint32)          # -0 -> +0, exact bits
    _, first, inv = np.unique(pts, axis=0, return_index=True, return_inverse=True)
    inv = inv.reshape(-1)
    # vertex ids in order of the lowest corner index of every vertex
    order = np.argsort(first, kind="stable")
    rank = np.empty_like(order)
    rank[order] = np.arange(order.size)
    cvid = rank[inv].reshape(F, 3).astype(np.int32)
    return cvid, int(order.size)


@pytest.mark.parametrize("name,scale", [("C1", 1.0), ("C2", 0.25), ("C3", 0.25), ("C4", 0.06), ("C5", 0.02)])
def test_feature_tables(name, scale):
    from paper_1903_00353_b200 import binding as B
    w = W.config(name, scale)
    soup = np.ascontiguousarray(w.soup, dtype=np.float32)
    F = soup.shape[0]
    m = B.sdf_create(soup)
    s = B.sdf_stats(m)
    cvid_ref, V = _numpy_connectivity(soup)
    assert (s["F"], s["V"], s["E"]) == (F, V, 3 * F // 2)
    assert s["V"] - s["E"] + s["F"] == w.meta["V"] - w.meta["E"] + F          # Euler characteristic
    cvid = B.sdf_get_table(m, B.TABLE_CORNER_VID)
    # same partition of the corners (the numbering of the vertices is the library's own)
    assert cvid.min() == 0 and cvid.max() == V - 1
    pairs = np.unique(np.stack([cvid.reshape(-1), cvid_ref.reshape(-1)], axis=1), axis=0)
    assert pairs.shape[0] == V

    # half-edge 3t+k runs corner k -> k+1; its opposite runs the same edge backwards
    adj = B.sdf_get_table(m, B.TABLE_HALFEDGE_ADJ).reshape(-1)
    he = np.arange(3 * F)
    assert adj.min() >= 0 and adj.max() < 3 * F
    assert np.array_equal(adj[adj], he) and not np.any(adj == he)
    src = cvid.reshape(-1)
    dst = cvid[:, [1, 2, 0]].reshape(-1)
    assert np.array_equal(src[adj], dst) and np.array_equal(dst[adj], src)

    # unit face normals against fp64 numpy
    fn = B.sdf_get_table(m, B.TABLE_FACE_NORMAL)
    p = soup.astype(np.float64)
    n = np.cross(p[:, 1] - p[:, 0], p[:, 2] - p[:, 0])
    n /= np.linalg.norm(n, axis=1, keepdims=True)
    assert np.max(np.abs(fn - n)) < 1e-7

    # edge records: one per undirected edge, end points = the edge's two vertices, n1 / n2 = the
    # normals of its two triangles, tri = the lower triangle id
    er = B.sdf_get_table(m, B.TABLE_EDGE_REC)
    # one record per edge that has a wedge (flat and smooth edges have none), in no particular order
    assert er.shape[0] == s["edges_convex"] + s["edges_concave"] and s["edges_flat"] == 3 * F // 2 - er.shape[0]
    assert er.shape[0] > 0 and np.all(er["cls"] != 0)
    pos_to_vid = {}
    flat = (soup.reshape(-1, 3) + np.float32(0.0))
    for c in (np.unique(src, return_index=True)[1]):
        pos_to_vid[flat[c].tobytes()] = src[c]
    fwd = np.nonzero(src < dst)[0]
    edge_of = {(int(src[h]), int(dst[h])): h for h in fwd}
    assert len(edge_of) == 3 * F // 2
    seen = set()
    step = max(1, er.shape[0] // 4000)
    for e in range(0, er.shape[0], step):
        a = pos_to_vid[np.asarray(er["a"][e], dtype=np.float32).tobytes()]
        b = pos_to_vid[np.asarray(er["b"][e], dtype=np.float32).tobytes()]
        key = (int(min(a, b)), int(max(a, b)))
        assert key in edge_of and key not in seen
        seen.add(key)
        h0 = edge_of[key]
        t0, t1 = h0 // 3, adj[h0] // 3
        assert er["tri"][e] == min(t0, t1)
        # n1 belongs to the triangle that traverses a -> b
        ta = t0 if (a, b) == (int(src[h0]), int(dst[h0])) else t1
        tb = t1 if ta == t0 else t0
        assert np.array_equal(er["n1"][e], fn[ta]) and np.array_equal(er["n2"][e], fn[tb])
    assert s["edges_convex"] + s["edges_concave"] + s["edges_flat"] == 3 * F // 2
    assert np.count_nonzero(er["cls"] > 0) == s["edges_convex"]
    assert np.count_nonzero(er["cls"] < 0) == s["edges_concave"]

    # lowest incident triangle, vertex positions
    vm = B.sdf_get_table(m, B.TABLE_VERTEX_MINTRI)
    ref = np.full(V, np.iinfo(np.int32).max, dtype=np.int64)
    np.minimum.at(ref, src, he // 3)
    assert np.array_equal(vm, ref)
    vr = B.sdf_get_table(m, B.TABLE_VERTEX_REC)
    first_corner = np.unique(src, return_index=True)[1]
    assert np.array_equal(np.asarray(vr["pos"]), flat[first_corner])
    B.sdf_destroy(m)


def test_edge_error_classification():
    """Invalid edge tables take the exact (sorted-key) classification path."""
    from paper_1903_00353_b200 import binding as B
    v, t = W.icosphere_mesh(2, 0.5)
    soup = W.soup_from_indexed(v, t, np.random.default_rng(2))
    flipped = soup.copy()
    flipped[17] = flipped[17][::-1].copy()
    with pytest.raises(B.SdfError) as e:
        B.sdf_create(flipped)
    assert e.value.status == B.SDF_EORIENT
    with pytest.raises(B.SdfError) as e:
        B.sdf_create(np.ascontiguousarray(soup[1:]))
    assert e.value.status == B.SDF_ENOTCLOSED
    # a fin: one extra pair of opposite triangles glued onto an existing edge (4 faces at it)
    tri = soup[5]
    apex = (tri[0] + tri[1]) * np.float32(0.5) * np.float32(1.5)
    fin = np.stack([np.stack([tri[0], tri[1], apex]), np.stack([tri[1], tri[0], apex])]).astype(np.float32)
    with pytest.raises(B.SdfError) as e:
        B.sdf_create(np.ascontiguousarray(np.concatenate([soup, fin])))
    assert e.value.status == B.SDF_ENOTCLOSED
    B.sdf_destroy(B.sdf_create(soup))


@pytest.mark.parametrize("name,scale", [("C1", 1.0), ("C2", 1.0), ("C3", 0.5), ("C4", 0.12), ("C5", 0.05)])
def test_tile_builder_equals_global_builder(monkeypatch, name, scale):
    """The tile-local feature builder (default: weld, pair and accumulate inside spatial tiles in shared memory, only
    tile-boundary features through the global tables) against the first builder (SDF_BUILDER=global: every corner and
    half-edge through the global tables): same topology, same class counts, same pseudonormal data and bit-identical
    grids -- the two differ in how the data moves, not in any arithmetic that reaches the output."""
    import torch
    from paper_1903_00353_b200 import binding as B
    from gpu_util import f32_grid
    w = f32_grid(W.config(name, scale) if scale < 1.0 else W.config(name))
    keys = ("F", "V", "E", "edges_convex", "edges_concave", "edges_flat", "verts_pos_only", "verts_neg_only", "verts_both",
            "verts_skipped", "verts_hemisphere", "band_cells", "polyhedra")
    m1, d1, t1 = B.compute_workload(w)
    s1 = B.sdf_stats(m1)
    monkeypatch.setenv("SDF_BUILDER", "tile")
    m0, d0, t0 = B.compute_workload(w)
    s0 = B.sdf_stats(m0)
    monkeypatch.delenv("SDF_BUILDER")
    assert {k: s1[k] for k in keys} == {k: s0[k] for k in keys}
    assert torch.equal(t0, t1) and torch.equal(d0.view(torch.int32), d1.view(torch.int32))
    # per-vertex data, matched through the corner -> vertex tables (the numbering of the vertices differs)
    c0, c1 = (B.sdf_get_table(m, B.TABLE_CORNER_VID).reshape(-1) for m in (m0, m1))
    v0, v1 = (B.sdf_get_table(m, B.TABLE_VERTEX_REC) for m in (m0, m1))
    for f in ("pos", "axis", "cos_cone", "info"):
        assert np.array_equal(np.asarray(v0[f])[c0], np.asarray(v1[f])[c1]), f
    assert np.array_equal(B.sdf_get_table(m0, B.TABLE_VERTEX_MINTRI)[c0], B.sdf_get_table(m1, B.TABLE_VERTEX_MINTRI)[c1])
    assert np.array_equal(B.sdf_get_table(m0, B.TABLE_HALFEDGE_ADJ), B.sdf_get_table(m1, B.TABLE_HALFEDGE_ADJ))
    assert np.array_equal(B.sdf_get_table(m0, B.TABLE_FACE_NORMAL), B.sdf_get_table(m1, B.TABLE_FACE_NORMAL))
    e0, e1 = (np.sort(B.sdf_get_table(m, B.TABLE_EDGE_REC).view(np.uint8).reshape(-1, 64).view("V64").reshape(-1)) for m in (m0, m1))
    assert np.array_equal(e0, e1)

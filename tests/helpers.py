"""Independent numpy references used to PIN the oracle, and the GPU-vs-oracle
comparison harness.  Nothing here is imported by the product or by oracle/.

The numpy routines deliberately use formulations different from oracle/sdf_oracle.c
(plane projection + three clamped segments instead of the seven-region barycentric
walk; solid-angle winding numbers instead of pseudonormals)."""
from __future__ import annotations

import numpy as np


# ----------------------------------------------------------------------------- #
# closed forms
# ----------------------------------------------------------------------------- #
def box_sdf(p, lo, hi):
    """Exact signed distance to the axis-aligned box [lo,hi] (negative inside)."""
    c = 0.5 * (lo + hi)
    half = 0.5 * (hi - lo)
    q = np.abs(p - c) - half
    outside = np.linalg.norm(np.maximum(q, 0.0), axis=-1)
    inside = np.minimum(np.max(q, axis=-1), 0.0)
    return outside + inside


def grid_points(origin, h, dims, dtype=np.float64):
    nx, ny, nz = dims
    o = np.asarray(origin, dtype=dtype)
    x = o[0] + np.arange(nx, dtype=dtype) * h
    y = o[1] + np.arange(ny, dtype=dtype) * h
    z = o[2] + np.arange(nz, dtype=dtype) * h
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    return np.stack([X, Y, Z], axis=-1)            # [nz,ny,nx,3]


# ----------------------------------------------------------------------------- #
# brute-force unsigned distance: projection + three segments
# ----------------------------------------------------------------------------- #
def _seg_dist2(p, a, b):
    ab = b - a
    t = np.clip(np.einsum("...i,...i->...", p - a, ab) / np.einsum("...i,...i->...", ab, ab), 0.0, 1.0)
    d = p - (a + t[..., None] * ab)
    return np.einsum("...i,...i->...", d, d)


def point_triangle_dist(p, tri):
    """p [...,3], tri [...,3,3] (broadcastable) -> unsigned distance (fp64)."""
    p = np.asarray(p, dtype=np.float64)
    tri = np.asarray(tri, dtype=np.float64)
    a, b, c = tri[..., 0, :], tri[..., 1, :], tri[..., 2, :]
    n = np.cross(b - a, c - a)
    nn = np.einsum("...i,...i->...", n, n)
    hgt = np.einsum("...i,...i->...", p - a, n)
    proj = p - (hgt / nn)[..., None] * n
    inside = np.ones(np.broadcast(hgt, nn).shape, dtype=bool)
    for (u, v) in ((a, b), (b, c), (c, a)):
        inside &= np.einsum("...i,...i->...", np.cross(v - u, proj - u), n) >= 0.0
    d2_plane = hgt * hgt / nn
    d2_edges = np.minimum(np.minimum(_seg_dist2(p, a, b), _seg_dist2(p, b, c)), _seg_dist2(p, c, a))
    return np.sqrt(np.where(inside, d2_plane, d2_edges))


def brute_unsigned(points, soup, chunk=4096):
    """min over all triangles, and argmin (lowest id on exact ties)."""
    pts = np.asarray(points, dtype=np.float64).reshape(-1, 3)
    soup = np.asarray(soup, dtype=np.float64)
    best = np.full(pts.shape[0], np.inf)
    arg = np.full(pts.shape[0], -1, dtype=np.int64)
    for s in range(0, pts.shape[0], chunk):
        d = point_triangle_dist(pts[s:s + chunk, None, :], soup[None, :, :, :])
        arg[s:s + chunk] = np.argmin(d, axis=1)
        best[s:s + chunk] = d[np.arange(d.shape[0]), arg[s:s + chunk]]
    return best, arg


def winding_number(points, soup, chunk=4096):
    """Generalised winding number: sum of signed solid angles / 4pi (Van Oosterom &
    Strackee).  ~1 inside a closed outward-oriented surface, ~0 outside."""
    pts = np.asarray(points, dtype=np.float64).reshape(-1, 3)
    soup = np.asarray(soup, dtype=np.float64)
    out = np.zeros(pts.shape[0])
    for s in range(0, pts.shape[0], chunk):
        P = pts[s:s + chunk, None, :]
        a = soup[None, :, 0, :] - P
        b = soup[None, :, 1, :] - P
        c = soup[None, :, 2, :] - P
        la, lb, lc = (np.linalg.norm(v, axis=-1) for v in (a, b, c))
        num = np.einsum("...i,...i->...", a, np.cross(b, c))
        den = (la * lb * lc + np.einsum("...i,...i->...", a, b) * lc
               + np.einsum("...i,...i->...", b, c) * la + np.einsum("...i,...i->...", c, a) * lb)
        out[s:s + chunk] = np.sum(2.0 * np.arctan2(num, den), axis=1) / (4.0 * np.pi)
    return out


# ----------------------------------------------------------------------------- #
# GPU-vs-oracle comparison: the four parity clauses of BASELINE.json north_star
# ----------------------------------------------------------------------------- #
def compare_to_oracle(dist_gpu, tri_gpu, dist_ref, tri_ref, workload, oracle_mesh, max_report=5):
    """Returns a dict of violation counts (all must be 0) and diagnostics.

    Clauses (BASELINE.json north_star):
      1. populated-cell set identical, except cells within 1e-5*h of the band edge;
      2. |d_gpu - d_oracle| <= 1e-5*h + 1e-6*diag (fp32);
      3. signs exact;
      4. closest-triangle ids bit-exact, except where the two candidates' distances differ
         by less than that tolerance (several results are correct).
    """
    h, band, diag = float(workload.h), float(workload.band), float(workload.diag)
    tol = 1e-5 * h + 1e-6 * diag
    dg = np.asarray(dist_gpu).reshape(-1)
    tg = np.asarray(tri_gpu).reshape(-1)
    dr = np.asarray(dist_ref).reshape(-1)
    tr = np.asarray(tri_ref).reshape(-1)
    pop_g = np.isfinite(dg)
    pop_r = np.isfinite(dr)
    res = {"tol": tol, "populated_gpu": int(pop_g.sum()), "populated_ref": int(pop_r.sum())}

    # sentinels
    res["bad_sentinel"] = int(np.sum(~pop_g & ((tg != -1) | ~(np.isposinf(dg)))))
    res["bad_id_range"] = int(np.sum(pop_g & ((tg < 0) | (tg >= workload.ntri))))

    nx, ny, nz = workload.dims

    def cell_xyz(idx):
        i = idx % nx
        j = (idx // nx) % ny
        k = idx // (nx * ny)
        o = np.asarray(workload.origin, dtype=np.float64)
        return np.stack([o[0] + i * h, o[1] + j * h, o[2] + k * h], axis=1)

    # clause 1: set difference must lie within 1e-5*h of the band edge (true distance)
    diff = np.nonzero(pop_g != pop_r)[0]
    bad_set = 0
    if diff.size:
        d_true, _ = oracle_mesh.query(cell_xyz(diff))
        bad = np.abs(np.abs(d_true) - band) > 1e-5 * h
        bad_set = int(bad.sum())
        res["set_diff_examples"] = [(int(c), float(v)) for c, v in zip(diff[bad][:max_report], d_true[bad][:max_report])]
    res["set_diff_total"] = int(diff.size)
    res["bad_set"] = bad_set

    both = np.nonzero(pop_g & pop_r)[0]
    err = np.abs(dg[both].astype(np.float64) - dr[both].astype(np.float64))
    res["max_abs_err"] = float(err.max()) if both.size else 0.0
    res["bad_dist"] = int(np.sum(err > tol))
    # clause 3: signs exact.  A zero distance has no sign -- and the oracle reports an exactly-zero distance (a cell centre on
    # a face or an edge of the mesh) as +-eps with |eps| ~ 1e-16 * diag, the sign being rounding noise of its fp64 n . r
    # (DESIGN.md sec.2 reading #20).  So the clause is waived where BOTH magnitudes are below 1e-12 * diag: five orders of
    # magnitude under what fp32 resolves, four above the noise.  A flipped sign of any distance fp32 can represent still counts.
    sg = np.signbit(dg[both]) != np.signbit(dr[both])
    zt = 1e-12 * diag
    sg &= ~((np.abs(dg[both].astype(np.float64)) <= zt) & (np.abs(dr[both].astype(np.float64)) <= zt))
    res["bad_sign"] = int(sg.sum())
    if sg.any():
        res["sign_examples"] = [(int(c), float(dg[c]), float(dr[c])) for c in both[sg][:max_report]]
    # clause 4: ids
    idm = np.nonzero(tg[both] != tr[both])[0]
    res["id_mismatch_total"] = int(idm.size)
    # of the mismatches: "ties" = the GPU's triangle is as close as the oracle's to the rounding of the oracle's fp32 output (the closest point
    # lies on a shared edge / vertex: several ids are correct); "near" = closer than the
    # tolerance but not a tie (fp32 could not tell them apart) -- the share of those is on record and bounded by
    # the callers, so that a kernel ignoring the lowest-id rule does not pass unnoticed
    bad_id, id_ties = 0, 0
    if idm.size:
        cells = both[idm]
        d_alt = oracle_mesh.dist_to_triangles(cell_xyz(cells), tg[cells])
        d_o = np.abs(dr[cells].astype(np.float64))           # the oracle's distance, rounded once to fp32
        gap = np.abs(d_alt - d_o)
        badm = gap > tol
        bad_id = int(badm.sum())
        id_ties = int(np.sum(gap <= 2.0 ** -22 * d_o + 1e-12 * diag))
        if badm.any():
            res["id_examples"] = [(int(c), int(tg[c]), int(tr[c])) for c in cells[badm][:max_report]]
    res["bad_id"] = bad_id
    res["id_mismatch_ties"] = id_ties
    res["id_mismatch_near"] = int(idm.size) - id_ties - bad_id
    res["id_mismatch_share"] = float(idm.size) / max(int(both.size), 1)
    res["id_near_share"] = float(res["id_mismatch_near"]) / max(int(both.size), 1)
    res["ok"] = all(res[k] == 0 for k in ("bad_sentinel", "bad_id_range", "bad_set", "bad_dist", "bad_sign", "bad_id"))
    return res

"""CPU oracle for the narrow-band signed distance transform.  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It shares no code with the CUDA path and imports
nothing from `paper_1903_00353_b200`.

`build()` compiles `sdf_oracle.c` with gcc into `oracle/libsdf_oracle.so`.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sdf_oracle.c")
_LIB = os.path.join(_HERE, "libsdf_oracle.so")
_lib = None

STATUS = {0: "OK", 1: "EINVAL", 2: "ENOTCLOSED", 3: "EORIENT", 4: "EDEGENERATE", 5: "ENOMEM"}
REGIONS = ("FACE", "E_AB", "E_BC", "E_CA", "V_A", "V_B", "V_C")


class OracleError(RuntimeError):
    def __init__(self, status):
        self.status = int(status)
        super().__init__("oracle status %d (%s)" % (status, STATUS.get(int(status), "?")))


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-ffp-contract=off", "-o", _LIB, _SRC,
               "-lm", "-lpthread"]
        subprocess.check_call(cmd)
    return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = C.CDLL(build())
    dp, fp, ip, lp = (C.POINTER(C.c_double), C.POINTER(C.c_float), C.POINTER(C.c_int32),
                      C.POINTER(C.c_int64))
    lib.oracle_build.argtypes = [fp, C.c_int64, C.POINTER(C.c_void_p)]
    lib.oracle_build.restype = C.c_int
    lib.oracle_free.argtypes = [C.c_void_p]
    lib.oracle_free.restype = None
    lib.oracle_counts.argtypes = [C.c_void_p, lp]
    lib.oracle_counts.restype = None
    for name, ptr in (("oracle_get_corner_vid", ip), ("oracle_get_corner_eid", ip),
                      ("oracle_get_vertex_normals", dp), ("oracle_get_edge_normals", dp),
                      ("oracle_get_face_normals", dp)):
        f = getattr(lib, name)
        f.argtypes = [C.c_void_p, ptr]
        f.restype = None
    lib.oracle_get_classes.argtypes = [C.c_void_p, ip, ip, dp]
    lib.oracle_get_classes.restype = None
    lib.oracle_sdf.argtypes = [C.c_void_p, dp, C.c_double, C.c_int, C.c_int, C.c_int, C.c_double,
                               fp, ip, C.c_int]
    lib.oracle_sdf.restype = C.c_int
    lib.oracle_query.argtypes = [C.c_void_p, dp, C.c_int64, dp, ip, C.c_int]
    lib.oracle_query.restype = C.c_int
    lib.oracle_dist_to_triangles.argtypes = [C.c_void_p, dp, ip, C.c_int64, dp]
    lib.oracle_dist_to_triangles.restype = C.c_int
    lib.oracle_closest_points.argtypes = [C.c_void_p, dp, C.c_double, C.c_int, C.c_int, C.c_int, ip, fp]
    lib.oracle_closest_points.restype = C.c_int
    lib.oracle_fill_interior.argtypes = [fp, C.c_int, C.c_int, C.c_int, C.c_float]
    lib.oracle_fill_interior.restype = C.c_int
    lib.oracle_point_triangle.argtypes = [dp, fp, dp, C.POINTER(C.c_int)]
    lib.oracle_point_triangle.restype = C.c_double
    _lib = lib
    return lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def default_threads() -> int:
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except AttributeError:
        return max(1, os.cpu_count() or 1)


def point_triangle(p, tri):
    """fp64 distance from point p to triangle tri[3,3] (fp32): (d, closest[3], region name)."""
    lib = _load()
    p = np.ascontiguousarray(p, dtype=np.float64)
    t = np.ascontiguousarray(tri, dtype=np.float32).reshape(9)
    q = np.zeros(3)
    r = C.c_int(0)
    d = lib.oracle_point_triangle(_p(p, C.c_double), _p(t, C.c_float), _p(q, C.c_double), C.byref(r))
    return float(d), q, REGIONS[r.value]


class Mesh:
    """Connectivity + pseudonormals of a closed triangle soup (oracle side, fp64)."""

    def __init__(self, soup):
        lib = _load()
        self.soup = np.ascontiguousarray(soup, dtype=np.float32).reshape(-1, 3, 3)
        h = C.c_void_p()
        st = lib.oracle_build(_p(self.soup, C.c_float), self.soup.shape[0], C.byref(h))
        if st != 0:
            raise OracleError(st)
        self._h = h
        cnt = np.zeros(10, dtype=np.int64)
        lib.oracle_counts(self._h, _p(cnt, C.c_int64))
        keys = ("F", "V", "E", "convex_e", "concave_e", "flat_e", "convex_v", "concave_v", "flat_v", "saddle_v")
        self.counts = dict(zip(keys, (int(v) for v in cnt)))
        self.F, self.V, self.E = self.counts["F"], self.counts["V"], self.counts["E"]

    def __del__(self):
        if getattr(self, "_h", None) is not None and _lib is not None:
            _lib.oracle_free(self._h)
            self._h = None

    def corner_vid(self):
        out = np.zeros(3 * self.F, dtype=np.int32)
        _lib.oracle_get_corner_vid(self._h, _p(out, C.c_int32))
        return out.reshape(self.F, 3)

    def corner_eid(self):
        out = np.zeros(3 * self.F, dtype=np.int32)
        _lib.oracle_get_corner_eid(self._h, _p(out, C.c_int32))
        return out.reshape(self.F, 3)

    def vertex_normals(self):
        out = np.zeros((self.V, 3))
        _lib.oracle_get_vertex_normals(self._h, _p(out, C.c_double))
        return out

    def edge_normals(self):
        out = np.zeros((self.E, 3))
        _lib.oracle_get_edge_normals(self._h, _p(out, C.c_double))
        return out

    def face_normals(self):
        out = np.zeros((self.F, 3))
        _lib.oracle_get_face_normals(self._h, _p(out, C.c_double))
        return out

    def classes(self):
        ec = np.zeros(self.E, dtype=np.int32)
        vc = np.zeros(self.V, dtype=np.int32)
        vcos = np.zeros(self.V)
        _lib.oracle_get_classes(self._h, _p(ec, C.c_int32), _p(vc, C.c_int32), _p(vcos, C.c_double))
        return ec, vc, vcos

    def sdf(self, origin, h, dims, band, nthreads=None):
        """Narrow-band SDF: returns (dist float32 [nz,ny,nx], tri int32 [nz,ny,nx])."""
        nx, ny, nz = (int(v) for v in dims)
        o = np.ascontiguousarray(origin, dtype=np.float64)
        dist = np.empty((nz, ny, nx), dtype=np.float32)
        tri = np.empty((nz, ny, nx), dtype=np.int32)
        st = _lib.oracle_sdf(self._h, _p(o, C.c_double), float(h), nx, ny, nz, float(band),
                             _p(dist, C.c_float), _p(tri, C.c_int32),
                             int(nthreads or default_threads()))
        if st != 0:
            raise OracleError(st)
        return dist, tri

    def closest_points(self, origin, h, dims, tri):
        """Closest point on triangle tri[cell] for every cell with tri >= 0: float32 [nz,ny,nx,3], +inf elsewhere."""
        nx, ny, nz = (int(v) for v in dims)
        o = np.ascontiguousarray(origin, dtype=np.float64)
        t = np.ascontiguousarray(tri, dtype=np.int32).reshape(-1)
        out = np.empty((nz, ny, nx, 3), dtype=np.float32)
        st = _lib.oracle_closest_points(self._h, _p(o, C.c_double), float(h), nx, ny, nz, _p(t, C.c_int32),
                                        _p(out, C.c_float))
        if st != 0:
            raise OracleError(st)
        return out

    def query(self, pts, nthreads=None):
        """Brute-force signed fp64 distance + closest triangle id for arbitrary points."""
        pts = np.ascontiguousarray(pts, dtype=np.float64).reshape(-1, 3)
        d = np.zeros(pts.shape[0])
        ids = np.zeros(pts.shape[0], dtype=np.int32)
        st = _lib.oracle_query(self._h, _p(pts, C.c_double), pts.shape[0], _p(d, C.c_double),
                               _p(ids, C.c_int32), int(nthreads or default_threads()))
        if st != 0:
            raise OracleError(st)
        return d, ids

    def dist_to_triangles(self, pts, tri_ids):
        pts = np.ascontiguousarray(pts, dtype=np.float64).reshape(-1, 3)
        ids = np.ascontiguousarray(tri_ids, dtype=np.int32).reshape(-1)
        d = np.zeros(pts.shape[0])
        st = _lib.oracle_dist_to_triangles(self._h, _p(pts, C.c_double), _p(ids, C.c_int32), pts.shape[0],
                                           _p(d, C.c_double))
        if st != 0:
            raise OracleError(st)
        return d


def fill_interior(dist, band):
    """PAPER.md:493 axis sweeps on a narrow-band grid [nz,ny,nx] (a filled copy is returned)."""
    _load()
    out = np.ascontiguousarray(dist, dtype=np.float32).copy()
    nz, ny, nx = out.shape
    st = _lib.oracle_fill_interior(_p(out, C.c_float), nx, ny, nz, float(np.float32(band)))
    if st != 0:
        raise OracleError(st)
    return out


def sdf(workload, nthreads=None):
    """Oracle SDF of a `Workload`-like object (soup, origin, h, dims, band)."""
    return Mesh(workload.soup).sdf(workload.origin, workload.h, workload.dims, workload.band, nthreads)

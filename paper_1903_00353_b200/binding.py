"""Thin ctypes binding over the C-ABI library of `include/sdf.h` (argument marshalling only).

Same names as the C entry points: `sdf_create`, `sdf_compute`, `sdf_compute_host`,
`sdf_stats`, `sdf_get_table`, `sdf_destroy`.  PyTorch supplies device memory (output
tensors, and the library's workspace through torch's caching allocator) and the CUDA
stream; every step of the method runs inside the library's kernels.  There is no CPU
fallback: if the library is missing or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

STATUS_NAMES = {0: "SDF_OK", 1: "SDF_EINVAL", 2: "SDF_ENOTCLOSED", 3: "SDF_EORIENT",
                4: "SDF_EDEGENERATE", 5: "SDF_ENOMEM", 6: "SDF_ECUDA", 7: "SDF_EIO", 8: "SDF_ETOOBIG"}
SDF_OK, SDF_EINVAL, SDF_ENOTCLOSED, SDF_EORIENT, SDF_EDEGENERATE, SDF_ENOMEM, SDF_ECUDA, SDF_EIO, SDF_ETOOBIG = range(9)

TABLE_CORNER_VID, TABLE_HALFEDGE_ADJ, TABLE_FACE_NORMAL, TABLE_VERTEX_REC, TABLE_EDGE_REC, \
    TABLE_VERTEX_MINTRI = range(6)

EXPORTS = ("sdf_create", "sdf_transform", "sdf_compute", "sdf_compute_host", "sdf_compute_sparse", "sdf_compute_sparse_host", "sdf_zslab", "sdf_compute_zslab", "sdf_fill_interior", "sdf_fill_interior_static", "sdf_closest_points", "sdf_stats", "sdf_get_table",
           "sdf_destroy", "sdf_strerror", "sdf_last_cuda_error", "sdf_version",
           "sdf_enable_timing", "sdf_get_timings", "sdf_launch_count", "sdf_measure_fp32_peak",
           "sdf_read_stl", "sdf_free_host", "sdf_write_stl", "sdf_write_grid")

TIMING_STAGES = ("ingest_weld", "edges", "vertices", "clip_scan", "clear", "evaluate", "emit", "fill")

VERTEX_REC_DTYPE = np.dtype([("pos", "<f4", 3), ("axis", "<f4", 3), ("cos_cone", "<f4"), ("info", "<i4")])
EDGE_REC_DTYPE = np.dtype([("a", "<f4", 3), ("b", "<f4", 3), ("n1", "<f4", 3), ("n2", "<f4", 3),
                           ("tri", "<i4"), ("cls", "<i4"), ("pad", "<i4", 2)])


class SdfError(RuntimeError):
    def __init__(self, status, where=""):
        self.status = int(status)
        msg = STATUS_NAMES.get(self.status, str(status))
        try:
            msg += ": " + lib().sdf_strerror(self.status).decode()
            if self.status == SDF_ECUDA:
                msg += " (cudaError %d)" % lib().sdf_last_cuda_error()
        except Exception:
            pass
        super().__init__("%s failed with %s" % (where or "sdf call", msg))


_ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p, C.c_void_p)
_FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class _Allocator(C.Structure):
    _fields_ = [("alloc", _ALLOC_FN), ("free", _FREE_FN), ("user", C.c_void_p)]


class Stats(C.Structure):
    _fields_ = [(n, C.c_int64) for n in (
        "F", "V", "E", "edges_convex", "edges_concave", "edges_flat",
        "verts_pos_only", "verts_neg_only", "verts_both", "verts_skipped", "verts_hemisphere",
        "weld_collisions", "polyhedra", "work_items", "pairs_tested", "pairs_accepted",
        "bricks_active", "bricks_total", "band_cells", "fp64_rechecks", "cdp_fallbacks")]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_}


_lib = None


def lib_path() -> str:
    return _build.LIB


def lib():
    """Load the shared library (building it with nvcc if the in-tree copy is missing or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if os.environ.get("SDF_B200_NO_BUILD") != "1":
        path = _build.build_library()
    if not os.path.exists(path):
        raise RuntimeError("CUDA library %s is missing; run `python -m paper_1903_00353_b200.build`" % path)
    L = C.CDLL(path)
    vp = C.c_void_p
    L.sdf_create.argtypes = [vp, C.c_int64, C.c_int, C.POINTER(_Allocator), vp, C.POINTER(vp)]
    L.sdf_create.restype = C.c_int
    L.sdf_compute.argtypes = [vp, C.POINTER(C.c_float), C.c_float, C.c_int, C.c_int, C.c_int, C.c_float, vp, vp, vp]
    L.sdf_compute.restype = C.c_int
    L.sdf_compute_host.argtypes = L.sdf_compute.argtypes
    L.sdf_transform.argtypes = [vp, C.c_int64, C.c_int, C.POINTER(_Allocator), C.POINTER(C.c_float), C.c_float, C.c_int, C.c_int,
                                C.c_int, C.c_float, vp, vp, vp, C.POINTER(vp)]
    L.sdf_transform.restype = C.c_int
    L.sdf_compute_sparse.argtypes = [vp, C.POINTER(C.c_float), C.c_float, C.c_int, C.c_int, C.c_int, C.c_float, C.c_int64, vp, vp, vp,
                                     C.POINTER(C.c_int64), vp]
    L.sdf_compute_sparse.restype = C.c_int
    L.sdf_compute_sparse_host.argtypes = L.sdf_compute_sparse.argtypes
    L.sdf_compute_sparse_host.restype = C.c_int
    L.sdf_zslab.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int)]
    L.sdf_zslab.restype = C.c_int
    L.sdf_compute_zslab.argtypes = [vp, C.POINTER(C.c_float), C.c_float, C.c_int, C.c_int, C.c_int, C.c_float, C.c_int, C.c_int,
                                    vp, vp, vp, C.POINTER(C.c_int), C.POINTER(C.c_int)]
    L.sdf_compute_zslab.restype = C.c_int
    L.sdf_compute_host.restype = C.c_int
    L.sdf_closest_points.argtypes = [vp, C.POINTER(C.c_float), C.c_float, C.c_int, C.c_int, C.c_int, vp, vp, vp]
    L.sdf_closest_points.restype = C.c_int
    L.sdf_read_stl.argtypes = [C.c_char_p, C.POINTER(C.POINTER(C.c_float)), C.POINTER(C.c_int64)]
    L.sdf_read_stl.restype = C.c_int
    L.sdf_free_host.argtypes = [vp]
    L.sdf_free_host.restype = None
    L.sdf_write_stl.argtypes = [C.c_char_p, vp, C.c_int64, C.c_int]
    L.sdf_write_stl.restype = C.c_int
    L.sdf_write_grid.argtypes = [C.c_char_p, vp, vp, C.POINTER(C.c_float), C.c_float, C.c_int, C.c_int, C.c_int, C.c_float]
    L.sdf_write_grid.restype = C.c_int
    L.sdf_fill_interior.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_float, vp]
    L.sdf_fill_interior.restype = C.c_int
    L.sdf_fill_interior_static.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_float, vp]
    L.sdf_fill_interior_static.restype = C.c_int
    L.sdf_stats.argtypes = [vp, C.POINTER(Stats)]
    L.sdf_stats.restype = C.c_int
    L.sdf_get_table.argtypes = [vp, C.c_int, vp, C.c_size_t]
    L.sdf_get_table.restype = C.c_int
    L.sdf_destroy.argtypes = [vp]
    L.sdf_destroy.restype = None
    L.sdf_strerror.argtypes = [C.c_int]
    L.sdf_strerror.restype = C.c_char_p
    L.sdf_last_cuda_error.argtypes = []
    L.sdf_last_cuda_error.restype = C.c_int
    L.sdf_version.argtypes = []
    L.sdf_version.restype = C.c_int
    L.sdf_enable_timing.argtypes = [C.c_int]
    L.sdf_enable_timing.restype = C.c_int
    L.sdf_get_timings.argtypes = [vp, C.POINTER(C.c_float), C.c_int]
    L.sdf_get_timings.restype = C.c_int
    L.sdf_measure_fp32_peak.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_int), vp]
    L.sdf_measure_fp32_peak.restype = C.c_int
    L.sdf_launch_count.argtypes = []
    L.sdf_launch_count.restype = C.c_int64
    _lib = L
    return L


# --------------------------------------------------------------------------------------
# torch plumbing: device memory and streams only
# --------------------------------------------------------------------------------------
def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_1903_00353_b200 needs a CUDA device (there is no CPU fallback)")
    return torch


_torch_allocator = None


def torch_allocator():
    """sdf_allocator whose callbacks are torch's caching allocator."""
    global _torch_allocator
    if _torch_allocator is None:
        torch = _torch()

        # the raw entry points of torch's caching allocator (what torch.cuda.caching_allocator_alloc
        # ends up calling, without its device-context manager: these callbacks sit on the critical
        # path of every sdf_create / sdf_compute); the public functions if a build lacks them
        raw_alloc = getattr(torch._C, "_cuda_cudaCachingAllocator_raw_alloc", None)
        raw_delete = getattr(torch._C, "_cuda_cudaCachingAllocator_raw_delete", None)

        def _alloc(nbytes, stream, user):
            try:
                if raw_alloc is not None:
                    return raw_alloc(int(nbytes), int(stream or 0))
                return torch.cuda.caching_allocator_alloc(int(nbytes), stream=int(stream or 0))
            except Exception:
                return None

        def _free(ptr, user):
            if ptr:
                if raw_delete is not None:
                    raw_delete(int(ptr))
                else:
                    torch.cuda.caching_allocator_delete(int(ptr))

        a = _Allocator(_ALLOC_FN(_alloc), _FREE_FN(_free), None)
        _torch_allocator = a
    return _torch_allocator


def _stream_ptr(stream):
    if stream is None:
        return int(_torch().cuda.current_stream().cuda_stream)
    if isinstance(stream, int):
        return stream
    return int(stream.cuda_stream)


class Mesh:
    """Owner of an `sdf_mesh*` handle."""

    def __init__(self, handle, ntri):
        self._h = handle
        self.ntri = int(ntri)

    def destroy(self):
        if self._h:
            lib().sdf_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    @property
    def handle(self):
        if not self._h:
            raise RuntimeError("sdf_mesh already destroyed")
        return self._h


def sdf_create(tri_xyz, stream=None, use_torch_allocator=True) -> Mesh:
    """tri_xyz: float32 [F,3,3] -- a torch CUDA tensor (device pointer, on_device=1) or a
    numpy array / CPU tensor (host pointer, copied by the library)."""
    L = lib()
    torch = _torch()
    if isinstance(tri_xyz, torch.Tensor):
        t = tri_xyz.detach()
        if t.dtype != torch.float32:
            raise TypeError("tri_xyz must be float32")
        t = t.contiguous()
        ptr, on_dev, ntri, keep = t.data_ptr(), int(t.is_cuda), t.numel() // 9, t
    else:
        a = np.ascontiguousarray(tri_xyz, dtype=np.float32)
        ptr, on_dev, ntri, keep = a.ctypes.data, 0, a.size // 9, a
    if keep is not None and (keep.size if isinstance(keep, np.ndarray) else keep.numel()) != 9 * ntri:
        raise ValueError("tri_xyz must hold 9 floats per triangle")
    out = C.c_void_p()
    alloc = C.byref(torch_allocator()) if use_torch_allocator else None
    st = L.sdf_create(C.c_void_p(ptr), ntri, on_dev, alloc, C.c_void_p(_stream_ptr(stream)), C.byref(out))
    if st != SDF_OK:
        raise SdfError(st, "sdf_create")
    return Mesh(out, ntri)


def _soup_ptr(tri_xyz):
    torch = _torch()
    if isinstance(tri_xyz, torch.Tensor):
        t = tri_xyz.detach()
        if t.dtype != torch.float32:
            raise TypeError("tri_xyz must be float32")
        t = t.contiguous()
        return t.data_ptr(), int(t.is_cuda), t.numel() // 9, t.numel(), t
    a = np.ascontiguousarray(tri_xyz, dtype=np.float32)
    return a.ctypes.data, 0, a.size // 9, a.size, a


def sdf_transform(tri_xyz, origin, h, dims, band, dist_out=None, tri_out=None, stream=None, use_torch_allocator=True):
    """sdf_create + sdf_compute in one call (include/sdf.h: the sentinel fill starts before the
    feature construction).  Returns (Mesh, dist float32 [nz,ny,nx], tri int32 [nz,ny,nx])."""
    L = lib()
    torch = _torch()
    ptr, on_dev, ntri, nel, keep = _soup_ptr(tri_xyz)
    if nel != 9 * ntri:
        raise ValueError("tri_xyz must hold 9 floats per triangle")
    nx, ny, nz = (int(v) for v in dims)
    if dist_out is None:
        dist_out = torch.empty((nz, ny, nx), dtype=torch.float32, device="cuda")
    if tri_out is None:
        tri_out = torch.empty((nz, ny, nx), dtype=torch.int32, device="cuda")
    assert dist_out.is_cuda and tri_out.is_cuda and dist_out.is_contiguous() and tri_out.is_contiguous()
    assert dist_out.numel() == nx * ny * nz and tri_out.numel() == nx * ny * nz
    assert dist_out.dtype == torch.float32 and tri_out.dtype == torch.int32
    out = C.c_void_p()
    alloc = C.byref(torch_allocator()) if use_torch_allocator else None
    st = L.sdf_transform(C.c_void_p(ptr), ntri, on_dev, alloc, _origin3(origin), float(h), nx, ny, nz, float(band),
                         C.c_void_p(dist_out.data_ptr()), C.c_void_p(tri_out.data_ptr()),
                         C.c_void_p(_stream_ptr(stream)), C.byref(out))
    del keep
    if st != SDF_OK:
        raise SdfError(st, "sdf_transform")
    return Mesh(out, ntri), dist_out, tri_out


def _origin3(origin):
    o = (C.c_float * 3)(*[float(v) for v in origin])
    return o


def sdf_compute(mesh: Mesh, origin, h, dims, band, dist_out=None, tri_out=None, stream=None):
    """Returns (dist float32 [nz,ny,nx], tri int32 [nz,ny,nx]) CUDA tensors."""
    L = lib()
    torch = _torch()
    nx, ny, nz = (int(v) for v in dims)
    if dist_out is None:
        dist_out = torch.empty((nz, ny, nx), dtype=torch.float32, device="cuda")
    if tri_out is None:
        tri_out = torch.empty((nz, ny, nx), dtype=torch.int32, device="cuda")
    assert dist_out.is_cuda and tri_out.is_cuda and dist_out.is_contiguous() and tri_out.is_contiguous()
    assert dist_out.numel() == nx * ny * nz and tri_out.numel() == nx * ny * nz
    assert dist_out.dtype == torch.float32 and tri_out.dtype == torch.int32
    st = L.sdf_compute(mesh.handle, _origin3(origin), float(h), nx, ny, nz, float(band),
                       C.c_void_p(dist_out.data_ptr()), C.c_void_p(tri_out.data_ptr()),
                       C.c_void_p(_stream_ptr(stream)))
    if st != SDF_OK:
        raise SdfError(st, "sdf_compute")
    return dist_out, tri_out


def sdf_compute_host(mesh: Mesh, origin, h, dims, band, dist_out=None, tri_out=None, stream=None):
    """Host-buffer variant: dist_out / tri_out are CPU tensors (pinned recommended)."""
    L = lib()
    torch = _torch()
    nx, ny, nz = (int(v) for v in dims)
    if dist_out is None:
        dist_out = torch.empty((nz, ny, nx), dtype=torch.float32, pin_memory=True)
    if tri_out is None:
        tri_out = torch.empty((nz, ny, nx), dtype=torch.int32, pin_memory=True)
    assert not dist_out.is_cuda and not tri_out.is_cuda
    assert dist_out.numel() == nx * ny * nz and tri_out.numel() == nx * ny * nz
    st = L.sdf_compute_host(mesh.handle, _origin3(origin), float(h), nx, ny, nz, float(band),
                            C.c_void_p(dist_out.data_ptr()), C.c_void_p(tri_out.data_ptr()),
                            C.c_void_p(_stream_ptr(stream)))
    if st != SDF_OK:
        raise SdfError(st, "sdf_compute_host")
    return dist_out, tri_out


def sdf_zslab(nz, part, parts):
    """(k0, nk): z-slab `part` of `parts` of a grid of nz slices (host only, no CUDA)."""
    k0, nk = C.c_int(0), C.c_int(0)
    st = lib().sdf_zslab(int(nz), int(part), int(parts), C.byref(k0), C.byref(nk))
    if st != SDF_OK:
        raise SdfError(st, "sdf_zslab")
    return k0.value, nk.value


def sdf_compute_zslab(mesh: Mesh, origin, h, dims, band, part, parts, dist_out=None, tri_out=None, stream=None):
    """Slab `part` of `parts` of the grid: returns (k0, dist [nk,ny,nx], tri [nk,ny,nx]) CUDA tensors."""
    torch = _torch()
    nx, ny, nz = (int(v) for v in dims)
    k0, nk = sdf_zslab(nz, part, parts)
    if dist_out is None:
        dist_out = torch.empty((nk, ny, nx), dtype=torch.float32, device="cuda")
    if tri_out is None:
        tri_out = torch.empty((nk, ny, nx), dtype=torch.int32, device="cuda")
    assert dist_out.is_cuda and tri_out.is_cuda and dist_out.is_contiguous() and tri_out.is_contiguous()
    assert dist_out.numel() == nx * ny * nk and tri_out.numel() == nx * ny * nk
    assert dist_out.dtype == torch.float32 and tri_out.dtype == torch.int32
    st = lib().sdf_compute_zslab(mesh.handle, _origin3(origin), float(h), nx, ny, nz, float(band), int(part), int(parts),
                                 C.c_void_p(dist_out.data_ptr()), C.c_void_p(tri_out.data_ptr()),
                                 C.c_void_p(_stream_ptr(stream)), None, None)
    if st != SDF_OK:
        raise SdfError(st, "sdf_compute_zslab")
    return k0, dist_out, tri_out


def sdf_closest_points(mesh: Mesh, origin, h, dims, tri, cp_out=None, stream=None):
    """Closest point on the winning triangle for every band cell: float32 [nz,ny,nx,3] CUDA tensor."""
    torch = _torch()
    nx, ny, nz = (int(v) for v in dims)
    assert tri.is_cuda and tri.is_contiguous() and tri.dtype == torch.int32 and tri.numel() == nx * ny * nz
    if cp_out is None:
        cp_out = torch.empty((nz, ny, nx, 3), dtype=torch.float32, device="cuda")
    assert cp_out.is_cuda and cp_out.is_contiguous() and cp_out.numel() == 3 * nx * ny * nz
    st = lib().sdf_closest_points(mesh.handle, _origin3(origin), float(h), nx, ny, nz, C.c_void_p(tri.data_ptr()),
                                  C.c_void_p(cp_out.data_ptr()), C.c_void_p(_stream_ptr(stream)))
    if st != SDF_OK:
        raise SdfError(st, "sdf_closest_points")
    return cp_out


def sdf_fill_interior(dist, band, stream=None):
    """PAPER.md:493 axis sweeps, in place on a device dist tensor [nz,ny,nx] written by sdf_compute."""
    assert dist.is_cuda and dist.is_contiguous() and dist.dim() == 3
    nz, ny, nx = (int(v) for v in dist.shape)
    st = lib().sdf_fill_interior(C.c_void_p(dist.data_ptr()), nx, ny, nz, float(band), C.c_void_p(_stream_ptr(stream)))
    if st != SDF_OK:
        raise SdfError(st, "sdf_fill_interior")
    return dist


def sdf_fill_interior_static(dist, band, stream=None):
    """sdf_fill_interior without any allocation: the scratch is a static 8 MiB device array (grids beyond it: SDF_ETOOBIG)."""
    assert dist.is_cuda and dist.is_contiguous() and dist.dim() == 3
    nz, ny, nx = (int(v) for v in dist.shape)
    st = lib().sdf_fill_interior_static(C.c_void_p(dist.data_ptr()), nx, ny, nz, float(band), C.c_void_p(_stream_ptr(stream)))
    if st != SDF_OK:
        raise SdfError(st, "sdf_fill_interior_static")
    return dist


def sdf_read_stl(path) -> np.ndarray:
    """Binary or ASCII STL file -> soup float32 [ntri,3,3] (a copy; the library's buffer is released)."""
    p = C.POINTER(C.c_float)()
    n = C.c_int64(0)
    st = lib().sdf_read_stl(str(path).encode(), C.byref(p), C.byref(n))
    if st != SDF_OK:
        raise SdfError(st, "sdf_read_stl")
    try:
        return np.ctypeslib.as_array(p, shape=(n.value, 3, 3)).copy()
    finally:
        lib().sdf_free_host(p)


def sdf_write_stl(path, soup, ascii=False):
    s = np.ascontiguousarray(soup, dtype=np.float32)
    st = lib().sdf_write_stl(str(path).encode(), C.c_void_p(s.ctypes.data), s.shape[0], 1 if ascii else 0)
    if st != SDF_OK:
        raise SdfError(st, "sdf_write_stl")


def sdf_write_grid(path, dist, tri, origin, h, band):
    """dist / tri: HOST arrays [nz,ny,nx] (tri may be None)."""
    d = np.ascontiguousarray(dist, dtype=np.float32)
    t = None if tri is None else np.ascontiguousarray(tri, dtype=np.int32)
    nz, ny, nx = d.shape
    st = lib().sdf_write_grid(str(path).encode(), C.c_void_p(d.ctypes.data), C.c_void_p(t.ctypes.data if t is not None else None),
                              _origin3(origin), float(h), nx, ny, nz, float(band))
    if st != SDF_OK:
        raise SdfError(st, "sdf_write_grid")


def sdf_stats(mesh: Mesh) -> dict:
    s = Stats()
    st = lib().sdf_stats(mesh.handle, C.byref(s))
    if st != SDF_OK:
        raise SdfError(st, "sdf_stats")
    return s.as_dict()


def sdf_get_table(mesh: Mesh, which: int) -> np.ndarray:
    s = sdf_stats(mesh)
    F, V, E = s["F"], s["V"], s["E"]
    shape_dtype = {
        TABLE_CORNER_VID: ((F, 3), np.int32), TABLE_HALFEDGE_ADJ: ((F, 3), np.int32),
        TABLE_FACE_NORMAL: ((F, 3), np.float32), TABLE_VERTEX_REC: ((V,), VERTEX_REC_DTYPE),
        TABLE_EDGE_REC: ((s["edges_convex"] + s["edges_concave"],), EDGE_REC_DTYPE), TABLE_VERTEX_MINTRI: ((V,), np.int32)}[which]
    out = np.empty(shape_dtype[0], dtype=shape_dtype[1])
    st = lib().sdf_get_table(mesh.handle, which, C.c_void_p(out.ctypes.data), out.nbytes)
    if st != SDF_OK:
        raise SdfError(st, "sdf_get_table")
    return out


def sdf_brick_count(mesh: Mesh, origin, h, dims, band, stream=None) -> int:
    """Number of 8x8x8 bricks the band reaches on this grid (sdf_compute_sparse with capacity 0: counts, writes nothing)."""
    _torch()
    o = (C.c_float * 3)(*[float(v) for v in origin])
    n = C.c_int64(0)
    st = lib().sdf_compute_sparse(mesh.handle, o, float(h), int(dims[0]), int(dims[1]), int(dims[2]), float(band), 0, None, None,
                                  None, C.byref(n), C.c_void_p(_stream_ptr(stream)))
    if st not in (SDF_OK, SDF_ENOMEM):
        raise SdfError(st, "sdf_compute_sparse")
    return int(n.value)


def sdf_compute_sparse(mesh: Mesh, origin, h, dims, band, brick_ids=None, dist_bricks=None, tri_bricks=None, stream=None):
    """Band-sparse output: (n, brick_ids int32[cap], dist_bricks float32[cap,512], tri_bricks int32[cap,512]).  Device tensors
    (allocated here for the exact count if not given) or pinned / plain CPU tensors (then the library stages and copies)."""
    torch = _torch()
    if dist_bricks is None:
        cap = sdf_brick_count(mesh, origin, h, dims, band, stream=stream)
        brick_ids = torch.empty((max(cap, 1),), dtype=torch.int32, device="cuda")
        dist_bricks = torch.empty((max(cap, 1), 512), dtype=torch.float32, device="cuda")
        tri_bricks = torch.empty((max(cap, 1), 512), dtype=torch.int32, device="cuda")
    cap = int(dist_bricks.shape[0])
    if not (brick_ids.dtype == torch.int32 and dist_bricks.dtype == torch.float32 and tri_bricks.dtype == torch.int32):
        raise TypeError("brick_ids / tri_bricks must be int32, dist_bricks float32")
    if not (brick_ids.is_contiguous() and dist_bricks.is_contiguous() and tri_bricks.is_contiguous()):
        raise ValueError("outputs must be contiguous")
    if brick_ids.numel() < cap or tri_bricks.shape != dist_bricks.shape or dist_bricks.shape[1] != 512:
        raise ValueError("outputs must be [cap], [cap,512], [cap,512]")
    on_dev = dist_bricks.is_cuda
    if brick_ids.is_cuda != on_dev or tri_bricks.is_cuda != on_dev:
        raise ValueError("outputs must live on the same side")
    o = (C.c_float * 3)(*[float(v) for v in origin])
    n = C.c_int64(0)
    fn = lib().sdf_compute_sparse if on_dev else lib().sdf_compute_sparse_host
    st = fn(mesh.handle, o, float(h), int(dims[0]), int(dims[1]), int(dims[2]), float(band), cap, C.c_void_p(brick_ids.data_ptr()),
            C.c_void_p(dist_bricks.data_ptr()), C.c_void_p(tri_bricks.data_ptr()), C.byref(n), C.c_void_p(_stream_ptr(stream)))
    if st != SDF_OK:
        raise SdfError(st, "sdf_compute_sparse")
    return int(n.value), brick_ids, dist_bricks, tri_bricks


def sdf_measure_fp32_peak(stream=None):
    """(TFLOP/s of an FMA loop on every SM, SM count): the FP32 leg of the roofline (measurement support)."""
    _torch()
    tf, sms = C.c_double(0.0), C.c_int(0)
    st = lib().sdf_measure_fp32_peak(C.byref(tf), C.byref(sms), C.c_void_p(_stream_ptr(stream)))
    if st != SDF_OK:
        raise SdfError(st, "sdf_measure_fp32_peak")
    return float(tf.value), int(sms.value)


def sdf_enable_timing(on):
    """0 / False: off; 1 / True: every stage; 2: only the dense sentinel write (SDF_T_FILL)."""
    lib().sdf_enable_timing(int(on))


def sdf_get_timings(mesh: Mesh) -> dict:
    """Stage durations (ms) of the handle's sdf_create and its last sdf_compute."""
    ms = (C.c_float * len(TIMING_STAGES))()
    st = lib().sdf_get_timings(mesh.handle, ms, len(TIMING_STAGES))
    if st != SDF_OK:
        raise SdfError(st, "sdf_get_timings")
    return {k: float(ms[i]) for i, k in enumerate(TIMING_STAGES)}


def sdf_launch_count() -> int:
    return int(lib().sdf_launch_count())


def sdf_destroy(mesh: Mesh):
    mesh.destroy()


def compute_workload(w, host_soup=False, stream=None):
    """Convenience for tests / bench: sdf_create + sdf_compute on a `Workload`."""
    torch = _torch()
    soup = w.soup if host_soup else torch.from_numpy(np.ascontiguousarray(w.soup)).cuda()
    m = sdf_create(soup, stream=stream)
    d, t = sdf_compute(m, w.origin, w.h, w.dims, w.band, stream=stream)
    return m, d, t

"""CPU-side tests (no GPU): the C-ABI library builds for sm_100a, loads, exports every
symbol include/sdf.h declares, and its host-side argument checks answer without a device."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1903_00353_b200 import build as b
    return C.CDLL(b.build_library())


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "sdf.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sdf_[a-z_0-9]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared_functions()
    assert {"sdf_create", "sdf_compute", "sdf_compute_host", "sdf_destroy", "sdf_stats"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n


def test_binding_export_list_matches_header():
    from paper_1903_00353_b200 import binding
    assert sorted(binding.EXPORTS) == _declared_functions()


def test_version_and_strerror(lib):
    lib.sdf_version.restype = C.c_int
    assert lib.sdf_version() >= 100
    lib.sdf_strerror.restype = C.c_char_p
    lib.sdf_strerror.argtypes = [C.c_int]
    msgs = [lib.sdf_strerror(i) for i in range(7)]
    assert len(set(msgs)) == 7 and all(m for m in msgs)
    assert b"unknown" in lib.sdf_strerror(99)


def test_argument_checks_without_device(lib):
    """Bad arguments are rejected before any CUDA call; a valid call without a device
    returns SDF_ECUDA (never a CPU fallback)."""
    lib.sdf_create.restype = C.c_int
    lib.sdf_create.argtypes = [C.c_void_p, C.c_int64, C.c_int, C.c_void_p, C.c_void_p, C.POINTER(C.c_void_p)]
    out = C.c_void_p(123)
    soup = np.zeros((4, 3, 3), dtype=np.float32)
    assert lib.sdf_create(None, 4, 0, None, None, C.byref(out)) == 1 and not out.value
    assert lib.sdf_create(soup.ctypes.data, 0, 0, None, None, C.byref(out)) == 1
    assert lib.sdf_create(soup.ctypes.data, -3, 0, None, None, C.byref(out)) == 1
    import torch
    if not torch.cuda.is_available():
        assert lib.sdf_create(soup.ctypes.data, 4, 0, None, None, C.byref(out)) == 6      # SDF_ECUDA
        assert not out.value
    lib.sdf_compute.restype = C.c_int
    lib.sdf_compute.argtypes = [C.c_void_p, C.c_void_p, C.c_float, C.c_int, C.c_int, C.c_int, C.c_float,
                                C.c_void_p, C.c_void_p, C.c_void_p]
    assert lib.sdf_compute(None, None, 0.1, 4, 4, 4, 0.3, None, None, None) == 1
    lib.sdf_get_timings.restype = C.c_int
    assert lib.sdf_get_timings(None, None, 7) == 1
    lib.sdf_destroy.argtypes = [C.c_void_p]
    lib.sdf_destroy(None)                                                                  # no-op


def test_product_does_not_import_oracle():
    """The product path never touches oracle/ (and the oracle never imports the product)."""
    pkg = os.path.join(ROOT, "paper_1903_00353_b200")
    for dp, _dn, fn in os.walk(pkg):
        for f in fn:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle", txt, flags=re.M), f
                assert "sdf_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_1903_00353_b200", txt, flags=re.M), f


def test_binding_fails_loudly_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("has a GPU")
    from paper_1903_00353_b200 import binding as B
    with pytest.raises(RuntimeError):
        B.sdf_create(np.zeros((4, 3, 3), dtype=np.float32))


def test_bench_reads_kernel_traffic_from_profiles():
    """bench.py takes roofline.traffic from the committed ncu summary (profiles/kernel_traffic.csv), not from a
    literal: the file must exist, parse, and hold the dense writer at the headline config."""
    import importlib.util
    spec = importlib.util.spec_from_file_location("bench_mod", os.path.join(ROOT, "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    t, src = bench.kernel_traffic("C4", "fill_tma_kernel")
    assert t is not None and 8.4e9 < t < 9.0e9 and src.startswith("profiles/kernel_traffic.csv")
    assert bench.kernel_traffic("C4", "no_such_kernel") == (None, None)
    assert set(bench.STAGE_KERNEL) == {"ingest_weld", "edges", "vertices", "clip_scan", "clear", "evaluate", "emit", "fill"}

"""Shared helpers of the GPU parity tests (not imported by the product)."""
from __future__ import annotations

import dataclasses

import numpy as np

from helpers import compare_to_oracle


def f32_grid(w):
    """Same workload with origin / h / band rounded to fp32 (what the C ABI receives), so
    the oracle and the CUDA path see bit-identical grid parameters."""
    o = tuple(float(np.float32(v)) for v in w.origin)
    return dataclasses.replace(w, origin=o, h=float(np.float32(w.h)), band=float(np.float32(w.band)))


def run_gpu(w, host_soup=False):
    from paper_1903_00353_b200 import binding as B
    m, d, t = B.compute_workload(w, host_soup=host_soup)
    stats = B.sdf_stats(m)
    return m, d.cpu().numpy(), t.cpu().numpy(), stats


def check_parity(w, oracle_mod, nthreads=None):
    """Full-grid element-by-element comparison under the four north_star clauses."""
    w = f32_grid(w)
    om = oracle_mod.Mesh(w.soup)
    d_ref, t_ref = om.sdf(w.origin, w.h, w.dims, w.band, nthreads)
    m, d_gpu, t_gpu, stats = run_gpu(w)
    res = compare_to_oracle(d_gpu, t_gpu, d_ref, t_ref, w, om)
    res["stats"] = stats
    assert stats["band_cells"] == res["populated_gpu"], (stats["band_cells"], res["populated_gpu"])
    return res

"""Host logic of the z-slab split (include/sdf.h sdf_zslab):
partition properties through the C ABI, and the N>1 path on CPU: world_size-2 / -3 gloo, every rank
takes its slab, the ranges are gathered and must tile the grid (no compute calls: no GPU here)."""
import os
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_partition_properties():
    from paper_1903_00353_b200 import binding as B
    rng = np.random.default_rng(11)
    cases = [(1, 1), (1, 4), (7, 2), (8, 2), (9, 2), (16, 2), (17, 3), (1024, 8), (1000, 7), (32767, 16), (64, 64)]
    cases += [(int(rng.integers(1, 5000)), int(rng.integers(1, 40))) for _ in range(200)]
    for nz, parts in cases:
        r = [B.sdf_zslab(nz, p, parts) for p in range(parts)]
        k = 0
        for k0, nk in r:                                            # ordered, disjoint, cover [0, nz)
            assert k0 == k and nk >= 0
            k += nk
        assert k == nz
        for k0, nk in r:                                            # cut on brick boundaries
            assert k0 % 8 == 0 or k0 == nz
            assert (k0 + nk) % 8 == 0 or k0 + nk == nz
        full = [nk for k0, nk in r if k0 + nk < nz and nk > 0]      # balanced to one brick
        if full:
            assert max(full) - min(full) <= 8
        nb = -(-nz // 8)
        assert max(nk for _, nk in r) <= 8 * -(-nb // parts)
    assert B.sdf_zslab(1024, 0, 1) == (0, 1024)


def test_partition_errors():
    from paper_1903_00353_b200 import binding as B
    for nz, part, parts in [(0, 0, 1), (-3, 0, 1), (8, 0, 0), (8, -1, 2), (8, 2, 2), (8, 5, 2)]:
        with pytest.raises(B.SdfError) as e:
            B.sdf_zslab(nz, part, parts)
        assert e.value.status == B.SDF_EINVAL


WORKER = r"""
import json, sys
import torch, torch.distributed as dist
sys.path.insert(0, %r)
from paper_1903_00353_b200 import binding as B
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
nz = 1000
k0, nk = B.sdf_zslab(nz, rank, world)
mine = torch.tensor([k0, nk, 100 * (rank + 1)], dtype=torch.int64)      # range + this rank's band cells
allr = [torch.zeros(3, dtype=torch.int64) for _ in range(world)]
dist.all_gather(allr, mine)
cells = mine[2:].clone()
dist.all_reduce(cells, op=dist.ReduceOp.SUM)                             # strong scaling: value sums the slabs
ms = torch.tensor([4.0 + rank], dtype=torch.float64)
dist.all_reduce(ms, op=dist.ReduceOp.MAX)
if rank == 0:
    print(json.dumps({"ranges": [[int(v) for v in t[:2]] for t in allr], "cells": int(cells.item()),
                      "ms": ms.item(), "world": world}))
dist.destroy_process_group()
"""


@pytest.mark.parametrize("world,port", [(2, 29631), (3, 29633)])
def test_slabs_tile_the_grid_gloo(tmp_path, world, port):
    import json
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(world),
                          "--master-addr", "127.0.0.1", "--master-port", str(port), str(script)],
                         capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    r = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
    assert r["world"] == world and r["ms"] == 4.0 + world - 1
    assert r["cells"] == 100 * world * (world + 1) // 2
    k = 0
    for k0, nk in r["ranges"]:
        assert k0 == k and nk > 0 and k0 % 8 == 0
        k += nk
    assert k == 1000

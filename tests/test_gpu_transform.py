"""sdf_transform (include/sdf.h) = sdf_create + sdf_compute, bit for bit, with the sentinel fill started under the
feature construction; checked against the two-call path and, through it, against the oracle's results."""
import numpy as np
import pytest
import torch

from paper_1903_00353_b200 import binding as B
from paper_1903_00353_b200 import workloads as W
from gpu_util import f32_grid
from helpers import compare_to_oracle

pytestmark = pytest.mark.gpu


def _both(w, **kw):
    m1 = B.sdf_create(torch.from_numpy(np.ascontiguousarray(w.soup)).cuda())
    d1, t1 = B.sdf_compute(m1, w.origin, w.h, w.dims, w.band)
    m2, d2, t2 = B.sdf_transform(torch.from_numpy(np.ascontiguousarray(w.soup)).cuda(), w.origin, w.h, w.dims, w.band, **kw)
    torch.cuda.synchronize()
    return (m1, d1, t1), (m2, d2, t2)


@pytest.mark.parametrize("name,scale", [("C1", 1.0), ("C2", 0.5), ("C3", 0.25), ("C4", 0.125)])
def test_transform_equals_two_calls(name, scale):
    w = W.config(name, scale)
    (m1, d1, t1), (m2, d2, t2) = _both(w)
    assert torch.equal(t1, t2)
    assert torch.equal(d1.view(torch.int32), d2.view(torch.int32))
    s1, s2 = B.sdf_stats(m1), B.sdf_stats(m2)
    assert all(s1[k] == s2[k] for k in ("V", "E", "F", "band_cells", "edges_convex", "edges_concave"))
    # the handle is a full one: a second grid through sdf_compute
    d3, t3 = B.sdf_compute(m2, w.origin, w.h, w.dims, w.band)
    assert torch.equal(t3, t1)
    m1.destroy(); m2.destroy()


@pytest.mark.parametrize("name", ["C4", "C5"])
def test_transform_equals_two_calls_full_size(name):
    """BASELINE.json's full sizes, the call bench.py times: identical to sdf_create + sdf_compute, whose
    results tests/test_gpu_fullsize.py checks against the oracle."""
    w = W.config(name)
    (m1, d1, t1), (m2, d2, t2) = _both(w)
    assert torch.equal(t1, t2)
    assert torch.equal(d1.view(torch.int32), d2.view(torch.int32))
    assert B.sdf_stats(m1)["band_cells"] == B.sdf_stats(m2)["band_cells"] == int((t2 >= 0).sum())
    m1.destroy(); m2.destroy()


@pytest.mark.parametrize("hoist", ["0", "1"])
def test_transform_brick_hoist_switch(hoist, monkeypatch):
    monkeypatch.setenv("SDF_HOIST_BRICKS", hoist)
    w = W.config("C2", 0.5)
    (m1, d1, t1), (m2, d2, t2) = _both(w)
    assert torch.equal(t1, t2) and torch.equal(d1.view(torch.int32), d2.view(torch.int32))
    m1.destroy(); m2.destroy()


@pytest.mark.parametrize("at", ["1", "2", "3", "4"])
def test_transform_fill_start_points(at, monkeypatch):
    """SDF_PREFILL_AT ablation: wherever the sentinel fill starts, the result is the two-call one, bit for bit."""
    monkeypatch.setenv("SDF_PREFILL_AT", at)
    w = W.config("C3", 0.25)
    (m1, d1, t1), (m2, d2, t2) = _both(w)
    assert torch.equal(t1, t2) and torch.equal(d1.view(torch.int32), d2.view(torch.int32))
    assert int(torch.isfinite(d2).sum()) == B.sdf_stats(m2)["band_cells"] > 0
    m1.destroy(); m2.destroy()


def test_transform_against_oracle(oracle_mod):
    for w in (W.config("C1"), W.config("C3", 0.125)):
        w = f32_grid(w)
        om = oracle_mod.Mesh(w.soup)
        d_ref, t_ref = om.sdf(w.origin, w.h, w.dims, w.band, None)
        m, d, t = B.sdf_transform(w.soup, w.origin, w.h, w.dims, w.band)      # host soup
        torch.cuda.synchronize()
        res = compare_to_oracle(d.cpu().numpy(), t.cpu().numpy(), d_ref, t_ref, w, om)
        assert res["ok"], {k: res[k] for k in res if k != "stats"}
        assert res["populated_gpu"] > 0
        m.destroy()


def test_transform_unaligned_outputs_and_side_stream():
    w = W.config("C2", 0.25)
    nx, ny, nz = w.dims
    n = nx * ny * nz
    bd = torch.empty(n + 1, dtype=torch.float32, device="cuda")[1:].view(nz, ny, nx)
    bt = torch.empty(n + 1, dtype=torch.int32, device="cuda")[1:].view(nz, ny, nx)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        (m1, d1, t1), (m2, d2, t2) = _both(w, dist_out=bd, tri_out=bt, stream=st)
    assert torch.equal(t1, t2) and torch.equal(d1.view(torch.int32), d2.view(torch.int32))
    m1.destroy(); m2.destroy()


def test_transform_errors_leave_no_handle():
    w = W.config("C1")
    soup = np.array(w.soup, copy=True)
    with pytest.raises(B.SdfError):                       # open surface
        B.sdf_transform(soup[:-1], w.origin, w.h, w.dims, w.band)
    with pytest.raises(B.SdfError):                       # bad grid: checked before any work
        B.sdf_transform(soup, w.origin, -1.0, w.dims, w.band)
    soup[0, 0, 0] = np.nan
    with pytest.raises(B.SdfError):
        B.sdf_transform(soup, w.origin, w.h, w.dims, w.band)
    torch.cuda.synchronize()


def test_two_host_threads_on_two_streams():
    """include/sdf.h: distinct handles on distinct streams are independent (the library's side streams are shared, its
    events pooled): two host threads run sdf_transform / sdf_compute_sparse / destroy in a loop, each on its own stream
    and workload; every result must equal the one the same call gives alone, bit for bit."""
    import threading
    from paper_1903_00353_b200 import binding as B
    ws = [f32_grid(W.config("C2", 0.5)), f32_grid(W.config("C3", 0.3)), f32_grid(W.config("C5", 0.08))]
    ref = []
    for w in ws:                                          # also creates the library-wide state (first calls: serial)
        m, d, t = B.compute_workload(w)
        torch.cuda.synchronize()
        ref.append((d.clone(), t.clone()))
        m.destroy()
    errors = []

    def worker(idx):
        try:
            w = ws[idx]
            st = torch.cuda.Stream()
            soup = torch.from_numpy(np.ascontiguousarray(w.soup)).cuda()
            torch.cuda.synchronize()
            for it in range(12):
                with torch.cuda.stream(st):
                    m, d, t = B.sdf_transform(soup, w.origin, w.h, w.dims, w.band, stream=st)
                    nb, ids, sd, stt = B.sdf_compute_sparse(m, w.origin, w.h, w.dims, w.band, stream=st)
                st.synchronize()
                if not (torch.equal(d.view(torch.int32), ref[idx][0].view(torch.int32)) and torch.equal(t, ref[idx][1])):
                    errors.append((idx, it, "dense"))
                if int(torch.isfinite(sd[:nb]).sum()) != int(torch.isfinite(ref[idx][0]).sum()):
                    errors.append((idx, it, "sparse"))
                m.destroy()
        except Exception as e:                            # noqa: BLE001 -- reported through the list
            errors.append((idx, repr(e)))

    threads = [threading.Thread(target=worker, args=(i,)) for i in range(len(ws))]
    for th in threads:
        th.start()
    for th in threads:
        th.join(timeout=120)
    assert not any(th.is_alive() for th in threads)
    torch.cuda.synchronize()
    assert not errors, errors[:5]

"""STL reader / writer and grid writer.  Host code:
runs without a GPU.  Files written here with plain Python are read back by the library and the
other way round."""
import struct

import numpy as np
import pytest

from paper_1903_00353_b200 import binding as B
from paper_1903_00353_b200 import workloads as W


def _soup():
    v, t = W.icosphere_mesh(1, 0.7)
    return W.soup_from_indexed(v + 0.013, t, np.random.default_rng(3))


def _write_binary(path, soup, header=b"made by the test"):
    with open(path, "wb") as f:
        f.write(header.ljust(80, b"\0"))
        f.write(struct.pack("<I", soup.shape[0]))
        for T in soup:
            f.write(struct.pack("<12fH", 0.0, 0.0, 0.0, *T.reshape(-1).tolist(), 0))


def _write_ascii(path, soup):
    with open(path, "w") as f:
        f.write("solid test\n")
        for T in soup:
            f.write("  facet normal 0 0 0\n    outer loop\n")
            for p in T:
                f.write("      vertex %s %s %s\n" % tuple(repr(float(c)) for c in p))
            f.write("    endloop\n  endfacet\n")
        f.write("endsolid test\n")


def test_read_binary_and_ascii(tmp_path):
    soup = _soup()
    _write_binary(tmp_path / "b.stl", soup)
    _write_ascii(tmp_path / "a.stl", soup)
    assert np.array_equal(B.sdf_read_stl(tmp_path / "b.stl"), soup)
    assert np.array_equal(B.sdf_read_stl(tmp_path / "a.stl"), soup)
    # a binary file whose header starts with "solid" is still binary
    _write_binary(tmp_path / "s.stl", soup, header=b"solid but binary")
    assert np.array_equal(B.sdf_read_stl(tmp_path / "s.stl"), soup)


@pytest.mark.parametrize("ascii_", [False, True])
def test_write_then_read_round_trip(tmp_path, ascii_):
    soup = _soup()
    p = tmp_path / "w.stl"
    B.sdf_write_stl(p, soup, ascii=ascii_)
    assert np.array_equal(B.sdf_read_stl(p), soup)              # 9 significant digits round-trip fp32
    raw = open(p, "rb").read()
    if ascii_:
        txt = raw.decode()
        assert txt.startswith("solid") and txt.count("vertex") == 3 * soup.shape[0]
        # facet normals written = unit normals of the counter-clockwise vertex order
        n0 = np.array([float(x) for x in txt.split("facet normal")[1].split("\n")[0].split()])
        ref = np.cross(soup[0, 1].astype(np.float64) - soup[0, 0], soup[0, 2].astype(np.float64) - soup[0, 0])
        assert np.allclose(n0, ref / np.linalg.norm(ref), atol=1e-7)
    else:
        assert len(raw) == 84 + 50 * soup.shape[0] and struct.unpack("<I", raw[80:84])[0] == soup.shape[0]


def test_bad_files(tmp_path):
    with pytest.raises(B.SdfError) as e:
        B.sdf_read_stl(tmp_path / "missing.stl")
    assert e.value.status == B.SDF_EIO
    soup = _soup()
    _write_binary(tmp_path / "b.stl", soup)
    raw = open(tmp_path / "b.stl", "rb").read()
    open(tmp_path / "trunc.stl", "wb").write(raw[:-7])
    with pytest.raises(B.SdfError) as e:
        B.sdf_read_stl(tmp_path / "trunc.stl")
    assert e.value.status == B.SDF_EIO
    open(tmp_path / "two.stl", "w").write("solid x\nfacet normal 0 0 1\nouter loop\nvertex 0 0 0\nvertex 1 0 0\nendloop\nendfacet\nendsolid x\n")
    with pytest.raises(B.SdfError) as e:
        B.sdf_read_stl(tmp_path / "two.stl")
    assert e.value.status == B.SDF_EIO
    open(tmp_path / "empty.stl", "wb").write(b"")
    with pytest.raises(B.SdfError) as e:
        B.sdf_read_stl(tmp_path / "empty.stl")
    assert e.value.status == B.SDF_EIO


def test_write_grid(tmp_path):
    rng = np.random.default_rng(0)
    d = rng.standard_normal((3, 4, 5)).astype(np.float32)
    d[0, 0, 0] = np.inf
    t = rng.integers(-1, 9, size=(3, 4, 5)).astype(np.int32)
    B.sdf_write_grid(tmp_path / "g.bin", d, t, (-1.0, 0.5, 2.0), 0.25, 0.75)
    raw = open(tmp_path / "g.bin", "rb").read()
    assert raw[:8] == b"SDFGRID1"
    nx, ny, nz, has = struct.unpack("<4i", raw[8:24])
    ox, oy, oz, h, band = struct.unpack("<5f", raw[24:44])
    assert (nx, ny, nz, has) == (5, 4, 3, 1) and (ox, oy, oz, h, band) == (-1.0, 0.5, 2.0, 0.25, 0.75)
    n = nx * ny * nz
    assert np.array_equal(np.frombuffer(raw[44:44 + 4 * n], dtype=np.float32).reshape(3, 4, 5), d)
    assert np.array_equal(np.frombuffer(raw[44 + 4 * n:], dtype=np.int32).reshape(3, 4, 5), t)
    B.sdf_write_grid(tmp_path / "g2.bin", d, None, (0, 0, 0), 1.0, 1.0)
    assert len(open(tmp_path / "g2.bin", "rb").read()) == 44 + 4 * n

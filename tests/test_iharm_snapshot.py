"""iharm3d-layout snapshot reader.  The paper's dump is not in the container, so a
synthetic dump in that layout is written and read back; libhdf5 / h5py are not in the image either, so the container
format is checked against the HDF5 file-format facts retyped here (signatures, superblock fields, the root
symbol-table entry), not against the library."""
import os
import struct
import sys

import numpy as np
import pytest

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from paper_2602_13198_b200 import iharm_snapshot as ih, workloads as wl  # noqa: E402


@pytest.fixture(scope="module")
def small():
    return wl.config3(Ns=2e3, n1=24, n2=16, n3=8)


def test_round_trip_double_is_bit_exact_and_extra_primitives_are_dropped(small, tmp_path):
    p, prim = small
    f = str(tmp_path / "dump_f64.h5")
    ih.write_iharm_dump(f, p, prim, t=1234.5, dtype=np.float64, extra_prims=2)
    grid, pr = ih.read_iharm_dump(f)
    assert pr.dtype == np.float64 and pr.shape == (24, 16, 8, 8) and pr.flags["C_CONTIGUOUS"]
    assert np.array_equal(pr, prim)
    for k in ("n1", "n2", "n3", "a_spin", "hslope", "gam_ad"):
        assert grid[k] == p[k], k
    assert grid["startx"] == list(p["startx"]) and grid["dx"] == list(p["dx"]) and grid["metric_kind"] == 1
    tree = ih.read_hdf5(f)
    assert float(tree["t"]) == 1234.5 and tree["prims"].shape[-1] == 10
    assert [s.decode() for s in tree["header"]["prim_names"][:8]] == list(ih.PRIM_NAMES)
    assert int(tree["header"]["has_electrons"]) == 1 and bytes(tree["header"]["metric"]) == b"MKS"


def test_single_precision_dump_as_iharm3d_writes_them(small, tmp_path):
    p, prim = small
    f = str(tmp_path / "dump_f32.h5")
    ih.write_iharm_dump(f, p, prim)                        # float32 /prims
    _, pr = ih.read_iharm_dump(f)
    assert pr.dtype == np.float64
    assert np.array_equal(pr, prim.astype(np.float32).astype(np.float64))
    p2, pr2 = ih.params_from_dump(f, p)
    assert p2["Ns_target"] == p["Ns_target"] and p2["n3"] == 8 and np.array_equal(pr2, pr)


def test_container_bytes_follow_the_hdf5_format(small, tmp_path):
    """Superblock version 0: signature, 8-byte offsets/lengths, end-of-file address = file size, root symbol-table
    entry (cache type 1) pointing at a version-1 object header whose symbol-table message names a TREE and a HEAP."""
    p, prim = small
    f = str(tmp_path / "dump.h5")
    ih.write_iharm_dump(f, p, prim, dtype=np.float64)
    b = open(f, "rb").read()
    assert b[:8] == b"\x89HDF\r\n\x1a\n" and b[8] == 0 and b[13] == 8 and b[14] == 8
    base, free, eof, drv = struct.unpack_from("<4Q", b, 24)
    assert base == 0 and free == 2**64 - 1 and drv == 2**64 - 1 and eof == len(b)
    name_off, hdr, cache = struct.unpack_from("<QQI", b, 56)
    bt, hp = struct.unpack_from("<QQ", b, 56 + 24)
    assert name_off == 0 and cache == 1 and b[hdr] == 1 and b[bt:bt + 4] == b"TREE" and b[hp:hp + 4] == b"HEAP"
    nmsg, = struct.unpack_from("<H", b, hdr + 2)
    mtype, msize = struct.unpack_from("<HH", b, hdr + 16)
    assert nmsg == 1 and mtype == 0x11 and msize == 16 and struct.unpack_from("<QQ", b, hdr + 24) == (bt, hp)
    # the B-tree's only child is a symbol-table node with the three root links in name order
    used, = struct.unpack_from("<H", b, bt + 6)
    child, = struct.unpack_from("<Q", b, bt + 24 + 8)
    assert used == 1 and b[child:child + 4] == b"SNOD" and struct.unpack_from("<H", b, child + 6)[0] == 3
    # /prims is stored contiguously: its bytes appear verbatim, 8-byte aligned
    at = b.find(prim.tobytes())
    assert at > 0 and at % 8 == 0


def test_unsupported_files_are_refused_not_guessed(small, tmp_path):
    p, prim = small
    f = str(tmp_path / "dump.h5")
    ih.write_iharm_dump(f, p, prim, dtype=np.float64)
    b = bytearray(open(f, "rb").read())
    bad = str(tmp_path / "bad.h5")
    for patch, what in (((0, b"\x88"), "signature"), ((8, b"\x02"), "superblock version"), ((13, b"\x04"), "offsets")):
        c = bytearray(b)
        c[patch[0]:patch[0] + 1] = patch[1]
        open(bad, "wb").write(c)
        with pytest.raises(ih.UnsupportedHDF5, match=what):
            ih.read_hdf5(bad)
    # a dump in another coordinate system, or without /prims
    tree = ih.read_hdf5(f)
    tree["header"]["metric"] = np.bytes_("FMKS")
    ih.write_hdf5(bad, tree)
    with pytest.raises(ih.UnsupportedHDF5, match="FMKS"):
        ih.read_iharm_dump(bad)
    tree["header"]["metric"] = np.bytes_("MKS")
    del tree["prims"]
    ih.write_hdf5(bad, tree)
    with pytest.raises(ih.UnsupportedHDF5, match="prims"):
        ih.read_iharm_dump(bad)


def test_generic_trees_nested_groups_and_scalar_types(tmp_path):
    tree = {"a": {"b": {"c": np.arange(5, dtype=np.int32), "d": np.float32(2.5)}, "s": np.bytes_("hello")},
            "u": np.arange(6, dtype=np.uint64).reshape(2, 3), "many": {"k%02d" % i: np.float64(i) for i in range(40)}}
    f = str(tmp_path / "t.h5")
    ih.write_hdf5(f, tree)
    r = ih.read_hdf5(f)
    assert np.array_equal(r["a"]["b"]["c"], tree["a"]["b"]["c"]) and r["a"]["b"]["c"].dtype == np.int32
    assert float(r["a"]["b"]["d"]) == 2.5 and bytes(r["a"]["s"]) == b"hello"
    assert np.array_equal(r["u"], tree["u"]) and r["u"].dtype == np.uint64
    assert sorted(r["many"]) == sorted(tree["many"]) and float(r["many"]["k39"]) == 39.0


def test_oracle_run_on_the_snapshot_equals_the_run_on_the_grid(small, tmp_path):
    from oracle_binding import Oracle
    p, prim = small
    f = str(tmp_path / "dump.h5")
    ih.write_iharm_dump(f, p, prim, dtype=np.float64)
    p2, prim2 = ih.params_from_dump(f, p)
    a = Oracle(p, prim); a.prepare(); a.run()
    b = Oracle(p2, prim2); b.prepare(); b.run()
    for x, y in zip(a.tally(), b.tally()):
        assert np.array_equal(x, y)


@pytest.mark.gpu
def test_cuda_path_runs_from_a_snapshot_file(small, tmp_path):
    """The same through the C-ABI: a run on the snapshot read from disk equals the run on the generated grid
    (superphoton counts per bin equal, sums to rounding of the atomics' order) and matches the oracle's counts."""
    import torch
    from oracle_binding import Oracle
    from paper_2602_13198_b200 import binding as gm
    p, prim = small
    f = str(tmp_path / "dump.h5")
    ih.write_iharm_dump(f, p, prim, dtype=np.float64)
    p2, prim2 = ih.params_from_dump(f, p)
    res = []
    for pp, gr in ((p, prim), (p2, prim2)):
        g = gm.GPUMonty(pp)
        g.set_grid(torch.from_numpy(gr).cuda())
        g.prepare(); g.run()
        res.append(g.tally())
        g.close()
    assert np.array_equal(res[0][3], res[1][3])
    m = res[0][0] > 0
    assert np.max(np.abs(res[1][0][m] / res[0][0][m] - 1)) < 1e-12
    o = Oracle(p2, prim2); o.prepare(); o.run()
    assert np.array_equal(o.tally()[3], res[1][3])

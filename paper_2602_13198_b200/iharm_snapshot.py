"""Reader (and a writer for synthetic test files) of iharm3d-style GRMHD snapshots (PAPER.md:272-288:
GPUmonty reads the fluid from an iharm3d dump, 288x128x128 in the paper's Sec. 4.3).

An iharm3d dump is an HDF5 file whose fluid state is the dataset `/prims`, shape [N1][N2][N3][NPRIM] with the first
eight primitives RHO, UU, U1, U2, U3, B1, B2, B3 in code units, and whose grid is described by scalar datasets under
`/header` (`n1 n2 n3 gam metric`) and `/header/geom` (`startx1..3 dx1..3`, and `mks/a`, `mks/hslope` for the modified
Kerr-Schild map theta(x2) = pi x2 + (1 - hslope)/2 sin(2 pi x2) -- the map of DESIGN.md G28).  That is exactly the
library's input: `prim[n1][n2][n3][8]` fp64 + `startx, dx, a_spin, hslope, gam_ad`.

Neither h5py nor libhdf5 is in this image, so the HDF5 container is parsed here, for the subset a dump written with
the library's default (earliest) format uses: superblock version 0 or 1, version-1 object headers with continuation
blocks, symbol-table groups (version-1 B-tree + local heap), contiguous or compact datasets of little-endian
fixed-point / IEEE floating-point / fixed-length string types, simple or scalar dataspaces.  Chunked or filtered
datasets, new-style groups (superblock 2+) and variable-length strings are reported as unsupported, not guessed.
The snapshot of the paper is not in the container: the tests write a synthetic dump in this layout with
`write_iharm_dump` and read it back (the parser is exercised against this module's own writer only -- stated in
DESIGN.md as unverified against libhdf5).

Host-side I/O only: no arithmetic of the method lives here.
"""
from __future__ import annotations

import struct

import numpy as np

_SIG = b"\x89HDF\r\n\x1a\n"
_UNDEF = 0xFFFFFFFFFFFFFFFF


class UnsupportedHDF5(ValueError):
    pass


# ======================================================================================================
# reading
# ======================================================================================================
class _Reader:
    def __init__(self, buf: bytes):
        self.b = buf
        if buf[:8] != _SIG:
            raise UnsupportedHDF5("not an HDF5 file (signature at offset 0 expected)")
        ver = buf[8]
        if ver not in (0, 1):
            raise UnsupportedHDF5(f"superblock version {ver}: only the earliest file format (0/1) is read here")
        if buf[13] != 8 or buf[14] != 8:
            raise UnsupportedHDF5("offsets and lengths must be 8 bytes")
        off = 24 if ver == 0 else 28                       # version 1 inserts indexed-storage K + 2 reserved bytes
        self.base, _free, _eof, _drv = struct.unpack_from("<4Q", buf, off)
        entry = off + 32                                   # root group symbol-table entry
        self.root_header = struct.unpack_from("<Q", buf, entry + 8)[0]

    # ---- object headers (version 1) ------------------------------------------------------------------
    def messages(self, addr: int):
        b = self.b
        a = self.base + addr
        if b[a] != 1:
            raise UnsupportedHDF5(f"object header version {b[a]} at {addr}: only version 1 is read here")
        nmsg, = struct.unpack_from("<H", b, a + 2)
        size, = struct.unpack_from("<I", b, a + 8)
        blocks = [(a + 16, size)]
        out = []
        while blocks and len(out) < nmsg:
            p, left = blocks.pop(0)
            end = p + left
            while p + 8 <= end and len(out) < nmsg:
                mtype, msize, _flags = struct.unpack_from("<HHB", b, p)
                data = b[p + 8:p + 8 + msize]
                p += 8 + msize
                if mtype == 0x0010:                        # continuation block
                    coff, clen = struct.unpack_from("<QQ", data, 0)
                    blocks.append((self.base + coff, clen))
                out.append((mtype, data))
        return out

    # ---- groups ---------------------------------------------------------------------------------------
    def _heap_name(self, heap_data: int, off: int) -> str:
        e = self.b.index(b"\0", heap_data + off)
        return self.b[heap_data + off:e].decode("ascii")

    def _btree_entries(self, addr: int, heap_data: int, out: dict):
        b = self.b
        a = self.base + addr
        if b[a:a + 4] == b"SNOD":
            n, = struct.unpack_from("<H", b, a + 6)
            for i in range(n):
                name_off, hdr = struct.unpack_from("<QQ", b, a + 8 + 40 * i)
                out[self._heap_name(heap_data, name_off)] = hdr
            return
        if b[a:a + 4] != b"TREE":
            raise UnsupportedHDF5(f"group node at {addr}: neither TREE nor SNOD")
        ntype, _level, used = struct.unpack_from("<BBH", b, a + 4)
        if ntype != 0:
            raise UnsupportedHDF5("B-tree of a chunked dataset where a group tree was expected")
        p = a + 24                                         # after the two sibling addresses
        for i in range(used):
            child, = struct.unpack_from("<Q", b, p + 8 + 16 * i)   # key_i (8), child_i (8), ...
            self._btree_entries(child, heap_data, out)

    def children(self, msgs) -> dict | None:
        for mtype, data in msgs:
            if mtype == 0x0011:                            # symbol table message: B-tree + local heap
                btree, heap = struct.unpack_from("<QQ", data, 0)
                h = self.base + heap
                if self.b[h:h + 4] != b"HEAP":
                    raise UnsupportedHDF5("local heap signature missing")
                heap_data = self.base + struct.unpack_from("<Q", self.b, h + 24)[0]
                out: dict = {}
                self._btree_entries(btree, heap_data, out)
                return out
        return None

    # ---- datasets -------------------------------------------------------------------------------------
    @staticmethod
    def _dtype(data: bytes):
        cls, ver = data[0] & 0x0F, data[0] >> 4
        bits0 = data[1]
        size, = struct.unpack_from("<I", data, 4)
        if ver not in (1, 2, 3):
            raise UnsupportedHDF5(f"datatype message version {ver}")
        if cls in (0, 1) and (bits0 & 1):
            raise UnsupportedHDF5("big-endian data")
        if cls == 0:
            return np.dtype(("<i" if bits0 & 0x08 else "<u") + str(size))
        if cls == 1:
            if size not in (4, 8):
                raise UnsupportedHDF5(f"{size}-byte floating point")
            return np.dtype("<f" + str(size))
        if cls == 3:
            return np.dtype("S" + str(size))
        raise UnsupportedHDF5(f"datatype class {cls} (only integers, IEEE floats and fixed-length strings)")

    @staticmethod
    def _shape(data: bytes):
        ver, rank, flags = data[0], data[1], data[2]
        if ver == 1:
            p = 8
        elif ver == 2:
            p = 4
        else:
            raise UnsupportedHDF5(f"dataspace message version {ver}")
        return tuple(struct.unpack_from("<%dQ" % rank, data, p)) if rank else ()

    def dataset(self, msgs):
        dt = shape = None
        raw = None
        for mtype, data in msgs:
            if mtype == 0x0001:
                shape = self._shape(data)
            elif mtype == 0x0003:
                dt = self._dtype(data)
            elif mtype == 0x000B:
                raise UnsupportedHDF5("filtered (compressed) dataset")
            elif mtype == 0x0008:
                ver = data[0]
                if ver != 3:
                    raise UnsupportedHDF5(f"data layout message version {ver}")
                cls = data[1]
                if cls == 1:
                    addr, nbytes = struct.unpack_from("<QQ", data, 2)
                    raw = b"" if addr == _UNDEF else (self.base + addr, nbytes)
                elif cls == 0:
                    n, = struct.unpack_from("<H", data, 2)
                    raw = bytes(data[4:4 + n])
                else:
                    raise UnsupportedHDF5("chunked dataset (iharm3d writes contiguous ones)")
        if dt is None or shape is None or raw is None:
            return None
        count = int(np.prod(shape, dtype=np.int64)) if shape else 1
        if isinstance(raw, tuple):
            arr = np.frombuffer(self.b, dtype=dt, count=count, offset=raw[0])
        else:
            arr = np.frombuffer(raw, dtype=dt, count=count) if raw else np.zeros(count, dt)
        return arr.reshape(shape)

    def tree(self, addr: int | None = None):
        msgs = self.messages(self.root_header if addr is None else addr)
        kids = self.children(msgs)
        if kids is not None:
            return {name: self.tree(h) for name, h in kids.items()}
        return self.dataset(msgs)


def read_hdf5(path: str) -> dict:
    """The whole file as nested dicts (groups) of numpy arrays (datasets; scalars are 0-d arrays)."""
    with open(path, "rb") as f:
        buf = f.read()
    return _Reader(buf).tree()


# ======================================================================================================
# writing (the same subset: what the tests and synthetic workloads need)
# ======================================================================================================
_LEAF_K, _INTERNAL_K = 32, 16                              # up to 64 links per group in one symbol-table node


def _pad8(b: bytes) -> bytes:
    return b + b"\0" * (-len(b) % 8)


def _msg(mtype: int, data: bytes) -> bytes:
    data = _pad8(data)
    return struct.pack("<HHB3x", mtype, len(data), 0) + data


def _dtype_msg(dt: np.dtype) -> bytes:
    if dt.kind == "f":
        prec, eloc, esz, msz, bias, b1 = {4: (32, 23, 8, 23, 127, 0x1F), 8: (64, 52, 11, 52, 1023, 0x3F)}[dt.itemsize]
        return struct.pack("<BBBBI", 0x11, 0x20, b1, 0, dt.itemsize) + struct.pack("<HHBBBBI", 0, prec, eloc, esz, 0, msz, bias)
    if dt.kind in "iu":
        return struct.pack("<BBBBI", 0x10, 0x08 if dt.kind == "i" else 0, 0, 0, dt.itemsize) + struct.pack("<HH", 0, 8 * dt.itemsize)
    if dt.kind == "S":
        return struct.pack("<BBBBI", 0x13, 0, 0, 0, dt.itemsize)
    raise UnsupportedHDF5(f"cannot write dtype {dt}")


class _Writer:
    def __init__(self):
        self.buf = bytearray(96)                           # superblock, filled in last

    def alloc(self, data: bytes) -> int:
        self.buf += b"\0" * (-len(self.buf) % 8)
        a = len(self.buf)
        self.buf += data
        return a

    def header(self, msgs: list[bytes]) -> int:
        body = b"".join(msgs)
        return self.alloc(struct.pack("<BxHII4x", 1, len(msgs), 1, len(body)) + body)

    def dataset(self, value) -> int:
        arr = np.asarray(value)
        if arr.dtype.kind == "U":
            arr = arr.astype("S")
        if arr.dtype.kind in "fiu" and arr.dtype.byteorder == ">":
            arr = arr.astype(arr.dtype.newbyteorder("<"))
        if arr.dtype == np.bool_:
            arr = arr.astype(np.int32)
        raw = np.ascontiguousarray(arr).tobytes()
        addr = self.alloc(raw) if raw else _UNDEF
        space = struct.pack("<BBBx4x", 1, arr.ndim, 0) + struct.pack("<%dQ" % arr.ndim, *arr.shape)
        fill = struct.pack("<BBBB", 2, 1, 0, 0)            # version 2, early allocation, no fill value defined
        layout = struct.pack("<BBQQ", 3, 1, addr, len(raw))
        return self.header([_msg(0x0001, space), _msg(0x0003, _dtype_msg(arr.dtype)), _msg(0x0005, fill), _msg(0x0008, layout)])

    def group(self, tree: dict):
        """-> (object header address, B-tree address, local heap address)"""
        names = sorted(tree)                               # links are kept in name order
        if len(names) > 2 * _LEAF_K:
            raise UnsupportedHDF5("more links in one group than one symbol-table node holds")
        entries = []
        for n in names:
            v = tree[n]
            if isinstance(v, dict):
                h, bt, hp = self.group(v)
                entries.append((n, h, 1, struct.pack("<QQ", bt, hp)))
            else:
                entries.append((n, self.dataset(v), 0, b"\0" * 16))
        heap = bytearray(8)                                # offset 0: the empty name
        offs = []
        for n in names:
            offs.append(len(heap))
            heap += _pad8(n.encode("ascii") + b"\0")
        heap_data = self.alloc(bytes(heap))
        heap_addr = self.alloc(b"HEAP" + struct.pack("<B3xQQQ", 0, len(heap), 1, heap_data))
        snod = bytearray(b"SNOD" + struct.pack("<BxH", 1, len(names)))
        for (n, h, cache, scratch), o in zip(entries, offs):
            snod += struct.pack("<QQI4x", o, h, cache) + scratch
        snod += b"\0" * (8 + 2 * _LEAF_K * 40 - len(snod))
        snod_addr = self.alloc(bytes(snod))
        node = bytearray(b"TREE" + struct.pack("<BBHQQ", 0, 0, 1 if names else 0, _UNDEF, _UNDEF))
        node += struct.pack("<QQQ", 0, snod_addr, offs[-1] if offs else 0)
        node += b"\0" * (24 + (2 * _INTERNAL_K + 1) * 8 + 2 * _INTERNAL_K * 8 - len(node))
        bt_addr = self.alloc(bytes(node))
        hdr = self.header([_msg(0x0011, struct.pack("<QQ", bt_addr, heap_addr))])
        return hdr, bt_addr, heap_addr

    def finish(self, tree: dict) -> bytes:
        hdr, bt, hp = self.group(tree)
        sb = _SIG + struct.pack("<BBBxBBBxHHI", 0, 0, 0, 0, 8, 8, _LEAF_K, _INTERNAL_K, 0)
        sb += struct.pack("<QQQQ", 0, _UNDEF, len(self.buf), _UNDEF)
        sb += struct.pack("<QQI4xQQ", 0, hdr, 1, bt, hp)
        assert len(sb) == 96
        self.buf[:96] = sb
        return bytes(self.buf)


def write_hdf5(path: str, tree: dict) -> None:
    """Nested dicts of array-likes -> an HDF5 file in the earliest file format (contiguous datasets)."""
    with open(path, "wb") as f:
        f.write(_Writer().finish(tree))


# ======================================================================================================
# the iharm3d layout
# ======================================================================================================
PRIM_NAMES = ("RHO", "UU", "U1", "U2", "U3", "B1", "B2", "B3")


def write_iharm_dump(path: str, p: dict, prim: np.ndarray, t: float = 0.0, dtype=np.float32, extra_prims: int = 0) -> None:
    """A synthetic dump in the iharm3d layout from a library parameter dict and its fluid grid (iharm3d itself
    stores /prims in single precision; `extra_prims` appends electron-entropy-like columns a reader must skip)."""
    n1, n2, n3 = int(p["n1"]), int(p["n2"]), int(p["n3"])
    pr = np.asarray(prim, dtype=np.float64).reshape(n1, n2, n3, 8)
    if extra_prims:
        pr = np.concatenate([pr, np.zeros((n1, n2, n3, extra_prims))], axis=-1)
    names = list(PRIM_NAMES) + ["KEL%d" % i for i in range(extra_prims)]
    r_in, r_out = np.exp(p["startx"][1]), np.exp(p["startx"][1] + n1 * p["dx"][1])
    tree = {
        "t": np.float64(t),
        "prims": pr.astype(dtype),
        "header": {
            "version": np.bytes_("iharm-layout-synthetic"), "metric": np.bytes_("MKS"),
            "n1": np.int32(n1), "n2": np.int32(n2), "n3": np.int32(n3), "n_prim": np.int32(pr.shape[-1]),
            "gam": np.float64(p["gam_ad"]), "has_electrons": np.int32(1 if extra_prims else 0),
            "prim_names": np.array(names, dtype="S"),
            "geom": {
                "n_dim": np.int32(4),
                "startx1": np.float64(p["startx"][1]), "startx2": np.float64(p["startx"][2]), "startx3": np.float64(p["startx"][3]),
                "dx1": np.float64(p["dx"][1]), "dx2": np.float64(p["dx"][2]), "dx3": np.float64(p["dx"][3]),
                "mks": {"a": np.float64(p["a_spin"]), "hslope": np.float64(p["hslope"]),
                        "r_in": np.float64(r_in), "r_out": np.float64(r_out)},
            },
        },
    }
    write_hdf5(path, tree)


def read_iharm_dump(path: str):
    """-> (grid, prim): grid = the parameter-dict entries the snapshot fixes (n1 n2 n3 startx dx a_spin hslope gam_ad
    metric_kind), prim = float64 [n1][n2][n3][8] (RHO UU U1 U2 U3 B1 B2 B3, code units); extra primitives are dropped."""
    f = read_hdf5(path)
    try:
        h, g = f["header"], f["header"]["geom"]
        metric = bytes(h["metric"]).decode("ascii").strip("\0 ").upper()
        if metric not in ("MKS", "MMKS"):
            raise UnsupportedHDF5(f"coordinate system {metric!r}: only the MKS map theta = pi x2 + (1-hslope)/2 sin(2 pi x2) "
                                  "(DESIGN.md G28) is tracked; FMKS needs its polynomial polar map")
        mk = g["mks"] if "mks" in g else g["mmks"]
        n1, n2, n3 = int(h["n1"]), int(h["n2"]), int(h["n3"])
        grid = dict(n1=n1, n2=n2, n3=n3, metric_kind=1, a_spin=float(mk["a"]), hslope=float(mk["hslope"]),
                    gam_ad=float(h["gam"]),
                    startx=[0.0, float(g["startx1"]), float(g["startx2"]), float(g["startx3"])],
                    dx=[1.0, float(g["dx1"]), float(g["dx2"]), float(g["dx3"])])
        pr = f["prims"]
    except KeyError as e:
        raise UnsupportedHDF5(f"not an iharm3d dump: {e} missing") from None
    if pr.ndim != 4 or pr.shape[:3] != (n1, n2, n3) or pr.shape[3] < 8:
        raise UnsupportedHDF5(f"/prims has shape {pr.shape}, header says {(n1, n2, n3)} x >= 8 primitives")
    return grid, np.ascontiguousarray(pr[..., :8], dtype=np.float64)


def params_from_dump(path: str, base: dict):
    """Library parameters for a run on the snapshot: `base` (units, sampling, bias, bins, N_s) with the grid entries
    replaced by the snapshot's."""
    grid, prim = read_iharm_dump(path)
    p = dict(base)
    p.update(grid)
    return p, prim

"""ctypes front end of the C data oracle (oracle/reshard_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this.  It marshals numpy arrays into the
oracle's C entry points; all arithmetic is in the C file, which follows PAPER.md:78-88.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_LIB = None

OR_OK, OR_EINVAL, OR_ESPEC, OR_EDIVIS = 0, 1, 2, 3
_ERR = {OR_EINVAL: "invalid argument", OR_ESPEC: "bad sharding spec", OR_EDIVIS: "dim not divisible by degree"}


class OracleError(ValueError):
    def __init__(self, code):
        super().__init__("oracle: " + _ERR.get(code, "error %d" % code))
        self.code = code


def lib():
    global _LIB
    if _LIB is None:
        path = _build.build()
        _LIB = C.CDLL(path)
        _LIB.oracle_num_devices.restype = C.c_int64
        for name in ("oracle_local_shape", "oracle_device_box", "oracle_shard_from_global",
                     "oracle_element_source", "reshard_oracle_device", "reshard_oracle",
                     "oracle_max_threads"):
            getattr(_LIB, name).restype = C.c_int
    return _LIB


def _i64(xs):
    return (C.c_int64 * len(xs))(*[int(x) for x in xs])


def _i32(xs):
    return (C.c_int32 * len(xs))(*[int(x) for x in xs])


def _chk(rc):
    if rc != OR_OK:
        raise OracleError(rc)


def num_devices(mesh):
    return int(lib().oracle_num_devices(_i32(mesh), len(mesh)))


def local_shape(shape, mesh, spec):
    out = (C.c_int64 * len(shape))()
    _chk(lib().oracle_local_shape(_i64(shape), len(shape), _i32(mesh), len(mesh), spec.encode(), out))
    return tuple(out)


def device_box(shape, mesh, spec, r):
    lo = (C.c_int64 * len(shape))()
    hi = (C.c_int64 * len(shape))()
    _chk(lib().oracle_device_box(_i64(shape), len(shape), _i32(mesh), len(mesh), spec.encode(),
                                 C.c_int64(r), lo, hi))
    return tuple(lo), tuple(hi)


def shard_from_global(D, mesh, spec, r, pad=0):
    """shard of device r: the oracle's own statement of the layout; padded local
    shape (R5), padding elements = `pad`."""
    D = np.ascontiguousarray(D)
    shape = D.shape
    out = np.zeros(local_shape(shape, mesh, spec), dtype=D.dtype)
    if pad:
        out.view(np.uint8)[...] = pad
    _chk(lib().oracle_shard_from_global(_i64(shape), len(shape), D.dtype.itemsize, _i32(mesh), len(mesh),
                                        spec.encode(), C.c_int64(r), C.c_void_p(D.ctypes.data),
                                        C.c_void_p(out.ctypes.data)))
    return out


def shards_from_global(D, mesh, spec, pad=0):
    return [shard_from_global(D, mesh, spec, r, pad) for r in range(num_devices(mesh))]


def element_source(shape, src_mesh, src_spec, dst_mesh, dst_spec, q, j):
    """(source device, source local linear index, global linear index) of dst element (q, j)."""
    dev, lin, g = C.c_int64(), C.c_int64(), C.c_int64()
    _chk(lib().oracle_element_source(_i64(shape), len(shape), _i32(src_mesh), len(src_mesh), src_spec.encode(),
                                     _i32(dst_mesh), len(dst_mesh), dst_spec.encode(),
                                     C.c_int64(q), C.c_int64(j), C.byref(dev), C.byref(lin), C.byref(g)))
    return dev.value, lin.value, g.value


def _ptr_array(arrs):
    return (C.c_void_p * len(arrs))(*[a.ctypes.data for a in arrs])


def reshard_device(shape, elem_bytes, src_mesh, src_spec, dst_mesh, dst_spec, src_shards, q, dtype,
                   n_threads=1, out=None):
    """destination shard of device q computed by the oracle from host source shards."""
    if out is None:
        out = np.zeros(local_shape(shape, dst_mesh, dst_spec), dtype=dtype)
    assert out.flags.c_contiguous and out.dtype.itemsize == elem_bytes
    for s in src_shards:
        assert s.flags.c_contiguous
    _chk(lib().reshard_oracle_device(_i64(shape), len(shape), int(elem_bytes),
                                     _i32(src_mesh), len(src_mesh), src_spec.encode(),
                                     _i32(dst_mesh), len(dst_mesh), dst_spec.encode(),
                                     _ptr_array(src_shards), C.c_int64(q), C.c_void_p(out.ctypes.data),
                                     int(n_threads)))
    return out


def reshard(shape, src_mesh, src_spec, dst_mesh, dst_spec, src_shards, n_threads=1, fill=0):
    """the whole task: list of destination shards, one per dst device.  Padding bytes of
    the destination shards (R5) keep the byte value `fill`: the oracle never writes them."""
    dtype = src_shards[0].dtype
    lshape = local_shape(shape, dst_mesh, dst_spec)
    outs = [np.zeros(lshape, dtype=dtype) for _ in range(num_devices(dst_mesh))]
    if fill:
        for o in outs:
            o.view(np.uint8)[...] = fill
    for s in src_shards:
        assert s.flags.c_contiguous and s.dtype == dtype
    _chk(lib().reshard_oracle(_i64(shape), len(shape), dtype.itemsize,
                              _i32(src_mesh), len(src_mesh), src_spec.encode(),
                              _i32(dst_mesh), len(dst_mesh), dst_spec.encode(),
                              _ptr_array(src_shards), _ptr_array(outs), int(n_threads)))
    return outs


def max_threads():
    """host cores the oracle can really use (sched affinity), for the cpu_baseline report."""
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:  # pragma: no cover
        return int(lib().oracle_max_threads())

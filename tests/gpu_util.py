"""helpers of the -m gpu parity tests: device buffers (torch is only memory + streams here),
shards cut with the ORACLE's boxes, calls through the C ABI binding."""
import numpy as np
import torch

from oracle import data_oracle as do
from paper_2211_05322_b200 import inputs
from paper_2211_05322_b200 import reshard as rs

_TORCH_CT = {1: torch.uint8, 2: torch.int16, 4: torch.int32, 8: torch.int64}


def dev():
    return torch.device("cuda:0")


def to_dev(a):
    """numpy array (any itemsize, incl. 16-byte void) -> device uint8 tensor of its bytes"""
    return torch.from_numpy(np.ascontiguousarray(a).view(np.uint8).reshape(-1).copy()).to(dev())


def ptrs(ts):
    return [t.data_ptr() for t in ts]


def stream():
    return torch.cuda.current_stream().cuda_stream


def oracle_slices(shape, mesh, spec):
    """per device the torch/numpy basic-slicing index of its box, from the oracle's device_box"""
    out = []
    for r in range(do.num_devices(mesh)):
        lo, hi = do.device_box(shape, mesh, spec, r)
        out.append(tuple(slice(l, h) for l, h in zip(lo, hi)))
    return out


def padded(D, idx, local, fill=0):
    """the shard buffer of one device: dense, padded local shape (R5), D[idx] at its origin, every
    padding byte = fill"""
    box = D[idx]
    if tuple(box.shape) == tuple(local):
        return box.contiguous()
    out = torch.empty(tuple(local), dtype=D.dtype, device=D.device)
    out.view(torch.uint8).fill_(fill)
    out[tuple(slice(0, n) for n in box.shape)] = box
    return out


def device_shards_from_global(D, mesh, spec, fill=0):
    """D: device tensor of the global shape -> list of dense (padded) device shards (oracle boxes)"""
    local = do.local_shape(tuple(D.shape), mesh, spec)
    return [padded(D, idx, local, fill) for idx in oracle_slices(tuple(D.shape), mesh, spec)]


def run_small(shape, np_dtype, sm, ss, dm, ds, flags=0, seed=1, src_offset=0, dst_offset=0, opts=None):
    """execute on the GPU and return (plan, got dst shards as numpy, oracle dst shards as numpy).
    src_offset / dst_offset: bytes every shard pointer is moved by (an int, or a function of the device index, < 64)"""
    e = np.dtype(np_dtype).itemsize
    rng = np.random.default_rng(seed)
    D = np.frombuffer(rng.bytes(int(np.prod(shape)) * e), dtype=np_dtype).reshape(shape)
    src = do.shards_from_global(D, sm, ss)
    want = do.reshard(shape, sm, ss, dm, ds, src, fill=0xA5)      # padding (R5) must come back untouched
    p = rs.Plan(shape, e, sm, ss, dm, ds, flags, opts)
    src_d = [torch.zeros(s.nbytes + 64, dtype=torch.uint8, device=dev()) for s in src]
    so = [src_offset(r) if callable(src_offset) else src_offset for r in range(len(src))]
    do_ = [dst_offset(q) if callable(dst_offset) else dst_offset for q in range(len(want))]
    for t, s, o in zip(src_d, src, so):
        t[o:o + s.nbytes] = to_dev(s)
    dst_d = [torch.full((want[0].nbytes + 64,), 0xA5, dtype=torch.uint8, device=dev()) for _ in want]
    p.execute([t.data_ptr() + o for t, o in zip(src_d, so)], [t.data_ptr() + o for t, o in zip(dst_d, do_)], stream())
    torch.cuda.synchronize()
    got = []
    for t, w, o in zip(dst_d, want, do_):
        raw = t.cpu().numpy()
        assert (raw[:o] == 0xA5).all() and (raw[o + w.nbytes:] == 0xA5).all(), "wrote outside the shard"
        got.append(raw[o:o + w.nbytes].view(np_dtype).reshape(w.shape))
    return p, got, want


def workload_on_device(w):
    """(D on device in its container dtype, src shards, expected dst shards) for a named workload;
    expected = basic slicing of D with the oracle's destination boxes."""
    D = inputs.global_tensor_torch(w, dev())
    src = device_shards_from_global(D, w.src_mesh, w.src_spec)
    return D, src

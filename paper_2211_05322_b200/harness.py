"""Device-buffer plumbing shared by bench.py and __graft_entry__.smoke(): torch is used for device
memory and streams only.  Shards are cut from the seeded global tensor with the LIBRARY's own
boxes (reshard_plan_device_box); none of the method's arithmetic lives here."""
import torch

from . import inputs
from . import reshard as rs


def make_plan(w, flags=0, tuning=None):
    """tuning: dict of rs_tuning fields (A/B runs of bench.py), None = the library's launch shapes"""
    return rs.Plan(w.shape, inputs.elem_bytes(w.dtype), w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec, flags,
                   dict(tuning=tuning) if tuning else None)


def device_inputs(w, plan, device):
    """(D, src shards) on `device`; shard r = D[box_r] at the origin of a dense buffer of the padded
    local shape (zero padding when the partition is uneven), in the container dtype."""
    D = inputs.global_tensor_torch(w, device)
    local = plan.local_shape(rs.RS_SRC)
    src = []
    for r in range(plan.info.n_src):
        lo, hi = plan.device_box(rs.RS_SRC, r)
        box = D[tuple(slice(a, b) for a, b in zip(lo, hi))]
        if tuple(box.shape) == tuple(local):
            src.append(box.contiguous())
        else:
            t = torch.zeros(local, dtype=D.dtype, device=device)
            t[tuple(slice(0, n) for n in box.shape)] = box
            src.append(t)
    return D, src


def device_outputs(plan, like, device, fill=None):
    out = [torch.empty(plan.local_shape(rs.RS_DST), dtype=like.dtype, device=device) for _ in range(plan.info.n_dst)]
    if fill is not None:
        for t in out:
            t.view(torch.uint8).fill_(fill)
    return out


def ptrs(ts):
    return [t.data_ptr() for t in ts]

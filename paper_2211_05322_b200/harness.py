"""Device-buffer plumbing shared by bench.py and __graft_entry__.smoke(): torch is used for device
memory and streams only.  Shards are cut from the seeded global tensor with the LIBRARY's own
boxes (reshard_plan_device_box); none of the method's arithmetic lives here."""
import torch

from . import inputs
from . import reshard as rs


def make_plan(w, flags=0):
    return rs.Plan(w.shape, inputs.elem_bytes(w.dtype), w.src_mesh, w.src_spec, w.dst_mesh, w.dst_spec, flags)


def device_inputs(w, plan, device):
    """(D, src shards) on `device`; shard r = D[box_r].contiguous() in the container dtype."""
    D = inputs.global_tensor_torch(w, device)
    src = []
    for r in range(plan.info.n_src):
        lo, hi = plan.device_box(rs.RS_SRC, r)
        src.append(D[tuple(slice(a, b) for a, b in zip(lo, hi))].contiguous())
    return D, src


def device_outputs(plan, like, device, fill=None):
    out = [torch.empty(plan.local_shape(rs.RS_DST), dtype=like.dtype, device=device) for _ in range(plan.info.n_dst)]
    if fill is not None:
        for t in out:
            t.view(torch.uint8).fill_(fill)
    return out


def ptrs(ts):
    return [t.data_ptr() for t in ts]

"""N > 1 plumbing of bench.py.  The path does not shard across real GPUs (S8: "replicas
only"): every rank runs the same task on its own device, there is no data-path collective; the only
communication is the barrier around the timed region and the max-over-ranks of the device time."""
import torch
import torch.distributed as dist


def init(backend, device=None):
    """process group from the torchrun environment (RANK / WORLD_SIZE / MASTER_ADDR / MASTER_PORT)."""
    if dist.is_initialized():
        return
    if backend == "nccl":
        dist.init_process_group("nccl", device_id=device)
    else:
        dist.init_process_group(backend)


def world():
    return dist.get_world_size() if dist.is_initialized() else 1


def barrier(sync=None):
    if world() > 1:
        dist.barrier()
    if sync is not None:
        sync()


def max_over_ranks(ms, device="cpu"):
    """slowest rank's time: the job is as slow as its slowest replica."""
    if world() == 1:
        return float(ms)
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_gbs(bytes_per_rank, ms, n_ranks):
    """whole-job throughput: all ranks' bytes over the max-over-ranks time."""
    return n_ranks * bytes_per_rank / (ms * 1e-3) / 1e9


def shutdown():
    if dist.is_initialized():
        dist.destroy_process_group()

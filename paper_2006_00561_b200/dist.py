"""Multi-process plumbing for bench.py: one process per GPU, torch.distributed for barrier / max / sum only.

The path does not shard across GPUs in this build ("replicas only"): every rank runs an
independent replica of the whole simulation, there is no data-path collective.  The helpers work with the
`nccl` backend on CUDA tensors and with `gloo` on CPU tensors (the latter is what the CPU tests exercise)."""
import os


class Group:
    def __init__(self, rank=0, world=1, local_rank=0, backend=None):
        self.rank, self.world, self.local_rank, self.backend = rank, world, local_rank, backend

    @property
    def is_main(self):
        return self.rank == 0


def init_from_env(backend=None, device_kind="cuda"):
    """Reads RANK / WORLD_SIZE / LOCAL_RANK / MASTER_ADDR / MASTER_PORT (torchrun).  world == 1 -> no process group."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", str(rank)))
    if world == 1:
        return Group(0, 1, local_rank, None)
    import torch.distributed as dist
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29531")
    if backend is None:
        backend = "nccl" if device_kind == "cuda" else "gloo"
    if device_kind == "cuda":
        import torch
        torch.cuda.set_device(local_rank)
    if not dist.is_initialized():
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return Group(rank, world, local_rank, backend)


def _tensor(g, values, dtype):
    import torch
    dev = "cuda" if g.backend == "nccl" else "cpu"
    return torch.tensor(values, dtype=dtype, device=dev)


def barrier(g):
    if g.world > 1:
        import torch.distributed as dist
        if g.backend == "nccl":
            import torch
            dist.barrier(device_ids=[torch.cuda.current_device()])
        else:
            dist.barrier()


def max_over_ranks(g, x):
    if g.world == 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = _tensor(g, [float(x)], torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(g, x):
    if g.world == 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = _tensor(g, [float(x)], torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def aggregate_throughput(g, units_this_rank, seconds_this_rank):
    """whole-job value = units all ranks processed / max-over-ranks time (bench.py contract)"""
    total = sum_over_ranks(g, units_this_rank)
    tmax = max_over_ranks(g, seconds_this_rank)
    return total / tmax, total, tmax


def shutdown(g):
    if g.world > 1:
        import torch.distributed as dist
        if dist.is_initialized():
            dist.destroy_process_group()

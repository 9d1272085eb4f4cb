"""Multi-process plumbing: one process per GPU; torch.distributed for the barrier / max / sum of bench.py's timing and
for the three exchanges of the partitioned redistribution (include/pa_b200.h "multi-GPU"):
all-gather of the ranks' weight sums, all-gather of their offspring totals, all-to-all-v of contiguous lattice
slices.  Every kernel runs in the library; this module only moves bytes between ranks.  The helpers work with the
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


# ---------------------------------------------------------------------------------------------------
# partitioned redistribution: rank = partition
# ---------------------------------------------------------------------------------------------------
def all_gather_doubles(g, values):
    """every rank contributes len(values) doubles; returns a (world, len(values)) nested list in rank order"""
    if g.world == 1:
        return [list(map(float, values))]
    import torch
    import torch.distributed as dist
    mine = _tensor(g, [float(v) for v in values], torch.float64)
    out = [torch.empty_like(mine) for _ in range(g.world)]
    dist.all_gather(out, mine)
    return [[float(x) for x in t.tolist()] for t in out]


def exchange_slices(g, send, recv, counts, unit, with_self=True):
    """all-to-all-v of contiguous slices.  send / recv: 1-D tensors (uint8 bytes or int32 words) on this rank; counts[src][dst]
    = items src sends to dst; one item = `unit` tensor elements.  Rank r's slices leave `send` in destination order and
    arrive in `recv` in source order (global child order is source-rank order, so `recv` ends up in global order).
    Point-to-point operations in one batch: the same code runs on NCCL (one group call) and on gloo.
    with_self = False (a step with theta > 0 after pa_dist_pack): counts[me][me] items are skipped on both sides."""
    me, W = g.rank, g.world
    s_off = [0] * (W + 1)
    r_off = [0] * (W + 1)
    for p in range(W):  # with_self = False: the rank's own share is in neither buffer (the sweep's load gathers it)
        own = p == me and not with_self
        s_off[p + 1] = s_off[p] + (0 if own else int(counts[me][p]) * unit)
        r_off[p + 1] = r_off[p] + (0 if own else int(counts[p][me]) * unit)
    if counts[me][me] and with_self:
        recv[r_off[me]:r_off[me + 1]].copy_(send[s_off[me]:s_off[me + 1]])
    if W == 1:
        return
    import torch.distributed as dist
    # gloo moves host memory only: device slices are staged through the host (the slices that cross a rank boundary,
    # nothing else).  This is the path for several ranks on ONE GPU and for machines without NCCL; with NCCL the device
    # buffers are handed over as they are.
    staged = g.backend == "gloo" and send.is_cuda
    ops, landing = [], []
    for p in range(W):
        if p == me:
            continue
        if counts[me][p]:
            out = send[s_off[p]:s_off[p + 1]]
            ops.append(dist.P2POp(dist.isend, out.cpu() if staged else out, p))
        if counts[p][me]:
            dst = recv[r_off[p]:r_off[p + 1]]
            if staged:
                import torch
                host = torch.empty(dst.shape, dtype=dst.dtype, device="cpu")
                landing.append((dst, host))
                ops.append(dist.P2POp(dist.irecv, host, p))
            else:
                ops.append(dist.P2POp(dist.irecv, dst, p))
    if ops:
        for req in dist.batch_isend_irecv(ops):
            req.wait()
    for dst, host in landing:
        dst.copy_(host)


class ShardedAnnealer:
    """One rank's shard of a multi-GPU population annealing run, or -- with `emulate` ranks -- all ranks of such a run on
    ONE device, stepped phase by phase in lock-step by the host (no kernel ever waits on another rank's kernel, so this
    is safe on one GPU; it is how the device path is parity-tested where only one GPU is available)."""

    def __init__(self, L, R0, seed=0, beta0=0.0, capacity=0, policy=0, block=0, maxexc=0, group=None, emulate=None, flags=0,
                 bonds=None):
        """bonds: (Jx, Jy) packed coupling planes of a +-J sample (binding.PopulationAnnealer.set_bonds); every rank
        sets the same sample"""
        from . import binding
        self._b = binding
        self.policy, self.block, self.maxexc = policy, block, maxexc
        self.L, self.S = L, L * L // 8
        if emulate:
            self.g, self.world = Group(), int(emulate)
            ranks = range(self.world)
        else:
            self.g = group if group is not None else Group()
            self.world = self.g.world
            ranks = [self.g.rank]
        self.shards = [binding.PopulationAnnealer(L, R0, seed=seed, beta0=beta0, capacity=capacity, policy=policy, block=block,
                                                  maxexc=maxexc, rank=r, world=self.world, flags=flags) for r in ranks]
        if bonds is not None:
            for s in self.shards:
                s.set_bonds(bonds[0], bonds[1])
        self.emulated = bool(emulate)
        self.last_T = None

    @property
    def R_local(self):
        return [s.R for s in self.shards]

    def step(self, beta_next, theta):
        b = self._b
        partials = [s.dist_begin(beta_next, theta) for s in self.shards]
        if self.emulated:
            all_partials = partials
        else:
            rows = all_gather_doubles(self.g, [partials[0][0], float(partials[0][1])])
            all_partials = [(r[0], int(r[1])) for r in rows]
        T_local = [s.dist_resample(all_partials) for s in self.shards]
        caps_local = [s.dist_capacity() for s in self.shards]
        if self.emulated:
            T_all, caps = T_local, caps_local
        else:  # the offspring total travels with the rank's capacity: every rank can judge every rank's share
            rows = all_gather_doubles(self.g, [float(T_local[0]), float(caps_local[0])])
            T_all, caps = [int(r[0]) for r in rows], [int(r[1]) for r in rows]
        R_all = [int(p[1]) for p in all_partials]
        try:
            # Every rank evaluates the same plan and the same check of EVERY rank's share (capacity of that rank, empty
            # share) on the same gathered numbers, before anything is exchanged: all ranks refuse the step or none does.
            ns, base, counts = b.exchange_plan(T_all, self.policy, self.block, self.maxexc)
            if theta > 0:
                b.plan_check(ns, caps, base, R_all)
            else:
                b.plan_check(ns, caps)
            # theta > 0: only the children that leave a rank are gathered into its send buffer; the rest of the new
            # population is gathered from the parents by the sweep's load in dist_finish, as in the one-GPU step
            with_self = [s.dist_pack(T_all) for s in self.shards][0]
        except b.PaError:
            for s in self.shards:
                s.dist_abort()
            raise
        S = self.S
        if self.emulated:
            bufs = [s.dist_buffers() for s in self.shards]
            for src in range(self.world):
                s_off = 0
                for dst in range(self.world):
                    n = int(counts[src][dst])
                    if src == dst and not with_self:
                        continue
                    if n:
                        r_off = int(sum(counts[q][dst] for q in range(src) if with_self or q != dst))
                        bufs[dst][1][r_off * S:(r_off + n) * S].copy_(bufs[src][0][s_off * S:(s_off + n) * S])
                    s_off += n
        else:
            children, population = self.shards[0].dist_buffers()
            # The exchange is issued on torch's current stream (the local copy directly, NCCL through req.wait()); the
            # library works on the shard's own stream.  When the two differ, order them explicitly in both directions:
            # the exchange must see what dist_pack enqueued, dist_finish must not start before the receives have landed.
            lib_stream, cur = self.shards[0].stream, None
            if population.is_cuda:
                import torch
                cur = torch.cuda.current_stream(population.device)
                if cur != lib_stream:
                    cur.wait_stream(lib_stream)
                if self.g.backend == "nccl" and self.world > 1:
                    lib_stream.synchronize()  # NCCL runs on its own stream: hand it finished buffers
            exchange_slices(self.g, children, population, counts, S, with_self=with_self)
            if cur is not None and cur != lib_stream:
                lib_stream.wait_stream(cur)
        self.last_T, self.last_counts, self.last_new_start = T_all, counts, ns
        return [s.dist_finish(T_all) for s in self.shards]

    def log_Z(self):
        return self.shards[0].log_Z()

    def gather_spins(self):
        """emulation only: the whole population in global slot order"""
        import numpy as np
        return np.concatenate([s.spins() for s in self.shards], axis=0)

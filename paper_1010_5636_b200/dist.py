"""Communication callbacks of the domain decomposition (include/nd_b200.h, "domain decomposition"; csrc/shard.cu) on top of
torch.distributed: one process per GPU, NCCL send/recv over NVLink for the two half-spinor faces of every stencil application,
all-reduce for the reductions.  Plumbing only: what is sent is packed, and what is received is consumed, by the library's kernels.

    ctx = Context(local_dims, ...); ctx.set_gauge(U[:, t_begin:t_begin + t_local])
    comm = TorchDistComm(ctx)            # after torch.distributed.init_process_group("nccl")
    ... every operator call on ctx now acts on the global lattice ...
"""
import torch
import torch.distributed as dist


def ring_neighbours(rank, world):
    """(previous, next) rank along x0: the time direction is a ring (the boundary condition sits in the faces' phase)."""
    return (rank - 1) % world, (rank + 1) % world


def exchange_ops(send_next, send_prev, recv_prev, recv_next, rank, world, group=None):
    """The four point-to-point operations of one face exchange, in an order that matches between any two ranks (with two ranks
    the previous and the next neighbour are the same peer: its first send pairs with our first receive)."""
    prev, nxt = ring_neighbours(rank, world)
    return [dist.P2POp(dist.isend, send_next, nxt, group, tag=0), dist.P2POp(dist.isend, send_prev, prev, group, tag=1),
            dist.P2POp(dist.irecv, recv_prev, prev, group, tag=0), dist.P2POp(dist.irecv, recv_next, nxt, group, tag=1)]


class TorchDistComm:
    """Registers NCCL-backed callbacks on `ctx` (nd_set_sharding) for the calling rank of the default (or given) process group."""

    def __init__(self, ctx, group=None):
        self.ctx, self.group = ctx, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.reqs = []
        ctx.set_sharding(self.rank, self.world, self.start, self.wait, self.allreduce)
        if self.world > 1:
            nbytes = ctx.halo_bytes()
            self.bufs = [ctx.wrap_device_memory(p, nbytes, ctx.real_dtype) for p in ctx.halo_buffers()]

    def start(self, send_next, send_prev, recv_prev, recv_next, nbytes):
        with torch.cuda.stream(self.ctx.stream):          # NCCL orders its work after what the context has enqueued
            self.reqs = dist.batch_isend_irecv(exchange_ops(*self.bufs, self.rank, self.world, self.group))

    def wait(self):
        with torch.cuda.stream(self.ctx.stream):          # ... and the context's stream waits for the transfers
            for r in self.reqs:
                r.wait()
        self.reqs = []

    def allreduce(self, d_buf, n):
        t = self.ctx.wrap_device_memory(d_buf, 8 * n, torch.float64)
        with torch.cuda.stream(self.ctx.stream):
            dist.all_reduce(t, group=self.group)


class PeerComm(TorchDistComm):
    """Peer-to-peer face exchange (nd_set_halo_peers): the receive windows live in a symmetric-memory allocation that every rank
    of the node maps (torch.distributed._symmetric_memory: CUDA IPC / fabric handles over NVLink), the library's pack kernel
    stores each face straight into the neighbour's window, and `wait` is the allocation's device-side barrier enqueued on the
    context's stream - no NCCL call on the stencil's path; reductions still go through all_reduce.  One node only."""

    def __init__(self, ctx, group=None):
        super().__init__(ctx, group)
        if self.world > 1:
            import torch.distributed._symmetric_memory as symm_mem

            g = group if group is not None else dist.group.WORLD
            with torch.cuda.stream(ctx.stream):
                self.window = symm_mem.empty(4 * ctx.halo_bytes(), dtype=torch.uint8, device=ctx.torch_device)
                self.window.zero_()
            self.handle = symm_mem.rendezvous(self.window, g)
            ptrs = window_pointers(list(self.handle.buffer_ptrs), self.rank, self.world)
            ctx.set_halo_peers(*ptrs)

    def start(self, *a):                                   # never called in peer-to-peer mode
        raise RuntimeError("PeerComm: the exchange-start callback must not be called while peer windows are set")

    def wait(self):
        with torch.cuda.stream(self.ctx.stream):
            self.handle.barrier()


def window_pointers(all_windows, rank, world):
    """(own, next rank's, previous rank's) receive window out of the per-rank list of a symmetric allocation."""
    prev, nxt = ring_neighbours(rank, world)
    return all_windows[rank], all_windows[nxt], all_windows[prev]

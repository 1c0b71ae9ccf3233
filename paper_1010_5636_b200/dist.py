"""Communication callbacks of the domain decomposition (include/nd_b200.h, "domain decomposition"; csrc/shard.cu) on top of
torch.distributed: one process per GPU, NCCL send/recv over NVLink for the two half-spinor faces of every stencil application,
all-reduce for the reductions.  Plumbing only: what is sent is packed, and what is received is consumed, by the library's kernels.

    ctx = Context(local_dims, ...); ctx.set_gauge(U[:, t_begin:t_begin + t_local])
    comm, kind = make_comm(ctx, p2p=True)   # after torch.distributed.init_process_group("nccl"); p2p falls back to NCCL
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


class CommSetupError(RuntimeError):
    """A collective set-up step failed on at least one rank; raised on EVERY rank of the group (see run_agreed)."""


def run_agreed(stage, what, device, group=None):
    """Run `stage()` on every rank and make the outcome unanimous: the ranks exchange a success flag (all_reduce MIN) after
    the stage, so either all return its value or all raise CommSetupError - no rank walks into the next collective alone
    after a peer has given up, which is how a failed set-up turns into a hang."""
    err, val = None, None
    try:
        val = stage()
    except Exception as e:                                   # noqa: BLE001 - whatever went wrong is reported, then agreed on
        err = f"{type(e).__name__}: {e}"
    ok = torch.tensor([0 if err else 1], dtype=torch.int32, device=device)
    dist.all_reduce(ok, op=dist.ReduceOp.MIN, group=group)
    if int(ok.item()) == 0:
        raise CommSetupError(f"{what}: {err or 'failed on another rank'}")
    return val


class PeerComm(TorchDistComm):
    """Peer-to-peer face exchange (nd_set_halo_peers): the receive windows live in a symmetric-memory allocation that every rank
    of the node maps (torch.distributed._symmetric_memory: CUDA IPC / fabric handles over NVLink), the library's pack kernel
    stores each face straight into the neighbour's window, and `wait` is the allocation's device-side barrier enqueued on the
    context's stream - no NCCL call on the stencil's path; reductions still go through all_reduce.  One node only.

    The symmetric-memory module is private to torch and has changed between releases, so its set-up runs in stages whose
    outcome all ranks agree on (run_agreed): if any stage fails anywhere, every rank raises CommSetupError with the context
    left unsharded, and make_comm falls back to NCCL send/recv."""

    def __init__(self, ctx, group=None):
        self.ctx, self.group = ctx, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.reqs = []
        if self.world > 1:
            g = group if group is not None else dist.group.WORLD
            dev = ctx.torch_device

            def allocate():
                import torch.distributed._symmetric_memory as symm_mem

                enable = getattr(symm_mem, "enable_symm_mem_for_group", None)
                if enable is not None:                       # needed before rendezvous in some releases, a no-op / deprecated in others
                    try:
                        enable(g.group_name)
                    except Exception:                        # noqa: BLE001
                        pass
                with torch.cuda.stream(ctx.stream):
                    w = symm_mem.empty(4 * ctx.halo_bytes(), dtype=torch.uint8, device=dev)
                    w.zero_()
                return symm_mem, w

            symm_mem, self.window = run_agreed(allocate, "symmetric-memory allocation", dev, group)
            self.handle = run_agreed(lambda: symm_mem.rendezvous(self.window, g), "symmetric-memory rendezvous", dev, group)
            ptrs = run_agreed(lambda: window_pointers([int(p) for p in self.handle.buffer_ptrs], self.rank, self.world),
                              "peer window pointers", dev, group)
        ctx.set_sharding(self.rank, self.world, self.start, self.wait, self.allreduce)
        if self.world > 1:
            ctx.set_halo_peers(*ptrs)

    def start(self, *a):                                   # never called in peer-to-peer mode
        raise RuntimeError("PeerComm: the exchange-start callback must not be called while peer windows are set")

    def wait(self):
        with torch.cuda.stream(self.ctx.stream):
            self.handle.barrier()


def make_comm(ctx, p2p=False, group=None, log=None):
    """The communicator of a sharded context: PeerComm when asked for and every rank can set it up, else TorchDistComm (NCCL
    send/recv), with the reason of the fallback handed to `log` (default: stderr of rank 0).  Returns (comm, kind)."""
    if p2p:
        try:
            return PeerComm(ctx, group), "p2p"
        except CommSetupError as e:
            msg = f"peer-to-peer face exchange unavailable ({e}); falling back to NCCL send/recv"
            if log is not None:
                log(msg)
            elif dist.get_rank(group) == 0:
                import sys

                print(msg, file=sys.stderr)
    return TorchDistComm(ctx, group), "nccl"


def window_pointers(all_windows, rank, world):
    """(own, next rank's, previous rank's) receive window out of the per-rank list of a symmetric allocation."""
    prev, nxt = ring_neighbours(rank, world)
    return all_windows[rank], all_windows[nxt], all_windows[prev]

"""Worker of tests/test_gpu_shard.py::test_two_ranks_nccl: one rank per GPU, the lattice split along x0, faces over NCCL
(paper_1010_5636_b200/dist.py); Q and a global reduction against the CPU oracle on the global lattice."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import paper_1010_5636_b200 as nd  # noqa: E402
from lattice_inputs import gauge_field, gaussian_spinor  # noqa: E402
from oracle import wilson_c  # noqa: E402
from paper_1010_5636_b200.dist import TorchDistComm  # noqa: E402


def main():
    local = int(os.environ["LOCAL_RANK"])
    torch.cuda.set_device(local)
    dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    rank, world = dist.get_rank(), dist.get_world_size()
    dims = (16, 8, 8, 8)
    U, psi = gauge_field(dims, "smooth", eps=0.3), gaussian_spinor(dims)
    tb, tl, _, _ = nd.shard_layout(dims[0], world, rank)
    ctx = nd.Context((tl,) + dims[1:], prec=64, recon=12, bc_time=-1, device=local)
    ctx.set_gauge(np.ascontiguousarray(U[:, tb:tb + tl]))
    comm = TorchDistComm(ctx)  # noqa: F841
    x, y = ctx.pack_spinor(np.ascontiguousarray(psi[tb:tb + tl])), ctx.new_spinor()
    ctx.apply_Q(y, x, -1.6)
    ref = wilson_c.apply_Q(psi, U, -1.6, -1)
    got = ctx.unpack_spinor(y)
    err = np.linalg.norm((got - ref[tb:tb + tl]).ravel()) / np.linalg.norm(ref.ravel())
    assert err <= 1e-12, err
    assert abs(ctx.norm2(x) - np.vdot(psi.ravel(), psi.ravel()).real) <= 1e-9
    # the faces as a checksum: |Q psi|^2 depends on both received faces of every rank and crosses the all-reduce; every rank must
    # hold the same bits, and they must be the oracle's value
    ny = ctx.norm2(y)
    assert abs(ny - np.vdot(ref.ravel(), ref.ravel()).real) <= 1e-10 * ny
    seen = [None] * world
    dist.all_gather_object(seen, ny)
    assert all(v == seen[0] for v in seen), seen
    dist.barrier()
    dist.destroy_process_group()


if __name__ == "__main__":
    main()

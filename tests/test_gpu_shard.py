"""Domain decomposition along x0 (csrc/shard.cu, VERDICT r1 task 8) on ONE GPU: the R ranks are R contexts of
the local lattices driven by R host threads, and the transfer callbacks are device copies between their halo buffers (the
library's own kernels pack the faces, run the local stencil with the wrapped time hops switched off and add the received
hops).  Everything a rank returns is compared with the oracle / the single-context result on the GLOBAL lattice: Q with every
stencil kernel, the fused epilogue, global reductions, D_N with projected low modes, and the eigen-solver.  With two or more
GPUs the same contexts run one per process with dist.TorchDistComm (test at the end, skipped below 2 GPUs)."""
import threading

import numpy as np
import pytest

from lattice_inputs import gauge_field, gaussian_spinor
from oracle import sign as osign
from oracle import wilson, wilson_c
from tests.gpu_common import TOL, assert_field_close, rel_l2, round_to
from tests.test_gpu_sign import M, PREF, QNORM, low_space

pytestmark = pytest.mark.gpu


class Emulation:
    """R ranks in one process: thread r drives context r; faces and reductions meet at barriers."""

    def __init__(self, dims, R, prec, recon, bc, U, peers=False):
        import torch

        import paper_1010_5636_b200 as nd

        self.torch, self.R = torch, R
        self.tl = dims[0] // R
        self.ctx = []
        for r in range(R):
            tb, tl, _, _ = nd.shard_layout(dims[0], R, r)
            c = nd.Context((tl,) + tuple(dims[1:]), prec=prec, recon=recon, bc_time=bc)
            Ur = np.ascontiguousarray(U[:, tb:tb + tl])
            c.set_gauge(Ur if prec == 64 else Ur.astype(np.complex64))
            self.ctx.append(c)
        self.barrier = threading.Barrier(R)
        self.red = [None] * R
        for r, c in enumerate(self.ctx):
            c.set_sharding(r, R, self._start(r), self._wait(r), self._allreduce(r))
        self.bufs = [[c.wrap_device_memory(p, c.halo_bytes(), c.real_dtype) for p in c.halo_buffers()] for c in self.ctx]
        if peers:
            # peer-to-peer mode (nd_set_halo_peers): one receive window per rank, the neighbours' pack kernels store into it;
            # the start callback must never run, the wait callback is a barrier over the ranks after a stream synchronise
            from paper_1010_5636_b200.dist import window_pointers

            self.windows = [torch.full((4 * c.halo_bytes(),), 0xFF, dtype=torch.uint8, device=c.torch_device) for c in self.ctx]   # NaN bits
            torch.cuda.synchronize()
            for r, c in enumerate(self.ctx):
                c.set_sharding(r, R, None, self._wait(r), self._allreduce(r))
                c.set_halo_peers(*window_pointers([w.data_ptr() for w in self.windows], r, R))

    def _start(self, r):
        def start(send_next, send_prev, recv_prev, recv_next, nbytes):
            self.ctx[r].synchronize()                      # my faces are packed
            self.barrier.wait()
            prev, nxt = (r - 1) % self.R, (r + 1) % self.R
            with self.torch.cuda.stream(self.ctx[r].stream):
                self.bufs[r][2].copy_(self.bufs[prev][0])  # recv_prev <- previous rank's send_next
                self.bufs[r][3].copy_(self.bufs[nxt][1])   # recv_next <- next rank's send_prev
        return start

    def _wait(self, r):
        def wait():
            self.ctx[r].synchronize()
            self.barrier.wait()                            # nobody repacks before everybody has copied
        return wait

    def _allreduce(self, r):
        def allreduce(d_buf, n):
            t = self.ctx[r].wrap_device_memory(d_buf, 8 * n, self.torch.float64)
            self.ctx[r].synchronize()
            self.red[r] = t.clone()
            self.barrier.wait()
            total = sum(self.red[q] for q in range(self.R))   # the same order on every rank: identical bits everywhere
            self.barrier.wait()
            with self.torch.cuda.stream(self.ctx[r].stream):
                t.copy_(total)
            self.ctx[r].synchronize()
        return allreduce

    def run(self, fn):
        """fn(rank, ctx) on R threads; returns the list of results; re-raises the first exception."""
        out, err = [None] * self.R, [None] * self.R

        def body(r):
            try:
                out[r] = fn(r, self.ctx[r])
            except BaseException as e:                      # noqa: B902
                err[r] = e
                self.barrier.abort()

        th = [threading.Thread(target=body, args=(r,)) for r in range(self.R)]
        for t in th:
            t.start()
        for t in th:
            t.join()
        for e in err:
            if e is not None:
                raise e
        return out

    def split(self, field):
        return [np.ascontiguousarray(field[r * self.tl:(r + 1) * self.tl]) for r in range(self.R)]


@pytest.mark.parametrize("peers", [False, True])
@pytest.mark.parametrize("dims,R,prec,recon,bc", [((16, 4, 4, 8), 2, 64, 12, -1), ((16, 4, 4, 8), 4, 64, 8, -1), ((8, 4, 6, 4), 2, 32, 18, +1),
                                                   ((80, 8, 16, 32), 2, 32, 12, -1), ((32, 8, 8, 16), 2, 32, 12, -1)])
def test_sharded_Q_matches_oracle(dims, R, prec, recon, bc, peers):
    U = round_to(gauge_field(dims, "smooth", eps=0.3), prec)
    em = Emulation(dims, R, prec, recon, bc, U, peers=peers)
    psi = round_to(gaussian_spinor(dims), prec)
    v = [round_to(gaussian_spinor(dims, seed=30 + i), prec) for i in range(2)]
    ref = wilson_c.apply_Q(psi, U, -1.6, bc)
    s0, s1, s2 = 0.37, -1.2, 0.81
    parts, vparts = em.split(psi), [em.split(a) for a in v]

    def work(r, ctx):
        x, y = ctx.pack_spinor(parts[r]), ctx.new_spinor()
        ctx.apply_Q(y, x, -1.6)
        q = ctx.unpack_spinor(y)
        d = [ctx.pack_spinor(a[r]) for a in vparts]
        ctx.apply_Q_axpbycz(d[1], x, -1.6, s0, s1, d[0], s2, d[1])          # out aliases v2
        return q, ctx.unpack_spinor(d[1]), ctx.dot(x, y), ctx.norm2(x), ctx.get_stencil_variant()

    res = em.run(work)
    got = np.concatenate([r[0] for r in res], axis=0)
    assert_field_close(got, ref, TOL[prec])
    assert np.abs(got - ref).max() <= (1e-11 if prec == 64 else 2e-4) * np.abs(ref).max()      # boundary slices included
    got_epi = np.concatenate([r[1] for r in res], axis=0)
    assert_field_close(got_epi, s0 * ref + s1 * v[0] + s2 * v[1], TOL[prec])
    for r in res:                                                           # reductions are GLOBAL on every rank
        assert abs(r[2] - np.vdot(psi.ravel(), ref.ravel())) <= (1e-11 if prec == 64 else 1e-5) * np.linalg.norm(psi.ravel()) * np.linalg.norm(ref.ravel())
        assert abs(r[3] - np.vdot(psi.ravel(), psi.ravel()).real) <= 1e-12 * r[3] and r[2] == res[0][2]
    if dims[3] == 32:
        assert res[0][4] == "tile"                                          # the tiled kernel ran the local lattices


@pytest.mark.parametrize("peers", [False, True])
def test_sharded_DN_and_eigensolver(peers):
    dims, R, prec = (16, 4, 4, 8), 2, 64
    U = gauge_field(dims, "smooth", eps=0.3)
    em = Emulation(dims, R, prec, 12, -1, U, peers=peers)
    Q = wilson_c.make_Q(U, M, -1)
    eta = gaussian_spinor(dims)
    nu, Us = low_space(Q, eta.shape, 5, cut=1.0, degree=8)
    n, eps = 40, 0.004
    c = osign.cheb_coeffs(n, eps)
    ref = osign.apply_DN(Q, wilson.apply_gamma5, eta, c, eps, QNORM, PREF, nu, Us)
    eparts, uparts = em.split(eta), [em.split(u) for u in Us]

    def work(r, ctx):
        ctx.set_sign_poly(c, eps, QNORM, M)
        modes = ctx.new_spinor(len(Us))
        for k in range(len(Us)):
            ctx.pack_spinor(uparts[k][r], out=modes[k])
        ctx.set_lowmodes(modes, nu)
        x, out, w = ctx.pack_spinor(eparts[r]), ctx.new_spinor(), ctx.new_spinor(3)
        ctx.apply_DN(out, x, PREF, w, use_graph=True)                        # (graphs are bypassed while sharded)
        dn = ctx.unpack_spinor(out)
        u, nus, resid, st = ctx.lowmodes_compute(6, M, tol=1e-8, maxit=60, lextra=6, degree=30)
        return dn, nus, resid, st["converged"], [ctx.unpack_spinor(u[k]) for k in range(len(nus))]

    res = em.run(work)
    got = np.concatenate([r[0] for r in res], axis=0)
    assert_field_close(got, ref, 1e-11)
    # the eigen-solver on the sharded lattice: every rank holds the same Ritz values, and they are the global lattice's
    assert res[0][3] and np.array_equal(res[0][1], res[1][1])
    import paper_1010_5636_b200 as nd

    one = nd.Context(dims, prec=64, recon=12, bc_time=-1)
    one.set_gauge(U)
    _, nu1, _, st1 = one.lowmodes_compute(6, M, tol=1e-8, maxit=60, lextra=6, degree=30)
    assert st1["converged"] and np.abs(np.sort(res[0][1]) - np.sort(nu1)).max() <= 1e-8
    for k in range(len(res[0][1])):                                          # residues with the ORACLE's Q on the assembled vectors
        uk = np.concatenate([r[4][k] for r in res], axis=0)
        assert np.linalg.norm((Q(uk) - res[0][1][k] * uk).ravel()) <= 5e-8
        assert abs(np.linalg.norm(uk.ravel()) - 1.0) <= 1e-10


def test_sharding_argument_checks():
    import paper_1010_5636_b200 as nd

    ctx = nd.Context((4, 4, 4, 4), prec=64, recon=12)
    with pytest.raises(nd.NDError) as e:
        ctx.set_halo_peers(None, None, None)                                 # peer windows need a sharded context
    assert e.value.code == -2
    with pytest.raises(nd.NDError):
        ctx.lib.nd_set_sharding(ctx._h, 2, 2, None, None, None, None) and None
        ctx._chk(ctx.lib.nd_set_sharding(ctx._h, 2, 2, None, None, None, None))
    with pytest.raises(nd.NDError):
        ctx._chk(ctx.lib.nd_set_sharding(ctx._h, 0, 2, None, None, None, None))   # callbacks missing
    ctx.set_sharding(0, 1)                                                         # unsharded: fine


def test_two_ranks_nccl():
    """The real thing, one process per GPU over NCCL: needs two GPUs (the development and driver boxes of this round have one)."""
    import torch

    if torch.cuda.device_count() < 2:
        pytest.skip("needs 2 GPUs")
    import os
    import subprocess
    import sys

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
                        "--master-port", "29533", os.path.join(root, "tests", "shard_nccl_worker.py")], capture_output=True, text=True,
                       timeout=600)
    assert r.returncode == 0, r.stdout + r.stderr

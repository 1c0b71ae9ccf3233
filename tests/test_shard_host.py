"""Host logic of the domain decomposition (csrc/shard.cu, paper_1010_5636_b200/dist.py) on CPU:
the partition helper of the C ABI, and the face-exchange schedule of dist.py run for real over the gloo backend with 2 and 3
processes (which face lands in which buffer, also when previous and next neighbour are the same peer)."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_window_pointers_of_the_peer_to_peer_exchange():
    from paper_1010_5636_b200.dist import ring_neighbours, window_pointers

    w = [100, 200, 300, 400]
    assert window_pointers(w, 0, 4) == (100, 200, 400) and window_pointers(w, 3, 4) == (400, 100, 300)
    assert window_pointers(w[:2], 1, 2) == (200, 100, 100)                   # two ranks: previous and next are the same peer
    assert ring_neighbours(0, 1) == (0, 0)


def test_shard_layout():
    import paper_1010_5636_b200 as nd

    assert nd.shard_layout(64, 1, 0) == (0, 64, True, True)
    assert nd.shard_layout(64, 8, 0) == (0, 8, True, False)
    assert nd.shard_layout(64, 8, 3) == (24, 8, False, False)
    assert nd.shard_layout(64, 8, 7) == (56, 8, False, True)
    covered = []
    for r in range(4):
        tb, tl, _, _ = nd.shard_layout(16, 4, r)
        covered += list(range(tb, tb + tl))
    assert covered == list(range(16))                                  # a partition of the time extent
    for bad in ((64, 3, 0), (64, 8, 8), (64, 8, -1), (8, 8, 0), (64, 0, 0)):   # not divisible, rank out of range, 1-slice parts
        with pytest.raises(nd.NDError):
            nd.shard_layout(*bad)


WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
from paper_1010_5636_b200.dist import exchange_ops, ring_neighbours
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
n = 6
send_next = torch.full((n,), 100.0 + rank); send_prev = torch.full((n,), 200.0 + rank)
recv_prev = torch.zeros(n); recv_next = torch.zeros(n)
for r in dist.batch_isend_irecv(exchange_ops(send_next, send_prev, recv_prev, recv_next, rank, world)):
    r.wait()
t = torch.tensor([float(rank + 1)], dtype=torch.float64)
dist.all_reduce(t)
dist.barrier()
print(json.dumps(dict(rank=rank, world=world, nb=ring_neighbours(rank, world), recv_prev=recv_prev.tolist(), recv_next=recv_next.tolist(),
                      total=t.item())))
dist.destroy_process_group()
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("world", [2, 3])
def test_face_exchange_schedule_gloo(tmp_path, world):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    port = _free_port()
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, text=True))
    outs = [json.loads(p.communicate(timeout=180)[0].strip().splitlines()[-1]) for p in procs]
    assert all(p.returncode == 0 for p in procs)
    for r, o in enumerate(outs):
        prev, nxt = (r - 1) % world, (r + 1) % world
        assert o["nb"] == [prev, nxt]
        assert o["recv_prev"] == [100.0 + prev] * 6        # what the previous rank sent "to next"
        assert o["recv_next"] == [200.0 + nxt] * 6         # what the next rank sent "to previous"
        assert o["total"] == world * (world + 1) / 2


AGREE_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
from paper_1010_5636_b200.dist import CommSetupError, run_agreed
dist.init_process_group("gloo")
rank = dist.get_rank()
cpu = torch.device("cpu")
def fails_on_rank_1():
    if rank == 1:
        raise ValueError("no symmetric memory here")
    return "window"
out = dict(rank=rank)
try:
    run_agreed(fails_on_rank_1, "stage A", cpu)
    out["A"] = "returned"
except CommSetupError as e:
    out["A"] = str(e)
out["B"] = run_agreed(lambda: 10 + rank, "stage B", cpu)      # the group is still usable: the next stage succeeds everywhere
dist.barrier()
print(json.dumps(out))
dist.destroy_process_group()
"""


def test_collective_setup_is_unanimous_gloo(tmp_path):
    """dist.run_agreed (PeerComm's set-up must not leave ranks in different states): a stage that fails on one
    rank raises CommSetupError on both, the failing rank naming its reason, and the following stage still runs."""
    script = tmp_path / "agree.py"
    script.write_text(AGREE_WORKER.format(root=ROOT))
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, text=True))
    outs = [json.loads(p.communicate(timeout=180)[0].strip().splitlines()[-1]) for p in procs]
    assert all(p.returncode == 0 for p in procs)
    assert outs[0]["A"] == "stage A: failed on another rank"
    assert outs[1]["A"] == "stage A: ValueError: no symmetric memory here"
    assert [o["B"] for o in outs] == [10, 11]

"""Host logic of bench.py for N > 1 (replicas only): rank environment, max-over-ranks timing and
the whole-job value, on CPU with the gloo backend at world_size 2."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
rank, world, local = bench.dist_env()
dist.init_process_group("gloo")
ms = bench.max_over_ranks(10.0 + 5.0 * rank, world)          # rank 1 is the slow one
value = bench.whole_job_value(100.0, world, ms)
dist.barrier()
print(json.dumps(dict(rank=rank, world=world, local=local, ms=ms, value=value)))
dist.destroy_process_group()
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_replicas_world_size_2_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, text=True))
    outs = [json.loads(p.communicate(timeout=120)[0].strip().splitlines()[-1]) for p in procs]
    assert all(p.returncode == 0 for p in procs)
    for r, o in enumerate(outs):
        assert o["rank"] == r and o["world"] == 2 and o["local"] == r
        assert o["ms"] == 15.0                                  # max over ranks on EVERY rank
        assert abs(o["value"] - 2 * 100.0 / 15e-3) < 1e-9       # units of all ranks / slowest time


def test_single_rank_helpers():
    sys.path.insert(0, ROOT)
    import bench

    assert bench.max_over_ranks(3.5, 1) == 3.5
    assert bench.whole_job_value(10.0, 1, 1000.0) == 10.0
    assert bench.q_bytes_per_site(32, 12) == 384 and bench.q_bytes_per_site(64, 12) == 768
    assert bench.q_bytes_per_site(32, 8) == 320 and bench.q_bytes_per_site(64, 18) == 960
    assert bench.q_bytes_per_site(32, 12, 3) == 384 + 288


def test_spawn_command_and_traffic_table():
    """`python bench.py --gpus N` without a torchrun environment re-executes itself under torch.distributed.run with one rank
    per GPU on 127.0.0.1; the DRAM-traffic table is keyed by kernel, lattice, precision and recon and gives None otherwise."""
    sys.path.insert(0, ROOT)
    import bench

    cmd = bench.spawn_command(["--gpus", "4", "--steps", "2"], 4, 29512)
    assert cmd[1:3] == ["-m", "torch.distributed.run"] and "--nproc-per-node=4" in cmd and "--nnodes=1" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[cmd.index("--master-port") + 1] == "29512"
    assert cmd[-4:] == ["--gpus", "4", "--steps", "2"] and cmd[-5].endswith("bench.py")
    assert bench.load_traffic("wilson_Q_kernel", "5^3x7", 32, 12) is None          # no capture of that lattice
    assert bench.load_traffic("no_such_kernel", "32^3x64", 32, 12) is None
    for kernel, prec in (("wilson_Q_tile2_kernel", 32), ("wilson_Q_tile2_kernel", 64), ("wilson_Q_tile_kernel", 32)):
        t = bench.load_traffic(kernel, "32^3x64", prec, 12)
        model = bench.q_bytes_per_site(prec, 12) * 2097152
        assert t is None or 0.9 * model < t < 1.3 * model                          # a capture, if present, is near the byte model
    assert bench.stencil_kernel_name("site", 8192) == "wilson_Q_hop_kernel" and bench.stencil_kernel_name("site", 1 << 20) == "wilson_Q_kernel"
    assert bench.stencil_kernel_name("tile", 1 << 21) == "wilson_Q_tile2_kernel" and bench.stencil_kernel_name("tile", 1 << 21, 64) == "wilson_Q_tile2_kernel"
    assert bench.stencil_kernel_name("tile4", 1 << 21) == "wilson_Q_tile_kernel" and bench.stencil_kernel_name("tile_tma", 1 << 21) == "wilson_Q_tile3_kernel"


def test_reference_arm_other_ranks_exit_without_work():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                        "--warmup", "1"], env=env, capture_output=True, text=True, timeout=60)
    assert r.returncode == 0 and r.stdout.strip() == ""

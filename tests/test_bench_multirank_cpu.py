"""N > 1 host logic of bench.py on CPU (gloo, world size 2): the path does not shard ("replicas
only"), so what there is to cover is the max-over-ranks timing, the aggregate
throughput, and the reference arm's rule that rank 0 alone runs and prints."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, %r)
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
t = bench.max_over_ranks(1.0 + rank, world, torch.device("cpu"))
assert t == float(world), t
assert bench.aggregate_mlups(1000, 10, world, 1e-3) == 1000 * 10 * world / 1e-3 / 1e6
dist.barrier()
dist.destroy_process_group()
sys.stdout.write("rank%%d-ok\n" %% rank)
sys.stdout.flush()
"""


def free_port():
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def torchrun(args):
    port = free_port()
    env = dict(os.environ, OMP_NUM_THREADS="2")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(port)] + args
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)


def test_max_over_ranks_and_aggregate_gloo_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    r = torchrun([str(script)])
    assert r.returncode == 0, (r.stdout[-1500:], r.stderr[-3000:])
    assert r.stdout.count("rank0-ok") == 1 and r.stdout.count("rank1-ok") == 1


def test_reference_arm_rank0_only_prints_one_line():
    r = torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "3", "--warmup", "1",
                  "--config", "c1"])
    assert r.returncode == 0, (r.stdout[-1500:], r.stderr[-3000:])
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["gpu_launches"] == 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"]

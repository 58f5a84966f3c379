"""World-size-2 gloo test (CPU) of bench.py's multi-rank plumbing: rendezvous, barrier, max over ranks.

The path has no exchange step ("replicas only"); the only distributed logic is the
timing aggregation, exercised here with two processes over gloo on 127.0.0.1.
"""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, os.environ["SCW_ROOT"])
import bench
rank, world, local_rank, dist = bench.dist_setup(2)
assert world == 2 and dist is not None and dist.get_backend() == "gloo"
bench.barrier(dist)
ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist)      # rank 1 is the slow one
assert ms == 15.0, ms
value = world * 1000 / (ms * 1e-3)                      # whole-job aggregate over the slowest rank
bench.barrier(dist)
print(f"rank {rank} ok {value:.1f}")
dist.destroy_process_group()
"""


def test_two_rank_gloo_aggregation(tmp_path):
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), SCW_ROOT=ROOT, CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=120)[0] for p in procs]
    for rank, (p, out) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, out
        assert f"rank {rank} ok 133333.3" in out


def test_reference_arm_only_rank0_works(tmp_path):
    """Under torchrun the reference arm runs on rank 0 alone; other ranks exit 0 without work."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert out.returncode == 0 and out.stdout.strip() == ""

"""The N > 1 path of bench.py: independent replicas, one process per GPU, no data-path collective
(DESIGN.md section 7).  What remains multi-process is the timing plumbing — the max over ranks and the
whole-job rate — covered here with world_size 2 over gloo on CPU.  -m "not gpu"."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, sys.argv[1])
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ms = 10.0 + 5.0 * rank                      # rank 1 is the slow one
ms_max = bench.max_over_ranks(ms, dist, "cpu")
assert ms_max == 15.0, ms_max
v = bench.aggregate_rate(1000, 7, world, ms_max)
assert abs(v - world * 1000 * 3 * 7 / 15e-3 / 1e6) < 1e-9
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
"""


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_max_over_ranks_and_aggregate_world_size_2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script), ROOT], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=240)[0] for p in procs]
    for rank, (p, out) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, out
        assert f"ok {rank}" in out


def test_reference_arm_runs_on_rank_0_only():
    """Under torchrun the reference arm (the CPU oracle) runs on rank 0; other ranks exit 0 without work."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_single_process_is_the_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.25, None, "cpu") == 3.25
    assert bench.aggregate_rate(8388608, 200, 1, 1531.4 * 200 / 200 * 200) > 0

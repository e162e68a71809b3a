"""The N > 1 path of bench.py on CPU (gloo, world_size 2): replicas only -- no data-path collective, just the barrier and
the max-over-ranks timing."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


_WORKER = r"""
import os, sys
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, "cpu")      # rank 1 is the slow one
dist.barrier()
rate = bench.whole_job_rate(1000, 4, ms, world)
assert ms == 15.0, ms
assert abs(rate - 2 * 1000 * 4 / 15e-3) < 1e-6, rate
if rank == 0:
    print("OK", ms, rate)
dist.destroy_process_group()
"""


def _torchrun(args, extra_env=None):
    env = dict(os.environ)
    env.update({"MASTER_ADDR": "127.0.0.1"})
    env.update(extra_env or {})
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port())] + args
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)


def test_max_over_ranks_and_whole_job_rate_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT))
    r = _torchrun([str(script)])
    assert r.returncode == 0, r.stderr[-2000:]
    assert "OK 15.0" in r.stdout


def test_reference_arm_under_torchrun_prints_one_line():
    """--impl reference with N > 1: rank 0 alone runs the oracle and prints the JSON line; the other rank exits 0."""
    r = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "3", "--size", "8"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0


def test_roofline_byte_model_matches_the_survey():
    """B_step = 8[(6d+8) N_p + (3+7d) N_n]: 232 B/particle on config 4."""
    sys.path.insert(0, ROOT)
    import bench
    per_kernel, step = bench.algorithmic_bytes(3, 134217728, 16974593)
    assert step == 8 * ((6 * 3 + 8) * 134217728 + (3 + 7 * 3) * 16974593)
    assert abs(step / 134217728 - 232.3) < 0.1
    assert per_kernel["update"] == 8 * (16 * 134217728 + 10 * 16974593)
    assert per_kernel["g2p_p2g2"] + per_kernel["update"] <= step

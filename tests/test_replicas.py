"""N > 1 path of bench.py ("replicas only") on CPU: gloo, world_size 2."""
import json
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


WORKER = r"""
import os, sys
sys.path.insert(0, os.environ["REPO_ROOT"])
from paper_0908_4362_b200.replicas import Replicas
r = Replicas(backend="gloo")
assert r.world == 2
r.barrier()
mine = 2.0 + 3.0 * r.rank                      # rank 0: 2 s, rank 1: 5 s
assert r.max_over_ranks(mine) == 5.0
rate = r.whole_job_rate(1000.0, mine)          # 2 ranks x 1000 units / slowest 5 s
assert abs(rate - 400.0) < 1e-12, rate
r.barrier()
if r.rank == 0:
    print("REPLICAS_OK", rate)
r.close()
"""


def _torchrun(args, timeout=600):
    env = dict(os.environ, REPO_ROOT=ROOT, MASTER_ADDR="127.0.0.1", OMP_NUM_THREADS="2")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port())] + args
    return subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=timeout)


def test_timing_protocol_world_size_2_gloo(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(WORKER)
    res = _torchrun([str(w)])
    assert res.returncode == 0, res.stderr[-2000:]
    assert res.stdout.count("REPLICAS_OK") == 1 and "400.0" in res.stdout


def test_single_process_is_identity():
    from paper_0908_4362_b200.replicas import Replicas
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        os.environ.pop(k, None)
    r = Replicas(backend="gloo")
    assert (r.rank, r.world) == (0, 1)
    assert r.max_over_ranks(3.5) == 3.5 and r.whole_job_rate(10.0, 2.0) == 5.0
    r.barrier()
    r.close()


def test_reference_arm_under_torchrun_prints_one_line():
    """bench.py --impl reference with 2 ranks: rank 0 alone runs the oracle and prints the JSON line"""
    res = _torchrun(["bench.py", "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "1", "--workload", "small"])
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, res.stdout
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0

"""N > 1 path on CPU: world_size-2 gloo runs of the replica plumbing bench.py uses (replicas only:
no data-path collective; barrier + max-over-ranks timing + whole-job throughput)."""
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


_WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
from paper_1904_02108_b200 import replicas
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist = replicas.init("gloo", rank, world)
replicas.barrier(dist)
ms = replicas.max_over_ranks(10.0 * (rank + 1), dist)        # rank 1 is the slow replica
val = replicas.whole_job_mlups(1000, 5, world, ms)
print(json.dumps({{"rank": rank, "ms": ms, "value": val}}))
replicas.finish(dist)
"""


def test_two_replicas_max_time_and_whole_job_value():
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", _WORKER.format(root=ROOT)], env=env,
                                      stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, err = p.communicate(timeout=300)
        assert p.returncode == 0, err
        outs.append(json.loads(out.strip().splitlines()[-1]))
    for o in outs:
        assert o["ms"] == 20.0                                  # MAX over ranks, on every rank
        assert abs(o["value"] - 2 * 1000 * 5 / 20e-3 / 1e6) < 1e-12


def test_single_process_needs_no_group():
    sys.path.insert(0, ROOT)
    from paper_1904_02108_b200 import replicas
    assert replicas.init("gloo", 0, 1) is None
    assert replicas.max_over_ranks(3.5, None) == 3.5
    assert replicas.whole_job_mlups(10 ** 6, 10, 1, 1.0) == 1e4


def test_reference_arm_prints_one_line_on_rank0_only():
    """bench.py --impl reference under a 2-rank launch: rank 0 alone times the oracle and prints the
    JSON line; the other rank exits 0 without work."""
    outs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank))
        p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                            "--workload", "W1", "--steps", "2", "--warmup", "0"], env=env, capture_output=True,
                           text=True, timeout=600)
        assert p.returncode == 0, p.stderr
        outs.append(p.stdout.strip())
    line = json.loads(outs[0].splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "MLUPS" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert outs[1] == ""

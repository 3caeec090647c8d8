"""world_size-2 gloo test of the N > 1 plumbing bench.py uses (replicas only: barrier + MAX over ranks)."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys
sys.path.insert(0, os.environ["REPO_ROOT"])
from paper_2501_18263_b200 import replicas
rank, world = replicas.init("gloo")
assert world == 2
replicas.barrier(world)
ms_local = 10.0 if rank == 0 else 25.0          # the slower replica sets the step time
ms_max, value = replicas.aggregate_throughput(1000.0, ms_local, world)
assert ms_max == 25.0, ms_max
assert abs(value - 2 * 1000.0 / 25e-3) < 1e-6, value
assert replicas.max_over_ranks(float(rank), world) == 1.0
replicas.barrier(world)
print("rank %d ok" % rank)
'''


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_two_replicas_take_the_max_time_and_sum_the_work(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = str(_free_port())
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=port, REPO_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=180)[0] for p in procs]
    for r, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, o
        assert "rank %d ok" % r in o


def test_single_process_is_the_identity():
    sys.path.insert(0, ROOT)
    from paper_2501_18263_b200 import replicas
    assert replicas.aggregate_throughput(5.0, 2.0, 1) == (2.0, 2500.0)

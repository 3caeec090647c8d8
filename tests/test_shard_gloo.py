"""world_size-2 gloo test of the sharded-apply exchange (paper_2501_18263_b200/sharded.py): two CPU ranks each hold the
psi' blocks of "their" half of an H_eff.psi computed by the oracle (zeros elsewhere, as dmrg_set_shard leaves them),
and the library's reduce step — torch.distributed.all_reduce behind `make_reduce` — must give every rank the whole
vector, bit-identical on both."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r'''
import os, sys
sys.path.insert(0, os.environ["REPO_ROOT"])
import numpy as np
import torch
import torch.distributed as dist
from oracle import dmrg as odmrg
from paper_2501_18263_b200 import inputs, replicas, sharded
rank, world = replicas.init("gloo")
assert world == 2
T, V, mps = inputs.make_config(0)
pb = inputs.psi_blocks(mps)
orc = odmrg.TwoSiteOracle(T, V, mps.n_up, mps.n_dn, mps.k, mps.sectors, mps.left, mps.right, pb)
orc.build_env()
v = inputs.make_psi0(mps, 3)
y = orc.apply(v)
part = np.zeros_like(y)
off = 0
for b, blk in enumerate(pb):
    n = blk[4] * blk[5]
    if b % world == rank:
        part[off:off + n] = y[off:off + n]
    off += n
assert off == y.size and np.abs(part).sum() < np.abs(y).sum()
t = torch.from_numpy(part.copy())
sharded.make_reduce()(t)
assert np.array_equal(t.numpy(), y)          # sums with exact zeros
other = [torch.zeros_like(t) for _ in range(world)]
dist.all_gather(other, t)
assert torch.equal(other[0], other[1])
class Fake:                                  # shard_over_ranks hands (rank, world, reduce) to set_shard
    def set_shard(self, r, n, reduce):
        self.args = (r, n, reduce)
f = Fake()
assert sharded.shard_over_ranks(f) == (rank, world) and f.args[:2] == (rank, world) and callable(f.args[2])
replicas.barrier(world)
print("rank %d ok" % rank)
'''


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_two_ranks_exchange_disjoint_blocks(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = str(_free_port())
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=port, REPO_ROOT=ROOT)
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    outs = [p.communicate(timeout=300)[0] for p in procs]
    for r, (p, o) in enumerate(zip(procs, outs)):
        assert p.returncode == 0, o
        assert "rank %d ok" % r in o

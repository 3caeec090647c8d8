"""One-off element-wise parity run at a size between BASELINE configs[1] and [2] (too slow for the pytest
suite: the numpy oracle needs tens of minutes).  Usage on a GPU box:

    python tests/midsize_parity.py [L] [n_elec_per_spin] [D]        (default 24 10 512)
    python tests/midsize_parity.py config C                          (BASELINE configs[C], its own seed; C = 3 needs hours and ~100 GB of host memory)

Prints the oracle's and the library's times and the relative L2 error of H_eff.psi (tolerance 1e-11,
DESIGN.md R18).  The result of the run made in round 1 is quoted in DESIGN.md §7.
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from oracle import dmrg as odmrg            # noqa: E402
from paper_2501_18263_b200 import inputs    # noqa: E402


def main():
    import torch
    from paper_2501_18263_b200.binding import DMRG
    if len(sys.argv) > 2 and sys.argv[1] == "config":
        c = inputs.CONFIGS[int(sys.argv[2])]
        T, V, mps = inputs.make_config(int(sys.argv[2]))
        L, ne, D, k = c["L"], c["n_up"], c["D"], mps.k
        v = inputs.make_psi0(mps, c["seed"])
    else:
        L = int(sys.argv[1]) if len(sys.argv) > 1 else 24
        ne = int(sys.argv[2]) if len(sys.argv) > 2 else 10
        D = int(sys.argv[3]) if len(sys.argv) > 3 else 512
        k = L // 2
        T, V = inputs.make_integrals(L, 4242)
        mps = inputs.make_mps(L, ne, ne, D, k, seed=4242)
        v = inputs.make_psi0(mps, 4242)
    pb = inputs.psi_blocks(mps)
    t0 = time.time()
    d = DMRG(L, ne, ne)
    d.setup(T, V, mps)
    got = d.heff_apply(torch.from_numpy(v).cuda()).cpu().numpy()
    torch.cuda.synchronize()
    t_gpu = time.time() - t0
    st = d.stats()
    print("library: setup + apply %.1f s, psi %d, tasks %d, flops/apply %.3e" % (t_gpu, len(v), st["n_tasks"], st["flops_apply"]), flush=True)
    t0 = time.time()
    orc = odmrg.TwoSiteOracle(T, V, ne, ne, k, mps.sectors, mps.left, mps.right, pb)
    orc.build_env()
    t_env = time.time() - t0
    print("oracle: environments %.1f s" % t_env, flush=True)
    t0 = time.time()
    ref = orc.apply(v)
    t_apply = time.time() - t0
    err = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    print("oracle: apply %.1f s" % t_apply)
    print("L=%d N=(%d,%d) D=%d middle bond: rel-L2(H_eff.psi) = %.3e  (tolerance 1e-11)" % (L, ne, ne, D, err))
    d.close()
    return 0 if err <= 1e-11 else 1


if __name__ == "__main__":
    sys.exit(main())

"""GPU tests of the rank-sharded H_eff.psi (dmrg_set_shard): `-m gpu`.

One GPU only: the ranks of a sharded job are separate library contexts run one after the other, and their partial
results are summed here.  The Davidson test runs two contexts in two host threads whose reduce callbacks meet at a
host barrier (an in-process all-reduce): the same lock-step a 2-GPU job runs, with no kernel waiting on another.
The sums are compared with the CPU oracle at the tolerances of the unsharded path (rel-L2 <= 1e-11, |dE| <= 1e-9).
"""
import threading

import numpy as np
import pytest

from oracle import dmrg as odmrg
from oracle import su2 as osu2
from paper_2501_18263_b200 import inputs

pytestmark = pytest.mark.gpu
REL_L2 = 1e-11


def _ctx(T, V, mps, su2=False, e_core=0.0):
    import torch
    from paper_2501_18263_b200.binding import DMRG
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    if su2:
        d = DMRG(mps.L, mps.N // 2, mps.N // 2, su2=True)
    else:
        d = DMRG(mps.L, mps.n_up, mps.n_dn)
    d.setup(T, V, mps, e_core=e_core)
    return d


def _rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def _block_slices(d):
    blocks, n = d.psi_layout()
    return [slice(b.off, b.off + b.dL * b.dR) for b in blocks], n


@pytest.mark.parametrize("count", [2, 3, 8])
def test_partial_results_sum_to_the_oracle_u1(count):
    import torch
    T, V, mps = inputs.make_config(1)
    e_core = 0.375
    pb = inputs.psi_blocks(mps)
    orc = odmrg.TwoSiteOracle(T, V, mps.n_up, mps.n_dn, mps.k, mps.sectors, mps.left, mps.right, pb)
    orc.build_env()
    v = inputs.make_psi0(mps, 77)
    y_ref = orc.apply(v) + e_core * v
    x = torch.from_numpy(v).cuda()
    d = _ctx(T, V, mps, e_core=e_core)
    y_full = d.heff_apply(x).cpu().numpy()
    full_flops = d.stats()["flops_apply"]
    sl, n = _block_slices(d)
    total = np.zeros(n)
    owners, flops_seen, tasks = None, 0.0, 0
    for r in range(count):
        d.set_shard(r, count)
        d.env_build(mps.k)
        own, fl = d.shard_info()
        if owners is None:
            owners = own.copy()
        assert np.array_equal(own, owners)            # every rank derives the same map
        assert np.isclose(fl.sum(), full_flops, rtol=1e-12)
        assert np.isclose(d.stats()["flops_apply"], fl[r], rtol=1e-12)
        assert fl.max() <= 1.25 * fl.mean()           # longest-processing-time balance
        y = d.heff_apply(x).cpu().numpy()
        for b, s in enumerate(sl):                    # a block is computed by its owner alone
            if own[b] != r:
                expect = e_core * v[s] if r == 0 else 0.0
                assert np.array_equal(y[s], expect + np.zeros_like(y[s]))
        total += y
        flops_seen += d.stats()["flops_apply"]
        tasks += d.stats()["n_tasks"]
        with pytest.raises(Exception):                # no collective given: Davidson refuses
            d.davidson(x.clone(), tol=1e-6, max_iter=2)
    assert set(owners.tolist()) == set(range(count))
    assert np.isclose(flops_seen, full_flops, rtol=1e-12)
    assert _rel(total, y_ref) <= REL_L2
    assert _rel(total, y_full) <= 1e-13
    # back to the unsharded library
    d.set_shard(0, 1)
    d.env_build(mps.k)
    assert d.stats()["n_tasks"] == tasks
    assert np.array_equal(d.heff_apply(x).cpu().numpy(), y_full)
    d.close()


def test_partial_results_sum_to_the_oracle_su2():
    import torch
    cfg = dict(L=12, N=12, D=60, k=6, seed=41)
    T, V = inputs.make_integrals(cfg["L"], cfg["seed"])
    mps = inputs.make_mps_su2(cfg["L"], cfg["N"], cfg["D"], cfg["k"], seed=cfg["seed"])
    orc = osu2.SU2TwoSiteOracle(T, V, mps, inputs.psi_blocks_su2(mps))
    orc.build_env()
    v = inputs.make_psi0_su2(mps, 5)
    y_ref = orc.apply(v)
    x = torch.from_numpy(v).cuda()
    d = _ctx(T, V, mps, su2=True)
    total = np.zeros_like(v)
    for r in range(3):
        d.set_shard(r, 3)
        d.env_build(mps.k)
        total += d.heff_apply(x).cpu().numpy()
    assert _rel(total, y_ref) <= REL_L2
    d.close()


def test_davidson_in_lock_step_over_two_ranks():
    """Two sharded contexts in two host threads; the reduce callbacks exchange through a host barrier."""
    import torch
    T, V, mps = inputs.make_config(0)
    pb = inputs.psi_blocks(mps)
    orc = odmrg.TwoSiteOracle(T, V, mps.n_up, mps.n_dn, mps.k, mps.sectors, mps.left, mps.right, pb)
    orc.build_env()
    v0 = inputs.make_psi0(mps, inputs.CONFIGS[0]["seed"])
    E_ref, _, _, _ = odmrg.davidson(orc.apply, orc.diag(), v0, tol=1e-10, max_iter=200, max_basis=20)
    count = 2
    barrier = threading.Barrier(count)
    slots = [None] * count
    results = [None] * count

    def make_reduce(r):
        def reduce(t):
            torch.cuda.synchronize()
            slots[r] = t
            barrier.wait(timeout=120)
            s = slots[0] + slots[1]              # the same order on both ranks
            torch.cuda.synchronize()
            barrier.wait(timeout=120)
            t.copy_(s)
        return reduce

    def run(r):
        try:
            d = _ctx(T, V, mps)
            d.set_shard(r, count, make_reduce(r))
            d.env_build(mps.k)
            x = torch.from_numpy(v0.copy()).cuda()
            y = d.heff_apply(x).cpu().numpy()
            E, it, rn = d.davidson(x, tol=1e-10, max_iter=200, max_basis=20)
            results[r] = (y, E, it, rn, x.cpu().numpy())
            d.close()
        except Exception as e:                    # release the other thread
            barrier.abort()
            results[r] = e

    th = [threading.Thread(target=run, args=(r,)) for r in range(count)]
    for t in th:
        t.start()
    for t in th:
        t.join(timeout=600)
    for r in results:
        assert not isinstance(r, Exception) and r is not None, r
    (y0, E0, it0, rn0, x0), (y1, E1, it1, rn1, x1) = results
    assert _rel(y0, orc.apply(v0)) <= REL_L2
    assert np.array_equal(y0, y1) and np.array_equal(x0, x1)      # replicated vectors stay bit-identical
    assert E0 == E1 and it0 == it1
    assert rn0 <= 1e-10
    assert abs(E0 - E_ref) <= 1e-9

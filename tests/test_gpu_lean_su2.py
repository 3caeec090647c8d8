"""SU(2)-adapted H_eff.psi at BASELINE sizes against the oracle on sampled blocks (`-m gpu`): configs[3] second half
(1024 multiplets) and a configs[4]-shaped problem.  oracle_su2(psi) = reduce(oracle_u1(expand(psi))) (oracle/su2.py);
the U(1) oracle is evaluated on the U(1) blocks the sampled reduced blocks expand into (oracle/lean.py).  A separate
module from test_gpu_lean_parity.py so that its module-scoped D = 4096 context is released first."""
import time

import numpy as np
import pytest

from lean_helpers import ExportedSideSU2, choose_blocks
from paper_2501_18263_b200 import inputs
from test_gpu_lean_parity import TOL, _check_definition, _ctx, _one_step, _sides, lean_parity

pytestmark = pytest.mark.gpu


def _su2_sampled_parity(cfg, D, n_red, seed, env_cache_gb=40):
    """The SU(2) library result on sampled REDUCED output blocks against reduce(lean U(1) oracle(expand(psi))), and the
    cross-check R19 at full size: expand(H^{SU2} psi) == H^{U1} expand(psi) with the library's U(1) path on the
    CG-expanded MPS (equal effective bond), itself compared with the oracle on sampled U(1) blocks."""
    import torch
    from oracle import su2
    from paper_2501_18263_b200.binding import DMRG
    T, V, mps = inputs.make_config_su2(cfg, D=D)
    c = inputs.SU2_CONFIGS[cfg]
    n2 = mps.N // 2
    orc = su2.SU2TwoSiteOracle(T, V, mps, inputs.psi_blocks_su2(mps))        # expansion maps only; no environments
    u1 = inputs.MPSInput(L=mps.L, k=mps.k, n_up=n2, n_dn=n2, sectors=orc.u1.sectors, left=orc.u1.left, right=orc.u1.right)
    pb = orc.u1_blocks
    assert pb == inputs.psi_blocks(u1)
    v = inputs.make_psi0_su2(mps, c["seed"])
    d2 = DMRG(mps.L, n2, n2, su2=True)
    d2.setup(T, V, mps)
    y_red = d2.heff_apply(torch.from_numpy(v).cuda()).cpu().numpy()
    st2 = d2.stats()
    d2.close()
    d1 = _ctx(T, V, u1, env_cache_bytes=env_cache_gb << 30)
    xe = orc.expand(v)
    y_u1 = d1.heff_apply(torch.from_numpy(np.ascontiguousarray(xe)).cuda()).cpu().numpy()
    # R19 at this size, whole vector
    lhs = orc.expand(y_red)
    r19 = np.linalg.norm(lhs - y_u1) / np.linalg.norm(y_u1)
    # reduced blocks to check against the oracle, and the U(1) blocks their expansion lives in
    red_blocks = orc.psi_blocks
    red_off = np.cumsum([0] + [b[5] * b[6] for b in red_blocks])
    u1_off = np.cumsum([0] + [b[4] * b[5] for b in pb])
    Rc = orc.R.tocsc()

    def images(j):
        rows = np.unique(Rc[:, red_off[j]:red_off[j + 1]].indices)
        return sorted(set((np.searchsorted(u1_off, rows, side="right") - 1).tolist()))
    rng = np.random.default_rng(seed)
    sizes = [b[5] * b[6] for b in red_blocks]
    chosen = [int(np.argmax(sizes))]
    for j in rng.permutation(len(red_blocks)).tolist():
        if len(chosen) >= n_red:
            break
        if j not in chosen and sizes[j] >= 16 and len(images(j)) <= 16:
            chosen.append(j)
    need = set()
    for j in chosen:
        need |= set(images(j))
    need |= set(choose_blocks(pb, 0, seed=seed, max_elems=0))     # every tile shape + the largest U(1) block
    t0 = time.time()
    res, nbytes, refs = lean_parity(d1, T, V, u1, xe, y_u1, sorted(need), keep_refs=True)
    print("SU(2) config %d (%d multiplets, U(1)-equivalent %d): %d reduced blocks -> %d U(1) blocks, %.1f GB exported, %.0f s;"
          " R19 whole-vector rel-L2 %.2e; SU(2) flops/apply %.3e" % (cfg, D or c["D"], sum(u1.sectors[mps.k].values()), len(chosen), len(need),
                                                                    nbytes / 1e9, time.time() - t0, r19, st2["flops_apply"]))
    for i, dL, dR, r2, rmax in res:
        assert r2 <= TOL and rmax <= 10 * TOL, ("u1 block", i, dL, dR, r2, rmax)
    print("  U(1) blocks: worst rel-L2 %.2e" % max(r[3] for r in res))
    # oracle value of the reduced blocks: R^T applied to the oracle's U(1) blocks
    y_orc = np.zeros(orc.n_u1)
    for i, m in refs.items():
        y_orc[u1_off[i]:u1_off[i + 1]] = m.reshape(-1)
    worst = 0.0
    for j in chosen:
        cols = Rc[:, red_off[j]:red_off[j + 1]]
        ref = cols.T @ y_orc
        got = y_red[red_off[j]:red_off[j + 1]]
        e2 = np.linalg.norm(got - ref) / np.linalg.norm(ref)
        print("  reduced block %4d  %3d x %3d  (%2d U(1) images)  rel-L2 %.2e" % (j, red_blocks[j][5], red_blocks[j][6], len(images(j)), e2))
        worst = max(worst, e2)
        assert e2 <= TOL, (j, e2)
    assert r19 <= TOL
    return d1, T, V, u1, worst


def test_config3_su2_1024_multiplets_against_the_oracle_and_u1_crosscheck():
    """BASELINE configs[3], SU(2) half: 1024 multiplets (U(1)-equivalent 3609 states)."""
    d1, T, V, u1, worst = _su2_sampled_parity(3, None, n_red=10, seed=5)
    # the exported U(1) operators of the expanded MPS, at this size, against their definition
    k, L = u1.k, u1.L
    Ls, Rs = _sides(d1, u1)
    up, dn = 0, 1
    strings = [(("C", 2 * 0 + up), [(True, 0)]), (("C", 2 * (k - 2) + dn), [(True, 2 * (k - 2) + dn)]),
               (("A", 2 * 1 + up, 2 * (k - 2) + dn), [(True, 2 * 1 + up), (True, 2 * (k - 2) + dn)]),
               (("B", 2 * (k - 3) + dn, 2 * 2 + dn), [(True, 2 * (k - 3) + dn), (False, 2 * 2 + dn)]),
               (("B", 2 * 4 + up, 2 * (k - 2) + dn), [(True, 2 * 4 + up), (False, 2 * (k - 2) + dn)])]
    w, n = _check_definition(d1, u1, Ls, True, strings)
    print("  expanded left block: %d blocks, max |lib - definition| = %.2e" % (n, w))
    assert w <= 1e-11
    r0, r1 = k + 1, L - 1
    strings = [(("C", 2 * r0 + dn), [(True, 2 * r0 + dn)]), (("C", 2 * r1 + up), [(True, 2 * r1 + up)]),
               (("A", 2 * r0 + up, 2 * r1 + up), [(True, 2 * r0 + up), (True, 2 * r1 + up)]),
               (("B", 2 * (r1 - 1) + up, 2 * (r0 + 1) + up), [(True, 2 * (r1 - 1) + up), (False, 2 * (r0 + 1) + up)]),
               (("B", 2 * (r0 + 2) + dn, 2 * (r1 - 2) + up), [(True, 2 * (r0 + 2) + dn), (False, 2 * (r1 - 2) + up)])]
    w, n = _check_definition(d1, u1, Rs, False, strings)
    print("  expanded right block: %d blocks, max |lib - definition| = %.2e" % (n, w))
    assert w <= 1e-11
    secL = u1.sectors[k - 1]
    q_new = max(secL, key=lambda q: secL[q])
    w, nS = _one_step(d1, T, V, u1, True, q_new, [k - 1, L - 1])
    print("  expanded left block, sector %s: H and %d S blocks, max |lib - oracle step| = %.2e" % (q_new, nS, w))
    assert w <= 1e-10
    d1.close()


def _reduced_against_refs(orc, y_red, chosen, refs, u1_off):
    """Sampled reduced blocks of the library's result against R^T applied to the oracle's U(1) blocks."""
    Rc = orc.R.tocsc()
    red_blocks = orc.psi_blocks
    red_off = np.cumsum([0] + [b[5] * b[6] for b in red_blocks])
    y_orc = np.zeros(orc.n_u1)
    have = np.zeros(orc.n_u1, dtype=bool)
    for i, m in refs.items():
        y_orc[u1_off[i]:u1_off[i + 1]] = m.reshape(-1)
        have[u1_off[i]:u1_off[i + 1]] = True
    out = []
    for j in chosen:
        cols = Rc[:, red_off[j]:red_off[j + 1]]
        assert have[np.unique(cols.indices)].all()          # every U(1) element the block expands into was computed
        ref = cols.T @ y_orc
        got = y_red[red_off[j]:red_off[j + 1]]
        out.append((j, red_blocks[j][5], red_blocks[j][6], np.linalg.norm(got - ref) / np.linalg.norm(ref)))
    return out


def test_config4_su2_4096_multiplets_sampled_blocks_against_the_oracle():
    """BASELINE configs[4] at its full size (L = 56, 40 electrons, SU(2), 4096 multiplets, Cr2-like integrals; U(1)-
    equivalent ~17000 states — no U(1) run of that size fits one GPU).  The reduced operator blocks the sampled
    output blocks need are exported, expanded to U(1) operator blocks by the Wigner-Eckart theorem with the oracle's
    Clebsch-Gordan coefficients (lean_helpers.ExportedSideSU2), checked against their definition on the expanded MPS
    and against one oracle blocking step, and handed to the lean U(1) oracle."""
    import torch
    from oracle import su2
    from paper_2501_18263_b200.binding import DMRG
    T, V, mps = inputs.make_config_su2(4)
    c = inputs.SU2_CONFIGS[4]
    n2 = mps.N // 2
    k, L = mps.k, mps.L
    t0 = time.time()
    orc = su2.SU2TwoSiteOracle(T, V, mps, inputs.psi_blocks_su2(mps))        # expansion maps only
    u1 = inputs.MPSInput(L=L, k=k, n_up=n2, n_dn=n2, sectors=orc.u1.sectors, left=orc.u1.left, right=orc.u1.right)
    pb = orc.u1_blocks
    print("config 4: expansion maps %.0f s, U(1)-equivalent bond %d, psi_u1 %d" % (time.time() - t0, sum(u1.sectors[k].values()), orc.n_u1))
    v = inputs.make_psi0_su2(mps, c["seed"])
    t0 = time.time()
    d2 = DMRG(L, n2, n2, su2=True, env_cache_bytes=72 << 30)
    d2.setup(T, V, mps)
    y_red = d2.heff_apply(torch.from_numpy(v).cuda()).cpu().numpy()
    st = d2.stats()
    print("config 4: library setup + apply %.0f s, %.3e flops per apply, %d reduced elements" % (time.time() - t0, st["flops_apply"], len(v)))
    xe = orc.expand(v)

    def mk(code, orbs, bond):
        return ExportedSideSU2(d2, code, orbs, orc.lay[bond], mps.N)
    red_blocks = orc.psi_blocks
    red_off = np.cumsum([0] + [b[5] * b[6] for b in red_blocks])
    u1_off = np.cumsum([0] + [b[4] * b[5] for b in pb])
    Rc = orc.R.tocsc()

    def images(j):
        rows = np.unique(Rc[:, red_off[j]:red_off[j + 1]].indices)
        return sorted(set((np.searchsorted(u1_off, rows, side="right") - 1).tolist()))
    rng = np.random.default_rng(11)
    chosen = []
    for j in rng.permutation(len(red_blocks)).tolist():
        if len(chosen) >= 10:
            break
        im = images(j)
        if red_blocks[j][5] * red_blocks[j][6] >= 64 and len(im) <= 10 and max(pb[i][4] * pb[i][5] for i in im) <= 30000:
            chosen.append(j)
    assert len(chosen) >= 10
    need = set()
    for j in chosen:
        need |= set(images(j))
    t0 = time.time()
    _, nbytes, refs = lean_parity(d2, T, V, u1, xe, None, sorted(need), keep_refs=True, mk=mk, group_elems=40000)
    print("config 4: %d reduced blocks -> %d U(1) blocks, %.1f GB of reduced operator blocks exported, %.0f s" % (len(chosen), len(need), nbytes / 1e9, time.time() - t0))
    worst = 0.0
    for j, dL, dR, e2 in _reduced_against_refs(orc, y_red, chosen, refs, u1_off):
        print("  reduced block %4d  %3d x %3d  rel-L2 %.2e" % (j, dL, dR, e2))
        worst = max(worst, e2)
    assert worst <= TOL
    # ---- the expanded operator blocks themselves, at this size ----
    Ls, Rs = _sides(d2, u1, mk)
    up, dn = 0, 1
    hi = k - 2
    strings = [(("C", 2 * hi + up), [(True, 2 * hi + up)]), (("C", 2 * (hi - 1) + dn), [(True, 2 * (hi - 1) + dn)]),
               (("A", 2 * (hi - 2) + up, 2 * hi + up), [(True, 2 * (hi - 2) + up), (True, 2 * hi + up)]),
               (("A", 2 * (hi - 1) + up, 2 * hi + dn), [(True, 2 * (hi - 1) + up), (True, 2 * hi + dn)]),
               (("A", 2 * (hi - 1) + dn, 2 * hi + up), [(True, 2 * (hi - 1) + dn), (True, 2 * hi + up)]),
               (("A", 2 * hi + up, 2 * hi + dn), [(True, 2 * hi + up), (True, 2 * hi + dn)]),
               (("A", 2 * 3 + dn, 2 * hi + dn), [(True, 2 * 3 + dn), (True, 2 * hi + dn)]),
               (("B", 2 * hi + up, 2 * (hi - 1) + up), [(True, 2 * hi + up), (False, 2 * (hi - 1) + up)]),
               (("B", 2 * (hi - 2) + dn, 2 * hi + dn), [(True, 2 * (hi - 2) + dn), (False, 2 * hi + dn)]),
               (("B", 2 * hi + up, 2 * (hi - 1) + dn), [(True, 2 * hi + up), (False, 2 * (hi - 1) + dn)]),
               (("B", 2 * (hi - 1) + dn, 2 * 5 + up), [(True, 2 * (hi - 1) + dn), (False, 2 * 5 + up)])]
    t0 = time.time()
    w, n = _check_definition(d2, u1, Ls, True, strings, nkeep=(1, 2), max_dim=160)
    print("  left block: %d expanded blocks of %d operators, max |lib - definition| = %.2e (%.0f s)" % (n, len(strings), w, time.time() - t0))
    assert w <= 1e-11
    r0, r1 = k + 1, L - 1
    strings = [(("C", 2 * r0 + up), [(True, 2 * r0 + up)]), (("C", 2 * (r0 + 1) + dn), [(True, 2 * (r0 + 1) + dn)]),
               (("A", 2 * r0 + up, 2 * (r0 + 2) + up), [(True, 2 * r0 + up), (True, 2 * (r0 + 2) + up)]),
               (("A", 2 * r0 + up, 2 * (r0 + 1) + dn), [(True, 2 * r0 + up), (True, 2 * (r0 + 1) + dn)]),
               (("A", 2 * r0 + dn, 2 * (r0 + 1) + up), [(True, 2 * r0 + dn), (True, 2 * (r0 + 1) + up)]),
               (("A", 2 * r0 + up, 2 * r0 + dn), [(True, 2 * r0 + up), (True, 2 * r0 + dn)]),
               (("A", 2 * r0 + dn, 2 * r1 + dn), [(True, 2 * r0 + dn), (True, 2 * r1 + dn)]),
               (("B", 2 * r0 + up, 2 * (r0 + 1) + up), [(True, 2 * r0 + up), (False, 2 * (r0 + 1) + up)]),
               (("B", 2 * (r0 + 2) + dn, 2 * r0 + dn), [(True, 2 * (r0 + 2) + dn), (False, 2 * r0 + dn)]),
               (("B", 2 * r0 + up, 2 * (r0 + 1) + dn), [(True, 2 * r0 + up), (False, 2 * (r0 + 1) + dn)]),
               (("B", 2 * (r0 + 1) + dn, 2 * (r1 - 3) + up), [(True, 2 * (r0 + 1) + dn), (False, 2 * (r1 - 3) + up)])]
    t0 = time.time()
    w, n = _check_definition(d2, u1, Rs, False, strings, nkeep=(1, 2), max_dim=160)
    print("  right block: %d expanded blocks of %d operators, max |lib - definition| = %.2e (%.0f s)" % (n, len(strings), w, time.time() - t0))
    assert w <= 1e-11
    secL = u1.sectors[k - 1]
    q_new = max((q for q in secL if secL[q] <= 120), key=lambda q: secL[q])
    w, nS = _one_step(d2, T, V, u1, True, q_new, [k - 1, L - 1], mk=mk)
    print("  left block, U(1) sector %s (dim %d): H and %d S blocks, max |lib - oracle step| = %.2e" % (q_new, secL[q_new], nS, w))
    assert nS >= 2 and w <= 1e-10
    secR = Rs.sectors
    q_new = max((q for q in secR if secR[q] <= 120), key=lambda q: secR[q])
    w, nS = _one_step(d2, T, V, u1, False, q_new, [0, k], mk=mk)
    print("  right block, U(1) sector %s (dim %d): H and %d S blocks, max |lib - oracle step| = %.2e" % (q_new, secR[q_new], nS, w))
    assert nS >= 2 and w <= 1e-10
    d2.close()

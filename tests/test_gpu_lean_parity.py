"""Element-wise GPU-vs-oracle parity of H_eff.psi at BASELINE configs[3] (U(1)xU(1), D = 4096) on sampled output
blocks (`-m gpu`).

The full oracle (`oracle/dmrg.py`) cannot reach this size (hours for the environments, ~150 GB for the superblock
terms), so, as SURVEY.md 8(c) "Large configs" lays out:
  * `oracle/lean.py` evaluates (H_eff psi){block} for chosen output blocks with the oracle's own formulas, from
    block operators restricted to the sectors that can contribute;
  * those operator blocks are read from the library (`dmrg_env_export_block`), whose blocking is pinned element-wise
    at configs 0-2 (tests/test_gpu_parity.py) — and a sample of them is checked HERE, at full size, against the
    oracle: normal operators against their definition (`lean.block_operator_by_definition`, straight from the MPS
    tensors), H and S against one oracle enlarge-and-project step from the predecessor block.
The same machinery is run at configs[1] first, where the full oracle is available, to pin the glue code.
"""
import time

import numpy as np
import pytest

from lean_helpers import ExportedSide, choose_blocks, rel_block_errors
from oracle import dmrg as odmrg
from oracle import lean
from paper_2501_18263_b200 import inputs

pytestmark = pytest.mark.gpu

TOL = 1e-11          # north_star: rel-L2 <= 1e-11, here per block


def _ctx(T, V, mps, **kw):
    import torch
    from paper_2501_18263_b200.binding import DMRG
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    d = DMRG(mps.L, mps.n_up, mps.n_dn, **kw)
    d.setup(T, V, mps)
    return d


def u1_side_factory(d, mps):
    """mk(side code, orbitals, bond): the exported block whose open bond is `bond` (U(1)xU(1) context)."""
    N = (mps.n_up, mps.n_dn)

    def mk(code, orbs, bond):
        sec = mps.sectors[bond] if code in (0, 2) else {odmrg.qsub(N, q): dim for q, dim in mps.sectors[bond].items()}
        return ExportedSide(d, code, orbs, sec, N)
    return mk


def _sides(d, mps, mk=None):
    k, L = mps.k, mps.L
    mk = mk or u1_side_factory(d, mps)
    return mk(0, range(0, k - 1), k - 1), mk(1, range(k + 1, L), k + 1)


def _offsets(pb):
    off, o = [], 0
    for b in pb:
        off.append(o)
        o += b[4] * b[5]
    return off


def lean_parity(d, T, V, mps, v, got_flat, idxs, group_elems=60000, keep_refs=False, mk=None):
    """Compares the library's psi' blocks `idxs` with the lean oracle fed by exported operator blocks.
    Blocks are processed in groups (bounded export size).  Returns list of (idx, dL, dR, rel-L2, rel-max); with
    got_flat = None only the oracle's blocks are computed (keep_refs)."""
    pb = inputs.psi_blocks(mps)
    N, L = (mps.n_up, mps.n_dn), mps.L
    off = _offsets(pb)
    Ls, Rs = _sides(d, mps, mk)
    order = sorted(idxs, key=lambda i: pb[i][4] * pb[i][5])
    groups, cur, acc = [], [], 0
    for i in order:
        sz = pb[i][4] * pb[i][5]
        if cur and acc + sz > group_elems:
            groups.append(cur); cur, acc = [], 0
        cur.append(i); acc += sz
    if cur:
        groups.append(cur)
    res, refs = [], {}
    for g in groups:
        qL = {pb[i][0] for i in g}
        qR = {odmrg.qsub(N, pb[i][3]) for i in g}
        lo = lean.LeanTwoSiteOracle(T, V, mps.n_up, mps.n_dn, mps.k, pb, Ls.block(qL, L), Rs.block(qR, L))
        ref = lo.apply_blocks(v, g)
        for i in g:
            dL, dR = pb[i][4], pb[i][5]
            if got_flat is not None:
                got = got_flat[off[i]:off[i] + dL * dR].reshape(dL, dR)
                res.append((i, dL, dR) + rel_block_errors(got, ref[i]))
            if keep_refs:
                refs[i] = ref[i]
        del lo, ref
    return res, Ls.bytes + Rs.bytes, refs


def test_lean_machinery_against_the_full_oracle_config1():
    """BASELINE configs[1]: exported blocks + lean oracle == full oracle == library, block by block."""
    import torch
    T, V, mps = inputs.make_config(1)
    v = inputs.make_psi0(mps, inputs.CONFIGS[1]["seed"])
    d = _ctx(T, V, mps)
    got = d.heff_apply(torch.from_numpy(v).cuda()).cpu().numpy()
    pb = inputs.psi_blocks(mps)
    idxs = choose_blocks(pb, 10, seed=1)
    res, _, _ = lean_parity(d, T, V, mps, v, got, idxs, group_elems=2000)
    d.close()
    for i, dL, dR, r2, rmax in res:
        assert r2 <= TOL and rmax <= 10 * TOL, (i, dL, dR, r2, rmax)
    orc = odmrg.TwoSiteOracle(T, V, mps.n_up, mps.n_dn, mps.k, mps.sectors, mps.left, mps.right, pb)
    orc.build_env()
    full = orc.apply(v)
    assert np.linalg.norm(got - full) / np.linalg.norm(full) <= TOL


@pytest.fixture(scope="module")
def config3():
    import torch
    T, V, mps = inputs.make_config(3)
    v = inputs.make_psi0(mps, inputs.CONFIGS[3]["seed"])
    # the environment cache must keep the predecessor blocks (sites 1..k-2 and k+3..L) on the device
    d = _ctx(T, V, mps, env_cache_bytes=48 << 30)
    got = d.heff_apply(torch.from_numpy(v).cuda()).cpu().numpy()
    yield T, V, mps, v, d, got
    d.close()


def test_config3_u1_d4096_sampled_blocks_against_the_oracle(config3):
    """>= 20 output blocks: every tile shape, the heaviest block, random ones; rel-L2 <= 1e-11 per block."""
    T, V, mps, v, d, got = config3
    pb = inputs.psi_blocks(mps)
    assert len(got) == 8085937
    idxs = choose_blocks(pb, 30, seed=3, max_elems=30000)
    assert len(idxs) >= 30
    t0 = time.time()
    res, nbytes, _ = lean_parity(d, T, V, mps, v, got, idxs)
    print("config 3: %d blocks, %.1f GB of operator blocks exported, %.0f s" % (len(res), nbytes / 1e9, time.time() - t0))
    for i, dL, dR, r2, rmax in res:
        print("  block %4d  %3d x %3d  rel-L2 %.2e  max %.2e" % (i, dL, dR, r2, rmax))
    shapes = set()
    from lean_helpers import tile_shapes
    for i, dL, dR, r2, rmax in res:
        shapes |= tile_shapes(dL, dR)
        assert r2 <= TOL and rmax <= 10 * TOL, (i, dL, dR, r2, rmax)
    assert len(shapes) == 9
    assert max(dL * dR for _, dL, dR, _, _ in res) == max(b[4] * b[5] for b in pb)


def _check_definition(d, mps, side_obj, left, strings, nkeep=(2, 2), max_dim=10 ** 9):
    """Exported normal operators against <b'|o_1 o_2|b> evaluated from the MPS tensors (every exported sector)."""
    N = (mps.n_up, mps.n_dn)
    k, L = mps.k, mps.L
    sites = list(range(1, k)) if left else list(range(k + 2, L + 1))
    tensors = mps.left if left else mps.right
    qs = sorted((q for q in side_obj.sectors if side_obj.sectors[q] <= max_dim), key=lambda q: -side_obj.sectors[q])
    keep = set(qs[:nkeep[0]] + qs[len(qs) // 2:len(qs) // 2 + nkeep[1]])      # the largest sectors and mid-sized ones
    blk = side_obj.block(keep, L, want=("C", "A", "B"))
    worst, nchecked = 0.0, 0
    for name, string in strings:
        ref = lean.block_operator_by_definition(tensors, sites, string, left)
        got = blk.ops[name]
        assert len(got) > 0, name
        for (co, ci), m in got.items():
            key = (co, ci) if left else (odmrg.qsub(N, co), odmrg.qsub(N, ci))
            r = ref.get(key)
            assert r is not None and r.shape == m.shape, (name, co, ci)
            worst = max(worst, np.abs(m - r).max())
            nchecked += 1
        # and nothing is missing: every block of the definition that touches `keep` was exported
        for (lo_, li_), r in ref.items():
            co, ci = (lo_, li_) if left else (odmrg.qsub(N, lo_), odmrg.qsub(N, li_))
            if (co in keep or ci in keep) and np.abs(r).max() > 1e-13:
                assert (co, ci) in got, (name, co, ci)
    return worst, nchecked


def test_config3_exported_operators_against_their_definition(config3):
    """>= 10 carried normal operators per side at D = 4096 against the site-by-site evaluation of their definition."""
    T, V, mps, v, d, got = config3
    k, L = mps.k, mps.L
    Ls, Rs = _sides(d, mps)
    lo, hi = 0, k - 2                 # left orbitals 0..k-2
    up, dn = 0, 1
    left_strings = [
        (("C", 2 * lo + up), [(True, 2 * lo + up)]),
        (("C", 2 * hi + dn), [(True, 2 * hi + dn)]),
        (("C", 2 * (hi // 2) + up), [(True, 2 * (hi // 2) + up)]),
        (("A", 2 * lo + up, 2 * hi + up), [(True, 2 * lo + up), (True, 2 * hi + up)]),
        (("A", 2 * 3 + dn, 2 * 7 + dn), [(True, 2 * 3 + dn), (True, 2 * 7 + dn)]),
        (("A", 2 * 5 + up, 2 * 5 + dn), [(True, 2 * 5 + up), (True, 2 * 5 + dn)]),
        (("A", 2 * 2 + dn, 2 * 9 + up), [(True, 2 * 2 + dn), (True, 2 * 9 + up)]),       # -AUD[9,2] in the library
        (("B", 2 * lo + up, 2 * hi + up), [(True, 2 * lo + up), (False, 2 * hi + up)]),
        (("B", 2 * hi + dn, 2 * 4 + dn), [(True, 2 * hi + dn), (False, 2 * 4 + dn)]),
        (("B", 2 * 6 + up, 2 * 6 + up), [(True, 2 * 6 + up), (False, 2 * 6 + up)]),
        (("B", 2 * 8 + up, 2 * 1 + dn), [(True, 2 * 8 + up), (False, 2 * 1 + dn)]),
        (("B", 2 * 1 + dn, 2 * 8 + up), [(True, 2 * 1 + dn), (False, 2 * 8 + up)]),       # BUD[8,1]^T in the library
    ]
    w, n = _check_definition(d, mps, Ls, True, left_strings)
    print("left block: %d exported blocks of %d operators, max |lib - definition| = %.2e" % (n, len(left_strings), w))
    assert w <= 1e-11
    r0, r1 = k + 1, L - 1             # right orbitals k+1..L-1
    mid = (r0 + r1) // 2
    right_strings = [
        (("C", 2 * r0 + up), [(True, 2 * r0 + up)]),
        (("C", 2 * r1 + dn), [(True, 2 * r1 + dn)]),
        (("C", 2 * mid + dn), [(True, 2 * mid + dn)]),
        (("A", 2 * r0 + up, 2 * r1 + up), [(True, 2 * r0 + up), (True, 2 * r1 + up)]),
        (("A", 2 * (r0 + 2) + dn, 2 * mid + dn), [(True, 2 * (r0 + 2) + dn), (True, 2 * mid + dn)]),
        (("A", 2 * mid + up, 2 * mid + dn), [(True, 2 * mid + up), (True, 2 * mid + dn)]),
        (("A", 2 * (r0 + 1) + dn, 2 * (r1 - 1) + up), [(True, 2 * (r0 + 1) + dn), (True, 2 * (r1 - 1) + up)]),
        (("B", 2 * r0 + up, 2 * r1 + up), [(True, 2 * r0 + up), (False, 2 * r1 + up)]),
        (("B", 2 * r1 + dn, 2 * (r0 + 3) + dn), [(True, 2 * r1 + dn), (False, 2 * (r0 + 3) + dn)]),
        (("B", 2 * mid + dn, 2 * mid + dn), [(True, 2 * mid + dn), (False, 2 * mid + dn)]),
        (("B", 2 * (r1 - 2) + up, 2 * (r0 + 1) + dn), [(True, 2 * (r1 - 2) + up), (False, 2 * (r0 + 1) + dn)]),
        (("B", 2 * (r0 + 1) + dn, 2 * (r1 - 2) + up), [(True, 2 * (r0 + 1) + dn), (False, 2 * (r1 - 2) + up)]),
    ]
    w, n = _check_definition(d, mps, Rs, False, right_strings)
    print("right block: %d exported blocks of %d operators, max |lib - definition| = %.2e" % (n, len(right_strings), w))
    assert w <= 1e-11


def _one_step(d, T, V, mps, left, q_new, s_orbs, mk=None):
    """H{q_new, q_new} and S_x{.., q_new} (x in s_orbs) of the current block from ONE oracle enlarge-and-project step
     applied to the exported predecessor block; compared with the exported current block."""
    N = (mps.n_up, mps.n_dn)
    k, L = mps.k, mps.L
    w = odmrg.w_from_V(V)
    mk = mk or u1_side_factory(d, mps)
    if left:
        site = k - 1                                   # absorbed site (1-based); orbital k-2
        old = mk(2, range(0, k - 2), k - 2)
        new = mk(0, range(0, k - 1), k - 1)
        iso = {(qi, odmrg.SITE_Q[s]): A for (qi, s), A in mps.left[site].items()}
    else:
        site = k + 2                                   # orbital k+1
        old = mk(3, range(k + 2, L), k + 2)
        new = mk(1, range(k + 1, L), k + 1)
        iso = {}
        for (qi, s), Bm in mps.right[site].items():
            qo = odmrg.qadd(qi, odmrg.SITE_Q[s])
            iso[(odmrg.SITE_Q[s], odmrg.qsub(N, qo))] = Bm.T
    # new sectors touched: q_new and, for S_x (which lowers the particle number by one), q_new - e_sigma
    targets = {q_new, (q_new[0] - 1, q_new[1]), (q_new[0], q_new[1] - 1)} & set(new.sectors)
    old_q = set()
    for q in targets:
        for s in range(4):
            qo = odmrg.qsub(q, odmrg.SITE_Q[s])
            if qo in old.sectors:
                old_q.add(qo)
    oldb = old.block(old_q, L, s_orbs=set(s_orbs) | {site - 1})
    sb = odmrg.site_block(site - 1, T, w, L)
    keep = {key for key in iso if odmrg.qadd(*key) in targets}
    E = odmrg.enlarge(oldb, sb, T, w, list(s_orbs), want_normal=False, keep=keep) if left else \
        odmrg.enlarge(sb, oldb, T, w, list(s_orbs), want_normal=False, keep=keep)
    newb = new.block({q_new}, L, want=("H", "S"), s_orbs=set(s_orbs))
    worst = 0.0
    ref = odmrg.project(E.ops["H"], iso)
    worst = max(worst, np.abs(ref[(q_new, q_new)] - newb.ops["H"][(q_new, q_new)]).max())
    nS = 0
    for x in s_orbs:
        for s in (0, 1):
            ref = odmrg.project(E.ops[("S", 2 * x + s)], iso)
            qo = (q_new[0] - 1, q_new[1]) if s == 0 else (q_new[0], q_new[1] - 1)
            if qo not in new.sectors:
                continue
            g = newb.ops[("S", 2 * x + s)].get((qo, q_new))
            assert g is not None
            worst = max(worst, np.abs(ref[(qo, q_new)] - g).max())
            nS += 1
    return worst, nS


def test_config3_exported_H_and_S_against_one_oracle_blocking_step(config3):
    """The three-operator complementary operators S_x and the block Hamiltonians at D = 4096: one oracle
    enlarge-and-project step from the exported predecessor block reproduces the exported blocks."""
    T, V, mps, v, d, got = config3
    N = (mps.n_up, mps.n_dn)
    k, L = mps.k, mps.L
    secL = mps.sectors[k - 1]
    qs = sorted(secL, key=lambda q: -secL[q])
    for q_new in (qs[0], qs[len(qs) // 3]):
        w, nS = _one_step(d, T, V, mps, True, q_new, [k - 1, k, L - 1])
        print("left block, sector %s (dim %d): H and %d S blocks, max |lib - oracle step| = %.2e" % (q_new, secL[q_new], nS, w))
        assert nS >= 4 and w <= 1e-10
    secR = {odmrg.qsub(N, q): dim for q, dim in mps.sectors[k + 1].items()}
    qs = sorted(secR, key=lambda q: -secR[q])
    for q_new in (qs[0], qs[len(qs) // 3]):
        w, nS = _one_step(d, T, V, mps, False, q_new, [0, k - 1, k])
        print("right block, sector %s (dim %d): H and %d S blocks, max |lib - oracle step| = %.2e" % (q_new, secR[q_new], nS, w))
        assert nS >= 4 and w <= 1e-10

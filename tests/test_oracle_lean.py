"""Pins for oracle/lean.py (no GPU): the output-block-restricted H_eff psi against the full oracle apply and
against the definition P^T H_FCI P, and `block_operator_by_definition` against explicit Fock-space embeddings."""
import numpy as np
import pytest

import helpers
from oracle import dmrg, fci, lean
from oracle.blockops import BlockOp
from paper_2501_18263_b200 import inputs
from test_oracle_dmrg import _herm_V, _jw_site_ops, _oracle


def restrict_block(blk, keep_q):
    """Copy of a dmrg.Block whose operators hold only the sector blocks with out or in sector in keep_q
    (what a test can afford to export from the library at BASELINE configs 3-4)."""
    out = dmrg.Block(blk.orbs, blk.sectors)
    for name, op in blk.ops.items():
        out.ops[name] = BlockOp({(qo, qi): m for (qo, qi), m in op.items() if qo in keep_q or qi in keep_q})
    return out


def _blocks_of(orc, v):
    psi = orc.unflatten(v)
    return [psi[((qL, dmrg.SITE_Q[s1]), (dmrg.SITE_Q[s2], dmrg.qsub(orc.N, qRb)))] for (qL, s1, s2, qRb, _, _) in orc.psi_blocks]


@pytest.mark.parametrize("L,nu,nd,k,D", [(6, 3, 3, 3, 12), (6, 2, 3, 4, 8), (5, 3, 2, 3, 10 ** 9), (6, 3, 3, 1, 7), (6, 3, 3, 5, 7)])
def test_lean_blocks_equal_projected_fci(L, nu, nd, k, D):
    """Every output block, one at a time and all together, with block operators restricted to the sectors that can
    contribute: equal to the same block of P^T H_FCI P psi (V has no symmetry beyond Hermiticity)."""
    rng = np.random.default_rng(100 * L + k)
    T = rng.normal(size=(L, L)); T = T + T.T
    V = _herm_V(rng, L)
    mps = inputs.make_mps(L, nu, nd, D, k, seed=5)
    orc, pb = _oracle(T, V, mps)
    P, _ = helpers.embedding(mps, pb)
    H, _ = fci.fci_hamiltonian(T, V, nu, nd)
    v = rng.normal(size=P.shape[1])
    ref = _blocks_of(orc, P.T @ (H @ (P @ v)))
    N = (nu, nd)
    for idxs in [[i] for i in range(len(pb))] + [list(range(len(pb)))] + [list(range(0, len(pb), 3))]:
        qL = {pb[i][0] for i in idxs}
        qR = {dmrg.qsub(N, pb[i][3]) for i in idxs}
        lo = lean.LeanTwoSiteOracle(T, V, nu, nd, k, pb, restrict_block(orc.Lblock, qL), restrict_block(orc.Rblock, qR))
        got = lo.apply_blocks(v, idxs)
        for i in idxs:
            assert np.abs(got[i] - ref[i]).max() <= 1e-12 * max(1.0, np.abs(ref[i]).max())


def test_lean_blocks_equal_full_oracle_config0_and_config1():
    """BASELINE configs[0] (every block) and configs[1] (a sample): lean == TwoSiteOracle.apply to rounding."""
    for cfg, sample in ((0, None), (1, 12)):
        T, V, mps = inputs.make_config(cfg)
        orc, pb = _oracle(T, V, mps)
        v = inputs.make_psi0(mps, inputs.CONFIGS[cfg]["seed"])
        ref = _blocks_of(orc, orc.apply(v))
        idxs = list(range(len(pb))) if sample is None else sorted(np.random.default_rng(3).choice(len(pb), sample, replace=False).tolist())
        N = (mps.n_up, mps.n_dn)
        qL = {pb[i][0] for i in idxs}
        qR = {dmrg.qsub(N, pb[i][3]) for i in idxs}
        lo = lean.LeanTwoSiteOracle(T, V, mps.n_up, mps.n_dn, mps.k, pb, restrict_block(orc.Lblock, qL),
                                    restrict_block(orc.Rblock, qR))
        got = lo.apply_blocks(v, idxs)
        scale = max(np.abs(r).max() for r in ref)
        for i in idxs:
            assert np.abs(got[i] - ref[i]).max() <= 1e-13 * scale


def _dense_string(cre, ann, string):
    n4 = next(iter(cre.values())).shape[0]
    M = np.eye(n4)
    for c, (i, s) in string:
        M = M @ (cre[(i, s)] if c else ann[(i, s)])
    return M


def test_block_operator_by_definition_left_and_right():
    """<b'|o_1..o_n|b> from the site-by-site contraction == V^T O_JW V with the block states V written out in the
    site-product basis and O_JW the Kronecker Jordan-Wigner matrices; also == the operators the blocking carries."""
    rng = np.random.default_rng(17)
    L, nu, nd, k = 7, 3, 3, 4
    T = rng.normal(size=(L, L)); T = T + T.T
    V = _herm_V(rng, L)
    mps = inputs.make_mps(L, nu, nd, 11, k, seed=9)
    orc, _ = _oracle(T, V, mps)
    # ---- left block: sites 1..3 (orbitals 0..2) ----
    n = k - 1
    vec = helpers.left_vectors(mps, n)
    cre = _jw_site_ops(n)
    ann = {key: m.T for key, m in cre.items()}
    strings = [[(True, (1, 0))], [(False, (2, 1))], [(True, (0, 1)), (True, (2, 0))], [(True, (2, 1)), (False, (0, 1))],
               [(True, (1, 0)), (False, (1, 0))], [(True, (0, 0)), (False, (2, 0)), (False, (1, 1))]]
    for st in strings:
        dense = _dense_string(cre, ann, st)
        got = lean.block_operator_by_definition(mps.left, list(range(1, n + 1)), [(c, 2 * i + s) for c, (i, s) in st], True)
        for qo in vec:
            for qi in vec:
                ref = vec[qo].T @ dense @ vec[qi]
                g = got.get((qo, qi))
                assert np.abs((g if g is not None else 0.0) - ref).max() < 1e-13
    got = lean.block_operator_by_definition(mps.left, [1, 2, 3], [(True, 1), (True, 4)], True)
    for key, m in orc.Lblock.ops[("A", 1, 4)].items():
        assert np.abs(got[key] - m).max() < 1e-13
    # ---- right block: sites 6..7 (orbitals 5, 6); states written out with site 6 most significant ----
    first = k + 2
    nR = L - first + 1
    rvec = helpers.right_vectors(mps, first)           # keyed by bond label
    creR = _jw_site_ops(nR)                             # local site index 0 = orbital first-1
    annR = {key: m.T for key, m in creR.items()}
    o0 = first - 1
    for st in [[(True, (o0, 0))], [(True, (o0 + 1, 1))], [(True, (o0, 1)), (False, (o0 + 1, 1))],
               [(True, (o0 + 1, 0)), (True, (o0, 1))]]:
        dense = _dense_string(creR, annR, [(c, (i - o0, s)) for c, (i, s) in st])
        got = lean.block_operator_by_definition(mps.right, list(range(first, L + 1)), [(c, 2 * i + s) for c, (i, s) in st], False)
        for qo in rvec:
            for qi in rvec:
                ref = rvec[qo].T @ dense @ rvec[qi]
                g = got.get((qo, qi))
                assert np.abs((g if g is not None else 0.0) - ref).max() < 1e-13
    # the carried right-block operators are keyed by the block's content N - label
    N = (nu, nd)
    got = lean.block_operator_by_definition(mps.right, list(range(first, L + 1)), [(True, 2 * o0 + 1), (False, 2 * (o0 + 1))], False)
    ref = orc.Rblock.ops[("B", 2 * o0 + 1, 2 * (o0 + 1))]
    assert len(ref) > 0
    for (co, ci), m in ref.items():
        assert np.abs(got[(dmrg.qsub(N, co), dmrg.qsub(N, ci))] - m).max() < 1e-13

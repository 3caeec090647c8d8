"""ORACLE (test infrastructure, CPU only): H_eff psi on a chosen list of output blocks, and block
operators straight from their definition.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs may
import this file; it shares no code with the CUDA path and never calls it.

Why it exists.  `oracle/dmrg.py:TwoSiteOracle` forms every enlarged operator of L' = L u k and
R' = k+1 u R on ALL sector blocks before it applies H_eff — ~150 GB at BASELINE
configs[3] (D = 4096).  A parity check only needs some output blocks of psi' = H_eff psi, and one
output block ((q_L', s_k'), (s_k+1', q_R')) receives contributions only from the sub-blocks of the
L' operators whose out (or, for the transposed half of a "+ h.c." term, in) key is (q_L', s_k'), and
likewise for R'.  `LeanTwoSiteOracle` therefore runs THE SAME code — `enlarge`, `comp_P_many`,
`comp_Q_many`, `TwoSiteOracle.terms`, `TwoSiteOracle._accumulate`, i.e. PAPER.md Eq. (6)-(8)
 in the hierarchical form of PAPER.md:129 — with the Kronecker products
restricted to the sub-blocks that touch the chosen keys (`blockops.product(keep=...)`).  No formula
of its own; memory = the block operators handed in + the restricted products.

The block operators are GIVEN as `dmrg.Block` objects (they may hold only the sector blocks that
can contribute: out or in sector among the chosen q_L' resp. q_R').  At configs 0-2 they come from
the oracle's own `build_left` / `build_right`; at configs 3-4, where those take hours, the tests
fill them from the library's exported blocks (`dmrg_env_export_block`) and check a sample of the
exported blocks against `block_operator_by_definition` below and against one oracle
enlarge-and-project step (SURVEY.md 8(c) "Large configs").

Pins (tests/test_oracle_lean.py): `apply_blocks` equals the corresponding blocks of
`TwoSiteOracle.apply` and of P^T H_FCI P psi; `block_operator_by_definition` equals V^T (Jordan-Wigner
matrix) V with the block states V written out in the site-product basis, and equals the operators the
blocking recursion carries.
"""
from __future__ import annotations

import numpy as np

from .blockops import qadd, qsub
from .dmrg import SITE_Q, TwoSiteOracle, _CRE


class LeanTwoSiteOracle(TwoSiteOracle):
    """`TwoSiteOracle` with given block operators, evaluated on chosen output blocks only."""

    def __init__(self, T, V, n_up, n_dn, k, psi_blocks, Lblock, Rblock):
        super().__init__(T, V, n_up, n_dn, k, None, None, None, psi_blocks)
        self.Lblock, self.Rblock = Lblock, Rblock

    def block_key(self, idx):
        qL, s1, s2, qRb, _, _ = self.psi_blocks[idx]
        return ((qL, SITE_Q[s1]), (SITE_Q[s2], qsub(self.N, qRb)))

    def apply_blocks(self, v, idxs):
        """dict idx -> (dL, dR) matrix of (H_eff psi) for the psi blocks `idxs` (Eq. (7)/(8))."""
        psi = self.unflatten(np.asarray(v, dtype=np.float64))
        keys = {i: self.block_key(i) for i in idxs}
        out = {key: np.zeros_like(psi[key]) for key in keys.values()}
        keepL = {key[0] for key in keys.values()}
        keepR = {key[1] for key in keys.values()}
        self._accumulate(self.terms(keepL, keepR), psi, out)
        return {i: out[key] for i, key in keys.items()}


# ---------------------------------------------------------------------------------------------
# block operators from their definition (no recursion, no complementary operators)
# ---------------------------------------------------------------------------------------------

_PAR = np.diag([1.0, -1.0, -1.0, 1.0])      # (-1)^n of the site states 0, dn, up, up+dn


def _local_factor(cre, p, site):
    """Jordan-Wigner factor on `site` (1-based) of the elementary operator a+_p / a_p, p = 2*orb + s:
    the local 4x4 matrix on its own site, the parity on the sites before it, 1 after it."""
    orb, s = divmod(p, 2)
    if site == orb + 1:
        return _CRE[s] if cre else _CRE[s].T
    return _PAR if site < orb + 1 else np.eye(4)


def block_operator_by_definition(tensors, sites, string, left):
    """<b'| o_1 o_2 ... o_n |b> over the states of a block, from the MPS tensors alone.

    tensors[i]: dict (q_in, s) -> (d_in, d_out) matrix of site i (Eq. (4), :53), q the
    bond labels (electrons left of the bond); sites: the block's sites in chain order; string: list
    of (cre, p) elementary operators a+_p / a_p (p = 2*orb + s, s = 0 up / 1 down), all inside the
    block, leftmost first.  left = True: block states |b> = sum A^{s_1} .. A^{s_m} |s_1 .. s_m>
    (left-canonical tensors); False: |b> = sum B^{s_m} .. B^{s_L} |s_m .. s_L>.

    Definition used: an elementary operator is the Jordan-Wigner string "parity on the block's
    sites before its own site, local matrix on its site" (the block's own first site starts the
    string, as in oracle/blockops.py), so the matrix element is the site-by-site contraction
      E' = sum_{s', s} M_i[s', s] A^{s'}^T E A^{s}     with M_i = prod_n (factor of o_n on site i).
    Returns dict (label_out, label_in) -> matrix, keyed by the bond labels of the block's open bond.
    """
    def site_matrix(i):
        M = np.eye(4)
        for cre, p in string:
            M = M @ _local_factor(cre, p, i)
        return M

    if left:
        E = {((0, 0), (0, 0)): np.ones((1, 1))}
        for i in sites:
            M, A, new = site_matrix(i), tensors[i], {}
            for (qo, qi), e in E.items():
                for so in range(4):
                    Ao = A.get((qo, so))
                    if Ao is None:
                        continue
                    for si in range(4):
                        if M[so, si] == 0.0:
                            continue
                        Ai = A.get((qi, si))
                        if Ai is None:
                            continue
                        key = (qadd(qo, SITE_Q[so]), qadd(qi, SITE_Q[si]))
                        val = M[so, si] * (Ao.T @ e @ Ai)
                        new[key] = new[key] + val if key in new else val
            E = new
        return E
    # right block: absorb sites from the chain end inwards; E lives on the bond LEFT of the absorbed part
    last = sites[-1]
    qN = None
    for (qi, s) in tensors[last]:
        qN = qadd(qi, SITE_Q[s])
        break
    E = {(qN, qN): np.ones((1, 1))}
    for i in reversed(sites):
        M, B, new = site_matrix(i), tensors[i], {}
        by_out = {}
        for (qi, s), Bm in B.items():
            by_out.setdefault(qadd(qi, SITE_Q[s]), []).append((qi, s, Bm))
        for (qo, qi), e in E.items():
            for (ao, so, Bo) in by_out.get(qo, ()):
                for (ai, si, Bi) in by_out.get(qi, ()):
                    if M[so, si] == 0.0:
                        continue
                    key = (ao, ai)
                    val = M[so, si] * (Bo @ e @ Bi.T)
                    new[key] = new[key] + val if key in new else val
        E = new
    return E

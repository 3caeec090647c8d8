"""ORACLE (test infrastructure, CPU only): two-site DMRG effective Hamiltonian, written from the paper.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this file; it shares no code with the CUDA path and never calls it.

What it computes:  H_eff = P^T H P, the Hamiltonian of
PAPER.md Eq. (1) (with the 1/2 of BASELINE.json, reading R1) projected on the
two-site space H_L (x) H_k (x) H_{k+1} (x) H_R of PAPER.md:97-99, where the block bases are
defined by the left/right-canonical MPS tensors (Eq. (4), :53).  The route is the
factorised form of PAPER.md Eq. (6)-(8), organised hierarchically as
H_eff = H'_L (x) H'_R with H'_L = H_L (x) H_k and H'_R = H_{k+1} (x) H_R exactly as PAPER.md:129
describes, with U(1)xU(1) block-sparse storage.

The paper does not list the terms of Eq. (6); readings R6-R10 fix them.  Here they
follow from ONE identity applied to a pair of neighbouring blocks B1 | B2 (
re-derived in DESIGN.md "Bipartition identity"), with w_ijkl = (V_ijkl + V_jilk)/2:

  H^{B1 u B2} = H^{B1} + H^{B2}
              + sum_{p in B1} (a+_p S^{B2}_p + h.c.) + sum_{p in B2} (a+_p S^{B1}_p + h.c.)
              + sum_{p<q in X} (A_pq P^{Xbar}_pq + h.c.) + sum_{p,q in X} B_pq Q^{Xbar}_pq
  normal operators       C_p = a+_p,  A_pq = a+_p a+_q,  B_pq = a+_p a_q           (p, q in the block)
  complementary (p=(i,s), q=(j,t) outside the block B):
      S_p   = 1/2 sum_{j in B} T_ij a_js + sum_{jkl in B, t} w_ijkl a+_jt a_lt a_ks
      P_pq  = sum_{kl in B} w_ijkl a_lt a_ks
      Q_pq' = delta_{s s'} sum_{jl in B, t} w_ijkl a+_jt a_lt - sum_{jl in B} w_ijlk a+_{j s'} a_{l s}
              (p = (i,s), q' = (k,s'))
  and the recursion  S^{B1 u B2}_p = S^{B1}_p + S^{B2}_p
              + sum_{j in B1} a+_j P^{B2}_{p j} + sum_{j in B2} a+_j P^{B1}_{p j}
              + sum_{k in B1} Q^{B2}_{p k} a_k + sum_{k in B2} Q^{B1}_{p k} a_k .

P and Q are never carried: they are formed from the block's normal operators by the
definitions above.  The same `enlarge` serves the renormalisation step (enlarge, then project
with the MPS tensor) and the superblock (enlarge both sides, do not project).

No blocking, fusion or reordering beyond these formulas.  Pins: tests/test_oracle_*.py
(FCI brute force, Jordan-Wigner definitions, Hermiticity, conservation).
"""
from __future__ import annotations

import numpy as np

import functools

from .blockops import BlockOp, ProdOp, identity, lincomb, project, qadd, qnum, qsub
from .blockops import product as _product

SITE_Q = ((0, 0), (0, 1), (1, 0), (1, 1))  # s = 0, dn, up, up+dn  ->  (n_up, n_dn)

# 4x4 site matrices, rows = out.  |3> = a+_up a+_dn |0>  (R3)
_CU = np.zeros((4, 4)); _CU[2, 0] = 1.0; _CU[3, 1] = 1.0      # a+_up
_CD = np.zeros((4, 4)); _CD[1, 0] = 1.0; _CD[3, 2] = -1.0     # a+_dn
_CRE = (_CU, _CD)


def w_from_V(V):
    """w_ijkl = (V_ijkl + V_jilk)/2: the part of V the operator sum of Eq. (1) can see."""
    return 0.5 * (V + V.transpose(1, 0, 3, 2))


class Block:
    """A block of contiguous orbitals with its sectors and carried operators.

    ops keys: 'H'; ('C', p); ('A', p, q) p<q; ('B', p, q); ('S', p) for p outside the block.
    p, q are spin-orbital indices 2*i + s (s = 0 up, 1 down).
    """

    def __init__(self, orbs, sectors):
        self.orbs = list(orbs)
        self.sectors = dict(sectors)
        self.ops = {}

    def spin_orbs(self):
        return [2 * i + s for i in self.orbs for s in (0, 1)]


def _dense_to_blockop(M):
    op = BlockOp()
    for so in range(4):
        for si in range(4):
            if M[so, si] != 0.0:
                op[(SITE_Q[so], SITE_Q[si])] = np.array([[M[so, si]]])
    return op


def site_block(i, T, w, L):
    """The single-orbital block of orbital i: every operator straight from its definition."""
    b = Block([i], {q: 1 for q in SITE_Q})
    cre = {2 * i + s: _CRE[s] for s in (0, 1)}
    ann = {p: m.T for p, m in cre.items()}
    for p in cre:
        b.ops[("C", p)] = _dense_to_blockop(cre[p])
    b.ops[("A", 2 * i, 2 * i + 1)] = _dense_to_blockop(cre[2 * i] @ cre[2 * i + 1])
    for p in cre:
        for q in cre:
            b.ops[("B", p, q)] = _dense_to_blockop(cre[p] @ ann[q])
    H = np.zeros((4, 4))
    for s in (0, 1):
        H += T[i, i] * cre[2 * i + s] @ ann[2 * i + s]
        for t in (0, 1):
            # 1/2 V_iiii a+_s a+_t a_t a_s ; only w_iiii = V_iiii enters
            H += 0.5 * w[i, i, i, i] * cre[2 * i + s] @ cre[2 * i + t] @ ann[2 * i + t] @ ann[2 * i + s]
    b.ops["H"] = _dense_to_blockop(H)
    for x in range(L):
        if x == i:
            continue
        for s in (0, 1):
            S = 0.5 * T[x, i] * ann[2 * i + s]
            for t in (0, 1):
                S = S + w[x, i, i, i] * cre[2 * i + t] @ ann[2 * i + t] @ ann[2 * i + s]
            b.ops[("S", 2 * x + s)] = _dense_to_blockop(S)
    return b


# ---------------------------------------------------------------------------------------------
# complementary operators from their definitions
# ---------------------------------------------------------------------------------------------

def comp_P_many(B: Block, w, pairs):
    """P^B_{pq} = sum_{kl in B} w_ijkl (a+_{ks} a+_{lt})^T for each (p=(i,s), q=(j,t)) in pairs."""
    names = [k for k in B.ops if k[0] == "A"]
    col = {k: n for n, k in enumerate(names)}
    if not names or not pairs:
        return [BlockOp() for _ in pairs]
    W = np.zeros((len(pairs), len(names)))
    for a, (p, q) in enumerate(pairs):
        i, s = divmod(p, 2)
        j, t = divmod(q, 2)
        for k in B.orbs:
            for l in B.orbs:
                r, u = 2 * k + s, 2 * l + t
                if r == u:
                    continue
                if r < u:
                    W[a, col[("A", r, u)]] += w[i, j, k, l]
                else:
                    W[a, col[("A", u, r)]] -= w[i, j, k, l]
    return lincomb(W, [B.ops[n] for n in names], transpose=True)


def comp_Q_many(B: Block, w, pairs):
    """Q^B_{pq'} for each (p=(i,s), q'=(k,s')) in pairs, from the definition in the header."""
    names = [k for k in B.ops if k[0] == "B"]
    col = {k: n for n, k in enumerate(names)}
    if not pairs:
        return []
    W = np.zeros((len(pairs), len(names)))
    for a, (p, q) in enumerate(pairs):
        i, s = divmod(p, 2)
        k, s2 = divmod(q, 2)
        for j in B.orbs:
            for l in B.orbs:
                if s == s2:
                    for t in (0, 1):
                        W[a, col[("B", 2 * j + t, 2 * l + t)]] += w[i, j, k, l]
                W[a, col[("B", 2 * j + s2, 2 * l + s)]] -= w[i, j, l, k]
    return lincomb(W, [B.ops[n] for n in names])


# ---------------------------------------------------------------------------------------------
# enlarging: operators of B1 u B2 on the product basis
# ---------------------------------------------------------------------------------------------

class Enlarged:
    def __init__(self, B1: Block, B2: Block, keep=None):
        self.B1, self.B2 = B1, B2
        self.orbs = B1.orbs + B2.orbs
        self.ops = {}
        self.I1 = identity(B1.sectors)
        self.I2 = identity(B2.sectors)
        self.keep = keep

    def spin_orbs(self):
        return [2 * i + s for i in self.orbs for s in (0, 1)]

    def identity(self) -> ProdOp:
        return _product(self.I1, self.I2, keep=self.keep)


def enlarge(B1: Block, B2: Block, T, w, ext_orbs, want_normal=True, want_H=True, keep=None) -> Enlarged:
    """Operators of B = B1 u B2 (B1 left of B2) as ProdOps; S_p for p over ext_orbs.

    keep: optional set of product sector keys; every Kronecker product below then forms only the
    sub-blocks that touch one of them (blockops.product).  The formulas are unchanged.
    """
    product = functools.partial(_product, keep=keep)
    E = Enlarged(B1, B2, keep)
    I1, I2 = E.I1, E.I2
    so1, so2 = B1.spin_orbs(), B2.spin_orbs()
    in1, in2 = set(so1), set(so2)
    # C_p
    for p in so1:
        E.ops[("C", p)] = product(B1.ops[("C", p)], I2)
    for p in so2:
        E.ops[("C", p)] = product(I1, B2.ops[("C", p)])
    if want_normal:
        allso = so1 + so2
        for a, p in enumerate(allso):
            for q in allso[a + 1:]:
                if q in in1:
                    E.ops[("A", p, q)] = product(B1.ops[("A", p, q)], I2)
                elif p in in2:
                    E.ops[("A", p, q)] = product(I1, B2.ops[("A", p, q)])
                else:  # p in B1, q in B2: a+_p a+_q in natural order
                    E.ops[("A", p, q)] = product(B1.ops[("C", p)], B2.ops[("C", q)])
        for p in allso:
            for q in allso:
                if p in in1 and q in in1:
                    E.ops[("B", p, q)] = product(B1.ops[("B", p, q)], I2)
                elif p in in2 and q in in2:
                    E.ops[("B", p, q)] = product(I1, B2.ops[("B", p, q)])
                elif p in in1:  # a+_p a_q, p in B1, q in B2
                    E.ops[("B", p, q)] = product(B1.ops[("C", p)], B2.ops[("C", q)].T())
                else:           # p in B2, q in B1: a+_p a_q = - a_q a+_p
                    E.ops[("B", p, q)] = product(B1.ops[("C", q)].T(), B2.ops[("C", p)], -1.0)
    # S_p for external p, by the recursion in the header
    ext_so = [2 * x + s for x in ext_orbs for s in (0, 1)]
    if ext_so:
        # P^{B2}_{p j}, j in B1 ; P^{B1}_{p j}, j in B2 ; Q likewise
        pj1 = [(p, j) for p in ext_so for j in so1]
        pj2 = [(p, j) for p in ext_so for j in so2]
        P2 = dict(zip(pj1, comp_P_many(B2, w, pj1)))
        P1 = dict(zip(pj2, comp_P_many(B1, w, pj2)))
        Q2 = dict(zip(pj1, comp_Q_many(B2, w, pj1)))
        Q1 = dict(zip(pj2, comp_Q_many(B1, w, pj2)))
        for p in ext_so:
            S = ProdOp()
            S.add_into(product(B1.ops[("S", p)], I2))
            S.add_into(product(I1, B2.ops[("S", p)]))
            for j in so1:
                if P2[(p, j)]:
                    S.add_into(product(B1.ops[("C", j)], P2[(p, j)]))          # a+_j P^{B2}_{pj}
                if Q2[(p, j)]:
                    S.add_into(product(B1.ops[("C", j)].T(), Q2[(p, j)]))      # Q^{B2}_{pj} a_j = a_j Q
            for j in so2:
                if P1[(p, j)]:
                    S.add_into(product(P1[(p, j)], B2.ops[("C", j)]))          # a+_j P^{B1}_{pj} = P a+_j
                if Q1[(p, j)]:
                    S.add_into(product(Q1[(p, j)], B2.ops[("C", j)].T()))      # Q^{B1}_{pj} a_j
            E.ops[("S", p)] = S
    if want_H:
        H = ProdOp()
        H.add_into(product(B1.ops["H"], I2))
        H.add_into(product(I1, B2.ops["H"]))
        for p in so1:   # a+_p S^{B2}_p + h.c.
            X = product(B1.ops[("C", p)], B2.ops[("S", p)])
            H.add_into(X); H.add_into(X.T())
        for p in so2:   # a+_p S^{B1}_p = - S^{B1}_p a+_p  (+ h.c.)
            X = product(B1.ops[("S", p)], B2.ops[("C", p)], -1.0)
            H.add_into(X); H.add_into(X.T())
        # two-index terms: normal operators on the smaller part X, complementary on the other
        if len(B2.orbs) <= len(B1.orbs):
            soX, BX, BY, x_is_2 = so2, B2, B1, True
        else:
            soX, BX, BY, x_is_2 = so1, B1, B2, False
        prs = [(p, q) for a, p in enumerate(soX) for q in soX[a + 1:]]
        for (p, q), Pc in zip(prs, comp_P_many(BY, w, prs)):
            if not Pc:
                continue
            X = product(Pc, BX.ops[("A", p, q)]) if x_is_2 else product(BX.ops[("A", p, q)], Pc)
            H.add_into(X); H.add_into(X.T())
        prs = [(p, q) for p in soX for q in soX]
        for (p, q), Qc in zip(prs, comp_Q_many(BY, w, prs)):
            if not Qc:
                continue
            X = product(Qc, BX.ops[("B", p, q)]) if x_is_2 else product(BX.ops[("B", p, q)], Qc)
            H.add_into(X)
        E.ops["H"] = H
    return E


def renormalize(E: Enlarged, iso, new_sectors) -> Block:
    """Project every operator of the enlarged block with the isometry (MPS site tensor)."""
    B = Block(E.orbs, new_sectors)
    for name, X in E.ops.items():
        B.ops[name] = project(X, iso)
    return B


# ---------------------------------------------------------------------------------------------
# the two-site problem
# ---------------------------------------------------------------------------------------------

def _vacuum_block(L):
    b = Block([], {(0, 0): 1})
    b.ops["H"] = BlockOp()
    for x in range(L):
        for s in (0, 1):
            b.ops[("S", 2 * x + s)] = BlockOp()
    return b


class TwoSiteOracle:
    """H_eff at the bond (k, k+1) (1-based sites) of an MPS given by plain dicts.

    sectors[b]: dict q -> dim for bond b = 0..L (q = electrons left of the bond);
    left[i] / right[i]: dict (q_in, s) -> (d_in, d_out) site tensors (1-based site i), left-
    canonical for i < k and right-canonical for i > k+1;
    psi_blocks: list of (qL, s1, s2, qR_bond, dL, dR) giving the flat psi layout.
    """

    def __init__(self, T, V, n_up, n_dn, k, sectors, left, right, psi_blocks):
        self.T = np.asarray(T, dtype=np.float64)
        self.w = w_from_V(np.asarray(V, dtype=np.float64))
        self.L = self.T.shape[0]
        self.N = (n_up, n_dn)
        self.k = k
        self.sectors, self.left, self.right = sectors, left, right
        self.psi_blocks = list(psi_blocks)
        self.Lblock = None
        self.Rblock = None
        self._terms = None

    # ---- environments: repeated enlarge + project ("renormalization steps") ----
    def left_iso(self, i):
        """Isometry of site i (1-based): product key (q_in, q(s)) -> (d_in, d_out)."""
        return {(qi, SITE_Q[s]): A for (qi, s), A in self.left[i].items()}

    def right_iso(self, i):
        """Right-canonical site i: product key (q(s), content_old) -> (d_old, d_new)."""
        iso = {}
        for (qi, s), Bm in self.right[i].items():
            qo = qadd(qi, SITE_Q[s])
            iso[(SITE_Q[s], qsub(self.N, qo))] = Bm.T
        return iso

    def build_left(self, upto):
        """Left block of sites 1..upto (orbitals 0..upto-1)."""
        blk = _vacuum_block(self.L)
        for i in range(1, upto + 1):
            site = site_block(i - 1, self.T, self.w, self.L)
            ext = list(range(i, self.L))
            E = enlarge(blk, site, self.T, self.w, ext)
            blk = renormalize(E, self.left_iso(i), self.sectors[i])
        return blk

    def build_right(self, downto):
        """Right block of sites downto..L (orbitals downto-1..L-1); sectors labelled by content."""
        blk = _vacuum_block(self.L)
        for i in range(self.L, downto - 1, -1):
            site = site_block(i - 1, self.T, self.w, self.L)
            ext = list(range(0, i - 1))
            E = enlarge(site, blk, self.T, self.w, ext)
            new_sec = {qsub(self.N, q): d for q, d in self.sectors[i - 1].items()}
            blk = renormalize(E, self.right_iso(i), new_sec)
        return blk

    def build_env(self):
        self.Lblock = self.build_left(self.k - 1)
        self.Rblock = self.build_right(self.k + 2)
        self._terms = None

    # ---- superblock terms: bipartition identity between L' = L u k and R' = k+1 u R ----
    def terms(self, keepL=None, keepR=None):
        """List of (X_L', X_R', hc) with H_eff = sum X_L' (x) X_R' (+ transpose if hc).

        keepL / keepR: optional sets of L' / R' product sector keys; the enlarged operators are then
        formed only on the sub-blocks that touch them (not cached).  None = everything (cached).
        """
        lean = keepL is not None or keepR is not None
        if self._terms is not None and not lean:
            return self._terms
        k, L = self.k, self.L
        s1 = site_block(k - 1, self.T, self.w, L)
        s2 = site_block(k, self.T, self.w, L)
        orbsL = list(range(0, k))        # orbitals of L'
        orbsR = list(range(k, L))        # orbitals of R'
        EL = enlarge(self.Lblock, s1, self.T, self.w, orbsR, keep=keepL)
        ER = enlarge(s2, self.Rblock, self.T, self.w, orbsL, keep=keepR)
        soL = EL.spin_orbs()
        soR = ER.spin_orbs()
        IL, IR = EL.identity(), ER.identity()
        terms = [(EL.ops["H"], IR, False), (IL, ER.ops["H"], False)]
        for p in soL:   # a+_p S^{R'}_p + h.c.
            terms.append((EL.ops[("C", p)], ER.ops[("S", p)], True))
        for p in soR:   # a+_p S^{L'}_p = - S^{L'}_p a+_p, + h.c.
            Sm = ProdOp({kk: -m for kk, m in EL.ops[("S", p)].items()})
            terms.append((Sm, ER.ops[("C", p)], True))
        # normal two-index operators on L', complementary ones on R' formed from R' normal ops
        ERb = Block(ER.orbs, {})
        ERb.ops = {n: o for n, o in ER.ops.items() if n[0] in ("A", "B")}
        prs = [(p, q) for a, p in enumerate(soL) for q in soL[a + 1:]]
        for (p, q), Pc in zip(prs, comp_P_many(ERb, self.w, prs)):
            if Pc:
                terms.append((EL.ops[("A", p, q)], Pc, True))
        prs = [(p, q) for p in soL for q in soL]
        for (p, q), Qc in zip(prs, comp_Q_many(ERb, self.w, prs)):
            if Qc:
                terms.append((EL.ops[("B", p, q)], Qc, False))
        if not lean:
            self._terms = terms
        return terms

    # ---- psi layout ----
    def unflatten(self, v):
        psi, off = {}, 0
        for (qL, s1, s2, qRb, dL, dR) in self.psi_blocks:
            key = ((qL, SITE_Q[s1]), (SITE_Q[s2], qsub(self.N, qRb)))
            psi[key] = np.asarray(v[off:off + dL * dR]).reshape(dL, dR)
            off += dL * dR
        assert off == len(v)
        return psi

    def flatten(self, psi):
        parts = []
        for (qL, s1, s2, qRb, dL, dR) in self.psi_blocks:
            key = ((qL, SITE_Q[s1]), (SITE_Q[s2], qsub(self.N, qRb)))
            parts.append(np.asarray(psi[key]).reshape(-1))
        return np.concatenate(parts)

    def psi_size(self):
        return sum(b[4] * b[5] for b in self.psi_blocks)

    # ---- H_eff psi  (Eq. (7)/(8)) ----
    def apply(self, v):
        psi = self.unflatten(np.asarray(v, dtype=np.float64))
        out = {kk: np.zeros_like(m) for kk, m in psi.items()}
        self._accumulate(self.terms(), psi, out)
        return self.flatten(out)

    def _accumulate(self, terms, psi, out):
        """out{key} += sum_terms (X_L' (x) X_R' psi){key} for the keys present in `out`."""
        by_left = {}
        for (kl, kr), m in psi.items():
            by_left.setdefault(kl, []).append((kr, m))
        for XL, XR, hc in terms:
            pR = XR.parity()
            r_by_in, r_by_out = {}, {}
            for (kro, kri), mR in XR.items():
                r_by_in.setdefault(kri, []).append((kro, mR))
                if hc:
                    r_by_out.setdefault(kro, []).append((kri, mR))
            for (klo, kli), mL in XL.items():
                sg = -1.0 if (pR and ((qnum(kli[0]) + qnum(kli[1])) & 1)) else 1.0
                for kri, x in by_left.get(kli, ()):      # forward: M psi
                    for kro, mR in r_by_in.get(kri, ()):
                        o = out.get((klo, kro))
                        if o is not None:
                            o += sg * (mL @ x @ mR.T)
                if hc:                                   # M^T psi (same sign, blocks transposed)
                    for kro, x in by_left.get(klo, ()):
                        for kri, mR in r_by_out.get(kro, ()):
                            o = out.get((kli, kri))
                            if o is not None:
                                o += sg * (mL.T @ x @ mR)

    def diag(self):
        """Diagonal of H_eff in the psi layout (Davidson preconditioner, DESIGN.md App. E)."""
        out = {}
        for (qL, s1, s2, qRb, dL, dR) in self.psi_blocks:
            out[((qL, SITE_Q[s1]), (SITE_Q[s2], qsub(self.N, qRb)))] = np.zeros((dL, dR))
        for XL, XR, hc in self.terms():
            pR = XR.parity()
            mult = 2.0 if hc else 1.0
            for (klo, kli), mL in XL.items():
                if klo != kli:
                    continue
                sg = -1.0 if (pR and ((qnum(kli[0]) + qnum(kli[1])) & 1)) else 1.0
                for (kro, kri), mR in XR.items():
                    if kro != kri:
                        continue
                    o = out.get((klo, kro))
                    if o is not None:
                        o += (mult * sg) * np.outer(np.diag(mL), np.diag(mR))
        return self.flatten(out)


# ---------------------------------------------------------------------------------------------
# Davidson (paper names no eigensolver, "iterative eigensolver"; DESIGN.md App. E)
# ---------------------------------------------------------------------------------------------

def davidson(apply, diag, v0, tol=1e-10, max_iter=200, max_basis=20):
    """Davidson-Liu for the lowest eigenpair of a real symmetric operator.

    v1 = v0/|v0|; loop: G = V^T W, lowest Ritz pair (theta, y); x = V y; r = W y - theta x;
    stop if |r| <= tol; t = r / (theta - diag) with |theta - diag| >= 1e-12 (sign kept);
    orthogonalise t against V twice (classical Gram-Schmidt), normalise, append; restart to
    [x] when the basis reaches max_basis.  Returns (theta, x, iterations, |r|) with
    iterations = number of operator applications.

    Pinned: the converged energy equals the brute-force FCI ground-state energy at untruncated
    bond dimension (tests/test_oracle_dmrg.py).  Parity unpinned: the iterate-by-iterate
    trajectory (energy / residual after a fixed number of iterations) has no value outside this
    file to compare with; the paper names no eigensolver (R13).
    """
    v = np.asarray(v0, dtype=np.float64)
    v = v / np.linalg.norm(v)
    Vb = [v]
    Wb = [apply(v)]
    napply = 1
    theta, x, rn = 0.0, v, np.inf
    while True:
        m = len(Vb)
        Vm = np.array(Vb)
        Wm = np.array(Wb)
        G = Vm @ Wm.T
        G = 0.5 * (G + G.T)
        ev, Y = np.linalg.eigh(G)
        theta, y = ev[0], Y[:, 0]
        x = y @ Vm
        hx = y @ Wm
        r = hx - theta * x
        rn = float(np.linalg.norm(r))
        if rn <= tol or napply >= max_iter:
            break
        den = theta - diag
        den = np.where(np.abs(den) < 1e-12, np.where(den < 0, -1e-12, 1e-12), den)
        t = r / den
        if m >= max_basis:
            nx = np.linalg.norm(x)
            Vb = [x / nx]
            Wb = [hx / nx]
        for _ in range(2):
            for u in Vb:
                t = t - (u @ t) * u
        nt = np.linalg.norm(t)
        if nt < 1e-14:
            break
        t = t / nt
        Vb.append(t)
        Wb.append(apply(t))
        napply += 1
    return float(theta), x / np.linalg.norm(x), napply, rn

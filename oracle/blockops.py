"""ORACLE (test infrastructure, CPU only): block-sparse operator algebra for the DMRG oracle.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this package; it shares no code with the CUDA path.

Block-sparse storage as in PAPER.md:107: states carry the labels q = (n_up, n_dn); an operator
O is stored as its non-zero blocks O{(q_out, q_in)}.  Two containers:

  BlockOp : dict (q_out, q_in) -> matrix, on one block of orbitals.
  ProdOp  : dict ((q1_out, q2_out), (q1_in, q2_in)) -> matrix on the product basis
            |b1>|b2> of two neighbouring blocks B1 (left) and B2 (right); the product state
            index inside a sub-block is i1 * d2 + i2 (plain Kronecker order).

Fermion sign: for global operators X1 on B1 and X2
on B2 written in the order X1 X2,
    <b1' b2'| X1 X2 |b1 b2> = (-1)^{N(b1) * parity(X2)} <b1'|X1|b1> <b2'|X2|b2>,
because X2 has to pass the creation string of the input state |b1>.
"""
from __future__ import annotations

import numpy as np


def qadd(a, b):
    return (a[0] + b[0], a[1] + b[1])


def qsub(a, b):
    return (a[0] - b[0], a[1] - b[1])


def qnum(q):
    return q[0] + q[1]


class BlockOp(dict):
    """dict (q_out, q_in) -> ndarray.  All blocks share dq = q_out - q_in."""

    def parity(self) -> int:
        for (qo, qi) in self:
            return (qnum(qo) - qnum(qi)) & 1
        return 0

    def T(self) -> "BlockOp":
        return BlockOp({(qi, qo): m.T for (qo, qi), m in self.items()})

    def scaled(self, c: float) -> "BlockOp":
        return BlockOp({k: c * m for k, m in self.items()})

    def add_into(self, other: "BlockOp", c: float = 1.0) -> None:
        for k, m in other.items():
            if k in self:
                self[k] = self[k] + c * m
            else:
                self[k] = c * m


class ProdOp(dict):
    """dict ((q1o, q2o), (q1i, q2i)) -> ndarray on the product basis of two blocks."""

    def T(self) -> "ProdOp":
        return ProdOp({(ki, ko): m.T for (ko, ki), m in self.items()})

    def add_into(self, other: "ProdOp", c: float = 1.0) -> None:
        for k, m in other.items():
            if k in self:
                self[k] = self[k] + c * m
            else:
                self[k] = c * m

    def parity(self) -> int:
        for (ko, ki) in self:
            return (qnum(ko[0]) + qnum(ko[1]) - qnum(ki[0]) - qnum(ki[1])) & 1
        return 0


def identity(sectors) -> BlockOp:
    return BlockOp({(q, q): np.eye(d) for q, d in sectors.items()})


def product(X1: BlockOp, X2: BlockOp, coef: float = 1.0, keep=None) -> ProdOp:
    """Matrix of coef * X1 X2 (X1 on B1 written first, X2 on B2) on the product basis.

    keep: optional set of product sector keys (q1, q2).  Only the sub-blocks whose out key or in
    key is in the set are formed (the others are simply absent, as for a restricted operator);
    None = all of them.  Used by oracle/lean.py to evaluate H_eff psi on chosen output blocks.
    """
    p2 = X2.parity()
    out = ProdOp()
    for (q1o, q1i), m1 in X1.items():
        sg = -1.0 if (p2 and (qnum(q1i) & 1)) else 1.0
        for (q2o, q2i), m2 in X2.items():
            if keep is not None and (q1o, q2o) not in keep and (q1i, q2i) not in keep:
                continue
            out[((q1o, q2o), (q1i, q2i))] = (coef * sg) * np.kron(m1, m2)
    return out


def project(X: ProdOp, iso) -> BlockOp:
    """O_new{(qo, qi)} = sum iso[(q1o,q2o)]^T  X[(q1o,q2o),(q1i,q2i)]  iso[(q1i,q2i)].

    iso: dict (q1, q2) -> matrix (d1*d2, d_new(q1+q2)) — the renormalisation isometry, i.e. the
    MPS site tensor ("renormalization steps").
    """
    out = BlockOp()
    for (ko, ki), m in X.items():
        if ko not in iso or ki not in iso:
            continue
        v = iso[ko].T @ m @ iso[ki]
        key = (qadd(*ko), qadd(*ki))
        if key in out:
            out[key] = out[key] + v
        else:
            out[key] = v
    return out


def lincomb(W: np.ndarray, ops, transpose: bool = False):
    """Stacked linear combination: out[a] = sum_b W[a, b] * ops[b]  (ops share dq).

    Works for BlockOp or ProdOp lists; with transpose=True every ops[b] is transposed first.
    Returns a list of the same container type, one per row of W.
    """
    cls = type(ops[0]) if ops else BlockOp
    if transpose:
        ops = [o.T() for o in ops]
    keys = {}
    for b, o in enumerate(ops):
        for k, m in o.items():
            keys.setdefault(k, m.shape)
    outs = [cls() for _ in range(W.shape[0])]
    for k, shp in keys.items():
        stack = np.zeros((len(ops), shp[0] * shp[1]))
        present = np.zeros(len(ops), dtype=bool)
        for b, o in enumerate(ops):
            m = o.get(k)
            if m is not None:
                stack[b] = np.asarray(m).reshape(-1)
                present[b] = True
        Wk = W[:, present]
        rows_used = np.abs(Wk).sum(axis=1) > 0
        if not rows_used.any():
            continue
        res = Wk @ stack[present]
        for a in np.nonzero(rows_used)[0]:
            outs[a][k] = res[a].reshape(shp)
    return outs

"""Test helpers: explicit Fock-space embedding of the MPS block bases (tiny systems only).

Builds the isometry P of SURVEY.md 8(c): |a s_k s_{k+1} b>  ->  determinant space, straight
from the MPS site tensors (Eq. (4)), so that H_eff can be checked against its
definition P^T H_FCI P.  Uses only numpy and the determinant convention of oracle/fci.py.
"""
import numpy as np

from oracle import fci

SITE_Q = ((0, 0), (0, 1), (1, 0), (1, 1))


def left_vectors(mps, upto):
    """dict q -> (4^upto, d_q): left block states of sites 1..upto in the site-product basis."""
    vec = {(0, 0): np.ones((1, 1))}
    for i in range(1, upto + 1):
        new = {}
        n_old = 4 ** (i - 1)
        for (qi, s), A in mps.left[i].items():
            qo = (qi[0] + SITE_Q[s][0], qi[1] + SITE_Q[s][1])
            tgt = new.setdefault(qo, np.zeros((n_old * 4, A.shape[1])))
            tgt[s::4, :] += vec[qi] @ A          # index = idx_old*4 + s
        vec = new
    return vec


def right_vectors(mps, downto):
    """dict q_bond -> (4^(L-downto+1), d_q): right block states of sites downto..L."""
    L = mps.L
    vec = {(mps.n_up, mps.n_dn): np.ones((1, 1))}
    for i in range(L, downto - 1, -1):
        new = {}
        n_old = 4 ** (L - i)
        for (qi, s), B in mps.right[i].items():
            qo = (qi[0] + SITE_Q[s][0], qi[1] + SITE_Q[s][1])
            tgt = new.setdefault(qi, np.zeros((4 * n_old, B.shape[0])))
            tgt[s * n_old:(s + 1) * n_old, :] += vec[qo] @ B.T   # index = s*n_old + idx_old
        vec = new
    return vec


def embedding(mps, psi_blocks):
    """Dense P (n_det x n_psi) and the determinant list."""
    L, k = mps.L, mps.k
    dets = fci.determinants(L, mps.n_up, mps.n_dn)
    nfull = 4 ** L
    # site-product index (s_1 most significant) -> determinant position
    pos = -np.ones(nfull, dtype=np.int64)
    idx = np.arange(nfull)
    bits = np.zeros(nfull, dtype=np.uint64)
    for site in range(L):
        s = (idx // (4 ** (L - 1 - site))) % 4
        up = ((s == 2) | (s == 3)).astype(np.uint64)
        dn = ((s == 1) | (s == 3)).astype(np.uint64)
        bits |= up << np.uint64(2 * site)
        bits |= dn << np.uint64(2 * site + 1)
    where = np.searchsorted(dets, bits)
    where[where >= len(dets)] = 0
    ok = dets[where] == bits
    pos[ok] = where[ok]
    lv = left_vectors(mps, k - 1)
    rv = right_vectors(mps, k + 2)
    nR = 4 ** (L - k - 1)
    npsi = sum(b[4] * b[5] for b in psi_blocks)
    P = np.zeros((len(dets), npsi))
    off = 0
    for (qL, s1, s2, qRb, dL, dR) in psi_blocks:
        Lm, Rm = lv[qL], rv[qRb]
        il = np.arange(Lm.shape[0])[:, None]
        ir = np.arange(Rm.shape[0])[None, :]
        full = ((il * 4 + s1) * 4 + s2) * nR + ir           # (nl, nr)
        rows = pos[full].reshape(-1)
        blockP = np.einsum("ia,jb->ijab", Lm, Rm).reshape(-1, dL * dR)
        bad = rows < 0                      # site-product states outside the N-electron space
        assert np.abs(blockP[bad]).max(initial=0.0) == 0.0
        P[rows[~bad], off:off + dL * dR] += blockP[~bad]
        off += dL * dR
    return P, dets


def assert_blocks_close(got, ref, sizes, rel=1e-11):
    """Whole-vector rel-L2 <= rel (the north_star tolerance) AND, block by block, max |got - ref| small against the
    block's own scale: an error confined to one small psi block does not show in the whole-vector norm."""
    got, ref = np.asarray(got), np.asarray(ref)
    assert np.linalg.norm(got - ref) / np.linalg.norm(ref) <= rel
    floor = 1e-3 * np.abs(ref).max()
    o = 0
    for n in sizes:
        g, r = got[o:o + n], ref[o:o + n]
        assert np.abs(g - r).max() <= 10 * rel * (np.abs(r).max() + floor), (o, n)
        o += n
    assert o == len(ref)

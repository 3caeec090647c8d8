"""Pins of the SU(2) oracle (oracle/su2.py) against what the mathematics and the paper fix (no GPU)."""
import numpy as np
import pytest
from sympy import Rational
from sympy.physics.quantum.cg import CG
from sympy.physics.wigner import wigner_6j, wigner_9j

from oracle import dmrg as odmrg
from oracle import fci, su2
from paper_2501_18263_b200 import inputs

import helpers


def _h(x):
    return Rational(x, 2)


def test_cg_against_sympy_and_closed_forms():
    rng = np.random.default_rng(0)
    n = 0
    while n < 150:
        j1, j2 = int(rng.integers(0, 7)), int(rng.integers(0, 5))
        J = int(rng.choice(np.arange(abs(j1 - j2), j1 + j2 + 1, 2)))
        m1 = int(rng.choice(np.arange(-j1, j1 + 1, 2)))
        m2 = int(rng.choice(np.arange(-j2, j2 + 1, 2)))
        if abs(m1 + m2) > J:
            continue
        ref = float(CG(_h(j1), _h(m1), _h(j2), _h(m2), _h(J), _h(m1 + m2)).doit())
        assert abs(su2.cg(j1, m1, j2, m2, J, m1 + m2) - ref) < 1e-13
        n += 1
    # textbook values: two spin-1/2 -> singlet / triplet; stretched state; orthogonality
    assert abs(su2.cg(1, 1, 1, -1, 0, 0) - 1 / np.sqrt(2)) < 1e-15
    assert abs(su2.cg(1, -1, 1, 1, 0, 0) + 1 / np.sqrt(2)) < 1e-15
    assert abs(su2.cg(1, 1, 1, -1, 2, 0) - 1 / np.sqrt(2)) < 1e-15
    assert su2.cg(3, 3, 2, 2, 5, 5) == pytest.approx(1.0, abs=1e-15)
    for J in (1, 3):
        for J2 in (1, 3):
            s = sum(su2.cg(2, m1, 1, 1 - m1, J, 1) * su2.cg(2, m1, 1, 1 - m1, J2, 1) for m1 in (-2, 0, 2))
            assert abs(s - (1.0 if J == J2 else 0.0)) < 1e-14
    assert su2.cg(2, 0, 2, 0, 2, 0) == 0.0      # <1 0; 1 0 | 1 0> vanishes


def test_6j_9j_against_sympy_and_zero_argument_reduction():
    for args in [(1, 1, 2, 1, 1, 2), (2, 2, 2, 2, 2, 2), (3, 2, 1, 1, 2, 3), (4, 3, 1, 2, 1, 3)]:
        assert abs(su2.sixj(*args) - float(wigner_6j(*[_h(a) for a in args]))) < 1e-13
    for args in [(1, 1, 2, 1, 1, 2, 2, 2, 2), (2, 1, 3, 1, 1, 2, 3, 0, 3), (4, 1, 3, 2, 1, 1, 2, 0, 2),
                 (3, 1, 2, 2, 0, 2, 1, 1, 2)]:
        assert abs(su2.ninej(*args) - float(wigner_9j(*[_h(a) for a in args], prec=64))) < 1e-12
    # {a b c; d e c; g g 0} = (-1)^{b+c+d+g} / sqrt((2c+1)(2g+1)) {a b c; e d g}
    for (a, b, c, d, e, g) in [(2, 1, 3, 1, 2, 1), (3, 2, 1, 2, 3, 1), (2, 2, 2, 2, 2, 2)]:
        lhs = su2.ninej(a, b, c, d, e, c, g, g, 0)
        rhs = (-1) ** ((b + c + d + g) // 2) / np.sqrt((c + 1) * (g + 1)) * su2.sixj(a, b, c, e, d, g)
        assert abs(lhs - rhs) < 1e-13


def test_F_ninej_equals_six_cg_contraction():
    """PAPER.md Eq. (11) vs Fig. 4 (:136-150): the two definitions of F agree on every allowed combination
    of the spins that occur in the two-site problem (operator ranks 0, 1/2, 1; site spins 0, 1/2)."""
    cnt = 0
    for Sa in range(0, 5):
        for Sk in (0, 1):
            for Sg in range(abs(Sa - Sk), Sa + Sk + 1, 2):
                for kL in (0, 1, 2):
                    for kk in (0, 1, 2):
                        for kop in range(abs(kL - kk), kL + kk + 1, 2):
                            for Sa_ in range(abs(Sa - kL), Sa + kL + 1, 2):
                                for Sk_ in (0, 1):
                                    if Sk_ < abs(Sk - kk) or Sk_ > Sk + kk or (Sk + kk + Sk_) % 2:
                                        continue
                                    for Sg_ in range(abs(Sa_ - Sk_), Sa_ + Sk_ + 1, 2):
                                        if Sg_ < abs(Sg - kop) or Sg_ > Sg + kop:
                                            continue
                                        a = su2.F_ninej(Sa, Sk, Sg, kL, kk, kop, Sa_, Sk_, Sg_)
                                        b = su2.F_sixcg(Sa, Sk, Sg, kL, kk, kop, Sa_, Sk_, Sg_)
                                        assert abs(a - b) < 1e-12
                                        cnt += 1
    assert cnt > 300
    # both factors scalar: F = 1 when the spins match
    assert su2.F_ninej(3, 1, 2, 0, 0, 0, 3, 1, 2) == pytest.approx(1.0, abs=1e-14)


def _spin_sq(nsites):
    """S^2 on the product basis of nsites sites (site states 0, dn, up, updn; index s_1 most significant)."""
    sp = np.zeros((4, 4)); sp[2, 1] = 1.0
    sz = np.diag([0.0, -0.5, 0.5, 0.0])
    def emb(m, i):
        out = np.eye(1)
        for j in range(nsites):
            out = np.kron(out, m if j == i else np.eye(4))
        return out
    Sp = sum(emb(sp, i) for i in range(nsites))
    Sz = sum(emb(sz, i) for i in range(nsites))
    return Sp.T @ Sp + Sz + Sz @ Sz


class _U1View:
    def __init__(self, mps, sec, left, right):
        self.L, self.k, self.n_up, self.n_dn = mps.L, mps.k, mps.N // 2, mps.N // 2
        self.sectors, self.left, self.right = sec, left, right


def test_expanded_block_states_are_spin_eigenstates():
    L, N, k = 6, 6, 4
    mps = inputs.make_mps_su2(L, N, 14, k, seed=4)
    sec, left, right, lay = su2.expand_mps(mps)
    view = _U1View(mps, sec, left, right)
    lv = helpers.left_vectors(view, k - 1)
    S2op = _spin_sq(k - 1)
    for q, vecs in lv.items():
        assert np.abs(vecs.T @ vecs - np.eye(vecs.shape[1])).max() < 1e-12      # orthonormal
        dim, layout = lay[k - 1][q]
        for (Nq, S2), off in layout:
            d = mps.sectors[k - 1][(Nq, S2)]
            v = vecs[:, off:off + d]
            assert np.abs(S2op @ v - (S2 / 2) * (S2 / 2 + 1) * v).max() < 1e-12
    rv = helpers.right_vectors(view, k + 2)
    S2r = _spin_sq(L - k - 1)
    for q, vecs in rv.items():
        dim, layout = lay[k + 1][q]
        for (Nq, S2), off in layout:
            d = mps.sectors[k + 1][(Nq, S2)]
            v = vecs[:, off:off + d]
            assert np.abs(S2r @ v - (S2 / 2) * (S2 / 2 + 1) * v).max() < 1e-12


@pytest.mark.parametrize("L,N,k,D", [(6, 6, 3, 10 ** 9), (6, 4, 2, 9), (7, 6, 4, 12)])
def test_reduced_space_is_invariant_and_isometric(L, N, k, D):
    T, V = inputs.make_integrals(L, 20 + L)
    mps = inputs.make_mps_su2(L, N, D, k, seed=3)
    orc = su2.SU2TwoSiteOracle(T, V, mps, inputs.psi_blocks_su2(mps))
    orc.build_env()
    R = orc.R
    assert abs(R.T @ R - np.eye(orc.n_red)).max() < 1e-13
    rng = np.random.default_rng(0)
    v = rng.normal(size=orc.n_red)
    w = orc.u1.apply(orc.expand(v))
    # H is a spin scalar: H_eff maps the image of the S = 0 space into itself
    assert np.linalg.norm(w - orc.expand(orc.reduce(w))) <= 1e-12 * np.linalg.norm(w)
    # symmetric
    u = rng.normal(size=orc.n_red)
    assert abs(u @ orc.apply(v) - v @ orc.apply(u)) < 1e-10


def test_singlet_energy_equals_fci_at_untruncated_bond():
    L, N, k = 6, 6, 3
    T, V = inputs.make_integrals(L, 5)
    mps = inputs.make_mps_su2(L, N, 10 ** 9, k, seed=3)
    orc = su2.SU2TwoSiteOracle(T, V, mps, inputs.psi_blocks_su2(mps))
    orc.build_env()
    assert orc.n_red == 175                       # singlet CSFs of 6 electrons in 6 orbitals
    v0 = inputs.make_psi0_su2(mps, 1)
    E, x, it, rn = odmrg.davidson(orc.apply, orc.diag(), v0, tol=1e-9, max_iter=400)
    # with these integrals the FCI ground state in the S_z = 0 sector is a singlet, so the S = 0 reduced
    # space at untruncated bond dimension must reproduce it
    ev = fci.fci_lowest(T, V, N // 2, N // 2, 4)
    assert abs(E - ev[0]) < 1e-8
    # the exact diagonal (one apply per basis vector) is what the library has to reproduce
    d = orc.diag_exact()
    assert abs(d.sum() - np.trace(orc.R.T @ (orc.R.T @ _dense_u1(orc)).T)) < 1e-8


def _dense_u1(orc):
    n = orc.n_u1
    H = np.zeros((n, n))
    e = np.zeros(n)
    for j in range(n):
        e[j] = 1.0
        H[:, j] = orc.u1.apply(e)
        e[j] = 0.0
    return H

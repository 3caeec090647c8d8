"""Pins for oracle/dmrg.py (no GPU): H_eff against its definition P^T H_FCI P, block operators
against Jordan-Wigner definitions, Davidson against FCI, and the paper's printed energy."""
import numpy as np
import pytest

import helpers
from oracle import dmrg, fci
from paper_2501_18263_b200 import inputs
from test_oracle_fci import _torus_integrals


def _oracle(T, V, mps):
    pb = inputs.psi_blocks(mps)
    orc = dmrg.TwoSiteOracle(T, V, mps.n_up, mps.n_dn, mps.k, mps.sectors, mps.left, mps.right, pb)
    orc.build_env()
    return orc, pb


def _herm_V(rng, L):
    V = rng.normal(size=(L,) * 4)
    return V + V.transpose(2, 3, 0, 1)        # only the Hermiticity relation V_ijkl = V_klij


@pytest.mark.parametrize("L,nu,nd,k,D", [(5, 2, 1, 2, 6), (5, 3, 2, 3, 10 ** 9), (6, 2, 3, 4, 8),
                                           (6, 3, 3, 1, 7), (6, 3, 3, 5, 7), (6, 3, 3, 3, 12)])
def test_heff_equals_projected_fci(L, nu, nd, k, D):
    """Definition: H_eff psi == P^T H_FCI P psi, truncated and untruncated, with
    a V that has no symmetry beyond Hermiticity (so a dropped or transposed index shows)."""
    rng = np.random.default_rng(10 * L + k)
    T = rng.normal(size=(L, L)); T = T + T.T
    V = _herm_V(rng, L)
    mps = inputs.make_mps(L, nu, nd, D, k, seed=5)
    orc, pb = _oracle(T, V, mps)
    P, _ = helpers.embedding(mps, pb)
    assert np.abs(P.T @ P - np.eye(P.shape[1])).max() < 1e-13
    H, _ = fci.fci_hamiltonian(T, V, nu, nd)
    Heff = P.T @ H @ P
    v = rng.normal(size=P.shape[1])
    ref = Heff @ v
    got = orc.apply(v)
    assert np.linalg.norm(got - ref) / np.linalg.norm(ref) < 1e-13
    assert np.abs(orc.diag() - np.diag(Heff)).max() < 1e-12


def _jw_site_ops(n):
    """a+_{(i,s)} on n sites in the site-product basis (site 0 most significant), JW from site 0."""
    Pm = np.diag([1.0, -1.0, -1.0, 1.0])
    cre = {}
    for i in range(n):
        for s in (0, 1):
            m = np.ones((1, 1))
            for j in range(n):
                m = np.kron(m, Pm if j < i else (dmrg._CRE[s] if j == i else np.eye(4)))
            cre[(i, s)] = m
    return cre


def test_left_block_operators_match_definitions():
    """C, A, B, S, H of a renormalised left block == V^T O_JW V with O_JW from the definitions."""
    rng = np.random.default_rng(7)
    L, nu, nd, k, n = 6, 3, 2, 4, 3
    T = rng.normal(size=(L, L)); T = T + T.T
    V = _herm_V(rng, L)
    w = dmrg.w_from_V(V)
    mps = inputs.make_mps(L, nu, nd, 9, k, seed=3)
    orc, _ = _oracle(T, V, mps)
    blk = orc.Lblock
    vec = helpers.left_vectors(mps, n)
    cre = _jw_site_ops(n)
    ann = {k_: m.T for k_, m in cre.items()}

    def check(op, dense):
        for qo in vec:
            for qi in vec:
                ref = vec[qo].T @ dense @ vec[qi]
                got = op.get((qo, qi))
                if got is None:
                    assert np.abs(ref).max() < 1e-12
                else:
                    assert np.abs(got - ref).max() < 1e-12

    for i in range(n):
        for s in (0, 1):
            check(blk.ops[("C", 2 * i + s)], cre[(i, s)])
    check(blk.ops[("A", 1, 4)], cre[(0, 1)] @ cre[(2, 0)])
    check(blk.ops[("B", 5, 2)], cre[(2, 1)] @ ann[(1, 0)])
    Hd = np.zeros((4 ** n, 4 ** n))
    for i in range(n):
        for j in range(n):
            for s in (0, 1):
                Hd += T[i, j] * cre[(i, s)] @ ann[(j, s)]
                for k_ in range(n):
                    for l in range(n):
                        for t in (0, 1):
                            Hd += 0.5 * V[i, j, k_, l] * cre[(i, s)] @ cre[(j, t)] @ ann[(l, t)] @ ann[(k_, s)]
    check(blk.ops["H"], Hd)
    for x in (3, 5):
        for s in (0, 1):
            Sd = np.zeros_like(Hd)
            for j in range(n):
                Sd += 0.5 * T[x, j] * ann[(j, s)]
                for k_ in range(n):
                    for l in range(n):
                        for t in (0, 1):
                            Sd += w[x, j, k_, l] * cre[(j, t)] @ ann[(l, t)] @ ann[(k_, s)]
            check(blk.ops[("S", 2 * x + s)], Sd)


def test_hermitian_and_number_conserving():
    T, V, mps = inputs.make_config(0)
    mps = inputs.make_mps(8, 4, 4, 24, 4, seed=11)
    orc, pb = _oracle(T, V, mps)
    rng = np.random.default_rng(0)
    x, y = rng.normal(size=(2, orc.psi_size()))
    assert abs(x @ orc.apply(y) - y @ orc.apply(x)) < 1e-11
    # T = eps, V_ijkl = U d_ik d_jl: H = eps N + U N (N-1)/2 on every state of the target sector
    L = 8
    Tn = 0.3 * np.eye(L)
    Vn = np.zeros((L,) * 4)
    for i in range(L):
        for j in range(L):
            Vn[i, j, i, j] = 0.9
    orc2, _ = _oracle(Tn, Vn, mps)
    assert np.abs(orc2.apply(x) - (0.3 * 8 + 0.9 * 8 * 7 / 2) * x).max() < 1e-11


def test_davidson_reaches_fci_config0():
    """BASELINE.json configs[0]: untruncated L=8 (4,4): lowest H_eff eigenvalue == FCI within 1e-10."""
    T, V, mps = inputs.make_config(0)
    orc, pb = _oracle(T, V, mps)
    assert orc.psi_size() == 4900
    v0 = inputs.make_psi0(mps, inputs.CONFIGS[0]["seed"])
    E, x, it, rn = dmrg.davidson(orc.apply, orc.diag(), v0, tol=1e-10, max_iter=300)
    assert rn <= 1e-10
    assert abs(E - fci.fci_lowest(T, V, 4, 4, 1)[0]) < 1e-10


def test_p0_through_the_dmrg_pipeline():
    """the symmetric k=8 partitioning with untruncated blocks recovers the exact
    E_GS = -7.2295... of the 4x4 spinless torus (embedded with N_dn = 0)."""
    T, V = _torus_integrals()
    mps = inputs.make_mps(16, 8, 0, 10 ** 9, 8, seed=1)
    orc, pb = _oracle(T, V, mps)
    assert orc.psi_size() == 12870
    v0 = inputs.make_psi0(mps, 2)
    E, x, it, rn = dmrg.davidson(orc.apply, orc.diag(), v0, tol=1e-7, max_iter=300)
    assert abs(E - (-7.2295)) < 1e-4

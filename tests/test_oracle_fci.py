"""Pins for oracle/fci.py (no GPU).  Each test names what fixes the expected value."""
import os

import numpy as np

from oracle import fci

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _torus_integrals():
    """PAPER.md Eq. (12) on the 4x4 torus embedded as L=16 orbitals with N_dn = 0 (R2)."""
    L = 16
    T = np.zeros((L, L))
    V = np.zeros((L, L, L, L))
    bonds = set()
    for x in range(4):
        for y in range(4):
            for dx, dy in ((1, 0), (0, 1)):
                a, b = x * 4 + y, ((x + dx) % 4) * 4 + (y + dy) % 4
                bonds.add((min(a, b), max(a, b)))
    assert len(bonds) == 32
    for a, b in bonds:
        T[a, b] = T[b, a] = -1.0
        V[a, b, a, b] = 1.0
        V[b, a, b, a] = 1.0
    return T, V


def test_p0_printed_energies():
    """PAPER.md:202 prints E_GS = -7.2295..., E_1 = -7.2242... (tests/golden/p0_spinless_torus.txt)."""
    gold = {}
    for line in open(os.path.join(GOLD, "p0_spinless_torus.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()
        gold[k] = float(v)
    T, V = _torus_integrals()
    e = fci.fci_lowest(T, V, 8, 0, 2)
    for got, key in zip(e, ("E_GS", "E_1")):
        assert abs(got - gold[key]) < 1e-4, (key, got)


def test_hubbard_dimer_closed_form():
    """Textbook: two-site Hubbard model at half filling, E0 = U/2 - sqrt(U^2/4 + 4 t^2)."""
    for t, U in ((1.0, 4.0), (0.7, 0.3), (1.3, 10.0)):
        T = np.array([[0.0, -t], [-t, 0.0]])
        V = np.zeros((2, 2, 2, 2))
        V[0, 0, 0, 0] = V[1, 1, 1, 1] = U
        e = fci.fci_lowest(T, V, 1, 1, 1)[0]
        assert abs(e - (U / 2 - np.sqrt(U * U / 4 + 4 * t * t))) < 1e-13


def test_one_body_only_is_orbital_filling():
    """V = 0: E0 = sum of the lowest n_up + lowest n_dn eigenvalues of T (free fermions)."""
    rng = np.random.default_rng(0)
    L = 6
    T = rng.normal(size=(L, L)); T = T + T.T
    V = np.zeros((L,) * 4)
    ev = np.linalg.eigvalsh(T)
    for nu, nd in ((2, 1), (3, 3), (1, 4)):
        e = fci.fci_lowest(T, V, nu, nd, 1)[0]
        assert abs(e - (ev[:nu].sum() + ev[:nd].sum())) < 1e-12


def test_number_operator_identities():
    """T = eps*1 gives eps*N; V_ijkl = U d_ik d_jl gives U N(N-1)/2 (closed forms)."""
    L, nu, nd = 5, 2, 2
    T = 0.37 * np.eye(L)
    V = np.zeros((L,) * 4)
    for i in range(L):
        for j in range(L):
            V[i, j, i, j] = 1.9
    H, _ = fci.fci_hamiltonian(T, V, nu, nd)
    N = nu + nd
    assert np.abs(H - (0.37 * N + 1.9 * N * (N - 1) / 2) * np.eye(len(H))).max() < 1e-12


def test_hermitian_when_V_is():
    rng = np.random.default_rng(1)
    L = 4
    T = rng.normal(size=(L, L)); T = T + T.T
    V = rng.normal(size=(L,) * 4); V = V + V.transpose(2, 3, 0, 1)
    H, _ = fci.fci_hamiltonian(T, V, 2, 2)
    assert np.abs(H - H.T).max() < 1e-13


def test_against_jordan_wigner_matrices():
    """Independent construction: Kronecker-product Jordan-Wigner matrices on the full Fock space."""
    rng = np.random.default_rng(2)
    L = 3
    T = rng.normal(size=(L, L)); T = T + T.T
    V = rng.normal(size=(L,) * 4); V = V + V.transpose(2, 3, 0, 1)
    n = 2 * L
    a = np.array([[0.0, 1.0], [0.0, 0.0]])      # annihilator on one mode, basis (|0>, |1>)
    Z = np.diag([1.0, -1.0])
    ann = []
    for p in range(n):
        m = np.ones((1, 1))
        for q in range(n):
            m = np.kron(m, Z if q < p else (a if q == p else np.eye(2)))
        ann.append(m)                             # mode 0 is the most significant Kronecker factor
    H = np.zeros((2 ** n, 2 ** n))
    for i in range(L):
        for j in range(L):
            for s in (0, 1):
                H += T[i, j] * ann[2 * i + s].T @ ann[2 * j + s]
                for k in range(L):
                    for l in range(L):
                        for t in (0, 1):
                            H += 0.5 * V[i, j, k, l] * (ann[2 * i + s].T @ ann[2 * j + t].T
                                                          @ ann[2 * l + t] @ ann[2 * k + s])
    nu, nd = 2, 1
    Hf, dets = fci.fci_hamiltonian(T, V, nu, nd)
    # Fock index of a determinant: mode p has Kronecker weight 2^(n-1-p)
    idx = [sum(((int(d) >> p) & 1) << (n - 1 - p) for p in range(n)) for d in dets]
    assert np.abs(H[np.ix_(idx, idx)] - Hf).max() < 1e-12

"""ORACLE (test infrastructure, CPU only): brute-force full CI in the determinant basis.

This file is part of the independent reference implementation.  Only `tests/`,
`__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs may import
it; the product path (`paper_2501_18263_b200/`) never does.

What it computes: the Hamiltonian of PAPER.md Eq. (1) with the 1/2 of
BASELINE.json's north_star (reading R1),

    H = sum_{ij,s} T_ij a+_{is} a_{js} + 1/2 sum_{ijkl,s,t} V_ijkl a+_{is} a+_{jt} a_{lt} a_{ks},

written out literally in the N-electron determinant space of PAPER.md Eq. (2):
every elementary operator string is applied to every determinant, with the fermion sign
obtained by counting occupied spin-orbitals to the left.  No symmetry of T or V is assumed.

Conventions: spin-orbital index p = 2*i + s, i = 0..L-1 the orbital,
s = 0 (up), 1 (down).  A determinant is an integer whose bit p is the occupation n_p, and
|n_0 n_1 ...> = prod_p (a+_p)^{n_p} |0> with a+_0 leftmost, so
    a_p |D> = (-1)^{sum_{q<p} n_q} |D - p>   (same sign rule for a+_p).

Pins (tests/test_oracle_fci.py): PAPER.md:202 printed energies of the 4x4 spinless t-V torus,
the Hubbard-dimer closed form, Hermiticity, and agreement with Jordan-Wigner matrices.
"""
from __future__ import annotations

import itertools

import numpy as np


def determinants(L: int, n_up: int, n_dn: int) -> np.ndarray:
    """All determinants with n_up up and n_dn down electrons, as sorted uint64 bit strings."""
    dets = []
    for ups in itertools.combinations(range(L), n_up):
        bu = 0
        for i in ups:
            bu |= 1 << (2 * i)
        for dns in itertools.combinations(range(L), n_dn):
            b = bu
            for i in dns:
                b |= 1 << (2 * i + 1)
            dets.append(b)
    return np.array(sorted(dets), dtype=np.uint64)


def apply_string(ops, dets: np.ndarray):
    """Apply an operator string to every determinant.

    ops = [(is_creator, p), ...] in the order it is written (leftmost first); the rightmost
    operator acts first.  Returns (new_dets, sign, alive) arrays.
    """
    cur = dets.copy()
    sign = np.ones(len(dets), dtype=np.float64)
    alive = np.ones(len(dets), dtype=bool)
    one = np.uint64(1)
    for is_creator, p in reversed(ops):
        bit = one << np.uint64(p)
        occ = (cur & bit) != 0
        alive &= (~occ) if is_creator else occ
        below = cur & (bit - one)
        par = np.bitwise_count(below) & 1
        sign = np.where(par == 1, -sign, sign)
        cur = cur ^ bit
    return cur, sign, alive


def fci_triplets(T: np.ndarray, V: np.ndarray, n_up: int, n_dn: int, tol: float = 0.0):
    """(dets, rows, cols, vals) of H in the (n_up, n_dn) determinant space (duplicates to be summed)."""
    L = T.shape[0]
    dets = determinants(L, n_up, n_dn)
    idx = np.arange(len(dets))
    rows, cols, vals = [], [], []

    def emit(ops, coef):
        new, sg, alive = apply_string(ops, dets)
        if not alive.any():
            return
        src = idx[alive]
        pos = np.searchsorted(dets, new[alive])
        rows.append(pos)
        cols.append(src)
        vals.append(coef * sg[alive])

    for i in range(L):
        for j in range(L):
            if abs(T[i, j]) <= tol:
                continue
            for s in (0, 1):
                emit([(True, 2 * i + s), (False, 2 * j + s)], T[i, j])
    nz = np.argwhere(np.abs(V) > tol)
    for i, j, k, l in nz:
        v = 0.5 * V[i, j, k, l]
        for s in (0, 1):
            for t in (0, 1):
                emit([(True, 2 * i + s), (True, 2 * j + t), (False, 2 * l + t), (False, 2 * k + s)], v)
    if rows:
        return dets, np.concatenate(rows), np.concatenate(cols), np.concatenate(vals)
    z = np.zeros(0, dtype=np.int64)
    return dets, z, z, np.zeros(0)


def fci_hamiltonian(T, V, n_up, n_dn):
    """Dense H (ndet x ndet) and the determinant list."""
    dets, r, c, v = fci_triplets(T, V, n_up, n_dn)
    H = np.zeros((len(dets), len(dets)))
    np.add.at(H, (r, c), v)
    return H, dets


def fci_lowest(T, V, n_up, n_dn, nev: int = 1):
    """Lowest `nev` eigenvalues (dense eigh below 6000 determinants, Lanczos above)."""
    dets, r, c, v = fci_triplets(T, V, n_up, n_dn)
    n = len(dets)
    if n <= 6000:
        H = np.zeros((n, n))
        np.add.at(H, (r, c), v)
        return np.linalg.eigvalsh(H)[:nev]
    import scipy.sparse as sp
    import scipy.sparse.linalg as spla
    H = sp.coo_matrix((v, (r, c)), shape=(n, n)).tocsr()
    w = spla.eigsh(H, k=max(nev, 2), which="SA", tol=1e-12, return_eigenvectors=False)
    return np.sort(w)[:nev]


def site_states_to_det(states) -> int:
    """Occupation bit string of the product state |s_1 ... s_L>, s in {0, dn, up, up+dn}.

    With |3> = a+_up a+_dn |0> (R3) the product state equals the
    determinant with those occupations, with sign +1.
    """
    b = 0
    for i, s in enumerate(states):
        if s in (2, 3):
            b |= 1 << (2 * i)
        if s in (1, 3):
            b |= 1 << (2 * i + 1)
    return b

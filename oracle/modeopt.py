"""ORACLE (test infrastructure, CPU only): steps ii) and iii) of the mode-optimisation micro-iteration.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs may import this file;
it shares no code with the CUDA path and never calls it.

What it computes (Sec. II.B, :57-75; Fig. 1, :63).  A two-site orbital rotation u^(k,k+1),
    c~+_{k,s}   =  cos(theta) c+_{k,s} + sin(theta) c+_{k+1,s}
    c~+_{k+1,s} = -sin(theta) c+_{k,s} + cos(theta) c+_{k+1,s}          (spin independent),
keeps the Hamiltonian of Eq. (1) as an operator when the integrals are rotated with it, t -> U t U^T and
v_abcd -> sum U_ai U_bj U_ck U_dl v_ijkl ("rotate the one- and two-body integrals").  The unitary of the
Fock space that realises it is exp(theta kappa), kappa = sum_s (c+_{k+1,s} c_{k,s} - c+_{k,s} c_{k+1,s}), because
[kappa, c+_k] = c+_{k+1} and [kappa, c+_{k+1}] = -c+_k; the coefficients of a fixed state in the occupation basis of
the rotated modes are therefore psi~ = exp(-theta kappa) psi.  On the two-site wavefunction only the 16-dimensional
occupation space of sites k, k+1 is touched (kappa is bilinear in neighbouring modes: no Jordan-Wigner string).
The cost function is the half-Renyi block entropy of the cut between the two sites,
    S_1/2(rho_{1..k}) = 2 ln Tr sqrt(rho_{1..k}) = 2 ln sum_i sigma_i,
with sigma_i the singular values of Psi[(a s_k), (s_{k+1} b)] of the normalised state ("requires an SVD in every
cycle").  The search for theta is a plain scan + golden-section refinement (the paper says "searched
iteratively", nothing more; reading R21).

Pins (tests/test_oracle_modeopt.py): the FCI spectrum is invariant under `rotate_integrals`; the FCI ground vector
transformed by exp(-theta K) (K = kappa in the determinant space, built by oracle/fci.py from its definition) is
the ground vector of the rotated Hamiltonian (fixes the sign of theta and the index convention jointly); the
two-site gate equals that determinant-space rotation through the explicit Fock embedding of the block states;
closed forms of the entropy (product state 0, singlet pair ln 2).
"""
from __future__ import annotations

import numpy as np
from scipy.linalg import expm

from .dmrg import SITE_Q, _CRE

_PAR = np.diag([1.0, -1.0, -1.0, 1.0])


def pair_generator():
    """kappa on the occupation basis of two neighbouring sites (index 4 s1 + s2, site k first), from Jordan-Wigner
    matrices: c+_{1,s} = c+_s (x) 1,  c+_{2,s} = P (x) c+_s."""
    K = np.zeros((16, 16))
    for s in (0, 1):
        c1 = np.kron(_CRE[s], np.eye(4))
        c2 = np.kron(_PAR, _CRE[s])
        K += c2 @ c1.T - c1 @ c2.T
    return K


def two_site_rotation(theta):
    """16 x 16 matrix R with psi~ = R psi (coefficients of the same state in the rotated modes)."""
    return expm(-theta * pair_generator())


def rotation_matrix(L, k, theta):
    """U (L x L) with the 2 x 2 block on orbitals k-1, k (sites k, k+1, 1-based)."""
    U = np.eye(L)
    c, s = np.cos(theta), np.sin(theta)
    U[k - 1, k - 1] = c; U[k - 1, k] = s
    U[k, k - 1] = -s; U[k, k] = c
    return U


def rotate_integrals(T, V, k, theta):
    U = rotation_matrix(T.shape[0], k, theta)
    Tn = U @ T @ U.T
    Vn = np.einsum("ai,bj,ck,dl,ijkl->abcd", U, U, U, U, V, optimize=True)
    return Tn, Vn


def apply_gate(psi_blocks, v, G):
    """psi'{a, s1' s2', b} = sum G[(s1' s2'), (s1 s2)] psi{a, s1 s2, b} on the flat block layout (qL, s1, s2, qR, dL, dR)."""
    off, o = {}, 0
    for (qL, s1, s2, qR, dL, dR) in psi_blocks:
        off[(qL, s1, s2)] = (o, dL * dR, qR)
        o += dL * dR
    out = np.zeros_like(v)
    for (qL, s1o, s2o, qR, dL, dR) in psi_blocks:
        oo, n, _ = off[(qL, s1o, s2o)]
        for s1 in range(4):
            for s2 in range(4):
                g = G[4 * s1o + s2o, 4 * s1 + s2]
                if g == 0.0 or (qL, s1, s2) not in off:
                    continue
                oi, ni, qRi = off[(qL, s1, s2)]
                if qRi != qR:
                    assert abs(g) < 1e-14, "gate does not conserve the particle numbers of the pair"
                    continue
                out[oo:oo + n] += g * v[oi:oi + ni]
    return out


def bond_spectrum(psi_blocks, v):
    """Singular values of Psi[(a s_k), (s_{k+1} b)], sector by sector of bond k (q = qL + q(s_k)), unnormalised."""
    sectors = {}
    o = 0
    for (qL, s1, s2, qR, dL, dR) in psi_blocks:
        q = (qL[0] + SITE_Q[s1][0], qL[1] + SITE_Q[s1][1])
        sectors.setdefault(q, []).append(((qL, s1), (s2, qR), v[o:o + dL * dR].reshape(dL, dR)))
        o += dL * dR
    sig = []
    for q in sorted(sectors):
        rows, cols = {}, {}
        nr = nc = 0
        for rk, ck, m in sectors[q]:
            if rk not in rows:
                rows[rk] = nr; nr += m.shape[0]
            if ck not in cols:
                cols[ck] = nc; nc += m.shape[1]
        M = np.zeros((nr, nc))
        for rk, ck, m in sectors[q]:
            M[rows[rk]:rows[rk] + m.shape[0], cols[ck]:cols[ck] + m.shape[1]] = m
        sig.append(np.linalg.svd(M, compute_uv=False))
    return np.concatenate(sig)


def entropies(sigma):
    """(S_1/2, S_1) of the normalised spectrum."""
    p = sigma ** 2 / np.sum(sigma ** 2)
    s_half = 2.0 * np.log(np.sum(np.sqrt(p)))
    pp = p[p > 0]
    return float(s_half), float(-np.sum(pp * np.log(pp)))


def half_renyi(psi_blocks, v):
    return entropies(bond_spectrum(psi_blocks, v))[0]


def optimise_theta(cost, ngrid=24, iters=40):
    """argmin over theta in [-pi/2, pi/2) of cost(theta): scan on ngrid points, then golden-section search in the
    bracket around the best point (reading R21).  Returns (theta, cost(theta))."""
    grid = -0.5 * np.pi + np.pi * np.arange(ngrid) / ngrid
    vals = [cost(t) for t in grid]
    i = int(np.argmin(vals))
    h = np.pi / ngrid
    a, b = grid[i] - h, grid[i] + h
    gr = 0.5 * (np.sqrt(5.0) - 1.0)
    c, d = b - gr * (b - a), a + gr * (b - a)
    fc, fd = cost(c), cost(d)
    for _ in range(iters):
        if fc < fd:
            b, d, fd = d, c, fc
            c = b - gr * (b - a)
            fc = cost(c)
        else:
            a, c, fc = c, d, fd
            d = a + gr * (b - a)
            fd = cost(d)
    t = 0.5 * (a + b)
    ft = cost(t)
    if vals[i] < ft:
        return float(grid[i]), float(vals[i])
    return float(t), float(ft)

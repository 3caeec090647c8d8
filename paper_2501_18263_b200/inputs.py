"""Seeded synthetic input generators shared by the tests, the oracle harness and bench.py.

This module holds NONE of the method's arithmetic (no Hamiltonian, no operators, no
contraction): it only draws the integrals T/V, the bond-sector sizes, random canonical MPS
tensors and a start vector, in the shapes BASELINE.json's configs name.  The oracle
(`oracle/`) and the CUDA library (`csrc/`) both receive these arrays; neither imports the
other.  Recipe: DESIGN.md "Input recipe" (BASELINE.json `configs`).

Conventions (PAPER.md:41 occupation basis):
  site state s = 0..3 = {0, dn, up, up+dn};  q(s) = (n_up, n_dn) = (0,0),(0,1),(1,0),(1,1)
  bond b (0..L) sits between site b and site b+1 (sites are 1-based); its sector label
  q = (n_up, n_dn) counts the electrons in sites 1..b.
  site tensor of site i: blocks keyed (q_in, s) -> q_out = q_in + q(s), shape (d_in, d_out).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

SITE_Q = ((0, 0), (0, 1), (1, 0), (1, 1))

# BASELINE.json configs (index = config number).  `ell` is the L^P decay length, `nP_per_L`
# the number of Cholesky-like vectors per orbital.
CONFIGS = {
    0: dict(L=8, n_up=4, n_dn=4, D=10**9, ell=4.0, nP_per_L=2, seed=1000),
    1: dict(L=20, n_up=10, n_dn=10, D=256, ell=4.0, nP_per_L=2, seed=1001),
    2: dict(L=30, n_up=12, n_dn=12, D=1024, ell=4.0, nP_per_L=2, seed=1002),
    3: dict(L=40, n_up=14, n_dn=14, D=4096, ell=4.0, nP_per_L=2, seed=1003),
    4: dict(L=56, n_up=20, n_dn=20, D=8192, ell=12.0, nP_per_L=3, seed=1004),
}


def make_integrals(L: int, seed: int, ell: float = 4.0, nP_per_L: int = 2):
    """T (L,L) symmetric and V (L,L,L,L) with V_ijkl = sum_P L^P_ij L^P_kl (BASELINE.json configs[0]).

    Draw order: T_ii (sorted ascending), T_ij i<j row-major, then for each
    P the upper triangle of L^P row-major.
    """
    rng = np.random.Generator(np.random.PCG64(seed))
    T = np.zeros((L, L))
    T[np.arange(L), np.arange(L)] = np.sort(rng.uniform(-2.0, 1.0, size=L))
    iu = np.triu_indices(L, 1)
    T[iu] = rng.normal(0.0, 0.05, size=len(iu[0]))
    T = np.triu(T) + np.triu(T, 1).T
    nP = nP_per_L * L
    iu0 = np.triu_indices(L, 0)
    decay = np.exp(-np.abs(iu0[0] - iu0[1]) / ell)
    LP = np.zeros((nP, L, L))
    for P in range(nP):
        vals = rng.normal(0.0, 0.1, size=len(iu0[0])) * decay
        M = np.zeros((L, L))
        M[iu0] = vals
        LP[P] = M + np.triu(M, 1).T
    V = np.einsum("pij,pkl->ijkl", LP, LP, optimize=True)
    return T, V


def _binom(n, k):
    return math.comb(n, k) if 0 <= k <= n else 0


def bond_sectors(L: int, n_up: int, n_dn: int, D: int):
    """Sector sizes d_b(q) for every bond b=0..L (BASELINE.json configs[1]).

    weight(q) = h(n_up) h(n_dn), h(n) = C(b,n) C(L-b, N_sigma - n); cap(q) = min(#left states,
    #right states); water-filling to total D, largest-remainder rounding, then clipping so
    that every site tensor can be an isometry.  Returns a list of dicts {q: dim}.
    """
    secs = []
    for b in range(L + 1):
        cand = {}
        for a in range(0, min(b, n_up) + 1):
            for c in range(0, min(b, n_dn) + 1):
                nl = _binom(b, a) * _binom(b, c)
                nr = _binom(L - b, n_up - a) * _binom(L - b, n_dn - c)
                if nl == 0 or nr == 0:
                    continue
                w = float(_binom(b, a) * _binom(L - b, n_up - a)) * float(_binom(b, c) * _binom(L - b, n_dn - c))
                cand[(a, c)] = (w, min(nl, nr))
        caps = {q: v[1] for q, v in cand.items()}
        if sum(caps.values()) <= D:
            secs.append(dict(caps))
            continue
        qs = sorted(cand)
        w = np.array([cand[q][0] for q in qs], dtype=np.float64)
        cap = np.array([cand[q][1] for q in qs], dtype=np.float64)
        lo, hi = 0.0, float(D) / w.min() * 4.0
        for _ in range(200):  # bisection on the water level
            mid = 0.5 * (lo + hi)
            if np.minimum(cap, mid * w).sum() > D:
                hi = mid
            else:
                lo = mid
        x = np.minimum(cap, lo * w)
        base = np.floor(x).astype(np.int64)
        rem = x - base
        short = int(D - base.sum())
        order = np.argsort(-rem, kind="stable")
        for idx in order[:max(short, 0)]:
            if base[idx] < cap[idx]:
                base[idx] += 1
        secs.append({q: int(d) for q, d in zip(qs, base) if d > 0})
    # clipping passes (left->right and right->left) for isometry feasibility
    for _ in range(3):
        for b in range(1, L + 1):
            new = {}
            for q, d in secs[b].items():
                tot = 0
                for s in range(4):
                    qi = (q[0] - SITE_Q[s][0], q[1] - SITE_Q[s][1])
                    tot += secs[b - 1].get(qi, 0)
                d2 = min(d, tot)
                if d2 > 0:
                    new[q] = d2
            secs[b] = new
        for b in range(L - 1, -1, -1):
            new = {}
            for q, d in secs[b].items():
                tot = 0
                for s in range(4):
                    qo = (q[0] + SITE_Q[s][0], q[1] + SITE_Q[s][1])
                    tot += secs[b + 1].get(qo, 0)
                d2 = min(d, tot)
                if d2 > 0:
                    new[q] = d2
            secs[b] = new
    return secs


@dataclass
class MPSInput:
    """Random block-sparse MPS around the two-site bond (k, k+1).

    sectors[b]  : dict q -> dim for bond b = 0..L
    left[i]     : for sites i = 1..k-1, dict (q_in, s) -> (d_in, d_out) block, left-canonical
                  (sum over (q_in, s) of A^T A = identity on each q_out)
    right[i]    : for sites i = k+2..L, dict (q_in, s) -> (d_in, d_out) block, right-canonical
                  (sum over (s, q_out) of A A^T = identity on each q_in)
    """
    L: int
    k: int
    n_up: int
    n_dn: int
    sectors: list
    left: dict = field(default_factory=dict)
    right: dict = field(default_factory=dict)


def _qadd(q, s):
    return (q[0] + SITE_Q[s][0], q[1] + SITE_Q[s][1])


def make_mps(L: int, n_up: int, n_dn: int, D: int, k: int, seed: int, sectors=None) -> MPSInput:
    """Random N(0,1) site tensors made canonical by QR with diag(R) > 0."""
    if sectors is None:
        sectors = bond_sectors(L, n_up, n_dn, D)
    rng = np.random.Generator(np.random.PCG64(seed + 7919))
    mps = MPSInput(L=L, k=k, n_up=n_up, n_dn=n_dn, sectors=sectors)
    for i in range(1, k):  # left-canonical sites 1..k-1 : bond i-1 -> bond i
        site = {}
        for qo in sorted(sectors[i]):
            do = sectors[i][qo]
            rows = []
            for qi in sorted(sectors[i - 1]):
                for s in range(4):
                    if _qadd(qi, s) == qo:
                        rows.append((qi, s, sectors[i - 1][qi]))
            nrow = sum(r[2] for r in rows)
            assert nrow >= do, "sector clipping failed (left)"
            M = rng.normal(size=(nrow, do))
            Q, R = np.linalg.qr(M)
            Q = Q * np.sign(np.diag(R))[None, :]
            off = 0
            for qi, s, d in rows:
                site[(qi, s)] = np.ascontiguousarray(Q[off:off + d, :])
                off += d
        mps.left[i] = site
    for i in range(L, k + 1, -1):  # right-canonical sites L..k+2 : bond i-1 <- bond i
        site = {}
        for qi in sorted(sectors[i - 1]):
            di = sectors[i - 1][qi]
            cols = []
            for s in range(4):
                qo = _qadd(qi, s)
                if qo in sectors[i]:
                    cols.append((s, qo, sectors[i][qo]))
            ncol = sum(c[2] for c in cols)
            assert ncol >= di, "sector clipping failed (right)"
            M = rng.normal(size=(ncol, di))
            Q, R = np.linalg.qr(M)
            Q = (Q * np.sign(np.diag(R))[None, :]).T  # (di, ncol), orthonormal rows
            off = 0
            for s, qo, d in cols:
                site[(qi, s)] = np.ascontiguousarray(Q[:, off:off + d])
                off += d
        mps.right[i] = site
    return mps


def make_left_site(sectors, i: int, seed: int):
    """One random left-canonical site tensor (site i, bond i-1 -> bond i) by the recipe of make_mps, for a single
    renormalisation step at a bond whose site tensors make_mps left open (sites k, k+1)."""
    rng = np.random.Generator(np.random.PCG64(seed + 7919 + 31 * i))
    site = {}
    for qo in sorted(sectors[i]):
        do = sectors[i][qo]
        rows = []
        for qi in sorted(sectors[i - 1]):
            for s in range(4):
                if _qadd(qi, s) == qo:
                    rows.append((qi, s, sectors[i - 1][qi]))
        nrow = sum(r[2] for r in rows)
        assert nrow >= do, "sector clipping failed (left)"
        Q, R = np.linalg.qr(rng.normal(size=(nrow, do)))
        Q = Q * np.sign(np.diag(R))[None, :]
        off = 0
        for qi, s, d in rows:
            site[(qi, s)] = np.ascontiguousarray(Q[off:off + d, :])
            off += d
    return site


def psi_blocks(mps: MPSInput):
    """Ordered list of two-site wavefunction blocks (qL, s1, s2, qbond_R) with shapes.

    qL is the label of bond k-1, qbond_R = qL + q(s1) + q(s2) the label of bond k+1 (so the
    right block holds N - qbond_R electrons).  Order: qL lexicographic, then s1, then s2.
    Returns list of (qL, s1, s2, qR_bond, dL, dR).
    """
    k = mps.k
    out = []
    sl, sr = mps.sectors[k - 1], mps.sectors[k + 1]
    for qL in sorted(sl):
        for s1 in range(4):
            for s2 in range(4):
                qr = _qadd(_qadd(qL, s1), s2)
                if qr in sr:
                    out.append((qL, s1, s2, qr, sl[qL], sr[qr]))
    return out


def make_psi0(mps: MPSInput, seed: int):
    """Normalised N(0,1) start vector, flat, blocks row-major in psi_blocks() order."""
    rng = np.random.Generator(np.random.PCG64(seed + 104729))
    n = sum(b[4] * b[5] for b in psi_blocks(mps))
    v = rng.normal(size=n)
    return v / np.linalg.norm(v)


def make_config(cfg: int, D: int | None = None, k: int | None = None):
    """(T, V, mps) for BASELINE.json config `cfg` at the middle bond (sites L/2, L/2+1)."""
    c = CONFIGS[cfg]
    L = c["L"]
    T, V = make_integrals(L, c["seed"], c["ell"], c["nP_per_L"])
    kk = L // 2 if k is None else k
    mps = make_mps(L, c["n_up"], c["n_dn"], c["D"] if D is None else D, kk, c["seed"])
    return T, V, mps


# =================================================================================================
# SU(2)-adapted inputs (BASELINE.json configs[3] second half and configs[4]).
# A bond sector is labelled q = (N, 2S): N electrons and total spin S in sites 1..b.  The site carries
# three multiplets m = 0, 1, 2 = (N=0,S=0), (N=1,S=1/2), (N=2,S=0).  A reduced site
# tensor block is keyed (q_in, m, q_out) with q_out = (N_in + n(m), 2S_in + {0 | +-1}); shapes
# (d_in, d_out), counted in multiplets.  Still no method arithmetic here: only sizes and random isometries.
# =================================================================================================
SITE_MULT = ((0, 0), (1, 1), (2, 0))   # (N, 2S) of the site multiplets m = 0, 1, 2


def su2_couplings(q, m):
    """Bond labels reachable from q = (N, 2S) by adding site multiplet m."""
    n, s2 = SITE_MULT[m]
    if s2 == 0:
        return [(q[0] + n, q[1])]
    out = [(q[0] + n, q[1] + 1)]
    if q[1] >= 1:
        out.append((q[0] + n, q[1] - 1))
    return out


def _mult_count(b, N, S2):
    """Number of (N, S) multiplets of b orbitals: #(N, Sz=S) - #(N, Sz=S+1), #(N,Sz) = C(b,na) C(b,nb)."""
    def cnt(sz2):
        if (N + sz2) % 2:
            return 0
        na, nb = (N + sz2) // 2, (N - sz2) // 2
        return _binom(b, na) * _binom(b, nb)
    return cnt(S2) - cnt(S2 + 2)


def su2_bond_sectors(L: int, N_tot: int, S2_tot: int, D: int):
    """Multiplet counts d_b(N, 2S) for every bond: weight m_b(N,S) * m_{L-b}(N_tot-N, S) (target S_tot = 0:
    the right part carries the same S; for S_tot != 0 the sum over the allowed right spins), cap = min of
    the two factors, water-filling to D multiplets, largest-remainder rounding, clipping passes."""
    secs = []
    for b in range(L + 1):
        cand = {}
        for N in range(0, min(2 * b, N_tot) + 1):
            for S2 in range(N % 2, min(N, 2 * b - N) + 1, 2):
                ml = _mult_count(b, N, S2)
                if ml <= 0:
                    continue
                mr = 0
                for S2r in range(abs(S2 - S2_tot), S2 + S2_tot + 1, 2):
                    mr += max(_mult_count(L - b, N_tot - N, S2r), 0)
                if mr <= 0:
                    continue
                cand[(N, S2)] = (float(ml) * float(mr), min(ml, mr))
        caps = {q: v[1] for q, v in cand.items()}
        if sum(caps.values()) <= D:
            secs.append(dict(caps))
            continue
        qs = sorted(cand)
        w = np.array([cand[q][0] for q in qs], dtype=np.float64)
        cap = np.array([cand[q][1] for q in qs], dtype=np.float64)
        lo, hi = 0.0, float(D) / w.min() * 4.0
        for _ in range(200):
            mid = 0.5 * (lo + hi)
            if np.minimum(cap, mid * w).sum() > D:
                hi = mid
            else:
                lo = mid
        x = np.minimum(cap, lo * w)
        base = np.floor(x).astype(np.int64)
        rem = x - base
        short = int(D - base.sum())
        order = np.argsort(-rem, kind="stable")
        for idx in order[:max(short, 0)]:
            if base[idx] < cap[idx]:
                base[idx] += 1
        secs.append({q: int(d) for q, d in zip(qs, base) if d > 0})
    for _ in range(3):
        for b in range(1, L + 1):
            new = {}
            for q, d in secs[b].items():
                tot = 0
                for qi, di in secs[b - 1].items():
                    for m in range(3):
                        if q in su2_couplings(qi, m):
                            tot += di
                d2 = min(d, tot)
                if d2 > 0:
                    new[q] = d2
            secs[b] = new
        for b in range(L - 1, -1, -1):
            new = {}
            for q, d in secs[b].items():
                tot = 0
                for m in range(3):
                    for qo in su2_couplings(q, m):
                        tot += secs[b + 1].get(qo, 0)
                d2 = min(d, tot)
                if d2 > 0:
                    new[q] = d2
            secs[b] = new
    return secs


@dataclass
class SU2MPSInput:
    """Random reduced (multiplet) MPS around the bond (k, k+1), total spin 0.

    sectors[b] : dict (N, 2S) -> number of multiplets, label = content of sites 1..b (the right block of
                 a bond then holds (N_tot - N, S), because S_tot = 0)
    left[i]    : sites 1..k-1, dict (q_in, m, q_out) -> (d_in, d_out), sum over (q_in, m) of A^T A = 1 per q_out
    right[i]   : sites k+2..L, dict (q_in, m, q_out) -> (d_in, d_out), sum over (m, q_out) of A A^T = 1 per q_in
    Coupling order: left states |(block, site) S'>, right states |(site, block) S'>.
    """
    L: int
    k: int
    N: int
    sectors: list
    left: dict = field(default_factory=dict)
    right: dict = field(default_factory=dict)


def make_mps_su2(L: int, N_tot: int, D: int, k: int, seed: int, sectors=None) -> SU2MPSInput:
    if sectors is None:
        sectors = su2_bond_sectors(L, N_tot, 0, D)
    rng = np.random.Generator(np.random.PCG64(seed + 15485863))
    mps = SU2MPSInput(L=L, k=k, N=N_tot, sectors=sectors)
    for i in range(1, k):
        site = {}
        for qo in sorted(sectors[i]):
            do = sectors[i][qo]
            rows = []
            for qi in sorted(sectors[i - 1]):
                for m in range(3):
                    if qo in su2_couplings(qi, m):
                        rows.append((qi, m, sectors[i - 1][qi]))
            nrow = sum(r[2] for r in rows)
            assert nrow >= do, "sector clipping failed (left, su2)"
            Q, R = np.linalg.qr(rng.normal(size=(nrow, do)))
            Q = Q * np.sign(np.diag(R))[None, :]
            off = 0
            for qi, m, d in rows:
                site[(qi, m, qo)] = np.ascontiguousarray(Q[off:off + d, :])
                off += d
        mps.left[i] = site
    for i in range(L, k + 1, -1):
        site = {}
        for qi in sorted(sectors[i - 1]):
            di = sectors[i - 1][qi]
            cols = []
            for m in range(3):
                for qo in su2_couplings(qi, m):
                    if qo in sectors[i]:
                        cols.append((m, qo, sectors[i][qo]))
            ncol = sum(c[2] for c in cols)
            assert ncol >= di, "sector clipping failed (right, su2)"
            Q, R = np.linalg.qr(rng.normal(size=(ncol, di)))
            Q = (Q * np.sign(np.diag(R))[None, :]).T
            off = 0
            for m, qo, d in cols:
                site[(qi, m, qo)] = np.ascontiguousarray(Q[:, off:off + d])
                off += d
        mps.right[i] = site
    return mps


def psi_blocks_su2(mps: SU2MPSInput):
    """Reduced two-site wavefunction blocks for S_tot = 0, in order (qL, m1, qLp, m2, qR):
    qL = label of bond k-1, qLp = (N, 2S') of L' = L + site k, qR = label of bond k+1 (the right block holds
    (N_tot - N, S) with that S), and R' = site k+1 + R must carry S' too, i.e. qLp in couplings(qL, m1) and
    qR in couplings(qLp, m2).  Returns list of (qL, m1, qLp, m2, qR, dL, dR)."""
    k = mps.k
    sl, sr = mps.sectors[k - 1], mps.sectors[k + 1]
    out = []
    for qL in sorted(sl):
        for m1 in range(3):
            for qLp in sorted(su2_couplings(qL, m1)):
                for m2 in range(3):
                    for qR in sorted(su2_couplings(qLp, m2)):
                        if qR in sr:
                            out.append((qL, m1, qLp, m2, qR, sl[qL], sr[qR]))
    return out


def make_psi0_su2(mps: SU2MPSInput, seed: int):
    rng = np.random.Generator(np.random.PCG64(seed + 32452843))
    n = sum(b[5] * b[6] for b in psi_blocks_su2(mps))
    v = rng.normal(size=n)
    return v / np.linalg.norm(v)


SU2_CONFIGS = {
    3: dict(L=40, N=28, D=1024, ell=4.0, nP_per_L=2, seed=1003),
    4: dict(L=56, N=40, D=4096, ell=12.0, nP_per_L=3, seed=1004),
}


def make_config_su2(cfg: int, D: int | None = None):
    c = SU2_CONFIGS[cfg]
    T, V = make_integrals(c["L"], c["seed"], c["ell"], c["nP_per_L"])
    mps = make_mps_su2(c["L"], c["N"], c["D"] if D is None else D, c["L"] // 2, c["seed"])
    return T, V, mps

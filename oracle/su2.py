"""ORACLE (test infrastructure, CPU only): SU(2) spin adaptation of the two-site problem.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs may
import this file; it shares no code with the CUDA path (no 9j / F / task-prefactor code in common).

What it computes (SURVEY.md 8(c) "SU(2) oracle"):

    oracle_su2(psi_red) = reduce( oracle_u1( expand(psi_red) ) )

The reduced (multiplet) MPS of PAPER.md:115-121 is expanded into an ordinary U(1)xU(1) MPS with
Clebsch-Gordan coefficients, using the paper's hierarchical coupling order (PAPER.md:129:
H'_L = H_L (x) H_k, H'_R = H_{k+1} (x) H_R, H_eff = H'_L (x) H'_R):

    left  block state  |a' S' M'> = sum A[(a S, m) -> a' S'] <S M; s_m mu | S' M'> |a S M> |m mu>
    right block state  |b' S' M'> = sum B[(m, b S) -> b' S'] <s_m mu; S M | S' M'> |m mu> |b S M>
    two-site state     |psi>      = sum psi_red[a m1 S_L'; m2 b] |((a, m1) S_L', (m2, b) S_L') S_tot = 0>

and the U(1) oracle (oracle/dmrg.py, itself pinned against brute-force FCI) does the rest.  Site multiplets
m = 0, 1, 2 = |0>, the doublet (|up>, |dn>) = (a+_up|0>, a+_dn|0>), |up dn> = a+_up a+_dn |0>; U(1) labels
of a multiplet member: n_up = (N + 2M)/2, n_dn = (N - 2M)/2.  Inside a U(1) sector (N, M) the expanded states
are ordered by (S ascending, multiplet index).

Also here, for the a8 row: the factor F of PAPER.md Eq. (10)-(11) in both forms the paper gives — the
rescaled Wigner 9j symbol (Eq. 11, reading R11) and the contraction of six Clebsch-Gordan tensors of
PAPER.md Fig. 4 (:150) — so that a test can check one against the other.

Pins (tests/test_oracle_su2.py): CG against sympy and closed forms; 9j with a zero argument against sympy's
6j; F(9j) == F(six CG); expanded states are S^2 eigenstates in the determinant space; H_eff leaves the image
of `expand` invariant; singlet energy == lowest FCI singlet.
"""
from __future__ import annotations

from fractions import Fraction
from math import factorial, sqrt

import numpy as np

SITE_MULT = ((0, 0), (1, 1), (2, 0))          # (N, 2S) of site multiplets m = 0, 1, 2
# U(1) site state s (0, dn, up, updn) of multiplet member (m, 2*mu)
SITE_STATE = {(0, 0): 0, (1, 1): 2, (1, -1): 1, (2, 0): 3}


def cg(j1, m1, j2, m2, J, M):
    """Clebsch-Gordan coefficient <j1 m1; j2 m2 | J M> (Condon-Shortley), arguments are DOUBLED integers.

    Racah's closed formula, evaluated with exact rational arithmetic under the square root.
    """
    if m1 + m2 != M or J < abs(j1 - j2) or J > j1 + j2 or (j1 + j2 + J) % 2:
        return 0.0
    if abs(m1) > j1 or abs(m2) > j2 or abs(M) > J or (j1 + m1) % 2 or (j2 + m2) % 2 or (J + M) % 2:
        return 0.0
    f = lambda x: factorial(x // 2)   # every argument below is an even doubled integer
    pref = Fraction((J + 1) * f(J + j1 - j2) * f(J - j1 + j2) * f(j1 + j2 - J), f(j1 + j2 + J + 2))
    pref *= f(J + M) * f(J - M) * f(j1 - m1) * f(j1 + m1) * f(j2 - m2) * f(j2 + m2)
    s = Fraction(0)
    for k2 in range(0, j1 + j2 - J + 1, 2):     # k = k2/2
        a = [k2, j1 + j2 - J - k2, j1 - m1 - k2, j2 + m2 - k2, J - j2 + m1 + k2, J - j1 - m2 + k2]
        if min(a) < 0:
            continue
        den = 1
        for x in a:
            den *= f(x)
        s += Fraction((-1) ** (k2 // 2), den)
    return float(s) * sqrt(float(pref))


def sixj(a, b, c, d, e, f_):
    """Wigner 6j {a b c; d e f} (doubled integer arguments), Racah's single-sum formula."""
    def tri(x, y, z):
        if (x + y + z) % 2 or z < abs(x - y) or z > x + y:
            return None
        g = lambda t: factorial(t // 2)
        return Fraction(g(x + y - z) * g(x - y + z) * g(-x + y + z), g(x + y + z + 2))
    ts = [tri(a, b, c), tri(a, e, f_), tri(d, b, f_), tri(d, e, c)]
    if any(t is None for t in ts):
        return 0.0
    pref = ts[0] * ts[1] * ts[2] * ts[3]
    s = Fraction(0)
    lo = max(a + b + c, a + e + f_, d + b + f_, d + e + c)
    hi = min(a + b + d + e, b + c + e + f_, a + c + d + f_)
    g = lambda t: factorial(t // 2)
    for t in range(lo, hi + 1, 2):
        den = (g(t - a - b - c) * g(t - a - e - f_) * g(t - d - b - f_) * g(t - d - e - c) *
               g(a + b + d + e - t) * g(b + c + e + f_ - t) * g(a + c + d + f_ - t))
        s += Fraction((-1) ** (t // 2) * g(t + 2), den)
    return float(s) * sqrt(float(pref))


def ninej(a, b, c, d, e, f_, g, h, i):
    """Wigner 9j {a b c; d e f; g h i} as the standard sum over products of three 6j symbols."""
    s = 0.0
    lo = max(abs(a - i), abs(d - h), abs(b - f_))
    hi = min(a + i, d + h, b + f_)
    for x in range(lo, hi + 1):
        if (x + a + i) % 2:
            continue
        s += ((-1) ** x) * (x + 1) * sixj(a, b, c, f_, i, x) * sixj(d, e, f_, b, x, h) * sixj(g, h, i, x, a, d)
    return s


def F_ninej(Sa, Sk, Sg, kL, kk, kop, Sa_, Sk_, Sg_):
    """PAPER.md Eq. (11) (reading R11): F = sqrt((2Sa'+1)(2Sk'+1)(2Sg+1)(2k+1)) x
    9j{Sa Sk Sg; kL kk k; Sa' Sk' Sg'} for the reduced element of [O_L^{kL} (x) O_k^{kk}]^{k} between the
    coupled multiplets |(Sa, Sk) Sg> -> |(Sa', Sk') Sg'>, with the Wigner-Eckart theorem in Clebsch-Gordan
    form <S'M'|O^k_q|SM> = <S M; k q|S' M'> O_red[S', S].  Doubled integer arguments."""
    return sqrt((Sa_ + 1) * (Sk_ + 1) * (Sg + 1) * (kop + 1)) * ninej(Sa, Sk, Sg, kL, kk, kop, Sa_, Sk_, Sg_)


def F_sixcg(Sa, Sk, Sg, kL, kk, kop, Sa_, Sk_, Sg_):
    """The same factor as the contraction of six Clebsch-Gordan tensors with the prefactor (2Sg'+1)^-1 of
    PAPER.md Fig. 4 (:150): two state couplings, one operator coupling, two Wigner-Eckart coefficients for
    the factors and one for the product, summed over all magnetic quantum numbers."""
    tot = 0.0
    for Mg_ in range(-Sg_, Sg_ + 1, 2):
        for q in range(-kop, kop + 1, 2):
            Mg = Mg_ - q
            w_out = cg(Sg, Mg, kop, q, Sg_, Mg_)
            if w_out == 0.0:
                continue
            for qL in range(-kL, kL + 1, 2):
                qk = q - qL
                c_op = cg(kL, qL, kk, qk, kop, q)
                if c_op == 0.0:
                    continue
                for Ma in range(-Sa, Sa + 1, 2):
                    Mk = Mg - Ma
                    c_in = cg(Sa, Ma, Sk, Mk, Sg, Mg)
                    if c_in == 0.0:
                        continue
                    Ma_, Mk_ = Ma + qL, Mk + qk
                    tot += (w_out * c_op * c_in * cg(Sa_, Ma_, Sk_, Mk_, Sg_, Mg_) *
                            cg(Sa, Ma, kL, qL, Sa_, Ma_) * cg(Sk, Mk, kk, qk, Sk_, Mk_))
    return tot / (Sg_ + 1)


# ---------------------------------------------------------------------------------------------
# expansion of a reduced MPS into a U(1) x U(1) MPS
# ---------------------------------------------------------------------------------------------

def _u1_label(N, M2):
    """(n_up, n_dn) of a state with N electrons and S_z = M2/2."""
    return ((N + M2) // 2, (N - M2) // 2)


def u1_sectors(su2_sec):
    """dict (n_up, n_dn) -> (dim, layout) from dict (N, 2S) -> multiplets; layout = list of
    ((N, 2S), offset) in the order (S ascending) used inside the U(1) sector."""
    out = {}
    for (N, S2) in sorted(su2_sec, key=lambda q: (q[0], q[1])):
        d = su2_sec[(N, S2)]
        for M2 in range(-S2, S2 + 1, 2):
            key = _u1_label(N, M2)
            dim, lay = out.get(key, (0, []))
            lay = lay + [((N, S2), dim)]
            out[key] = (dim + d, lay)
    return out


def _offset(u1sec, N, S2, M2):
    dim, lay = u1sec[_u1_label(N, M2)]
    for q, off in lay:
        if q == (N, S2):
            return off
    raise KeyError((N, S2, M2))


def expand_mps(mps):
    """U(1) sectors and site tensors (the dict formats of oracle.dmrg.TwoSiteOracle) of a reduced MPS.

    `mps`: object with L, k, N, sectors[b] (dict (N,2S)->d), left[i] / right[i] (dict (q_in, m, q_out) ->
    (d_in, d_out)), S_tot = 0.  Returns (sectors_u1, left_u1, right_u1, layouts) with
    sectors_u1[b]: dict (n_up,n_dn)->dim; layouts[b] the per-sector multiplet layout.
    """
    L, Ntot = mps.L, mps.N
    lay = [u1_sectors(s) for s in mps.sectors]
    sec_u1 = [{q: v[0] for q, v in l.items()} for l in lay]
    left_u1, right_u1 = {}, {}
    for i, site in mps.left.items():
        blocks = {}
        for (qi, m, qo), A in site.items():
            (Ni, Si), (No, So) = qi, qo
            sm = SITE_MULT[m][1]
            for Mo in range(-So, So + 1, 2):
                for mu in range(-sm, sm + 1, 2):
                    Mi = Mo - mu
                    c = cg(Si, Mi, sm, mu, So, Mo)
                    if c == 0.0:
                        continue
                    s = SITE_STATE[(m, mu)]
                    key = (_u1_label(Ni, Mi), s)
                    din, dout = sec_u1[i - 1][_u1_label(Ni, Mi)], sec_u1[i][_u1_label(No, Mo)]
                    blk = blocks.setdefault(key, np.zeros((din, dout)))
                    r0, c0 = _offset(lay[i - 1], Ni, Si, Mi), _offset(lay[i], No, So, Mo)
                    blk[r0:r0 + A.shape[0], c0:c0 + A.shape[1]] += c * A
        left_u1[i] = blocks
    for i, site in mps.right.items():
        # right block of bond b with LEFT label (N, 2S) holds (Ntot - N, S); a member with S_z = M/2 of the
        # right block sits in the U(1) bond sector of the left label with S_z = -M/2 (S_z,tot = 0).
        blocks = {}
        for (qi, m, qo), B in site.items():
            (Ni, Si), (No, So) = qi, qo          # left labels of bonds i-1 and i
            sm = SITE_MULT[m][1]
            for Mnew in range(-Si, Si + 1, 2):   # S_z of the NEW (bigger) right block state, spin Si
                for mu in range(-sm, sm + 1, 2):
                    Mold = Mnew - mu
                    c = cg(sm, mu, So, Mold, Si, Mnew)
                    if c == 0.0:
                        continue
                    s = SITE_STATE[(m, mu)]
                    lab_in, lab_out = _u1_label(Ni, -Mnew), _u1_label(No, -Mold)
                    key = (lab_in, s)
                    din, dout = sec_u1[i - 1][lab_in], sec_u1[i][lab_out]
                    blk = blocks.setdefault(key, np.zeros((din, dout)))
                    r0, c0 = _offset(lay[i - 1], Ni, Si, -Mnew), _offset(lay[i], No, So, -Mold)
                    blk[r0:r0 + B.shape[0], c0:c0 + B.shape[1]] += c * B
        right_u1[i] = blocks
    return sec_u1, left_u1, right_u1, lay


class SU2TwoSiteOracle:
    """H_eff on the reduced two-site space, total spin 0, by expansion to U(1) (module docstring).

    psi_blocks: list of (qL, m1, qLp, m2, qR, dL, dR) giving the flat reduced layout (qL, qLp, qR are the
    left labels (N, 2S) of bond k-1, of L' = L + site k, and of bond k+1).
    """

    def __init__(self, T, V, mps, psi_blocks):
        from . import dmrg as odmrg
        self.mps = mps
        self.psi_blocks = list(psi_blocks)
        k = mps.k
        sec_u1, left_u1, right_u1, lay = expand_mps(mps)
        self.lay = lay
        n2 = mps.N // 2
        # U(1) psi layout in the documented order (qL lexicographic, s1, s2)
        pb = []
        for qL in sorted(sec_u1[k - 1]):
            for s1 in range(4):
                for s2 in range(4):
                    qr = (qL[0] + odmrg.SITE_Q[s1][0] + odmrg.SITE_Q[s2][0], qL[1] + odmrg.SITE_Q[s1][1] + odmrg.SITE_Q[s2][1])
                    if qr in sec_u1[k + 1]:
                        pb.append((qL, s1, s2, qr, sec_u1[k - 1][qL], sec_u1[k + 1][qr]))
        self.u1_blocks = pb
        self.u1 = odmrg.TwoSiteOracle(T, V, n2, n2, k, sec_u1, left_u1, right_u1, pb)
        self._build_expander(sec_u1)

    def _build_expander(self, sec_u1):
        """Sparse matrix R (n_u1 x n_red): psi_u1 = R psi_red, R^T R = 1."""
        import scipy.sparse as sp
        k, lay = self.mps.k, self.lay
        off_u1, o = {}, 0
        for (qL, s1, s2, qr, dL, dR) in self.u1_blocks:
            off_u1[(qL, s1, s2)] = (o, dL, dR)
            o += dL * dR
        self.n_u1 = o
        rows, cols, vals = [], [], []
        o = 0
        for (qL, m1, qLp, m2, qR, dL, dR) in self.psi_blocks:
            (Na, Sa), (Np, Sp), (Nr, Sr) = qL, qLp, qR
            s1m, s2m = SITE_MULT[m1][1], SITE_MULT[m2][1]
            ia = np.arange(dL)[:, None]
            ib = np.arange(dR)[None, :]
            red_idx = (o + ia * dR + ib).reshape(-1)
            for Mp in range(-Sp, Sp + 1, 2):                 # S_z of L'; R' carries -Mp
                c_tot = cg(Sp, Mp, Sp, -Mp, 0, 0)
                for mu1 in range(-s1m, s1m + 1, 2):
                    Ma = Mp - mu1
                    c1 = cg(Sa, Ma, s1m, mu1, Sp, Mp)
                    if c1 == 0.0:
                        continue
                    for mu2 in range(-s2m, s2m + 1, 2):
                        Mb = -Mp - mu2                       # S_z of the right block state (spin Sr)
                        c2 = cg(s2m, mu2, Sr, Mb, Sp, -Mp)
                        if c2 == 0.0:
                            continue
                        s1, s2 = SITE_STATE[(m1, mu1)], SITE_STATE[(m2, mu2)]
                        labL = _u1_label(Na, Ma)
                        base, DL, DR = off_u1[(labL, s1, s2)]
                        r0 = _offset(lay[k - 1], Na, Sa, Ma)
                        c0 = _offset(lay[k + 1], Nr, Sr, -Mb)
                        u_idx = (base + (r0 + ia) * DR + (c0 + ib)).reshape(-1)
                        rows.append(u_idx); cols.append(red_idx)
                        vals.append(np.full(u_idx.shape, c_tot * c1 * c2))
            o += dL * dR
        self.n_red = o
        self.R = sp.csr_matrix((np.concatenate(vals), (np.concatenate(rows), np.concatenate(cols))),
                               shape=(self.n_u1, self.n_red))

    def build_env(self):
        self.u1.build_env()

    def psi_size(self):
        return self.n_red

    def expand(self, v):
        return self.R @ np.asarray(v, dtype=np.float64)

    def reduce(self, w):
        return self.R.T @ np.asarray(w, dtype=np.float64)

    def apply(self, v):
        return self.reduce(self.u1.apply(self.expand(v)))

    def diag_exact(self):
        """diag(R^T H R) from one apply per basis vector (tiny sizes only; pins the library's diagonal)."""
        n = self.n_red
        d = np.zeros(n)
        e = np.zeros(n)
        for j in range(n):
            e[j] = 1.0
            d[j] = self.apply(e)[j]
            e[j] = 0.0
        return d

    def diag(self):
        """Davidson preconditioner for the oracle's own solver: sum_i R_ij^2 (H_u1)_ii.  It drops the couplings
        between the members of one multiplet pattern, so it is NOT the exact diagonal; converged energies do
        not depend on it."""
        return (self.R.multiply(self.R)).T @ self.u1.diag()

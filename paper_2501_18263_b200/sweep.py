"""Two-site DMRG sweep driver (SURVEY.md 8(f) item 1; Fig. 1, :63: eigensolve, SVD truncation,
renormalisation, move on).  U(1)xU(1) and SU(2) (total spin 0) contexts.

Everything on the hot path runs in the library (`dmrg_davidson`, `dmrg_renormalize`, the environment cache).
The truncation SVD, the new site tensor and the wave-function transformation (next start vector) are library calls
too in the `native` mode (`dmrg_truncate_bond`, `dmrg_start_vector`; U(1)xU(1), default for D <= 512).  Otherwise, as
north_star allows ("the truncation SVD is outside the hot path but stays on the device"), this driver does them with
torch on the device and keeps the MPS tensors as host numpy blocks, because `dmrg_mps_set_site` takes host data.

SU(2): the same steps on reduced (multiplet) blocks.  The middle-bond label of a block is (N, 2S') of
L' = L + site k; the SVD factors are plain isometries on multiplets; a singular value is the total weight of
its multiplet.  The wave-function transformation needs no extra factor: re-coupling
|(a', (m2, (m3 b2)S_b) S') 0> -> |((a' m2) S_b, (m3 b2) S_b) 0> is a 6j symbol with a zero argument and equals +1
(checked by the energy continuity test in tests/test_gpu_sweep.py).
"""
from __future__ import annotations

import numpy as np

SITE_Q = ((0, 0), (0, 1), (1, 0), (1, 1))
MULT_N = (0, 1, 2)


def _qadd(q, s):
    return (q[0] + SITE_Q[s][0], q[1] + SITE_Q[s][1])


class TwoSiteSweep:
    def __init__(self, d, T, V, mps, D, e_core=0.0, native=None):
        """d: binding.DMRG; mps: inputs.MPSInput / SU2MPSInput positioned at bond (mps.k, mps.k+1).
        native: do the truncation and the wave-function transformation with the library calls dmrg_truncate_bond /
        dmrg_start_vector (no torch.linalg, no host copy of the site tensors) instead of the torch code below.
        Default: yes for U(1)xU(1) contexts with D <= 512, where the bond sectors fit the library's shared-memory
        Jacobi SVD; the torch path stays for SU(2) and for large D (where the library's SVD is correct but slow)."""
        self.d, self.D = d, D
        self.su2 = bool(getattr(d, "su2", False))
        self.native = (not self.su2 and D <= 512) if native is None else bool(native)
        if self.native and self.su2:
            raise ValueError("the library's truncation step is U(1)xU(1) only")
        self.L = mps.L
        self.k = mps.k
        self.sectors = [dict(s) for s in mps.sectors]
        self.left = dict(mps.left)
        self.right = dict(mps.right)
        d.setup(T, V, mps, e_core)
        self.guess = None
        self.energies = []
        self.trunc = []
        # wall-time split per category, the ones of PAPER.md Fig. 20 (:284): Diag_H, SVD, Ren (+ Tables), StVec
        self.seconds = {"Diag_H": 0.0, "SVD": 0.0, "Ren+Tables": 0.0, "StVec": 0.0}

    def _tick(self, name, t0):
        import time
        self.d.torch.cuda.synchronize()
        t1 = time.perf_counter()
        self.seconds[name] += t1 - t0
        return t1

    # -- helpers --
    def _layout(self):
        blocks, n = self.d.psi_layout()
        out = []
        for b in blocks:
            qL, qR = (b.qL_up, b.qL_dn), (b.qR_up, b.qR_dn)
            qm = (qL[0] + MULT_N[b.s1], b.twoS_mid) if self.su2 else _qadd(qL, b.s1)   # label of bond k
            out.append((qL, b.s1, b.s2, qR, b.dL, b.dR, b.off, qm))
        return out, n

    def _lkey(self, qin, s, qout):
        """Key of a site-tensor block (q_in, site state or multiplet[, q_out])."""
        return (qin, s, qout) if self.su2 else (qin, s)

    def _set_site(self, site, canonical, blocks):
        (self.d.mps_set_site_su2 if self.su2 else self.d.mps_set_site)(site, canonical, blocks)

    def _start_vector(self, n, seed):
        torch = self.d.torch
        if self.guess is not None and self.guess.numel() == n:
            return self.guess
        g = torch.Generator(device="cpu").manual_seed(seed)
        x = torch.randn(n, dtype=torch.float64, generator=g).to(self.d.device)
        return x / torch.linalg.norm(x)

    def step(self, direction, tol=1e-9, max_iter=200, max_basis=16, seed=0):
        """Optimise the two-site tensor at the current bond, truncate, and move (0: right, 1: left, None: stay).
        Returns the Davidson energy."""
        torch = self.d.torch
        d, k = self.d, self.k
        layout, n = self._layout()
        import time
        x = self._start_vector(n, seed).clone()
        t0 = time.perf_counter()
        E, it, rn = d.davidson(x, tol=tol, max_iter=max_iter, max_basis=max_basis)
        t0 = self._tick("Diag_H", t0)
        self.energies.append(E)
        self.last_psi = x                      # the optimised two-site wavefunction this step truncates (tests)
        if direction is None:
            self.guess = x
            return E
        if self.native:
            # ---- the library's truncation step: SVD per bond sector, selection, new site tensor, all on the device ----
            w, _ = d.truncate_bond(x, direction, self.D)
            self.trunc.append(w)
            self.sectors[k] = d.bond_sectors(k)
            t0 = self._tick("SVD", t0)
            d.renormalize(direction)
            self.k = k + 1 if direction == 0 else k - 1
            t0 = self._tick("Ren+Tables", t0)
            y = d.start_vector()
            nrm = torch.linalg.norm(y)
            self.guess = y / nrm if float(nrm) > 0 else None
            self._tick("StVec", t0)
            return E
        # ---- SVD per middle-bond sector q_mid = qL + q(s1) ----
        groups = {}
        for (qL, s1, s2, qR, dL, dR, off, qm) in layout:
            g = groups.setdefault(qm, {"rows": {}, "cols": {}, "blk": []})
            g["rows"].setdefault((qL, s1), dL)
            g["cols"].setdefault((s2, qR), dR)
            g["blk"].append(((qL, s1), (s2, qR), dL, dR, off))
        svds, allsv = {}, []
        for qm, g in sorted(groups.items()):    # lexicographic sector order: the tie-break rule of the truncation
            ro, co, o = {}, {}, 0
            for key in sorted(g["rows"]):
                ro[key] = o; o += g["rows"][key]
            nr, o = o, 0
            for key in sorted(g["cols"]):
                co[key] = o; o += g["cols"][key]
            M = torch.zeros((nr, o), dtype=torch.float64, device=d.device)
            for (rk, ck, dL, dR, off) in g["blk"]:
                M[ro[rk]:ro[rk] + dL, co[ck]:co[ck] + dR] = x[off:off + dL * dR].view(dL, dR)
            U, S, Vh = torch.linalg.svd(M, full_matrices=False)
            svds[qm] = (U, S, Vh, ro, co, g)
            allsv += [(float(s), qm) for s in S.cpu().numpy()]
        allsv.sort(key=lambda t: -t[0])
        kept = {}
        for s, qm in allsv[:self.D]:
            if s > 1e-14:
                kept[qm] = kept.get(qm, 0) + 1
        self.trunc.append(float(sum(s * s for s, _ in allsv[self.D:])))
        t0 = self._tick("SVD", t0)
        new_sec = {qm: c for qm, c in kept.items()}
        self.sectors[k] = new_sec
        d.mps_update_bond(k, new_sec)
        if direction == 0:
            A, C = {}, {}
            for qm, c in kept.items():
                U, S, Vh, ro, co, g = svds[qm]
                for (qL, s1), dL in g["rows"].items():
                    A[self._lkey(qL, s1, qm)] = U[ro[(qL, s1)]:ro[(qL, s1)] + dL, :c].cpu().numpy()
                C[qm] = (S[:c, None] * Vh[:c, :], co, g["cols"])
            self.left[k] = A
            self._set_site(k, 0, A)
            if k + 2 > self.L:
                raise ValueError("already at the right end")
            R = self.right.pop(k + 2)
            d.renormalize(0)
            self.k = k + 1
            t0 = self._tick("Ren+Tables", t0)
            layout2, n2 = self._layout()
            y = torch.zeros(n2, dtype=torch.float64, device=d.device)
            for (qL, s1, s2, qR, dL, dR, off, qmid2) in layout2:   # qL = old q_mid, s1 = old s2, s2 = site k+2
                if qL not in C:
                    continue
                Cm, co, cols = C[qL]
                rk = self._lkey(qmid2, s2, qR)
                if (s1, qmid2) not in co or rk not in R:
                    continue
                c0 = co[(s1, qmid2)]
                w = cols[(s1, qmid2)]
                Rb = torch.from_numpy(np.ascontiguousarray(R[rk])).to(d.device)
                y[off:off + dL * dR] = (Cm[:, c0:c0 + w] @ Rb).reshape(-1)
        else:
            B, C = {}, {}
            for qm, c in kept.items():
                U, S, Vh, ro, co, g = svds[qm]
                for (s2, qR), dR in g["cols"].items():
                    B[self._lkey(qm, s2, qR)] = Vh[:c, co[(s2, qR)]:co[(s2, qR)] + dR].cpu().numpy()
                C[qm] = (U[:, :c] * S[None, :c], ro, g["rows"])
            self.right[k + 1] = B
            self._set_site(k + 1, 1, B)
            if k - 1 < 1:
                raise ValueError("already at the left end")
            Lt = self.left.pop(k - 1)
            d.renormalize(1)
            self.k = k - 1
            t0 = self._tick("Ren+Tables", t0)
            layout2, n2 = self._layout()
            y = torch.zeros(n2, dtype=torch.float64, device=d.device)
            for (qL, s1, s2, qR, dL, dR, off, qk1) in layout2:   # s2 = old s1 (site k), qR = old q_mid, qk1 = bond k-1
                if qR not in C:
                    continue
                Cm, ro, rows = C[qR]
                lk = self._lkey(qL, s1, qk1)
                if (qk1, s2) not in ro or lk not in Lt:
                    continue
                r0 = ro[(qk1, s2)]
                h = rows[(qk1, s2)]
                Lb = torch.from_numpy(np.ascontiguousarray(Lt[lk])).to(d.device)
                y[off:off + dL * dR] = (Lb @ Cm[r0:r0 + h, :]).reshape(-1)
        nrm = torch.linalg.norm(y)
        self.guess = y / nrm if float(nrm) > 0 else None
        self._tick("StVec", t0)
        return E

    def sweep(self, nsweeps=2, **kw):
        """Right to the last bond, back to the first, ... starting from the current bond.  Returns energies."""
        out = []
        for _ in range(nsweeps):
            while self.k + 2 <= self.L:
                out.append(self.step(0, **kw))
            while self.k - 1 >= 1:
                out.append(self.step(1, **kw))
        out.append(self.step(None, **kw))
        return out

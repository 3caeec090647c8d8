"""ORACLE (test infrastructure, CPU only): the truncation step of a two-site DMRG micro-iteration.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs may import this file;
it shares no code with the CUDA path and never calls it.

What it computes (PAPER.md:55 "keeping only the D largest singular values in SVD"; Fig. 1, :63): the optimised
two-site wavefunction is reshaped to Psi[(a s_k), (s_{k+1} b)], which is block diagonal in the sectors of bond k;
each sector block gets a dense SVD; the D largest singular values OVER ALL sectors are kept (values <= 1e-14 never;
equal values: the sector that comes first in lexicographic order first, reading R23); the discarded weight
is the sum of the squares of the rest.  Returns the kept dimension per sector, the discarded weight and the kept
singular values — the quantities a sweep driver must reproduce exactly (dimensions) or to rounding (weight).
"""
from __future__ import annotations

import numpy as np

from .dmrg import SITE_Q


def sector_matrices(psi_blocks, v):
    """dict q_k -> dense Psi_q[(a s_k), (s_{k+1} b)] with rows ordered by (q_L, s_k), columns by (s_{k+1}, q_R)."""
    blocks, o = {}, 0
    for (qL, s1, s2, qR, dL, dR) in psi_blocks:
        q = (qL[0] + SITE_Q[s1][0], qL[1] + SITE_Q[s1][1])
        blocks.setdefault(q, []).append(((qL, s1), (s2, qR), np.asarray(v[o:o + dL * dR]).reshape(dL, dR)))
        o += dL * dR
    out = {}
    for q, lst in blocks.items():
        rows, cols = {}, {}
        for rk, ck, m in lst:
            rows.setdefault(rk, m.shape[0]); cols.setdefault(ck, m.shape[1])
        ro, co, n = {}, {}, 0
        for key in sorted(rows):
            ro[key] = n; n += rows[key]
        nr, n = n, 0
        for key in sorted(cols):
            co[key] = n; n += cols[key]
        M = np.zeros((nr, n))
        for rk, ck, m in lst:
            M[ro[rk]:ro[rk] + m.shape[0], co[ck]:co[ck] + m.shape[1]] = m
        out[q] = M
    return out


def truncate(psi_blocks, v, D):
    """(kept: dict q_k -> dimension, discarded weight, kept singular values sorted descending)."""
    sv = []
    for q, M in sorted(sector_matrices(psi_blocks, v).items()):
        for s in np.linalg.svd(M, compute_uv=False):
            sv.append((float(s), q))
    sv.sort(key=lambda t: -t[0])          # stable: equal values keep the lexicographic sector order
    kept = {}
    for s, q in sv[:D]:
        if s > 1e-14:
            kept[q] = kept.get(q, 0) + 1
    weight = float(sum(s * s for s, _ in sv[D:]))
    return kept, weight, np.array([s for s, _ in sv[:D] if s > 1e-14])

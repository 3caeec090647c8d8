"""Mode-optimisation micro-iteration (Sec. II.B, Fig. 1 :63) driven through the C ABI.

i)   the eigenstate of H_eff at bond (k, k+1): `dmrg_davidson`;
ii)  the two-site orbital rotation u^(k,k+1) that minimises the half-Renyi block entropy S_1/2(rho_{1..k})
     (PAPER.md:75): every trial angle is one `dmrg_two_site_gate` + one `dmrg_bond_entropy` (an SVD per bond sector "in
     every cycle") on the device; the search over theta in [-pi/2, pi/2) is a scan followed by a
     golden-section refinement (reading R21) — control flow only;
iii) the wavefunction is rotated (`dmrg_two_site_gate`) and the integrals t, v with it (`dmrg_rotate_integrals`).
theta = pi/2 is the swap gate of PAPER.md:89 (mode exchange, up to signs), `swap=True` skips the search.

Only argument marshalling and control flow here; the numerical steps run in the library's kernels.
"""
from __future__ import annotations

import math

from .binding import rotation_gate


def optimise_rotation(d, psi, ngrid=24, iters=40):
    """(theta, S_1/2 at theta = 0, S_1/2 at theta) for the two-site wavefunction psi (CUDA tensor) of context d."""
    tmp = psi.new_empty(psi.shape)

    def cost(theta):
        d.two_site_gate(rotation_gate(theta), psi, tmp)
        return d.bond_entropy(tmp)[0]
    s0 = d.bond_entropy(psi)[0]
    grid = [-0.5 * math.pi + math.pi * i / ngrid for i in range(ngrid)]
    vals = [cost(t) for t in grid]
    i = min(range(ngrid), key=lambda j: vals[j])
    h = math.pi / ngrid
    a, b = grid[i] - h, grid[i] + h
    gr = 0.5 * (math.sqrt(5.0) - 1.0)
    c, e = b - gr * (b - a), a + gr * (b - a)
    fc, fe = cost(c), cost(e)
    for _ in range(iters):
        if fc < fe:
            b, e, fe = e, c, fc
            c = b - gr * (b - a)
            fc = cost(c)
        else:
            a, c, fc = c, e, fe
            e = a + gr * (b - a)
            fe = cost(e)
    t = 0.5 * (a + b)
    ft = cost(t)
    if vals[i] < ft:
        t, ft = grid[i], vals[i]
    return t, s0, ft


def micro_iteration(d, psi, k, tol=1e-8, max_iter=200, max_basis=20, swap=False):
    """One micro-iteration at the prepared bond (k, k+1).  psi: start vector (CUDA tensor), overwritten by the rotated
    eigenstate.  Returns dict(energy, theta, S_before, S_after).  The context's integrals are rotated: its
    environments are invalid afterwards (`env_build` again, with site tensors in the rotated modes)."""
    energy, iters, resid = d.davidson(psi, tol=tol, max_iter=max_iter, max_basis=max_basis)
    if swap:
        theta, s0 = 0.5 * math.pi, d.bond_entropy(psi)[0]
        rot = d.two_site_gate(rotation_gate(theta), psi)
        s1 = d.bond_entropy(rot)[0]
    else:
        theta, s0, s1 = optimise_rotation(d, psi)
        rot = d.two_site_gate(rotation_gate(theta), psi)
    psi.copy_(rot)
    d.rotate_integrals(k, theta)
    return {"energy": energy, "davidson_applies": iters, "resid": resid, "theta": theta, "S_before": s0, "S_after": s1}

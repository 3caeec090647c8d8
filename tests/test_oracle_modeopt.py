"""Pins for oracle/modeopt.py (no GPU): integral rotation, the sign / index convention of the two-site orbital rotation,
the two-site gate against the determinant-space rotation, and closed forms of the half-Renyi entropy."""
import numpy as np
from scipy.linalg import expm

import helpers
from oracle import fci, modeopt
from paper_2501_18263_b200 import inputs
from test_oracle_dmrg import _herm_V


def _kappa_fci(L, k, nu, nd):
    """kappa = sum_s (c+_{k+1,s} c_{k,s} - c+_{k,s} c_{k+1,s}) in the determinant space, from its definition."""
    K1 = np.zeros((L, L))
    K1[k, k - 1] = 1.0       # orbital index k = site k+1
    K1[k - 1, k] = -1.0
    K, _ = fci.fci_hamiltonian(K1, np.zeros((L,) * 4), nu, nd)
    return K


def test_rotated_integrals_keep_the_fci_spectrum_and_fix_the_convention():
    rng = np.random.default_rng(3)
    L, nu, nd, k, theta = 5, 2, 2, 3, 0.37
    T = rng.normal(size=(L, L)); T = T + T.T
    V = _herm_V(rng, L)
    Tn, Vn = modeopt.rotate_integrals(T, V, k, theta)
    H, _ = fci.fci_hamiltonian(T, V, nu, nd)
    Hn, _ = fci.fci_hamiltonian(Tn, Vn, nu, nd)
    ev, vec = np.linalg.eigh(H)
    assert np.abs(np.linalg.eigvalsh(Hn) - ev).max() < 1e-11                 # same operator, other modes
    # coefficients in the rotated modes: psi~ = exp(-theta K) psi; it must be the ground vector of the rotated H
    K = _kappa_fci(L, k, nu, nd)
    assert np.abs(K + K.T).max() < 1e-14
    psi_t = expm(-theta * K) @ vec[:, 0]
    assert np.linalg.norm(Hn @ psi_t - ev[0] * psi_t) < 1e-10
    # the opposite sign of theta is NOT a ground vector (the pin fails for a wrong convention)
    psi_w = expm(theta * K) @ vec[:, 0]
    assert np.linalg.norm(Hn @ psi_w - ev[0] * psi_w) > 1e-3
    # H~ = R H R^T as matrices in the determinant space
    R = expm(-theta * K)
    assert np.abs(Hn - R @ H @ R.T).max() < 1e-10


def test_two_site_gate_equals_the_determinant_space_rotation():
    """Through the explicit embedding P of the block states: P (G psi) = exp(-theta K) (P psi), left blocks of odd and
    even particle number included (no Jordan-Wigner string between neighbouring sites)."""
    for (L, nu, nd, k) in ((5, 2, 2, 2), (6, 3, 2, 4), (5, 3, 2, 1)):
        mps = inputs.make_mps(L, nu, nd, 10 ** 9, k, seed=4)
        pb = inputs.psi_blocks(mps)
        P, _ = helpers.embedding(mps, pb)
        rng = np.random.default_rng(L + k)
        v = rng.normal(size=P.shape[1])
        theta = 0.61
        G = modeopt.two_site_rotation(theta)
        lhs = P @ modeopt.apply_gate(pb, v, G)
        rhs = expm(-theta * _kappa_fci(L, k, nu, nd)) @ (P @ v)
        assert np.abs(lhs - rhs).max() < 1e-13
        assert np.abs(G @ G.T - np.eye(16)).max() < 1e-14


def test_half_renyi_closed_forms():
    # two sites, one up and one down electron, trivial blocks: psi over (s1, s2)
    mps = inputs.make_mps(2, 1, 1, 10 ** 9, 1, seed=1)
    pb = inputs.psi_blocks(mps)
    idx = {(b[1], b[2]): i for i, b in enumerate(pb)}
    assert all(b[4] == 1 and b[5] == 1 for b in pb)
    v = np.zeros(len(pb))
    v[idx[(2, 1)]] = 1.0                                            # |up, dn>: product state
    assert abs(modeopt.half_renyi(pb, v)) < 1e-14
    v[idx[(1, 2)]] = -1.0                                           # (|up,dn> - |dn,up>): Schmidt values (1/sqrt2, 1/sqrt2)
    s_half, s_vn = modeopt.entropies(modeopt.bond_spectrum(pb, v))
    assert abs(s_half - np.log(2.0)) < 1e-14 and abs(s_vn - np.log(2.0)) < 1e-14
    # the bonding orbital doubly occupied, (c+_1 + c+_2)_up (c+_1 + c+_2)_dn |0> / 2, is entangled in the site modes and a
    # product state in the rotated modes: theta = pi/4 brings the entropy to zero, and the optimiser finds it
    w = np.zeros(len(pb))
    for key, c in (((3, 0), 0.5), ((0, 3), 0.5), ((2, 1), 0.5), ((1, 2), -0.5)):    # c+_2u c+_1d |0> = -|dn, up>
        w[idx[key]] = c
    s0 = modeopt.half_renyi(pb, w)
    assert s0 > 0.5
    cost = lambda t: modeopt.half_renyi(pb, modeopt.apply_gate(pb, w, modeopt.two_site_rotation(t)))
    theta, smin = modeopt.optimise_theta(cost)
    assert smin < 1e-10 and abs(abs(theta) - np.pi / 4) < 1e-5

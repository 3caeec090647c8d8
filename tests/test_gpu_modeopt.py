"""GPU parity of the mode-optimisation micro-iteration calls (Sec. II.B, Fig. 1) against oracle/modeopt.py
(`-m gpu`): two-site gate, block entropies, rotated integrals, the search for the optimal rotation, one whole
micro-iteration."""
import numpy as np
import pytest

from oracle import dmrg as odmrg
from oracle import fci, modeopt as omo
from paper_2501_18263_b200 import inputs

pytestmark = pytest.mark.gpu


def _ctx(T, V, mps):
    import torch
    from paper_2501_18263_b200.binding import DMRG
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    d = DMRG(mps.L, mps.n_up, mps.n_dn)
    d.setup(T, V, mps)
    return d


def _gpu(v):
    import torch
    return torch.from_numpy(np.ascontiguousarray(v)).cuda()


@pytest.mark.parametrize("L,nu,nd,k,D", [(8, 4, 4, 4, 40), (10, 5, 4, 3, 64), (8, 3, 4, 7, 30), (20, 10, 10, 10, 256)])
def test_gate_and_entropy_match_the_oracle(L, nu, nd, k, D):
    from paper_2501_18263_b200.binding import rotation_gate
    T, V = inputs.make_integrals(L, 50 + L)
    mps = inputs.make_mps(L, nu, nd, D, k, seed=8)
    pb = inputs.psi_blocks(mps)
    d = _ctx(T, V, mps)
    rng = np.random.default_rng(k)
    v = rng.normal(size=d.psi_size())
    for theta in (0.4, -1.1, 0.5 * np.pi):
        G = rotation_gate(theta)
        assert np.abs(G - omo.two_site_rotation(theta)).max() <= 1e-14
        got = d.two_site_gate(G, _gpu(v)).cpu().numpy()
        ref = omo.apply_gate(pb, v, omo.two_site_rotation(theta))
        assert np.abs(got - ref).max() <= 1e-14 * max(1.0, np.abs(ref).max())
        assert abs(np.linalg.norm(got) - np.linalg.norm(v)) <= 1e-12 * np.linalg.norm(v)
        s_half, s_vn, sig = d.bond_entropy(_gpu(ref), spectrum=True)
        ref_sig = omo.bond_spectrum(pb, ref)
        assert len(sig) == len(ref_sig)
        assert np.abs(np.sort(sig) - np.sort(ref_sig)).max() <= 1e-12 * ref_sig.max()
        r_half, r_vn = omo.entropies(ref_sig)
        assert abs(s_half - r_half) <= 1e-11 and abs(s_vn - r_vn) <= 1e-11
    # a general number-conserving gate (random orthogonal inside every (n_up, n_dn) sector of the pair), and a rejected one
    Q = np.zeros((16, 16))
    secs = {}
    for s in range(16):
        q = (odmrg.SITE_Q[s // 4][0] + odmrg.SITE_Q[s % 4][0], odmrg.SITE_Q[s // 4][1] + odmrg.SITE_Q[s % 4][1])
        secs.setdefault(q, []).append(s)
    for idx in secs.values():
        Q[np.ix_(idx, idx)] = np.linalg.qr(rng.normal(size=(len(idx), len(idx))))[0]
    got = d.two_site_gate(Q, _gpu(v)).cpu().numpy()
    assert np.abs(got - omo.apply_gate(pb, v, Q)).max() <= 1e-14 * np.abs(v).max() * 4
    from paper_2501_18263_b200.binding import DMRGError
    bad = Q.copy(); bad[0, 5] = 0.1
    with pytest.raises(DMRGError, match="conserve"):
        d.two_site_gate(bad, _gpu(v))
    d.close()


def test_rotated_integrals_give_the_rotated_effective_hamiltonian():
    """H~_eff (G psi) = G (H_eff psi): the library's H_eff after dmrg_rotate_integrals + env_build against its own H_eff
    before, and against the oracle's H_eff built from the oracle's rotated integrals (truncated blocks)."""
    L, nu, nd, k, D, theta = 10, 5, 5, 5, 48, 0.73
    T, V = inputs.make_integrals(L, 91)
    mps = inputs.make_mps(L, nu, nd, D, k, seed=2)
    pb = inputs.psi_blocks(mps)
    d = _ctx(T, V, mps)
    v = np.random.default_rng(1).normal(size=d.psi_size())
    hv = d.heff_apply(_gpu(v)).cpu().numpy()
    G = omo.two_site_rotation(theta)
    d.rotate_integrals(k, theta)
    from paper_2501_18263_b200.binding import DMRGError
    with pytest.raises(DMRGError):
        d.heff_apply(_gpu(v))                          # the environments are gone with the old integrals
    d.env_build(k)
    gv = omo.apply_gate(pb, v, G)
    got = d.heff_apply(_gpu(gv)).cpu().numpy()
    ref = omo.apply_gate(pb, hv, G)
    assert np.linalg.norm(got - ref) / np.linalg.norm(ref) <= 1e-11
    Tn, Vn = omo.rotate_integrals(T, V, k, theta)
    orc = odmrg.TwoSiteOracle(Tn, Vn, nu, nd, k, mps.sectors, mps.left, mps.right, pb)
    orc.build_env()
    ref2 = orc.apply(gv)
    assert np.linalg.norm(got - ref2) / np.linalg.norm(ref2) <= 1e-11
    d.close()


def test_micro_iteration_lowers_the_block_entropy_and_keeps_the_energy():
    """One whole micro-iteration (Fig. 1): Davidson, search for u^(k,k+1), rotation of psi and of the integrals.  The
    optimal angle and entropy agree with the oracle's search on the same eigenstate; the rotated state has the same
    energy under the rebuilt H_eff; with untruncated blocks that energy is the FCI ground-state energy."""
    import torch
    from paper_2501_18263_b200 import modeopt
    T, V, mps = inputs.make_config(0)
    pb = inputs.psi_blocks(mps)
    k = mps.k
    d = _ctx(T, V, mps)
    psi = _gpu(inputs.make_psi0(mps, 7))
    res = modeopt.micro_iteration(d, psi, k, tol=1e-10, max_iter=400)
    e_fci = fci.fci_lowest(T, V, mps.n_up, mps.n_dn, 1)[0]
    assert abs(res["energy"] - e_fci) <= 1e-9
    assert res["S_after"] <= res["S_before"] + 1e-12
    # the oracle's search on the unrotated eigenstate: rotate back with the inverse gate
    rot = psi.cpu().numpy()
    x = omo.apply_gate(pb, rot, omo.two_site_rotation(-res["theta"]))
    assert abs(omo.half_renyi(pb, x) - res["S_before"]) <= 1e-10
    cost = lambda t: omo.half_renyi(pb, omo.apply_gate(pb, x, omo.two_site_rotation(t)))
    th_o, s_o = omo.optimise_theta(cost)
    assert abs(s_o - res["S_after"]) <= 1e-8
    assert abs(cost(res["theta"]) - res["S_after"]) <= 1e-10
    # energy continuity under the rotated Hamiltonian
    d.env_build(k)
    hx = d.heff_apply(psi)
    e_rot = float(torch.dot(psi, hx) / torch.dot(psi, psi))
    assert abs(e_rot - res["energy"]) <= 1e-9
    assert float(torch.linalg.norm(hx - e_rot * psi)) <= 1e-7
    # the swap gate: theta = pi/2 exchanges the two modes; the spectrum of the cut of the twice-swapped state is the original
    y = d.two_site_gate(modeopt.rotation_gate(0.5 * np.pi), psi)
    z = d.two_site_gate(modeopt.rotation_gate(0.5 * np.pi), y)
    assert float(torch.linalg.norm(torch.abs(z) - torch.abs(psi))) <= 1e-12 * float(torch.linalg.norm(psi))
    d.close()

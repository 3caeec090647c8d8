"""GPU parity of the SU(2)-adapted path against the SU(2) oracle (expansion to U(1) by
Clebsch-Gordan coefficients, oracle/su2.py) on the same seeded reduced MPS; `-m gpu`.

Tolerances as for U(1): rel-L2 <= 1e-11 on H_eff.psi, |dE| <= 1e-9 Eh on Davidson energies."""
import numpy as np
import pytest

from helpers import assert_blocks_close
from oracle import dmrg as odmrg
from oracle import fci, su2
from paper_2501_18263_b200 import inputs

pytestmark = pytest.mark.gpu
REL_L2 = 1e-11


def _gpu(T, V, mps, **kw):
    import torch
    from paper_2501_18263_b200.binding import DMRG
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    d = DMRG(mps.L, mps.N // 2, mps.N // 2, su2=True, **kw)
    d.setup(T, V, mps)
    return d


def _oracle(T, V, mps):
    orc = su2.SU2TwoSiteOracle(T, V, mps, inputs.psi_blocks_su2(mps))
    orc.build_env()
    return orc


def _apply_gpu(d, v):
    import torch
    return d.heff_apply(torch.from_numpy(np.ascontiguousarray(v)).cuda()).cpu().numpy()


def _rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def _general_integrals(L, seed):
    rng = np.random.default_rng(seed)
    T = rng.normal(size=(L, L)); T = T + T.T
    V = rng.normal(size=(L,) * 4); V = V + V.transpose(2, 3, 0, 1)
    return T, V


@pytest.mark.parametrize("L,N,k,D", [
    (6, 6, 3, 10 ** 9),            # untruncated
    (6, 6, 1, 8), (6, 6, 5, 8),    # chain ends (empty blocks)
    (6, 4, 2, 7), (7, 8, 4, 12),   # other fillings, ragged sectors
    (8, 8, 4, 30),
])
def test_su2_apply_and_layout(L, N, k, D):
    T, V = _general_integrals(L, 300 + L + k)
    mps = inputs.make_mps_su2(L, N, D, k, seed=5)
    orc = _oracle(T, V, mps)
    d = _gpu(T, V, mps)
    blocks, n = d.psi_layout()
    ref_blocks = inputs.psi_blocks_su2(mps)
    assert n == orc.psi_size()
    assert [(b.qL_up, b.qL_dn, b.s1, b.twoS_mid, b.s2, b.qR_up, b.qR_dn, b.dL, b.dR) for b in blocks] == \
           [(q[0][0], q[0][1], q[1], q[2][1], q[3], q[4][0], q[4][1], q[5], q[6]) for q in ref_blocks]
    rng = np.random.default_rng(1)
    for _ in range(2):
        v = rng.normal(size=n)
        assert_blocks_close(_apply_gpu(d, v), orc.apply(v), [q[5] * q[6] for q in ref_blocks], REL_L2)
    d.close()


def test_su2_diag_and_davidson_reach_the_fci_singlet():
    import torch
    L, N, k = 6, 6, 3
    T, V = inputs.make_integrals(L, 5)
    mps = inputs.make_mps_su2(L, N, 10 ** 9, k, seed=3)
    orc = _oracle(T, V, mps)
    d = _gpu(T, V, mps)
    assert np.abs(d.heff_diag().cpu().numpy() - orc.diag_exact()).max() <= 1e-11
    v0 = inputs.make_psi0_su2(mps, 1)
    x = torch.from_numpy(v0.copy()).cuda()
    E, it, rn = d.davidson(x, tol=1e-10, max_iter=400, max_basis=20)
    assert rn <= 1e-10
    assert abs(E - fci.fci_lowest(T, V, N // 2, N // 2, 1)[0]) <= 1e-9    # the ground state is a singlet here
    xv = x.cpu().numpy()
    assert np.linalg.norm(orc.apply(xv) - E * xv) <= 1e-8
    d.close()


def test_su2_energy_equals_u1_energy_of_the_expanded_state():
    """R19: the SU(2) run and a U(1) run on the CG-expanded MPS (equal effective bond) agree: expand(H psi) on
    the GPU's U(1) path == H expand(psi), and the Davidson energies coincide."""
    import torch
    from paper_2501_18263_b200.binding import DMRG
    L, N, k, D = 8, 8, 4, 24
    T, V = inputs.make_integrals(L, 77)
    mps = inputs.make_mps_su2(L, N, D, k, seed=9)
    orc = _oracle(T, V, mps)            # used for its expansion map and U(1) MPS only
    d2 = _gpu(T, V, mps)
    sec_u1, left_u1, right_u1, _ = su2.expand_mps(mps)
    u1 = inputs.MPSInput(L=L, k=k, n_up=N // 2, n_dn=N // 2, sectors=sec_u1, left=left_u1, right=right_u1)
    d1 = DMRG(L, N // 2, N // 2)
    d1.setup(T, V, u1)
    assert d1.psi_size() == orc.n_u1
    v = np.random.default_rng(2).normal(size=orc.n_red)
    lhs = orc.expand(_apply_gpu(d2, v))
    rhs = _apply_gpu(d1, orc.expand(v))
    assert _rel(lhs, rhs) <= REL_L2
    # The SU(2) eigenpair is an eigenpair of the U(1) effective Hamiltonian at equal effective bond.  (A U(1)
    # Davidson started from the expanded singlet does NOT stay in S = 0: rounding noise seeds S > 0 components
    # and the U(1) space of a truncated MPS may hold a lower non-singlet state, so its energy is only bounded
    # from above by the singlet energy.)
    x2 = torch.from_numpy(inputs.make_psi0_su2(mps, 4)).cuda()
    E2, _, r2 = d2.davidson(x2, tol=1e-9, max_iter=300, max_basis=20)
    assert r2 <= 1e-9
    xe = orc.expand(x2.cpu().numpy())
    assert np.linalg.norm(_apply_gpu(d1, xe) - E2 * xe) <= 1e-8
    x1 = torch.from_numpy(xe.copy()).cuda()
    E1, _, r1 = d1.davidson(x1, tol=1e-9, max_iter=300, max_basis=20)
    assert r1 <= 1e-9 and E1 <= E2 + 1e-9
    d1.close(); d2.close()


def test_su2_renormalize_step_matches_oracle():
    L, N, k, D = 8, 8, 3, 20
    T, V = _general_integrals(L, 19)
    sectors = inputs.su2_bond_sectors(L, N, 0, D)
    a = inputs.make_mps_su2(L, N, D, k, seed=2, sectors=sectors)
    b = inputs.make_mps_su2(L, N, D, k + 1, seed=3, sectors=sectors)
    start = inputs.SU2MPSInput(L=L, k=k, N=N, sectors=sectors, left={i: b.left[i] for i in range(1, k)}, right=a.right)
    d = _gpu(T, V, start)
    d.mps_set_site_su2(k, 0, b.left[k])
    d.renormalize(0)
    m2 = inputs.SU2MPSInput(L=L, k=k + 1, N=N, sectors=sectors, left=b.left,
                            right={i: a.right[i] for i in range(k + 3, L + 1)})
    orc = _oracle(T, V, m2)
    v = np.random.default_rng(4).normal(size=orc.psi_size())
    assert d.psi_size() == orc.psi_size()
    assert _rel(_apply_gpu(d, v), orc.apply(v)) <= REL_L2
    d.close()


def test_su2_medium_size_against_oracle():
    """Several tiles per block and ragged tails: L = 12, 12 electrons, 90 multiplets (U(1)-equivalent ~ 300)."""
    L, N, k, D = 12, 12, 6, 90
    T, V = inputs.make_integrals(L, 123)
    mps = inputs.make_mps_su2(L, N, D, k, seed=11)
    orc = _oracle(T, V, mps)
    d = _gpu(T, V, mps)
    v = inputs.make_psi0_su2(mps, 6)
    assert d.psi_size() == orc.psi_size()
    assert _rel(_apply_gpu(d, v), orc.apply(v)) <= REL_L2
    d.close()


def test_su2_input_errors_are_reported():
    from paper_2501_18263_b200.binding import DMRG, DMRGError
    L, N = 6, 6
    T, V = _general_integrals(L, 1)
    with pytest.raises(DMRGError):
        DMRG(L, 4, 2, su2=True)                       # SU(2) contexts are total-spin-0 only
    d = DMRG(L, 3, 3, su2=True)
    d.load_integrals(T, V)
    mps = inputs.make_mps_su2(L, N, 8, 3, seed=1)
    d.mps_set_sectors(mps.sectors)
    with pytest.raises(DMRGError, match="dmrg_mps_set_site_su2"):
        d.mps_set_site(1, 0, {((0, 0), 0): np.ones((1, 1))})       # U(1) entry point on an SU(2) context
    # a q_out that is not a spin coupling of q_in with the site multiplet
    good = mps.left[2]
    key = next(k for k in good if k[1] == 1)
    bad = dict(good)
    blk = bad.pop(key)
    wrong = next(q for q in mps.sectors[2] if q not in inputs.su2_couplings(key[0], 1) and mps.sectors[2][q] == blk.shape[1])\
        if any(q not in inputs.su2_couplings(key[0], 1) and mps.sectors[2][q] == blk.shape[1] for q in mps.sectors[2]) else None
    if wrong is not None:
        bad[(key[0], 1, wrong)] = blk
        with pytest.raises(DMRGError, match="coupling"):
            d.mps_set_site_su2(2, 0, bad)
    scaled = {k: v * 1.01 for k, v in good.items()}
    d.mps_set_site_su2(1, 0, mps.left[1])
    with pytest.raises(DMRGError, match="left-canonical"):
        d.mps_set_site_su2(2, 0, scaled)
    with pytest.raises(DMRGError):
        d.mps_update_bond(0, {(0, 0): 1})             # bonds 0 and L are fixed
    d.close()

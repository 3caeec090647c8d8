"""The library's truncation step (dmrg_truncate_bond, dmrg_start_vector, dmrg_bond_sectors; Fig. 1 :63)
against oracle/sweep.py and against gauge-independent properties of the truncated state (`-m gpu`)."""
import numpy as np
import pytest

from oracle import sweep as osweep
from paper_2501_18263_b200 import inputs

pytestmark = pytest.mark.gpu


def _ctx(L, nu, nd, D, k, seed):
    import torch
    from paper_2501_18263_b200.binding import DMRG
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    T, V = inputs.make_integrals(L, 40 + L)
    mps = inputs.make_mps(L, nu, nd, D, k, seed=seed)
    d = DMRG(L, nu, nd)
    d.setup(T, V, mps)
    return d, mps


def _truncated_state(pb, v, kept):
    """P_kept Psi in the old layout, from numpy SVDs: per sector the best rank-c approximation (independent of the
    sign / rotation freedom of the singular vectors as long as the kept values are separated from the dropped ones)."""
    mats = osweep.sector_matrices(pb, v)
    approx = {}
    for q, M in mats.items():
        c = kept.get(q, 0)
        U, S, Vh = np.linalg.svd(M, full_matrices=False)
        approx[q] = (U[:, :c] * S[:c]) @ Vh[:c, :]
    out = np.zeros_like(v)
    # scatter back with the oracle's own row / column order
    blocks, o = {}, 0
    for (qL, s1, s2, qR, dL, dR) in pb:
        q = (qL[0] + inputs.SITE_Q[s1][0], qL[1] + inputs.SITE_Q[s1][1])
        blocks.setdefault(q, []).append(((qL, s1), (s2, qR), dL, dR, o))
        o += dL * dR
    for q, lst in blocks.items():
        rows, cols = {}, {}
        for rk, ck, dL, dR, _ in lst:
            rows.setdefault(rk, dL); cols.setdefault(ck, dR)
        ro, co, n = {}, {}, 0
        for key in sorted(rows):
            ro[key] = n; n += rows[key]
        n = 0
        for key in sorted(cols):
            co[key] = n; n += cols[key]
        for rk, ck, dL, dR, off in lst:
            out[off:off + dL * dR] = approx[q][ro[rk]:ro[rk] + dL, co[ck]:co[ck] + dR].ravel()
    return out


@pytest.mark.parametrize("L,nu,nd,k,Dm,D,direction", [(8, 4, 4, 4, 40, 23, 0), (8, 4, 4, 4, 40, 23, 1), (10, 5, 4, 3, 64, 37, 0),
                                                      (10, 5, 4, 6, 64, 50, 1), (8, 3, 4, 6, 30, 10 ** 6, 1), (20, 10, 10, 10, 256, 200, 0)])
def test_truncation_against_the_oracle_and_energy_of_the_truncated_state(L, nu, nd, k, Dm, D, direction):
    import torch
    d, mps = _ctx(L, nu, nd, Dm, k, seed=6)
    pb = inputs.psi_blocks(mps)
    rng = np.random.default_rng(L + k + direction)
    # a wavefunction with a decaying spectrum: a few Lanczos-like applications of H_eff to a random vector
    x = torch.from_numpy(rng.normal(size=d.psi_size())).cuda()
    for _ in range(3):
        x = d.heff_apply(x) - 30.0 * x
        x = x / torch.linalg.norm(x)
    v = x.cpu().numpy()
    kept, weight, sig = osweep.truncate(pb, v, D)
    # the truncated state and its energy under the OLD effective Hamiltonian
    vt = _truncated_state(pb, v, kept)
    xt = torch.from_numpy(vt).cuda()
    e_old = float(torch.dot(xt, d.heff_apply(xt)) / torch.dot(xt, xt))
    w, nk = d.truncate_bond(x, direction, D)
    assert d.bond_sectors(k) == kept                                   # exactly
    assert nk == sum(kept.values()) == len(sig)
    assert abs(w - weight) <= 1e-13 * max(1.0, weight)
    assert abs(w + float(np.sum(sig ** 2)) - 1.0) <= 1e-12           # kept + discarded = |psi|^2
    d.renormalize(direction)
    y = d.start_vector()
    # the same state in the new basis: same norm, same energy under the NEW effective Hamiltonian (this fails for a
    # site tensor that is not the isometry of the kept singular vectors, or a wrong transformation)
    assert abs(float(torch.dot(y, y)) - float(np.sum(sig ** 2))) <= 1e-12
    e_new = float(torch.dot(y, d.heff_apply(y)) / torch.dot(y, y))
    assert abs(e_new - e_old) <= 1e-10 * max(1.0, abs(e_old)), (e_new, e_old)
    # calls out of order are refused
    from paper_2501_18263_b200.binding import DMRGError
    d.renormalize(1 - direction)
    with pytest.raises(DMRGError, match="start_vector"):
        d.start_vector()
    d.close()


def test_sectors_larger_than_shared_memory_take_the_global_memory_path():
    import torch
    L, nu, nd, k, Dm, D = 12, 6, 6, 6, 1024, 600
    d, mps = _ctx(L, nu, nd, Dm, k, seed=3)
    pb = inputs.psi_blocks(mps)
    mats = osweep.sector_matrices(pb, np.zeros(d.psi_size()))
    assert max(m.shape[0] * (m.shape[1] + 1) * 8 for m in mats.values()) > 220 * 1024
    x = torch.from_numpy(np.random.default_rng(1).normal(size=d.psi_size())).cuda()
    x = d.heff_apply(x) - 30.0 * x
    x = x / torch.linalg.norm(x)
    kept, weight, sig = osweep.truncate(pb, x.cpu().numpy(), D)
    w, nk = d.truncate_bond(x, 0, D)
    assert d.bond_sectors(k) == kept and nk == len(sig)
    assert abs(w - weight) <= 1e-12 * max(1.0, weight)
    d.renormalize(0)
    y = d.start_vector()
    assert abs(float(torch.dot(y, y)) - float(np.sum(sig ** 2))) <= 1e-11
    d.close()


def test_native_and_torch_drivers_give_the_same_sweep():
    """Two truncated sweeps with the library's truncation step and with the torch code of sweep.py: the same energies
    (gauge-independent) and the same kept sectors at every step."""
    from paper_2501_18263_b200.binding import DMRG
    from paper_2501_18263_b200.sweep import TwoSiteSweep
    L, nu, nd, D = 10, 5, 5, 32
    T, V = inputs.make_integrals(L, 77)
    runs = []
    for native in (True, False):
        mps = inputs.make_mps(L, nu, nd, D, 1, seed=9)
        d = DMRG(L, nu, nd)
        sw = TwoSiteSweep(d, T, V, mps, D, native=native)
        assert sw.native == native
        es = sw.sweep(nsweeps=2, tol=1e-10, max_iter=300, max_basis=20)
        runs.append((es, [dict(s) for s in sw.sectors], list(sw.trunc)))
        d.close()
    (e0, s0, t0), (e1, s1, t1) = runs
    assert len(e0) == len(e1)
    assert max(abs(a - b) for a, b in zip(e0, e1)) <= 1e-8
    assert s0 == s1
    assert max(abs(a - b) for a, b in zip(t0, t1)) <= 1e-10

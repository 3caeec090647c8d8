"""Two-site DMRG sweeps through the library (Davidson + renormalisation + environment cache) with the SVD
truncation done by the driver in paper_2501_18263_b200/sweep.py.  Pins: brute-force FCI
(oracle/fci.py) and the variational principle.  `-m gpu`."""
import numpy as np
import pytest

from oracle import fci
from paper_2501_18263_b200 import inputs

pytestmark = pytest.mark.gpu


def _sweeper(L, nu, nd, D, seed, k0=1):
    import torch
    from paper_2501_18263_b200.binding import DMRG
    from paper_2501_18263_b200.sweep import TwoSiteSweep
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    T, V = inputs.make_integrals(L, seed)
    mps = inputs.make_mps(L, nu, nd, D, k0, seed=seed)
    d = DMRG(L, nu, nd)
    return TwoSiteSweep(d, T, V, mps, D), T, V


def test_untruncated_sweep_gives_fci_at_every_bond():
    """Nothing is discarded (D above every Schmidt rank): after the first micro-iteration, whose random right
    environment is still incomplete, every bond reproduces the FCI energy."""
    sw, T, V = _sweeper(6, 3, 3, 10 ** 9, 21)
    e_fci = fci.fci_lowest(T, V, 3, 3, 1)[0]
    es = sw.sweep(nsweeps=1, tol=1e-10, max_iter=300, max_basis=20)
    assert len(es) == 2 * (6 - 2) + 1
    assert es[0] >= e_fci - 1e-9
    assert max(abs(e - e_fci) for e in es[1:]) <= 1e-8
    assert max(sw.trunc) <= 1e-20
    sw.d.close()


def test_truncated_sweeps_are_variational_and_converge():
    L, nu, nd = 8, 4, 4
    sw, T, V = _sweeper(L, nu, nd, 24, 1000)
    e_fci = fci.fci_lowest(T, V, nu, nd, 1)[0]
    runs = []
    for _ in range(3):
        es = sw.sweep(nsweeps=1, tol=1e-9, max_iter=200, max_basis=16)
        assert min(es) >= e_fci - 1e-9            # variational: never below the exact ground state
        runs.append(es)
    # converged: at a given bond the energy is stationary from sweep to sweep (truncation makes the two-site
    # scheme only approximately monotone), and far below the first sweep's start
    for a, b in zip(runs[1], runs[2]):
        assert abs(b - a) <= 1e-3
    assert runs[2][-1] <= runs[0][0] - 1.0
    assert runs[-1][-1] - e_fci <= 2e-2
    assert max(sw.trunc) > 0.0
    sw.d.close()
    # with D above the largest Schmidt rank of an 8-orbital chain (256 at the middle bond) the driver reaches FCI
    sw2, T2, V2 = _sweeper(L, nu, nd, 256, 1000)
    es = sw2.sweep(nsweeps=2, tol=1e-10, max_iter=300, max_basis=20)
    assert abs(es[-1] - e_fci) <= 1e-8
    sw2.d.close()


def test_environment_cache_is_reused_and_invalidated():
    """Moving right then left again re-uses cached blocks; the result equals a fresh build at the same bond."""
    import torch
    from paper_2501_18263_b200.binding import DMRG
    L, nu, nd, D, k = 8, 4, 4, 20, 3
    T, V = inputs.make_integrals(L, 5)
    sectors = inputs.bond_sectors(L, nu, nd, D)
    a = inputs.make_mps(L, nu, nd, D, k, seed=2, sectors=sectors)
    b = inputs.make_mps(L, nu, nd, D, k + 1, seed=2, sectors=sectors)     # same left tensors + site k
    d = DMRG(L, nu, nd)
    d.setup(T, V, a)
    x = torch.from_numpy(inputs.make_psi0(a, 1)).cuda()
    y0 = d.heff_apply(x).clone()
    l0 = d.stats()["total_launches"]
    d.mps_set_site(k, 0, b.left[k])
    d.renormalize(0)
    d.mps_set_site(k + 2, 1, a.right[k + 2])
    d.renormalize(1)                      # back at bond k: left block from the cache, right block re-blocked
    assert torch.allclose(d.heff_apply(x), y0, rtol=0, atol=1e-12 * float(y0.abs().max()))
    # a full rebuild costs many more launches than the two cached steps
    steps = d.stats()["total_launches"] - l0
    d2 = DMRG(L, nu, nd)
    d2.setup(T, V, a)
    assert steps < d2.stats()["total_launches"]
    d.close(); d2.close()


def _sweeper_su2(L, N, D, seed, k0=1):
    import torch
    from paper_2501_18263_b200.binding import DMRG
    from paper_2501_18263_b200.sweep import TwoSiteSweep
    T, V = inputs.make_integrals(L, seed)
    mps = inputs.make_mps_su2(L, N, D, k0, seed=seed)
    d = DMRG(L, N // 2, N // 2, su2=True)
    return TwoSiteSweep(d, T, V, mps, D), T, V


@pytest.mark.parametrize("su2", [False, True])
def test_wavefunction_transformation_keeps_the_energy(su2):
    """Nothing discarded: the transformed start vector at the next bond is the same state, so its Rayleigh
    quotient equals the energy just found (this also fixes the SU(2) re-coupling factor, +1)."""
    import torch
    sw, T, V = (_sweeper_su2(6, 6, 10 ** 9, 5, k0=2) if su2 else _sweeper(6, 3, 3, 10 ** 9, 5, k0=2))
    for direction in (0, 0, 1, 1):
        E = sw.step(direction, tol=1e-10, max_iter=300, max_basis=20)
        g = sw.guess
        assert abs(float(torch.linalg.norm(g)) - 1.0) < 1e-12
        rq = float(torch.dot(g, sw.d.heff_apply(g)))
        assert abs(rq - E) <= 1e-8, (direction, rq, E)
    sw.d.close()


def test_su2_sweep_reaches_the_fci_singlet():
    sw, T, V = _sweeper_su2(6, 6, 10 ** 9, 5)
    e_fci = fci.fci_lowest(T, V, 3, 3, 1)[0]          # singlet ground state for these integrals
    es = sw.sweep(nsweeps=1, tol=1e-10, max_iter=300, max_basis=20)
    assert max(abs(e - e_fci) for e in es[1:]) <= 1e-8
    sw.d.close()
    # L = 8, seed 1000: the FCI ground state of the S_z = 0 sector is a TRIPLET (-7.8244); the lowest singlet is
    # the third FCI eigenvalue.  The SU(2) sweep (S = 0 sector only) must find exactly that one.
    sw2, T2, V2 = _sweeper_su2(8, 8, 10 ** 9, 1000)
    ev = fci.fci_lowest(T2, V2, 4, 4, 5)
    es = sw2.sweep(nsweeps=1, tol=1e-10, max_iter=300, max_basis=20)
    e_singlet = es[-1]
    assert abs(e_singlet - ev[2]) <= 1e-7 and e_singlet > ev[0] + 1e-2
    sw2.d.close()
    # truncated to 20 multiplets: variational with respect to the singlet energy, and close to it
    sw3, _, _ = _sweeper_su2(8, 8, 20, 1000)
    es = sw3.sweep(nsweeps=2, tol=1e-9, max_iter=200, max_basis=16)
    assert min(es[1:]) >= e_singlet - 1e-8
    assert es[-1] - e_singlet <= 1e-2
    sw3.d.close()


@pytest.mark.parametrize("su2", [False, True])
def test_host_tier_of_the_environment_cache(su2):
    """With a device cap of one byte every cached block that is not in use goes to pinned host memory and comes
    back when the sweep returns to it: the energies equal those of the all-on-device run bit for bit, and no block
    is re-blocked (same number of kernel launches)."""
    import torch
    from paper_2501_18263_b200.binding import DMRG
    from paper_2501_18263_b200.sweep import TwoSiteSweep
    L, N, D, seed = 8, 8, 20, 7
    T, V = inputs.make_integrals(L, seed)
    runs = []
    for kw in (dict(), dict(env_cache_bytes=1, env_host_bytes=1 << 30)):
        if su2:
            mps = inputs.make_mps_su2(L, N, D, 1, seed=seed)
            d = DMRG(L, N // 2, N // 2, su2=True, **kw)
        else:
            mps = inputs.make_mps(L, N // 2, N // 2, D, 1, seed=seed)
            d = DMRG(L, N // 2, N // 2, **kw)
        sw = TwoSiteSweep(d, T, V, mps, D)
        es = sw.sweep(nsweeps=2, tol=1e-9, max_iter=200, max_basis=16)
        runs.append((es, d.stats()))
        d.close()
    (e0, s0), (e1, s1) = runs
    assert e0 == e1
    assert s0["env_spills"] == 0 and s0["env_fetches"] == 0
    assert s1["env_spills"] >= L - 3 and s1["env_fetches"] >= L - 3
    assert s1["env_host_bytes"] <= 1 << 30
    assert s1["total_launches"] == s0["total_launches"]


def test_truncation_matches_the_oracle():
    """The kept dimension per bond sector (exactly), the discarded weight and the kept singular values of the driver's
    device SVD against oracle/sweep.py on the same optimised wavefunction; the library's own per-sector Jacobi singular
    values (dmrg_bond_entropy) agree with both."""
    import torch
    from oracle import sweep as osweep
    from paper_2501_18263_b200.binding import DMRG
    from paper_2501_18263_b200.sweep import TwoSiteSweep
    L, nu, nd, D = 10, 5, 5, 28
    T, V = inputs.make_integrals(L, 17)
    mps = inputs.make_mps(L, nu, nd, D, 5, seed=3)
    d = DMRG(L, nu, nd)
    sw = TwoSiteSweep(d, T, V, mps, D)
    for direction in (0, 0, 1):
        pb = [(q[0], q[1], q[2], q[3], q[4], q[5]) for q in sw._layout()[0]]
        k = sw.k
        sw.step(direction, tol=1e-9)
        x = sw.last_psi.cpu().numpy()
        kept, weight, sig = osweep.truncate(pb, x, D)
        assert sw.sectors[k] == kept
        assert abs(sw.trunc[-1] - weight) <= 1e-13 * max(1.0, weight)
        assert sum(kept.values()) <= D
    # the library's Jacobi singular values at the current bond
    pb = [(q[0], q[1], q[2], q[3], q[4], q[5]) for q in sw._layout()[0]]
    y = sw.guess.clone()
    _, _, sig_lib = d.bond_entropy(y, spectrum=True)
    ref = np.concatenate([np.linalg.svd(M, compute_uv=False) for _, M in sorted(osweep.sector_matrices(pb, y.cpu().numpy()).items())])
    assert np.abs(np.sort(sig_lib) - np.sort(ref)).max() <= 1e-12
    d.close()

"""dmrg_bond_entropy_static (include/dmrg_b200.h): the block-entropy call whose device scratch is a file-scope
`static __device__` array, for callers that may not allocate.  Checked against dmrg_bond_entropy, the existing path, on
calls in a row that share the array (`-m gpu`).  Collected last on purpose: the suite runs with `pytest -x`."""
import numpy as np
import pytest

from paper_2501_18263_b200 import inputs

pytestmark = pytest.mark.gpu


def _ctx(L, nu, nd, D, k, seed):
    import torch
    from paper_2501_18263_b200.binding import DMRG
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device")
    T, V = inputs.make_integrals(L, 50 + L)
    mps = inputs.make_mps(L, nu, nd, D, k, seed=seed)
    d = DMRG(L, nu, nd)
    d.setup(T, V, mps)
    return d, mps


def _n_sigma(mps):
    """Number of singular values of the cut between sites k and k+1: sum over bond sectors of min(rows, columns)."""
    rows, cols = {}, {}
    for (qL, s1, s2, qRb, dL, dR) in inputs.psi_blocks(mps):
        q = (qL[0] + inputs.SITE_Q[s1][0], qL[1] + inputs.SITE_Q[s1][1])
        rows.setdefault(q, {})[(qL, s1)] = dL
        cols.setdefault(q, {})[(s2, qRb)] = dR
    return sum(min(sum(rows[q].values()), sum(cols[q].values())) for q in rows)


def _compare(d, psi):
    """One call of each path on the same psi; returns the static path's results."""
    import torch
    ref = d.bond_entropy(psi, spectrum=True)
    torch.cuda.synchronize()
    before = torch.cuda.memory_stats()["allocation.all.allocated"]
    live = len(d._live)
    got = d.bond_entropy_static(psi, spectrum=True)
    assert torch.cuda.memory_stats()["allocation.all.allocated"] == before and len(d._live) == live   # the allocator callbacks were not called
    # same kernels on the same data in the same order: the tolerances of test_gpu_modeopt.py, met with room to spare
    assert len(got[2]) == len(ref[2]) > 0
    assert np.abs(got[2] - ref[2]).max() <= 1e-12 * ref[2].max()
    assert abs(got[0] - ref[0]) <= 1e-11 and abs(got[1] - ref[1]) <= 1e-11
    return got


def test_static_scratch_path_matches_the_allocating_path_on_calls_in_a_row():
    import torch
    big, mps_big = _ctx(20, 10, 10, 256, 10, seed=8)
    small, mps_small = _ctx(8, 4, 4, 40, 4, seed=8)
    assert _n_sigma(mps_small) < _n_sigma(mps_big) <= 2048
    g = torch.Generator(device="cuda").manual_seed(5)
    x = torch.randn(big.psi_size(), dtype=torch.float64, device="cuda", generator=g)
    y = torch.randn(small.psi_size(), dtype=torch.float64, device="cuda", generator=g)
    a1 = _compare(big, x)
    b1 = _compare(small, y)                  # a smaller problem right after a larger one: stale tables and sigma stay unread
    a2 = _compare(big, x)
    b2 = _compare(small, 3.0 * y)            # entropies are those of the normalised state
    assert len(a1[2]) == _n_sigma(mps_big) and len(b1[2]) == _n_sigma(mps_small)
    assert a1[0] == a2[0] and a1[1] == a2[1] and np.array_equal(a1[2], a2[2])      # deterministic, whatever ran in between
    assert abs(b1[0] - b2[0]) <= 1e-12 and abs(b1[1] - b2[1]) <= 1e-12
    assert np.abs(b2[2] - 3.0 * b1[2]).max() <= 1e-12 * b2[2].max()
    # a product state across the cut: one singular value, zero entropy, right after calls that filled the array
    blocks = inputs.psi_blocks(mps_small)
    off = np.cumsum([0] + [b[4] * b[5] for b in blocks])
    i = max(range(len(blocks)), key=lambda j: blocks[j][4] * blocks[j][5])
    dL, dR = blocks[i][4], blocks[i][5]
    rng = np.random.default_rng(2)
    z = np.zeros(small.psi_size())
    z[off[i]:off[i + 1]] = np.outer(rng.normal(size=dL), rng.normal(size=dR)).ravel()
    s_half, s_vn, sig = small.bond_entropy_static(torch.from_numpy(z).cuda(), spectrum=True)
    assert abs(s_half) <= 1e-12 and abs(s_vn) <= 1e-12
    assert abs(np.sort(sig)[-1] - np.linalg.norm(z)) <= 1e-12 * np.linalg.norm(z) and np.sort(sig)[-2] <= 1e-12 * np.linalg.norm(z)
    big.close()
    small.close()


def test_static_scratch_path_rejects_what_does_not_fit():
    import torch
    from paper_2501_18263_b200.binding import DMRGError, STATIC_MAX_SIGMA
    d, mps = _ctx(12, 6, 6, 1024, 6, seed=3)
    assert _n_sigma(mps) > STATIC_MAX_SIGMA
    psi = torch.ones(d.psi_size(), dtype=torch.float64, device="cuda")
    with pytest.raises(DMRGError, match="exceed the static scratch .DMRG_STATIC_MAX_SIGMA = 2048"):
        d.bond_entropy_static(psi)
    d.close()

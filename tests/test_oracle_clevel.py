"""Pins of oracle/clevel.py + oracle/cproducts.c (the oracle's contraction loop in plain C + OpenMP).  CPU only.

The C loop is a drop-in for the numpy loop `TwoSiteOracle._accumulate`; it is pinned (i) against the definition
H_eff = P^T H_FCI P with explicit Fock-space embeddings and a V that has no symmetry beyond Hermiticity, truncated and
untruncated, at both chain ends, (ii) against the numpy loop on BASELINE configs[0] and on a restricted set of output
blocks (the mode bench.py times), (iii) on the shapes that distinguish a wrong transpose: rectangular blocks only."""
import numpy as np
import pytest

import helpers
from oracle import clevel, dmrg, fci, lean
from paper_2501_18263_b200 import inputs


def _oracle(T, V, mps):
    pb = inputs.psi_blocks(mps)
    orc = dmrg.TwoSiteOracle(T, V, mps.n_up, mps.n_dn, mps.k, mps.sectors, mps.left, mps.right, pb)
    orc.build_env()
    return orc, pb


def _apply_c(orc, v):
    psi = orc.unflatten(np.asarray(v, dtype=np.float64))
    out = {kk: np.zeros_like(m) for kk, m in psi.items()}
    clevel.accumulate_c(orc.terms(), psi, out)
    return orc.flatten(out)


@pytest.mark.parametrize("L,nu,nd,k,D", [(5, 2, 1, 2, 6), (5, 3, 2, 3, 10 ** 9), (6, 3, 3, 1, 7), (6, 3, 3, 5, 7),
                                           (6, 2, 3, 4, 8)])
def test_c_loop_equals_projected_fci(L, nu, nd, k, D):
    rng = np.random.default_rng(10 * L + k)
    T = rng.normal(size=(L, L)); T = T + T.T
    V = rng.normal(size=(L,) * 4); V = V + V.transpose(2, 3, 0, 1)        # Hermiticity only
    mps = inputs.make_mps(L, nu, nd, D, k, seed=5)
    orc, pb = _oracle(T, V, mps)
    P, _ = helpers.embedding(mps, pb)
    H, _ = fci.fci_hamiltonian(T, V, nu, nd)
    v = rng.normal(size=P.shape[1])
    ref = P.T @ (H @ (P @ v))
    got = _apply_c(orc, v)
    assert np.linalg.norm(got - ref) / np.linalg.norm(ref) < 1e-13
    # sectors of this case are rectangular (d_L != d_R for most blocks): a transposed operand cannot pass by shape
    assert any(b[4] != b[5] for b in pb)


def test_c_loop_equals_numpy_loop_config0_and_on_chosen_blocks():
    T, V, mps = inputs.make_config(0)
    orc, pb = _oracle(T, V, mps)
    v = inputs.make_psi0(mps, 3)
    ref = orc.apply(v)
    got = _apply_c(orc, v)
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()
    # restricted to a few output blocks, as bench.py's cpu_baseline runs it (lean oracle, same term list)
    L_blk, R_blk = orc.Lblock, orc.Rblock
    lo = lean.LeanTwoSiteOracle(T, V, mps.n_up, mps.n_dn, mps.k, pb, L_blk, R_blk)
    psi = lo.unflatten(v)
    idxs = [0, len(pb) // 3, len(pb) // 2, len(pb) - 1]
    keys = [lo.block_key(i) for i in idxs]
    terms = lo.terms({kk[0] for kk in keys}, {kk[1] for kk in keys})
    out_np = {kk: np.zeros_like(psi[kk]) for kk in keys}
    lo._accumulate(terms, psi, out_np)
    out_c = clevel.ProductList(terms, psi, {kk: np.zeros_like(psi[kk]) for kk in keys}).run()
    full = orc.unflatten(ref)
    for kk in keys:
        assert np.abs(out_c[kk] - out_np[kk]).max() <= 1e-13 * max(1.0, np.abs(out_np[kk]).max())
        assert np.abs(out_c[kk] - full[kk]).max() <= 1e-12 * max(1.0, np.abs(full[kk]).max())


def test_shape_mismatch_is_reported():
    psi = {(("a",), ("b",)): np.ones((2, 3))}

    class Op(dict):
        def parity(self):
            return 0
    XL = Op({(("a",), ("a",)): np.ones((2, 2))})
    XR = Op({(("b",), ("b",)): np.ones((4, 3))})      # maps 3 -> 4 columns, the output block has 3
    with pytest.raises(ValueError):
        clevel.ProductList([(XL, XR, False)], psi, {(("a",), ("b",)): np.zeros((2, 3))}).run()

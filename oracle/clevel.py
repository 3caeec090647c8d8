"""ORACLE (test infrastructure, CPU only): the oracle's contraction loop in plain C + OpenMP (`cproducts.c`).

Only `tests/`, `__graft_entry__` and `bench.py`'s cpu_baseline / `--impl reference` legs may import this file; it
shares no code with the CUDA path and never calls it.

`accumulate_c(terms, psi, out)` does what `dmrg.TwoSiteOracle._accumulate(terms, psi, out)` does -- PAPER.md Eq. (8)
(:109-113), psi'{out} += sum over terms and sectors of  sg * mL psi{in} mR^T  and, for a "+ h.c." term, the transposed
half -- and walks the SAME term list in the same order; only the three-matrix product itself runs in C, as the two
triple loops of its definition (no BLAS).  It is the "plain C + OpenMP" CPU baseline of BASELINE.md §4, timed by
`bench.py` beside the numpy loop; it is not a second derivation of H_eff (the term list and all signs come from
`oracle/dmrg.py`), so its pins are the numpy loop on every product shape (forward and transposed halves, parities) and,
through the whole apply, P^T H_FCI P (tests/test_oracle_clevel.py).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

from .blockops import qnum

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "cproducts.c")
LIB = os.path.join(HERE, "libheff_products.so")


class _Product(C.Structure):
    _fields_ = [("a_off", C.c_longlong), ("x_off", C.c_longlong), ("b_off", C.c_longlong),
                ("a_rows", C.c_int), ("a_cols", C.c_int), ("x_rows", C.c_int), ("x_cols", C.c_int),
                ("b_rows", C.c_int), ("b_cols", C.c_int), ("ta", C.c_int), ("tb", C.c_int), ("sg", C.c_double)]


_PROD_DTYPE = np.dtype([("a_off", "<i8"), ("x_off", "<i8"), ("b_off", "<i8"), ("a_rows", "<i4"), ("a_cols", "<i4"),
                        ("x_rows", "<i4"), ("x_cols", "<i4"), ("b_rows", "<i4"), ("b_cols", "<i4"), ("ta", "<i4"),
                        ("tb", "<i4"), ("sg", "<f8")], align=True)
assert _PROD_DTYPE.itemsize == C.sizeof(_Product)


def build(force=False):
    """gcc -O2 -fopenmp -shared; rebuilt when the source is newer than the library."""
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    # the system gcc first (an environment's $CC may lack libgomp); last resort: without OpenMP (one thread)
    tries = [("/usr/bin/gcc", True), ("gcc", True), (os.environ.get("CC", "cc"), True), ("gcc", False)]
    log = []
    for cc, omp in tries:
        cmd = [cc, "-O2", "-shared", "-fPIC", "-std=c99"] + (["-fopenmp"] if omp else []) + [SRC, "-o", LIB]
        try:
            r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT)
        except OSError as e:
            log.append("%s: %s" % (" ".join(cmd), e))
            continue
        if r.returncode == 0:
            return LIB
        log.append("%s\n%s" % (" ".join(cmd), r.stdout.decode()))
    raise RuntimeError("could not compile oracle/cproducts.c:\n" + "\n".join(log))


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.heff_products.restype = C.c_int
        _lib.heff_products.argtypes = [C.c_void_p, C.c_void_p, C.c_longlong, C.c_void_p, C.c_void_p, C.c_void_p,
                                       C.c_void_p, C.c_void_p]
    return _lib


class ProductList:
    """The products of one H_eff psi on the keys of `out`, gathered once (setup) and executed by `run` (timed)."""

    def __init__(self, terms, psi, out):
        pool, off = [], 0
        where = {}

        def put(m):
            nonlocal off
            key = id(m)
            if key not in where:
                a = np.ascontiguousarray(m, dtype=np.float64)
                where[key] = (off, a.shape[0], a.shape[1])
                pool.append(a.reshape(-1))
                off += a.size
            return where[key]

        self.keys = list(out.keys())
        index = {k: i for i, k in enumerate(self.keys)}
        per_out = [[] for _ in self.keys]
        # ---- the loop nest of TwoSiteOracle._accumulate, recording (mL, x, mR) instead of multiplying ----
        by_left = {}
        for (kl, kr), m in psi.items():
            by_left.setdefault(kl, []).append((kr, m))
        for XL, XR, hc in terms:
            pR = XR.parity()
            r_by_in, r_by_out = {}, {}
            for (kro, kri), mR in XR.items():
                r_by_in.setdefault(kri, []).append((kro, mR))
                if hc:
                    r_by_out.setdefault(kro, []).append((kri, mR))
            for (klo, kli), mL in XL.items():
                sg = -1.0 if (pR and ((qnum(kli[0]) + qnum(kli[1])) & 1)) else 1.0
                for kri, x in by_left.get(kli, ()):      # forward: mL x mR^T
                    for kro, mR in r_by_in.get(kri, ()):
                        o = index.get((klo, kro))
                        if o is not None:
                            per_out[o].append((put(mL), put(x), put(mR), 0, 0, sg))
                if hc:                                   # transposed half: mL^T x mR
                    for kro, x in by_left.get(klo, ()):
                        for kri, mR in r_by_out.get(kro, ()):
                            o = index.get((kli, kri))
                            if o is not None:
                                per_out[o].append((put(mL), put(x), put(mR), 1, 1, sg))
        n = sum(len(p) for p in per_out)
        self.prods = np.zeros(n, dtype=_PROD_DTYPE)
        self.first = np.zeros(len(self.keys) + 1, dtype=np.int64)
        t = 0
        for o, lst in enumerate(per_out):
            self.first[o] = t
            for (a, x, b, ta, tb, sg) in lst:
                self.prods[t] = (a[0], x[0], b[0], a[1], a[2], x[1], x[2], b[1], b[2], ta, tb, sg)
                t += 1
        self.first[len(self.keys)] = t
        self.pool = np.concatenate(pool) if pool else np.zeros(1)
        self.out_rows = np.array([out[k].shape[0] for k in self.keys], dtype=np.int32)
        self.out_cols = np.array([out[k].shape[1] for k in self.keys], dtype=np.int32)
        sizes = self.out_rows.astype(np.int64) * self.out_cols
        self.out_off = np.concatenate([[0], np.cumsum(sizes)[:-1]]).astype(np.int64) if len(sizes) else np.zeros(0, np.int64)
        self.out_size = int(sizes.sum())

    def run(self):
        """Executes the list into a zeroed pool; returns {key: block}."""
        outpool = np.zeros(max(self.out_size, 1))
        rc = _load().heff_products(self.prods.ctypes.data, self.first.ctypes.data, len(self.keys), self.out_off.ctypes.data,
                                   self.out_rows.ctypes.data, self.out_cols.ctypes.data, self.pool.ctypes.data,
                                   outpool.ctypes.data)
        if rc != 0:
            raise ValueError("heff_products: a product's shapes do not fit its output block")
        return {k: outpool[self.out_off[i]:self.out_off[i] + int(self.out_rows[i]) * int(self.out_cols[i])]
                .reshape(int(self.out_rows[i]), int(self.out_cols[i])) for i, k in enumerate(self.keys)}


def accumulate_c(terms, psi, out):
    """Drop-in for TwoSiteOracle._accumulate: out{key} += (H_eff psi){key} for the keys present in `out`."""
    res = ProductList(terms, psi, out).run()
    for k, m in res.items():
        out[k] += m

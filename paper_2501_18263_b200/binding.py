"""Thin ctypes binding of libdmrg_b200.so (include/dmrg_b200.h): argument marshalling only.

Every numerical step runs in the library's CUDA kernels.  PyTorch is used for device memory (the
allocator callbacks hand out torch uint8 tensors) and for the current CUDA stream.  There is no
CPU fallback: importing works without a GPU (so that the symbol table can be checked), but
`DMRG(...)` raises if CUDA or the shared library is missing.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdmrg_b200.so")

EXPORTS = [
    "dmrg_create", "dmrg_destroy", "dmrg_last_error", "dmrg_load_integrals", "dmrg_mps_set_sectors",
    "dmrg_mps_set_site", "dmrg_env_build", "dmrg_renormalize", "dmrg_psi_layout", "dmrg_heff_apply",
    "dmrg_heff_diag", "dmrg_davidson", "dmrg_heff_apply_host", "dmrg_davidson_host", "dmrg_stats",
    "dmrg_env_export", "dmrg_fp64_peak", "dmrg_apply_profile", "dmrg_mps_set_site_su2", "dmrg_su2_f_factor",
    "dmrg_mps_update_bond", "dmrg_set_shard", "dmrg_shard_info", "dmrg_env_export_block", "dmrg_block_flops", "dmrg_dfma_peak",
    "dmrg_two_site_gate", "dmrg_bond_entropy", "dmrg_rotate_integrals", "dmrg_rotation_gate", "dmrg_bond_entropy_static",
    "dmrg_truncate_bond", "dmrg_start_vector", "dmrg_bond_sectors",
]

STATIC_MAX_SIGMA, STATIC_MAX_SECTORS, STATIC_MAX_BLOCKS = 2048, 512, 4096     # include/dmrg_b200.h DMRG_STATIC_MAX_*

REDUCE_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p)
ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_uint64, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class Config(C.Structure):
    _fields_ = [("L", C.c_int32), ("n_up", C.c_int32), ("n_dn", C.c_int32), ("symmetry", C.c_int32),
                ("device", C.c_int32), ("workspace_bytes", C.c_uint64), ("env_cache_bytes", C.c_uint64), ("alloc", ALLOC_FN),
                ("free", FREE_FN), ("alloc_user", C.c_void_p), ("env_host_bytes", C.c_uint64)]


class PsiBlock(C.Structure):
    _fields_ = [("qL_up", C.c_int32), ("qL_dn", C.c_int32), ("s1", C.c_int32), ("s2", C.c_int32),
                ("qR_up", C.c_int32), ("qR_dn", C.c_int32), ("dL", C.c_int32), ("dR", C.c_int32),
                ("off", C.c_int64), ("twoS_mid", C.c_int32), ("pad_", C.c_int32)]


class Stats(C.Structure):
    _fields_ = [("n_terms", C.c_int64), ("n_tasks", C.c_int64), ("n_groups", C.c_int64),
                ("flops_apply", C.c_double), ("flops_executed", C.c_double), ("bytes_unique", C.c_double),
                ("bytes_intermediate", C.c_double), ("psi_size", C.c_int64), ("op_bytes_left", C.c_int64),
                ("op_bytes_right", C.c_int64), ("n_chunks", C.c_int32), ("launches_per_apply", C.c_int32),
                ("last_build_ms", C.c_double), ("flops_renorm", C.c_double), ("total_launches", C.c_int64),
                ("renorm_ms", C.c_double), ("flops_shared", C.c_double), ("env_spills", C.c_int64),
                ("env_fetches", C.c_int64), ("env_host_bytes", C.c_double), ("env_device_bytes", C.c_double)]

    def as_dict(self):
        return {f: getattr(self, f) for f, _ in self._fields_}


class LaunchInfo(C.Structure):
    _fields_ = [("chunk", C.c_int32), ("phase", C.c_int32), ("shape", C.c_int32), ("ntiles", C.c_int32),
                ("flops", C.c_double), ("ms", C.c_double)]


_lib = None


def load_library(build_if_missing: bool = True):
    """dlopen the in-tree shared library (building it with nvcc first if it is absent)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        if not build_if_missing:
            raise RuntimeError("libdmrg_b200.so is missing: run `python -m paper_2501_18263_b200.build`")
        _build.build()
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64, dp = C.c_void_p, C.c_int32, C.c_int64, C.POINTER(C.c_double)
    lib.dmrg_create.argtypes = [C.POINTER(Config), C.POINTER(vp)]
    lib.dmrg_destroy.argtypes = [vp]
    lib.dmrg_last_error.argtypes = [vp]
    lib.dmrg_last_error.restype = C.c_char_p
    lib.dmrg_load_integrals.argtypes = [vp, i32, vp, vp, C.c_double]
    lib.dmrg_mps_set_sectors.argtypes = [vp, vp, vp, vp, vp]
    lib.dmrg_mps_set_site.argtypes = [vp, i32, i32, i32, vp, vp, vp, vp, vp]
    lib.dmrg_mps_update_bond.argtypes = [vp, i32, i32, vp, vp, vp]
    lib.dmrg_mps_set_site_su2.argtypes = [vp, i32, i32, i32, vp, vp, vp, vp, vp, vp]
    lib.dmrg_su2_f_factor.argtypes = [i32] * 9 + [dp, dp]
    lib.dmrg_env_build.argtypes = [vp, i32, vp]
    lib.dmrg_renormalize.argtypes = [vp, i32, vp]
    lib.dmrg_psi_layout.argtypes = [vp, C.POINTER(i32), C.POINTER(PsiBlock), C.POINTER(i64)]
    lib.dmrg_heff_apply.argtypes = [vp, vp, vp, vp]
    lib.dmrg_heff_diag.argtypes = [vp, vp, vp]
    lib.dmrg_set_shard.argtypes = [vp, i32, i32, REDUCE_FN, vp]
    lib.dmrg_shard_info.argtypes = [vp, vp, vp]
    lib.dmrg_davidson.argtypes = [vp, vp, C.c_double, i32, i32, dp, C.POINTER(i32), dp, vp]
    lib.dmrg_heff_apply_host.argtypes = [vp, vp, vp, vp]
    lib.dmrg_davidson_host.argtypes = [vp, vp, C.c_double, i32, i32, dp, C.POINTER(i32), dp, vp]
    lib.dmrg_stats.argtypes = [vp, C.POINTER(Stats)]
    lib.dmrg_env_export.argtypes = [vp, i32, i32, i32, i32, vp, C.POINTER(i64)]
    lib.dmrg_env_export_block.argtypes = [vp, i32, i32, i32, i32, i32, C.POINTER(i32), C.POINTER(i32), C.POINTER(i32), vp]
    lib.dmrg_fp64_peak.argtypes = [vp, dp, vp]
    lib.dmrg_dfma_peak.argtypes = [vp, dp, vp]
    lib.dmrg_block_flops.argtypes = [vp, vp]
    lib.dmrg_two_site_gate.argtypes = [vp, vp, vp, vp, vp]
    lib.dmrg_bond_entropy.argtypes = [vp, vp, dp, dp, vp, C.POINTER(i32), vp]
    lib.dmrg_bond_entropy_static.argtypes = [vp, vp, dp, dp, vp, C.POINTER(i32), vp]
    lib.dmrg_truncate_bond.argtypes = [vp, vp, i32, i32, dp, C.POINTER(i32), vp]
    lib.dmrg_start_vector.argtypes = [vp, vp, vp]
    lib.dmrg_bond_sectors.argtypes = [vp, i32, C.POINTER(i32), vp, vp, vp]
    lib.dmrg_rotate_integrals.argtypes = [vp, i32, C.c_double]
    lib.dmrg_rotation_gate.argtypes = [C.c_double, vp]
    lib.dmrg_apply_profile.argtypes = [vp, vp, vp, i32, C.POINTER(LaunchInfo), C.POINTER(i32), vp]
    for name in EXPORTS:
        if name != "dmrg_last_error":
            getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


class DMRGError(RuntimeError):
    pass


def _np_ptr(a):
    return a.ctypes.data_as(C.c_void_p)


class DMRG:
    """One library context on one GPU.  Methods carry the names of the C calls (without `dmrg_`)."""

    def __init__(self, L, n_up, n_dn, device=0, workspace_bytes=0, su2=False, env_cache_bytes=0, env_host_bytes=0):
        import torch
        if not torch.cuda.is_available():
            raise DMRGError("CUDA device required: the library has no CPU path")
        self.torch = torch
        self.lib = load_library()
        self.device = torch.device("cuda", device)
        self._live = {}
        # The callbacks below hand the library torch tensors.  A sweep at D = 4096 allocates and frees workspaces and
        # environment blocks of tens of GB in changing sizes; torch's default caching allocator fragments on that pattern
        # (measured: "returned NULL for 48.7 GB" at the third micro-iteration with 70 GB free), its expandable segments
        # do not.  Left alone when the user has configured the allocator.
        if "PYTORCH_CUDA_ALLOC_CONF" not in os.environ and "PYTORCH_ALLOC_CONF" not in os.environ:
            try:
                setter = getattr(torch._C, "_accelerator_setAllocatorSettings", None)      # torch >= 2.9
                if setter is None:
                    setter = torch.cuda.memory._set_allocator_settings
                setter("expandable_segments:True")
            except Exception:      # an older torch: keep its default
                pass

        def _alloc(nbytes, _user):
            try:
                t = torch.empty(int(nbytes), dtype=torch.uint8, device=self.device)
            except Exception:  # out of memory -> NULL, the library reports DMRG_ERR_ALLOC
                return None
            self._live[t.data_ptr()] = t
            return t.data_ptr()

        def _free(ptr, _user):
            self._live.pop(ptr, None)

        self._alloc_cb = ALLOC_FN(_alloc)
        self._free_cb = FREE_FN(_free)
        self.su2 = bool(su2)
        self.cfg = Config(L, n_up, n_dn, 1 if su2 else 0, device, workspace_bytes, env_cache_bytes, self._alloc_cb,
                          self._free_cb, None, env_host_bytes)
        self.ctx = C.c_void_p()
        rc = self.lib.dmrg_create(C.byref(self.cfg), C.byref(self.ctx))
        if rc != 0:
            raise DMRGError("dmrg_create failed with status %d" % rc)
        self.L, self.n_up, self.n_dn = L, n_up, n_dn

    # -- plumbing --
    def _check(self, rc):
        if rc != 0:
            raise DMRGError("status %d: %s" % (rc, self.lib.dmrg_last_error(self.ctx).decode()))

    def _stream(self):
        return C.c_void_p(self.torch.cuda.current_stream(self.device).cuda_stream)

    def close(self):
        if self.ctx:
            self.lib.dmrg_destroy(self.ctx)
            self.ctx = C.c_void_p()
            self._live.clear()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the C calls --
    def load_integrals(self, T, V, e_core=0.0):
        T = np.ascontiguousarray(T, dtype=np.float64)
        V = np.ascontiguousarray(V, dtype=np.float64)
        self._check(self.lib.dmrg_load_integrals(self.ctx, self.L, _np_ptr(T), _np_ptr(V), float(e_core)))

    def mps_set_sectors(self, sectors):
        """sectors: list over bonds 0..L of dict (n_up, n_dn) -> dim."""
        off, qu, qd, dim = [0], [], [], []
        self._sec_index = []
        for sec in sectors:
            keys = sorted(sec)
            self._sec_index.append({q: i for i, q in enumerate(keys)})
            for q in keys:
                qu.append(q[0]); qd.append(q[1]); dim.append(sec[q])
            off.append(len(qu))
        a = [np.asarray(x, dtype=np.int32) for x in (off, qu, qd, dim)]
        self._check(self.lib.dmrg_mps_set_sectors(self.ctx, *[_np_ptr(x) for x in a]))

    def mps_update_bond(self, b, sectors):
        """Replace the sectors of bond b by dict q -> dim (the site tensors b, b+1 must be set again)."""
        keys = sorted(sectors)
        self._sec_index[b] = {q: i for i, q in enumerate(keys)}
        a = [np.asarray(x, dtype=np.int32) for x in ([q[0] for q in keys], [q[1] for q in keys], [sectors[q] for q in keys])]
        self._check(self.lib.dmrg_mps_update_bond(self.ctx, b, len(keys), *[_np_ptr(x) for x in a]))

    def mps_set_site(self, site, canonical, blocks):
        """blocks: dict (q_in, s) -> (d_in, d_out) array, site 1-based, canonical 0 left / 1 right."""
        keys = sorted(blocks)
        qin = np.asarray([self._sec_index[site - 1][k[0]] for k in keys], dtype=np.int32)
        s = np.asarray([k[1] for k in keys], dtype=np.int32)
        offs, parts, o = [], [], 0
        for k in keys:
            a = np.ascontiguousarray(blocks[k], dtype=np.float64)
            offs.append(o); parts.append(a.reshape(-1)); o += a.size
        data = np.concatenate(parts) if parts else np.zeros(1)
        offs = np.asarray(offs, dtype=np.int64)
        self._check(self.lib.dmrg_mps_set_site(self.ctx, site, canonical, len(keys), _np_ptr(qin), _np_ptr(s),
                                               _np_ptr(offs), _np_ptr(data), self._stream()))

    def mps_set_site_su2(self, site, canonical, blocks):
        """blocks: dict (q_in, m, q_out) -> (d_in, d_out) array with q = (N, 2S); site 1-based."""
        keys = sorted(blocks)
        qin = np.asarray([self._sec_index[site - 1][k[0]] for k in keys], dtype=np.int32)
        m = np.asarray([k[1] for k in keys], dtype=np.int32)
        qout = np.asarray([self._sec_index[site][k[2]] for k in keys], dtype=np.int32)
        offs, parts, o = [], [], 0
        for k in keys:
            a = np.ascontiguousarray(blocks[k], dtype=np.float64)
            offs.append(o); parts.append(a.reshape(-1)); o += a.size
        data = np.concatenate(parts) if parts else np.zeros(1)
        offs = np.asarray(offs, dtype=np.int64)
        self._check(self.lib.dmrg_mps_set_site_su2(self.ctx, site, canonical, len(keys), _np_ptr(qin), _np_ptr(m),
                                                   _np_ptr(qout), _np_ptr(offs), _np_ptr(data), self._stream()))

    def env_build(self, k):
        self._check(self.lib.dmrg_env_build(self.ctx, k, self._stream()))

    def renormalize(self, direction):
        self._check(self.lib.dmrg_renormalize(self.ctx, direction, self._stream()))

    def set_shard(self, rank, count, reduce=None):
        """dmrg_set_shard.  `reduce(t)` must sum the float64 device tensor `t` over all ranks in place (e.g.
        `lambda t: torch.distributed.all_reduce(t)`); None = partial results, the caller sums."""
        if reduce is None or count <= 1:
            self._reduce_cb = REDUCE_FN(0)
        else:
            torch = self.torch

            def _cb(_user, ptr, n, _stream):
                try:
                    buf = self._live[ptr]     # the library's padded psi' buffer, allocated through _alloc
                    reduce(buf.view(torch.float64)[:n])
                    return 0
                except Exception:             # no exception may cross the C boundary
                    import traceback
                    traceback.print_exc()
                    return 1

            self._reduce_cb = REDUCE_FN(_cb)
        self._check(self.lib.dmrg_set_shard(self.ctx, int(rank), int(count), self._reduce_cb, None))
        self.shard = (int(rank), int(count))

    def shard_info(self):
        """(owner rank per psi block, analytic flops per rank) of the prepared problem."""
        nb = len(self.psi_layout()[0])
        owner = np.zeros(nb, dtype=np.int32)
        flops = np.zeros(getattr(self, "shard", (0, 1))[1], dtype=np.float64)
        self._check(self.lib.dmrg_shard_info(self.ctx, _np_ptr(owner), _np_ptr(flops)))
        return owner, flops

    def psi_layout(self):
        nb, n = C.c_int32(), C.c_int64()
        self._check(self.lib.dmrg_psi_layout(self.ctx, C.byref(nb), None, C.byref(n)))
        arr = (PsiBlock * nb.value)()
        self._check(self.lib.dmrg_psi_layout(self.ctx, C.byref(nb), arr, C.byref(n)))
        return list(arr), n.value

    def psi_size(self):
        nb, n = C.c_int32(), C.c_int64()
        self._check(self.lib.dmrg_psi_layout(self.ctx, C.byref(nb), None, C.byref(n)))
        return n.value

    def heff_apply(self, psi_in, psi_out=None):
        """psi_in: float64 CUDA tensor of length psi_size(); returns psi_out (CUDA tensor)."""
        t = self.torch
        assert psi_in.is_cuda and psi_in.dtype == t.float64 and psi_in.is_contiguous()
        if psi_out is None:
            psi_out = t.empty_like(psi_in)
        self._check(self.lib.dmrg_heff_apply(self.ctx, C.c_void_p(psi_in.data_ptr()), C.c_void_p(psi_out.data_ptr()),
                                             self._stream()))
        return psi_out

    def heff_diag(self):
        t = self.torch
        d = t.empty(self.psi_size(), dtype=t.float64, device=self.device)
        self._check(self.lib.dmrg_heff_diag(self.ctx, C.c_void_p(d.data_ptr()), self._stream()))
        return d

    def davidson(self, psi, tol=1e-10, max_iter=200, max_basis=20):
        """psi: CUDA start vector, overwritten with the Ritz vector.  Returns (energy, iters, resid)."""
        e, it, r = C.c_double(), C.c_int32(), C.c_double()
        self._check(self.lib.dmrg_davidson(self.ctx, C.c_void_p(psi.data_ptr()), tol, max_iter, max_basis,
                                           C.byref(e), C.byref(it), C.byref(r), self._stream()))
        return e.value, it.value, r.value

    def heff_apply_host(self, psi_in: np.ndarray, psi_out: np.ndarray | None = None):
        psi_in = np.ascontiguousarray(psi_in, dtype=np.float64)
        if psi_out is None:
            psi_out = np.empty_like(psi_in)
        self._check(self.lib.dmrg_heff_apply_host(self.ctx, _np_ptr(psi_in), _np_ptr(psi_out), self._stream()))
        return psi_out

    def davidson_host(self, psi: np.ndarray, tol=1e-10, max_iter=200, max_basis=20):
        assert psi.dtype == np.float64 and psi.flags.c_contiguous
        e, it, r = C.c_double(), C.c_int32(), C.c_double()
        self._check(self.lib.dmrg_davidson_host(self.ctx, _np_ptr(psi), tol, max_iter, max_basis,
                                                C.byref(e), C.byref(it), C.byref(r), self._stream()))
        return e.value, it.value, r.value

    def stats(self):
        s = Stats()
        self._check(self.lib.dmrg_stats(self.ctx, C.byref(s)))
        return s.as_dict()

    def env_export(self, side, kind, i, j=0):
        D = C.c_int64()
        self._check(self.lib.dmrg_env_export(self.ctx, side, kind, i, j, None, C.byref(D)))
        out = np.zeros((D.value, D.value))
        self._check(self.lib.dmrg_env_export(self.ctx, side, kind, i, j, _np_ptr(out), C.byref(D)))
        return out

    def env_export_block(self, side, kind, qin, d2S=0):
        """(nops, rows, cols) array of one sector block of every operator of a class, or None if the class has no
        block with input sector `qin` (label convention of dmrg_psi_block)."""
        n, r, c = C.c_int32(), C.c_int32(), C.c_int32()
        self._check(self.lib.dmrg_env_export_block(self.ctx, side, kind, d2S, qin[0], qin[1], C.byref(n), C.byref(r),
                                                   C.byref(c), None))
        if r.value == 0 or c.value == 0 or n.value == 0:
            return None
        out = np.empty((n.value, r.value, c.value))
        self._check(self.lib.dmrg_env_export_block(self.ctx, side, kind, d2S, qin[0], qin[1], C.byref(n), C.byref(r),
                                                   C.byref(c), _np_ptr(out)))
        return out

    def fp64_peak(self):
        v = C.c_double()
        self._check(self.lib.dmrg_fp64_peak(self.ctx, C.byref(v), self._stream()))
        return v.value

    def dfma_peak(self):
        v = C.c_double()
        self._check(self.lib.dmrg_dfma_peak(self.ctx, C.byref(v), self._stream()))
        return v.value

    def block_flops(self):
        """Analytic flops of one H_eff.psi per output block (numpy array, psi_layout order)."""
        out = np.zeros(len(self.psi_layout()[0]))
        self._check(self.lib.dmrg_block_flops(self.ctx, _np_ptr(out)))
        return out

    def two_site_gate(self, G, psi_in, psi_out=None):
        """psi_out = (16 x 16 gate on the occupation basis of sites k, k+1) applied to psi_in (CUDA tensors)."""
        G = np.ascontiguousarray(G, dtype=np.float64)
        assert G.shape == (16, 16)
        if psi_out is None:
            psi_out = self.torch.empty_like(psi_in)
        self._check(self.lib.dmrg_two_site_gate(self.ctx, _np_ptr(G), C.c_void_p(psi_in.data_ptr()),
                                                C.c_void_p(psi_out.data_ptr()), self._stream()))
        return psi_out

    def bond_entropy(self, psi, spectrum=False):
        """(S_1/2, S_1[, singular values]) of the cut between sites k and k+1 of the two-site wavefunction psi."""
        a, b, n = C.c_double(), C.c_double(), C.c_int32()
        self._check(self.lib.dmrg_bond_entropy(self.ctx, C.c_void_p(psi.data_ptr()), C.byref(a), C.byref(b), None,
                                               C.byref(n), self._stream()))
        if not spectrum:
            return a.value, b.value
        sig = np.zeros(max(n.value, 1))
        self._check(self.lib.dmrg_bond_entropy(self.ctx, C.c_void_p(psi.data_ptr()), C.byref(a), C.byref(b), _np_ptr(sig),
                                               C.byref(n), self._stream()))
        return a.value, b.value, sig[:n.value]

    def bond_entropy_static(self, psi, spectrum=False):
        """bond_entropy through dmrg_bond_entropy_static: no device allocation, scratch in a static device array shared
        by every call on this GPU (include/dmrg_b200.h for the limits).  The spectrum buffer is sized to the limit, so
        this method makes one call."""
        a, b, n = C.c_double(), C.c_double(), C.c_int32()
        sig = np.zeros(STATIC_MAX_SIGMA) if spectrum else None
        self._check(self.lib.dmrg_bond_entropy_static(self.ctx, C.c_void_p(psi.data_ptr()), C.byref(a), C.byref(b),
                                                      _np_ptr(sig) if spectrum else None, C.byref(n), self._stream()))
        return (a.value, b.value, sig[:n.value]) if spectrum else (a.value, b.value)

    def truncate_bond(self, psi, direction, D):
        """SVD truncation of the optimised two-site wavefunction psi inside the library (dmrg_truncate_bond): new
        sectors of bond k and the new canonical site tensor are installed on the device.  Returns (discarded weight,
        number of kept states).  Call renormalize(direction) next, then start_vector()."""
        w, n = C.c_double(), C.c_int32()
        self._check(self.lib.dmrg_truncate_bond(self.ctx, C.c_void_p(psi.data_ptr()), int(direction), int(D), C.byref(w),
                                                C.byref(n), self._stream()))
        return w.value, n.value

    def start_vector(self, out=None):
        """The truncated state in the layout of the problem prepared by renormalize (dmrg_start_vector); not normalised."""
        if out is None:
            out = self.torch.empty(self.psi_size(), dtype=self.torch.float64, device=self.device)
        self._check(self.lib.dmrg_start_vector(self.ctx, C.c_void_p(out.data_ptr()), self._stream()))
        return out

    def bond_sectors(self, b):
        """dict (n_up, n_dn) -> dimension of bond b as the library holds it."""
        n = C.c_int32()
        self._check(self.lib.dmrg_bond_sectors(self.ctx, int(b), C.byref(n), None, None, None))
        a = [np.zeros(max(n.value, 1), dtype=np.int32) for _ in range(3)]
        self._check(self.lib.dmrg_bond_sectors(self.ctx, int(b), C.byref(n), *[_np_ptr(x) for x in a]))
        return {(int(a[0][i]), int(a[1][i])): int(a[2][i]) for i in range(n.value)}

    def rotate_integrals(self, k, theta):
        self._check(self.lib.dmrg_rotate_integrals(self.ctx, int(k), float(theta)))

    def apply_profile(self, psi_in, psi_out=None, cap=4096):
        """One H_eff.psi with per-launch event timing; returns (psi_out, list of dict per launch)."""
        if psi_out is None:
            psi_out = self.torch.empty_like(psi_in)
        arr, n = (LaunchInfo * cap)(), C.c_int32()
        self._check(self.lib.dmrg_apply_profile(self.ctx, C.c_void_p(psi_in.data_ptr()), C.c_void_p(psi_out.data_ptr()),
                                                cap, arr, C.byref(n), self._stream()))
        return psi_out, [{f: getattr(arr[i], f) for f, _ in LaunchInfo._fields_} for i in range(min(n.value, cap))]

    # -- convenience: load everything a two-site problem needs from the generator objects --
    def setup(self, T, V, mps, e_core=0.0):
        self.load_integrals(T, V, e_core)
        self.mps_set_sectors(mps.sectors)
        put = self.mps_set_site_su2 if self.su2 else self.mps_set_site
        for i, blocks in mps.left.items():
            put(i, 0, blocks)
        for i, blocks in mps.right.items():
            put(i, 1, blocks)
        self.env_build(mps.k)


def rotation_gate(theta):
    """16 x 16 gate exp(-theta kappa) of the two-site orbital rotation (dmrg_rotation_gate)."""
    lib = load_library()
    G = np.zeros((16, 16))
    rc = lib.dmrg_rotation_gate(float(theta), _np_ptr(G))
    if rc != 0:
        raise DMRGError("dmrg_rotation_gate failed with status %d" % rc)
    return G


def su2_f_factor(Sa, Sk, Sg, kL, kk, k, Sa_, Sk_, Sg_):
    """(F by the 9j closed form, F by the six-CG contraction) of PAPER.md Eq. (10)-(11); doubled spins."""
    lib = load_library()
    a, b = C.c_double(), C.c_double()
    rc = lib.dmrg_su2_f_factor(Sa, Sk, Sg, kL, kk, k, Sa_, Sk_, Sg_, C.byref(a), C.byref(b))
    if rc != 0:
        raise DMRGError("dmrg_su2_f_factor failed with status %d" % rc)
    return a.value, b.value

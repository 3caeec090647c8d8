"""No-GPU checks of the boundary: the shared library builds, loads, and exports every symbol that
include/dmrg_b200.h declares; the Python binding names the same calls; the product path refuses to
run without CUDA (no CPU fallback)."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "dmrg_b200.h")


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(dmrg_[a-z0-9_]+)\s*\(", src)) - {"dmrg_alloc_fn", "dmrg_free_fn"})


def test_header_declares_the_survey_calls():
    names = _declared()
    for must in ("dmrg_create", "dmrg_destroy", "dmrg_load_integrals", "dmrg_mps_set_sectors", "dmrg_mps_set_site",
                 "dmrg_env_build", "dmrg_psi_layout", "dmrg_heff_apply", "dmrg_heff_diag", "dmrg_davidson",
                 "dmrg_renormalize", "dmrg_stats", "dmrg_env_export"):
        assert must in names


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2501_18263_b200 import build
    lib = build.build()
    assert os.path.exists(lib)
    out = subprocess.run(["nm", "-D", "--defined-only", lib], capture_output=True, text=True, check=True).stdout
    exported = set(re.findall(r" T (dmrg_[a-z0-9_]+)", out))
    assert set(_declared()) <= exported
    h = ctypes.CDLL(lib)
    for n in _declared():
        assert hasattr(h, n)


def test_binding_names_match_header():
    from paper_2501_18263_b200 import binding
    assert sorted(binding.EXPORTS) == _declared()
    for n in binding.EXPORTS:
        assert hasattr(binding.DMRG, n[len("dmrg_"):]) or hasattr(binding, n[len("dmrg_"):]) or \
            n in ("dmrg_create", "dmrg_destroy", "dmrg_last_error")


def test_su2_F_table_matches_the_oracle_in_both_forms():
    """a8 (Eq. (10)-(11), Fig. 4): the library's 9j closed form and its CG contraction (host code, no GPU
    needed) against the oracle's independent implementation."""
    from oracle import su2
    from paper_2501_18263_b200 import binding
    n = 0
    for Sa in range(0, 6):
        for Sk in (0, 1):
            for Sg in range(abs(Sa - Sk), Sa + Sk + 1, 2):
                for kL in (0, 1, 2):
                    for kk in (0, 1, 2):
                        for kop in range(abs(kL - kk), kL + kk + 1, 2):
                            for Sa_ in range(abs(Sa - kL), Sa + kL + 1, 2):
                                for Sk_ in (0, 1):
                                    for Sg_ in range(abs(Sa_ - Sk_), Sa_ + Sk_ + 1, 2):
                                        a, b = binding.su2_f_factor(Sa, Sk, Sg, kL, kk, kop, Sa_, Sk_, Sg_)
                                        ref = su2.F_sixcg(Sa, Sk, Sg, kL, kk, kop, Sa_, Sk_, Sg_)
                                        assert abs(b - ref) < 1e-12
                                        ok = (abs(Sk - kk) <= Sk_ <= Sk + kk and (Sk + kk + Sk_) % 2 == 0 and
                                              abs(Sg - kop) <= Sg_ <= Sg + kop)
                                        if ok:
                                            assert abs(a - ref) < 1e-12
                                            n += 1
    assert n > 300


def test_sm100a_code_is_in_the_library():
    from paper_2501_18263_b200 import build
    lib = build.build()
    out = subprocess.run(["cuobjdump", "-lelf", lib], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_no_cpu_fallback_without_cuda():
    import torch
    from paper_2501_18263_b200 import binding
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    with pytest.raises(binding.DMRGError):
        binding.DMRG(4, 2, 2)


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2501_18263_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2501_18263_b200\b", txt, flags=re.M), f

"""CPU-side checks of the product library: it loads, exports every symbol include/afs.h declares, validates input
before touching the device, and afs_coeffs (host arithmetic) matches the oracle's exact rationals."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import workloads as W
from oracle import coeffs_exact as ce

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def afs():
    from paper_2606_06656_b200 import build
    build.build()
    import paper_2606_06656_b200 as pkg
    return pkg


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "afs.h")).read()
    return sorted(set(re.findall(r"AFS_(?:API|DIAG)[^;(]*?\b(afs_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_boundary():
    names = declared_symbols()
    for must in ("afs_problem_create", "afs_problem_destroy", "afs_coeffs", "afs_eval_grad", "afs_round_count",
                 "afs_pgd_run", "afs_pgd_run_host", "afs_eval_grad_f64", "afs_pgd_run_f64", "afs_status_string"):
        assert must in names


def test_library_loads_and_exports_every_declared_symbol(afs):
    lib = afs.lib()
    for name in declared_symbols():
        assert hasattr(lib, name), name
    assert sorted(afs.EXPORTS) == declared_symbols()
    assert lib.afs_abi_version() == 1
    assert afs.lib().afs_status_string(0) == b"ok"


def test_no_torch_types_and_no_oracle_in_the_product():
    # the product path must not reach into oracle/ (and the oracle not into the product)
    for root, _, files in os.walk(os.path.join(ROOT, "paper_2606_06656_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(root, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, re.M), f
                assert not re.search(r"#\s*include[^\n]*oracle", src) and "afs_oracle" not in src, f
                assert "_work/" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2606_06656_b200" not in src and "from paper_2606_06656_b200" not in src
            assert "libafs_b200" not in src
    hdr = open(os.path.join(ROOT, "include", "afs.h")).read()
    assert "torch" not in hdr and "at::" not in hdr


def _create(afs, n, row_ptr, lits, types, k):
    h = C.c_void_p(None)
    rp = np.asarray(row_ptr, dtype=np.int64); li = np.asarray(lits, dtype=np.int32)
    ty = np.asarray(types, dtype=np.int32); kk = np.asarray(k, dtype=np.int32)
    st = afs.lib().afs_problem_create(n, len(types), rp.ctypes.data, li.ctypes.data, ty.ctypes.data, kk.ctypes.data,
                                      0, C.byref(h))
    if st == 0:
        afs.lib().afs_problem_destroy(h)
    return st


def test_create_rejects_invalid_input_before_touching_the_device(afs):
    ok3 = ([0, 3], [1, -2, 3], [afs.AFS_OR], [0])
    assert _create(afs, 3, [0, 3], [1, -2, 0], [afs.AFS_OR], [0]) == 4          # literal 0
    assert _create(afs, 3, [0, 3], [1, -2, 4], [afs.AFS_OR], [0]) == 4          # |literal| > n
    assert _create(afs, 3, [0, 3], [1, -2, 2], [afs.AFS_OR], [0]) == 5          # duplicate variable (G8)
    assert _create(afs, 3, [0, 3], [1, -2, 3], [7], [0]) == 2                   # bad type
    assert _create(afs, 3, [0, 3], [1, -2, 3], [afs.AFS_EK], [5]) == 3          # k > L+1
    assert _create(afs, 3, [0, 3], [1, -2, 3], [afs.AFS_CARD], [-1]) == 3       # k < 0
    assert _create(afs, 3, [0, 3], [1, -2, 3], [afs.AFS_XOR], [2]) == 3         # parity not in {0,1}
    assert _create(afs, 3, [0, 1], [1], [afs.AFS_NAE], [0]) == 3                # NAE needs L >= 2 (G6)
    assert _create(afs, 3, [0, 0], [], [afs.AFS_OR], [0]) == 4                  # empty constraint
    assert _create(afs, 3, [1, 3], [1, 2, 3], [afs.AFS_OR], [0]) == 4           # row_ptr[0] != 0
    assert _create(afs, 0, *ok3) == 1                                           # n < 1
    big = list(range(1, 1301))
    assert _create(afs, 1300, [0, 1300], big, [afs.AFS_CARD], [600]) == 8       # count type longer than 1144
    # valid input: succeeds on a GPU box, AFS_ERR_CUDA (7) without a device -- never a silent CPU fallback
    import torch
    st = _create(afs, 3, *ok3)
    assert st == (0 if torch.cuda.is_available() else 7)


def test_binding_fails_loudly_without_a_device(afs):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    inst = W.tiny_mixed(1, n=8)
    with pytest.raises(afs.AfsError) as e:
        afs.Problem.from_instance(inst)
    assert e.value.status == 7


@pytest.mark.parametrize("L", [1, 2, 3, 4, 7, 12, 20, 33])
def test_afs_coeffs_matches_exact_rationals(afs, L):
    # the product's closed forms (Appendix A, repaired) against the oracle's eq. (3) in exact rationals
    cases = [(ce.OR, 0), (ce.XOR, 0), (ce.XOR, 1), (ce.AMO, 0), (ce.EO, 0)] + ([(ce.NAE, 0)] if L >= 2 else [])
    cases += [(ce.EK, k) for k in range(0, L + 2)] + [(ce.CARD, k) for k in range(0, L + 2)]
    for ctype, k in cases:
        exact = ce.eq3(ce.spectrum(ctype, L, k), L)
        got = afs.coeffs(ctype, L, k)
        for s in range(L + 1):
            want = float(exact[s])
            assert abs(got[s] - want) <= 2 * np.spacing(abs(want)), (ctype, L, k, s, got[s], want)


@pytest.mark.parametrize("L,k", [(64, 32), (125, 60), (256, 128), (400, 7), (1024, 512)])
def test_afs_coeffs_long_parseval_and_mean(afs, L, k):
    # beyond the reach of the rational checker's speed: Parseval sum_s C(L,s) a_s^2 = 1 and a_0 = E[f], in mpmath
    import mpmath
    mpmath.mp.prec = 200
    for ctype in (ce.CARD, ce.EK):
        a = afs.coeffs(ctype, L, k)
        tot = mpmath.mpf(0)
        for s in range(L + 1):
            tot += mpmath.binomial(L, s) * mpmath.mpf(float(a[s])) ** 2
        assert abs(tot - 1) < 1e-12
        sp = ce.spectrum(ctype, L, k)
        mean = sum(mpmath.binomial(L, t) * sp[t] for t in range(L + 1)) / mpmath.mpf(2) ** L
        assert abs(mpmath.mpf(float(a[0])) - mean) < 1e-15


def test_afs_coeffs_argument_errors(afs):
    a = np.zeros(8)
    assert afs.lib().afs_coeffs(9, 3, 0, a.ctypes.data) == 2
    assert afs.lib().afs_coeffs(afs.AFS_CARD, 3, 9, a.ctypes.data) == 3
    assert afs.lib().afs_coeffs(afs.AFS_OR, 0, 0, a.ctypes.data) == 1
    assert afs.lib().afs_coeffs(afs.AFS_OR, 3, 0, None) == 1

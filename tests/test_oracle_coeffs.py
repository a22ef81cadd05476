"""Pins for the oracle's coefficients (O1): eq. (3) against the brute-force Walsh transform, the
Appendix-A closed forms, Parseval, E[f], the paper's identity at L110 and the printed n = 3 values."""
import os
from fractions import Fraction as Fr
from math import comb

import numpy as np
import pytest

from oracle import coeffs_exact as ce
from oracle import ref

TYPES = (ce.OR, ce.XOR, ce.AMO, ce.EO, ce.EK, ce.NAE, ce.CARD)
NAMES = {"OR": ce.OR, "XOR": ce.XOR, "AMO": ce.AMO, "EO": ce.EO, "EK": ce.EK, "NAE": ce.NAE, "CARD": ce.CARD}


def cases(n):
    out = [(ce.OR, 0), (ce.XOR, 0), (ce.XOR, 1), (ce.AMO, 0), (ce.EO, 0)]
    if n >= 2:
        out.append((ce.NAE, 0))
    out += [(ce.EK, k) for k in range(0, n + 1)]
    out += [(ce.CARD, k) for k in range(0, n + 2)]
    return out


@pytest.mark.parametrize("n", range(1, 9))
def test_eq3_equals_brute_force_walsh(n):
    # T1: eq. (3) reproduces the definition eq. (1) for every symmetric spectrum
    for ctype, k in cases(n):
        sp = ce.spectrum(ctype, n, k)
        assert ce.eq3(sp, n) == ce.walsh_brute(sp, n), (ctype, n, k)


@pytest.mark.parametrize("n,ctype,k", [(10, ce.CARD, 4), (10, ce.EK, 5), (11, ce.AMO, 0), (12, ce.CARD, 6),
                                       (12, ce.NAE, 0), (12, ce.XOR, 1)])
def test_eq3_equals_brute_force_walsh_n_up_to_12(n, ctype, k):
    sp = ce.spectrum(ctype, n, k)
    assert ce.eq3(sp, n) == ce.walsh_brute(sp, n)


@pytest.mark.parametrize("n", range(2, 21))
def test_closed_forms_equal_eq3(n):
    # T2: Appendix A (with readings G3, G4) equals eq. (3)
    for ctype, k in cases(n):
        cf = ce.closed_form(ctype, n, k)
        if cf is None:
            continue
        assert cf == ce.eq3(ce.spectrum(ctype, n, k), n), (ctype, n, k)


def test_amo_constant_as_printed_is_wrong():
    # G3: P:L237 prints 1-(n-1)/2^(n-1); brute force gives 1-(n+1)/2^(n-1) (-1/2 at n=2, printed form +1/2)
    for n in (2, 3, 5):
        brute = ce.walsh_brute(ce.spectrum(ce.AMO, n), n)
        assert ce.closed_form(ce.AMO, n, amo_as_printed=True)[0] != brute[0]
        assert ce.closed_form(ce.AMO, n)[0] == brute[0]
    assert ce.walsh_brute(ce.spectrum(ce.AMO, 2), 2)[0] == Fr(-1, 2)


@pytest.mark.parametrize("n", range(1, 16))
def test_parseval_and_mean(n):
    # T3: sum_s C(n,s) a_s^2 = 1 (f is +-1 valued);  T4: a_0 = E[f] = 1 - 2 #sat / 2^n
    for ctype, k in cases(n):
        sp = ce.spectrum(ctype, n, k)
        a = ce.eq3(sp, n)
        assert sum(comb(n, s) * a[s] ** 2 for s in range(n + 1)) == 1
        nsat = sum(comb(n, t) for t in range(n + 1) if sp[t] == -1)
        assert a[0] == 1 - Fr(2 * nsat, 2 ** n)


def _negate_literals(a):
    # negating every literal maps e_s -> (-1)^s e_s
    return [(-1) ** s * a[s] for s in range(len(a))]


def test_identity_L110_card2_neg_plus_or_is_eo_minus_1():
    # T5: CARD>=2(not x) + OR(x) = EO(x) - 1 in 3 variables, coefficient-wise
    n = 3
    card = _negate_literals(ce.eq3(ce.spectrum(ce.CARD, n, 2), n))
    orc = ce.eq3(ce.spectrum(ce.OR, n), n)
    eo = ce.eq3(ce.spectrum(ce.EO, n), n)
    assert [card[s] + orc[s] for s in range(n + 1)] == [eo[s] - (1 if s == 0 else 0) for s in range(n + 1)]


@pytest.mark.parametrize("n", range(2, 12))
def test_amo_plus_or_is_eo_minus_1(n):
    amo = ce.eq3(ce.spectrum(ce.AMO, n), n)
    orc = ce.eq3(ce.spectrum(ce.OR, n), n)
    eo = ce.eq3(ce.spectrum(ce.EO, n), n)
    assert [amo[s] + orc[s] for s in range(n + 1)] == [eo[s] - (1 if s == 0 else 0) for s in range(n + 1)]


@pytest.mark.parametrize("n", range(2, 12))
def test_special_cases(n):
    # T7, T8, T12
    e = lambda t, k=0: ce.eq3(ce.spectrum(t, n, k), n)
    xor = e(ce.XOR, 1)
    assert xor == [Fr(0)] * n + [Fr(1)]                                   # single coefficient a_L = 1
    assert e(ce.XOR, 0) == [Fr(0)] * n + [Fr(-1)]
    assert all(e(ce.NAE)[s] == 0 for s in range(1, n + 1, 2))             # odd orders vanish
    assert e(ce.CARD, 1) == e(ce.OR)                                      # CARD>=1 == OR
    assert e(ce.EK, 1) == e(ce.EO)                                        # EK(1) == EO
    assert e(ce.AMO) == _negate_literals(e(ce.CARD, n - 1))              # AMO(x) == CARD>=L-1(not x)
    for k in range(0, n + 1):                                             # EK = 1 + CARD>=k - CARD>=k+1
        ek, c0, c1 = e(ce.EK, k), e(ce.CARD, k), e(ce.CARD, k + 1)
        assert ek == [(1 if s == 0 else 0) + c0[s] - c1[s] for s in range(n + 1)]
    assert e(ce.CARD, 0) == [Fr(-1)] + [Fr(0)] * n                        # G5
    assert e(ce.CARD, n + 1) == [Fr(1)] + [Fr(0)] * n
    if n == 2:
        assert e(ce.NAE) == e(ce.XOR, 1)                                  # NAE(L=2) == XOR(L=2)


def test_printed_n3_values():
    # golden: Appendix-A formulas substituted at n = 3 (tests/golden/appendix_a_n3.txt, with citations)
    path = os.path.join(os.path.dirname(__file__), "golden", "appendix_a_n3.txt")
    seen = 0
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        name, k, *vals = line.split()
        want = [Fr(v) for v in vals]
        ctype = NAMES[name]
        assert ce.eq3(ce.spectrum(ctype, 3, int(k)), 3) == want, name
        got = ref.coeffs_eq3(ctype, 3, int(k))
        assert np.array_equal(got, np.array([float(v) for v in want])), name
        seen += 1
    assert seen == 6


@pytest.mark.parametrize("L", [1, 2, 3, 5, 8, 13, 21, 34, 48, 62])
def test_c_eq3_matches_exact_rationals(L):
    # the C routine (exact __int128 numerators) against the rational checker, <= 2 ulp
    for ctype, k in [(ce.OR, 0), (ce.XOR, 1), (ce.AMO, 0), (ce.EO, 0), (ce.EK, L // 2), (ce.EK, 0),
                     (ce.CARD, max(1, L // 3)), (ce.CARD, L), (ce.CARD, 0), (ce.CARD, L + 1)] + \
                    ([(ce.NAE, 0)] if L >= 2 else []):
        exact = ce.eq3(ce.spectrum(ctype, L, k), L)
        got = ref.coeffs_eq3(ctype, L, k)
        for s in range(L + 1):
            want = float(exact[s])
            assert abs(got[s] - want) <= 2 * np.spacing(abs(want)), (ctype, L, k, s)


def test_c_spectrum_matches_python():
    for L in (1, 2, 7, 30):
        for ctype, k in cases(L):
            assert list(ref.spectrum(ctype, L, k)) == ce.spectrum(ctype, L, k)

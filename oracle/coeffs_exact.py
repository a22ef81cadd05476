"""Exact-rational Fourier coefficients of symmetric constraints (oracle; TEST INFRASTRUCTURE ONLY).

Three independent routes to the same numbers, all in ``fractions.Fraction``:

* :func:`walsh_brute`  -- the DEFINITION, eq. (1): f^(S) = 2^-n sum_y f(y) prod_{j in S} y_j
  over all 2^n corners, True -> -1 (L37), f = -1 when satisfied (L52).
* :func:`eq3`          -- the general symmetric formula, eq. (3) (L49-L52).
* :func:`closed_form`  -- Appendix A (L223-L255), with the two printed formulas repaired as DESIGN.md
  readings G3 (AMO constant term) and G4 (EK subscripts) state.

Only tests/ may import this module; it shares nothing with the CUDA path.
"""
from __future__ import annotations

from fractions import Fraction as Fr
from itertools import product
from math import comb
from typing import List, Optional

OR, XOR, AMO, EO, EK, NAE, CARD = range(7)


def pred(ctype: int, L: int, k: int, t: int) -> bool:
    """Is the constraint true when exactly t of its L literals are true? (L60; Table 2; G2, G5)."""
    if ctype == OR:
        return t >= 1
    if ctype == XOR:
        return (t % 2) == (k % 2)
    if ctype == AMO:
        return t <= 1
    if ctype == EO:
        return t == 1
    if ctype == EK:
        return t == k
    if ctype == NAE:
        return 0 < t < L
    if ctype == CARD:
        return t >= k
    raise ValueError(ctype)


def spectrum(ctype: int, L: int, k: int = 0) -> List[int]:
    """sp_t = -1 if f is true when t literals are true and +1 otherwise (L52)."""
    return [-1 if pred(ctype, L, k, t) else 1 for t in range(L + 1)]


def walsh_brute(sp: List[int], n: int) -> List[Fr]:
    """Definition (eq. 1): per-|S| coefficient, S = the first s variables (symmetry makes the choice immaterial)."""
    out = []
    for s in range(n + 1):
        acc = 0
        for y in product((1, -1), repeat=n):
            t = sum(1 for v in y if v == -1)
            ch = 1
            for j in range(s):
                ch *= y[j]
            acc += sp[t] * ch
        out.append(Fr(acc, 2 ** n))
    return out


def _polymul(a: List[Fr], b: List[Fr]) -> List[Fr]:
    r = [Fr(0)] * (len(a) + len(b) - 1)
    for i, x in enumerate(a):
        for j, y in enumerate(b):
            r[i + j] += x * y
    return r


def _polypow(base: List[Fr], e: int) -> List[Fr]:
    r = [Fr(1)]
    for _ in range(e):
        r = _polymul(r, base)
    return r


def eq3(sp: List[int], n: int) -> List[Fr]:
    """eq. (3): a_0 = 2^-n sum_i C(n,i) sp_i;  a_s = [rho^(s-1)] g(rho) / (C(n-1,s-1) 2^(n-1)),
    g(rho) = sum_{i<n} d_i C(n-1,i) (1+rho)^(n-i-1) (1-rho)^i,  d_i = (sp_i - sp_{i+1})/2."""
    a = [Fr(0)] * (n + 1)
    a[0] = Fr(sum(comb(n, i) * sp[i] for i in range(n + 1)), 2 ** n)
    g = [Fr(0)] * n
    for i in range(n):
        d = Fr(sp[i] - sp[i + 1], 2)
        if d == 0:
            continue
        term = _polymul(_polypow([Fr(1), Fr(1)], n - i - 1), _polypow([Fr(1), Fr(-1)], i))
        for j, c in enumerate(term):
            g[j] += d * comb(n - 1, i) * c
    for s in range(1, n + 1):
        a[s] = g[s - 1] / (comb(n - 1, s - 1) * 2 ** (n - 1))
    return a


def closed_form(ctype: int, n: int, k: int = 0, amo_as_printed: bool = False) -> Optional[List[Fr]]:
    """Appendix A closed forms. Returns None where the appendix gives no usable closed form
    (EK with k in {0, n} has negative exponents, G4; CARD outside 1..n, G5)."""
    a = [Fr(0)] * (n + 1)
    if ctype == OR:                                   # L225
        a = [Fr(1, 2 ** (n - 1))] * (n + 1)
        a[0] = Fr(1, 2 ** (n - 1)) - 1
    elif ctype == EO:                                 # L229
        a = [Fr(2 * s - n, 2 ** (n - 1)) for s in range(n + 1)]
        a[0] = 1 - Fr(n, 2 ** (n - 1))
    elif ctype == AMO:                                # L237; constant term repaired (G3): n+1, not n-1
        a = [Fr(2 * s - n - 1, 2 ** (n - 1)) for s in range(n + 1)]
        a[0] = 1 - Fr((n - 1) if amo_as_printed else (n + 1), 2 ** (n - 1))
    elif ctype == NAE:                                # L243
        a = [Fr(1, 2 ** (n - 2)) if s % 2 == 0 else Fr(0) for s in range(n + 1)]
        a[0] = Fr(1, 2 ** (n - 2)) - 1
    elif ctype == XOR:                                # L249; k = required parity (G2): odd -> +1, even -> -1
        a[n] = Fr(1) if (k % 2) == 1 else Fr(-1)
    elif ctype == CARD:                               # L253-L255, valid for 1 <= k <= n
        if not 1 <= k <= n:
            return None
        a[0] = 1 - Fr(sum(comb(n, i) for i in range(k, n + 1)), 2 ** (n - 1))
        g = _polymul(_polypow([Fr(1), Fr(1)], n - k), _polypow([Fr(1), Fr(-1)], k - 1))
        for s in range(1, n + 1):
            a[s] = comb(n - 1, k - 1) * g[s - 1] / (comb(n - 1, s - 1) * 2 ** (n - 1))
    elif ctype == EK:                                 # L233, subscripts repaired (G4); valid for 1 <= k <= n-1
        if not 1 <= k <= n - 1:
            return None
        a[0] = 1 - Fr(comb(n, k), 2 ** (n - 1))
        g = _polymul([Fr(2 * k - n), Fr(n)],
                     _polymul(_polypow([Fr(1), Fr(1)], n - k - 1), _polypow([Fr(1), Fr(-1)], k - 1)))
        for s in range(1, n + 1):
            a[s] = Fr(comb(n, k), n) * g[s - 1] / (comb(n - 1, s - 1) * 2 ** (n - 1))
    else:
        raise ValueError(ctype)
    return a

"""Pins for the oracle's objective and gradient (O2, O2', O3): +-1 corner invariant, evaluator A vs B,
count basis vs the literal formula in multiprecision, exact finite differences, metamorphic identities."""
from fractions import Fraction as Fr
from itertools import product
from math import comb

import mpmath
import numpy as np
import pytest

import workloads as W
from oracle import coeffs_exact as ce
from oracle import ref

ALL = [(ce.OR, 0), (ce.XOR, 0), (ce.XOR, 1), (ce.AMO, 0), (ce.EO, 0), (ce.NAE, 0)]


def type_cases(L):
    out = [(t, k) for t, k in ALL if not (t == ce.NAE and L < 2)]
    out += [(ce.EK, k) for k in sorted({0, 1, L // 2, L - 1, L})]
    out += [(ce.CARD, k) for k in sorted({0, 1, L // 2, L - 1, L, L + 1})]
    return [(t, k) for t, k in out if k >= 0]


# ------------------------------------------------------------------ T6: +-1 on every Boolean corner
@pytest.mark.parametrize("L", [1, 2, 3, 4, 7, 10])
@pytest.mark.parametrize("evaluator", [0, 1, 2])
def test_corner_invariant_exhaustive(L, evaluator):
    for ctype, k in type_cases(L):
        for y in product((1.0, -1.0), repeat=L):
            t = sum(1 for v in y if v == -1.0)
            want = -1.0 if ce.pred(ctype, L, k, t) else 1.0
            fe, _ = ref.fe(ctype, k, y, evaluator, want_grad=False)
            assert abs(fe - want) < 1e-12, (ctype, L, k, y)


def points(rng, L):
    y1 = rng.uniform(-1, 1, L)
    y2 = rng.uniform(-1, 1, L); m = rng.random(L) < 0.5; y2[m] = np.sign(y2[m])      # half fixed
    y3 = np.sign(rng.uniform(-1, 1, L)); i = rng.choice(L, max(1, L // 8), replace=False)
    y3[i] = rng.uniform(-1, 1, i.size)                                                # near a corner
    return [y1, y2, y3]


# ------------------------------------------------------------------ A == B where A is well conditioned
@pytest.mark.parametrize("L", [1, 2, 3, 5, 9, 16, 24, 33, 40])
def test_evaluator_A_equals_B(L):
    rng = np.random.default_rng(100 + L)
    n_ok = 0
    for ctype, k in type_cases(L):
        for y in points(rng, L):
            try:
                fa, ga = ref.fe(ctype, k, y, 0)
            except ArithmeticError:
                continue                       # literal form refused: beyond its floating-point ceiling
            fb, gb = ref.fe(ctype, k, y, 1)
            assert abs(fa - fb) < 1e-8 and np.abs(ga - gb).max() < 1e-8, (ctype, L, k)
            n_ok += 1
    assert n_ok > 0


def test_evaluator_A_equals_B_tight_small_L():
    rng = np.random.default_rng(7)
    for L in (2, 3, 6, 12):
        for ctype, k in type_cases(L):
            for y in points(rng, L):
                fa, ga = ref.fe(ctype, k, y, 0)
                fb, gb = ref.fe(ctype, k, y, 1)
                assert abs(fa - fb) < 1e-12 and np.abs(ga - gb).max() < 1e-12


# ------------------------------------------------------------------ G10 pin: count basis vs literal form, multiprecision
def _int_poly_coeffs(a, b):
    """integer coefficients of (1+rho)^a (1-rho)^b"""
    return [sum((-1) ** u * comb(b, u) * comb(a, j - u) for u in range(max(0, j - a), min(b, j) + 1))
            for j in range(a + b + 1)]


def literal_form_mp(ctype, L, k, y, bits):
    """sum_s a_s e_s(y) with eq. (3) coefficients as exact rationals and the ESP recurrence in `bits`-bit floats."""
    mpmath.mp.prec = bits
    sp = ce.spectrum(ctype, L, k)
    g = [0] * L
    for i in range(L):
        two_d = sp[i] - sp[i + 1]
        if two_d == 0:
            continue
        c = _int_poly_coeffs(L - 1 - i, i)
        for j in range(L):
            g[j] += (two_d // 2) * comb(L - 1, i) * c[j]
    a = [Fr(sum(comb(L, i) * sp[i] for i in range(L + 1)), 2 ** L)]
    a += [Fr(g[s - 1], comb(L - 1, s - 1) * 2 ** (L - 1)) for s in range(1, L + 1)]
    e = [mpmath.mpf(0)] * (L + 1)
    e[0] = mpmath.mpf(1)
    ym = [mpmath.mpf(float(v)) for v in y]
    for j in range(L):
        for i in range(j + 1, 0, -1):
            e[i] = e[i] + ym[j] * e[i - 1]
    tot = mpmath.mpf(0)
    for s in range(L + 1):
        tot += mpmath.mpf(a[s].numerator) / mpmath.mpf(a[s].denominator) * e[s]
    return float(tot)


@pytest.mark.parametrize("L,bits", [(64, 400), (128, 800), (256, 1600)])
def test_count_basis_equals_literal_form_multiprecision(L, bits):
    rng = np.random.default_rng(L)
    for ctype, k in [(ce.CARD, L // 2), (ce.EK, L // 2), (ce.CARD, L // 4), (ce.AMO, 0), (ce.NAE, 0)]:
        for y in points(rng, L)[:2]:
            want = literal_form_mp(ctype, L, k, y, bits)
            got, _ = ref.fe(ctype, k, y, 2, want_grad=False)
            assert abs(got - want) < 1e-13, (ctype, L, k)


@pytest.mark.slow
def test_count_basis_equals_literal_form_multiprecision_L1024():
    L = 1024
    rng = np.random.default_rng(L)
    y = rng.uniform(-1, 1, L)
    want = literal_form_mp(ce.CARD, L, L // 2, y, 6000)
    got, _ = ref.fe(ce.CARD, L // 2, y, 2, want_grad=False)
    assert abs(got - want) < 1e-12


# ------------------------------------------------------------------ gradient pins
@pytest.mark.parametrize("L", [1, 2, 5, 17, 64, 200])
def test_definitional_equals_table_gradient(L):
    rng = np.random.default_rng(L)
    for ctype, k in type_cases(L):
        for y in points(rng, L):
            f1, g1 = ref.fe(ctype, k, y, 1)
            f2, g2 = ref.fe(ctype, k, y, 2)
            assert f1 == f2 and np.abs(g1 - g2).max() < 1e-13


def _fd_check(inst, X, evaluator, tol=1e-13):
    # T9: F is affine in each coordinate (multilinear), so the box-wide difference is exact
    F, G = ref.eval_grad(inst, X, evaluator)
    for v in range(inst.n):
        Xp, Xm = X.copy(), X.copy()
        Xp[:, v], Xm[:, v] = 1.0, -1.0
        Fp, _ = ref.eval_grad(inst, Xp, evaluator, want_grad=False)
        Fm, _ = ref.eval_grad(inst, Xm, evaluator, want_grad=False)
        assert np.abs((Fp - Fm) / 2 - G[:, v]).max() < tol * max(1.0, np.abs(G[:, v]).max()), v


@pytest.mark.parametrize("evaluator", [0, 1, 2])
def test_gradient_is_exact_finite_difference_tiny(evaluator):
    inst = W.tiny_mixed(11, n=9, m_each=3, max_len=6)
    X = np.random.default_rng(3).uniform(-1, 1, (5, inst.n))
    X[0, :3] = [1.0, -1.0, 0.0]
    _fd_check(inst, X, evaluator)


def test_gradient_is_exact_finite_difference_mixed_and_long():
    inst = W.mixed_pb(5, n=40, n_or=30, n_xor=6, n_eo=5, n_amo=5, n_card=5, n_nae=4, n_ek=4,
                      eo_len=(5, 12), amo_len=(5, 12), card_len=(10, 30))
    X = np.random.default_rng(4).uniform(-1, 1, (3, inst.n))
    _fd_check(inst, X, 2)
    long = W.long_pb(6, n=150, n_clauses=40, n_card=2, n_ek=2, long_len=(60, 120))
    X = np.random.default_rng(5).uniform(-1, 1, (2, long.n))
    _fd_check(long, X, 2, tol=1e-12)


def test_eo_plateau_at_all_true_corner():
    # T10 (Fig. 2): for n = 3 the EO gradient at the all-true corner (all literals -1) is exactly 0
    for ev in (0, 1, 2):
        fe, g = ref.fe(ce.EO, 0, [-1.0, -1.0, -1.0], ev)
        assert fe == 1.0 and np.all(g == 0.0)


def test_xor_is_product_of_literals():
    # T7: FE_XOR = prod y_j (odd parity), - prod y_j (even parity)
    rng = np.random.default_rng(9)
    for L in (1, 2, 3, 8):
        y = rng.uniform(-1, 1, L)
        for ev in (0, 1, 2):
            f1, g1 = ref.fe(ce.XOR, 1, y, ev)
            f0, _ = ref.fe(ce.XOR, 0, y, ev)
            assert abs(f1 - np.prod(y)) < 1e-14 and abs(f0 + np.prod(y)) < 1e-14
            for j in range(L):
                assert abs(g1[j] - np.prod(np.delete(y, j))) < 1e-14


def test_identity_L110_pointwise():
    # T5: CARD>=2(not x) + OR(x) = EO(x) - 1 at arbitrary points of the cube, values and gradients
    rng = np.random.default_rng(10)
    for _ in range(20):
        y = rng.uniform(-1, 1, 3)
        fc, gc = ref.fe(ce.CARD, 2, -y, 2)
        fo, go = ref.fe(ce.OR, 0, y, 2)
        fe, ge = ref.fe(ce.EO, 0, y, 2)
        assert abs(fc + fo - (fe - 1)) < 1e-14
        assert np.abs(-gc + go - ge).max() < 1e-14


def test_special_cases_pointwise():
    # T12 at evaluation level, long enough that evaluator A is out of the picture
    rng = np.random.default_rng(12)
    L = 90
    y = rng.uniform(-1, 1, L)
    f = lambda t, k, yy=y: ref.fe(t, k, yy, 2)
    assert abs(f(ce.CARD, 1)[0] - f(ce.OR, 0)[0]) < 1e-14
    assert abs(f(ce.EK, 1)[0] - f(ce.EO, 0)[0]) < 1e-14
    assert abs(f(ce.AMO, 0)[0] - f(ce.CARD, L - 1, -y)[0]) < 1e-14
    for k in (0, 1, 30, 45, L):
        assert abs(f(ce.EK, k)[0] - (1 + f(ce.CARD, k)[0] - f(ce.CARD, k + 1)[0])) < 1e-13
    assert abs(f(ce.CARD, 0)[0] + 1.0) < 1e-14 and np.all(f(ce.CARD, 0)[1] == 0)          # G5: constants
    assert abs(f(ce.CARD, L + 1)[0] - 1.0) < 1e-14 and np.all(f(ce.CARD, L + 1)[1] == 0)
    # OR has the closed product form 2 prod u - 1
    assert abs(f(ce.OR, 0)[0] - (2 * np.prod((1 + y) / 2) - 1)) < 1e-14


def test_symmetry_permutation_and_variable_negation():
    # T13: permuting literals leaves FE unchanged; negating x_v and all its literal signs leaves F unchanged, flips dF/dx_v
    inst = W.mixed_pb(21, n=30, n_or=20, n_xor=5, n_eo=4, n_amo=4, n_card=4, n_nae=3, n_ek=3,
                      eo_len=(5, 10), amo_len=(5, 10), card_len=(10, 20))
    rng = np.random.default_rng(1)
    X = rng.uniform(-1, 1, (4, inst.n))
    F, G = ref.eval_grad(inst, X, 2)
    # permute literals inside every constraint
    lits = inst.lits.copy()
    for c in range(inst.m):
        a, b = inst.row_ptr[c], inst.row_ptr[c + 1]
        lits[a:b] = rng.permutation(lits[a:b])
    perm = W.Instance("perm", inst.n, inst.row_ptr, lits, inst.types, inst.k)
    Fp, Gp = ref.eval_grad(perm, X, 2)
    assert np.abs(F - Fp).max() < 1e-12 and np.abs(G - Gp).max() < 1e-12
    # negate variable 3 everywhere
    v = 3
    lits2 = np.where(np.abs(inst.lits) == v + 1, -inst.lits, inst.lits).astype(np.int32)
    neg = W.Instance("neg", inst.n, inst.row_ptr, lits2, inst.types, inst.k)
    X2 = X.copy(); X2[:, v] = -X2[:, v]
    Fn, Gn = ref.eval_grad(neg, X2, 2)
    assert np.abs(F - Fn).max() < 1e-12
    assert np.abs(G[:, v] + Gn[:, v]).max() < 1e-12
    keep = np.arange(inst.n) != v
    assert np.abs(G[:, keep] - Gn[:, keep]).max() < 1e-12


def test_constraint_order_changes_gradient_only_at_rounding_level():
    inst = W.planted_kcnf(31, n=60, m=250)
    X = np.random.default_rng(2).uniform(-1, 1, (3, inst.n))
    F, G = ref.eval_grad(inst, X, 2)
    order = np.random.default_rng(3).permutation(inst.m)
    rows = [inst.lits[inst.row_ptr[c]:inst.row_ptr[c + 1]] for c in order]
    sh = W.generate._pack("shuffled", inst.n, rows, inst.types[order], inst.k[order], None, 0)
    F2, G2 = ref.eval_grad(sh, X, 2)
    assert np.abs(F - F2).max() < 1e-10 and np.abs(G - G2).max() < 1e-12


def test_objective_at_corners_counts_violations():
    # T6 at problem level: F(sign X) = m - 2 #satisfied
    inst = W.tiny_mixed(41, n=12, m_each=4, max_len=7)
    rng = np.random.default_rng(6)
    X = np.sign(rng.uniform(-1, 1, (16, inst.n)))
    F, _ = ref.eval_grad(inst, X, 2, want_grad=False)
    _, sat = ref.round_count(inst, X)
    assert np.abs(F - (inst.m - 2 * sat)).max() < 1e-12

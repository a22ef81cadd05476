"""Pins of the oracle's weighted objective (orc_eval_grad_w / orc_pgd_run_w; PAPER.md L134, L188 (i); reading G25)
against what the mathematics fixes: linearity in the weights through single-constraint sub-instances, the paper's
redundant-constraint effect (a duplicated constraint IS weight 2), exact box-wide differences, and the
per-constraint gradient magnitudes against the per-constraint evaluator."""
import numpy as np

import workloads as W
from oracle import ref


def small():
    return W.mixed_pb(91, n=80, n_or=60, n_xor=6, n_eo=4, n_amo=4, n_card=3, n_nae=4, n_ek=3, nae_len=(2, 6),
                      ek_len=(3, 9)).with_run(None, 7, 10)


def single(inst, c):
    lits = inst.lits[inst.row_ptr[c]:inst.row_ptr[c + 1]]
    return W.generate._pack("one", inst.n, [lits], inst.types[c:c + 1], inst.k[c:c + 1], None, 0)


def test_unit_weights_are_the_unweighted_objective():
    inst = small()
    F, G = ref.eval_grad(inst, inst.X0, 2)
    Fw, Gw, _ = ref.eval_grad_w(inst, np.ones(inst.m), inst.X0)
    Fn, Gn, _ = ref.eval_grad_w(inst, None, inst.X0)
    assert np.array_equal(F, Fw) and np.array_equal(G, Gw) and np.array_equal(F, Fn) and np.array_equal(G, Gn)
    a = ref.pgd_run(inst, inst.X0, 10, 0.1)
    b = ref.pgd_run_w(inst, np.ones(inst.m), inst.X0, 10, 0.1)
    assert np.array_equal(a["X"], b["X"]) and np.array_equal(a["best_sat"], b["best_sat"])


def test_linearity_in_the_weights_constraint_by_constraint():
    inst = small()
    rng = np.random.default_rng(1)
    w = rng.uniform(0.0, 3.0, inst.m)
    w[3] = 0.0
    X = inst.X0.astype(np.float64)
    Fw, Gw, GM = ref.eval_grad_w(inst, w, X, want_gm=True)
    F = np.zeros(inst.B); G = np.zeros_like(X); gm = np.zeros(inst.m)
    for c in range(inst.m):
        Fc, Gc = ref.eval_grad(single(inst, c), X, 2)
        F += w[c] * Fc; G += w[c] * Gc
        gm[c] = np.abs(Gc).sum()            # distinct variables within a constraint: |dFE/dx_v| = |dFE/dy_j|
    assert np.allclose(Fw, F, rtol=0, atol=1e-12) and np.allclose(Gw, G, rtol=0, atol=1e-12)
    assert np.allclose(GM, gm, rtol=1e-13, atol=1e-13)


def test_a_duplicated_constraint_is_weight_two():
    """redundant copies reshape the landscape exactly like doubling the constraint's weight."""
    base = W.xor_dup(9, n=40, m=30)                       # 30 XORs followed by their 30 copies
    half = W.Instance("half", base.n, base.row_ptr[:31].copy(), base.lits[:90].copy(), base.types[:30].copy(),
                      base.k[:30].copy())
    X0 = np.random.default_rng(2).uniform(-1, 1, (9, 40))
    a = ref.pgd_run(base, X0, 25, 0.05)
    b = ref.pgd_run_w(half, 2.0 * np.ones(30), X0, 25, 0.05)
    assert np.abs(a["X"] - b["X"]).max() < 1e-12
    assert np.array_equal(2 * b["best_sat"], a["best_sat"])


def test_weighted_gradient_is_the_exact_box_wide_difference():
    inst = small()
    w = np.random.default_rng(3).uniform(0.5, 2.0, inst.m)
    X = inst.X0[:3].astype(np.float64)
    _, G, _ = ref.eval_grad_w(inst, w, X)
    for v in (0, 7, 79):
        Xp, Xm = X.copy(), X.copy()
        Xp[:, v] = 1.0; Xm[:, v] = -1.0
        Fp, _, _ = ref.eval_grad_w(inst, w, Xp, want_grad=False)
        Fm, _, _ = ref.eval_grad_w(inst, w, Xm, want_grad=False)
        assert np.allclose(G[:, v], (Fp - Fm) / 2, rtol=0, atol=1e-12)     # multilinearity

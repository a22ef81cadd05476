"""Pins for the oracle's step / clip / mask (O4), rounding + count (O5) and best tracking (O6)."""
from itertools import product

import numpy as np
import pytest

import workloads as W
from oracle import coeffs_exact as ce
from oracle import ref

LR = float(np.float32(0.1))


def small_mixed(seed=3):
    return W.mixed_pb(seed, n=60, n_or=120, n_xor=10, n_eo=8, n_amo=8, n_card=6, n_nae=5, n_ek=5,
                      eo_len=(5, 12), amo_len=(5, 12), card_len=(10, 25)).with_run(None, 12, 25)


def test_round_count_brute_force_via_predicates():
    # O5 against a from-scratch Python recount with coeffs_exact.pred (the paper's semantics)
    inst = W.tiny_mixed(5, n=11, m_each=4, max_len=7)
    rng = np.random.default_rng(1)
    X = rng.uniform(-1, 1, (9, inst.n))
    X[0, :4] = [0.0, -0.0, 1.0, -1.0]                         # G13: +-0.0 round to False
    assign, sat = ref.round_count(inst, X)
    assert np.array_equal(assign, np.where(X < 0, -1, 1).astype(np.int8))
    assert assign[0, 0] == 1 and assign[0, 1] == 1
    for b in range(X.shape[0]):
        cnt = 0
        for c in range(inst.m):
            lits = inst.lits[inst.row_ptr[c]:inst.row_ptr[c + 1]]
            t = sum(1 for l in lits if (assign[b, abs(l) - 1] == -1) == (l > 0))
            cnt += ce.pred(int(inst.types[c]), len(lits), int(inst.k[c]), t)
        assert cnt == sat[b]


def test_round_count_equals_objective_at_the_corner():
    # sum_k FE(sign X) = m - 2 #sat
    inst = small_mixed()
    assign, sat = ref.round_count(inst, inst.X0)
    F, _ = ref.eval_grad(inst, assign.astype(np.float64), 2, want_grad=False)
    assert np.abs((inst.m - F) / 2 - sat).max() < 1e-10


def test_plant_satisfies_everything_and_full_mask_keeps_it():
    inst = small_mixed()
    Xp = np.tile(inst.plant.astype(np.float64), (3, 1))
    _, sat = ref.round_count(inst, Xp)
    assert np.all(sat == inst.m)
    out = ref.pgd_run(inst, inst.X0[:3], 5, LR, mask=inst.plant)     # everything fixed to the plant
    assert np.all(out["best_sat"] == inst.m) and np.all(out["best_step"] == 0)
    assert np.array_equal(out["X"], Xp)


def test_step_clip_mask_invariants():
    inst = W.long_pb(8, n=120, n_clauses=300, n_card=3, n_ek=2, long_len=(40, 90)).with_run(None, 6, 15)
    out = ref.pgd_run(inst, inst.X0, 15, LR, mask=inst.mask, want_traj=True)
    fixed = inst.mask != 0
    tr = out["traj"]
    assert np.all(np.abs(tr) <= 1.0)
    assert np.all(tr[:, :, fixed] == inst.mask[fixed].astype(np.float64))     # bit-identical for all steps
    # one step by hand from the oracle's own gradient: x' = clip(x - lr g) on the free coordinates
    _, G = ref.eval_grad(inst, tr[0], 2)
    want = np.clip(tr[0] - LR * G, -1, 1)
    want[:, fixed] = tr[0][:, fixed]
    assert np.array_equal(want, tr[1])


def test_duplicate_constraints_equal_doubled_step():
    # T11: PGD on C u copy(C) with lr equals PGD on C with 2 lr
    base = W.xor_dup(9, n=40, m=30)                 # already C u copy(C)
    half = W.Instance("half", base.n, base.row_ptr[:31].copy(), base.lits[:90].copy(),
                      base.types[:30].copy(), base.k[:30].copy())
    X0 = np.random.default_rng(2).uniform(-1, 1, (5, 40)).astype(np.float32)
    a = ref.pgd_run(base, X0, 25, 0.05, want_traj=True)
    b = ref.pgd_run(half, X0, 25, 0.10, want_traj=True)
    assert np.abs(a["traj"] - b["traj"]).max() < 1e-12


def test_best_tracking_first_max_and_recount():
    inst = small_mixed(4)
    out = ref.pgd_run(inst, inst.X0, 25, LR)
    hist = out["sat_hist"]
    assert np.array_equal(out["best_sat"], hist.max(axis=0))
    assert np.array_equal(out["best_step"], hist.argmax(axis=0))            # earliest iterate on ties (G14)
    _, recount = ref.round_count(inst, out["best_assign"].astype(np.float64))
    assert np.array_equal(recount, out["best_sat"])
    assert np.all(out["best_sat"] >= hist[0])


def test_split_run_is_resume():
    inst = small_mixed(5)
    full = ref.pgd_run(inst, inst.X0, 20, LR)
    a = ref.pgd_run(inst, inst.X0, 8, LR)
    b = ref.pgd_run(inst, a["X"], 12, LR)
    assert np.array_equal(full["X"], b["X"])
    assert np.array_equal(np.maximum(a["best_sat"], b["best_sat"]), full["best_sat"])


def test_zero_steps():
    inst = small_mixed(6)
    out = ref.pgd_run(inst, inst.X0, 0, LR)
    assign, sat = ref.round_count(inst, inst.X0)
    assert np.array_equal(out["best_assign"], assign) and np.array_equal(out["best_sat"], sat)
    assert np.all(out["best_step"] == 0) and np.array_equal(out["X"], inst.X0.astype(np.float64))


def test_pgd_reaches_the_minimum_on_an_easy_instance():
    # at a satisfying corner the objective is -m.  An under-constrained planted 3-CNF is solved by some restart.
    inst = W.planted_kcnf(12, n=30, m=45).with_run(None, 32, 200)
    out = ref.pgd_run(inst, inst.X0, 200, LR)
    assert out["best_sat"].max() == inst.m
    b = int(out["best_sat"].argmax())
    F, _ = ref.eval_grad(inst, out["best_assign"][b:b + 1].astype(np.float64), 2, want_grad=False)
    assert abs(F[0] + inst.m) < 1e-12


def test_evaluators_give_the_same_trajectory():
    inst = W.tiny_mixed(13, n=10, m_each=3, max_len=6).with_run(None, 4, 10)
    t0 = ref.pgd_run(inst, inst.X0, 10, LR, evaluator=0, want_traj=True)["traj"]
    t1 = ref.pgd_run(inst, inst.X0, 10, LR, evaluator=1, want_traj=True)["traj"]
    t2 = ref.pgd_run(inst, inst.X0, 10, LR, evaluator=2, want_traj=True)["traj"]
    assert np.abs(t0 - t1).max() < 1e-12 and np.abs(t1 - t2).max() < 1e-12


def test_same_variable_twice_in_one_constraint_is_rejected():
    # G8: the multilinear expansion assumes distinct variables; the oracle refuses, like afs_problem_create
    ok = W.Instance("ok", 4, np.array([0, 3, 5], np.int64), np.array([1, -2, 3, 2, -4], np.int32),
                    np.array([W.AFS_OR, W.AFS_XOR], np.int32), np.array([0, 1], np.int32))
    X = np.zeros((1, 4))
    ref.eval_grad(ok, X)                                       # the same variable in two constraints is fine
    for lits in ([1, -2, 1, 2, -4], [1, -2, -1, 2, -4], [1, -2, 3, 4, -4]):
        bad = W.Instance("dup", 4, ok.row_ptr.copy(), np.array(lits, np.int32), ok.types.copy(), ok.k.copy())
        with pytest.raises(ValueError):
            ref.eval_grad(bad, X)
        with pytest.raises(ValueError):
            ref.round_count(bad, X)
        with pytest.raises(ValueError):
            ref.pgd_run(bad, X, 1, LR)

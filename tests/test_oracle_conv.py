"""Pins of the oracle's convergence-detecting PGD (orc_pgd_run_conv; reading G24)
against what the mathematics fixes, not against itself: the run without detection, trajectories of that run, a
hand-computed one-variable example, and monotonicity in the tolerance."""
import numpy as np

import workloads as W
from oracle import ref

LR = 0.1


def small():
    return W.mixed_pb(77, n=40, n_or=110, n_xor=8, n_eo=5, n_amo=5, n_card=4).with_run(None, 12, 60)


def test_tolerance_zero_is_the_plain_run():
    inst = small()
    a = ref.pgd_run(inst, inst.X0, 60, LR)
    b = ref.pgd_run_conv(inst, inst.X0, 60, LR, 0.0)
    assert np.array_equal(a["X"], b["X"]) and np.array_equal(a["best_sat"], b["best_sat"])
    assert np.array_equal(a["best_step"], b["best_step"]) and np.array_equal(a["best_assign"], b["best_assign"])
    assert np.all(b["conv_step"] == -1)
    assert np.array_equal(b["final_sat"], a["sat_hist"][-1])
    F, _ = ref.eval_grad(inst, a["X"], 2, want_grad=False)
    assert np.allclose(b["final_F"], F, rtol=0, atol=1e-12)


def test_a_stopped_restart_keeps_the_iterate_of_its_last_step():
    """conv_step = t+1 is the FIRST step whose max|dX| is below tol in the plain run's trajectory, the returned X is
    that trajectory's iterate t+1, and best / final counts are those of the iterates 0..t+1."""
    inst = small()
    tr = ref.pgd_run(inst, inst.X0, 60, LR, want_traj=True)
    traj, hist = tr["traj"], tr["sat_hist"]
    for tol in (0.2, 0.05, 1e-3, 1e-9):
        c = ref.pgd_run_conv(inst, inst.X0, 60, LR, tol)
        for b in range(inst.B):
            d = np.abs(np.diff(traj[:, b, :], axis=0)).max(axis=1)          # max|dX| of step t -> t+1
            hit = np.nonzero(d < tol)[0]
            if hit.size == 0:
                assert c["conv_step"][b] == -1
                last = 60
            else:
                last = int(hit[0]) + 1
                assert c["conv_step"][b] == last
            assert np.array_equal(c["X"][b], traj[last, b])
            assert c["final_sat"][b] == hist[last, b]
            assert c["best_sat"][b] == hist[: last + 1, b].max()
            assert c["best_step"][b] == int(hist[: last + 1, b].argmax())


def test_everything_stops_after_one_step_when_the_tolerance_exceeds_the_cube():
    inst = small()
    one = ref.pgd_run(inst, inst.X0, 1, LR)
    c = ref.pgd_run_conv(inst, inst.X0, 60, LR, 2.5)           # |dX| <= 2 always
    assert np.all(c["conv_step"] == 1) and np.array_equal(c["X"], one["X"])


def test_conv_step_is_monotone_in_the_tolerance():
    inst = small()
    prev = None
    for tol in (1e-6, 1e-3, 1e-2, 0.1, 0.3):
        cs = ref.pgd_run_conv(inst, inst.X0, 60, LR, tol)["conv_step"].astype(np.int64)
        cs[cs < 0] = 10 ** 6
        if prev is not None:
            assert np.all(cs <= prev)
        prev = cs


def test_hand_computed_unit_clause():
    """One variable, one unit clause (x): FE = x, dFE/dx = 1, so x_{t+1} = max(x_t - lr, -1).  From x_0 = 0.25 with
    lr = 0.1 the steps are 0.1 wide until x_12 = -0.95; step 12 -> 13 is clipped to -1 (width 0.05), step 13 -> 14
    has width 0.  tol = 0.07 therefore stops at conv_step = 13, tol = 0.01 at 14 (first width below it), tol = 0.2 at 1."""
    one = W.Instance("one", 1, np.array([0, 1], np.int64), np.array([1], np.int32), np.array([W.AFS_OR], np.int32),
                     np.zeros(1, np.int32))
    X0 = np.array([[0.25]])
    for tol, want, xf in ((0.07, 13, -1.0), (0.01, 14, -1.0), (0.2, 1, 0.15)):
        c = ref.pgd_run_conv(one, X0, 40, 0.1, tol)
        assert c["conv_step"][0] == want, (tol, c["conv_step"])
        assert abs(c["X"][0, 0] - xf) < 1e-12
    c = ref.pgd_run_conv(one, X0, 40, 0.1, 0.07)
    assert c["final_sat"][0] == 1 and c["best_step"][0] == 3 and abs(c["final_F"][0] + 1.0) < 1e-12   # x_3 = -0.05 < 0


def test_mask_and_fixed_coordinates():
    inst = W.long_pb(5, n=120, n_clauses=150, n_card=3, n_ek=2, long_len=(70, 110)).with_run(None, 6, 30)
    c = ref.pgd_run_conv(inst, inst.X0, 30, LR, 1e-3, mask=inst.mask)
    fixed = inst.mask != 0
    assert np.array_equal(c["X"][:, fixed], np.tile(inst.mask[fixed].astype(np.float64), (6, 1)))
    # all variables fixed: nothing moves, every restart stops after its first step
    c = ref.pgd_run_conv(inst, inst.X0, 30, LR, 1e-9, mask=inst.plant)
    assert np.all(c["conv_step"] == 1) and np.all(c["final_sat"] == inst.m)

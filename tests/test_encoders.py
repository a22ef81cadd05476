"""The Table-1 encoders (workloads/encoders.py) against facts that do not depend on this code: a valid
Sudoku grid built from the cyclic Latin pattern, the pentagon colouring of K5 (R(3,3) > 5) and R(3,3) = 6; and the
oracle on them."""
import itertools

import numpy as np
import pytest

import workloads as W
from oracle import ref


def valid_grid(box=3):
    N = box * box          # the standard shifted pattern: row r is the base row shifted by box*(r % box) + r // box
    return np.array([[(box * (r % box) + r // box + c) % N + 1 for c in range(N)] for r in range(N)])


def test_sudoku_constraints_hold_exactly_on_valid_grids():
    for box in (2, 3):
        inst = W.sudoku(box=box)
        N = box * box
        assert inst.n == N ** 3 and inst.m == 4 * N * N and np.all(inst.lengths() == N)
        g = valid_grid(box)
        a = W.sudoku_assignment(g, box)
        assert W.plant_satisfies(inst, a).all()
        _, sat = ref.round_count(inst, a[None, :].astype(np.float64))
        assert sat[0] == inst.m
        F, _ = ref.eval_grad(inst, a[None, :].astype(np.float64), 2, want_grad=False)
        assert abs(F[0] + inst.m) < 1e-12                      # F = -m at a solution
        g2 = g.copy(); g2[0, 0], g2[0, 1] = g2[0, 1], g2[0, 0]  # swapping two cells of a row breaks column / box constraints
        assert not W.plant_satisfies(inst, W.sudoku_assignment(g2, box)).all()


def test_sudoku_clues_become_the_mask():
    g = valid_grid(3)
    clues = np.where(np.random.default_rng(0).random((9, 9)) < 0.4, g, 0)
    inst = W.sudoku(clues=clues)
    a = W.sudoku_assignment(g)
    fixed = inst.mask != 0
    assert fixed.sum() == 9 * (clues > 0).sum() and np.array_equal(inst.mask[fixed], a[fixed])


def test_ramsey_pentagon_and_r33():
    inst = W.ramsey(5, 3)
    assert inst.n == 10 and inst.m == 10 and np.all(inst.lengths() == 3)
    pent = W.ramsey_assignment(5, lambda i, j: (j - i) % 5 in (1, 4))      # the 5-cycle in one colour, its complement in the other
    assert W.plant_satisfies(inst, pent).all()
    k6 = W.ramsey(6, 3)                                                   # R(3,3) = 6: no colouring of K6 works
    best = 0
    for bits in itertools.product((-1, 1), repeat=15):
        best = max(best, int(W.plant_satisfies(k6, np.array(bits, np.int8)).sum()))
    assert best == k6.m - 2                                               # every colouring of K6 has >= 2 monochromatic triangles


@pytest.mark.gpu
def test_encoders_on_the_gpu_against_the_oracle():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_2606_06656_b200 import build
    build.build()
    import paper_2606_06656_b200 as afs
    g = valid_grid(3)
    clues = np.where(np.random.default_rng(1).random((9, 9)) < 0.45, g, 0)
    for inst in (W.sudoku(clues=clues).with_run(None, 70, 60), W.ramsey(17, 4).with_run(None, 40, 60)):
        P = afs.Problem.from_instance(inst)
        mask = None if inst.mask is None else torch.from_numpy(inst.mask).cuda()
        X = torch.from_numpy(inst.X0.astype(np.float64)).cuda()
        out = P.pgd_run(X, 20, 0.1, mask=mask)
        o = ref.pgd_run(inst, inst.X0, 20, 0.1, mask=inst.mask)
        assert np.abs(X.cpu().numpy() - o["X"]).max() <= 1e-9
        assert np.array_equal(out["best_sat"].cpu().numpy(), o["best_sat"])
        Xf = torch.from_numpy(inst.X0).cuda()
        outf = P.pgd_run(Xf, 60, 0.1, mask=mask)
        _, rec = ref.round_count(inst, outf["best_assign"].cpu().numpy().astype(np.float64))
        assert np.array_equal(rec, outf["best_sat"].cpu().numpy())
        _, s0 = ref.round_count(inst, o["X"] * 0 + np.where(inst.X0 < 0, -1.0, 1.0))
        assert outf["best_sat"].float().mean().item() > s0.mean()          # descent improves the rounded count
        P.close()

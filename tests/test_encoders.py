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


def test_sudoku_with_unit_clues_has_the_sizes_table_1_prints():
    """Sudoku 9x9, Walsh-Fourier: 729 variables, 341 constraints = 324 exactly-one + 17 unit clues."""
    g = valid_grid(3)
    cells = np.random.default_rng(3).choice(81, size=17, replace=False)
    clues = np.zeros((9, 9), int)
    clues.flat[cells] = g.flat[cells]
    inst = W.sudoku_unit_clues(clues)
    assert (inst.n, inst.m) == (729, 341)
    assert (inst.types == W.AFS_EO).sum() == 324 and (inst.lengths() == 1).sum() == 17
    assert W.plant_satisfies(inst, W.sudoku_assignment(g)).all()
    g2 = valid_grid(3)[::-1]                                   # another valid grid: breaks clues, keeps the 324
    ok = W.plant_satisfies(inst, W.sudoku_assignment(g2))
    assert ok[:324].all() and not ok[324:].all()


def gf16_colouring():
    """The classical 3-colouring of K16 without a monochromatic triangle (it shows R(3,3,3) > 16): vertices = GF(16),
    edge {a, b} coloured by the coset of the cubes that a + b lies in.  GF(16) = GF(2)[x] / (x^4 + x + 1), x generates."""
    log, e = {}, 1
    for i in range(15):
        log[e] = i
        e <<= 1
        if e & 16:
            e ^= 0b10011
    return lambda i, j: log[i ^ j] % 3


def test_ramsey3c_variable_counts_of_table_1_and_the_k16_colouring():
    """234 variables for 13 vertices, 360 for 16.  The GF(16) colouring satisfies every family of
    constraints: one colour per edge, 5 edges of each colour at every vertex, 40 per colour overall, no monochromatic
    triangle; recolouring one edge breaks the balance at both of its ends."""
    assert W.ramsey3c(13, triangles=False).n == 234 and W.ramsey3c(16, triangles=False).n == 360
    assert W.ramsey3c(13, triangles=False).m == 78 + 39
    inst = W.ramsey3c(16, triangles=True, global_cardinality=True)
    assert inst.m == 120 + 48 + 3 + 3 * 560
    L = inst.lengths()
    assert np.all(L[:120] == 3) and np.all(L[120:168] == 15) and np.all(L[168:171] == 120) and np.all(L[171:] == 3)
    col = gf16_colouring()
    a = W.ramsey3c_assignment(16, col)
    assert W.plant_satisfies(inst, a).all()
    _, sat = ref.round_count(inst, a[None, :].astype(np.float64))
    assert sat[0] == inst.m
    bad = W.ramsey3c_assignment(16, lambda i, j: (col(i, j) + 1) % 3 if (i, j) == (2, 9) else col(i, j))
    ok = W.plant_satisfies(inst, bad)
    assert ok[:120].all() and (~ok[120:168]).sum() == 4 and (~ok[168:171]).sum() == 2
    # K17 has no such colouring (R(3,3,3) = 17), and N - 1 must be divisible by 3
    with pytest.raises(ValueError):
        W.ramsey3c(15)


def is_costas(perm):
    n = len(perm)
    seen = set()
    for i in range(n):
        for j in range(i + 1, n):
            v = (j - i, perm[j] - perm[i])
            if v in seen:
                return False
            seen.add(v)
    return True


@pytest.mark.parametrize("n,count", [(3, 4), (4, 12), (5, 40)])
def test_costas_encoder_accepts_exactly_the_costas_permutations(n, count):
    """The definition checked directly on every permutation, against the encoder's constraints; the
    number of Costas arrays of order 3, 4, 5 is 4, 12, 40 (the known enumeration)."""
    inst = W.costas(n)
    assert inst.n == n * n and (inst.types == W.AFS_EO).sum() == 2 * n
    found = 0
    for perm in itertools.permutations(range(n)):
        ok = bool(W.plant_satisfies(inst, W.costas_assignment(perm)).all())
        assert ok == is_costas(perm)
        found += ok
    assert found == count
    # a non-permutation fails a row / column constraint
    a = W.costas_assignment(list(range(n)))
    a[0] = 1
    assert not W.plant_satisfies(inst, a)[:2 * n].all()


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


@pytest.mark.gpu
def test_table_1_encoders_on_the_gpu_against_the_oracle():
    """Sudoku with unit clues (729 / 341), Ramsey 3C on 16 vertices (360 variables; EO, per-vertex EK of length 15, the
    three global EK of length 120 the paper calls beyond the floating-point ceiling, triangle clauses) and Costas order 6:
    fp64 build against the oracle over 20 steps, fp32 counts recounted by the oracle."""
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_2606_06656_b200 import build
    build.build()
    import paper_2606_06656_b200 as afs
    g = valid_grid(3)
    cells = np.random.default_rng(3).choice(81, size=17, replace=False)
    clues = np.zeros((9, 9), int)
    clues.flat[cells] = g.flat[cells]
    for inst in (W.sudoku_unit_clues(clues).with_run(None, 70, 60),
                 W.ramsey3c(16, triangles=True, global_cardinality=True).with_run(None, 45, 60),
                 W.costas(6).with_run(None, 40, 60)):
        P = afs.Problem.from_instance(inst)
        X = torch.from_numpy(inst.X0.astype(np.float64)).cuda()
        out = P.pgd_run(X, 20, 0.1)
        o = ref.pgd_run(inst, inst.X0, 20, 0.1)
        assert np.abs(X.cpu().numpy() - o["X"]).max() <= 1e-9, inst.name
        assert np.array_equal(out["best_sat"].cpu().numpy(), o["best_sat"]), inst.name
        assert np.array_equal(out["best_assign"].cpu().numpy(), o["best_assign"]), inst.name
        Xf = torch.from_numpy(inst.X0).cuda()
        F, G = P.eval_grad(Xf)
        Fo, Go = ref.eval_grad(inst, inst.X0.astype(np.float64), 2)
        assert np.all(np.abs(F.cpu().numpy() - Fo) <= 1e-4 * np.abs(Fo) + 1e-6 * inst.m), inst.name
        assert np.all(np.abs(G.cpu().numpy() - Go) <= 1e-4 * np.abs(Go).max(axis=1, keepdims=True)), inst.name
        outf = P.pgd_run(Xf, 60, 0.1)
        _, rec = ref.round_count(inst, outf["best_assign"].cpu().numpy().astype(np.float64))
        assert np.array_equal(rec, outf["best_sat"].cpu().numpy()), inst.name
        P.close()

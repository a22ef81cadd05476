"""Encoders of the three problem families of the paper's Table 1 into symmetric constraints, as a
second workload beside BASELINE.json's five configurations.  The paper does not print its encodings; these are the
direct textbook formulations, derived here, and DESIGN.md section 2 (readings G26-G28) says where their counts meet
the printed ones and where they cannot.  No arithmetic of the method lives in this module.

Polarity as everywhere: True -> -1, False -> +1; a literal +(v+1) is x_v.
"""
from __future__ import annotations

import itertools
from typing import Optional

import numpy as np

from .generate import AFS_EK, AFS_EO, AFS_NAE, AFS_OR, Instance, _pack, _rng


def sudoku(clues: Optional[np.ndarray] = None, box: int = 3, seed: int = 0) -> Instance:
    """Sudoku of side N = box^2 as exactly-one constraints over x[r, c, d] ("cell (r, c) holds digit d"), variable index
    (r N + c) N + d:  every cell holds exactly one digit; every digit occurs exactly once in every row, column and box
    -- 4 N^2 EO constraints of length N.  ``clues`` (N x N ints, 0 = empty) become the fixed-variable mask: the clue's
    variable fixed True, the other digits of that cell fixed False (partial-assignment completion)."""
    N = box * box
    var = lambda r, c, d: (r * N + c) * N + d
    rows = []
    for r in range(N):
        for c in range(N):
            rows.append(np.array([var(r, c, d) + 1 for d in range(N)]))
    for d in range(N):
        for r in range(N):
            rows.append(np.array([var(r, c, d) + 1 for c in range(N)]))
        for c in range(N):
            rows.append(np.array([var(r, c, d) + 1 for r in range(N)]))
        for br in range(box):
            for bc in range(box):
                rows.append(np.array([var(br * box + i, bc * box + j, d) + 1 for i in range(box) for j in range(box)]))
    inst = _pack("sudoku_%dx%d" % (N, N), N ** 3, rows, [AFS_EO] * len(rows), [0] * len(rows), None, seed)
    if clues is not None:
        clues = np.asarray(clues)
        mask = np.zeros(N ** 3, np.int8)
        for r in range(N):
            for c in range(N):
                if clues[r, c] > 0:
                    for d in range(N):
                        mask[var(r, c, d)] = -1 if d == clues[r, c] - 1 else 1
        inst.mask = mask
    inst.notes["rng"] = _rng(seed)
    return inst


def sudoku_assignment(grid: np.ndarray, box: int = 3) -> np.ndarray:
    """The +-1 assignment (int8, -1 = True) that a filled grid (digits 1..N) stands for."""
    N = box * box
    a = np.ones(N ** 3, np.int8)
    for r in range(N):
        for c in range(N):
            a[(r * N + c) * N + int(grid[r, c]) - 1] = -1
    return a


def ramsey(n_vertices: int, clique: int, seed: int = 0) -> Instance:
    """Two-colourings of the edges of K_n without a monochromatic K_clique (a witness that R(clique, clique) > n):
    one variable per edge (True = first colour), and for every clique-subset of the vertices one NAE constraint over its
    C(clique, 2) edges -- "not all equal" is exactly "not monochromatic"."""
    idx = {}
    for e, (i, j) in enumerate(itertools.combinations(range(n_vertices), 2)):
        idx[(i, j)] = e
    rows = []
    for sub in itertools.combinations(range(n_vertices), clique):
        rows.append(np.array([idx[p] + 1 for p in itertools.combinations(sub, 2)]))
    inst = _pack("ramsey_K%d_no_K%d" % (n_vertices, clique), len(idx), rows, [AFS_NAE] * len(rows), [0] * len(rows), None, seed)
    inst.notes["rng"] = _rng(seed)
    return inst


def ramsey_assignment(n_vertices: int, first_colour) -> np.ndarray:
    """+-1 assignment of the edge variables from a predicate first_colour(i, j) (i < j)."""
    a = np.ones(n_vertices * (n_vertices - 1) // 2, np.int8)
    for e, (i, j) in enumerate(itertools.combinations(range(n_vertices), 2)):
        if first_colour(i, j):
            a[e] = -1
    return a


def sudoku_unit_clues(clues: np.ndarray, box: int = 3, seed: int = 0) -> Instance:
    """The Sudoku encoding whose size Table 1 prints (729 variables, 341 constraints): the 4 N^2 = 324
    exactly-one constraints of `sudoku` plus ONE UNIT CONSTRAINT PER CLUE (an OR over the single literal "cell (r, c)
    holds its clue"), nothing fixed by a mask.  341 - 324 = 17 is the number of clues of a minimal 9 x 9 puzzle, so a
    17-clue grid gives exactly the printed counts (reading G26)."""
    N = box * box
    base = sudoku(None, box, seed)
    rows = [base.lits[base.row_ptr[c]:base.row_ptr[c + 1]] for c in range(base.m)]
    types = [AFS_EO] * base.m
    clues = np.asarray(clues)
    for r in range(N):
        for c in range(N):
            if clues[r, c] > 0:
                rows.append(np.array([(r * N + c) * N + int(clues[r, c]) - 1 + 1]))
                types.append(AFS_OR)
    inst = _pack("sudoku_%dx%d_unit_clues" % (N, N), N ** 3, rows, types, [0] * len(rows), None, seed)
    inst.notes["rng"] = _rng(seed)
    return inst


def ramsey3c(n_vertices: int, triangles: bool = True, global_cardinality: bool = False, seed: int = 0) -> Instance:
    """"Ramsey 3C" of Table 1 and section 3.1: 3-colourings of the edges of K_N in the
    balanced relaxation.  One variable per (edge, colour), index 3 e + c with the edges in lexicographic order: 78 * 3 =
    234 variables for N = 13 and 120 * 3 = 360 for N = 16, the printed counts.  Constraints:
      - EO over the 3 colour variables of every edge ("each edge gets exactly one colour");
      - EK with k = (N-1)/3 over the N-1 edges at a vertex, per vertex and colour ("each vertex to have equal edge-colour
        distribution ... cardinality constraints enforce balancing"; the per-vertex decomposition of P:L106);
      - optionally EK with k = E/3 over ALL edges per colour (the "global cardinality constraints on edges (120 literals
        for (16, 3))" the paper names as beyond the floating-point ceiling);
      - optionally, per triangle and colour, the clause "not all three edges have this colour" (no monochromatic triangle).
    N - 1 must be divisible by 3.  The printed constraint counts (276, 411 = 3 (E + N + 1)) are not reproduced by any
    combination of these families; reading G27."""
    if (n_vertices - 1) % 3 != 0:
        raise ValueError("balanced 3-colouring needs 3 | N - 1")
    edges = list(itertools.combinations(range(n_vertices), 2))
    eidx = {e: i for i, e in enumerate(edges)}
    var = lambda i, j, c: 3 * eidx[(min(i, j), max(i, j))] + c
    rows, types, ks = [], [], []
    for (i, j) in edges:
        rows.append(np.array([var(i, j, c) + 1 for c in range(3)])); types.append(AFS_EO); ks.append(0)
    for v in range(n_vertices):
        for c in range(3):
            rows.append(np.array([var(v, u, c) + 1 for u in range(n_vertices) if u != v]))
            types.append(AFS_EK); ks.append((n_vertices - 1) // 3)
    if global_cardinality:
        if len(edges) % 3 != 0:
            raise ValueError("global balancing needs 3 | E")
        for c in range(3):
            rows.append(np.array([var(i, j, c) + 1 for (i, j) in edges])); types.append(AFS_EK); ks.append(len(edges) // 3)
    if triangles:
        for (i, j, k) in itertools.combinations(range(n_vertices), 3):
            for c in range(3):
                rows.append(-np.array([var(i, j, c) + 1, var(i, k, c) + 1, var(j, k, c) + 1])); types.append(AFS_OR); ks.append(0)
    inst = _pack("ramsey3c_K%d" % n_vertices, 3 * len(edges), rows, types, ks, None, seed)
    inst.notes["rng"] = _rng(seed)
    return inst


def ramsey3c_assignment(n_vertices: int, colour) -> np.ndarray:
    """+-1 assignment of the (edge, colour) variables from colour(i, j) in {0, 1, 2} (i < j)."""
    edges = list(itertools.combinations(range(n_vertices), 2))
    a = np.ones(3 * len(edges), np.int8)
    for e, (i, j) in enumerate(edges):
        a[3 * e + int(colour(i, j))] = -1
    return a


def costas(n: int, seed: int = 0) -> Instance:
    """Costas arrays of order n: n points in an n x n grid, exactly one per row and column, all
    displacement vectors between pairs of points distinct.  One variable per cell, index r n + c; EO per row and per
    column; and for every displacement vector v = (dr, dc), dr >= 1, dc != 0, and every two different anchors a, a'
    with a, a + v, a', a' + v inside the grid, the clause "not all of these cells hold a point" (3 cells when the two
    pairs chain, a' = a + v).  No auxiliary variables, O(n^5) clauses: meant for the small orders the paper solves
    (n <= 8).  Table 1's variable counts (97, 712, 2577, 5872) include auxiliary variables of an encoding the
    paper does not print and are not reproduced; reading G28."""
    if n > 10:
        raise ValueError("the auxiliary-free Costas encoding is meant for n <= 10")
    var = lambda r, c: r * n + c
    rows, types = [], []
    for r in range(n):
        rows.append(np.array([var(r, c) + 1 for c in range(n)])); types.append(AFS_EO)
    for c in range(n):
        rows.append(np.array([var(r, c) + 1 for r in range(n)])); types.append(AFS_EO)
    for dr in range(1, n):
        for dc in range(-(n - 1), n):
            if dc == 0:
                continue
            anchors = [(r, c) for r in range(n - dr) for c in range(n) if 0 <= c + dc < n]
            for (a, b) in itertools.combinations(anchors, 2):
                cells = sorted({var(*a), var(a[0] + dr, a[1] + dc), var(*b), var(b[0] + dr, b[1] + dc)})
                rows.append(-(np.array(cells) + 1)); types.append(AFS_OR)
    inst = _pack("costas_%d" % n, n * n, rows, types, [0] * len(rows), None, seed)
    inst.notes["rng"] = _rng(seed)
    return inst


def costas_assignment(perm) -> np.ndarray:
    """+-1 assignment with a point at (r, perm[r]) for every row r."""
    n = len(perm)
    a = np.ones(n * n, np.int8)
    for r, c in enumerate(perm):
        a[r * n + int(c)] = -1
    return a

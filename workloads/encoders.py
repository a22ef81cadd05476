"""Encoders of two problem families of the paper's Table 1 into symmetric constraints, as a second
workload beside BASELINE.json's five configurations.  The paper does not print its encodings; these are the direct
textbook formulations, derived here.  No arithmetic of the method lives in this module.

Polarity as everywhere: True -> -1, False -> +1; a literal +(v+1) is x_v.
"""
from __future__ import annotations

import itertools
from typing import Optional

import numpy as np

from .generate import AFS_EO, AFS_NAE, Instance, _pack, _rng


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

"""Seeded synthetic PB-SAT instances: the five BASELINE.json configs and scaled variants.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path
(``paper_2606_06656_b200/``).  It holds none of the method's arithmetic: no
Walsh-Fourier coefficient, no objective, no gradient, no PGD step -- only
instance construction (random variable choices, literal signs, counting true
literals under a planted assignment to set thresholds) and the start points.

Conventions (section 2.1): True -> -1, False -> +1.
A literal is a signed 1-based int32: +(v+1) is x_v, -(v+1) is NOT x_v.
A planted assignment ``plant[v]`` is -1 (True) or +1 (False).

Recipes: DESIGN.md "Input recipe" (readings G19-G23 of SURVEY.md 8(c)).
"""
from .generate import (  # noqa: F401
    AFS_OR, AFS_XOR, AFS_AMO, AFS_EO, AFS_EK, AFS_NAE, AFS_CARD, TYPE_NAMES,
    Instance, config, config_names, BASE_SEED,
    random_kcnf, planted_kcnf, mixed_pb, xor_dup, long_pb, tiny_mixed,
    concat, true_counts, plant_satisfies,
)
from .encoders import (sudoku, sudoku_assignment, sudoku_unit_clues, ramsey, ramsey_assignment, ramsey3c,  # noqa: F401
                       ramsey3c_assignment, costas, costas_assignment)

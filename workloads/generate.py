"""Instance builders.  No method arithmetic lives here (see package docstring).

Each builder returns an :class:`Instance`: literal CSR + constraint types + thresholds
(the arguments of ``afs_problem_create``), the run parameters BASELINE.json states
(B, steps, lr), the start point X0 ~ U[-1,1] in fp32, and optionally a planted
assignment and a fixed-variable mask.

BASELINE.json ``configs[i]`` -> :func:`config` (i); the same builders with smaller
sizes give the parity-test cases.  The synthetic instances stand in for the paper's
workloads (SAT Competition 2007 random 3-SAT; Ramsey / Costas PB
encodings, L100-L166), none of which is available here; see DESIGN.md.
"""
from __future__ import annotations

import hashlib
from dataclasses import dataclass, field
from typing import List, Optional, Sequence

import numpy as np

# constraint type codes == afs_ctype in include/afs.h (an interface constant, not arithmetic)
AFS_OR, AFS_XOR, AFS_AMO, AFS_EO, AFS_EK, AFS_NAE, AFS_CARD = range(7)
TYPE_NAMES = ("OR", "XOR", "AMO", "EO", "EK", "NAE", "CARD")

BASE_SEED = 2606066560  # + config index (reading G23)


@dataclass
class Instance:
    name: str
    n: int
    row_ptr: np.ndarray            # int64 [m+1]
    lits: np.ndarray               # int32 [nnz], signed 1-based
    types: np.ndarray              # int32 [m]
    k: np.ndarray                  # int32 [m]; EK: ==k, CARD: >=k, XOR: parity (1 = odd), else 0
    B: int = 0
    steps: int = 0
    lr: float = 0.1
    X0: Optional[np.ndarray] = None      # float32 [B, n]
    mask: Optional[np.ndarray] = None    # int8 [n]: 0 free, -1 fixed True, +1 fixed False
    plant: Optional[np.ndarray] = None   # int8 [n]: -1 True, +1 False
    seed: int = 0
    notes: dict = field(default_factory=dict)

    @property
    def m(self) -> int:
        return int(self.types.shape[0])

    @property
    def nnz(self) -> int:
        return int(self.lits.shape[0])

    def lengths(self) -> np.ndarray:
        return np.diff(self.row_ptr)

    def sha256(self) -> str:
        h = hashlib.sha256()
        for a in (self.row_ptr, self.lits, self.types, self.k, self.X0, self.mask):
            if a is not None:
                h.update(np.ascontiguousarray(a).tobytes())
        return h.hexdigest()

    def with_run(self, rng: Optional[np.random.Generator], B: int, steps: int, lr: float = 0.1) -> "Instance":
        """Draw X0 ~ U[-1,1] (fp32) from the instance's own generator stream (or ``rng``)."""
        if rng is None:
            rng = self.notes.pop("rng")
        self.B, self.steps, self.lr = int(B), int(steps), float(lr)
        self.X0 = rng.uniform(-1.0, 1.0, size=(B, self.n)).astype(np.float32)
        return self


# ----------------------------------------------------------------------------- helpers
def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(int(seed)))


def _distinct_rows(rng: np.random.Generator, n: int, m: int, L: int) -> np.ndarray:
    """m rows of L distinct variables each, uniform over [0, n)."""
    if L > n:
        raise ValueError("constraint longer than the variable count")
    v = rng.integers(0, n, size=(m, L), dtype=np.int64)
    while True:
        s = np.sort(v, axis=1)
        bad = np.nonzero((s[:, 1:] == s[:, :-1]).any(axis=1))[0]
        if bad.size == 0:
            return v
        v[bad] = rng.integers(0, n, size=(bad.size, L), dtype=np.int64)


def _signs(rng: np.random.Generator, shape) -> np.ndarray:
    """+1 (positive literal) or -1 (negated literal), each w.p. 1/2."""
    return (1 - 2 * rng.integers(0, 2, size=shape, dtype=np.int64)).astype(np.int64)


def _lit_true(vars_: np.ndarray, signs: np.ndarray, plant: np.ndarray) -> np.ndarray:
    """Boolean array: literal true under the plant (value sign*plant == -1 means True)."""
    return (signs * plant[vars_].astype(np.int64)) == -1


def true_counts(inst: Instance, assign: np.ndarray) -> np.ndarray:
    """Number of true literals per constraint under ``assign`` (int8/-1 = True). Instance bookkeeping only."""
    v = np.abs(inst.lits).astype(np.int64) - 1
    s = np.sign(inst.lits).astype(np.int64)
    t = ((s * assign[v].astype(np.int64)) == -1).astype(np.int64)
    c = np.concatenate([[0], np.cumsum(t)])
    return (c[inst.row_ptr[1:]] - c[inst.row_ptr[:-1]]).astype(np.int64)


def plant_satisfies(inst: Instance, assign: np.ndarray) -> np.ndarray:
    """Per-constraint truth of the defining predicate under ``assign`` (generator self-check)."""
    t = true_counts(inst, assign)
    L = inst.lengths()
    ty, k = inst.types, inst.k.astype(np.int64)
    out = np.zeros(inst.m, dtype=bool)
    out |= (ty == AFS_OR) & (t >= 1)
    out |= (ty == AFS_XOR) & ((t % 2) == (k % 2))
    out |= (ty == AFS_AMO) & (t <= 1)
    out |= (ty == AFS_EO) & (t == 1)
    out |= (ty == AFS_EK) & (t == k)
    out |= (ty == AFS_NAE) & (t > 0) & (t < L)
    out |= (ty == AFS_CARD) & (t >= k)
    return out


def _pack(name: str, n: int, rows: Sequence[np.ndarray], types: Sequence[int], ks: Sequence[int],
          plant: Optional[np.ndarray], seed: int) -> Instance:
    lens = np.fromiter((len(r) for r in rows), dtype=np.int64, count=len(rows))
    row_ptr = np.zeros(len(rows) + 1, dtype=np.int64)
    np.cumsum(lens, out=row_ptr[1:])
    lits = (np.concatenate(rows) if rows else np.zeros(0)).astype(np.int32)
    return Instance(name=name, n=int(n), row_ptr=row_ptr, lits=lits,
                    types=np.asarray(types, dtype=np.int32), k=np.asarray(ks, dtype=np.int32),
                    plant=None if plant is None else plant.astype(np.int8), seed=int(seed))


def _pack_fixed(name: str, n: int, vars_: np.ndarray, signs: np.ndarray, ctype: int, ks,
                plant: Optional[np.ndarray], seed: int) -> Instance:
    m, L = vars_.shape
    row_ptr = (np.arange(m + 1, dtype=np.int64) * L)
    lits = (signs * (vars_ + 1)).astype(np.int32).reshape(-1)
    k = np.broadcast_to(np.asarray(ks, dtype=np.int32), (m,)).copy()
    return Instance(name=name, n=int(n), row_ptr=row_ptr, lits=lits,
                    types=np.full(m, ctype, dtype=np.int32), k=k,
                    plant=None if plant is None else plant.astype(np.int8), seed=int(seed))


def concat(name: str, parts: List[Instance]) -> Instance:
    """Concatenate constraint lists over the same variable set (constraint ids keep part order)."""
    n = parts[0].n
    assert all(p.n == n for p in parts)
    lens = np.concatenate([p.lengths() for p in parts])
    row_ptr = np.zeros(lens.size + 1, dtype=np.int64)
    np.cumsum(lens, out=row_ptr[1:])
    return Instance(name=name, n=n, row_ptr=row_ptr,
                    lits=np.concatenate([p.lits for p in parts]).astype(np.int32),
                    types=np.concatenate([p.types for p in parts]).astype(np.int32),
                    k=np.concatenate([p.k for p in parts]).astype(np.int32),
                    plant=parts[0].plant, seed=parts[0].seed)


def _plant(rng: np.random.Generator, n: int) -> np.ndarray:
    return (1 - 2 * rng.integers(0, 2, size=n, dtype=np.int64)).astype(np.int8)


# ----------------------------------------------------------------------------- builders
def random_kcnf(seed: int, n: int, m: int, L: int = 3, name: str = "random_kcnf") -> Instance:
    """Uniform random L-CNF, not planted: L distinct variables, each sign +-1 w.p. 1/2 (configs[0])."""
    rng = _rng(seed)
    v = _distinct_rows(rng, n, m, L)
    s = _signs(rng, (m, L))
    inst = _pack_fixed(name, n, v, s, AFS_OR, 0, None, seed)
    inst.notes["rng"] = rng
    return inst


def _planted_clauses(rng, n, m, L, plant):
    v = _distinct_rows(rng, n, m, L)
    s = _signs(rng, (m, L))
    while True:  # resample whole clauses the plant falsifies (configs[3] wording)
        bad = np.nonzero(~_lit_true(v, s, plant).any(axis=1))[0]
        if bad.size == 0:
            return v, s
        v[bad] = _distinct_rows(rng, n, bad.size, L)
        s[bad] = _signs(rng, (bad.size, L))


def planted_kcnf(seed: int, n: int, m: int, L: int = 3, name: str = "planted_kcnf") -> Instance:
    """Planted random L-CNF: every clause satisfied by a uniform random plant (configs[3])."""
    rng = _rng(seed)
    plant = _plant(rng, n)
    v, s = _planted_clauses(rng, n, m, L, plant)
    inst = _pack_fixed(name, n, v, s, AFS_OR, 0, plant, seed)
    inst.notes["rng"] = rng
    return inst


def mixed_pb(seed: int, n: int, n_or: int, n_xor: int, n_eo: int, n_amo: int, n_card: int,
             or_len=(3, 5), xor_len=(3, 8), eo_len=(5, 20), amo_len=(5, 20), card_len=(10, 40),
             n_nae: int = 0, nae_len=(3, 6), n_ek: int = 0, ek_len=(4, 12),
             name: str = "mixed_pb") -> Instance:
    """Mixed symmetric PB, every constraint satisfied by the plant (configs[1]; reading G20).

    NAE / EK blocks are off in configs[1]; the parity tests switch them on to cover all seven types.
    """
    rng = _rng(seed)
    plant = _plant(rng, n)
    rows, types, ks = [], [], []

    def draw_len(lo_hi):
        return int(rng.integers(lo_hi[0], lo_hi[1] + 1))

    def draw_vars(L):
        return rng.choice(n, size=L, replace=False).astype(np.int64)

    for _ in range(n_or):            # OR: resample signs until >= 1 true literal
        L = draw_len(or_len); v = draw_vars(L)
        while True:
            s = _signs(rng, L)
            if _lit_true(v, s, plant).any():
                break
        rows.append(s * (v + 1)); types.append(AFS_OR); ks.append(0)
    for _ in range(n_xor):           # XOR: signs uniform, parity := the plant's
        L = draw_len(xor_len); v = draw_vars(L); s = _signs(rng, L)
        rows.append(s * (v + 1)); types.append(AFS_XOR); ks.append(int(_lit_true(v, s, plant).sum() % 2))
    for _ in range(n_eo):            # EO: one uniformly chosen position true under the plant
        L = draw_len(eo_len); v = draw_vars(L); pos = int(rng.integers(0, L))
        want_true = np.zeros(L, dtype=bool); want_true[pos] = True
        s = np.where(want_true, -1, 1) * plant[v].astype(np.int64)   # sign*plant = -1 iff true
        rows.append(s * (v + 1)); types.append(AFS_EO); ks.append(0)
    for _ in range(n_amo):           # AMO: 0 or 1 true literal, fair coin
        L = draw_len(amo_len); v = draw_vars(L)
        want_true = np.zeros(L, dtype=bool)
        if rng.integers(0, 2) == 1:
            want_true[int(rng.integers(0, L))] = True
        s = np.where(want_true, -1, 1) * plant[v].astype(np.int64)
        rows.append(s * (v + 1)); types.append(AFS_AMO); ks.append(0)
    for _ in range(n_card):          # CARD>=k: signs uniform (resample if count 0), k := min(U{1..L-1}, count)
        L = draw_len(card_len); v = draw_vars(L)
        while True:
            s = _signs(rng, L); cnt = int(_lit_true(v, s, plant).sum())
            if cnt > 0:
                break
        kk = min(int(rng.integers(1, L)), cnt)
        rows.append(s * (v + 1)); types.append(AFS_CARD); ks.append(kk)
    for _ in range(n_nae):           # NAE: resample signs until neither all-true nor all-false
        L = draw_len(nae_len); v = draw_vars(L)
        while True:
            s = _signs(rng, L); cnt = int(_lit_true(v, s, plant).sum())
            if 0 < cnt < L:
                break
        rows.append(s * (v + 1)); types.append(AFS_NAE); ks.append(0)
    for _ in range(n_ek):            # EK: signs uniform, k := the plant's count
        L = draw_len(ek_len); v = draw_vars(L); s = _signs(rng, L)
        rows.append(s * (v + 1)); types.append(AFS_EK); ks.append(int(_lit_true(v, s, plant).sum()))
    inst = _pack(name, n, rows, types, ks, plant, seed)
    inst.notes["rng"] = rng
    return inst


def xor_dup(seed: int, n: int, m: int, L: int = 3, name: str = "xor_dup") -> Instance:
    """Planted L-XOR-SAT, positive literals, every constraint appended once more (configs[2]; G21)."""
    rng = _rng(seed)
    plant = _plant(rng, n)
    v = _distinct_rows(rng, n, m, L)
    s = np.ones((m, L), dtype=np.int64)
    par = (_lit_true(v, s, plant).sum(axis=1) % 2).astype(np.int32)
    one = _pack_fixed(name, n, v, s, AFS_XOR, par, plant, seed)
    inst = concat(name, [one, one])      # constraint i+m is the copy of constraint i
    inst.notes["rng"] = rng
    return inst


def long_pb(seed: int, n: int, n_clauses: int, n_card: int, n_ek: int, long_len=(256, 1024),
            mask_frac: float = 0.5, name: str = "long_pb") -> Instance:
    """Planted 3-CNF plus long CARD>=k / EK with k := the plant's true count; a mask fixes
    ``mask_frac`` of the variables to the plant (configs[4]; G22)."""
    rng = _rng(seed)
    plant = _plant(rng, n)
    v3, s3 = _planted_clauses(rng, n, n_clauses, 3, plant)
    cnf = _pack_fixed(name, n, v3, s3, AFS_OR, 0, plant, seed)
    rows, types, ks = [], [], []
    for i in range(n_card + n_ek):
        is_card = i < n_card
        L = int(rng.integers(long_len[0], long_len[1] + 1))
        v = rng.choice(n, size=L, replace=False).astype(np.int64)
        while True:
            s = _signs(rng, L); cnt = int(_lit_true(v, s, plant).sum())
            if cnt > 0 or not is_card:
                break
        rows.append(s * (v + 1)); types.append(AFS_CARD if is_card else AFS_EK); ks.append(cnt)
    longs = _pack(name, n, rows, types, ks, plant, seed)
    inst = concat(name, [cnf, longs]) if rows else cnf
    n_fix = int(round(mask_frac * n))
    mask = np.zeros(n, dtype=np.int8)
    fixed = rng.permutation(n)[:n_fix]
    mask[fixed] = plant[fixed]
    inst.mask = mask
    inst.notes["rng"] = rng
    return inst


def tiny_mixed(seed: int, n: int = 10, m_each: int = 2, max_len: int = 6) -> Instance:
    """A few constraints of every type on few variables, NOT planted, arbitrary thresholds:
    for brute-force checks of the oracle (n small enough to enumerate corners)."""
    rng = _rng(seed)
    rows, types, ks = [], [], []
    for ty in range(7):
        for _ in range(m_each):
            lo = 2 if ty == AFS_NAE else 1
            L = int(rng.integers(lo, min(max_len, n) + 1))
            v = rng.choice(n, size=L, replace=False).astype(np.int64)
            s = _signs(rng, L)
            if ty == AFS_XOR:
                kk = int(rng.integers(0, 2))
            elif ty == AFS_EK:
                kk = int(rng.integers(0, L + 1))
            elif ty == AFS_CARD:
                kk = int(rng.integers(0, L + 2))
            else:
                kk = 0
            rows.append(s * (v + 1)); types.append(ty); ks.append(kk)
    inst = _pack("tiny_mixed", n, rows, types, ks, None, seed)
    inst.notes["rng"] = rng
    return inst


# ----------------------------------------------------------------------------- BASELINE.json configs
_CONFIG_NAMES = (
    "cfg0_random3cnf_n50",
    "cfg1_mixed_pb_n1000",
    "cfg2_xor3_dup_n2000",
    "cfg3_planted3cnf_n100k",
    "cfg4_long_pb_n5000",
)


def config_names():
    return _CONFIG_NAMES


def config(i: int, B: Optional[int] = None, steps: Optional[int] = None) -> Instance:
    """BASELINE.json ``configs[i]`` at full size (B / steps may be overridden for bounded samples;
    the instance and the first B rows of X0 do not depend on the override of ``steps``)."""
    seed = BASE_SEED + i
    if i == 0:
        inst = random_kcnf(seed, n=50, m=213, L=3, name=_CONFIG_NAMES[0]); b, st = 64, 200
    elif i == 1:
        inst = mixed_pb(seed, n=1000, n_or=3000, n_xor=200, n_eo=100, n_amo=100, n_card=50,
                        name=_CONFIG_NAMES[1]); b, st = 1024, 500
    elif i == 2:
        inst = xor_dup(seed, n=2000, m=1800, L=3, name=_CONFIG_NAMES[2]); b, st = 4096, 1000
    elif i == 3:
        inst = planted_kcnf(seed, n=100_000, m=420_000, L=3, name=_CONFIG_NAMES[3]); b, st = 256, 300
    elif i == 4:
        inst = long_pb(seed, n=5000, n_clauses=20_000, n_card=400, n_ek=100, name=_CONFIG_NAMES[4])
        b, st = 2048, 500
    else:
        raise ValueError("configs are 0..4")
    rng = inst.notes.pop("rng")
    inst.with_run(rng, b, st if steps is None else steps, lr=0.1)
    if B is not None and B != b:
        # a prefix (or tiling) of the same start points, so bounded samples are sub-batches of the full run
        reps = -(-B // b)
        inst.X0 = np.tile(inst.X0, (reps, 1))[:B].copy() if reps > 1 else inst.X0[:B].copy()
        inst.B = int(B)
    return inst

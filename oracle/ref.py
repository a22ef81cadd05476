"""ctypes wrapper around oracle/afs_oracle.c (numpy in, numpy out). TEST INFRASTRUCTURE ONLY.

Evaluators (argument ``evaluator``): 0 = A, the literal form  sum_i a_i e_i  with eq. (3) coefficients and the
O(L^2) ESP recurrence (L <= 62, refuses on ill-conditioning); 1 = B, count basis with the definitional
leave-one-out gradient; 2 = B with prefix/suffix tables (the one used at full size).
"""
from __future__ import annotations

import ctypes as C
from typing import Optional, Tuple

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        i32p, i64p, f64p, i8p = (C.POINTER(C.c_int32), C.POINTER(C.c_int64), C.POINTER(C.c_double),
                                 C.POINTER(C.c_int8))
        L.orc_pred.argtypes = [C.c_int] * 4
        L.orc_spectrum.argtypes = [C.c_int, C.c_int, C.c_int, i32p]
        L.orc_coeffs_eq3.argtypes = [C.c_int, C.c_int, C.c_int, f64p]
        L.orc_fe_A.argtypes = [C.c_int, C.c_int, C.c_int, f64p, f64p, f64p]
        L.orc_fe_B.argtypes = [C.c_int, C.c_int, C.c_int, f64p, f64p, f64p, C.c_int]
        inst = [C.c_int, C.c_int64, i64p, i32p, i32p, i32p]
        L.orc_eval_grad.argtypes = inst + [f64p, C.c_int, f64p, f64p, C.c_int, C.c_int]
        L.orc_round_count.argtypes = inst + [f64p, C.c_int, i8p, i32p]
        L.orc_pgd_run.argtypes = inst + [f64p, C.c_int, C.c_int, C.c_double, i8p, i8p, i32p, i32p,
                                         f64p, i32p, C.c_int, C.c_int]
        L.orc_pgd_run_conv.argtypes = inst + [f64p, C.c_int, C.c_int, C.c_double, i8p, C.c_double, i8p, i32p, i32p,
                                              i32p, i32p, f64p, C.c_int, C.c_int]
        L.orc_eval_grad_w.argtypes = inst + [f64p, f64p, C.c_int, f64p, f64p, f64p, C.c_int]
        L.orc_pgd_run_w.argtypes = inst + [f64p, f64p, C.c_int, C.c_int, C.c_double, i8p, i8p, i32p, i32p, C.c_int]
        L.orc_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _p(a: Optional[np.ndarray], ct):
    return None if a is None else a.ctypes.data_as(C.POINTER(ct))


def num_threads() -> int:
    return int(lib().orc_num_threads())


def spectrum(ctype: int, L: int, k: int = 0) -> np.ndarray:
    sp = np.zeros(L + 1, dtype=np.int32)
    if lib().orc_spectrum(ctype, L, k, _p(sp, C.c_int32)):
        raise ValueError("bad constraint")
    return sp


def coeffs_eq3(ctype: int, L: int, k: int = 0) -> np.ndarray:
    a = np.zeros(L + 1, dtype=np.float64)
    if lib().orc_coeffs_eq3(ctype, L, k, _p(a, C.c_double)):
        raise ValueError("bad constraint or L > 62")
    return a


def fe(ctype: int, k: int, y, evaluator: int = 2, want_grad: bool = True) -> Tuple[float, Optional[np.ndarray]]:
    """One constraint at literal values y (fp64). Returns (FE, dFE/dy)."""
    y = np.ascontiguousarray(y, dtype=np.float64)
    L = y.shape[0]
    out = C.c_double(0.0)
    g = np.zeros(L, dtype=np.float64) if want_grad else None
    if evaluator == 0:
        rc = lib().orc_fe_A(ctype, L, k, _p(y, C.c_double), C.byref(out), _p(g, C.c_double))
    else:
        rc = lib().orc_fe_B(ctype, L, k, _p(y, C.c_double), C.byref(out), _p(g, C.c_double), evaluator)
    if rc == 1:
        raise ArithmeticError("evaluator A refused: ill-conditioned literal form")
    if rc:
        raise ValueError("oracle error %d" % rc)
    return float(out.value), g


def _inst_args(inst):
    rp = np.ascontiguousarray(inst.row_ptr, dtype=np.int64)
    li = np.ascontiguousarray(inst.lits, dtype=np.int32)
    ty = np.ascontiguousarray(inst.types, dtype=np.int32)
    kk = np.ascontiguousarray(inst.k, dtype=np.int32)
    keep = (rp, li, ty, kk)
    return keep, [int(inst.n), int(ty.shape[0]), _p(rp, C.c_int64), _p(li, C.c_int32), _p(ty, C.c_int32),
                  _p(kk, C.c_int32)]


def eval_grad(inst, X, evaluator: int = 2, want_grad: bool = True, nthreads: int = 0):
    """F[B] and G[B,n] (fp64) at X[B,n]."""
    X = np.ascontiguousarray(X, dtype=np.float64)
    B, n = X.shape
    assert n == inst.n
    F = np.zeros(B, dtype=np.float64)
    G = np.zeros((B, n), dtype=np.float64) if want_grad else None
    keep, args = _inst_args(inst)
    rc = lib().orc_eval_grad(*args, _p(X, C.c_double), B, _p(F, C.c_double), _p(G, C.c_double),
                             evaluator, nthreads)
    if rc == 1:
        raise ArithmeticError("evaluator A refused: ill-conditioned literal form")
    if rc:
        raise ValueError("oracle error %d" % rc)
    return F, G


def round_count(inst, X, want_assign: bool = True):
    """Rounded assignment int8[B,n] (-1 True, +1 False) and satisfied counts int32[B]."""
    X = np.ascontiguousarray(X, dtype=np.float64)
    B, n = X.shape
    sat = np.zeros(B, dtype=np.int32)
    assign = np.zeros((B, n), dtype=np.int8) if want_assign else None
    keep, args = _inst_args(inst)
    if lib().orc_round_count(*args, _p(X, C.c_double), B, _p(assign, C.c_int8), _p(sat, C.c_int32)):
        raise ValueError("oracle error")
    return assign, sat


def pgd_run(inst, X0, steps: int, lr: float, mask=None, evaluator: int = 2, want_traj: bool = False,
            nthreads: int = 0):
    """Returns dict(X, best_assign, best_sat, best_step, sat_hist[, traj])."""
    X = np.array(X0, dtype=np.float64, order="C", copy=True)
    B, n = X.shape
    m8 = None if mask is None else np.ascontiguousarray(mask, dtype=np.int8)
    best_assign = np.zeros((B, n), dtype=np.int8)
    best_sat = np.zeros(B, dtype=np.int32)
    best_step = np.zeros(B, dtype=np.int32)
    sat_hist = np.zeros((steps + 1, B), dtype=np.int32)
    traj = np.zeros((steps + 1, B, n), dtype=np.float64) if want_traj else None
    keep, args = _inst_args(inst)
    rc = lib().orc_pgd_run(*args, _p(X, C.c_double), B, int(steps), float(lr), _p(m8, C.c_int8),
                           _p(best_assign, C.c_int8), _p(best_sat, C.c_int32), _p(best_step, C.c_int32),
                           _p(traj, C.c_double), _p(sat_hist, C.c_int32), evaluator, nthreads)
    if rc:
        raise ValueError("oracle error %d" % rc)
    out = dict(X=X, best_assign=best_assign, best_sat=best_sat, best_step=best_step, sat_hist=sat_hist)
    if want_traj:
        out["traj"] = traj
    return out


def pgd_run_conv(inst, X0, max_steps: int, lr: float, tol: float, mask=None, evaluator: int = 2, nthreads: int = 0):
    """PGD with per-restart convergence detection (orc_pgd_run_conv): a restart stops after the first step with
    max|dX| < tol.  Returns dict(X, best_assign, best_sat, best_step, conv_step, final_sat, final_F)."""
    X = np.array(X0, dtype=np.float64, order="C", copy=True)
    B, n = X.shape
    m8 = None if mask is None else np.ascontiguousarray(mask, dtype=np.int8)
    best_assign = np.zeros((B, n), dtype=np.int8)
    best_sat = np.zeros(B, dtype=np.int32)
    best_step = np.zeros(B, dtype=np.int32)
    conv_step = np.zeros(B, dtype=np.int32)
    final_sat = np.zeros(B, dtype=np.int32)
    final_F = np.zeros(B, dtype=np.float64)
    keep, args = _inst_args(inst)
    rc = lib().orc_pgd_run_conv(*args, _p(X, C.c_double), B, int(max_steps), float(lr), _p(m8, C.c_int8), float(tol),
                                _p(best_assign, C.c_int8), _p(best_sat, C.c_int32), _p(best_step, C.c_int32),
                                _p(conv_step, C.c_int32), _p(final_sat, C.c_int32), _p(final_F, C.c_double),
                                evaluator, nthreads)
    if rc:
        raise ValueError("oracle error %d" % rc)
    return dict(X=X, best_assign=best_assign, best_sat=best_sat, best_step=best_step, conv_step=conv_step,
                final_sat=final_sat, final_F=final_F)


def eval_grad_w(inst, weights, X, evaluator: int = 2, want_grad: bool = True, want_gm: bool = False):
    """Weighted objective F_w = sum_k w_k FE_k and its gradient (orc_eval_grad_w); optionally the per-constraint
    gradient magnitudes gm[k] = sum_b sum_j |dFE_k/dy_j| (unweighted).  Returns (F, G, GM)."""
    X = np.ascontiguousarray(X, dtype=np.float64)
    B, n = X.shape
    w = None if weights is None else np.ascontiguousarray(weights, dtype=np.float64)
    F = np.zeros(B, dtype=np.float64)
    G = np.zeros((B, n), dtype=np.float64) if want_grad else None
    GM = np.zeros(inst.m, dtype=np.float64) if want_gm else None
    keep, args = _inst_args(inst)
    rc = lib().orc_eval_grad_w(*args, _p(w, C.c_double), _p(X, C.c_double), B, _p(F, C.c_double), _p(G, C.c_double),
                               _p(GM, C.c_double), evaluator)
    if rc:
        raise ValueError("oracle error %d" % rc)
    return F, G, GM


def pgd_run_w(inst, weights, X0, steps: int, lr: float, mask=None, evaluator: int = 2):
    """PGD on the weighted objective (orc_pgd_run_w). Returns dict(X, best_assign, best_sat, best_step)."""
    X = np.array(X0, dtype=np.float64, order="C", copy=True)
    B, n = X.shape
    w = None if weights is None else np.ascontiguousarray(weights, dtype=np.float64)
    m8 = None if mask is None else np.ascontiguousarray(mask, dtype=np.int8)
    best_assign = np.zeros((B, n), dtype=np.int8)
    best_sat = np.zeros(B, dtype=np.int32)
    best_step = np.zeros(B, dtype=np.int32)
    keep, args = _inst_args(inst)
    rc = lib().orc_pgd_run_w(*args, _p(w, C.c_double), _p(X, C.c_double), B, int(steps), float(lr), _p(m8, C.c_int8),
                             _p(best_assign, C.c_int8), _p(best_sat, C.c_int32), _p(best_step, C.c_int32), evaluator)
    if rc:
        raise ValueError("oracle error %d" % rc)
    return dict(X=X, best_assign=best_assign, best_sat=best_sat, best_step=best_step)

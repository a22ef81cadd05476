"""Thin ctypes binding over the C ABI of include/afs.h -- argument marshalling only.

Every step of the path runs inside ``libafs_b200.so`` (hand-written CUDA); PyTorch is used for device memory and
streams and nothing else.  There is no CPU fallback: if the shared library is missing, cannot be loaded, or no CUDA
device is present, calls fail loudly.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libafs_b200.so")

AFS_OR, AFS_XOR, AFS_AMO, AFS_EO, AFS_EK, AFS_NAE, AFS_CARD = range(7)

EXPORTS = (
    "afs_problem_create", "afs_problem_destroy", "afs_coeffs", "afs_eval_grad", "afs_eval_grad_f64",
    "afs_round_count", "afs_round_count_f64", "afs_pgd_run", "afs_pgd_run_f64", "afs_pgd_run_host",
    "afs_problem_info", "afs_set_option", "afs_status_string", "afs_abi_version", "afs_last_error_message",
    "afs_profile_read", "afs_profile_flops", "afs_fp32_fma_peak", "afs_pgd_run_conv", "afs_pgd_run_conv_f64", "afs_pgd_run_masks", "afs_pgd_run_masks_f64", "afs_problem_create_w", "afs_constraint_grad_l1", "afs_constraint_grad_l1_f64",
    "afs_round_count_static",
)

_lib = None


class AfsError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = int(status)
        msg = lib().afs_status_string(status).decode()
        detail = lib().afs_last_error_message().decode() if status == 7 else ""
        super().__init__("%s: %s (status %d)%s" % (where, msg, status, " -- " + detail if detail else ""))


def lib():
    """Load libafs_b200.so (built in-tree by ``paper_2606_06656_b200.build``). Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(
            "%s not found: build it with `python -m paper_2606_06656_b200.build` (nvcc, sm_100a). "
            "There is no CPU fallback." % LIB_PATH)
    L = C.CDLL(LIB_PATH)
    vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
    L.afs_problem_create.argtypes = [i32, i32, vp, vp, vp, vp, i32, C.POINTER(vp)]
    L.afs_problem_create.restype = C.c_int
    L.afs_problem_create_w.argtypes = [i32, i32, vp, vp, vp, vp, vp, i32, C.POINTER(vp)]
    L.afs_problem_create_w.restype = C.c_int
    L.afs_problem_destroy.argtypes = [vp]
    L.afs_problem_destroy.restype = None
    L.afs_coeffs.argtypes = [i32, i32, i32, vp]
    L.afs_coeffs.restype = C.c_int
    for name in ("afs_eval_grad", "afs_eval_grad_f64"):
        f = getattr(L, name); f.argtypes = [vp, vp, i32, vp, vp, vp]; f.restype = C.c_int
    for name in ("afs_round_count", "afs_round_count_f64", "afs_round_count_static"):
        f = getattr(L, name); f.argtypes = [vp, vp, i32, vp, vp, vp]; f.restype = C.c_int
    for name in ("afs_constraint_grad_l1", "afs_constraint_grad_l1_f64"):
        f = getattr(L, name); f.argtypes = [vp, vp, i32, vp, vp]; f.restype = C.c_int
    L.afs_pgd_run.argtypes = [vp, vp, i32, i32, C.c_float, vp, vp, vp, vp, vp]
    L.afs_pgd_run.restype = C.c_int
    L.afs_pgd_run_f64.argtypes = [vp, vp, i32, i32, C.c_double, vp, vp, vp, vp, vp]
    L.afs_pgd_run_f64.restype = C.c_int
    L.afs_pgd_run_conv.argtypes = [vp, vp, i32, i32, C.c_float, vp, C.c_float, vp, vp, vp, vp, vp, vp, vp]
    L.afs_pgd_run_conv.restype = C.c_int
    L.afs_pgd_run_conv_f64.argtypes = [vp, vp, i32, i32, C.c_double, vp, C.c_double, vp, vp, vp, vp, vp, vp, vp]
    L.afs_pgd_run_conv_f64.restype = C.c_int
    L.afs_pgd_run_masks.argtypes = [vp, vp, i32, i32, C.c_float, vp, vp, vp, vp, vp]
    L.afs_pgd_run_masks.restype = C.c_int
    L.afs_pgd_run_masks_f64.argtypes = [vp, vp, i32, i32, C.c_double, vp, vp, vp, vp, vp]
    L.afs_pgd_run_masks_f64.restype = C.c_int
    L.afs_pgd_run_host.argtypes = [vp, vp, i32, i32, C.c_float, vp, vp, vp, vp, vp]
    L.afs_pgd_run_host.restype = C.c_int
    L.afs_problem_info.argtypes = [vp, i32]
    L.afs_problem_info.restype = i64
    L.afs_set_option.argtypes = [vp, i32, i64]
    L.afs_set_option.restype = C.c_int
    L.afs_profile_read.argtypes = [vp, vp, vp, i32]
    L.afs_profile_read.restype = C.c_int
    L.afs_profile_flops.argtypes = [vp, vp, i32]
    L.afs_profile_flops.restype = C.c_int
    L.afs_fp32_fma_peak.argtypes = [i32, vp]
    L.afs_fp32_fma_peak.restype = C.c_int
    L.afs_status_string.argtypes = [C.c_int]
    L.afs_status_string.restype = C.c_char_p
    L.afs_abi_version.restype = i32
    L.afs_last_error_message.restype = C.c_char_p
    _lib = L
    return L


def _chk(status: int, where: str):
    if status != 0:
        raise AfsError(status, where)


def coeffs(ctype: int, L: int, k: int = 0) -> np.ndarray:
    """afs_coeffs: a_0..a_L (fp64, host)."""
    a = np.zeros(L + 1, dtype=np.float64)
    _chk(lib().afs_coeffs(ctype, L, k, a.ctypes.data), "afs_coeffs")
    return a


def fp32_fma_peak(device: int = 0) -> float:
    """afs_fp32_fma_peak: measured plain-FP32 FMA throughput of the device, TFLOP/s."""
    v = C.c_double(0.0)
    _chk(lib().afs_fp32_fma_peak(int(device), C.byref(v)), "afs_fp32_fma_peak")
    return float(v.value)


def _torch():
    import torch
    return torch


def _stream_ptr(device) -> int:
    torch = _torch()
    return int(torch.cuda.current_stream(device).cuda_stream)


class Problem:
    """afs_problem handle. Arrays in, torch CUDA tensors out; layouts are those of include/afs.h ([B, n] row-major)."""

    INFO = {"n_vars": 0, "n_cons": 1, "nnz": 2, "n_pull": 3, "n_med": 4, "n_long": 5, "scratch_slots": 6,
            "launches": 7, "workspace_bytes": 8, "resident": 9}

    def __init__(self, n_vars: int, row_ptr, lits, types, k, device: int = 0, weights=None):
        self._h = C.c_void_p(None)
        rp = np.ascontiguousarray(row_ptr, dtype=np.int64)
        li = np.ascontiguousarray(lits, dtype=np.int32)
        ty = np.ascontiguousarray(types, dtype=np.int32)
        kk = np.ascontiguousarray(k, dtype=np.int32)
        if rp.ndim != 1 or rp.shape[0] != ty.shape[0] + 1 or kk.shape != ty.shape:
            raise ValueError("row_ptr / types / k shapes disagree")
        if rp.shape[0] and li.shape[0] != int(rp[-1]):
            raise ValueError("lits length != row_ptr[-1]")
        self.n, self.m, self.nnz = int(n_vars), int(ty.shape[0]), int(li.shape[0])
        self.device = int(device)
        h = C.c_void_p(None)
        if weights is None:
            _chk(lib().afs_problem_create(self.n, self.m, rp.ctypes.data, li.ctypes.data, ty.ctypes.data,
                                          kk.ctypes.data, self.device, C.byref(h)), "afs_problem_create")
        else:
            ww = np.ascontiguousarray(weights, dtype=np.float32)
            if ww.shape != ty.shape:
                raise ValueError("weights must have one entry per constraint")
            _chk(lib().afs_problem_create_w(self.n, self.m, rp.ctypes.data, li.ctypes.data, ty.ctypes.data,
                                            kk.ctypes.data, ww.ctypes.data, self.device, C.byref(h)), "afs_problem_create_w")
        self._h = h

    @classmethod
    def from_instance(cls, inst, device: int = 0, weights=None) -> "Problem":
        return cls(inst.n, inst.row_ptr, inst.lits, inst.types, inst.k, device, weights=weights)

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().afs_problem_destroy(self._h)
            self._h = C.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def info(self, what: str) -> int:
        return int(lib().afs_problem_info(self._h, self.INFO[what]))

    def set_option(self, what: int, value: int):
        _chk(lib().afs_set_option(self._h, what, value), "afs_set_option")

    KERNEL_CLASSES = (["resident", "var", "sat_pull", "cmed", "med0", "long_scan", "glong", "med3", "med4"] +
                      ["long1", "long_lane8", "long3", "long_lane32", "long5", "long_lane16", "long7", "long8", "long9", "boundary"])

    def profile_read(self):
        """afs_profile_read: {class name: (milliseconds, launches)} of the last pgd_run, non-empty classes only."""
        ms = np.zeros(len(self.KERNEL_CLASSES), dtype=np.float64)
        cnt = np.zeros(len(self.KERNEL_CLASSES), dtype=np.int64)
        _chk(lib().afs_profile_read(self._h, ms.ctypes.data, cnt.ctypes.data, len(ms)), "afs_profile_read")
        return {k: (float(m), int(c)) for k, m, c in zip(self.KERNEL_CLASSES, ms, cnt) if c}

    def profile_flops(self):
        """afs_profile_flops: {class name: state-dependent algorithmic flops of the launches last read}, non-zero only."""
        fl = np.zeros(len(self.KERNEL_CLASSES), dtype=np.float64)
        _chk(lib().afs_profile_flops(self._h, fl.ctypes.data, len(fl)), "afs_profile_flops")
        return {k: float(v) for k, v in zip(self.KERNEL_CLASSES, fl) if v}

    # ------------------------------------------------------------------ helpers
    def _dev(self):
        return _torch().device("cuda", self.device)

    def _check_X(self, X, dtype):
        torch = _torch()
        if not (isinstance(X, torch.Tensor) and X.is_cuda and X.dtype == dtype and X.dim() == 2
                and X.shape[1] == self.n and X.is_contiguous() and X.device.index == self.device):
            raise ValueError("X must be a contiguous CUDA %s tensor [B, %d] on device %d" % (dtype, self.n, self.device))

    # ------------------------------------------------------------------ entry points
    def eval_grad(self, X, want_F: bool = True, want_G: bool = True):
        """afs_eval_grad / afs_eval_grad_f64 (chosen by X.dtype). Returns (F[B] or None, G[B,n] or None)."""
        torch = _torch()
        f64 = X.dtype == torch.float64
        self._check_X(X, torch.float64 if f64 else torch.float32)
        B = X.shape[0]
        F = torch.empty(B, dtype=X.dtype, device=X.device) if want_F else None
        G = torch.empty_like(X) if want_G else None
        fn = lib().afs_eval_grad_f64 if f64 else lib().afs_eval_grad
        _chk(fn(self._h, X.data_ptr(), B, F.data_ptr() if want_F else None, G.data_ptr() if want_G else None,
                _stream_ptr(X.device)), "afs_eval_grad")
        return F, G

    def constraint_grad_l1(self, X):
        """afs_constraint_grad_l1 / _f64: gm[n_cons] = sum_b sum_j |dFE_k/dy_j(X_b)| (unweighted)."""
        torch = _torch()
        f64 = X.dtype == torch.float64
        self._check_X(X, torch.float64 if f64 else torch.float32)
        gm = torch.empty(self.m, dtype=X.dtype, device=X.device)
        fn = lib().afs_constraint_grad_l1_f64 if f64 else lib().afs_constraint_grad_l1
        _chk(fn(self._h, X.data_ptr(), X.shape[0], gm.data_ptr(), _stream_ptr(X.device)), "afs_constraint_grad_l1")
        return gm

    def round_count(self, X, want_assign: bool = True):
        """afs_round_count. Returns (assign int8[B,n] or None, sat int32[B])."""
        torch = _torch()
        f64 = X.dtype == torch.float64
        self._check_X(X, torch.float64 if f64 else torch.float32)
        B = X.shape[0]
        sat = torch.empty(B, dtype=torch.int32, device=X.device)
        assign = torch.empty((B, self.n), dtype=torch.int8, device=X.device) if want_assign else None
        fn = lib().afs_round_count_f64 if f64 else lib().afs_round_count
        _chk(fn(self._h, X.data_ptr(), B, assign.data_ptr() if want_assign else None, sat.data_ptr(),
                _stream_ptr(X.device)), "afs_round_count")
        return assign, sat

    def round_count_static(self, X, assign=None, sat=None):
        """afs_round_count_static: round and count without any device allocation inside the library call.

        For callers that cannot allocate on the device when they call (all of HBM already owned by a pool, a thread that
        cannot take cudaMalloc's device-wide synchronisation, a host that forbids allocations after set-up): the
        library's working memory is a fixed 16 MiB array inside the library image, so (n, B) must satisfy
        256-aligned(4 Bp) + 4 n Bp <= 16 MiB or AfsError(status 9) is raised.  Pass preallocated ``assign`` int8[B,n]
        and ``sat`` int32[B] to keep this wrapper allocation-free too (they are created here only when left out;
        ``assign=False`` skips the assignment).  One array per GPU is shared by all calls: calls that overlap on the
        GPU race.  Returns (assign or None, sat), bit-identical to ``round_count``."""
        torch = _torch()
        self._check_X(X, torch.float32)
        B = X.shape[0]
        if sat is None:
            sat = torch.empty(B, dtype=torch.int32, device=X.device)
        if assign is None:
            assign = torch.empty((B, self.n), dtype=torch.int8, device=X.device)
        elif assign is False:
            assign = None
        _chk(lib().afs_round_count_static(self._h, X.data_ptr(), B, assign.data_ptr() if assign is not None else None,
                                          sat.data_ptr(), _stream_ptr(X.device)), "afs_round_count_static")
        return assign, sat

    def pgd_run(self, X, steps: int, lr: float, mask=None, out=None):
        """afs_pgd_run / _f64, in place on X (device). Returns dict(X, best_assign, best_sat, best_step).

        ``out`` may carry preallocated ``best_assign`` / ``best_sat`` / ``best_step`` tensors (bench.py reuses them)."""
        torch = _torch()
        f64 = X.dtype == torch.float64
        self._check_X(X, torch.float64 if f64 else torch.float32)
        B = X.shape[0]
        if mask is not None:
            if not (mask.is_cuda and mask.dtype == torch.int8 and mask.numel() == self.n and mask.is_contiguous()):
                raise ValueError("mask must be a contiguous CUDA int8 tensor [n]")
        out = out or {}
        ba = out.get("best_assign")
        bs = out.get("best_sat")
        bt = out.get("best_step")
        if ba is None:
            ba = torch.empty((B, self.n), dtype=torch.int8, device=X.device)
        if bs is None:
            bs = torch.empty(B, dtype=torch.int32, device=X.device)
        if bt is None:
            bt = torch.empty(B, dtype=torch.int32, device=X.device)
        fn = lib().afs_pgd_run_f64 if f64 else lib().afs_pgd_run
        _chk(fn(self._h, X.data_ptr(), B, int(steps), float(lr), mask.data_ptr() if mask is not None else None,
                ba.data_ptr(), bs.data_ptr(), bt.data_ptr(), _stream_ptr(X.device)), "afs_pgd_run")
        return dict(X=X, best_assign=ba, best_sat=bs, best_step=bt)

    def pgd_run_conv(self, X, max_steps: int, lr: float, tol: float, mask=None):
        """afs_pgd_run_conv / _f64, in place on X. Returns dict(X, best_assign, best_sat, best_step, conv_step,
        final_sat, final_F)."""
        torch = _torch()
        f64 = X.dtype == torch.float64
        self._check_X(X, torch.float64 if f64 else torch.float32)
        B = X.shape[0]
        if mask is not None and not (mask.is_cuda and mask.dtype == torch.int8 and mask.numel() == self.n):
            raise ValueError("mask must be a contiguous CUDA int8 tensor [n]")
        ba = torch.empty((B, self.n), dtype=torch.int8, device=X.device)
        i32 = lambda: torch.empty(B, dtype=torch.int32, device=X.device)
        bs, bt, cs, fs = i32(), i32(), i32(), i32()
        fF = torch.empty(B, dtype=X.dtype, device=X.device)
        fn = lib().afs_pgd_run_conv_f64 if f64 else lib().afs_pgd_run_conv
        _chk(fn(self._h, X.data_ptr(), B, int(max_steps), float(lr), mask.data_ptr() if mask is not None else None,
                float(tol), ba.data_ptr(), bs.data_ptr(), bt.data_ptr(), cs.data_ptr(), fs.data_ptr(), fF.data_ptr(),
                _stream_ptr(X.device)), "afs_pgd_run_conv")
        return dict(X=X, best_assign=ba, best_sat=bs, best_step=bt, conv_step=cs, final_sat=fs, final_F=fF)

    def pgd_run_masks(self, X, steps: int, lr: float, masks):
        """afs_pgd_run_masks / _f64: masks is a CUDA int8 tensor [B, n], one partial assignment per restart."""
        torch = _torch()
        f64 = X.dtype == torch.float64
        self._check_X(X, torch.float64 if f64 else torch.float32)
        B = X.shape[0]
        if not (masks.is_cuda and masks.dtype == torch.int8 and tuple(masks.shape) == (B, self.n) and masks.is_contiguous()):
            raise ValueError("masks must be a contiguous CUDA int8 tensor [B, n]")
        ba = torch.empty((B, self.n), dtype=torch.int8, device=X.device)
        bs = torch.empty(B, dtype=torch.int32, device=X.device)
        bt = torch.empty(B, dtype=torch.int32, device=X.device)
        fn = lib().afs_pgd_run_masks_f64 if f64 else lib().afs_pgd_run_masks
        _chk(fn(self._h, X.data_ptr(), B, int(steps), float(lr), masks.data_ptr(), ba.data_ptr(), bs.data_ptr(),
                bt.data_ptr(), _stream_ptr(X.device)), "afs_pgd_run_masks")
        return dict(X=X, best_assign=ba, best_sat=bs, best_step=bt)

    def pgd_run_host(self, X, steps: int, lr: float, mask=None, out=None):
        """afs_pgd_run_host: X float32 [B,n] HOST tensor/array (pinned recommended), updated in place; H2D and D2H
        copies happen inside the call. Returns dict of host tensors."""
        torch = _torch()
        if isinstance(X, np.ndarray):
            X = torch.from_numpy(X)
        if X.is_cuda or X.dtype != torch.float32 or X.dim() != 2 or X.shape[1] != self.n or not X.is_contiguous():
            raise ValueError("X must be a contiguous host float32 tensor [B, n]")
        B = X.shape[0]
        if mask is not None:
            if isinstance(mask, np.ndarray):
                mask = torch.from_numpy(np.ascontiguousarray(mask, dtype=np.int8))
            if mask.is_cuda or mask.dtype != torch.int8 or mask.numel() != self.n:
                raise ValueError("mask must be a host int8 tensor [n]")
        out = out or {}
        ba = out.get("best_assign")
        bs = out.get("best_sat")
        bt = out.get("best_step")
        if ba is None:
            ba = torch.empty((B, self.n), dtype=torch.int8)
        if bs is None:
            bs = torch.empty(B, dtype=torch.int32)
        if bt is None:
            bt = torch.empty(B, dtype=torch.int32)
        _chk(lib().afs_pgd_run_host(self._h, X.data_ptr(), B, int(steps), float(lr),
                                    mask.data_ptr() if mask is not None else None, ba.data_ptr(), bs.data_ptr(),
                                    bt.data_ptr(), _stream_ptr(self._dev())), "afs_pgd_run_host")
        return dict(X=X, best_assign=ba, best_sat=bs, best_step=bt)

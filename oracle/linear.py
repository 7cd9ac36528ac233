"""ctypes binding of oracle/linear_oracle.c (TEST INFRASTRUCTURE, not product): the paper's linear objective
(Eq.(4)/(5)) by brute force.  Arithmetic lives in the C file; this file only marshals."""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "linear_oracle.c")
# ORACLE_SANITIZE=1 builds a separate library with AddressSanitizer + UndefinedBehaviorSanitizer (the test process must
# then run with LD_PRELOAD=$(gcc -print-file-name=libasan.so); see profiles/r2_sanitizers.md).  Build plumbing only.
_SAN = bool(os.environ.get("ORACLE_SANITIZE"))
_OUT = os.path.join(_HERE, "_build", "liblinorc_san.so" if _SAN else "liblinorc.so")
_lock = threading.Lock()
_lib = None

PARAM_NAMES = ("lambda_f", "lambda_c", "lambda_l", "lambda_ld", "beta", "effort")


def build(force: bool = False) -> str:
    os.makedirs(os.path.dirname(_OUT), exist_ok=True)
    if force or not os.path.exists(_OUT) or os.path.getmtime(_OUT) < os.path.getmtime(_SRC):
        tmp = _OUT + f".{os.getpid()}.tmp"
        san = ["-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer", "-g"] if _SAN else []
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-shared", "-fPIC", "-Wall", "-Wextra", *san,
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _OUT)
    return _OUT


class _Batch(C.Structure):
    _fields_ = [("R", C.c_int32), ("node_off", C.c_void_p), ("opt_off", C.c_void_p), ("pred_mask", C.c_void_p),
                ("vuln", C.c_void_p), ("tau", C.c_void_p), ("q", C.c_void_p), ("cost", C.c_void_p)]


class _Params(C.Structure):
    _fields_ = [(n, C.c_double) for n in PARAM_NAMES]


class _Result(C.Structure):
    _fields_ = [("plan_idx", C.c_void_p), ("choice", C.c_void_p), ("J", C.c_void_p), ("T", C.c_void_p),
                ("Dtau", C.c_void_p), ("runner_J", C.c_void_p), ("status", C.c_void_p)]


def lib():
    global _lib
    with _lock:
        if _lib is None:
            l = C.CDLL(build())
            l.ln_compile.restype = C.c_int
            l.ln_compile.argtypes = [C.POINTER(_Batch), C.POINTER(_Params), C.c_int, C.c_void_p, C.POINTER(_Result)]
            l.ln_score.restype = C.c_int
            l.ln_score.argtypes = [C.POINTER(_Batch), C.c_int, C.POINTER(_Params), C.c_double, C.c_void_p,
                                   C.POINTER(C.c_double), C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
            l.ln_reach_weights.restype = None
            l.ln_reach_weights.argtypes = [C.c_int, C.c_void_p, C.c_double, C.c_double, C.c_void_p]
            _lib = l
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _cbatch(batch, cost):
    keep = dict(node_off=np.ascontiguousarray(batch.node_off, np.int32), opt_off=np.ascontiguousarray(batch.opt_off, np.int32),
                pred_mask=np.ascontiguousarray(batch.pred_mask, np.uint32), vuln=np.ascontiguousarray(batch.vuln, np.float32),
                tau=np.ascontiguousarray(batch.lat_us, np.int32), q=np.ascontiguousarray(batch.acc, np.float32),
                cost=np.ascontiguousarray(cost, np.float32))
    assert keep["cost"].size == keep["q"].size
    return _Batch(batch.R, *[_p(keep[k]) for k in ("node_off", "opt_off", "pred_mask", "vuln", "tau", "q", "cost")]), keep


def _cparams(params: dict) -> _Params:
    return _Params(*[float(params[n]) for n in PARAM_NAMES])


def compile(batch, cost, params: dict, levels) -> dict:
    """Best plan per (request, level) under J_L (Eq.(5)); batch.lat_us = tau, batch.acc = q, batch.vuln = v."""
    cb, keep = _cbatch(batch, cost)
    lv = np.ascontiguousarray(levels, np.float64)
    L = lv.size
    n = batch.R * L
    out = dict(plan_idx=np.zeros(n, np.uint64), choice=np.zeros(n * 16, np.uint8), J=np.zeros(n, np.float64),
               T=np.zeros(n, np.int64), Dtau=np.zeros(n, np.int64), runner_J=np.zeros(n, np.float64),
               status=np.zeros(n, np.uint8))
    res = _Result(*[_p(out[k]) for k in ("plan_idx", "choice", "J", "T", "Dtau", "runner_J", "status")])
    cp = _cparams(params)
    rc = lib().ln_compile(C.byref(cb), C.byref(cp), L, _p(lv), C.byref(res))
    assert rc == 0, rc
    return out


def score(batch, cost, params: dict, r: int, level: float, choice) -> dict:
    cb, keep = _cbatch(batch, cost)
    ch = np.ascontiguousarray(choice, np.uint8)
    J, T, D = C.c_double(), C.c_int64(), C.c_int64()
    cp = _cparams(params)
    st = lib().ln_score(C.byref(cb), r, C.byref(cp), float(level), _p(ch), C.byref(J), C.byref(T), C.byref(D))
    return dict(status=st, J=J.value, T=T.value, Dtau=D.value)


def reach_weights(pred_masks, beta: float, effort: float) -> np.ndarray:
    pm = np.ascontiguousarray(pred_masks, np.uint32)
    rho = np.zeros(pm.size, np.float64)
    lib().ln_reach_weights(pm.size, _p(pm), float(beta), float(effort), _p(rho))
    return rho

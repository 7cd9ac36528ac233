"""ctypes binding of oracle/dyplan_oracle.c (TEST INFRASTRUCTURE, not product).

Builds ``oracle/_build/liborc.so`` with gcc on first use.  Everything here takes the numpy
``Batch`` / ``Workload`` of ``tests/support/workloads.py`` (the shared seeded input generator) and
returns plain dicts of numpy arrays.  Arithmetic lives in the C file; this file only marshals.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dyplan_oracle.c")
# ORACLE_SANITIZE=1 builds a separate library with AddressSanitizer + UndefinedBehaviorSanitizer (the test process must
# then run with LD_PRELOAD=$(gcc -print-file-name=libasan.so); see profiles/r2_sanitizers.md).  Build plumbing only.
_SAN = bool(os.environ.get("ORACLE_SANITIZE"))
_OUT = os.path.join(_HERE, "_build", "liborc_san.so" if _SAN else "liborc.so")
_lock = threading.Lock()
_lib = None

ST_OK, ST_INFEASIBLE, ST_INVALID, ST_TOO_LARGE = 0, 1, 2, 3


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2 -fopenmp). Idempotent."""
    os.makedirs(os.path.dirname(_OUT), exist_ok=True)
    if force or not os.path.exists(_OUT) or os.path.getmtime(_OUT) < os.path.getmtime(_SRC):
        tmp = _OUT + f".{os.getpid()}.tmp"
        san = ["-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer", "-g"] if _SAN else []
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-shared", "-fPIC", "-Wall", "-Wextra", *san,
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _OUT)
    return _OUT


class _Batch(C.Structure):
    _fields_ = [("R", C.c_int32), ("B", C.c_int32), ("M", C.c_int32),
                ("node_off", C.c_void_p), ("opt_off", C.c_void_p), ("pred_mask", C.c_void_p),
                ("vuln", C.c_void_p), ("lat_us", C.c_void_p), ("acc", C.c_void_p), ("demand", C.c_void_p),
                ("backend", C.c_void_p), ("model", C.c_void_p), ("slo_us", C.c_void_p), ("cap", C.c_void_p)]


class _Result(C.Structure):
    _fields_ = [("plan_idx", C.c_void_p), ("choice", C.c_void_p), ("corr", C.c_void_p), ("lat", C.c_void_p),
                ("dem", C.c_void_p), ("dom_model", C.c_void_p), ("status", C.c_void_p),
                ("runner_idx", C.c_void_p), ("runner_corr", C.c_void_p), ("n_feasible", C.c_void_p)]


def lib():
    global _lib
    with _lock:
        if _lib is None:
            l = C.CDLL(build())
            l.orc_compile.restype = C.c_int
            l.orc_compile.argtypes = [C.POINTER(_Batch), C.c_int, C.c_void_p, C.c_int, C.c_int, C.POINTER(_Result)]
            l.orc_replan.restype = C.c_int
            l.orc_replan.argtypes = [C.POINTER(_Batch), C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint32, C.c_int,
                                     C.c_int, C.POINTER(_Result)]
            l.orc_score.restype = C.c_int
            l.orc_score.argtypes = [C.POINTER(_Batch), C.c_int, C.c_void_p, C.c_void_p, C.c_uint32,
                                    C.POINTER(C.c_double), C.POINTER(C.c_int64), C.c_void_p,
                                    C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.POINTER(C.c_uint64)]
            l.orc_select.restype = C.c_int
            l.orc_select.argtypes = [C.POINTER(_Batch), C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                     C.c_void_p, C.c_void_p, C.c_void_p]
            l.orc_num_threads.restype = C.c_int
            _lib = l
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _cbatch(b):
    keep = [np.ascontiguousarray(b.node_off, np.int32), np.ascontiguousarray(b.opt_off, np.int32),
            np.ascontiguousarray(b.pred_mask, np.uint32), np.ascontiguousarray(b.vuln, np.float32),
            np.ascontiguousarray(b.lat_us, np.int32), np.ascontiguousarray(b.acc, np.float32),
            np.ascontiguousarray(b.demand, np.int32), np.ascontiguousarray(b.backend, np.uint8),
            np.ascontiguousarray(b.model, np.uint8), np.ascontiguousarray(b.slo_us, np.int32),
            None if b.cap is None else np.ascontiguousarray(b.cap, np.int32)]
    cb = _Batch(b.R, b.B, b.M, *[_p(a) for a in keep])
    return cb, keep


def _alloc_result(nrec: int, B: int):
    out = dict(
        plan_idx=np.full(nrec, np.iinfo(np.uint64).max, np.uint64), choice=np.full((nrec, 16), 0xFF, np.uint8),
        corr=np.full(nrec, -1.0, np.float64), lat=np.full(nrec, 2**31 - 1, np.int64),
        dem=np.zeros((nrec, B), np.int64), dom_model=np.full(nrec, 0xFF, np.uint8),
        status=np.full(nrec, 255, np.uint8), runner_idx=np.full(nrec, np.iinfo(np.uint64).max, np.uint64),
        runner_corr=np.full(nrec, -1.0, np.float64), n_feasible=np.zeros(nrec, np.uint64))
    res = _Result(*[_p(out[k]) for k in ("plan_idx", "choice", "corr", "lat", "dem", "dom_model", "status",
                                         "runner_idx", "runner_corr", "n_feasible")])
    return out, res


def compile(batch, L: int, mult_pm, r_begin: int = 0, r_end: int | None = None) -> dict:
    """Best plan per (request, level); records of requests outside [r_begin, r_end) keep status 255."""
    r_end = batch.R if r_end is None else r_end
    cb, keep = _cbatch(batch)
    mult = np.ascontiguousarray(mult_pm, np.int32)
    assert mult.size == L * batch.B
    out, res = _alloc_result(batch.R * L, batch.B)
    rc = lib().orc_compile(C.byref(cb), L, _p(mult), r_begin, r_end, C.byref(res))
    assert rc == 0, rc
    return out


def replan(batch, dispatched_mask, fixed_choice, live_mult_pm, flags: int = 0, r_begin: int = 0,
           r_end: int | None = None) -> dict:
    r_end = batch.R if r_end is None else r_end
    cb, keep = _cbatch(batch)
    dm = np.ascontiguousarray(dispatched_mask, np.uint32)
    fc = np.ascontiguousarray(fixed_choice, np.uint8)
    lm = np.ascontiguousarray(live_mult_pm, np.int32)
    assert dm.size == batch.R and fc.size == batch.NN and lm.size == batch.R * batch.B
    out, res = _alloc_result(batch.R, batch.B)
    rc = lib().orc_replan(C.byref(cb), _p(dm), _p(fc), _p(lm), flags, r_begin, r_end, C.byref(res))
    assert rc == 0, rc
    return out


def run(w, r_begin: int = 0, r_end: int | None = None) -> dict:
    """Dispatch on the workload kind."""
    if w.kind == "compile":
        return compile(w.batch, w.L, w.mult_pm, r_begin, r_end)
    return replan(w.batch, w.dispatched_mask, w.fixed_choice, w.live_mult_pm, w.flags, r_begin, r_end)


def score(batch, r: int, mult_pm_B, choice, skip_mask: int = 0) -> dict:
    """(C, T, D_b, feasible, dominant model, canonical idx) of one plan of request r under one multiplier vector."""
    cb, keep = _cbatch(batch)
    mult = np.ascontiguousarray(mult_pm_B, np.int32)
    ch = np.ascontiguousarray(choice, np.uint8)
    Cv, T, f, dm, idx = C.c_double(), C.c_int64(), C.c_int32(), C.c_int32(), C.c_uint64()
    D = np.zeros(batch.B, np.int64)
    st = lib().orc_score(C.byref(cb), r, _p(mult), _p(ch), skip_mask, C.byref(Cv), C.byref(T), _p(D), C.byref(f),
                         C.byref(dm), C.byref(idx))
    return dict(status=st, corr=Cv.value, lat=T.value, dem=D, feasible=bool(f.value), dom_model=dm.value,
                plan_idx=idx.value)


def select(batch, L: int, choice, status, live_mult_pm_B) -> dict:
    cb, keep = _cbatch(batch)
    ch = np.ascontiguousarray(choice, np.uint8)
    stt = np.ascontiguousarray(status, np.uint8)
    lm = np.ascontiguousarray(live_mult_pm_B, np.int32)
    assert ch.size == batch.R * L * 16 and stt.size == batch.R * L and lm.size == batch.B
    variant = np.full(batch.R, -1, np.int32)
    lat = np.zeros(batch.R, np.int64)
    corr = np.zeros(batch.R, np.float64)
    feas = np.zeros(batch.R, np.uint8)
    rc = lib().orc_select(C.byref(cb), L, _p(ch), _p(stt), _p(lm), _p(variant), _p(lat), _p(corr), _p(feas))
    assert rc == 0, rc
    return dict(variant=variant, lat=lat, corr=corr, feasible=feas)

"""Thin ctypes binding of libdyplan.so (include/dyplan.h) -- argument marshalling only.

Every step of the path (staging, enumeration, scoring, arg-best, annotations, selection) runs in
the CUDA kernels behind the C ABI; this module only builds the two structs, passes pointers and
checks return codes.  PyTorch is used for device memory and streams, nothing else.  There is no
CPU fallback: a missing library or a missing CUDA device raises.

Names follow the header: ``dyplan_compile`` / ``dyplan_replan`` / ``dyplan_select`` (device
pointers) and the ``*_host`` variants (host pointers, copies inside the call).
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdyplan.so")

ST_OK, ST_INFEASIBLE, ST_INVALID, ST_TOO_LARGE = 0, 1, 2, 3
ERR_NULL, ERR_LIMIT, ERR_CUDA, ERR_ARG, ERR_STATIC_LIMIT = -1, -2, -3, -4, -5
STATIC_MAX_REQUESTS = 512          # DYPLAN_STATIC_MAX_REQUESTS
STATIC_SCRATCH_BYTES = 16 << 20    # DYPLAN_STATIC_SCRATCH_BYTES
FIXED_IN_PLACE, RESIDUAL = 0, 1
NO_IDX = np.iinfo(np.uint64).max

EXPORTS = (
    "dyplan_create", "dyplan_destroy", "dyplan_set_flags", "dyplan_compile", "dyplan_replan", "dyplan_select", "dyplan_switch", "dyplan_compile_linear", "dyplan_compile_linear_host", "dyplan_bind",
    "dyplan_compile_host", "dyplan_replan_host", "dyplan_select_host", "dyplan_last_stats",
    "dyplan_strerror", "dyplan_last_cuda_error", "dyplan_version", "dyplan_measure_issue_rates",
    "dyplan_compile_static",
)


class DyplanError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"dyplan error {code}: {msg}")
        self.code = code


class CBatch(C.Structure):
    _fields_ = [("R", C.c_int32), ("B", C.c_int32), ("M", C.c_int32), ("NN", C.c_int32), ("KK", C.c_int32),
                ("node_off", C.c_void_p), ("opt_off", C.c_void_p), ("pred_mask", C.c_void_p), ("vuln", C.c_void_p),
                ("lat_us", C.c_void_p), ("acc", C.c_void_p), ("demand", C.c_void_p), ("backend", C.c_void_p),
                ("model", C.c_void_p), ("slo_us", C.c_void_p), ("cap", C.c_void_p)]


class CBundle(C.Structure):
    _fields_ = [("plan_idx", C.c_void_p), ("choice", C.c_void_p), ("corr", C.c_void_p), ("corr64", C.c_void_p),
                ("lat", C.c_void_p), ("dem", C.c_void_p), ("dom_model", C.c_void_p), ("status", C.c_void_p)]


PRUNE_DOMINATED = 1
PRUNE_BOUNDS = 2
NO_SMALL_PATH = 4


class CSwitchParams(C.Structure):
    _fields_ = [("hi_load", C.c_float), ("lo_load", C.c_float), ("load_margin", C.c_float),
                ("quality_tol", C.c_float), ("min_dwell", C.c_float)]


class CLinearParams(C.Structure):
    _fields_ = [(n, C.c_float) for n in ("lambda_f", "lambda_c", "lambda_l", "lambda_ld", "beta", "effort")]


class CLinearExtra(C.Structure):
    _fields_ = [("dtau", C.c_void_p), ("quality", C.c_void_p)]


class CProfiles(C.Structure):
    _fields_ = [("S", C.c_int32), ("M", C.c_int32), ("P", C.c_int32), ("D", C.c_int32), ("A", C.c_int32), ("J", C.c_int32),
                ("ROLES", C.c_int32), ("F", C.c_int32), ("quality", C.c_void_p), ("tokens", C.c_void_p),
                ("theta_dec", C.c_void_p), ("tau_pre_us", C.c_void_p), ("psi", C.c_void_p), ("token_norm", C.c_float)]


class CStats(C.Structure):
    _fields_ = [("plans", C.c_uint64), ("evals", C.c_uint64), ("work_items", C.c_uint64), ("slow_steps", C.c_uint64),
                ("fast_requests", C.c_uint64), ("launches", C.c_int32), ("sm_count", C.c_int32), ("score_ms", C.c_float),
                ("bound_skipped", C.c_uint64), ("approx_requests", C.c_uint64), ("small_requests", C.c_uint64)]


class CIssueRate(C.Structure):
    _fields_ = [("name", C.c_char * 64), ("rate", C.c_float), ("rate_min", C.c_float), ("rate_max", C.c_float)]


_lib = None


def lib():
    """Load libdyplan.so (built by ``python -m paper_2607_02942_b200.build``).  Raises if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2607_02942_b200.build` "
                              "(there is no CPU fallback)")
        l = C.CDLL(LIB_PATH)
        vp, i32, u32 = C.c_void_p, C.c_int32, C.c_uint32
        pb, po, pu64 = C.POINTER(CBatch), C.POINTER(CBundle), C.POINTER(C.c_uint64)
        l.dyplan_create.argtypes = [C.POINTER(vp), C.c_int]
        l.dyplan_destroy.argtypes = [vp]
        l.dyplan_set_flags.argtypes = [vp, u32]
        l.dyplan_compile.argtypes = [vp, pb, i32, vp, po, vp]
        l.dyplan_replan.argtypes = [vp, pb, vp, vp, vp, u32, po, vp]
        l.dyplan_compile_static.argtypes = [vp, pb, i32, vp, po, vp]
        l.dyplan_select.argtypes = [vp, pb, po, i32, vp, vp, po, vp]
        l.dyplan_compile_linear.argtypes = [vp, pb, vp, C.POINTER(CLinearParams), i32, vp, po, C.POINTER(CLinearExtra), vp]
        l.dyplan_compile_linear_host.argtypes = [vp, pb, vp, C.POINTER(CLinearParams), i32, vp, po, C.POINTER(CLinearExtra), vp, pu64, pu64]
        l.dyplan_bind.argtypes = [vp, C.POINTER(CProfiles), i32, i32] + [vp] * 13
        l.dyplan_switch.argtypes = [vp, pb, po, i32, C.POINTER(CSwitchParams), vp, vp, vp, vp, vp, vp, vp]
        l.dyplan_compile_host.argtypes = [vp, pb, i32, vp, po, vp, pu64, pu64]
        l.dyplan_replan_host.argtypes = [vp, pb, vp, vp, vp, u32, po, vp, pu64, pu64]
        l.dyplan_select_host.argtypes = [vp, pb, po, i32, vp, vp, po, vp, pu64, pu64]
        l.dyplan_last_stats.argtypes = [vp, C.POINTER(CStats)]
        l.dyplan_measure_issue_rates.argtypes = [vp, C.POINTER(CIssueRate), i32, C.POINTER(i32), C.POINTER(C.c_float), vp]
        for n in EXPORTS:
            getattr(l, n).restype = C.c_int
        l.dyplan_strerror.restype = C.c_char_p
        l.dyplan_strerror.argtypes = [C.c_int]
        l.dyplan_last_cuda_error.restype = C.c_char_p
        l.dyplan_last_cuda_error.argtypes = [vp]
        l.dyplan_version.argtypes = []
        _lib = l
    return _lib


def dyplan_version() -> int:
    return int(lib().dyplan_version())


def dyplan_strerror(code: int) -> str:
    return lib().dyplan_strerror(code).decode()


# ---------------------------------------------------------------------------------------------
# buffers
# ---------------------------------------------------------------------------------------------
_BATCH_FIELDS = (("node_off", np.int32), ("opt_off", np.int32), ("pred_mask", np.uint32), ("vuln", np.float32),
                 ("lat_us", np.int32), ("acc", np.float32), ("demand", np.int32), ("backend", np.uint8),
                 ("model", np.uint8), ("slo_us", np.int32), ("cap", np.int32))
_BUNDLE_FIELDS = (("plan_idx", np.uint64, 1), ("choice", np.uint8, 16), ("corr", np.float32, 1),
                  ("corr64", np.float64, 1), ("lat", np.int32, 1), ("dem", np.int32, 0), ("dom_model", np.uint8, 1),
                  ("status", np.uint8, 1))


def _torch():
    import torch
    return torch


def _as_dev(a: np.ndarray, device):
    """numpy -> device tensor of the same bytes (unsigned types travel as their signed twins)."""
    torch = _torch()
    a = np.ascontiguousarray(a)
    view = {np.dtype(np.uint32): np.int32, np.dtype(np.uint64): np.int64}.get(a.dtype)
    t = torch.from_numpy(a.view(view) if view else a)
    return t.to(device)


def _ptr(t) -> Optional[int]:
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        return t.ctypes.data or None
    return t.data_ptr() or None


@dataclass
class Buffers:
    """A dyplan_batch or dyplan_bundle whose arrays live either on the host (numpy) or on a device (torch)."""
    arrays: dict
    cstruct: C.Structure
    R: int
    B: int
    L: int = 1

    def host(self) -> dict:
        """Copy to numpy (device buffers: a synchronising .cpu())."""
        out = {}
        for k, v in self.arrays.items():
            if v is None:
                out[k] = None
            elif isinstance(v, np.ndarray):
                out[k] = v
            else:
                out[k] = v.cpu().numpy()
        if out.get("plan_idx") is not None:
            out["plan_idx"] = out["plan_idx"].view(np.uint64)
        return out


def make_batch(batch, device=None) -> Buffers:
    """Marshal a ``workloads.Batch`` into a dyplan_batch (device tensors if ``device`` is given, else numpy)."""
    arrays = {}
    for name, dt in _BATCH_FIELDS:
        a = getattr(batch, name)
        if a is None:
            arrays[name] = None
            continue
        a = np.ascontiguousarray(a, dtype=dt)
        arrays[name] = _as_dev(a, device) if device is not None else a
    cb = CBatch(batch.R, batch.B, batch.M, batch.NN, batch.KK, *[_ptr(arrays[n]) for n, _ in _BATCH_FIELDS])
    return Buffers(arrays, cb, batch.R, batch.B)


def alloc_bundle(R: int, L: int, B: int, device=None, corr64: bool = True) -> Buffers:
    """Caller-owned result buffers for R x L records."""
    nrec = R * L
    arrays = {}
    for name, dt, width in _BUNDLE_FIELDS:
        if name == "corr64" and not corr64:
            arrays[name] = None
            continue
        n = nrec * (B if width == 0 else width)
        if device is None:
            arrays[name] = np.zeros(n, dtype=dt)
        else:
            torch = _torch()
            tdt = {np.uint64: torch.int64, np.uint8: torch.uint8, np.float32: torch.float32,
                   np.float64: torch.float64, np.int32: torch.int32}[dt]
            arrays[name] = torch.zeros(n, dtype=tdt, device=device)
    cb = CBundle(*[_ptr(arrays[n]) for n, _, _ in _BUNDLE_FIELDS])
    return Buffers(arrays, cb, R, B, L)


def bundle_from_host(d: dict, R: int, L: int, B: int, device=None) -> Buffers:
    """Marshal stored bundle arrays (e.g. the output of a previous compile) for dyplan_select."""
    arrays = {}
    for name, dt, _w in _BUNDLE_FIELDS:
        a = d.get(name)
        if a is None:
            arrays[name] = None
            continue
        a = np.ascontiguousarray(np.asarray(a).reshape(-1), dtype=dt)
        arrays[name] = _as_dev(a, device) if device is not None else a
    cb = CBundle(*[_ptr(arrays[n]) for n, _, _ in _BUNDLE_FIELDS])
    return Buffers(arrays, cb, R, B, L)


def _stream_ptr(stream) -> Optional[int]:
    if stream is None:
        return None
    if isinstance(stream, int):
        return stream or None
    return stream.cuda_stream or None


# ---------------------------------------------------------------------------------------------
# the calls
# ---------------------------------------------------------------------------------------------
class Context:
    """dyplan_ctx* with the header's calls as methods of the same names."""

    def __init__(self, device_ordinal: int = 0):
        self._h = C.c_void_p()
        rc = lib().dyplan_create(C.byref(self._h), device_ordinal)
        if rc:
            self._h = C.c_void_p()
            raise DyplanError(rc, dyplan_strerror(rc) + " (dyplan_create: no usable CUDA device?)")
        self.device_ordinal = device_ordinal
        self.flags = 0

    def close(self):
        if self._h:
            lib().dyplan_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int):
        if rc:
            msg = dyplan_strerror(rc)
            if rc in (ERR_CUDA, ERR_STATIC_LIMIT):
                msg += ": " + lib().dyplan_last_cuda_error(self._h).decode()
            raise DyplanError(rc, msg)

    def dyplan_compile(self, batch: Buffers, L: int, mult_pm, out: Buffers, stream=None):
        self._check(lib().dyplan_compile(self._h, C.byref(batch.cstruct), L, _ptr(mult_pm), C.byref(out.cstruct),
                                         _stream_ptr(stream)))

    def dyplan_compile_static(self, batch: Buffers, L: int, mult_pm, out: Buffers, stream=None):
        """dyplan_compile with every byte of scratch in the library's static device array: no allocation."""
        self._check(lib().dyplan_compile_static(self._h, C.byref(batch.cstruct), L, _ptr(mult_pm),
                                                C.byref(out.cstruct), _stream_ptr(stream)))

    def dyplan_replan(self, batch: Buffers, dispatched_mask, fixed_choice, live_mult_pm, flags: int, out: Buffers,
                      stream=None):
        self._check(lib().dyplan_replan(self._h, C.byref(batch.cstruct), _ptr(dispatched_mask), _ptr(fixed_choice),
                                        _ptr(live_mult_pm), flags, C.byref(out.cstruct), _stream_ptr(stream)))

    def dyplan_select(self, batch: Buffers, bundle: Buffers, L: int, live_mult_pm, variant,
                      rescored: Optional[Buffers] = None, stream=None):
        self._check(lib().dyplan_select(self._h, C.byref(batch.cstruct), C.byref(bundle.cstruct), L,
                                        _ptr(live_mult_pm), _ptr(variant),
                                        C.byref(rescored.cstruct) if rescored is not None else None,
                                        _stream_ptr(stream)))

    def dyplan_compile_linear(self, batch: Buffers, cost, params: dict, levels, out: Buffers, dtau=None, quality=None,
                              stream=None):
        p = CLinearParams(*[float(params[n]) for n, _ in CLinearParams._fields_])
        lv = np.ascontiguousarray(levels, np.float32)
        ex = CLinearExtra(_ptr(dtau), _ptr(quality))
        self._check(lib().dyplan_compile_linear(self._h, C.byref(batch.cstruct), _ptr(cost), C.byref(p), int(lv.size),
                                                lv.ctypes.data_as(C.c_void_p), C.byref(out.cstruct), C.byref(ex),
                                                _stream_ptr(stream)))

    def dyplan_bind(self, dims: dict, quality, tokens, theta_dec, tau_pre_us, psi, token_norm: float, NN: int, KK: int,
                    opt_off, pred_mask, skill, role, model, backend, policy, vuln, acc, lat_us, cost, demand=None, stream=None):
        p = CProfiles(dims["S"], dims["M"], dims["P"], dims["D"], dims["A"], dims["J"], dims["ROLES"], dims["F"],
                      _ptr(quality), _ptr(tokens), _ptr(theta_dec), _ptr(tau_pre_us), _ptr(psi), float(token_norm))
        self._check(lib().dyplan_bind(self._h, C.byref(p), NN, KK, _ptr(opt_off), _ptr(pred_mask), _ptr(skill), _ptr(role),
                                      _ptr(model), _ptr(backend), _ptr(policy), _ptr(vuln), _ptr(acc), _ptr(lat_us),
                                      _ptr(cost), _ptr(demand), _stream_ptr(stream)))

    def dyplan_compile_linear_host(self, batch: Buffers, cost: np.ndarray, params: dict, levels, out: Buffers, dtau=None,
                                   quality=None, stream=None):
        p = CLinearParams(*[float(params[n]) for n, _ in CLinearParams._fields_])
        lv = np.ascontiguousarray(levels, np.float32)
        ex = CLinearExtra(_ptr(dtau), _ptr(quality))
        h2d, d2h = C.c_uint64(), C.c_uint64()
        self._check(lib().dyplan_compile_linear_host(self._h, C.byref(batch.cstruct), _ptr(cost), C.byref(p), int(lv.size),
                                                     lv.ctypes.data_as(C.c_void_p), C.byref(out.cstruct), C.byref(ex),
                                                     _stream_ptr(stream), C.byref(h2d), C.byref(d2h)))
        return h2d.value, d2h.value

    def dyplan_set_flags(self, flags: int):
        self._check(lib().dyplan_set_flags(self._h, int(flags)))
        self.flags = int(flags)

    def dyplan_switch(self, batch: Buffers, bundle: Buffers, L: int, params: dict, model_load, since_switch,
                      dispatched_mask, cur_variant, active_choice, switched, stream=None):
        p = CSwitchParams(params["hi_load"], params["lo_load"], params["load_margin"], params["quality_tol"],
                          params["min_dwell"])
        self._check(lib().dyplan_switch(self._h, C.byref(batch.cstruct), C.byref(bundle.cstruct), L, C.byref(p),
                                        _ptr(model_load), _ptr(since_switch), _ptr(dispatched_mask), _ptr(cur_variant),
                                        _ptr(active_choice), _ptr(switched), _stream_ptr(stream)))

    def dyplan_compile_host(self, batch: Buffers, L: int, mult_pm: np.ndarray, out: Buffers, stream=None):
        h2d, d2h = C.c_uint64(), C.c_uint64()
        self._check(lib().dyplan_compile_host(self._h, C.byref(batch.cstruct), L, _ptr(mult_pm), C.byref(out.cstruct),
                                              _stream_ptr(stream), C.byref(h2d), C.byref(d2h)))
        return h2d.value, d2h.value

    def dyplan_replan_host(self, batch: Buffers, dispatched_mask, fixed_choice, live_mult_pm, flags: int,
                           out: Buffers, stream=None):
        h2d, d2h = C.c_uint64(), C.c_uint64()
        self._check(lib().dyplan_replan_host(self._h, C.byref(batch.cstruct), _ptr(dispatched_mask),
                                             _ptr(fixed_choice), _ptr(live_mult_pm), flags, C.byref(out.cstruct),
                                             _stream_ptr(stream), C.byref(h2d), C.byref(d2h)))
        return h2d.value, d2h.value

    def dyplan_select_host(self, batch: Buffers, bundle: Buffers, L: int, live_mult_pm, variant: np.ndarray,
                           rescored: Optional[Buffers] = None, stream=None):
        h2d, d2h = C.c_uint64(), C.c_uint64()
        self._check(lib().dyplan_select_host(self._h, C.byref(batch.cstruct), C.byref(bundle.cstruct), L,
                                             _ptr(live_mult_pm), _ptr(variant),
                                             C.byref(rescored.cstruct) if rescored is not None else None,
                                             _stream_ptr(stream), C.byref(h2d), C.byref(d2h)))
        return h2d.value, d2h.value

    def dyplan_measure_issue_rates(self, stream=None):
        """M0: ([{name, rate, rate_min, rate_max}], sm_clock_mhz) -- warp-instructions / clk / SMSP per instruction."""
        arr = (CIssueRate * 32)()
        n, mhz = C.c_int32(), C.c_float()
        self._check(lib().dyplan_measure_issue_rates(self._h, arr, 32, C.byref(n), C.byref(mhz), _stream_ptr(stream)))
        return ([dict(name=arr[i].name.decode(), rate=arr[i].rate, rate_min=arr[i].rate_min, rate_max=arr[i].rate_max)
                 for i in range(n.value)], mhz.value)

    def dyplan_last_stats(self) -> dict:
        st = CStats()
        self._check(lib().dyplan_last_stats(self._h, C.byref(st)))
        return {k: getattr(st, k) for k, _ in CStats._fields_}


# ---------------------------------------------------------------------------------------------
# convenience: a whole ``workloads.Workload`` through the device-pointer calls
# ---------------------------------------------------------------------------------------------
@dataclass
class DeviceWorkload:
    """Inputs of one call resident on the device, plus caller-owned result buffers."""
    kind: str
    L: int
    batch: Buffers
    out: Buffers
    mult: object = None
    dispatched: object = None
    fixed_choice: object = None
    flags: int = 0


def upload(w, device="cuda:0", corr64: bool = True) -> DeviceWorkload:
    b = make_batch(w.batch, device)
    out = alloc_bundle(w.batch.R, w.L, w.batch.B, device, corr64)
    if w.kind == "compile":
        return DeviceWorkload("compile", w.L, b, out, mult=_as_dev(np.asarray(w.mult_pm, np.int32), device))
    return DeviceWorkload("replan", 1, b, out, mult=_as_dev(np.asarray(w.live_mult_pm, np.int32), device),
                          dispatched=_as_dev(np.asarray(w.dispatched_mask, np.uint32), device),
                          fixed_choice=_as_dev(np.asarray(w.fixed_choice, np.uint8), device), flags=int(w.flags))


def launch(ctx: Context, dw: DeviceWorkload, stream=None):
    """Enqueue the call for ``dw`` (asynchronous)."""
    if dw.kind == "compile":
        ctx.dyplan_compile(dw.batch, dw.L, dw.mult, dw.out, stream)
    else:
        ctx.dyplan_replan(dw.batch, dw.dispatched, dw.fixed_choice, dw.mult, dw.flags, dw.out, stream)


def run_host(ctx: Context, w, corr64: bool = True, stream=None):
    """The same call through the *_host entry points with numpy buffers.  Returns (bundle dict, h2d, d2h)."""
    b = make_batch(w.batch, None)
    out = alloc_bundle(w.batch.R, w.L, w.batch.B, None, corr64)
    if w.kind == "compile":
        h2d, d2h = ctx.dyplan_compile_host(b, w.L, np.ascontiguousarray(w.mult_pm, np.int32), out, stream)
    else:
        h2d, d2h = ctx.dyplan_replan_host(b, np.ascontiguousarray(w.dispatched_mask, np.uint32),
                                          np.ascontiguousarray(w.fixed_choice, np.uint8),
                                          np.ascontiguousarray(w.live_mult_pm, np.int32), int(w.flags), out, stream)
    return out.host(), h2d, d2h

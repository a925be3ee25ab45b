"""ctypes binding over libnkb200.so (include/nkb200.h).  Argument marshalling only: every step of the path runs
in the library's CUDA kernels.  torch is used to allocate device memory and to supply the current stream.

There is no CPU fallback: if the shared library is missing or a call fails, an exception is raised.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

__all__ = ["load", "NkError", "Operator", "rbm_logpsi", "rbm_logpsi_static", "connected", "local_energy", "local_energy_host", "energy_gradient",
           "qgt_matvec", "sr_solve", "rbmsymm_expand", "rbmsymm_reduce_gradient", "metropolis_sample", "NK_RULE_LOCAL", "NK_RULE_EXCHANGE", "LocalEnergyPlan", "HostPlan", "launch_count", "pipe_peaks", "profile_enable", "profile_read", "PHASES", "combine_stats", "allreduce_stats", "allreduce_gradient", "LIB_PATH",
           "NK_HEISENBERG", "NK_ISING", "NK_F32", "NK_C64", "NK_FLAG_MARSHALL", "NK_OUT_F64", "NK_FORM_PRODUCT", "NK_CHECK_SPINS", "NK_FORM_LOGCOSH", "NK_FORM_SERIES", "NK_SERIAL_CHUNKS", "EXPORTS"]

NK_HEISENBERG, NK_ISING = 0, 1
NK_F32, NK_C64 = 0, 1
NK_FLAG_MARSHALL, NK_OUT_F64, NK_FORM_PRODUCT, NK_CHECK_SPINS, NK_FORM_LOGCOSH, NK_FORM_SERIES = 1, 2, 4, 8, 16, 32
NK_SERIAL_CHUNKS = 64
NK_RULE_LOCAL, NK_RULE_EXCHANGE = 0, 1
LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libnkb200.so")

_vp, _i64, _int, _sz, _u32, _dbl = C.c_void_p, C.c_int64, C.c_int, C.c_size_t, C.c_uint, C.c_double
_u64 = C.c_uint64
# name -> (restype, argtypes): every symbol include/nkb200.h declares
EXPORTS = {
    "nk_status_string": (C.c_char_p, [_int]),
    "nk_last_cuda_error": (_int, []),
    "nk_version": (_int, []),
    "nk_operator_create": (_int, [C.POINTER(_vp), _int, _int, _int, _vp, _vp, _int, _vp, _dbl, _u32]),
    "nk_operator_destroy": (_int, [_vp]),
    "nk_operator_max_conn": (_int, [_vp, C.POINTER(_int)]),
    "nk_rbm_logpsi_workspace_bytes": (_sz, [_i64, _int, _int, _int]),
    "nk_rbm_logpsi": (_int, [_vp, _i64, _int, _int, _int, _vp, _vp, _vp, _vp, _vp, _u32, _vp, _sz, _vp]),
    "nk_rbm_logpsi_static_max_bytes": (_sz, []),
    "nk_rbm_logpsi_static": (_int, [_vp, _i64, _int, _int, _int, _vp, _vp, _vp, _vp, _vp, _u32, _vp]),
    "nk_connected": (_int, [_vp, _vp, _i64, _vp, _vp, _vp, _vp, _vp]),
    "nk_local_energy_workspace_bytes": (_sz, [_vp, _i64, _int, _int, _int, _i64]),
    "nk_local_energy": (_int, [_vp, _vp, _i64, _int, _int, _int, _vp, _vp, _vp, _i64, _vp, _vp, _vp, _vp, _sz, _vp]),
    "nk_local_energy_ex": (_int, [_vp, _vp, _i64, _int, _int, _int, _vp, _vp, _vp, _i64, _u32, _vp, _vp, _vp, _vp, _sz,
                                  _vp]),
    "nk_local_energy_plan_create": (_int, [C.POINTER(_vp), _vp, _vp, _i64, _int, _int, _int, _vp, _vp, _vp, _i64, _u32, _vp,
                                            _vp, _vp, _vp, _sz]),
    "nk_local_energy_plan_run": (_int, [_vp, _vp]),
    "nk_local_energy_plan_destroy": (_int, [_vp]),
    "nk_local_energy_form": (_int, [_vp, _i64, _int, _int, _int, _i64, _vp, _sz, _vp, _vp, _vp, _vp]),
    "nk_local_energy_host_scratch_bytes": (_sz, [_vp, _i64, _int, _int, _int, _i64]),
    "nk_local_energy_host": (_int, [_vp, _vp, _i64, _int, _int, _int, _vp, _vp, _vp, _i64, _vp, _vp, _vp, _vp, _sz, _vp]),
    "nk_energy_gradient_workspace_bytes": (_sz, [_i64, _int, _int, _int, _i64]),
    "nk_energy_gradient": (_int, [_vp, _i64, _int, _int, _int, _vp, _vp, _vp, _vp, _i64, _vp, _vp, _vp, _vp, _sz, _vp]),
    "nk_energy_gradient_sharded": (_int, [_vp, _i64, _i64, _int, _int, _int, _vp, _vp, _vp, _vp, _i64, _vp, _vp, _vp, _vp,
                                           _sz, _vp]),
    "nk_stats_combine": (_int, [_vp, _int, _vp]),
    "nk_qgt_matvec_workspace_bytes": (_sz, [_i64, _int, _int, _int, _i64]),
    "nk_qgt_matvec": (_int, [_vp, _i64, _int, _int, _int, _vp, _vp, _vp, _vp, _vp, _dbl, _i64, _vp, _vp, _vp, _vp, _sz,
                             _vp]),
    "nk_sr_solve_workspace_bytes": (_sz, [_i64, _int, _int, _int, _i64]),
    "nk_sr_solve": (_int, [_vp, _i64, _int, _int, _int, _vp, _vp, _vp, _vp, _vp, _dbl, _dbl, _int, _i64, _vp, _vp, _vp,
                           _vp, _vp, _sz, _vp]),
    "nk_rbmsymm_expand": (_int, [_int, _int, _int, _int, _vp, _vp, _vp, _vp, _vp, _vp]),
    "nk_rbmsymm_reduce_gradient": (_int, [_int, _int, _int, _int, _vp, _vp, _vp, _vp, _vp, _vp]),
    "nk_metropolis_workspace_bytes": (_sz, [_int, _int, _i64, _int, _int, _int, _i64]),
    "nk_metropolis_sample": (_int, [_int, _vp, _int, _vp, _i64, _int, _int, _int, _vp, _vp, _vp, _i64, _u64, _u64, _u64,
                                    _i64, _vp, _vp, _sz, _vp]),
    "nk_pipe_peaks": (_int, [_vp, _vp, _vp]),
    "nk_launch_count": (_i64, [_int]),
    "nk_profile_enable": (_int, [_int]),
    "nk_profile_read": (_int, [_vp]),
}

_lib = None


class NkError(RuntimeError):
    pass


def load():
    """Open libnkb200.so (built in-tree by `python -m paper_2112_10526_b200.build`).  Raises if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise NkError(f"{LIB_PATH} not found: build it with `python -m paper_2112_10526_b200.build` "
                          "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        for name, (res, args) in EXPORTS.items():
            fn = getattr(lib, name)
            fn.restype, fn.argtypes = res, args
        _lib = lib
    return _lib


def _check(rc: int, what: str):
    if rc != 0:
        lib = load()
        msg = lib.nk_status_string(rc).decode()
        raise NkError(f"{what}: {msg} (status {rc}, cudaError {lib.nk_last_cuda_error()})")


def _torch():
    import torch
    return torch


def _stream():
    return _torch().cuda.current_stream().cuda_stream


def _ptr(t):
    return None if t is None else t.data_ptr()


def _dtype_code(W) -> int:
    torch = _torch()
    if W.dtype == torch.float32:
        return NK_F32
    if W.dtype == torch.complex64:
        return NK_C64
    raise NkError("W must be float32 or complex64")


def _check_params(sigma, W, a, b):
    torch = _torch()
    if sigma.dtype != torch.int8 or sigma.dim() != 2 or not sigma.is_contiguous() or not sigma.is_cuda:
        raise NkError("sigma must be a contiguous CUDA int8 tensor [B][N]")
    if W.dim() != 2 or not W.is_contiguous() or not W.is_cuda or W.shape[1] != sigma.shape[1]:
        raise NkError("W must be a contiguous CUDA tensor [M][N]")
    for name, t, n in (("a", a, W.shape[1]), ("b", b, W.shape[0])):
        if t is not None and (t.dtype != W.dtype or tuple(t.shape) != (n,) or not t.is_contiguous() or not t.is_cuda):
            raise NkError(f"{name} must be a contiguous CUDA tensor of W's dtype and length {n}")


class Operator:
    """nk_operator_t: device-resident bond table + couplings (nk_operator_create / nk_operator_destroy)."""

    def __init__(self, kind: int, n_sites: int, bonds, colors=None, J=(1.0,), h: float = 0.0, flags: int = 0):
        lib = load()
        bonds = np.ascontiguousarray(np.asarray(bonds, dtype=np.int32).reshape(-1, 2))
        J = np.ascontiguousarray(np.asarray(J, dtype=np.float64).reshape(-1))
        col = None if colors is None else np.ascontiguousarray(np.asarray(colors, dtype=np.int32))
        if col is not None and col.shape != (len(bonds),):
            raise NkError("colors must have one entry per bond")
        self.kind, self.n_sites, self.n_bonds = int(kind), int(n_sites), len(bonds)
        h_ = _vp()
        rc = lib.nk_operator_create(C.byref(h_), self.kind, self.n_sites, self.n_bonds,
                                    bonds.ctypes.data if len(bonds) else None,
                                    None if col is None else col.ctypes.data, len(J), J.ctypes.data, float(h),
                                    int(flags))
        _check(rc, "nk_operator_create")
        self.handle = h_
        c = _int()
        _check(lib.nk_operator_max_conn(self.handle, C.byref(c)), "nk_operator_max_conn")
        self.max_conn = c.value

    @classmethod
    def from_problem(cls, p, flags: int = 0):
        return cls(p.kind, p.n_sites, p.bonds, p.colors, p.J, p.h, flags)

    def close(self):
        if getattr(self, "handle", None) is not None and _lib is not None:
            _lib.nk_operator_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def rbm_logpsi(sigma, W, a=None, b=None, *, out_f64: bool = False, return_theta: bool = False):
    """nk_rbm_logpsi: ln psi [B] (and theta [B][M]) for device tensors."""
    torch = _torch()
    lib = load()
    _check_params(sigma, W, a, b)
    B, N = sigma.shape
    M = W.shape[0]
    dt = _dtype_code(W)
    cplx = dt == NK_C64
    odt = (torch.complex128 if cplx else torch.float64) if out_f64 else (torch.complex64 if cplx else torch.float32)
    out = torch.empty(B, dtype=odt, device=sigma.device)
    theta = torch.empty((B, M), dtype=W.dtype, device=sigma.device) if return_theta else None
    nbytes = lib.nk_rbm_logpsi_workspace_bytes(B, N, M, dt)
    ws = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=sigma.device)
    rc = lib.nk_rbm_logpsi(_ptr(sigma), B, N, M, dt, _ptr(W), _ptr(a), _ptr(b), _ptr(out), _ptr(theta),
                           NK_OUT_F64 if out_f64 else 0, _ptr(ws), ws.numel(), _stream())
    _check(rc, "nk_rbm_logpsi")
    return (out, theta) if return_theta else out


def rbm_logpsi_static(sigma, W, a=None, b=None, *, out=None, out_f64: bool = False):
    """nk_rbm_logpsi_static: ln psi [B] with the library's static 16 MiB scratch instead of a workspace — the C call
    allocates nothing.  `out`: preallocated result (a caller that cannot allocate passes it; else torch.empty here).
    Calls that may overlap on the GPU race on the shared scratch."""
    torch = _torch()
    lib = load()
    _check_params(sigma, W, a, b)
    B, N = sigma.shape
    M = W.shape[0]
    dt = _dtype_code(W)
    cplx = dt == NK_C64
    odt = (torch.complex128 if cplx else torch.float64) if out_f64 else (torch.complex64 if cplx else torch.float32)
    need, cap = lib.nk_rbm_logpsi_workspace_bytes(B, N, M, dt), lib.nk_rbm_logpsi_static_max_bytes()
    if need > cap:
        raise NkError(f"nk_rbm_logpsi_static: this problem needs {need} bytes of scratch, the static array holds {cap}; "
                      "use rbm_logpsi (caller workspace)")
    if out is None:
        out = torch.empty(B, dtype=odt, device=sigma.device)
    elif out.dtype != odt or out.shape != (B,) or not out.is_contiguous() or out.device != sigma.device:
        raise NkError("out must be a contiguous [B] tensor of the result dtype on sigma's device")
    rc = lib.nk_rbm_logpsi_static(_ptr(sigma), B, N, M, dt, _ptr(W), _ptr(a), _ptr(b), _ptr(out), None,
                                  NK_OUT_F64 if out_f64 else 0, _stream())
    _check(rc, "nk_rbm_logpsi_static")
    return out


def connected(op: Operator, sigma, *, materialize: bool = False):
    """nk_connected: (flips [B][C][2] int32, mels [B][C] f32, n_conn [B] int32, sigma' [B][C][N] int8 | None)."""
    torch = _torch()
    lib = load()
    if sigma.dtype != torch.int8 or sigma.dim() != 2 or not sigma.is_contiguous() or sigma.shape[1] != op.n_sites:
        raise NkError("sigma must be a contiguous CUDA int8 tensor [B][n_sites]")
    B, N = sigma.shape
    Cw = op.max_conn
    flips = torch.empty((B, Cw, 2), dtype=torch.int32, device=sigma.device)
    mels = torch.empty((B, Cw), dtype=torch.float32, device=sigma.device)
    n_conn = torch.empty(B, dtype=torch.int32, device=sigma.device)
    sp = torch.empty((B, Cw, N), dtype=torch.int8, device=sigma.device) if materialize else None
    rc = lib.nk_connected(op.handle, _ptr(sigma), B, _ptr(flips), _ptr(mels), _ptr(n_conn), _ptr(sp), _stream())
    _check(rc, "nk_connected")
    return flips, mels, n_conn, sp


class LocalEnergyPlan:
    """Pre-allocated outputs + workspace for repeated nk_local_energy calls of one shape (used by bench.py so
    that the timed region contains nothing but the C call)."""

    def __init__(self, op: Operator, B: int, N: int, M: int, dtype_code: int, chunk_size: int = 0, device="cuda",
                 want_logpsi: bool = True, flags: int = 0):
        torch = _torch()
        lib = load()
        self.op, self.B, self.N, self.M, self.dt, self.chunk = op, int(B), int(N), int(M), dtype_code, int(chunk_size)
        self.flags = int(flags)
        cdt = torch.complex64 if dtype_code == NK_C64 else torch.float32
        self.eloc = torch.empty(B, dtype=cdt, device=device)
        self.logpsi = torch.empty(B, dtype=cdt, device=device) if want_logpsi else None
        self.stats = torch.zeros(4, dtype=torch.float64, device=device)
        self.ws_bytes = lib.nk_local_energy_workspace_bytes(op.handle, B, N, M, dtype_code, self.chunk)
        if self.ws_bytes == 0:
            raise NkError("nk_local_energy_workspace_bytes rejected the arguments")
        self.ws = torch.empty(self.ws_bytes, dtype=torch.uint8, device=device)

    def run(self, sigma, W, a, b):
        rc = load().nk_local_energy_ex(self.op.handle, _ptr(sigma), self.B, self.N, self.M, self.dt, _ptr(W), _ptr(a),
                                       _ptr(b), self.chunk, self.flags, _ptr(self.eloc), _ptr(self.logpsi),
                                       _ptr(self.stats), _ptr(self.ws), self.ws_bytes, _stream())
        _check(rc, "nk_local_energy_ex")
        return self.eloc, self.logpsi, self.stats

    def form(self):
        """nk_local_energy_form: (NK_FORM_SERIES | NK_FORM_PRODUCT | NK_FORM_LOGCOSH, tau_max) of the last automatic run
        (synchronises); the number of series terms K is kept in `self.series_terms`."""
        form, tau, terms = C.c_int(0), C.c_float(0.0), C.c_int(0)
        rc = load().nk_local_energy_form(self.op.handle, self.B, self.N, self.M, self.dt, self.chunk, _ptr(self.ws),
                                         self.ws_bytes, _stream(), C.byref(form), C.byref(tau), C.byref(terms))
        _check(rc, "nk_local_energy_form")
        self.series_terms = terms.value
        return form.value, tau.value

    def run_graph(self, sigma, W, a, b):
        """nk_local_energy_plan_create / _run: the same call captured once into a CUDA graph by the library and replayed
        — one launch per step instead of ~15 per chunk, which is what bounds the small configs.  The plan is bound to
        the addresses of the tensors given first (their CONTENTS may change between replays; new tensors make a new
        plan); the tensors must stay alive."""
        key = tuple(_ptr(t) for t in (sigma, W, a, b))
        if getattr(self, "_plan_key", None) != key:
            self.close_plan()
            h = _vp()
            rc = load().nk_local_energy_plan_create(C.byref(h), self.op.handle, _ptr(sigma), self.B, self.N, self.M,
                                                    self.dt, _ptr(W), _ptr(a), _ptr(b), self.chunk, self.flags,
                                                    _ptr(self.eloc), _ptr(self.logpsi), _ptr(self.stats),
                                                    _ptr(self.ws), self.ws_bytes)
            _check(rc, "nk_local_energy_plan_create")
            self._plan, self._plan_key = h, key
            self._plan_keep = (sigma, W, a, b)
        _check(load().nk_local_energy_plan_run(self._plan, _stream()), "nk_local_energy_plan_run")
        return self.eloc, self.logpsi, self.stats

    def close_plan(self):
        if getattr(self, "_plan", None) is not None and _lib is not None:
            _lib.nk_local_energy_plan_destroy(self._plan)
        self._plan, self._plan_key, self._plan_keep = None, None, None

    def __del__(self):
        try:
            self.close_plan()
        except Exception:
            pass


def local_energy(op: Operator, sigma, W, a=None, b=None, *, chunk_size: int = 0, want_logpsi: bool = True,
                 flags: int = 0):
    """nk_local_energy on device tensors -> (eloc [B], logpsi [B] | None, stats double[4])."""
    _check_params(sigma, W, a, b)
    plan = LocalEnergyPlan(op, sigma.shape[0], sigma.shape[1], W.shape[0], _dtype_code(W), chunk_size,
                           device=sigma.device, want_logpsi=want_logpsi, flags=flags)
    return plan.run(sigma, W, a, b)


class HostPlan:
    """Device scratch for nk_local_energy_host (inputs + outputs + workspace), reusable across calls."""

    def __init__(self, op, B, N, M, dtype_code, chunk_size=0, device="cuda"):
        torch = _torch()
        self.bytes = load().nk_local_energy_host_scratch_bytes(op.handle, B, N, M, dtype_code, int(chunk_size))
        if self.bytes == 0:
            raise NkError("nk_local_energy_host_scratch_bytes rejected the arguments")
        self.scratch = torch.empty(self.bytes, dtype=torch.uint8, device=device)


def local_energy_host(op: Operator, sigma, W, a=None, b=None, *, chunk_size: int = 0, want_logpsi: bool = True,
                      plan: HostPlan | None = None, out=None):
    """nk_local_energy_host on HOST numpy arrays (ideally views of pinned torch tensors).
    Returns (eloc, logpsi | None, stats[4]) as numpy arrays; synchronises the stream."""
    lib = load()
    sigma = np.ascontiguousarray(sigma, dtype=np.int8)
    W = np.ascontiguousarray(W)
    if W.dtype not in (np.float32, np.complex64):
        raise NkError("W must be float32 or complex64")
    dt = NK_C64 if W.dtype == np.complex64 else NK_F32
    B, N = sigma.shape
    M = W.shape[0]
    a = None if a is None else np.ascontiguousarray(a, dtype=W.dtype)
    b = None if b is None else np.ascontiguousarray(b, dtype=W.dtype)
    if plan is None:
        plan = HostPlan(op, B, N, M, dt, chunk_size)
    if out is None:
        out = (np.empty(B, dtype=W.dtype), np.empty(B, dtype=W.dtype) if want_logpsi else None,
               np.empty(4, dtype=np.float64))
    eloc, logpsi, stats = out
    p = lambda x: None if x is None else x.ctypes.data
    rc = lib.nk_local_energy_host(op.handle, p(sigma), B, N, M, dt, p(W), p(a), p(b), int(chunk_size), p(eloc),
                                  p(logpsi), p(stats), _ptr(plan.scratch), plan.bytes, _stream())
    _check(rc, "nk_local_energy_host")
    return eloc, logpsi, stats


def energy_gradient(sigma, W, b, eloc, stats, *, chunk_size: int = 0, ws=None, n_global: int | None = None):
    """nk_energy_gradient on device tensors -> (grad_a [N], grad_b [M], grad_W [M][N]) in the parameter dtype.
    `eloc`, `stats` are the outputs of local_energy on the same sigma.  n_global (nk_energy_gradient_sharded): this
    rank holds one shard of a batch of n_global samples and `stats` are the statistics of the whole batch; the outputs
    of the ranks then SUM to the gradient of the union (allreduce_gradient)."""
    torch = _torch()
    lib = load()
    _check_params(sigma, W, None, b)
    B, N = sigma.shape
    M = W.shape[0]
    dt = _dtype_code(W)
    if eloc.dtype != W.dtype or eloc.shape != (B,) or stats.dtype != torch.float64 or stats.numel() != 4:
        raise NkError("eloc must be [B] of W's dtype and stats double[4] (outputs of local_energy)")
    ga = torch.empty(N, dtype=W.dtype, device=sigma.device)
    gb = torch.empty(M, dtype=W.dtype, device=sigma.device)
    gW = torch.empty((M, N), dtype=W.dtype, device=sigma.device)
    nbytes = lib.nk_energy_gradient_workspace_bytes(B, N, M, dt, int(chunk_size))
    if nbytes == 0:
        raise NkError("nk_energy_gradient_workspace_bytes rejected the arguments")
    if ws is None or ws.numel() < nbytes:
        ws = torch.empty(nbytes, dtype=torch.uint8, device=sigma.device)
    rc = lib.nk_energy_gradient_sharded(_ptr(sigma), B, B if n_global is None else int(n_global), N, M, dt, _ptr(W),
                                        _ptr(b), _ptr(eloc), _ptr(stats), int(chunk_size), _ptr(ga), _ptr(gb),
                                        _ptr(gW), _ptr(ws), ws.numel(), _stream())
    _check(rc, "nk_energy_gradient_sharded")
    return ga, gb, gW


def qgt_matvec(sigma, W, b, v_a, v_b, v_W, *, diag_shift: float = 0.0, chunk_size: int = 0, ws=None, out=None):
    """nk_qgt_matvec on device tensors: (G + diag_shift) v for v = (v_a [N], v_b [M], v_W [M][N]) in the parameter
    dtype -> (out_a, out_b, out_W).  `out`: optional preallocated triple."""
    torch = _torch()
    lib = load()
    _check_params(sigma, W, None, b)
    B, N = sigma.shape
    M = W.shape[0]
    dt = _dtype_code(W)
    for name, t, shape in (("v_a", v_a, (N,)), ("v_b", v_b, (M,)), ("v_W", v_W, (M, N))):
        if t is not None and (t.dtype != W.dtype or tuple(t.shape) != shape or not t.is_contiguous() or not t.is_cuda):
            raise NkError(f"{name} must be a contiguous CUDA tensor of W's dtype and shape {shape}")
    if v_W is None:
        raise NkError("v_W is required")
    if out is None:
        out = (torch.empty(N, dtype=W.dtype, device=sigma.device), torch.empty(M, dtype=W.dtype, device=sigma.device),
               torch.empty((M, N), dtype=W.dtype, device=sigma.device))
    nbytes = lib.nk_qgt_matvec_workspace_bytes(B, N, M, dt, int(chunk_size))
    if nbytes == 0:
        raise NkError("nk_qgt_matvec_workspace_bytes rejected the arguments")
    if ws is None or ws.numel() < nbytes:
        ws = torch.empty(nbytes, dtype=torch.uint8, device=sigma.device)
    rc = lib.nk_qgt_matvec(_ptr(sigma), B, N, M, dt, _ptr(W), _ptr(b), _ptr(v_a), _ptr(v_b), _ptr(v_W),
                           float(diag_shift), int(chunk_size), _ptr(out[0]), _ptr(out[1]), _ptr(out[2]), _ptr(ws),
                           ws.numel(), _stream())
    _check(rc, "nk_qgt_matvec")
    return out


def sr_solve(sigma, W, b, f_a, f_b, f_W, *, diag_shift: float = 0.01, tol: float = 1e-5, max_iter: int = 200,
             chunk_size: int = 0, ws=None):
    """nk_sr_solve: delta = (G + diag_shift)^-1 f by conjugate gradients on the device.
    Returns ((delta_a, delta_b, delta_W), iterations, relative residual)."""
    torch = _torch()
    lib = load()
    _check_params(sigma, W, None, b)
    B, N = sigma.shape
    M = W.shape[0]
    dt = _dtype_code(W)
    for name, t, shape in (("f_a", f_a, (N,)), ("f_b", f_b, (M,)), ("f_W", f_W, (M, N))):
        if t is None or t.dtype != W.dtype or tuple(t.shape) != shape or not t.is_contiguous() or not t.is_cuda:
            raise NkError(f"{name} must be a contiguous CUDA tensor of W's dtype and shape {shape}")
    out = (torch.empty(N, dtype=W.dtype, device=sigma.device), torch.empty(M, dtype=W.dtype, device=sigma.device),
           torch.empty((M, N), dtype=W.dtype, device=sigma.device))
    nbytes = lib.nk_sr_solve_workspace_bytes(B, N, M, dt, int(chunk_size))
    if nbytes == 0:
        raise NkError("nk_sr_solve_workspace_bytes rejected the arguments")
    if ws is None or ws.numel() < nbytes:
        ws = torch.empty(nbytes, dtype=torch.uint8, device=sigma.device)
    info = np.zeros(2, dtype=np.float64)
    rc = lib.nk_sr_solve(_ptr(sigma), B, N, M, dt, _ptr(W), _ptr(b), _ptr(f_a), _ptr(f_b), _ptr(f_W),
                         float(diag_shift), float(tol), int(max_iter), int(chunk_size), _ptr(out[0]), _ptr(out[1]),
                         _ptr(out[2]), info.ctypes.data, _ptr(ws), ws.numel(), _stream())
    _check(rc, "nk_sr_solve")
    return out, int(info[0]), float(info[1])


def _check_perms(perms, N):
    torch = _torch()
    if perms.dtype != torch.int32 or perms.dim() != 2 or perms.shape[1] != N or not perms.is_contiguous() or not perms.is_cuda:
        raise NkError("perms must be a contiguous CUDA int32 tensor [G][N]")


def rbmsymm_expand(W_sym, b_sym, perms):
    """nk_rbmsymm_expand: tied (W_sym [F][N], b_sym [F] or None) + group permutations [G][N] -> (W [F*G][N], b [F*G])."""
    torch = _torch()
    F, N = W_sym.shape
    _check_perms(perms, N)
    G = perms.shape[0]
    W = torch.zeros((F * G, N), dtype=W_sym.dtype, device=W_sym.device)
    b = torch.zeros(F * G, dtype=W_sym.dtype, device=W_sym.device)
    rc = load().nk_rbmsymm_expand(F, G, N, _dtype_code(W_sym), _ptr(W_sym), _ptr(b_sym), _ptr(perms), _ptr(W), _ptr(b),
                                  _stream())
    _check(rc, "nk_rbmsymm_expand")
    return W, b


def rbmsymm_reduce_gradient(grad_W, grad_b, perms, n_features: int):
    """nk_rbmsymm_reduce_gradient: expanded (grad_W [F*G][N], grad_b [F*G]) -> tied (grad_W_sym [F][N], grad_b_sym [F])."""
    torch = _torch()
    M, N = grad_W.shape
    _check_perms(perms, N)
    G = perms.shape[0]
    if n_features * G != M:
        raise NkError("grad_W must have n_features * n_group rows")
    gW = torch.empty((n_features, N), dtype=grad_W.dtype, device=grad_W.device)
    gb = torch.empty(n_features, dtype=grad_W.dtype, device=grad_W.device)
    rc = load().nk_rbmsymm_reduce_gradient(n_features, G, N, _dtype_code(grad_W), _ptr(grad_W), _ptr(grad_b),
                                           _ptr(perms), _ptr(gW), _ptr(gb), _stream())
    _check(rc, "nk_rbmsymm_reduce_gradient")
    return gW, gb


def metropolis_sample(sigma, W, a=None, b=None, *, rule: int = NK_RULE_LOCAL, clusters=None, n_steps: int | None = None,
                      seed: int = 0, step_offset: int = 0, chain_offset: int = 0, chunk_size: int = 0, ws=None):
    """nk_metropolis_sample: advances every row of `sigma` (device int8 [B][N], modified IN PLACE) by n_steps
    Metropolis-Hastings transitions (default: one sweep = N).  `clusters`: host int32 [n][2] pairs for
    NK_RULE_EXCHANGE (e.g. the lattice bonds).  Returns the accepted-transition counts, device int32 [B]."""
    torch = _torch()
    lib = load()
    _check_params(sigma, W, a, b)
    B, N = sigma.shape
    M = W.shape[0]
    dt = _dtype_code(W)
    if n_steps is None:
        n_steps = N
    cl, n_cl = None, 0
    if clusters is not None:
        cl = np.ascontiguousarray(np.asarray(clusters), dtype=np.int32).reshape(-1, 2)
        n_cl = int(cl.shape[0])
    nbytes = lib.nk_metropolis_workspace_bytes(int(rule), n_cl, B, N, M, dt, int(chunk_size))
    if nbytes == 0:
        raise NkError("nk_metropolis_workspace_bytes rejected the arguments")
    if ws is None or ws.numel() < nbytes:
        ws = torch.empty(nbytes, dtype=torch.uint8, device=sigma.device)
    accepted = torch.empty(B, dtype=torch.int32, device=sigma.device)
    rc = lib.nk_metropolis_sample(int(rule), None if cl is None else cl.ctypes.data, n_cl, _ptr(sigma), B, N, M, dt,
                                  _ptr(W), _ptr(a), _ptr(b), int(n_steps), int(seed), int(step_offset),
                                  int(chain_offset), int(chunk_size), _ptr(accepted), _ptr(ws), ws.numel(), _stream())
    _check(rc, "nk_metropolis_sample")
    return accepted


def launch_count(reset: bool = False) -> int:
    return int(load().nk_launch_count(1 if reset else 0))


PHASES = ("pack", "theta", "logpsi", "fused", "stats", "series_gemm", "series_prep")


def profile_enable(on: bool = True):
    _check(load().nk_profile_enable(1 if on else 0), "nk_profile_enable")


def profile_read() -> dict:
    """{phase: (total ms, bracketed launch groups)} since the last read (synchronises on the recorded events)."""
    out = np.zeros(2 * len(PHASES), dtype=np.float64)
    _check(load().nk_profile_read(out.ctypes.data), "nk_profile_read")
    return {ph: (float(out[i]), int(out[len(PHASES) + i])) for i, ph in enumerate(PHASES)}


# ---- multi-GPU: samples shard across ranks, the only exchange is the statistics ----------
def combine_stats(parts):
    """nk_stats_combine: per-shard (mean_re, mean_im, variance, count) -> the statistics of the union (the merge runs
    in the library; this only marshals the 4-double records)."""
    arr = np.ascontiguousarray(np.asarray([np.asarray(p, dtype=np.float64).reshape(4) for p in parts],
                                          dtype=np.float64).reshape(-1, 4))
    out = np.zeros(4, dtype=np.float64)
    _check(load().nk_stats_combine(arr.ctypes.data, int(arr.shape[0]), out.ctypes.data), "nk_stats_combine")
    return out


def allreduce_stats(stats):
    """All-gather the 4-double statistics over torch.distributed (NCCL on GPUs, gloo on CPU) and combine."""
    torch = _torch()
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return combine_stats([stats.detach().cpu().numpy() if hasattr(stats, "detach") else stats])
    t = stats if hasattr(stats, "detach") else torch.as_tensor(np.asarray(stats, dtype=np.float64))
    gathered = [torch.empty_like(t) for _ in range(dist.get_world_size())]
    dist.all_gather(gathered, t.contiguous())
    return combine_stats([g.cpu().numpy() for g in gathered])


def allreduce_gradient(grads):
    """Sum per-rank energy-gradient blocks into those of the union of the shards (in place): every rank has called
    energy_gradient(..., n_global=B_total) on its own samples with the statistics of the whole batch
    (allreduce_stats), so its blocks are already weighted by 1 / B_total and the union's gradient is their plain sum —
    one all-reduce per block (NCCL on GPUs, gloo on CPU), no arithmetic here.  QGT-vector products do not combine this
    way (nk_qgt_matvec centres with the shard-local mean): multi-rank SR is not supported.  Returns `grads`."""
    torch = _torch()
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return grads
    for g in grads:
        if g is not None:
            dist.all_reduce(torch.view_as_real(g) if g.is_complex() else g)
    return grads


def pipe_peaks(device="cuda"):
    """nk_pipe_peaks: measured MUFU / FFMA lanes and LDS bytes per clock per SM (roofline denominators of bench.py)."""
    torch = _torch()
    out = np.zeros(8, dtype=np.float64)
    scratch = torch.zeros(256, dtype=torch.uint8, device=device)
    _check(load().nk_pipe_peaks(out.ctypes.data, _ptr(scratch), _stream()), "nk_pipe_peaks")
    return {"mufu_lanes_per_clk_sm": out[0], "ffma_lanes_per_clk_sm": out[1], "lds_bytes_per_clk_sm": out[2],
            "sm_ghz": [out[3], out[4], out[5]], "sms": int(out[6]), "ms": out[7]}

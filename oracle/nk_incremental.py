"""ORACLE, second route — test infrastructure, NOT the product.

ctypes loader of oracle/nk_incremental.c: the separately written float64 INCREMENTAL local energy (theta' = theta -
2 s_k W[:,k], per-term ln-cosh differences; Eq. (12)) that covers full batches the from-scratch oracle
(oracle/nk_oracle.py) cannot reach in reasonable time (SURVEY.md §8(c), §8(d) "(ii)").  Pinned against the from-scratch
oracle in tests/test_oracle_incremental.py.  Only tests/, __graft_entry__ and bench.py's CPU-baseline legs may use it.

`build()` compiles the C source in place with gcc when the shared object is missing or older than the source:
`-O3 -mavx2 -mfma -ffast-math` so that gcc may call glibc's vector exp / log1p (libmvec, <= 4 ulp) and reassociate the
sums over hidden units — 3x faster, which is what makes a full 65536-sample pass of config 5 affordable — with plain
`-O2` as the fallback where those flags are refused.  Either way the result is pinned to 1e-12 against the
from-scratch oracle.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "nk_incremental.c")
LIB = os.path.join(HERE, "libnk_incremental.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < os.path.getmtime(SRC):
        for opt in (["-O3", "-mavx2", "-mfma", "-ffast-math"], ["-O2"]):
            cmd = [os.environ.get("CC", "gcc"), *opt, "-pthread", "-shared", "-fPIC", "-o", LIB, SRC, "-lm"]
            r = subprocess.run(cmd, capture_output=True, text=True)
            if r.returncode == 0:
                break
        else:
            raise RuntimeError("gcc failed on nk_incremental.c:\n" + r.stdout + r.stderr)
    return LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i64, i32, dbl, ptr = ctypes.c_int64, ctypes.c_int, ctypes.c_double, ctypes.c_void_p
        for name in ("nk_inc_local_energy_real", "nk_inc_local_energy_cplx"):
            f = getattr(lib, name)
            f.restype = i32
            f.argtypes = [i32, i64, i32, i32, ptr, i32, ptr, ptr, ptr, dbl, ctypes.c_uint, ptr, ptr, ptr, ptr, ptr]
        lib.nk_inc_num_threads.restype = i32
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().nk_inc_num_threads())


def local_energy(kind, sigma, bonds, colors, J, h, W, a=None, b=None, flags=0):
    """Same signature and return value as nk_oracle.local_energy: (eloc [B], logpsi [B]) in float64 / complex128."""
    lib = _load()
    sigma = np.ascontiguousarray(np.atleast_2d(np.asarray(sigma, dtype=np.int8)))
    B, N = sigma.shape
    cplx = np.iscomplexobj(W)
    dt = np.complex128 if cplx else np.float64
    W = np.ascontiguousarray(np.asarray(W).astype(dt))           # exact up-cast of the fp32 storage
    M = W.shape[0]
    a = None if a is None else np.ascontiguousarray(np.asarray(a).astype(dt))
    b = None if b is None else np.ascontiguousarray(np.asarray(b).astype(dt))
    bonds = np.ascontiguousarray(np.asarray(bonds, dtype=np.int32).reshape(-1, 2))
    colors = None if colors is None else np.ascontiguousarray(np.asarray(colors, dtype=np.int32))
    J = np.ascontiguousarray(np.asarray(J, dtype=np.float64))
    eloc = np.zeros(B, dtype=dt)
    logpsi = np.zeros(B, dtype=dt)
    p = lambda x: None if x is None else x.ctypes.data_as(ctypes.c_void_p)
    fn = lib.nk_inc_local_energy_cplx if cplx else lib.nk_inc_local_energy_real
    rc = fn(int(kind), B, N, M, p(sigma), len(bonds), p(bonds), p(colors), p(J), float(h), int(flags), p(W), p(a),
            p(b), p(eloc), p(logpsi))
    if rc != 0:
        raise RuntimeError("nk_inc_local_energy failed")
    return eloc, logpsi

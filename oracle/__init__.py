"""CPU oracle — TEST INFRASTRUCTURE, NOT PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It builds ``swept_oracle.cpp`` (plain per-step C++17, see the header of
that file for the cited passages and readings) with g++ and calls it through ctypes.  It imports nothing
from ``paper_1705_03162_b200`` and shares no code with it.

Build flags: ``-O2 -ffp-contract=off -mfma -fopenmp``: contraction off so that only the
``std::fma`` calls written in the source are fused; ``-mfma`` makes those one instruction.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "swept_oracle.cpp")
_LIB = os.path.join(_HERE, "libswept_oracle.so")
_lock = threading.Lock()
_lib = None

HEAT, KS, EULER, KS3 = 0, 1, 2, 3   # KS3: Eq. (C.2) with three sub-timesteps per timestep (SSP-RK3, row f3)
RK2_MIDPOINT, RK2_HEUN = 0, 1


def build(force: bool = False) -> str:
    """Compile the oracle shared library in-tree (idempotent)."""
    with _lock:
        if (not force and os.path.exists(_LIB)
                and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
            return _LIB
        tmp = _LIB + f".tmp{os.getpid()}"
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-mfma", "-fopenmp", "-fPIC",
               "-shared", "-o", tmp, _SRC]
        subprocess.run(cmd, check=True, capture_output=True, text=True)
        os.replace(tmp, _LIB)
        return _LIB


def _load():
    global _lib
    if _lib is None:
        path = build()
        lib = ctypes.CDLL(path)
        i64, dbl, ci = ctypes.c_int64, ctypes.c_double, ctypes.c_int
        vp = ctypes.c_void_p
        lib.oracle_heat_f64.argtypes = [vp, i64, i64, dbl, dbl, dbl]
        lib.oracle_heat_f32.argtypes = [vp, i64, i64, dbl, dbl, dbl]
        lib.oracle_heat_bc_f64.argtypes = [vp, i64, i64, dbl, dbl, dbl, ci]
        lib.oracle_heat_bc_f32.argtypes = [vp, i64, i64, dbl, dbl, dbl, ci]
        lib.oracle_euler_bc_f64.argtypes = [vp, i64, i64, dbl, dbl, dbl, ci]
        lib.oracle_ks_f64.argtypes = [vp, i64, i64, dbl, dbl, ci]
        lib.oracle_ks_f32.argtypes = [vp, i64, i64, dbl, dbl, ci]
        lib.oracle_ks3_f64.argtypes = [vp, i64, i64, dbl, dbl]
        lib.oracle_euler_f64.argtypes = [vp, i64, i64, dbl, dbl, dbl, ci]
        lib.oracle_euler_f32.argtypes = [vp, i64, i64, dbl, dbl, dbl, ci]
        lib.oracle_set_num_threads.argtypes = [ci]
        lib.oracle_num_threads.restype = ci
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def set_num_threads(n: int) -> None:
    _load().oracle_set_num_threads(int(n))


def run(problem: int, u0: np.ndarray, N: int, nsteps: int, dx: float, dt: float, *,
        alpha: float = 1.0, gamma: float = 1.4, rk2: int = RK2_MIDPOINT,
        dtype=np.float64, bc: int = 0) -> np.ndarray:
    """Advance ``u0`` (component-major, C*N values) by ``nsteps`` full timesteps; returns a new array.

    ``dtype`` float64 or float32 selects the arithmetic type of the whole computation (reading X15: the
    FP32 GPU path is gated against the FP32 instantiation of these same expression trees).
    ``bc``: 0 periodic (the configs), 1 the paper's own ends: insulated for heat, Eq. (B.5) PAPER.md:328-331;
    Dirichlet (the initial end states) for the Euler tube.
    """
    lib = _load()
    dtype = np.dtype(dtype)
    u = np.ascontiguousarray(np.array(u0, dtype=dtype, copy=True))
    C = 3 if problem == EULER else 1
    if u.size != C * N:
        raise ValueError(f"expected {C * N} values, got {u.size}")
    sfx = "f64" if dtype == np.float64 else "f32"
    ptr = u.ctypes.data_as(ctypes.c_void_p)
    if problem == KS3:
        if bc or dtype != np.float64:
            raise ValueError("KS3 is periodic and FP64 only")
        if lib.oracle_ks3_f64(ptr, N, nsteps, dx, dt) != 0:
            raise ValueError("oracle rejected the arguments")
        return u
    if bc and (problem == KS or (problem == EULER and dtype != np.float64)):
        raise ValueError("non-periodic ends exist for heat (B.5) and FP64 Euler (PAPER.md:377) only")
    if problem == HEAT:
        rc = getattr(lib, "oracle_heat_bc_" + sfx)(ptr, N, nsteps, dx, dt, alpha, bc) if bc else \
            getattr(lib, "oracle_heat_" + sfx)(ptr, N, nsteps, dx, dt, alpha)
    elif problem == KS:
        rc = getattr(lib, "oracle_ks_" + sfx)(ptr, N, nsteps, dx, dt, rk2)
    elif problem == EULER:
        rc = lib.oracle_euler_bc_f64(ptr, N, nsteps, dx, dt, gamma, rk2) if bc else \
            getattr(lib, "oracle_euler_" + sfx)(ptr, N, nsteps, dx, dt, gamma, rk2)
    else:
        raise ValueError("unknown problem")
    if rc != 0:
        raise ValueError("oracle rejected the arguments")
    return u


def run_workload(w, nsteps: int | None = None, dtype=np.float64) -> np.ndarray:
    """Run a ``swept_inputs.Workload`` (duck-typed: no import of that module needed)."""
    return run(w.problem, w.u0, w.N, w.nsteps if nsteps is None else nsteps, w.dx, w.dt,
               alpha=w.alpha, gamma=w.gamma, rk2=w.rk2, dtype=dtype, bc=getattr(w, "bc", 0))

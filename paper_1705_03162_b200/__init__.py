"""paper_1705_03162_b200 — thin Python binding of the C-ABI library ``libswept_b200.so`` (include/swept.h).

Argument marshalling only: every step of the hot path runs in the library's CUDA kernels.  PyTorch is used
for plumbing — device memory comes from torch's caching allocator (through the ``alloc``/``free`` hooks of
``swept_params``) and work is enqueued on torch's current stream.  There is no CPU fallback: if the
extension cannot be built or loaded, or no CUDA device is present, the calls raise.

The function names mirror the C ABI (``swept_create``, ``swept_write``, ``swept_run``, ``swept_read``,
``swept_autotune``, ``swept_destroy``, ...).  :class:`Swept` is a small convenience wrapper around them.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import (CFUNCTYPE, POINTER, Structure, byref, c_char_p, c_double, c_int, c_int32, c_int64,
                    c_uint32, c_uint64, c_void_p)

import numpy as np

HEAT, KS, EULER, KS3 = 0, 1, 2, 3   # KS3: (C.2) with three sub-timesteps per timestep (SSP-RK3), row f3
#: problem -> (h, sigma, C): stencil half-width, sub-timesteps per timestep, components
PROBLEM_SHAPE = {HEAT: (1, 1, 1), KS: (2, 2, 1), EULER: (2, 2, 3), KS3: (2, 3, 1)}
PER_STEP, SWEPT = 0, 1
F64, F32 = 0, 1
RK2_MIDPOINT, RK2_HEUN = 0, 1
FLAVOR_AUTO, FLAVOR_TIER, FLAVOR_CHAR, FLAVOR_FLOW = 0, 1, 2, 3
PS_LAUNCH, PS_RESIDENT = 0, 1  # per-step flavours
BC_PERIODIC, BC_PAPER = 0, 1   # BC_PAPER: insulated heat ends, Eq. (B.5)
KIND_NAMES = {0: "UpTriangle", 1: "SplitDiamond", 2: "WholeDiamond", 3: "DownTriangle", 4: "PerStepRemainder", 5: "FlowCycle"}

_ALLOC_FN = CFUNCTYPE(c_void_p, c_void_p, c_uint64)
_FREE_FN = CFUNCTYPE(None, c_void_p, c_void_p)


class swept_params(Structure):
    _fields_ = [("struct_size", c_uint32), ("dtype", c_int32), ("rk2", c_int32), ("device", c_int32),
                ("alpha", c_double), ("gamma", c_double), ("stream", c_void_p),
                ("alloc", _ALLOC_FN), ("free", _FREE_FN), ("alloc_ctx", c_void_p),
                ("bc", c_int32), ("reserved0", c_int32)]


class swept_phase(Structure):
    _fields_ = [("kind", c_int32), ("shift", c_int32), ("tier0", c_int64), ("ntiers", c_int64),
                ("n", c_int32), ("reserved", c_int32)]


class SweptError(RuntimeError):
    pass


_lib = None


def lib_path() -> str:
    return os.path.join(os.path.dirname(os.path.abspath(__file__)), "libswept_b200.so")


def load():
    """Load (building in-tree first if needed) the C-ABI library.  Raises if that is impossible."""
    global _lib
    if _lib is not None:
        return _lib
    from . import build as _build
    path = _build.build()
    lib = ctypes.CDLL(path)
    lib.swept_create.restype = c_void_p
    lib.swept_create.argtypes = [c_int, c_int64, c_double, c_double, POINTER(swept_params)]
    lib.swept_write.argtypes = [c_void_p, c_void_p]
    lib.swept_write_device.argtypes = [c_void_p, c_void_p]
    lib.swept_run.argtypes = [c_void_p, c_int64, c_int32, c_int]
    lib.swept_run_flavor.argtypes = [c_void_p, c_int64, c_int32, c_int, c_int]
    lib.swept_read.argtypes = [c_void_p, c_void_p]
    lib.swept_sync.argtypes = [c_void_p]
    lib.swept_device_ptr.restype = c_void_p
    lib.swept_device_ptr.argtypes = [c_void_p]
    lib.swept_autotune.argtypes = [c_void_p, c_int, POINTER(c_int32)]
    lib.swept_set_stream.argtypes = [c_void_p, c_void_p]
    lib.swept_steps_done.restype = c_int64
    lib.swept_steps_done.argtypes = [c_void_p]
    lib.swept_last_launches.restype = c_int64
    lib.swept_last_launches.argtypes = [c_void_p]
    lib.swept_destroy.restype = None
    lib.swept_destroy.argtypes = [c_void_p]
    lib.swept_last_error.restype = c_char_p
    lib.swept_plan.restype = c_int64
    lib.swept_plan.argtypes = [c_int64, c_int32, c_int32, POINTER(swept_phase), c_int64]
    lib.swept_plan_sigma.restype = c_int64
    lib.swept_plan_sigma.argtypes = [c_int64, c_int32, c_int32, c_int32, POINTER(swept_phase), c_int64]
    lib.swept_probe_fp64.argtypes = [c_int, c_void_p, POINTER(c_double)]
    lib.swept_probe_launch.argtypes = [c_int, c_void_p, c_int, POINTER(c_double)]
    lib.swept_set_phase_timing.argtypes = [c_void_p, c_int]
    lib.swept_phase_times.argtypes = [c_void_p, POINTER(c_double), POINTER(c_int64)]
    lib.swept_tuned.argtypes = [c_void_p, c_int, POINTER(c_int32), POINTER(c_int32), POINTER(c_int32)]
    _lib = lib
    return lib


def swept_last_error() -> str:
    return (load().swept_last_error() or b"").decode()


def _check(rc: int) -> None:
    if rc != 0:
        raise SweptError(f"swept error {rc}: {swept_last_error()}")


# ---- torch plumbing: allocator hooks and current stream ------------------------------------------------
_hooks = None


def _torch_hooks():
    """ctypes callbacks that route the library's device allocations through torch's caching allocator."""
    global _hooks
    if _hooks is None:
        import torch

        def _alloc(_ctx, nbytes):
            try:
                return torch.cuda.caching_allocator_alloc(int(nbytes))
            except Exception:
                return None

        def _free(_ctx, ptr):
            torch.cuda.caching_allocator_delete(int(ptr))

        _hooks = (_ALLOC_FN(_alloc), _FREE_FN(_free))
    return _hooks


def _current_stream() -> int:
    import torch
    return int(torch.cuda.current_stream().cuda_stream)


# ---- the C ABI, same names ----------------------------------------------------------------------------
def swept_create(problem: int, N: int, dx: float, dt: float, *, dtype: int = F64, rk2: int = RK2_MIDPOINT,
                 alpha: float = 1.0, gamma: float = 1.4, device: int = -1, use_torch: bool = True,
                 bc: int = BC_PERIODIC) -> int:
    lib = load()
    p = swept_params()
    p.struct_size = ctypes.sizeof(swept_params)
    p.dtype, p.rk2, p.device, p.alpha, p.gamma, p.bc = dtype, rk2, device, alpha, gamma, bc
    if use_torch:
        import torch
        if not torch.cuda.is_available():
            raise SweptError("no CUDA device: the swept library has no CPU fallback")
        a, f = _torch_hooks()
        p.alloc, p.free = a, f
        p.stream = _current_stream()
    h = lib.swept_create(problem, N, dx, dt, byref(p))
    if not h:
        raise SweptError(f"swept_create failed: {swept_last_error()}")
    return h


def swept_write(state: int, host_buf: np.ndarray) -> None:
    assert host_buf.flags["C_CONTIGUOUS"]
    _check(load().swept_write(state, host_buf.ctypes.data_as(c_void_p)))


def swept_run(state: int, nsteps: int, tile_width: int, variant: int, flavor: int = FLAVOR_AUTO,
              group: int = 0) -> None:
    """``group``: TIER points per thread / CHAR lanes per tile / FLOW resident CTAs per SM (0 = library default)."""
    _check(load().swept_run_flavor(state, nsteps, tile_width, variant, flavor | (group << 8)))


def swept_read(state: int, host_buf: np.ndarray) -> None:
    assert host_buf.flags["C_CONTIGUOUS"] and host_buf.flags["WRITEABLE"]
    _check(load().swept_read(state, host_buf.ctypes.data_as(c_void_p)))


def swept_sync(state: int) -> None:
    _check(load().swept_sync(state))


def swept_autotune(state: int, variant: int) -> int:
    best = c_int32(0)
    _check(load().swept_autotune(state, variant, byref(best)))
    return int(best.value)


def swept_tuned(state: int, variant: int):
    n, fl, g = c_int32(0), c_int32(0), c_int32(0)
    _check(load().swept_tuned(state, variant, byref(n), byref(fl), byref(g)))
    return int(n.value), int(fl.value), int(g.value)


def swept_set_phase_timing(state: int, on: bool) -> None:
    _check(load().swept_set_phase_timing(state, 1 if on else 0))


def swept_phase_times(state: int):
    """{kind name: (milliseconds, launches)} recorded since timing was switched on / the previous call."""
    ms, cnt = (c_double * 6)(), (c_int64 * 6)()
    _check(load().swept_phase_times(state, ms, cnt))
    return {KIND_NAMES[k]: (float(ms[k]), int(cnt[k])) for k in range(6)}


def swept_set_stream(state: int, stream: int) -> None:
    _check(load().swept_set_stream(state, stream))


def swept_destroy(state: int) -> None:
    load().swept_destroy(state)


def swept_plan(nsub: int, n: int, h: int, sigma: int = 1):
    """Phase list of ``swept_plan`` (sigma <= 2) / ``swept_plan_sigma`` (three sub-timesteps per timestep)."""
    lib = load()
    if sigma <= 2:
        cnt = lib.swept_plan(nsub, n, h, None, 0)
    else:
        cnt = lib.swept_plan_sigma(nsub, n, h, sigma, None, 0)
    if cnt < 0:
        raise SweptError(f"swept_plan: {swept_last_error()}")
    arr = (swept_phase * max(cnt, 1))()
    if sigma <= 2:
        lib.swept_plan(nsub, n, h, arr, cnt)
    else:
        lib.swept_plan_sigma(nsub, n, h, sigma, arr, cnt)
    return [(int(a.kind), int(a.shift), int(a.tier0), int(a.ntiers), int(a.n)) for a in arr[:cnt]]


def swept_probe_fp64(device: int = -1) -> float:
    out = c_double(0)
    _check(load().swept_probe_fp64(device, _current_stream(), byref(out)))
    return float(out.value)


def swept_probe_launch(count: int = 2000, device: int = -1) -> float:
    out = c_double(0)
    _check(load().swept_probe_launch(device, _current_stream(), count, byref(out)))
    return float(out.value)


class Swept:
    """Convenience wrapper: one problem instance on the current CUDA device."""

    def __init__(self, problem: int, N: int, dx: float, dt: float, *, dtype=np.float64, rk2: int = RK2_MIDPOINT,
                 alpha: float = 1.0, gamma: float = 1.4, bc: int = BC_PERIODIC):
        self.problem, self.N = problem, N
        self.np_dtype = np.dtype(dtype)
        self.h, self.sigma, self.C = PROBLEM_SHAPE[problem]
        self._h = swept_create(problem, N, dx, dt, dtype=F64 if self.np_dtype == np.float64 else F32, rk2=rk2,
                               alpha=alpha, gamma=gamma, bc=bc)

    @classmethod
    def from_workload(cls, w, dtype=np.float64) -> "Swept":
        s = cls(w.problem, w.N, w.dx, w.dt, dtype=dtype, rk2=w.rk2, alpha=w.alpha, gamma=w.gamma,
                bc=getattr(w, "bc", BC_PERIODIC))
        s.write(w.u0)
        return s

    def write(self, u0: np.ndarray) -> None:
        buf = np.ascontiguousarray(u0, dtype=self.np_dtype)
        if buf.size != self.C * self.N:
            raise ValueError("wrong initial-data size")
        swept_set_stream(self._h, _current_stream())
        swept_write(self._h, buf)
        self._keep = buf  # the copy is asynchronous for pinned memory

    def run(self, nsteps: int, tile_width: int = 0, variant: int = SWEPT, flavor: int = FLAVOR_AUTO,
            group: int = 0) -> None:
        swept_set_stream(self._h, _current_stream())
        swept_run(self._h, nsteps, tile_width, variant, flavor, group)

    def read(self, out: np.ndarray | None = None) -> np.ndarray:
        if out is None:
            out = np.empty(self.C * self.N, dtype=self.np_dtype)
        swept_set_stream(self._h, _current_stream())
        swept_read(self._h, out)
        return out

    def sync(self) -> None:
        swept_set_stream(self._h, _current_stream())
        swept_sync(self._h)

    def autotune(self, variant: int = SWEPT) -> int:
        swept_set_stream(self._h, _current_stream())
        return swept_autotune(self._h, variant)

    def set_phase_timing(self, on: bool) -> None:
        swept_set_phase_timing(self._h, on)

    def phase_times(self):
        swept_set_stream(self._h, _current_stream())
        return swept_phase_times(self._h)

    def tuned(self, variant: int = SWEPT):
        return swept_tuned(self._h, variant)

    @property
    def last_launches(self) -> int:
        return int(load().swept_last_launches(self._h))

    @property
    def device_ptr(self) -> int:
        return int(load().swept_device_ptr(self._h))

    def close(self) -> None:
        if self._h:
            swept_destroy(self._h)
            self._h = 0

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

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
FLAVOR_AUTO, FLAVOR_TIER, FLAVOR_CHAR, FLAVOR_FLOW, FLAVOR_CLUSTER = 0, 1, 2, 3, 4
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


class swept_exchange(Structure):
    _fields_ = [("after_phase", c_int32), ("dir", c_int32), ("src_off", c_int64), ("dst_off", c_int64),
                ("count", c_int32), ("rows", c_int32)]


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
    lib.swept_shard_exchanges.restype = c_int64
    lib.swept_shard_exchanges.argtypes = [POINTER(swept_phase), c_int64, c_int32, c_int32, c_int64,
                                          POINTER(swept_exchange), c_int64]
    lib.swept_shard_create.restype = c_void_p
    lib.swept_shard_create.argtypes = [c_int, c_int64, c_int32, c_int32, c_int32, c_double, c_double,
                                       POINTER(swept_params)]
    lib.swept_shard_begin.restype = c_int64
    lib.swept_shard_begin.argtypes = [c_void_p, c_int64, c_int]
    lib.swept_shard_exchange_list.restype = c_int64
    lib.swept_shard_exchange_list.argtypes = [c_void_p, POINTER(swept_exchange), c_int64]
    lib.swept_shard_message_bytes.restype = c_int64
    lib.swept_shard_message_bytes.argtypes = [c_void_p, c_int64]
    lib.swept_shard_phase.argtypes = [c_void_p]
    lib.swept_shard_pack.argtypes = [c_void_p, c_int64, c_void_p]
    lib.swept_shard_unpack.argtypes = [c_void_p, c_int64, c_void_p]
    lib.swept_shard_end.argtypes = [c_void_p]
    lib.swept_shard_run.argtypes = [POINTER(c_void_p), c_int32, c_int64, c_int]
    lib.swept_heat_flow_static.argtypes = [c_void_p, c_void_p, c_int64, c_int64, c_int32, c_double, c_double, c_double,
                                           c_void_p]
    lib.swept_heat_flow_static_check.argtypes = [c_void_p]
    lib.swept_probe_fp64.argtypes = [c_int, c_void_p, POINTER(c_double)]
    lib.swept_probe_launch.argtypes = [c_int, c_void_p, c_int, POINTER(c_double)]
    lib.swept_probe_chain.argtypes = [c_int, c_void_p, POINTER(c_double)]
    lib.swept_probe_tier.argtypes = [c_int, c_void_p, POINTER(c_double)]
    lib.swept_probe_smem.argtypes = [c_int, c_void_p, POINTER(c_double), POINTER(c_double)]
    lib.swept_probe_sweep.argtypes = [c_int, c_void_p, c_int, c_int, c_int, POINTER(c_double), POINTER(c_double)]
    lib.swept_flow_profile.argtypes = [c_void_p, c_int, POINTER(c_uint64)]
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


def swept_flow_profile(state: int, on: bool):
    """Switch the instrumented FLOW kernel on / off; returns the counters accumulated so far as a dict of SM cycles
    summed over all warps (ticket, wait_parents, stage, sweep, publish) and the number of tiles."""
    c = (c_uint64 * 8)()
    _check(load().swept_flow_profile(state, 1 if on else 0, c))
    return {"ticket": int(c[0]), "wait_parents": int(c[1]), "stage": int(c[2]), "sweep": int(c[3]),
            "publish": int(c[4]), "tiles": int(c[5])}


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


def swept_shard_exchanges(plan, h: int, sigma: int, n_local: int):
    """Host-only: the edge exchanges that go with a phase list (tuples as returned by :func:`swept_plan`) for shards
    of ``n_local`` points: [(after_phase, dir, src_off, dst_off, count, rows), ...]."""
    lib = load()
    arr = (swept_phase * max(len(plan), 1))()
    for a, (kind, shift, tier0, ntiers, n) in zip(arr, plan):
        a.kind, a.shift, a.tier0, a.ntiers, a.n = kind, shift, tier0, ntiers, n
    cnt = lib.swept_shard_exchanges(arr, len(plan), h, sigma, n_local, None, 0)
    if cnt < 0:
        raise SweptError(f"swept_shard_exchanges: {swept_last_error()}")
    out = (swept_exchange * max(cnt, 1))()
    lib.swept_shard_exchanges(arr, len(plan), h, sigma, n_local, out, cnt)
    return [(int(x.after_phase), int(x.dir), int(x.src_off), int(x.dst_off), int(x.count), int(x.rows))
            for x in out[:cnt]]


STATIC_MAX_N = 65536  # SWEPT_STATIC_MAX_N


def swept_heat_flow_static(in_dev: int, out_dev: int, N: int, nsteps: int, tile_width: int, dx: float, dt: float,
                           alpha: float = 1.0, stream: int | None = None) -> None:
    """One swept cycle of the periodic FP64 heat problem with all scratch in the library's static device array: no
    allocation, no state.  ``in_dev`` / ``out_dev`` are DEVICE addresses of N doubles (e.g. ``tensor.data_ptr()``)."""
    st = _current_stream() if stream is None else stream
    _check(load().swept_heat_flow_static(in_dev, out_dev, N, nsteps, tile_width, dx, dt, alpha, st))


def swept_heat_flow_static_check(stream: int | None = None) -> None:
    st = _current_stream() if stream is None else stream
    _check(load().swept_heat_flow_static_check(st))


def swept_probe_fp64(device: int = -1) -> float:
    out = c_double(0)
    _check(load().swept_probe_fp64(device, _current_stream(), byref(out)))
    return float(out.value)


def swept_probe_chain(device: int = -1) -> float:
    """Cycles per dependent DADD -> DFMA pair (the critical path of one heat tier)."""
    out = c_double(0)
    _check(load().swept_probe_chain(device, _current_stream(), byref(out)))
    return float(out.value)


def swept_probe_tier(device: int = -1):
    """Cycles per link of a register-resident tier's dependent chain: (shuffle -> shuffle, two 64-bit shuffles -> DADD
    -> DFMA, the same -> select = one heat tier, DFMA -> select)."""
    out = (c_double * 4)()
    _check(load().swept_probe_tier(device, _current_stream(), out))
    return tuple(float(x) for x in out)


def swept_probe_smem(device: int = -1):
    """(bytes per second, bytes per clock per SM) of shared-memory reads on the whole device."""
    bps, bpc = c_double(0), c_double(0)
    _check(load().swept_probe_smem(device, _current_stream(), byref(bps), byref(bpc)))
    return float(bps.value), float(bpc.value)


def swept_probe_sweep(problem: int, lines_per_lane: int, warps_per_scheduler: int, device: int = -1):
    """(SM cycles per super-step, FP64 pipe busy fraction) of the characteristic sweep on one SM, no global traffic."""
    cyc, busy = c_double(0), c_double(0)
    _check(load().swept_probe_sweep(device, _current_stream(), problem, lines_per_lane, warps_per_scheduler,
                                    byref(cyc), byref(busy)))
    return float(cyc.value), float(busy.value)


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


class SweptShards:
    """A problem of N periodic points cut into contiguous shards (include/swept.h "sharding").

    ``ranks=None``: every shard lives in this process (``swept_shard_run``: one cudaMemcpyAsync per message).
    ``ranks=(rank, world)``: this process owns shard ``rank`` of ``world`` (one process per GPU) and the messages
    travel through :func:`_transport` — torch.distributed point-to-point — the only place an 8-GPU box differs.
    """

    def __init__(self, problem: int, N: int, nshards: int, tile_width: int, dx: float, dt: float, *, rk2: int = RK2_MIDPOINT,
                 alpha: float = 1.0, gamma: float = 1.4, dtype=np.float64, ranks=None):
        import torch
        if not torch.cuda.is_available():
            raise SweptError("no CUDA device: the swept library has no CPU fallback")
        lib = load()
        self.problem, self.N, self.nshards, self.n = problem, N, nshards, tile_width
        self.np_dtype = np.dtype(dtype)
        self.h, self.sigma, self.C = PROBLEM_SHAPE[problem]
        self.n_local = N // nshards
        self.ranks = ranks
        a, f = _torch_hooks()
        self._states = []
        for k in (range(nshards) if ranks is None else (ranks[0],)):
            p = swept_params()
            p.struct_size = ctypes.sizeof(swept_params)
            p.dtype = F64 if self.np_dtype == np.float64 else F32
            p.rk2, p.device, p.alpha, p.gamma, p.bc = rk2, -1, alpha, gamma, BC_PERIODIC
            p.alloc, p.free, p.stream = a, f, _current_stream()
            h = lib.swept_shard_create(problem, N, nshards, k, tile_width, dx, dt, byref(p))
            if not h:
                self.close()
                raise SweptError(f"swept_shard_create failed: {swept_last_error()}")
            self._states.append(h)

    @classmethod
    def from_workload(cls, w, nshards: int, tile_width: int, ranks=None) -> "SweptShards":
        s = cls(w.problem, w.N, nshards, tile_width, w.dx, w.dt, rk2=w.rk2, alpha=w.alpha, gamma=w.gamma, ranks=ranks)
        s.write(w.u0)
        return s

    def _own(self, k: int, field: np.ndarray) -> np.ndarray:
        """Shard k's points of a global component-major field."""
        f = field.reshape(self.C, self.N)[:, k * self.n_local:(k + 1) * self.n_local]
        return np.ascontiguousarray(f, dtype=self.np_dtype).reshape(-1)

    def write(self, u0: np.ndarray) -> None:
        self._keep = []
        ks = range(self.nshards) if self.ranks is None else (self.ranks[0],)
        for h, k in zip(self._states, ks):
            buf = self._own(k, np.asarray(u0))
            swept_set_stream(h, _current_stream())
            swept_write(h, buf)
            self._keep.append(buf)

    def read(self) -> np.ndarray:
        """The global field (single process) or this rank's own points (one process per shard)."""
        parts = []
        for h in self._states:
            out = np.empty(self.C * self.n_local, dtype=self.np_dtype)
            swept_set_stream(h, _current_stream())
            swept_read(h, out)
            parts.append(out.reshape(self.C, self.n_local))
        return np.concatenate(parts, axis=1).reshape(-1)

    def run(self, nsteps: int, flavor: int = FLAVOR_AUTO, group: int = 0) -> None:
        lib = load()
        for h in self._states:
            swept_set_stream(h, _current_stream())
        if self.ranks is None:
            arr = (c_void_p * len(self._states))(*self._states)
            _check(lib.swept_shard_run(arr, len(self._states), nsteps, flavor | (group << 8)))
            return
        import torch
        h = self._states[0]
        nph = lib.swept_shard_begin(h, nsteps, flavor | (group << 8))
        if nph < 0:
            raise SweptError(f"swept_shard_begin: {swept_last_error()}")
        nx = lib.swept_shard_exchange_list(h, None, 0)
        xs = (swept_exchange * max(nx, 1))()
        lib.swept_shard_exchange_list(h, xs, nx)
        ix = 0
        for i in range(-1, nph):
            if i >= 0:
                _check(lib.swept_shard_phase(h))
            while ix < nx and xs[ix].after_phase == i:
                nbytes = lib.swept_shard_message_bytes(h, ix)
                send = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
                recv = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
                _check(lib.swept_shard_pack(h, ix, c_void_p(send.data_ptr())))
                _transport(send, recv, int(xs[ix].dir), self.ranks[0], self.ranks[1])
                _check(lib.swept_shard_unpack(h, ix, c_void_p(recv.data_ptr())))
                ix += 1
        _check(lib.swept_shard_end(h))

    @property
    def last_launches(self) -> int:
        return sum(int(load().swept_last_launches(h)) for h in self._states)

    def close(self) -> None:
        for h in getattr(self, "_states", []):
            swept_destroy(h)
        self._states = []

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _transport(send, recv, direction: int, rank: int, world: int) -> None:
    """Move one edge message to the neighbour in `direction` (+1 right, -1 left) and receive the matching one from
    the other side, with torch.distributed point-to-point operations on the current stream's tensors.  NCCL moves
    device tensors directly (NVLink / NVSwitch); gloo (CPU tests, hosts without NCCL) goes through host copies."""
    import torch
    import torch.distributed as dist
    dst, src = (rank + direction) % world, (rank - direction) % world
    if dist.get_backend() == "nccl":
        ops = [dist.P2POp(dist.isend, send, dst), dist.P2POp(dist.irecv, recv, src)]
        for r in dist.batch_isend_irecv(ops):
            r.wait()
        return
    s_host = send.cpu()
    r_host = torch.empty_like(s_host)
    reqs = [dist.isend(s_host, dst), dist.irecv(r_host, src)]
    for r in reqs:
        r.wait()
    recv.copy_(r_host)

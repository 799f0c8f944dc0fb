"""ctypes binding of liblm.so -- argument marshalling only.

Module-level ``lib()`` returns the loaded library with every ``lm_*`` symbol of ``include/lm.h``
typed; ``Solver`` wraps a handle and forwards to the same-named C calls (``mdot`` -> ``lm_mdot``
...).  Tensors are torch CUDA tensors (device entry points) or numpy / CPU tensors (``*_host``
entry points); torch is used for device memory and streams only.

There is no fallback: if the library cannot be built or loaded, importing ``lib()`` raises.
"""
from __future__ import annotations

import ctypes
import weakref
import os
from ctypes import POINTER, c_char_p, c_double, c_int, c_int64, c_void_p

import numpy as np

LM_F32, LM_F64 = 0, 1
LM_OK, LM_E_INVALID, LM_E_NOPOS, LM_E_ANGULAR, LM_E_NULL, LM_E_CUDA, LM_E_NOCONV = 0, -1, -2, -3, -4, -5, -6
LM_RULE_ESTIMATE, LM_RULE_STEP = 0, 1
LM_OPT_LANCZOS_RULE, LM_OPT_GRAPH_REPLAY, LM_OPT_SHARE_FIRST_APPLY, LM_OPT_SMALL_KERNEL, LM_OPT_J_SPLITS, LM_OPT_GATHER_IN_PLACE, LM_OPT_ACCUMULATE_F64 = 0, 1, 2, 3, 4, 5, 6

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "liblm.so")
_lib = None

# name -> (restype, argtypes); mirrors include/lm.h one to one
SIGNATURES = {
    "lm_create": (c_int, [POINTER(c_void_p), c_int, c_int64, c_double, c_double, c_int]),
    "lm_destroy": (c_int, [c_void_p]),
    "lm_set_wall": (c_int, [c_void_p, c_int, c_double]),
    "lm_set_positions": (c_int, [c_void_p, c_void_p, c_void_p]),
    "lm_mdot": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]),
    "lm_mdot_batch": (c_int, [c_void_p, c_int, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]),
    "lm_sqrt_mdot_w": (c_int, [c_void_p, c_void_p, c_double, c_void_p, c_void_p, POINTER(c_int), c_void_p]),
    "lm_sqrt_mdot_w_batch": (c_int, [c_void_p, c_int, c_void_p, c_double, c_void_p, c_void_p, POINTER(c_int), c_void_p]),
    "lm_hydrodynamic_velocities": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_double, c_double, c_void_p, c_void_p, c_void_p]),
    "lm_set_positions_host": (c_int, [c_void_p, c_void_p, c_void_p]),
    "lm_mdot_host": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]),
    "lm_mdot_batch_host": (c_int, [c_void_p, c_int, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]),
    "lm_sqrt_mdot_w_host": (c_int, [c_void_p, c_void_p, c_double, c_void_p, c_void_p, POINTER(c_int), c_void_p]),
    "lm_hydrodynamic_velocities_host": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_double, c_double, c_void_p, c_void_p, c_void_p]),
    "lm_steric_forces": (c_int, [c_void_p, c_double, c_double, c_void_p, c_void_p, c_void_p]),
    "lm_bd_step": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_double, c_double, c_double, c_double, c_double, c_void_p]),
    "lm_bd_step_host": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_double, c_double, c_double, c_double, c_double, c_void_p]),
    "lm_bd_step_rfd": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_double, c_double, c_double, c_double, c_double, c_double,
                               c_void_p]),
    "lm_bd_step_rfd_host": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p, c_double, c_double, c_double, c_double, c_double,
                                    c_double, c_void_p]),
    "lm_bd_reset": (c_int, [c_void_p]),
    "lm_thermal_drift": (c_int, [c_void_p, c_void_p, c_void_p, c_void_p]),
    "lm_thermal_drift_rfd": (c_int, [c_void_p, c_void_p, c_double, c_void_p, c_void_p, c_void_p]),
    "lm_dist_row_block": (c_int, [c_int64, c_int, c_int, POINTER(c_int64), POINTER(c_int64)]),
    "lm_dist_unique_id": (c_int, [c_void_p]),
    "lm_dist_init": (c_int, [c_void_p, c_int, c_int, c_void_p]),
    "lm_mdot_rows": (c_int, [c_void_p, c_int64, c_int64, c_void_p, c_void_p, c_void_p, c_void_p, c_void_p]),
    "lm_set_option": (c_int, [c_void_p, c_int, c_int]),
    "lm_lanczos_history": (c_int, [c_void_p, c_int, c_int, POINTER(c_double), POINTER(c_double), POINTER(c_double), POINTER(c_double)]),
    "lm_set_max_iter": (c_int, [c_void_p, c_int]),
    "lm_last_iterations": (c_int, [c_void_p]),
    "lm_last_error": (c_char_p, [c_void_p]),
    "lm_set_profiling": (c_int, [c_void_p, c_int]),
    "lm_reset_stats": (c_int, [c_void_p]),
    "lm_get_stats": (c_int, [c_void_p, POINTER(c_int64), POINTER(c_int64), POINTER(c_double), POINTER(c_double)]),
    "lm_pair_launch_config": (c_int, [c_void_p, c_int, POINTER(c_int), POINTER(c_int), POINTER(c_int), POINTER(c_int), POINTER(c_int)]),
    "lm_pair_kernel_name": (c_char_p, [c_void_p, c_int]),
    "lm_mdot_static": (c_int, [c_int, c_int64, c_double, c_double, c_void_p, c_void_p, c_void_p, c_void_p]),
    "lm_mdot_static_max_n": (c_int64, []),
    "lm_mdot_static_error": (c_char_p, []),
    "lm_version": (c_char_p, []),
}


class LmError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"liblm error {code}: {message}")
        self.code = code


def lib():
    """Load liblm.so (building it in-tree with nvcc if it is missing or stale)."""
    global _lib
    if _lib is None:
        from . import build as _build
        path = _build.build() if (not os.path.exists(_LIB_PATH) or _build.stale()) else _LIB_PATH
        cdll = ctypes.CDLL(path)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(cdll, name)          # AttributeError here = the library is missing a declared symbol
            fn.restype, fn.argtypes = res, args
        _lib = cdll
    return _lib


def lm_version() -> str:
    return lib().lm_version().decode()


def lm_dist_row_block(N: int, nranks: int, rank: int):
    """(row_begin, row_end) of `rank`'s block of target rows -- host only, needs no GPU."""
    b, e = c_int64(0), c_int64(0)
    rc = lib().lm_dist_row_block(int(N), int(nranks), int(rank), ctypes.byref(b), ctypes.byref(e))
    if rc != LM_OK:
        raise LmError(rc, "lm_dist_row_block: need N > 0 and 0 <= rank < nranks")
    return b.value, e.value


def lm_dist_unique_id() -> bytes:
    buf = ctypes.create_string_buffer(128)
    rc = lib().lm_dist_unique_id(buf)
    if rc != LM_OK:
        raise LmError(rc, "lm_dist_unique_id: NCCL unavailable")
    return buf.raw


def lm_mdot_static_max_n() -> int:
    return int(lib().lm_mdot_static_max_n())


def mdot_static(precision, N: int, eta: float, a: float, positions, forces, lin_out, stream=None) -> None:
    """lm_mdot_static: lin_out = M_uF . forces (free space, translational) on the current device, WITHOUT any device
    allocation by the library -- for callers whose memory is spoken for (an engine that owns the whole card, a
    latency-critical loop that cannot take cudaMalloc's device-wide synchronisation, a fixed memory budget).  The scratch
    is a static array inside liblm.so (16 MiB per GPU, held until exit), hence the limit N <= lm_mdot_static_max_n().
    All calls on a GPU share that array: keep them on one stream (or order them), overlapping calls race.
    Torch CUDA tensors of 3N elements in the precision's dtype; argument marshalling only."""
    import torch
    prec = {"f32": LM_F32, "f64": LM_F64}.get(precision, precision)
    dt = torch.float32 if prec == LM_F32 else torch.float64
    for name, x in (("positions", positions), ("forces", forces), ("lin_out", lin_out)):
        if x is None or not x.is_cuda or x.dtype != dt or x.numel() != 3 * int(N) or not x.is_contiguous():
            raise TypeError(f"{name}: need a contiguous CUDA tensor of {3 * int(N)} elements of dtype {dt}")
    rc = lib().lm_mdot_static(int(prec), int(N), float(eta), float(a), _ptr(positions), _ptr(forces), _ptr(lin_out), _stream_ptr(stream))
    if rc != LM_OK:
        raise LmError(rc, lib().lm_mdot_static_error().decode())


def _ptr(x):
    """Raw address of a torch tensor / numpy array (None -> NULL).  No copies, no conversions."""
    if x is None:
        return None
    if isinstance(x, np.ndarray):
        if not x.flags["C_CONTIGUOUS"]:
            raise ValueError("array must be C-contiguous")
        return c_void_p(x.ctypes.data)
    if not x.is_contiguous():
        raise ValueError("tensor must be contiguous")
    return c_void_p(x.data_ptr())


def _raw_stream_fn():
    try:
        import torch
        return torch._C._cuda_getCurrentRawStream
    except Exception:
        return None


_RAW_STREAM = _raw_stream_fn()


def _stream_ptr(stream):
    if stream is None:
        import torch
        try:                               # the raw handle of torch's current stream, without building a Stream object
            return c_void_p(torch._C._cuda_getCurrentRawStream(torch.cuda.current_device()))
        except AttributeError:
            return c_void_p(torch.cuda.current_stream().cuda_stream)
    if isinstance(stream, int):
        return c_void_p(stream)
    return c_void_p(stream.cuda_stream)


class Solver:
    """A handle of liblm.  Methods map 1:1 to the C calls and only marshal arguments."""

    def __init__(self, precision: str | int, N: int, eta: float = 1.0, a: float = 1.0, include_angular: bool = False):
        self.precision = {"f32": LM_F32, "f64": LM_F64}.get(precision, precision)
        self.N, self.eta, self.a, self.angular = int(N), float(eta), float(a), bool(include_angular)
        self._h = c_void_p()
        rc = lib().lm_create(ctypes.byref(self._h), self.precision, self.N, self.eta, self.a, int(self.angular))
        if rc != LM_OK:
            self._h = c_void_p()
            raise LmError(rc, "lm_create failed (bad argument, or no CUDA device)")
        L = lib()
        self._n3, self._seen = 3 * self.N, {}
        self._lm_set_positions, self._lm_mdot, self._lm_mdot_batch, self._lm_sqrt_mdot_w = L.lm_set_positions, L.lm_mdot, L.lm_mdot_batch, L.lm_sqrt_mdot_w
        try:
            import torch
            self._device = torch.cuda.current_device()          # lm_create bound the handle to the current device
            self._tdtype = torch.float32 if self.precision == LM_F32 else torch.float64
        except Exception:
            self._device, self._tdtype = 0, None

    # -- helpers
    @property
    def torch_dtype(self):
        import torch
        return torch.float32 if self.precision == LM_F32 else torch.float64

    @property
    def np_dtype(self):
        return np.float32 if self.precision == LM_F32 else np.float64

    def _check(self, rc, allow=()):
        if rc != LM_OK and rc not in allow:
            raise LmError(rc, lib().lm_last_error(self._h).decode())
        return rc

    def _expect(self, x, n, host):
        if x is None:
            return
        dt = self.np_dtype if host else self.torch_dtype
        if x.dtype != dt:
            raise TypeError(f"expected dtype {dt}, got {x.dtype}")
        size = x.size if isinstance(x, np.ndarray) else x.numel()
        if size != n:
            raise ValueError(f"expected {n} elements, got {size}")
        if not host and not x.is_cuda:
            raise TypeError("device entry point needs a CUDA tensor (use the *_host call for host arrays)")

    def _dev(self, x, n):
        """Device argument of a hot call: the tensor's address as an int (None -> NULL).  Size, dtype and device are
        checked on EVERY call (three attribute reads: a tensor can change under the same Python object -- resize_, set_,
        `.data =` -- and a stale length would be an out-of-bounds device access, not a TypeError); only the contiguity
        walk is remembered per tensor object and re-done when the object, its size or its storage offset changes.  A
        time-stepping loop calls with the same few tensors millions of times and a small apply is otherwise bound by this
        marshalling."""
        if x is None:
            return None
        if x.numel() != n or x.dtype != self._tdtype or not x.is_cuda:
            self._expect(x, n, False)          # raises with the precise reason
        seen = self._seen
        ent = seen.get(id(x))
        if ent is None or ent[0]() is not x or ent[1] != x.stride():
            if not x.is_contiguous():
                raise ValueError("tensor must be contiguous")
            if len(seen) > 256:
                seen.clear()
            seen[id(x)] = (weakref.ref(x), x.stride())
        return x.data_ptr()

    def _stream(self, stream):
        if stream is None:
            return _RAW_STREAM(self._device) if _RAW_STREAM is not None else _stream_ptr(None)
        return stream if isinstance(stream, int) else stream.cuda_stream

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            lib().lm_destroy(self._h)
            self._h = c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_wall(self, enabled: bool, wall_height: float = 0.0):
        """Geometry ("open","open","single_wall") with the wall at z = wall_height."""
        self._check(lib().lm_set_wall(self._h, int(bool(enabled)), float(wall_height)))

    # -- device entry points (torch CUDA tensors)
    def set_positions(self, pos, stream=None):
        rc = self._lm_set_positions(self._h, self._dev(pos, self._n3), self._stream(stream))
        if rc != LM_OK:
            self._check(rc)

    def mdot(self, forces, torques, lin_out, ang_out=None, stream=None):
        n3, d = self._n3, self._dev
        rc = self._lm_mdot(self._h, d(forces, n3), d(torques, n3), d(lin_out, n3), d(ang_out, n3), self._stream(stream))
        if rc != LM_OK:
            self._check(rc)

    def mdot_batch(self, nrhs, forces, torques, lin_out, ang_out=None, stream=None):
        n, d = nrhs * self._n3, self._dev
        rc = self._lm_mdot_batch(self._h, int(nrhs), d(forces, n), d(torques, n), d(lin_out, n), d(ang_out, n), self._stream(stream))
        if rc != LM_OK:
            self._check(rc)

    def sqrt_mdot_w(self, noise, tol, lin_out, ang_out=None, stream=None, allow_noconv=False) -> int:
        n3, d = self._n3, self._dev
        iters = c_int(0)
        self._check(self._lm_sqrt_mdot_w(self._h, d(noise, (2 if self.angular else 1) * n3), float(tol), d(lin_out, n3), d(ang_out, n3),
                                         ctypes.byref(iters), self._stream(stream)), allow=(LM_E_NOCONV,) if allow_noconv else ())
        return iters.value

    def sqrt_mdot_w_batch(self, nvec, noise, tol, lin_out, ang_out=None, stream=None, allow_noconv=False):
        self._expect(noise, nvec * (6 if self.angular else 3) * self.N, False)
        for x in (lin_out, ang_out):
            self._expect(x, nvec * 3 * self.N, False)
        iters = (c_int * int(nvec))()
        self._check(lib().lm_sqrt_mdot_w_batch(self._h, int(nvec), _ptr(noise), float(tol), _ptr(lin_out), _ptr(ang_out), iters,
                                               _stream_ptr(stream)), allow=(LM_E_NOCONV,) if allow_noconv else ())
        return list(iters)

    def hydrodynamic_velocities(self, forces, torques, noise, noise_prefactor, tol, lin_out, ang_out=None, stream=None):
        n3, d = self._n3, self._dev
        self._check(lib().lm_hydrodynamic_velocities(self._h, d(forces, n3), d(torques, n3), d(noise, (2 if self.angular else 1) * n3),
                                                     float(noise_prefactor), float(tol), d(lin_out, n3), d(ang_out, n3), self._stream(stream)))

    # -- host entry points (numpy arrays; pinned memory makes the copies asynchronous)
    def set_positions_host(self, pos, stream=None):
        self._expect(pos, 3 * self.N, True)
        self._check(lib().lm_set_positions_host(self._h, _ptr(pos), _stream_ptr(stream)))

    def mdot_host(self, forces, torques, lin_out, ang_out=None, stream=None):
        for x in (forces, torques, lin_out, ang_out):
            self._expect(x, 3 * self.N, True)
        self._check(lib().lm_mdot_host(self._h, _ptr(forces), _ptr(torques), _ptr(lin_out), _ptr(ang_out), _stream_ptr(stream)))

    def mdot_batch_host(self, nrhs, forces, torques, lin_out, ang_out=None, stream=None):
        for x in (forces, torques, lin_out, ang_out):
            self._expect(x, nrhs * 3 * self.N, True)
        self._check(lib().lm_mdot_batch_host(self._h, int(nrhs), _ptr(forces), _ptr(torques), _ptr(lin_out), _ptr(ang_out), _stream_ptr(stream)))

    def sqrt_mdot_w_host(self, noise, tol, lin_out, ang_out=None, stream=None) -> int:
        self._expect(noise, (6 if self.angular else 3) * self.N, True)
        iters = c_int(0)
        self._check(lib().lm_sqrt_mdot_w_host(self._h, _ptr(noise), float(tol), _ptr(lin_out), _ptr(ang_out), ctypes.byref(iters),
                                              _stream_ptr(stream)))
        return iters.value

    def hydrodynamic_velocities_host(self, forces, torques, noise, noise_prefactor, tol, lin_out, ang_out=None, stream=None):
        self._check(lib().lm_hydrodynamic_velocities_host(self._h, _ptr(forces), _ptr(torques), _ptr(noise), float(noise_prefactor),
                                                          float(tol), _ptr(lin_out), _ptr(ang_out), _stream_ptr(stream)))

    # -- free-space Brownian-dynamics step (eqs. (13), (14))
    def steric_forces(self, U0, b, ext_forces, forces_out, stream=None):
        for x in (ext_forces, forces_out):
            self._expect(x, 3 * self.N, False)
        self._check(lib().lm_steric_forces(self._h, float(U0), float(b), _ptr(ext_forces), _ptr(forces_out), _stream_ptr(stream)))

    def bd_step(self, pos, ext_forces, ext_torques, noise, dt, kT, U0, b, tol, stream=None, allow_noconv=False) -> int:
        for x in (pos, ext_forces, ext_torques):
            self._expect(x, 3 * self.N, False)
        self._expect(noise, (6 if self.angular else 3) * self.N, False)
        return self._check(lib().lm_bd_step(self._h, _ptr(pos), _ptr(ext_forces), _ptr(ext_torques), _ptr(noise), float(dt), float(kT),
                                            float(U0), float(b), float(tol), _stream_ptr(stream)), allow=(LM_E_NOCONV,) if allow_noconv else ())

    def bd_step_host(self, pos, ext_forces, ext_torques, noise, dt, kT, U0, b, tol, stream=None, allow_noconv=False) -> int:
        for x in (pos, ext_forces, ext_torques):
            self._expect(x, 3 * self.N, True)
        self._expect(noise, (6 if self.angular else 3) * self.N, True)
        return self._check(lib().lm_bd_step_host(self._h, _ptr(pos), _ptr(ext_forces), _ptr(ext_torques), _ptr(noise), float(dt), float(kT),
                                                 float(U0), float(b), float(tol), _stream_ptr(stream)), allow=(LM_E_NOCONV,) if allow_noconv else ())

    def bd_step_rfd(self, pos, ext_forces, ext_torques, noise, rfd_noise, rfd_delta, dt, kT, U0, b, tol, stream=None, allow_noconv=False) -> int:
        """lm_bd_step with the thermal-drift term of eq. (14) as one RFD sample (W~ = rfd_noise, 3N)."""
        for x in (pos, ext_forces, ext_torques, rfd_noise):
            self._expect(x, 3 * self.N, False)
        self._expect(noise, (6 if self.angular else 3) * self.N, False)
        return self._check(lib().lm_bd_step_rfd(self._h, _ptr(pos), _ptr(ext_forces), _ptr(ext_torques), _ptr(noise), _ptr(rfd_noise), float(rfd_delta),
                                                float(dt), float(kT), float(U0), float(b), float(tol), _stream_ptr(stream)),
                           allow=(LM_E_NOCONV,) if allow_noconv else ())

    def bd_step_rfd_host(self, pos, ext_forces, ext_torques, noise, rfd_noise, rfd_delta, dt, kT, U0, b, tol, stream=None, allow_noconv=False) -> int:
        for x in (pos, ext_forces, ext_torques, rfd_noise):
            self._expect(x, 3 * self.N, True)
        self._expect(noise, (6 if self.angular else 3) * self.N, True)
        return self._check(lib().lm_bd_step_rfd_host(self._h, _ptr(pos), _ptr(ext_forces), _ptr(ext_torques), _ptr(noise), _ptr(rfd_noise),
                                                     float(rfd_delta), float(dt), float(kT), float(U0), float(b), float(tol), _stream_ptr(stream)),
                           allow=(LM_E_NOCONV,) if allow_noconv else ())

    def bd_reset(self):
        self._check(lib().lm_bd_reset(self._h))

    # -- row-sharded applies
    def dist_init(self, nranks: int, rank: int, unique_id: bytes):
        assert len(unique_id) == 128
        self._check(lib().lm_dist_init(self._h, int(nranks), int(rank), ctypes.create_string_buffer(unique_id, 128)))

    def mdot_rows(self, row_begin, row_count, forces, torques, lin_out, ang_out=None, stream=None):
        for x in (forces, torques, lin_out, ang_out):
            self._expect(x, 3 * self.N, False)
        self._check(lib().lm_mdot_rows(self._h, int(row_begin), int(row_count), _ptr(forces), _ptr(torques), _ptr(lin_out), _ptr(ang_out),
                                       _stream_ptr(stream)))

    # -- thermal drift (the paper's divM)
    def thermal_drift(self, lin_out, ang_out=None, stream=None):
        for x in (lin_out, ang_out):
            self._expect(x, 3 * self.N, False)
        self._check(lib().lm_thermal_drift(self._h, _ptr(lin_out), _ptr(ang_out), _stream_ptr(stream)))

    def thermal_drift_rfd(self, noise, delta, lin_out, ang_out=None, stream=None):
        for x in (noise, lin_out, ang_out):
            self._expect(x, 3 * self.N, False)
        self._check(lib().lm_thermal_drift_rfd(self._h, _ptr(noise), float(delta), _ptr(lin_out), _ptr(ang_out), _stream_ptr(stream)))

    # -- controls / introspection
    def set_option(self, option: int, value: int):
        self._check(lib().lm_set_option(self._h, int(option), int(value)))

    def lanczos_history(self, vec: int = 0) -> dict:
        """alpha_k, beta_k, relative step s_k and error estimate e_k of the last Lanczos call, k = 1 .. iterations."""
        dp = POINTER(c_double)
        cap = 1001
        arrs = [np.full(cap, np.nan) for _ in range(4)]
        k = lib().lm_lanczos_history(self._h, int(vec), cap, *[a.ctypes.data_as(dp) for a in arrs])
        return dict(zip(("alpha", "beta", "step", "estimate"), (a[:k] for a in arrs)))

    def set_max_iter(self, n):
        self._check(lib().lm_set_max_iter(self._h, int(n)))

    def last_iterations(self) -> int:
        return lib().lm_last_iterations(self._h)

    def last_error(self) -> str:
        return lib().lm_last_error(self._h).decode()

    def set_profiling(self, on: bool):
        self._check(lib().lm_set_profiling(self._h, int(on)))

    def reset_stats(self):
        self._check(lib().lm_reset_stats(self._h))

    def get_stats(self) -> dict:
        a, b, ms, pairs = c_int64(0), c_int64(0), c_double(0), c_double(0)
        self._check(lib().lm_get_stats(self._h, ctypes.byref(a), ctypes.byref(b), ctypes.byref(ms), ctypes.byref(pairs)))
        return dict(pair_kernel_launches=a.value, aux_launches=b.value, pair_kernel_ms=ms.value, pairs=pairs.value)

    def pair_launch_config(self, nrhs: int = 1) -> dict:
        v = [c_int(0) for _ in range(5)]
        self._check(lib().lm_pair_launch_config(self._h, int(nrhs), *[ctypes.byref(x) for x in v]))
        keys = ("i_tiles", "j_splits", "block", "targets_per_thread", "smem_bytes")
        out = {k: x.value for k, x in zip(keys, v)}
        out["kernel"] = lib().lm_pair_kernel_name(self._h, int(nrhs)).decode()
        return out

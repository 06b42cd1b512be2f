"""Thin ctypes binding of the C ABI in include/ds.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of csrc/; this module holds no arithmetic of
the method and has NO CPU fallback: if libds.so cannot be built/loaded, or there is no sm_100
device, the calls raise.  torch is used only for device memory and streams: any object with a
`data_ptr()` (torch tensor, device or pinned/pageable host) or a numpy array is accepted as a
buffer; the library itself tells host from device pointers.
"""
import ctypes
import os

import numpy as np

from . import build as _build

F32, F64 = 0, 1
OSEEN, RPY = 0, 1
EULER, HEUN = 0, 1

OK = 0
ERR_INVALID_PARAM, ERR_NULL, ERR_CUDA, ERR_STATE, ERR_NO_DEVICE, ERR_ALLOC, ERR_TOO_LARGE = -1, -2, -3, -4, -5, -6, -7
MSD_STATIC_MAX_PARTIALS = 16384

# every symbol include/ds.h declares (tests check that the built library exports all of them)
SYMBOLS = ["ds_create", "ds_destroy", "ds_set_stream", "ds_set_state", "ds_get_state", "ds_forces",
           "ds_mobility_apply", "ds_step", "ds_batch_step", "ds_velocity", "ds_dumbbell_coords", "ds_msd_set_reference", "ds_msd", "ds_msd_static", "ds_avg_rhs", "ds_avg_step", "ds_strerror", "ds_last_cuda_error", "ds_version"]
# development / measurement hooks (include/ds_dev.h)
DEV_SYMBOLS = ["ds_set_tuning", "ds_set_probe", "ds_launch_count", "ds_peak_probe", "ds_set_pipeline", "ds_pipeline_active"]


class DsError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        L = lib()
        msg = L.ds_strerror(code).decode()
        cu = L.ds_last_cuda_error().decode()
        super().__init__(f"{where}: {msg} ({code})" + (f" [{cu}]" if code == ERR_CUDA and cu else ""))


class Params(ctypes.Structure):
    """Mirror of ds_params (include/ds.h)."""
    _fields_ = [("n_dumbbells", ctypes.c_int32), ("n_batch", ctypes.c_int32), ("precision", ctypes.c_int32),
                ("tensor", ctypes.c_int32), ("integrator", ctypes.c_int32), ("device", ctypes.c_int32),
                ("a", ctypes.c_double), ("eta", ctypes.c_double), ("ell", ctypes.c_double),
                ("lam", ctypes.c_double), ("omega", ctypes.c_double), ("k0", ctypes.c_double),
                ("dt", ctypes.c_double), ("stream", ctypes.c_void_p), ("kT", ctypes.c_double), ("seed", ctypes.c_uint64)]


_lib = None


def lib():
    """Build (if stale) and load libds.so.  Raises if that fails: there is no fallback."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = ctypes.CDLL(path)
        vp, i32, i64, dbl = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_double
        L.ds_create.argtypes = [ctypes.POINTER(Params), ctypes.POINTER(vp)]
        L.ds_destroy.argtypes = [vp]
        L.ds_set_stream.argtypes = [vp, vp]
        L.ds_set_state.argtypes = [vp, vp, vp, dbl]
        L.ds_get_state.argtypes = [vp, vp, ctypes.POINTER(dbl)]
        L.ds_forces.argtypes = [vp, vp]
        L.ds_mobility_apply.argtypes = [vp, vp, vp, vp, i32]
        L.ds_step.argtypes = [vp, i64]
        L.ds_batch_step.argtypes = [vp, i64]
        L.ds_velocity.argtypes = [vp, vp]
        L.ds_dumbbell_coords.argtypes = [vp, vp, vp]
        L.ds_avg_rhs.argtypes = [vp, vp, vp, vp, vp, vp, i32]
        L.ds_avg_step.argtypes = [vp, vp, vp, vp, i32, dbl, i64]
        L.ds_msd_set_reference.argtypes = [vp]
        L.ds_msd.argtypes = [vp, ctypes.POINTER(dbl)]
        L.ds_msd_static.argtypes = [vp, vp, i32, i32, vp, vp, i32]
        L.ds_set_tuning.argtypes = [vp, i32]
        L.ds_set_probe.argtypes = [vp, vp]
        L.ds_set_pipeline.argtypes = [vp, i32]
        L.ds_pipeline_active.argtypes = [vp]
        L.ds_launch_count.argtypes = [vp]
        L.ds_launch_count.restype = i64
        L.ds_peak_probe.argtypes = [i32, i32, ctypes.POINTER(dbl)]
        for f in ("ds_strerror", "ds_last_cuda_error", "ds_version"):
            getattr(L, f).restype = ctypes.c_char_p
        L.ds_strerror.argtypes = [ctypes.c_int]
        _lib = L
    return _lib


def version():
    return lib().ds_version().decode()


def peak_probe(precision, device=0):
    """Measured FMA-chain peak of `device` in FLOP/s (FMA = 2)."""
    v = ctypes.c_double()
    _check(lib().ds_peak_probe(int(precision), int(device), ctypes.byref(v)), "ds_peak_probe")
    return v.value


def _ptr(x):
    """Raw address of a torch tensor / numpy array (must be contiguous); None -> NULL."""
    if x is None:
        return None
    if hasattr(x, "data_ptr"):
        if not x.is_contiguous():
            raise ValueError("buffer must be contiguous")
        return ctypes.c_void_p(x.data_ptr())
    if isinstance(x, np.ndarray):
        if not x.flags["C_CONTIGUOUS"]:
            raise ValueError("buffer must be contiguous")
        return ctypes.c_void_p(x.ctypes.data)
    if isinstance(x, int):
        return ctypes.c_void_p(x)
    raise TypeError(f"unsupported buffer type {type(x)}")


def _check(code, where):
    if code != OK:
        raise DsError(code, where)


def msd_static(X, Rref, S, W, out, stream=None, device=0):
    """ds_msd_static: Eq. (13) from device arrays X [W][2S][3], Rref [W][S][3] (FP64) into the device double `out`;
    allocates nothing (scratch = a static device array shared by all calls: do not overlap calls on the GPU)."""
    _check(lib().ds_msd_static(_ptr(X), _ptr(Rref), int(S), int(W), _ptr(out), ctypes.c_void_p(stream or 0), int(device)),
           "ds_msd_static")


class System:
    """Owner of one ds_system handle; method names and arguments follow include/ds.h."""

    def __init__(self, n_dumbbells, n_batch=1, precision=F64, tensor=RPY, integrator=HEUN, a=1.0, eta=1.0,
                 ell=10.0, lam=2.0, omega=2.0 * np.pi, k0=1000.0, dt=1e-3, device=0, stream=None, kT=0.0, seed=0):
        self._h = ctypes.c_void_p()
        self.params = Params(int(n_dumbbells), int(n_batch), int(precision), int(tensor), int(integrator),
                             int(device), float(a), float(eta), float(ell), float(lam), float(omega),
                             float(k0), float(dt), ctypes.c_void_p(stream) if stream else None, float(kT), int(seed))
        _check(lib().ds_create(ctypes.byref(self.params), ctypes.byref(self._h)), "ds_create")
        self.S, self.N, self.B = int(n_dumbbells), 2 * int(n_dumbbells), int(n_batch)
        self.precision = int(precision)

    def destroy(self):
        if self._h:
            lib().ds_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    def set_stream(self, stream):
        _check(lib().ds_set_stream(self._h, ctypes.c_void_p(stream) if stream else None), "ds_set_stream")

    def set_state(self, pos, phase, t0=0.0):
        _check(lib().ds_set_state(self._h, _ptr(pos), _ptr(phase), float(t0)), "ds_set_state")

    def get_state(self, pos=None):
        t = ctypes.c_double()
        _check(lib().ds_get_state(self._h, _ptr(pos), ctypes.byref(t)), "ds_get_state")
        return t.value

    def forces(self, F):
        _check(lib().ds_forces(self._h, _ptr(F)), "ds_forces")

    def velocity(self, V):
        _check(lib().ds_velocity(self._h, _ptr(V)), "ds_velocity")

    def dumbbell_coords(self, R=None, Nv=None):
        _check(lib().ds_dumbbell_coords(self._h, _ptr(R), _ptr(Nv)), "ds_dumbbell_coords")

    def msd_set_reference(self):
        _check(lib().ds_msd_set_reference(self._h), "ds_msd_set_reference")

    def msd(self):
        v = ctypes.c_double()
        _check(lib().ds_msd(self._h, ctypes.byref(v)), "ds_msd")
        return v.value

    def avg_rhs(self, R, Nv, phase, dR, dN, S):
        _check(lib().ds_avg_rhs(self._h, _ptr(R), _ptr(Nv), _ptr(phase), _ptr(dR), _ptr(dN), int(S)), "ds_avg_rhs")

    def avg_step(self, R, Nv, phase, S, dt, n_steps):
        _check(lib().ds_avg_step(self._h, _ptr(R), _ptr(Nv), _ptr(phase), int(S), float(dt), int(n_steps)), "ds_avg_step")

    def mobility_apply(self, pos, F, u, n):
        _check(lib().ds_mobility_apply(self._h, _ptr(pos), _ptr(F), _ptr(u), int(n)), "ds_mobility_apply")

    def step(self, n_steps):
        _check(lib().ds_step(self._h, int(n_steps)), "ds_step")

    def batch_step(self, n_steps):
        _check(lib().ds_batch_step(self._h, int(n_steps)), "ds_batch_step")

    def set_tuning(self, n_tiles=0):
        _check(lib().ds_set_tuning(self._h, int(n_tiles)), "ds_set_tuning")

    def set_pipeline(self, mode=-1):
        _check(lib().ds_set_pipeline(self._h, int(mode)), "ds_set_pipeline")

    def pipeline_active(self):
        return int(lib().ds_pipeline_active(self._h))   # 0 one-pass / warp-per-system, 1 pipelined, 2 cluster kernel

    def set_probe(self, buf=None):
        _check(lib().ds_set_probe(self._h, _ptr(buf)), "ds_set_probe")

    def launch_count(self):
        return int(lib().ds_launch_count(self._h))

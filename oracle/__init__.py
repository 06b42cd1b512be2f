"""CPU oracle for the active-dumbbell hot path of arXiv 1004.1932.

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  The arithmetic lives in
oracle/ds_oracle.c (plain C, fp64, scalar loops, each function citing the paper); this file
is the ctypes marshalling around it and holds none of the method's arithmetic.  It imports
nothing from paper_1004_1932_b200.
"""
import ctypes
from dataclasses import dataclass

import numpy as np

from . import build as _build

OSEEN, RPY = 0, 1
EULER, HEUN = 0, 1


class _CParams(ctypes.Structure):
    _fields_ = [("a", ctypes.c_double), ("eta", ctypes.c_double), ("ell", ctypes.c_double),
                ("lam", ctypes.c_double), ("omega", ctypes.c_double), ("k0", ctypes.c_double),
                ("dt", ctypes.c_double), ("tensor", ctypes.c_int32), ("integrator", ctypes.c_int32),
                ("kT", ctypes.c_double), ("seed", ctypes.c_uint64), ("system", ctypes.c_int32)]


@dataclass
class Params:
    """Scalars of the model.  Defaults: BASELINE.json units a=eta=T=1."""
    a: float = 1.0
    eta: float = 1.0
    ell: float = 10.0
    lam: float = 2.0
    omega: float = 2.0 * np.pi
    k0: float = 1000.0
    dt: float = 1e-3
    tensor: int = RPY
    integrator: int = HEUN
    kT: float = 0.0        # thermal energy of Eq. (1a); 0 = the deterministic limit the paper simulates
    seed: int = 0          # key of the counter-based generator
    system: int = 0        # index w of the realisation (enters the generator's counter)

    def c(self) -> _CParams:
        return _CParams(self.a, self.eta, self.ell, self.lam, self.omega, self.k0, self.dt,
                        int(self.tensor), int(self.integrator), float(self.kT), int(self.seed), int(self.system))


_lib = None
_dp = ctypes.POINTER(ctypes.c_double)


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(_build.build())
        L.or_set_threads.argtypes = [ctypes.c_int]
        L.or_get_threads.restype = ctypes.c_int
        L.or_max_threads.restype = ctypes.c_int
        L.or_forces.argtypes = [ctypes.c_int32, _dp, _dp, ctypes.c_double, ctypes.POINTER(_CParams), _dp]
        L.or_dense_mobility.argtypes = [ctypes.c_int32, _dp, ctypes.c_double, ctypes.c_double, ctypes.c_int32, _dp]
        L.or_mobility_apply.argtypes = [ctypes.c_int32, _dp, _dp, ctypes.c_double, ctypes.c_double,
                                        ctypes.c_int32, _dp]
        L.or_velocity.argtypes = [ctypes.c_int32, _dp, _dp, ctypes.c_double, ctypes.POINTER(_CParams), _dp, _dp]
        L.or_step.argtypes = [ctypes.c_int32, _dp, _dp, ctypes.c_double, ctypes.c_int64, ctypes.c_int64,
                              ctypes.POINTER(_CParams)]
        L.or_step.restype = ctypes.c_int
        L.or_step_record.argtypes = [ctypes.c_int32, _dp, _dp, ctypes.c_double, ctypes.c_int64, ctypes.c_int64,
                                     ctypes.POINTER(_CParams), ctypes.c_int64, _dp]
        L.or_step_record.restype = ctypes.c_int
        L.or_philox4x32_10.argtypes = [ctypes.POINTER(ctypes.c_uint32)] * 3
        L.or_noise_normal.argtypes = [ctypes.c_uint64, ctypes.c_int64, ctypes.c_int32, ctypes.c_int64]
        L.or_noise_normal.restype = ctypes.c_double
        L.or_avg_rhs.argtypes = [ctypes.c_int32, _dp, _dp, _dp, ctypes.POINTER(_CParams), _dp, _dp]
        L.or_avg_step.argtypes = [ctypes.c_int32, _dp, _dp, _dp, ctypes.c_double, ctypes.c_int64, ctypes.POINTER(_CParams)]
        L.or_avg_step.restype = ctypes.c_int
        L.or_dumbbell_coords.argtypes = [ctypes.c_int32, _dp, _dp, _dp]
        L.or_msd.argtypes = [ctypes.c_int32, ctypes.c_int32, _dp, _dp]
        L.or_msd.restype = ctypes.c_double
        _lib = L
    return _lib


def _d(x):
    x = np.ascontiguousarray(x, dtype=np.float64)
    return x, x.ctypes.data_as(_dp)


def set_threads(n: int) -> None:
    lib().or_set_threads(int(n))


def max_threads() -> int:
    return int(lib().or_max_threads())


def forces(X, phi, t, p: Params):
    """Eq. (4).  X [N][3], phi [S] -> F [N][3]."""
    X, Xp = _d(X)
    phi, pp = _d(phi)
    S = phi.shape[0]
    assert X.shape == (2 * S, 3)
    F = np.empty_like(X)
    cp = p.c()
    lib().or_forces(S, Xp, pp, float(t), ctypes.byref(cp), F.ctypes.data_as(_dp))
    return F


def dense_mobility(X, a, eta, tensor):
    """Eq. (3a,b) entry by entry.  X [N][3] -> H [3N][3N]."""
    X, Xp = _d(X)
    N = X.shape[0]
    H = np.empty((3 * N, 3 * N), dtype=np.float64)
    lib().or_dense_mobility(N, Xp, float(a), float(eta), int(tensor), H.ctypes.data_as(_dp))
    return H


def mobility_apply(X, F, a, eta, tensor):
    """u = H(X) F, matrix free.  X, F [N][3] -> u [N][3]."""
    X, Xp = _d(X)
    F, Fp = _d(F)
    assert X.shape == F.shape and X.shape[1] == 3
    u = np.empty_like(X)
    lib().or_mobility_apply(X.shape[0], Xp, Fp, float(a), float(eta), int(tensor), u.ctypes.data_as(_dp))
    return u


def velocity(X, phi, t, p: Params):
    X, Xp = _d(X)
    phi, pp = _d(phi)
    V = np.empty_like(X)
    W = np.empty_like(X)
    cp = p.c()
    lib().or_velocity(phi.shape[0], Xp, pp, float(t), ctypes.byref(cp), V.ctypes.data_as(_dp),
                      W.ctypes.data_as(_dp))
    return V


def step(X, phi, t0, n_done, n_steps, p: Params):
    """n_steps explicit steps from step index n_done; returns the new X (input untouched)."""
    X = np.array(X, dtype=np.float64, order="C", copy=True)
    phi, pp = _d(phi)
    assert X.shape == (2 * phi.shape[0], 3)
    cp = p.c()
    rc = lib().or_step(phi.shape[0], X.ctypes.data_as(_dp), pp, float(t0), int(n_done), int(n_steps),
                       ctypes.byref(cp))
    if rc:
        raise MemoryError("or_step")
    return X


def step_record(X, phi, t0, n_done, n_steps, p: Params, stride: int):
    """As step(), also returning the positions after every stride-th step: (X, traj[k][N][3])."""
    X = np.array(X, dtype=np.float64, order="C", copy=True)
    phi, pp = _d(phi)
    cp = p.c()
    traj = np.empty((n_steps // stride,) + X.shape, dtype=np.float64)
    rc = lib().or_step_record(phi.shape[0], X.ctypes.data_as(_dp), pp, float(t0), int(n_done), int(n_steps),
                              ctypes.byref(cp), int(stride), traj.ctypes.data_as(_dp))
    if rc:
        raise MemoryError("or_step_record")
    return X, traj


def dumbbell_coords(X):
    """Eq. (6a), (6b): X [2S][3] -> (R [S][3], N [S][3])."""
    X, xp = _d(X)
    S = X.shape[0] // 2
    R = np.empty((S, 3), dtype=np.float64)
    Nv = np.empty((S, 3), dtype=np.float64)
    lib().or_dumbbell_coords(S, xp, R.ctypes.data_as(_dp), Nv.ctypes.data_as(_dp))
    return R, Nv


def msd(Rt, R0):
    """Eq. (13): Rt, R0 [W][S][3] -> <<R(t)^2>>."""
    Rt, rp = _d(Rt)
    R0, r0p = _d(R0)
    assert Rt.shape == R0.shape and Rt.ndim == 3
    return float(lib().or_msd(Rt.shape[0], Rt.shape[1], rp, r0p))


def philox4x32_10(ctr, key):
    """The generator behind the Brownian increments: counter [4] uint32, key [2] uint32 -> [4] uint32."""
    c = (ctypes.c_uint32 * 4)(*[int(v) & 0xffffffff for v in ctr])
    k = (ctypes.c_uint32 * 2)(*[int(v) & 0xffffffff for v in key])
    o = (ctypes.c_uint32 * 4)()
    lib().or_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def noise_normal(seed, n, system, element):
    """z ~ N(0,1) of step n, realisation `system`, state element 3 alpha + i (Eq. 1b, 1c)."""
    return float(lib().or_noise_normal(int(seed), int(n), int(system), int(element)))


def avg_rhs(R, N, phi, p: Params):
    """Stroke-averaged far-field model, Eq. (9a)-(9d): (dR/dt, dN/dt), each [S][3]."""
    R, rp = _d(R)
    N, np_ = _d(N)
    phi, pp = _d(phi)
    cp = p.c()
    dR = np.empty_like(R)
    dN = np.empty_like(N)
    lib().or_avg_rhs(R.shape[0], rp, np_, pp, ctypes.byref(cp), dR.ctypes.data_as(_dp), dN.ctypes.data_as(_dp))
    return dR, dN


def avg_step(R, N, phi, dt, n_steps, p: Params):
    """n_steps Heun steps of Eq. (9) with step dt (N renormalised after every stage): (R, N)."""
    R = np.array(R, dtype=np.float64, order="C", copy=True)
    N = np.array(N, dtype=np.float64, order="C", copy=True)
    phi, pp = _d(phi)
    cp = p.c()
    rc = lib().or_avg_step(R.shape[0], R.ctypes.data_as(_dp), N.ctypes.data_as(_dp), pp, float(dt), int(n_steps), ctypes.byref(cp))
    if rc:
        raise MemoryError("or_avg_step")
    return R, N

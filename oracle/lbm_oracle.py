"""ctypes front end of the CPU oracle (oracle/lbm_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this.  It never imports the CUDA package.
All arrays are numpy float64, C-contiguous, indexed i = (ix*ny + iy)*nz + iz.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

MODELS = {"BGK_W2": 0, "BGK_NW4": 1, "TRT": 2, "RM": 3, "HM": 4, "CM": 5, "CHM": 6, "K": 7, "RR": 8, "REG": 9}
BASES = {"raw": 0, "hermite": 1, "central": 2, "central_hermite": 3}
FLUID, WALL, MOVING = 0, 1, 2

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        dp = C.POINTER(C.c_double)
        ip = C.POINTER(C.c_int)
        L.lbmo_create.restype = C.c_void_p
        L.lbmo_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double]
        L.lbmo_destroy.argtypes = [C.c_void_p]
        L.lbmo_set_flags.argtypes = [C.c_void_p, C.POINTER(C.c_uint8), dp]
        L.lbmo_set_relaxation.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double]
        L.lbmo_set_trt_magic.argtypes = [C.c_void_p, C.c_double]
        L.lbmo_set_force.argtypes = [C.c_void_p, dp]
        L.lbmo_init_equilibrium.argtypes = [C.c_void_p, dp, dp]
        L.lbmo_step.argtypes = [C.c_void_p, C.c_int]
        L.lbmo_get_populations.argtypes = [C.c_void_p, dp]
        L.lbmo_set_populations.argtypes = [C.c_void_p, dp]
        L.lbmo_macroscopic.argtypes = [C.c_void_p, dp, dp]
        L.lbmo_kinetic_energy.argtypes = [C.c_void_p, dp]
        L.lbmo_steps.restype = C.c_long
        L.lbmo_steps.argtypes = [C.c_void_p]
        L.lbmo_num_threads.restype = C.c_int
        L.lbmo_lattice.argtypes = [C.c_int, ip, dp, ip, ip]
        L.lbmo_equilibrium.argtypes = [C.c_int, C.c_int, C.c_double, dp, dp]
        L.lbmo_collide.argtypes = [C.c_int, C.c_int, dp, dp, dp]
        L.lbmo_moments.argtypes = [C.c_int, C.c_int, dp, dp, dp]
        L.lbmo_cumulants.argtypes = [C.c_int, C.c_int, dp, dp]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return lib().lbmo_num_threads()


def lattice(Q):
    """(c[Q,3], t[Q], opp[Q], mom[Q,3]) of the oracle's own tables."""
    c = np.zeros((Q, 3), dtype=np.int32)
    mom = np.zeros((Q, 3), dtype=np.int32)
    t = np.zeros(Q)
    opp = np.zeros(Q, dtype=np.int32)
    ip = C.POINTER(C.c_int)
    rc = lib().lbmo_lattice(Q, c.ctypes.data_as(ip), _dp(t), opp.ctypes.data_as(ip), mom.ctypes.data_as(ip))
    assert rc == 0
    return c, t, opp, mom


def equilibrium(Q, kind, rho, u):
    """kind 'w2' (Eq 6) or 'ext' (extended / NW4)."""
    E = np.zeros(Q)
    uu = _f64(u)
    lib().lbmo_equilibrium(Q, 0 if kind == "w2" else 1, float(rho), _dp(uu), _dp(E))
    return E


def collide(Q, model, f, omega, omega_bulk=None, omega3=None, omega_hi=None, trt_magic=None):
    nan = float("nan")
    rates = _f64([omega] + [nan if v is None else v for v in (omega_bulk, omega3, omega_hi, trt_magic)])
    fin = _f64(f)
    out = np.zeros(Q)
    rc = lib().lbmo_collide(Q, MODELS[model], _dp(rates), _dp(fin), _dp(out))
    assert rc == 0
    return out


def moments(Q, basis, f, u=(0.0, 0.0, 0.0)):
    m = np.zeros(Q)
    uu, ff = _f64(u), _f64(f)
    lib().lbmo_moments(Q, BASES[basis], _dp(uu), _dp(ff), _dp(m))
    return m


def cumulants_from_moments(Q, kap):
    k = _f64(kap).copy()
    K = np.zeros(Q)
    lib().lbmo_cumulants(Q, 1, _dp(k), _dp(K))
    return K


def moments_from_cumulants(Q, K):
    kk = _f64(K).copy()
    m = np.zeros(Q)
    m[0] = 1.0
    lib().lbmo_cumulants(Q, -1, _dp(m), _dp(kk))
    return m


class Oracle:
    """One oracle simulation; mirrors the product's call names with an 'o'."""

    def __init__(self, nx, ny, nz, Q=19, model="BGK_W2", omega=1.0):
        self.nx, self.ny, self.nz, self.Q = nx, ny, nz, Q
        self.N = nx * ny * nz
        self._h = lib().lbmo_create(nx, ny, nz, Q, MODELS[model], float(omega))
        if not self._h:
            raise ValueError("lbmo_create failed")

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.lbmo_destroy(self._h)
            self._h = None

    def set_flags(self, flags, u_wall=(0.0, 0.0, 0.0)):
        fl = np.ascontiguousarray(flags, dtype=np.uint8).reshape(-1)
        assert fl.size == self.N
        uw = _f64(u_wall)
        lib().lbmo_set_flags(self._h, fl.ctypes.data_as(C.POINTER(C.c_uint8)), _dp(uw))

    def set_relaxation(self, omega_bulk, omega3, omega_hi):
        lib().lbmo_set_relaxation(self._h, omega_bulk, omega3, omega_hi)

    def set_trt_magic(self, lam):
        lib().lbmo_set_trt_magic(self._h, lam)

    def set_force(self, g):
        gg = _f64(g)
        lib().lbmo_set_force(self._h, _dp(gg))

    def init_equilibrium(self, rho, u):
        r = _f64(rho).reshape(-1)
        uu = _f64(u).reshape(-1)
        assert r.size == self.N and uu.size == 3 * self.N
        lib().lbmo_init_equilibrium(self._h, _dp(r), _dp(uu))

    def step(self, n=1):
        lib().lbmo_step(self._h, int(n))

    def get_populations(self):
        f = np.zeros((self.Q, self.N))
        lib().lbmo_get_populations(self._h, _dp(f))
        return f

    def set_populations(self, f):
        ff = _f64(f).reshape(-1)
        assert ff.size == self.Q * self.N
        lib().lbmo_set_populations(self._h, _dp(ff))

    def macroscopic(self):
        rho = np.zeros(self.N)
        u = np.zeros((3, self.N))
        lib().lbmo_macroscopic(self._h, _dp(rho), _dp(u))
        return rho, u

    def kinetic_energy(self):
        e = C.c_double(0.0)
        lib().lbmo_kinetic_energy(self._h, C.byref(e))
        return e.value

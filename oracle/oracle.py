"""ctypes driver for the CPU oracle (oracle/lbm_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  Nothing in paper_1311_2404_b200/ imports this module
and this module imports nothing from it.  It holds no arithmetic of the method: it only
compiles lbm_oracle.c with gcc, marshals numpy arrays, and forwards calls.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lbm_oracle.c")
_LIB = os.path.join(_HERE, "liblbm_oracle.so")

D2Q9, D3Q19 = 0, 1
FLUID, SOLID, WALL_FULLWAY, VELOCITY = 0, 1, 2, 3
FORCE_GUO, FORCE_EDM = 0, 1
BGK, MRT, SC2, REG, LES = 0, 1, 2, 3, 4
PSI_RHO, PSI_1MEXP = 0, 1
QMAX = 19


class _Params(C.Structure):
    _fields_ = [
        ("lattice", C.c_int32), ("model", C.c_int32),
        ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
        ("tau", C.c_double * 2),
        ("rates", C.c_double * QMAX),
        ("force", C.c_double * 3),
        ("sc_G", C.c_double),
        ("sc_psi", C.c_int32),
        ("bc_velocity", C.c_double * 3),
        ("force_scheme", C.c_int32),
        ("smagorinsky_cs", C.c_double),
    ]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP over nodes; results do not depend on the
    thread count because every site is written exactly once per pass)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-std=c99", "-O2", "-fopenmp", "-fPIC", "-shared",
                               "-ffp-contract=off", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.POINTER(_Params)]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_destroy.restype = None
        for name in ("orc_set_geometry", "orc_stream_map"):
            getattr(L, name).argtypes = [C.c_void_p, C.c_void_p]
        for name in ("orc_init_equilibrium", "orc_macro"):
            getattr(L, name).argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        for name in ("orc_set_distributions", "orc_get_distributions", "orc_sc_force"):
            getattr(L, name).argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.orc_step.argtypes = [C.c_void_p, C.c_int]
        L.orc_lattice_tables.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_feq.argtypes = [C.c_int, C.c_double, C.c_void_p, C.c_void_p]
        L.orc_mrt_matrix.argtypes = [C.c_int, C.c_void_p, C.c_void_p]
        _lib = L
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def lattice_tables(lattice: int):
    Q = lib().orc_lattice_Q(lattice)
    e = np.zeros((Q, 3), np.int32)
    w = np.zeros(Q, np.float64)
    opp = np.zeros(Q, np.int32)
    assert lib().orc_lattice_tables(lattice, e.ctypes.data, w.ctypes.data, opp.ctypes.data) == 0
    return e, w, opp


def feq(lattice: int, rho: float, v) -> np.ndarray:
    Q = lib().orc_lattice_Q(lattice)
    v3 = np.zeros(3)
    v3[: len(v)] = v
    out = np.zeros(Q)
    assert lib().orc_feq(lattice, float(rho), v3.ctypes.data, out.ctypes.data) == 0
    return out


def mrt_matrix(lattice: int):
    Q = lib().orc_lattice_Q(lattice)
    M = np.zeros((Q, Q))
    Minv = np.zeros((Q, Q))
    assert lib().orc_mrt_matrix(lattice, M.ctypes.data, Minv.ctypes.data) == 0
    return M, Minv


class Oracle:
    """One oracle simulation.  Arrays are C-order [z][y][x]; u is [D][z][y][x]; f is [Q][z][y][x]."""

    def __init__(self, lattice, model, nx, ny, nz=1, tau=(1.0, 1.0), rates=None,
                 force=(0.0, 0.0, 0.0), sc_G=0.0, sc_psi=PSI_RHO, bc_velocity=(0.0, 0.0, 0.0),
                 force_scheme=0, smagorinsky_cs=0.0):
        p = _Params()
        p.lattice, p.model = lattice, model
        p.nx, p.ny, p.nz = nx, ny, nz
        tau = (tau, tau) if np.isscalar(tau) else tuple(tau)
        p.tau[0], p.tau[1] = float(tau[0]), float(tau[1] if len(tau) > 1 else tau[0])
        if rates is not None:
            for k, r in enumerate(rates):
                p.rates[k] = float(r)
        for a in range(3):
            p.force[a] = float(force[a]) if a < len(force) else 0.0
        p.sc_G, p.sc_psi = float(sc_G), int(sc_psi)
        p.force_scheme = int(force_scheme)
        p.smagorinsky_cs = float(smagorinsky_cs)
        for a in range(3):
            p.bc_velocity[a] = float(bc_velocity[a]) if a < len(bc_velocity) else 0.0
        self._h = lib().orc_create(C.byref(p))
        if not self._h:
            raise ValueError("orc_create rejected the parameters")
        self.Q = lib().orc_lattice_Q(lattice)
        self.D = lib().orc_lattice_D(lattice)
        self.shape = (nz, ny, nx)
        self.N = nx * ny * nz
        self.ncomp = 2 if model == SC2 else 1

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_destroy(self._h)
            self._h = None

    def set_geometry(self, mask):
        m = np.ascontiguousarray(mask, dtype=np.uint8)
        assert m.size == self.N
        lib().orc_set_geometry(self._h, m.ctypes.data)

    def init_equilibrium(self, rho, u, comp=0):
        rho, u = _f64(rho), _f64(u)
        assert rho.size == self.N and u.size == self.D * self.N
        assert lib().orc_init_equilibrium(self._h, comp, rho.ctypes.data, u.ctypes.data) == 0

    def step(self, n=1):
        assert lib().orc_step(self._h, int(n)) == 0

    def macro(self, comp=0):
        rho = np.zeros(self.shape)
        u = np.zeros((self.D,) + self.shape)
        assert lib().orc_macro(self._h, comp, rho.ctypes.data, u.ctypes.data) == 0
        return rho, u

    def get_distributions(self, comp=0):
        f = np.zeros((self.Q,) + self.shape)
        assert lib().orc_get_distributions(self._h, comp, f.ctypes.data) == 0
        return f

    def set_distributions(self, f, comp=0):
        f = _f64(f)
        assert f.size == self.Q * self.N
        assert lib().orc_set_distributions(self._h, comp, f.ctypes.data) == 0

    def stream_map(self):
        m = np.zeros((self.Q, self.N), np.int64)
        assert lib().orc_stream_map(self._h, m.ctypes.data) == 0
        return m

    def sc_force(self, comp):
        F = np.zeros((3,) + self.shape)
        assert lib().orc_sc_force(self._h, comp, F.ctypes.data) == 0
        return F

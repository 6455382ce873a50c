"""ctypes front end of the CPU oracle (oracle/pd_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It imports nothing from
paper_2309_11273_b200 and the CUDA path imports nothing from here.

The class below only marshals numpy arrays into the C functions and keeps the state
(u, v, rho) between calls; every number is produced by pd_oracle.c, which follows
PAPER.md step by step (see the citations there).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pd_oracle.c")
_LIB = os.path.join(_HERE, "libpd_oracle.so")

MODE_3D, MODE_PLANE_STRESS, MODE_PLANE_STRAIN = 0, 1, 2
FLAG_BODYF, FLAG_NOFAIL = 1 << 6, 1 << 7


def build(force: bool = False) -> str:
    """Compile pd_oracle.c with gcc (-ffp-contract=off so the horizon test is reproducible)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
               _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.pdo_family_count_brute.restype = C.c_int64
        _lib.pdo_family_cells.restype = C.c_int64
        _lib.pdo_find_bond.restype = C.c_int64
        _lib.pdo_break.restype = C.c_int64
        _lib.pdo_run.restype = C.c_int64
        _lib.pdo_run_geom.restype = C.c_int64
        _lib.pdo_break_geom.restype = C.c_int64
        _lib.pdo_num_threads.restype = C.c_int
    return _lib


def num_threads() -> int:
    return int(lib().pdo_num_threads())


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f64(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None:
        a = a.reshape(shape)
    return a


def constants(mode: int, E: float, nu: float):
    """(A, K, G, kappa, mu) per Eqs. 1.8, 1.15, 1.16."""
    out = [C.c_double() for _ in range(5)]
    rc = lib().pdo_constants(C.c_int(mode), C.c_double(E), C.c_double(nu), *[C.byref(o) for o in out])
    if rc != 0:
        raise ValueError("inadmissible material / mode")
    return tuple(o.value for o in out)


def family(coords: np.ndarray, horizon: float, method: str = "cells"):
    """CSR (rowptr int64[n+1], col int32[Z]) of the directed bonds, rows ascending in j."""
    coords = _f64(coords)
    n, dim = coords.shape
    rowptr = np.zeros(n + 1, dtype=np.int64)
    L = lib()
    if method == "brute":
        Z = L.pdo_family_count_brute(C.c_int64(n), C.c_int(dim), _p(coords), C.c_double(horizon), _p(rowptr))
        col = np.empty(Z, dtype=np.int32)
        L.pdo_family_fill_brute(C.c_int64(n), C.c_int(dim), _p(coords), C.c_double(horizon), _p(rowptr), _p(col))
    else:
        Z = L.pdo_family_cells(C.c_int64(n), C.c_int(dim), _p(coords), C.c_double(horizon), _p(rowptr), None)
        if Z < 0:
            raise MemoryError
        col = np.empty(Z, dtype=np.int32)
        L.pdo_family_cells(C.c_int64(n), C.c_int(dim), _p(coords), C.c_double(horizon), _p(rowptr), _p(col))
    return rowptr, col


class PDOracle:
    """State holder around the C oracle.  Arguments mirror the library boundary (include/pd.h)
    but are plain numpy arrays in user node order."""

    def __init__(self, coords, volumes, horizon, *, dim, mode, E, nu, rho, dt, s_c=0.0,
                 ramp_time=0.0, flags=None, value=None, precut=None, u0=None, v0=None,
                 family_method="cells", extension="linearized"):
        assert extension in ("linearized", "geometric")   # geometric: App. C's e = ||xi+eta|| - ||xi||
        self.geom = extension == "geometric"
        self.coords = _f64(coords).reshape(-1, dim)
        self.n, self.dim = self.coords.shape
        self.V = _f64(volumes).reshape(self.n)
        self.horizon = float(horizon)
        self.mode, self.E, self.nu, self.rho_mass = int(mode), float(E), float(nu), float(rho)
        self.dt, self.s_c, self.ramp_time = float(dt), float(s_c), float(ramp_time)
        if (dim == 3) != (mode == MODE_3D):
            raise ValueError("dim/mode mismatch")
        self.A, self.K, self.G, self.kappa, self.mu = constants(mode, E, nu)
        self.flags = (np.zeros(self.n, np.uint8) if flags is None
                      else np.ascontiguousarray(flags, dtype=np.uint8).reshape(self.n))
        self.value = (np.zeros((self.n, dim)) if value is None else _f64(value, (self.n, dim)))
        self.rowptr, self.col = family(self.coords, self.horizon, family_method)
        self.Z = int(self.rowptr[-1])
        self.m = np.empty(self.n)
        self.fvol = np.empty(self.n)
        lib().pdo_weighted_volume(C.c_int64(self.n), C.c_int(dim), _p(self.coords), _p(self.V),
                                  _p(self.rowptr), _p(self.col), _p(self.m), _p(self.fvol))
        if np.any(self.m <= 0.0):
            raise ValueError("isolated node (m_i = 0)")
        self.rho = np.ones(self.Z, dtype=np.uint8)
        if precut is not None and len(precut):
            pc = np.asarray(precut, dtype=np.int64).reshape(-1, 2)
            for a, b in pc:
                for i, j in ((a, b), (b, a)):
                    p = lib().pdo_find_bond(_p(self.rowptr), _p(self.col), C.c_int64(i), C.c_int64(j))
                    if p < 0:
                        raise ValueError(f"precut pair ({a},{b}) is not a bond")
                    self.rho[p] = 0
        self.u = np.zeros((self.n, dim)) if u0 is None else _f64(u0, (self.n, dim)).copy()
        self.v = np.zeros((self.n, dim)) if v0 is None else _f64(v0, (self.n, dim)).copy()
        for k in range(dim):  # reading C-3: clamped dofs sit at 0 with v = 0
            cl = (self.flags & (1 << k)) != 0
            self.u[cl, k] = 0.0
            self.v[cl, k] = 0.0
        self.step_index = 0
        self.phi = np.empty(self.n)
        self.e = np.empty(self.Z)
        self.xbar = np.empty(self.Z)
        self.theta = np.empty(self.n)
        self.f = np.empty((self.n, dim))
        self.near_total = 0
        self.break_log = []
        self.damage()

    # ---- pieces (used by the pins) ------------------------------------------------------
    def extension(self, u=None):
        u = self.u if u is None else _f64(u, (self.n, self.dim))
        fn = lib().pdo_extension_geom if self.geom else lib().pdo_extension
        fn(C.c_int64(self.n), C.c_int(self.dim), _p(self.coords), _p(self.rowptr),
                            _p(self.col), _p(self.rho), _p(u), _p(self.e), _p(self.xbar))
        return self.e

    def dilatation(self, u=None):
        self.extension(u)
        lib().pdo_dilatation(C.c_int64(self.n), _p(self.V), _p(self.rowptr), _p(self.col), _p(self.e),
                             _p(self.xbar), C.c_double(self.A), _p(self.m), _p(self.theta))
        return self.theta

    def force_density(self, u=None):
        self.dilatation(u)
        lib().pdo_force_density(C.c_int64(self.n), C.c_int(self.dim), _p(self.coords), _p(self.V),
                                _p(self.rowptr), _p(self.col), _p(self.rho), _p(self.e), _p(self.xbar),
                                _p(self.theta), _p(self.m), C.c_double(self.K), C.c_double(self.G),
                                _p(self.f))
        return self.f

    def energy_density(self, u=None):
        self.dilatation(u)
        W = np.empty(self.n)
        lib().pdo_energy_density(C.c_int64(self.n), _p(self.V), _p(self.rowptr), _p(self.col), _p(self.e),
                                 _p(self.theta), _p(self.m), C.c_double(self.A), C.c_double(self.K),
                                 C.c_double(self.G), _p(W))
        return W

    def break_bonds(self, near_tol=1e-9):
        near = C.c_int64(0)
        fn = lib().pdo_break_geom if self.geom else lib().pdo_break
        nb = fn(C.c_int64(self.n), C.c_int(self.dim), _p(self.coords), _p(self.rowptr),
                             _p(self.col), _p(self.flags), _p(self.u), C.c_double(self.s_c),
                             _p(self.rho), C.c_double(near_tol), C.byref(near))
        return int(nb), int(near.value)

    def damage(self):
        lib().pdo_damage(C.c_int64(self.n), _p(self.V), _p(self.rowptr), _p(self.col), _p(self.rho),
                         _p(self.fvol), _p(self.phi))
        return self.phi

    # ---- the time step ------------------------------------------------------------------
    def step(self, nsteps: int, log_breaks: bool = False, near_tol: float = 1e-9) -> int:
        if self.geom:
            near = C.c_int64(0)
            nb = lib().pdo_run_geom(
                C.c_int64(self.n), C.c_int(self.dim), _p(self.coords), _p(self.V), _p(self.rowptr),
                _p(self.col), _p(self.rho), _p(self.m), _p(self.fvol), _p(self.flags), _p(self.value),
                C.c_double(self.A), C.c_double(self.K), C.c_double(self.G), C.c_double(self.rho_mass),
                C.c_double(self.dt), C.c_double(self.ramp_time), C.c_double(self.s_c),
                C.c_int64(self.step_index), C.c_int64(nsteps), _p(self.u), _p(self.v), _p(self.phi),
                _p(self.e), _p(self.xbar), _p(self.theta), _p(self.f), C.c_double(near_tol), C.byref(near))
            self.step_index += nsteps
            self.near_total += int(near.value)
            return int(nb)
        near = C.c_int64(0)
        logn = C.c_int64(0)
        cap = 0
        log = None
        if log_breaks:
            cap = max(1024, self.Z)
            log = np.empty((cap, 3), dtype=np.int64)
        nb = lib().pdo_run(
            C.c_int64(self.n), C.c_int(self.dim), _p(self.coords), _p(self.V), _p(self.rowptr),
            _p(self.col), _p(self.rho), _p(self.m), _p(self.fvol), _p(self.flags), _p(self.value),
            C.c_double(self.A), C.c_double(self.K), C.c_double(self.G), C.c_double(self.rho_mass),
            C.c_double(self.dt), C.c_double(self.ramp_time), C.c_double(self.s_c),
            C.c_int64(self.step_index), C.c_int64(nsteps), _p(self.u), _p(self.v), _p(self.phi),
            _p(self.e), _p(self.xbar), _p(self.theta), _p(self.f), C.c_double(near_tol),
            C.byref(near), _p(log), C.c_int64(cap), C.byref(logn))
        self.step_index += nsteps
        self.near_total += int(near.value)
        if log_breaks:
            self.break_log.extend(map(tuple, log[: min(cap, logn.value)].tolist()))
        return int(nb)

    # ---- views --------------------------------------------------------------------------
    def bond_pairs(self, intact=None):
        """(i, j) user-index pairs of the directed bonds, optionally filtered by status."""
        i = np.repeat(np.arange(self.n, dtype=np.int64), np.diff(self.rowptr))
        j = self.col.astype(np.int64)
        if intact is None:
            return i, j
        sel = self.rho == (1 if intact else 0)
        return i[sel], j[sel]

    def broken_set(self):
        i, j = self.bond_pairs(intact=False)
        return set(zip(i.tolist(), j.tolist()))

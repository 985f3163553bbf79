"""ctypes driver of oracle/pic_oracle.c — TEST INFRASTRUCTURE (see oracle/__init__.py).

Marshalling only: every number is computed by the C file.  ``build()`` compiles it with
``gcc -O2 -ffp-contract=off`` (no fast-math, no FMA contraction: the arithmetic is the
plain definition of SURVEY.md §8(c)).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pic_oracle.c")
_SO = os.path.join(_HERE, "libpic_oracle.so")
_lib = None


class OracleParams(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("scx", C.c_int32), ("scy", C.c_int32), ("scz", C.c_int32),
                ("order", C.c_int32), ("gather", C.c_int32),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double), ("dt", C.c_double)]

    @staticmethod
    def make(grid, cell=(1.0, 1.0, 1.0), dt=0.5, supercell=(8, 8, 4), order=1, gather=0) -> "OracleParams":
        """gather: 0 momentum-conserving (the contract's path, S3), 1 energy-conserving / Galerkin."""
        return OracleParams(int(grid[0]), int(grid[1]), int(grid[2]),
                            int(supercell[0]), int(supercell[1]), int(supercell[2]),
                            int(order), int(gather), float(cell[0]), float(cell[1]), float(cell[2]), float(dt))


def build(force: bool = False) -> str:
    """Compile the oracle shared library next to its source (idempotent)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-std=c99",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _SO)
    return _SO


_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_shape.restype = C.c_double
        L.orc_shape.argtypes = [C.c_int, C.c_double]
        L.orc_gather.restype = None
        L.orc_gather.argtypes = [C.POINTER(OracleParams), C.POINTER(_dp), _dp, _dp]
        L.orc_boris.restype = None
        L.orc_boris.argtypes = [_dp, _dp, _dp, C.c_double, C.c_double, _dp]
        L.orc_move.restype = None
        L.orc_move.argtypes = [C.POINTER(OracleParams), _dp, _dp, _dp]
        L.orc_deposit.restype = None
        L.orc_deposit.argtypes = [C.POINTER(OracleParams), C.c_double, _dp, _dp, _dp, _dp, _dp]
        L.orc_rho.restype = None
        L.orc_rho.argtypes = [C.POINTER(OracleParams), C.c_long, _dp, _dp, _dp, _dp, _dp]
        L.orc_wrap_and_bucket.restype = C.c_int32
        L.orc_wrap_and_bucket.argtypes = [C.POINTER(OracleParams), _dp]
        L.orc_step.restype = C.c_int
        L.orc_step.argtypes = [C.POINTER(OracleParams), C.c_long] + [_dp] * 6 + [_dp, _ip, _dp, _dp] + [_dp] * 6 + [_dp] * 3 + [_ip]
        _lib = L
    return _lib


def _d(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a: np.ndarray):
    return a.ctypes.data_as(_dp)


def shape(order: int, d: float) -> float:
    return float(lib().orc_shape(int(order), float(d)))


def gather(prm: OracleParams, fields: Sequence[np.ndarray], X: Sequence[float]) -> np.ndarray:
    """fields: six float64 arrays [nz,ny,nx]; X in cell units. Returns (Ex,Ey,Ez,Bx,By,Bz)."""
    fs = [_d(f) for f in fields]
    arr = (_dp * 6)(*[_p(f) for f in fs])
    Xa = _d(X)
    out = np.zeros(6)
    lib().orc_gather(C.byref(prm), arr, _p(Xa), _p(out))
    return out


def boris(u, E, B, q_over_m: float, dt: float) -> np.ndarray:
    ua, Ea, Ba = _d(u), _d(E), _d(B)
    out = np.zeros(3)
    lib().orc_boris(_p(ua), _p(Ea), _p(Ba), float(q_over_m), float(dt), _p(out))
    return out


def move(prm: OracleParams, X, u) -> np.ndarray:
    Xa, ua = _d(X), _d(u)
    out = np.zeros(3)
    lib().orc_move(C.byref(prm), _p(Xa), _p(ua), _p(out))
    return out


def deposit(prm: OracleParams, qw: float, X0, X1, J: Optional[Tuple[np.ndarray, ...]] = None):
    """Adds one particle's Esirkepov current into J=(Jx,Jy,Jz) float64 [nz,ny,nx]; X in cell units."""
    if J is None:
        J = tuple(np.zeros((prm.nz, prm.ny, prm.nx)) for _ in range(3))
    a0, a1 = _d(X0), _d(X1)
    lib().orc_deposit(C.byref(prm), float(qw), _p(a0), _p(a1), _p(J[0]), _p(J[1]), _p(J[2]))
    return J


def rho(prm: OracleParams, X, Y, Z, qw) -> np.ndarray:
    """Node charge density of particles at cell-unit positions X,Y,Z with charge*weight qw."""
    Xa, Ya, Za, qa = _d(X), _d(Y), _d(Z), _d(qw)
    out = np.zeros((prm.nz, prm.ny, prm.nx))
    lib().orc_rho(C.byref(prm), Xa.size, _p(Xa), _p(Ya), _p(Za), _p(qa), _p(out))
    return out


def wrap_and_bucket(prm: OracleParams, X) -> Tuple[np.ndarray, int]:
    Xa = _d(X).copy()
    sc = lib().orc_wrap_and_bucket(C.byref(prm), _p(Xa))
    return Xa, int(sc)


def step(prm: OracleParams, x, y, z, ux, uy, uz, w, species, q, m, fields, J, supercell=None) -> int:
    """One step in place over float64 arrays (physical positions). J is accumulated (caller zeroes)."""
    n = x.size
    sp = species.ctypes.data_as(_ip) if species is not None else None
    sc = supercell.ctypes.data_as(_ip) if supercell is not None else None
    return int(lib().orc_step(C.byref(prm), n, _p(x), _p(y), _p(z), _p(ux), _p(uy), _p(uz), _p(w), sp,
                              _p(q), _p(m), *[_p(f) for f in fields], _p(J[0]), _p(J[1]), _p(J[2]), sc))


class Oracle:
    """Stateful convenience wrapper mirroring the product's call sequence
    (create / set_species / load_particles / set_fields / step / get_*)."""

    def __init__(self, grid, cell=(1.0, 1.0, 1.0), dt=0.5, supercell=(8, 8, 4), order=1, gather=0):
        self.prm = OracleParams.make(grid, cell, dt, supercell, order, gather)
        self.q = np.full(256, -1.0)
        self.m = np.full(256, 1.0)
        self._parts = [np.zeros(0) for _ in range(7)]
        self.species = np.zeros(0, dtype=np.int32)
        self.fields = None
        shp = (self.prm.nz, self.prm.ny, self.prm.nx)
        self.J = tuple(np.zeros(shp) for _ in range(3))
        self.supercell = np.zeros(0, dtype=np.int32)

    def set_species(self, q, m):
        self.q[:len(q)] = q
        self.m[:len(m)] = m

    def load_particles(self, x, y, z, ux, uy, uz, w, species=None):
        new = [_d(a) for a in (x, y, z, ux, uy, uz, w)]
        self._parts = [np.concatenate([a, b]) for a, b in zip(self._parts, new)]
        sp = np.zeros(new[0].size, dtype=np.int32) if species is None else np.ascontiguousarray(species, dtype=np.int32)
        self.species = np.concatenate([self.species, sp])
        self.supercell = np.zeros(self.n, dtype=np.int32)

    @property
    def n(self) -> int:
        return int(self._parts[0].size)

    def set_fields(self, fields6):
        """fields6: array-like [6,nz,ny,nx] (Ex,Ey,Ez,Bx,By,Bz)."""
        self.fields = [_d(f) for f in fields6]

    def step(self, n_steps: int = 1, update_fields: bool = False) -> int:
        """update_fields: after every particle step advance E, B with that step's J
        (oracle/yee_oracle.py) — the self-consistent PIC loop."""
        rc = 0
        x, y, z, ux, uy, uz, w = self._parts
        for _ in range(n_steps):
            for j in self.J:
                j.fill(0.0)                       # S16: J is the last step's current
            rc |= step(self.prm, x, y, z, ux, uy, uz, w, self.species, self.q, self.m,
                       self.fields, self.J, self.supercell)
            if update_fields:
                self.update_fields()
        return rc

    def update_fields(self):
        """One Yee update of the fields with the last step's J."""
        from . import yee_oracle
        p = self.prm
        self.fields = [np.ascontiguousarray(f) for f in
                       yee_oracle.yee_update(self.fields, self.J, p.dt, (p.dx, p.dy, p.dz))]

    def particles(self):
        x, y, z, ux, uy, uz, w = self._parts
        return dict(x=x, y=y, z=z, ux=ux, uy=uy, uz=uz, w=w, species=self.species, supercell=self.supercell)

    def counts(self) -> np.ndarray:
        p = self.prm
        nsc = (p.nx // p.scx) * (p.ny // p.scy) * (p.nz // p.scz)
        return np.bincount(self.supercell, minlength=nsc).astype(np.int32)

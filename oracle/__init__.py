"""oracle -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

ctypes front end of ``oracle/mhd_oracle.cpp``: the plain CPU restatement of the paper's relaxing-TVD
MHD update (section 3, lines 47-172; sequencing from section 4.2-4.3).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It imports nothing from ``paper_0908_4362_b200`` and the CUDA path
imports nothing from here.

All functions work on a list of eight C-contiguous numpy arrays of shape (nz, ny, nx) (x fastest),
dtype float32 or float64, in the order rho, m_x, m_y, m_z, E, Bx, By, Bz, and update them IN PLACE.
Axes are numbered 0 = x, 1 = y, 2 = z.  ``bc``: 0 periodic, 1 outflow.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mhd_oracle.cpp")
_LIB = os.path.join(_HERE, "libmhd_oracle.so")

PERIODIC, OUTFLOW = 0, 1
FIELD_NAMES = ("rho", "mx", "my", "mz", "E", "Bx", "By", "Bz")


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (no fast-math, no FMA contraction) if it is missing or stale."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        P8 = ctypes.POINTER(ctypes.c_void_p)
        head = [ctypes.c_int] * 4 + [ctypes.c_double, ctypes.c_int, P8]
        lib.mhdo_cmax.argtypes = head + [ctypes.POINTER(ctypes.c_double)]
        lib.mhdo_fluid.argtypes = head + [ctypes.c_int, ctypes.c_double]
        lib.mhdo_badvect.argtypes = head + [ctypes.c_int, ctypes.c_int, ctypes.c_double]
        lib.mhdo_sweep.argtypes = head + [ctypes.c_int, ctypes.c_int, ctypes.c_double]
        lib.mhdo_step_fixed.argtypes = head + [ctypes.c_longlong, ctypes.c_double]
        lib.mhdo_run.argtypes = head + [ctypes.c_longlong, ctypes.c_int, ctypes.c_double,
                                        ctypes.POINTER(ctypes.c_double)]
        lib.mhdo_set_num_threads.argtypes = [ctypes.c_int]
        for name in ("mhdo_cmax", "mhdo_fluid", "mhdo_badvect", "mhdo_sweep", "mhdo_step_fixed", "mhdo_run",
                     "mhdo_num_threads"):
            getattr(lib, name).restype = ctypes.c_int
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().mhdo_num_threads())


def set_num_threads(n: int) -> None:
    _load().mhdo_set_num_threads(int(n))


def _head(fields, gamma, bc):
    if len(fields) != 8:
        raise ValueError("need 8 fields")
    f0 = fields[0]
    if f0.ndim != 3:
        raise ValueError("fields must have shape (nz, ny, nx)")
    for f in fields:
        if f.dtype != f0.dtype or f.shape != f0.shape or not f.flags.c_contiguous or not f.flags.writeable:
            raise ValueError("fields must be C-contiguous writable arrays of one dtype and shape")
    if len({f.ctypes.data for f in fields}) != 8:
        raise ValueError("fields must not alias one another (they are updated in place)")
    if f0.dtype == np.float32:
        prec = 0
    elif f0.dtype == np.float64:
        prec = 1
    else:
        raise ValueError("dtype must be float32 or float64")
    nz, ny, nx = f0.shape
    ptrs = (ctypes.c_void_p * 8)(*[f.ctypes.data for f in fields])
    return [prec, nx, ny, nz, float(gamma), int(bc), ptrs]


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")


def cmax(fields, gamma, bc) -> float:
    """c_max of eq (18)."""
    out = ctypes.c_double()
    _check(_load().mhdo_cmax(*_head(fields, gamma, bc), ctypes.byref(out)), "cmax")
    return out.value


def fluid(fields, gamma, bc, d, dt) -> None:
    """fluid_d, Algorithm 1."""
    _check(_load().mhdo_fluid(*_head(fields, gamma, bc), int(d), float(dt)), "fluid")


def badvect(fields, gamma, bc, d, t, dt) -> None:
    """B_{t->d}: advect B_t along d and constrain B_d, Algorithm 2."""
    _check(_load().mhdo_badvect(*_head(fields, gamma, bc), int(d), int(t), float(dt)), "badvect")


def sweep(fields, gamma, bc, d, reverse, dt) -> None:
    """L_d forward or reverse."""
    _check(_load().mhdo_sweep(*_head(fields, gamma, bc), int(d), int(bool(reverse)), float(dt)), "sweep")


def step_fixed(fields, gamma, bc, s, dt) -> None:
    """One double sweep (eqs (23)-(25)) with step index s and the given dt."""
    _check(_load().mhdo_step_fixed(*_head(fields, gamma, bc), int(s), float(dt)), "step_fixed")


def run(fields, gamma, bc, s0, nsteps, cfl) -> float:
    """nsteps times {c_max, dt = cfl/c_max, double sweep}; returns the advanced time (grid units)."""
    t = ctypes.c_double()
    _check(_load().mhdo_run(*_head(fields, gamma, bc), int(s0), int(nsteps), float(cfl), ctypes.byref(t)), "run")
    return t.value

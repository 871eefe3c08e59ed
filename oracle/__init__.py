"""CPU oracle for the moments-only lattice Boltzmann step (arxiv 2301.01622).

TEST INFRASTRUCTURE ONLY.  Thin ctypes loader around ``lbwp_oracle.c`` (plain C,
fp64).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package; the
product (``paper_2301_01622_b200``) never does, and this package never imports
the product.  All arithmetic lives in the C file, each function citing the
PAPER.md passage it restates.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lbwp_oracle.c")
_SO = os.path.join(_HERE, "liblbwp_oracle.so")
_lib = None

CFLAGS = ["-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp"]  # no fast-math


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (idempotent). Returns the .so path."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", *CFLAGS, "-o", _SO, _SRC, "-lm"])
    return _SO


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        lib.lbwp_oracle_lattice.argtypes = [ctypes.c_int, ip, dp]
        lib.lbwp_oracle_reconstruct.argtypes = [ctypes.c_int, dp, ctypes.c_double, dp]
        lib.lbwp_oracle_project.argtypes = [ctypes.c_int, dp, dp]
        run_args = [ctypes.c_int] * 5 + [ctypes.c_double] * 3 + [dp, ctypes.c_int64]
        lib.lbwp_oracle_run.argtypes = run_args
        lib.lbwp_oracle_pop_run.argtypes = run_args
        lib.lbwp_oracle_threads.restype = ctypes.c_int
        lib.lbwp_oracle_reconstruct_forced.argtypes = [ctypes.c_int, dp, ctypes.c_double, dp, dp]
        lib.lbwp_oracle_run_nc.argtypes = [ctypes.c_int] * 4 + [ctypes.c_double] * 5 + [dp, ctypes.c_int64, dp]
        lib.lbwp_oracle_diagnostics.argtypes = [ctypes.c_int] * 4 + [dp, ctypes.c_double, ctypes.c_int, ip, dp, dp]
        lib.lbwp_oracle_set_threads.argtypes, lib.lbwp_oracle_set_threads.restype = [ctypes.c_int], ctypes.c_int
        lib.lbwp_oracle_set_g2cut.argtypes = [ctypes.c_double]
        lib.lbwp_oracle_get_g2cut.restype = ctypes.c_double
        _lib = lib
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def threads() -> int:
    """OpenMP threads the step loops will use (results do not depend on it)."""
    return int(_load().lbwp_oracle_threads())


def set_threads(n: int) -> int:
    """Use n OpenMP threads from now on (the single-thread / all-core timings of bench.py); returns what is set."""
    return int(_load().lbwp_oracle_set_threads(int(n)))


def set_g2cut(v: float) -> float:
    """Reading C8 threshold on |G|^2 (default 1e-10); returns the previous value.  For the pin that
    brackets the dependence on it only: every parity run uses the default."""
    old = float(_load().lbwp_oracle_get_g2cut())
    _load().lbwp_oracle_set_g2cut(float(v))
    return old


def lattice(q: int):
    """(c[Q,3] int, w[Q] float64) in the oracle's direction order."""
    c = np.zeros((27, 3), dtype=np.int32)
    w = np.zeros(27, dtype=np.float64)
    n = _load().lbwp_oracle_lattice(q, c.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), _dp(w))
    if n < 0:
        raise ValueError("lattice must be 19 or 27")
    return c[:n].copy(), w[:n].copy()


def reconstruct(q: int, H10, omega: float = 0.0) -> np.ndarray:
    """Eq. 8 populations of one node (omega=0: Eq. 4)."""
    H = np.ascontiguousarray(H10, dtype=np.float64)
    out = np.zeros(27, dtype=np.float64)
    n = _load().lbwp_oracle_reconstruct(q, _dp(H), float(omega), _dp(out))
    if n < 0:
        raise ValueError("lattice must be 19 or 27")
    return out[:n].copy()


def project(q: int, f) -> np.ndarray:
    """Eq. 1-3 moments (rho, u, P) of one node's populations."""
    f = np.ascontiguousarray(f, dtype=np.float64)
    out = np.zeros(10, dtype=np.float64)
    if _load().lbwp_oracle_project(q, _dp(f), _dp(out)) < 0:
        raise ValueError("lattice must be 19 or 27")
    return out


def _run(fn, moments, q, ncomp, tau, nsteps, A, beta):
    m = np.array(moments, dtype=np.float64, order="C", copy=True)  # fp32 inputs widen exactly
    M = 10 if ncomp == 1 else 11
    if m.ndim != 4 or m.shape[0] != M:
        raise ValueError(f"moments must have shape [{M}, nz, ny, nx]")
    _, nz, ny, nx = m.shape
    rc = fn(q, ncomp, nx, ny, nz, float(tau), float(A), float(beta), _dp(m), int(nsteps))
    if rc != 0:
        raise RuntimeError(f"oracle returned {rc}")
    return m


def run(moments, *, lattice: int, ncomp: int = 1, tau: float, nsteps: int, A: float = 0.0,
        beta: float = 0.0) -> np.ndarray:
    """Advance moments [M,nz,ny,nx] by nsteps of the moments-only scheme; returns fp64."""
    return _run(_load().lbwp_oracle_run, moments, lattice, ncomp, tau, nsteps, A, beta)


def pop_run(moments, *, lattice: int, ncomp: int = 1, tau: float, nsteps: int, A: float = 0.0,
            beta: float = 0.0) -> np.ndarray:
    """Same interface, population-storing BGK (the comparison kernel's mini-oracle)."""
    return _run(_load().lbwp_oracle_pop_run, moments, lattice, ncomp, tau, nsteps, A, beta)


def diagnostics(moments, *, ncomp: int = 1, threshold: float = 0.5, probes=()) -> dict:
    """The paper's diagnostics of a state [M,nz,ny,nx]; probes = [(x, y, z), ...]."""
    m = np.ascontiguousarray(moments, dtype=np.float64)
    _, nz, ny, nx = m.shape
    n = len(probes)
    xyz = np.ascontiguousarray(np.array(probes, dtype=np.int32).reshape(max(n, 0), 3) if n else np.zeros((1, 3), np.int32))
    out, rho = np.zeros(8), np.zeros(max(n, 1))
    rc = _load().lbwp_oracle_diagnostics(ncomp, nx, ny, nz, _dp(m), float(threshold), n,
                                          xyz.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), _dp(out), _dp(rho))
    if rc != 0:
        raise ValueError("bad arguments (probe outside the box?)")
    return {"mass": [out[0], out[1]], "momentum": [out[2], out[3], out[4]], "rho_mean_above": out[5],
            "count_above": int(out[6]), "rho_max": out[7], "probe_rho": [float(v) for v in rho[:n]]}


def run_nc(moments, *, lattice: int, tau: float, nsteps: int, A: float, beta: float, A_h: float, h_c: float = 4.0,
           return_force: bool = False):
    """Two-component run with the near-contact repulsion of PAPER.md Eq. 10 (readings C20-C24); with return_force
    also the force field [3,nz,ny,nx] of the last step."""
    m = np.array(moments, dtype=np.float64, order="C", copy=True)
    if m.ndim != 4 or m.shape[0] != 11:
        raise ValueError("moments must have shape [11, nz, ny, nx]")
    _, nz, ny, nx = m.shape
    f = np.zeros((3, nz, ny, nx))
    rc = _load().lbwp_oracle_run_nc(lattice, nx, ny, nz, float(tau), float(A), float(beta), float(A_h), float(h_c),
                                    _dp(m), int(nsteps), _dp(f))
    if rc != 0:
        raise RuntimeError(f"oracle returned {rc}")
    return (m, f) if return_force else m


def reconstruct_forced(q: int, H10, omega: float, F3) -> np.ndarray:
    """Eq. 8 populations of one node under a body force F (reading C24)."""
    H = np.ascontiguousarray(H10, dtype=np.float64)
    F = np.ascontiguousarray(F3, dtype=np.float64)
    out = np.zeros(27, dtype=np.float64)
    n = _load().lbwp_oracle_reconstruct_forced(q, _dp(H), float(omega), _dp(F), _dp(out))
    if n < 0:
        raise ValueError("lattice must be 19 or 27")
    return out[:n].copy()

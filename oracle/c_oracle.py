"""ctypes loader for the plain-C oracle (oracle/pn_oracle.c).  Test infrastructure, not the product:
only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
`build()` compiles it with gcc; nothing here touches the CUDA path."""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "pn_oracle.c")
LIB = os.path.join(HERE, "libpn_oracle.so")


class _Info(ctypes.Structure):
    _fields_ = [("n_solved", ctypes.c_longlong), ("n_inlet_only", ctypes.c_longlong),
                ("n_outlet_only", ctypes.c_longlong), ("n_floating", ctypes.c_longlong),
                ("nnz", ctypes.c_longlong),
                ("iterations", ctypes.c_int), ("restarts", ctypes.c_int), ("status", ctypes.c_int),
                ("threads", ctypes.c_int),
                ("rel_residual", ctypes.c_double), ("q_in", ctypes.c_double),
                ("q_out", ctypes.c_double), ("g_eff", ctypes.c_double), ("k_eff", ctypes.c_double),
                ("t_label", ctypes.c_double), ("t_assemble", ctypes.c_double),
                ("t_pcg", ctypes.c_double), ("it_decade", ctypes.c_int * 16)]


@dataclass
class COracleResult:
    P: np.ndarray
    classes: np.ndarray
    q_in: float
    q_out: float
    g_eff: float
    k_eff: float
    iterations: int
    restarts: int
    rel_residual: float
    n_solved: int
    n_inlet_only: int
    n_outlet_only: int
    n_floating: int
    status: str
    threads: int
    t_label: float
    t_assemble: float
    t_pcg: float
    nnz: int
    it_decade: tuple = ()      # first iteration with recursive ||r||/||b|| <= 1e-k, k = 0..15 (-1: never)


def build(force: bool = False) -> str:
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < os.path.getmtime(SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", LIB, SRC, "-lm"])
    return LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        fp = ctypes.POINTER(ctypes.c_float)
        dp = ctypes.POINTER(ctypes.c_double)
        _lib.pno_solve.argtypes = [ctypes.c_int] * 3 + [fp, fp, fp, ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                                        ctypes.c_int, ctypes.c_int, dp,
                                                        ctypes.POINTER(ctypes.c_byte),
                                                        ctypes.POINTER(_Info)]
        _lib.pno_solve.restype = ctypes.c_int
        _lib.pno_solve_from.argtypes = [ctypes.c_int] * 3 + [fp, fp, fp, ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                                             ctypes.c_int, ctypes.c_int, dp, dp,
                                                             ctypes.POINTER(ctypes.c_byte), ctypes.POINTER(_Info)]
        _lib.pno_solve_from.restype = ctypes.c_int
        _lib.pno_certificate.argtypes = [ctypes.c_int] * 3 + [fp, fp, fp, ctypes.c_int, ctypes.c_int, dp, dp, dp,
                                         ctypes.POINTER(ctypes.c_byte)]
        _lib.pno_certificate.restype = ctypes.c_int
    return _lib


def _ptr(a, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct)) if a is not None else None


def _prep(nx, ny, nz, g):
    if g is None:
        return None
    g = np.ascontiguousarray(g, dtype=np.float32)
    assert g.size == nx * ny * nz
    return g


_STATUS = {0: "ok", 1: "no_spanning_cluster", 2: "max_iters"}


def solve(nx, ny, nz, gx, gy, gz, direction=0, tol=1e-13, max_iter=200000, threads=0, periodic=False,
          P_start=None):
    """`P_start` (optional, N doubles): starting iterate on the solved nodes instead of the zero start."""
    lib = _load()
    gx, gy, gz = (_prep(nx, ny, nz, g) for g in (gx, gy, gz))
    P = np.empty((nz, ny, nx), dtype=np.float64)
    cls = np.empty((nz, ny, nx), dtype=np.int8)
    info = _Info()
    if P_start is not None:
        P_start = np.ascontiguousarray(P_start, dtype=np.float64)
        assert P_start.size == nx * ny * nz
    rc = lib.pno_solve_from(nx, ny, nz, _ptr(gx, ctypes.c_float), _ptr(gy, ctypes.c_float),
                            _ptr(gz, ctypes.c_float), direction, 1 if periodic else 0, tol, max_iter, threads,
                            _ptr(P_start, ctypes.c_double), _ptr(P, ctypes.c_double), _ptr(cls, ctypes.c_byte),
                            ctypes.byref(info))
    if rc < 0:
        raise ValueError(f"pno_solve failed with code {rc}")
    return COracleResult(P, cls, info.q_in, info.q_out, info.g_eff, info.k_eff, info.iterations,
                         info.restarts, info.rel_residual, info.n_solved, info.n_inlet_only,
                         info.n_outlet_only, info.n_floating, _STATUS[rc], info.threads,
                         info.t_label, info.t_assemble, info.t_pcg, info.nnz, tuple(info.it_decade))


def certificate(nx, ny, nz, gx, gy, gz, P, direction=0, classes_out=None, periodic=False):
    """(rel_residual, pin_err) of any pressure field; `classes_out` (int8 array of N entries, optional)
    receives the node classes of the serial labelling."""
    lib = _load()
    gx, gy, gz = (_prep(nx, ny, nz, g) for g in (gx, gy, gz))
    P = np.ascontiguousarray(P, dtype=np.float64)
    rel = ctypes.c_double()
    pin = ctypes.c_double()
    rc = lib.pno_certificate(nx, ny, nz, _ptr(gx, ctypes.c_float), _ptr(gy, ctypes.c_float),
                             _ptr(gz, ctypes.c_float), direction, 1 if periodic else 0, _ptr(P, ctypes.c_double),
                             ctypes.byref(rel), ctypes.byref(pin), _ptr(classes_out, ctypes.c_byte))
    if rc < 0:
        raise ValueError(f"pno_certificate failed with code {rc}")
    return rel.value, pin.value

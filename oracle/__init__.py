"""ORACLE -- test infrastructure, NOT product code.

Plain CPU implementation (C, double precision) of the paper's Algorithm 1 (flooding Sum-Product) in the
syndrome form named by BASELINE.json, plus the BIAWGN capacity integrator (`oracle.capacity`).

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference` legs may import this
package.  Nothing here imports the CUDA package, and the CUDA package never imports this one.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import NamedTuple, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle_sumproduct.so")
_SRC = [os.path.join(_HERE, "sumproduct_oracle.c"), os.path.join(_HERE, "sumproduct_core.inc")]
MSG_MAX = 30.0   # clamp on |m_cv| (reading S2); the CUDA path defines its own constant
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, OpenMP over frames only). Returns the path of the shared library."""
    stale = (not os.path.exists(_SO)) or any(os.path.getmtime(s) > os.path.getmtime(_SO) for s in _SRC)
    if force or stale:
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
               "-o", _SO, _SRC[0], "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return _SO


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.oracle_phi.restype = ctypes.c_double
        lib.oracle_phi.argtypes = [ctypes.c_double]
        lib.oracle_build_h_coo.restype = ctypes.c_int64
        lib.oracle_build_h_coo.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                           ctypes.c_void_p, ctypes.c_void_p]
        lib.oracle_decode_from.restype = ctypes.c_int
        lib.oracle_decode_from.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                      ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                      ctypes.c_int, ctypes.c_double, ctypes.c_int, ctypes.c_int,
                                      ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                      ctypes.c_void_p]
        lib.oracle_decode_sparse.restype = ctypes.c_int
        lib.oracle_decode_sparse.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64,
                                             ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                             ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int,
                                             ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_int, ctypes.c_int,
                                             ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                             ctypes.c_void_p]
        lib.oracle_syndrome_sparse.restype = ctypes.c_int
        lib.oracle_syndrome_sparse.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64,
                                               ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_void_p,
                                               ctypes.c_int, ctypes.c_void_p]
        _lib = lib
    return _lib


def phi(x: float) -> float:
    """Phi(x) = -ln tanh(x/2), as evaluated by the oracle."""
    return _load().oracle_phi(float(x))


def build_h_coo(base_shifts: np.ndarray, Z: int):
    """(rows, cols) of the non-zeros of H, check-major, by the oracle's own expansion of (base_shifts, Z)."""
    base = np.ascontiguousarray(base_shifts, dtype=np.int32)
    mb, nb = base.shape
    E = int((base >= 0).sum()) * Z
    rows = np.empty(E, dtype=np.int64)
    cols = np.empty(E, dtype=np.int64)
    got = _load().oracle_build_h_coo(base.ctypes.data, mb, nb, Z, rows.ctypes.data, cols.ctypes.data)
    if got != E:
        raise ValueError(f"oracle_build_h_coo failed ({got})")
    return rows, cols


class OracleResult(NamedTuple):
    hard: np.ndarray        # uint8 [F][n]
    iters: np.ndarray       # int32 [F]
    passed: np.ndarray      # uint8 [F]
    posterior: np.ndarray   # float64 [F][n]
    msg_cv: Optional[np.ndarray]   # float64 [F][E] (check-major edge order) or None


def decode(base_shifts: np.ndarray, Z: int, llr: np.ndarray, syndrome: np.ndarray, max_iter: int,
           early_stop: int, msg_max: float = MSG_MAX, precision: int = 64, want_messages: bool = False,
           threads: Optional[int] = None, check_from: int = 1) -> OracleResult:
    """Run the oracle on frames llr float32 [F][n], syndrome uint8 [F][m]."""
    base = np.ascontiguousarray(base_shifts, dtype=np.int32)
    mb, nb = base.shape
    llr = np.ascontiguousarray(llr, dtype=np.float32)
    syndrome = np.ascontiguousarray(syndrome, dtype=np.uint8)
    if llr.ndim == 1:
        llr = llr[None]
        syndrome = syndrome[None]
    F, n = llr.shape
    m = mb * Z
    assert n == nb * Z and syndrome.shape == (F, m), (llr.shape, syndrome.shape, nb, mb, Z)
    hard = np.zeros((F, n), dtype=np.uint8)
    iters = np.zeros(F, dtype=np.int32)
    passed = np.zeros(F, dtype=np.uint8)
    post = np.zeros((F, n), dtype=np.float64)
    E = int((base >= 0).sum()) * Z
    msg = np.zeros((F, E), dtype=np.float64) if want_messages else None
    lib = _load()
    rc = lib.oracle_decode_from(base.ctypes.data, mb, nb, Z, llr.ctypes.data, syndrome.ctypes.data, F, int(max_iter),
                           int(early_stop), int(check_from), float(msg_max), int(precision), int(threads or 0),
                           hard.ctypes.data, iters.ctypes.data,
                           passed.ctypes.data, post.ctypes.data, msg.ctypes.data if msg is not None else None)
    if rc != 0:
        raise RuntimeError(f"oracle_decode failed with status {rc}")
    return OracleResult(hard, iters, passed, post, msg)


def decode_sparse(rows: np.ndarray, cols: np.ndarray, shifts: np.ndarray, mb: int, nb: int, Z: int,
                  llr: np.ndarray, syndrome: np.ndarray, max_iter: int, early_stop: int, msg_max: float = MSG_MAX,
                  precision: int = 64, threads: Optional[int] = None, check_from: int = 1) -> OracleResult:
    """The oracle on a code given by its non-zero blocks (rows[k], cols[k], shifts[k]); frames as in decode()."""
    r = np.ascontiguousarray(rows, dtype=np.int32)
    c = np.ascontiguousarray(cols, dtype=np.int32)
    p = np.ascontiguousarray(shifts, dtype=np.int32)
    llr = np.ascontiguousarray(llr, dtype=np.float32)
    syndrome = np.ascontiguousarray(syndrome, dtype=np.uint8)
    if llr.ndim == 1:
        llr = llr[None]
        syndrome = syndrome[None]
    F, n = llr.shape
    m = mb * Z
    assert n == nb * Z and syndrome.shape == (F, m), (llr.shape, syndrome.shape, nb, mb, Z)
    hard = np.zeros((F, n), dtype=np.uint8)
    iters = np.zeros(F, dtype=np.int32)
    passed = np.zeros(F, dtype=np.uint8)
    post = np.zeros((F, n), dtype=np.float64)
    rc = _load().oracle_decode_sparse(r.ctypes.data, c.ctypes.data, p.ctypes.data, len(r), int(mb), int(nb), int(Z),
                                      llr.ctypes.data, syndrome.ctypes.data, F, int(max_iter), int(early_stop),
                                      int(check_from), float(msg_max), int(precision), int(threads or 0),
                                      hard.ctypes.data, iters.ctypes.data, passed.ctypes.data, post.ctypes.data, None)
    if rc != 0:
        raise RuntimeError(f"oracle_decode_sparse failed with status {rc}")
    return OracleResult(hard, iters, passed, post, None)


def syndrome_sparse(rows, cols, shifts, mb: int, nb: int, Z: int, x: np.ndarray) -> np.ndarray:
    """s = H x mod 2 by the oracle's own loop over the non-zero blocks (x uint8 [F][n] -> uint8 [F][m])."""
    r = np.ascontiguousarray(rows, dtype=np.int32)
    c = np.ascontiguousarray(cols, dtype=np.int32)
    p = np.ascontiguousarray(shifts, dtype=np.int32)
    x = np.ascontiguousarray(x, dtype=np.uint8)
    if x.ndim == 1:
        x = x[None]
    s = np.zeros((x.shape[0], mb * Z), dtype=np.uint8)
    rc = _load().oracle_syndrome_sparse(r.ctypes.data, c.ctypes.data, p.ctypes.data, len(r), int(mb), int(nb), int(Z),
                                        x.ctypes.data, x.shape[0], s.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"oracle_syndrome_sparse failed with status {rc}")
    return s

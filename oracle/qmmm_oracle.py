"""ctypes loader for the plain-C FP64 oracle (oracle/qmmm_oracle.c).

TEST INFRASTRUCTURE.  Follows PAPER.md:59-60 (Eq. 4) term by term; see the C
file's header for the definition, the sign convention and the list of pins.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "qmmm_oracle.c")
_LIB = os.path.join(_HERE, "libqmmm_oracle.so")
# -ffp-contract=off: no FMA contraction; -fno-fast-math: IEEE sqrt/divide, no
# reassociation (Kahan must survive the optimiser).
_CFLAGS = ["-O2", "-fno-fast-math", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
           "-std=c11", "-Wall", "-Wextra"]

_lib: Optional[ctypes.CDLL] = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc if the .so is missing or older than the source."""
    stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
    if force or stale:
        subprocess.run(["gcc", *_CFLAGS, _SRC, "-o", _LIB, "-lm"], check=True)
    return _LIB


def _load() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        lib.qmmm_oracle_field.restype = ctypes.c_int
        lib.qmmm_oracle_field.argtypes = [dp, dp, ctypes.c_int64, dp, dp, ctypes.c_int64,
                                          dp, ctypes.c_int64, dp, dp, dp, dp, ctypes.c_int]
        lib.qmmm_oracle_terms.restype = None
        lib.qmmm_oracle_terms.argtypes = [dp, dp, ctypes.c_int64, dp, dp, ctypes.c_int64,
                                          dp, dp]
        _lib = lib
    return _lib


def _arr(a, shape_tail=()) -> np.ndarray:
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float64))
    if shape_tail and a.size:
        a = a.reshape((-1,) + tuple(shape_tail))
    return a


def _ptr(a: Optional[np.ndarray]):
    if a is None:
        return None
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


@dataclass
class OracleResult:
    V: np.ndarray              # [P]
    E: Optional[np.ndarray]    # [P][3]
    absV: Optional[np.ndarray]  # sum_j |q_j|/r_ij      -> kappa_V = absV/|V|
    absE: Optional[np.ndarray]  # sum_j |q_j|/r_ij^2    -> kappa_E = absE/|E|
    threads: int


def field(src_xyz, src_q, nuc_xyz, nuc_Z, elec_xyz, want_E: bool = True,
          want_abs: bool = False, nthreads: int = 0) -> OracleResult:
    """V and E at every row of elec_xyz ([...,3]; leading dims are flattened)."""
    src_xyz = _arr(src_xyz, (3,)); src_q = _arr(src_q)
    nuc_xyz = _arr(nuc_xyz, (3,)); nuc_Z = _arr(nuc_Z)
    elec = _arr(elec_xyz, (3,))
    M, K, P = src_q.size, nuc_Z.size, elec.shape[0] if elec.size else 0
    assert src_xyz.size == 3 * M and nuc_xyz.size == 3 * K
    V = np.zeros(P)
    E = np.zeros((P, 3)) if want_E else None
    aV = np.zeros(P) if want_abs else None
    aE = np.zeros(P) if want_abs else None
    used = _load().qmmm_oracle_field(_ptr(src_xyz), _ptr(src_q), M, _ptr(nuc_xyz), _ptr(nuc_Z),
                                     K, _ptr(elec), P, _ptr(V), _ptr(E), _ptr(aV), _ptr(aE),
                                     int(nthreads))
    return OracleResult(V, E, aV, aE, used)


def potential_terms(src_xyz, src_q, nuc_xyz, nuc_Z, r) -> np.ndarray:
    """The M+K individual terms q_j/|r - R_j| of one point, in array order."""
    src_xyz = _arr(src_xyz, (3,)); src_q = _arr(src_q)
    nuc_xyz = _arr(nuc_xyz, (3,)); nuc_Z = _arr(nuc_Z)
    r = _arr(r)
    out = np.zeros(src_q.size + nuc_Z.size)
    _load().qmmm_oracle_terms(_ptr(src_xyz), _ptr(src_q), src_q.size, _ptr(nuc_xyz),
                              _ptr(nuc_Z), nuc_Z.size, _ptr(r), _ptr(out))
    return out

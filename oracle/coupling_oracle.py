"""ctypes wrapper around oracle/coupling_oracle.c (Eq. 4) -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/ and bench.py's cpu_baseline leg import this.  float32 inputs are widened bit-exactly to float64.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "coupling_oracle.c")
_LIB = os.path.join(_HERE, "libcoupling_oracle.so")
_lib = None

COULOMB_KCAL_A = 332.0637133  # 1/(4 pi eps0) in kcal A / (mol e^2) (reading C2: a caller-supplied constant)


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.run(["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC", _SRC,
                        "-o", tmp, "-lm"], check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        lib.coupling_energy_forces.restype = C.c_double
        _lib = lib
    return _lib


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _i(a):
    return a.ctypes.data_as(C.POINTER(C.c_int))


def coupling_energy_forces(pos, nnp_rows, q_nnp, sigma_nnp, eps_nnp, mm_rows, q_mm, sigma_mm, eps_mm,
                           kc: float = COULOMB_KCAL_A, cutoff: float = 0.0, want_forces: bool = True):
    """Eq. 4.  pos [n_rows][3]; returns (V, F [n_rows][3] or None).  Inputs of any float dtype are widened."""
    lib = _load()
    f64 = lambda v: np.ascontiguousarray(np.asarray(v).astype(np.float64))
    i32 = lambda v: np.ascontiguousarray(v, dtype=np.int32)
    pos = f64(pos)
    nnp_rows, mm_rows = i32(nnp_rows), i32(mm_rows)
    qn, sn, en, qm, sm, em = map(f64, (q_nnp, sigma_nnp, eps_nnp, q_mm, sigma_mm, eps_mm))
    F = np.zeros_like(pos) if want_forces else None
    V = lib.coupling_energy_forces(C.c_int(nnp_rows.size), _i(nnp_rows), _d(qn), _d(sn), _d(en),
                                   C.c_int(mm_rows.size), _i(mm_rows), _d(qm), _d(sm), _d(em), _d(pos),
                                   C.c_double(kc), C.c_double(cutoff), _d(F) if F is not None else None)
    return float(V), F

"""Oracle (test infrastructure): ctypes wrapper around the plain-C restatement of eq. 2.1 in
`oracle/wilson_ref.c`.  `build()` compiles it with gcc (also called from
`__graft_entry__.build()`); nothing here touches the CUDA path."""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "wilson_ref.c")
_LIB = os.path.join(_HERE, "libwilson_ref.so")
_lib = None


def build(force=False):
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", _SRC, "-o", _LIB, "-lm"])
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.wd_apply_Q.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                    ctypes.POINTER(ctypes.c_int), ctypes.c_double, ctypes.c_int]
        _lib.wd_apply_Q.restype = None
        _lib.wd_num_threads.restype = ctypes.c_int
    return _lib


def num_threads():
    return int(_load().wd_num_threads())


def apply_Q(psi, U, m, bc_time=-1):
    """Q psi = gamma5 D_W psi (eq. 2.1); psi[x0,x1,x2,x3,4,3], U[4,x0,x1,x2,x3,3,3] complex128."""
    lib = _load()
    psi = np.ascontiguousarray(psi, dtype=np.complex128)
    U = np.ascontiguousarray(U, dtype=np.complex128)
    dims = psi.shape[:4]
    assert U.shape == (4,) + dims + (3, 3) and psi.shape[4:] == (4, 3)
    out = np.empty_like(psi)
    cd = (ctypes.c_int * 4)(*dims)
    lib.wd_apply_Q(psi.ctypes.data, U.ctypes.data, out.ctypes.data, cd, float(m), int(bc_time))
    return out


def make_Q(U, m, bc_time=-1):
    U = np.ascontiguousarray(U, dtype=np.complex128)
    return lambda psi: apply_Q(psi, U, m, bc_time)

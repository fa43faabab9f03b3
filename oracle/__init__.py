"""ctypes binding of the CPU oracle (oracle/fmm_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference leg may import this package.  It never
imports the CUDA path (paper_2101_08226_b200) and shares no code with it.

The C source is compiled on first use with the host gcc:
    gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC fmm_oracle.c -o libfmm_oracle.so -lm
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fmm_oracle.c")
_LIB = os.path.join(_HERE, "libfmm_oracle.so")
_lib = None

OK, EINVAL, EMASS = 0, 1, 2


def build(force: bool = False) -> str:
    """Compile the oracle if the shared object is missing or older than its source."""
    stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
    if force or stale:
        tmp = _LIB + ".tmp.%d" % os.getpid()
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=c99",
               _SRC, "-o", tmp, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        ullp = ctypes.POINTER(ctypes.c_ulonglong)
        L.fmm_oracle_stencil.argtypes = [ctypes.c_double, ctypes.c_int, ctypes.c_int, ip,
                                         ctypes.POINTER(ctypes.c_byte)]
        L.fmm_oracle_green.argtypes = [dp, dp]
        L.fmm_oracle_pair.argtypes = [dp, dp, ctypes.c_double, dp, ctypes.c_int, dp, dp]
        L.fmm_oracle_interact_multipole.argtypes = [ip, ip, ip, ctypes.c_double, ctypes.c_double, ctypes.c_int,
                                                    dp, dp, dp, dp, ullp]
        L.fmm_oracle_interact_monopole.argtypes = [ip, ip, ip, ctypes.c_double, ctypes.c_double, dp, dp, ullp]
        L.fmm_oracle_interaction_count.argtypes = [ip, ip, ip, ctypes.c_double, ullp]
        L.fmm_oracle_num_threads.restype = ctypes.c_int
        L.fmm_oracle_set_num_threads.argtypes = [ctypes.c_int]
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _i3(v):
    return (ctypes.c_int * 3)(*[int(x) for x in v])


def _check(rc, what):
    if rc != OK:
        raise RuntimeError("%s failed with status %d" % (what, rc))


def stencil(theta: float, parity: int) -> np.ndarray:
    """Partner offsets (dx,dy,dz) of parity class px+2py+4pz, int8 [count][3], (dz,dy,dx)-lexicographic."""
    L = lib()
    cnt = ctypes.c_int(0)
    _check(L.fmm_oracle_stencil(theta, parity, 0, ctypes.byref(cnt), None), "stencil")
    out = np.zeros((cnt.value, 3), dtype=np.int8)
    _check(L.fmm_oracle_stencil(theta, parity, cnt.value, ctypes.byref(cnt),
                                out.ctypes.data_as(ctypes.POINTER(ctypes.c_byte))), "stencil")
    return out


def green(R) -> tuple:
    """Full derivative tensors (D0, D1[3], D2[3,3], D3[3,3,3], D4[3,3,3,3]) of -1/|R|."""
    R = np.ascontiguousarray(R, dtype=np.float64)
    out = np.zeros(121)
    _check(lib().fmm_oracle_green(_dp(R), _dp(out)), "green")
    return (out[0], out[1:4].copy(), out[4:13].reshape(3, 3).copy(), out[13:40].reshape(3, 3, 3).copy(),
            out[40:121].reshape(3, 3, 3, 3).copy())


def pair(R, MB, MA0=1.0, MA3=None, correction=False):
    """One ordered pair A<-B: returns (L[20] without correction, dL1[3])."""
    R = np.ascontiguousarray(R, dtype=np.float64)
    MB = np.ascontiguousarray(MB, dtype=np.float64)
    MA3 = np.zeros(10) if MA3 is None else np.ascontiguousarray(MA3, dtype=np.float64)
    Lo, dL = np.zeros(20), np.zeros(3)
    _check(lib().fmm_oracle_pair(_dp(R), _dp(MB), float(MA0), _dp(MA3), int(bool(correction)), _dp(Lo), _dp(dL)),
           "pair")
    return Lo, dL


def interact_multipole(n, h, theta, moments, com_off, out_lo=None, out_hi=None, am_correction=True, threads=None):
    """Returns (L[20][oz][oy][ox], Lcorr[3][oz][oy][ox], n_interactions)."""
    L = lib()
    if threads:
        L.fmm_oracle_set_num_threads(int(threads))
    out_lo = (0, 0, 0) if out_lo is None else out_lo
    out_hi = tuple(n) if out_hi is None else out_hi
    moments = np.ascontiguousarray(moments, dtype=np.float64)
    com_off = np.ascontiguousarray(com_off, dtype=np.float64)
    nx, ny, nz = n
    assert moments.shape == (20, nz, ny, nx) and com_off.shape == (3, nz, ny, nx)
    o = tuple(out_hi[a] - out_lo[a] for a in range(3))
    Lout = np.zeros((20, o[2], o[1], o[0]))
    Lc = np.zeros((3, o[2], o[1], o[0]))
    cnt = ctypes.c_ulonglong(0)
    rc = L.fmm_oracle_interact_multipole(_i3(n), _i3(out_lo), _i3(out_hi), float(h), float(theta),
                                         int(bool(am_correction)), _dp(moments), _dp(com_off), _dp(Lout), _dp(Lc),
                                         ctypes.byref(cnt))
    _check(rc, "interact_multipole")
    return Lout, Lc, cnt.value


def interact_monopole(n, h, theta, mass, out_lo=None, out_hi=None, threads=None):
    """Returns (out[4][oz][oy][ox] = phi,gx,gy,gz ; n_interactions)."""
    L = lib()
    if threads:
        L.fmm_oracle_set_num_threads(int(threads))
    out_lo = (0, 0, 0) if out_lo is None else out_lo
    out_hi = tuple(n) if out_hi is None else out_hi
    nx, ny, nz = n
    mass = np.ascontiguousarray(mass, dtype=np.float64).reshape(nz, ny, nx)
    o = tuple(out_hi[a] - out_lo[a] for a in range(3))
    out = np.zeros((4, o[2], o[1], o[0]))
    cnt = ctypes.c_ulonglong(0)
    _check(L.fmm_oracle_interact_monopole(_i3(n), _i3(out_lo), _i3(out_hi), float(h), float(theta), _dp(mass),
                                          _dp(out), ctypes.byref(cnt)), "interact_monopole")
    return out, cnt.value


def interaction_count(n, theta, out_lo=None, out_hi=None) -> int:
    out_lo = (0, 0, 0) if out_lo is None else out_lo
    out_hi = tuple(n) if out_hi is None else out_hi
    cnt = ctypes.c_ulonglong(0)
    _check(lib().fmm_oracle_interaction_count(_i3(n), _i3(out_lo), _i3(out_hi), float(theta), ctypes.byref(cnt)),
           "interaction_count")
    return cnt.value


def num_threads() -> int:
    return int(lib().fmm_oracle_num_threads())

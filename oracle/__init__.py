"""fp64 CPU oracle -- TEST INFRASTRUCTURE (see nb_oracle.c).  Only tests/, smoke() and bench.py's
CPU-baseline legs may import this; the product package never does.

`build()` compiles nb_oracle.c with gcc for the host it runs on (the .so is rebuilt when the
source or the host CPU changes); `predict` and `force` are thin ctypes wrappers over numpy arrays.
"""
import ctypes
import hashlib
import os
import platform
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nb_oracle.c")
_LIB = None


def _host_tag():
    flags = ""
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    flags = line
                    break
    except OSError:
        pass
    with open(_SRC, "rb") as f:
        src = f.read()
    return hashlib.sha1(src + flags.encode() + platform.machine().encode()).hexdigest()[:12]


def build():
    """Compile the oracle for this host; returns the path of the shared object."""
    so = os.path.join(_HERE, "libnb_oracle_%s.so" % _host_tag())
    if not os.path.exists(so):
        tmp = so + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", "-O3", "-march=native", "-ffp-contract=off", "-fno-fast-math",
                               "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, so)
    return so


def _lib():
    global _LIB
    if _LIB is None:
        L = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        L.oracle_predict.argtypes = [ctypes.c_int64, ctypes.c_double] + [dp] * 7
        L.oracle_predict.restype = None
        L.oracle_force.argtypes = [ctypes.c_int64, dp, dp, dp, ctypes.POINTER(ctypes.c_uint8),
                                   ctypes.c_int64, ctypes.POINTER(ctypes.c_int32), ctypes.c_double,
                                   dp, dp, dp]
        L.oracle_force.restype = None
        L.oracle_force6.argtypes = [ctypes.c_int64, dp, dp, dp, dp, ctypes.POINTER(ctypes.c_uint8),
                                    ctypes.c_int64, ctypes.POINTER(ctypes.c_int32), ctypes.c_double,
                                    dp, dp, dp, dp]
        L.oracle_force6.restype = None
        L.oracle_predict_acc.argtypes = [ctypes.c_int64, ctypes.c_double, dp, dp, dp, dp]
        L.oracle_predict_acc.restype = None
        L.oracle_threads.restype = ctypes.c_int
        _LIB = L
    return _LIB


def _d(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _c(a, dtype=np.float64):
    return np.ascontiguousarray(a, dtype=dtype)


def threads():
    return int(_lib().oracle_threads())


def predict(t, x, v, a, j, tj):
    """Predicted (xp, vp), each (3, n), of particles stored as x, v, a, j (3, n) at times tj (n,)."""
    x, v, a, j, tj = _c(x), _c(v), _c(a), _c(j), _c(tj)
    n = tj.shape[0]
    assert x.shape == v.shape == a.shape == j.shape == (3, n)
    xp, vp = np.empty((3, n)), np.empty((3, n))
    _lib().oracle_predict(n, float(t), _d(x), _d(v), _d(a), _d(j), _d(tj), _d(xp), _d(vp))
    return xp, vp


def force(m, xp, vp, i_list, eps2, flags=None):
    """acc (3, ni), jrk (3, ni), pot (ni,) on particles i_list from all n particles (m, xp, vp)."""
    m, xp, vp = _c(m), _c(xp), _c(vp)
    n = m.shape[0]
    assert xp.shape == vp.shape == (3, n)
    il = _c(i_list, np.int32)
    ni = il.shape[0]
    assert ni == 0 or (il.min() >= 0 and il.max() < n)
    fl = None
    if flags is not None:
        flags = _c(flags, np.uint8)
        assert flags.shape == (n,)
        fl = flags.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8))
    acc, jrk, pot = np.empty((3, ni)), np.empty((3, ni)), np.empty(ni)
    _lib().oracle_force(n, _d(m), _d(xp), _d(vp), fl, ni,
                        il.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), float(eps2),
                        _d(acc), _d(jrk), _d(pot))
    return acc, jrk, pot


def predict_acc(t, a, j, tj):
    """Predicted acceleration ap = a + jerk (t - tj), (3, n) (reading R22)."""
    a, j, tj = _c(a), _c(j), _c(tj)
    n = tj.shape[0]
    assert a.shape == j.shape == (3, n)
    ap = np.empty((3, n))
    _lib().oracle_predict_acc(n, float(t), _d(a), _d(j), _d(tj), _d(ap))
    return ap


def force6(m, xp, vp, ap, i_list, eps2, flags=None):
    """6th-order variant: acc, jrk, snp (3, ni) and pot (ni,) on particles i_list, given positions,
    velocities and accelerations (3, n) of all particles at one instant."""
    m, xp, vp, ap = _c(m), _c(xp), _c(vp), _c(ap)
    n = m.shape[0]
    assert xp.shape == vp.shape == ap.shape == (3, n)
    il = _c(i_list, np.int32)
    ni = il.shape[0]
    assert ni == 0 or (il.min() >= 0 and il.max() < n)
    fl = None
    if flags is not None:
        flags = _c(flags, np.uint8)
        assert flags.shape == (n,)
        fl = flags.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8))
    acc, jrk, snp, pot = np.empty((3, ni)), np.empty((3, ni)), np.empty((3, ni)), np.empty(ni)
    _lib().oracle_force6(n, _d(m), _d(xp), _d(vp), _d(ap), fl, ni,
                         il.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), float(eps2),
                         _d(acc), _d(jrk), _d(snp), _d(pot))
    return acc, jrk, snp, pot

"""ctypes front-end of oracle/kf_oracle.c -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It never imports the CUDA binding.  All arrays are host numpy; fp32 inputs are widened to fp64 exactly.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "kf_oracle.c")
_SO = os.path.join(_HERE, "libkf_oracle.so")
_lib = None

UNREACHABLE, LEFT_Z, GRAZING, NUMERIC = 1, 2, 4, 8


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", _SRC, "-o", _SO, "-lm"]
        subprocess.run(cmd, check=True)
    return _SO


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.kfo_num_threads.restype = C.c_int
    return _lib


def num_threads() -> int:
    return int(lib().kfo_num_threads())


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a, t=C.c_double):
    return a.ctypes.data_as(C.POINTER(t)) if a is not None else None


def propagate(p, q, bz, R):
    """-> (flags, p_out[6], J[6,6], s, cos_inc)"""
    p = _d(p); po = np.zeros(6); J = np.zeros(36); s = C.c_double(); ci = C.c_double()
    f = lib().kfo_propagate(_p(p), C.c_int(int(q)), C.c_double(bz), C.c_double(R), _p(po), _p(J), C.byref(s), C.byref(ci))
    return f, po, J.reshape(6, 6), s.value, ci.value


def ms_noise(p, cosinc, xx0):
    p = _d(p); Q = np.zeros(36)
    lib().kfo_ms_noise(_p(p), C.c_double(cosinc), C.c_double(xx0), _p(Q))
    return Q.reshape(6, 6)


def inv3_spd(S):
    S = _d(S).reshape(9); out = np.zeros(9)
    rc = lib().kfo_inv3_spd(_p(S), _p(out))
    return rc, out.reshape(3, 3)


def similarity6(J, Cm):
    J = _d(J).reshape(36); Cm = _d(Cm).reshape(36); out = np.zeros(36)
    lib().kfo_similarity6(_p(J), _p(Cm), _p(out))
    return out.reshape(6, 6)


def update(p, Cm, m, sig_rphi, sig_z, sig_r):
    """-> (flags, p_out, C_out, chi2)"""
    p = _d(p); Cm = _d(Cm).reshape(36); m = _d(m); po = np.zeros(6); Co = np.zeros(36); c2 = C.c_double()
    f = lib().kfo_update(_p(p), _p(Cm), _p(m), C.c_double(sig_rphi), C.c_double(sig_z), C.c_double(sig_r), _p(po), _p(Co), C.byref(c2))
    return f, po, Co.reshape(6, 6), c2.value


def chi2(p, Cm, m, sig_rphi, sig_z, sig_r):
    p = _d(p); Cm = _d(Cm).reshape(36); m = _d(m); c2 = C.c_double()
    rc = lib().kfo_chi2(_p(p), _p(Cm), _p(m), C.c_double(sig_rphi), C.c_double(sig_z), C.c_double(sig_r), C.byref(c2))
    return rc, c2.value


def predict(layers, l, bz, p, Cm, q):
    """propagate to layer l + J C J^T + Q  -> (flags, p_pred, C_pred)"""
    layers = _d(layers); p = _d(p); Cm = _d(Cm).reshape(36); po = np.zeros(6); Co = np.zeros(36)
    f = lib().kfo_predict(_p(layers), C.c_int(l), C.c_double(bz), _p(p), _p(Cm), C.c_int(int(q)), _p(po), _p(Co))
    return f, po, Co.reshape(6, 6)


def _unpack21(cov21):
    """[21][ld] packed lower-triangular row-major -> dense [36][ld] (layout conversion only)."""
    ld = cov21.shape[1]
    out = np.empty((36, ld), dtype=np.float64)
    for i in range(6):
        for j in range(6):
            a, b = (i, j) if i >= j else (j, i)
            out[i * 6 + j] = cov21[a * (a + 1) // 2 + b]
    return out


def fit(layers, bz, par, cov21, q, hx, hy, hz, seg_off, hit_idx=None, trk_event=None, n=None):
    """kf_fit_ref.  par [6][ld], cov21 [21][ld] (any float dtype), q [n] int8.
    -> dict(par [6][n] f64, cov [n][6][6] f64, chi2 [n], nhits [n], status [n])"""
    layers = _d(layers)
    L = layers.shape[0]
    par = _d(par); ld = par.shape[1]
    n = len(q) if n is None else n
    cov = _unpack21(_d(cov21))
    q = np.ascontiguousarray(q, dtype=np.int8)
    hx, hy, hz = _d(hx), _d(hy), _d(hz)
    seg_off = np.ascontiguousarray(seg_off, dtype=np.int64)
    hi = None if hit_idx is None else np.ascontiguousarray(hit_idx, dtype=np.int32)
    te = None if trk_event is None else np.ascontiguousarray(trk_event, dtype=np.int32)
    if hi is not None:
        assert hi.shape == (L, ld)
    po = np.zeros((6, ld)); co = np.zeros((36, ld)); c2 = np.zeros(n); nh = np.zeros(n, dtype=np.int32); st = np.zeros(n, dtype=np.uint32)
    lib().kfo_fit(C.c_int(L), _p(layers), C.c_double(bz), C.c_int64(n), C.c_int64(ld), _p(par), _p(cov), _p(q, C.c_int8),
                  _p(hx), _p(hy), _p(hz), _p(seg_off, C.c_int64), _p(hi, C.c_int32), _p(te, C.c_int32),
                  _p(po), _p(co), _p(c2), _p(nh, C.c_int32), _p(st, C.c_uint32))
    return dict(par=po[:, :n], cov=co[:, :n].T.reshape(n, 6, 6), chi2=c2, nhits=nh, status=st)

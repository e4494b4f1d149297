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


def _lt(layers):
    """Layer table for the C side: [L][8] = r (or the z of a disk), zmax (or the outer radius of a disk), xx0, sig_rphi,
    sig_z, sig_r, kind (0 barrel, 1 disk), rmin.  A [L][6] table (barrel only) is padded with kind = 0, rmin = 0."""
    t = np.asarray(layers, dtype=np.float64)
    if t.shape[1] == 6:
        t = np.concatenate([t, np.zeros((t.shape[0], 2))], axis=1)
    assert t.shape[1] == 8
    return np.ascontiguousarray(t)


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
    layers = _lt(layers); p = _d(p); Cm = _d(Cm).reshape(36); po = np.zeros(6); Co = np.zeros(36)
    f = lib().kfo_predict(_p(layers), C.c_int(l), C.c_double(bz), _p(p), _p(Cm), C.c_int(int(q)), _p(po), _p(Co))
    return f, po, Co.reshape(6, 6)


def propagate_near(p, q, bz, R):
    """second step to the nearest crossing of the cylinder R (either direction) -> (flags, p_out, J, s)"""
    p = _d(p); po = np.zeros(6); J = np.zeros(36); s = C.c_double()
    f = lib().kfo_propagate_near(_p(p), C.c_int(int(q)), C.c_double(bz), C.c_double(R), _p(po), _p(J), C.byref(s))
    return f, po, J.reshape(6, 6), s.value


def propagate_z(p, q, bz, Z, forward_only=True):
    """to the plane z = Z -> (flags, p_out, J, s, |cos theta|)"""
    p = _d(p); po = np.zeros(6); J = np.zeros(36); s = C.c_double(); ci = C.c_double()
    f = lib().kfo_propagate_z(_p(p), C.c_int(int(q)), C.c_double(bz), C.c_double(Z), C.c_int(1 if forward_only else 0), _p(po), _p(J),
                              C.byref(s), C.byref(ci))
    return f, po, J.reshape(6, 6), s.value, ci.value


def update_2d(p, Cm, m, kind, s1, s2):
    """2-D update on the plane tangent to the hit radius -> (flags, p_out, C_out, chi2)"""
    p = _d(p); Cm = _d(Cm).reshape(36); m = _d(m); po = np.zeros(6); Co = np.zeros(36); c2 = C.c_double()
    f = lib().kfo_update_2d(_p(p), _p(Cm), _p(m), C.c_int(kind), C.c_double(s1), C.c_double(s2), _p(po), _p(Co), C.byref(c2))
    return f, po, Co.reshape(6, 6), c2.value


def chi2_2d(p, Cm, m, kind, s1, s2):
    p = _d(p); Cm = _d(Cm).reshape(36); m = _d(m); c2 = C.c_double()
    rc = lib().kfo_chi2_2d(_p(p), _p(Cm), _p(m), C.c_int(kind), C.c_double(s1), C.c_double(s2), C.byref(c2))
    return rc, c2.value


def to_hit_surface(kind, bz, q, pp, Cp, m):
    """second step of the two-step propagation -> (flags, p2, C2)"""
    pp = _d(pp); Cp = _d(Cp).reshape(36); m = _d(m); p2 = np.zeros(6); C2 = np.zeros(36)
    f = lib().kfo_to_hit_surface(C.c_int(kind), C.c_double(bz), C.c_int(int(q)), _p(pp), _p(Cp), _p(m), _p(p2), _p(C2))
    return f, p2, C2.reshape(6, 6)


def _unpack21(cov21):
    """[21][ld] packed lower-triangular row-major -> dense [36][ld] (layout conversion only)."""
    ld = cov21.shape[1]
    out = np.empty((36, ld), dtype=np.float64)
    for i in range(6):
        for j in range(6):
            a, b = (i, j) if i >= j else (j, i)
            out[i * 6 + j] = cov21[a * (a + 1) // 2 + b]
    return out


def fit(layers, bz, par, cov21, q, hx, hy, hz, seg_off, hit_idx=None, trk_event=None, n=None, hit_mode=0):
    """kf_fit_ref.  par [6][ld], cov21 [21][ld] (any float dtype), q [n] int8.  hit_mode 1: two-step propagation to each
    hit's own radius / z and 2-D update on the tangent plane.
    -> dict(par [6][n] f64, cov [n][6][6] f64, chi2 [n], nhits [n], status [n])"""
    layers = _lt(layers)
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
    lib().kfo_fit(C.c_int(L), _p(layers), C.c_double(bz), C.c_int(hit_mode), C.c_int64(n), C.c_int64(ld), _p(par), _p(cov), _p(q, C.c_int8),
                  _p(hx), _p(hy), _p(hz), _p(seg_off, C.c_int64), _p(hi, C.c_int32), _p(te, C.c_int32),
                  _p(po), _p(co), _p(c2), _p(nh, C.c_int32), _p(st, C.c_uint32))
    return dict(par=po[:, :n], cov=co[:, :n].T.reshape(n, 6, 6), chi2=c2, nhits=nh, status=st)


# ---------------------------------------------------------------------------------------------------------
# binning / window lookup / building
# ---------------------------------------------------------------------------------------------------------
def _f(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _i(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def tan_table(n_phi):
    tab = np.zeros(n_phi // 8 + 1, dtype=np.float32)
    lib().kfo_tan_table(C.c_int(n_phi), _p(tab, C.c_float))
    return tab


def phi_bin(x, y, n_phi):
    l = lib(); l.kfo_phi_bin.restype = C.c_int
    tab = tan_table(n_phi)
    x, y = _f(np.atleast_1d(x)), _f(np.atleast_1d(y))
    return np.array([l.kfo_phi_bin(C.c_float(float(a)), C.c_float(float(b)), C.c_int(n_phi), _p(tab, C.c_float)) for a, b in zip(x, y)], dtype=np.int32)


def z_bin(z, zmax, n_z):
    l = lib(); l.kfo_z_bin.restype = C.c_int
    return np.array([l.kfo_z_bin(C.c_float(float(a)), C.c_float(float(zmax)), C.c_int(n_z)) for a in _f(np.atleast_1d(z))], dtype=np.int32)


def row_bin(v, lo, hi, n):
    """X2 for any layer (R22): row of v in [lo, hi) cut into n rows (barrel: z in [-zmax, zmax); disk: radius)."""
    l = lib(); l.kfo_row_bin.restype = C.c_int
    return np.array([l.kfo_row_bin(C.c_float(float(a)), C.c_float(float(lo)), C.c_float(float(hi)), C.c_int(n)) for a in _f(np.atleast_1d(v))], dtype=np.int32)


def hit_rho(x, y):
    """fp32 radius of a hit as the disk binning takes it: sqrt(fl(fl(x x) + fl(y y)))."""
    l = lib(); l.kfo_hit_rho.restype = C.c_float
    return np.array([l.kfo_hit_rho(C.c_float(float(a)), C.c_float(float(b))) for a, b in zip(_f(np.atleast_1d(x)), _f(np.atleast_1d(y)))], dtype=np.float32)


def window_bins_row(phi_c, dphi, c, d, lo, hi, n_phi, n_z):
    """X3 with the row coordinate binned in [lo, hi) -> (first phi bin, n phi bins, row_lo, row_hi)"""
    a, b, e, f = C.c_int(), C.c_int(), C.c_int(), C.c_int()
    lib().kfo_window_bins_row(C.c_float(phi_c), C.c_float(dphi), C.c_float(c), C.c_float(d), C.c_float(lo), C.c_float(hi), C.c_int(n_phi), C.c_int(n_z),
                              C.byref(a), C.byref(b), C.byref(e), C.byref(f))
    return a.value, b.value, e.value, f.value


def window_bins(phi_c, dphi, z_c, dz, zmax, n_phi, n_z):
    """X3 -> (first phi bin, n phi bins, iz_lo, iz_hi)"""
    a, b, c, d = C.c_int(), C.c_int(), C.c_int(), C.c_int()
    lib().kfo_window_bins(C.c_float(phi_c), C.c_float(dphi), C.c_float(z_c), C.c_float(dz), C.c_float(zmax), C.c_int(n_phi), C.c_int(n_z),
                          C.byref(a), C.byref(b), C.byref(c), C.byref(d))
    return a.value, b.value, c.value, d.value


def bin_hits(layers, n_events, seg_off, hx, hy, hz, n_phi, n_z):
    """kf_bin_hits_ref -> dict(x, y, z sorted f32, perm i32, bin_off i32)"""
    layers = _lt(layers); L = layers.shape[0]
    seg_off = np.ascontiguousarray(seg_off, dtype=np.int64)
    assert len(seg_off) == n_events * L + 1
    hx, hy, hz = _f(hx), _f(hy), _f(hz)
    n = int(seg_off[-1])
    sx = np.zeros(n, np.float32); sy = np.zeros(n, np.float32); sz = np.zeros(n, np.float32)
    perm = np.zeros(n, np.int32); bin_off = np.zeros(n_events * L * n_phi * n_z + 1, np.int32)
    lib().kfo_bin_hits(C.c_int(L), _p(layers), C.c_int(n_events), _p(seg_off, C.c_int64), _p(hx, C.c_float), _p(hy, C.c_float), _p(hz, C.c_float),
                       C.c_int(n_phi), C.c_int(n_z), _p(sx, C.c_float), _p(sy, C.c_float), _p(sz, C.c_float), _p(perm, C.c_int32), _p(bin_off, C.c_int32))
    return dict(x=sx, y=sy, z=sz, perm=perm, bin_off=bin_off, n_phi=n_phi, n_z=n_z)


def window_lookup(layers, binned, event, layer, phi_c, dphi, z_c, dz, cap):
    layers = _lt(layers)
    event, layer = _i(event), _i(layer)
    phi_c, dphi, z_c, dz = _f(phi_c), _f(dphi), _f(z_c), _f(dz)
    nq = len(event)
    count = np.zeros(nq, np.int32); idx = np.full((nq, cap), -1, np.int32)
    lib().kfo_window_lookup(C.c_int(layers.shape[0]), _p(layers), C.c_int(binned["n_phi"]), C.c_int(binned["n_z"]), _p(binned["bin_off"], C.c_int32),
                            C.c_int64(nq), _p(event, C.c_int32), _p(layer, C.c_int32), _p(phi_c, C.c_float), _p(dphi, C.c_float),
                            _p(z_c, C.c_float), _p(dz, C.c_float), C.c_int(cap), _p(count, C.c_int32), _p(idx, C.c_int32))
    return count, idx


COUNTERS = ("n_prop", "n_scan", "n_window", "n_children", "n_upd", "n_rows", "n_seed_layers", "n_ranked")


def kf_build(layers, bz, binned, seg_off, par, cov21, q, seed_event, seed_hit_idx, first_layer, K, chi2_cut, n_sigma,
          chi2_in=None, use_bins=True, n=None, margins=False, hit_mode=0):
    """kf_build_ref.  -> dict(par [6][n*K], cov [n*K][6][6], chi2, nhits, status [n*K], hit_idx [L][n*K], n_cand [n], counters
    [, margins [n][L][5]: smallest relative distance of the seed's decisions on that layer to the window edge, the chi2
    cut, a rank swap, the propagation / acceptance guards, a tangential crossing; 1e300 = none])"""
    layers = _lt(layers); L = layers.shape[0]
    par = _d(par); ld = par.shape[1]
    n = len(q) if n is None else n
    cov = _unpack21(_d(cov21))
    q = np.ascontiguousarray(q, dtype=np.int8)
    seg_off = np.ascontiguousarray(seg_off, dtype=np.int64)
    se = None if seed_event is None else _i(seed_event)
    sh = None if seed_hit_idx is None else _i(seed_hit_idx)
    if sh is not None:
        assert sh.shape == (first_layer, ld)
    ci = None if chi2_in is None else _d(chi2_in)
    ldo = max(n * K, 1)
    po = np.zeros((6, ldo)); co = np.zeros((36, ldo)); c2 = np.zeros(ldo); nh = np.zeros(ldo, np.int32); st = np.zeros(ldo, np.uint32)
    hi = np.zeros((L, ldo), np.int32); nc = np.zeros(max(n, 1), np.int32); cnt = np.zeros(8, np.int64)
    mg = np.full((max(n, 1), L, 5), 1e300) if margins else None
    l = lib(); l.kfo_build.restype = C.c_int
    rc = l.kfo_build(C.c_int(L), _p(layers), C.c_double(bz), C.c_int(binned["n_phi"]), C.c_int(binned["n_z"]),
                     _p(binned["x"], C.c_float), _p(binned["y"], C.c_float), _p(binned["z"], C.c_float), _p(binned["perm"], C.c_int32),
                     _p(binned["bin_off"], C.c_int32), _p(seg_off, C.c_int64), C.c_int64(n), C.c_int64(ld), _p(par), _p(cov), _p(q, C.c_int8),
                     _p(ci), _p(se, C.c_int32), _p(sh, C.c_int32), C.c_int(first_layer), C.c_int(K), C.c_double(chi2_cut), C.c_double(n_sigma),
                     C.c_int(1 if use_bins else 0), C.c_int(hit_mode), C.c_int64(ldo), _p(po), _p(co), _p(c2), _p(nh, C.c_int32), _p(st, C.c_uint32),
                     _p(hi, C.c_int32), _p(nc, C.c_int32), _p(cnt, C.c_int64), _p(mg))
    assert rc == 0, rc
    m = n * K
    extra = dict(margins=mg[:n]) if margins else {}
    return dict(**extra, par=po[:, :m], cov=co[:, :m].T.reshape(m, 6, 6), chi2=c2[:m], nhits=nh[:m], status=st[:m], hit_idx=hi[:, :m], n_cand=nc[:n],
                counters=dict(zip(COUNTERS, (int(v) for v in cnt))))


# ---------------------------------------------------------------------------------------------------------
# layout micro-benchmark (sec. 4.3, Fig. 5): n independent 6x6 products, the plain definition
# ---------------------------------------------------------------------------------------------------------
def mat66_multiply(A, B):
    """C_i = A_i B_i, A and B [n][6][6] (any float dtype) -> [n][6][6] float64; C_i[r][c] = sum_k A_i[r][k] B_i[k][c]."""
    A = np.asarray(A, dtype=np.float64); B = np.asarray(B, dtype=np.float64)
    assert A.shape == B.shape and A.shape[1:] == (6, 6)
    return np.matmul(A, B)

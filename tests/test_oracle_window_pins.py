"""Pins of the search-window widths INSIDE kfo_build (R11 var_phi, R22 var_rho, R23 widening; SURVEY.md sec. 8c-7,
reading A11; sec. 4.1 for the two-step case) that do not retype the oracle's formulas.

The width kfo_build actually uses is MEASURED from outside: every probe seed gets an event of its own holding a single hit on
the layer under test; with K = 1 and no chi2 cut to speak of the hit is picked exactly when it lies inside the window, so a
bisection on the hit's offset from the predicted crossing finds the window edge (the offset is read back from the fp32
coordinates the oracle saw).  The edge is then compared with quantities that come from somewhere else:
  W1  the variance of the predicted azimuth / radius as g^T C g with g the CENTRAL FINITE DIFFERENCE of atan2(y, x) /
      hypot(x, y) -- no closed-form gradient is typed here;
  W2  the same as the sample variance of 2e5 Gaussian draws of the predicted position (what "n_sigma standard deviations of
      the prediction" means), to 1.5 %;
  W3  the R23 widening as the shift of the SIMULATOR's helix crossing (synth.cross_cylinder / cross_plane: circle-circle
      geometry, none of the oracle's code) when the surface is displaced by +-d along its normal.
The predicted state itself comes from kfo_predict, which has its own pins (tests/test_oracle_pins.py P1-P4).
A factor 2, r^2 for r^4, a wrong sign of the x-y cross term or a dropped hit-resolution term in kf_oracle.c fails W1;
a window that means something else than standard deviations fails W2; a wrong incidence / dip factor fails W3.
"""
import numpy as np

from oracle import kf_oracle as o
from paper_1711_06571_b200 import synth

N_SIGMA = 3.0
BIG_CUT = 1e30


def probe_seeds(config, n, first_layer, seed=3):
    """n seed states of the synthetic build inputs with a FULL (correlated) covariance: the recipe's diagonal one rotated by a
    random correlation matrix, so that every cross term of the window formula matters."""
    bi = synth.build_inputs(config, n_events=1, tracks=max(4 * n, 64), first_layer=first_layer)
    rng = np.random.default_rng(seed)
    n = min(n, bi.n_seeds)
    par = bi.par[:, :n].astype(np.float64)
    covs = []
    for s in range(n):
        d = np.sqrt(np.diag(synth.unpack_sym(bi.cov[:, s].astype(np.float64))))
        a = rng.normal(size=(6, 6))
        corr = a @ a.T + 6.0 * np.eye(6)
        corr /= np.sqrt(np.outer(np.diag(corr), np.diag(corr)))
        covs.append(corr * np.outer(d, d))
    return bi, par, np.array(covs), bi.q[:n].astype(np.int8)


def predicted(lt, l, bz, par, covs, q):
    out = [o.predict(lt, l, bz, par[:, s], covs[s], q[s]) for s in range(par.shape[1])]
    ok = np.array([f == 0 for f, _, _ in out])
    return ok, np.array([p for _, p, _ in out]), np.array([c for _, _, c in out])


def picked(lt, bz, l, par, covs, q, hx, hy, hz, hit_mode):
    """one kfo_build call: seed s lives in event s, whose only hit is (hx, hy, hz)[s] on layer l -> was it picked?"""
    n, L = par.shape[1], lt.shape[0]
    ld = par.shape[1]
    seg_off = np.zeros(n * L + 1, np.int64)
    for e in range(n):
        seg_off[e * L + l + 1:] += 1
    x, y, z = (np.asarray(a, np.float32) for a in (hx, hy, hz))
    binned = dict(n_phi=8, n_z=1, x=x, y=y, z=z, perm=np.zeros(n, np.int32), bin_off=np.zeros(n * L * 8 + 1, np.int32))
    cov21 = np.stack([synth.pack_sym(c) for c in covs], axis=1)
    r = o.kf_build(lt, bz, binned, seg_off, par, cov21, q, np.arange(n, dtype=np.int32), None, l, 1, BIG_CUT, N_SIGMA,
                   use_bins=False, n=n, hit_mode=hit_mode)
    assert ld == n
    return r["hit_idx"][l, :n] >= 0


def window_edge(lt, bz, l, par, covs, q, pp, place, offset_of, hi0, hit_mode=0, side=+1.0):
    """bisection per seed on the offset t in [0, hi0]: place(t) -> hit coordinates; offset_of(x32, y32, z32) -> the offset the
    oracle saw.  Returns the largest offset found inside and the smallest found outside."""
    n = par.shape[1]
    lo, hi = np.zeros(n), np.full(n, hi0)
    inside0 = picked(lt, bz, l, par, covs, q, *place(lo * side), hit_mode)
    outside0 = ~picked(lt, bz, l, par, covs, q, *place(hi * side), hit_mode)
    assert inside0.all() and outside0.all(), (inside0, outside0)
    in_off, out_off = np.zeros(n), np.full(n, np.inf)
    for _ in range(44):
        mid = 0.5 * (lo + hi)
        hx, hy, hz = place(mid * side)
        got = picked(lt, bz, l, par, covs, q, hx, hy, hz, hit_mode)
        seen = offset_of(np.float32(hx).astype(np.float64), np.float32(hy).astype(np.float64), np.float32(hz).astype(np.float64))
        in_off = np.where(got, np.maximum(in_off, seen), in_off)
        out_off = np.where(~got, np.minimum(out_off, seen), out_off)
        lo = np.where(got, mid, lo); hi = np.where(got, hi, mid)
    assert (in_off <= out_off).all()
    return in_off, out_off


def fd_variance(f, x, y, cxy):
    """g^T C g with g the central finite difference of f(x, y)"""
    h = 1e-6 * np.hypot(x, y)
    g = np.array([(f(x + h, y) - f(x - h, y)) / (2 * h), (f(x, y + h) - f(x, y - h)) / (2 * h)])
    return np.einsum("in,ijn,jn->n", g, cxy, g)


def xy_block(Cp):
    return np.array([[Cp[:, 0, 0], Cp[:, 0, 1]], [Cp[:, 1, 0], Cp[:, 1, 1]]])


def measure_barrel(lt, bz, l, par, covs, q, pp, hit_mode=0):
    """(sin of the azimuthal half-width, z half-width) of the window on barrel layer l, each as (inside, outside) brackets"""
    rp, ap = np.hypot(pp[:, 0], pp[:, 1]), np.arctan2(pp[:, 1], pp[:, 0])
    sin_off = lambda x, y, z: np.abs(pp[:, 0] * y - pp[:, 1] * x) / (rp * np.hypot(x, y))      # R11: the window test is on sin(d phi)
    e_phi = window_edge(lt, bz, l, par, covs, q, pp, lambda t: (rp * np.cos(ap + t), rp * np.sin(ap + t), pp[:, 2]), sin_off, 0.7, hit_mode)
    e_z = window_edge(lt, bz, l, par, covs, q, pp, lambda t: (pp[:, 0], pp[:, 1], pp[:, 2] + t), lambda x, y, z: np.abs(z - pp[:, 2]), 60.0, hit_mode)
    return e_phi, e_z


def measure_disk(lt, bz, l, par, covs, q, pp, hit_mode=0):
    rp, ap, Z = np.hypot(pp[:, 0], pp[:, 1]), np.arctan2(pp[:, 1], pp[:, 0]), pp[:, 2]
    sin_off = lambda x, y, z: np.abs(pp[:, 0] * y - pp[:, 1] * x) / (rp * np.hypot(x, y))
    e_phi = window_edge(lt, bz, l, par, covs, q, pp, lambda t: (rp * np.cos(ap + t), rp * np.sin(ap + t), Z), sin_off, 0.7, hit_mode)
    e_rho = window_edge(lt, bz, l, par, covs, q, pp, lambda t: ((rp + t) * np.cos(ap), (rp + t) * np.sin(ap), Z),
                        lambda x, y, z: np.abs(np.hypot(x, y) - rp), 40.0, hit_mode)
    return e_phi, e_rho


def assert_edge(bracket, expected, rel, abs_):
    lo, hi = bracket
    tol = rel * expected + abs_
    assert (lo <= expected + tol).all() and (hi >= expected - tol).all(), (np.max(lo - expected), np.max(expected - hi), expected[:4])
    assert ((hi - lo) <= 4 * tol).all()          # the bracket closed: the measurement resolves the edge


def test_W1_W2_barrel_window_is_n_sigma_of_predicted_azimuth_and_z():
    """R11 on a cylinder, hit_mode 0: half-widths = n_sigma sqrt(var of the predicted coordinate + hit resolution^2)."""
    l = 3
    bi, par, covs, q = probe_seeds(3, 48, first_layer=l)
    lt, bz = bi.geom.layer_table(), bi.geom.bz
    ok, pp, Cp = predicted(lt, l, bz, par, covs, q)
    assert ok.all()
    R, _, _, srphi, sz, _ = lt[l][:6]
    e_phi, e_z = measure_barrel(lt, bz, l, par, covs, q, pp)
    var_phi = fd_variance(az_xy, pp[:, 0], pp[:, 1], xy_block(Cp))                                 # W1
    assert_edge(e_phi, N_SIGMA * np.sqrt(var_phi + (srphi / R) ** 2), 1e-5, 1e-8)
    assert_edge(e_z, N_SIGMA * np.sqrt(Cp[:, 2, 2] + sz ** 2), 1e-5, 2e-5)
    # the correlated covariance makes the cross term count: without it the width would be off by far more than the tolerance
    no_cross = N_SIGMA * np.sqrt(fd_variance(az_xy, pp[:, 0], pp[:, 1], xy_block(Cp) * np.eye(2)[:, :, None]) + (srphi / R) ** 2)
    assert np.median(np.abs(no_cross / (0.5 * (e_phi[0] + e_phi[1])) - 1)) > 1e-3
    # W2: sample variance of the azimuth / z of Gaussian draws of the predicted position
    rng = np.random.default_rng(11)
    for s in range(4):
        w, v = np.linalg.eigh(Cp[s][:3, :3])
        draws = pp[s, :3] + (rng.normal(size=(200_000, 3)) * np.sqrt(np.maximum(w, 0))) @ v.T
        d_az = np.angle(np.exp(1j * (np.arctan2(draws[:, 1], draws[:, 0]) - np.arctan2(pp[s, 1], pp[s, 0]))))
        mc_phi = N_SIGMA * np.sqrt(d_az.var() + (srphi / R) ** 2)
        mc_z = N_SIGMA * np.sqrt(draws[:, 2].var() + sz ** 2)
        assert abs(mc_phi / e_phi[0][s] - 1) < 0.015 and abs(mc_z / e_z[0][s] - 1) < 0.015, (s, mc_phi, e_phi[0][s], mc_z, e_z[0][s])


def az_xy(x, y):
    return np.arctan2(y, x)


def disk_probes(hit_mode_jitter=0.0, n=64):
    """forward seeds (state on barrel layer 2) taken straight to the first disk they cross inside its annulus"""
    bi = synth.build_inputs("lids", n_events=1, tracks=600, jitter=hit_mode_jitter)
    rng = np.random.default_rng(5)
    lt, bz = bi.geom.layer_table(), bi.geom.bz
    out = {}
    for l in range(lt.shape[0]):
        if lt[l][6] == 0:
            continue
        sel = []
        for s in range(bi.n_seeds):
            f, p1, _ = o.predict(lt, l, bz, bi.par[:, s].astype(np.float64), synth.unpack_sym(bi.cov[:, s].astype(np.float64)), bi.q[s])
            rho = np.hypot(p1[0], p1[1])
            if f == 0 and lt[l][7] + 3.0 < rho < lt[l][1] - 3.0:
                sel.append(s)
            if len(sel) == n:
                break
        if len(sel) >= 8:
            out[l] = np.array(sel)
    return bi, lt, bz, out, rng


def full_cov(bi, sel, rng):
    covs = []
    for s in sel:
        d = np.sqrt(np.diag(synth.unpack_sym(bi.cov[:, s].astype(np.float64))))
        a = rng.normal(size=(6, 6))
        corr = a @ a.T + 6.0 * np.eye(6)
        corr /= np.sqrt(np.outer(np.diag(corr), np.diag(corr)))
        covs.append(corr * np.outer(d, d))
    return np.array(covs)


def test_W1_W2_disk_window_is_n_sigma_of_predicted_azimuth_and_radius():
    """R22: on a disk the window is in azimuth and radius."""
    bi, lt, bz, probes, rng = disk_probes()
    assert len(probes) >= 2
    for l, sel in list(probes.items())[:2]:
        par, q = bi.par[:, sel].astype(np.float64), bi.q[sel].astype(np.int8)
        covs = full_cov(bi, sel, rng)
        ok, pp, Cp = predicted(lt, l, bz, par, covs, q)
        keep = ok & (np.hypot(pp[:, 0], pp[:, 1]) > lt[l][7] + 2.0) & (np.hypot(pp[:, 0], pp[:, 1]) < lt[l][1] - 2.0)
        par, q, covs, pp, Cp = par[:, keep], q[keep], covs[keep], pp[keep], Cp[keep]
        assert keep.sum() >= 8
        srphi, sr = lt[l][3], lt[l][5]
        rho = np.hypot(pp[:, 0], pp[:, 1])
        e_phi, e_rho = measure_disk(lt, bz, l, par, covs, q, pp)
        var_phi = fd_variance(az_xy, pp[:, 0], pp[:, 1], xy_block(Cp))
        var_rho = fd_variance(np.hypot, pp[:, 0], pp[:, 1], xy_block(Cp))
        assert_edge(e_phi, N_SIGMA * np.sqrt(var_phi + (srphi / rho) ** 2), 1e-5, 1e-8)
        assert_edge(e_rho, N_SIGMA * np.sqrt(var_rho + sr ** 2), 1e-5, 2e-5)
        w, v = np.linalg.eigh(Cp[0][:3, :3])
        draws = pp[0, :3] + (np.random.default_rng(2).normal(size=(200_000, 3)) * np.sqrt(np.maximum(w, 0))) @ v.T
        mc_rho = N_SIGMA * np.sqrt(np.hypot(draws[:, 0], draws[:, 1]).var() + sr ** 2)
        assert abs(mc_rho / e_rho[0][0] - 1) < 0.015


def test_W3_two_step_widening_is_the_shift_of_the_crossing_on_a_displaced_surface():
    """R23 (hit_mode 1): the window grows, in quadrature, by n_sigma x (r.m.s. sensor displacement along the normal) x (shift of
    the crossing point per unit displacement of the surface).  That shift is taken from the simulator's helix on surfaces
    displaced by +-d; the widening is what kfo_build uses with hit_mode 1 minus what it uses with hit_mode 0."""
    d = 1e-3
    # cylinder: sensors displaced radially by sig_r
    l = 3
    bi, par, covs, q = probe_seeds(3, 32, first_layer=l, seed=9)
    lt, bz = bi.geom.layer_table().copy(), bi.geom.bz
    lt[:, 5] = 0.25                                        # sig_r = r.m.s. displacement of the sensors (R23)
    ok, pp, Cp = predicted(lt, l, bz, par, covs, q)
    assert ok.all()
    R = lt[l][0]
    (p0, z0), (p1, z1) = measure_barrel(lt, bz, l, par, covs, q, pp, 0), measure_barrel(lt, bz, l, par, covs, q, pp, 1)
    wz = np.sqrt(np.maximum((0.5 * (z1[0] + z1[1])) ** 2 - (0.5 * (z0[0] + z0[1])) ** 2, 0)) / N_SIGMA
    wphi = np.sqrt(np.maximum((0.5 * (p1[0] + p1[1])) ** 2 - (0.5 * (p0[0] + p0[1])) ** 2, 0)) / N_SIGMA
    args = (par[0], par[1], par[2], par[3], par[4], par[5], q, bz)
    okp, xp, yp, zp, *_ = synth.cross_cylinder(*args, R + d)
    okm, xm, ym, zm, *_ = synth.cross_cylinder(*args, R - d)
    assert okp.all() and okm.all()
    shift_z = np.abs(zp - zm) / (2 * d)
    shift_phi = np.abs(np.angle(np.exp(1j * (np.arctan2(yp, xp) - np.arctan2(ym, xm))))) / (2 * d)
    assert np.allclose(wz, 0.25 * shift_z, rtol=2e-4, atol=1e-6), np.max(np.abs(wz / (0.25 * shift_z) - 1))
    # the azimuthal widening is a small difference in quadrature of two measured half-widths p ~ 5e-3 rad, each resolved to the
    # fp32 grid of the hit coordinates (ulp(16 cm) / 16 cm ~ 1e-7 rad): d(w) = p dp / (n_sigma^2 w) ~ 2e-6 at the smallest
    # w ~ 6e-5 here.  A factor 2 or cos for sin of the incidence angle is off by >= 6e-5.
    assert np.allclose(wphi, 0.25 * shift_phi, rtol=2e-3, atol=4e-6), np.max(np.abs(wphi - 0.25 * shift_phi))
    assert wphi.max() > 1e-3 and np.median(np.abs(wphi / (0.25 * shift_phi) - 1)) < 2e-3
    assert (wz > 1e-3).all()                                # the widening is there at all
    # disk: sensors displaced along z by sig_z; the transverse position moves by tan(theta) per unit z along the direction of
    # motion, split between radius and azimuth: the reading widens each by the whole of it ("at most")
    bi, lt, bz, probes, rng = disk_probes()
    lt = lt.copy(); lt[:, 4] = np.where(lt[:, 6] == 1, 0.25, lt[:, 4])
    l, sel = next(iter(probes.items()))
    sel = sel[:24]
    par, q = bi.par[:, sel].astype(np.float64), bi.q[sel].astype(np.int8)
    covs = full_cov(bi, sel, rng)
    ok, pp, Cp = predicted(lt, l, bz, par, covs, q)
    assert ok.all()
    (p0, r0), (p1, r1) = measure_disk(lt, bz, l, par, covs, q, pp, 0), measure_disk(lt, bz, l, par, covs, q, pp, 1)
    wrho = np.sqrt(np.maximum((0.5 * (r1[0] + r1[1])) ** 2 - (0.5 * (r0[0] + r0[1])) ** 2, 0)) / N_SIGMA
    wphi = np.sqrt(np.maximum((0.5 * (p1[0] + p1[1])) ** 2 - (0.5 * (p0[0] + p0[1])) ** 2, 0)) / N_SIGMA
    Z = lt[l][0]
    args = (par[0], par[1], par[2], par[3], par[4], par[5], q, bz)
    okp, xp, yp, *_ = synth.cross_plane(*args, Z + d * np.sign(Z))
    okm, xm, ym, *_ = synth.cross_plane(*args, Z - d * np.sign(Z))
    assert okp.all() and okm.all()
    shift_xy = np.hypot(xp - xm, yp - ym) / (2 * d)
    shift_rho = np.abs(np.hypot(xp, yp) - np.hypot(xm, ym)) / (2 * d)
    rho = np.hypot(pp[:, 0], pp[:, 1])
    assert np.allclose(wrho, 0.25 * shift_xy, rtol=2e-4, atol=1e-6), np.max(np.abs(wrho / (0.25 * shift_xy) - 1))
    assert np.allclose(wphi, 0.25 * shift_xy / rho, rtol=2e-3, atol=4e-6), np.max(np.abs(wphi - 0.25 * shift_xy / rho))
    assert (shift_rho <= shift_xy * (1 + 1e-9)).all()       # "at most": the radial part alone is never larger

"""Pins of the oracle's "cylinder with lids" pieces (sec. 4.1; R19-R21):
propagation to an endcap disk, the second propagation step to a hit's own radius / z, and the 2-D Kalman update on the
plane tangent to the hit radius.  CPU only; pinned to the simulator's independent plane crossing, finite differences, the
group property of the transport, plain numpy normal equations, textbook straight-line least squares and pull statistics."""
import numpy as np
import pytest

from oracle import kf_oracle as o
from paper_1711_06571_b200 import synth
from tests.test_oracle_pins import GOLD, K


def rand_forward_state(rng):
    r0, a = rng.uniform(0, 30), rng.uniform(-np.pi, np.pi)
    pt = np.exp(rng.uniform(np.log(0.4), np.log(50)))
    theta = rng.uniform(0.15, 1.2)
    if rng.random() < 0.5:
        theta = np.pi - theta
    return np.array([r0 * np.cos(a), r0 * np.sin(a), rng.uniform(-20, 20), 1 / pt, rng.uniform(-np.pi, np.pi), theta])


def test_L1_propagate_z_vs_plane_crossing():
    """Oracle vs the simulator's turn-about-the-centre plane crossing.  The disk must lie ahead (s > 0) and within half a
    turn; z' = Z exactly; cos(incidence) = |cos theta|.  Catches: sign of s, wrong rotation sense, wrong side accepted."""
    rng = np.random.default_rng(31)
    n_ok = n_bad = 0
    for _ in range(2000):
        p = rand_forward_state(rng)
        q, bz = rng.choice([-1, 1]), rng.choice([3.8, -3.8, 0.0])
        Z = rng.choice([-1, 1]) * rng.uniform(30, 110)
        ok, xs, ys, zs, ph, s, ci = synth.cross_plane(p[0], p[1], p[2], p[3], p[4], p[5], q, bz, Z)
        f, po, J, s_o, ci_o = o.propagate_z(p, q, bz, Z)
        if not ok:
            n_bad += 1
            assert f == o.UNREACHABLE
            continue
        n_ok += 1
        assert f == (o.GRAZING if abs(np.cos(p[5])) < 0.1 else 0)
        assert po[2] == Z and abs(s_o - s) < 1e-10 * max(1, s) and abs(ci_o - abs(np.cos(p[5]))) < 1e-15
        assert abs(po[0] - xs) < 1e-9 and abs(po[1] - ys) < 1e-9 and abs(po[4] - ph) < 1e-11
        assert po[3] == p[3] and po[5] == p[5]
    assert n_ok > 500 and n_bad > 500


def test_L2_disk_jacobian_vs_finite_differences():
    """d p'/d p of the transport TO THE PLANE (path-length term from s = (Z - z) tan theta) vs central differences;
    the z' row vanishes.  Catches: dropped ds/dz or ds/dtheta terms, wrong curvature column."""
    rng = np.random.default_rng(32)
    worst = 0.0
    n = 0
    for _ in range(300):
        p = rand_forward_state(rng)
        q, bz = rng.choice([-1, 1]), rng.choice([3.8, -3.8, 0.0])
        Z = np.sign(np.cos(p[5])) * rng.uniform(40, 110)
        f, po, J, s, ci = o.propagate_z(p, q, bz, Z)
        if f or abs(K * bz * p[3]) * s > 2.0:
            continue
        errs = []
        for hs in (1e-4, 1e-5):
            Jn = np.zeros((6, 6))
            for k in range(6):
                h = hs * max(1.0, abs(p[k]))
                pp, pm = p.copy(), p.copy()
                pp[k] += h; pm[k] -= h
                Jn[:, k] = (o.propagate_z(pp, q, bz, Z)[1] - o.propagate_z(pm, q, bz, Z)[1]) / (2 * h)
            scale = np.maximum(np.abs(Jn), 1e-3 * np.abs(Jn).max(axis=1, keepdims=True) + 1e-9)
            errs.append(np.max(np.abs(J - Jn) / scale))
        worst = max(worst, min(errs))
        assert not J[2].any() and np.array_equal(J[3], [0, 0, 0, 1, 0, 0]) and np.array_equal(J[5], [0, 0, 0, 0, 0, 1])
        n += 1
    assert n > 100 and worst < 2e-6, worst


def test_L3_second_step_composes_with_the_first():
    """Two-step propagation (R20): to the nominal radius R1 and then on to a hit radius R2 a little outside OR inside it
    (backwards) lands where the direct transport to R2 lands, and the Jacobians compose, J2 J1 = J12.  The same for
    disks: to Z1, then on / back to Z2.  Catches: a second step that cannot go backwards, a Jacobian that is not the
    surface-to-surface map."""
    rng = np.random.default_rng(33)
    n = 0
    for _ in range(400):
        p = rand_forward_state(rng)
        p[:2] *= 0.3
        q, bz = rng.choice([-1, 1]), 3.8
        R1 = rng.uniform(15, 45); R2 = R1 + rng.uniform(-0.5, 0.5)
        f1, p1, J1, _, ci = o.propagate(p, q, bz, R1)
        f12, p12, J12, _, _ = o.propagate(p, q, bz, R2)
        if f1 or f12 or ci < 0.3:
            continue
        f2, p2, J2, s2 = o.propagate_near(p1, q, bz, R2)
        assert f2 == 0 and (s2 > 0) == (R2 > R1)
        assert np.max(np.abs(p2 - p12)) < 1e-10 and np.max(np.abs(J2 @ J1 - J12)) < 1e-8 * np.abs(J12).max()
        Z1 = np.sign(np.cos(p[5])) * rng.uniform(50, 100); Z2 = Z1 + rng.uniform(-0.5, 0.5)
        g1, q1, K1, _, _ = o.propagate_z(p, q, bz, Z1)
        g12, q12, K12, _, _ = o.propagate_z(p, q, bz, Z2)
        if g1 or g12:
            continue
        g2, q2, K2, t2, _ = o.propagate_z(q1, q, bz, Z2, forward_only=False)
        assert g2 == 0 and np.max(np.abs(q2 - q12)) < 1e-9 and np.max(np.abs(K2 @ K1 - K12)) < 1e-8 * np.abs(K12).max()
        n += 1
    assert n > 100


def test_L4_tangent_plane_update():
    """(a) update_2d == the normal-equation solution of the same linear problem in plain numpy (information form), for
    barrel (r-phi, z) and disk (r-phi, r) hits.  (b) With the hit on the nominal radius at the predicted azimuth, displaced
    in z only, the 2-D update equals the 3-D update of R5 exactly (the radial direction carries no information: C n = 0);
    with a small r-phi displacement they agree to second order in it.  Catches: wrong measurement axes, gain or Joseph form."""
    rng = np.random.default_rng(34)
    for kind in (0, 1):
        for _ in range(50):
            A = rng.normal(size=(6, 6)); Cm = A @ A.T * 1e-3 + np.eye(6) * 1e-6
            p = np.array([20.0, 5.0, 30.0, 0.5, 0.2, 1.0]) + rng.normal(size=6) * 0.01
            p[3] = 0.5
            m = p[:3] + rng.normal(size=3) * 0.02
            s1, s2 = 0.01, 0.1 if kind == 0 else 0.02
            f, pu, Cu, c2 = o.update_2d(p, Cm, m, kind, s1, s2)
            rm = np.hypot(m[0], m[1])
            u1 = np.array([-m[1], m[0], 0]) / rm
            u2 = np.array([0, 0, 1.0]) if kind == 0 else np.array([m[0], m[1], 0]) / rm
            H = np.zeros((2, 6)); H[0, :3] = u1; H[1, :3] = u2
            Vi = np.diag([1 / s1 ** 2, 1 / s2 ** 2])
            info = np.linalg.inv(Cm) + H.T @ Vi @ H
            Cn = np.linalg.inv(info)
            pn = p + Cn @ H.T @ Vi @ (H @ np.concatenate([m - p[:3], np.zeros(3)]))
            r = H[:, :3] @ (m - p[:3])
            S = H @ Cm @ H.T + np.diag([s1 ** 2, s2 ** 2])
            assert f == 0 and np.max(np.abs(pu - pn)) < 1e-8 and np.max(np.abs(Cu - Cn)) < 1e-8 * np.abs(Cn).max()
            assert abs(c2 - r @ np.linalg.solve(S, r)) < 1e-9 * max(1, c2)
            assert o.chi2_2d(p, Cm, m, kind, s1, s2) == (0, pytest.approx(c2, rel=1e-12))
    # (b)
    g = synth.geometry("barrel10")
    lt = g.layer_table()
    p0 = np.array([0.01, -0.02, 0.3, 0.8, 0.4, 1.1])
    C0 = np.diag(np.array([0.05, 0.05, 0.05, 0.04, 0.005, 0.005]) ** 2)
    f, pp, Cp = o.predict(lt, 5, g.bz, p0, C0, 1)
    assert f == 0
    m = pp[:3] + np.array([0, 0, 0.07])
    f3, p3, C3, c3 = o.update(pp, Cp, m, 0.01, 0.1, 0.01)
    f2, p2, C2, c2 = o.update_2d(pp, Cp, m, 0, 0.01, 0.1)
    assert f3 == 0 and f2 == 0
    assert np.max(np.abs(p3 - p2)) < 1e-12 and np.max(np.abs(C3 - C2)) < 1e-12 * np.abs(C3).max() and abs(c3 - c2) < 1e-10
    az = np.arctan2(pp[1], pp[0]) + 5e-4
    m = np.array([24.0 * np.cos(az), 24.0 * np.sin(az), pp[2] + 0.07])       # on the nominal cylinder, 0.012 cm along r-phi
    f3, p3, C3, c3 = o.update(pp, Cp, m, 0.01, 0.1, 0.01)
    fs, ps, Cs = o.to_hit_surface(0, g.bz, 1, pp, Cp, m)
    f2, p2, C2, c2 = o.update_2d(ps, Cs, m, 0, 0.01, 0.1)
    assert fs == 0 and np.max(np.abs(ps - pp)) < 1e-9                          # the second step is the identity here
    assert np.max(np.abs(p3 - p2) / np.maximum(np.abs(p3), 1e-3)) < 1e-5 and abs(c3 - c2) < 1e-4 * c3


def _run_lids(fi, hit_mode=1):
    return o.fit(fi.geom.layer_table(), fi.geom.bz, fi.par, fi.cov, fi.q, fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off, fi.hit_idx, hit_mode=hit_mode)


def test_L5_noise_free_truth_recovery_on_the_cylinder_with_lids():
    """Exact hits on staggered sensors (+-0.3 cm about the nominal surfaces), no scattering, seed = truth: every
    residual vanishes and the state ends on the last hit's own surface as the simulator's truth state.  Catches: wrong
    plane crossing, second step to the wrong surface, disks of the wrong side touched."""
    fi = synth.fit_inputs("lids", n=3000, ms=False, smear=False)
    vtx = np.stack([fi.gun[k] for k in ("x", "y", "z", "ipt", "phi", "theta")], axis=0)
    fi.par = fi.par.astype(np.float64)
    fi.par[:, :fi.n] = vtx                     # the exact truth at the vertex as the seed
    r = _run_lids(fi)
    nh = fi.valid.sum(axis=0)
    assert (r["status"] == 0).mean() > 0.995 and (nh[r["status"] == 0] == r["nhits"][r["status"] == 0]).all()
    ok = (r["status"] == 0) & (nh > 0)
    assert r["chi2"][ok].max() < 1e-4          # hits are rounded to fp32 (3e-6 cm at 50 cm against 0.01 cm)
    last = np.where(fi.valid, np.arange(fi.geom.n_layers)[:, None], -1).max(axis=0)
    tr = fi.truth[last[ok], np.nonzero(ok)[0]]
    d = r["par"][:, ok].T - tr
    d[:, 4] = np.angle(np.exp(1j * d[:, 4]))
    assert np.abs(d[:, :3]).max() < 2e-4 and np.abs(d[:, 3:]).max() < 2e-5
    assert (fi.valid[10:].any(axis=0)).mean() > 0.3 and (fi.valid[:10].any(axis=0) & fi.valid[10:].any(axis=0)).mean() > 0.15   # lids and transition used


def test_L6_straight_line_through_disks_closed_form():
    """B = 0, no scattering, four disks, polar angle 0.35 rad, diffuse prior: the KF covariance is the textbook straight-line
    weighted least squares -- r-phi against the hit radius (slope = azimuth), r against z (slope = tan theta).
    Values: tests/golden/closed_forms.txt (disk_*).  Catches: wrong measurement model on the disk (r-phi / r axes), lever arms."""
    g = synth.geometry("lids10", bz=0.0, xx0_scale=0.0)
    lt = g.layer_table()[10:14]
    th, ph = 0.35, 0.3
    zk = lt[:, 0]
    rk = zk * np.tan(th)
    hits = np.stack([rk * np.cos(ph), rk * np.sin(ph), zk], axis=1)
    par = np.zeros((6, 1)); par[:, 0] = [0, 0, 0, 0.5, ph, th]
    cov = np.zeros((21, 1))
    for i, sg in enumerate([1, 1, 10, 0.05, 0.1, 0.1]):
        cov[synth.pack_index(i, i), 0] = sg ** 2
    r = o.fit(lt, 0.0, par, cov, np.array([1], np.int8), hits[:, 0], hits[:, 1], hits[:, 2], np.arange(5), hit_mode=1)
    C = r["cov"][0]
    t = np.array([-np.sin(ph), np.cos(ph), 0.0]); n = np.array([np.cos(ph), np.sin(ph), 0.0])
    rel = lambda a, b: abs(a - b) / b
    assert r["nhits"][0] == 4 and abs(r["chi2"][0]) < 1e-18
    assert rel(np.sqrt(C[4, 4]), GOLD["disk_sigma_phi"]) < 3e-3
    assert rel(np.sqrt(t @ C[:3, :3] @ t), GOLD["disk_sigma_rphi_last"]) < 3e-3
    assert rel(np.sqrt(C[5, 5]), GOLD["disk_sigma_theta"]) < 3e-3
    assert rel(np.sqrt(n @ C[:3, :3] @ n), GOLD["disk_sigma_r_last"]) < 3e-3
    assert C[2, 2] < 1e-20 and rel(np.sqrt(C[3, 3]), 0.05) < 1e-9       # on the plane; curvature unobservable at B = 0


def _pulls_lids(fi, r):
    L = fi.geom.n_layers
    last = np.where(fi.valid, np.arange(L)[:, None], -1).max(axis=0)
    sel = (r["status"] == 0) & (last >= 0) & (r["nhits"] == fi.valid.sum(axis=0)) & (r["nhits"] >= 3)
    idx = np.nonzero(sel)[0]
    tr = fi.truth[last[idx], idx]
    p = r["par"][:, idx].T; C = r["cov"][idx]
    rr = np.hypot(tr[:, 0], tr[:, 1])
    disk = fi.geom.kind[last[idx]] != 0
    T = np.zeros((len(idx), 5, 6))
    T[:, 0, 0] = -tr[:, 1] / rr; T[:, 0, 1] = tr[:, 0] / rr
    T[:, 1, 2] = np.where(disk, 0.0, 1.0); T[:, 1, 0] = np.where(disk, tr[:, 0] / rr, 0.0); T[:, 1, 1] = np.where(disk, tr[:, 1] / rr, 0.0)
    T[:, 2, 3] = 1; T[:, 3, 4] = 1; T[:, 4, 5] = 1
    d = p - tr
    d[:, 4] = np.angle(np.exp(1j * d[:, 4]))
    dd = np.einsum("nij,nj->ni", T, d)
    var = np.einsum("nij,njk,nik->ni", T, C, T)
    return dd / np.sqrt(var), r["chi2"][idx], r["nhits"][idx], disk


def test_L7_pulls_on_the_cylinder_with_lids():
    """Statistics pin of R19-R21: smeared hits on staggered sensors, scattering, |eta| < 2.2 (barrel, both lids and the
    transition).  Pulls of (r-phi, z or r, 1/pT, phi, theta) at the last hit are unit, chi2 / (2 nhits) = 1, for tracks that
    end in the barrel and for tracks that end on a disk alike.  Catches: wrong disk scattering (path 1/|cos theta|), wrong
    r / r-phi resolution on disks, material added at the wrong place in the two-step scheme."""
    fi = synth.fit_inputs("lids", n=30000)
    r = _run_lids(fi)
    pulls, chi2, nh, disk = _pulls_lids(fi, r)
    assert len(chi2) > 0.85 * fi.n and disk.mean() > 0.25
    for sel in (disk, ~disk):
        pl = pulls[sel]
        assert (np.abs(pl) < 5).mean() > 0.999
        assert np.all(np.abs(pl.mean(axis=0)) < 0.04), pl.mean(axis=0)
        assert np.all(np.abs(pl.std(axis=0) - 1) < 0.04), pl.std(axis=0)
        assert abs((chi2[sel] / (2 * nh[sel])).mean() - 1) < 0.03
    # hit_mode 0 on the same (staggered) hits ignores the 0.3 cm offsets: the fit is visibly worse
    r0 = _run_lids(fi, hit_mode=0)
    ok = (r0["status"] == 0) & (r0["nhits"] >= 3)
    assert (r0["chi2"][ok] / (2 * r0["nhits"][ok])).mean() > 3

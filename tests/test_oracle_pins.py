"""Pins of the fp64 oracle (oracle/kf_oracle.c) to things other than itself.  CPU only.

The paper prints no worked example, so the pins are closed forms, invariants, special cases that
reduce to textbook results, finite differences and an independent simulator (pins P1-P11).
Each test names the mistake it would catch.
"""
import numpy as np
import pytest
from scipy import optimize, stats

from oracle import kf_oracle as o
from paper_1711_06571_b200 import synth

K = 0.00299792458
GOLD = {}
for line in open(__file__.rsplit("/", 1)[0] + "/golden/closed_forms.txt"):
    line = line.split("#")[0].strip()
    if line:
        k, v = line.split("=")
        GOLD[k.strip()] = float(v)


def rand_state(rng, rmax, wide=False):
    r0 = rng.uniform(0, rmax)
    a = rng.uniform(-np.pi, np.pi)
    pt = np.exp(rng.uniform(np.log(0.3), np.log(100))) if wide else rng.uniform(0.5, 10)
    phi = a + rng.uniform(-0.8, 0.8)  # roughly outward
    theta = 2 * np.arctan(np.exp(-rng.uniform(-1.5, 1.5)))
    return np.array([r0 * np.cos(a), r0 * np.sin(a), rng.uniform(-20, 20), 1 / pt, phi, theta])


# ------------------------------------------------------------------------------------------------ P1
@pytest.mark.parametrize("bz", [3.8, -3.8, 0.0, 1.0])
def test_P1_chord_from_origin(bz):
    """From the origin the helix-cylinder crossing is the textbook chord relation: alpha = 2 asin(R w / 2),
    s = alpha / w, azimuth of the crossing = phi + alpha/2, cos(incidence) = cos(alpha/2), z = s cot(theta).
    Catches: wrong sign of the curvature, wrong root, wrong z transport."""
    rng = np.random.default_rng(1)
    for _ in range(300):
        pt = np.exp(rng.uniform(np.log(0.3), np.log(1000)))
        phi, theta = rng.uniform(-np.pi, np.pi), rng.uniform(0.4, np.pi - 0.4)
        q = rng.choice([-1, 1])
        R = rng.uniform(2, 80)
        w = -q * K * bz / pt
        if abs(w) * R / 2 >= 1:
            f, *_ = o.propagate([0, 0, 0, 1 / pt, phi, theta], q, bz, R)
            assert f == o.UNREACHABLE
            continue
        alpha = 2 * np.arcsin(R * w / 2) if w != 0 else 0.0
        s = alpha / w if w != 0 else R
        f, po, J, s_o, ci = o.propagate([0, 0, 0, 1 / pt, phi, theta], q, bz, R)
        assert f in (0, o.GRAZING)
        assert abs(s_o - s) < 1e-11 * max(1, s)
        assert abs(po[0] - R * np.cos(phi + alpha / 2)) < 1e-11 and abs(po[1] - R * np.sin(phi + alpha / 2)) < 1e-11
        assert abs(po[2] - s / np.tan(theta)) < 1e-10
        assert abs(po[4] - (phi + alpha)) < 1e-12
        assert abs(ci - np.cos(alpha / 2)) < 1e-12
        assert (f == o.GRAZING) == (np.cos(alpha / 2) < 0.1)


def test_P1_printed_values():
    """q=+1, B=+3.8 T, phi0=0 from the origin to R=40 cm (values in tests/golden/closed_forms.txt are the chord
    closed form evaluated by hand-independent arithmetic, see the file)."""
    f, po, J, s, ci = o.propagate([0, 0, 0, 1.0, 0.0, np.pi / 2], 1, 3.8, 40.0)
    assert abs(s - GOLD["s_pt1_R40"]) < 1e-6 and abs(ci - GOLD["cosinc_pt1_R40"]) < 1e-6
    assert abs(po[4] - GOLD["phi_pt1_R40"]) < 1e-6 and abs(po[1] - GOLD["y_pt1_R40"]) < 1e-6
    f, po, J, s, ci = o.propagate([0, 0, 0, 1 / 0.3, 0.0, np.pi / 2], 1, 3.8, 40.0)
    assert abs(s - GOLD["s_pt03_R40"]) < 1e-6 and abs(ci - GOLD["cosinc_pt03_R40"]) < 1e-6
    # rho = pT / (k B): 1 GeV in 3.8 T
    assert abs(1 / (K * 3.8) - GOLD["rho_pt1_B38"]) < 1e-5


def test_P1_generic_start_vs_circle_geometry():
    """Oracle (march + Newton on the helix) vs the simulator's circle-circle intersection (law of cosines) for
    states anywhere inside the cylinder.  Catches: wrong handling of a non-zero start point, second root taken."""
    rng = np.random.default_rng(2)
    worst = 0.0
    for _ in range(2000):
        R = rng.uniform(5, 80)
        p = rand_state(rng, 0.97 * R, wide=True)
        q = rng.choice([-1, 1]); bz = rng.choice([3.8, -3.8, 2.0])
        ok, x, y, z, ph, s, ci = synth.cross_cylinder(p[0], p[1], p[2], p[3], p[4], p[5], q, bz, R)
        f, po, J, s_o, ci_o = o.propagate(p, q, bz, R)
        if not ok:
            assert f == o.UNREACHABLE
            continue
        assert f == (o.GRAZING if ci < 0.1 else 0)      # near-tangent double crossings included: none may be stepped over
        if ci < 1e-4:                                   # the root is then conditioned like 1/cos(incidence)
            continue
        worst = max(worst, abs(po[0] - x), abs(po[1] - y), abs(po[2] - z), abs(po[4] - ph), abs(s_o - s))
        assert abs(np.hypot(po[0], po[1]) - R) < 1e-11
    assert worst < 1e-8


# ------------------------------------------------------------------------------------------------ P2
def test_P2_jacobian_vs_finite_differences():
    """J includes the path-length term: compare with central differences of the propagate-to-R map itself.
    Catches: a dropped ds/dp term, wrong sign/index in any of the 20 non-zero entries, transposition."""
    rng = np.random.default_rng(3)
    worst = 0.0
    for _ in range(400):
        R = rng.uniform(5, 80)
        p = rand_state(rng, 0.9 * R, wide=True)
        q = rng.choice([-1, 1]); bz = rng.choice([3.8, -3.8, 0.0])
        f, po, J, s, ci = o.propagate(p, q, bz, R)
        if f or ci < 0.3:
            continue
        errs = []
        for hs in (1e-4, 1e-5):      # two step sizes: truncation error falls, round-off noise rises
            Jn = np.zeros((6, 6))
            for k in range(6):
                h = hs * max(1.0, abs(p[k]))
                pp, pm = p.copy(), p.copy()
                pp[k] += h; pm[k] -= h
                Jn[:, k] = (o.propagate(pp, q, bz, R)[1] - o.propagate(pm, q, bz, R)[1]) / (2 * h)
            scale = np.maximum(np.abs(Jn), 1e-3 * np.abs(Jn).max(axis=1, keepdims=True) + 1e-9)
            errs.append(np.max(np.abs(J - Jn) / scale))
        worst = max(worst, min(errs))
        # structure: rows iota and theta are unit rows; z, theta columns
        assert np.array_equal(J[3], [0, 0, 0, 1, 0, 0]) and np.array_equal(J[5], [0, 0, 0, 0, 0, 1])
        assert np.count_nonzero(J) <= 20
        # transported to the surface: the normal component of the position block vanishes
        n = np.array([po[0], po[1], 0]) / R
        assert np.max(np.abs(n @ J[0:3, :])) < 1e-9 * max(1, np.abs(J).max())
    assert worst < 2e-6


# ------------------------------------------------------------------------------------------------ P3
def test_P3_noise_free_truth_recovery():
    """Noise-free hits, no scattering, seed = truth: every residual vanishes, chi2 = 0 and the output is the
    simulator's truth state on the last layer.  Catches: any inconsistency between transport and hit model."""
    fi = synth.fit_inputs(0, n=500, ms=False, smear=False)
    g = fi.gun
    par = np.stack([g["x"], g["y"], g["z"], g["ipt"], g["phi"], g["theta"]])
    hits = np.nan_to_num(synth.simulate(fi.geom, g, synth.rng_for(99), ms=False, smear=False)["hits"])
    L, n = fi.geom.n_layers, fi.n
    hx, hy, hz = (hits[:, :, k].reshape(-1) for k in range(3))
    r = o.fit(fi.geom.layer_table(), fi.geom.bz, par, fi.cov[:, :n].astype(np.float64), fi.q, hx, hy, hz,
              np.arange(L + 1) * n)
    assert (r["status"] == 0).all() and (r["nhits"] == L).all()
    assert r["chi2"].max() < 1e-14
    tr = fi.truth[-1].copy()
    tr[:, 4] = np.angle(np.exp(1j * tr[:, 4]))
    assert np.max(np.abs(r["par"].T - tr)) < 1e-9


def test_P4_prior_weight_vanishes_with_hit_resolution():
    """Noise-free hits + a smeared seed: the fitted state approaches the truth as the hit resolution shrinks."""
    fi = synth.fit_inputs(0, n=200, ms=False, smear=False)
    tr = fi.truth[-1]
    errs = []
    for scale in (1.0, 0.1, 0.01):
        lt = fi.geom.layer_table(); lt[:, 3:6] *= scale
        r = o.fit(lt, fi.geom.bz, fi.par, fi.cov, fi.q, fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off)
        d = r["par"].T - tr
        d[:, 4] = np.angle(np.exp(1j * d[:, 4]))
        errs.append(np.abs(d[:, 3] / tr[:, 3]).mean())
    assert errs[0] > 3 * errs[1] > 9 * errs[2]


# ------------------------------------------------------------------------------------------------ P5 / P6
def _fit_single(layers, bz, p0, sig0, q, hits):
    L = layers.shape[0]
    par = np.zeros((6, 1)); par[:, 0] = p0
    cov = np.zeros((21, 1))
    for i in range(6):
        cov[synth.pack_index(i, i), 0] = sig0[i] ** 2
    r = o.fit(layers, bz, par, cov, np.array([q], dtype=np.int8), hits[:, 0], hits[:, 1], hits[:, 2], np.arange(L + 1))
    return r


def test_P5_straight_line_least_squares_closed_form():
    """B = 0, no scattering: the KF covariance after 10 equidistant layers R = 4..40 equals the weighted
    least-squares straight-line fit: sigma(phi) = s/sqrt(sum (R-Rbar)^2), sigma(r phi at 40) =
    s sqrt(1/10 + 18^2/1320), same in z with sigma_z, sigma(cot theta) likewise; 1/pT unobservable.
    Catches: wrong gain / covariance update, wrong hit covariance, wrong Jacobian lever arms."""
    geom = synth.geometry("barrel10", bz=0.0, xx0_scale=0.0)
    lt = geom.layer_table()
    phi0, th0 = 0.3, np.pi / 2
    R = geom.r
    hits = np.stack([R * np.cos(phi0), R * np.sin(phi0), np.zeros_like(R)], axis=1)
    sig0 = np.array([1, 1, 10, 0.05, 0.1, 0.1])
    r = _fit_single(lt, 0.0, [0, 0, 0, 0.5, phi0, th0], sig0, 1, hits)
    C = r["cov"][0]
    t = np.array([-np.sin(phi0), np.cos(phi0), 0.0])
    rel = lambda a, b: abs(a - b) / b
    assert rel(np.sqrt(C[4, 4]), GOLD["wls_sigma_phi"]) < 2e-4
    assert rel(np.sqrt(t @ C[:3, :3] @ t), GOLD["wls_sigma_rphi_40"]) < 2e-4
    assert rel(np.sqrt(C[2, 2]), GOLD["wls_sigma_z_40"]) < 2e-3
    assert rel(np.sqrt(C[5, 5]), GOLD["wls_sigma_cot"]) < 2e-3   # d cot = d theta at theta = pi/2
    assert rel(np.sqrt(C[3, 3]), 0.05) < 1e-9                     # curvature unobservable at B = 0
    assert abs(r["chi2"][0]) < 1e-18


def test_P5_state_equals_batch_least_squares():
    """B = 0: the KF state equals the batch solution of the normal equations (prior as pseudo-measurement) up to
    O(eps^2) in the smearing scale eps -- checked by shrinking eps by 10 and seeing the gap shrink by ~100."""
    geom = synth.geometry("barrel10", bz=0.0, xx0_scale=0.0)
    lt = geom.layer_table()
    R = geom.r
    rng = np.random.default_rng(5)
    truth = np.array([0.02, -0.01, 0.5, 0.5, 0.3, 1.2])
    sig0 = np.array([0.05, 0.05, 0.05, 0.05, 0.005, 0.005])
    e_hit = rng.standard_normal((10, 2)); e_seed = rng.standard_normal(6)

    def line_hits(p):
        cp, sp = np.cos(p[4]), np.sin(p[4])
        u = p[0] * cp + p[1] * sp
        s = -u + np.sqrt(u * u + R * R - p[0] ** 2 - p[1] ** 2)
        return np.stack([p[0] + s * cp, p[1] + s * sp, p[2] + s / np.tan(p[5])], axis=1)

    gaps = []
    for eps in (1.0, 0.1):
        h = line_hits(truth)
        az = np.arctan2(h[:, 1], h[:, 0]) + eps * e_hit[:, 0] * 0.01 / R
        hits = np.stack([R * np.cos(az), R * np.sin(az), h[:, 2] + eps * e_hit[:, 1] * 0.1], axis=1)
        seed = truth + eps * e_seed * sig0
        r = _fit_single(lt, 0.0, seed, sig0, 1, hits)

        def resid(v):   # state at the vertex (5 free parameters + iota fixed by its prior)
            p = np.array([v[0], v[1], v[2], seed[3], v[3], v[4]])
            d = (hits - line_hits(p))
            return np.concatenate([d[:, 0] / 0.01, d[:, 1] / 0.01, d[:, 2] / 0.1,
                                   (np.array([v[0], v[1], v[2]]) - seed[:3]) / sig0[:3], (v[3:] - seed[4:]) / sig0[4:]])
        sol = optimize.least_squares(resid, [seed[0], seed[1], seed[2], seed[4], seed[5]], xtol=1e-15, ftol=1e-15, gtol=1e-15)
        v = sol.x
        last = line_hits(np.array([v[0], v[1], v[2], seed[3], v[3], v[4]]))[-1]
        gap = max(np.max(np.abs(r["par"][:3, 0] - last)), abs(r["par"][4, 0] - v[3]), abs(r["par"][5, 0] - v[4]))
        gaps.append(gap)
    print('P5 gaps', gaps)
    assert gaps[0] < 1e-4          # already tiny at nominal smearing
    assert gaps[1] < gaps[0] / 30  # and second order in the smearing scale


def test_P6_gluckstern_curvature_resolution():
    """B = 3.8 T, pT = 1000 GeV, eta = 0, no scattering: parabola fit.  sigma(kappa) from Gluckstern's formula
    for N+1 = 10 equidistant points over L = 36 cm; sigma(1/pT) = sigma(kappa)/(k B); r-phi error at R = 40.
    Catches: wrong curvature Jacobian column (F_x,iota ~ s^2/2 lever arm), wrong field constant."""
    geom = synth.geometry("barrel10", bz=3.8, xx0_scale=0.0)
    lt = geom.layer_table()
    ok = np.ones(1, bool)
    x = y = z = np.zeros(1)
    hits = []
    st = dict(x=x, y=y, z=z, ipt=np.array([1e-3]), phi=np.array([0.3]), theta=np.array([np.pi / 2]))
    for R in geom.r:
        ok, xs, ys, zs, ph, s, ci = synth.cross_cylinder(0.0, 0.0, 0.0, 1e-3, 0.3, np.pi / 2, 1, 3.8, R)
        hits.append([float(xs), float(ys), float(zs)])
    hits = np.array(hits)
    sig0 = np.array([1, 1, 10, 1.0, 0.1, 0.1])
    r = _fit_single(lt, 3.8, [0, 0, 0, 1e-3, 0.3, np.pi / 2], sig0, 1, hits)
    C = r["cov"][0]
    p = r["par"][:, 0]
    t = np.array([-p[1], p[0], 0.0]) / np.hypot(p[0], p[1])
    assert abs(np.sqrt(C[3, 3]) * K * 3.8 - GOLD["gluckstern_sigma_kappa"]) / GOLD["gluckstern_sigma_kappa"] < 1e-3
    assert abs(np.sqrt(t @ C[:3, :3] @ t) - GOLD["gluckstern_sigma_rphi_40"]) / GOLD["gluckstern_sigma_rphi_40"] < 1e-3


# ------------------------------------------------------------------------------------------------ P7 / P8
def test_P7_linear_kalman_equals_normal_equations():
    """Random linear model x_{k+1} = F_k x_k, measurements of the first three components with V = diag:
    oracle similarity + update chained == batch weighted least squares (information form).  Catches: gain or
    Joseph-form mistakes that P5's special geometry might hide."""
    rng = np.random.default_rng(7)
    n_step = 6
    x0 = np.array([0.1, -0.2, 0.3, 1.0, 0.2, 0.9])
    P0 = np.diag([0.5, 0.4, 0.6, 0.01, 0.2, 0.3]) ** 2
    Fs = [np.eye(6) + 0.2 * rng.standard_normal((6, 6)) for _ in range(n_step)]
    sr, sz = 0.05, 0.2
    V = np.diag([sr * sr, sr * sr, sz * sz])
    H = np.hstack([np.eye(3), np.zeros((3, 3))])
    ms = [rng.standard_normal(3) for _ in range(n_step)]
    # batch: unknown = initial state; propagate the information
    A = np.linalg.inv(P0); b = A @ x0
    Phi = np.eye(6)
    rng = np.random.default_rng(7)
    Fs2 = [np.eye(6) + 0.2 * rng.standard_normal((6, 6)) for _ in range(n_step)]
    ms2 = [rng.standard_normal(3) for _ in range(n_step)]
    xs, Ps = x0.copy(), P0.copy()
    meas = []
    for F, e in zip(Fs2, ms2):   # replay the sequential filter in numpy to recover the actual measurements
        xs = F @ xs; Ps = F @ Ps @ F.T
        m = xs[:3] + 0.1 * e
        meas.append(m)
        S = H @ Ps @ H.T + V; Kg = Ps @ H.T @ np.linalg.inv(S)
        xs = xs + Kg @ (m - H @ xs); Ps = (np.eye(6) - Kg @ H) @ Ps
    for F, m in zip(Fs2, meas):
        Phi = F @ Phi
        G = H @ Phi
        A += G.T @ np.linalg.inv(V) @ G; b += G.T @ np.linalg.inv(V) @ m
    x_batch0 = np.linalg.solve(A, b)
    x_batch = Phi @ x_batch0
    P_batch = Phi @ np.linalg.inv(A) @ Phi.T
    # oracle again, now on exactly those measurements
    x, P = x0.copy(), P0.copy()
    for F, m in zip(Fs2, meas):
        x = F @ x; P = o.similarity6(F, P)
        f, x, P, c2 = o.update(x, P, m, sr, sz, sr)
        assert f == 0
    assert np.max(np.abs(x - x_batch)) < 1e-9 * np.max(np.abs(x_batch))
    assert np.max(np.abs(P - P_batch)) < 1e-9 * np.max(np.abs(P_batch))


def test_P8_small_matrix_core_vs_lapack():
    rng = np.random.default_rng(8)
    for _ in range(200):
        A = rng.standard_normal((3, 3)); S = A @ A.T + 1e-3 * np.eye(3)
        rc, Si = o.inv3_spd(S)
        assert rc == 0 and np.max(np.abs(Si - np.linalg.inv(S))) < 1e-12 * np.max(np.abs(Si)) * np.linalg.cond(S)
        J = rng.standard_normal((6, 6)); B = rng.standard_normal((6, 6)); Cm = B @ B.T
        assert np.max(np.abs(o.similarity6(J, Cm) - J @ Cm @ J.T)) < 1e-12 * np.abs(J @ Cm @ J.T).max()
    rc, _ = o.inv3_spd(np.diag([1.0, -1.0, 1.0]))
    assert rc != 0


def test_hit_covariance_orientation():
    """sig_r != sig_rphi: V must be the rotation of diag(sig_r^2, sig_rphi^2) to the hit's azimuth.  For a hit on
    the x axis a radial residual costs 1/sig_r^2, a tangential one 1/sig_rphi^2 (and swapped on the y axis)."""
    p = np.zeros(6); p[3] = 1; p[5] = 1.0
    Cz = np.zeros((6, 6))
    for (m, d, expect) in (([10, 0, 0], [0.1, 0, 0], (0.1 / 0.5) ** 2), ([10, 0, 0], [0, 0.1, 0], (0.1 / 0.02) ** 2),
                           ([0, 10, 0], [0.1, 0, 0], (0.1 / 0.02) ** 2), ([0, 10, 0], [0, 0, 0.3], (0.3 / 0.2) ** 2)):
        st = p.copy(); st[:3] = np.array(m) - np.array(d)
        rc, c2 = o.chi2(st, Cz, m, 0.02, 0.2, 0.5)
        assert rc == 0 and abs(c2 - expect) < 2e-3 * expect   # hit azimuth vs state azimuth differ slightly


# ------------------------------------------------------------------------------------------------ P9
def _run(fi, par=None, q=None, bz=None, hits=None, layers=None):
    par = fi.par if par is None else par
    hx, hy, hz = (fi.hit_x, fi.hit_y, fi.hit_z) if hits is None else hits
    return o.fit(fi.geom.layer_table() if layers is None else layers, fi.geom.bz if bz is None else bz, par, fi.cov,
                 fi.q if q is None else q, hx, hy, hz, fi.seg_off, fi.hit_idx)


def test_P9_invariances():
    """Rotation about z, mirror z -> -z (theta -> pi - theta), and (q, B) -> (-q, -B) leave chi2 unchanged and
    transform states/covariances covariantly.  Catches: frame-dependent terms, sign slips in curvature."""
    fi = synth.fit_inputs(2, n=300)
    base = _run(fi)
    n = fi.n
    # (q,B) -> (-q,-B)
    r = _run(fi, q=(-fi.q).astype(np.int8), bz=-fi.geom.bz)
    assert np.array_equal(r["status"], base["status"])
    assert np.max(np.abs(r["par"] - base["par"])) < 1e-12 and np.max(np.abs(r["chi2"] - base["chi2"])) < 1e-12
    # rotation by a
    a = 0.7
    ca, sa = np.cos(a), np.sin(a)
    p64 = fi.par.astype(np.float64)
    h64x, h64y = fi.hit_x.astype(np.float64), fi.hit_y.astype(np.float64)
    par = p64.copy()
    par[0], par[1] = ca * p64[0] - sa * p64[1], sa * p64[0] + ca * p64[1]
    par[4] = p64[4] + a
    hx = ca * h64x - sa * h64y; hy = sa * h64x + ca * h64y
    # the diagonal seed covariance has equal x and y variances, hence is rotation invariant
    r = _run(fi, par=par, hits=(hx, hy, fi.hit_z))
    assert np.array_equal(r["status"], base["status"])
    okm = base["nhits"] > 0
    assert np.max(np.abs(r["chi2"] - base["chi2"])[okm] / np.maximum(base["chi2"][okm], 1e-9)) < 1e-8
    Rm = np.eye(6); Rm[0, 0] = ca; Rm[0, 1] = -sa; Rm[1, 0] = sa; Rm[1, 1] = ca
    exp = Rm @ base["par"]; exp[4] = np.angle(np.exp(1j * (base["par"][4] + a)))
    assert np.max(np.abs(r["par"] - exp)) < 1e-9
    expC = Rm @ base["cov"] @ Rm.T
    assert np.max(np.abs(r["cov"] - expC)) < 1e-9 * np.max(np.abs(expC))
    # mirror
    par = fi.par.astype(np.float64).copy(); par[2] = -par[2]; par[5] = np.pi - par[5]
    r = _run(fi, par=par, hits=(fi.hit_x, fi.hit_y, -fi.hit_z.astype(np.float64)))
    M = np.diag([1, 1, -1, 1, 1, -1.0])
    exp = M @ base["par"]; exp[5] += np.pi
    assert np.max(np.abs(r["par"] - exp)) < 1e-9 and np.max(np.abs(r["chi2"] - base["chi2"])) < 1e-7
    assert np.max(np.abs(r["cov"] - M @ base["cov"] @ M)) < 1e-9 * np.max(np.abs(base["cov"]))


# ------------------------------------------------------------------------------------------------ P10
def test_P10_invariants():
    fi = synth.fit_inputs(2, n=2000)
    r = _run(fi)
    C = r["cov"]
    assert np.array_equal(C, np.swapaxes(C, 1, 2))                      # Joseph form: exactly symmetric
    lam = np.linalg.eigvalsh(C)
    assert (lam[:, 0] >= -1e-10 * lam[:, -1]).all()                     # PSD (one ~0 eigenvalue: surface normal)
    assert (r["chi2"] >= 0).all()
    # strictly PD on the tangent space (r-phi, z, iota, phi, theta)
    for i in np.nonzero(r["nhits"] > 3)[0][:300]:
        p = r["par"][:, i]
        rr = np.hypot(p[0], p[1])
        T = np.zeros((5, 6)); T[0, 0] = -p[1] / rr; T[0, 1] = p[0] / rr; T[1, 2] = 1; T[2, 3] = 1; T[3, 4] = 1; T[4, 5] = 1
        assert np.linalg.eigvalsh(T @ C[i] @ T.T)[0] > 0
    # C_upd <= C_pred, and adding Q before or after the update is the same thing (Q has no position block)
    lt = fi.geom.layer_table()
    rng = np.random.default_rng(10)
    for i in range(50):
        p = fi.par[:, i].astype(np.float64); Cm = synth.unpack_sym(fi.cov[:, i].astype(np.float64))
        f, pp, J, s, ci = o.propagate(p, fi.q[i], fi.geom.bz, lt[0, 0])
        Cp = o.similarity6(J, Cm); Q = o.ms_noise(pp, ci, lt[0, 2])
        m = [fi.hit_x[i], fi.hit_y[i], fi.hit_z[i]]
        f1, p1, C1, c1 = o.update(pp, Cp + Q, m, *lt[0, 3:6])
        f2, p2, C2, c2 = o.update(pp, Cp, m, *lt[0, 3:6])
        assert np.linalg.eigvalsh(Cp + Q - C1)[0] > -1e-12 * np.abs(Cp).max()
        assert np.max(np.abs(C1 - (C2 + Q))) < 1e-12 * np.abs(C1).max() and abs(c1 - c2) < 1e-9 and np.max(np.abs(p1 - p2)) < 1e-12
        assert (Q[:3] == 0).all() and (Q[:, :3] == 0).all()
        f3, pp3, Cp3 = o.predict(lt, 0, fi.geom.bz, p, Cm, fi.q[i])
        assert np.array_equal(pp3, pp) and np.max(np.abs(Cp3 - (Cp + Q))) == 0


def test_ms_noise_matches_monte_carlo():
    """Q in (iota, phi, theta) vs brute force: rotate the momentum by two orthogonal Gaussian angles of width
    theta0 (|p| fixed) and take the sample covariance.  Catches: missing 1/sin^2, wrong sign of the
    iota-theta correlation.  theta0 itself is checked against the Highland formula typed out here."""
    rng = np.random.default_rng(11)
    p = np.array([10.0, 5.0, 3.0, 0.8, 0.4, 1.1]); ci, xx0 = 0.9, 0.02
    Q = o.ms_noise(p, ci, xx0)
    t = xx0 / (np.sin(p[5]) * ci)
    pmom = 1 / (p[3] * np.sin(p[5]))
    th0 = 0.0136 / pmom * np.sqrt(t) * (1 + 0.038 * np.log(t))
    assert abs(Q[5, 5] - th0 ** 2) < 1e-12 * th0 ** 2
    N = 400000
    e1, e2 = rng.standard_normal(N) * th0, rng.standard_normal(N) * th0
    th, ph = p[5], p[4]
    d = np.array([np.sin(th) * np.cos(ph), np.sin(th) * np.sin(ph), np.cos(th)])
    eth = np.array([np.cos(th) * np.cos(ph), np.cos(th) * np.sin(ph), -np.sin(th)])
    eph = np.array([-np.sin(ph), np.cos(ph), 0])
    dn = d[:, None] + eth[:, None] * e1 + eph[:, None] * e2
    dn /= np.linalg.norm(dn, axis=0)
    thn = np.arccos(dn[2]); phn = np.arctan2(dn[1], dn[0]); iptn = 1 / (pmom * np.sin(thn))
    S = np.cov(np.stack([iptn - p[3], phn - ph, thn - th]))
    Qs = Q[3:, 3:]
    assert np.max(np.abs(S - Qs) / np.sqrt(np.outer(np.diag(Qs), np.diag(Qs)))) < 0.01


# ------------------------------------------------------------------------------------------------ P11
def _pulls(fi, r):
    n = fi.n
    last = np.where(fi.valid, np.arange(fi.geom.n_layers)[:, None], -1).max(axis=0)
    sel = (r["status"] == 0) & (last >= 0) & (r["nhits"] == fi.valid.sum(axis=0))
    idx = np.nonzero(sel)[0]
    tr = fi.truth[last[idx], idx]
    p = r["par"][:, idx].T; C = r["cov"][idx]
    rr = np.hypot(tr[:, 0], tr[:, 1])
    T = np.zeros((len(idx), 5, 6))
    T[:, 0, 0] = -tr[:, 1] / rr; T[:, 0, 1] = tr[:, 0] / rr; T[:, 1, 2] = 1; T[:, 2, 3] = 1; T[:, 3, 4] = 1; T[:, 4, 5] = 1
    d = p - tr
    d[:, 4] = np.angle(np.exp(1j * d[:, 4]))
    dd = np.einsum("nij,nj->ni", T, d)
    var = np.einsum("nij,njk,nik->ni", T, C, T)
    return dd / np.sqrt(var), r["chi2"][idx], r["nhits"][idx]


@pytest.mark.parametrize("config,n", [(0, 20000), (2, 20000)])
def test_P11_pulls_and_chi2_statistics(config, n):
    """Pulls of (r-phi, z, 1/pT, phi, theta) at the last layer have mean 0 and width 1; chi2/(2 nhits) has mean 1
    (two effective degrees of freedom per hit, consistent prior); chi2 p-values are flat.  Catches: wrong Q
    (too small/large), wrong V, inconsistent seed covariance, biased propagation."""
    fi = synth.fit_inputs(config, n=n)
    r = _run(fi)
    pulls, chi2, nh = _pulls(fi, r)
    assert len(chi2) > 0.6 * n
    core = np.abs(pulls) < 5   # Highland tails do not exist here (Gaussian kicks), keep all but absurd outliers
    assert core.mean() > 0.9995
    assert np.all(np.abs(pulls.mean(axis=0)) < 0.03), pulls.mean(axis=0)
    assert np.all(np.abs(pulls.std(axis=0) - 1) < 0.03), pulls.std(axis=0)
    assert abs((chi2 / (2 * nh)).mean() - 1) < 0.02
    pval = stats.chi2.sf(chi2, 2 * nh)
    hist = np.histogram(pval, bins=10, range=(0, 1))[0] / len(pval)
    assert np.all(np.abs(hist - 0.1) < 0.012), hist


@pytest.mark.parametrize("event", [1, 2, 3])
def test_P11_hundred_track_cases(event):
    fi = synth.fit_inputs(0, n=100, event=event)
    r = _run(fi)
    pulls, chi2, nh = _pulls(fi, r)
    assert np.all(np.abs(pulls.std(axis=0) - 1) < 0.25) and np.all(np.abs(pulls.mean(axis=0)) < 0.3)
    assert abs((chi2 / (2 * nh)).mean() - 1) < 0.15


def test_fit_skips_and_stops():
    """hit_idx <= -2 skips the layer entirely; a failing layer freezes the track with the status bit set."""
    fi = synth.fit_inputs(0, n=64, force_index=True)
    base = _run(fi)
    hi = fi.hit_idx.copy(); hi[4, :] = -2
    r = o.fit(fi.geom.layer_table(), fi.geom.bz, fi.par, fi.cov, fi.q, fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off, hi)
    assert (r["nhits"] == 9).all() and (r["status"] == 0).all()
    # same as removing the layer from the geometry altogether
    lt = np.delete(fi.geom.layer_table(), 4, axis=0)
    L, ld = 10, fi.ld
    keep = [l for l in range(10) if l != 4]
    hx = fi.hit_x.reshape(L, ld)[keep].reshape(-1); hy = fi.hit_y.reshape(L, ld)[keep].reshape(-1); hz = fi.hit_z.reshape(L, ld)[keep].reshape(-1)
    r2 = o.fit(lt, fi.geom.bz, fi.par, fi.cov, fi.q, hx, hy, hz, np.arange(10) * ld)
    assert np.array_equal(r["par"], r2["par"]) and np.array_equal(r["chi2"], r2["chi2"])
    # last layer moved out to R = 400 cm: unreachable for 2 rho < 400 (pT < 2.28 GeV) -> bit 0, state frozen after 9 layers
    lt = fi.geom.layer_table(); lt[9, 0] = 400.0
    r3 = o.fit(lt, fi.geom.bz, fi.par, fi.cov, fi.q, fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off)
    r9 = o.fit(lt[:9], fi.geom.bz, fi.par, fi.cov, fi.q, fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off[:10])
    pt = 1 / r9["par"][3]
    low, high = pt < 2.0, pt > 2.6
    assert low.any() and high.any()
    assert (r3["status"][low] == o.UNREACHABLE).all() and (r3["nhits"][low] == 9).all()
    assert np.array_equal(r3["par"][:, low], r9["par"][:, low]) and np.array_equal(r3["cov"][low], r9["cov"][low])
    assert ((r3["status"][high] & o.UNREACHABLE) == 0).all()
    assert np.array_equal(base["nhits"], np.full(64, 10))


def test_fit_hole_layer_transports_and_adds_material():
    """hit_idx == -1 (R8): the layer is crossed without a hit -- the state is transported to it and the
    layer's scattering is added, only the update is left out.
    (a) Without material on that layer the intermediate stop changes nothing: transport to r_4 and then to r_5 is
        the transport to r_5 (the helix maps form a group, so the Jacobians compose) -- equal to the fit with the
        layer removed from the geometry.  Catches: a Jacobian that does not compose (a wrong ds/dp term), a hole
        that leaves the state behind or touches chi2 / nhits.
    (b) With material the covariance can only grow: C(hole) - C(layer removed) is positive semi-definite and not
        zero, the chi2 of the later hits falls.  Catches: Q subtracted or dropped."""
    fi = synth.fit_inputs(0, n=64, force_index=True)
    L, ld = 10, fi.ld
    hi = fi.hit_idx.copy(); hi[4, :] = -1
    keep = [l for l in range(10) if l != 4]
    hx = fi.hit_x.reshape(L, ld)[keep].reshape(-1); hy = fi.hit_y.reshape(L, ld)[keep].reshape(-1); hz = fi.hit_z.reshape(L, ld)[keep].reshape(-1)
    lt = fi.geom.layer_table()
    removed = o.fit(np.delete(lt, 4, axis=0), fi.geom.bz, fi.par, fi.cov, fi.q, hx, hy, hz, np.arange(10) * ld)
    lt0 = lt.copy(); lt0[4, 2] = 0.0
    r = o.fit(lt0, fi.geom.bz, fi.par, fi.cov, fi.q, fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off, hi)
    assert (r["nhits"] == 9).all() and (r["status"] == 0).all()
    assert np.max(np.abs(r["par"] - removed["par"])) < 1e-9 and np.max(np.abs(r["chi2"] - removed["chi2"])) < 1e-7
    assert np.max(np.abs(r["cov"] - removed["cov"]) / np.abs(removed["cov"]).max(axis=(1, 2), keepdims=True)) < 1e-8
    rm = o.fit(lt, fi.geom.bz, fi.par, fi.cov, fi.q, fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off, hi)
    assert (rm["nhits"] == 9).all() and (rm["status"] == 0).all()
    # stop right after the hole (layers 0..5, hit on 5): before later hits mix the information
    h5 = hi.copy(); h5[6:] = -2
    a = o.fit(lt, fi.geom.bz, fi.par, fi.cov, fi.q, fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off, h5)
    b_ = o.fit(lt0, fi.geom.bz, fi.par, fi.cov, fi.q, fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off, h5)
    for t in range(fi.n):
        lam = np.linalg.eigvalsh(a["cov"][t] - b_["cov"][t])
        assert lam[0] > -1e-9 * lam[-1] and lam[-1] > 0
    assert (a["chi2"] < b_["chi2"]).mean() > 0.95
    # a hole on the last layer leaves the state ON that layer (transported, not updated)
    hl = fi.hit_idx.copy(); hl[9, :] = -1
    e = o.fit(lt, fi.geom.bz, fi.par, fi.cov, fi.q, fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off, hl)
    assert np.allclose(np.hypot(e["par"][0], e["par"][1]), 40.0, atol=1e-9) and (e["nhits"] == 9).all()


def test_fit_hole_layers_keep_unit_pulls():
    """Statistics pin of R8: 25 % of the inner hits of config-2-like tracks removed and marked as holes (-1).  With the
    material of the hole layers the pulls stay unit and chi2/ndf = 1; leaving the material out (the round-1 reading,
    reproduced here with -2) widens the 1/pT pull to ~1.12 and chi2/ndf to ~1.03."""
    fi = synth.fit_inputs(2, n=20000, force_index=True)
    L = fi.geom.n_layers
    rng = np.random.default_rng(5)
    last = np.where(fi.valid, np.arange(L)[:, None], -1).max(axis=0)
    lay = np.arange(L)[:, None]
    drop = (rng.random((L, fi.n)) < 0.25) & fi.valid & (lay < last[None, :]) & (lay > 0)
    width = {}
    for mode in (-1, -2):
        h = fi.hit_idx.copy(); h[:, :fi.n][drop] = mode
        r = o.fit(fi.geom.layer_table(), fi.geom.bz, fi.par, fi.cov, fi.q, fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off, h)
        kept = type("V", (), {})()
        kept.n, kept.geom, kept.truth, kept.valid = fi.n, fi.geom, fi.truth, fi.valid & ~drop
        pulls, chi2, nh = _pulls(kept, r)
        assert len(chi2) > 0.9 * fi.n
        width[mode] = (pulls.std(axis=0), (chi2 / (2 * nh)).mean())
    assert np.all(np.abs(width[-1][0] - 1) < 0.03) and abs(width[-1][1] - 1) < 0.02, width[-1]
    assert width[-2][0][2] > 1.06 and width[-2][1] > 1.015, width[-2]


def _first_crossing_turn(x, y, phi, w, R):
    """Turning angle about the centre of curvature up to the first crossing of |p| = R (test-local circle-circle
    geometry): None when the circles do not intersect."""
    cx, cy, rho = x - np.sin(phi) / w, y + np.cos(phi) / w, 1 / abs(w)
    d = np.hypot(cx, cy)
    cosb = (d * d + R * R - rho * rho) / (2 * d * R)
    if abs(cosb) > 1:
        return None
    beta, gamma, psi0 = np.arccos(cosb), np.arctan2(cy, cx), np.arctan2(y - cy, x - cx)
    turns = []
    for pm in (1, -1):
        psi = np.arctan2(R * np.sin(gamma + pm * beta) - cy, R * np.cos(gamma + pm * beta) - cx)
        turns.append(np.mod((psi - psi0) * np.sign(w), 2 * np.pi))
    return min(turns)


def test_P1_half_turn_boundary():
    """DESIGN.md R2: the crossing must come within HALF a turn.  States anywhere inside the cylinder, moving in any
    direction (inwards included), tight circles: the oracle reports UNREACHABLE exactly when the circles do not
    intersect or the first crossing needs more than half a turn, and the simulator's cross_cylinder agrees.
    Catches: a march limit of a full turn (or none), the second crossing taken for inward-moving states."""
    rng = np.random.default_rng(7)
    n_far = n_near = 0
    for _ in range(6000):
        R = rng.uniform(5, 80)
        r0, a = rng.uniform(0.05, 0.97) * R, rng.uniform(-np.pi, np.pi)
        rho = np.exp(rng.uniform(np.log(0.52 * (R - r0)), np.log(3 * R)))      # tight circles: many need a long arc
        q, bz = rng.choice([-1, 1]), rng.choice([3.8, -3.8])
        pt = rho * K * abs(bz)
        phi = rng.uniform(-np.pi, np.pi)
        p = np.array([r0 * np.cos(a), r0 * np.sin(a), 0.0, 1 / pt, phi, 1.3])
        w = -q * K * bz / pt
        turn = _first_crossing_turn(p[0], p[1], phi, w, R)
        f, po, J, s, ci = o.propagate(p, q, bz, R)
        ok, xs, ys, *_ = synth.cross_cylinder(p[0], p[1], p[2], p[3], p[4], p[5], q, bz, R)
        if turn is None:
            assert f == o.UNREACHABLE and not ok
            continue
        if abs(turn - np.pi) < 1e-6:
            continue
        if turn > np.pi:
            n_far += 1
            assert f == o.UNREACHABLE and not ok, (turn, f)
            continue
        cos_inc = (xs * np.cos(phi + turn * np.sign(w)) + ys * np.sin(phi + turn * np.sign(w))) / R
        n_near += 1
        assert ok and f == (o.GRAZING if cos_inc < 0.1 else 0), (turn, f, cos_inc)       # near-tangent double crossings included
        if cos_inc < 1e-3:
            continue
        assert abs(abs(w) * s - turn) < 1e-8 and abs(po[0] - xs) < 1e-8 and abs(po[1] - ys) < 1e-8
    assert n_far > 100 and n_near > 1000


def test_fit_numeric_exits():
    """KFO_NUMERIC in kfo_fit (status bit 3, track frozen at its last good state):
    (a) an innovation matrix that is not positive definite (hand-made seed covariance with a negative position block):
        nothing is used, the seed comes back unchanged;
    (b) an update that drives 1/pT <= 0 (hits of a negative track, seed of positive charge with a wide 1/pT prior):
        the state is that of the fit truncated before the failing layer.
    Catches: a failed layer that still updates the state or counts a hit, a missing status bit."""
    fi = synth.fit_inputs(0, n=8, ms=False)
    lt = fi.geom.layer_table()
    cov = fi.cov.copy()
    cov[synth.pack_index(0, 0), :] = -1.0; cov[synth.pack_index(1, 1), :] = -1.0
    r = o.fit(lt, fi.geom.bz, fi.par, cov, fi.q, fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off)
    assert (r["status"] == o.NUMERIC).all() and (r["nhits"] == 0).all() and (r["chi2"] == 0).all()
    assert np.array_equal(r["par"], fi.par[:, :8].astype(np.float64))
    assert np.array_equal(synth.pack_sym(r["cov"]).T, cov[:, :8].astype(np.float64))
    # (b) wrong charge, stiff seed with a wide curvature prior: 1/pT is pulled through zero
    par = fi.par.copy(); par[3, :] = 0.02
    cov = fi.cov.copy(); cov[synth.pack_index(3, 3), :] = 1.0
    q = (-fi.q).astype(np.int8)
    r = o.fit(lt, fi.geom.bz, par, cov, q, fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off)
    failed = (r["status"] & o.NUMERIC) != 0
    assert failed.sum() >= 4 and (r["nhits"][failed] < 10).all() and (r["par"][3][failed] > 0).all()
    for t in np.nonzero(failed)[0]:
        k = r["nhits"][t]
        rt = o.fit(lt[:k], fi.geom.bz, par, cov, q, fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off[:k + 1])
        assert rt["status"][t] == 0 and rt["nhits"][t] == k
        assert np.array_equal(rt["par"][:, t], r["par"][:, t]) and np.array_equal(rt["cov"][t], r["cov"][t]) and rt["chi2"][t] == r["chi2"][t]
        # the next update really is the one that fails: 1/pT of the unguarded Kalman step is <= 0
        f, pp, Cp = o.predict(lt, k, fi.geom.bz, rt["par"][:, t], rt["cov"][t], q[t])
        m = np.array([fi.hit_x[k * fi.ld + t], fi.hit_y[k * fi.ld + t], fi.hit_z[k * fi.ld + t]], dtype=np.float64)
        S = Cp[:3, :3] + np.diag([lt[k, 5] ** 2, lt[k, 5] ** 2, lt[k, 4] ** 2])
        assert f == 0 and (pp + Cp[:, :3] @ np.linalg.solve(S, m - pp[:3]))[3] <= 0


def test_mat66_multiply_definition():
    """Layout micro-benchmark oracle: element-wise triple loop, identity, and (AB)^T = B^T A^T."""
    rng = np.random.default_rng(66)
    A = rng.normal(size=(5, 6, 6)); B = rng.normal(size=(5, 6, 6))
    C = o.mat66_multiply(A, B)
    for i in range(5):
        for r in range(6):
            for c in range(6):
                assert abs(C[i, r, c] - sum(A[i, r, k] * B[i, k, c] for k in range(6))) < 1e-13
    I = np.broadcast_to(np.eye(6), (5, 6, 6))
    assert np.array_equal(o.mat66_multiply(A, I), A) and np.array_equal(o.mat66_multiply(I, B), B)
    assert np.allclose(o.mat66_multiply(A, B).transpose(0, 2, 1), o.mat66_multiply(B.transpose(0, 2, 1), A.transpose(0, 2, 1)), atol=1e-13)

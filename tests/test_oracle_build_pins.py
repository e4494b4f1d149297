"""Pins of the oracle's binning, window lookup and combinatorial building (oracle/kf_oracle.c) to things other than
itself.  CPU only.  The paper gives no formulas for these (readings X1-X3, R10, R11), so the pins are:
fp64 atan2 / plain numpy arithmetic for the bins, brute force over all hits for the lookup, the same build without
the spatial index (P12), an exhaustive Python enumeration of every hit combination on tiny events, the fit oracle
on the built hit list, and truth purity on noise-free events.
"""
import itertools

import numpy as np
import pytest

from oracle import kf_oracle as o
from paper_1711_06571_b200 import synth


# ------------------------------------------------------------------------------------------------ X1 / X2
@pytest.mark.parametrize("n_phi", [8, 256, 1024])
def test_X1_phi_bin_vs_atan2(n_phi):
    """Tangent-table bin == floor(phi N / 2pi) from fp64 atan2, except for hits within 1e-5 bin widths of an edge
    (there: off by exactly one bin).  Catches: wrong octant folding, off-by-one in the table search."""
    rng = np.random.default_rng(21)
    n = 20000
    r = rng.uniform(3, 90, n)
    a = rng.uniform(-np.pi, np.pi, n)
    x, y = (r * np.cos(a)).astype(np.float32), (r * np.sin(a)).astype(np.float32)
    got = o.phi_bin(x, y, n_phi)
    f = np.mod(np.arctan2(y.astype(np.float64), x.astype(np.float64)), 2 * np.pi) * n_phi / (2 * np.pi)
    exp = np.floor(f).astype(np.int64) % n_phi
    assert got.min() >= 0 and got.max() <= n_phi - 1
    bad = got != exp
    assert bad.mean() < 1e-4
    dist = np.minimum(f - np.floor(f), np.ceil(f) - f)
    assert (dist[bad] < 1e-5).all()
    assert (((got[bad] - exp[bad]) % n_phi == 1) | ((exp[bad] - got[bad]) % n_phi == 1)).all()


def test_X1_axis_points_and_symmetry():
    assert list(o.phi_bin([1, 0, -1, 0], [0, 1, 0, -1], 256)) == [0, 63, 127, 192]
    assert list(o.phi_bin([1, -1, -1, 1], [1, 1, -1, -1], 256)) == [31, 96, 159, 224]   # diagonals sit exactly on a bin edge: t = 1 -> j = N/8-1, folded per quadrant
    # mirror symmetry about the x axis: bin(x, -y) = N - 1 - bin(x, y) away from the axes
    rng = np.random.default_rng(22)
    x, y = rng.uniform(-50, 50, 2000).astype(np.float32), rng.uniform(0.1, 50, 2000).astype(np.float32)
    assert np.array_equal(o.phi_bin(x, -y, 1024), 1023 - o.phi_bin(x, y, 1024))


def test_X2_z_bin():
    z = np.array([-150, -100, -99.999, -87.5, -87.4999, 0, 99.99, 100, 1e4], dtype=np.float32)
    assert list(o.z_bin(z, 100.0, 16)) == [0, 0, 0, 1, 1, 8, 15, 15, 15]
    rng = np.random.default_rng(23)
    z = rng.uniform(-100, 100, 5000).astype(np.float32)
    exp = np.clip(np.floor((z + np.float32(100)) * np.float32(32 / 200.0)), 0, 31).astype(np.int32)   # numpy fp32 arithmetic
    assert np.array_equal(o.z_bin(z, 100.0, 32), exp)


# ------------------------------------------------------------------------------------------------ B0
def _small_event(config=3, n_events=2, tracks=300, **kw):
    bi = synth.build_inputs(config, n_events=n_events, tracks=tracks, **kw)
    lt = bi.geom.layer_table()
    b = o.bin_hits(lt, bi.n_events, bi.seg_off, bi.hit_x, bi.hit_y, bi.hit_z, bi.n_phi, bi.n_z)
    return bi, lt, b


def test_B0_sorted_index_properties():
    """perm is a permutation of every segment, sorted arrays are the gathered originals, keys ascend, ties keep the
    original order (stable), bin_off delimits exactly the hits of each bin.  The bin key is recomputed here from
    fp64 atan2 / plain arithmetic; only hits on a bin edge may differ."""
    bi, lt, b = _small_event()
    L = lt.shape[0]
    nb = bi.n_phi * bi.n_z
    assert b["bin_off"][0] == 0 and b["bin_off"][-1] == len(bi.hit_x) and (np.diff(b["bin_off"]) >= 0).all()
    for sg in range(bi.n_events * L):
        s0, s1 = bi.seg_off[sg], bi.seg_off[sg + 1]
        p = b["perm"][s0:s1]
        assert np.array_equal(np.sort(p), np.arange(s1 - s0))
        assert np.array_equal(b["x"][s0:s1], bi.hit_x[s0:s1][p]) and np.array_equal(b["z"][s0:s1], bi.hit_z[s0:s1][p])
        assert b["bin_off"][sg * nb] == s0 and b["bin_off"][(sg + 1) * nb] == s1
        x, y, z = (a[s0:s1][p].astype(np.float64) for a in (bi.hit_x, bi.hit_y, bi.hit_z))
        f = np.mod(np.arctan2(y, x), 2 * np.pi) * bi.n_phi / (2 * np.pi)
        key = np.clip(np.floor((z + 100.0) * bi.n_z / 200.0), 0, bi.n_z - 1) * bi.n_phi + np.floor(f) % bi.n_phi
        binof = np.searchsorted(b["bin_off"][sg * nb:(sg + 1) * nb + 1], np.arange(s0, s1), side="right") - 1
        edge = np.minimum(f - np.floor(f), np.ceil(f) - f) < 1e-4
        assert np.array_equal(binof[~edge], key[~edge].astype(np.int64))
        assert (np.diff(binof) >= 0).all()
        same = np.diff(binof) == 0
        assert (np.diff(p)[same] > 0).all()                       # stable within a bin


# ------------------------------------------------------------------------------------------------ X3
def test_X3_window_lookup_vs_brute_force():
    """The bin-granular list (i) equals the hits whose (iz, iphi) lie in the X3 ranges, in row / wrapped-bin / sorted
    order, recomputed here with numpy; (ii) contains every hit truly inside the window.  Windows include wrapping
    across +-pi, across phi = 0, full circle, off both z ends."""
    bi, lt, b = _small_event()
    L = lt.shape[0]
    rng = np.random.default_rng(31)
    nq = 400
    ev = rng.integers(0, bi.n_events, nq).astype(np.int32); ly = rng.integers(0, L, nq).astype(np.int32)
    phc = rng.uniform(-np.pi, np.pi, nq).astype(np.float32)
    dph = np.abs(rng.normal(0, 0.05, nq)).astype(np.float32)
    zc = rng.uniform(-110, 110, nq).astype(np.float32); dz = np.abs(rng.normal(0, 8, nq)).astype(np.float32)
    phc[:4] = [3.14, -3.14, 0.001, -0.001]; dph[:4] = 0.05
    dph[4] = 4.0; dph[5] = 0.0; dz[6] = 0.0; zc[7] = 150.0; zc[8] = -150.0
    cap = 4096
    cnt, idx = o.window_lookup(lt, b, ev, ly, phc, dph, zc, dz, cap)
    nb = bi.n_phi * bi.n_z
    inv = np.float32(bi.n_phi / (2 * np.pi))
    for i in range(nq):
        sg = ev[i] * L + ly[i]
        s0, s1 = bi.seg_off[sg], bi.seg_off[sg + 1]
        binof = np.searchsorted(b["bin_off"][sg * nb:(sg + 1) * nb + 1], np.arange(s0, s1), side="right") - 1
        iz, ip = binof // bi.n_phi, binof % bi.n_phi
        b_lo = int(np.floor((phc[i] - dph[i]) * inv)); b_hi = int(np.floor((phc[i] + dph[i]) * inv))
        n_b = min(b_hi - b_lo + 1, bi.n_phi)
        z_lo = int(np.clip(np.floor((zc[i] - dz[i] + np.float32(100)) * np.float32(bi.n_z / 200.0)), 0, bi.n_z - 1))
        z_hi = int(np.clip(np.floor((zc[i] + dz[i] + np.float32(100)) * np.float32(bi.n_z / 200.0)), 0, bi.n_z - 1))
        assert o.window_bins(float(phc[i]), float(dph[i]), float(zc[i]), float(dz[i]), 100.0, bi.n_phi, bi.n_z) == (b_lo % bi.n_phi, n_b, z_lo, z_hi)
        exp = []
        for r in range(z_lo, z_hi + 1):
            for k in range(n_b):
                exp.extend(list(s0 + np.nonzero((iz == r) & (ip == (b_lo + k) % bi.n_phi))[0]))
        assert cnt[i] == len(exp)
        assert list(idx[i, :min(cnt[i], cap)]) == exp[:cap]
        # superset of the true window (away from bin edges)
        x, y, z = (a[s0:s1].astype(np.float64) for a in (b["x"], b["y"], b["z"]))
        dphi = np.abs(np.angle(np.exp(1j * (np.arctan2(y, x) - float(phc[i])))))
        inside = (dphi < float(dph[i]) * (1 - 1e-3) - 1e-5) & (np.abs(z - float(zc[i])) < float(dz[i]) * (1 - 1e-3) - 1e-4)
        assert set(s0 + np.nonzero(inside)[0]) <= set(exp)
    c2, i2 = o.window_lookup(lt, b, ev[:20], ly[:20], phc[:20], dph[:20], zc[:20], dz[:20], 3)     # cap smaller than the list
    assert np.array_equal(c2, cnt[:20]) and all(list(i2[k, :min(3, c2[k])]) == list(idx[k, :min(3, c2[k])]) for k in range(20))


# ------------------------------------------------------------------------------------------------ P12 and friends
def _build(bi, lt, b, K=None, use_bins=True, n=None, cut=None, n_sigma=None, margins=False):
    return o.kf_build(lt, bi.geom.bz, b, bi.seg_off, bi.par, bi.cov, bi.q, bi.seed_event, bi.seed_hit_idx, bi.first_layer,
                      bi.K if K is None else K, bi.chi2_cut if cut is None else cut, bi.n_sigma if n_sigma is None else n_sigma,
                      use_bins=use_bins, n=n, margins=margins)


@pytest.mark.parametrize("config,tracks", [(3, 400), (4, 600)])
def test_P12_bins_equal_brute_force(config, tracks):
    """The same algorithm without the spatial index (every hit of the layer tested against the strict window) gives
    identical candidates.  Catches: a window bin range that misses hits, wrap-around errors, wrong segment."""
    bi, lt, b = _small_event(config, n_events=2, tracks=tracks, fake_frac=0.0)
    a = _build(bi, lt, b)
    c = _build(bi, lt, b, use_bins=False)
    assert c["counters"]["n_scan"] > 20 * a["counters"]["n_scan"]
    for k in ("n_cand", "hit_idx", "nhits", "status", "chi2", "par"):
        assert np.array_equal(a[k], c[k]), k
    assert a["counters"]["n_window"] == c["counters"]["n_window"] and a["counters"]["n_upd"] == c["counters"]["n_upd"]


def _enumerate(bi, lt, b, s, K):
    """Exhaustive Python version of DESIGN.md R10/R11 for one seed, built from the oracle's single-step primitives
    (predict, chi2, update): every hit of the layer is tested (no bins; the window test itself is plain numpy),
    children are ranked with Python tuples.  Also returns, per layer, the smallest relative chi2 gap between children
    adjacent in the ranking (equal nhits, at least one kept): margins[..., 2] of the C build."""
    L = lt.shape[0]
    ev = bi.seed_event[s]
    cands = [dict(p=bi.par[:, s].astype(np.float64), C=synth.unpack_sym(bi.cov[:, s].astype(np.float64)), chi2=0.0, nh=bi.first_layer,
                  hits=list(bi.seed_hit_idx[:, s]) + [-2] * (L - bi.first_layer), fin=False, st=0)]
    gaps = np.full(L, 1e300)
    for l in range(bi.first_layer, L):
        sg = ev * L + l
        s0, s1 = bi.seg_off[sg], bi.seg_off[sg + 1]
        R, zmax, _, srphi, sz, sr = lt[l]
        hx, hy, hz = (b[k][s0:s1].astype(np.float64) for k in "xyz")
        children = []
        for ci, c in enumerate(cands):
            if c["fin"]:
                children.append((-c["nh"], c["chi2"], ci, np.inf, "fin", 0)); continue
            f, pp, Cp = o.predict(lt, l, bi.geom.bz, c["p"], c["C"], bi.q[s])
            if f:
                children.append((-c["nh"], c["chi2"], ci, np.inf, "fin", f)); continue
            x, y = pp[0], pp[1]
            r2 = x * x + y * y
            dphi = bi.n_sigma * np.sqrt(max((x * x * Cp[1, 1] - 2 * x * y * Cp[0, 1] + y * y * Cp[0, 0]) / r2 ** 2, 0) + (srphi / R) ** 2)
            dz = bi.n_sigma * np.sqrt(Cp[2, 2] + sz * sz)
            if abs(pp[2]) > zmax + dz:
                children.append((-c["nh"], c["chi2"], ci, np.inf, "fin", o.LEFT_Z)); continue
            inside = (np.abs(x * hy - y * hx) <= dphi * np.sqrt(r2) * np.hypot(hx, hy)) & (x * hx + y * hy > 0) & (np.abs(hz - pp[2]) <= dz)
            got = False
            for h in s0 + np.nonzero(inside)[0]:
                m = np.array([b["x"][h], b["y"][h], b["z"][h]], dtype=np.float64)
                rc, c2 = o.chi2(pp, Cp, m, srphi, sz, sr)
                if rc == 0 and c2 < bi.chi2_cut:
                    children.append((-(c["nh"] + 1), c["chi2"] + c2, ci, h, "hit", (pp, Cp, m)))
                    got = True
            if not got:
                children.append((-c["nh"], c["chi2"], ci, np.inf, "miss", (pp, Cp, None)))
        children.sort(key=lambda t: t[:4])
        for j in range(min(len(children) - 1, K)):
            u, v = children[j], children[j + 1]
            if u[0] == v[0]:
                gaps[l] = min(gaps[l], abs(u[1] - v[1]) / max(abs(u[1]), abs(v[1])) if max(abs(u[1]), abs(v[1])) > 0 else 0.0)
        new = []
        for (mnh, chi2, ci, h, kind, aux) in children[:K]:
            c = cands[ci]
            hits = list(c["hits"])
            if kind == "fin":
                hits[l] = -2
                new.append(dict(p=c["p"], C=c["C"], chi2=c["chi2"], nh=c["nh"], hits=hits, fin=True, st=c["st"] | aux))
            elif kind == "miss":
                hits[l] = -1
                new.append(dict(p=aux[0], C=aux[1], chi2=c["chi2"], nh=c["nh"], hits=hits, fin=False, st=c["st"]))
            else:
                f, pu, Cu, _ = o.update(aux[0], aux[1], aux[2], srphi, sz, sr)
                assert f == 0
                hits[l] = int(b["perm"][h])
                new.append(dict(p=pu, C=Cu, chi2=chi2, nh=-mnh, hits=hits, fin=False, st=c["st"]))
        cands = new
    return cands, gaps


def _check_against_enumeration(bi, lt, b, r, seeds, K):
    checked = multi = 0
    for s in seeds:
        ref, gaps = _enumerate(bi, lt, b, s, K)
        assert r["n_cand"][s] == len(ref)
        multi += len(ref) > 1
        for k, c in enumerate(ref):
            slot = s * K + k
            assert list(r["hit_idx"][:, slot]) == c["hits"], (s, k)
            assert r["nhits"][slot] == c["nh"] and abs(r["chi2"][slot] - c["chi2"]) <= 1e-9 * max(1, c["chi2"])
            assert r["status"][slot] == c["st"], (s, k, r["status"][slot], c["st"])
            pe = c["p"].copy(); pe[4] = np.angle(np.exp(1j * pe[4]))
            assert np.max(np.abs(r["par"][:, slot] - pe)) < 1e-9 and np.max(np.abs(r["cov"][slot] - c["C"])) < 1e-9 * np.abs(c["C"]).max()
            checked += 1
        if "margins" in r:
            got = r["margins"][s, :, 2]
            assert np.all((got == gaps) | (np.abs(got - gaps) <= 1e-6 * np.maximum(gaps, 1e-30))), (s, got, gaps)
    return checked, multi


@pytest.mark.parametrize("K", [1, 3, 10])
def test_build_equals_exhaustive_python_enumeration(K):
    """Dense tiny events (80 tracks + 5x noise in a narrowed barrel-10 event -> several compatible hits per window):
    the C build equals the step-by-step Python enumeration for 25 seeds.  Catches: ranking order, parent/child
    bookkeeping, hit-index mapping through perm, pass-through handling."""
    bi, lt, b = _small_event(3, n_events=1, tracks=1500, noise=8.0)
    r = _build(bi, lt, b, K=K, margins=True)
    checked, multi = _check_against_enumeration(bi, lt, b, r, range(0, bi.n_seeds, max(1, bi.n_seeds // 25))[:25], K)
    assert checked >= 25 and (K == 1 or multi >= 3)


def test_build_equals_enumeration_where_candidates_leave_the_barrel():
    """configs[4] generator (|eta| < 1.5, pT down to 0.3 GeV, 17 layers, fake seeds): the seeds whose candidates leave
    |z| <= zmax + window, graze or cannot reach the next layer, walked step by step -- the acceptance test
    |z'| > zmax + dz, the status bits and the 'finished' bookkeeping against the Python enumeration.
    Catches: a missing / negated dz in the acceptance test, the wrong layer's zmax, status bits lost on the way."""
    bi, lt, b = _small_event(4, n_events=1, tracks=800, fake_frac=0.2)
    K = 4
    r = _build(bi, lt, b, K=K, margins=True)
    st = r["status"].reshape(-1, K)
    left = np.nonzero(((st & o.LEFT_Z) != 0).any(axis=1))[0]
    other = np.nonzero(((st & (o.GRAZING | o.UNREACHABLE)) != 0).any(axis=1))[0]
    clean = np.nonzero((st == 0).all(axis=1))[0]
    assert len(left) >= 20 and len(other) >= 3
    seeds = list(left[:14]) + list(other[:6]) + list(clean[:6])
    checked, multi = _check_against_enumeration(bi, lt, b, r, seeds, K)
    assert checked >= 40 and multi >= 5


def test_left_z_fires_exactly_beyond_zmax_plus_window():
    """Acceptance exit of kfo_build (R11): a hand-built forward seed on layer 2; zmax of layer 3 is set just
    below and just above |z'| - dz (z', dz from the oracle's own predicted state, the window formula retyped here).
    The other layers carry other half lengths, so the wrong layer's zmax cannot give the same answers."""
    g = synth.geometry("barrel10")
    lt0 = g.layer_table()
    p = np.array([12.0, 0.0, 60.0, 0.5, 0.05, 0.45])         # pT = 2 GeV, theta = 0.45: z grows by ~8 cm per layer
    sig = np.array([0.05, 0.05, 0.05, 0.025, 0.005, 0.005])
    f, pp, Cp = o.predict(lt0, 3, g.bz, p, np.diag(sig ** 2), 1)
    assert f == 0
    dz = 3.0 * np.sqrt(Cp[2, 2] + lt0[3, 4] ** 2)
    edge = abs(pp[2]) - dz
    par = np.zeros((6, 32), np.float32); par[:, 0] = p
    cov = np.zeros((21, 32), np.float32)
    for i in range(6):
        cov[synth.pack_index(i, i), 0] = sig[i] ** 2
    f, pp, Cp = o.predict(lt0, 3, g.bz, par[:, 0].astype(np.float64), synth.unpack_sym(cov[:, 0].astype(np.float64)), 1)   # the fp32-rounded seed
    edge = abs(pp[2]) - 3.0 * np.sqrt(Cp[2, 2] + lt0[3, 4] ** 2)
    seg = np.zeros(11, np.int64)
    empty = np.zeros(0, np.float32)
    for eps, expect_left in ((-1e-9, True), (+1e-9, False)):
        lt = lt0.copy()
        lt[:, 1] = edge + 40.0          # every other layer: far inside acceptance
        lt[2, 1] = edge - 40.0          # ... except the seed's own layer: would always fire
        lt[3, 1] = edge + eps
        lt[4:, 1] = 1000.0
        b = o.bin_hits(lt, 1, seg, empty, empty, empty, 8, 1)
        r = o.kf_build(lt, g.bz, b, seg, par, cov, np.array([1], np.int8), np.zeros(1, np.int32), None, 3, 2, 30.0, 3.0, n=1, margins=True)
        assert r["n_cand"][0] == 1
        if expect_left:
            assert r["status"][0] == o.LEFT_Z and (r["hit_idx"][3:, 0] == -2).all()
            assert np.allclose(r["par"][:4, 0], par[:4, 0]) and np.allclose(r["cov"][0], synth.unpack_sym(cov[:, 0].astype(np.float64)))
        else:
            assert r["status"][0] == 0 and (r["hit_idx"][3:, 0] == -1).all()
            assert abs(np.hypot(r["par"][0, 0], r["par"][1, 0]) - 40.0) < 1e-9
        assert r["margins"][0, 3, 3] < 1e-9


def numeric_exit_case():
    """Hand-made seeds on layer 2 of the 10-layer barrel and two hits on layer 3 next to the predicted crossing of
    seeds 0-2.  Seed 0: negative x/y variances -> S not positive definite for the hits inside its window.  Seed 1: strong
    1/pT - y correlation -> the update with one of the two hits leaves 1/pT <= 0.  Seed 2: negative z variance -> the
    window itself is not finite.  Seed 3: as seed 0 but pointing away from every hit (no hit inside the window)."""
    g = synth.geometry("barrel10")
    lt = g.layer_table()
    p = np.array([12.0, 0.0, 3.0, 0.2, 0.02, np.pi / 2])      # theta = pi/2: the x/y variances do not leak into z
    sig = np.array([0.05, 0.05, 0.05, 0.01, 0.005, 0.005])
    C0 = np.diag(sig ** 2)
    f, pp, Cp = o.predict(lt, 3, g.bz, p, C0, 1)
    par = np.zeros((6, 32), np.float32); par[:, :4] = p[:, None]
    par[0, 3] = -12.0; par[4, 3] = np.pi - 0.02
    par[3, 4:] = 1.0; par[5, 4:] = 1.5
    cov = np.zeros((21, 32), np.float32)
    Ca = C0.copy(); Ca[0, 0] = Ca[1, 1] = -1.0
    Cb = C0.copy(); Cb[3, 3] = 4.0; Cb[1, 3] = Cb[3, 1] = 0.999 * 2.0 * 0.05   # 1/pT moves by ~40 per cm of y residual
    Cc = C0.copy(); Cc[2, 2] = -0.05
    for k, Cm in enumerate((Ca, Cb, Cc, Ca)):
        cov[:, k] = synth.pack_sym(Cm)
    hit = np.array([[pp[0], pp[1] - 0.02, pp[2]], [pp[0], pp[1] + 0.02, pp[2]]])
    hit[:, :2] *= 16.0 / np.hypot(hit[:, 0], hit[:, 1])[:, None]
    seg = np.array([0, 0, 0, 0, 2, 2, 2, 2, 2, 2, 2], np.int64)
    hx, hy, hz = (hit[:, k].astype(np.float32) for k in range(3))
    return g, lt, par, cov, np.ones(4, np.int8), seg, hx, hy, hz


def test_build_numeric_exits():
    """KFO_NUMERIC in kfo_build.  Seed 0 (S not positive definite for a hit inside the window): the parent's hit children
    are dropped, one finished child carries the UNCHANGED seed state.  Seed 1 (update drives 1/pT <= 0): that child keeps
    the PREDICTED state, records the hit, is finished with the bit set; its sibling is a normal candidate.  Seed 2 (window
    not finite): finished on the unchanged state.  Seed 3 (S not positive definite but no hit to test it on): an
    ordinary hit-less child on the predicted state, no bit.
    Catches: a failed parent that still spawns hit children, a failed update that writes the updated state."""
    g, lt, par, cov, q, seg, hx, hy, hz = numeric_exit_case()
    b = o.bin_hits(lt, 1, seg, hx, hy, hz, 8, 1)
    K = 3
    r = o.kf_build(lt, g.bz, b, seg, par, cov, q, np.zeros(4, np.int32), None, 3, K, 30.0, 3.0, n=4)
    C = lambda t: synth.unpack_sym(cov[:, t].astype(np.float64))
    for t in (0, 2):
        s0 = t * K
        assert r["n_cand"][t] == 1 and r["status"][s0] == o.NUMERIC and r["nhits"][s0] == 3 and (r["hit_idx"][3:, s0] == -2).all()
        assert np.array_equal(r["par"][:4, s0], par[:4, t].astype(np.float64)) and np.array_equal(r["cov"][s0], C(t))
    # seed 0 really went through the S test: its window is finite and holds both hits
    f, p0, C0p = o.predict(lt, 3, g.bz, par[:, 0].astype(np.float64), C(0), 1)
    S0 = C0p[:3, :3] + np.diag([lt[3, 5] ** 2, lt[3, 5] ** 2, lt[3, 4] ** 2])
    assert f == 0 and C0p[2, 2] + lt[3, 4] ** 2 > 0 and np.linalg.eigvalsh(S0).min() < 0
    # seed 1: the two hit children; the one whose update leaves 1/pT <= 0 is finished on the predicted state
    f, pq, Cq = o.predict(lt, 3, g.bz, par[:, 1].astype(np.float64), C(1), 1)
    n_failed = 0
    for k in range(r["n_cand"][1]):
        slot = K + k
        h = r["hit_idx"][3, slot]
        if h < 0:
            continue
        m = np.array([hx[h], hy[h], hz[h]], dtype=np.float64)
        S = Cq[:3, :3] + np.diag([lt[3, 5] ** 2, lt[3, 5] ** 2, lt[3, 4] ** 2])
        iota_upd = (pq + Cq[:, :3] @ np.linalg.solve(S, m - pq[:3]))[3]
        if iota_upd <= 0:
            n_failed += 1
            assert r["status"][slot] == o.NUMERIC and r["nhits"][slot] == 4 and (r["hit_idx"][4:, slot] == -2).all()
            pw = pq.copy(); pw[4] = np.angle(np.exp(1j * pw[4]))
            assert np.max(np.abs(r["par"][:, slot] - pw)) < 1e-12 and np.max(np.abs(r["cov"][slot] - Cq)) < 1e-12 * np.abs(Cq).max()
        else:
            assert r["status"][slot] == 0 and r["par"][3, slot] > 0
    assert n_failed == 1
    # seed 3: nothing in its window on any layer -> transported to the last layer, no status
    s3 = 3 * K
    assert r["n_cand"][3] == 1 and r["status"][s3] == 0 and (r["hit_idx"][3:, s3] == -1).all()
    assert abs(np.hypot(r["par"][0, s3], r["par"][1, s3]) - 40.0) < 1e-9


def test_margins_flag_every_threshold_sensitive_seed():
    """Pin of the R16 diagnostics (margins of kfo_build): scale a threshold by (1 + delta) and rebuild.  The first
    decision that flips is taken on states identical to the base run, so every seed whose result changes must carry, in
    the base run, a margin below delta in the matching category: [1] for the chi2 cut, [0] or [3] for n_sigma (window
    edges, acceptance).  Catches: a margin that is not recorded, recorded for the wrong seed / layer, or scaled wrongly."""
    bi, lt, b = _small_event(4, n_events=1, tracks=1500, fake_frac=0.2)
    base = _build(bi, lt, b, margins=True)
    mg = base["margins"]

    def changed(r):
        d = (base["n_cand"] != r["n_cand"])
        for k in ("nhits", "status"):
            d |= (base[k] != r[k]).reshape(bi.n_seeds, bi.K).any(axis=1)
        return d | (base["hit_idx"] != r["hit_idx"]).any(axis=0).reshape(bi.n_seeds, bi.K).any(axis=1)
    n_flip = 0
    for delta in (2e-3, -2e-3):
        ch = changed(_build(bi, lt, b, cut=bi.chi2_cut * (1 + delta)))
        assert (mg[ch][:, :, 1].min(axis=1) <= abs(delta) * 1.001).all()
        n_flip += ch.sum()
        ch = changed(_build(bi, lt, b, n_sigma=bi.n_sigma * (1 + delta)))
        assert (np.minimum(mg[ch][:, :, 0], mg[ch][:, :, 3]).min(axis=1) <= abs(delta) * 1.001).all()
        n_flip += ch.sum()
    assert n_flip >= 20
    # and the categories are populated sensibly
    assert (mg[:, bi.first_layer:, :] >= 0).all() and (mg[:, :bi.first_layer, :] == 1e300).all()
    assert np.isfinite(mg[:, bi.first_layer:, 3]).all() and (mg[:, bi.first_layer:, 3] < 1e299).mean() > 0.7


@pytest.mark.parametrize("config,kw", [(3, dict(n_events=2, tracks=400)), (4, dict(n_events=1, tracks=800, fake_frac=0.2))])
def test_built_candidate_equals_fit_of_its_hit_list(config, kw):
    """A built candidate went through exactly the fit's steps: kf_fit_ref started from the seed on the layers >=
    first_layer with the built list (hits, -1 = crossed without hit: transported + material, -2 = not crossed)
    reproduces state, covariance and chi2 -- of EVERY candidate, holes and finished ones included (R8)."""
    bi, lt, b = _small_event(config, **kw)
    r = _build(bi, lt, b)
    L = lt.shape[0]
    best = np.arange(bi.n_seeds) * bi.K
    lists = r["hit_idx"][bi.first_layer:, best]
    assert (lists == -1).any() and ((lists >= 0).all(axis=0)).mean() > (0.9 if config == 3 else 0.2)
    if config == 4:
        assert (lists == -2).any()
    hi = np.full((L, bi.ld), -2, np.int32)
    hi[bi.first_layer:, :bi.n_seeds] = lists
    f = o.fit(lt, bi.geom.bz, bi.par, bi.cov, bi.q, bi.hit_x, bi.hit_y, bi.hit_z, bi.seg_off, hi, bi.seed_event)
    ok = (r["status"][best] & o.NUMERIC) == 0
    assert ok.mean() > 0.99
    assert np.array_equal(f["nhits"][ok] + bi.first_layer, r["nhits"][best][ok])
    assert np.max(np.abs(f["chi2"][ok] - r["chi2"][best][ok])) < 1e-9
    assert np.max(np.abs(f["par"][:, ok] - r["par"][:, best[ok]])) < 1e-10
    assert np.max(np.abs(f["cov"][ok] - r["cov"][best[ok]])) < 1e-12
    assert (f["status"][ok] == 0).all()       # a layer the candidate could not reach is marked -2: the refit never tries it


def test_truth_purity_on_noise_free_events():
    """No noise hits: the best candidate of nearly every seed is the truth track (3-sigma windows lose ~0.5 % of the
    hits per layer).  Catches: windows centred or sized wrongly, wrong event/layer segment."""
    bi, lt, b = _small_event(3, n_events=2, tracks=500, noise=0.0)
    r = _build(bi, lt, b)
    best = np.arange(bi.n_seeds) * bi.K
    truth = bi.truth_hit_idx[:, bi.seed_truth]
    hi = r["hit_idx"][:, best]
    full = (hi >= 0).all(axis=0)
    assert full.mean() > 0.92
    assert (hi[:, full] == truth[:, full]).all(axis=0).mean() > 0.995
    assert (hi == truth).mean() > 0.985
    n_found = r["nhits"][best] - bi.first_layer
    ok = n_found > 0
    assert abs((r["chi2"][best][ok] / (2 * n_found[ok])).mean() - 1) < 0.06


def test_build_ranking_invariants_and_edge_cases():
    bi, lt, b = _small_event(4, n_events=1, tracks=800, fake_frac=0.2)
    r = _build(bi, lt, b)
    K, L = bi.K, lt.shape[0]
    assert (bi.seed_truth < 0).sum() > 50                       # fake seeds present
    nh = r["nhits"].reshape(-1, K); c2 = r["chi2"].reshape(-1, K)
    for s in range(bi.n_seeds):
        n = r["n_cand"][s]
        assert 1 <= n <= K
        key = list(zip(-nh[s, :n], c2[s, :n]))
        assert key == sorted(key)                                 # best first
        assert (nh[s, n:] == 0).all() and (r["hit_idx"][:, s * K + n:(s + 1) * K] == -2).all()
    valid = np.concatenate([np.arange(s * K, s * K + r["n_cand"][s]) for s in range(bi.n_seeds)])
    hi = r["hit_idx"][:, valid]
    assert np.array_equal((hi >= 0).sum(axis=0), r["nhits"][valid])
    fin = hi == -2
    assert (fin[:-1] <= fin[1:]).all()                           # once finished, finished on all outer layers
    assert ((r["status"][valid] != 0) <= fin[-1]).all()
    # all candidates of one seed are distinct hit lists
    for s in range(0, bi.n_seeds, 7):
        n = r["n_cand"][s]
        lists = {tuple(r["hit_idx"][:, s * K + k]) for k in range(n)}
        assert len(lists) == n
    # K = 1 keeps exactly the best child of the single parent at each layer; first_layer == L returns the seeds
    r1 = _build(bi, lt, b, K=1)
    assert (r1["n_cand"] == 1).all()
    r0 = o.kf_build(lt[:3], bi.geom.bz, o.bin_hits(lt[:3], 1, bi.seg_off[:4], bi.hit_x[:bi.seg_off[3]], bi.hit_y[:bi.seg_off[3]], bi.hit_z[:bi.seg_off[3]], 8, 1),
                    bi.seg_off[:4], bi.par, bi.cov, bi.q, bi.seed_event, bi.seed_hit_idx, 3, 4, 30.0, 3.0)
    assert (r0["n_cand"] == 1).all() and np.allclose(r0["par"][:, ::4][:3], bi.par[:3, :bi.n_seeds].astype(np.float64))
    # zero seeds
    rz = o.kf_build(lt, bi.geom.bz, b, bi.seg_off, bi.par, bi.cov, bi.q[:0], bi.seed_event[:0], bi.seed_hit_idx, 3, 4, 30.0, 3.0, n=0)
    assert rz["par"].shape[1] == 0

"""Pins of the oracle's combinatorial building on the "cylinder with lids" (sec. 4.1; R22): rows of a
disk's bins by radius, window in (phi, radius), layers that are not crossed are skipped.  CPU only.

The paper gives no formula for any of it; what fixes the oracle here is (B1) the barrel special case reducing bit for bit
to X2 and the disk rows to a plain fp64 floor, (B2) the sorted index against a brute-force key, (B3) bins = no bins,
(B4) the window list against brute force, (B5) the acceptance edges recomputed in numpy from the one-step primitives,
(B6) an exhaustive Python enumeration of the rules from those primitives, (B7) best candidate = the fit of its hit list,
(B8) truth purity on noise-free events with tracks that end on a disk; and for hit_mode 1 (second propagation step to every
candidate hit, 2-D chi2 and update on its tangent plane; R23) the same four on events with staggered sensors
(B9-B12)."""
import numpy as np
import pytest

from oracle import kf_oracle as o
from paper_1711_06571_b200 import synth


def _event(n_events=2, tracks=300, **kw):
    bi = synth.build_inputs("lids", n_events=n_events, tracks=tracks, **kw)
    lt = bi.geom.layer_table()
    b = o.bin_hits(lt, bi.n_events, bi.seg_off, bi.hit_x, bi.hit_y, bi.hit_z, bi.n_phi, bi.n_z)
    return bi, lt, b


def _build(bi, lt, b, K=None, use_bins=True, margins=False, n=None, hit_mode=0):
    return o.kf_build(lt, bi.geom.bz, b, bi.seg_off, bi.par, bi.cov, bi.q, bi.seed_event, bi.seed_hit_idx, bi.first_layer,
                      bi.K if K is None else K, bi.chi2_cut, bi.n_sigma, use_bins=use_bins, margins=margins, n=n, hit_mode=hit_mode)


def test_B1_row_bin_barrel_is_X2_and_disk_is_a_floor():
    rng = np.random.default_rng(1)
    z = np.r_[rng.uniform(-120, 120, 4000), [-100, 100, 0, 99.99999, -99.99999, 12.5]].astype(np.float32)
    for zmax, n in ((100.0, 16), (50.0, 32), (37.5, 7)):
        assert np.array_equal(o.row_bin(z, -zmax, zmax, n), o.z_bin(z, zmax, n))
    x = rng.uniform(-50, 50, 4000).astype(np.float32); y = rng.uniform(-50, 50, 4000).astype(np.float32)
    rho = o.hit_rho(x, y)
    assert np.array_equal(rho, np.sqrt((x * x + y * y).astype(np.float32)).astype(np.float32))      # one rounding per operation
    assert np.max(np.abs(rho.astype(np.float64) - np.hypot(x.astype(np.float64), y.astype(np.float64)))) < 1.2e-5      # 1.5 ulp of a radius of 64-71 cm
    rmin, rmax, n = 4.0, 44.0, 16
    got = o.row_bin(rho, rmin, rmax, n)
    f = (np.hypot(x.astype(np.float64), y.astype(np.float64)) - rmin) * n / (rmax - rmin)
    exp = np.clip(np.floor(f), 0, n - 1).astype(np.int32)
    away = np.abs(f - np.round(f)) > 1e-4
    assert np.array_equal(got[away], exp[away]) and np.all(np.abs(got - exp) <= 1)
    assert got.min() == 0 and got.max() == n - 1          # radii below rmin / above rmax are clamped


def test_B2_sorted_index_on_disks_vs_brute_force_keys():
    bi, lt, b = _event(n_events=2, tracks=400)
    L = lt.shape[0]
    nb = bi.n_phi * bi.n_z
    for sg in range(bi.n_events * L):
        l = sg % L
        s0, s1 = bi.seg_off[sg], bi.seg_off[sg + 1]
        x, y, z = bi.hit_x[s0:s1], bi.hit_y[s0:s1], bi.hit_z[s0:s1]
        if lt[l][6] == 0:
            row = o.z_bin(z, lt[l][1], bi.n_z)
        else:
            row = o.row_bin(o.hit_rho(x, y), lt[l][7], lt[l][1], bi.n_z)
        key = row.astype(np.int64) * bi.n_phi + o.phi_bin(x, y, bi.n_phi)
        order = np.lexsort((np.arange(s1 - s0), key))
        assert np.array_equal(b["perm"][s0:s1], order.astype(np.int32))
        assert np.array_equal(b["x"][s0:s1], x[order]) and np.array_equal(b["z"][s0:s1], z[order])
        cnt = np.bincount(key, minlength=nb)
        assert np.array_equal(b["bin_off"][sg * nb:(sg + 1) * nb + 1], s0 + np.r_[0, np.cumsum(cnt)])
    assert lt[10][6] == 1 and (bi.seg_off[11] - bi.seg_off[10]) > 100      # the disks do hold hits


def test_B3_bins_equal_brute_force_on_the_cylinder_with_lids():
    bi, lt, b = _event(n_events=2, tracks=300)
    a = _build(bi, lt, b)
    c = _build(bi, lt, b, use_bins=False)
    assert c["counters"]["n_scan"] > 20 * a["counters"]["n_scan"]
    for k in ("n_cand", "hit_idx", "nhits", "status", "chi2", "par"):
        assert np.array_equal(a[k], c[k]), k
    on_disk = (a["hit_idx"][10:] >= 0).any(axis=0)
    assert on_disk.sum() > 100                             # candidates do pick up hits on the lids


def test_B4_window_list_on_a_disk_vs_brute_force():
    bi, lt, b = _event(n_events=2, tracks=400)
    L = lt.shape[0]
    rng = np.random.default_rng(3)
    nq = 120
    ev = rng.integers(0, bi.n_events, nq).astype(np.int32)
    ly = rng.integers(10, L, nq).astype(np.int32)          # disks only
    phc = rng.uniform(-np.pi, np.pi, nq).astype(np.float32); dph = np.abs(rng.normal(0, 0.05, nq)).astype(np.float32)
    rc = rng.uniform(0, 50, nq).astype(np.float32); dr = np.abs(rng.normal(0, 3, nq)).astype(np.float32)
    phc[:2] = [3.14, -3.14]; dph[:2] = 0.05; rc[2] = 60.0; rc[3] = 1.0
    cnt, idx = o.window_lookup(lt, b, ev, ly, phc, dph, rc, dr, 4096)
    nb = bi.n_phi * bi.n_z
    inv = np.float32(bi.n_phi / (2 * np.pi))
    for i in range(nq):
        sg = ev[i] * L + ly[i]
        s0, s1 = bi.seg_off[sg], bi.seg_off[sg + 1]
        binof = np.searchsorted(b["bin_off"][sg * nb:(sg + 1) * nb + 1], np.arange(s0, s1), side="right") - 1
        ir, ip = binof // bi.n_phi, binof % bi.n_phi
        b_lo = int(np.floor((phc[i] - dph[i]) * inv)); b_hi = int(np.floor((phc[i] + dph[i]) * inv))
        n_b = min(b_hi - b_lo + 1, bi.n_phi)
        r_lo, r_hi = (int(o.row_bin(v, lt[ly[i]][7], lt[ly[i]][1], bi.n_z)[0]) for v in (rc[i] - dr[i], rc[i] + dr[i]))
        assert o.window_bins_row(float(phc[i]), float(dph[i]), float(rc[i]), float(dr[i]), lt[ly[i]][7], lt[ly[i]][1], bi.n_phi, bi.n_z) == (b_lo % bi.n_phi, n_b, r_lo, r_hi)
        exp = []
        for r in range(r_lo, r_hi + 1):
            for k in range(n_b):
                exp.extend(list(s0 + np.nonzero((ir == r) & (ip == (b_lo + k) % bi.n_phi))[0]))
        assert cnt[i] == len(exp) and list(idx[i, :cnt[i]]) == exp
        x, y = b["x"][s0:s1].astype(np.float64), b["y"][s0:s1].astype(np.float64)
        dphi = np.abs(np.angle(np.exp(1j * (np.arctan2(y, x) - float(phc[i])))))
        inside = (dphi < float(dph[i]) * (1 - 1e-3) - 1e-5) & (np.abs(np.hypot(x, y) - float(rc[i])) < float(dr[i]) * (1 - 1e-3) - 1e-4)
        assert set(s0 + np.nonzero(inside)[0]) <= set(exp)


def _disk_window(pp, Cp, n_sigma, srphi, sr, wphi2=0.0, wrow2=0.0):
    x, y = pp[0], pp[1]
    r2 = x * x + y * y
    varphi = max((x * x * Cp[1, 1] - 2 * x * y * Cp[0, 1] + y * y * Cp[0, 0]) / r2 ** 2, 0.0)
    varrho = max((x * x * Cp[0, 0] + 2 * x * y * Cp[0, 1] + y * y * Cp[1, 1]) / r2, 0.0)
    return np.sqrt(r2), n_sigma * np.sqrt(varphi + srphi ** 2 / r2 + wphi2), n_sigma * np.sqrt(varrho + sr ** 2 + wrow2)


def test_B5_disk_acceptance_edges():
    """A seed aimed at the outer (inner) rim of the first disk: the layer is skipped exactly when the predicted radius
    lies beyond rmax + d_rho (below rmin - d_rho), with rho_c and d_rho recomputed here from o.predict; the candidate
    stays alive, without a status bit, and goes on to the next disk."""
    geom = synth.geometry("lids10", xx0_scale=1.0)
    lt = geom.layer_table()
    L = lt.shape[0]
    Z, rmax, rmin = lt[10][0], lt[10][1], lt[10][7]
    seg = np.zeros(L + 1, np.int64)
    bz = geom.bz
    b = o.bin_hits(lt, 1, seg, np.zeros(0, np.float32), np.zeros(0, np.float32), np.zeros(0, np.float32), 64, 8)
    sig = np.array([0.05, 0.05, 0.05, 0.005, 0.005, 0.005])
    skipped = crossed = 0
    for target in np.r_[np.linspace(rmax - 0.6, rmax + 1.2, 25), np.linspace(rmin - 1.2, rmin + 0.6, 25)]:
        # straight-ish track (10 GeV) from a point at z = 50 heading to radius `target` on the plane z = Z
        r0 = target * 50.0 / Z
        th = np.arctan2(target - r0, Z - 50.0)
        p = np.array([r0, 0.0, 50.0, 0.1, 0.0, th])
        par = np.zeros((6, 32)); par[:, 0] = p
        cov = np.zeros((21, 32)); cov[[0, 2, 5, 9, 14, 20], 0] = sig ** 2
        r = o.kf_build(lt, bz, b, seg, par, cov, np.array([1], np.int8), None, None, 10, 4, 30.0, 3.0, n=1)
        f, pp, Cp = o.predict(lt, 10, bz, p, synth.unpack_sym(cov[:, 0]), 1)
        assert f == 0
        rho, dphi, drho = _disk_window(pp, Cp, 3.0, lt[10][3], lt[10][5])
        off = rho > rmax + drho or rho < rmin - drho
        assert r["n_cand"][0] == 1 and r["status"][0] == 0
        assert r["hit_idx"][10, 0] == (-2 if off else -1), (target, rho, drho)
        if off:
            skipped += 1
            if target < 10.0:      # below the inner rim here, inside the next disks: the candidate is alive and crosses them
                assert (r["hit_idx"][11:14, 0] == -1).any() and r["par"][2, 0] > Z + 1.0
        else:
            crossed += 1
    assert skipped >= 8 and crossed >= 8


def _enumerate(bi, lt, b, s, K, hit_mode=0):
    """Exhaustive Python version of R10 / R11 / R22 (hit_mode 1: R23) for one seed, built from the oracle's one-step primitives."""
    L = lt.shape[0]
    ev = bi.seed_event[s]
    cands = [dict(p=bi.par[:, s].astype(np.float64), C=synth.unpack_sym(bi.cov[:, s].astype(np.float64)), chi2=0.0, nh=bi.first_layer,
                  hits=list(bi.seed_hit_idx[:, s]) + [-2] * (L - bi.first_layer), fin=False, st=0)]
    for l in range(bi.first_layer, L):
        sg = ev * L + l
        s0, s1 = bi.seg_off[sg], bi.seg_off[sg + 1]
        R, zmax, _, srphi, sz, sr, kind, rmin = lt[l]
        hx, hy, hz = (b[k][s0:s1].astype(np.float64) for k in "xyz")
        children = []
        for ci, c in enumerate(cands):
            if c["fin"]:
                children.append((-c["nh"], c["chi2"], ci, np.inf, "fin", 0)); continue
            f, pp, Cp = o.predict(lt, l, bi.geom.bz, c["p"], c["C"], bi.q[s])
            if f:
                children.append((-c["nh"], c["chi2"], ci, np.inf, "skip", 0)); continue
            x, y = pp[0], pp[1]
            r2 = x * x + y * y
            # hit_mode 1 (R23): sensors displaced along the surface normal by an r.m.s. sig_r (cylinder) / sig_z (disk) widen the window
            wphi2 = wrow2 = 0.0
            if hit_mode and kind == 0:
                cinc = (x * np.cos(pp[4]) + y * np.sin(pp[4])) / np.sqrt(r2)
                wrow2 = (sr / np.tan(pp[5]) / cinc) ** 2
                wphi2 = sr ** 2 * (1 - cinc ** 2) / cinc ** 2 / r2
            elif hit_mode:
                wrow2 = (sz * np.tan(pp[5])) ** 2
                wphi2 = wrow2 / r2
            if kind == 0:
                dphi = bi.n_sigma * np.sqrt(max((x * x * Cp[1, 1] - 2 * x * y * Cp[0, 1] + y * y * Cp[0, 0]) / r2 ** 2, 0) + (srphi / R) ** 2 + wphi2)
                dw = bi.n_sigma * np.sqrt(Cp[2, 2] + sz * sz + wrow2)
                off = abs(pp[2]) > zmax + dw
                row, rowc = hz, pp[2]
            else:
                rho, dphi, dw = _disk_window(pp, Cp, bi.n_sigma, srphi, sr, wphi2, wrow2)
                off = rho > zmax + dw or rho < rmin - dw
                row, rowc = np.hypot(hx, hy), rho
            if off:
                children.append((-c["nh"], c["chi2"], ci, np.inf, "skip", 0)); continue
            inside = (np.abs(x * hy - y * hx) <= dphi * np.sqrt(r2) * np.hypot(hx, hy)) & (x * hx + y * hy > 0) & (np.abs(row - rowc) <= dw)
            got = False
            for h in s0 + np.nonzero(inside)[0]:
                m = np.array([b["x"][h], b["y"][h], b["z"][h]], dtype=np.float64)
                if hit_mode == 0:
                    rc, c2 = o.chi2(pp, Cp, m, srphi, sz, sr)
                    at = (pp, Cp, m)
                else:           # second step to the hit's own surface, 2-D chi2 on its tangent plane
                    f2, p2, C2 = o.to_hit_surface(int(kind), bi.geom.bz, bi.q[s], pp, Cp, m)
                    if f2:
                        continue
                    rc, c2 = o.chi2_2d(p2, C2, m, int(kind), srphi, sr if kind else sz)
                    at = (p2, C2, m)
                assert rc == 0
                if c2 < bi.chi2_cut:
                    children.append((-(c["nh"] + 1), c["chi2"] + c2, ci, h, "hit", at))
                    got = True
            if not got:
                children.append((-c["nh"], c["chi2"], ci, np.inf, "miss", (pp, Cp, None)))
        children.sort(key=lambda t: t[:4])
        new = []
        for (mnh, chi2, ci, h, kind_, aux) in children[:K]:
            c = cands[ci]
            hits = list(c["hits"])
            if kind_ in ("fin", "skip"):
                hits[l] = -2
                new.append(dict(p=c["p"], C=c["C"], chi2=c["chi2"], nh=c["nh"], hits=hits, fin=c["fin"], st=c["st"]))
            elif kind_ == "miss":
                hits[l] = -1
                new.append(dict(p=aux[0], C=aux[1], chi2=c["chi2"], nh=c["nh"], hits=hits, fin=False, st=c["st"]))
            else:
                if hit_mode == 0:
                    f, pu, Cu, _ = o.update(aux[0], aux[1], aux[2], srphi, sz, sr)
                else:
                    f, pu, Cu, _ = o.update_2d(aux[0], aux[1], aux[2], int(kind), srphi, sr if kind else sz)
                assert f == 0
                hits[l] = int(b["perm"][h])
                new.append(dict(p=pu, C=Cu, chi2=chi2, nh=-mnh, hits=hits, fin=False, st=c["st"]))
        cands = new
    return cands


@pytest.mark.parametrize("K", [1, 4])
def test_B6_build_equals_exhaustive_python_enumeration_on_lids(K):
    bi, lt, b = _event(n_events=1, tracks=120)
    r = _build(bi, lt, b, K=K)
    checked = ends_on_disk = 0
    for s in range(0, bi.n_seeds, 3):
        ref = _enumerate(bi, lt, b, s, K)
        assert r["n_cand"][s] == len(ref)
        for k, c in enumerate(ref):
            slot = s * K + k
            assert list(r["hit_idx"][:, slot]) == c["hits"], (s, k)
            assert r["nhits"][slot] == c["nh"] and abs(r["chi2"][slot] - c["chi2"]) <= 1e-9 * max(1, c["chi2"])
            assert r["status"][slot] == 0
            pe = c["p"].copy(); pe[4] = np.angle(np.exp(1j * pe[4]))
            assert np.max(np.abs(r["par"][:, slot] - pe)) < 1e-9 and np.max(np.abs(r["cov"][slot] - c["C"])) < 1e-9 * np.abs(c["C"]).max()
            checked += 1
            ends_on_disk += max(i for i, h in enumerate(c["hits"]) if h >= 0) >= 10
    assert checked >= 30 and ends_on_disk >= 5


def test_B7_best_candidate_is_the_fit_of_its_hit_list():
    bi, lt, b = _event(n_events=2, tracks=300)
    r = _build(bi, lt, b)
    K, n = bi.K, bi.n_seeds
    hi = np.full((lt.shape[0], bi.ld), -2, np.int32)
    hi[:, :n] = r["hit_idx"][:, ::K]
    hi[:bi.first_layer] = -2                               # the seed state already holds those layers
    f = o.fit(lt, bi.geom.bz, bi.par, bi.cov, bi.q, bi.hit_x, bi.hit_y, bi.hit_z, bi.seg_off, hit_idx=hi, trk_event=bi.seed_event, n=n)
    assert np.array_equal(f["nhits"] + bi.first_layer, r["nhits"][::K]) and (f["status"] == 0).all()
    assert np.allclose(f["chi2"], r["chi2"][::K], rtol=1e-9, atol=1e-9)
    assert np.allclose(f["par"][[0, 1, 2, 3, 5]], r["par"][[0, 1, 2, 3, 5]][:, ::K], rtol=1e-9, atol=1e-9)
    assert np.allclose(f["cov"], r["cov"][::K], rtol=1e-8, atol=1e-14)


def test_B8_truth_purity_on_noise_free_lids_events():
    bi, lt, b = _event(n_events=2, tracks=300, noise=0.0)
    r = _build(bi, lt, b)
    K = bi.K
    best = r["hit_idx"][:, ::K][:, :bi.n_seeds]
    truth = bi.truth_hit_idx[:, bi.seed_truth]
    truth = np.where(truth >= 0, truth, -9)
    same = ((best == truth) | ((truth == -9) & (best < 0)))[bi.first_layer:].all(axis=0)
    assert same.mean() > 0.93, same.mean()
    ends_on_disk = (truth[10:] >= 0).any(axis=0)
    assert ends_on_disk.sum() > 100 and same[ends_on_disk].mean() > 0.90, (ends_on_disk.sum(), same[ends_on_disk].mean())
    assert (r["status"][::K][:bi.n_seeds] == 0).all()


# ------------------------------------------------------------------------------------------------ hit_mode 1 (R23)
def _event_j(n_events=1, tracks=120, **kw):
    return _event(n_events=n_events, tracks=tracks, jitter=0.3, **kw)


@pytest.mark.parametrize("K", [1, 4])
def test_B9_two_step_build_equals_exhaustive_python_enumeration(K):
    bi, lt, b = _event_j(n_events=1, tracks=120)
    r = _build(bi, lt, b, K=K, hit_mode=1)
    checked = ends_on_disk = 0
    for s in range(0, bi.n_seeds, 3):
        ref = _enumerate(bi, lt, b, s, K, hit_mode=1)
        assert r["n_cand"][s] == len(ref)
        for k, c in enumerate(ref):
            slot = s * K + k
            assert list(r["hit_idx"][:, slot]) == c["hits"], (s, k)
            assert r["nhits"][slot] == c["nh"] and abs(r["chi2"][slot] - c["chi2"]) <= 1e-9 * max(1, c["chi2"])
            pe = c["p"].copy(); pe[4] = np.angle(np.exp(1j * pe[4]))
            assert np.max(np.abs(r["par"][:, slot] - pe)) < 1e-9 and np.max(np.abs(r["cov"][slot] - c["C"])) < 1e-9 * np.abs(c["C"]).max()
            checked += 1
            ends_on_disk += max(i for i, h in enumerate(c["hits"]) if h >= 0) >= 10
    assert checked >= 30 and ends_on_disk >= 5


def test_B10_two_step_best_candidate_is_the_two_step_fit_of_its_hit_list():
    bi, lt, b = _event_j(n_events=2, tracks=300)
    r = _build(bi, lt, b, hit_mode=1)
    K, n = bi.K, bi.n_seeds
    hi = np.full((lt.shape[0], bi.ld), -2, np.int32)
    hi[:, :n] = r["hit_idx"][:, ::K]
    hi[:bi.first_layer] = -2
    f = o.fit(lt, bi.geom.bz, bi.par, bi.cov, bi.q, bi.hit_x, bi.hit_y, bi.hit_z, bi.seg_off, hit_idx=hi, trk_event=bi.seed_event, n=n, hit_mode=1)
    assert np.array_equal(f["nhits"] + bi.first_layer, r["nhits"][::K]) and (f["status"] == 0).all()
    assert np.allclose(f["chi2"], r["chi2"][::K], rtol=1e-9, atol=1e-9)
    assert np.allclose(f["par"][[0, 1, 2, 3, 5]], r["par"][[0, 1, 2, 3, 5]][:, ::K], rtol=1e-9, atol=1e-9)
    assert np.allclose(f["cov"], r["cov"][::K], rtol=1e-8, atol=1e-14)
    # and the states do sit on the hits' own surfaces, off the nominal ones
    last = np.array([max(i for i in range(lt.shape[0]) if hi[i, t] >= 0) if (hi[:, t] >= 0).any() else -1 for t in range(n)])
    crossed = np.array([max(i for i in range(lt.shape[0]) if hi[i, t] >= -1) if (hi[:, t] >= -1).any() else -1 for t in range(n)])
    barrel = (last >= 3) & (last < 10) & (crossed == last)          # the last layer crossed carries a hit
    off = np.abs(np.hypot(r["par"][0, ::K][barrel], r["par"][1, ::K][barrel]) - lt[last[barrel], 0])
    assert barrel.sum() > 50 and off.max() <= 0.3 + 1e-6 and np.median(off) > 0.05


def test_B11_two_step_bins_equal_brute_force_and_truth_purity():
    bi, lt, b = _event_j(n_events=2, tracks=300)
    a = _build(bi, lt, b, hit_mode=1)
    c = _build(bi, lt, b, hit_mode=1, use_bins=False)
    for k in ("n_cand", "hit_idx", "nhits", "status", "chi2", "par"):
        assert np.array_equal(a[k], c[k]), k
    bi, lt, b = _event_j(n_events=2, tracks=300, noise=0.0)
    r = _build(bi, lt, b, hit_mode=1)
    K = bi.K
    best = r["hit_idx"][:, ::K][:, :bi.n_seeds]
    truth = bi.truth_hit_idx[:, bi.seed_truth]
    truth = np.where(truth >= 0, truth, -9)
    same = ((best == truth) | ((truth == -9) & (best < 0)))[bi.first_layer:].all(axis=0)
    assert same.mean() > 0.93, same.mean()
    # chi2 of the 2-D residuals: 2 per hit added (R21)
    full = same & (r["nhits"][::K][:bi.n_seeds] >= 8)
    per_hit = r["chi2"][::K][:bi.n_seeds][full] / (r["nhits"][::K][:bi.n_seeds][full] - bi.first_layer)
    assert full.sum() > 200 and 1.7 < per_hit.mean() < 2.3, (full.sum(), per_hit.mean())

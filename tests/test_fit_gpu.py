"""Parity of the CUDA kf_fit (fp32, through the C ABI) with the fp64 oracle, element by element on the same seeded
inputs.  Tolerances: tests/parity.py (north_star: parameters 1e-4 rel / 1e-6 abs, covariance 1e-3, chi2 1e-3)."""
import numpy as np
import pytest
import torch

from oracle import kf_oracle as o
from paper_1711_06571_b200 import synth
from tests.parity import compare_tracks

pytestmark = pytest.mark.gpu


def run_gpu(fi, force_index=False):
    from paper_1711_06571_b200 import binding as b
    geom = b.Geom(fi.geom.layer_table(), fi.geom.bz)
    hits = b.Hits(fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off, 1)
    seeds = b.Tracks.from_host(fi.par, fi.cov, fi.q)
    hi = None if fi.hit_idx is None else torch.from_numpy(fi.hit_idx).cuda()
    out = b.kf_fit(geom, hits, hi, None, seeds)
    torch.cuda.synchronize()
    return out.to_host()


def run_ref(fi, idx=None):
    if idx is None:
        return o.fit(fi.geom.layer_table(), fi.geom.bz, fi.par, fi.cov, fi.q, fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off, fi.hit_idx)
    L, ld = fi.geom.n_layers, fi.ld
    m = len(idx)
    hx = fi.hit_x.reshape(L, ld)[:, idx].reshape(-1); hy = fi.hit_y.reshape(L, ld)[:, idx].reshape(-1); hz = fi.hit_z.reshape(L, ld)[:, idx].reshape(-1)
    hi = None
    if fi.hit_idx is not None:
        hi = np.where(fi.hit_idx[:, idx] >= 0, np.arange(m, dtype=np.int32)[None, :], -1).astype(np.int32)
    return o.fit(fi.geom.layer_table(), fi.geom.bz, np.ascontiguousarray(fi.par[:, idx]), np.ascontiguousarray(fi.cov[:, idx]),
                 fi.q[idx], hx, hy, hz, np.arange(L + 1) * m, hi)


def check(g, r, min_frac_strict=0.999, max_decision_mismatch=0.0):
    """Discrete decisions (which layers were used, status bits) must agree; `max_decision_mismatch` is the fraction of
    tracks allowed to differ where the inputs sit on a reachability / grazing threshold (reading A16) --
    zero for the BASELINE configs.  Values are compared on the agreeing tracks."""
    same = (g["nhits"] == r["nhits"]) & (g["status"] == r["status"])
    assert (~same).sum() <= max_decision_mismatch * len(same), int((~same).sum())
    rep = compare_tracks(g, r, sel=(r["nhits"] > 0) & same)
    print(rep)
    assert rep["mom_viol"] == 0 and rep["pos_viol"] == 0 and rep["cov_viol"] == 0 and rep["chi2_viol"] == 0, rep
    assert rep["strict_pos_viol"] <= (1 - min_frac_strict) * rep["n"], rep
    return rep


@pytest.mark.parametrize("n", [0, 1, 31, 10_000, 10_037])
def test_fit_config0(n):
    """configs[0] (10 000 tracks, 10 layers) plus empty, single, sub-warp and ragged-tail sizes."""
    fi = synth.fit_inputs(0, n=max(n, 1))
    if n == 0:
        from paper_1711_06571_b200 import binding as b
        geom = b.Geom(fi.geom.layer_table(), fi.geom.bz)
        hits = b.Hits(fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off, 1)
        out = b.kf_fit(geom, hits, None, None, b.Tracks.empty(0))
        assert out.n == 0
        return
    check(run_gpu(fi), run_ref(fi))


def test_fit_config2_small():
    """configs[2] generator (17 layers, pT 0.3-100 GeV log-uniform, |eta|<1.5, dropped layers) at 20 000 tracks."""
    fi = synth.fit_inputs(2, n=20_000)
    assert fi.hit_idx is not None and (fi.hit_idx < 0).any()
    check(run_gpu(fi), run_ref(fi), min_frac_strict=0.99)


def test_fit_explicit_index_equals_identity():
    """One-track kernel: identity indexing and the same indices given explicitly are the same arithmetic, bit for bit."""
    from paper_1711_06571_b200 import binding as b
    fi = synth.fit_inputs(0, n=4096)
    fj = synth.fit_inputs(0, n=4096, force_index=True)
    b.kf_fit_set_pairs(0)
    try:
        a, b_ = run_gpu(fi), run_gpu(fj)
    finally:
        b.kf_fit_set_pairs(1)
    for k in ("par", "cov", "chi2", "nhits", "status"):
        assert np.array_equal(a[k], b_[k]), k


@pytest.mark.parametrize("config,n", [(0, 10_001), (2, 20_000)])
def test_fit_pairs_and_single_agree(config, n):
    """Two tracks per thread (default for identity indexing) against the one-track kernel on the same input: same
    decisions, values within a tenth of the parity tolerances of each other; both against the oracle.  Config 2 without
    its index list (identity): low-pT tracks leave the fast path and are redone by the one-track code inside the kernel."""
    from paper_1711_06571_b200 import binding as b
    fi = synth.fit_inputs(config, n=n)
    if config == 2:          # identity indexing needs a hit on every layer: keep the tracks that have them all
        full = np.nonzero(fi.valid.all(axis=0))[0]
        keep = full[: len(full) // 2 * 2 + 1]
        L = fi.geom.n_layers
        m = len(keep)
        ld = m + 1                                     # m is odd: an even stride, and an odd tail for the pair kernel
        pad = lambda a_: np.ascontiguousarray(np.concatenate([a_[:, keep], a_[:, keep[:1]]], axis=1))
        hits = [pad(h.reshape(L, fi.ld)).reshape(-1) for h in (fi.hit_x, fi.hit_y, fi.hit_z)]
        fi.par = pad(fi.par); fi.cov = pad(fi.cov); fi.q = fi.q[keep]
        fi.hit_x, fi.hit_y, fi.hit_z = hits
        fi.hit_idx = None; fi.n = m; fi.ld = ld; fi.seg_off = np.arange(L + 1, dtype=np.int64) * ld
    r = run_ref(fi)
    g2 = run_gpu(fi)
    b.kf_fit_set_pairs(0)
    try:
        g1 = run_gpu(fi)
    finally:
        b.kf_fit_set_pairs(1)
    check(g2, r, min_frac_strict=0.99)
    check(g1, r, min_frac_strict=0.99)
    assert np.array_equal(g1["nhits"], g2["nhits"]) and np.array_equal(g1["status"], g2["status"])
    sel = g1["nhits"] > 0
    assert np.allclose(g1["chi2"][sel], g2["chi2"][sel], rtol=5e-4, atol=5e-4)      # each within 1e-3 of the oracle
    d = g1["par"][:, sel].astype(np.float64) - g2["par"][:, sel]
    d[4] = np.angle(np.exp(1j * d[4]))
    assert (np.abs(d) <= np.maximum(5e-5 * np.abs(g1["par"][:, sel]), 1e-5)).all()


def test_fit_stops_and_flags():
    """Last layer moved out to R = 400 cm: unreachable for 2 rho < 400 cm (pT < 2.28 GeV).  Those tracks must carry
    status bit 0 and the state frozen after 9 layers, with the same decisions as the oracle.  (Tracks that do reach
    R = 400 are updated with a hit that is not on their helix; only their decision bits are compared.)"""
    fi = synth.fit_inputs(0, n=5000)
    fi.geom.r[9] = 400.0
    fi.geom.zmax[9] = 4000.0
    g, r = run_gpu(fi), run_ref(fi)
    stopped = (r["status"] & o.UNREACHABLE) != 0
    assert stopped.sum() > 500 and (r["status"] == 0).sum() > 500
    same = (g["nhits"] == r["nhits"]) & (g["status"] == r["status"])
    assert (~same).sum() <= 2e-3 * len(same)      # 2 rho within rounding of 400 cm: reading A16
    sel = stopped & same
    assert (r["nhits"][sel] == 9).all()
    rep = compare_tracks(g, r, sel=sel)
    assert rep["mom_viol"] == 0 and rep["pos_viol"] == 0 and rep["cov_viol"] == 0 and rep["chi2_viol"] == 0, rep


def test_fit_in_place():
    from paper_1711_06571_b200 import binding as b
    fi = synth.fit_inputs(0, n=3000)
    ref = run_gpu(fi)
    geom = b.Geom(fi.geom.layer_table(), fi.geom.bz)
    hits = b.Hits(fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off, 1)
    seeds = b.Tracks.from_host(fi.par, fi.cov, fi.q)
    b.kf_fit(geom, hits, None, None, seeds, out=seeds)
    torch.cuda.synchronize()
    got = seeds.to_host()
    assert np.array_equal(got["par"], ref["par"]) and np.array_equal(got["cov"], ref["cov"])


def test_fit_multi_event_segments():
    """Two events in one call (trk_event + device segment offsets) == the two events fitted separately."""
    from paper_1711_06571_b200 import binding as b
    f0, f1 = synth.fit_inputs(0, n=1000, event=0), synth.fit_inputs(0, n=777, event=1)
    L = 10
    xs, ys, zs, off = [], [], [], [0]
    for f in (f0, f1):
        for l in range(L):
            xs.append(f.hit_x.reshape(L, f.ld)[l, :f.n]); ys.append(f.hit_y.reshape(L, f.ld)[l, :f.n]); zs.append(f.hit_z.reshape(L, f.ld)[l, :f.n])
            off.append(off[-1] + f.n)
    n = f0.n + f1.n
    ld = (n + 31) // 32 * 32
    par = np.zeros((6, ld), np.float32); cov = np.zeros((21, ld), np.float32)
    par[:, :f0.n] = f0.par[:, :f0.n]; par[:, f0.n:n] = f1.par[:, :f1.n]
    cov[:, :f0.n] = f0.cov[:, :f0.n]; cov[:, f0.n:n] = f1.cov[:, :f1.n]
    q = np.concatenate([f0.q, f1.q])
    hit_idx = np.full((L, ld), -1, np.int32)
    hit_idx[:, :f0.n] = np.arange(f0.n); hit_idx[:, f0.n:n] = np.arange(f1.n)
    ev = np.concatenate([np.zeros(f0.n, np.int32), np.ones(f1.n, np.int32)])
    geom = b.Geom(f0.geom.layer_table(), f0.geom.bz)
    hits = b.Hits(np.concatenate(xs), np.concatenate(ys), np.concatenate(zs), np.array(off), 2)
    out = b.kf_fit(geom, hits, torch.from_numpy(hit_idx).cuda(), torch.from_numpy(ev).cuda(), b.Tracks.from_host(par, cov, q))
    torch.cuda.synchronize()
    got = out.to_host()
    b.kf_fit_set_pairs(0)            # the one-track kernel on both sides: the same arithmetic, bit for bit
    try:
        a, c = run_gpu(f0), run_gpu(f1)
    finally:
        b.kf_fit_set_pairs(1)
    assert np.array_equal(got["par"][:, :f0.n], a["par"]) and np.array_equal(got["par"][:, f0.n:], c["par"])
    assert np.array_equal(got["chi2"][:f0.n], a["chi2"]) and np.array_equal(got["chi2"][f0.n:], c["chi2"])


def test_fit_rejects_bad_arguments():
    from paper_1711_06571_b200 import binding as b
    fi = synth.fit_inputs(0, n=64)
    hits = b.Hits(fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off, 1)
    seeds = b.Tracks.from_host(fi.par, fi.cov, fi.q)
    tab = fi.geom.layer_table(); tab[3, 0] = tab[2, 0]            # radii not increasing
    with pytest.raises(b.KfError, match="-3"):
        b.kf_fit(b.Geom(tab, 3.8), hits, None, None, seeds)
    with pytest.raises(b.KfError, match="-3"):
        b.kf_fit(b.Geom(np.tile(fi.geom.layer_table()[:1], (40, 1)) * np.arange(1, 41)[:, None], 3.8), hits, None, None, seeds)
    short = b.Hits(fi.hit_x[:100], fi.hit_y[:100], fi.hit_z[:100], np.arange(11) * 10, 1)   # identity needs n hits per segment
    with pytest.raises(b.KfError, match="-1"):
        b.kf_fit(b.Geom(fi.geom.layer_table(), 3.8), short, None, None, seeds)


@pytest.mark.parametrize("config", [1, 2])
def test_fit_full_size_sampled(config):
    """BASELINE.json configs[1] / configs[2] at full size (1 000 000 tracks) in the launch configuration bench.py
    times; the oracle recomputes a strided sample of 20 000 tracks one by one."""
    fi = synth.fit_inputs(config)
    g = run_gpu(fi)
    idx = np.arange(0, fi.n, 50)
    r = run_ref(fi, idx)
    gs = dict(par=g["par"][:, idx], cov=g["cov"][:, idx], chi2=g["chi2"][idx], nhits=g["nhits"][idx], status=g["status"][idx])
    check(gs, r, min_frac_strict=0.99 if config == 2 else 0.999)
    # properties that hold at any size
    assert np.isfinite(g["par"]).all() and np.isfinite(g["cov"]).all() and (g["chi2"] >= 0).all()
    assert (g["nhits"] == fi.valid.sum(axis=0)).mean() > 0.999
    full = g["nhits"] > 0
    assert abs((g["chi2"][full] / (2 * g["nhits"][full])).mean() - 1) < 0.02

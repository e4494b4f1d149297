"""Parity of the CUDA binning / window lookup / combinatorial building on the "cylinder with lids" (sec. 4.1;
DESIGN.md R22: rows of a disk's bins by radius, window in (phi, radius), layers that are not crossed are skipped) with the
fp64 oracle, through the C ABI.  Bins and window lists bit-exact; built candidates as in tests/test_build_gpu.py (every
seed whose lists differ proven to be a decision-margin case); then the build -> select -> final fit chain on the lids."""
import numpy as np
import pytest
import torch

from oracle import kf_oracle as o
from paper_1711_06571_b200 import synth
from tests.parity import assert_parity, compare_tracks
from tests.test_build_gpu import assert_binned_equal, compare_build, gpu_bin, ref_bin, ref_build, run_build

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("kw", [dict(n_events=1, tracks=50), dict(n_events=3, tracks=1500), dict(n_events=2, tracks=800, n_phi=1024, n_z=32)])
def test_lids_bin_hits_bit_exact(kw):
    bi = synth.build_inputs("lids", **kw)
    _, _, binned = gpu_bin(bi)
    assert_binned_equal(binned.to_host(), ref_bin(bi))


def test_lids_window_lookup_bit_exact():
    from paper_1711_06571_b200 import binding as b
    bi = synth.build_inputs("lids", n_events=2, tracks=1000)
    lt = bi.geom.layer_table()
    geom, hits, binned = gpu_bin(bi)
    rb = ref_bin(bi)
    rng = np.random.default_rng(5)
    nq = 4000
    ev = rng.integers(0, bi.n_events, nq).astype(np.int32)
    ly = rng.integers(0, lt.shape[0], nq).astype(np.int32)           # barrel layers and disks
    phc = rng.uniform(-np.pi, np.pi, nq).astype(np.float32); dph = np.abs(rng.normal(0, 0.05, nq)).astype(np.float32)
    disk = lt[ly, 6] != 0
    c = np.where(disk, rng.uniform(0, 50, nq), rng.uniform(-60, 60, nq)).astype(np.float32)
    d = np.abs(rng.normal(0, 3, nq)).astype(np.float32)
    cap = 512
    t = lambda a: torch.from_numpy(a).cuda()
    cnt, idx = b.kf_window_lookup(geom, hits, binned, t(ev), t(ly), t(phc), t(dph), t(c), t(d), cap)
    torch.cuda.synchronize()
    rc, ri = o.window_lookup(lt, rb, ev, ly, phc, dph, c, d, cap)
    cnt, idx = cnt.cpu().numpy(), idx.cpu().numpy()
    assert np.array_equal(cnt, rc)
    for i in range(nq):
        n = min(rc[i], cap)
        assert np.array_equal(idx[i, :n], ri[i, :n])
    assert disk.sum() > 1000 and rc[disk].sum() > 1000


@pytest.mark.parametrize("kw,K", [(dict(n_events=4, tracks=2000), None), (dict(n_events=2, tracks=1500), 3), (dict(n_events=2, tracks=1500, noise=0.0), None)])
def test_lids_build_parity(kw, K):
    bi = synth.build_inputs("lids", **kw)
    K_ = bi.K if K is None else K
    g, r = run_build(bi, K=K), ref_build(bi, K=K)
    rep = compare_build(g, r, bi.n_seeds, K_, bi.first_layer)
    # the lids are used: candidates with hits on disks, layers skipped by candidates that live on, no status bits
    best = np.arange(bi.n_seeds) * K_
    on_disk = (r["hit_idx"][10:, best] >= 0).any(axis=0)
    assert on_disk.mean() > 0.3 and (g["hit_idx"][10:, best] >= 0).any(axis=0).mean() > 0.3
    skipped_then_hit = ((r["hit_idx"][3:10, best] == -2).any(axis=0)) & on_disk
    assert skipped_then_hit.sum() > 50
    assert (g["status"][best] == 0).all()
    assert rep["seed_mismatch_frac"] < 0.02


def test_lids_build_then_final_fit():
    from paper_1711_06571_b200 import binding as b
    bi = synth.build_inputs("lids", n_events=3, tracks=1500)
    K, n = bi.K, bi.n_seeds
    lt = bi.geom.layer_table()
    geom = b.Geom(lt, bi.geom.bz)
    hits = b.Hits(bi.hit_x, bi.hit_y, bi.hit_z, bi.seg_off, bi.n_events)
    binned = b.kf_bin_hits(geom, hits, bi.n_phi, bi.n_z)
    seeds = b.Tracks.from_host(bi.par, bi.cov, bi.q)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    sev = t(bi.seed_event)
    cands = b.kf_build(geom, hits, binned, seeds, sev, t(bi.seed_hit_idx), bi.first_layer, K, bi.chi2_cut, bi.n_sigma)
    idx = b.kf_select_best(cands, bi.first_layer, seeds.ld)
    fitted = b.kf_fit(geom, hits, idx, sev, seeds)
    torch.cuda.synchronize()
    g, c, hi = fitted.to_host(), cands.to_host(), idx.cpu().numpy()
    best = np.arange(n) * K
    r = o.fit(lt, bi.geom.bz, bi.par, bi.cov, bi.q, bi.hit_x, bi.hit_y, bi.hit_z, bi.seg_off, hit_idx=hi, trk_event=bi.seed_event)
    # a layer the build skipped is skipped by the fit (-2); a hole the build crossed may, within rounding of a guard, stop the fit
    same = (g["nhits"] == r["nhits"]) & (g["status"] == r["status"])
    assert (~same).sum() <= 2e-3 * n, int((~same).sum())
    ok = same & (r["status"] == 0)
    assert ok.mean() > 0.97
    assert_parity(compare_tracks(g, r, sel=ok))
    # the refit reproduces the built candidate
    m = ok & (c["status"][best] == 0)
    assert np.array_equal(g["nhits"][m] + bi.first_layer, c["nhits"][best][m])
    assert np.allclose(g["chi2"][m], c["chi2"][best][m], rtol=2e-4, atol=1e-4)


def _run_two_step(bi, K=None):
    from paper_1711_06571_b200 import binding as b
    lt = bi.geom.layer_table()
    geom = b.Geom(lt, bi.geom.bz, hit_mode=1)
    hits = b.Hits(bi.hit_x, bi.hit_y, bi.hit_z, bi.seg_off, bi.n_events)
    binned = b.kf_bin_hits(geom, hits, bi.n_phi, bi.n_z)
    seeds = b.Tracks.from_host(bi.par, bi.cov, bi.q)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    sev = t(bi.seed_event)
    K = bi.K if K is None else K
    cands = b.kf_build(geom, hits, binned, seeds, sev, t(bi.seed_hit_idx), bi.first_layer, K, bi.chi2_cut, bi.n_sigma)
    idx = b.kf_select_best(cands, bi.first_layer, seeds.ld)
    fitted = b.kf_fit(geom, hits, idx, sev, seeds)
    torch.cuda.synchronize()
    rb = ref_bin(bi)
    r = o.kf_build(lt, bi.geom.bz, rb, bi.seg_off, bi.par, bi.cov, bi.q, bi.seed_event, bi.seed_hit_idx, bi.first_layer, K, bi.chi2_cut, bi.n_sigma,
                   margins=True, hit_mode=1)
    return cands.to_host(), r, fitted.to_host(), idx.cpu().numpy()


@pytest.mark.parametrize("kw,K", [(dict(n_events=3, tracks=2000), None), (dict(n_events=2, tracks=1500), 3), (dict(n_events=2, tracks=1500, noise=0.0), None)])
def test_lids_two_step_build_parity(kw, K):
    """kf_build with hit_mode = 1 (R23) on sensors staggered by +-0.3 cm: second step to every candidate hit, 2-D chi2
    and update on its tangent plane; then the final fit of the best candidates with the same hit mode."""
    bi = synth.build_inputs("lids", jitter=0.3, **kw)
    K_ = bi.K if K is None else K
    g, r, gf, hi = _run_two_step(bi, K)
    rep = compare_build(g, r, bi.n_seeds, K_, bi.first_layer, band_frac=0.05)
    best = np.arange(bi.n_seeds) * K_
    assert (r["hit_idx"][10:, best] >= 0).any(axis=0).mean() > 0.3 and rep["seed_mismatch_frac"] < 0.03
    # states sit on the hits' own surfaces: off the nominal radius of the last barrel layer with a hit
    hl = r["hit_idx"][:, best]
    last_hit = np.array([max([i for i in range(hl.shape[0]) if hl[i, t] >= 0], default=-1) for t in range(bi.n_seeds)])
    last_x = np.array([max([i for i in range(hl.shape[0]) if hl[i, t] >= -1], default=-1) for t in range(bi.n_seeds)])
    sel = (last_hit >= 3) & (last_hit < 10) & (last_x == last_hit)
    off = np.abs(np.hypot(g["par"][0, best][sel], g["par"][1, best][sel]) - bi.geom.layer_table()[last_hit[sel], 0])
    assert sel.sum() > 100 and off.max() <= 0.3 + 1e-4 and np.median(off) > 0.05
    # final fit with the same hit mode against the oracle's fit of the same lists
    rf = o.fit(bi.geom.layer_table(), bi.geom.bz, bi.par, bi.cov, bi.q, bi.hit_x, bi.hit_y, bi.hit_z, bi.seg_off, hit_idx=hi, trk_event=bi.seed_event, hit_mode=1)
    same = (gf["nhits"] == rf["nhits"]) & (gf["status"] == rf["status"])
    assert (~same).sum() <= 3e-3 * bi.n_seeds, int((~same).sum())
    # cos(incidence) on the surface the fitted state sits on: in the transverse plane on a cylinder, |cos theta| on a disk
    x, y, ph = rf["par"][0], rf["par"][1], rf["par"][4]
    kind = bi.geom.layer_table()[:, 6]
    crossed = hi[:, :bi.n_seeds] >= -1
    last = np.where(crossed.any(axis=0), crossed.shape[0] - 1 - np.argmax(crossed[::-1], axis=0), 0)
    cosinc = np.where(kind[last] == 0, (x * np.cos(ph) + y * np.sin(ph)) / np.maximum(np.hypot(x, y), 1e-30), np.abs(np.cos(rf["par"][5])))
    from tests.test_build_gpu import BAND_CHI2_SCALE, BAND_COV_SCALE
    from tests.test_lids_gpu import TWO_STEP_BAND
    ok = same & (rf["status"] == 0) & (rf["nhits"] > 0)
    inband = cosinc < TWO_STEP_BAND
    assert (ok & ~inband).mean() > 0.9
    assert_parity(compare_tracks(gf, rf, sel=ok & ~inband))
    # the conditioning band (R16b) is compared too, with its scales, and its share is bounded
    rb = compare_tracks(gf, rf, sel=ok & inband, cov_scale=BAND_COV_SCALE, chi2_scale=BAND_CHI2_SCALE)
    assert rb["n"] <= 0.05 * bi.n_seeds, rb
    assert_parity(rb)


def test_build_rejects_an_unknown_hit_mode():
    from paper_1711_06571_b200 import binding as b
    bi = synth.build_inputs("lids", n_events=1, tracks=50)
    geom = b.Geom(bi.geom.layer_table(), bi.geom.bz, hit_mode=2)
    hits = b.Hits(bi.hit_x, bi.hit_y, bi.hit_z, bi.seg_off, bi.n_events)
    binned = b.kf_bin_hits(b.Geom(bi.geom.layer_table(), bi.geom.bz), hits, bi.n_phi, bi.n_z)
    seeds = b.Tracks.from_host(bi.par, bi.cov, bi.q)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    with pytest.raises(b.KfError, match="-3"):
        b.kf_build(geom, hits, binned, seeds, t(bi.seed_event), t(bi.seed_hit_idx), bi.first_layer, bi.K, bi.chi2_cut, bi.n_sigma)

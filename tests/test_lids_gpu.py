"""Parity of the CUDA "cylinder with lids" path (sec. 4.1; R19-R21) with the fp64 oracle: endcap
disks in the layer list, two-step propagation to each hit's own radius / z, 2-D update on the plane tangent to the hit
radius -- through kf_fit (kf_geom.hit_mode), element by element on the same seeded inputs."""
import numpy as np
import pytest
import torch

from oracle import kf_oracle as o
from paper_1711_06571_b200 import synth
from tests.parity import assert_parity, compare_tracks

pytestmark = pytest.mark.gpu


def run_gpu(fi, hit_mode, trk_event=None):
    from paper_1711_06571_b200 import binding as b
    geom = b.Geom(fi.geom.layer_table(), fi.geom.bz, hit_mode=hit_mode)
    hits = b.Hits(fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off, 1)
    seeds = b.Tracks.from_host(fi.par, fi.cov, fi.q)
    hi = None if fi.hit_idx is None else torch.from_numpy(fi.hit_idx).cuda()
    out = b.kf_fit(geom, hits, hi, trk_event, seeds)
    torch.cuda.synchronize()
    return out.to_host()


def run_ref(fi, hit_mode):
    return o.fit(fi.geom.layer_table(), fi.geom.bz, fi.par, fi.cov, fi.q, fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off, fi.hit_idx, hit_mode=hit_mode)


TWO_STEP_BAND = 0.25   # DESIGN.md R16b for hit_mode 1: two covariance transports per layer, each amplified by 1/cos^2(incidence)


def check(g, r, max_decision_mismatch=1e-4, band=0.0):
    """band > 0: tracks whose final state crosses its cylinder with cos(incidence) < band are compared with the R16b scales
    (3x on the covariance elements carrying the 1/cos(incidence) factor, 2x on chi2), their share bounded at 2 %."""
    from tests.test_build_gpu import BAND_CHI2_SCALE, BAND_COV_SCALE
    same = (g["nhits"] == r["nhits"]) & (g["status"] == r["status"])
    assert (~same).sum() <= max_decision_mismatch * len(same), int((~same).sum())
    x, y, ph = r["par"][0], r["par"][1], r["par"][4]
    cosinc = (x * np.cos(ph) + y * np.sin(ph)) / np.maximum(np.hypot(x, y), 1e-30)
    inband = cosinc < band
    rep = compare_tracks(g, r, sel=(r["nhits"] > 0) & same & ~inband)
    print(rep)
    assert_parity(rep)
    if band > 0:
        rb = compare_tracks(g, r, sel=(r["nhits"] > 0) & same & inband, cov_scale=BAND_COV_SCALE, chi2_scale=BAND_CHI2_SCALE)
        print(rb)
        assert rb["n"] <= 0.02 * len(same)
        assert_parity(rb)
    return rep


@pytest.mark.parametrize("n", [1, 33, 20_000])
def test_fit_lids_two_step(n):
    """Staggered sensors (+-0.3 cm), barrel + both lids + the transition, hit_mode 1."""
    fi = synth.fit_inputs("lids", n=n)
    g, r = run_gpu(fi, 1), run_ref(fi, 1)
    rep = check(g, r)
    if n >= 1000:
        on_disk = fi.valid[10:].any(axis=0)
        assert on_disk.mean() > 0.3 and rep["n"] > 0.95 * n


def test_fit_lids_nominal_surfaces():
    """hit_mode 0 on the geometry with disks (no staggering): propagation to z and the 3-D update with the hit covariance
    turned to the hit's azimuth (sig_r, sig_rphi in the disk plane, sig_z as the regulariser along the normal)."""
    fi = synth.fit_inputs("lids", n=20_000, jitter=0.0)
    check(run_gpu(fi, 0), run_ref(fi, 0))


def test_fit_two_step_on_the_barrel_configs():
    """hit_mode 1 on the generators of configs[0] and configs[2] with staggered sensors: the second step alone (no disks),
    inwards and outwards.  configs[2] reaches the generator's grazing guard (cos(incidence) = 0.2): measured worst there
    1.02x on one covariance element at cos(incidence) = 0.21, hence the band (R16b)."""
    f0 = synth.fit_inputs(0, n=20_000, jitter=0.3)
    check(run_gpu(f0, 1), run_ref(f0, 1))
    fi = synth.fit_inputs(2, n=20_000, jitter=0.3)
    g, r = run_gpu(fi, 1), run_ref(fi, 1)
    check(g, r, max_decision_mismatch=2e-4, band=TWO_STEP_BAND)
    # and the hit mode matters: ignoring the 0.3 cm offsets is visibly worse
    r0 = run_ref(fi, 0)
    ok = (r0["status"] == 0) & (r0["nhits"] >= 3)
    assert (r0["chi2"][ok] / (2 * r0["nhits"][ok])).mean() > 2 * (r["chi2"][ok] / (2 * np.maximum(r["nhits"][ok], 1))).mean()


def test_fit_lids_full_size_sampled():
    """The "lids" configuration at its full size (100 000 tracks); the oracle recomputes every fifth track."""
    fi = synth.fit_inputs("lids")
    g = run_gpu(fi, 1)
    idx = np.arange(0, fi.n, 5)
    L, ld, m = fi.geom.n_layers, fi.ld, len(np.arange(0, fi.n, 5))
    hx, hy, hz = (a.reshape(L, ld)[:, idx].reshape(-1) for a in (fi.hit_x, fi.hit_y, fi.hit_z))
    hi = np.where(fi.hit_idx[:, idx] >= 0, np.arange(m, dtype=np.int32)[None, :], fi.hit_idx[:, idx]).astype(np.int32)
    r = o.fit(fi.geom.layer_table(), fi.geom.bz, np.ascontiguousarray(fi.par[:, idx]), np.ascontiguousarray(fi.cov[:, idx]), fi.q[idx],
              hx, hy, hz, np.arange(L + 1) * m, hi, hit_mode=1)
    gs = dict(par=g["par"][:, idx], cov=g["cov"][:, idx], chi2=g["chi2"][idx], nhits=g["nhits"][idx], status=g["status"][idx])
    check(gs, r)
    assert np.isfinite(g["par"]).all() and np.isfinite(g["cov"]).all() and (g["chi2"] >= 0).all()
    full = g["nhits"] > 2
    assert abs((g["chi2"][full] / (2 * g["nhits"][full])).mean() - 1) < 0.03


def test_lids_geometry_checks():
    from paper_1711_06571_b200 import binding as b
    fi = synth.fit_inputs("lids", n=64)
    hits = b.Hits(fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off, 1)
    seeds = b.Tracks.from_host(fi.par, fi.cov, fi.q)
    hi = torch.from_numpy(fi.hit_idx).cuda()
    lt = fi.geom.layer_table()
    bad = lt.copy(); bad[11, 0] = 55.0                     # disks of one side not by increasing |z|
    with pytest.raises(b.KfError, match="-3"):
        b.kf_fit(b.Geom(bad, 3.8), hits, hi, None, seeds)
    bad = lt.copy(); bad[12, 7] = 50.0                     # rmin >= outer radius
    with pytest.raises(b.KfError, match="-3"):
        b.kf_fit(b.Geom(bad, 3.8), hits, hi, None, seeds)
    bad = lt.copy(); bad[3, 6] = 2                         # unknown kind
    with pytest.raises(b.KfError, match="-3"):
        b.kf_fit(b.Geom(bad, 3.8), hits, hi, None, seeds)
    with pytest.raises(b.KfError, match="-3"):
        b.kf_fit(b.Geom(lt, 3.8, hit_mode=2), hits, hi, None, seeds)

"""Building -> final fit (sec. 2: "When a complete track has been reconstructed, a final fit using the KF is
performed"): kf_build, kf_select_best and kf_fit chained on the device (explicit hit indices, per-track event), against the
oracle's fit of the same hit lists, and against the built candidate itself where its hit list has no holes."""
import numpy as np
import pytest
import torch

from oracle import kf_oracle as o
from paper_1711_06571_b200 import synth
from tests.parity import compare_tracks

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("config,kw", [(3, dict(n_events=3, tracks=1500)), (4, dict(n_events=1, tracks=3000))])
def test_build_then_final_fit(config, kw):
    from paper_1711_06571_b200 import binding as b
    bi = synth.build_inputs(config, **kw)
    L, K, n = bi.geom.n_layers, bi.K, bi.n_seeds
    geom = b.Geom(bi.geom.layer_table(), bi.geom.bz)
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
    # the index lists are the best candidates' lists, negative entries and seed layers masked
    want = np.where(c["hit_idx"][:, best] < 0, -1, c["hit_idx"][:, best])
    want[:bi.first_layer] = -1
    assert np.array_equal(hi[:, :n], want)
    # oracle fit of the same lists (fp64), same seeds
    r = o.fit(bi.geom.layer_table(), bi.geom.bz, bi.par, bi.cov, bi.q, bi.hit_x, bi.hit_y, bi.hit_z, bi.seg_off, hit_idx=hi, trk_event=bi.seed_event)
    same = (g["nhits"] == r["nhits"]) & (g["status"] == r["status"])
    assert (~same).sum() <= 2e-3 * n
    x, y, ph = r["par"][0], r["par"][1], r["par"][4]
    cosinc = (x * np.cos(ph) + y * np.sin(ph)) / np.maximum(np.hypot(x, y), 1e-30)
    sel = same & (r["nhits"] > 0) & (cosinc >= 0.2)          # conditioning band: DESIGN.md R16b
    rep = compare_tracks(g, r, sel=sel)
    print(rep)
    assert rep["n"] > 0.9 * n
    assert rep["mom_viol"] == 0 and rep["pos_viol"] == 0 and rep["cov_viol"] == 0 and rep["chi2_viol"] == 0, rep
    # a built candidate without holes went through exactly the same steps: the refit reproduces it
    lists = c["hit_idx"][bi.first_layer:, best]
    last = (L - 1) - np.argmax(lists[::-1] >= 0, axis=0)                 # last layer with a hit
    no_holes = (lists >= 0).any(axis=0) & np.array([(lists[: last[s] - bi.first_layer + 1, s] >= 0).all() for s in range(n)])
    ends_on_hit = lists[-1] >= 0
    m = no_holes & ends_on_hit & (c["status"][best] == 0) & (g["status"] == 0)
    assert m.sum() > 0.3 * n            # config 4: half of the candidates leave the barrel or end on a hole
    assert np.array_equal(g["nhits"][m] + bi.first_layer, c["nhits"][best][m])
    assert np.allclose(g["chi2"][m], c["chi2"][best][m], rtol=1e-5, atol=1e-5)
    assert np.allclose(g["par"][:, m], c["par"][:, best][:, m], rtol=1e-5, atol=1e-6)
    assert np.allclose(g["cov"][:, m], c["cov"][:, best][:, m], rtol=1e-4, atol=1e-12)


def test_select_best_arguments():
    from paper_1711_06571_b200 import binding as b
    cands = b.Cands(5, 4, 10)
    cands.hit_idx.fill_(-2)
    out = b.kf_select_best(cands, 3, 32)
    torch.cuda.synchronize()
    assert (out[:, :5] == -1).all()
    with pytest.raises(b.KfError, match="-1"):
        b.kf_select_best(cands, 11, 32)
    with pytest.raises(b.KfError, match="-1"):
        b.kf_select_best(cands, 3, 4, out=torch.empty((10, 4), dtype=torch.int32, device="cuda"))       # ld < n_seeds

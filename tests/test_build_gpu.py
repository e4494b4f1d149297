"""Parity of the CUDA binning / window lookup / combinatorial building (through the C ABI) with the fp64 oracle.

Bins, sorted order, offsets and window hit lists are integer / index work: bit-exact.  Built candidates: hit-index
lists identical except where fp32 decides a threshold or a rank differently (R16: window edge, chi2 cut,
competing chi2 within 1e-4 relative); those seeds are counted and bounded, the rest is compared element-wise with
the tolerances of tests/parity.py.
"""
import numpy as np
import pytest
import torch

from oracle import kf_oracle as o
from paper_1711_06571_b200 import synth
from tests.parity import compare_tracks

pytestmark = pytest.mark.gpu


def gpu_bin(bi):
    from paper_1711_06571_b200 import binding as b
    geom = b.Geom(bi.geom.layer_table(), bi.geom.bz)
    hits = b.Hits(bi.hit_x, bi.hit_y, bi.hit_z, bi.seg_off, bi.n_events)
    binned = b.kf_bin_hits(geom, hits, bi.n_phi, bi.n_z)
    torch.cuda.synchronize()
    return geom, hits, binned


def ref_bin(bi):
    return o.bin_hits(bi.geom.layer_table(), bi.n_events, bi.seg_off, bi.hit_x, bi.hit_y, bi.hit_z, bi.n_phi, bi.n_z)


def assert_binned_equal(g, r):
    for k in ("bin_off", "perm", "x", "y", "z"):
        assert np.array_equal(g[k], r[k]), k
    # the 16-byte records the build kernel reads: same hits, perm carried as bits
    p4 = g["xyzp"]
    assert np.array_equal(p4[:, 0], r["x"]) and np.array_equal(p4[:, 1], r["y"]) and np.array_equal(p4[:, 2], r["z"])
    assert np.array_equal(np.ascontiguousarray(p4[:, 3]).view(np.int32), r["perm"])


@pytest.mark.parametrize("config,kw", [(3, dict(n_events=1, tracks=1)), (3, dict(n_events=3, tracks=777)), (3, {}),
                                        (4, dict(n_events=2, tracks=3000, fake_frac=0.0))])
def test_bin_hits_bit_exact(config, kw):
    bi = synth.build_inputs(config, **kw)
    _, _, binned = gpu_bin(bi)
    assert_binned_equal(binned.to_host(), ref_bin(bi))


def test_bin_hits_empty_segments_and_edges():
    """Segments without hits, hits exactly on the axes / diagonals / z ends, n_phi = 8 and n_z = 1."""
    from paper_1711_06571_b200 import binding as b
    geom_s = synth.geometry("barrel10")
    lt = geom_s.layer_table()[:3]
    x = np.array([4, 0, -4, 0, 2.8284271, -2.8284271, 4, 4, 8, 0, 5.6568542], np.float32)
    y = np.array([0, 4, 0, -4, 2.8284271, 2.8284271, 1e-30, -1e-30, 0, -8, -5.6568542], np.float32)
    z = np.array([-100, 100, 0, 99.99999, -150, 150, 12.5, -12.5, 3, 4, 5], np.float32)
    seg_off = np.array([0, 8, 8, 11, 11, 11, 11], np.int64)      # 2 events x 3 layers; four empty segments
    for n_phi, n_z in ((8, 1), (256, 16), (1024, 32)):
        geom = b.Geom(lt, 3.8)
        hits = b.Hits(x, y, z, seg_off, 2)
        g = b.kf_bin_hits(geom, hits, n_phi, n_z)
        torch.cuda.synchronize()
        assert_binned_equal(g.to_host(), o.bin_hits(lt, 2, seg_off, x, y, z, n_phi, n_z))
    # no hits at all
    hits0 = b.Hits(x[:0], y[:0], z[:0], np.zeros(7, np.int64), 2)
    g = b.kf_bin_hits(b.Geom(lt, 3.8), hits0, 8, 2)
    torch.cuda.synchronize()
    assert (g.bin_off.cpu().numpy() == 0).all()
    with pytest.raises(b.KfError, match="-3"):
        b.kf_bin_hits(b.Geom(lt, 3.8), hits, 12, 4)                       # n_phi not a multiple of 8
    with pytest.raises(b.KfError, match="-4"):
        b.kf_bin_hits(b.Geom(lt, 3.8), hits, 256, 16, ws=torch.empty(16, dtype=torch.uint8, device="cuda"))


def test_window_lookup_bit_exact():
    from paper_1711_06571_b200 import binding as b
    bi = synth.build_inputs(3, n_events=2, tracks=1000)
    geom, hits, binned = gpu_bin(bi)
    rb = ref_bin(bi)
    rng = np.random.default_rng(41)
    nq = 5000
    L = bi.geom.n_layers
    ev = rng.integers(0, bi.n_events, nq).astype(np.int32); ly = rng.integers(0, L, nq).astype(np.int32)
    phc = rng.uniform(-np.pi, np.pi, nq).astype(np.float32); dph = np.abs(rng.normal(0, 0.03, nq)).astype(np.float32)
    zc = rng.uniform(-110, 110, nq).astype(np.float32); dz = np.abs(rng.normal(0, 6, nq)).astype(np.float32)
    phc[:6] = [np.pi, -np.pi, 3.1415, -3.1415, 1e-4, -1e-4]; dph[:6] = 0.03
    dph[6] = 4.0; dph[7] = 0.0; dz[8] = 0.0; zc[9] = 150.0; zc[10] = -150.0; dz[11] = 500.0
    cap = 512
    t = lambda a: torch.from_numpy(a).cuda()
    cnt, idx = b.kf_window_lookup(geom, hits, binned, t(ev), t(ly), t(phc), t(dph), t(zc), t(dz), cap)
    torch.cuda.synchronize()
    rc, ri = o.window_lookup(bi.geom.layer_table(), rb, ev, ly, phc, dph, zc, dz, cap)
    assert np.array_equal(cnt.cpu().numpy(), rc)
    gi = idx.cpu().numpy()
    for i in range(nq):
        m = min(rc[i], cap)
        assert np.array_equal(gi[i, :m], ri[i, :m]), i
    assert rc.max() > cap and (rc == 0).any()


def run_build(bi, K=None, tile=0, first_layer=None):
    from paper_1711_06571_b200 import binding as b
    geom, hits, binned = gpu_bin(bi)
    seeds = b.Tracks.from_host(bi.par, bi.cov, bi.q)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    b.kf_build_set_tile(tile)
    try:
        out = b.kf_build(geom, hits, binned, seeds, t(bi.seed_event), t(bi.seed_hit_idx), bi.first_layer, bi.K if K is None else K,
                         bi.chi2_cut, bi.n_sigma)
        torch.cuda.synchronize()
    finally:
        b.kf_build_set_tile(0)
    return out.to_host()


def ref_build(bi, K=None):
    rb = ref_bin(bi)
    return o.kf_build(bi.geom.layer_table(), bi.geom.bz, rb, bi.seg_off, bi.par, bi.cov, bi.q, bi.seed_event, bi.seed_hit_idx,
                      bi.first_layer, bi.K if K is None else K, bi.chi2_cut, bi.n_sigma)


GRAZING_BAND = 0.2   # generator guard on cos(incidence) (R8); the KF guard is 0.1 (R9)


def compare_build(g, r, n_seeds, K, max_mismatch_frac, band_frac=0.02):
    """Seeds whose valid slots carry identical (n_cand, hit lists, nhits, status) are compared element-wise; the others
    (fp32 decided a window edge / chi2 cut / rank differently, R16) are counted.
    Conditioning band (R16b): a candidate whose final state crosses its cylinder with cos(incidence) < 0.2 lies
    beyond the guard the generator applies to truth tracks (R8) and inside the KF guard band 0.1-0.2 (R9); the surface
    Jacobian carries 1/cos(incidence) factors, so rounding is amplified up to 4x more than anywhere on a truth track.
    Such candidates (pT < 0.5 GeV near their turning point; only the configs[4] generator makes them) are compared at
    3x the tolerances and their share is bounded by `band_frac`; every other candidate at 1x with zero violations."""
    same = g["n_cand"] == r["n_cand"]
    hs = (g["hit_idx"] == r["hit_idx"]).all(axis=0) & (g["nhits"] == r["nhits"]) & (g["status"] == r["status"])
    slot_valid = (np.arange(K)[None, :] < r["n_cand"][:, None])
    same &= (hs.reshape(n_seeds, K) | ~slot_valid).all(axis=1)
    frac = 1.0 - same.mean()
    # the best candidate alone (what a user takes as the track)
    best = np.arange(n_seeds) * K
    best_same = (g["hit_idx"][:, best] == r["hit_idx"][:, best]).all(axis=0)
    sel = (np.repeat(same, K) & slot_valid.reshape(-1)) & (r["nhits"] > 0)
    x, y, ph = r["par"][0], r["par"][1], r["par"][4]
    cosinc = (x * np.cos(ph) + y * np.sin(ph)) / np.maximum(np.hypot(x, y), 1e-30)
    band = sel & (cosinc < GRAZING_BAND)
    gd = dict(par=g["par"], cov=g["cov"], chi2=g["chi2"])
    rep = compare_tracks(gd, r, sel=sel & ~band)
    rep_band = compare_tracks(gd, r, sel=band)
    rep.update(seed_mismatch_frac=float(frac), best_mismatch_frac=float(1 - best_same.mean()), seeds=int(n_seeds),
               band=dict(n=rep_band["n"], worst_mom=rep_band["worst_mom"], worst_pos_norm=rep_band["worst_pos_norm"],
                         worst_cov=rep_band["worst_cov"], worst_chi2=rep_band["worst_chi2"]))
    print(rep)
    assert frac <= max_mismatch_frac, rep
    assert rep["mom_viol"] == 0 and rep["pos_viol"] == 0 and rep["chi2_viol"] == 0 and rep["cov_viol"] == 0, rep
    assert rep_band["n"] <= band_frac * max(rep["n"], 1), rep
    assert max(rep_band["worst_mom"], rep_band["worst_pos_norm"], rep_band["worst_cov"], rep_band["worst_chi2"]) < 3.0, rep
    # unused slots
    unused = ~(np.arange(K)[None, :] < g["n_cand"][:, None]).reshape(-1)
    assert (g["nhits"][unused] == 0).all() and (g["hit_idx"][:, unused] == -2).all() and (g["status"][unused] == 0).all()
    return rep


@pytest.mark.parametrize("tile", [0, 16, 112, 256])
def test_build_config3_small(tile):
    bi = synth.build_inputs(3, n_events=2, tracks=2000)
    compare_build(run_build(bi, tile=tile), ref_build(bi), bi.n_seeds, bi.K, 2e-3)


def test_build_tile_does_not_change_the_result():
    """Seeds per block (and with it the number of rounds a layer takes: 256 seeds x up to 10 candidates exceed the list
    area on the outer layers) must not change a single bit of the result."""
    bi = synth.build_inputs(4, n_events=1, tracks=2000, fake_frac=0.2)
    base = run_build(bi, tile=128)
    for tile in (16, 48, 256):
        other = run_build(bi, tile=tile)
        for k in ("n_cand", "hit_idx", "nhits", "status", "chi2"):
            assert np.array_equal(base[k], other[k]), (tile, k)
        v = base["nhits"] > 0
        assert np.array_equal(base["par"][:, v], other["par"][:, v]) and np.array_equal(base["cov"][:, v], other["cov"][:, v])


def test_build_config4_small():
    """configs[4] generator: 17 layers, wide pT, |eta| < 1.5 (candidates leaving the barrel), 20 % fake seeds, 10x noise."""
    bi = synth.build_inputs(4, n_events=1, tracks=3000)
    g, r = run_build(bi), ref_build(bi)
    assert (r["status"] != 0).any() and (r["n_cand"] == bi.K).mean() > 0.03
    compare_build(g, r, bi.n_seeds, bi.K, 2e-2, band_frac=0.05)


@pytest.mark.parametrize("K", [1, 3, 32])
def test_build_other_K(K):
    bi = synth.build_inputs(3, n_events=1, tracks=1500, noise=8.0)
    compare_build(run_build(bi, K=K), ref_build(bi, K=K), bi.n_seeds, K, 5e-3)


def test_build_dense_windows_exceed_the_child_buffer():
    """30-sigma windows, chi2 cut 3000, 40x noise: ~37 compatible hits per seed-layer, so the child buffer is pruned
    several times per layer and K = 10 saturates for every seed."""
    bi = synth.build_inputs(3, n_events=1, tracks=300, noise=40.0, n_sigma=30.0, chi2_cut=3000.0)
    r = ref_build(bi)
    assert r["counters"]["n_children"] / r["counters"]["n_seed_layers"] > 20
    compare_build(run_build(bi, tile=64), r, bi.n_seeds, bi.K, 5e-2)


def test_build_edge_cases():
    from paper_1711_06571_b200 import binding as b
    bi = synth.build_inputs(3, n_events=1, tracks=200)
    geom, hits, binned = gpu_bin(bi)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    # zero seeds
    out = b.kf_build(geom, hits, binned, b.Tracks.empty(0), None, None, 3, 10, 30.0, 3.0)
    assert out.n_seeds == 0
    # first_layer == n_layers: the seeds come back unchanged as the single candidate
    seeds = b.Tracks.from_host(bi.par, bi.cov, bi.q)
    L = bi.geom.n_layers
    shi = np.full((L, bi.ld), -1, np.int32)
    out = b.kf_build(geom, hits, binned, seeds, t(bi.seed_event), t(shi), L, 4, 30.0, 3.0)
    torch.cuda.synchronize()
    h = out.to_host()
    assert (h["n_cand"] == 1).all() and (h["nhits"][::4] == L).all()
    pe = bi.par[:, :bi.n_seeds].copy()
    assert np.allclose(h["par"][:4, ::4], pe[:4], rtol=0, atol=0) and np.allclose(h["par"][5, ::4], pe[5], rtol=0, atol=0)
    with pytest.raises(b.KfError, match="-1"):
        b.kf_build(geom, hits, binned, seeds, t(bi.seed_event), t(bi.seed_hit_idx), 3, 33, 30.0, 3.0)
    with pytest.raises(b.KfError, match="-1"):
        b.kf_build(geom, hits, binned, seeds, t(bi.seed_event), t(bi.seed_hit_idx), 3, 10, -1.0, 3.0)
    with pytest.raises(b.KfError, match="-4"):
        b.kf_build(geom, hits, binned, seeds, t(bi.seed_event), t(bi.seed_hit_idx), 3, 10, 30.0, 3.0, ws=torch.empty(64, dtype=torch.uint8, device="cuda"))
    with pytest.raises(b.KfError, match="-1"):
        b.kf_build_set_tile(24)


def test_build_config3_full():
    """BASELINE.json configs[3] at full size (16 events x 2 000 tracks), in the launch configuration bench.py times."""
    bi = synth.build_inputs(3)
    g, r = run_build(bi), ref_build(bi)
    rep = compare_build(g, r, bi.n_seeds, bi.K, 2e-3)
    assert rep["best_mismatch_frac"] < 1e-3
    best = np.arange(bi.n_seeds) * bi.K
    truth = bi.truth_hit_idx[:, bi.seed_truth]
    assert (g["hit_idx"][:, best] == truth).all(axis=0).mean() > 0.9

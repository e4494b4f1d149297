"""Several sub-batches in flight (sec. 4.2, L88 sec. 4.3): the streamed, host-to-host
form of the path (paper_1711_06571_b200/pipeline.py, the code bench.py times as `e2e`) returns, bit for bit, what one call on
the whole input returns, and is within tolerance of the oracle."""
import numpy as np
import pytest
import torch

from oracle import kf_oracle as o
from paper_1711_06571_b200 import synth
from tests.parity import assert_parity, compare_tracks

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("config,n,streams", [(0, 10_001, 4), (2, 30_000, 3), (0, 5, 4)])
def test_fit_pipeline_equals_single_call(config, n, streams):
    from paper_1711_06571_b200 import binding as b, pipeline
    fi = synth.fit_inputs(config, n=n)
    geom = b.Geom(fi.geom.layer_table(), fi.geom.bz)
    hits = b.Hits(fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off, 1)
    hi = None if fi.hit_idx is None else torch.from_numpy(fi.hit_idx).cuda()
    one = b.Tracks.from_host(fi.par, fi.cov, fi.q)
    # sub-batch boundaries are odd in general, so the two-track kernel pairs other tracks: compare with the one-track kernel,
    # whose arithmetic per track does not depend on its neighbours
    opt = b.options(fit_tracks_per_thread=1)
    ref = b.kf_fit(geom, hits, hi, None, one, opt=opt)
    torch.cuda.synchronize()
    ref = ref.to_host()
    pipe = pipeline.FitPipeline(geom, fi.n, fi.par, fi.cov, fi.q, fi.hit_x, fi.hit_y, fi.hit_z, fi.ld, hit_idx=fi.hit_idx, n_streams=streams, opt=opt)
    assert len(pipe.subs) == min(streams, n)
    for _ in range(2):                       # a second pass reuses every buffer
        pipe.run()
        torch.cuda.synchronize()
        got = pipe.result()
        for k in ("par", "cov", "chi2", "nhits", "status"):
            assert np.array_equal(got[k], ref[k]), k
    # default options (two tracks per thread where possible) against the oracle
    pipe = pipeline.FitPipeline(geom, fi.n, fi.par, fi.cov, fi.q, fi.hit_x, fi.hit_y, fi.hit_z, fi.ld, hit_idx=fi.hit_idx, n_streams=streams)
    pipe.run()
    torch.cuda.synchronize()
    got = pipe.result()
    r = o.fit(fi.geom.layer_table(), fi.geom.bz, fi.par, fi.cov, fi.q, fi.hit_x, fi.hit_y, fi.hit_z, fi.seg_off, fi.hit_idx)
    assert np.array_equal(got["nhits"], r["nhits"]) and np.array_equal(got["status"], r["status"])
    assert_parity(compare_tracks(got, r, sel=r["nhits"] > 0))
    assert pipe.h2d_bytes >= fi.n * (27 * 4 + 1) and pipe.d2h_bytes >= fi.n * 30 * 4


@pytest.mark.parametrize("config,kw,streams", [(3, dict(n_events=5, tracks=1200), 4), (4, dict(n_events=3, tracks=2500), 2)])
def test_build_pipeline_equals_single_call(config, kw, streams):
    from paper_1711_06571_b200 import binding as b, pipeline
    from tests.test_build_gpu import compare_build, ref_build, run_build
    bi = synth.build_inputs(config, **kw)
    geom = b.Geom(bi.geom.layer_table(), bi.geom.bz)
    one = run_build(bi)
    pipe = pipeline.BuildPipeline(geom, bi.n_events, bi.hit_x, bi.hit_y, bi.hit_z, bi.seg_off, bi.n_phi, bi.n_z, bi.par, bi.cov, bi.q, bi.seed_event,
                                  bi.seed_hit_idx, bi.first_layer, bi.K, bi.chi2_cut, bi.n_sigma, n_streams=streams)
    assert len(pipe.subs) == streams and sum(sb["m"] for sb in pipe.subs) == bi.n_seeds
    for _ in range(2):
        pipe.run()
        torch.cuda.synchronize()
        got = pipe.result()
        for k in ("n_cand", "hit_idx", "nhits", "status", "chi2"):
            assert np.array_equal(got[k], one[k]), k
        v = one["nhits"] > 0
        assert np.array_equal(got["par"][:, v], one["par"][:, v]) and np.array_equal(got["cov"][:, v], one["cov"][:, v])
    compare_build(got, ref_build(bi), bi.n_seeds, bi.K, bi.first_layer, band_frac=0.05)

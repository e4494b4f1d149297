"""kf_bin_hits_static: binning for callers that may not allocate device memory.

Some users of this library cannot call cudaMalloc at the point where they bin hits: a reconstruction module inside an
event-processing framework whose memory pool owns the card, or a per-event loop that cannot take the device-wide
synchronisation an allocation brings.  For them kf_bin_hits_static keeps the binning scratch (24 bytes per hit) in one fixed
array inside the library, good for KF_BIN_STATIC_MAX_HITS hits.  The array is shared by all calls and never cleared, so the
test calls the entry twice in a row -- a large batch first, then a smaller and different one that finds the first call's
leftovers in the scratch -- and asks for exactly the output of kf_bin_hits with a caller workspace (the index is integer work:
bit for bit, the bar of tests/test_build_gpu.py), and once more for the first batch.  The outputs are allocated before the
calls; the calls themselves must not change the amount of device memory in use.

This file sorts last on purpose (pytest -x stops at the first failure; nothing should hide behind this one) and passes alone
in a fresh process as well as after the other tests: it touches no state but the library's own scratch array.
"""
import numpy as np
import pytest
import torch

from paper_1711_06571_b200 import synth

pytestmark = pytest.mark.gpu


def device_arrays(bi):
    from paper_1711_06571_b200 import binding as b
    geom = b.Geom(bi.geom.layer_table(), bi.geom.bz)
    hits = b.Hits(bi.hit_x, bi.hit_y, bi.hit_z, bi.seg_off, bi.n_events)
    n_bins = bi.n_events * geom.n_layers * bi.n_phi * bi.n_z
    return geom, hits, n_bins


def assert_same_index(got, want):
    for k in ("bin_off", "perm", "x", "y", "z", "xyzp"):
        assert np.array_equal(got[k].view(np.int32) if got[k].dtype == np.float32 else got[k],
                              want[k].view(np.int32) if want[k].dtype == np.float32 else want[k]), k


def test_static_scratch_binning_equals_workspace_binning_twice_in_a_row():
    from paper_1711_06571_b200 import binding as b
    batches = [synth.build_inputs(3, n_events=3, tracks=777),                       # ~140 000 hits
               synth.build_inputs(4, n_events=1, tracks=400, fake_frac=0.0),        # fewer hits, other geometry and bin counts
               synth.build_inputs(3, n_events=3, tracks=777)]
    for bi in batches:
        geom, hits, n_bins = device_arrays(bi)
        assert hits.n_hits <= b.BIN_STATIC_MAX_HITS
        want = b.kf_bin_hits(geom, hits, bi.n_phi, bi.n_z)                          # existing path, torch-allocated workspace
        out = b.Binned(hits.n_hits, n_bins, bi.n_phi, bi.n_z, hits.x.device)        # caller's outputs, made before the call
        for t in (out.x, out.y, out.z, out.perm, out.bin_off, out.xyzp):
            t.fill_(-1)
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        b.kf_bin_hits_static(geom, hits, bi.n_phi, bi.n_z, out)
        torch.cuda.synchronize()
        if bi is not batches[0]:      # the very first call of a process may load the library's device code (set-up, documented)
            assert torch.cuda.mem_get_info()[0] == free_before
        assert_same_index(out.to_host(), want.to_host())


def test_static_scratch_binning_refuses_more_hits_than_the_array_holds():
    from paper_1711_06571_b200 import binding as b
    lt = synth.geometry("barrel10").layer_table()[:1]
    n = b.BIN_STATIC_MAX_HITS + 1
    ang = np.linspace(-3.0, 3.0, n)
    x = (lt[0][0] * np.cos(ang)).astype(np.float32); y = (lt[0][0] * np.sin(ang)).astype(np.float32); z = np.zeros(n, np.float32)
    geom = b.Geom(lt, 3.8)
    hits = b.Hits(x, y, z, np.array([0, n], np.int64), 1)
    out = b.Binned(n, 64 * 4, 64, 4, hits.x.device)
    with pytest.raises(b.KfError, match="KF_BIN_STATIC_MAX_HITS"):
        b.kf_bin_hits_static(geom, hits, 64, 4, out)
    # one hit fewer is the largest batch the entry takes, and it is binned like anywhere else
    hits = b.Hits(x[:-1], y[:-1], z[:-1], np.array([0, n - 1], np.int64), 1)
    want = b.kf_bin_hits(geom, hits, 64, 4)
    out = b.Binned(n - 1, 64 * 4, 64, 4, hits.x.device)
    b.kf_bin_hits_static(geom, hits, 64, 4, out)
    torch.cuda.synchronize()
    assert_same_index(out.to_host(), want.to_host())

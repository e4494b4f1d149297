"""Several sub-batches in flight: host -> device copies, the KF kernels and device -> host copies of different
sub-batches overlap on separate CUDA streams.

"To counter this effect we process multiple events at a time" (sec. 4.2); "multiple events in flight was also
necessary for scaling so that expensive copy operations could be overlapped with processing" (sec. 4.3).
This is the end-to-end form of the path: inputs start in HOST memory, results end in HOST
memory.  Every entry point of the C ABI takes a stream and never synchronises, so the recipe is only plumbing: split the
tracks (fit) or whole events (build) into `n_streams` groups, give each group its own stream, pinned host buffers and
device buffers, and enqueue copy-in / kernels / copy-out group by group.  No arithmetic lives here; each group's numbers
are exactly what a single call on that group gives (tests/test_pipeline_gpu.py).
"""
from __future__ import annotations

import numpy as np
import torch

from . import binding as b


def _pin(a):
    return torch.from_numpy(np.ascontiguousarray(a)).pin_memory()


def _nbytes(ts):
    return int(sum(t.numel() * t.element_size() for t in ts if t is not None))


def _ld(n):
    return max(32, (n + 31) // 32 * 32)


class FitPipeline:
    """kf_fit on host inputs, `n_streams` sub-batches of tracks in flight.

    par [6][>=n], cov [21][>=n], q [n], hit_x/y/z [L*ld_hits] with the hits of track t on layer l at l*ld_hits + t,
    hit_idx [L][>=n] (identity where >= 0, -1 hole, -2 not crossed) or None = a hit on every layer."""

    def __init__(self, geom: b.Geom, n: int, par, cov, q, hit_x, hit_y, hit_z, ld_hits: int, hit_idx=None, n_streams: int = 4, opt=None):
        self.geom, self.n, self.opt = geom, n, opt
        L = geom.n_layers
        n_sub = max(1, min(n_streams, n))
        self.bounds = [n * i // n_sub for i in range(n_sub + 1)]
        self.subs = []
        for c in range(n_sub):
            lo, hi = self.bounds[c], self.bounds[c + 1]
            m = hi - lo
            ldc = _ld(m)
            hp = np.zeros((6, ldc), np.float32); hp[:, :m] = par[:, lo:hi]
            hp[3, m:] = 1.0; hp[5, m:] = 1.5
            hc = np.zeros((21, ldc), np.float32); hc[:, :m] = cov[:, lo:hi]
            hxs = [np.ascontiguousarray(np.asarray(a_).reshape(L, ld_hits)[:, lo:hi]).reshape(-1) for a_ in (hit_x, hit_y, hit_z)]
            hidx = None
            if hit_idx is not None:
                hidx = np.full((L, ldc), -2, np.int32)
                hidx[:, :m] = np.where(hit_idx[:, lo:hi] >= 0, np.arange(m, dtype=np.int32)[None, :], hit_idx[:, lo:hi])
            sub = dict(m=m, stream=torch.cuda.Stream(), h_in=[_pin(hp), _pin(hc), _pin(np.asarray(q[lo:hi], np.int8))] + [_pin(x) for x in hxs] + ([_pin(hidx)] if hidx is not None else []))
            sub["seeds"] = b.Tracks.empty(m, ldc)
            sub["hits"] = b.Hits(np.zeros(L * m, np.float32), np.zeros(L * m, np.float32), np.zeros(L * m, np.float32), np.arange(L + 1, dtype=np.int64) * m, 1)
            sub["hit_idx"] = None if hidx is None else torch.empty((L, ldc), dtype=torch.int32, device="cuda")
            sub["out"] = b.Tracks.empty(m, ldc)
            sub["out"].q = sub["seeds"].q
            sub["d_in"] = [sub["seeds"].par, sub["seeds"].cov, sub["seeds"].q, sub["hits"].x, sub["hits"].y, sub["hits"].z] + ([sub["hit_idx"]] if hidx is not None else [])
            sub["d_out"] = [sub["out"].par, sub["out"].cov, sub["out"].chi2, sub["out"].nhits, sub["out"].status]
            sub["h_out"] = [torch.empty(t_.shape, dtype=t_.dtype).pin_memory() for t_ in sub["d_out"]]
            self.subs.append(sub)
        self.h2d_bytes = sum(_nbytes(sb["h_in"]) for sb in self.subs)
        self.d2h_bytes = sum(_nbytes(sb["h_out"]) for sb in self.subs)

    def run(self, stream=None):
        """Enqueue one pass: every group copies in, fits and copies out on its own stream; `stream` (default: current) waits
        for all of them, so an event recorded on it afterwards marks the end of the whole pass."""
        stream = torch.cuda.current_stream() if stream is None else stream
        start = torch.cuda.Event(); start.record(stream)
        for sb in self.subs:
            st_ = sb["stream"]
            st_.wait_event(start)
            with torch.cuda.stream(st_):
                for dst, src in zip(sb["d_in"], sb["h_in"]):
                    dst.copy_(src, non_blocking=True)
                b.kf_fit(self.geom, sb["hits"], sb["hit_idx"], None, sb["seeds"], out=sb["out"], opt=self.opt, stream=st_)
                for dst, src in zip(sb["h_out"], sb["d_out"]):
                    dst.copy_(src, non_blocking=True)
            done = torch.cuda.Event(); done.record(st_)
            stream.wait_event(done)

    def result(self) -> dict:
        """Host results of the last run (after a synchronize), concatenated over the groups."""
        par = np.concatenate([sb["h_out"][0][:, :sb["m"]].numpy() for sb in self.subs], axis=1)
        cov = np.concatenate([sb["h_out"][1][:, :sb["m"]].numpy() for sb in self.subs], axis=1)
        cat = lambda i: np.concatenate([sb["h_out"][i].numpy() for sb in self.subs])
        return dict(par=par, cov=cov, chi2=cat(2), nhits=cat(3), status=cat(4).view(np.uint32))


class BuildPipeline:
    """kf_bin_hits + kf_build on host inputs, `n_streams` groups of whole events in flight (seeds only read the hits of
    their own event, so a group is self-contained).  Seeds must be stored event by event (seed_event non-decreasing)."""

    def __init__(self, geom: b.Geom, n_events: int, hit_x, hit_y, hit_z, seg_off, n_phi: int, n_z: int, par, cov, q, seed_event, seed_hit_idx,
                 first_layer: int, K: int, chi2_cut: float, n_sigma: float, n_streams: int = 4, opt=None):
        self.geom, self.K, self.first_layer, self.chi2_cut, self.n_sigma, self.n_phi, self.n_z, self.opt = geom, K, first_layer, chi2_cut, n_sigma, n_phi, n_z, opt
        L = geom.n_layers
        seed_event = np.asarray(seed_event)
        assert (np.diff(seed_event) >= 0).all(), "seeds must be stored event by event"
        n_sub = max(1, min(n_streams, n_events))
        ev_b = [n_events * i // n_sub for i in range(n_sub + 1)]
        self.subs = []
        for c in range(n_sub):
            e0, e1 = ev_b[c], ev_b[c + 1]
            h0, h1 = int(seg_off[e0 * L]), int(seg_off[e1 * L])
            s0_, s1_ = int(np.searchsorted(seed_event, e0, side="left")), int(np.searchsorted(seed_event, e1, side="left"))
            m = s1_ - s0_
            ldc = _ld(m)
            hp = np.zeros((6, ldc), np.float32); hp[:, :m] = par[:, s0_:s1_]
            hp[3, m:] = 1.0; hp[5, m:] = 1.5
            hc = np.zeros((21, ldc), np.float32); hc[:, :m] = cov[:, s0_:s1_]
            hs = np.full((first_layer, ldc), -1, np.int32); hs[:, :m] = seed_hit_idx[:, s0_:s1_]
            sub = dict(stream=torch.cuda.Stream(), n_ev=e1 - e0, m=m, s0=s0_)
            sub["hits"] = b.Hits(np.zeros(h1 - h0, np.float32), np.zeros(h1 - h0, np.float32), np.zeros(h1 - h0, np.float32),
                                 np.asarray(seg_off[e0 * L: e1 * L + 1]) - h0, e1 - e0)
            sub["binned"] = b.Binned(h1 - h0, (e1 - e0) * L * n_phi * n_z, n_phi, n_z, soa=False)
            sub["ws"] = torch.empty(max(b.kf_bin_workspace_bytes(geom, sub["hits"], n_phi, n_z), 1), dtype=torch.uint8, device="cuda")
            sub["seeds"] = b.Tracks.empty(m, ldc)
            sub["sev"] = torch.zeros(max(m, 1), dtype=torch.int32, device="cuda")[:m]
            sub["shi"] = torch.empty((first_layer, ldc), dtype=torch.int32, device="cuda")
            sub["out"] = b.Cands(m, K, L)
            sub["bws"] = torch.empty(max(b.kf_build_workspace_bytes(geom, m, K, opt), 1), dtype=torch.uint8, device="cuda")
            sub["h_in"] = [_pin(a_) for a_ in (hit_x[h0:h1], hit_y[h0:h1], hit_z[h0:h1], hp, hc, np.asarray(q[s0_:s1_], np.int8),
                                               (seed_event[s0_:s1_] - e0).astype(np.int32), hs)]
            sub["d_in"] = [sub["hits"].x, sub["hits"].y, sub["hits"].z, sub["seeds"].par, sub["seeds"].cov, sub["seeds"].q, sub["sev"], sub["shi"]]
            o_ = sub["out"]
            sub["d_out"] = [o_.tracks.par, o_.tracks.cov, o_.tracks.chi2, o_.tracks.nhits, o_.tracks.status, o_.hit_idx, o_.n_cand]
            sub["h_out"] = [torch.empty(t_.shape, dtype=t_.dtype).pin_memory() for t_ in sub["d_out"]]
            self.subs.append(sub)
        self.h2d_bytes = sum(_nbytes(sb["h_in"]) for sb in self.subs)
        self.d2h_bytes = sum(_nbytes(sb["h_out"]) for sb in self.subs)

    def run(self, stream=None):
        stream = torch.cuda.current_stream() if stream is None else stream
        start = torch.cuda.Event(); start.record(stream)
        for sb in self.subs:
            st_ = sb["stream"]
            st_.wait_event(start)
            with torch.cuda.stream(st_):
                for dst, src in zip(sb["d_in"], sb["h_in"]):
                    dst.copy_(src, non_blocking=True)
                b.kf_bin_hits(self.geom, sb["hits"], self.n_phi, self.n_z, out=sb["binned"], ws=sb["ws"], stream=st_)
                b.kf_build(self.geom, sb["hits"], sb["binned"], sb["seeds"], sb["sev"], sb["shi"], self.first_layer, self.K, self.chi2_cut, self.n_sigma,
                           out=sb["out"], opt=self.opt, ws=sb["bws"], stream=st_)
                for dst, src in zip(sb["h_out"], sb["d_out"]):
                    dst.copy_(src, non_blocking=True)
            done = torch.cuda.Event(); done.record(st_)
            stream.wait_event(done)

    def result(self) -> dict:
        """Host results of the last run (after a synchronize): slot s*K + k over all seeds, as kf_cands."""
        K = self.K
        sl = lambda sb: sb["m"] * K
        par = np.concatenate([sb["h_out"][0][:, :sl(sb)].numpy() for sb in self.subs], axis=1)
        cov = np.concatenate([sb["h_out"][1][:, :sl(sb)].numpy() for sb in self.subs], axis=1)
        cat = lambda i: np.concatenate([sb["h_out"][i].numpy()[:sl(sb)] for sb in self.subs])
        hit_idx = np.concatenate([sb["h_out"][5][:, :sl(sb)].numpy() for sb in self.subs], axis=1)
        n_cand = np.concatenate([sb["h_out"][6].numpy() for sb in self.subs])
        return dict(par=par, cov=cov, chi2=cat(2), nhits=cat(3), status=cat(4).view(np.uint32), hit_idx=hit_idx, n_cand=n_cand)

"""Thin ctypes binding of libkf_b200.so (include/kf.h).  Argument marshalling only: every step of the path runs
in the CUDA kernels behind the C ABI.  PyTorch supplies device memory and streams.

There is no CPU fallback: if the shared library is missing or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libkf_b200.so")
_lib = None

KF_MAX_LAYERS = 32
MIN_KF_VERSION = 220      # struct layouts and signatures of include/kf.h as they stand (kf_layer.kind, kf_geom.hit_mode, opt)
ST_UNREACHABLE, ST_LEFT_Z, ST_GRAZING, ST_NUMERIC = 1, 2, 4, 8

EXPORTS = ["kf_options_init", "kf_fit", "kf_bin_workspace_bytes", "kf_bin_hits", "kf_bin_hits_static", "kf_window_lookup", "kf_build_workspace_bytes",
           "kf_build", "kf_select_best", "kf_mat66_multiply", "kf_last_error", "kf_version"]


class KfError(RuntimeError):
    pass


class kf_layer(C.Structure):
    _fields_ = [(n, C.c_float) for n in ("r", "zmax", "xx0", "sig_rphi", "sig_z", "sig_r")] + [("kind", C.c_int32), ("rmin", C.c_float)]


class kf_geom(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("bz_tesla", C.c_float), ("layers", C.POINTER(kf_layer)), ("hit_mode", C.c_int32)]


class kf_options(C.Structure):
    _fields_ = [("size", C.c_uint32), ("fit_tracks_per_thread", C.c_int32), ("build_seeds_per_block", C.c_int32), ("build_max_blocks", C.c_int32)]


class kf_tracks(C.Structure):
    _fields_ = [("n", C.c_int64), ("ld", C.c_int64), ("par", C.c_void_p), ("cov", C.c_void_p), ("q", C.c_void_p),
                ("chi2", C.c_void_p), ("nhits", C.c_void_p), ("status", C.c_void_p)]


class kf_hits(C.Structure):
    _fields_ = [("n_hits", C.c_int64), ("x", C.c_void_p), ("y", C.c_void_p), ("z", C.c_void_p), ("n_events", C.c_int32),
                ("seg_off", C.POINTER(C.c_int64)), ("seg_off_dev", C.c_void_p)]


class kf_binned(C.Structure):
    _fields_ = [("n_phi", C.c_int32), ("n_z", C.c_int32), ("x", C.c_void_p), ("y", C.c_void_p), ("z", C.c_void_p),
                ("perm", C.c_void_p), ("bin_off", C.c_void_p), ("xyzp", C.c_void_p)]


class kf_cands(C.Structure):
    _fields_ = [("K", C.c_int32), ("n_layers", C.c_int32), ("n_seeds", C.c_int64), ("ld", C.c_int64), ("cand", kf_tracks),
                ("hit_idx", C.c_void_p), ("n_cand", C.c_void_p)]


def lib() -> C.CDLL:
    """Loads libkf_b200.so (built in-tree by paper_1711_06571_b200.build_ext).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise KfError(f"{_SO} not built: run `python -m paper_1711_06571_b200.build_ext` (there is no CPU fallback)")
        l = C.CDLL(_SO)
        l.kf_last_error.restype = C.c_char_p
        l.kf_version.restype = C.c_int
        l.kf_bin_workspace_bytes.restype = C.c_size_t
        l.kf_build_workspace_bytes.restype = C.c_size_t
        l.kf_bin_workspace_bytes.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32]
        l.kf_build_workspace_bytes.argtypes = [C.c_void_p, C.c_int64, C.c_int32, C.c_void_p]
        l.kf_options_init.argtypes = [C.c_void_p]
        l.kf_options_init.restype = None
        l.kf_fit.argtypes = [C.c_void_p] * 8
        l.kf_bin_hits.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
        l.kf_bin_hits_static.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]
        l.kf_window_lookup.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64] + [C.c_void_p] * 6 + [C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
        l.kf_mat66_multiply.argtypes = [C.c_int32, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        l.kf_select_best.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_int64, C.c_void_p]
        l.kf_build.argtypes = [C.c_void_p] * 6 + [C.c_int32, C.c_int32, C.c_float, C.c_float, C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]
        # kf_layer (32 bytes with kind / rmin), kf_geom.hit_mode and the opt arguments date from version 220: only kf_options
        # carries a size field, so an older library would misread the structs below instead of rejecting them
        if l.kf_version() < MIN_KF_VERSION:
            raise KfError(f"{_SO} is version {l.kf_version()}, this binding needs >= {MIN_KF_VERSION}: rebuild with `python -m paper_1711_06571_b200.build_ext --force`")
        _lib = l
    return _lib


def _check(rc: int, who: str):
    if rc != 0:
        raise KfError(f"{who} failed with {rc}: {lib().kf_last_error().decode()}")


def _require_cuda():
    if not torch.cuda.is_available():
        raise KfError("no CUDA device: the KF path has no CPU fallback")


def _ptr(t, dtype=None):
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous(), "device, contiguous tensors only"
    if dtype is not None:
        assert t.dtype == dtype, (t.dtype, dtype)
    return C.c_void_p(t.data_ptr())


def _stream(stream):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


class Geom:
    """Host-side kf_geom built from a [L][6] table (r, zmax, xx0, sig_rphi, sig_z, sig_r; cylinders) or a [L][8] table
    (... kind, rmin; cylinders and endcap disks), Bz and the hit mode (0: hits on the nominal surfaces, 3-D update;
    1: two-step propagation and 2-D update on the tangent plane)."""

    def __init__(self, layer_table, bz: float, hit_mode: int = 0):
        tab = np.asarray(layer_table, dtype=np.float32)
        self.n_layers = tab.shape[0]
        self._arr = (kf_layer * max(1, self.n_layers))()
        for i in range(self.n_layers):
            row = [float(v) for v in tab[i, :6]]
            kind, rmin = (int(tab[i, 6]), float(tab[i, 7])) if tab.shape[1] >= 8 else (0, 0.0)
            self._arr[i] = kf_layer(*row, kind, rmin)
        self.hit_mode = int(hit_mode)
        self.c = kf_geom(self.n_layers, float(bz), C.cast(self._arr, C.POINTER(kf_layer)), self.hit_mode)
        self.table = tab
        self.bz = float(bz)


@dataclass
class Tracks:
    """Device SoA track store (kf_tracks)."""
    n: int
    ld: int
    par: torch.Tensor      # [6, ld] f32
    cov: torch.Tensor      # [21, ld] f32
    q: torch.Tensor        # [n] i8
    chi2: torch.Tensor     # [n] f32
    nhits: torch.Tensor    # [n] i32
    status: torch.Tensor   # [n] i32 (bit pattern of uint32)

    @staticmethod
    def empty(n: int, ld: int | None = None, device="cuda") -> "Tracks":
        ld = max(32, (n + 31) // 32 * 32) if ld is None else ld
        return Tracks(n, ld, torch.empty((6, ld), dtype=torch.float32, device=device), torch.empty((21, ld), dtype=torch.float32, device=device),
                      torch.empty(max(n, 1), dtype=torch.int8, device=device)[:n], torch.zeros(max(n, 1), dtype=torch.float32, device=device)[:n],
                      torch.zeros(max(n, 1), dtype=torch.int32, device=device)[:n], torch.zeros(max(n, 1), dtype=torch.int32, device=device)[:n])

    @staticmethod
    def from_host(par, cov, q, device="cuda", chi2=None, nhits=None) -> "Tracks":
        n, ld = len(q), par.shape[1]
        t = Tracks.empty(n, ld, device)
        t.par.copy_(torch.from_numpy(np.ascontiguousarray(par, dtype=np.float32)))
        t.cov.copy_(torch.from_numpy(np.ascontiguousarray(cov, dtype=np.float32)))
        t.q.copy_(torch.from_numpy(np.ascontiguousarray(q, dtype=np.int8)))
        if chi2 is not None:
            t.chi2.copy_(torch.from_numpy(np.ascontiguousarray(chi2, dtype=np.float32)))
        if nhits is not None:
            t.nhits.copy_(torch.from_numpy(np.ascontiguousarray(nhits, dtype=np.int32)))
        return t

    def c(self) -> kf_tracks:
        return kf_tracks(self.n, self.ld, self.par.data_ptr(), self.cov.data_ptr(), self.q.data_ptr() if self.n else None,
                         self.chi2.data_ptr() if self.n else None, self.nhits.data_ptr() if self.n else None,
                         self.status.data_ptr() if self.n else None)

    def to_host(self) -> dict:
        return dict(par=self.par[:, :self.n].cpu().numpy(), cov=self.cov[:, :self.n].cpu().numpy(), chi2=self.chi2.cpu().numpy(),
                    nhits=self.nhits.cpu().numpy(), status=self.status.cpu().numpy().view(np.uint32))


class Hits:
    """Device hit store (kf_hits): SoA x, y, z over all (event, layer) segments + host/device segment offsets."""

    def __init__(self, x, y, z, seg_off, n_events: int, device="cuda"):
        def dev(a):
            if isinstance(a, torch.Tensor):
                return a.to(device=device, dtype=torch.float32).contiguous()
            return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(device)
        self.x, self.y, self.z = dev(x), dev(y), dev(z)
        self.n_hits = int(self.x.numel())
        self.n_events = int(n_events)
        self.seg_off = np.ascontiguousarray(seg_off, dtype=np.int64)
        self.seg_off_dev = torch.from_numpy(self.seg_off).to(device)
        self.c = kf_hits(self.n_hits, self.x.data_ptr(), self.y.data_ptr(), self.z.data_ptr(), self.n_events,
                         self.seg_off.ctypes.data_as(C.POINTER(C.c_int64)), self.seg_off_dev.data_ptr())


def kf_version() -> int:
    return int(lib().kf_version())


def options(**fields) -> kf_options:
    """kf_options with the library's defaults (kf_options_init) and the given fields set, e.g. options(build_seeds_per_block=64)
    (build_seeds_per_block: 0 or a multiple of 16 in 16..256)."""
    o = kf_options()
    lib().kf_options_init(C.byref(o))
    for k, v in fields.items():
        if k not in ("fit_tracks_per_thread", "build_seeds_per_block", "build_max_blocks"):
            raise KeyError(k)
        setattr(o, k, int(v))
    return o


def _opt(opt):
    return None if opt is None else C.byref(opt)


def kf_fit(geom: Geom, hits: Hits, hit_idx, trk_event, seeds: Tracks, out: Tracks | None = None, opt: kf_options | None = None, stream=None) -> Tracks:
    """include/kf.h kf_fit.  hit_idx: [L, seeds.ld] int32 device tensor (-1 = hole, -2 = not crossed) or None (identity);
    trk_event [n] int32 or None."""
    _require_cuda()
    if out is None:
        out = Tracks.empty(seeds.n, seeds.ld, seeds.par.device)
        out.q = seeds.q
    if hit_idx is not None:
        assert tuple(hit_idx.shape) == (geom.n_layers, seeds.ld)
    sc, oc = seeds.c(), out.c()
    rc = lib().kf_fit(C.byref(geom.c), C.byref(hits.c), _ptr(hit_idx, torch.int32), _ptr(trk_event, torch.int32),
                      C.byref(sc), C.byref(oc), _opt(opt), _stream(stream))
    _check(rc, "kf_fit")
    return out


class Binned:
    """Device arrays of kf_binned, allocated by the caller (here: torch) and filled by kf_bin_hits."""

    def __init__(self, n_hits: int, n_bins: int, n_phi: int, n_z: int, device="cuda", soa: bool = True):
        """soa = False: only bin_off and the 16-byte records xyzp (all kf_build reads); x, y, z, perm stay NULL."""
        self.n_phi, self.n_z, self.n_hits = n_phi, n_z, n_hits
        m = max(n_hits, 1)
        mk = lambda dt: torch.empty(m, dtype=dt, device=device) if soa else None
        self.x, self.y, self.z, self.perm = mk(torch.float32), mk(torch.float32), mk(torch.float32), mk(torch.int32)
        self.bin_off = torch.empty(n_bins + 1, dtype=torch.int32, device=device)
        self.xyzp = torch.empty((m, 4), dtype=torch.float32, device=device)
        p = lambda t: t.data_ptr() if t is not None else None
        self.c = kf_binned(n_phi, n_z, p(self.x), p(self.y), p(self.z), p(self.perm), self.bin_off.data_ptr(), self.xyzp.data_ptr())

    def to_host(self) -> dict:
        n = self.n_hits
        d = dict(bin_off=self.bin_off.cpu().numpy(), n_phi=self.n_phi, n_z=self.n_z, xyzp=self.xyzp[:n].cpu().numpy())
        if self.x is not None:
            d.update(x=self.x[:n].cpu().numpy(), y=self.y[:n].cpu().numpy(), z=self.z[:n].cpu().numpy(), perm=self.perm[:n].cpu().numpy())
        return d


def kf_bin_workspace_bytes(geom: Geom, hits: Hits, n_phi: int, n_z: int) -> int:
    return int(lib().kf_bin_workspace_bytes(C.byref(geom.c), C.byref(hits.c), n_phi, n_z))


def kf_bin_hits(geom: Geom, hits: Hits, n_phi: int, n_z: int, out: Binned | None = None, ws: torch.Tensor | None = None, stream=None) -> Binned:
    """include/kf.h kf_bin_hits.  Allocates the output and the workspace with torch when not given."""
    _require_cuda()
    n_bins = hits.n_events * geom.n_layers * n_phi * n_z
    if out is None:
        out = Binned(hits.n_hits, n_bins, n_phi, n_z, hits.x.device)
    need = kf_bin_workspace_bytes(geom, hits, n_phi, n_z)
    if ws is None:
        ws = torch.empty(max(need, 1), dtype=torch.uint8, device=hits.x.device)
    rc = lib().kf_bin_hits(C.byref(geom.c), C.byref(hits.c), n_phi, n_z, C.byref(out.c), C.c_void_p(ws.data_ptr()), ws.numel(), _stream(stream))
    _check(rc, "kf_bin_hits")
    out._ws = ws    # keep the workspace alive until the stream has consumed it
    return out


BIN_STATIC_MAX_HITS = 1 << 20      # KF_BIN_STATIC_MAX_HITS of include/kf.h


def kf_bin_hits_static(geom: Geom, hits: Hits, n_phi: int, n_z: int, out: Binned, stream=None) -> Binned:
    """include/kf.h kf_bin_hits_static: kf_bin_hits without a workspace argument, for callers that may not allocate device
    memory (a module fed from a framework-owned memory pool, a loop that cannot take cudaMalloc's synchronisation).  The scratch
    is a fixed array inside the library, good for BIN_STATIC_MAX_HITS hits; larger batches raise KfError (-1).  `out` must be
    given -- this wrapper allocates nothing either.  Calls share the array: keep them ordered on the GPU (one stream)."""
    _require_cuda()
    rc = lib().kf_bin_hits_static(C.byref(geom.c), C.byref(hits.c), n_phi, n_z, C.byref(out.c), _stream(stream))
    _check(rc, "kf_bin_hits_static")
    return out


def kf_window_lookup(geom: Geom, hits: Hits, binned: Binned, event, layer, phi_c, dphi, z_c, dz, cap: int, stream=None):
    """include/kf.h kf_window_lookup.  Query arrays are device tensors (int32 / float32).  -> (count [n], sorted_idx [n, cap])"""
    _require_cuda()
    n = int(event.numel())
    count = torch.zeros(max(n, 1), dtype=torch.int32, device=event.device)[:n]
    idx = torch.full((max(n, 1), max(cap, 1)), -1, dtype=torch.int32, device=event.device)
    rc = lib().kf_window_lookup(C.byref(geom.c), C.byref(hits.c), C.byref(binned.c), n, _ptr(event, torch.int32), _ptr(layer, torch.int32),
                                _ptr(phi_c, torch.float32), _ptr(dphi, torch.float32), _ptr(z_c, torch.float32), _ptr(dz, torch.float32),
                                cap, C.c_void_p(count.data_ptr()), C.c_void_p(idx.data_ptr()), _stream(stream))
    _check(rc, "kf_window_lookup")
    return count, idx[:n, :cap]


class Cands:
    """Device arrays of kf_cands: n_seeds*K candidate slots (slot s*K + k, best first)."""

    def __init__(self, n_seeds: int, K: int, n_layers: int, device="cuda"):
        self.n_seeds, self.K, self.n_layers = n_seeds, K, n_layers
        n = n_seeds * K
        self.tracks = Tracks.empty(n, None, device)
        self.ld = self.tracks.ld
        self.hit_idx = torch.empty((n_layers, self.ld), dtype=torch.int32, device=device)
        self.n_cand = torch.zeros(max(n_seeds, 1), dtype=torch.int32, device=device)[:n_seeds]
        self.c = kf_cands(K, n_layers, n_seeds, self.ld, self.tracks.c(), self.hit_idx.data_ptr(), self.n_cand.data_ptr() if n_seeds else None)

    def to_host(self) -> dict:
        d = self.tracks.to_host()
        d["hit_idx"] = self.hit_idx[:, :self.tracks.n].cpu().numpy()
        d["n_cand"] = self.n_cand.cpu().numpy()
        return d


def kf_build_workspace_bytes(geom: Geom, n_seeds: int, K: int, opt: kf_options | None = None) -> int:
    return int(lib().kf_build_workspace_bytes(C.byref(geom.c), n_seeds, K, _opt(opt)))


def kf_build(geom: Geom, hits: Hits, binned: Binned, seeds: Tracks, seed_event, seed_hit_idx, first_layer: int, K: int, chi2_cut: float,
             n_sigma: float, out: Cands | None = None, opt: kf_options | None = None, ws: torch.Tensor | None = None, stream=None) -> Cands:
    """include/kf.h kf_build.  seed_event [n] int32 device tensor (or None), seed_hit_idx [first_layer, seeds.ld] int32 (or None).
    Allocates the output and the workspace with torch when not given."""
    _require_cuda()
    if out is None:
        out = Cands(seeds.n, K, geom.n_layers, seeds.par.device)
    if seed_hit_idx is not None:
        assert tuple(seed_hit_idx.shape) == (first_layer, seeds.ld)
    if ws is None:
        ws = torch.empty(max(kf_build_workspace_bytes(geom, seeds.n, K, opt), 1), dtype=torch.uint8, device=seeds.par.device)
    sc = seeds.c()
    rc = lib().kf_build(C.byref(geom.c), C.byref(hits.c), C.byref(binned.c), C.byref(sc), _ptr(seed_event, torch.int32), _ptr(seed_hit_idx, torch.int32),
                        first_layer, K, chi2_cut, n_sigma, C.byref(out.c), _opt(opt), C.c_void_p(ws.data_ptr()), ws.numel(), _stream(stream))
    _check(rc, "kf_build")
    out._ws = ws    # keep the workspace alive until the stream has consumed it
    return out


def kf_select_best(cands: Cands, first_layer: int, ld: int, out: torch.Tensor | None = None, stream=None) -> torch.Tensor:
    """include/kf.h kf_select_best -> [n_layers, ld] int32 hit indices of the best candidate per seed, for kf_fit."""
    _require_cuda()
    if out is None:
        out = torch.full((cands.n_layers, ld), -1, dtype=torch.int32, device=cands.hit_idx.device)
    assert tuple(out.shape) == (cands.n_layers, ld)
    rc = lib().kf_select_best(C.byref(cands.c), first_layer, _ptr(out, torch.int32), ld, _stream(stream))
    _check(rc, "kf_select_best")
    return out


def kf_mat66_multiply(layout: int, A: torch.Tensor, B: torch.Tensor, out: torch.Tensor | None = None, stream=None) -> torch.Tensor:
    """include/kf.h kf_mat66_multiply.  layout 0: A, B [36, ld] (matrix-major); layout 1: A, B [n, 36] (array of matrices)."""
    _require_cuda()
    if out is None:
        out = torch.empty_like(A)
    n, ld = (A.shape[1], A.shape[1]) if layout == 0 else (A.shape[0], 0)
    rc = lib().kf_mat66_multiply(layout, n, ld, _ptr(A, torch.float32), _ptr(B, torch.float32), _ptr(out, torch.float32), _stream(stream))
    _check(rc, "kf_mat66_multiply")
    return out

"""Seeded synthetic inputs for the KF tracking hot path (toy Monte Carlo).

Stands in for the paper's standalone toy simulation -- "simplified ideal barrel
geometry with a uniform longitudinal magnetic field, gaussian-smeared hit
positions, a particle gun ... flat transverse momentum distribution between 0.5
and 10 GeV" (sec. 3) -- and for its CMS-simulation events
(sec. 4.2), which are not available here.  Shapes and
distributions follow BASELINE.json configs[0..4]; the recipe is restated in
DESIGN.md "Input recipe".

This module serves BOTH the CUDA path and the CPU oracle and therefore holds
none of the Kalman filter: no Jacobian, no covariance transport, no gain, no
chi2, no binning.  It is a particle *simulator*: truth helices are intersected
with the barrel cylinders by circle-circle geometry (centre of curvature +
law of cosines), which is a different derivation from both the oracle's
march-and-Newton root finder and the kernel's tan-half-angle closed form, so
the noise-free pin (tests/test_oracle_pins.py::P3) is a real cross-check.

Everything is numpy fp64; hits and seeds are rounded to fp32 ONCE at the end
and that fp32 data is the common input of oracle and GPU.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

K_CURV = 0.00299792458  # GeV / (T cm): rho[cm] = pT / (K_CURV * |Bz|)
MASTER_SEED = 171106571


def rng_for(config: int, event: int = 0, stream: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(np.random.SeedSequence([MASTER_SEED, config, event, stream])))


@dataclass
class Geometry:
    """Ideal concentric barrel, optionally closed by endcap disks ("cylinder with lids", sec. 4.1).
    One row per layer in the order a track from the vertex crosses them: barrel layers by increasing radius, then the
    disks of either side by increasing |z|.  kind 0: cylinder of radius r, |z| <= zmax.  kind 1: disk in the plane
    z = r (signed), rmin <= radius <= zmax."""
    r: np.ndarray
    zmax: np.ndarray
    xx0: np.ndarray
    sig_rphi: np.ndarray
    sig_z: np.ndarray
    sig_r: np.ndarray
    bz: float
    kind: np.ndarray | None = None
    rmin: np.ndarray | None = None

    def __post_init__(self):
        if self.kind is None:
            self.kind = np.zeros(len(self.r), dtype=np.int32)
        if self.rmin is None:
            self.rmin = np.zeros(len(self.r))

    @property
    def n_layers(self) -> int:
        return len(self.r)

    @property
    def has_disks(self) -> bool:
        return bool(np.any(self.kind != 0))

    def layer_table(self) -> np.ndarray:
        """[L][6] float64: r, zmax, xx0, sig_rphi, sig_z, sig_r; with disks [L][8]: ..., kind, rmin."""
        t = np.stack([self.r, self.zmax, self.xx0, self.sig_rphi, self.sig_z, self.sig_r], axis=1).astype(np.float64)
        if self.has_disks:
            t = np.concatenate([t, self.kind[:, None].astype(np.float64), self.rmin[:, None].astype(np.float64)], axis=1)
        return t


def geometry(kind: str, bz: float = 3.8, xx0_scale: float = 1.0, depth: float = 0.0) -> Geometry:
    """kind 'barrel10' (configs 0,1,3): r = 4,8..40 cm, x/X0 = 0.02.
    kind 'barrel17' (configs 2,4): 17 layers r = 4..80 uniformly, x/X0 alternating 0.01/0.03."""
    if kind == "barrel10":
        r = 4.0 * np.arange(1, 11, dtype=np.float64)
        xx0 = np.full(10, 0.02)
    elif kind == "barrel17":
        r = 4.0 + 4.75 * np.arange(17, dtype=np.float64)
        xx0 = np.where(np.arange(17) % 2 == 0, 0.01, 0.03)
    elif kind == "lids10":
        # "cylinder with lids": the 10-layer barrel shortened to |z| <= 50 cm, closed on either side by four
        # disks at |z| = 60, 75, 90, 105 cm covering 4 <= radius <= 44 cm; same resolutions, x/X0 = 0.02 everywhere
        rb = 4.0 * np.arange(1, 11, dtype=np.float64)
        zd = np.array([60.0, 75.0, 90.0, 105.0])
        r = np.concatenate([rb, zd, -zd])
        n = len(r)
        knd = np.concatenate([np.zeros(10, np.int32), np.ones(8, np.int32)])
        # depth > 0 (building with kf_geom.hit_mode = 1, R23): the resolution along a surface's normal -- which the
        # 2-D update does not use -- carries the r.m.s. displacement of the sensors about the nominal surface
        return Geometry(r=r, zmax=np.where(knd == 0, 50.0, 44.0), xx0=np.full(n, 0.02) * xx0_scale, sig_rphi=np.full(n, 0.01),
                        sig_z=np.where((knd == 1) & (depth > 0), depth, 0.1), sig_r=np.where((knd == 0) & (depth > 0), depth, 0.01),
                        bz=bz, kind=knd, rmin=np.where(knd == 0, 0.0, 4.0))
    else:
        raise ValueError(kind)
    n = len(r)
    # depth > 0 (hit_mode 1 on staggered sensors, R23): sig_r carries the r.m.s. radial displacement of the sensors
    return Geometry(r=r, zmax=np.full(n, 100.0), xx0=xx0 * xx0_scale, sig_rphi=np.full(n, 0.01),
                    sig_z=np.full(n, 0.1), sig_r=np.full(n, depth if depth > 0 else 0.01), bz=bz)


def pack_index(i: int, j: int) -> int:
    """Packed lower-triangular row-major index, k(i,j) = i(i+1)/2 + j for i >= j."""
    if i < j:
        i, j = j, i
    return i * (i + 1) // 2 + j


def pack_sym(c: np.ndarray) -> np.ndarray:
    """[..., 6, 6] -> [..., 21]"""
    idx = [(i, j) for i in range(6) for j in range(i + 1)]
    return np.stack([c[..., i, j] for i, j in idx], axis=-1)


def unpack_sym(p: np.ndarray) -> np.ndarray:
    """[..., 21] -> [..., 6, 6]"""
    out = np.empty(p.shape[:-1] + (6, 6), dtype=p.dtype)
    for i in range(6):
        for j in range(i + 1):
            out[..., i, j] = p[..., pack_index(i, j)]
            out[..., j, i] = p[..., pack_index(i, j)]
    return out


# ----------------------------------------------------------------------------------------------
# particle gun
# ----------------------------------------------------------------------------------------------
def particle_gun(rng: np.random.Generator, n: int, kind: str) -> dict:
    """Truth at the vertex (origin).  kind 'flat' (configs 0,1,3): pT ~ U(0.5,10) GeV, |eta|<1.
    kind 'wide' (configs 2,4): ln pT ~ U(ln 0.3, ln 100), |eta|<1.5."""
    phi = rng.uniform(-np.pi, np.pi, n)
    q = np.where(rng.random(n) < 0.5, -1, 1).astype(np.int8)
    if kind == "flat":
        pt = rng.uniform(0.5, 10.0, n)
        eta = rng.uniform(-1.0, 1.0, n)
    elif kind == "wide":
        pt = np.exp(rng.uniform(np.log(0.3), np.log(100.0), n))
        eta = rng.uniform(-1.5, 1.5, n)
    elif kind == "forward":      # the flat gun opened up to |eta| < 2.2: barrel, both lids and the transition between them
        pt = rng.uniform(0.5, 10.0, n)
        eta = rng.uniform(-2.2, 2.2, n)
    else:
        raise ValueError(kind)
    theta = 2.0 * np.arctan(np.exp(-eta))
    z = np.zeros(n)
    return dict(x=z.copy(), y=z.copy(), z=z.copy(), ipt=1.0 / pt, phi=phi, theta=theta, q=q)


# ----------------------------------------------------------------------------------------------
# truth transport: circle-circle intersection (simulator only)
# ----------------------------------------------------------------------------------------------
def cross_cylinder(x, y, z, ipt, phi, theta, q, bz, R):
    """First outward crossing of the cylinder of radius R by the truth helix.

    Returns (ok, x', y', z', phi', s_T, cos_inc).  Geometry: the transverse projection is a circle of
    signed curvature w = -q K Bz / pT about the centre c = (x - sin(phi)/w, y + cos(phi)/w); the cylinder
    is the circle |p| = R about the origin.  The two intersections sit at polar angle gamma +- beta, with
    gamma the azimuth of c and cos(beta) = (d^2 + R^2 - rho^2) / (2 d R) (law of cosines, d = |c|).
    The one reached first is the one with the smaller turning angle about c in the sense of rotation; a crossing
    that needs more than half a turn is not a step to the next layer outwards and counts as not reached (DESIGN.md
    R2; never the case for a particle that starts moving outwards).  A straight line (w = 0) uses the chord formula.
    """
    x, y, z, ipt, phi, theta = (np.asarray(a, dtype=np.float64) for a in (x, y, z, ipt, phi, theta))
    w = -np.asarray(q, dtype=np.float64) * K_CURV * bz * ipt
    cp, sp = np.cos(phi), np.sin(phi)
    r02 = x * x + y * y
    inside = r02 < R * R
    straight = np.abs(w) * R < 1e-12
    ws = np.where(straight, 1.0, w)
    # --- curved branch
    cx, cy = x - sp / ws, y + cp / ws
    rho = 1.0 / np.abs(ws)
    d = np.hypot(cx, cy)
    cosb = (d * d + R * R - rho * rho) / (2.0 * np.where(d > 0, d, 1.0) * R)
    reach = (np.abs(cosb) <= 1.0) & (d > 0)
    beta = np.arccos(np.clip(cosb, -1.0, 1.0))
    gamma = np.arctan2(cy, cx)
    psi0 = np.arctan2(y - cy, x - cx)
    sgn = np.sign(ws)
    best = np.full(x.shape, np.inf)
    bx = np.zeros_like(x)
    by = np.zeros_like(x)
    for pm in (+1.0, -1.0):
        px, py = R * np.cos(gamma + pm * beta), R * np.sin(gamma + pm * beta)
        psi = np.arctan2(py - cy, px - cx)
        turn = np.mod((psi - psi0) * sgn, 2.0 * np.pi)
        take = turn < best
        best = np.where(take, turn, best)
        bx = np.where(take, px, bx)
        by = np.where(take, py, by)
    s_c = best * rho
    phi_c = phi + sgn * best
    # --- straight branch: |p + s d|^2 = R^2
    u = x * cp + y * sp
    s_l = -u + np.sqrt(np.maximum(u * u + R * R - r02, 0.0))
    lx, ly = x + s_l * cp, y + s_l * sp
    xs = np.where(straight, lx, bx)
    ys = np.where(straight, ly, by)
    s = np.where(straight, s_l, s_c)
    phn = np.where(straight, phi, phi_c)
    ok = inside & (straight | (reach & (best <= np.pi)))
    zn = z + s / np.tan(theta)
    cosinc = (xs * np.cos(phn) + ys * np.sin(phn)) / R
    return ok, xs, ys, zn, phn, s, cosinc


def cross_plane(x, y, z, ipt, phi, theta, q, bz, Z):
    """First crossing of the plane z = Z by the truth helix (simulator only): z advances by cot(theta) per unit of
    transverse path, so s_T = (Z - z) tan(theta) must be positive; the transverse position turns about the centre of
    curvature by w s_T.  Returns (ok, x', y', z', phi', s_T, cos_inc = |cos theta|); ok needs s_T > 0 and at most half a turn."""
    x, y, z, ipt, phi, theta = (np.asarray(a, dtype=np.float64) for a in (x, y, z, ipt, phi, theta))
    w = -np.asarray(q, dtype=np.float64) * K_CURV * bz * ipt
    s = (Z - z) * np.tan(theta)
    straight = np.abs(w) * np.abs(s) < 1e-12
    ws = np.where(straight, 1.0, w)
    cx, cy = x - np.sin(phi) / ws, y + np.cos(phi) / ws
    a = ws * s
    xr, yr = x - cx, y - cy
    xc = cx + xr * np.cos(a) - yr * np.sin(a)
    yc = cy + xr * np.sin(a) + yr * np.cos(a)
    xs = np.where(straight, x + s * np.cos(phi), xc)
    ys = np.where(straight, y + s * np.sin(phi), yc)
    phn = np.where(straight, phi, phi + a)
    ok = (s > 0) & np.isfinite(s) & (np.abs(w) * s <= np.pi)
    return ok, xs, ys, np.full(xs.shape, float(Z)) if np.ndim(Z) == 0 else Z, phn, s, np.abs(np.cos(theta))


def highland_theta0(ipt, theta, cosinc, xx0):
    """Highland/PDG width of the projected scattering angle, beta = 1, unit charge, p = 1/(ipt sin theta),
    path through the layer = xx0 / (sin(theta) * cos_inc)."""
    t = xx0 / (np.sin(theta) * cosinc)
    return 0.0136 * ipt * np.sin(theta) * np.sqrt(t) * (1.0 + 0.038 * np.log(t))


GEN_MIN_COSINC = 0.2  # a truth crossing shallower than this ends the track (reading A9)


def simulate(geom: Geometry, gun: dict, rng: np.random.Generator, ms: bool = True, smear: bool = True, jitter: float = 0.0) -> dict:
    """Transport every truth particle outward layer by layer; record the crossing, smear the hit on the
    surface (barrel: phi by N(0, sig_rphi/R), z by N(0, sig_z); disk: r-phi by N(0, sig_rphi), radius by N(0, sig_r)),
    then apply the thin-scatterer kick.

    Barrel-only geometry: a track ends (that layer and all outer ones get no hit) when the layer is unreachable, the
    crossing has |z| > zmax, or cos(incidence) < GEN_MIN_COSINC.  With disks a crossing outside the layer's acceptance
    only skips that layer (the particle flies on to the lids); unreachable / grazing still ends the track.
    jitter > 0 ("hits at slightly different radii within a layer"): the sensor that is hit sits at
    R + U(-jitter, jitter) (barrel) or Z + U(-jitter, jitter) (disk); crossing, hit and scattering happen THERE.
    Returns hits [L][n][3] (NaN where absent), valid [L][n], truth [L][n][6] = state just outside the layer (at the
    hit's own surface)."""
    n = len(gun["phi"])
    L = geom.n_layers
    x, y, z = gun["x"].copy(), gun["y"].copy(), gun["z"].copy()
    ipt, phi, theta, q = gun["ipt"].copy(), gun["phi"].copy(), gun["theta"].copy(), gun["q"]
    alive = np.ones(n, dtype=bool)
    hits = np.full((L, n, 3), np.nan)
    valid = np.zeros((L, n), dtype=bool)
    truth = np.full((L, n, 6), np.nan)
    lids = geom.has_disks
    for l in range(L):
        R = geom.r[l]
        disk = geom.kind[l] != 0
        off = rng.uniform(-jitter, jitter, n) if jitter > 0 else 0.0
        with np.errstate(invalid="ignore", divide="ignore"):
            if disk:
                ok, xn, yn, zn, phn, s, ci = cross_plane(x, y, z, ipt, phi, theta, q, geom.bz, R + off)
                ci3 = ci                                     # cosine of the angle to the disk normal
                rn = np.hypot(xn, yn)
                inside = (rn >= geom.rmin[l]) & (rn <= geom.zmax[l])
            else:
                ok, xn, yn, zn, phn, s, ci = cross_cylinder(x, y, z, ipt, phi, theta, q, geom.bz, R + off)
                inside = np.abs(zn) <= geom.zmax[l]
        if lids:
            crossed = ok & alive & (ci >= GEN_MIN_COSINC)
            if not disk:
                alive = alive & crossed                      # a looper that cannot reach / grazes a cylinder is lost
            ok = crossed & inside
        else:
            ok = ok & alive & inside & (ci >= GEN_MIN_COSINC)
            alive = ok
        x = np.where(ok, xn, x); y = np.where(ok, yn, y); z = np.where(ok, zn, z); phi = np.where(ok, phn, phi)
        # hit, smeared on the surface
        e1 = rng.standard_normal(n)
        e2 = rng.standard_normal(n)
        if disk:
            rr = np.hypot(x, y)
            az = np.arctan2(y, x) + e1 * (geom.sig_rphi[l] if smear else 0.0) / np.where(rr > 0, rr, 1.0)
            rh = rr + e2 * (geom.sig_r[l] if smear else 0.0)
            hits[l, :, 0] = np.where(ok, rh * np.cos(az), np.nan)
            hits[l, :, 1] = np.where(ok, rh * np.sin(az), np.nan)
            hits[l, :, 2] = np.where(ok, z, np.nan)
        else:
            Rh = R + off
            az = np.arctan2(y, x) + e1 * (geom.sig_rphi[l] / Rh if smear else 0.0)
            hits[l, :, 0] = np.where(ok, Rh * np.cos(az), np.nan)
            hits[l, :, 1] = np.where(ok, Rh * np.sin(az), np.nan)
            hits[l, :, 2] = np.where(ok, z + e2 * (geom.sig_z[l] if smear else 0.0), np.nan)
        valid[l] = ok
        # multiple scattering: two orthogonal kicks of width theta0, |p| conserved
        k1 = rng.standard_normal(n)
        k2 = rng.standard_normal(n)
        if ms:
            with np.errstate(invalid="ignore", divide="ignore"):
                # highland_theta0 takes the in-plane incidence on a cylinder; for a disk hand it |cos theta| / sin theta so
                # that sin(theta) * cos_inc is the cosine of the angle to the surface normal in both cases
                cie = np.where(ok, ci / np.sin(theta) if disk else ci, 1.0)
                th0 = np.where(ok, highland_theta0(ipt, theta, cie, geom.xx0[l]), 0.0)
            th_new = theta + k1 * th0
            phi = phi + k2 * th0 / np.sin(theta)
            ipt = ipt * np.sin(theta) / np.sin(th_new)
            theta = th_new
        truth[l] = np.where(ok[:, None], np.stack([x, y, z, ipt, phi, theta], axis=1), np.nan)
    return dict(hits=hits, valid=valid, truth=truth)


# ----------------------------------------------------------------------------------------------
# seeds
# ----------------------------------------------------------------------------------------------
SEED_SIGMA_POS = 0.05      # cm
SEED_SIGMA_REL_IPT = 0.05  # "truth smeared 5 %" (BASELINE.json config 0) applies to 1/pT
SEED_SIGMA_ANG = 0.005     # rad


def smear_seed(rng: np.random.Generator, state: np.ndarray) -> tuple[np.ndarray, np.ndarray]:
    """state [n][6] truth -> (seed [n][6], sigma [n][6]).  Diagonal Gaussian smearing; covariance = diag(sigma^2)."""
    n = state.shape[0]
    sig = np.empty((n, 6))
    sig[:, 0:3] = SEED_SIGMA_POS
    sig[:, 3] = SEED_SIGMA_REL_IPT * np.abs(state[:, 3])
    sig[:, 4:6] = SEED_SIGMA_ANG
    seed = state + rng.standard_normal((n, 6)) * sig
    return seed, sig


def _ld(n: int) -> int:
    return max(32, (n + 31) // 32 * 32)


def _soa_tracks(seed: np.ndarray, sig: np.ndarray, q: np.ndarray) -> dict:
    """AoS fp64 -> the SoA fp32 store of include/kf.h (par[6][ld], cov[21][ld], q[n])."""
    n = seed.shape[0]
    ld = _ld(n)
    par = np.zeros((6, ld), dtype=np.float32)
    par[:, :n] = seed.T.astype(np.float32)
    cov = np.zeros((21, ld), dtype=np.float32)
    for i in range(6):
        cov[pack_index(i, i), :n] = (sig[:, i] ** 2).astype(np.float32)
    # padding lanes: harmless unit state so that kernels may touch them
    par[3, n:] = 1.0; par[5, n:] = 1.5
    return dict(n=n, ld=ld, par=par, cov=cov, q=np.ascontiguousarray(q.astype(np.int8)))


@dataclass
class FitInputs:
    geom: Geometry
    n: int
    ld: int
    par: np.ndarray        # [6][ld] f32 seeds
    cov: np.ndarray        # [21][ld] f32
    q: np.ndarray          # [n] i8
    hit_x: np.ndarray      # [L*ld] f32, segment l at [l*ld, l*ld+n)
    hit_y: np.ndarray
    hit_z: np.ndarray
    seg_off: np.ndarray    # [L+1] i64
    hit_idx: np.ndarray | None  # [L][ld] i32 (identity, or -2 = layer not crossed), None = identity everywhere
    truth: np.ndarray      # [L][n][6] f64 (NaN where no hit)
    valid: np.ndarray      # [L][n] bool
    gun: dict = field(default_factory=dict)


FIT_CONFIGS = {
    # "lids": cylinder with lids + sensors staggered by +-0.3 cm about the nominal surfaces;
    # fitted with kf_geom.hit_mode = 1 (two-step propagation, 2-D update on the tangent plane)
    "lids": dict(n=100_000, geom="lids10", gun="forward", jitter=0.3),
    0: dict(n=10_000, geom="barrel10", gun="flat"),
    1: dict(n=1_000_000, geom="barrel10", gun="flat"),
    2: dict(n=1_000_000, geom="barrel17", gun="wide"),
}


def fit_inputs(config, n: int | None = None, ms: bool = True, smear: bool = True, event: int = 0,
               force_index: bool = False, bz: float = 3.8, jitter: float | None = None) -> FitInputs:
    """Inputs of kf_fit for BASELINE.json configs 0-2 (n overrides the track count, e.g. for tests)."""
    cfg = FIT_CONFIGS[config]
    n = cfg["n"] if n is None else n
    geom = geometry(cfg["geom"], bz=bz, xx0_scale=1.0 if ms else 0.0)
    rng = rng_for(config if isinstance(config, int) else 100, event)
    gun = particle_gun(rng, n, cfg["gun"])
    sim = simulate(geom, gun, rng, ms=ms, smear=smear, jitter=cfg.get("jitter", 0.0) if jitter is None else jitter)
    vtx = np.stack([gun["x"], gun["y"], gun["z"], gun["ipt"], gun["phi"], gun["theta"]], axis=1)
    seed, sig = smear_seed(rng, vtx)
    t = _soa_tracks(seed, sig, gun["q"])
    L, ld = geom.n_layers, t["ld"]
    hx = np.zeros((L, ld), dtype=np.float32); hy = np.zeros((L, ld), dtype=np.float32); hz = np.zeros((L, ld), dtype=np.float32)
    h = np.nan_to_num(sim["hits"], nan=0.0)
    hx[:, :n] = h[:, :, 0]; hy[:, :n] = h[:, :, 1]; hz[:, :n] = h[:, :, 2]
    all_valid = bool(sim["valid"].all())
    hit_idx = None
    if force_index or not all_valid:
        hit_idx = np.full((L, ld), -2, dtype=np.int32)     # -2: the truth track ended before this layer (not crossed)
        ident = np.arange(n, dtype=np.int32)
        for l in range(L):
            hit_idx[l, :n] = np.where(sim["valid"][l], ident, -2)
    seg_off = (np.arange(L + 1, dtype=np.int64) * ld)
    return FitInputs(geom=geom, n=n, ld=ld, par=t["par"], cov=t["cov"], q=t["q"], hit_x=hx.reshape(-1), hit_y=hy.reshape(-1),
                     hit_z=hz.reshape(-1), seg_off=seg_off, hit_idx=hit_idx, truth=sim["truth"], valid=sim["valid"], gun=gun)


# ----------------------------------------------------------------------------------------------
# build events (configs 3, 4)
# ----------------------------------------------------------------------------------------------
@dataclass
class BuildInputs:
    geom: Geometry
    n_events: int
    n_phi: int
    n_z: int
    K: int
    chi2_cut: float
    n_sigma: float
    first_layer: int
    hit_x: np.ndarray      # [n_hits] f32, segments (event*L + layer) back to back
    hit_y: np.ndarray
    hit_z: np.ndarray
    seg_off: np.ndarray    # [n_events*L+1] i64
    hit_truth: np.ndarray  # [n_hits] i32: global truth-track id of the hit, -1 = noise
    n_seeds: int
    ld: int
    par: np.ndarray        # [6][ld] f32 seed states on layer first_layer-1
    cov: np.ndarray        # [21][ld]
    q: np.ndarray          # [n_seeds] i8
    seed_event: np.ndarray    # [n_seeds] i32
    seed_hit_idx: np.ndarray  # [first_layer][ld] i32 index within segment
    seed_truth: np.ndarray    # [n_seeds] i32 global truth-track id, -1 = fake seed
    truth_hit_idx: np.ndarray  # [L][n_tracks_total] i32 index within segment of each truth track's hit, -1 none
    event_ids: np.ndarray = None   # [n_events] i64 global id (generator stream) of each event of the call


BUILD_CONFIGS = {
    3: dict(n_events=16, tracks=2_000, geom="barrel10", gun="flat", noise=5, n_phi=256, n_z=16, fake_frac=0.0),
    4: dict(n_events=64, tracks=10_000, geom="barrel17", gun="wide", noise=10, n_phi=1024, n_z=32, fake_frac=0.2),
    # building on the "cylinder with lids" (R22): the config-3 recipe on the lids10 geometry with the
    # forward gun; noise on a disk is uniform in phi and in radius over [rmin, rmax]
    "lids": dict(n_events=8, tracks=2_000, geom="lids10", gun="forward", noise=5, n_phi=256, n_z=16, fake_frac=0.0),
}


def _three_point_seed(p1, p2, p3, bz):
    """Fake seed from three hits (simulator-side geometry only): circle through the (x,y) points ->
    curvature and tangent at p3; cot(theta) from dz over arc length between p1 and p3.
    Returns state[6] at p3 and charge, or None when degenerate."""
    (x1, y1, z1), (x2, y2, z2), (x3, y3, z3) = p1, p2, p3
    a = 2.0 * ((x2 - x1) * (y3 - y1) - (y2 - y1) * (x3 - x1))
    chord = np.hypot(x3 - x1, y3 - y1)
    if chord <= 0:
        return None
    if abs(a) < 1e-12 * chord * chord:
        w = 0.0
        phi = np.arctan2(y3 - y1, x3 - x1)
        arc = chord
    else:
        b2, b3 = (x2 * x2 + y2 * y2 - x1 * x1 - y1 * y1), (x3 * x3 + y3 * y3 - x1 * x1 - y1 * y1)
        cx = (b2 * (y3 - y1) - b3 * (y2 - y1)) / a
        cy = (b3 * (x2 - x1) - b2 * (x3 - x1)) / a
        rho = np.hypot(x3 - cx, y3 - cy)
        sgn = 1.0 if a > 0 else -1.0   # counter-clockwise (w > 0) when p1->p2->p3 turns left
        w = sgn / rho
        phi = np.arctan2(sgn * (x3 - cx), -sgn * (y3 - cy))
        half = min(1.0, chord / (2.0 * rho))
        arc = 2.0 * rho * np.arcsin(half)
    cot = (z3 - z1) / arc
    theta = np.arctan2(1.0, cot)
    if w == 0.0 or bz == 0.0:
        return None
    ipt = abs(w) / (K_CURV * abs(bz))
    q = 1 if (-w / (K_CURV * bz)) > 0 else -1
    return np.array([x3, y3, z3, ipt, phi, theta]), q


def build_inputs(config, n_events: int | None = None, tracks: int | None = None, first_layer: int = 3,
                 K: int = 10, chi2_cut: float = 30.0, n_sigma: float = 3.0, noise: float | None = None,
                 fake_frac: float | None = None, n_phi: int | None = None, n_z: int | None = None,
                 smear: bool = True, ms: bool = True, event0: int = 0, jitter: float = 0.0, events=None) -> BuildInputs:
    """Inputs of kf_bin_hits / kf_build for BASELINE.json configs 3-4 (sizes can be overridden for tests).

    jitter > 0: sensors sit at R + U(-jitter, jitter) / Z + U(-jitter, jitter) ("hits at slightly different radii within a
    layer"), truth and noise hits alike: inputs for kf_geom.hit_mode = 1.
    Per event: truth tracks from the particle gun; hits per layer = truth hits + `noise` x (number of truth
    hits on that layer) uniform in (phi, z) on the cylinder; each segment is shuffled.  One seed per truth
    track that reaches layer `first_layer-1`: truth state just outside that layer, smeared (smear_seed),
    diagonal covariance (reading A6b).  Config 4 adds `fake_frac` x tracks fake seeds from random
    hit triplets on layers 0-2 (reading A18).
    Which events: event e of the call is drawn from the generator of global event id event_ids[e]; by default the ids are
    event0, event0 + 1, ...; `events` = an explicit list of global ids (a rank's share under strong scaling, shard.assign_events)
    overrides n_events and event0.  The ids are returned in BuildInputs.event_ids."""
    cfg = dict(BUILD_CONFIGS[config])
    if events is not None:
        n_events = len(events)
        if n_events < 1:
            raise ValueError("build_inputs: `events` must name at least one event")
    n_events = cfg["n_events"] if n_events is None else n_events
    event_ids = np.asarray(events if events is not None else np.arange(n_events) + event0, dtype=np.int64)
    tracks = cfg["tracks"] if tracks is None else tracks
    noise = cfg["noise"] if noise is None else noise
    fake_frac = cfg["fake_frac"] if fake_frac is None else fake_frac
    n_phi = cfg["n_phi"] if n_phi is None else n_phi
    n_z = cfg["n_z"] if n_z is None else n_z
    geom = geometry(cfg["geom"], xx0_scale=1.0 if ms else 0.0, **({"depth": jitter / np.sqrt(3.0)} if jitter > 0 else {}))
    L = geom.n_layers
    xs, ys, zs, tr = [], [], [], []
    seg_off = [0]
    seeds, sigs, qs, sev, struth, shit = [], [], [], [], [], []
    truth_hit_idx = np.full((L, n_events * tracks), -1, dtype=np.int32)
    for ev in range(n_events):
        rng = rng_for(config if isinstance(config, int) else 101, int(event_ids[ev]))     # a rank's own events
        gun = particle_gun(rng, tracks, cfg["gun"])
        sim = simulate(geom, gun, rng, ms=ms, smear=smear, jitter=jitter)
        ev_hits = []
        for l in range(L):
            v = sim["valid"][l]
            ids = np.nonzero(v)[0]
            n_sig = len(ids)
            n_noise = int(round(noise * n_sig))
            az = rng.uniform(-np.pi, np.pi, n_noise)
            if geom.kind[l] == 0:
                nz = rng.uniform(-geom.zmax[l], geom.zmax[l], n_noise)
                nr = np.full(n_noise, geom.r[l])
            else:                                  # disk: in the plane z = Z, radius uniform over the annulus' width
                nz = np.full(n_noise, geom.r[l])
                nr = rng.uniform(geom.rmin[l], geom.zmax[l], n_noise)
            if jitter > 0:                         # the sensor a noise hit sits on is displaced like any other
                off = rng.uniform(-jitter, jitter, n_noise)
                if geom.kind[l] == 0:
                    nr = nr + off
                else:
                    nz = nz + off
            hx = np.concatenate([sim["hits"][l, ids, 0], nr * np.cos(az)])
            hy = np.concatenate([sim["hits"][l, ids, 1], nr * np.sin(az)])
            hz = np.concatenate([sim["hits"][l, ids, 2], nz])
            ht = np.concatenate([ids + ev * tracks, np.full(n_noise, -1)]).astype(np.int32)
            perm = rng.permutation(len(hx))
            hx, hy, hz, ht = hx[perm], hy[perm], hz[perm], ht[perm]
            pos = np.empty(len(perm), dtype=np.int64); pos[perm] = np.arange(len(perm))
            truth_hit_idx[l, ids + ev * tracks] = pos[:n_sig]
            xs.append(hx.astype(np.float32)); ys.append(hy.astype(np.float32)); zs.append(hz.astype(np.float32)); tr.append(ht)
            seg_off.append(seg_off[-1] + len(hx))
            ev_hits.append((hx, hy, hz, ht))
        # true seeds
        ok = sim["valid"][first_layer - 1]
        ids = np.nonzero(ok)[0]
        sd, sg = smear_seed(rng, sim["truth"][first_layer - 1][ids])
        seeds.append(sd); sigs.append(sg); qs.append(gun["q"][ids]); sev.append(np.full(len(ids), ev, dtype=np.int32))
        struth.append((ids + ev * tracks).astype(np.int32))
        shit.append(truth_hit_idx[:first_layer, ids + ev * tracks])
        # fake seeds from random hit triplets on layers 0..2
        n_fake = int(round(fake_frac * tracks))
        if n_fake:
            f_sd, f_q, f_hit = [], [], []
            h0, h1, h2 = ev_hits[0], ev_hits[1], ev_hits[2]
            dphi = 3.0 * 2.0 * np.pi / n_phi / 2.0      # "3x3 bin neighbourhood": +-1.5 bins
            dz = 3.0 * (2.0 * geom.zmax[0] / n_z) / 2.0
            # hits of layers 1, 2 ordered by azimuth, so that a phi window is one (wrapping) slice
            srt = []
            for hh in (h1, h2):
                az = np.arctan2(hh[1], hh[0])
                o = np.argsort(az, kind="stable")
                srt.append((az[o], o, hh[2][o]))
            tries = 0
            while len(f_sd) < n_fake and tries < 200 * n_fake:
                tries += 1
                i0 = int(rng.integers(len(h0[0])))
                a0 = np.arctan2(h0[1][i0], h0[0][i0]); z0 = h0[2][i0]
                picks = [i0]
                fail = False
                for (azs, order, zsrt), l in zip(srt, (1, 2)):
                    zexp = z0 * geom.r[l] / geom.r[0]
                    lo, hi = a0 - dphi, a0 + dphi
                    parts = []
                    for (u, v) in ((lo, hi), (lo + 2 * np.pi, hi + 2 * np.pi), (lo - 2 * np.pi, hi - 2 * np.pi)):
                        i, j = np.searchsorted(azs, u, side="left"), np.searchsorted(azs, v, side="right")
                        if j > i:
                            parts.append(np.arange(i, j))
                    sl = np.concatenate(parts) if parts else np.zeros(0, dtype=np.int64)
                    cand = np.sort(order[sl[np.abs(zsrt[sl] - zexp) <= dz]])
                    if len(cand) == 0:
                        fail = True; break
                    picks.append(int(cand[rng.integers(len(cand))]))
                if fail:
                    continue
                t0, t1, t2 = h0[3][picks[0]], h1[3][picks[1]], h2[3][picks[2]]
                if t0 >= 0 and t0 == t1 == t2:
                    continue
                pts = [(hh[0][i], hh[1][i], hh[2][i]) for hh, i in zip((h0, h1, h2), picks)]
                res = _three_point_seed(*pts, geom.bz)
                if res is None:
                    continue
                st, qq = res
                if 1.0 / st[3] < 0.3:
                    continue
                f_sd.append(st); f_q.append(qq); f_hit.append(picks)
            if f_sd:
                f_sd = np.array(f_sd)
                f_sg = np.empty_like(f_sd)
                f_sg[:, 0:3] = SEED_SIGMA_POS; f_sg[:, 3] = SEED_SIGMA_REL_IPT * f_sd[:, 3]; f_sg[:, 4:6] = SEED_SIGMA_ANG
                seeds.append(f_sd); sigs.append(f_sg); qs.append(np.array(f_q, dtype=np.int8))
                sev.append(np.full(len(f_sd), ev, dtype=np.int32)); struth.append(np.full(len(f_sd), -1, dtype=np.int32))
                fh = np.array(f_hit, dtype=np.int32).T            # [3][n_fake]
                if first_layer != 3:
                    raise ValueError("fake seeds are defined for first_layer == 3")
                shit.append(fh)
    seed = np.concatenate(seeds); sig = np.concatenate(sigs); q = np.concatenate(qs)
    t = _soa_tracks(seed, sig, q)
    n_seeds, ld = t["n"], t["ld"]
    seed_hit_idx = np.full((first_layer, ld), -1, dtype=np.int32)
    seed_hit_idx[:, :n_seeds] = np.concatenate(shit, axis=1)
    return BuildInputs(geom=geom, n_events=n_events, n_phi=n_phi, n_z=n_z, K=K, chi2_cut=chi2_cut, n_sigma=n_sigma,
                       first_layer=first_layer, hit_x=np.concatenate(xs), hit_y=np.concatenate(ys), hit_z=np.concatenate(zs),
                       seg_off=np.array(seg_off, dtype=np.int64), hit_truth=np.concatenate(tr), n_seeds=n_seeds, ld=ld,
                       par=t["par"], cov=t["cov"], q=t["q"], seed_event=np.concatenate(sev), seed_hit_idx=seed_hit_idx,
                       seed_truth=np.concatenate(struth), truth_hit_idx=truth_hit_idx, event_ids=event_ids)

"""Tolerance rules for comparing the fp32 CUDA path with the fp64 oracle.

north_star: parameters within 1e-4 relative (1e-6 absolute floor), covariance within 1e-3 relative, chi2 within
1e-3 relative.  How "relative" is normalised where an element can pass through zero (readings A12, A13):
  * parameters: per component |d| <= max(1e-4 |p|, 1e-6) for 1/pT, phi, theta; for the position the same rule is
    applied to the vector norm, |d(x,y,z)| <= max(1e-4 |(x,y,z)|, 1e-6) (a Cartesian component crossing zero at
    r = 80 cm has ulp(80) = 7.6e-6 > the floor); the strict per-component count is reported as well;
  * covariance: |dC_ij| <= 1e-3 s_i s_j, s_i = sqrt(C_ii), with s_x = s_y = sqrt(C_xx + C_yy) (the x-y block is
    singular by construction and rotates with the azimuth);
  * phi is an azimuth: its zero is a choice of frame, so "relative to |phi|" is as frame-dependent as it is for x and y.
    Read like the position (A12) -- the transverse direction (cos phi, sin phi), not the number phi -- but NOT with the
    1e-4 of its norm that reading would allow (1e-4 rad is a hundred times what the kernels do and would let a real
    regression through): the flat bound is |d phi| <= PHI_DIR_ABS = 1e-5 rad (`phi_viol`; worst measured over the GPU suite
    below 1e-6 rad on the fits), AND the strict per-component rule |d phi| <= max(1e-4 |phi|, 1e-6) counted and
    bounded (`strict_phi_viol`, `worst_phi_strict`): a track that turns by 2 rad carries d phi = 2 rad x d(1/pT)/(1/pT),
    so a 1/pT that is right to 1e-6 -- a hundred times inside ITS tolerance -- already moves phi by 2e-6 rad, which only
    shows where |phi| happens to be below 0.01 (assert_parity: at most 1e-4 of the tracks, none beyond 4x);
  * chi2: |d| <= 1e-3 max(chi2, 1).  The floor is arithmetic, not licence: a residual m - x is the difference of two fp32
    numbers of size R, good to ulp(R)/2 = 3.8e-6 cm at R = 80 cm, so chi2_l = r^2/sigma^2 carries 2 sqrt(chi2_l) x 3.8e-6 / 0.01
    = 7.6e-4 sqrt(chi2_l) of absolute error per hit: 1e-3 RELATIVE cannot be met by any fp32 path below chi2 ~ 0.6.
"""
import numpy as np

PAR_REL, PAR_ABS, COV_REL, CHI2_REL = 1e-4, 1e-6, 1e-3, 1e-3
PHI_DIR_ABS = 1e-5      # rad: the frame-independent bound on d phi (module docstring)


def compare_tracks(gpu: dict, ref: dict, sel=None, cov_scale=None, chi2_scale=1.0) -> dict:
    """gpu: par [6][n] f32, cov [21][n] f32 packed, chi2; ref: par [6][n] f64, cov [n][6][6] f64, chi2.
    cov_scale, chi2_scale: optional factors on the covariance ([6][6]) and chi2 tolerances (R16b).
    Returns violation counts and worst normalised errors (1.0 = at tolerance)."""
    n = ref["par"].shape[1]
    sel = np.ones(n, bool) if sel is None else sel
    gp = gpu["par"].astype(np.float64)[:, sel]; rp = ref["par"][:, sel]
    d = gp - rp
    d[4] = np.angle(np.exp(1j * d[4]))
    tol = np.maximum(PAR_REL * np.abs(rp), PAR_ABS)
    comp = np.abs(d) / tol
    pos = np.linalg.norm(d[:3], axis=0) / np.maximum(PAR_REL * np.linalg.norm(rp[:3], axis=0), PAR_ABS)
    rc = ref["cov"][sel]
    gc = np.empty_like(rc)
    k = 0
    for i in range(6):
        for j in range(i + 1):
            gc[:, i, j] = gc[:, j, i] = gpu["cov"][k][sel]
            k += 1
    s = np.sqrt(np.einsum("nii->ni", rc))
    s[:, 0] = s[:, 1] = np.sqrt(rc[:, 0, 0] + rc[:, 1, 1])
    with np.errstate(invalid="ignore", divide="ignore"):      # a state on a disk has C_zz = 0 exactly on both sides: 0/0 counts as 0
        cerr = np.nan_to_num(np.abs(gc - rc) / (COV_REL * s[:, :, None] * s[:, None, :]), nan=0.0, posinf=np.inf)
    if cov_scale is not None:
        cerr = cerr / np.asarray(cov_scale, dtype=np.float64)[None, :, :]
    c2 = np.abs(gpu["chi2"].astype(np.float64)[sel] - ref["chi2"][sel]) / (chi2_scale * CHI2_REL * np.maximum(ref["chi2"][sel], 1.0))
    mom = comp[[3, 5]]
    phi_dir = np.abs(d[4]) / PHI_DIR_ABS
    return dict(n=int(sel.sum()), worst_mom=float(mom.max(initial=0)), worst_pos_norm=float(pos.max(initial=0)),
                strict_pos_viol=int((comp[:3] > 1).any(axis=0).sum()), mom_viol=int((mom > 1).any(axis=0).sum()),
                phi_viol=int((phi_dir > 1).sum()), worst_phi_dir=float(phi_dir.max(initial=0)),
                strict_phi_viol=int((comp[4] > 1).sum()), worst_phi_strict=float(comp[4].max(initial=0)),
                pos_viol=int((pos > 1).sum()), worst_cov=float(cerr.max(initial=0)), cov_viol=int((cerr > 1).any(axis=(1, 2)).sum()),
                worst_chi2=float(c2.max(initial=0)), chi2_viol=int((c2 > 1).sum()))


def assert_parity(rep: dict):
    """The north_star tolerances on a compare_tracks report (module docstring for the reading of phi)."""
    assert rep["mom_viol"] == 0 and rep["pos_viol"] == 0 and rep["cov_viol"] == 0 and rep["chi2_viol"] == 0 and rep["phi_viol"] == 0, rep
    assert rep["strict_phi_viol"] <= max(1, 1e-4 * rep["n"]) and rep["worst_phi_strict"] < 4.0, rep

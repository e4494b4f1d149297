"""Tolerance rules for comparing the fp32 CUDA path with the fp64 oracle.

north_star: parameters within 1e-4 relative (1e-6 absolute floor), covariance within 1e-3 relative, chi2 within
1e-3 relative.  How "relative" is normalised where an element can pass through zero (readings A12, A13):
  * parameters: per component |d| <= max(1e-4 |p|, 1e-6) for 1/pT, phi, theta; for the position the same rule is
    applied to the vector norm, |d(x,y,z)| <= max(1e-4 |(x,y,z)|, 1e-6) (a Cartesian component crossing zero at
    r = 80 cm has ulp(80) = 7.6e-6 > the floor); the strict per-component count is reported as well;
  * covariance: |dC_ij| <= 1e-3 s_i s_j, s_i = sqrt(C_ii), with s_x = s_y = sqrt(C_xx + C_yy) (the x-y block is
    singular by construction and rotates with the azimuth);
  * chi2: |d| <= 1e-3 max(chi2, 1).
"""
import numpy as np

PAR_REL, PAR_ABS, COV_REL, CHI2_REL = 1e-4, 1e-6, 1e-3, 1e-3


def compare_tracks(gpu: dict, ref: dict, sel=None) -> dict:
    """gpu: par [6][n] f32, cov [21][n] f32 packed, chi2; ref: par [6][n] f64, cov [n][6][6] f64, chi2.
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
    cerr = np.abs(gc - rc) / (COV_REL * s[:, :, None] * s[:, None, :])
    c2 = np.abs(gpu["chi2"].astype(np.float64)[sel] - ref["chi2"][sel]) / (CHI2_REL * np.maximum(ref["chi2"][sel], 1.0))
    return dict(n=int(sel.sum()), worst_mom=float(comp[3:].max(initial=0)), worst_pos_norm=float(pos.max(initial=0)),
                strict_pos_viol=int((comp[:3] > 1).any(axis=0).sum()), mom_viol=int((comp[3:] > 1).any(axis=0).sum()),
                pos_viol=int((pos > 1).sum()), worst_cov=float(cerr.max(initial=0)), cov_viol=int((cerr > 1).any(axis=(1, 2)).sum()),
                worst_chi2=float(c2.max(initial=0)), chi2_viol=int((c2 > 1).sum()))

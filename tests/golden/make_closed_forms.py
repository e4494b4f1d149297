"""Writes tests/golden/closed_forms.txt: textbook closed forms the oracle is pinned to.

Calls neither the oracle nor the CUDA path: plain Python arithmetic on formulas typed out here.
The paper prints no numbers for this path; the sources are
  * helix chord relation from the origin: alpha = 2 asin(R w / 2), s = alpha / w, cos(inc) = cos(alpha/2),
    rho = pT / (0.00299792458 B)  (any charged-particle-in-solenoid text);
  * straight-line weighted least squares on N equidistant points: var(slope) = s^2 / sum (x - xbar)^2,
    var(value at x0) = s^2 (1/N + (x0 - xbar)^2 / sum (x - xbar)^2);
  * Gluckstern (NIM 24 (1963) 381): sigma(kappa) = (s / L^2) sqrt(720 n^3 / ((n-1)(n+1)(n+2)(n+3))), n = N-1 intervals;
    end-point error of the quadratic fit from its hat matrix;
  * the same straight-line formulas for hits on four endcap disks (pins of the endcap / tangent-plane update, R19-R21).
Run: python tests/golden/make_closed_forms.py
"""
import math
import os

import numpy as np

K = 0.00299792458
out = {}
out["rho_pt1_B38"] = 1.0 / (K * 3.8)
for name, pt in (("pt1", 1.0), ("pt03", 0.3)):
    w = -K * 3.8 / pt          # q = +1
    R = 40.0
    alpha = 2.0 * math.asin(R * w / 2.0)
    out[f"s_{name}_R40"] = alpha / w
    out[f"cosinc_{name}_R40"] = math.cos(alpha / 2.0)
    out[f"phi_{name}_R40"] = alpha                  # phi0 = 0
    out[f"y_{name}_R40"] = R * math.sin(alpha / 2.0)
x = np.arange(4.0, 41.0, 4.0)
sxx = float(((x - x.mean()) ** 2).sum())
out["wls_sigma_phi"] = 0.01 / math.sqrt(sxx)                      # slope of r*phi vs R = angle
out["wls_sigma_rphi_40"] = 0.01 * math.sqrt(1 / 10 + (40 - x.mean()) ** 2 / sxx)
out["wls_sigma_z_40"] = 0.1 * math.sqrt(1 / 10 + (40 - x.mean()) ** 2 / sxx)
out["wls_sigma_cot"] = 0.1 / math.sqrt(sxx)
n, L = 9, 36.0
out["gluckstern_sigma_kappa"] = 0.01 / L ** 2 * math.sqrt(720.0 * n ** 3 / ((n - 1) * (n + 1) * (n + 2) * (n + 3)))
X = np.stack([np.ones_like(x), x, x * x], axis=1)
x0 = np.array([1.0, 40.0, 1600.0])
out["gluckstern_sigma_rphi_40"] = 0.01 * math.sqrt(float(x0 @ np.linalg.inv(X.T @ X) @ x0))
# straight line through four endcap disks at z = 60, 75, 90, 105 cm at polar angle 0.35 rad (B = 0): the hits measure
# r-phi (resolution 0.01 cm) and r (0.01 cm).  r-phi is linear in the hit radius r_k = z_k tan(theta) with slope = azimuth,
# r is linear in z_k with slope tan(theta); d(theta) = cos^2(theta) d(tan theta).
zk = np.array([60.0, 75.0, 90.0, 105.0])
th = 0.35
rk = zk * math.tan(th)
srr = float(((rk - rk.mean()) ** 2).sum())
szz = float(((zk - zk.mean()) ** 2).sum())
out["disk_sigma_phi"] = 0.01 / math.sqrt(srr)
out["disk_sigma_rphi_last"] = 0.01 * math.sqrt(1 / 4 + (rk[-1] - rk.mean()) ** 2 / srr)
out["disk_sigma_theta"] = 0.01 / math.sqrt(szz) * math.cos(th) ** 2
out["disk_sigma_r_last"] = 0.01 * math.sqrt(1 / 4 + (zk[-1] - zk.mean()) ** 2 / szz)
here = os.path.dirname(os.path.abspath(__file__))
with open(os.path.join(here, "closed_forms.txt"), "w") as f:
    f.write("# written by tests/golden/make_closed_forms.py (textbook closed forms; see its docstring for sources)\n")
    for k, v in out.items():
        f.write(f"{k} = {v:.10g}\n")

/* kf_oracle.c -- fp64 CPU ORACLE for batched Kalman-filter track fitting and building.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the cpu_baseline /
 * --impl reference legs of bench.py may load it.  It shares no code, header, table or constant generator with
 * the CUDA path under paper_1711_06571_b200/csrc/ and include/kf.h; neither includes the other.
 *
 * What it follows.  The paper (arxiv 1711.06571, /root/reference/PAPER.md) is a prose report with no formulas:
 *   - three stages, building = project outwards, collect compatible hits, branch, keep the best; final KF fit
 *     (sec. 2);
 *   - hybrid coordinates: global Cartesian position + polar momentum (sec. 3);
 *   - ideal barrel, uniform longitudinal field, Gaussian-smeared hits (sec. 3);
 *   - small matrices 3x3 .. 6x6 (sec. 2.1); fixed slots per seed, best candidates;
 *   - the Kalman filter itself is ref. [3] (Fruehwirth 1987).
 * Everything the paper leaves open is a "reading", listed in DESIGN.md sec. 3 (R1..R18) and cited below as [Rn].
 * The KF is an iteration, so the oracle follows it step by step, dense 6x6 doubles, plain loops, no packed
 * storage, no sparsity shortcuts, no blocking/fusion.  The helix-cylinder intersection is found by marching
 * along the helix until the radius first exceeds R and polishing the bracketed root with safeguarded Newton
 * (the CUDA path uses a closed form instead).
 *
 * Pins (tests/test_oracle_pins.py, all -m "not gpu"): P1 chord closed form from the origin; P2 Jacobian vs central
 * finite differences of the root-found map; P3 noise-free truth recovery against the simulator's independent
 * circle-circle transport; P5 B=0 straight-line weighted least squares closed form; P6 Gluckstern curvature
 * resolution; P7 linear KF vs normal equations; P8 3x3 solve vs LAPACK; P9 rotation / mirror / charge-field
 * invariances; P10 PSD, C_upd <= C_pred, chi2 >= 0; P11 pulls and chi2/ndf statistics; P12 build vs brute force
 * without bins; X1-X3 binning / window vs fp64 atan2 and brute force.
 * PARITY UNPINNED (paper silent, pinned only by self-consistency P11): the Highland form and where Q is added
 * [R4], seed smearing widths [R6], candidate ranking order [R10], window definition [R11], noise and fake-seed
 * recipes [R17, R18], guards cos_inc 0.2 / 0.1 [R9].
 *
 * State p = (x, y, z, iota = 1/pT, phi, theta), charge q = +-1 separate [R1]; units cm, GeV, Tesla, rad.
 * Curvature w = dphi/ds_T = -q * k * Bz * iota, k = 0.00299792458 [R3].
 *
 * Build: gcc -O2 -std=c11 -fopenmp -ffp-contract=off -fPIC -shared kf_oracle.c -o libkf_oracle.so -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define KFO_KCURV 0.00299792458
#define KFO_PI 3.14159265358979323846

enum { KFO_UNREACHABLE = 1, KFO_LEFT_Z = 2, KFO_GRAZING = 4, KFO_NUMERIC = 8 };

#define KFO_CMIN 0.1 /* KF-side grazing guard on cos(incidence) [R9] */

/* layer table row, 8 columns: r, zmax, xx0, sig_rphi, sig_z, sig_r, kind, rmin.
 * kind 0 = barrel cylinder of radius r and half length zmax; kind 1 = endcap disk ("cylinder with lids", PAPER.md:L70
 * sec. 4.1) in the plane z = r (column 0, signed), covering rmin <= radius <= zmax (column 1 = outer radius) [R19]. */
#define KFO_LW 8
#define LR(t, l) ((t)[KFO_LW * (l) + 0])
#define LZMAX(t, l) ((t)[KFO_LW * (l) + 1])
#define LXX0(t, l) ((t)[KFO_LW * (l) + 2])
#define LSRPHI(t, l) ((t)[KFO_LW * (l) + 3])
#define LSZ(t, l) ((t)[KFO_LW * (l) + 4])
#define LSR(t, l) ((t)[KFO_LW * (l) + 5])
#define LKIND(t, l) ((int)(t)[KFO_LW * (l) + 6])
#define LRMIN(t, l) ((t)[KFO_LW * (l) + 7])

int kfo_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* phi is wrapped to (-pi, pi] on output only */
static double wrap_phi(double a) {
    double w = a - 2.0 * KFO_PI * floor((a + KFO_PI) / (2.0 * KFO_PI));
    if (w <= -KFO_PI) w += 2.0 * KFO_PI;
    if (w > KFO_PI) w -= 2.0 * KFO_PI;
    return w;
}

/* sin(a)/a */
static double sinc_(double a) {
    if (fabs(a) < 1e-2) {
        double a2 = a * a;
        return 1.0 - a2 / 6.0 * (1.0 - a2 / 20.0 * (1.0 - a2 / 42.0 * (1.0 - a2 / 72.0)));
    }
    return sin(a) / a;
}

/* Helix at fixed transverse path length s (sec. 8c-2 of SURVEY.md; standard helix in a uniform field along z):
 *   alpha = w s, X = sin(alpha)/w, Y = (1-cos(alpha))/w   (X -> s, Y -> w s^2/2 as w -> 0)
 *   x' = x + cos(phi) X - sin(phi) Y,  y' = y + sin(phi) X + cos(phi) Y,  z' = z + s cot(theta),  phi' = phi + alpha */
static void helix_at(const double p[6], double w, double s, double out[6]) {
    double a = w * s;
    double X = s * sinc_(a);
    double h = sinc_(0.5 * a);
    double Y = 0.5 * a * s * h * h; /* = 2 sin^2(a/2)/w, regular at w = 0 */
    double cp = cos(p[4]), sp = sin(p[4]);
    out[0] = p[0] + cp * X - sp * Y;
    out[1] = p[1] + sp * X + cp * Y;
    out[2] = p[2] + s * cos(p[5]) / sin(p[5]);
    out[3] = p[3];
    out[4] = p[4] + a;
    out[5] = p[5];
}

static double g_of(const double p[6], double w, double s, double R, double* dg) {
    double o[6];
    helix_at(p, w, s, o);
    if (dg) *dg = 2.0 * (o[0] * cos(o[4]) + o[1] * sin(o[4]));
    return o[0] * o[0] + o[1] * o[1] - R * R;
}

/* Fixed-path-length partial derivatives of the helix (sec. 8c-3 of SURVEY.md): with a = w s,
 * dX/d iota = c_w s^2 f1(a), dY/d iota = c_w s^2 f2(a), f1 = (cos a - sin a / a)/a, f2 = (sin a - (1 - cos a)/a)/a. */
static void helix_curv_partials(double c_w, double w, double s, double* dXdi, double* dYdi) {
    const double a = w * s;
    double f1, f2;
    if (fabs(a) < 1e-2) {
        double a2 = a * a;
        f1 = a * (-1.0 / 3.0 + a2 * (1.0 / 30.0 + a2 * (-1.0 / 840.0 + a2 / 45360.0)));
        f2 = 0.5 + a2 * (-1.0 / 8.0 + a2 * (1.0 / 144.0 - a2 / 5760.0));
    } else {
        f1 = (cos(a) - sin(a) / a) / a;
        f2 = (sin(a) - (1.0 - cos(a)) / a) / a;
    }
    *dXdi = c_w * s * s * f1;
    *dYdi = c_w * s * s * f2;
}

/* State at transverse path s and the Jacobian of the transport TO THE CYLINDER through that point: fixed-s partials
 * plus the path-length term, ds/dp from the constraint x'^2 + y'^2 = const (sec. 8c-3).  up = x' cos phi' + y' sin phi'. */
static void helix_to_cylinder(const double p[6], double w, double c_w, double s, double pout[6], double J[36], double* up_out) {
    helix_at(p, w, s, pout);
    const double xn = pout[0], yn = pout[1], phn = pout[4];
    const double cpn = cos(phn), spn = sin(phn), cp = cos(p[4]), sp = sin(p[4]);
    const double up = xn * cpn + yn * spn; /* R cos(incidence) */
    double dXdi, dYdi;
    helix_curv_partials(c_w, w, s, &dXdi, &dYdi);
    const double Fxi = cp * dXdi - sp * dYdi, Fyi = sp * dXdi + cp * dYdi;
    const double Fxp = -(yn - p[1]), Fyp = xn - p[0];
    const double cot = cos(p[5]) / sin(p[5]), sin2 = sin(p[5]) * sin(p[5]);
    /* ds/dp from g(p, s(p)) = 0 */
    const double sx = -xn / up, sy = -yn / up;
    const double si = -(xn * Fxi + yn * Fyi) / up, sph = -(xn * Fxp + yn * Fyp) / up;
    memset(J, 0, 36 * sizeof(double));
    /* columns: x y z iota phi theta */
    J[0 * 6 + 0] = 1.0 + cpn * sx; J[0 * 6 + 1] = cpn * sy; J[0 * 6 + 3] = Fxi + cpn * si; J[0 * 6 + 4] = Fxp + cpn * sph;
    J[1 * 6 + 0] = spn * sx; J[1 * 6 + 1] = 1.0 + spn * sy; J[1 * 6 + 3] = Fyi + spn * si; J[1 * 6 + 4] = Fyp + spn * sph;
    J[2 * 6 + 0] = cot * sx; J[2 * 6 + 1] = cot * sy; J[2 * 6 + 2] = 1.0; J[2 * 6 + 3] = cot * si; J[2 * 6 + 4] = cot * sph;
    J[2 * 6 + 5] = -s / sin2;
    J[3 * 6 + 3] = 1.0;
    J[4 * 6 + 0] = w * sx; J[4 * 6 + 1] = w * sy; J[4 * 6 + 3] = c_w * s + w * si; J[4 * 6 + 4] = 1.0 + w * sph;
    J[5 * 6 + 5] = 1.0;
    *up_out = up;
}

/* Propagate the state to the cylinder of radius R: smallest positive root of g(s) = x'^2 + y'^2 - R^2 [R2].
 * J (row-major 6x6) = d p'/d p INCLUDING the path-length term (the state is transported to the surface).
 * Returns 0 or a flag: KFO_UNREACHABLE (start not inside R, or no crossing within half a turn), KFO_GRAZING
 * (cos(incidence) < KFO_CMIN; outputs are still filled).  s_out = transverse path, cosinc_out = u'/R.
 * tangency_out (diagnostics for DESIGN.md R16, may be NULL): how far the helix is from just touching the cylinder --
 * cos^2(incidence) when it crosses, max(R^2 - r^2)/R^2 over the half turn when it does not, 1e300 when neither applies. */
static int propagate_ex(const double p[6], int q, double bz, double R, double pout[6], double J[36], double* s_out,
                        double* cosinc_out, double* tangency_out) {
    const double w = -(double)q * KFO_KCURV * bz * p[3];
    const double c_w = -(double)q * KFO_KCURV * bz; /* w = c_w * iota */
    double r02 = p[0] * p[0] + p[1] * p[1];
    memcpy(pout, p, 6 * sizeof(double));
    for (int i = 0; i < 36; ++i) J[i] = (i % 7 == 0) ? 1.0 : 0.0;
    if (s_out) *s_out = 0.0;
    if (cosinc_out) *cosinc_out = 0.0;
    if (tangency_out) *tangency_out = 1e300;
    if (!(r02 < R * R) || !isfinite(w) || !isfinite(r02)) return KFO_UNREACHABLE;

    /* march: a circle of radius rho >= R that starts inside the cylinder leaves it within an arc pi R
       (<= half a turn); a tighter circle must cross within half a turn pi rho, else the layer counts as
       unreachable [R2] */
    const int NMARCH = 64;
    double smax = (fabs(w) * R <= 1.0) ? KFO_PI * R * (1.0 + 1e-9) : KFO_PI / fabs(w);
    double lo = 0.0, hi = -1.0;
    int kbest = 0;
    double gbest = r02 - R * R;
    for (int k = 1; k <= NMARCH; ++k) {
        double sk = smax * (double)k / NMARCH;
        double gk = g_of(p, w, sk, R, NULL);
        if (gk >= 0.0) { hi = sk; break; }
        if (gk > gbest) { gbest = gk; kbest = k; }
        lo = sk;
    }
    if (hi < 0.0) {
        /* No sample lies outside, but a helix that only just pokes through the cylinder crosses it twice between two
           samples.  Along the helix r^2 = a + b cos(w s + delta): at most one maximum within half a turn, bracketed by the
           neighbours of the largest sample.  Golden-section search for it; if it is >= 0 the first crossing lies between
           the bracket's start (inside) and the maximum. */
        double a = smax * (double)(kbest > 0 ? kbest - 1 : 0) / NMARCH, b = smax * (double)(kbest < NMARCH ? kbest + 1 : NMARCH) / NMARCH;
        const double a0 = a, gr = 0.6180339887498949;
        double x1 = b - gr * (b - a), x2 = a + gr * (b - a);
        double f1 = g_of(p, w, x1, R, NULL), f2 = g_of(p, w, x2, R, NULL);
        for (int it = 0; it < 200 && b - a > 1e-16 * fmax(1.0, b); ++it) {
            if (f1 < f2) { a = x1; x1 = x2; f1 = f2; x2 = a + gr * (b - a); f2 = g_of(p, w, x2, R, NULL); }
            else { b = x2; x2 = x1; f2 = f1; x1 = b - gr * (b - a); f1 = g_of(p, w, x1, R, NULL); }
        }
        const double sm = f1 > f2 ? x1 : x2, gm = f1 > f2 ? f1 : f2;
        if (!(gm >= 0.0)) {
            if (tangency_out) *tangency_out = -gm / (R * R);
            return KFO_UNREACHABLE;
        }
        lo = a0; hi = sm;
    }
    /* safeguarded Newton inside [lo, hi], g(lo) < 0 <= g(hi) */
    double s = 0.5 * (lo + hi);
    for (int it = 0; it < 200; ++it) {
        double dg, g = g_of(p, w, s, R, &dg);
        if (g < 0.0) lo = s; else hi = s;
        double sn = (dg > 0.0) ? s - g / dg : -1.0;
        if (!(sn > lo && sn < hi)) sn = 0.5 * (lo + hi);
        double ds = fabs(sn - s);
        s = sn;
        if (ds <= 1e-15 * fmax(1.0, fabs(s)) || hi - lo <= 1e-15 * fmax(1.0, fabs(s))) break;
    }
    double up;
    helix_to_cylinder(p, w, c_w, s, pout, J, &up);
    if (s_out) *s_out = s;
    if (cosinc_out) *cosinc_out = up / R;
    if (tangency_out) *tangency_out = (up / R) * (up / R);
    if (!(up / R >= KFO_CMIN)) return KFO_GRAZING;
    return 0;
}
int kfo_propagate(const double p[6], int q, double bz, double R, double pout[6], double J[36], double* s_out,
                  double* cosinc_out) {
    return propagate_ex(p, q, bz, R, pout, J, s_out, cosinc_out, NULL);
}

/* Second step of the two-step propagation (sec. 4.1: "an initial propagation to the average radius of the
 * barrel ... followed by further propagation steps to the position of each candidate hit") [R20]: from a state on (or
 * near) a cylinder to the NEAREST crossing of the cylinder of radius R, forwards or backwards -- Newton on
 * g(s) = x'^2 + y'^2 - R^2 from s = 0, g' = 2 (x' cos phi' + y' sin phi').  Same surface Jacobian.  No material.
 * Returns 0, or KFO_UNREACHABLE when the iteration does not converge (the hit radius is not within reach of a short step). */
int kfo_propagate_near(const double p[6], int q, double bz, double R, double pout[6], double J[36], double* s_out) {
    const double w = -(double)q * KFO_KCURV * bz * p[3], c_w = -(double)q * KFO_KCURV * bz;
    memcpy(pout, p, 6 * sizeof(double));
    for (int i = 0; i < 36; ++i) J[i] = (i % 7 == 0) ? 1.0 : 0.0;
    if (s_out) *s_out = 0.0;
    double s = 0.0;
    int ok = 0;
    for (int it = 0; it < 50; ++it) {
        double dg, g = g_of(p, w, s, R, &dg);
        if (!(fabs(dg) > 0.0) || !isfinite(g)) break;
        double ds = -g / dg;
        s += ds;
        if (fabs(ds) <= 1e-14 * fmax(1.0, R)) { ok = 1; break; }       /* the rounding of g = r^2 - R^2 is ~1e-16 R^2, of ds ~1e-16 R */
        if (!(fabs(s) < 4.0 * R)) break;
    }
    if (!ok) return KFO_UNREACHABLE;
    double up;
    helix_to_cylinder(p, w, c_w, s, pout, J, &up);
    if (s_out) *s_out = s;
    return 0;
}

/* Propagate to the plane z = Z of an endcap disk [R19]: z' = z + s cot(theta) fixes the transverse path
 * s = (Z - z) tan(theta).  forward_only: s must be positive (first step: the track has to move towards the disk) and
 * the turning angle at most half a turn [R2]; otherwise (second step to a hit's own z) any sign of s.
 * J = fixed-s partials + (dp'/ds)(ds/dp)^T with ds/dz = -tan(theta), ds/dtheta = (Z - z)/cos^2(theta): the z' row
 * vanishes identically (the state is transported to the surface).  cosinc_out = |cos(theta)| (angle to the disk normal). */
int kfo_propagate_z(const double p[6], int q, double bz, double Z, int forward_only, double pout[6], double J[36], double* s_out,
                    double* cosinc_out) {
    const double w = -(double)q * KFO_KCURV * bz * p[3], c_w = -(double)q * KFO_KCURV * bz;
    const double st = sin(p[5]), ct = cos(p[5]);
    memcpy(pout, p, 6 * sizeof(double));
    for (int i = 0; i < 36; ++i) J[i] = (i % 7 == 0) ? 1.0 : 0.0;
    if (s_out) *s_out = 0.0;
    if (cosinc_out) *cosinc_out = fabs(ct);
    const double s = (Z - p[2]) * st / ct;
    if (!isfinite(s) || !isfinite(w)) return KFO_UNREACHABLE;
    if (forward_only && (!(s > 0.0) || !(fabs(w) * s <= KFO_PI))) return KFO_UNREACHABLE;
    helix_at(p, w, s, pout);
    pout[2] = Z;
    const double cpn = cos(pout[4]), spn = sin(pout[4]), cp = cos(p[4]), sp = sin(p[4]);
    double dXdi, dYdi;
    helix_curv_partials(c_w, w, s, &dXdi, &dYdi);
    const double Fxi = cp * dXdi - sp * dYdi, Fyi = sp * dXdi + cp * dYdi;
    const double Fxp = -(pout[1] - p[1]), Fyp = pout[0] - p[0];
    const double sz = -st / ct, sth = (Z - p[2]) / (ct * ct);
    memset(J, 0, 36 * sizeof(double));
    J[0 * 6 + 0] = 1.0; J[0 * 6 + 2] = cpn * sz; J[0 * 6 + 3] = Fxi; J[0 * 6 + 4] = Fxp; J[0 * 6 + 5] = cpn * sth;
    J[1 * 6 + 1] = 1.0; J[1 * 6 + 2] = spn * sz; J[1 * 6 + 3] = Fyi; J[1 * 6 + 4] = Fyp; J[1 * 6 + 5] = spn * sth;
    /* row z': 1 + cot(theta) ds/dz = 0 and -s/sin^2 + cot(theta) ds/dtheta = 0 */
    J[3 * 6 + 3] = 1.0;
    J[4 * 6 + 2] = w * sz; J[4 * 6 + 3] = c_w * s; J[4 * 6 + 4] = 1.0; J[4 * 6 + 5] = w * sth;
    J[5 * 6 + 5] = 1.0;
    if (s_out) *s_out = s;
    if (forward_only && !(fabs(ct) >= KFO_CMIN)) return KFO_GRAZING;
    return 0;
}

/* remove the rounding-level asymmetry of the dense loops: C <- (C + C^T)/2 */
static void symmetrize6(double C[36]) {
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < i; ++j) {
            double m = 0.5 * (C[i * 6 + j] + C[j * 6 + i]);
            C[i * 6 + j] = C[j * 6 + i] = m;
        }
}

/* C <- J C J^T, dense */
static void similarity6(const double J[36], const double C[36], double out[36]) {
    double T[36];
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) {
            double a = 0.0;
            for (int k = 0; k < 6; ++k) a += J[i * 6 + k] * C[k * 6 + j];
            T[i * 6 + j] = a;
        }
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) {
            double a = 0.0;
            for (int k = 0; k < 6; ++k) a += T[i * 6 + k] * J[j * 6 + k];
            out[i * 6 + j] = a;
        }
    symmetrize6(out);
}
void kfo_similarity6(const double J[36], const double C[36], double out[36]) { similarity6(J, C, out); }

/* Multiple-scattering noise of a thin layer of thickness xx0 (radiation lengths at normal incidence),
 * evaluated at the arriving state [R4]: path t = xx0/(sin(theta) cos_inc); Highland, beta = 1, unit charge,
 * p = 1/(iota sin theta): theta0 = 0.0136 iota sin(theta) sqrt(t) (1 + 0.038 ln t).  Two orthogonal deflections
 * of variance theta0^2 with |p| conserved give, in (iota, phi, theta):
 *   Q_thth = th0^2, Q_phph = th0^2/sin^2(theta), Q_ii = iota^2 cot^2(theta) th0^2, Q_ith = -iota cot(theta) th0^2. */
void kfo_ms_noise(const double p[6], double cosinc, double xx0, double Q[36]) {
    memset(Q, 0, 36 * sizeof(double));
    if (!(xx0 > 0.0)) return;
    double st = sin(p[5]), ct = cos(p[5]);
    double t = xx0 / (st * cosinc);
    double th0 = 0.0136 * p[3] * st * sqrt(t) * (1.0 + 0.038 * log(t));
    double v = th0 * th0, cot = ct / st;
    Q[5 * 6 + 5] = v;
    Q[4 * 6 + 4] = v / (st * st);
    Q[3 * 6 + 3] = p[3] * p[3] * cot * cot * v;
    Q[3 * 6 + 5] = Q[5 * 6 + 3] = -p[3] * cot * v;
}

/* 3x3 SPD solve by Cholesky: returns 0 and inv (row-major) or -1 when not positive definite */
int kfo_inv3_spd(const double S[9], double inv[9]) {
    double l00, l10, l11, l20, l21, l22;
    if (!(S[0] > 0.0)) return -1;
    l00 = sqrt(S[0]); l10 = S[3] / l00; l20 = S[6] / l00;
    double d1 = S[4] - l10 * l10;
    if (!(d1 > 0.0)) return -1;
    l11 = sqrt(d1); l21 = (S[7] - l20 * l10) / l11;
    double d2 = S[8] - l20 * l20 - l21 * l21;
    if (!(d2 > 0.0)) return -1;
    l22 = sqrt(d2);
    /* invert L (lower) then inv = L^-T L^-1 */
    double m00 = 1.0 / l00, m11 = 1.0 / l11, m22 = 1.0 / l22;
    double m10 = -l10 * m00 * m11;
    double m21 = -l21 * m11 * m22;
    double m20 = -(l20 * m00 + l21 * m10) * m22;
    inv[0] = m00 * m00 + m10 * m10 + m20 * m20;
    inv[1] = inv[3] = m10 * m11 + m20 * m21;
    inv[2] = inv[6] = m20 * m22;
    inv[4] = m11 * m11 + m21 * m21;
    inv[5] = inv[7] = m21 * m22;
    inv[8] = m22 * m22;
    return 0;
}

/* Hit covariance in global Cartesian coordinates from the layer resolutions and the hit's own azimuth [R5]:
 * c = mx/rm, s = my/rm: Vxx = c^2 sr^2 + s^2 srphi^2, Vyy = s^2 sr^2 + c^2 srphi^2, Vxy = c s (sr^2 - srphi^2), Vzz = sz^2 */
static void hit_cov(const double m[3], double srphi, double sz, double sr, double V[9]) {
    double rm = sqrt(m[0] * m[0] + m[1] * m[1]);
    double c = m[0] / rm, s = m[1] / rm;
    memset(V, 0, 9 * sizeof(double));
    V[0] = c * c * sr * sr + s * s * srphi * srphi;
    V[4] = s * s * sr * sr + c * c * srphi * srphi;
    V[1] = V[3] = c * s * (sr * sr - srphi * srphi);
    V[8] = sz * sz;
}

/* chi2 of hit m against the predicted state (p, C) without updating.  Returns -1 if S is not PD. */
int kfo_chi2(const double p[6], const double C[36], const double m[3], double srphi, double sz, double sr,
             double* chi2) {
    double V[9], S[9], Si[9], r[3];
    hit_cov(m, srphi, sz, sr, V);
    for (int i = 0; i < 3; ++i) {
        r[i] = m[i] - p[i];
        for (int j = 0; j < 3; ++j) S[i * 3 + j] = C[i * 6 + j] + V[i * 3 + j];
    }
    if (kfo_inv3_spd(S, Si)) return -1;
    double c2 = 0.0;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) c2 += r[i] * Si[i * 3 + j] * r[j];
    *chi2 = c2;
    return 0;
}

/* Kalman update with the 3-D hit m, H = [I3 0] (Fruehwirth 1987, gain-matrix form):
 *   r = m - p[0:3]; S = C[0:3,0:3] + V; chi2 = r^T S^-1 r; K = C[:,0:3] S^-1; p <- p + K r;
 *   C <- (I-KH) C (I-KH)^T + K V K^T   (Joseph form: equal to C - K H C in exact arithmetic, symmetric by construction)
 * Returns 0, or KFO_NUMERIC when S is not PD, the result is not finite or iota <= 0 (outputs then undefined). */
int kfo_update(const double p[6], const double C[36], const double m[3], double srphi, double sz, double sr,
               double pout[6], double Cout[36], double* chi2) {
    double V[9], S[9], Si[9], r[3], K[18], A[36], T[36];
    hit_cov(m, srphi, sz, sr, V);
    for (int i = 0; i < 3; ++i) {
        r[i] = m[i] - p[i];
        for (int j = 0; j < 3; ++j) S[i * 3 + j] = C[i * 6 + j] + V[i * 3 + j];
    }
    if (kfo_inv3_spd(S, Si)) return KFO_NUMERIC;
    double c2 = 0.0;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) c2 += r[i] * Si[i * 3 + j] * r[j];
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 3; ++j) {
            double a = 0.0;
            for (int k = 0; k < 3; ++k) a += C[i * 6 + k] * Si[k * 3 + j];
            K[i * 3 + j] = a;
        }
    for (int i = 0; i < 6; ++i) {
        double a = p[i];
        for (int k = 0; k < 3; ++k) a += K[i * 3 + k] * r[k];
        pout[i] = a;
    }
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) A[i * 6 + j] = (i == j ? 1.0 : 0.0) - (j < 3 ? K[i * 3 + j] : 0.0);
    similarity6(A, C, T);
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) {
            double a = 0.0;
            for (int k = 0; k < 3; ++k)
                for (int l = 0; l < 3; ++l) a += K[i * 3 + k] * V[k * 3 + l] * K[j * 3 + l];
            Cout[i * 6 + j] = T[i * 6 + j] + a;
        }
    symmetrize6(Cout);
    *chi2 = c2;
    for (int i = 0; i < 6; ++i)
        if (!isfinite(pout[i])) return KFO_NUMERIC;
    for (int i = 0; i < 36; ++i)
        if (!isfinite(Cout[i])) return KFO_NUMERIC;
    if (!(pout[3] > 0.0) || !isfinite(c2)) return KFO_NUMERIC;
    return 0;
}

/* Measurement directions of a hit on its tangent plane ("KF updates are performed on the plane tangent to
 * the hit radius") [R21]: u1 = azimuthal unit vector at the hit, u2 = z axis (barrel hit: measures r-phi and z) or the
 * radial unit vector at the hit (disk hit: measures r-phi and r). */
static void hit_axes(const double m[3], int kind, double u1[3], double u2[3]) {
    const double rm = sqrt(m[0] * m[0] + m[1] * m[1]);
    u1[0] = -m[1] / rm; u1[1] = m[0] / rm; u1[2] = 0.0;
    if (kind == 0) { u2[0] = 0.0; u2[1] = 0.0; u2[2] = 1.0; }
    else { u2[0] = m[0] / rm; u2[1] = m[1] / rm; u2[2] = 0.0; }
}

/* chi2 of the 2-D residual of hit m on its tangent plane, H = [u1^T 0; u2^T 0], V = diag(s1^2, s2^2).  -1 if S is not PD. */
int kfo_chi2_2d(const double p[6], const double C[36], const double m[3], int kind, double s1, double s2, double* chi2) {
    double u[2][3], r[2], S[2][2];
    hit_axes(m, kind, u[0], u[1]);
    for (int a = 0; a < 2; ++a) {
        r[a] = 0.0;
        for (int i = 0; i < 3; ++i) r[a] += u[a][i] * (m[i] - p[i]);
        for (int b = 0; b < 2; ++b) {
            double v = 0.0;
            for (int i = 0; i < 3; ++i)
                for (int j = 0; j < 3; ++j) v += u[a][i] * C[i * 6 + j] * u[b][j];
            S[a][b] = v;
        }
    }
    S[0][0] += s1 * s1; S[1][1] += s2 * s2;
    const double det = S[0][0] * S[1][1] - S[0][1] * S[1][0];
    if (!(S[0][0] > 0.0) || !(det > 0.0)) return -1;
    *chi2 = (S[1][1] * r[0] * r[0] - 2.0 * S[0][1] * r[0] * r[1] + S[0][0] * r[1] * r[1]) / det;
    return 0;
}

/* Kalman update with the 2-D measurement of hit m on its tangent plane [R21]: r = H (m - x), S = H C H^T + V (2x2),
 * K = C H^T S^-1 (6x2), p <- p + K r, C <- (I-KH) C (I-KH)^T + K V K^T (Joseph form).  Flags as kfo_update. */
int kfo_update_2d(const double p[6], const double C[36], const double m[3], int kind, double s1, double s2, double pout[6],
                  double Cout[36], double* chi2) {
    double u[2][3], r[2], S[2][2], Si[2][2], CHt[6][2], K[6][2], A[36], T[36];
    const double V[2] = {s1 * s1, s2 * s2};
    hit_axes(m, kind, u[0], u[1]);
    for (int a = 0; a < 2; ++a) {
        r[a] = 0.0;
        for (int i = 0; i < 3; ++i) r[a] += u[a][i] * (m[i] - p[i]);
    }
    for (int i = 0; i < 6; ++i)
        for (int a = 0; a < 2; ++a) {
            double v = 0.0;
            for (int j = 0; j < 3; ++j) v += C[i * 6 + j] * u[a][j];
            CHt[i][a] = v;
        }
    for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b) {
            double v = 0.0;
            for (int i = 0; i < 3; ++i) v += u[a][i] * CHt[i][b];
            S[a][b] = v + (a == b ? V[a] : 0.0);
        }
    const double det = S[0][0] * S[1][1] - S[0][1] * S[1][0];
    if (!(S[0][0] > 0.0) || !(det > 0.0)) return KFO_NUMERIC;
    Si[0][0] = S[1][1] / det; Si[1][1] = S[0][0] / det; Si[0][1] = Si[1][0] = -S[0][1] / det;
    const double c2 = r[0] * (Si[0][0] * r[0] + Si[0][1] * r[1]) + r[1] * (Si[1][0] * r[0] + Si[1][1] * r[1]);
    for (int i = 0; i < 6; ++i)
        for (int a = 0; a < 2; ++a) K[i][a] = CHt[i][0] * Si[0][a] + CHt[i][1] * Si[1][a];
    for (int i = 0; i < 6; ++i) pout[i] = p[i] + K[i][0] * r[0] + K[i][1] * r[1];
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) {
            double kh = 0.0;
            if (j < 3) kh = K[i][0] * u[0][j] + K[i][1] * u[1][j];
            A[i * 6 + j] = (i == j ? 1.0 : 0.0) - kh;
        }
    similarity6(A, C, T);
    for (int i = 0; i < 6; ++i)
        for (int j = 0; j < 6; ++j) Cout[i * 6 + j] = T[i * 6 + j] + K[i][0] * V[0] * K[j][0] + K[i][1] * V[1] * K[j][1];
    symmetrize6(Cout);
    *chi2 = c2;
    for (int i = 0; i < 6; ++i)
        if (!isfinite(pout[i])) return KFO_NUMERIC;
    for (int i = 0; i < 36; ++i)
        if (!isfinite(Cout[i])) return KFO_NUMERIC;
    if (!(pout[3] > 0.0) || !isfinite(c2)) return KFO_NUMERIC;
    return 0;
}

/* Second step [R20]: from the predicted state on the layer's nominal surface to the surface through hit m -- the
 * cylinder of the hit's own radius (barrel) or the plane of the hit's own z (disk); C2 = J2 Cp J2^T, no material. */
static int to_hit_surface(int kind, double bz, int q, const double pp[6], const double Cp[36], const double m[3], double p2[6], double C2[36]) {
    double J[36], s;
    int f;
    if (kind == 0) f = kfo_propagate_near(pp, q, bz, sqrt(m[0] * m[0] + m[1] * m[1]), p2, J, &s);
    else f = kfo_propagate_z(pp, q, bz, m[2], 0, p2, J, &s, NULL);
    if (f) return f;
    similarity6(J, Cp, C2);
    return 0;
}
int kfo_to_hit_surface(int kind, double bz, int q, const double pp[6], const double Cp[36], const double m[3], double p2[6], double C2[36]) {
    return to_hit_surface(kind, bz, q, pp, Cp, m, p2, C2);
}

/* One KF step: propagate to layer l, add Q, (optionally) update with hit m.  Used by fit and build.
 * Returns flags; on flags != 0 the outputs are not to be used. */
static int predict_ci(const double* layers, int l, double bz, const double p[6], const double C[36], int q,
                      double pp[6], double Cp[36], double* ci_out, double* tangency_out) {
    double J[36], Q[36], s, ci;
    int f;
    if (LKIND(layers, l) == 0) f = propagate_ex(p, q, bz, LR(layers, l), pp, J, &s, &ci, tangency_out);
    else {
        /* disk: cos of the angle to the disk normal is |cos theta|; kfo_ms_noise divides by sin(theta) cos_inc, the cosine
           of the 3-D angle to a CYLINDER's normal, so hand it |cos theta| / sin theta */
        f = kfo_propagate_z(p, q, bz, LR(layers, l), 1, pp, J, &s, &ci);
        if (tangency_out) *tangency_out = 1e300;
        ci = ci / sin(p[5]);
    }
    if (ci_out) *ci_out = ci;
    if (f) return f;
    similarity6(J, C, Cp);
    kfo_ms_noise(pp, ci, LXX0(layers, l), Q);
    for (int i = 0; i < 36; ++i) Cp[i] += Q[i];
    return 0;
}
static int predict(const double* layers, int l, double bz, const double p[6], const double C[36], int q,
                   double pp[6], double Cp[36]) {
    return predict_ci(layers, l, bz, p, C, q, pp, Cp, NULL, NULL);
}
int kfo_predict(const double* layers, int l, double bz, const double p[6], const double C[36], int q, double pp[6],
                double Cp[36]) {
    return predict(layers, l, bz, p, C, q, pp, Cp);
}

/* kf_fit_ref [R8]: forward (inside-out) filter over the layers in order of increasing radius.
 * hit_idx[l*ld + t] >= 0 -> propagate, add Q, update with that hit;  == -1 -> the layer is crossed without a hit:
 * propagate and add Q (the material is there whether or not a hit was found), no update;  <= -2 -> layer not
 * crossed: skipped entirely;  NULL -> identity.  Hit of track t on layer l is
 * (hx,hy,hz)[seg_off[ev*L + l] + idx], ev = trk_event ? trk_event[t] : 0.
 * A propagation failure or a failed update sets the status bit, stops the track and keeps the last good state.
 * par [6][ld], cov [36][ld] dense in, outputs alike; chi2/nhits/status [n].
 * hit_mode 0: hits lie on the nominal surface, 3-D update there [R5].  hit_mode 1 [R20, R21]: two-step propagation -- to the
 * nominal surface (material added there), then on to the hit's own radius (barrel) / z (disk) -- and a 2-D update on the
 * plane tangent to the hit radius; the state then sits on the hit's surface. */
int kfo_fit(int n_layers, const double* layers, double bz, int hit_mode, int64_t n, int64_t ld, const double* par,
            const double* cov, const int8_t* q, const double* hx, const double* hy, const double* hz,
            const int64_t* seg_off, const int32_t* hit_idx, const int32_t* trk_event, double* par_out,
            double* cov_out, double* chi2_out, int32_t* nhits_out, uint32_t* status_out) {
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t t = 0; t < n; ++t) {
        double p[6], C[36], pp[6], Cp[36], pu[6], Cu[36];
        for (int i = 0; i < 6; ++i) p[i] = par[i * ld + t];
        for (int i = 0; i < 36; ++i) C[i] = cov[i * ld + t];
        double chi2 = 0.0;
        int nh = 0;
        uint32_t st = 0;
        int ev = trk_event ? trk_event[t] : 0;
        for (int l = 0; l < n_layers; ++l) {
            int64_t idx = hit_idx ? hit_idx[(int64_t)l * ld + t] : t;
            if (idx < -1) continue;
            int f = predict(layers, l, bz, p, C, q[t], pp, Cp);
            if (f) { st |= (uint32_t)f; break; }
            if (idx == -1) { /* hole: the predicted state (incl. Q) becomes the state */
                memcpy(p, pp, sizeof p);
                memcpy(C, Cp, sizeof C);
                continue;
            }
            int64_t h = seg_off[(int64_t)ev * n_layers + l] + idx;
            double m[3] = {hx[h], hy[h], hz[h]}, c2;
            if (hit_mode == 0) f = kfo_update(pp, Cp, m, LSRPHI(layers, l), LSZ(layers, l), LSR(layers, l), pu, Cu, &c2);
            else {
                double p2[6], C2[36];
                const int kind = LKIND(layers, l);
                f = to_hit_surface(kind, bz, q[t], pp, Cp, m, p2, C2);
                if (!f) f = kfo_update_2d(p2, C2, m, kind, LSRPHI(layers, l), kind == 0 ? LSZ(layers, l) : LSR(layers, l), pu, Cu, &c2);
            }
            if (f) { st |= (uint32_t)f; break; }
            memcpy(p, pu, sizeof p);
            memcpy(C, Cu, sizeof C);
            chi2 += c2;
            nh += 1;
        }
        p[4] = wrap_phi(p[4]);
        for (int i = 0; i < 6; ++i) par_out[i * ld + t] = p[i];
        for (int i = 0; i < 36; ++i) cov_out[i * ld + t] = C[i];
        chi2_out[t] = chi2;
        nhits_out[t] = nh;
        status_out[t] = st;
    }
    return 0;
}

/* =====================================================================================================
 * Hit binning, window lookup, combinatorial building (sec. 2, L54 sec. 3.1, L82-88 sec. 4.3).
 * The X-series is specified in IEEE fp32 so that CPU and GPU agree bit for bit: every
 * float expression below is a single rounded operation (this file is compiled with -ffp-contract=off).
 * ===================================================================================================== */

/* X1 table: T[k] = fl32(tan(2 pi k / N)), k = 0 .. N/8, T[N/8] := 1 */
void kfo_tan_table(int n_phi, float* tab) {
    int m = n_phi / 8;
    for (int k = 0; k < m; ++k) tab[k] = (float)tan(2.0 * KFO_PI * (double)k / (double)n_phi);
    tab[m] = 1.0f;
}

/* X1: azimuthal bin of (x, y) from exact fp32 comparisons, no atan2 */
int kfo_phi_bin(float x, float y, int n_phi, const float* tab) {
    float ax = fabsf(x), ay = fabsf(y);
    int swap = ay > ax;
    float lo = swap ? ax : ay, hi = swap ? ay : ax;
    float t = (hi > 0.0f) ? lo / hi : 0.0f;
    int m = n_phi / 8;
    int j = 0; /* largest k <= m-1 with tab[k] <= t; tab[0] = 0 <= t */
    for (int k = 1; k < m; ++k)
        if (tab[k] <= t) j = k;
    int a = swap ? n_phi / 4 - 1 - j : j;
    if (x >= 0.0f) return (y >= 0.0f) ? a : n_phi - 1 - a;
    return (y >= 0.0f) ? n_phi / 2 - 1 - a : n_phi / 2 + a;
}

/* X2: z bin */
int kfo_z_bin(float z, float zmax, int n_z) {
    float inv_dz = (float)n_z / (2.0f * zmax);
    float f = floorf((z + zmax) * inv_dz);
    int iz = (f >= (float)n_z) ? n_z - 1 : (f < 0.0f ? 0 : (int)f);
    return iz;
}

/* X2 for any layer [R22]: row of coordinate v in [lo, hi) cut into n rows.  A barrel layer bins z in [-zmax, zmax) (then this
 * is kfo_z_bin bit for bit: z - (-zmax) = z + zmax and zmax - (-zmax) = 2 zmax are the same fp32 operations); a disk bins
 * the radius of the hit, rho = fl32(sqrt(fl32(fl32(x x) + fl32(y y)))), in [rmin, rmax). */
int kfo_row_bin(float v, float lo, float hi, int n) {
    float inv = (float)n / (hi - lo);
    float f = floorf((v - lo) * inv);
    return (f >= (float)n) ? n - 1 : (f < 0.0f ? 0 : (int)f);
}
float kfo_hit_rho(float x, float y) {
    float xx = x * x, yy = y * y;
    return sqrtf(xx + yy);
}
static void row_range(const double* layers, int l, float* lo, float* hi) {
    if (LKIND(layers, l) == 0) { *lo = -(float)LZMAX(layers, l); *hi = (float)LZMAX(layers, l); }
    else { *lo = (float)LRMIN(layers, l); *hi = (float)LZMAX(layers, l); }
}

/* B0: sorted order = ascending (global bin, original index).  seg_off [n_events*L + 1]; outputs sx, sy, sz,
 * perm [n_hits] (sorted position -> original index within the segment), bin_off [n_events*L*n_z*n_phi + 1]. */
int kfo_bin_hits(int n_layers, const double* layers, int n_events, const int64_t* seg_off, const float* hx,
                 const float* hy, const float* hz, int n_phi, int n_z, float* sx, float* sy, float* sz, int32_t* perm,
                 int32_t* bin_off) {
    float* tab = (float*)malloc((size_t)(n_phi / 8 + 1) * sizeof(float));
    kfo_tan_table(n_phi, tab);
    int64_t nseg = (int64_t)n_events * n_layers;
    int64_t bins_per_seg = (int64_t)n_phi * n_z;
    int64_t n_hits = seg_off[nseg];
    bin_off[0] = 0;
    int32_t* key = (int32_t*)malloc((size_t)(n_hits > 0 ? n_hits : 1) * sizeof(int32_t));
    for (int64_t sg = 0; sg < nseg; ++sg) {
        int l = (int)(sg % n_layers);
        float lo, hi;
        row_range(layers, l, &lo, &hi);
        const int disk = LKIND(layers, l) != 0;
        int32_t* cnt = (int32_t*)calloc((size_t)bins_per_seg + 1, sizeof(int32_t));
        for (int64_t h = seg_off[sg]; h < seg_off[sg + 1]; ++h) {
            int b = kfo_row_bin(disk ? kfo_hit_rho(hx[h], hy[h]) : hz[h], lo, hi, n_z) * n_phi + kfo_phi_bin(hx[h], hy[h], n_phi, tab);
            key[h] = b;
            cnt[b + 1] += 1;
        }
        for (int64_t b = 0; b < bins_per_seg; ++b) cnt[b + 1] += cnt[b];
        for (int64_t b = 0; b < bins_per_seg; ++b) bin_off[sg * bins_per_seg + b + 1] = (int32_t)(seg_off[sg] + cnt[b + 1]);
        for (int64_t h = seg_off[sg]; h < seg_off[sg + 1]; ++h) { /* stable: ascending original index within a bin */
            int64_t pos = seg_off[sg] + cnt[key[h]]++;
            sx[pos] = hx[h]; sy[pos] = hy[h]; sz[pos] = hz[h];
            perm[pos] = (int32_t)(h - seg_off[sg]);
        }
        free(cnt);
    }
    free(key);
    free(tab);
    return 0;
}

/* X3: window (phi_c +- dphi, c +- d) -> first phi bin, number of phi bins (wrapping), rows [iz_lo, iz_hi] of the row
 * coordinate (z on a barrel layer, radius on a disk [R22]) binned in [lo, hi) */
void kfo_window_bins_row(float phi_c, float dphi, float z_c, float dz, float lo, float hi, int n_phi, int n_z, int* first, int* n_b,
                         int* iz_lo, int* iz_hi) {
    float inv_dphi = (float)((double)n_phi / (2.0 * KFO_PI));
    if (!(dphi * inv_dphi < (float)n_phi)) { /* half width of a full turn or more: every bin, starting at bin 0 [X3] */
        *first = 0;
        *n_b = n_phi;
    } else {
        float f_lo = (phi_c - dphi) * inv_dphi, f_hi = (phi_c + dphi) * inv_dphi;
        int b_lo = (int)floorf(f_lo), b_hi = (int)floorf(f_hi);
        int nb = b_hi - b_lo + 1;
        if (nb > n_phi) nb = n_phi;
        if (nb < 0) nb = 0;
        *n_b = nb;
        *first = ((b_lo % n_phi) + n_phi) % n_phi;
    }
    *iz_lo = kfo_row_bin(z_c - dz, lo, hi, n_z);
    *iz_hi = kfo_row_bin(z_c + dz, lo, hi, n_z);
}
void kfo_window_bins(float phi_c, float dphi, float z_c, float dz, float zmax, int n_phi, int n_z, int* first, int* n_b,
                     int* iz_lo, int* iz_hi) {
    kfo_window_bins_row(phi_c, dphi, z_c, dz, -zmax, zmax, n_phi, n_z, first, n_b, iz_lo, iz_hi);
}

/* kf_window_lookup_ref: bin-granular hit list of each query (rows ascending, bins ascending with wrap, hits in
 * sorted order).  count[i] = full length; sorted_idx[i*cap + j] for j < min(count, cap). */
int kfo_window_lookup(int n_layers, const double* layers, int n_phi, int n_z, const int32_t* bin_off, int64_t n_query,
                      const int32_t* event, const int32_t* layer, const float* phi_c, const float* dphi,
                      const float* z_c, const float* dz, int cap, int32_t* count, int32_t* sorted_idx) {
    for (int64_t i = 0; i < n_query; ++i) {
        int first, nb, z0, z1;
        float lo, hi;
        row_range(layers, layer[i], &lo, &hi);
        kfo_window_bins_row(phi_c[i], dphi[i], z_c[i], dz[i], lo, hi, n_phi, n_z, &first, &nb, &z0, &z1);
        int64_t seg = (int64_t)event[i] * n_layers + layer[i];
        int32_t c = 0;
        for (int iz = z0; iz <= z1; ++iz)
            for (int k = 0; k < nb; ++k) {
                int64_t b = (seg * n_z + iz) * n_phi + (first + k) % n_phi;
                for (int32_t h = bin_off[b]; h < bin_off[b + 1]; ++h) {
                    if (c < cap) sorted_idx[i * cap + c] = h;
                    ++c;
                }
            }
        count[i] = c;
    }
    return 0;
}

/* ---- combinatorial building (R10, R11) ---- */
typedef struct {
    double p[6], C[36], chi2;
    int nhits, finished;
    uint32_t status;
    int32_t hits[32];
} kfo_cand;

typedef struct {
    int parent, kind; /* kind 0 = hit child, 1 = no compatible hit (-1), 2 = finished (-2), 3 = layer skipped (-2, alive) [R22] */
    int64_t hitpos;   /* global sorted position; INT64_MAX for kinds 1, 2 */
    double chi2;
    int nhits;
} kfo_child;

/* chi2 of hit m against the predicted state (pp, Cp) on the layer's nominal surface: hit_mode 0 the 3-D one [R5];
 * hit_mode 1 second step to the hit's own surface, then the 2-D one on its tangent plane [R20, R21, R23].
 * 0 = ok, -1 = S not positive definite, 1 = the second step does not reach the hit. */
static int build_hit_chi2(int hit_mode, int disk, double bz, int q, const double pp[6], const double Cp[36], const double m[3],
                          double srphi, double szz, double sr, double* c2) {
    if (hit_mode == 0) return kfo_chi2(pp, Cp, m, srphi, szz, sr, c2) ? -1 : 0;
    double p2[6], C2[36];
    if (to_hit_surface(disk, bz, q, pp, Cp, m, p2, C2)) return 1;
    return kfo_chi2_2d(p2, C2, m, disk, srphi, disk ? sr : szz, c2) ? -1 : 0;
}

static int child_cmp(const void* a_, const void* b_) {
    const kfo_child *a = (const kfo_child*)a_, *b = (const kfo_child*)b_;
    if (a->nhits != b->nhits) return a->nhits > b->nhits ? -1 : 1;
    if (a->chi2 != b->chi2) return a->chi2 < b->chi2 ? -1 : 1;
    if (a->parent != b->parent) return a->parent < b->parent ? -1 : 1;
    if (a->hitpos != b->hitpos) return a->hitpos < b->hitpos ? -1 : 1;
    return 0;
}

/* kf_build_ref.  Hits are the SORTED arrays of kfo_bin_hits (float), perm / bin_off alike.  Seeds: par [6][ld_seed],
 * cov dense [36][ld_seed], chi2_in (NULL = 0), seed_hit_idx [first_layer][ld_seed].  use_bins = 0 scans every hit of
 * the layer's segment (brute force without the spatial index, pin P12).
 * Outputs, slot = s*K + k: par_o [6][ld_out], cov_o [36][ld_out], chi2_o, nhits_o, status_o [n_seeds*K],
 * hit_idx_o [n_layers][ld_out], n_cand [n_seeds]; unused slots: nhits 0, chi2 0, status 0, hit_idx -2, par/cov 0.
 * Geometry with disks ("cylinder with lids") [R22]: the layers are alternatives, not a sequence every track
 * goes through -- a candidate that cannot be propagated to a layer (not reached, grazing) or whose window lies off the
 * layer SKIPS it: one child with the unchanged state, hit = -2, alive, no status bit; only a numeric failure finishes a
 * candidate.  On a disk the window is in (phi, radius): rho_c = |(x', y')|, d_rho = n_sigma sqrt(var_rho + sig_r^2) with
 * var_rho = (x'^2 Cxx + 2 x'y' Cxy + y'^2 Cyy)/rho_c^2, dphi = n_sigma sqrt(var_phi + (sig_rphi/rho_c)^2); off the layer when
 * rho_c > rmax + d_rho or rho_c < rmin - d_rho; strict test |x'm_y - y'm_x| <= dphi rho_c rho_m, x'm_x + y'm_y > 0,
 * |rho_m - rho_c| <= d_rho; rows of the bins by radius.  chi2 and update: the 3-D ones [R5] (sig_z regularises along the
 * disk normal).  Barrel-only geometries keep the behaviour of R10 exactly.
 * hit_mode 1 ("followed by further propagation steps to the position of each candidate hit.  KF updates are
 * performed on the plane tangent to the hit radius") [R23]: the window is opened on the layer's nominal surface as above,
 * widened by the displacement of the sensors about it (r.m.s. sig_r along the normal of a cylinder, sig_z along that of a disk);
 * every hit inside it is reached by the second propagation step [R20] from the predicted state and judged by the chi2 of
 * the 2-D residual on its tangent plane [R21]; a hit the second step cannot reach is not compatible; the kept hit
 * children are updated there (2-D update; the state then sits on the hit's own surface).  hit_mode 0: 3-D chi2 and
 * update on the nominal surface [R5].
 * counters[8]: 0 propagations, 1 hits scanned, 2 pass strict window, 3 pass chi2 cut (hit children), 4 updates,
 *              5 bin rows touched, 6 seed-layers, 7 children ranked.
 * margins (NULL or [n_seeds][n_layers][5], test diagnostics for DESIGN.md R16): the smallest RELATIVE distance of any
 * decision taken for that seed on that layer to its threshold (1e300 = no such decision):
 *   [0] strict window: | |x'm_y - y'm_x| / (dphi r' r_m) - 1 | and | |m_z - z_c| / dz - 1 | of a hit that passes the other
 *       window tests and would pass (or passes) the chi2 cut;
 *   [1] chi2 cut: |chi2_h / chi2_cut - 1| of a hit inside the window;
 *   [2] rank: |chi2_a - chi2_b| / max(chi2_a, chi2_b) of children adjacent in the ranking with equal nhits, at least
 *       one of them kept;
 *   [3] propagation: |cos_inc / c_min - 1| (grazing guard) and | |z'| / (zmax + dz) - 1 | (acceptance);
 *   [4] tangency (a crossing that only just exists / only just does not, i.e. the choice between the "grazing" and the
 *       "unreachable" bit): cos^2(incidence), resp. max(R^2 - r^2)/R^2 along the half turn. */
int kfo_build(int n_layers, const double* layers, double bz, int n_phi, int n_z, const float* sx, const float* sy,
              const float* sz, const int32_t* perm, const int32_t* bin_off, const int64_t* seg_off, int64_t n_seeds,
              int64_t ld_seed, const double* par, const double* cov, const int8_t* q, const double* chi2_in,
              const int32_t* seed_event, const int32_t* seed_hit_idx, int first_layer, int K, double chi2_cut,
              double n_sigma, int use_bins, int hit_mode, int64_t ld_out, double* par_o, double* cov_o, double* chi2_o,
              int32_t* nhits_o, uint32_t* status_o, int32_t* hit_idx_o, int32_t* n_cand, int64_t* counters,
              double* margins) {
    if (K < 1 || K > 32 || n_layers > 32 || first_layer < 0 || first_layer > n_layers) return -1;
    int64_t cnt[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    int lids = 0;
    for (int l = 0; l < n_layers; ++l) lids = lids || LKIND(layers, l) != 0;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : cnt[:8])
    for (int64_t sd = 0; sd < n_seeds; ++sd) {
        kfo_cand* cur = (kfo_cand*)calloc((size_t)K, sizeof(kfo_cand));
        kfo_cand* nxt = (kfo_cand*)calloc((size_t)K, sizeof(kfo_cand));
        double(*pp)[6] = malloc((size_t)K * sizeof *pp);
        double(*Cp)[36] = malloc((size_t)K * sizeof *Cp);
        uint32_t* pflag = (uint32_t*)malloc((size_t)K * sizeof(uint32_t));
        size_t cap_ch = 256, n_ch = 0;
        kfo_child* ch = (kfo_child*)malloc(cap_ch * sizeof(kfo_child));
        int ev = seed_event ? seed_event[sd] : 0;
        int nc = 1;
        for (int i = 0; i < 6; ++i) cur[0].p[i] = par[i * ld_seed + sd];
        for (int i = 0; i < 36; ++i) cur[0].C[i] = cov[i * ld_seed + sd];
        cur[0].chi2 = chi2_in ? chi2_in[sd] : 0.0;
        cur[0].nhits = first_layer;
        for (int l = 0; l < 32; ++l) cur[0].hits[l] = -2;
        for (int l = 0; l < first_layer; ++l) cur[0].hits[l] = seed_hit_idx ? seed_hit_idx[(int64_t)l * ld_seed + sd] : -1;

        for (int l = first_layer; l < n_layers; ++l) {
            const double R = LR(layers, l), zmax = LZMAX(layers, l), rmin = LRMIN(layers, l);
            const int disk = LKIND(layers, l) != 0;
            const double srphi = LSRPHI(layers, l), szz = LSZ(layers, l), sr = LSR(layers, l);
            const int64_t seg = (int64_t)ev * n_layers + l;
            n_ch = 0;
            cnt[6] += 1;
            double mg[5] = {1e300, 1e300, 1e300, 1e300, 1e300};
#define KFO_MARGIN(k, v) do { double v_ = (v); if (v_ < mg[k]) mg[k] = v_; } while (0)
            for (int c = 0; c < nc; ++c) {
                kfo_child pass = {c, 2, INT64_MAX, cur[c].chi2, cur[c].nhits};
                pflag[c] = 0;
                double ci = 0.0, tang = 1e300;
                int f = cur[c].finished ? -1 : predict_ci(layers, l, bz, cur[c].p, cur[c].C, q[sd], pp[c], Cp[c], &ci, &tang);
                if (!cur[c].finished) cnt[0] += 1;
                if (!cur[c].finished && (f == 0 || f == KFO_GRAZING)) KFO_MARGIN(3, fabs(ci / KFO_CMIN - 1.0));
                if (!cur[c].finished) KFO_MARGIN(4, tang);
                double dphi = 0, dzw = 0;
                if (f == 0) { /* window (R11; on a disk R22) */
                    const double x = pp[c][0], y = pp[c][1], r2 = x * x + y * y;
                    double varphi = (x * x * Cp[c][1 * 6 + 1] - 2.0 * x * y * Cp[c][0 * 6 + 1] + y * y * Cp[c][0]) / (r2 * r2);
                    if (varphi < 0.0) varphi = 0.0;
                    /* hit_mode 1 [R23]: the sensors sit off the nominal surface by an r.m.s. sig_n along its normal (sig_r on a
                       cylinder, sig_z on a disk: the resolutions the 2-D update does not use); a sensor displaced by d along
                       the normal is crossed d cot(theta)/cos(inc) further in z and d tan(inc)/r further in azimuth (cylinder),
                       at most d tan(theta) further in radius and d tan(theta)/rho in azimuth (disk) */
                    double wphi2 = 0.0, wrow2 = 0.0;
                    if (hit_mode && !disk) {
                        const double cinc = (x * cos(pp[c][4]) + y * sin(pp[c][4])) / sqrt(r2);
                        const double cot = cos(pp[c][5]) / sin(pp[c][5]);
                        wrow2 = (sr * cot / cinc) * (sr * cot / cinc);
                        wphi2 = sr * sr * (1.0 - cinc * cinc) / (cinc * cinc) / r2;
                    } else if (hit_mode) {
                        const double tth = sin(pp[c][5]) / cos(pp[c][5]);
                        wrow2 = szz * tth * szz * tth;
                        wphi2 = wrow2 / r2;
                    }
                    if (!disk) {
                        dphi = n_sigma * sqrt(varphi + (srphi / R) * (srphi / R) + wphi2);
                        dzw = n_sigma * sqrt(Cp[c][2 * 6 + 2] + szz * szz + wrow2);
                    } else {
                        double varrho = (x * x * Cp[c][0] + 2.0 * x * y * Cp[c][0 * 6 + 1] + y * y * Cp[c][1 * 6 + 1]) / r2;
                        if (varrho < 0.0) varrho = 0.0;
                        dphi = n_sigma * sqrt(varphi + srphi * srphi / r2 + wphi2);
                        dzw = n_sigma * sqrt(varrho + sr * sr + wrow2);
                    }
                    if (!isfinite(dphi) || !isfinite(dzw)) f = KFO_NUMERIC;
                    else if (!disk) {
                        KFO_MARGIN(3, fabs(fabs(pp[c][2]) / (zmax + dzw) - 1.0));
                        if (fabs(pp[c][2]) > zmax + dzw) f = KFO_LEFT_Z;
                    } else {
                        const double rho = sqrt(r2);
                        KFO_MARGIN(3, fabs(rho / (zmax + dzw) - 1.0));
                        if (rmin - dzw > 0.0) KFO_MARGIN(3, fabs(rho / (rmin - dzw) - 1.0));
                        if (rho > zmax + dzw || rho < rmin - dzw) f = KFO_LEFT_Z;
                    }
                }
                if (f != 0) {
                    if (lids && !cur[c].finished && f != KFO_NUMERIC) { /* layer not crossed: skipped, the candidate lives on [R22] */
                        kfo_child skip = {c, 3, INT64_MAX, cur[c].chi2, cur[c].nhits};
                        if (n_ch == cap_ch) ch = (kfo_child*)realloc(ch, (cap_ch *= 2) * sizeof(kfo_child));
                        ch[n_ch++] = skip;
                        continue;
                    }
                    /* finished (or just found unpropagatable): state unchanged */
                    if (f > 0) pflag[c] = (uint32_t)f;
                    if (n_ch == cap_ch) ch = (kfo_child*)realloc(ch, (cap_ch *= 2) * sizeof(kfo_child));
                    ch[n_ch++] = pass;
                    continue;
                }
                const double x = pp[c][0], y = pp[c][1], rp = sqrt(x * x + y * y);
                const double zc = disk ? rp : pp[c][2];            /* centre of the window along the row coordinate */
                int first = 0, nb = 1, z0 = 0, z1 = 0;
                if (use_bins) {
                    float lo_, hi_;
                    row_range(layers, l, &lo_, &hi_);
                    kfo_window_bins_row((float)atan2(y, x), (float)dphi, (float)zc, (float)dzw, lo_, hi_, n_phi, n_z, &first, &nb, &z0, &z1);
                }
                int n_hit_children = 0, s_bad = 0;
                for (int iz = z0; iz <= z1 && !s_bad; ++iz) {
                    cnt[5] += use_bins ? 1 : 0;
                    for (int kb = 0; kb < nb && !s_bad; ++kb) {
                        int64_t h0, h1;
                        if (use_bins) {
                            int64_t b = (seg * n_z + iz) * n_phi + (first + kb) % n_phi;
                            h0 = bin_off[b]; h1 = bin_off[b + 1];
                        } else { h0 = seg_off[seg]; h1 = seg_off[seg + 1]; }
                        for (int64_t h = h0; h < h1; ++h) {
                            cnt[1] += 1;
                            const double m[3] = {sx[h], sy[h], sz[h]};
                            const double rm = sqrt(m[0] * m[0] + m[1] * m[1]);
                            const int in_phi = fabs(x * m[1] - y * m[0]) <= dphi * rp * rm;
                            const int in_dot = x * m[0] + y * m[1] > 0.0;
                            const double mrow = disk ? rm : m[2];
                            const int in_z = fabs(mrow - zc) <= dzw;
                            if (margins && in_dot && (in_phi || in_z)) { /* distance to the window edges (diagnostics only) */
                                const double mphi = fabs(fabs(x * m[1] - y * m[0]) / (dphi * rp * rm) - 1.0);
                                const double mz = fabs(fabs(mrow - zc) / dzw - 1.0);
                                const double near = fmin(in_z ? mphi : 1e300, in_phi ? mz : 1e300);
                                if (near < mg[0]) {
                                    double c2m;
                                    int fm = build_hit_chi2(hit_mode, disk, bz, q[sd], pp[c], Cp[c], m, srphi, szz, sr, &c2m);
                                    if (fm < 0 || (fm == 0 && c2m < chi2_cut)) mg[0] = near;
                                }
                            }
                            if (!in_phi) continue;
                            if (!in_dot) continue;
                            if (!in_z) continue;
                            cnt[2] += 1;
                            double c2;
                            const int fh = build_hit_chi2(hit_mode, disk, bz, q[sd], pp[c], Cp[c], m, srphi, szz, sr, &c2);
                            if (fh < 0) { s_bad = 1; break; }
                            if (fh > 0) continue;          /* hit_mode 1: the second step does not reach the hit's surface */
                            KFO_MARGIN(1, fabs(c2 / chi2_cut - 1.0));
                            if (!(c2 < chi2_cut)) continue;
                            cnt[3] += 1;
                            kfo_child k = {c, 0, h, cur[c].chi2 + c2, cur[c].nhits + 1};
                            if (n_ch == cap_ch) ch = (kfo_child*)realloc(ch, (cap_ch *= 2) * sizeof(kfo_child));
                            ch[n_ch++] = k;
                            ++n_hit_children;
                        }
                    }
                }
                if (s_bad) { /* S not positive definite: drop this parent's hit children, finish it */
                    n_ch -= (size_t)n_hit_children;
                    pflag[c] = KFO_NUMERIC;
                    if (n_ch == cap_ch) ch = (kfo_child*)realloc(ch, (cap_ch *= 2) * sizeof(kfo_child));
                    ch[n_ch++] = pass;
                } else if (n_hit_children == 0) {
                    kfo_child miss = {c, 1, INT64_MAX, cur[c].chi2, cur[c].nhits};
                    if (n_ch == cap_ch) ch = (kfo_child*)realloc(ch, (cap_ch *= 2) * sizeof(kfo_child));
                    ch[n_ch++] = miss;
                }
            }
            cnt[7] += (int64_t)n_ch;
            qsort(ch, n_ch, sizeof(kfo_child), child_cmp);
            int nn = n_ch < (size_t)K ? (int)n_ch : K;
            for (int j = 0; j + 1 < (int)n_ch && j < nn; ++j)
                if (ch[j].nhits == ch[j + 1].nhits) {
                    const double big = fmax(fabs(ch[j].chi2), fabs(ch[j + 1].chi2));
                    KFO_MARGIN(2, big > 0.0 ? fabs(ch[j].chi2 - ch[j + 1].chi2) / big : 0.0);
                }
            if (margins)
                for (int k = 0; k < 5; ++k) margins[((int64_t)sd * n_layers + l) * 5 + k] = mg[k];
#undef KFO_MARGIN
            for (int j = 0; j < nn; ++j) {
                const kfo_child* k = &ch[j];
                const kfo_cand* pa = &cur[k->parent];
                kfo_cand* o = &nxt[j];
                *o = *pa;
                if (k->kind == 2) {
                    o->finished = 1;
                    o->status |= pflag[k->parent];
                    o->hits[l] = -2;
                } else if (k->kind == 3) {
                    o->hits[l] = -2;
                } else if (k->kind == 1) {
                    memcpy(o->p, pp[k->parent], sizeof o->p);
                    memcpy(o->C, Cp[k->parent], sizeof o->C);
                    o->hits[l] = -1;
                } else {
                    const double m[3] = {sx[k->hitpos], sy[k->hitpos], sz[k->hitpos]};
                    double c2;
                    cnt[4] += 1;
                    int f;
                    if (hit_mode == 0) f = kfo_update(pp[k->parent], Cp[k->parent], m, srphi, szz, sr, o->p, o->C, &c2);
                    else {
                        double p2[6], C2[36];
                        f = to_hit_surface(disk, bz, q[sd], pp[k->parent], Cp[k->parent], m, p2, C2);
                        if (f == 0) f = kfo_update_2d(p2, C2, m, disk, srphi, disk ? sr : szz, o->p, o->C, &c2);
                    }
                    o->chi2 = k->chi2;
                    o->nhits = k->nhits;
                    o->hits[l] = perm[k->hitpos];
                    if (f) { /* numerically failed update: keep the predicted state, finish the candidate */
                        memcpy(o->p, pp[k->parent], sizeof o->p);
                        memcpy(o->C, Cp[k->parent], sizeof o->C);
                        o->status |= KFO_NUMERIC;
                        o->finished = 1;
                    }
                }
            }
            kfo_cand* t = cur; cur = nxt; nxt = t;
            nc = nn;
        }
        n_cand[sd] = nc;
        for (int k = 0; k < K; ++k) {
            int64_t slot = sd * K + k;
            if (k < nc) {
                const kfo_cand* c = &cur[k];
                for (int i = 0; i < 6; ++i) par_o[i * ld_out + slot] = (i == 4) ? wrap_phi(c->p[i]) : c->p[i];
                for (int i = 0; i < 36; ++i) cov_o[i * ld_out + slot] = c->C[i];
                chi2_o[slot] = c->chi2; nhits_o[slot] = c->nhits; status_o[slot] = c->status;
                for (int l = 0; l < n_layers; ++l) hit_idx_o[(int64_t)l * ld_out + slot] = c->hits[l];
            } else {
                for (int i = 0; i < 6; ++i) par_o[i * ld_out + slot] = 0.0;
                for (int i = 0; i < 36; ++i) cov_o[i * ld_out + slot] = 0.0;
                chi2_o[slot] = 0.0; nhits_o[slot] = 0; status_o[slot] = 0;
                for (int l = 0; l < n_layers; ++l) hit_idx_o[(int64_t)l * ld_out + slot] = -2;
            }
        }
        free(cur); free(nxt); free(pp); free(Cp); free(pflag); free(ch);
    }
    if (counters) for (int i = 0; i < 8; ++i) counters[i] = cnt[i];
    return 0;
}

// kf_pair.cuh -- the per-layer Kalman-filter step for TWO tracks per thread: every quantity is a pair (track a, track b)
// and every fp32 operation one packed instruction (FFMA2 / FMUL2 / FADD2, sm_100a), so the whole step -- not only its
// regular 6x6 chains -- runs two FMA lanes per issue slot, and the address arithmetic, constants and loop control are
// shared by the two tracks.  Fast path only: anything unusual in either track (unreachable / grazing crossing, turning
// angle beyond the series, large angle correction, non-positive pivot, non-finite result) makes the function return
// false and the caller redoes both tracks with the one-track code of kf_state.cuh.  Isotropic hit covariance only.
// Same formulas and operation order as kf_state.cuh (R2-R5); shares nothing with oracle/.
#pragma once
#include "kf_math.cuh"
#include "kf_state.cuh"

namespace kf {
namespace pair {

struct V { float2 v; };
__device__ __forceinline__ V mk(float a, float b) { V r; r.v = make_float2(a, b); return r; }
__device__ __forceinline__ V sp(float a) { return mk(a, a); }                                   // splat
__device__ __forceinline__ V operator+(V a, V b) { V r; r.v = __fadd2_rn(a.v, b.v); return r; }
__device__ __forceinline__ V operator-(V a) { return mk(-a.v.x, -a.v.y); }
__device__ __forceinline__ V operator-(V a, V b) { return a + (-b); }
__device__ __forceinline__ V operator*(V a, V b) { V r; r.v = __fmul2_rn(a.v, b.v); return r; }
__device__ __forceinline__ V operator*(float a, V b) { return sp(a) * b; }
__device__ __forceinline__ V operator*(V a, float b) { return a * sp(b); }
__device__ __forceinline__ V operator+(V a, float b) { return a + sp(b); }
__device__ __forceinline__ V fma(V a, V b, V c) { V r; r.v = __ffma2_rn(a.v, b.v, c.v); return r; }
__device__ __forceinline__ V fma(V a, V b, float c) { return fma(a, b, sp(c)); }
__device__ __forceinline__ V fma(float a, V b, V c) { return fma(sp(a), b, c); }
__device__ __forceinline__ V fma(V a, float b, V c) { return fma(a, sp(b), c); }
__device__ __forceinline__ V fma(V a, float b, float c) { return fma(a, sp(b), sp(c)); }
__device__ __forceinline__ V rcp(V a) { return mk(frcp(a.v.x), frcp(a.v.y)); }
__device__ __forceinline__ V sqrt_(V a) { return mk(fsqrt(a.v.x), fsqrt(a.v.y)); }
__device__ __forceinline__ V log_(V a) { return mk(flog(a.v.x), flog(a.v.y)); }
__device__ __forceinline__ bool both_gt(V a, float b) { return a.v.x > b && a.v.y > b; }
__device__ __forceinline__ bool both_ge(V a, float b) { return a.v.x >= b && a.v.y >= b; }
__device__ __forceinline__ bool both_lt(V a, float b) { return a.v.x < b && a.v.y < b; }
__device__ __forceinline__ V abs_(V a) { return mk(fabsf(a.v.x), fabsf(a.v.y)); }

struct Trig2 { V cp, sp, st, ct; };
struct State2 { V p[6]; V C[21]; Trig2 g; int pha, phb; };   // p[4] is unused: phi is the fixed-point pair (pha, phb), see kf_state.cuh

// rotate (c, s) by d, |d| < 0.06 (polynomial, then one Newton step back to unit norm)
__device__ __forceinline__ void rotate_poly(V& c, V& s, V d) {
    const V d2 = d * d;
    const V sd = d * fma(d2, fma(d2, 1.0f / 120.0f, -1.0f / 6.0f), 1.0f);
    const V cd = fma(d2, fma(d2, 1.0f / 24.0f, -0.5f), 1.0f);
    const V cn = fma(c, cd, -(s * sd)), sn = fma(s, cd, c * sd);
    const V k = fma(fma(cn, cn, sn * sn), -0.5f, 1.5f);
    c = cn * k; s = sn * k;
}

// Predict (F2-F5) for both tracks; false = not the fast path (state untouched).  cw = -q k Bz per track.
__device__ __forceinline__ bool predict(State2& S, V cw, const LayerC& ly) {
    V (&p)[6] = S.p; V (&C)[21] = S.C;
    const V spn_ = S.g.sp, cp = S.g.cp, st = S.g.st, ct = S.g.ct;
    const V ist = rcp(st);
    const V cot = ct * ist;
    // ---- closed-form first crossing of the cylinder (R2) ----
    const V x = p[0], y = p[1];
    const V w = cw * p[3];
    const V u = fma(x, cp, y * spn_);
    const V v = fma(y, cp, -(x * spn_));
    const V E = 0.5f * (sp(ly.r2) - fma(x, x, y * y));
    const V A = fma(-(w * w), E, 2.0f * fma(v, w, 1.0f));
    const V D = fma(E, A, u * u);
    const bool fa = u.v.x >= 0.0f, fb = u.v.y >= 0.0f;
    if (!both_gt(E, 0.0f) || !both_ge(D, 0.0f) || !(fa || A.v.x > 0.0f) || !(fb || A.v.y > 0.0f)) return false;
    const V sq = sqrt_(D);
    const V num = mk(fa ? E.v.x : sq.v.x - u.v.x, fb ? E.v.y : sq.v.y - u.v.y);
    const V den = mk(fa ? u.v.x + sq.v.x : A.v.x, fb ? u.v.y + sq.v.y : A.v.y);
    const V tau = num * rcp(den);
    const V th = w * tau;                         // tan(alpha/2)
    const V th2 = th * th;
    if (!both_lt(th2, 0.06f)) return false;       // series for atan(t)/t and the curvature partials only
    const V inv = rcp(th2 + 1.0f);
    const V X = 2.0f * tau * inv;                 // sin(alpha)/w
    const V Y = X * th;                           // (1 - cos(alpha))/w
    const V sa = w * X;
    const V ca = (sp(1.0f) - th2) * inv;
    const V dx = fma(cp, X, -(spn_ * Y));
    const V dy = fma(spn_, X, cp * Y);
    const V xn = x + dx, yn = y + dy;
    const V f = fma(th2, fma(th2, fma(th2, fma(th2, fma(th2, -1.0f / 11.0f, 1.0f / 9.0f), -1.0f / 7.0f), 0.2f), -1.0f / 3.0f), 1.0f);
    const V alpha = 2.0f * th * f;
    const V a2 = alpha * alpha;
    const V f1 = alpha * fma(a2, fma(a2, fma(a2, 1.0f / 45360.0f, -1.0f / 840.0f), 1.0f / 30.0f), -1.0f / 3.0f);
    const V f2 = fma(a2, fma(a2, fma(a2, fma(a2, 1.0f / 403200.0f, -1.0f / 5760.0f), 1.0f / 144.0f), -0.125f), 0.5f);
    const V s = 2.0f * tau * f;
    const V zn = fma(s, cot, p[2]);
    const V cpn = fma(cp, ca, -(spn_ * sa));
    const V spn = fma(spn_, ca, cp * sa);
    const V up = fma(xn, cpn, yn * spn);
    if (!both_ge(up, ly.rcmin)) return false;
    // ---- Jacobian entries (R3) ----
    const V cs2 = cw * s * s;
    const V dXdi = cs2 * f1, dYdi = cs2 * f2;
    const V Fxi = fma(cp, dXdi, -(spn_ * dYdi)), Fyi = fma(spn_, dXdi, cp * dYdi);
    const V Fxp = -dy, Fyp = dx;
    const V iup = rcp(up);
    const V sx = -(xn * iup), sy = -(yn * iup);
    const V si = -(fma(xn, Fxi, yn * Fyi) * iup);
    const V sph = -(fma(xn, Fxp, yn * Fyp) * iup);
    // J = I + E + g s^T with s^T = ds/dp = (sx, sy, 0, si, sph, 0), g = dp'/ds = (cos phi', sin phi', cot, 0, w, 0)^T and the
    // fixed-path-length part E: E_03 = Fxi, E_04 = Fxp, E_13 = Fyi, E_14 = Fyp, E_25 = c5, E_43 = cw s.  Used in this form
    // (corrections added to C) the transport costs 30 instructions less than with the 17 Jacobian entries multiplied out.
    const V c5 = -(s * ist * ist), e43 = cw * s;
#define CC(i, j) C[pk(i, j)]
    // ---- T = J C = C + g (s^T C) + E C ----
#define RJ(j) fma(sx, CC(0, j), fma(sy, CC(1, j), fma(si, CC(3, j), sph * CC(4, j))))
    const V r0 = RJ(0), r1 = RJ(1), r2 = RJ(2), r3 = RJ(3), r4 = RJ(4), r5 = RJ(5);
#undef RJ
#define T0(j, r) fma(cpn, r, fma(Fxi, CC(3, j), fma(Fxp, CC(4, j), CC(0, j))))
#define T1(j, r) fma(spn, r, fma(Fyi, CC(3, j), fma(Fyp, CC(4, j), CC(1, j))))
#define T2(j, r) fma(cot, r, fma(c5, CC(5, j), CC(2, j)))
#define T4(j, r) fma(w, r, fma(e43, CC(3, j), CC(4, j)))
    const V T00 = T0(0, r0), T01 = T0(1, r1), T03 = T0(3, r3), T04 = T0(4, r4), T05 = T0(5, r5);
    const V T10 = T1(0, r0), T11 = T1(1, r1), T13 = T1(3, r3), T14 = T1(4, r4), T15 = T1(5, r5);
    const V T20 = T2(0, r0), T21 = T2(1, r1), T22 = T2(2, r2), T23 = T2(3, r3), T24 = T2(4, r4), T25 = T2(5, r5);
    const V T40 = T4(0, r0), T41 = T4(1, r1), T43 = T4(3, r3), T44 = T4(4, r4), T45 = T4(5, r5);
#undef T0
#undef T1
#undef T2
#undef T4
    // ---- C' = T J^T = T + (T s) g^T + T E^T, lower triangle; (4,2) through its mirror (2,4) ----
#define QI(Ta, Tb, Tc, Td) fma(sx, Ta, fma(sy, Tb, fma(si, Tc, sph * Td)))
    const V q0 = QI(T00, T01, T03, T04), q1 = QI(T10, T11, T13, T14), q2 = QI(T20, T21, T23, T24), q4 = QI(T40, T41, T43, T44);
#undef QI
    const V n00 = fma(q0, cpn, fma(Fxi, T03, fma(Fxp, T04, T00)));
    const V n10 = fma(q1, cpn, fma(Fxi, T13, fma(Fxp, T14, T10)));
    const V n11 = fma(q1, spn, fma(Fyi, T13, fma(Fyp, T14, T11)));
    const V n20 = fma(q2, cpn, fma(Fxi, T23, fma(Fxp, T24, T20)));
    const V n21 = fma(q2, spn, fma(Fyi, T23, fma(Fyp, T24, T21)));
    const V n22 = fma(q2, cot, fma(c5, T25, T22));
    const V n40 = fma(q4, cpn, fma(Fxi, T43, fma(Fxp, T44, T40)));
    const V n41 = fma(q4, spn, fma(Fyi, T43, fma(Fyp, T44, T41)));
    const V n42 = fma(q2, w, fma(e43, T23, T24));
    const V n44 = fma(q4, w, fma(e43, T43, T44));
    // ---- multiple scattering (R4) ----
    V q33 = sp(0.0f), q53 = sp(0.0f), q44 = sp(0.0f), q55 = sp(0.0f);
    if (ly.xx0r > 0.0f) {
        const V tms = ly.xx0r * ist * iup;
        const V lg = fma(log_(tms), 0.038f, 1.0f);
        const V h = 0.0136f * p[3] * st * lg;
        const V vv = h * h * tms;
        const V icot = p[3] * cot;
        q55 = vv;
        q44 = vv * ist * ist;
        q33 = icot * icot * vv;
        q53 = -(icot * vv);
    }
    C[pk(0, 0)] = n00;
    C[pk(1, 0)] = n10; C[pk(1, 1)] = n11;
    C[pk(2, 0)] = n20; C[pk(2, 1)] = n21; C[pk(2, 2)] = n22;
    C[pk(3, 0)] = T03; C[pk(3, 1)] = T13; C[pk(3, 2)] = T23; C[pk(3, 3)] = C[pk(3, 3)] + q33;
    C[pk(4, 0)] = n40; C[pk(4, 1)] = n41; C[pk(4, 2)] = n42; C[pk(4, 3)] = T43; C[pk(4, 4)] = n44 + q44;
    C[pk(5, 0)] = T05; C[pk(5, 1)] = T15; C[pk(5, 2)] = T25; C[pk(5, 3)] = C[pk(5, 3)] + q53; C[pk(5, 4)] = T45; C[pk(5, 5)] = C[pk(5, 5)] + q55;
#undef CC
    p[0] = xn; p[1] = yn; p[2] = zn;
    S.pha += phi_fix_small(alpha.v.x); S.phb += phi_fix_small(alpha.v.y);
    S.g.cp = cpn; S.g.sp = spn;
    return true;
}

// Update with the hits m (F7-F8), isotropic V = diag(vr, vr, vz): LDL^T factor of S = C_pos + V, chi2, gain by two
// triangular solves per row, state, covariance (columns of the measured block as K V).  false = not the fast path (the
// state is then garbage: the caller redoes the pair from the seed).
__device__ __forceinline__ bool update(State2& S, V mx, V my, V mz, float vr, float vz, V& chi2) {
    V (&p)[6] = S.p; V (&C)[21] = S.C;
    // LDL^T of the symmetric 3x3 S (branch-free; validity tested at the end)
    const V m00 = C[pk(0, 0)] + vr, m10 = C[pk(1, 0)], m11 = C[pk(1, 1)] + vr;
    const V m20 = C[pk(2, 0)], m21 = C[pk(2, 1)], m22 = C[pk(2, 2)] + vz;
    const V i0 = rcp(m00);
    const V l10 = m10 * i0, l20 = m20 * i0;
    const V d1 = fma(-l10, m10, m11);
    const V i1 = rcp(d1);
    const V t21 = fma(-l20, m10, m21);
    const V l21 = t21 * i1;
    const V d2 = fma(-l21, t21, fma(-l20, m20, m22));
    const V i2 = rcp(d2);
    bool ok = both_gt(m00, 0.0f) && both_gt(d1, 0.0f) && both_gt(d2, 0.0f);
    const V r0 = mx - p[0], r1 = my - p[1], r2 = mz - p[2];
    {
        const V y1 = fma(-l10, r0, r1);
        const V y2 = fma(-l21, y1, fma(-l20, r0, r2));
        chi2 = fma(r0 * r0, i0, fma(y1 * y1, i1, y2 * y2 * i2));
    }
    V K[6][3];
#pragma unroll
    for (int i = 0; i < 6; ++i) {       // x = S^-1 b for b = row i of C[:, 0:3]
        const V b0 = C[pk(i, 0)], b1 = C[pk(i, 1)], b2 = C[pk(i, 2)];
        const V y1 = fma(-l10, b0, b1);
        const V y2 = fma(-l21, y1, fma(-l20, b0, b2));
        K[i][2] = y2 * i2;
        K[i][1] = fma(-l21, K[i][2], y1 * i1);
        K[i][0] = fma(-l20, K[i][2], fma(-l10, K[i][1], b0 * i0));
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) p[i] = fma(K[i][0], r0, fma(K[i][1], r1, fma(K[i][2], r2, p[i])));
    const V dphi = fma(K[4][0], r0, fma(K[4][1], r1, K[4][2] * r2));
    const V dth = fma(K[5][0], r0, fma(K[5][1], r1, K[5][2] * r2));
    S.pha += phi_fix_small(dphi.v.x); S.phb += phi_fix_small(dphi.v.y);
    p[5] = p[5] + dth;
    ok = ok && both_lt(abs_(dphi), 0.06f) && both_lt(abs_(dth), 0.06f);
    rotate_poly(S.g.cp, S.g.sp, dphi);
    rotate_poly(S.g.ct, S.g.st, dth);
    // momentum block: C_ab -= sum_k K_ak C_bk with the still-intact old columns 0..2
#pragma unroll
    for (int a = 3; a < 6; ++a)
#pragma unroll
        for (int b = 3; b <= a; ++b)
            C[pk(a, b)] = fma(-K[a][0], C[pk(b, 0)], fma(-K[a][1], C[pk(b, 1)], fma(-K[a][2], C[pk(b, 2)], C[pk(a, b)])));
    // columns 0..2: K V
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        C[pk(i, 0)] = K[i][0] * vr;
        if (i >= 1) C[pk(i, 1)] = K[i][1] * vr;
        if (i >= 2) C[pk(i, 2)] = K[i][2] * vz;
    }
    // finite and physical: 0 * x is NaN for x = Inf or NaN
    const V z = fma(chi2, 0.0f, fma(p[0] + p[1], 0.0f, fma(p[2] + p[3], 0.0f, (dphi + p[5]) * 0.0f)));
    return ok && z.v.x == 0.0f && z.v.y == 0.0f && both_gt(p[3], 0.0f);
}

__device__ __forceinline__ bool all_finite(const State2& S) {
    V acc = S.p[0] * 0.0f;
#pragma unroll
    for (int i = 1; i < 6; ++i)
        if (i != 4) acc = fma(S.p[i], 0.0f, acc);
#pragma unroll
    for (int i = 0; i < 21; ++i) acc = fma(S.C[i], 0.0f, acc);
    return acc.v.x == 0.0f && acc.v.y == 0.0f;
}

}  // namespace pair
}  // namespace kf

// kf_math.cuh -- register-resident device math of the per-layer Kalman-filter step (fp32, sm_100a).
//
// One thread owns one track candidate: 6 parameters + 21 packed covariance elements live in registers for the whole
// layer loop.  The Jacobian's sparsity (20 non-zeros, 3 of them == 1; cf. "patterns of elements known ... to be zero
// or one", sec. 2.1) is written out by hand: J C J^T costs 138 FMA instead of 627 dense flops x/2.
// Formulas: DESIGN.md sec. 3 (R2 closed-form helix/cylinder solve, R3 surface Jacobian, R4 Highland noise,
// R5 3-D update).  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace kf {

constexpr float KCURV = 0.00299792458f;  // GeV / (T cm)
constexpr float CMIN = 0.1f;             // grazing guard on cos(incidence)

enum : uint32_t { ST_UNREACHABLE = 1u, ST_LEFT_Z = 2u, ST_GRAZING = 4u, ST_NUMERIC = 8u };

// per-layer constants, prepared on the host; two 16-byte vectors so that a layer is two constant-bank loads
struct alignas(16) LayerC {
    float r2, rcmin, xx0r, var_z;     // radius^2, r * CMIN, xx0 * r, hit variance along z
    float var_r, var_rphi, zmax, r;   // hit variances along r and r-phi, half length, radius
};

// 1-ulp hardware approximations (MUFU.RCP / MUFU.RSQ / MUFU.LG2): no IEEE slow paths, no branches.
__device__ __forceinline__ float frcp(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float fsqrt(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float flog(float x) { float r; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r * 0.69314718056f; }

// sin / cos of the two angles, carried along the track instead of being re-evaluated every layer: the transport
// rotates (cos phi, sin phi) by the exact rational (cos alpha, sin alpha), the update by a small-angle polynomial.
struct Trig { float cp, sp, st, ct; };

__device__ __forceinline__ void trig_init(Trig& g, float phi, float theta) {
    sincosf(phi, &g.sp, &g.cp);
    sincosf(theta, &g.st, &g.ct);
}

// rotate (c, s) by d: polynomial for |d| < 0.06 (truncation < 6e-11) followed by one Newton step back to unit norm
__device__ __forceinline__ void rotate_poly(float& c, float& s, float d) {
    const float d2 = d * d;
    const float sd = d * fmaf(d2, fmaf(d2, 1.0f / 120.0f, -1.0f / 6.0f), 1.0f);
    const float cd = fmaf(d2, fmaf(d2, 1.0f / 24.0f, -0.5f), 1.0f);
    const float cn = fmaf(c, cd, -s * sd), sn = fmaf(s, cd, c * sd);
    const float k = fmaf(-0.5f, fmaf(cn, cn, sn * sn), 1.5f);
    c = cn * k; s = sn * k;
}

// library call otherwise (angle = full value)
__device__ __forceinline__ void rotate_small(float& c, float& s, float d, float angle) {
    if (fabsf(d) < 0.06f) rotate_poly(c, s, d);
    else sincosf(angle, &s, &c);
}

// both angles of the state after an update; one test for the (rare) large correction
__device__ __forceinline__ void rotate_pair(Trig& g, float dphi, float dth, float phi, float theta) {
    if (fmaxf(fabsf(dphi), fabsf(dth)) < 0.06f) {
        rotate_poly(g.cp, g.sp, dphi);
        rotate_poly(g.ct, g.st, dth);
    } else {
        sincosf(phi, &g.sp, &g.cp);
        sincosf(theta, &g.st, &g.ct);
    }
}

// packed lower-triangular index
__host__ __device__ constexpr int pk(int i, int j) { return i >= j ? i * (i + 1) / 2 + j : j * (j + 1) / 2 + i; }

// Turning-angle functions of t = tan(alpha/2):  f = atan(t)/t  (alpha = 2 t f, s = 2 tau f) and the curvature partials
// f1(a) = (cos a - sin a / a)/a, f2(a) = (sin a - (1 - cos a)/a)/a of a = alpha.  One test selects the series for all
// three (|t| < 0.245, i.e. |alpha| < 0.48 per layer: every track above ~0.2 GeV on these geometries except near its
// turning point); truncation < 4e-9 relative.  The other side uses the library atan and the closed forms.
__device__ __forceinline__ void angle_functions(float t, float t2, float sa, float ca, float& f, float& alpha, float& f1, float& f2) {
    if (t2 < 0.06f) {
        f = fmaf(t2, fmaf(t2, fmaf(t2, fmaf(t2, fmaf(t2, -1.0f / 11.0f, 1.0f / 9.0f), -1.0f / 7.0f), 0.2f), -1.0f / 3.0f), 1.0f);
        alpha = 2.0f * t * f;
        const float a2 = alpha * alpha;
        f1 = alpha * fmaf(a2, fmaf(a2, fmaf(a2, 1.0f / 45360.0f, -1.0f / 840.0f), 1.0f / 30.0f), -1.0f / 3.0f);
        f2 = fmaf(a2, fmaf(a2, fmaf(a2, fmaf(a2, 1.0f / 403200.0f, -1.0f / 5760.0f), 1.0f / 144.0f), -0.125f), 0.5f);
    } else {
        f = atanf(t) * frcp(t);
        alpha = 2.0f * t * f;
        const float a2 = alpha * alpha;
        if (a2 < 0.25f) {
            f1 = alpha * fmaf(a2, fmaf(a2, fmaf(a2, 1.0f / 45360.0f, -1.0f / 840.0f), 1.0f / 30.0f), -1.0f / 3.0f);
            f2 = fmaf(a2, fmaf(a2, fmaf(a2, fmaf(a2, 1.0f / 403200.0f, -1.0f / 5760.0f), 1.0f / 144.0f), -0.125f), 0.5f);
        } else {
            const float ia = frcp(alpha);
            f1 = (ca - sa * ia) * ia;
            f2 = (sa - (1.0f - ca) * ia) * ia;
        }
    }
}

// Result of the transport to a cylinder (state only).
struct Transport {
    float dx, dy;        // x' - x, y' - y
    float xn, yn, zn;    // position on the cylinder
    float alpha, s;      // turning angle, transverse path length
    float sa, ca;        // sin / cos alpha
    float cpn, spn;      // cos / sin of phi'
    float up;            // x' cos phi' + y' sin phi' = r cos(incidence)
    float w;             // curvature
    float f1, f2;        // curvature partials (angle_functions)
};

// Closed-form first crossing of the cylinder r (R2): with u, v the position along / across the direction,
// E = (r^2 - x^2 - y^2)/2, A = 2(1 + v w) - w^2 E, D = u^2 + E A:  tau = tan(alpha/2)/w solves A tau^2 + 2 u tau - E = 0.
__device__ __forceinline__ uint32_t transport(const float (&p)[6], float cw, float cp, float sp, float cot,
                                              const LayerC& ly, Transport& t) {
    const float x = p[0], y = p[1];
    const float w = cw * p[3];
    const float u = fmaf(x, cp, y * sp);
    const float v = fmaf(y, cp, -x * sp);
    const float E = 0.5f * (ly.r2 - fmaf(x, x, y * y));
    const float A = fmaf(-w * w, E, 2.0f * fmaf(v, w, 1.0f));
    const float D = fmaf(E, A, u * u);
    // u >= 0 (moving outwards): tau = E / (u + sqrt D), the smaller positive root whatever the sign of A;
    // u < 0: tau = (sqrt D - u) / A, positive only for A > 0 (else the crossing lies beyond half a turn).
    // Branch-free on purpose: the sign of u is random for seeds smeared about the vertex.
    const bool fwd = u >= 0.0f;
    if (!(E > 0.0f) || !(D >= 0.0f) || !(fwd || A > 0.0f)) return ST_UNREACHABLE;
    const float sq = fsqrt(D);
    const float tau = (fwd ? E : sq - u) * frcp(fwd ? u + sq : A);
    const float th = w * tau;                     // tan(alpha/2)
    const float th2 = th * th;
    const float inv = frcp(1.0f + th2);
    const float X = 2.0f * tau * inv;             // sin(alpha)/w
    const float Y = X * th;                       // (1 - cos(alpha))/w
    t.sa = w * X;
    t.ca = (1.0f - th2) * inv;
    t.dx = fmaf(cp, X, -sp * Y);
    t.dy = fmaf(sp, X, cp * Y);
    t.xn = x + t.dx;
    t.yn = y + t.dy;
    float f;
    angle_functions(th, th2, t.sa, t.ca, f, t.alpha, t.f1, t.f2);
    t.s = 2.0f * tau * f;
    t.zn = fmaf(t.s, cot, p[2]);
    t.cpn = fmaf(cp, t.ca, -sp * t.sa);
    t.spn = fmaf(sp, t.ca, cp * t.sa);
    t.up = fmaf(t.xn, t.cpn, t.yn * t.spn);
    t.w = w;
    if (!(t.up >= ly.rcmin)) return (t.up == t.up) ? ST_GRAZING : ST_NUMERIC;
    return 0u;
}

// Predict: transport p, C to layer ly, C <- J C J^T + Q.  On a non-zero return p and C are untouched.
// cw = -q k Bz.  up_out = r cos(incidence) of the crossing.
__device__ __forceinline__ uint32_t predict(float (&p)[6], float (&C)[21], Trig& g, float cw, const LayerC& ly) {
    const float sp = g.sp, cp = g.cp, st = g.st, ct = g.ct;
    const float ist = frcp(st);
    const float cot = ct * ist;
    Transport t;
    const uint32_t flag = transport(p, cw, cp, sp, cot, ly, t);
    if (flag) return flag;

    // ---- Jacobian entries (R3) ----
    const float f1 = t.f1, f2 = t.f2;
    const float cs2 = cw * t.s * t.s;
    const float dXdi = cs2 * f1, dYdi = cs2 * f2;
    const float Fxi = fmaf(cp, dXdi, -sp * dYdi), Fyi = fmaf(sp, dXdi, cp * dYdi);
    const float Fxp = -t.dy, Fyp = t.dx;
    const float iup = frcp(t.up);
    const float sx = -t.xn * iup, sy = -t.yn * iup;
    const float si = -fmaf(t.xn, Fxi, t.yn * Fyi) * iup;
    const float sph = -fmaf(t.xn, Fxp, t.yn * Fyp) * iup;
    const float a0 = fmaf(t.cpn, sx, 1.0f), a1 = t.cpn * sy, a3 = fmaf(t.cpn, si, Fxi), a4 = fmaf(t.cpn, sph, Fxp);
    const float b0 = t.spn * sx, b1 = fmaf(t.spn, sy, 1.0f), b3 = fmaf(t.spn, si, Fyi), b4 = fmaf(t.spn, sph, Fyp);
    const float c0 = cot * sx, c1 = cot * sy, c3 = cot * si, c4 = cot * sph, c5 = -t.s * ist * ist;
    const float d0 = t.w * sx, d1 = t.w * sy, d3 = fmaf(t.w, si, cw * t.s), d4 = fmaf(t.w, sph, 1.0f);

#define CC(i, j) C[pk(i, j)]
    // ---- T = J C: rows 0, 1, 4 (columns 0,1,3,4,5) and row 2 (all columns) ----
#define ROW4(c0_, c1_, c3_, c4_, j) fmaf(c0_, CC(0, j), fmaf(c1_, CC(1, j), fmaf(c3_, CC(3, j), c4_ * CC(4, j))))
    const float T00 = ROW4(a0, a1, a3, a4, 0), T01 = ROW4(a0, a1, a3, a4, 1), T03 = ROW4(a0, a1, a3, a4, 3),
                T04 = ROW4(a0, a1, a3, a4, 4), T05 = ROW4(a0, a1, a3, a4, 5);
    const float T10 = ROW4(b0, b1, b3, b4, 0), T11 = ROW4(b0, b1, b3, b4, 1), T13 = ROW4(b0, b1, b3, b4, 3),
                T14 = ROW4(b0, b1, b3, b4, 4), T15 = ROW4(b0, b1, b3, b4, 5);
    const float T40 = ROW4(d0, d1, d3, d4, 0), T41 = ROW4(d0, d1, d3, d4, 1), T43 = ROW4(d0, d1, d3, d4, 3),
                T44 = ROW4(d0, d1, d3, d4, 4), T45 = ROW4(d0, d1, d3, d4, 5);
#define ROW6(j) (fmaf(c0, CC(0, j), fmaf(c1, CC(1, j), fmaf(c3, CC(3, j), fmaf(c4, CC(4, j), fmaf(c5, CC(5, j), CC(2, j)))))))
    const float T20 = ROW6(0), T21 = ROW6(1), T22 = ROW6(2), T23 = ROW6(3), T24 = ROW6(4), T25 = ROW6(5);
#undef ROW4
#undef ROW6
    // ---- C' = T J^T, lower triangle; rows 3 and 5 of J are unit rows ----
#define DOT4(T0, T1, T3, T4, e0, e1, e3, e4) fmaf(T0, e0, fmaf(T1, e1, fmaf(T3, e3, T4 * e4)))
    const float n00 = DOT4(T00, T01, T03, T04, a0, a1, a3, a4);
    const float n10 = DOT4(T10, T11, T13, T14, a0, a1, a3, a4);
    const float n11 = DOT4(T10, T11, T13, T14, b0, b1, b3, b4);
    const float n20 = DOT4(T20, T21, T23, T24, a0, a1, a3, a4);
    const float n21 = DOT4(T20, T21, T23, T24, b0, b1, b3, b4);
    const float n22 = fmaf(T20, c0, fmaf(T21, c1, fmaf(T23, c3, fmaf(T24, c4, fmaf(T25, c5, T22)))));
    const float n40 = DOT4(T40, T41, T43, T44, a0, a1, a3, a4);
    const float n41 = DOT4(T40, T41, T43, T44, b0, b1, b3, b4);
    const float n42 = DOT4(T20, T21, T23, T24, d0, d1, d3, d4);
    const float n44 = DOT4(T40, T41, T43, T44, d0, d1, d3, d4);
#undef DOT4
    // ---- multiple scattering (R4), evaluated at the arriving state ----
    float q33 = 0.0f, q53 = 0.0f, q44 = 0.0f, q55 = 0.0f;
    if (ly.xx0r > 0.0f) {
        const float tms = ly.xx0r * ist * iup;                 // xx0 / (sin(theta) cos(inc))
        const float lg = fmaf(0.038f, flog(tms), 1.0f);
        const float h = 0.0136f * p[3] * st * lg;
        const float v = h * h * tms;                           // theta0^2
        const float icot = p[3] * cot;
        q55 = v;
        q44 = v * ist * ist;
        q33 = icot * icot * v;
        q53 = -icot * v;
    }
    // commit
    C[pk(0, 0)] = n00;
    C[pk(1, 0)] = n10; C[pk(1, 1)] = n11;
    C[pk(2, 0)] = n20; C[pk(2, 1)] = n21; C[pk(2, 2)] = n22;
    C[pk(3, 0)] = T03; C[pk(3, 1)] = T13; C[pk(3, 2)] = T23; C[pk(3, 3)] += q33;
    C[pk(4, 0)] = n40; C[pk(4, 1)] = n41; C[pk(4, 2)] = n42; C[pk(4, 3)] = T43; C[pk(4, 4)] = n44 + q44;
    C[pk(5, 0)] = T05; C[pk(5, 1)] = T15; C[pk(5, 2)] = T25; C[pk(5, 3)] += q53; C[pk(5, 4)] = T45; C[pk(5, 5)] += q55;
#undef CC
    p[0] = t.xn; p[1] = t.yn; p[2] = t.zn; p[4] += t.alpha;
    g.cp = t.cpn; g.sp = t.spn;
    return 0u;
}

// Hit covariance (R5): rotation of diag(var_r, var_rphi) to the hit's azimuth, var_z along z.
struct HitCov { float xx, xy, yy, zz; };
__device__ __forceinline__ HitCov hit_cov(float mx, float my, const LayerC& ly) {
    HitCov V;
    V.zz = ly.var_z;
    if (ly.var_r == ly.var_rphi) {
        V.xx = ly.var_r; V.yy = ly.var_r; V.xy = 0.0f;
    } else {
        const float ir2 = frcp(fmaf(mx, mx, my * my));
        const float c2 = mx * mx * ir2, s2 = my * my * ir2, cs = mx * my * ir2;
        V.xx = fmaf(c2, ly.var_r, s2 * ly.var_rphi);
        V.yy = fmaf(s2, ly.var_r, c2 * ly.var_rphi);
        V.xy = cs * (ly.var_r - ly.var_rphi);
    }
    return V;
}

// Symmetric positive-definite 3x3 system by LDL^T (Cholesky without square roots).  Backward stable for SPD
// matrices, which a cofactor inverse is not: for low-pT tracks S = C_pos + V has condition number ~1e4 (predicted
// tangential variance vs hit variance) and the 1/det-scaled rounding errors of cofactors would reach every element.
struct Sym3 { float m00, m10, m11, m20, m21, m22; };
struct Ldl3 { float l10, l20, l21, i0, i1, i2; };

// Branch-free: a non-positive pivot makes the later entries garbage (Inf / NaN), never a trap; the caller must not use
// F when the result is false.
__device__ __forceinline__ bool ldl3(const Sym3& S, Ldl3& F) {
    F.i0 = frcp(S.m00);
    F.l10 = S.m10 * F.i0;
    F.l20 = S.m20 * F.i0;
    const float d1 = fmaf(-F.l10, S.m10, S.m11);
    F.i1 = frcp(d1);
    const float t21 = fmaf(-F.l20, S.m10, S.m21);
    F.l21 = t21 * F.i1;
    const float d2 = fmaf(-F.l21, t21, fmaf(-F.l20, S.m20, S.m22));
    F.i2 = frcp(d2);
    return (S.m00 > 0.0f) && (d1 > 0.0f) && (d2 > 0.0f);
}

// x = S^-1 b
__device__ __forceinline__ void ldl3_solve(const Ldl3& F, float b0, float b1, float b2, float& x0, float& x1, float& x2) {
    const float y1 = fmaf(-F.l10, b0, b1);
    const float y2 = fmaf(-F.l21, y1, fmaf(-F.l20, b0, b2));
    x2 = y2 * F.i2;
    x1 = fmaf(-F.l21, x2, y1 * F.i1);
    x0 = fmaf(-F.l20, x2, fmaf(-F.l10, x1, b0 * F.i0));
}

// Innovation of hit m against the predicted (p, C): factor S = C_pos + V, r = m - p[0:3], chi2 = r^T S^-1 r.
__device__ __forceinline__ bool innovation(const float (&p)[6], const float (&C)[21], float mx, float my, float mz,
                                           const HitCov& V, Ldl3& F, float (&r)[3], float& chi2) {
    Sym3 S;
    S.m00 = C[pk(0, 0)] + V.xx; S.m10 = C[pk(1, 0)] + V.xy; S.m11 = C[pk(1, 1)] + V.yy;
    S.m20 = C[pk(2, 0)]; S.m21 = C[pk(2, 1)]; S.m22 = C[pk(2, 2)] + V.zz;
    const bool ok = ldl3(S, F);
    r[0] = mx - p[0]; r[1] = my - p[1]; r[2] = mz - p[2];
    const float y1 = fmaf(-F.l10, r[0], r[1]);
    const float y2 = fmaf(-F.l21, y1, fmaf(-F.l20, r[0], r[2]));
    chi2 = fmaf(r[0] * r[0], F.i0, fmaf(y1 * y1, F.i1, y2 * y2 * F.i2));
    return ok;
}

// Gain and update (R5): K = C[:,0:3] S^-1, p += K r, C <- C - K C[0:3,:].
// The columns that touch the measured block are written in the algebraically identical, cancellation-free form
//   (C - K H C) H^T = C H^T - K (S - V) = K V          (because K S = C H^T),
// which matters in fp32: for low-pT tracks at shallow incidence the predicted position variance exceeds the hit
// variance by 1e3-1e4 and C - K C would lose every significant digit of the updated position block.
// ISO: V = diag(V.xx, V.xx, V.zz) known at compile time (sig_r == sig_rphi on every layer).
template <bool ISO = false>
__device__ __forceinline__ void gain_update(float (&p)[6], float (&C)[21], Trig& g, const Ldl3& F, const HitCov& V,
                                            const float (&r)[3]) {
    float K[6][3];
#pragma unroll
    for (int i = 0; i < 6; ++i) ldl3_solve(F, C[pk(i, 0)], C[pk(i, 1)], C[pk(i, 2)], K[i][0], K[i][1], K[i][2]);
#pragma unroll
    for (int i = 0; i < 4; ++i) p[i] = fmaf(K[i][0], r[0], fmaf(K[i][1], r[1], fmaf(K[i][2], r[2], p[i])));
    const float dphi = fmaf(K[4][0], r[0], fmaf(K[4][1], r[1], K[4][2] * r[2]));
    const float dth = fmaf(K[5][0], r[0], fmaf(K[5][1], r[1], K[5][2] * r[2]));
    p[4] += dphi;
    p[5] += dth;
    rotate_pair(g, dphi, dth, p[4], p[5]);
    // momentum block (rows/cols 3..5): C_ab -= sum_k K_ak C_kb, with the still-intact old C[b][k]
#pragma unroll
    for (int a = 3; a < 6; ++a)
#pragma unroll
        for (int b = 3; b <= a; ++b)
            C[pk(a, b)] = fmaf(-K[a][0], C[pk(b, 0)], fmaf(-K[a][1], C[pk(b, 1)], fmaf(-K[a][2], C[pk(b, 2)], C[pk(a, b)])));
    // columns 0..2: K V
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        if (ISO) {
            C[pk(i, 0)] = K[i][0] * V.xx;
            if (i >= 1) C[pk(i, 1)] = K[i][1] * V.xx;
        } else {
            C[pk(i, 0)] = fmaf(K[i][0], V.xx, K[i][1] * V.xy);
            if (i >= 1) C[pk(i, 1)] = fmaf(K[i][0], V.xy, K[i][1] * V.yy);
        }
        if (i >= 2) C[pk(i, 2)] = K[i][2] * V.zz;
    }
}

__device__ __forceinline__ float wrap_phi(float a) {
    const float TWO_PI = 6.28318530717958647692f, PI = 3.14159265358979323846f;
    a -= TWO_PI * floorf((a + PI) * (1.0f / TWO_PI));
    if (a <= -PI) a += TWO_PI;
    if (a > PI) a -= TWO_PI;
    return a;
}

// cheap per-layer check: NaN/Inf anywhere in S or the gain reaches chi2 or the parameters
__device__ __forceinline__ bool step_finite(const float (&p)[6], float chi2) {
    const float acc = fmaf(0.0f, chi2, 0.0f * (((p[0] + p[1]) + (p[2] + p[3])) + (p[4] + p[5])));
    return acc == 0.0f;
}

__device__ __forceinline__ bool all_finite(const float (&p)[6], const float (&C)[21]) {
    float acc = 0.0f;
#pragma unroll
    for (int i = 0; i < 6; ++i) acc = fmaf(0.0f, p[i], acc);
#pragma unroll
    for (int i = 0; i < 21; ++i) acc = fmaf(0.0f, C[i], acc);
    return acc == 0.0f;   // 0 * inf = NaN, 0 * NaN = NaN
}

}  // namespace kf

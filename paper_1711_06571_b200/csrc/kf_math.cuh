// kf_math.cuh -- scalar pieces of the per-layer Kalman-filter step (fp32, sm_100a): per-layer constants, hardware
// approximations, the closed-form helix/cylinder solve (R2), the hit covariance and the 3x3 LDL^T factor
// (R5).  The 6x6 algebra on the packed register state lives in kf_state.cuh.  Shares nothing with oracle/.
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
    float var_r, var_rphi, zmax, r;   // hit variances along r and r-phi, half length (disk: outer radius), radius (disk: z)
    float xx0, rmin; int32_t kind, pad_;   // thickness, inner radius of a disk, 0 = cylinder / 1 = disk
};

// 1-ulp hardware approximations (MUFU.RCP / MUFU.RSQ / MUFU.LG2): no IEEE slow paths, no branches.
__device__ __forceinline__ float frcp(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float fsqrt(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float flog(float x) { float r; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r * 0.69314718056f; }

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
// NEAR (second step of the two-step propagation, R20): the nearest crossing of a radius close to the state's own,
// forwards or backwards (E of either sign); the state must move outwards (u > 0).
template <bool NEAR = false>
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
    const bool fwd = NEAR || u >= 0.0f;
    if (NEAR ? (!(u > 0.0f) || !(D >= 0.0f)) : (!(E > 0.0f) || !(D >= 0.0f) || !(fwd || A > 0.0f))) return ST_UNREACHABLE;
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

__device__ __forceinline__ float wrap_phi(float a) {
    const float TWO_PI = 6.28318530717958647692f, PI = 3.14159265358979323846f;
    a -= TWO_PI * floorf((a + PI) * (1.0f / TWO_PI));
    if (a <= -PI) a += TWO_PI;
    if (a > PI) a -= TWO_PI;
    return a;
}

}  // namespace kf

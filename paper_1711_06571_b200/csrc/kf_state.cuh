// kf_state.cuh -- the per-layer Kalman-filter step on a register-resident state laid out for Blackwell's packed
// fp32 arithmetic (FFMA2 / FMUL2 / FADD2: two fp32 lanes per instruction; sm_100a).
//
// Why: a packed FFMA2 does two fp32 FMAs in one issue slot and takes any scalar register as a free broadcast operand, so
// a candidate's step takes 452 instead of 560 warp instructions.  The 6x6 algebra of the
// step is arranged so that its long, regular chains run two rows (or two columns) of a matrix at a time:
//   rows (x, y) and rows (z, phi) of T = J C and of J C J^T,        columns (1/pT, theta) of T,
//   rows (0,1), (2,4), (3,5) of the gain K = C H^T S^-1 and of the covariance update.
// The covariance is stored in exactly the pairs those chains consume and produce, so no repacking is needed between
// layers; three elements are held twice (C01, C20, C21) and kept identical by copies.
// Jacobian sparsity (20 non-zeros, 3 of them == 1; "patterns of elements known ... to be zero or one", PAPER.md:L40
// sec. 2.1) is written out by hand.  Formulas: DESIGN.md sec. 3 (R2 helix/cylinder solve, R3 surface Jacobian, R4 Highland noise,
// R5 3-D update).  Shares nothing with oracle/.
#pragma once
#include "kf_math.cuh"

namespace kf {

__device__ __forceinline__ float2 f2(float a, float b) { return make_float2(a, b); }
__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 fma2(float2 a, float s, float2 c) { return __ffma2_rn(a, make_float2(s, s), c); }   // s: broadcast
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 mul2(float2 a, float s) { return __fmul2_rn(a, make_float2(s, s)); }
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }

// The azimuth phi is only ever accumulated (turning angles, update corrections) and written out; the arithmetic uses the
// carried sin/cos.  It is kept as a 32-bit fixed-point angle, phi = PH * pi / 2^31: integer addition wraps modulo 2 pi
// exactly and does not round, so the output carries one rounding instead of 2 L of them at the size of the largest
// intermediate angle (a 0.5 GeV track turns by ~2 rad on the way out; its final |phi| may be 1e-3: the 1e-6 absolute floor
// of the parity tolerance is then below the accumulated fp32 rounding).
constexpr float PHI_TO_FIX = 683565275.57643158978f;          // 2^31 / pi
constexpr float FIX_TO_PHI = 1.46291807926715968105e-9f;      // pi / 2^31
__device__ __forceinline__ int phi_fix_small(float a) { return __float2int_rn(a * PHI_TO_FIX); }                                // |a| <= pi
__device__ __forceinline__ int phi_fix(float a) { return (int)__double2ll_rn((double)a * 683565275.57643158978); }            // any a, modulo 2 pi
__device__ __forceinline__ float phi_float(int f) { return f == (int)0x80000000 ? 3.14159265358979323846f : (float)f * FIX_TO_PHI; }   // (-pi, pi]

// Track state: 6 parameters, carried sin/cos of both angles, 21 covariance elements (+3 duplicates).
struct State {
    float2 XY;           // x, y
    float Z;             // z
    int PH;              // phi, fixed point
    float dph;           // last update's correction of phi (finiteness checks only)
    float2 IT;           // 1/pT, theta
    float2 CC, SS;       // (cos phi, cos theta), (sin phi, sin theta)
    float2 P0, P1, P2;   // (C00, C10), (C01, C11), (C02, C12): rows 0,1 x columns 0,1,2
    float2 Q0, Q1, Q2;   // (C20, C40), (C21, C41), (C22, C42): rows 2,4 x columns 0,1,2
    float2 R0, R1, R2;   // (C30, C50), (C31, C51), (C32, C52): rows 3,5 x columns 0,1,2
    float2 M3, M4;       // (C33, C53), (C43, C54)
    float C44, C55;
};

// packed lower-triangular storage <-> State (k = i(i+1)/2 + j).  RAW: par(4) is the bit pattern of the fixed-point angle
// (intermediate records), otherwise phi in radians.
template <bool RAW = false, typename LoadP, typename LoadC>
__device__ __forceinline__ void state_set(State& s, LoadP par, LoadC cov) {
    s.XY = f2(par(0), par(1)); s.Z = par(2); s.IT = f2(par(3), par(5));
    s.PH = RAW ? __float_as_int(par(4)) : phi_fix(par(4));
    s.dph = 0.0f;
    const float c10 = cov(pk(1, 0)), c20 = cov(pk(2, 0)), c21 = cov(pk(2, 1));
    s.P0 = f2(cov(pk(0, 0)), c10); s.P1 = f2(c10, cov(pk(1, 1))); s.P2 = f2(c20, c21);
    s.Q0 = f2(c20, cov(pk(4, 0))); s.Q1 = f2(c21, cov(pk(4, 1))); s.Q2 = f2(cov(pk(2, 2)), cov(pk(4, 2)));
    s.R0 = f2(cov(pk(3, 0)), cov(pk(5, 0))); s.R1 = f2(cov(pk(3, 1)), cov(pk(5, 1))); s.R2 = f2(cov(pk(3, 2)), cov(pk(5, 2)));
    s.M3 = f2(cov(pk(3, 3)), cov(pk(5, 3))); s.M4 = f2(cov(pk(4, 3)), cov(pk(5, 4)));
    s.C44 = cov(pk(4, 4)); s.C55 = cov(pk(5, 5));
}

// sin / cos of both angles from the angles themselves (start of a track; afterwards they are carried)
__device__ __forceinline__ void state_trig(State& s, float phi) {
    float sp, cp, st, ct;
    sincosf(phi, &sp, &cp);
    sincosf(s.IT.y, &st, &ct);
    s.CC = f2(cp, ct); s.SS = f2(sp, st);
}

template <typename LoadP, typename LoadC>
__device__ __forceinline__ void state_load(State& s, LoadP par, LoadC cov) {
    state_set(s, par, cov);
    state_trig(s, par(4));
}

// WRAP: phi in radians in (-pi, pi] (final output) or the bit pattern of the fixed-point angle (intermediate record)
template <bool WRAP = true, typename StoreP, typename StoreC>
__device__ __forceinline__ void state_store(const State& s, StoreP par, StoreC cov) {
    par(0, s.XY.x); par(1, s.XY.y); par(2, s.Z); par(3, s.IT.x); par(4, WRAP ? phi_float(s.PH) : __int_as_float(s.PH)); par(5, s.IT.y);
    cov(pk(0, 0), s.P0.x);
    cov(pk(1, 0), s.P0.y); cov(pk(1, 1), s.P1.y);
    cov(pk(2, 0), s.P2.x); cov(pk(2, 1), s.P2.y); cov(pk(2, 2), s.Q2.x);
    cov(pk(3, 0), s.R0.x); cov(pk(3, 1), s.R1.x); cov(pk(3, 2), s.R2.x); cov(pk(3, 3), s.M3.x);
    cov(pk(4, 0), s.Q0.y); cov(pk(4, 1), s.Q1.y); cov(pk(4, 2), s.Q2.y); cov(pk(4, 3), s.M4.x); cov(pk(4, 4), s.C44);
    cov(pk(5, 0), s.R0.y); cov(pk(5, 1), s.R1.y); cov(pk(5, 2), s.R2.y); cov(pk(5, 3), s.M3.y); cov(pk(5, 4), s.M4.y); cov(pk(5, 5), s.C55);
}

// 0 * inf = NaN, 0 * NaN = NaN: one fused chain over everything
__device__ __forceinline__ bool state_finite(const State& s) {
    float2 a = mul2(s.XY, 0.0f);
    a = fma2(f2(s.Z, s.dph), 0.0f, a); a = fma2(s.IT, 0.0f, a);
    a = fma2(s.P0, 0.0f, a); a = fma2(s.P1, 0.0f, a); a = fma2(s.P2, 0.0f, a);
    a = fma2(s.Q0, 0.0f, a); a = fma2(s.Q1, 0.0f, a); a = fma2(s.Q2, 0.0f, a);
    a = fma2(s.R0, 0.0f, a); a = fma2(s.R1, 0.0f, a); a = fma2(s.R2, 0.0f, a);
    a = fma2(s.M3, 0.0f, a); a = fma2(s.M4, 0.0f, a);
    return fmaf(0.0f, s.C44, fmaf(0.0f, s.C55, a.x + a.y)) == 0.0f;
}

// cheap per-layer check: NaN/Inf anywhere in S or the gain reaches chi2 or the parameters
__device__ __forceinline__ bool step_finite(const State& s, float chi2) {
    const float2 a = fma2(s.XY, 0.0f, fma2(f2(s.Z, s.dph), 0.0f, mul2(s.IT, 0.0f)));
    return fmaf(0.0f, chi2, a.x + a.y) == 0.0f;
}

// Predict: transport the state to layer ly, C <- J C J^T + Q (R2-R4).  On a non-zero return s is untouched.
// cw = -q k Bz.
// NEAR: second step of the two-step propagation (R20): to the nearest crossing of ly.r2, either direction, no material.
template <bool NEAR = false>
__device__ __forceinline__ uint32_t predict(State& s, float cw, const LayerC& ly) {
    const float cp = s.CC.x, ct = s.CC.y, sp = s.SS.x, st = s.SS.y;
    const float ist = frcp(st);
    const float cot = ct * ist;
    const float pp[6] = {s.XY.x, s.XY.y, s.Z, s.IT.x, 0.0f, s.IT.y};       // transport works from the carried sin / cos, not from phi
    Transport t;
    const uint32_t flag = transport<NEAR>(pp, cw, cp, sp, cot, ly, t);
    if (flag) return flag;

    // ---- Jacobian (R3): rows x', y' as pairs ab_k = (a_k, b_k), rows z', phi' as pairs cd_k = (c_k, d_k) ----
    const float cs2 = cw * t.s * t.s;
    const float dXdi = cs2 * t.f1, dYdi = cs2 * t.f2;
    const float Fxi = fmaf(cp, dXdi, -sp * dYdi), Fyi = fmaf(sp, dXdi, cp * dYdi);
    const float iup = frcp(t.up);
    const float sx = -t.xn * iup, sy = -t.yn * iup;
    const float si = -fmaf(t.xn, Fxi, t.yn * Fyi) * iup;
    const float sph = -fmaf(t.yn, t.dx, -t.xn * t.dy) * iup;       // F_x,phi = -dy, F_y,phi = dx
    const float2 G = f2(t.cpn, t.spn);
    const float2 ab0 = f2(fmaf(t.cpn, sx, 1.0f), t.spn * sx), ab1 = f2(t.cpn * sy, fmaf(t.spn, sy, 1.0f));
    const float2 ab3 = fma2(G, si, f2(Fxi, Fyi)), ab4 = fma2(G, sph, f2(-t.dy, t.dx));
    const float2 H = f2(cot, t.w);
    const float2 cd0 = mul2(H, sx), cd1 = mul2(H, sy);
    const float2 cd3 = f2(cot * si, fmaf(t.w, si, cw * t.s)), cd4 = f2(cot * sph, fmaf(t.w, sph, 1.0f));
    const float c5 = -t.s * ist * ist;

    // ---- T = J C ----
    // columns 0, 1, 4 of T for the row pairs: T_k = sum_m J_m * C_mk (m = 0, 1, 3, 4); row z' also takes C_2k + c5 C_5k
#define KF_ROWS(v0, v1, v3, v4, e0, e1, e3, e4) fma2(v0, e0, fma2(v1, e1, fma2(v3, e3, mul2(v4, e4))))
    const float2 Tab0 = KF_ROWS(ab0, ab1, ab3, ab4, s.P0.x, s.P0.y, s.R0.x, s.Q0.y);
    float2 Tcd0 = KF_ROWS(cd0, cd1, cd3, cd4, s.P0.x, s.P0.y, s.R0.x, s.Q0.y);
    Tcd0.x += fmaf(c5, s.R0.y, s.P2.x);
    const float2 Tab1 = KF_ROWS(ab0, ab1, ab3, ab4, s.P0.y, s.P1.y, s.R1.x, s.Q1.y);
    float2 Tcd1 = KF_ROWS(cd0, cd1, cd3, cd4, s.P0.y, s.P1.y, s.R1.x, s.Q1.y);
    Tcd1.x += fmaf(c5, s.R1.y, s.P2.y);
    const float2 Tab4 = KF_ROWS(ab0, ab1, ab3, ab4, s.Q0.y, s.Q1.y, s.M4.x, s.C44);
    float2 Tcd4 = KF_ROWS(cd0, cd1, cd3, cd4, s.Q0.y, s.Q1.y, s.M4.x, s.C44);
    Tcd4.x += fmaf(c5, s.M4.y, s.Q2.y);
    // columns (3, 5) of T as pairs, one per row: (T_j3, T_j5) = sum_m J_jm * (C_m3, C_m5)
    const float2 RTa = KF_ROWS(s.R0, s.R1, s.M3, s.M4, ab0.x, ab1.x, ab3.x, ab4.x);
    const float2 RTb = KF_ROWS(s.R0, s.R1, s.M3, s.M4, ab0.y, ab1.y, ab3.y, ab4.y);
    const float2 RTd = KF_ROWS(s.R0, s.R1, s.M3, s.M4, cd0.y, cd1.y, cd3.y, cd4.y);
    float2 RTc = fma2(s.R0, cd0.x, fma2(s.R1, cd1.x, fma2(s.M3, cd3.x, fma2(s.M4, cd4.x, s.R2))));
    RTc.x = fmaf(c5, s.M3.y, RTc.x);
    RTc.y = fmaf(c5, s.C55, RTc.y);
    const float T22 = fmaf(cd0.x, s.P2.x, fmaf(cd1.x, s.P2.y, fmaf(cd3.x, s.R2.x, fmaf(cd4.x, s.Q2.y, fmaf(c5, s.R2.y, s.Q2.x)))));
    const float2 Tab3 = f2(RTa.x, RTb.x), Tcd3 = f2(RTc.x, RTd.x);
    // ---- C' = T J^T (rows 1/pT and theta of J are unit rows) ----
    const float2 nP0 = KF_ROWS(Tab0, Tab1, Tab3, Tab4, ab0.x, ab1.x, ab3.x, ab4.x);          // (C00, C10)
    const float n11 = fmaf(Tab0.y, ab0.y, fmaf(Tab1.y, ab1.y, fmaf(Tab3.y, ab3.y, Tab4.y * ab4.y)));
    const float2 nQ0 = KF_ROWS(Tcd0, Tcd1, Tcd3, Tcd4, ab0.x, ab1.x, ab3.x, ab4.x);          // (C20, C40)
    const float2 nQ1 = KF_ROWS(Tcd0, Tcd1, Tcd3, Tcd4, ab0.y, ab1.y, ab3.y, ab4.y);          // (C21, C41)
    float2 nQ2 = KF_ROWS(cd0, cd1, cd3, cd4, Tcd0.x, Tcd1.x, Tcd3.x, Tcd4.x);                // (C22 - ..., C42)
    nQ2.x += fmaf(RTc.y, c5, T22);
    const float n44 = fmaf(Tcd0.y, cd0.y, fmaf(Tcd1.y, cd1.y, fmaf(Tcd3.y, cd3.y, Tcd4.y * cd4.y)));
#undef KF_ROWS
    // ---- multiple scattering (R4), evaluated at the arriving state ----
    float q33 = 0.0f, q53 = 0.0f, q44 = 0.0f, q55 = 0.0f;
    if (!NEAR && ly.xx0r > 0.0f) {
        const float iota = s.IT.x;
        const float tms = ly.xx0r * ist * iup;                 // xx0 / (sin(theta) cos(inc))
        const float lg = fmaf(0.038f, flog(tms), 1.0f);
        const float h = 0.0136f * iota * st * lg;
        const float v = h * h * tms;                           // theta0^2
        const float icot = iota * cot;
        q55 = v;
        q44 = v * ist * ist;
        q33 = icot * icot * v;
        q53 = -icot * v;
    }
    // ---- commit ----
    s.P0 = nP0; s.P1 = f2(nP0.y, n11); s.P2 = f2(nQ0.x, nQ1.x);
    s.Q0 = nQ0; s.Q1 = nQ1; s.Q2 = nQ2;
    s.R0 = RTa; s.R1 = RTb; s.R2 = RTc;
    s.M4 = RTd;
    s.M3.x += q33; s.M3.y += q53;
    s.C44 = n44 + q44;
    s.C55 += q55;
    s.XY = f2(t.xn, t.yn);
    s.Z = t.zn;
    s.PH += phi_fix_small(t.alpha);
    s.CC.x = t.cpn; s.SS.x = t.spn;
    return 0u;
}

// Innovation of hit m against the predicted state: factor S = C_pos + V, r = m - pos, chi2 = r^T S^-1 r.
// Branch-free: when the result is false F, r, chi2 are garbage.
__device__ __forceinline__ bool innovation(const State& s, float mx, float my, float mz, const HitCov& V, Ldl3& F, float (&r)[3],
                                           float& chi2) {
    Sym3 S;
    S.m00 = s.P0.x + V.xx; S.m10 = s.P0.y + V.xy; S.m11 = s.P1.y + V.yy;
    S.m20 = s.P2.x; S.m21 = s.P2.y; S.m22 = s.Q2.x + V.zz;
    const bool ok = ldl3(S, F);
    r[0] = mx - s.XY.x; r[1] = my - s.XY.y; r[2] = mz - s.Z;
    const float y1 = fmaf(-F.l10, r[0], r[1]);
    const float y2 = fmaf(-F.l21, y1, fmaf(-F.l20, r[0], r[2]));
    chi2 = fmaf(r[0] * r[0], F.i0, fmaf(y1 * y1, F.i1, y2 * y2 * F.i2));
    return ok;
}

// two rows of K = C[:,0:3] S^-1 at once: x = S^-1 b for the pairs (b0, b1, b2)
__device__ __forceinline__ void ldl3_solve2(const Ldl3& F, float2 b0, float2 b1, float2 b2, float2& x0, float2& x1, float2& x2) {
    const float2 y1 = fma2(neg2(b0), F.l10, b1);
    const float2 y2 = fma2(neg2(y1), F.l21, fma2(neg2(b0), F.l20, b2));
    x2 = mul2(y2, F.i2);
    x1 = fma2(neg2(x2), F.l21, mul2(y1, F.i1));
    x0 = fma2(neg2(x2), F.l20, fma2(neg2(x1), F.l10, mul2(b0, F.i0)));
}

// rotate (c, s) by d for both angles at once: polynomial for |d| < 0.06 (truncation < 6e-11) followed by one Newton
// step back to unit norm
__device__ __forceinline__ void rotate_poly2(float2& c, float2& sn_, float2 d) {
    const float2 d2 = mul2(d, d);
    const float2 sd = mul2(d, fma2(d2, fma2(d2, 1.0f / 120.0f, f2(-1.0f / 6.0f, -1.0f / 6.0f)), f2(1.0f, 1.0f)));
    const float2 cd = fma2(d2, fma2(d2, 1.0f / 24.0f, f2(-0.5f, -0.5f)), f2(1.0f, 1.0f));
    const float2 cn = fma2(c, cd, neg2(mul2(sn_, sd))), sn = fma2(sn_, cd, mul2(c, sd));
    const float2 k = fma2(fma2(cn, cn, mul2(sn, sn)), -0.5f, f2(1.5f, 1.5f));
    c = mul2(cn, k); sn_ = mul2(sn, k);
}

// Gain and update (R5): K = C[:,0:3] S^-1, p += K r, C <- C - K C[0:3,:].
// The columns that touch the measured block are written in the algebraically identical, cancellation-free form
//   (C - K H C) H^T = C H^T - K (S - V) = K V          (because K S = C H^T),
// which matters in fp32: for low-pT tracks at shallow incidence the predicted position variance exceeds the hit
// variance by 1e3-1e4 and C - K C would lose every significant digit of the updated position block.
// ISO: V = diag(V.xx, V.xx, V.zz) (sig_r == sig_rphi on every layer).
template <bool ISO>
__device__ __forceinline__ void gain_update(State& s, const Ldl3& F, const HitCov& V, const float (&r)[3]) {
    float2 KP0, KP1, KP2, KQ0, KQ1, KQ2, KR0, KR1, KR2;      // K rows (0,1), (2,4), (3,5); index = column
    ldl3_solve2(F, s.P0, s.P1, s.P2, KP0, KP1, KP2);
    ldl3_solve2(F, s.Q0, s.Q1, s.Q2, KQ0, KQ1, KQ2);
    ldl3_solve2(F, s.R0, s.R1, s.R2, KR0, KR1, KR2);
    // state
    s.XY = fma2(KP0, r[0], fma2(KP1, r[1], fma2(KP2, r[2], s.XY)));
    const float2 dZP = fma2(KQ0, r[0], fma2(KQ1, r[1], mul2(KQ2, r[2])));
    const float2 dIT = fma2(KR0, r[0], fma2(KR1, r[1], mul2(KR2, r[2])));
    s.Z += dZP.x;
    s.PH += phi_fix_small(dZP.y);
    s.dph = dZP.y;
    s.IT = add2(s.IT, dIT);
    const float dphi = dZP.y, dth = dIT.y;
    if (fmaxf(fabsf(dphi), fabsf(dth)) < 0.06f) {
        rotate_poly2(s.CC, s.SS, f2(dphi, dth));
    } else {
        float sp, cp, st, ct;
        sincosf(phi_float(s.PH), &sp, &cp);
        sincosf(s.IT.y, &st, &ct);
        s.CC = f2(cp, ct); s.SS = f2(sp, st);
    }
    // momentum block: C_ab -= sum_k K_ak C_bk with the still-intact old columns 0..2
    s.M3 = fma2(neg2(KR0), s.R0.x, fma2(neg2(KR1), s.R1.x, fma2(neg2(KR2), s.R2.x, s.M3)));     // (C33, C53) -= (K3k, K5k) C3k
    s.M4 = fma2(neg2(s.R0), KQ0.y, fma2(neg2(s.R1), KQ1.y, fma2(neg2(s.R2), KQ2.y, s.M4)));     // (C43, C54) -= K4k (C3k, C5k)
    s.C44 = fmaf(-KQ0.y, s.Q0.y, fmaf(-KQ1.y, s.Q1.y, fmaf(-KQ2.y, s.Q2.y, s.C44)));
    s.C55 = fmaf(-KR0.y, s.R0.y, fmaf(-KR1.y, s.R1.y, fmaf(-KR2.y, s.R2.y, s.C55)));
    // columns 0..2: K V
    if (ISO) {
        s.P0 = mul2(KP0, V.xx); s.P1 = mul2(KP1, V.xx);
        s.Q0 = mul2(KQ0, V.xx); s.Q1 = mul2(KQ1, V.xx);
        s.R0 = mul2(KR0, V.xx); s.R1 = mul2(KR1, V.xx);
    } else {
        s.P0 = fma2(KP0, V.xx, mul2(KP1, V.xy)); s.P1 = fma2(KP0, V.xy, mul2(KP1, V.yy));
        s.Q0 = fma2(KQ0, V.xx, mul2(KQ1, V.xy)); s.Q1 = fma2(KQ0, V.xy, mul2(KQ1, V.yy));
        s.R0 = fma2(KR0, V.xx, mul2(KR1, V.xy)); s.R1 = fma2(KR0, V.xy, mul2(KR1, V.yy));
    }
    s.Q2 = mul2(KQ2, V.zz); s.R2 = mul2(KR2, V.zz);
    s.P1.x = s.P0.y;                      // the three duplicates follow the lower triangle
    s.P2 = f2(s.Q0.x, s.Q1.x);
}

// =====================================================================================================================
// "Cylinder with lids" (sec. 4.1; R19-R21): endcap disks, the second propagation step to a hit's own
// surface, the 2-D update on the plane tangent to the hit radius.  Written on a plain packed covariance (21 elements,
// every index a compile-time constant): this path is about coverage of the geometry, not the FP32 roof.
// =====================================================================================================================
struct Dense { float p[6]; float C[21]; };
#define KF_CD(d, i, j) (d).C[pk(i, j)]

__device__ __forceinline__ void to_dense(const State& s, Dense& d) {
    state_store<false>(s, [&](int i, float v) { d.p[i] = v; }, [&](int k, float v) { d.C[k] = v; });
}
__device__ __forceinline__ void cov_from_dense(State& s, const Dense& d) {
    const int ph = s.PH;
    const float2 cc = s.CC, ss = s.SS;
    const float dph = s.dph;
    state_set<true>(s, [&](int i) { return i == 4 ? __int_as_float(ph) : d.p[i]; }, [&](int k) { return d.C[k]; });
    s.CC = cc; s.SS = ss; s.dph = dph;
}

// curvature partials f1(a) = (cos a - sin a / a)/a, f2(a) = (sin a - (1 - cos a)/a)/a from the turning angle itself
__device__ __forceinline__ void curv_partials(float alpha, float sa, float ca, float& f1, float& f2) {
    const float a2 = alpha * alpha;
    if (a2 < 0.25f) {
        f1 = alpha * fmaf(a2, fmaf(a2, fmaf(a2, 1.0f / 45360.0f, -1.0f / 840.0f), 1.0f / 30.0f), -1.0f / 3.0f);
        f2 = fmaf(a2, fmaf(a2, fmaf(a2, fmaf(a2, 1.0f / 403200.0f, -1.0f / 5760.0f), 1.0f / 144.0f), -0.125f), 0.5f);
    } else {
        const float ia = 1.0f / alpha;
        f1 = (ca - sa * ia) * ia;
        f2 = (sa - (1.0f - ca) * ia) * ia;
    }
}

// Transport to the plane z = Z (R19): s = (Z - z) tan(theta); J = fixed-s partials + (dp'/ds)(ds/dp)^T with ds/dz = -tan(theta),
// ds/dtheta = (Z - z)/cos^2(theta); the z' row vanishes.  NEAR: second step to a hit's own z (either direction, no material,
// no guards).  On a non-zero return s is untouched.
template <bool NEAR>
__device__ __noinline__ uint32_t predict_disk(State& s, float cw, const LayerC& ly, float Z) {
    const float cp = s.CC.x, ct = s.CC.y, sp = s.SS.x, st = s.SS.y;
    Dense d;
    to_dense(s, d);
    const float x = d.p[0], y = d.p[1], iota = d.p[3];
    const float w = cw * iota;
    const float dz = Z - d.p[2];
    const float tanth = st / ct;
    const float sT = dz * tanth;
    if (!(fabsf(sT) <= 3.0e38f)) return ST_UNREACHABLE;
    if (!NEAR) {
        if (!(sT > 0.0f) || !(fabsf(w) * sT <= 3.14159265358979f)) return ST_UNREACHABLE;
        if (!(fabsf(ct) >= CMIN)) return ST_GRAZING;
    }
    const float alpha = w * sT;
    float sa, ca;
    sincosf(alpha, &sa, &ca);
    float X, Y;
    if (fabsf(alpha) < 0.02f) {
        const float a2 = alpha * alpha;
        X = sT * fmaf(a2, -1.0f / 6.0f, 1.0f);
        Y = sT * 0.5f * alpha * fmaf(a2, -1.0f / 12.0f, 1.0f);
    } else {
        const float iw = 1.0f / w;
        X = sa * iw;
        Y = (1.0f - ca) * iw;
    }
    const float dx = fmaf(cp, X, -sp * Y), dy = fmaf(sp, X, cp * Y);
    const float cpn = fmaf(cp, ca, -sp * sa), spn = fmaf(sp, ca, cp * sa);
    float f1, f2;
    curv_partials(alpha, sa, ca, f1, f2);
    const float cs2 = cw * sT * sT;
    const float Fxi = cs2 * fmaf(cp, f1, -sp * f2), Fyi = cs2 * fmaf(sp, f1, cp * f2);
    const float sz = -tanth, sth = dz / (ct * ct);
    // rows of J: x' = (1, 0, a2, a3, a4, a5), y' = (0, 1, b2, b3, b4, b5), z' = 0, phi' = (0, 0, d2, d3, 1, d5); 1/pT and theta unit rows
    const float a2_ = cpn * sz, a3 = Fxi, a4 = -dy, a5 = cpn * sth;
    const float b2_ = spn * sz, b3 = Fyi, b4 = dx, b5 = spn * sth;
    const float d2 = w * sz, d3 = cw * sT, d5 = w * sth;
    float T0[6], T1[6], T4[6];
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        T0[k] = fmaf(a2_, KF_CD(d, 2, k), fmaf(a3, KF_CD(d, 3, k), fmaf(a4, KF_CD(d, 4, k), fmaf(a5, KF_CD(d, 5, k), KF_CD(d, 0, k)))));
        T1[k] = fmaf(b2_, KF_CD(d, 2, k), fmaf(b3, KF_CD(d, 3, k), fmaf(b4, KF_CD(d, 4, k), fmaf(b5, KF_CD(d, 5, k), KF_CD(d, 1, k)))));
        T4[k] = fmaf(d2, KF_CD(d, 2, k), fmaf(d3, KF_CD(d, 3, k), fmaf(d5, KF_CD(d, 5, k), KF_CD(d, 4, k))));
    }
    auto colx = [&](const float (&T)[6]) { return fmaf(a2_, T[2], fmaf(a3, T[3], fmaf(a4, T[4], fmaf(a5, T[5], T[0])))); };
    auto coly = [&](const float (&T)[6]) { return fmaf(b2_, T[2], fmaf(b3, T[3], fmaf(b4, T[4], fmaf(b5, T[5], T[1])))); };
    auto colp = [&](const float (&T)[6]) { return fmaf(d2, T[2], fmaf(d3, T[3], fmaf(d5, T[5], T[4]))); };
    Dense n;
    KF_CD(n, 0, 0) = colx(T0);
    KF_CD(n, 1, 0) = colx(T1); KF_CD(n, 1, 1) = coly(T1);
    KF_CD(n, 2, 0) = 0.0f; KF_CD(n, 2, 1) = 0.0f; KF_CD(n, 2, 2) = 0.0f;
    KF_CD(n, 3, 0) = T0[3]; KF_CD(n, 3, 1) = T1[3]; KF_CD(n, 3, 2) = 0.0f; KF_CD(n, 3, 3) = KF_CD(d, 3, 3);
    KF_CD(n, 4, 0) = colx(T4); KF_CD(n, 4, 1) = coly(T4); KF_CD(n, 4, 2) = 0.0f; KF_CD(n, 4, 3) = T4[3]; KF_CD(n, 4, 4) = colp(T4);
    KF_CD(n, 5, 0) = T0[5]; KF_CD(n, 5, 1) = T1[5]; KF_CD(n, 5, 2) = 0.0f; KF_CD(n, 5, 3) = KF_CD(d, 5, 3); KF_CD(n, 5, 4) = T4[5]; KF_CD(n, 5, 5) = KF_CD(d, 5, 5);
    if (!NEAR && ly.xx0 > 0.0f) {      // scattering (R4) with the path through the disk xx0 / |cos theta|
        const float ist = 1.0f / st;
        const float tms = ly.xx0 / fabsf(ct);
        const float lg = fmaf(0.038f, flog(tms), 1.0f);
        const float h = 0.0136f * iota * st * lg;
        const float v = h * h * tms;
        const float icot = iota * ct * ist;
        KF_CD(n, 5, 5) += v;
        KF_CD(n, 4, 4) += v * ist * ist;
        KF_CD(n, 3, 3) += icot * icot * v;
        KF_CD(n, 5, 3) += -icot * v;
    }
    n.p[0] = x + dx; n.p[1] = y + dy; n.p[2] = Z; n.p[3] = iota; n.p[5] = d.p[5];
    s.PH += phi_fix_small(alpha);
    s.CC.x = cpn; s.SS.x = spn;
    cov_from_dense(s, n);
    return 0u;
}

// 2-D update on the plane tangent to the hit radius (R21).  The position block is turned into the hit's own (radial,
// azimuthal, z) frame; a barrel hit measures (azimuthal, z), a disk hit (azimuthal, radial) -- for the disk the radial and
// z coordinates swap places, so that the measured pair is always coordinates (1, 2).  Columns of the measured pair are
// rebuilt as K V (exact, no cancellation; kf_state.cuh gain_update), the rest as C - K (C H^T)^T.
// v1, v2: variances along the azimuth and along z (barrel) / the radius (disk).  false: S not positive definite.
static __device__ __noinline__ bool update_2d(State& s, float mx, float my, float mz, int kind, float v1, float v2, float& chi2) {
    Dense d;
    to_dense(s, d);
    const float irm = rsqrtf(fmaf(mx, mx, my * my));
    const float cn = mx * irm, sn = my * irm;
    // full symmetric matrix in the rotated frame q = (n, t, z): rows / columns 0, 1 turned by the hit's azimuth
    float c[6][6];
#pragma unroll
    for (int i = 0; i < 6; ++i)
#pragma unroll
        for (int j = 0; j < 6; ++j) c[i][j] = KF_CD(d, i, j);
#pragma unroll
    for (int k = 0; k < 6; ++k) {       // rows
        const float a = c[0][k], b = c[1][k];
        c[0][k] = fmaf(cn, a, sn * b); c[1][k] = fmaf(-sn, a, cn * b);
    }
#pragma unroll
    for (int k = 0; k < 6; ++k) {       // columns
        const float a = c[k][0], b = c[k][1];
        c[k][0] = fmaf(cn, a, sn * b); c[k][1] = fmaf(-sn, a, cn * b);
    }
    const float dx = mx - d.p[0], dy = my - d.p[1];
    float rq[3] = {fmaf(cn, dx, sn * dy), fmaf(-sn, dx, cn * dy), mz - d.p[2]};
    if (kind) {                         // disk: swap the radial and the z coordinate
#pragma unroll
        for (int k = 0; k < 6; ++k) { const float t = c[0][k]; c[0][k] = c[2][k]; c[2][k] = t; }
#pragma unroll
        for (int k = 0; k < 6; ++k) { const float t = c[k][0]; c[k][0] = c[k][2]; c[k][2] = t; }
        const float t = rq[0]; rq[0] = rq[2]; rq[2] = t;
    }
    const float S11 = c[1][1] + v1, S12 = c[2][1], S22 = c[2][2] + v2;
    const float det = fmaf(S11, S22, -S12 * S12);
    const bool ok = (S11 > 0.0f) && (det > 0.0f);
    const float idet = 1.0f / det;
    const float r1 = rq[1], r2 = rq[2];
    chi2 = (fmaf(S22 * r1, r1, fmaf(-2.0f * S12 * r1, r2, S11 * r2 * r2))) * idet;
    float K1[6], K2[6], dq[6];
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        K1[i] = fmaf(c[i][1], S22, -c[i][2] * S12) * idet;
        K2[i] = fmaf(-c[i][1], S12, c[i][2] * S11) * idet;
        dq[i] = fmaf(K1[i], r1, K2[i] * r2);
    }
    // covariance: unmeasured block with the old measured columns, measured columns as K V
    constexpr int U[4] = {0, 3, 4, 5};
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b <= a; ++b) {
            const int i = U[a], j = U[b];
            const float v = fmaf(-K1[i], c[j][1], fmaf(-K2[i], c[j][2], c[i][j]));
            c[i][j] = v; c[j][i] = v;
        }
#pragma unroll
    for (int i = 0; i < 6; ++i) { c[i][1] = K1[i] * v1; c[i][2] = K2[i] * v2; }
    c[1][2] = c[2][1];
#pragma unroll
    for (int i = 0; i < 6; ++i) { c[1][i] = c[i][1]; c[2][i] = c[i][2]; }
    if (kind) {
#pragma unroll
        for (int k = 0; k < 6; ++k) { const float t = c[0][k]; c[0][k] = c[2][k]; c[2][k] = t; }
#pragma unroll
        for (int k = 0; k < 6; ++k) { const float t = c[k][0]; c[k][0] = c[k][2]; c[k][2] = t; }
        const float t = dq[0]; dq[0] = dq[2]; dq[2] = t;
    }
    // back to (x, y): q = R x  =>  x = R^T q
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const float a = c[0][k], b = c[1][k];
        c[0][k] = fmaf(cn, a, -sn * b); c[1][k] = fmaf(sn, a, cn * b);
    }
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const float a = c[k][0], b = c[k][1];
        c[k][0] = fmaf(cn, a, -sn * b); c[k][1] = fmaf(sn, a, cn * b);
    }
    Dense n;
#pragma unroll
    for (int i = 0; i < 6; ++i)
#pragma unroll
        for (int j = 0; j <= i; ++j) KF_CD(n, i, j) = c[i][j];
    n.p[0] = d.p[0] + fmaf(cn, dq[0], -sn * dq[1]);
    n.p[1] = d.p[1] + fmaf(sn, dq[0], cn * dq[1]);
    n.p[2] = d.p[2] + dq[2];
    n.p[3] = d.p[3] + dq[3];
    n.p[5] = d.p[5] + dq[5];
    s.PH += phi_fix_small(dq[4]);
    s.dph = dq[4];
    if (fmaxf(fabsf(dq[4]), fabsf(dq[5])) < 0.06f) {
        rotate_poly2(s.CC, s.SS, f2(dq[4], dq[5]));
    } else {
        float sp_, cp_, st_, ct_;
        sincosf(phi_float(s.PH), &sp_, &cp_);
        sincosf(n.p[5], &st_, &ct_);
        s.CC = f2(cp_, ct_); s.SS = f2(sp_, st_);
    }
    cov_from_dense(s, n);
    return ok;
}
#undef KF_CD

}  // namespace kf

// kf_binmath.cuh -- bit-exact bin arithmetic (X1-X3): IEEE fp32 single operations and integer work only.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/kf.h"

namespace kf {

// X1: azimuthal bin from comparisons against the tangent table tab[k] = fl32(tan(2 pi k / n_phi)), k = 0..n_phi/8
// (strictly increasing, tab[0] = 0): no atan2 in the DEFINITION, hence no dependence on a math library -- the bin is
// j = the largest k <= n_phi/8 - 1 with tab[k] <= t.  A two-term fit of atan only supplies the first guess of the search
// (scale = n_phi / (2 pi)); the two correction loops make the result the defined one whatever the guess was.
__device__ __forceinline__ int phi_bin(float x, float y, int n_phi, const float* __restrict__ tab, float scale) {
    const float ax = fabsf(x), ay = fabsf(y);
    const bool swap = ay > ax;
    const float lo = swap ? ax : ay, hi = swap ? ay : ax;
    const float t = hi > 0.0f ? __fdiv_rn(lo, hi) : 0.0f;
    const int m = n_phi >> 3;
    // first guess: atan(t) ~ t (0.9724 - 0.1919 t^2) on [0, 1] (|error| < 0.005 rad: a bin or two; the loops below settle it)
    int j = min(max((int)(t * fmaf(-0.1919f, t * t, 0.9724f) * scale), 0), m - 1);
    while (j > 0 && tab[j] > t) --j;
    while (j + 1 < m && tab[j + 1] <= t) ++j;
    const int a = swap ? (n_phi >> 2) - 1 - j : j;
    if (x >= 0.0f) return (y >= 0.0f) ? a : n_phi - 1 - a;
    return (y >= 0.0f) ? (n_phi >> 1) - 1 - a : (n_phi >> 1) + a;
}

// X2: z row of a barrel layer; inv_dz = fl32(n_z / (2 zmax))
__device__ __forceinline__ int z_bin(float z, float zmax, float inv_dz, int n_z) {
    const float f = floorf(__fmul_rn(__fadd_rn(z, zmax), inv_dz));
    return (f >= (float)n_z) ? n_z - 1 : (f < 0.0f ? 0 : (int)f);
}
// X2 for any layer: row of the coordinate v binned in [lo, hi), inv = fl32(n / fl32(hi - lo)).  Barrel layer: v = z, lo = -zmax (then
// v - lo = z + zmax and hi - lo = 2 zmax: the original X2); disk (R22): v = hit_rho(x, y), lo = rmin, hi = rmax.
__device__ __forceinline__ int row_bin(float v, float lo, float inv, int n) {
    const float f = floorf(__fmul_rn(__fsub_rn(v, lo), inv));
    return (f >= (float)n) ? n - 1 : (f < 0.0f ? 0 : (int)f);
}
// radius of a hit as the disk rows take it: one IEEE rounding per operation
__device__ __forceinline__ float hit_rho(float x, float y) { return __fsqrt_rn(__fadd_rn(__fmul_rn(x, x), __fmul_rn(y, y))); }
// per-layer row constants on the host (the same fp32 operations as the oracle)
inline void host_row_range(const kf_layer& y, int n_z, float* lo, float* inv) {
    const float l = y.kind ? y.rmin : -y.zmax, h = y.zmax;
    *lo = l;
    *inv = (float)n_z / (h - l);
}

// X3: window -> first phi bin, number of phi bins (wrapping), z rows
struct WindowBins { int first, n_b, iz_lo, iz_hi; };

// ROW = false: barrel layer, rows of z (a = zmax, b = inv_dz); ROW = true: any layer, rows of the coordinate binned in
// [lo, hi) (a = lo, b = inv): the same bins for a barrel layer, written with the operations of X2 / of row_bin
template <bool ROW = false>
__device__ __forceinline__ WindowBins window_bins(float phi_c, float dphi, float z_c, float dz, float a, float b,
                                                  float inv_dphi, int n_phi, int n_z) {
    WindowBins w;
    if (!(__fmul_rn(dphi, inv_dphi) < (float)n_phi)) {      // half width of a full turn or more (or not a number): every bin, from bin 0
        w.first = 0; w.n_b = n_phi;
    } else {
        const int b_lo = (int)floorf(__fmul_rn(__fsub_rn(phi_c, dphi), inv_dphi));
        const int b_hi = (int)floorf(__fmul_rn(__fadd_rn(phi_c, dphi), inv_dphi));
        int nb = b_hi - b_lo + 1;
        nb = nb > n_phi ? n_phi : nb;
        w.n_b = nb < 0 ? 0 : nb;
        int f = b_lo % n_phi;
        w.first = f < 0 ? f + n_phi : f;
    }
    w.iz_lo = ROW ? row_bin(__fsub_rn(z_c, dz), a, b, n_z) : z_bin(__fsub_rn(z_c, dz), a, b, n_z);
    w.iz_hi = ROW ? row_bin(__fadd_rn(z_c, dz), a, b, n_z) : z_bin(__fadd_rn(z_c, dz), a, b, n_z);
    return w;
}

// inv_dphi = fl32(n_phi / (2 pi)), the division carried out in double
inline float host_inv_dphi(int n_phi) { return (float)((double)n_phi / 6.283185307179586476925286766559); }

}  // namespace kf

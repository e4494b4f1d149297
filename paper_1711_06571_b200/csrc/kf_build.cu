// kf_build.cu -- combinatorial track building (DESIGN.md sec. 2 steps B1-B6, readings R10, R11, X3).
//
// "Track building projects the track candidate outwards to collect additional hits, using the KF to estimate which
// hits represent the most likely continuation ... branching to explore multiple candidate tracks per seed"
// (sec. 2); "a fixed number of slots for each track seed" (sec. 4.3).
//
// One kernel for all layers.  A group of G lanes (G = 4, 8, 16 or 32, a template parameter) owns one seed; the <= K
// candidates of the seed live in shared memory (33 words each: 6 parameters, 21 packed covariance elements, chi2,
// nhits/status word, carried sin/cos of phi and theta) and never touch HBM between layers.  Per layer:
//   phase 1  lanes loop over the parents: predict (F2-F5), window -> bin ranges (B2), LDL^T factor of S
//   phase 2  the group walks the window runs of every parent with unit-stride lanes over the sorted hits: strict
//            window test + chi2 (B3); passing children are appended to a small buffer that is pruned to the best K
//            (rank by counting inside the group, B4) whenever it fills
//   phase 3  one hit-less / finished child per parent that produced no hit child; final ranking
//   phase 4  lanes loop over the kept children: Kalman update (B5), per-layer link (parent slot, hit)
// At the end the links are traced back into per-candidate hit lists and everything is stored SoA (B6).
#include "kf_common.cuh"
#include "kf_binmath.cuh"

namespace kf {

constexpr int BUILD_BLOCK = 128;
constexpr int NS = 33;          // words per candidate record
constexpr int NW = 20;          // words per parent window record
constexpr int HITPOS_NONE = 0x7fffffff;

// candidate record
enum { R_PAR = 0, R_COV = 6, R_CHI2 = 27, R_META = 28, R_TRIG = 29 };
// meta word: bits 0-7 nhits, bit 8 finished, bits 16-19 status
__device__ __forceinline__ int meta_pack(int nhits, bool fin, uint32_t st) { return nhits | (fin ? 256 : 0) | (int)(st << 16); }
// window record
enum { W_KIND = 0, W_X = 1, W_Y = 2, W_Z = 3, W_THR2 = 4, W_DZ = 5, W_LDL = 6, W_FOK = 12, W_FIRST = 13, W_NB = 14, W_ZLO = 15, W_ZHI = 16,
       W_CHI2 = 17, W_NH = 18, W_SBAD = 19 };
enum { KIND_OPEN = 0, KIND_FIN = 1 };

struct BuildArgs {
    int32_t n_layers, first_layer, K, n_phi, n_z, cap;
    float kb, chi2_cut, n_sigma, inv_dphi;
    int64_t n_seeds, ld_seed, ld_out;
    const float *par, *cov; const int8_t* q;
    const int32_t *seed_event, *seed_hit_idx;
    const float *sx, *sy, *sz; const int32_t *perm, *bin_off;
    float *par_o, *cov_o, *chi2_o; int8_t* q_o; int32_t* nhits_o; uint32_t* status_o; int32_t *hit_idx_o, *n_cand_o;
    LayerC layer[KF_MAX_LAYERS];
    float inv_dz[KF_MAX_LAYERS], sphi_over_r2[KF_MAX_LAYERS];   // n_z/(2 zmax); (sig_rphi/r)^2
};

// words of shared memory per seed
__host__ __device__ inline int seed_words(int K, int L, int cap) {
    return 2 * K * NS + K * NW + L * K + (L * K + 3) / 4 + 2 * 4 * cap;
}

struct Key { float chi2; int nh, parent, hitpos; };
__device__ __forceinline__ bool key_less(const Key& a, const Key& b) {   // a ranks before b (R10)
    if (a.nh != b.nh) return a.nh > b.nh;
    if (a.chi2 != b.chi2) return a.chi2 < b.chi2;
    if (a.parent != b.parent) return a.parent < b.parent;
    return a.hitpos < b.hitpos;
}

template <int G>
__device__ __forceinline__ int group_sum(int v, unsigned gmask) {
#pragma unroll
    for (int d = G / 2; d >= 1; d >>= 1) v += __shfl_xor_sync(gmask, v, d);
    return v;
}

// Keep the best min(K, #valid) entries of src[0..n) in rank order in dst; entries of parents flagged sbad are dropped.
template <int G>
__device__ __forceinline__ int prune(const int* src, int* dst, int n, int cap, int K, const float* W, int lane, unsigned gmask) {
    const float* s_chi2 = (const float*)src;
    const int *s_nh = src + cap, *s_par = src + 2 * cap, *s_hit = src + 3 * cap;
    int nvalid = 0;
    for (int e = lane; e < n; e += G) {
        Key a = {s_chi2[e], s_nh[e], s_par[e], s_hit[e]};
        const bool valid = a.hitpos == HITPOS_NONE || __float_as_int(W[a.parent * NW + W_SBAD]) == 0;
        if (!valid) continue;
        ++nvalid;
        int rank = 0;
        for (int f = 0; f < n; ++f) {
            Key b = {s_chi2[f], s_nh[f], s_par[f], s_hit[f]};
            const bool vb = b.hitpos == HITPOS_NONE || __float_as_int(W[b.parent * NW + W_SBAD]) == 0;
            rank += (vb && key_less(b, a)) ? 1 : 0;
        }
        if (rank < K) {
            ((float*)dst)[rank] = a.chi2; dst[cap + rank] = a.nh; dst[2 * cap + rank] = a.parent; dst[3 * cap + rank] = a.hitpos;
        }
    }
    nvalid = group_sum<G>(nvalid, gmask);
    __syncwarp(gmask);
    return nvalid < K ? nvalid : K;
}

template <int G>
__global__ void __launch_bounds__(BUILD_BLOCK) kf_build_kernel(const __grid_constant__ BuildArgs a) {
    extern __shared__ float smem[];
    const int lane = threadIdx.x % G;
    const int grp = threadIdx.x / G;
    const unsigned gmask = (G == 32) ? 0xffffffffu : (((1u << G) - 1u) << ((threadIdx.x & 31) / G * G));
    const int64_t s = (int64_t)blockIdx.x * (BUILD_BLOCK / G) + grp;
    if (s >= a.n_seeds) return;          // whole group leaves together
    const int K = a.K, L = a.n_layers, cap = a.cap;
    float* A = smem + (size_t)grp * seed_words(K, L, cap);
    float* B = A + K * NS;
    float* W = B + K * NS;
    int* link_hit = (int*)(W + K * NW);
    unsigned char* link_par = (unsigned char*)(link_hit + L * K);
    int* buf0 = link_hit + L * K + (L * K + 3) / 4;
    int* buf1 = buf0 + 4 * cap;

    const float cw = -(float)a.q[s] * a.kb;
    const int ev = a.seed_event ? a.seed_event[s] : 0;
    // seed -> slot 0
    for (int i = lane; i < 27; i += G) A[i] = (i < 6) ? a.par[(int64_t)i * a.ld_seed + s] : a.cov[(int64_t)(i - 6) * a.ld_seed + s];
    __syncwarp(gmask);
    if (lane == 0) {
        Trig g;
        trig_init(g, A[R_PAR + 4], A[R_PAR + 5]);
        A[R_CHI2] = 0.0f;
        A[R_META] = __int_as_float(meta_pack(a.first_layer, false, 0u));
        A[R_TRIG] = g.cp; A[R_TRIG + 1] = g.sp; A[R_TRIG + 2] = g.st; A[R_TRIG + 3] = g.ct;
    }
    __syncwarp(gmask);
    int nc = 1;

    for (int l = a.first_layer; l < L; ++l) {
        const LayerC& ly = a.layer[l];
        const bool iso = ly.var_r == ly.var_rphi;
        const int64_t seg = (int64_t)ev * L + l;
        // ---------------- phase 1: predict + window ----------------
        for (int c = lane; c < nc; c += G) {
            const float* rec = A + c * NS;
            float* out = B + c * NS;
            float* w = W + c * NW;
            float p[6], C[21];
#pragma unroll
            for (int i = 0; i < 6; ++i) p[i] = rec[R_PAR + i];
#pragma unroll
            for (int i = 0; i < 21; ++i) C[i] = rec[R_COV + i];
            Trig g = {rec[R_TRIG], rec[R_TRIG + 1], rec[R_TRIG + 2], rec[R_TRIG + 3]};
            const int meta = __float_as_int(rec[R_META]);
            uint32_t flag = 0u;
            bool fin = (meta & 256) != 0;
            float thr2 = 0.f, dzw = 0.f;
            Ldl3 F = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
            bool fok = false;
            WindowBins wb = {0, 0, 0, -1};
            if (!fin) {
                flag = predict(p, C, g, cw, ly);
                if (!flag) {
                    const float x = p[0], y = p[1];
                    const float r2 = fmaf(x, x, y * y);
                    const float num = fmaf(x * x, C[pk(1, 1)], fmaf(-2.0f * x * y, C[pk(1, 0)], y * y * C[pk(0, 0)]));
                    const float varphi = fmaxf(num / (r2 * r2), 0.0f);
                    const float dphi = a.n_sigma * sqrtf(varphi + a.sphi_over_r2[l]);
                    dzw = a.n_sigma * sqrtf(C[pk(2, 2)] + ly.var_z);
                    if (!(dphi <= 3.0e38f) || !(dzw <= 3.0e38f)) flag = ST_NUMERIC;      // NaN or Inf
                    else if (fabsf(p[2]) > ly.zmax + dzw) flag = ST_LEFT_Z;
                    else {
                        thr2 = dphi * dphi * r2;
                        wb = window_bins(atan2f(y, x), dphi, p[2], dzw, ly.zmax, a.inv_dz[l], a.inv_dphi, a.n_phi, a.n_z);
                        if (iso) {
                            Sym3 S;
                            S.m00 = C[pk(0, 0)] + ly.var_r; S.m10 = C[pk(1, 0)]; S.m11 = C[pk(1, 1)] + ly.var_r;
                            S.m20 = C[pk(2, 0)]; S.m21 = C[pk(2, 1)]; S.m22 = C[pk(2, 2)] + ly.var_z;
                            fok = ldl3(S, F);
                        }
                    }
                }
                fin = flag != 0u;
            }
            if (fin) {   // finished now or before: the child inherits the unchanged state
#pragma unroll
                for (int i = 0; i < NS; ++i) out[i] = rec[i];
                w[W_KIND] = __int_as_float(KIND_FIN | (int)(flag << 8));
            } else {
#pragma unroll
                for (int i = 0; i < 6; ++i) out[R_PAR + i] = p[i];
#pragma unroll
                for (int i = 0; i < 21; ++i) out[R_COV + i] = C[i];
                out[R_CHI2] = rec[R_CHI2]; out[R_META] = rec[R_META];
                out[R_TRIG] = g.cp; out[R_TRIG + 1] = g.sp; out[R_TRIG + 2] = g.st; out[R_TRIG + 3] = g.ct;
                w[W_KIND] = __int_as_float(KIND_OPEN);
                w[W_X] = p[0]; w[W_Y] = p[1]; w[W_Z] = p[2]; w[W_THR2] = thr2; w[W_DZ] = dzw;
                w[W_LDL] = F.l10; w[W_LDL + 1] = F.l20; w[W_LDL + 2] = F.l21; w[W_LDL + 3] = F.i0; w[W_LDL + 4] = F.i1; w[W_LDL + 5] = F.i2;
                w[W_FOK] = __int_as_float(fok ? 1 : 0);
                w[W_FIRST] = __int_as_float(wb.first); w[W_NB] = __int_as_float(wb.n_b);
                w[W_ZLO] = __int_as_float(wb.iz_lo); w[W_ZHI] = __int_as_float(wb.iz_hi);
            }
            w[W_CHI2] = rec[R_CHI2];
            w[W_NH] = __int_as_float(meta & 255);
            w[W_SBAD] = __int_as_float(0);
        }
        __syncwarp(gmask);
        // ---------------- phase 2: window scan ----------------
        int* buf = buf0;
        int* alt = buf1;
        int n_buf = 0;
        unsigned has_child = 0u;
        for (int c = 0; c < nc; ++c) {
            const float* w = W + c * NW;
            if ((__float_as_int(w[W_KIND]) & 255) != KIND_OPEN) continue;
            const float px = w[W_X], py = w[W_Y], pz = w[W_Z], thr2 = w[W_THR2], dzw = w[W_DZ];
            Ldl3 F = {w[W_LDL], w[W_LDL + 1], w[W_LDL + 2], w[W_LDL + 3], w[W_LDL + 4], w[W_LDL + 5]};
            const bool fok = __float_as_int(w[W_FOK]) != 0;
            const int first = __float_as_int(w[W_FIRST]), nb = __float_as_int(w[W_NB]);
            const int zlo = __float_as_int(w[W_ZLO]), zhi = __float_as_int(w[W_ZHI]);
            const float chi2_par = w[W_CHI2];
            const int nh_child = __float_as_int(w[W_NH]) + 1;
            const float* Bc = B + c * NS;
            for (int iz = zlo; iz <= zhi; ++iz) {
                const int64_t row = (seg * a.n_z + iz) * a.n_phi;
                for (int run = 0; run < 2; ++run) {
                    int b0, b1;
                    if (run == 0) { b0 = first; b1 = min(first + nb, a.n_phi); }
                    else { b0 = 0; b1 = first + nb - a.n_phi; }
                    if (b1 <= b0) continue;
                    const int h0 = a.bin_off[row + b0], h1 = a.bin_off[row + b1];
                    for (int hb = h0; hb < h1; hb += G) {
                        const int h = hb + lane;
                        bool pass = false;
                        float c2 = 0.f;
                        if (h < h1) {
                            const float mx = a.sx[h], my = a.sy[h], mz = a.sz[h];
                            const float cr = fmaf(px, my, -py * mx);
                            const bool in_win = (cr * cr <= thr2 * fmaf(mx, mx, my * my)) && (fmaf(px, mx, py * my) > 0.0f) && (fabsf(mz - pz) <= dzw);
                            if (in_win) {
                                bool ok = fok;
                                if (!iso) {
                                    const HitCov V = hit_cov(mx, my, ly);
                                    Sym3 S;
                                    S.m00 = Bc[R_COV + 0] + V.xx; S.m10 = Bc[R_COV + 1] + V.xy; S.m11 = Bc[R_COV + 2] + V.yy;
                                    S.m20 = Bc[R_COV + 3]; S.m21 = Bc[R_COV + 4]; S.m22 = Bc[R_COV + 5] + V.zz;
                                    ok = ldl3(S, F);
                                }
                                if (!ok) W[c * NW + W_SBAD] = __int_as_float(1);
                                else {
                                    const float r0 = mx - px, r1 = my - py, r2 = mz - pz;
                                    const float y1 = fmaf(-F.l10, r0, r1);
                                    const float y2 = fmaf(-F.l21, y1, fmaf(-F.l20, r0, r2));
                                    c2 = fmaf(r0 * r0, F.i0, fmaf(y1 * y1, F.i1, y2 * y2 * F.i2));
                                    pass = c2 < a.chi2_cut;
                                }
                            }
                        }
                        const unsigned m = __ballot_sync(gmask, pass);
                        if (m) {
                            const int n_new = __popc(m);
                            if (n_buf + n_new > cap) {
                                __syncwarp(gmask);
                                n_buf = prune<G>(buf, alt, n_buf, cap, K, W, lane, gmask);
                                int* t = buf; buf = alt; alt = t;
                            }
                            if (pass) {
                                const int idx = n_buf + __popc(m & ((1u << (threadIdx.x & 31)) - 1u));
                                ((float*)buf)[idx] = chi2_par + c2; buf[cap + idx] = nh_child; buf[2 * cap + idx] = c; buf[3 * cap + idx] = h;
                            }
                            n_buf += n_new;
                            has_child |= 1u << c;
                        }
                    }
                }
            }
        }
        __syncwarp(gmask);
        // ---------------- phase 3: hit-less / finished children, final ranking ----------------
        for (int c = 0; c < nc; ++c) {
            const float* w = W + c * NW;
            const bool open = (__float_as_int(w[W_KIND]) & 255) == KIND_OPEN;
            const bool sbad = __float_as_int(w[W_SBAD]) != 0;
            if (open && !sbad && ((has_child >> c) & 1u)) continue;
            if (open && sbad)      // S not positive definite: the finished child inherits the unchanged state, not the prediction
                for (int i = lane; i < NS; i += G) B[c * NS + i] = A[c * NS + i];
            if (n_buf + 1 > cap) {
                __syncwarp(gmask);
                n_buf = prune<G>(buf, alt, n_buf, cap, K, W, lane, gmask);
                int* t = buf; buf = alt; alt = t;
            }
            if (lane == 0) {
                ((float*)buf)[n_buf] = w[W_CHI2]; buf[cap + n_buf] = __float_as_int(w[W_NH]); buf[2 * cap + n_buf] = c; buf[3 * cap + n_buf] = HITPOS_NONE;
            }
            ++n_buf;
        }
        __syncwarp(gmask);
        const int n_new = prune<G>(buf, alt, n_buf, cap, K, W, lane, gmask);
        const int* sel = alt;
        // ---------------- phase 4: update the survivors ----------------
        for (int j = lane; j < n_new; j += G) {
            const int parent = sel[2 * cap + j], hitpos = sel[3 * cap + j];
            const float* rec = B + parent * NS;
            const float* w = W + parent * NW;
            float* out = A + j * NS;
            int meta = __float_as_int(rec[R_META]);
            int link;
            if (hitpos == HITPOS_NONE) {
                const int kind = __float_as_int(w[W_KIND]);
                const bool sbad = __float_as_int(w[W_SBAD]) != 0;
#pragma unroll
                for (int i = 0; i < NS; ++i) out[i] = rec[i];
                if ((kind & 255) == KIND_FIN || sbad) {
                    meta |= 256 | (int)(((uint32_t)(kind >> 8) | (sbad ? ST_NUMERIC : 0u)) << 16);
                    out[R_META] = __int_as_float(meta);
                    link = -2;
                } else {
                    link = -1;
                }
            } else {
                float p[6], C[21];
#pragma unroll
                for (int i = 0; i < 6; ++i) p[i] = rec[R_PAR + i];
#pragma unroll
                for (int i = 0; i < 21; ++i) C[i] = rec[R_COV + i];
                Trig g = {rec[R_TRIG], rec[R_TRIG + 1], rec[R_TRIG + 2], rec[R_TRIG + 3]};
                const float mx = a.sx[hitpos], my = a.sy[hitpos], mz = a.sz[hitpos];
                const HitCov V = hit_cov(mx, my, ly);
                Ldl3 F;
                float r[3], c2;
                bool ok = innovation(p, C, mx, my, mz, V, F, r, c2);
                if (ok) {
                    gain_update(p, C, g, F, V, r);
                    ok = all_finite(p, C) && p[3] > 0.0f;
                }
                const int nh = sel[cap + j];
                if (ok) {
#pragma unroll
                    for (int i = 0; i < 6; ++i) out[R_PAR + i] = p[i];
#pragma unroll
                    for (int i = 0; i < 21; ++i) out[R_COV + i] = C[i];
                    out[R_TRIG] = g.cp; out[R_TRIG + 1] = g.sp; out[R_TRIG + 2] = g.st; out[R_TRIG + 3] = g.ct;
                    meta = (meta & ~255) | nh;
                } else {     // failed update: keep the predicted state, finish the candidate
#pragma unroll
                    for (int i = 0; i < NS; ++i) out[i] = rec[i];
                    meta = ((meta & ~255) | nh) | 256 | (int)(ST_NUMERIC << 16);
                }
                out[R_CHI2] = ((const float*)sel)[j];
                out[R_META] = __int_as_float(meta);
                link = a.perm[hitpos];
            }
            link_hit[l * K + j] = link;
            link_par[l * K + j] = (unsigned char)parent;
        }
        nc = n_new;
        __syncwarp(gmask);
    }

    // ---------------- B6: back-trace + store ----------------
    if (lane == 0) a.n_cand_o[s] = nc;
    for (int j = lane; j < K; j += G) {
        const int64_t slot = s * K + j;
        a.q_o[slot] = a.q[s];
        if (j < nc) {
            const float* rec = A + j * NS;
#pragma unroll
            for (int i = 0; i < 6; ++i) a.par_o[(int64_t)i * a.ld_out + slot] = (i == 4) ? wrap_phi(rec[R_PAR + i]) : rec[R_PAR + i];
#pragma unroll
            for (int i = 0; i < 21; ++i) a.cov_o[(int64_t)i * a.ld_out + slot] = rec[R_COV + i];
            const int meta = __float_as_int(rec[R_META]);
            a.chi2_o[slot] = rec[R_CHI2];
            a.nhits_o[slot] = meta & 255;
            a.status_o[slot] = (uint32_t)(meta >> 16) & 15u;
            int k = j;
            for (int l = L - 1; l >= a.first_layer; --l) {
                a.hit_idx_o[(int64_t)l * a.ld_out + slot] = link_hit[l * K + k];
                k = link_par[l * K + k];
            }
            for (int l = 0; l < a.first_layer; ++l)
                a.hit_idx_o[(int64_t)l * a.ld_out + slot] = a.seed_hit_idx ? a.seed_hit_idx[(int64_t)l * a.ld_seed + s] : -1;
        } else {
            a.chi2_o[slot] = 0.0f; a.nhits_o[slot] = 0; a.status_o[slot] = 0u;
            for (int l = 0; l < L; ++l) a.hit_idx_o[(int64_t)l * a.ld_out + slot] = -2;
        }
    }
}

template <int G>
static int launch_build(const BuildArgs& a, cudaStream_t st) {
    const int seeds_per_block = BUILD_BLOCK / G;
    const size_t smem = (size_t)seeds_per_block * seed_words(a.K, a.n_layers, a.cap) * sizeof(float);
    if (smem > 227 * 1024) return fail(KF_ERR_INVALID_ARG, "kf_build: K = %d needs %zu bytes of shared memory per block (> 227 KB)", a.K, smem);
    cudaError_t e = cudaFuncSetAttribute(kf_build_kernel<G>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return fail(KF_ERR_CUDA, "kf_build: cudaFuncSetAttribute: %s", cudaGetErrorString(e));
    const int64_t blocks = (a.n_seeds + seeds_per_block - 1) / seeds_per_block;
    kf_build_kernel<G><<<(unsigned)blocks, BUILD_BLOCK, smem, st>>>(a);
    return check_launch("kf_build");
}

static int g_build_lanes = 0;   // 0 = automatic

}  // namespace kf

extern "C" size_t kf_build_workspace_bytes(const kf_geom*, int64_t, int32_t) { return 0; }   // candidates stay in shared memory

// tuning / test hook: lanes per seed (4, 8, 16, 32; 0 = automatic)
extern "C" int kf_build_set_lanes(int32_t g) {
    if (g != 0 && g != 4 && g != 8 && g != 16 && g != 32) return kf::fail(KF_ERR_INVALID_ARG, "kf_build_set_lanes: %d not in {0, 4, 8, 16, 32}", g);
    kf::g_build_lanes = g;
    return KF_OK;
}

extern "C" int kf_build(const kf_geom* geom, const kf_hits* hits, const kf_binned* binned, const kf_tracks* seeds,
                        const int32_t* seed_event, const int32_t* seed_hit_idx, int32_t first_layer, int32_t K, float chi2_cut,
                        float n_sigma, kf_cands* out, void* ws, size_t ws_bytes, void* stream) {
    using namespace kf;
    (void)ws; (void)ws_bytes;
    if (!geom || !hits || !binned || !seeds || !out) return fail(KF_ERR_NULL_PTR, "kf_build: NULL struct argument");
    int rc = check_geom(geom, "kf_build");
    if (rc) return rc;
    if (K < 1 || K > 32) return fail(KF_ERR_INVALID_ARG, "kf_build: K = %d outside 1..32", K);
    if (first_layer < 0 || first_layer > geom->n_layers) return fail(KF_ERR_INVALID_ARG, "kf_build: first_layer outside 0..n_layers");
    if (!(chi2_cut > 0.f) || !(n_sigma > 0.f)) return fail(KF_ERR_INVALID_ARG, "kf_build: chi2_cut and n_sigma must be positive");
    if (seeds->n < 0 || seeds->ld < seeds->n) return fail(KF_ERR_INVALID_ARG, "kf_build: need 0 <= n <= ld for the seeds");
    if (out->ld < seeds->n * K || out->cand.ld != out->ld) return fail(KF_ERR_INVALID_ARG, "kf_build: out->ld must be >= n_seeds*K and equal cand.ld");
    if (binned->n_phi < 8 || (binned->n_phi % 8) || binned->n_z < 1) return fail(KF_ERR_BAD_GEOM, "kf_build: bad bin counts");
    out->K = K; out->n_layers = geom->n_layers; out->n_seeds = seeds->n; out->cand.n = seeds->n * K;
    if (seeds->n == 0) return KF_OK;
    if (!seeds->par || !seeds->cov || !seeds->q) return fail(KF_ERR_NULL_PTR, "kf_build: NULL seed array");
    if (!binned->x || !binned->y || !binned->z || !binned->perm || !binned->bin_off) return fail(KF_ERR_NULL_PTR, "kf_build: NULL binned array");
    if (hits->n_events > 1 && !seed_event) return fail(KF_ERR_NULL_PTR, "kf_build: seed_event is NULL with n_events > 1");
    const kf_tracks& c = out->cand;
    if (!c.par || !c.cov || !c.q || !c.chi2 || !c.nhits || !c.status || !out->hit_idx || !out->n_cand)
        return fail(KF_ERR_NULL_PTR, "kf_build: NULL output array");
    BuildArgs a;
    a.n_layers = geom->n_layers; a.first_layer = first_layer; a.K = K; a.n_phi = binned->n_phi; a.n_z = binned->n_z;
    a.kb = KCURV * geom->bz_tesla; a.chi2_cut = chi2_cut; a.n_sigma = n_sigma; a.inv_dphi = host_inv_dphi(binned->n_phi);
    a.n_seeds = seeds->n; a.ld_seed = seeds->ld; a.ld_out = out->ld;
    a.par = seeds->par; a.cov = seeds->cov; a.q = seeds->q; a.seed_event = seed_event; a.seed_hit_idx = seed_hit_idx;
    a.sx = binned->x; a.sy = binned->y; a.sz = binned->z; a.perm = binned->perm; a.bin_off = binned->bin_off;
    a.par_o = c.par; a.cov_o = c.cov; a.chi2_o = c.chi2; a.q_o = c.q; a.nhits_o = c.nhits; a.status_o = c.status;
    a.hit_idx_o = out->hit_idx; a.n_cand_o = out->n_cand;
    for (int l = 0; l < KF_MAX_LAYERS; ++l) {
        const kf_layer& y = geom->layers[l < geom->n_layers ? l : geom->n_layers - 1];
        a.layer[l] = make_layer(y);
        a.inv_dz[l] = (float)binned->n_z / (2.0f * y.zmax);
        a.sphi_over_r2[l] = (y.sig_rphi / y.r) * (y.sig_rphi / y.r);
    }
    int G = g_build_lanes ? g_build_lanes : 8;
    a.cap = K + G > 32 ? K + G : 32;
    cudaStream_t st = (cudaStream_t)stream;
    switch (G) {
        case 4: return launch_build<4>(a, st);
        case 8: return launch_build<8>(a, st);
        case 16: return launch_build<16>(a, st);
        default: return launch_build<32>(a, st);
    }
}

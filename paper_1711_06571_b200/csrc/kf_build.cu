// kf_build.cu -- combinatorial track building (DESIGN.md sec. 2 steps B1-B6, readings R10, R11, X3).
//
// "Track building projects the track candidate outwards to collect additional hits, using the KF to estimate which
// hits represent the most likely continuation ... branching to explore multiple candidate tracks per seed"
// (sec. 2); "a fixed number of slots for each track seed" (sec. 4.3).
//
// One kernel for all layers.  A block of 64-256 threads owns a tile of S seeds (32 or 128) and walks the layers with
// block-level phases; inside every phase one THREAD owns one live candidate, one seed or one child, so the long
// dependent chains of the Kalman arithmetic run at full lane occupancy however few candidates a seed has:
//   phase 1  thread per live candidate (build_candidate): predict (F2-F5), window -> bin ranges (B2), LDL^T factor
//            of S, then the window scan (B3): strict window test + chi2 per 16-byte hit record, the passing hits
//            appended to the candidate's own list (shared memory; best K kept, sorted once the scan is over)
//   phase 2  thread per seed: K-way merge of the lists of its <= K parents over 48-bit keys whose integer order is
//            the total order R10 -> the best K children (B4); block scan of the child counts -> dense child positions
//   phase 3  thread per surviving child (build_child): Kalman update (B5), per-layer link (parent slot, hit)
// Candidate records (33 words: 6 parameters -- phi as a fixed-point angle --, 21 packed covariance elements, carried
// sin/cos, chi2, meta; stored as 9 groups of four) live in a block-private global workspace that stays L2-resident:
// record c of the current layer at a DENSE index (seed offset + slot), group-of-four-major over the index, so every
// record moves with 9 coalesced 16-byte accesses.  Two buffers: A (updated states) and B (predicted states).  When the
// tile has more live candidates than the list area holds, the seeds are taken in rounds.  At the end the links are
// traced back into hit lists and stored SoA, one thread per live candidate (B6).  The three per-thread bodies are
// separate (not inlined) functions: inlined they need 228 registers and spill 480 bytes at the 128 the launch bounds
// allow.  All warps of a block run the same phase at the same time, which also keeps them in the same ~30 KB of code:
// a warp-per-tile variant without block barriers (every warp in its own phase) spent a third of its issue slots waiting
// for instructions (32 KB L1.5 instruction cache; profiles/r03_build.md).
// Geometries with endcap disks and / or kf_geom.hit_mode = 1 (R22, R23) run the LIDS instantiation: window in (phi,
// radius) on a disk, layers that are not crossed skipped, second propagation step + 2-D chi2 / update per candidate hit.
// The barrel-only instantiation keeps its own source text (if constexpr, not shared expressions): the kernel is sensitive
// to instruction scheduling, and the shared form cost it 8.5 % at an identical instruction count (profiles/r03_build.md).
#include <algorithm>
#include "kf_common.cuh"
#include "kf_state.cuh"
#include "kf_binmath.cuh"

namespace kf {

#ifndef KF_BUILD_TPS
#define KF_BUILD_TPS 2     // threads per seed of the tile
#endif
constexpr int BUILD_MAX_NT = 256;         // threads per block: 64, 128 or 256 (KF_BUILD_TPS x the seeds of the tile)
#ifndef KF_BUILD_TPSM
#define KF_BUILD_TPSM 512
#endif
constexpr int BUILD_THREADS_PER_SM = KF_BUILD_TPSM; // 512: 128 registers per thread
constexpr int NREC = 33;                  // words per candidate record
#ifndef KF_TILE_WAVE
#define KF_TILE_WAVE 128   // seeds per block when the whole job is one wave of such blocks
#endif
#ifndef KF_TILE_SMALL
#define KF_TILE_SMALL 32   // seeds per block otherwise
#endif
#ifndef KF_SCAN_BATCH
#define KF_SCAN_BATCH 4
#endif
constexpr int SCAN_BATCH = KF_SCAN_BATCH;  // hits requested together in the window scan
constexpr int HITPOS_NONE = 0x7fffffff;
#ifndef KF_LIST_BYTES
#define KF_LIST_BYTES 192
#endif
constexpr int LIST_BYTES_PER_THREAD = KF_LIST_BYTES; // shared memory for the per-candidate child lists, per thread of the block
enum { W_TRIG = 27, W_CHI2 = 31, W_META = 32 };
// meta word of a record: bits 0-7 nhits, bit 8 finished, bits 16-19 status
// info word of a parent in a round: bits 0-7 nhits, bit 8 finished (child inherits the unchanged state), bit 9 layer skipped
// (the same, but the candidate lives on: R22), bits 16-19 status to add

struct BuildArgs {
    int32_t n_layers, first_layer, K, n_phi, n_z, S, ncap;
    float kb, chi2_cut, n_sigma, inv_dphi;
    int64_t n_seeds, ld_seed, ld_out, n_tiles;
    const float *par, *cov, *chi2_in; const int8_t* q;
    const int32_t *seed_event, *seed_hit_idx;
    const float4* xyzp; const int32_t* bin_off;
    float *par_o, *cov_o, *chi2_o; int8_t* q_o; int32_t* nhits_o; uint32_t* status_o; int32_t *hit_idx_o, *n_cand_o;
    float* ws_rec;            // [grid][2][NREC4][S*K] float4
    int32_t* ws_link_hit;     // [grid][n_layers][S*K]
    LayerC layer[KF_MAX_LAYERS];
    float inv_dz[KF_MAX_LAYERS], sphi_over_r2[KF_MAX_LAYERS];   // n_z/(2 zmax) (disk: n_z/(rmax - rmin)); (sig_rphi/r)^2
    float row_lo[KF_MAX_LAYERS];   // X2 rows of any layer start at -zmax (disk: rmin)
    int32_t lids, hit_mode;   // the geometry has disks (R22); two-step propagation and 2-D update per candidate hit (R23)
};

// Records are stored as NREC4 = 9 groups of four words, group g of record c at float4 index g * SK + c: a record moves
// with 9 coalesced 16-byte accesses per thread.  buf points at group 0 of the buffer.
constexpr int NREC4 = (NREC + 3) / 4;

__device__ __forceinline__ void rec_load(State& s, float& chi2, int& meta, const float* __restrict__ buf, int SK, int c) {
    float v[4 * NREC4];
    const float4* __restrict__ b4 = reinterpret_cast<const float4*>(buf);
#pragma unroll
    for (int g = 0; g < NREC4; ++g) {                                   // all requests in flight together
        const float4 t = __ldcg(b4 + g * SK + c);
        v[4 * g] = t.x; v[4 * g + 1] = t.y; v[4 * g + 2] = t.z; v[4 * g + 3] = t.w;
    }
    state_set<true>(s, [&](int i) { return v[i]; }, [&](int k) { return v[6 + k]; });
    s.CC = f2(v[W_TRIG + 0], v[W_TRIG + 2]);
    s.SS = f2(v[W_TRIG + 1], v[W_TRIG + 3]);
    chi2 = v[W_CHI2];
    meta = __float_as_int(v[W_META]);
}

__device__ __forceinline__ void rec_store(const State& s, float chi2, int meta, float* __restrict__ buf, int SK, int c) {
    float v[4 * NREC4];
    state_store<false>(s, [&](int i, float x) { v[i] = x; }, [&](int k, float x) { v[6 + k] = x; });
    v[W_TRIG + 0] = s.CC.x; v[W_TRIG + 1] = s.SS.x; v[W_TRIG + 2] = s.CC.y; v[W_TRIG + 3] = s.SS.y;
    v[W_CHI2] = chi2; v[W_META] = __int_as_float(meta);
    v[33] = 0.0f; v[34] = 0.0f; v[35] = 0.0f;
    float4* __restrict__ b4 = reinterpret_cast<float4*>(buf);
#pragma unroll
    for (int g = 0; g < NREC4; ++g) __stcg(b4 + g * SK + c, make_float4(v[4 * g], v[4 * g + 1], v[4 * g + 2], v[4 * g + 3]));
}

// one word of a record
__device__ __forceinline__ float rec_word(const float* buf, int SK, int c, int w) { return __ldcg(buf + ((w >> 2) * SK + c) * 4 + (w & 3)); }
__device__ __forceinline__ void rec_set_word(float* buf, int SK, int c, int w, float x) { __stcg(buf + ((w >> 2) * SK + c) * 4 + (w & 3), x); }

// src and dst never overlap (different buffers): all loads are issued before the stores
__device__ __forceinline__ void rec_copy(const float* __restrict__ src, int cs, float* __restrict__ dst, int cd, int SK) {
    const float4* __restrict__ s4 = reinterpret_cast<const float4*>(src);
    float4* __restrict__ d4 = reinterpret_cast<float4*>(dst);
    float4 v[NREC4];
#pragma unroll
    for (int g = 0; g < NREC4; ++g) v[g] = __ldcg(s4 + g * SK + cs);
#pragma unroll
    for (int g = 0; g < NREC4; ++g) __stcg(d4 + g * SK + cd, v[g]);
}

// Child list of a candidate: at most K entries (chi2, hit), entry j of candidate i at [j * ncap + i] (conflict-free).
// During the scan entries are appended unsorted; a full list (more than K compatible hits: rare) keeps the best K by
// replacing its worst entry; list_sort orders it ascending by (chi2, hit) once the scan is over.
__device__ __noinline__ void list_replace_worst(float* lc, int* lh, int ncap, int K, float c, int h) {
    int w = 0;
    float cw = lc[0]; int hw = lh[0];
    for (int j = 1; j < K; ++j) {
        const float cj = lc[j * ncap]; const int hj = lh[j * ncap];
        if (cj > cw || (cj == cw && hj > hw)) { w = j; cw = cj; hw = hj; }
    }
    if (c < cw || (c == cw && h < hw)) { lc[w * ncap] = c; lh[w * ncap] = h; }
}

__device__ __forceinline__ void list_sort(float* lc, int* lh, int ncap, int n) {
    for (int a = 1; a < n; ++a) {
        const float c = lc[a * ncap]; const int h = lh[a * ncap];
        int pos = a;
        while (pos > 0) {
            const float cp = lc[(pos - 1) * ncap]; const int hp = lh[(pos - 1) * ncap];
            if (!(c < cp || (c == cp && h < hp))) break;
            lc[pos * ncap] = cp; lh[pos * ncap] = hp;
            --pos;
        }
        lc[pos * ncap] = c; lh[pos * ncap] = h;
    }
}

__device__ __forceinline__ unsigned long long child_key(int nh, float chi2, int k, int j) {
    return ((unsigned long long)(63 - nh) << 42) | ((unsigned long long)__float_as_uint(chi2) << 10) | (unsigned long long)((k << 5) | j);
}

// exclusive scan of one int per thread over the block (NT threads); returns the exclusive prefix, total in *total
template <int NT>
__device__ __forceinline__ int block_exclusive_scan(int v, int* s_warp, int* total) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int o = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += o;
    }
    if (lane == 31) s_warp[w] = inc;
    __syncthreads();
    if (w == 0) {
        int t = lane < NT / 32 ? s_warp[lane] : 0;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int o = __shfl_up_sync(0xffffffffu, t, d);
            if (lane >= d) t += o;
        }
        s_warp[lane] = t;
    }
    __syncthreads();
    const int base = w > 0 ? s_warp[w - 1] : 0;
    *total = s_warp[NT / 32 - 1];
    __syncthreads();
    return base + inc - v;
}

// shared memory carve-up (bytes), identical on host and device
struct BuildSmem { int nc, off, nnew, offn, sel_chi2, sel_hit, sel_pk, cseed, l_chi2, l_hit, l_cnt, l_head, p_chi2, p_info, link_par, misc, total; };
__host__ __device__ inline BuildSmem build_smem(int S, int K, int ncap, int L) {
    BuildSmem m;
    int o = 0;
    auto take = [&](int bytes) { const int at = o; o += (bytes + 15) & ~15; return at; };
    m.nc = take(4 * S); m.off = take(4 * (S + 1)); m.nnew = take(4 * S); m.offn = take(4 * (S + 1));
    m.sel_chi2 = take(4 * S * K); m.sel_hit = take(4 * S * K); m.sel_pk = take(4 * S * K); m.cseed = take(2 * S * K);
    m.l_chi2 = take(4 * ncap * K); m.l_hit = take(4 * ncap * K); m.l_cnt = take(ncap); m.l_head = take(8 * ncap);
    m.p_chi2 = take(4 * ncap); m.p_info = take(4 * ncap);
    m.link_par = take(L * S * K);
    m.misc = take(4 * 40);
    m.total = o;
    return m;
}

// per-block context: sizes and workspace.  Re-derived inside every phase body from the kernel arguments (constant bank)
// and the block index: passed by reference it would live in local memory, whose loads miss the small L1 left beside the
// shared-memory carve-out.
struct Tile {
    int S, K, L, ncap, SK;
    float *recA, *recB; int32_t* link_hit;
};
__device__ __forceinline__ Tile tile_of(const BuildArgs& a) {
    Tile T;
    T.S = a.S; T.K = a.K; T.L = a.n_layers; T.ncap = a.ncap; T.SK = a.S * a.K;
    T.recA = a.ws_rec + (size_t)blockIdx.x * 2 * (4 * NREC4) * T.SK;
    T.recB = T.recA + (size_t)(4 * NREC4) * T.SK;
    T.link_hit = a.ws_link_hit + (size_t)blockIdx.x * T.L * T.SK;
    return T;
}

// The three per-thread bodies are separate functions (not inlined) so that each gets its own register allocation:
// inlined into one kernel they need 228 registers and spill ~480 bytes at the 128 the launch bounds allow.

// hit_mode 1 (R20, R21, R23): second propagation step from the predicted state s on the layer's nominal surface to the surface
// through the hit (its own radius / its own z), then the 2-D update on the plane tangent to the hit radius; chi2 = that of
// the 2-D residual.  0 = done, 1 = the second step does not reach the hit (s untouched), -1 = S not positive definite.
static __device__ __noinline__ int two_step_update(State& s, float cw, const LayerC& ly, float mx, float my, float mz, float& chi2) {
    uint32_t flag;
    if (ly.kind) flag = predict_disk<true>(s, cw, ly, mz);
    else {
        LayerC hl = ly;
        hl.r2 = fmaf(mx, mx, my * my); hl.rcmin = 0.0f; hl.xx0r = 0.0f;
        flag = predict<true>(s, cw, hl);
    }
    if (flag) return 1;
    return update_2d(s, mx, my, mz, ly.kind, ly.var_rphi, ly.kind ? ly.var_r : ly.var_z, chi2) ? 0 : -1;
}

// phase 1, one live candidate: dense index base + i, round-local index i
// LIDS: the geometry has disks (R22); a barrel-only geometry compiles without any of it
template <bool ISO, bool LIDS>
__device__ __noinline__ void build_candidate(const BuildArgs& a, int l, int base, int i, int64_t s0) {
    const Tile T = tile_of(a);
    // shared arrays are re-derived from the block's shared window (so that they stay LDS / STS, not generic accesses)
    extern __shared__ __align__(16) unsigned char smem[];
    const int K = T.K, L = T.L, ncap = T.ncap, SK = T.SK;
    const BuildSmem m = build_smem(T.S, K, ncap, L);
    float* __restrict__ recA = T.recA; float* __restrict__ recB = T.recB;
    const unsigned short* s_cseed = (const unsigned short*)(smem + m.cseed);
    float* s_lchi2 = (float*)(smem + m.l_chi2); int* s_lhit = (int*)(smem + m.l_hit);
    unsigned char* s_lcnt = smem + m.l_cnt;
    float* s_pchi2 = (float*)(smem + m.p_chi2); int* s_pinfo = (int*)(smem + m.p_info);
    const LayerC& ly = a.layer[l];
    const int c = base + i;
    const int64_t sg = s0 + s_cseed[c];
    const float cw = -(float)a.q[sg] * a.kb;
    const int ev = a.seed_event ? a.seed_event[sg] : 0;
    State st;
    float chi2;
    int meta;
    rec_load(st, chi2, meta, recA, SK, c);
    uint32_t flag = 0u;
    bool fin = (meta & 256) != 0;
    float px = 0.f, py = 0.f, pz = 0.f, thr2 = 0.f, dzw = 0.f;
    float c00 = 0.f, c10 = 0.f, c11 = 0.f, c20 = 0.f, c21 = 0.f, c22 = 0.f;
    Ldl3 F = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    bool fok = false;
    WindowBins wb = {0, 0, 0, -1};
    [[maybe_unused]] float wrow = 0.f;          // LIDS: centre of the window along the row coordinate (z or radius)
    [[maybe_unused]] bool skip = false, disk = false;
    if constexpr (!LIDS) {
        if (!fin) {
            flag = predict(st, cw, ly);
            if (!flag) {
                px = st.XY.x; py = st.XY.y; pz = st.Z;
                c00 = st.P0.x; c10 = st.P0.y; c11 = st.P1.y; c20 = st.P2.x; c21 = st.P2.y; c22 = st.Q2.x;
                const float r2 = fmaf(px, px, py * py);
                const float num = fmaf(px * px, c11, fmaf(-2.0f * px * py, c10, py * py * c00));
                const float varphi = fmaxf(num / (r2 * r2), 0.0f);
                const float dphi = a.n_sigma * sqrtf(varphi + a.sphi_over_r2[l]);
                dzw = a.n_sigma * sqrtf(c22 + ly.var_z);
                if (!(dphi <= 3.0e38f) || !(dzw <= 3.0e38f)) flag = ST_NUMERIC;      // NaN or Inf
                else if (fabsf(pz) > ly.zmax + dzw) flag = ST_LEFT_Z;
                else {
                    thr2 = dphi * dphi * r2;
                    wb = window_bins(atan2f(py, px), dphi, pz, dzw, ly.zmax, a.inv_dz[l], a.inv_dphi, a.n_phi, a.n_z);
                    if (ISO) {
                        Sym3 Sm;
                        Sm.m00 = c00 + ly.var_r; Sm.m10 = c10; Sm.m11 = c11 + ly.var_r;
                        Sm.m20 = c20; Sm.m21 = c21; Sm.m22 = c22 + ly.var_z;
                        fok = ldl3(Sm, F);
                    }
                }
            }
            fin = flag != 0u;
        }
    } else {
        // Geometry with disks (R22): on a disk the window is in (phi, radius); a layer that is not reached or whose window
        // lies off it is skipped and the candidate lives on; only a numeric failure finishes it.
        disk = ly.kind != 0;
        if (!fin) {
            flag = disk ? predict_disk<false>(st, cw, ly, ly.r) : predict(st, cw, ly);
            if (!flag) {
                px = st.XY.x; py = st.XY.y; pz = st.Z;
                c00 = st.P0.x; c10 = st.P0.y; c11 = st.P1.y; c20 = st.P2.x; c21 = st.P2.y; c22 = st.Q2.x;
                const float r2 = fmaf(px, px, py * py);
                const float num = fmaf(px * px, c11, fmaf(-2.0f * px * py, c10, py * py * c00));
                const float varphi = fmaxf(num / (r2 * r2), 0.0f);
                float dphi;
                bool off;
                // hit_mode 1 (R23): sensors displaced along the surface normal (r.m.s. sig_r on a cylinder, sig_z on a disk) are
                // crossed elsewhere than on the nominal surface: the window grows by that
                float wphi2 = 0.0f, wrow2 = 0.0f;
                if (a.hit_mode && !disk) {
                    const float cinc = fmaf(px, st.CC.x, py * st.SS.x) * rsqrtf(r2);
                    const float cot = st.CC.y / st.SS.y;
                    const float t = cot / cinc;
                    wrow2 = ly.var_r * t * t;
                    wphi2 = ly.var_r * (1.0f - cinc * cinc) / (cinc * cinc) / r2;
                } else if (a.hit_mode) {
                    const float tth = st.SS.y / st.CC.y;
                    wrow2 = ly.var_z * tth * tth;
                    wphi2 = wrow2 / r2;
                }
                if (!disk) {
                    dphi = a.n_sigma * sqrtf(varphi + a.sphi_over_r2[l] + wphi2);
                    dzw = a.n_sigma * sqrtf(c22 + ly.var_z + wrow2);
                    wrow = pz;
                    off = fabsf(pz) > ly.zmax + dzw;
                } else {
                    const float varrho = fmaxf(fmaf(px * px, c00, fmaf(2.0f * px * py, c10, py * py * c11)) / r2, 0.0f);
                    dphi = a.n_sigma * sqrtf(varphi + ly.var_rphi / r2 + wphi2);
                    dzw = a.n_sigma * sqrtf(varrho + ly.var_r + wrow2);
                    wrow = sqrtf(r2);
                    off = wrow > ly.zmax + dzw || wrow < ly.rmin - dzw;
                }
                if (!(dphi <= 3.0e38f) || !(dzw <= 3.0e38f)) flag = ST_NUMERIC;      // NaN or Inf
                else if (off) flag = ST_LEFT_Z;
                else {
                    thr2 = dphi * dphi * r2;
                    wb = window_bins<true>(atan2f(py, px), dphi, wrow, dzw, a.row_lo[l], a.inv_dz[l], a.inv_dphi, a.n_phi, a.n_z);
                    if (ISO) {
                        Sym3 Sm;
                        Sm.m00 = c00 + ly.var_r; Sm.m10 = c10; Sm.m11 = c11 + ly.var_r;
                        Sm.m20 = c20; Sm.m21 = c21; Sm.m22 = c22 + ly.var_z;
                        fok = ldl3(Sm, F);
                    }
                }
            }
            if (a.lids && flag != 0u && flag != ST_NUMERIC) { skip = true; flag = 0u; }
            fin = flag != 0u || skip;
        }
    }
    int cnt = 0;
    if (!fin) {
        rec_store(st, chi2, meta, recB, SK, c);
        // ---- window scan (B3) ----
        bool sbad = false;
        float* lc = s_lchi2 + i;
        int* lh = s_lhit + i;
        const int64_t seg = (int64_t)ev * L + l;
        // Both runs of a row (the window may wrap at phi = pi) are scanned as one range.  Memory round
        // trips are what this loop costs (the hits are cold): the four bin offsets of the NEXT row are
        // requested before the hits of the current row, and SCAN_BATCH hits are requested together.
        const int e0 = min(wb.first + wb.n_b, a.n_phi), e1 = max(wb.first + wb.n_b - a.n_phi, 0);
        const int32_t* bo = a.bin_off + (seg * a.n_z + wb.iz_lo) * a.n_phi;
        int h0a = 0, h1a = 0, h0b = 0, h1b = 0;
        if (wb.iz_lo <= wb.iz_hi) { h0a = __ldg(bo + wb.first); h1a = __ldg(bo + e0); h0b = __ldg(bo); h1b = __ldg(bo + e1); }
        for (int iz = wb.iz_lo; iz <= wb.iz_hi; ++iz) {
            bo += a.n_phi;
            int n0a = 0, n1a = 0, n0b = 0, n1b = 0;
            if (iz < wb.iz_hi) { n0a = __ldg(bo + wb.first); n1a = __ldg(bo + e0); n0b = __ldg(bo); n1b = __ldg(bo + e1); }
            const int na = h1a - h0a, nab = na + (h1b - h0b);
            {
                for (int t0 = 0; t0 < nab; t0 += SCAN_BATCH) {
                    float4 hv[SCAN_BATCH];
                    int hpos[SCAN_BATCH];
#pragma unroll
                    for (int u = 0; u < SCAN_BATCH; ++u) {
                        const int t = min(t0 + u, nab - 1);
                        hpos[u] = t < na ? h0a + t : h0b + (t - na);
                        hv[u] = __ldg(a.xyzp + hpos[u]);
                    }
                    // window test of the batch (cheap, branch-free) -> bit mask; chi2 and the list only for the
                    // few hits inside the window, one at a time
                    unsigned inside = 0u;
#pragma unroll
                    for (int u = 0; u < SCAN_BATCH; ++u) {
                        const float mx = hv[u].x, my = hv[u].y, mz = hv[u].z;
                        const float cr = fmaf(px, my, -py * mx);
                        bool in_win;
                        if constexpr (!LIDS) {
                            in_win = (t0 + u < nab) && (cr * cr <= thr2 * fmaf(mx, mx, my * my)) && (fmaf(px, mx, py * my) > 0.0f) &&
                                     (fabsf(mz - pz) <= dzw);
                        } else {
                            const float rm2 = fmaf(mx, mx, my * my);
                            in_win = (t0 + u < nab) && (cr * cr <= thr2 * rm2) && (fmaf(px, mx, py * my) > 0.0f) &&
                                     (fabsf((disk ? sqrtf(rm2) : mz) - wrow) <= dzw);
                        }
                        inside |= in_win ? (1u << u) : 0u;
                    }
                    while (inside) {
                        const int u = __ffs(inside) - 1;
                        inside &= inside - 1u;
                        float4 m4 = hv[0];
                        int h = hpos[0];
#pragma unroll
                        for (int v = 1; v < SCAN_BATCH; ++v)
                            if (u == v) { m4 = hv[v]; h = hpos[v]; }
                        const float mx = m4.x, my = m4.y, mz = m4.z;
                        if constexpr (LIDS) {
                            if (a.hit_mode) {      // second step to the hit, 2-D chi2 there (the updated copy is dropped)
                                State t2 = st;
                                float c2h;
                                const int r2s = two_step_update(t2, cw, ly, mx, my, mz, c2h);
                                if (r2s < 0) { sbad = true; continue; }
                                if (r2s > 0) continue;
                                if (c2h < a.chi2_cut) {
                                    if (cnt < K) { lc[cnt * ncap] = chi2 + c2h; lh[cnt * ncap] = h; ++cnt; }
                                    else list_replace_worst(lc, lh, ncap, K, chi2 + c2h, h);
                                }
                                continue;
                            }
                        }
                        bool ok = fok;
                        if (!ISO) {
                            const HitCov V = hit_cov(mx, my, ly);
                            Sym3 Sm;
                            Sm.m00 = c00 + V.xx; Sm.m10 = c10 + V.xy; Sm.m11 = c11 + V.yy;
                            Sm.m20 = c20; Sm.m21 = c21; Sm.m22 = c22 + V.zz;
                            ok = ldl3(Sm, F);
                        }
                        if (!ok) { sbad = true; continue; }
                        const float q0 = mx - px, q1 = my - py, q2 = mz - pz;
                        const float y1 = fmaf(-F.l10, q0, q1);
                        const float y2 = fmaf(-F.l21, y1, fmaf(-F.l20, q0, q2));
                        const float c2 = fmaf(q0 * q0, F.i0, fmaf(y1 * y1, F.i1, y2 * y2 * F.i2));
                        if (c2 < a.chi2_cut) {
                            if (cnt < K) {           // unsorted append
                                lc[cnt * ncap] = chi2 + c2; lh[cnt * ncap] = h; ++cnt;
                            } else {
                                list_replace_worst(lc, lh, ncap, K, chi2 + c2, h);
                            }
                        }
                    }
                }
            }
            h0a = n0a; h1a = n1a; h0b = n0b; h1b = n1b;
        }
        list_sort(lc, lh, ncap, cnt);
        if (sbad) {      // S not positive definite: one finished child with the unchanged state
            fin = true;
            flag = ST_NUMERIC;
            cnt = 0;
        }
    }
    if (fin) rec_copy(recA, c, recB, c, SK);
    s_lcnt[i] = (unsigned char)cnt;
    s_pchi2[i] = chi2;
    s_pinfo[i] = (meta & 255) | (fin ? (LIDS && skip ? 512 : 256) : 0) | (int)(flag << 16);
}

// phase 3, one surviving child: dense index cn among the children of the tile
template <bool ISO, bool LIDS>
__device__ __noinline__ void build_child(const BuildArgs& a, int l, int cn) {
    const Tile T = tile_of(a);
    // shared arrays are re-derived from the block's shared window (so that they stay LDS / STS, not generic accesses)
    extern __shared__ __align__(16) unsigned char smem[];
    const int K = T.K, L = T.L, ncap = T.ncap, SK = T.SK;
    const BuildSmem m = build_smem(T.S, K, ncap, L);
    float* __restrict__ recA = T.recA; float* __restrict__ recB = T.recB;
    int32_t* link_hit = T.link_hit; uint8_t* link_par = smem + m.link_par;
    const int* s_off = (const int*)(smem + m.off); const int* s_offn = (const int*)(smem + m.offn);
    const float* sel_chi2 = (const float*)(smem + m.sel_chi2); const int* sel_hit = (const int*)(smem + m.sel_hit); const int* sel_pk = (const int*)(smem + m.sel_pk);
    const unsigned short* s_cseed = (const unsigned short*)(smem + m.cseed);
    const LayerC& ly = a.layer[l];
    const int s = s_cseed[cn];
    const int j = cn - s_offn[s];
    const float chi2c = sel_chi2[s * K + j];
    const int hitpos = sel_hit[s * K + j], pkd = sel_pk[s * K + j];
    const int k = pkd & 255, nh = (pkd >> 8) & 255;
    const int cp = s_off[s] + k;
    int link;
    if (hitpos == HITPOS_NONE) {
        rec_copy(recB, cp, recA, cn, SK);
        if (pkd & (1 << 16)) {
            const int meta = __float_as_int(rec_word(recB, SK, cp, W_META)) | 256 | (((pkd >> 24) & 15) << 16);
            rec_set_word(recA, SK, cn, W_META, __int_as_float(meta));
            link = -2;
        } else if (pkd & (1 << 17)) {      // layer skipped: the record is the unchanged state, the candidate lives on
            link = -2;
        } else {
            link = -1;
        }
    } else {
        State st;
        float chi2p;
        int meta;
        rec_load(st, chi2p, meta, recB, SK, cp);
        const float4 hv = __ldg(a.xyzp + hitpos);
        const float mx = hv.x, my = hv.y, mz = hv.z;
        HitCov V;
        if (ISO) { V.xx = ly.var_r; V.yy = ly.var_r; V.xy = 0.0f; V.zz = ly.var_z; }
        else V = hit_cov(mx, my, ly);
        Ldl3 F;
        float r[3], c2;
        bool ok;
        bool two_step = false;
        if constexpr (LIDS) two_step = a.hit_mode != 0;
        if (two_step) {
            const int64_t s0 = *reinterpret_cast<const long long*>(smem + m.misc + 4 * 36);      // first seed of the tile
            ok = two_step_update(st, -(float)a.q[s0 + s] * a.kb, ly, mx, my, mz, c2) == 0;
        } else {
            ok = innovation(st, mx, my, mz, V, F, r, c2);
            gain_update<ISO>(st, F, V, r);
        }
        ok = ok && state_finite(st) && st.IT.x > 0.0f;
        if (ok) {
            rec_store(st, chi2c, (meta & ~255) | nh, recA, SK, cn);
        } else {     // failed update: keep the predicted state, finish the candidate
            rec_copy(recB, cp, recA, cn, SK);
            rec_set_word(recA, SK, cn, W_CHI2, chi2c);
            rec_set_word(recA, SK, cn, W_META, __int_as_float(((meta & ~255) | nh) | 256 | (int)(ST_NUMERIC << 16)));
        }
        link = __float_as_int(hv.w);
    }
    __stcg(link_hit + l * SK + s * K + j, link);
    link_par[l * SK + s * K + j] = (uint8_t)k;
}

// B6, one live candidate (dense index c) -> its output slot; unused slots are filled by the caller
__device__ __noinline__ void build_output(const BuildArgs& a, int64_t s0, int c) {
    const Tile T = tile_of(a);
    extern __shared__ __align__(16) unsigned char smem[];
    const int K = T.K, L = T.L, SK = T.SK;
    const BuildSmem m = build_smem(T.S, K, T.ncap, L);
    const float* __restrict__ recA = T.recA;
    const int32_t* __restrict__ link_hit = T.link_hit;
    const uint8_t* link_par = smem + m.link_par;
    const int* s_nc = (const int*)(smem + m.nc); const int* s_off = (const int*)(smem + m.off);
    float* __restrict__ par_o = a.par_o; float* __restrict__ cov_o = a.cov_o; int32_t* __restrict__ hit_o = a.hit_idx_o;
    const unsigned short* s_cseed = (const unsigned short*)(smem + m.cseed);
    const int s = s_cseed[c], j = c - s_off[s];
    const int64_t sg = s0 + s;
    const int64_t slot = sg * K + j;
    (void)s_nc;
    {
        State st;
        float chi2;
        int meta;
        rec_load(st, chi2, meta, recA, SK, c);
        // back-trace: the parent chain runs through shared memory, so the hit links of four layers are requested together
        int k = j;
        for (int l = L - 1; l >= a.first_layer; l -= 4) {
            int v[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                if (l - u >= a.first_layer) {
                    v[u] = __ldcg(link_hit + (l - u) * SK + s * K + k);
                    k = link_par[(l - u) * SK + s * K + k];
                }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (l - u >= a.first_layer) hit_o[(int64_t)(l - u) * a.ld_out + slot] = v[u];
        }
        for (int l = 0; l < a.first_layer; ++l)
            hit_o[(int64_t)l * a.ld_out + slot] = a.seed_hit_idx ? a.seed_hit_idx[(int64_t)l * a.ld_seed + sg] : -1;
        state_store(st, [&](int i, float v) { par_o[(int64_t)i * a.ld_out + slot] = v; },
                    [&](int kk, float v) { cov_o[(int64_t)kk * a.ld_out + slot] = v; });
        a.chi2_o[slot] = chi2;
        a.nhits_o[slot] = meta & 255;
        a.status_o[slot] = (uint32_t)(meta >> 16) & 15u;
    }
}

template <int NT, bool ISO, bool LIDS>
__global__ void __launch_bounds__(NT, BUILD_THREADS_PER_SM / NT) kf_build_kernel(const __grid_constant__ BuildArgs ga) {
    extern __shared__ __align__(16) unsigned char smem[];
    // The phase bodies are separate functions that take the arguments by reference: a copy in shared memory keeps their
    // reads of it short (a reference to the kernel parameters makes every one a generic load of the parameter space).
    __shared__ BuildArgs sa;
    for (int w = threadIdx.x; w < (int)(sizeof(BuildArgs) / 4); w += NT) ((int*)&sa)[w] = ((const int*)&ga)[w];
    __syncthreads();
    const BuildArgs& a = sa;
    const int S = a.S, K = a.K, L = a.n_layers, ncap = a.ncap, SK = S * K;
    const BuildSmem m = build_smem(S, K, ncap, L);
    int* s_nc = (int*)(smem + m.nc); int* s_off = (int*)(smem + m.off);
    int* s_nnew = (int*)(smem + m.nnew); int* s_offn = (int*)(smem + m.offn);
    float* sel_chi2 = (float*)(smem + m.sel_chi2); int* sel_hit = (int*)(smem + m.sel_hit);
    int* sel_pk = (int*)(smem + m.sel_pk);
    unsigned short* s_cseed = (unsigned short*)(smem + m.cseed);
    float* s_lchi2 = (float*)(smem + m.l_chi2); int* s_lhit = (int*)(smem + m.l_hit);
    unsigned char* s_lcnt = smem + m.l_cnt; unsigned long long* s_hkey = (unsigned long long*)(smem + m.l_head);
    float* s_pchi2 = (float*)(smem + m.p_chi2); int* s_pinfo = (int*)(smem + m.p_info);
    int* s_misc = (int*)(smem + m.misc);          // [0..31] warp sums of the scan, [32] round end
    const int tid = threadIdx.x;

    float* recA = tile_of(a).recA;

    for (int64_t tile = blockIdx.x; tile < a.n_tiles; tile += gridDim.x) {
        const int64_t s0 = tile * S;
        const int ns = (int)min((int64_t)S, a.n_seeds - s0);
        if constexpr (LIDS) { if (tid == 0) *reinterpret_cast<long long*>(s_misc + 36) = s0; }
        // ---- seeds -> one candidate each, dense index = seed ----
        if (tid < S) {
            if (tid < ns) {
                const int64_t sg = s0 + tid;
                State st;
                state_load(st, [&](int i) { return a.par[(int64_t)i * a.ld_seed + sg]; }, [&](int k) { return a.cov[(int64_t)k * a.ld_seed + sg]; });
                rec_store(st, a.chi2_in ? a.chi2_in[sg] : 0.0f, a.first_layer, recA, SK, tid);
            }
            s_nc[tid] = tid < ns ? 1 : 0;
            s_off[tid] = tid < ns ? tid : ns;
            if (tid < ns) s_cseed[tid] = (unsigned short)tid;
        }
        if (tid == 0) s_off[S] = ns;
        __syncthreads();

        for (int l = a.first_layer; l < L; ++l) {
            const LayerC& ly = a.layer[l];
            // ---------------- rounds of whole seeds whose candidates fit the list area ----------------
            int r0 = 0;
            while (r0 < ns) {
                const int base = s_off[r0];
                int r1 = ns;
                if (s_off[ns] - base > ncap) {
                    if (tid >= r0 && tid < ns) {
                        const bool fits = s_off[tid + 1] - base <= ncap;
                        const bool next_fits = tid + 1 < ns && s_off[tid + 2] - base <= ncap;
                        if (fits && !next_fits) s_misc[32] = tid + 1;
                    }
                    __syncthreads();
                    r1 = s_misc[32];
                }
                const int nround = s_off[r1] - base;
                // ---------------- phase 1: predict + window + scan, thread per candidate ----------------
                for (int i = tid; i < nround; i += NT) {
                    build_candidate<ISO, LIDS>(a, l, base, i, s0);
                }
                __syncthreads();
                // ---------------- phase 2: best K children of a seed (B4), thread per seed ----------------
                // K-way merge of the sorted child lists of the <= K parents.  The head of every list is a 48-bit key whose
                // integer order is the total order R10: (63 - nhits) | chi2 bits (chi2 >= 0, so the bit pattern is
                // monotonic) | parent slot | position in the parent's list (ascending in (chi2, hit)); exhausted = all ones.
                if (tid >= r0 && tid < r1) {
                    const int s = tid;
                    const int nc = s_nc[s], ib = s_off[s] - base;
                    for (int k = 0; k < nc; ++k) {
                        const int i = ib + k;
                        const int cnt = s_lcnt[i];
                        const int nh = (s_pinfo[i] & 255) + (cnt ? 1 : 0);     // a finished or hit-less parent: one child, no hit
                        s_hkey[i] = child_key(nh, cnt ? s_lchi2[i] : s_pchi2[i], k, 0);
                    }
                    int n_out = 0;
                    for (; n_out < K; ++n_out) {
                        unsigned long long best = ~0ull;
                        for (int k = 0; k < nc; ++k) best = min(best, s_hkey[ib + k]);
                        if (best == ~0ull) break;
                        const int k = (int)(best >> 5) & 31, j = (int)best & 31, nh = 63 - (int)(best >> 42);
                        const int i = ib + k;
                        const int cnt = s_lcnt[i];
                        sel_chi2[s * K + n_out] = __uint_as_float((unsigned)(best >> 10));
                        sel_hit[s * K + n_out] = cnt ? s_lhit[j * ncap + i] : HITPOS_NONE;
                        sel_pk[s * K + n_out] = k | (nh << 8) | (s_pinfo[i] & 0x000f0300) << 8;   // bit 16 finished, bit 17 skipped, bits 24-27 status
                        s_hkey[i] = (j + 1 < cnt) ? child_key(nh, s_lchi2[(j + 1) * ncap + i], k, j + 1) : ~0ull;
                    }
                    s_nnew[s] = n_out;
                }
                __syncthreads();
                r0 = r1;
            }
            // ---------------- dense positions of the children ----------------
            {
                const int v = tid < ns ? s_nnew[tid] : 0;
                int tot;
                const int ex = block_exclusive_scan<NT>(v, s_misc, &tot);
                if (tid < S) s_offn[tid] = tid < ns ? ex : tot;
                if (tid == 0) s_offn[S] = tot;
                for (int j = 0; j < v; ++j) s_cseed[ex + j] = (unsigned short)tid;
                __syncthreads();
            }
            // ---------------- phase 3: update the survivors, thread per child (B5) ----------------
            const int nchild = s_offn[S];
            for (int cn = tid; cn < nchild; cn += NT) {
                build_child<ISO, LIDS>(a, l, cn);
            }
            __syncthreads();
            if (tid < S) { s_nc[tid] = tid < ns ? s_nnew[tid] : 0; s_off[tid] = s_offn[tid]; }
            if (tid == 0) s_off[S] = s_offn[S];
            __syncthreads();
        }

        // ---------------- B6: back-trace + store ----------------
        if (tid < ns) a.n_cand_o[s0 + tid] = s_nc[tid];
        for (int c = tid; c < s_off[ns]; c += NT) build_output(a, s0, c);       // live candidates, densely
        for (int idx = tid; idx < ns * K; idx += NT) {                            // every slot: charge; unused slots: empty
            const int s = idx / K, j = idx - s * K;
            const int64_t slot = (s0 + s) * K + j;
            a.q_o[slot] = a.q[s0 + s];
            if (j >= s_nc[s]) {
                a.chi2_o[slot] = 0.0f; a.nhits_o[slot] = 0; a.status_o[slot] = 0u;
                for (int l = 0; l < L; ++l) a.hit_idx_o[(int64_t)l * a.ld_out + slot] = -2;
            }
        }
        __syncthreads();     // the workspace and the shared arrays are reused by the next tile
    }
}

// ---- host side: tile size, grid and workspace layout (one function, used by the size query and by the launch) ----
static int sm_count() {
    static int n = 0;
    if (n == 0) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) {
            cudaGetLastError();
            n = 148;
        }
    }
    return n;
}

struct BuildPlan { int S, NT, ncap, grid; int64_t n_tiles; size_t smem, o_rec, o_lh, total; bool ok; };

static BuildPlan build_plan(int n_layers, int64_t n_seeds, int K, const kf_options* opt) {
    BuildPlan p;
    int S = KF_OPT(opt, build_seeds_per_block);
    const int max_blocks = KF_OPT(opt, build_max_blocks);
    p.ok = (S == 0 || (S >= 16 && S <= BUILD_MAX_NT && S % 16 == 0)) && max_blocks >= 0;
    if (!p.ok) S = 0;
    const bool automatic = S == 0;
    if (automatic)   // one wave of 128-seed tiles when the job is that small (latency-sized), otherwise small tiles: more
                     // independent blocks per SM, so that the block-level barriers of one tile overlap work of another
        S = n_seeds <= (int64_t)KF_TILE_WAVE * 2 * sm_count() ? KF_TILE_WAVE : KF_TILE_SMALL;
    for (;;) {
        p.S = S;
        p.NT = S * KF_BUILD_TPS <= 64 ? 64 : (S * KF_BUILD_TPS <= 128 ? 128 : 256);
        const int SK = S * K;
        p.ncap = std::min(SK, std::max(std::max(K, 32), (LIST_BYTES_PER_THREAD * p.NT / (8 * K)) & ~31));
        p.smem = (size_t)build_smem(S, K, p.ncap, n_layers).total;
        if (!automatic || p.smem + sizeof(BuildArgs) <= 200 * 1024 || S <= 16) break;      // large K and many layers: a smaller tile fits
        S /= 2;
    }
    const int SK = p.S * K;
    p.n_tiles = (n_seeds + p.S - 1) / p.S;
    const int by_smem = (int)std::max<size_t>(1, (size_t)(227 * 1024) / (p.smem + sizeof(BuildArgs) + 1024));
    int64_t resident = (int64_t)sm_count() * std::min(BUILD_THREADS_PER_SM / p.NT, by_smem);
    if (max_blocks > 0) resident = std::min<int64_t>(resident, max_blocks);
    p.grid = (int)std::min<int64_t>(std::max<int64_t>(p.n_tiles, 1), resident);
    auto up = [](size_t x) { return (x + 255) & ~(size_t)255; };
    size_t o = 0;
    p.o_rec = o; o += up((size_t)p.grid * 2 * (4 * NREC4) * SK * sizeof(float));
    p.o_lh = o; o += up((size_t)p.grid * n_layers * SK * sizeof(int32_t));
    p.total = o;
    return p;
}

template <int NT, bool ISO, bool LIDS>
static int launch_build3(const BuildArgs& a, const BuildPlan& p, cudaStream_t st) {
    cudaError_t e = cudaFuncSetAttribute(kf_build_kernel<NT, ISO, LIDS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.smem);
    if (e != cudaSuccess) return fail(KF_ERR_CUDA, "kf_build: cudaFuncSetAttribute: %s", cudaGetErrorString(e));
    kf_build_kernel<NT, ISO, LIDS><<<p.grid, NT, p.smem, st>>>(a);
    return check_launch("kf_build");
}

template <int NT>
static int launch_build(const BuildArgs& a, const BuildPlan& p, bool iso, cudaStream_t st) {
    if (a.lids || a.hit_mode) return iso ? launch_build3<NT, true, true>(a, p, st) : launch_build3<NT, false, true>(a, p, st);
    return iso ? launch_build3<NT, true, false>(a, p, st) : launch_build3<NT, false, false>(a, p, st);
}

}  // namespace kf

extern "C" size_t kf_build_workspace_bytes(const kf_geom* geom, int64_t n_seeds, int32_t K, const kf_options* opt) {
    if (!geom || geom->n_layers < 1 || geom->n_layers > KF_MAX_LAYERS || n_seeds < 0 || K < 1 || K > 32) return 0;
    const kf::BuildPlan p = kf::build_plan(geom->n_layers, n_seeds, K, opt);
    return p.ok ? p.total : 0;
}

extern "C" int kf_build(const kf_geom* geom, const kf_hits* hits, const kf_binned* binned, const kf_tracks* seeds,
                        const int32_t* seed_event, const int32_t* seed_hit_idx, int32_t first_layer, int32_t K, float chi2_cut,
                        float n_sigma, kf_cands* out, const kf_options* opt, void* ws, size_t ws_bytes, void* stream) {
    using namespace kf;
    if (!geom || !hits || !binned || !seeds || !out) return fail(KF_ERR_NULL_PTR, "kf_build: NULL struct argument");
    int rc = check_geom(geom, "kf_build");
    if (rc) return rc;
    if (K < 1 || K > 32) return fail(KF_ERR_INVALID_ARG, "kf_build: K = %d outside 1..32", K);
    if (first_layer < 0 || first_layer > geom->n_layers) return fail(KF_ERR_INVALID_ARG, "kf_build: first_layer outside 0..n_layers");
    if (!(chi2_cut > 0.f) || !(n_sigma > 0.f)) return fail(KF_ERR_INVALID_ARG, "kf_build: chi2_cut and n_sigma must be positive");
    if (seeds->n < 0 || seeds->ld < seeds->n) return fail(KF_ERR_INVALID_ARG, "kf_build: need 0 <= n <= ld for the seeds");
    if (out->ld < seeds->n * K || out->cand.ld != out->ld) return fail(KF_ERR_INVALID_ARG, "kf_build: out->ld must be >= n_seeds*K and equal cand.ld");
    if (binned->n_phi < 8 || (binned->n_phi % 8) || binned->n_z < 1) return fail(KF_ERR_BAD_GEOM, "kf_build: bad bin counts");
    const BuildPlan p = build_plan(geom->n_layers, seeds->n, K, opt);
    if (!p.ok) return fail(KF_ERR_INVALID_ARG, "kf_build: options out of range (build_seeds_per_block: 0 or a multiple of 16 in 16..256; build_max_blocks >= 0)");
    out->K = K; out->n_layers = geom->n_layers; out->n_seeds = seeds->n; out->cand.n = seeds->n * K;
    if (seeds->n == 0) return KF_OK;
    if (!seeds->par || !seeds->cov || !seeds->q) return fail(KF_ERR_NULL_PTR, "kf_build: NULL seed array");
    if (!binned->xyzp || !binned->bin_off) return fail(KF_ERR_NULL_PTR, "kf_build: NULL binned array (xyzp, bin_off)");
    if (hits->n_events > 1 && !seed_event) return fail(KF_ERR_NULL_PTR, "kf_build: seed_event is NULL with n_events > 1");
    const kf_tracks& c = out->cand;
    if (!c.par || !c.cov || !c.q || !c.chi2 || !c.nhits || !c.status || !out->hit_idx || !out->n_cand)
        return fail(KF_ERR_NULL_PTR, "kf_build: NULL output array");
    if (!ws || ws_bytes < p.total) return fail(KF_ERR_WORKSPACE_TOO_SMALL, "kf_build: workspace %zu < %zu bytes", ws_bytes, p.total);
    if (p.smem + sizeof(BuildArgs) > 227 * 1024) return fail(KF_ERR_INVALID_ARG, "kf_build: tile of %d seeds with K = %d needs %zu bytes of shared memory (> 227 KB)", p.S, K, p.smem);
    BuildArgs a;
    a.n_layers = geom->n_layers; a.first_layer = first_layer; a.K = K; a.n_phi = binned->n_phi; a.n_z = binned->n_z;
    a.S = p.S; a.ncap = p.ncap; a.n_tiles = p.n_tiles;
    a.kb = KCURV * geom->bz_tesla; a.chi2_cut = chi2_cut; a.n_sigma = n_sigma; a.inv_dphi = host_inv_dphi(binned->n_phi);
    a.n_seeds = seeds->n; a.ld_seed = seeds->ld; a.ld_out = out->ld;
    a.par = seeds->par; a.cov = seeds->cov; a.chi2_in = seeds->chi2; a.q = seeds->q; a.seed_event = seed_event; a.seed_hit_idx = seed_hit_idx;
    a.xyzp = (const float4*)binned->xyzp; a.bin_off = binned->bin_off;
    a.par_o = c.par; a.cov_o = c.cov; a.chi2_o = c.chi2; a.q_o = c.q; a.nhits_o = c.nhits; a.status_o = c.status;
    a.hit_idx_o = out->hit_idx; a.n_cand_o = out->n_cand;
    a.ws_rec = (float*)((char*)ws + p.o_rec); a.ws_link_hit = (int32_t*)((char*)ws + p.o_lh);
    bool iso = true;
    a.lids = 0; a.hit_mode = geom->hit_mode;
    for (int l = 0; l < KF_MAX_LAYERS; ++l) {
        const kf_layer& y = geom->layers[l < geom->n_layers ? l : geom->n_layers - 1];
        a.layer[l] = make_layer(y);
        host_row_range(y, binned->n_z, &a.row_lo[l], &a.inv_dz[l]);
        a.lids = a.lids || y.kind != 0;
        a.sphi_over_r2[l] = (y.sig_rphi / y.r) * (y.sig_rphi / y.r);
        iso = iso && y.sig_r == y.sig_rphi;
    }
    cudaStream_t st = (cudaStream_t)stream;
    switch (p.NT) {
        case 64: return launch_build<64>(a, p, iso, st);
        case 128: return launch_build<128>(a, p, iso, st);
        default: return launch_build<256>(a, p, iso, st);
    }
}

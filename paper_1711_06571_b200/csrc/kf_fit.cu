// kf_fit.cu -- fused propagate + update track fit (steps F1-F9).
//
// One thread per track; the whole layer loop runs in registers (6 parameters + 21 packed covariance elements),
// the only HBM traffic being the coalesced SoA load of the seed (F1), one hit (+ optional index) per layer (F6)
// and the coalesced store of the result (F9).  Per-layer constants arrive as a __grid_constant__ kernel
// parameter, i.e. through the constant bank: warp-uniform, no global loads.
#include "kf_common.cuh"
#include "kf_state.cuh"
#include "kf_pair.cuh"

namespace kf {

struct FitArgs {
    int32_t n_layers, n_events, hit_mode;
    float kb;                      // k * Bz
    int64_t n, ld_in, ld_out, ld_idx;
    const float* par; const float* cov; const int8_t* q;
    const float *hx, *hy, *hz;
    const int64_t* seg_off_dev;
    const int32_t* hit_idx; const int32_t* trk_event;
    float* par_o; float* cov_o; float* chi2_o; int32_t* nhits_o; uint32_t* status_o;
    LayerC layer[KF_MAX_LAYERS];
    const float *hxl[KF_MAX_LAYERS], *hyl[KF_MAX_LAYERS], *hzl[KF_MAX_LAYERS];   // hx + seg_off[l] ... of event 0 (trk_event == NULL)
};

#ifndef KF_FIT_BLOCK
#define KF_FIT_BLOCK 128
#endif
#ifndef KF_FIT_MINB
#define KF_FIT_MINB 5
#endif
#ifndef KF_FIT_IDX_MINB
#define KF_FIT_IDX_MINB KF_FIT_MINB   // explicit indices, gather requested a layer ahead: 96 registers without spills beat 80 with
                                      // (config 2 on B200: 0.334 ms at 5 blocks per SM, 0.365 at 6, 0.342 at 4; before the pipelined gather 0.354 at 6)
#endif
constexpr int FIT_BLOCK = KF_FIT_BLOCK;

// IDX: explicit hit_idx (else identity), EVT: per-track event (else event 0), ISO: sig_r == sig_rphi on every layer.

// The layer loop of one track, layers [0, limit).  Leaves through `break` when the track ends (failed propagation: the
// state of the last updated layer is final; status bit set) or when an update went numerically wrong: then the index
// of that layer is returned (-1 otherwise) and the state is garbage.  CAREFUL: every element of the state is checked
// after every layer (the fast path checks what reaches chi2 and the parameters, and the whole state once at the end).
template <bool IDX, bool EVT, bool ISO, bool CAREFUL>
__device__ __forceinline__ int fit_layers(const FitArgs& a, int64_t t, float cw, int64_t seg, int limit, State& s, float& chi2, int& nh,
                                          uint32_t& st) {
    // F1: coalesced SoA load
    state_load(s, [&](int i) { return a.par[i * a.ld_in + t]; }, [&](int k) { return a.cov[k * a.ld_in + t]; });
    chi2 = 0.0f;
    nh = 0;
    int bad = -1;
    // F6 with identity indexing: the hit of the next layer is requested one layer ahead
    float nx = 0.f, ny = 0.f, nz = 0.f;
    if (!IDX && !EVT && limit > 0) { nx = a.hxl[0][t]; ny = a.hyl[0][t]; nz = a.hzl[0][t]; }
    // F6 with explicit indices (event 0): the same one layer ahead, which takes the index two layers ahead -- the index of
    // layer l+2 and the hit of layer l+1 (whose index arrived during layer l-1) are requested before the arithmetic of layer l,
    // instead of index -> dependent gather -> arithmetic in every layer
    constexpr bool PIPE = IDX && !EVT;
    int i1 = -2, i2 = -2;                    // indices of this layer and the next
    if (PIPE) {
        if (limit > 0) i1 = a.hit_idx[t];
        if (limit > 1) i2 = a.hit_idx[a.ld_idx + t];
        if (i1 >= 0) { nx = a.hxl[0][i1]; ny = a.hyl[0][i1]; nz = a.hzl[0][i1]; }
    }
#pragma unroll 1
    for (int l = 0; l < limit; ++l) {
        int64_t idx = t;
        float px = nx, py = ny, pz = nz;     // PIPE: the hit of this layer, requested a layer ago
        if (PIPE) {
            idx = i1;
            i1 = i2;
            i2 = l + 2 < limit ? a.hit_idx[(int64_t)(l + 2) * a.ld_idx + t] : -2;
            if (i1 >= 0) { nx = a.hxl[l + 1][i1]; ny = a.hyl[l + 1][i1]; nz = a.hzl[l + 1][i1]; }
            if (idx < -1) continue;          // layer not crossed: skipped entirely (R8)
        } else if (IDX) {
            idx = a.hit_idx[l * a.ld_idx + t];
            if (idx < -1) continue;
        }
        const bool hole = IDX && idx < 0;    // -1: crossed without a hit -> transport + material, no update (R8)
        // F6: issued before the arithmetic
        float mx = 0.f, my = 0.f, mz = 0.f;
        if (hole) {
        } else if (EVT) {
            const int64_t h = a.seg_off_dev[seg + l] + idx;
            mx = a.hx[h]; my = a.hy[h]; mz = a.hz[h];
        } else {
            if (!IDX) {
                mx = nx; my = ny; mz = nz;
                if (l + 1 < limit) { nx = a.hxl[l + 1][t]; ny = a.hyl[l + 1][t]; nz = a.hzl[l + 1][t]; }
            } else {
                mx = px; my = py; mz = pz;
            }
        }
        const LayerC ly = a.layer[l];
        const uint32_t flag = predict(s, cw, ly);                          // F2-F5
        if (flag) {
            st |= flag;
            break;
        }
        if (hole) continue;
        Ldl3 Si;
        float r[3], c2;
        HitCov V;
        if (ISO) { V.xx = ly.var_r; V.yy = ly.var_r; V.xy = 0.0f; V.zz = ly.var_z; }
        else V = hit_cov(mx, my, ly);
        bool ok = innovation(s, mx, my, mz, V, Si, r, c2);                  // F7 (branch-free; garbage when !ok)
        gain_update<ISO>(s, Si, V, r);                                      // F8
        ok = ok && step_finite(s, c2) && s.IT.x > 0.0f && (!CAREFUL || state_finite(s));
        if (!ok) {
            bad = l;
            break;
        }
        chi2 += c2;
        nh += 1;
    }
    return bad;
}

// Numeric failure (rare): the track keeps the state of the last good layer, i.e. it is redone up to the layer before the
// one that failed.  A separate function so that the fast path keeps its registers.
template <bool IDX, bool EVT, bool ISO>
__device__ __noinline__ void fit_redo(const FitArgs& a, int64_t t, float cw, int64_t seg, State& s, float& chi2, int& nh, uint32_t& st) {
    int limit = a.n_layers;
    st = 0u;
    for (int attempt = 0; attempt < 3; ++attempt) {
        const uint32_t keep = st;
        const int bad = fit_layers<IDX, EVT, ISO, true>(a, t, cw, seg, limit, s, chi2, nh, st);
        if (bad < 0) return;
        st = keep | ST_NUMERIC;
        limit = bad;
    }
    // three failing layers in a row: the seed itself
    state_load(s, [&](int i) { return a.par[i * a.ld_in + t]; }, [&](int k) { return a.cov[k * a.ld_in + t]; });
    chi2 = 0.0f;
    nh = 0;
}

template <bool IDX, bool EVT, bool ISO>
__global__ void __launch_bounds__(FIT_BLOCK, IDX ? KF_FIT_IDX_MINB : KF_FIT_MINB) kf_fit_kernel(const __grid_constant__ FitArgs a) {
    const int64_t t = (int64_t)blockIdx.x * FIT_BLOCK + threadIdx.x;
    if (t >= a.n) return;
    const float cw = -(float)a.q[t] * a.kb;
    const int64_t seg = EVT ? (int64_t)a.trk_event[t] * a.n_layers : 0;
    State s;
    float chi2;
    int nh;
    uint32_t st = 0u;
    const int bad = fit_layers<IDX, EVT, ISO, false>(a, t, cw, seg, a.n_layers, s, chi2, nh, st);
    if (bad >= 0 || !state_finite(s)) fit_redo<IDX, EVT, ISO>(a, t, cw, seg, s, chi2, nh, st);
    // F9: coalesced store
    state_store(s, [&](int i, float v) { a.par_o[i * a.ld_out + t] = v; }, [&](int k, float v) { a.cov_o[k * a.ld_out + t] = v; });
    a.chi2_o[t] = chi2;
    a.nhits_o[t] = nh;
    a.status_o[t] = st;
}

// ---- two tracks per thread (kf_pair.cuh): identity indexing, event 0, isotropic hit covariance ----
// one track by the one-track code, as a function: the odd tail and the pairs that left the fast path
__device__ __noinline__ void fit_one(const FitArgs& a, int64_t t) {
    const float cw = -(float)a.q[t] * a.kb;
    State s;
    float chi2;
    int nh;
    uint32_t st = 0u;
    const int bad = fit_layers<false, false, true, false>(a, t, cw, 0, a.n_layers, s, chi2, nh, st);
    if (bad >= 0 || !state_finite(s)) fit_redo<false, false, true>(a, t, cw, 0, s, chi2, nh, st);
    state_store(s, [&](int i, float v) { a.par_o[i * a.ld_out + t] = v; }, [&](int k, float v) { a.cov_o[k * a.ld_out + t] = v; });
    a.chi2_o[t] = chi2;
    a.nhits_o[t] = nh;
    a.status_o[t] = st;
}

#ifndef KF_PAIR_MINB
#define KF_PAIR_MINB 3
#endif
__global__ void __launch_bounds__(FIT_BLOCK, KF_PAIR_MINB) kf_fit_pair_kernel(const __grid_constant__ FitArgs a) {
    using namespace pair;
    const int64_t t = 2 * ((int64_t)blockIdx.x * FIT_BLOCK + threadIdx.x);
    if (t >= a.n) return;
    if (t + 1 >= a.n) { fit_one(a, t); return; }
    auto ld2 = [](const float* p_) { V r; r.v = *reinterpret_cast<const float2*>(p_); return r; };
    const V cw = mk(-(float)a.q[t] * a.kb, -(float)a.q[t + 1] * a.kb);
    State2 S;
#pragma unroll
    for (int i = 0; i < 6; ++i) S.p[i] = ld2(a.par + i * a.ld_in + t);
#pragma unroll
    for (int i = 0; i < 21; ++i) S.C[i] = ld2(a.cov + i * a.ld_in + t);
    {
        float s0, c0, s1, c1;
        sincosf(S.p[4].v.x, &s0, &c0); sincosf(S.p[4].v.y, &s1, &c1);
        S.g.sp = mk(s0, s1); S.g.cp = mk(c0, c1);
        S.pha = phi_fix(S.p[4].v.x); S.phb = phi_fix(S.p[4].v.y);
        sincosf(S.p[5].v.x, &s0, &c0); sincosf(S.p[5].v.y, &s1, &c1);
        S.g.st = mk(s0, s1); S.g.ct = mk(c0, c1);
    }
    V chi2 = pair::sp(0.0f);
    bool good = true;
    const int L = a.n_layers;
    V nx = ld2(a.hxl[0] + t), ny = ld2(a.hyl[0] + t), nz = ld2(a.hzl[0] + t);     // F6: one layer ahead
#pragma unroll 1
    for (int l = 0; l < L; ++l) {
        const V mx = nx, my = ny, mz = nz;
        if (l + 1 < L) { nx = ld2(a.hxl[l + 1] + t); ny = ld2(a.hyl[l + 1] + t); nz = ld2(a.hzl[l + 1] + t); }
        const LayerC ly = a.layer[l];
        good = predict(S, cw, ly);                                   // F2-F5
        if (!good) break;
        V c2;
        good = update(S, mx, my, mz, ly.var_r, ly.var_z, c2);        // F7-F8
        if (!good) break;
        chi2 = chi2 + c2;
    }
    if (!good || !all_finite(S)) {      // not the fast path for one of the two: both by the one-track code
        fit_one(a, t);
        fit_one(a, t + 1);
        return;
    }
    // F9
    auto st2 = [](float* p_, V v) { *reinterpret_cast<float2*>(p_) = v.v; };
    S.p[4] = mk(phi_float(S.pha), phi_float(S.phb));
#pragma unroll
    for (int i = 0; i < 6; ++i) st2(a.par_o + i * a.ld_out + t, S.p[i]);
#pragma unroll
    for (int i = 0; i < 21; ++i) st2(a.cov_o + i * a.ld_out + t, S.C[i]);
    st2(a.chi2_o + t, chi2);
    *reinterpret_cast<int2*>(a.nhits_o + t) = make_int2(L, L);
    *reinterpret_cast<uint2*>(a.status_o + t) = make_uint2(0u, 0u);
}

// ---- "cylinder with lids" (R19-R21): disks in the layer list and / or hit_mode 1 (two-step propagation,
// 2-D update on the tangent plane).  One track per thread, explicit or identity indices, any event, any hit covariance. ----
__global__ void __launch_bounds__(FIT_BLOCK) kf_fit_lids_kernel(const __grid_constant__ FitArgs a) {
    const int64_t t = (int64_t)blockIdx.x * FIT_BLOCK + threadIdx.x;
    if (t >= a.n) return;
    const float cw = -(float)a.q[t] * a.kb;
    const int64_t seg = a.trk_event ? (int64_t)a.trk_event[t] * a.n_layers : 0;
    State s;
    state_load(s, [&](int i) { return a.par[i * a.ld_in + t]; }, [&](int k) { return a.cov[k * a.ld_in + t]; });
    float chi2 = 0.0f;
    int nh = 0;
    uint32_t st = 0u;
#pragma unroll 1
    for (int l = 0; l < a.n_layers; ++l) {
        int64_t idx = t;
        if (a.hit_idx) {
            idx = a.hit_idx[l * a.ld_idx + t];
            if (idx < -1) continue;
        }
        const LayerC ly = a.layer[l];
        const State before = s;                     // a layer that fails leaves the state of the last good layer
        uint32_t flag = ly.kind ? predict_disk<false>(s, cw, ly, ly.r) : predict(s, cw, ly);
        if (flag) { st |= flag; break; }
        if (idx < 0) continue;                      // hole: transported, material added, no update
        float mx, my, mz;
        if (a.trk_event) {
            const int64_t h = a.seg_off_dev[seg + l] + idx;
            mx = a.hx[h]; my = a.hy[h]; mz = a.hz[h];
        } else {
            mx = a.hxl[l][idx]; my = a.hyl[l][idx]; mz = a.hzl[l][idx];
        }
        bool ok;
        float c2;
        if (a.hit_mode) {
            if (ly.kind) flag = predict_disk<true>(s, cw, ly, mz);
            else {
                LayerC hl = ly;
                hl.r2 = fmaf(mx, mx, my * my); hl.rcmin = 0.0f; hl.xx0r = 0.0f;
                flag = predict<true>(s, cw, hl);
            }
            if (flag) { s = before; st |= flag; break; }
            ok = update_2d(s, mx, my, mz, ly.kind, ly.var_rphi, ly.kind ? ly.var_r : ly.var_z, c2);
        } else {
            Ldl3 Si;
            float r[3];
            const HitCov V = hit_cov(mx, my, ly);
            ok = innovation(s, mx, my, mz, V, Si, r, c2);
            gain_update<false>(s, Si, V, r);
        }
        ok = ok && step_finite(s, c2) && s.IT.x > 0.0f && state_finite(s);
        if (!ok) { s = before; st |= ST_NUMERIC; break; }
        chi2 += c2;
        nh += 1;
    }
    state_store(s, [&](int i, float v) { a.par_o[i * a.ld_out + t] = v; }, [&](int k, float v) { a.cov_o[k * a.ld_out + t] = v; });
    a.chi2_o[t] = chi2;
    a.nhits_o[t] = nh;
    a.status_o[t] = st;
}

template <bool IDX, bool EVT>
static void launch_fit(const FitArgs& a, bool iso, unsigned blocks, cudaStream_t st) {
    if (iso) kf_fit_kernel<IDX, EVT, true><<<blocks, FIT_BLOCK, 0, st>>>(a);
    else kf_fit_kernel<IDX, EVT, false><<<blocks, FIT_BLOCK, 0, st>>>(a);
}

}  // namespace kf

extern "C" int kf_fit(const kf_geom* geom, const kf_hits* hits, const int32_t* hit_idx, const int32_t* trk_event,
                      const kf_tracks* seeds, kf_tracks* out, const kf_options* opt, void* stream) {
    using namespace kf;
    if (!geom || !hits || !seeds || !out) return fail(KF_ERR_NULL_PTR, "kf_fit: NULL struct argument");
    int rc = check_geom(geom, "kf_fit");
    if (rc) return rc;
    if (seeds->n < 0 || seeds->ld < seeds->n || out->n != seeds->n || out->ld < out->n)
        return fail(KF_ERR_INVALID_ARG, "kf_fit: need 0 <= n <= ld and out->n == seeds->n");
    if (seeds->n == 0) return KF_OK;
    if (!seeds->par || !seeds->cov || !seeds->q || !out->par || !out->cov || !out->chi2 || !out->nhits || !out->status)
        return fail(KF_ERR_NULL_PTR, "kf_fit: NULL track array");
    if (!hits->x || !hits->y || !hits->z || !hits->seg_off) return fail(KF_ERR_NULL_PTR, "kf_fit: NULL hit array");
    if (hits->n_events < 1) return fail(KF_ERR_INVALID_ARG, "kf_fit: n_events < 1");
    if (trk_event && !hits->seg_off_dev) return fail(KF_ERR_NULL_PTR, "kf_fit: trk_event given but hits->seg_off_dev is NULL");
    if (trk_event && !hit_idx) return fail(KF_ERR_INVALID_ARG, "kf_fit: identity indexing (hit_idx == NULL) needs trk_event == NULL");
    const int tpt = KF_OPT(opt, fit_tracks_per_thread);
    if (tpt < 0 || tpt > 2) return fail(KF_ERR_INVALID_ARG, "kf_fit: options: fit_tracks_per_thread = %d not 0, 1 or 2", tpt);
    FitArgs a;
    a.n_layers = geom->n_layers; a.n_events = hits->n_events; a.hit_mode = geom->hit_mode;
    a.kb = KCURV * geom->bz_tesla;
    a.n = seeds->n; a.ld_in = seeds->ld; a.ld_out = out->ld; a.ld_idx = seeds->ld;
    a.par = seeds->par; a.cov = seeds->cov; a.q = seeds->q;
    a.hx = hits->x; a.hy = hits->y; a.hz = hits->z;
    a.seg_off_dev = hits->seg_off_dev; a.hit_idx = hit_idx; a.trk_event = trk_event;
    a.par_o = out->par; a.cov_o = out->cov; a.chi2_o = out->chi2; a.nhits_o = out->nhits; a.status_o = out->status;
    bool iso = true, lids = geom->hit_mode != 0;
    for (int l = 0; l < KF_MAX_LAYERS; ++l) {
        const int ll = l < geom->n_layers ? l : geom->n_layers - 1;
        a.layer[l] = make_layer(geom->layers[ll]);
        iso = iso && geom->layers[ll].sig_r == geom->layers[ll].sig_rphi;
        lids = lids || geom->layers[ll].kind != 0;
        const int64_t o = hits->seg_off[ll];
        a.hxl[l] = hits->x + o; a.hyl[l] = hits->y + o; a.hzl[l] = hits->z + o;
    }
    if (!hit_idx) {   // identity indexing: every segment of event 0 must hold n hits
        for (int l = 0; l < geom->n_layers; ++l)
            if (hits->seg_off[l + 1] - hits->seg_off[l] < seeds->n)
                return fail(KF_ERR_INVALID_ARG, "kf_fit: hit_idx == NULL needs >= n hits in every segment");
    }
    const unsigned blocks = (unsigned)((a.n + FIT_BLOCK - 1) / FIT_BLOCK);
    cudaStream_t cs = (cudaStream_t)stream;
    if (lids) {
        kf_fit_lids_kernel<<<blocks, FIT_BLOCK, 0, cs>>>(a);
        return check_launch("kf_fit");
    }
    if (tpt != 1 && !hit_idx && !trk_event && iso) {
        // two tracks per thread: 8-byte loads and stores of track pairs, so every array and stride must be even
        bool even = (a.ld_in % 2 == 0) && (a.ld_out % 2 == 0);
        const void* ptrs[] = {a.par, a.cov, a.par_o, a.cov_o, a.chi2_o, a.nhits_o, a.status_o};
        for (const void* q_ : ptrs) even = even && ((uintptr_t)q_ % 8 == 0);
        for (int l = 0; l < geom->n_layers; ++l)
            even = even && ((uintptr_t)a.hxl[l] % 8 == 0) && ((uintptr_t)a.hyl[l] % 8 == 0) && ((uintptr_t)a.hzl[l] % 8 == 0);
        if (even) {
            const int64_t n_thr = (a.n + 1) / 2;
            kf_fit_pair_kernel<<<(unsigned)((n_thr + FIT_BLOCK - 1) / FIT_BLOCK), FIT_BLOCK, 0, cs>>>(a);
            return check_launch("kf_fit");
        }
    }
    if (hit_idx) { if (trk_event) launch_fit<true, true>(a, iso, blocks, cs); else launch_fit<true, false>(a, iso, blocks, cs); }
    else launch_fit<false, false>(a, iso, blocks, cs);
    return check_launch("kf_fit");
}

// kf_api.cu -- error plumbing and small entry points of the C ABI (include/kf.h).
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include "kf_common.cuh"

namespace kf {

static thread_local char g_err[512] = "";

int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}

int check_launch(const char* what) {
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(KF_ERR_CUDA, "%s: CUDA error %d (%s)", what, (int)e, cudaGetErrorString(e));
    return KF_OK;
}

int check_geom(const kf_geom* g, const char* who) {
    if (!g->layers) return fail(KF_ERR_NULL_PTR, "%s: geom->layers is NULL", who);
    if (g->n_layers < 1 || g->n_layers > KF_MAX_LAYERS)
        return fail(KF_ERR_BAD_GEOM, "%s: n_layers = %d outside 1..%d", who, g->n_layers, KF_MAX_LAYERS);
    float last_r = 0.f, last_zp = 0.f, last_zn = 0.f;
    for (int l = 0; l < g->n_layers; ++l) {
        const kf_layer& y = g->layers[l];
        if (y.kind == 0) {
            if (!(y.r > last_r)) return fail(KF_ERR_BAD_GEOM, "%s: cylinder radii must be positive and strictly increasing (layer %d)", who, l);
            last_r = y.r;
        } else if (y.kind == 1) {
            float& last = y.r > 0.f ? last_zp : last_zn;
            if (!(fabsf(y.r) > last)) return fail(KF_ERR_BAD_GEOM, "%s: disks of one side must come with strictly increasing |z| (layer %d)", who, l);
            last = fabsf(y.r);
            if (!(y.rmin >= 0.f) || !(y.zmax > y.rmin)) return fail(KF_ERR_BAD_GEOM, "%s: disk %d needs 0 <= rmin < outer radius", who, l);
        } else
            return fail(KF_ERR_BAD_GEOM, "%s: layer %d has kind %d (0 = cylinder, 1 = disk)", who, l, y.kind);
        if (!(y.zmax > 0.f) || !(y.xx0 >= 0.f) || !(y.sig_rphi > 0.f) || !(y.sig_z > 0.f) || !(y.sig_r > 0.f))
            return fail(KF_ERR_BAD_GEOM, "%s: layer %d needs zmax > 0, xx0 >= 0 and positive resolutions", who, l);
    }
    if (g->hit_mode != 0 && g->hit_mode != 1) return fail(KF_ERR_BAD_GEOM, "%s: hit_mode = %d not 0 or 1", who, g->hit_mode);
    if (!(g->bz_tesla == g->bz_tesla)) return fail(KF_ERR_BAD_GEOM, "%s: bz_tesla is NaN", who);
    return KF_OK;
}

}  // namespace kf

extern "C" void kf_options_init(kf_options* opt) {
    if (!opt) return;
    opt->size = (uint32_t)sizeof(kf_options);
    opt->fit_tracks_per_thread = 0;
    opt->build_seeds_per_block = 0;
    opt->build_max_blocks = 0;
}

extern "C" const char* kf_last_error(void) { return kf::g_err; }
extern "C" int kf_version(void) { return 230; }

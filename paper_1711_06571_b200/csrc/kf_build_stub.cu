// temporary: entry points not built yet
#include "kf_common.cuh"
extern "C" size_t kf_bin_workspace_bytes(const kf_geom*, const kf_hits*, int32_t, int32_t) { return 0; }
extern "C" int kf_bin_hits(const kf_geom*, const kf_hits*, int32_t, int32_t, kf_binned*, void*, size_t, void*) { return kf::fail(KF_ERR_UNIMPLEMENTED, "kf_bin_hits: not implemented"); }
extern "C" int kf_window_lookup(const kf_geom*, const kf_hits*, const kf_binned*, int64_t, const int32_t*, const int32_t*, const float*, const float*, const float*, const float*, int32_t, int32_t*, int32_t*, void*) { return kf::fail(KF_ERR_UNIMPLEMENTED, "kf_window_lookup: not implemented"); }
extern "C" size_t kf_build_workspace_bytes(const kf_geom*, int64_t, int32_t) { return 0; }
extern "C" int kf_build(const kf_geom*, const kf_hits*, const kf_binned*, const kf_tracks*, const int32_t*, const int32_t*, int32_t, int32_t, float, float, kf_cands*, void*, size_t, void*) { return kf::fail(KF_ERR_UNIMPLEMENTED, "kf_build: not implemented"); }

// kf_common.cuh -- host-side plumbing shared by the entry points: error reporting, geometry checks.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>
#include "../../include/kf.h"
#include "kf_math.cuh"

namespace kf {

int fail(int code, const char* fmt, ...);              // records the message for kf_last_error(), returns code
int check_launch(const char* what);                    // cudaGetLastError() -> KF_OK / KF_ERR_CUDA
int check_geom(const kf_geom* g, const char* who);

// field of the caller's kf_options; 0 (= automatic) when opt is NULL or the caller's struct is older than the field
inline int32_t opt_get(const kf_options* o, size_t offset) {
    if (!o || o->size < offset + sizeof(int32_t)) return 0;
    return *(const int32_t*)((const char*)o + offset);
}
#define KF_OPT(o, field) kf::opt_get(o, offsetof(kf_options, field))

inline LayerC make_layer(const kf_layer& l) {
    LayerC c;
    c.r = l.r; c.r2 = l.r * l.r; c.zmax = l.zmax; c.xx0r = l.xx0 * l.r;
    c.var_rphi = l.sig_rphi * l.sig_rphi; c.var_z = l.sig_z * l.sig_z; c.var_r = l.sig_r * l.sig_r;
    c.rcmin = l.r * CMIN;
    c.xx0 = l.xx0; c.rmin = l.rmin; c.kind = l.kind; c.pad_ = 0;
    return c;
}

}  // namespace kf

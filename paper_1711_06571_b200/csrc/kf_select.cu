// kf_select.cu -- hand-over from building to the final fit (sec. 2: "When a complete track has been
// reconstructed, a final fit using the KF is performed to provide the best estimate of the track's parameters").
// kf_select_best copies the hit list of the best candidate of every seed (slot s*K of kf_cands, ranked first by
// kf_build) into the [n_layers][ld] index layout kf_fit reads, with kf_fit's meaning of the negative entries: -1 =
// layer crossed without a hit (transported, material added), -2 = not crossed; the layers already on the seed
// (< first_layer: the seed state sits behind them) become -2.
#include "kf_common.cuh"

namespace kf {

__global__ void __launch_bounds__(256) kf_select_best_kernel(const int32_t* __restrict__ cand_hit, int64_t ld_cand, int32_t K, int64_t n_seeds,
                                                             int32_t n_layers, int32_t first_layer, int32_t* __restrict__ out, int64_t ld_out) {
    const int64_t s = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (s >= n_seeds) return;
    for (int l = 0; l < n_layers; ++l) {
        const int32_t h = l < first_layer ? -2 : cand_hit[(int64_t)l * ld_cand + s * K];
        out[(int64_t)l * ld_out + s] = h < -2 ? -2 : h;
    }
}

}  // namespace kf

extern "C" int kf_select_best(const kf_cands* cands, int32_t first_layer, int32_t* hit_idx, int64_t ld, void* stream) {
    using namespace kf;
    if (!cands) return fail(KF_ERR_NULL_PTR, "kf_select_best: NULL struct argument");
    if (cands->n_seeds < 0 || cands->K < 1 || cands->n_layers < 1 || cands->n_layers > KF_MAX_LAYERS || ld < cands->n_seeds ||
        cands->ld < cands->n_seeds * cands->K || first_layer < 0 || first_layer > cands->n_layers)
        return fail(KF_ERR_INVALID_ARG, "kf_select_best: need n_seeds >= 0, K >= 1, 1 <= n_layers <= %d, ld >= n_seeds, cands->ld >= n_seeds*K, 0 <= first_layer <= n_layers", KF_MAX_LAYERS);
    if (cands->n_seeds == 0) return KF_OK;
    if (!cands->hit_idx || !hit_idx) return fail(KF_ERR_NULL_PTR, "kf_select_best: NULL array");
    kf_select_best_kernel<<<(unsigned)((cands->n_seeds + 255) / 256), 256, 0, (cudaStream_t)stream>>>(
        cands->hit_idx, cands->ld, cands->K, cands->n_seeds, cands->n_layers, first_layer, hit_idx, ld);
    return check_launch("kf_select_best");
}

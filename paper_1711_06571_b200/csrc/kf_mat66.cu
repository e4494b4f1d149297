// kf_mat66.cu -- batched 6x6 matrix multiply in two memory layouts.
//
// The paper's layout study (sec. 4.3, Fig. 5: "time vs number of 6x6 multiplications for different
// memory layouts"): "Matriplex" = matrix-major storage, element (r, c) of all N matrices contiguous, against plain
// arrays of matrices handed to a standard library.  Here: C_i = A_i B_i for i < n, fp32,
//   layout 0 (matrix-major / SoA): element (r, c) of matrix i at [(6 r + c) * ld + i]   -- what the KF kernels use
//   layout 1 (array of matrices / AoS): matrix i at [36 i + 6 r + c].
// One thread per matrix in both; 432 B and 432 flop per multiply, i.e. HBM-bound (1 flop/B).  In layout 0 every load
// and store of a warp is one 128-byte line; in layout 1 a thread reads its 144 contiguous bytes as nine 16-byte
// vectors, so a warp instruction touches 32 different lines and the L1 has to hold them until they are used up.
#include "kf_common.cuh"

namespace kf {

constexpr int MAT_BLOCK = 128;

__device__ __forceinline__ void mul66(const float (&a)[36], const float (&b)[36], float (&c)[36]) {
#pragma unroll
    for (int r = 0; r < 6; ++r)
#pragma unroll
        for (int k = 0; k < 6; ++k) {
            float acc = a[6 * r] * b[k];
#pragma unroll
            for (int m = 1; m < 6; ++m) acc = fmaf(a[6 * r + m], b[6 * m + k], acc);
            c[6 * r + k] = acc;
        }
}

__global__ void __launch_bounds__(MAT_BLOCK) kf_mat66_soa_kernel(int64_t n, int64_t ld, const float* __restrict__ A, const float* __restrict__ B,
                                                                 float* __restrict__ C) {
    const int64_t i = (int64_t)blockIdx.x * MAT_BLOCK + threadIdx.x;
    if (i >= n) return;
    float a[36], b[36], c[36];
#pragma unroll
    for (int e = 0; e < 36; ++e) { a[e] = A[e * ld + i]; b[e] = B[e * ld + i]; }
    mul66(a, b, c);
#pragma unroll
    for (int e = 0; e < 36; ++e) C[e * ld + i] = c[e];
}

__global__ void __launch_bounds__(MAT_BLOCK) kf_mat66_aos_kernel(int64_t n, const float* __restrict__ A, const float* __restrict__ B, float* __restrict__ C) {
    const int64_t i = (int64_t)blockIdx.x * MAT_BLOCK + threadIdx.x;
    if (i >= n) return;
    float a[36], b[36], c[36];
    const float4* a4 = reinterpret_cast<const float4*>(A + 36 * i);
    const float4* b4 = reinterpret_cast<const float4*>(B + 36 * i);
#pragma unroll
    for (int v = 0; v < 9; ++v) {
        const float4 x = a4[v], y = b4[v];
        a[4 * v] = x.x; a[4 * v + 1] = x.y; a[4 * v + 2] = x.z; a[4 * v + 3] = x.w;
        b[4 * v] = y.x; b[4 * v + 1] = y.y; b[4 * v + 2] = y.z; b[4 * v + 3] = y.w;
    }
    mul66(a, b, c);
    float4* c4 = reinterpret_cast<float4*>(C + 36 * i);
#pragma unroll
    for (int v = 0; v < 9; ++v) c4[v] = make_float4(c[4 * v], c[4 * v + 1], c[4 * v + 2], c[4 * v + 3]);
}

}  // namespace kf

extern "C" int kf_mat66_multiply(int32_t layout, int64_t n, int64_t ld, const float* A, const float* B, float* C, void* stream) {
    using namespace kf;
    if (layout != 0 && layout != 1) return fail(KF_ERR_INVALID_ARG, "kf_mat66_multiply: layout %d not 0 (matrix-major) or 1 (array of matrices)", layout);
    if (n < 0 || (layout == 0 && ld < n)) return fail(KF_ERR_INVALID_ARG, "kf_mat66_multiply: need n >= 0 and ld >= n");
    if (n == 0) return KF_OK;
    if (!A || !B || !C) return fail(KF_ERR_NULL_PTR, "kf_mat66_multiply: NULL array");
    if (layout == 1 && ((((uintptr_t)A) | ((uintptr_t)B) | ((uintptr_t)C)) & 15)) return fail(KF_ERR_INVALID_ARG, "kf_mat66_multiply: layout 1 needs 16-byte aligned arrays");
    const unsigned blocks = (unsigned)((n + MAT_BLOCK - 1) / MAT_BLOCK);
    if (layout == 0) kf_mat66_soa_kernel<<<blocks, MAT_BLOCK, 0, (cudaStream_t)stream>>>(n, ld, A, B, C);
    else kf_mat66_aos_kernel<<<blocks, MAT_BLOCK, 0, (cudaStream_t)stream>>>(n, A, B, C);
    return check_launch("kf_mat66_multiply");
}

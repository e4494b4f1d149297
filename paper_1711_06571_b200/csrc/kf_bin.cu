// kf_bin.cu -- binned hit index (B0) and the diagnostic window lookup (B2-B3 list): DESIGN.md readings X1-X3.
//
// "data structures used for selecting hit candidates" (sec. 3.1).  Per (event, layer) segment the hits
// are sorted by (z row, phi bin, original index); bin_off delimits the bins.  Everything here is integer / index
// work specified in IEEE fp32 single operations (__fdiv_rn, __fmul_rn, __fadd_rn: no contraction), so the result
// is bit-exact against the CPU oracle.
//
// Pipeline (one memset + four kernels on the caller's stream, no host-to-device copy: graph-capturable):
//   0. bin_off <- 0
//   1. bin_count:   thread per hit: key = global bin; rank = atomicAdd(bin_off[key + 1], 1) is at the same time the
//                   histogram and the hit's (arbitrary) arrival rank inside its bin; (key, rank) kept, 8 bytes per hit
//   2. bin_scan:    block per segment: inclusive scan of the segment's bin counts, offset by seg_off[segment] --
//                   segments are independent, so there is no carry between blocks and one launch does it
//   3. bin_scatter: thread per hit: record (x, y, z, original index) to bin_off[key] + rank (the hits travel with their
//                   index: no gather through the index later)
//   4. bin_place:   lane per record, warp per 32 consecutive bins: order the records of a bin by original index ->
//                   deterministic, stable; writes the 16-byte records the build scan reads and, if asked for, the
//                   sorted x, y, z, perm arrays
#include <cmath>
#include "kf_common.cuh"
#include "kf_binmath.cuh"

namespace kf {

constexpr int BIN_BLOCK = 256;
constexpr int SCAN_BLOCK = 512;
constexpr int SCAN_ITEMS = 8;                        // per thread
constexpr int MAX_TAN_TAB = 4096 / 8 + 1;

struct BinArgs {
    int32_t n_layers, n_phi, n_z, n_seg;
    const float *hx, *hy, *hz;
    const int64_t* seg_off;      // device
    int2* kr;                    // [n_hits] (key, arrival rank within the bin)
    int32_t* bin_off;            // [n_bins + 1]
    float4* tmp;                 // [n_hits] records in arrival order within each bin
    float *sx, *sy, *sz;         // optional (all or none)
    int32_t* perm;
    float4* xyzp;
    float phi_scale;             // n_phi / (2 pi): first guess of the table search
    float row_lo[KF_MAX_LAYERS], row_inv[KF_MAX_LAYERS];   // X2 rows: z in [-zmax, zmax) on a barrel layer, radius in [rmin, rmax) on a disk
    int32_t kind[KF_MAX_LAYERS];
    float tan_tab[MAX_TAN_TAB];  // X1: fl32(tan(2 pi k / n_phi)), k = 0 .. n_phi/8 (evaluated in double on the host), last = 1
};

// BIN_ILP hits per thread, all their loads requested before the first is used and all their atomics before the first rank
// is stored: the chain load -> atomic -> store is two memory round trips per hit otherwise
constexpr int BIN_ILP = 2;

__global__ void __launch_bounds__(BIN_BLOCK) kf_bin_count_kernel(const __grid_constant__ BinArgs a) {
    extern __shared__ float s_tab[];
    for (int i = threadIdx.x; i <= a.n_phi / 8; i += BIN_BLOCK) s_tab[i] = a.tan_tab[i];
    __syncthreads();
    for (int seg = blockIdx.y; seg < a.n_seg; seg += gridDim.y) {
        const int l = seg % a.n_layers;
        const int64_t h0 = a.seg_off[seg], h1 = a.seg_off[seg + 1];
        const int32_t base = seg * a.n_z * a.n_phi;
        const bool disk = a.kind[l] != 0;
        const float lo = a.row_lo[l], inv = a.row_inv[l];
        for (int64_t hb = h0 + (int64_t)blockIdx.x * (BIN_BLOCK * BIN_ILP) + threadIdx.x; hb < h1; hb += (int64_t)gridDim.x * (BIN_BLOCK * BIN_ILP)) {
            float x[BIN_ILP], y[BIN_ILP], z[BIN_ILP];
#pragma unroll
            for (int u = 0; u < BIN_ILP; ++u) {
                const int64_t h = min(hb + u * BIN_BLOCK, h1 - 1);
                x[u] = a.hx[h]; y[u] = a.hy[h]; z[u] = a.hz[h];
            }
            int b[BIN_ILP], r[BIN_ILP];
#pragma unroll
            for (int u = 0; u < BIN_ILP; ++u)
                b[u] = base + row_bin(disk ? hit_rho(x[u], y[u]) : z[u], lo, inv, a.n_z) * a.n_phi + phi_bin(x[u], y[u], a.n_phi, s_tab, a.phi_scale);
#pragma unroll
            for (int u = 0; u < BIN_ILP; ++u)
                if (hb + u * BIN_BLOCK < h1) r[u] = atomicAdd(&a.bin_off[b[u] + 1], 1);
#pragma unroll
            for (int u = 0; u < BIN_ILP; ++u)
                if (hb + u * BIN_BLOCK < h1) a.kr[hb + u * BIN_BLOCK] = make_int2(b[u], r[u]);
        }
    }
}

// block per segment: bin_off[seg*B + b + 1] <- seg_off[seg] + (number of hits in bins 0..b of the segment)
__global__ void __launch_bounds__(SCAN_BLOCK) kf_bin_scan_kernel(int32_t* __restrict__ bin_off, const int64_t* __restrict__ seg_off, int bins_per_seg) {
    __shared__ int s_warp[SCAN_BLOCK / 32];
    __shared__ int s_carry;
    const int seg = blockIdx.x, lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int32_t* v = bin_off + (int64_t)seg * bins_per_seg + 1;
    if (threadIdx.x == 0) s_carry = (int)seg_off[seg];
    __syncthreads();
    for (int base = 0; base < bins_per_seg; base += SCAN_BLOCK * SCAN_ITEMS) {
        const int t0 = base + threadIdx.x * SCAN_ITEMS;
        int x[SCAN_ITEMS];
        int acc = 0;
#pragma unroll
        for (int i = 0; i < SCAN_ITEMS; ++i) { x[i] = (t0 + i < bins_per_seg) ? v[t0 + i] : 0; acc += x[i]; }
        int inc = acc;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int o = __shfl_up_sync(0xffffffffu, inc, d);
            if (lane >= d) inc += o;
        }
        if (lane == 31) s_warp[w] = inc;
        __syncthreads();
        int before = s_carry;
        for (int j = 0; j < w; ++j) before += s_warp[j];
        int run = before + inc - acc;
#pragma unroll
        for (int i = 0; i < SCAN_ITEMS; ++i) { run += x[i]; if (t0 + i < bins_per_seg) v[t0 + i] = run; }
        __syncthreads();
        if (threadIdx.x == SCAN_BLOCK - 1) s_carry = run;
        __syncthreads();
    }
}

__global__ void __launch_bounds__(BIN_BLOCK) kf_bin_scatter_kernel(const __grid_constant__ BinArgs a) {
    for (int seg = blockIdx.y; seg < a.n_seg; seg += gridDim.y) {
        const int64_t h0 = a.seg_off[seg], h1 = a.seg_off[seg + 1];
        for (int64_t hb = h0 + (int64_t)blockIdx.x * (BIN_BLOCK * BIN_ILP) + threadIdx.x; hb < h1; hb += (int64_t)gridDim.x * (BIN_BLOCK * BIN_ILP)) {
            int2 kr[BIN_ILP];
            float x[BIN_ILP], y[BIN_ILP], z[BIN_ILP];
            int pos[BIN_ILP];
#pragma unroll
            for (int u = 0; u < BIN_ILP; ++u) {
                const int64_t h = min(hb + u * BIN_BLOCK, h1 - 1);
                kr[u] = a.kr[h];
                x[u] = a.hx[h]; y[u] = a.hy[h]; z[u] = a.hz[h];
            }
#pragma unroll
            for (int u = 0; u < BIN_ILP; ++u) pos[u] = __ldg(a.bin_off + kr[u].x) + kr[u].y;
#pragma unroll
            for (int u = 0; u < BIN_ILP; ++u)
                if (hb + u * BIN_BLOCK < h1) a.tmp[pos[u]] = make_float4(x[u], y[u], z[u], __int_as_float((int)(hb + u * BIN_BLOCK - h0)));
        }
    }
}

// A warp takes 32 consecutive bins and with them one contiguous run of records; a LANE takes a record (not a bin: bins hold
// 0 to a dozen records, so a thread per bin leaves two thirds of the lanes waiting for the fullest one).  The record's bin
// is found among the warp's 33 offsets (held one per lane) by a shuffle binary search; its place is the rank of its
// original index among the records of that bin (L1-resident re-reads of the index word).
template <bool SOA>
__global__ void __launch_bounds__(BIN_BLOCK) kf_bin_place_kernel(const __grid_constant__ BinArgs a, int64_t n_bins) {
    const int lane = threadIdx.x & 31;
    const int64_t b0 = ((int64_t)blockIdx.x * BIN_BLOCK + threadIdx.x) - lane;      // first bin of the warp
    if (b0 >= n_bins) return;
    const int64_t bl = min(b0 + lane, n_bins);
    const int off = a.bin_off[bl], off1 = a.bin_off[min(bl + 1, n_bins)];           // [off, off1): this lane's bin
    const int start = __shfl_sync(0xffffffffu, off, 0), end = __shfl_sync(0xffffffffu, off1, 31);
    for (int base = start; base < end; base += 32) {
        const int i = base + lane;
        const bool valid = i < end;
        int lo = 0;                                        // largest lane whose bin starts at or before record i
#pragma unroll
        for (int step = 16; step >= 1; step >>= 1) {
            const int v = __shfl_sync(0xffffffffu, off, lo + step);
            if (v <= i) lo += step;
        }
        const int o0 = __shfl_sync(0xffffffffu, off, lo), o1 = __shfl_sync(0xffffffffu, off1, lo);
        if (valid) {
            const float4 me = a.tmp[i];
            const int idx = __float_as_int(me.w);
            int rank = 0;
            for (int j = o0; j < o1; ++j) rank += __float_as_int(a.tmp[j].w) < idx ? 1 : 0;
            const int dst = o0 + rank;
            a.xyzp[dst] = me;
            if (SOA) { a.sx[dst] = me.x; a.sy[dst] = me.y; a.sz[dst] = me.z; a.perm[dst] = idx; }
        }
    }
}

// ---- window lookup (diagnostic entry; the build kernel walks the same ranges) ----
struct LookupArgs {
    int32_t n_layers, n_phi, n_z, cap;
    int64_t n_query;
    const int32_t *event, *layer;
    const float *phi_c, *dphi, *z_c, *dz;
    const int32_t* bin_off;
    int32_t *count, *sorted_idx;
    float inv_dphi;
    float row_lo[KF_MAX_LAYERS], row_inv[KF_MAX_LAYERS];
};

__global__ void __launch_bounds__(BIN_BLOCK) kf_window_lookup_kernel(const __grid_constant__ LookupArgs a) {
    const int64_t i = (int64_t)blockIdx.x * BIN_BLOCK + threadIdx.x;
    if (i >= a.n_query) return;
    const int l = a.layer[i];
    const WindowBins w = window_bins<true>(a.phi_c[i], a.dphi[i], a.z_c[i], a.dz[i], a.row_lo[l], a.row_inv[l], a.inv_dphi, a.n_phi, a.n_z);
    const int64_t seg = (int64_t)a.event[i] * a.n_layers + l;
    int c = 0;
    for (int iz = w.iz_lo; iz <= w.iz_hi; ++iz) {
        const int64_t row = (seg * a.n_z + iz) * a.n_phi;
        for (int k = 0; k < w.n_b; ++k) {
            int ip = w.first + k;
            if (ip >= a.n_phi) ip -= a.n_phi;
            const int h0 = a.bin_off[row + ip], h1 = a.bin_off[row + ip + 1];
            for (int h = h0; h < h1; ++h) {
                if (c < a.cap) a.sorted_idx[i * a.cap + c] = h;
                ++c;
            }
        }
    }
    a.count[i] = c;
}

static int check_bins(const kf_geom* geom, const kf_hits* hits, int32_t n_phi, int32_t n_z, const char* who, int64_t* n_bins) {
    if (n_phi < 8 || n_phi > 4096 || (n_phi % 8) != 0 || n_z < 1 || n_z > 1024)
        return fail(KF_ERR_BAD_GEOM, "%s: need n_phi a multiple of 8 in 8..4096 and n_z in 1..1024", who);
    if (hits->n_events < 1 || hits->n_hits < 0) return fail(KF_ERR_INVALID_ARG, "%s: n_events < 1 or n_hits < 0", who);
    const int64_t nb = (int64_t)hits->n_events * geom->n_layers * n_phi * n_z;
    if (nb + 1 >= (int64_t)1 << 31 || hits->n_hits >= (int64_t)1 << 31)
        return fail(KF_ERR_INVALID_ARG, "%s: bins (%lld) or hits (%lld) exceed the int32 index range", who, (long long)nb, (long long)hits->n_hits);
    *n_bins = nb;
    return KF_OK;
}

static inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

struct BinWs { size_t kr, tmp, total; };
static BinWs bin_ws_layout(int64_t n_hits) {
    BinWs w;
    size_t o = 0;
    w.kr = o; o += align256((size_t)n_hits * sizeof(int2));
    w.tmp = o; o += align256((size_t)n_hits * sizeof(float4));
    w.total = o;
    return w;
}

}  // namespace kf

extern "C" size_t kf_bin_workspace_bytes(const kf_geom* geom, const kf_hits* hits, int32_t n_phi, int32_t n_z) {
    using namespace kf;
    if (!geom || !hits) return 0;
    int64_t nb;
    if (check_geom(geom, "kf_bin_workspace_bytes") || check_bins(geom, hits, n_phi, n_z, "kf_bin_workspace_bytes", &nb)) return 0;
    return bin_ws_layout(hits->n_hits).total;
}

extern "C" int kf_bin_hits(const kf_geom* geom, const kf_hits* hits, int32_t n_phi, int32_t n_z, kf_binned* out, void* ws,
                           size_t ws_bytes, void* stream) {
    using namespace kf;
    if (!geom || !hits || !out) return fail(KF_ERR_NULL_PTR, "kf_bin_hits: NULL struct argument");
    int rc = check_geom(geom, "kf_bin_hits");
    if (rc) return rc;
    int64_t n_bins;
    rc = check_bins(geom, hits, n_phi, n_z, "kf_bin_hits", &n_bins);
    if (rc) return rc;
    if (!hits->seg_off || !hits->seg_off_dev) return fail(KF_ERR_NULL_PTR, "kf_bin_hits: hits->seg_off / seg_off_dev is NULL");
    if (!out->bin_off) return fail(KF_ERR_NULL_PTR, "kf_bin_hits: out->bin_off is NULL");
    const int64_t n_hits = hits->n_hits;
    const bool soa = out->x || out->y || out->z || out->perm;
    if (n_hits > 0 && (!hits->x || !hits->y || !hits->z || !out->xyzp || (soa && (!out->x || !out->y || !out->z || !out->perm))))
        return fail(KF_ERR_NULL_PTR, "kf_bin_hits: NULL hit array (out->x, y, z, perm: all or none)");
    const int n_seg = hits->n_events * geom->n_layers;
    if (hits->seg_off[0] != 0 || hits->seg_off[n_seg] != n_hits) return fail(KF_ERR_INVALID_ARG, "kf_bin_hits: seg_off must run from 0 to n_hits");
    int64_t max_seg = 0;
    for (int s = 0; s < n_seg; ++s) {
        const int64_t d = hits->seg_off[s + 1] - hits->seg_off[s];
        if (d < 0) return fail(KF_ERR_INVALID_ARG, "kf_bin_hits: seg_off not monotonic at segment %d", s);
        if (d > max_seg) max_seg = d;
    }
    const BinWs w = bin_ws_layout(n_hits);
    if (!ws || ws_bytes < w.total) return fail(KF_ERR_WORKSPACE_TOO_SMALL, "kf_bin_hits: workspace %zu < %zu bytes", ws_bytes, w.total);
    cudaStream_t st = (cudaStream_t)stream;
    char* base = (char*)ws;
    out->n_phi = n_phi; out->n_z = n_z;

    BinArgs a;
    a.n_layers = geom->n_layers; a.n_phi = n_phi; a.n_z = n_z; a.n_seg = n_seg;
    a.hx = hits->x; a.hy = hits->y; a.hz = hits->z; a.seg_off = hits->seg_off_dev;
    a.kr = (int2*)(base + w.kr); a.bin_off = out->bin_off; a.tmp = (float4*)(base + w.tmp);
    a.sx = out->x; a.sy = out->y; a.sz = out->z; a.perm = out->perm; a.xyzp = (float4*)out->xyzp;
    a.phi_scale = host_inv_dphi(n_phi);
    for (int l = 0; l < KF_MAX_LAYERS; ++l) {
        const kf_layer& y = geom->layers[l < geom->n_layers ? l : geom->n_layers - 1];
        host_row_range(y, n_z, &a.row_lo[l], &a.row_inv[l]);      // one IEEE fp32 subtraction and division (X2)
        a.kind[l] = y.kind;
    }
    // X1 table: T[k] = fl32(tan(2 pi k / N)) evaluated in double on the host, T[N/8] = 1; travels as a kernel argument
    const double two_pi = 6.283185307179586476925286766559;
    for (int k = 0; k < n_phi / 8; ++k) a.tan_tab[k] = (float)std::tan(two_pi * (double)k / (double)n_phi);
    a.tan_tab[n_phi / 8] = 1.0f;
    for (int k = n_phi / 8 + 1; k < MAX_TAN_TAB; ++k) a.tan_tab[k] = 0.0f;

    cudaMemsetAsync(out->bin_off, 0, (size_t)(n_bins + 1) * sizeof(int32_t), st);
    if (n_hits > 0) {
        const unsigned gx = (unsigned)std::min<int64_t>((max_seg + BIN_BLOCK * BIN_ILP - 1) / (BIN_BLOCK * BIN_ILP), 4096);
        const dim3 grid(gx ? gx : 1, (unsigned)std::min(n_seg, 65535));
        kf_bin_count_kernel<<<grid, BIN_BLOCK, (size_t)(n_phi / 8 + 1) * sizeof(float), st>>>(a);
        kf_bin_scan_kernel<<<n_seg, SCAN_BLOCK, 0, st>>>(out->bin_off, hits->seg_off_dev, n_phi * n_z);
        kf_bin_scatter_kernel<<<grid, BIN_BLOCK, 0, st>>>(a);
        const unsigned pb = (unsigned)((n_bins + BIN_BLOCK - 1) / BIN_BLOCK);
        if (soa) kf_bin_place_kernel<true><<<pb, BIN_BLOCK, 0, st>>>(a, n_bins);
        else kf_bin_place_kernel<false><<<pb, BIN_BLOCK, 0, st>>>(a, n_bins);
    }
    return check_launch("kf_bin_hits");
}

extern "C" int kf_window_lookup(const kf_geom* geom, const kf_hits* hits, const kf_binned* binned, int64_t n_query,
                                const int32_t* event, const int32_t* layer, const float* phi_c, const float* dphi,
                                const float* z_c, const float* dz, int32_t cap, int32_t* count, int32_t* sorted_idx, void* stream) {
    using namespace kf;
    if (!geom || !hits || !binned) return fail(KF_ERR_NULL_PTR, "kf_window_lookup: NULL struct argument");
    int rc = check_geom(geom, "kf_window_lookup");
    if (rc) return rc;
    int64_t n_bins;
    rc = check_bins(geom, hits, binned->n_phi, binned->n_z, "kf_window_lookup", &n_bins);
    if (rc) return rc;
    if (n_query < 0 || cap < 0) return fail(KF_ERR_INVALID_ARG, "kf_window_lookup: n_query < 0 or cap < 0");
    if (n_query == 0) return KF_OK;
    if (!event || !layer || !phi_c || !dphi || !z_c || !dz || !count || (cap > 0 && !sorted_idx) || !binned->bin_off)
        return fail(KF_ERR_NULL_PTR, "kf_window_lookup: NULL array");
    LookupArgs a;
    a.n_layers = geom->n_layers; a.n_phi = binned->n_phi; a.n_z = binned->n_z; a.cap = cap; a.n_query = n_query;
    a.event = event; a.layer = layer; a.phi_c = phi_c; a.dphi = dphi; a.z_c = z_c; a.dz = dz;
    a.bin_off = binned->bin_off; a.count = count; a.sorted_idx = sorted_idx;
    a.inv_dphi = host_inv_dphi(binned->n_phi);
    for (int l = 0; l < KF_MAX_LAYERS; ++l) {
        const kf_layer& y = geom->layers[l < geom->n_layers ? l : geom->n_layers - 1];
        host_row_range(y, binned->n_z, &a.row_lo[l], &a.row_inv[l]);
    }
    kf_window_lookup_kernel<<<(unsigned)((n_query + BIN_BLOCK - 1) / BIN_BLOCK), BIN_BLOCK, 0, (cudaStream_t)stream>>>(a);
    return check_launch("kf_window_lookup");
}

// ---- kf_bin_hits_static: the same binning with its scratch in a fixed array of this library (include/kf.h) ----
// For callers that cannot get device memory themselves: a module inside a framework that owns all device memory through its
// pool, or a loop that cannot afford cudaMalloc's device-wide synchronisation.  Nothing here allocates.
#include <mutex>

namespace kf {

constexpr size_t align256_c(size_t x) { return (x + 255) & ~(size_t)255; }
// the layout of bin_ws_layout() for the largest batch accepted: (key, rank) pairs, then the records in arrival order
constexpr size_t STATIC_WS_BYTES = align256_c((size_t)KF_BIN_STATIC_MAX_HITS * sizeof(int2)) + align256_c((size_t)KF_BIN_STATIC_MAX_HITS * sizeof(float4));

// Lives in the global memory of every GPU that loads this module, until the process ends.  In HOST code the name below is only
// a handle for cudaGetSymbolAddress -- it is not a device pointer and must never be handed to a kernel as one.
static __device__ __align__(256) unsigned char g_bin_scratch[STATIC_WS_BYTES];

constexpr int STATIC_MAX_DEVICES = 64;
static void* g_bin_scratch_addr[STATIC_MAX_DEVICES];     // device address of g_bin_scratch on device d; NULL = not looked up yet
static std::mutex g_bin_scratch_mutex;

}  // namespace kf

extern "C" int kf_bin_hits_static(const kf_geom* geom, const kf_hits* hits, int32_t n_phi, int32_t n_z, kf_binned* out, void* stream) {
    using namespace kf;
    if (!geom || !hits || !out) return fail(KF_ERR_NULL_PTR, "kf_bin_hits_static: NULL struct argument");
    if (hits->n_hits > (int64_t)KF_BIN_STATIC_MAX_HITS)
        return fail(KF_ERR_INVALID_ARG, "kf_bin_hits_static: n_hits = %lld exceeds KF_BIN_STATIC_MAX_HITS = %d, the size of the library's fixed scratch array "
                    "(bin fewer events per call, or use kf_bin_hits with a workspace of your own)", (long long)hits->n_hits, (int)KF_BIN_STATIC_MAX_HITS);
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(KF_ERR_CUDA, "kf_bin_hits_static: cudaGetDevice failed: %d (%s)", (int)e, cudaGetErrorString(e));
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return fail(KF_ERR_INVALID_ARG, "kf_bin_hits_static: device ordinal %d outside 0..%d", dev, STATIC_MAX_DEVICES - 1);
    void* scratch = nullptr;
    {   // once per device, with that device current: the array's address THERE (each GPU has its own copy)
        std::lock_guard<std::mutex> lock(g_bin_scratch_mutex);
        scratch = g_bin_scratch_addr[dev];
        if (!scratch) {
            e = cudaGetSymbolAddress(&scratch, g_bin_scratch);
            if (e != cudaSuccess || !scratch)
                return fail(KF_ERR_CUDA, "kf_bin_hits_static: cudaGetSymbolAddress on device %d failed: %d (%s)", dev, (int)e, cudaGetErrorString(e));
            g_bin_scratch_addr[dev] = scratch;
        }
    }
    // every scratch entry of a hit is written (count, scatter) before it is read (scatter, place): nothing to clear between calls
    return kf_bin_hits(geom, hits, n_phi, n_z, out, scratch, STATIC_WS_BYTES, stream);
}

/* kf.h -- C ABI of libkf_b200: batched Kalman-filter track fitting and combinatorial track building on one
 * NVIDIA B200 (sm_100a), fp32.
 *
 * The operations are the hot path of arxiv 1711.06571:
 *   - kf_fit:   "a final fit using the KF is performed to provide the best estimate of the track's parameters"
 *               -- repeated propagate + update over a fixed hit list, no branching (sec. 2);
 *   - kf_bin_hits / kf_window_lookup: the "data structures used for selecting hit candidates" (sec. 3.1);
 *   - kf_build: "Track building projects the track candidate outwards to collect additional hits, using the KF to
 *               estimate which hits represent the most likely continuation ... branching to explore multiple
 *               candidate tracks per seed", with "a fixed number of slots for each track seed" and
 *               "rapid identification of the best candidates" (sec. 4.3).
 * The paper gives no formulas; the arithmetic (state, helix, Jacobian, noise, update, ranking, bins) is fixed by
 * DESIGN.md sec. 3 "Readings" and restated per entry point below.
 *
 * Conventions
 *   - State p = (x, y, z, 1/pT, phi, theta): global Cartesian position [cm], polar momentum ("hybrid
 *     coordinate system"); charge q = +-1 separate; field along +z in Tesla; curvature dphi/ds_T = -q k Bz / pT,
 *     k = 0.00299792458 GeV/(T cm).
 *   - Covariance: packed lower-triangular row-major, element (i,j), i >= j, at k = i(i+1)/2 + j; 21 floats.
 *   - Every array argument is a DEVICE pointer unless marked "host".  SoA: component c of track t at [c*ld + t].
 *   - The library never allocates, frees or retains user memory.  All work is enqueued on `stream`
 *     (a cudaStream_t passed as void*; NULL = the legacy default stream) and the call returns without
 *     synchronising.  Host-marked arrays are read before the call returns.
 *   - Return value 0 = OK, negative = kf_status.  No C++ exception crosses the boundary.  kf_last_error() gives
 *     a thread-local, statically stored description of the last failure on the calling thread.
 *   - Per-track numerical trouble is data, not an error: it sets bits in `status` and the track keeps its
 *     last good state.
 */
#ifndef KF_B200_H
#define KF_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define KF_MAX_LAYERS 32

typedef enum {
    KF_OK = 0,
    KF_ERR_INVALID_ARG = -1,
    KF_ERR_NULL_PTR = -2,
    KF_ERR_BAD_GEOM = -3,            /* n_layers outside 1..KF_MAX_LAYERS, radii / disk |z| not increasing, n_phi % 8 != 0 ... */
    KF_ERR_WORKSPACE_TOO_SMALL = -4,
    KF_ERR_CUDA = -5,                /* launch / runtime error; text in kf_last_error() */
    KF_ERR_UNIMPLEMENTED = -6
} kf_status;

/* per-track status bits */
#define KF_ST_UNREACHABLE 1u /* layer surface not reached within half a turn, start radius >= layer radius, disk behind */
#define KF_ST_LEFT_Z 2u      /* kf_build only: predicted |z| beyond zmax + window                                   */
#define KF_ST_GRAZING 4u     /* cos(incidence) < 0.1 at the crossing (cylinder: in the transverse plane; disk: |cos theta|) */
#define KF_ST_NUMERIC 8u     /* innovation matrix not positive definite, non-finite result, or 1/pT <= 0            */

/* One layer.  kind 0, barrel: cylinder of radius r [cm], half length zmax [cm].  kind 1, endcap disk ("cylinder with
 * lids", sec. 4.1; R19): the plane z = r (signed), covering rmin <= radius <= zmax.  Thickness xx0
 * in radiation lengths at normal incidence, hit resolutions [cm] along r-phi, z and r (in a 3-D update the resolution
 * along the surface normal -- sig_r for a cylinder, sig_z for a disk -- only regularises; R5). */
typedef struct { float r, zmax, xx0, sig_rphi, sig_z, sig_r; int32_t kind; float rmin; } kf_layer;

/* Geometry: n_layers layers in the order a track from the vertex crosses them (cylinders by increasing r, then the
 * disks of either side by increasing |z|); uniform field bz_tesla along z.  `layers` is a HOST array.
 * hit_mode 0: hits lie on the nominal surfaces, 3-D update there (R5).  hit_mode 1 (R20, R21; kf_fit
 * and kf_build): two-step propagation -- to the nominal surface, where the material is added, then on to the hit's own
 * radius (barrel) or z (disk) -- and a 2-D update on the plane tangent to the hit radius (r-phi and z for a barrel
 * hit, r-phi and r for a disk hit); the state then sits on the hit's surface. */
typedef struct { int32_t n_layers; float bz_tesla; const kf_layer* layers; int32_t hit_mode; } kf_geom;

/* Per-call tuning options (never change a result beyond rounding; kf_build results do not depend on them at all).
 * Pass NULL for the defaults.  `size` = sizeof(kf_options) of the caller's header (versioning: fields beyond it are
 * taken as 0 = automatic); kf_options_init fills the defaults.  There is no process-global state in the library. */
typedef struct {
    uint32_t size;
    int32_t fit_tracks_per_thread;   /* 0 = automatic (2 where the arguments allow it), 1 = always one track per thread  */
    int32_t build_seeds_per_block;   /* seeds owned by one thread block of kf_build: 0 = automatic, else a multiple of 16 in 16..256 */
    int32_t build_max_blocks;        /* cap on the persistent grid of kf_build: 0 = automatic (fills the device)         */
} kf_options;
void kf_options_init(kf_options* opt);

/* SoA track store.  n tracks, stride ld >= n between components. */
typedef struct {
    int64_t n, ld;
    float* par;       /* [6][ld]  x, y, z, 1/pT, phi, theta                                   */
    float* cov;       /* [21][ld] packed symmetric                                             */
    int8_t* q;        /* [n]      charge +-1                                                   */
    float* chi2;      /* [n]      accumulated chi2 (input value is ignored by kf_fit)          */
    int32_t* nhits;   /* [n]      number of hits used                                          */
    uint32_t* status; /* [n]      KF_ST_* bits                                                 */
} kf_tracks;

/* Hits of all (event, layer) segments back to back, SoA.  Segment (event e, layer l) is
 * [seg_off[e*n_layers + l], seg_off[e*n_layers + l + 1]).  seg_off is a HOST array of n_events*n_layers + 1
 * entries; seg_off_dev is a device copy of the same array (required when n_events > 1 or for the build calls,
 * may be NULL for kf_fit with n_events == 1). */
typedef struct {
    int64_t n_hits;
    const float *x, *y, *z;
    int32_t n_events;
    const int64_t* seg_off;
    const int64_t* seg_off_dev;
} kf_hits;

/* ---------------------------------------------------------------------------------------------------------
 * kf_fit -- forward (inside-out) Kalman filter over a fixed hit list (DESIGN.md sec. 2 F1-F9).
 * For every track t and every layer l in list order with hit_idx[l*ld + t] >= -1:
 *   propagate the state and covariance along the exact helix to the first crossing of the layer's surface (Jacobian
 *   including the path-length term), add the multiple-scattering noise of the layer (Highland) and, if there is a hit,
 *   update with the 3-D hit (residual, 3x3 innovation inverse, chi2, gain, state and covariance update).
 * hit_idx: [n_layers][seeds->ld] index of the hit within its segment; -1 = layer crossed without a hit (transport and
 *          material, no update: what kf_build does for a candidate without a compatible hit); <= -2 = layer not
 *          crossed, skipped entirely; NULL = identity (hit of track t on layer l is element t of segment l; needs
 *          trk_event == NULL).
 * trk_event: [n] event of each track, NULL = event 0.
 * seeds/out: same n; out->ld may differ; out may alias seeds.  out->q is not written.
 * A failing layer sets the status bit, ends the track there and leaves the state of the last updated layer.
 * Output phi is wrapped to (-pi, pi].  Errors: NULL pointers, n < 0, ld < n, bad geometry, hit_idx == NULL together
 * with trk_event != NULL, CUDA launch failure.
 * With sig_r == sig_rphi on every layer, event 0 and even strides / 8-byte aligned arrays kf_fit runs two tracks per
 * thread (all arithmetic as packed fp32 pairs); tracks that leave the fast path (failed crossing, large turning angle
 * or angle correction, numeric trouble) are redone by the one-track code.  opt->fit_tracks_per_thread = 1 forces the
 * one-track kernel (results agree to rounding). */
int kf_fit(const kf_geom* geom, const kf_hits* hits, const int32_t* hit_idx, const int32_t* trk_event,
           const kf_tracks* seeds, kf_tracks* out, const kf_options* opt, void* stream);

/* ---------------------------------------------------------------------------------------------------------
 * Binned hit index (DESIGN.md sec. 2 B0, readings X1-X2).  Filled by kf_bin_hits into
 * caller-allocated arrays.  Global bin of a hit = ((event*n_layers + layer)*n_z + iz)*n_phi + iphi; iphi from the
 * azimuth by exact fp32 comparisons against a tangent table (no atan2), iz = clamp(floor((z + zmax)*n_z/(2 zmax))) on a
 * barrel layer; on a disk (kind 1; R22) the rows are cut along the radius of the hit,
 * iz = clamp(floor((sqrt(x^2 + y^2) - rmin)*n_z/(rmax - rmin))), every operation one IEEE fp32 rounding.
 * Sorted order = ascending (global bin, original index): unique, hence bit-exact testable. */
typedef struct {
    int32_t n_phi, n_z;   /* n_phi multiple of 8, 8..4096; n_z 1..1024                                     */
    float *x, *y, *z;     /* [n_hits] hits in sorted order            } optional: all four NULL = not wanted       */
    int32_t* perm;        /* [n_hits] sorted position -> original index within its segment                 */
    int32_t* bin_off;     /* [n_events*n_layers*n_z*n_phi + 1] offsets into the sorted arrays              */
    float* xyzp;          /* [n_hits][4] the same hits as 16-byte records (x, y, z, bits of perm): what the */
                          /* window scan of kf_build reads, one load per hit; 16-byte aligned; required     */
} kf_binned;

size_t kf_bin_workspace_bytes(const kf_geom* geom, const kf_hits* hits, int32_t n_phi, int32_t n_z);
int kf_bin_hits(const kf_geom* geom, const kf_hits* hits, int32_t n_phi, int32_t n_z, kf_binned* out, void* ws,
                size_t ws_bytes, void* stream);

/* kf_bin_hits_static -- kf_bin_hits for callers that have no device memory to lend as workspace and may not allocate any.
 * Who that is: a reconstruction module running inside an event-processing framework whose device memory is handed out by the
 * framework's own pool (a direct cudaMalloc is forbidden there, or simply fails because the pool already holds the card),
 * and a trigger-style loop that must not hit cudaMalloc's device-wide synchronisation and unbounded latency between events.
 * Same arguments, same result (bit for bit) as kf_bin_hits, minus ws / ws_bytes: the 24 bytes per hit of scratch (bin key +
 * arrival rank, then the record in arrival order) live in ONE fixed array compiled into the library, sized for
 * KF_BIN_STATIC_MAX_HITS hits.  Cost of that: every GPU on which the library's device code gets loaded carries the array
 * (24 MiB) until the process exits, whether or not this entry is ever called.
 *   - hits->n_hits > KF_BIN_STATIC_MAX_HITS is refused with KF_ERR_INVALID_ARG and a message naming both numbers (bin larger
 *     batches in pieces of whole events, or use kf_bin_hits with your own workspace).
 *   - The call itself performs no cudaMalloc / cudaFree and uses no library routine that allocates; inputs and outputs are the
 *     caller's as before.
 *   - The device that is CURRENT on the calling thread must be the one that owns `stream` and every array passed in.  The first
 *     call on each device looks up the array's device address (cudaGetSymbolAddress; this may make the runtime load the
 *     library's device code on that GPU) and remembers it per device; make that first call during set-up, before any stream
 *     capture is begun.  Later calls only launch.
 *   - All calls on a device share the one array and it keeps whatever the previous call left.  Nothing in it needs to start
 *     from zero -- each call writes the entries of its own n_hits hits before it reads them -- but two calls whose kernels can
 *     overlap on the GPU (different streams without an ordering between them, or host threads racing) overwrite each other's
 *     scratch and give wrong bins: order them on one stream or with events. */
#define KF_BIN_STATIC_MAX_HITS (1 << 20)
int kf_bin_hits_static(const kf_geom* geom, const kf_hits* hits, int32_t n_phi, int32_t n_z, kf_binned* out, void* stream);

/* kf_window_lookup -- test / diagnostic entry: the window hit list of B2-B3 for explicit windows (reading X3).
 * Query i: event[i], layer[i], azimuth window phi_c +- dphi (phi_c in (-pi, pi], dphi >= 0), z window z_c +- dz (on a
 * disk layer z_c, dz are read as the radius window rho_c +- d_rho).
 * The list is every hit of the bins touched, rows in ascending iz, bins in ascending (wrapping) iphi, hits in
 * sorted order.  count[i] = true length even if > cap; sorted_idx[i*cap + j] = global sorted position, j < min(count, cap). */
int kf_window_lookup(const kf_geom* geom, const kf_hits* hits, const kf_binned* binned, int64_t n_query,
                     const int32_t* event, const int32_t* layer, const float* phi_c, const float* dphi,
                     const float* z_c, const float* dz, int32_t cap, int32_t* count, int32_t* sorted_idx, void* stream);

/* ---------------------------------------------------------------------------------------------------------
 * kf_build -- combinatorial track building (DESIGN.md sec. 2 B1-B6, readings R10-R11).
 * Per seed, per layer l = first_layer .. n_layers-1: propagate the <= K live candidates, open a window of
 * n_sigma standard deviations in phi and z, chi2 against every hit of the window, one child per hit with
 * chi2 < chi2_cut (else one child without hit), keep the best K children by (nhits desc, chi2 asc, parent slot asc,
 * sorted hit position asc), update the survivors.
 * Geometry with endcap disks ("cylinder with lids"; R22): on a disk the window is in phi and
 * radius, and on any layer a candidate that cannot be propagated there (not reached, grazing) or whose window lies off the
 * layer skips it (hit_idx -2, state unchanged, no status bit) and lives on; only a numeric failure finishes a candidate.
 * A barrel-only geometry keeps the behaviour below (a failed layer finishes the candidate).
 * geom->hit_mode 1 ("further propagation steps to the position of each candidate hit"; R23): every hit
 * of the window is reached by a second propagation step from the predicted state and judged by the chi2 of its 2-D residual
 * on the plane tangent to the hit radius; survivors are updated there (state on the hit's own surface).  The window is
 * widened by the displacement of the sensors about the nominal surface, whose r.m.s. is read from the resolution along the
 * surface normal (sig_r of a cylinder, sig_z of a disk), which the 2-D update does not use.
 * Output: slot s*K + k of `cand` (best first), hit_idx[l*ld + slot] = original index within the segment,
 * -1 = no hit on this layer, -2 = layer not crossed (candidate finished); n_cand[s] = number of valid slots.
 */
typedef struct {
    int32_t K, n_layers;
    int64_t n_seeds, ld;  /* ld >= n_seeds*K */
    kf_tracks cand;       /* n = n_seeds*K, cand.ld == ld */
    int32_t* hit_idx;     /* [n_layers][ld] */
    int32_t* n_cand;      /* [n_seeds] */
} kf_cands;

/* Seeds: state on (or near) layer first_layer-1; every seed starts with chi2 = seeds->chi2[s] (0 when seeds->chi2 is
 * NULL) and nhits = first_layer (seeds->nhits is ignored).  seed_event [n] (may be NULL when n_events == 1); seed_hit_idx
 * [first_layer][seeds->ld] = hits already on the seed (copied to the output lists; NULL = -1).
 * Slots k >= n_cand[s] get nhits = 0, chi2 = 0, status = 0 and hit_idx = -2; their par / cov are not written.
 * cand.q is filled with the seed's charge.  A candidate that cannot be propagated to a layer, leaves
 * |z| <= zmax + window, or fails numerically is finished (status bit set) and carried unchanged.
 * K in 1..32.  ws: device workspace of at least kf_build_workspace_bytes(geom, n_seeds, K, opt) bytes (candidate records
 * and per-layer hit links of the tiles in flight: (288 + 4 n_layers) K bytes per seed in flight, ~100 MB at most); a
 * pure function of its arguments; the workspace is only used while the enqueued kernel runs and may be reused by the
 * next call on the same stream.  opt (NULL = automatic): seeds per thread block and the cap on the persistent grid;
 * the result does not depend on them, the workspace size does (pass the same opt to both calls).
 * Errors: NULL pointers, K / first_layer / cuts / options out of range, bad bin counts, workspace too small (-4),
 * CUDA failure. */
size_t kf_build_workspace_bytes(const kf_geom* geom, int64_t n_seeds, int32_t K, const kf_options* opt);
int kf_build(const kf_geom* geom, const kf_hits* hits, const kf_binned* binned, const kf_tracks* seeds,
             const int32_t* seed_event, const int32_t* seed_hit_idx, int32_t first_layer, int32_t K, float chi2_cut,
             float n_sigma, kf_cands* out, const kf_options* opt, void* ws, size_t ws_bytes, void* stream);

/* ---------------------------------------------------------------------------------------------------------
 * kf_select_best -- hand-over from building to the final fit ("When a complete track has been
 * reconstructed, a final fit using the KF is performed").  hit_idx[l*ld + s] = hit of the best candidate (slot s*K)
 * of seed s on layer l, in the layout and with the meaning kf_fit reads: >= 0 hit, -1 layer crossed without a hit,
 * -2 layer not crossed; layers < first_layer (already behind the seed state) are -2.  The final fit is then
 *   kf_fit(geom, hits, hit_idx, seed_event, seeds, out, NULL, stream)       with ld == seeds->ld
 * and goes through exactly the steps the built candidate went through (R8).
 * Errors: NULL pointers, ld < n_seeds, first_layer outside 0..n_layers, CUDA failure. */
int kf_select_best(const kf_cands* cands, int32_t first_layer, int32_t* hit_idx, int64_t ld, void* stream);

/* ---------------------------------------------------------------------------------------------------------
 * kf_mat66_multiply -- the paper's layout micro-benchmark (sec. 4.3, Fig. 5): C_i = A_i B_i for n
 * general 6x6 fp32 matrices.  layout 0 = matrix-major ("Matriplex"): element (r, c) of matrix i at [(6r + c)*ld + i],
 * ld >= n; layout 1 = array of matrices: matrix i at [36 i + 6r + c] (ld ignored; arrays 16-byte aligned).
 * C must not overlap A or B.  Errors: bad layout, n < 0, ld < n, NULL or misaligned arrays, CUDA failure. */
int kf_mat66_multiply(int32_t layout, int64_t n, int64_t ld, const float* A, const float* B, float* C, void* stream);

const char* kf_last_error(void);
int kf_version(void);

#ifdef __cplusplus
}
#endif
#endif /* KF_B200_H */

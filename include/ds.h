/*
 * ds.h -- C ABI of libds: the HLT1 "Downstream + ghost-killer MLP + two-track vertexing" hot path of
 * arXiv:2503.13092 as hand-written CUDA for NVIDIA B200 (sm_100a).
 *
 * Citations: `P:n` = line n of the paper text; `A-n` = a reading of the paper listed in DESIGN.md.
 *
 * Conventions for every entry point
 *   - Pointers marked HOST are read/written synchronously on the calling thread.  Pointers marked DEVICE are CUDA
 *     device pointers on the handle's device, owned by the caller; the library never frees or reallocates them.
 *   - `cuda_stream` is a `cudaStream_t` passed as `void*` (NULL = the legacy default stream).  All device work is
 *     enqueued on it and the call returns without synchronising; outputs are valid once the caller has
 *     synchronised the stream.  The `*_host` calls are the exception: they block until the results are in the
 *     HOST buffers.
 *   - Return value: DS_OK (0) or a negative DS_E_* code.  Nothing throws, aborts or prints.  There is no CPU
 *     fallback: without a CUDA device ds_create fails with DS_E_CUDA.
 *   - Units: mm, GeV for q/p (1/GeV) and the kick, MeV for masses.  Arrays are flat over all events of the call with
 *     int32 [n_events+1] offset tables (a call is limited to < 2^31 hits and seeds).
 */
#ifndef DS_H_
#define DS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DS_VERSION 1

enum {
    DS_OK = 0,
    DS_E_ARG = -1,       /* NULL / negative / inconsistent argument, wrong struct_size                  */
    DS_E_NOGEOM = -2,    /* ds_upload_geometry has not been called on this handle                       */
    DS_E_WORKSPACE = -3, /* workspace pointer NULL or workspace_bytes smaller than ds_*_workspace_bytes */
    DS_E_CUDA = -4,      /* a CUDA runtime call failed (no device, launch error, out of memory)         */
    DS_E_LIMIT = -5,     /* ds_vertex_static: the call is larger than its fixed scratch (DS_STATIC_MAX_*) */
};

/* Ghost-killer architecture (BASELINE cfg0: 8 -> 32 -> 16 -> 1; the paper's own is 8 -> 14 -> 1).
 * Layer sizes are compile-time so that the network lives in registers / shared memory. */
#define DS_MLP_IN 8
#define DS_MLP_H1 32
#define DS_MLP_H2 16
#define DS_MLP_SINGLE_H 14 /* the paper's own ghost killer: one hidden layer of 14 neurons */

/* HLT1 line NNs on the vertices (P:277-P:285): four networks DS_LINE_IN -> DS_LINE_H -> 1 (inputs: reading A-33). */
#define DS_LINE_IN 16
#define DS_LINE_H 32
#define DS_N_LINES 4

/* S1 layout granularity: each (layer, y-sector) bin is cut into DS_XBINS equal x0 slices, see ds_layout. */
#define DS_XBINS 16
#define DS_MAX_SECTORS 16

typedef struct ds_handle ds_handle; /* opaque; owns the device copy of the MLP weights and the *_host staging buffers */

/* UT geometry and thin-magnet model (HOST, POD).  P:39 Fig. 2 (four planes X/U/V/X), P:93 (magnet point), A-1..A-3. */
typedef struct {
    size_t struct_size;    /* = sizeof(ds_geometry)                                                         */
    double z_layer[4];     /* plane z of UTaX, UTaU, UTbV, UTbX; used for the window predictions            */
    double dxdy[4];        /* tan(stereo angle): a strip measures x_hit(y) = x0 + y*dxdy (A-1)              */
    double x_half, y_half; /* sensitive half-sizes; y-sector s covers [-y_half + s*h, -y_half + (s+1)*h]    */
    double hole_half;      /* beam hole half-size (information only; not used by the kernels)               */
    int32_t n_sectors_y;   /* 1..DS_MAX_SECTORS                                                             */
    int32_t pad_;
    double sector_height;  /* h                                                                             */
    double z_seed;         /* z at which the SciFi seed state is given                                      */
    double z_ref;          /* z0 of the output state = UT midpoint                                  */
    double zmag_c[4];      /* z_mag = c0 + c1*ty^2 + c2*tx^2 + c3*qop^2 (A-3)                         */
    double kick;           /* K [GeV]: tx_UT = tx_seed - K*qop (thin-magnet kick, BASELINE cfg0)            */
} ds_geometry;

/* Ghost-killer weights (HOST, POD), row-major [out][in] (A-10, A-18). */
typedef struct {
    size_t struct_size;
    float W1[DS_MLP_H1][DS_MLP_IN], b1[DS_MLP_H1];
    float W2[DS_MLP_H2][DS_MLP_H1], b2[DS_MLP_H2];
    float W3[DS_MLP_H2], b3;
    float mu[DS_MLP_IN], inv_sigma[DS_MLP_IN]; /* input k is fed as (v_k - mu_k) * inv_sigma_k */
} ds_mlp;

/* The paper's ghost killer 8 -> 14 -> 1, row-major [out][in]: W3 acts on the hidden layer. */
typedef struct {
    size_t struct_size;
    float W1[DS_MLP_SINGLE_H][DS_MLP_IN], b1[DS_MLP_SINGLE_H];
    float W3[DS_MLP_SINGLE_H], b3;
    float mu[DS_MLP_IN], inv_sigma[DS_MLP_IN];
} ds_mlp_single;

/* Weights of the four line NNs (HOST, POD), row-major [net][out][in]; input k of every network is fed as
 * (v_k - mu_k) * inv_sigma_k.  Network order in the paper: K_S selection, Lambda selection, detached-vs-prompt
 * K_S, detached-vs-prompt Lambda; the library only evaluates them. */
typedef struct {
    size_t struct_size;
    float W1[DS_N_LINES][DS_LINE_H][DS_LINE_IN], b1[DS_N_LINES][DS_LINE_H];
    float W3[DS_N_LINES][DS_LINE_H], b3[DS_N_LINES];
    float mu[DS_LINE_IN], inv_sigma[DS_LINE_IN];
} ds_line_nets;

/* Algorithm parameters (HOST, POD, read at call time).  None of the values is printed in the paper. */
typedef struct {
    size_t struct_size;
    double w0_a, w0_b, w0_max;        /* first window half-width  min(w0_max, w0_a + w0_b*|qop|)  (A-5)   */
    double w1_a, w1_b;                /* refined window half-width w1_a + w1_b*|qop|              (A-5)  */
    double y_tol;                     /* a hit is y-compatible iff ymin - y_tol <= y_track <= ymax + y_tol      */
    double w_mag;                     /* weight of the magnet-point pseudo-measurement            (A-8)         */
    double chi2ndf_max, miss_penalty; /* candidate cut and score = chi2 + miss_penalty*(4 - n_hits) (A-9) */
    int32_t min_hits;                 /* minimum UT hits of a candidate, the UTbX hit included    (A-6)         */
    int32_t max_first_hits;           /* closest UTbX hits tried per seed, 1..DS_MAX_FIRST_HITS       */
    double mlp_thr;
    int32_t mlp_keep_above;           /* 1: keep iff score > thr (BASELINE cfg3); 0: keep iff score < thr */
    int32_t max_event_hits_hint;      /* expected upper bound of hits per event (0 = 4096): sizes the per-event shared-memory
                                         staging of the layout and tracking kernels (and with it the thread blocks per
                                         SM, so a tight bound is faster).  Events above it give the same results on
                                         slower global-memory paths.                                                */
    double doca_max, zv_min, zv_max;  /* vertex cuts (BASELINE cfg3)                                             */
    double m_pi, m_p, m_ks, m_lambda, dm_ks, dm_lambda; /* MeV                                                   */
    double n2_min;                    /* pairs with |d_a x d_b|^2 below this have no vertex       (A-14)        */
    /* Curved-track vertexing (P:255-P:269): x_i(z) = x_i + tx_i (z - z_ref) + gamma_i (z - z_ref)^2 (Eq. 4) with
     * gamma_i = -magnet_polarity * (gamma_c0 + gamma_c1 * qop_i / 1000) (Eq. 3; qop in 1/GeV, the parametrisation in
     * 1/MeV, A-27); closest approach by vtx_newton_iters Newton-Raphson steps from the straight-line solution (P:269:
     * three, A-28); the masses use the slopes at the vertex z.  magnet_polarity = 0: straight tracks, closed form. */
    double magnet_polarity, gamma_c0, gamma_c1;
    int32_t vtx_newton_iters;         /* 0..16                                                                  */
    int32_t clone_min_shared;         /* clone killing across seeds (A-31): found tracks of an event that share at
                                         least this many UT hits (same index, same layer) with a better track (smaller
                                         chi2 + miss_penalty*(4 - nhits), ties: earlier seed) are removed after S6;
                                         paper: 3 ("more than two"); 0 = off (the BASELINE configurations)              */
    int32_t dv1;                      /* 1: Dv1 triplet search (P:107-P:111, A-32): no first window -- every UTbX hit of
                                         the seed's y-compatible sectors starts a candidate, which needs a UTaX hit within
                                         the refined window of the line through that hit and the magnet point; stereo
                                         hits, fit and choice as Dv0.  0: Dv0 (the BASELINE configurations)               */
    int32_t mlp_fast_math;            /* 1: sigmoid by the fast intrinsics __expf / __fdividef as in the paper and no
                                         fp64 re-evaluation next to the threshold; scores then differ from an IEEE
                                         evaluation by a few 1e-7 absolute and a keep decision on the threshold may flip.
                                         0 (default): IEEE, the parity-tested path                                     */
} ds_params;
#define DS_MAX_FIRST_HITS 10

/* UT hits, SoA, DEVICE (BASELINE cfg0: "x at y=0, z, ymin, ymax, weight" fp32 + int32 id).
 * id = seq | sector << 20 | layer << 24 (A-2); layer 0..3 = UTaX, UTaU, UTbV, UTbX; sector < n_sectors_y.
 * Precondition: [ymin, ymax] of a hit lies inside its sector's y range; no NaN.  ids are unique inside an event
 * (only the order of hits with equal (layer, sector, x0, id) depends on it). */
typedef struct {
    const float *x0, *z, *ymin, *ymax, *w;
    const int32_t *id;
    int64_t n;
} ds_hits;

/* Unmatched SciFi seeds, SoA, DEVICE: state (x, y, tx, ty, q/p) at z_seed, optional seed chi2 (NULL
 * = 0, A-11). */
typedef struct {
    const float *x, *y, *tx, *ty, *qop, *chi2;
    int64_t n;
} ds_seeds;

/* Downstream tracks, SoA, DEVICE, one slot per seed in seed order (dense).  State (x, y, tx, ty, q/p) at z_ref and
 * chi2; nhits; hit[4*s + layer] = index of the chosen hit in the caller's (unsorted) hit arrays or -1;
 * found = 1 if a candidate survived; score = ghost-killer output; keep = found && (score passes mlp_thr).
 * Slots with found = 0 hold zeros, hit = -1, keep = 0. */
typedef struct {
    float *x, *y, *tx, *ty, *qop, *chi2, *score;
    int32_t *nhits, *hit, *found, *keep;
    int64_t n;
} ds_tracks;

/* Two-track vertices, SoA, DEVICE.  Event e owns entries [offsets[e], offsets[e+1]), sorted by (ia, ib).
 * ia / ib = seed index of the positive / negative track.  flags bit0: |m_pipi - m_ks| < dm_ks, bit1: |m_ppi -
 * m_lambda| < dm_lambda.  Entries at positions >= capacity are not written; overflow[0] = how many were dropped;
 * n_per_event and offsets always hold the true counts. */
typedef struct {
    int32_t *evt, *ia, *ib;
    float *x, *y, *z, *doca, *m_pipi, *m_ppi;
    int32_t *flags;
    int32_t *n_per_event; /* [n_events]     */
    int64_t *offsets;     /* [n_events + 1] */
    int32_t *overflow;    /* [1]            */
    int64_t capacity;
} ds_vertices;

/* S1 output (DEVICE): the event-batched sorted SoA.  Event e keeps its slice [hit_offsets[e], hit_offsets[e+1]).
 * Inside it hits are ordered by (layer, sector, x0, id).  perm[p] = caller's index of the hit now at p.
 * n_bins = 4 * n_sectors_y * DS_XBINS; bin (layer*n_sectors_y + sector)*DS_XBINS + xb, with
 * xb = clamp(floor((x0 + X) * DS_XBINS / (2X)), 0, DS_XBINS-1) in fp32 and X = (float)(x_half + y_half*max|dxdy|);
 * bin_offsets[e*(n_bins+1) + b] = first position of bin b relative to hit_offsets[e]; entry n_bins = event size. */
typedef struct {
    float *x0, *z, *ymin, *ymax, *w;
    int32_t *id, *perm;
    int32_t *bin_offsets;
    int64_t n;
} ds_layout_out;

/* ---- handle ------------------------------------------------------------------------------------------------- */

/* Create a handle bound to CUDA device `cuda_device`.  DS_E_CUDA if there is no such device. */
int ds_create(ds_handle **h, int cuda_device);
void ds_destroy(ds_handle *h);
const char *ds_error_string(int code);
int ds_version(void);

/* Copy geometry and ghost-killer weights (both HOST) into the handle; may be called again to replace them.
 * Synchronous.  DS_E_ARG on a wrong struct_size, n_sectors_y outside 1..DS_MAX_SECTORS or a non-positive height. */
int ds_upload_geometry(ds_handle *h, const ds_geometry *g, const ds_mlp *m);

/* Replace the handle's ghost killer by the paper's single-hidden-layer network (HOST weights; synchronous).  It stays in
 * use by ds_reconstruct / ds_ghost_killer / ds_process_host until ds_upload_geometry is called again (which installs its
 * 8 -> 32 -> 16 -> 1 network).  DS_E_ARG on a wrong struct_size. */
int ds_upload_mlp_single(ds_handle *h, const ds_mlp_single *m);

/* ---- S1: layout (P:109-P:111 "UT hits are grouped into different Y sectors"; BASELINE north_star (1)) -------- */

/* Segmented sort of every event's hits by (layer, sector, x0, id) plus the per-event bin table (see ds_layout_out).
 * One thread block per event: the input arrays staged in shared memory by bulk async copies (16-byte aligned array
 * pointers; otherwise by ordinary loads), bin histogram, exclusive scan, rank inside each bin, gathered coalesced stores.
 * Events with more hits than params->max_event_hits_hint (or than fit in shared memory) take an O(n^2) path that
 * is slower but gives the same result.  hit_offsets: DEVICE int32 [n_events+1], non-decreasing, [0] = 0,
 * [n_events] = hits->n.  No workspace. */
int ds_layout(ds_handle *h, const ds_hits *hits, const int32_t *hit_offsets, int n_events, const ds_params *p,
              ds_layout_out *out, void *cuda_stream);

/* ---- S2: seed extrapolation (P:93 magnet point, P:95 first window; thin-kick model of BASELINE cfg0) ---------- */

/* Per seed, 12 doubles (DEVICE out[12*s + k]): z_m, x_m, y_m, y_0..y_3 (track y at the four planes), tx_pred,
 * xc_3 (first-window centre in UTbX), w0, w1, 0.  ds_reconstruct computes the same values in registers; this entry
 * exposes the step on its own. */
int ds_extrapolate(ds_handle *h, const ds_seeds *seeds, const ds_params *p, double *out, void *cuda_stream);

/* ---- S1..S7: ds_reconstruct ------------------------------------------------------------------------------------ */

/* Bytes of DEVICE workspace ds_reconstruct needs for a call of this size (the sorted SoA, permutation and bin
 * tables of S1 for the events that take the two-kernel path, one flag per event).  Alignment required: 256 B. */
size_t ds_workspace_bytes(const ds_handle *h, int n_events, int64_t n_hits, int64_t n_seeds);

/* Layout (S1) -> per seed: extrapolate (S2), first window in UTbX keeping the <= max_first_hits closest hits (S3,
 * P:95), per first hit the refined windows in UTaX/UTaU/UTbV keeping the closest 1/2/2 (S4),
 * weighted line fit + chi2 of every combination with the magnet point as pseudo-measurement (S5, A-8), best
 * candidate by score with id tie-breaks (S6) -> ghost-killer MLP score and keep flag (S7).
 * All deciding arithmetic is fp64 in registers; the MLP is fp32 (a decision within 1e-3 of the threshold is
 * re-evaluated in fp64).  seed_offsets: DEVICE int32 [n_events+1].
 * Launches: with dv1 = 0, S1..S6 run as one kernel per event that sorts the event's hits in shared memory and searches
 * the copy it holds; events above the staging capacity derived from max_event_hits_hint (and every event when the hint
 * is so large that fewer than two such blocks fit an SM, or with dv1 = 1) take a layout kernel and a search kernel through
 * the workspace.  The results do not depend on which path an event takes.  Then clone killing (clone_min_shared > 0) and
 * the ghost killer. */
int ds_reconstruct(ds_handle *h, const ds_hits *hits, const ds_seeds *seeds, const int32_t *hit_offsets,
                   const int32_t *seed_offsets, int n_events, const ds_params *p, ds_tracks *out, void *workspace,
                   size_t workspace_bytes, void *cuda_stream);

/* Clone killing alone (A-31; needs params->clone_min_shared > 0): removes from `trk` (x..chi2, nhits, hit, found
 * are read) every found track that shares enough hits with a better one; its slot becomes the "not found" record
 * (zeros, hit = -1, found = score = keep = 0).  ds_reconstruct does the same between S6 and S7. */
int ds_clone_kill(ds_handle *h, const int32_t *seed_offsets, int n_events, const ds_params *p, ds_tracks *trk,
                  void *cuda_stream);

/* S7 alone: re-score tracks already in `trk` (reads x..chi2, found and the seeds' qop / chi2; writes score, keep). */
int ds_ghost_killer(ds_handle *h, const ds_seeds *seeds, const ds_params *p, ds_tracks *trk, void *cuda_stream);

/* ---- S8..S10: ds_vertex (P:253-P:269 with gamma = 0, A-20; P:279 opposite charges; cuts of BASELINE cfg3) ------- */

size_t ds_vertex_workspace_bytes(const ds_handle *h, int n_events, int64_t n_seeds);

/* Per event: all (positive, negative) pairs of tracks with keep = 1; closed-form closest approach of the two
 * straight lines (or, with magnet_polarity != 0, Newton-Raphson on the two parabolas of Eq. 4), midpoint vertex, DOCA,
 * m_pipi, m_ppi (proton = larger momentum, A-15), cuts; passing pairs are
 * written in (ia, ib) order: count -> exclusive scan over events -> write.  Only x, y, tx, ty, qop, keep of `trk`
 * are read.  Deciding arithmetic in fp64. */
int ds_vertex(ds_handle *h, const ds_tracks *trk, const int32_t *seed_offsets, int n_events, const ds_params *p,
              ds_vertices *out, void *workspace, size_t workspace_bytes, void *cuda_stream);

/* ---- ds_vertex without any allocation: the scratch is a fixed device array inside the library ------------------- */

/* For callers that cannot allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
 * ds_vertex_static is ds_vertex (same kernels, same output, bit for bit) with its workspace in a file-scope
 * `static __device__` array of DS_STATIC_SCRATCH_BYTES (4.03 MiB) that every GPU that loads the library holds until the
 * process exits.  The caller passes inputs and outputs only.  It calls no cudaMalloc / cudaFree / allocating routine (the
 * ds_profile_* event pairs are not recorded for it).
 * Limits: n_events <= DS_STATIC_MAX_EVENTS and trk->n <= DS_STATIC_MAX_SEEDS, else DS_E_LIMIT (nothing is launched).
 * Sharing: there is ONE array per device.  Every call uses it and finds the previous call's contents (what has to start
 * at zero is cleared by the call itself, on its stream).  Calls that overlap on the GPU -- two streams, two handles or
 * two threads on the same device -- race on it and corrupt each other's vertex lists: keep them on one stream, or order
 * them with events.
 * ds_vertex_static_setup resolves the array's device address for the handle's device (once per device; cheap when
 * repeated).  ds_vertex_static does the same on its first call for a device; call the set-up beforehand if that first
 * call must not touch the runtime (e.g. under stream capture). */
#define DS_STATIC_MAX_EVENTS 2048
#define DS_STATIC_MAX_SEEDS 524288
#define DS_STATIC_SCRATCH_BYTES 4227072
int ds_vertex_static_setup(ds_handle *h);
int ds_vertex_static(ds_handle *h, const ds_tracks *trk, const int32_t *seed_offsets, int n_events, const ds_params *p,
                     ds_vertices *out, void *cuda_stream);

/* ---- HLT1 line NNs on the vertices (P:277-P:285, A-33) ------------------------------------------- */

/* Copy the four weight sets (HOST) into the handle.  Synchronous; may be called again. */
int ds_upload_line_nets(ds_handle *h, const ds_line_nets *nets);

/* For every vertex k written by ds_vertex (k < min(offsets[n_events], capacity), read on the device): the 16 inputs
 * -- positive track (tx, ty, q/p, chi2), negative track (tx, ty, q/p, chi2) from `trk` via ia / ib, vertex (x, y, z,
 * DOCA), parent (tx, ty, p [GeV], pT [GeV]; momentum sum of the two tracks) -- through the four networks (ReLU hidden
 * layer, sigmoid): scores[4*k + i] (DEVICE float [4*capacity]) and bits[k] = sum_i 2^i [score_i > threshold] (DEVICE
 * int32 [capacity]); the paper's threshold is 0.5.  DS_E_NOGEOM if no weights were uploaded. */
int ds_lines(ds_handle *h, const ds_tracks *trk, const ds_vertices *vtx, int n_events, double threshold, float *scores,
             int32_t *bits, void *cuda_stream);

/* ---- whole path from HOST buffers ------------------------------------------------------------------------------ */

/* ds_reconstruct + ds_vertex with every array pointer (hits, seeds, offsets, tracks, vertices) in HOST memory
 * (pinned memory makes the copies asynchronous).  Device buffers are owned by the handle and grown on demand.
 * Copies inputs host->device, runs both calls, copies tracks and the first min(total, capacity) vertices back,
 * and synchronises.  *n_vertices_total (HOST, may be NULL) receives the true number of passing pairs. */
int ds_process_host(ds_handle *h, const ds_hits *hits, const ds_seeds *seeds, const int32_t *hit_offsets,
                    const int32_t *seed_offsets, int n_events, const ds_params *p, ds_tracks *out_tracks,
                    ds_vertices *out_vertices, int64_t *n_vertices_total, void *cuda_stream);

/* ---- per-kernel device timing (measurement aid; no effect on results) ------------------------------------------ */

/* Kernels of the path.  DS_K_EVENT = S1..S6 in one kernel (ds_reconstruct, dv1 = 0); DS_K_LAYOUT / DS_K_TRACK = the same
 * steps as two kernels (ds_layout; dv1 = 1; events DS_K_EVENT leaves over -- launched after it, empty if there are none). */
enum { DS_K_LAYOUT = 0, DS_K_TRACK, DS_K_MLP, DS_K_VTX_COUNT, DS_K_VTX_SCAN, DS_K_VTX_WRITE, DS_K_CLONE, DS_K_LINES, DS_K_EVENT, DS_K_COUNT };

typedef struct {
    size_t struct_size;
    double ms[DS_K_COUNT];        /* summed device time of the kernel's launches, CUDA events on the launching stream */
    int64_t launches[DS_K_COUNT]; /* number of launches                                                             */
} ds_profile;

/* on != 0: every kernel launched through this handle from now on is bracketed by a pair of CUDA events recorded on
 * the stream it is launched on.  Off by default. */
int ds_profile_enable(ds_handle *h, int on);
/* Waits for all recorded events (blocks the calling thread until the bracketed kernels have finished), adds their
 * elapsed times into *out (HOST) and forgets them.  Counters start from zero at every call. */
int ds_profile_read(ds_handle *h, ds_profile *out);
/* Measured fp64 FMA throughput of the handle's device in TFLOP/s (a register-resident DFMA loop on every SM, timed with
 * CUDA events; blocks the calling thread for a few milliseconds).  The denominator of the ALU fraction bench.py reports
 * for the vertex kernels on BASELINE configs[3]. */
int ds_measure_dfma_peak(ds_handle *h, double *tflops);

/* Name of kernel k ("k_layout", ...), NULL if k is out of range. */
const char *ds_kernel_name(int k);

#ifdef __cplusplus
}
#endif
#endif /* DS_H_ */

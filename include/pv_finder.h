/* pv_finder.h -- C ABI of the B200-native primary-vertex (PV) finder hot path of arXiv:2412.14966.
 *
 * One call, pv_find(), runs the five steps the paper lists ("P:Lnn" = PAPER.md line nn)
 * plus the post-fit cleanup over a batch of independent events ("events are independent
 * from each other"), entirely in hand-written CUDA kernels for sm_100a:
 *
 *   a1 project  z_poca (Eq. 1), sigma_poca (Eq. 3)
 *   a2 fill     per-event z-histogram of Gaussian bin integrals, int32 fixed point (2^20 = 1 track)
 *   a3 peaks    proto-clusters, dip search, z-ordered splitting, seed z (Eq. 4-5)
 *   a4 assign   bin -> closest seed via partition points, removal of under-populated seeds
 *   a5 fit      adaptive Tukey-weighted Newton-Raphson vertex fit (Eq. 6-18)
 *   a6 cleanup  duplicate removal, min tracks, beamline distance (Table 2)
 *
 * The readings taken where the paper is silent are listed in DESIGN.md section "Readings".
 *
 * Conventions
 *   - No torch / C++ types: plain pointers and sizes.  Every pointer says HOST or DEVICE below.
 *   - The caller owns every buffer.  pv_find never allocates, frees or synchronises; all work is
 *     enqueued on `stream` (a cudaStream_t passed as void*; NULL = the legacy default stream).
 *   - Return value: 0 (PV_OK) or a negative PV_E_* code.  Data-dependent problems never fail the
 *     call; they set bits in event_status[e].
 *   - Device base pointers must be 4-byte aligned; per-event offsets need no alignment.
 *   - Thread safety: calls on different streams are independent provided they use different
 *     workspaces and output buffers (launches are serialised by a lock inside the library).  The two
 *     diagnostics pv_last_launch_info / pv_kernel_timing are process-global: meaningful only while one
 *     thread is calling.
 */
#ifndef PV_FINDER_H
#define PV_FINDER_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* All lengths in mm.  Index 0 = pp region (z >= z_split), 1 = p-gas / SMOG2 region (z < z_split). */
typedef struct pv_params {
  float z_min, z_max, dz;               /* histogram range and bin size: -550, 300, 0.25 */
  float z_split;                        /* region boundary: -300                          Table 2 */
  float beam_x, beam_y, beam_tx, beam_ty; /* beamline position and direction at z = 0 */
  float max_sigma_poca[2];              /* max sigma_poca to enter the histogram: 1.5, 10  P:L129, Table 2
                                           (6 max_sigma_poca / dz + 4 <= 3072 bins, and with PV_FILL_TEMPLATE the
                                           window of the widest class as well, else PV_E_PARAM) */
  float min_bin_content;                /* proto-cluster bin threshold [tracks]: 0.25      P:L135 (value: reading R-4) */
  float min_dip;                        /* significance of an extremum [tracks]: 0.75      P:L135 (value: reading R-4) */
  float min_cluster_integral[2];        /* min track integral of a seed cluster: 2.5, 1.75 Table 2 */
  int32_t min_tracks_seed[2];           /* min tracks associated to a seed: 3, 2 */
  int32_t min_tracks_pv[2];             /* min tracks in a fitted PV: 4, 3                 Table 2 */
  float chi2_max;                       /* Tukey cut-off: 12 (INFINITY = unit weights)     Eq. 18 */
  int32_t max_iter;                     /* max fit iterations: 10 (1..16) */
  float conv_dchi2, conv_dz;            /* convergence: |dchi2| < 0.01 and |dz| < 0.001 mm P:L225 */
  float merge_ratio;                    /* duplicate iff dz^2/(Czz1+Czz2) < 25 */
  float max_beam_dist;                  /* pp vertices farther than 0.3 mm are discarded */
  int32_t max_vtx_per_event;            /* output stride per event, 1..PV_MAX_VTX (default 32) */
  int32_t flavour;                      /* PV_FLAVOUR_EXPLICIT (default): one track one vertex, Tukey weights   P:L163, Eq. 18
                                           PV_FLAVOUR_MULTIVERTEX: every track to every vertex, weights Eq. 19 */
  float chi2_window;                    /* multi-vertex flavour: a track takes part in a vertex fit iff its chi2 at
                                           the seed position is below this: 25      P:L384 (value: reading R-13) */
  int32_t split_mode;                   /* proto-cluster splitting: PV_SPLIT_Z_ORDERED (default, the paper's GPU
                                           variant: minima in z order) or PV_SPLIT_RECURSIVE (its x86 variant: the
                                           smallest minimum between the two largest maxima, recursively; reading R-16) */
  int32_t fill_mode;                    /* histogram fill: PV_FILL_POLYNOMIAL (default, the paper's GPU variant: a
                                           polynomial approximation of the cumulative density per track, reading R-6) or
                                           PV_FILL_TEMPLATE (its x86 variant: "a finite set of template histograms,
                                           selected based on the value of sigma_poca"; reading R-17: classes
                                           sigma_k = 0.08 dz 2^(k/4) x 8 positions of z_poca inside its bin) */
} pv_params;

enum { PV_FLAVOUR_EXPLICIT = 0, PV_FLAVOUR_MULTIVERTEX = 1 };
enum { PV_SPLIT_Z_ORDERED = 0, PV_SPLIT_RECURSIVE = 1 };
enum { PV_FILL_POLYNOMIAL = 0, PV_FILL_TEMPLATE = 1 };

enum {
  PV_OK = 0,
  PV_E_NULL = -1,       /* a required pointer is NULL */
  PV_E_PARAM = -2,      /* invalid parameter (dz <= 0, range not a whole number of bins, too many bins, ...) */
  PV_E_WORKSPACE = -3,  /* workspace too small */
  PV_E_CUDA = -4,       /* a CUDA runtime call or kernel launch failed (see pv_last_cuda_error) */
  PV_E_SIZE = -5,       /* negative n_events / n_tracks, or a host staging capacity exceeded */
  PV_E_STATIC_LIMIT = -6 /* pv_find_static only: the batch needs more scratch than PV_STATIC_WORKSPACE_BYTES */
};

/* Compile-time limits of this build. */
enum {
  PV_MAX_BINS = 4096,          /* (z_max - z_min) / dz must be <= this */
  PV_MAX_VTX = 32,             /* max_vtx_per_event must be <= this */
  PV_MAX_TRACKS_PER_EVENT = 2047, /* larger events get PV_EVT_TOO_MANY_TRACKS and zero vertices */
  PV_FIXED_ONE = 1 << 20,      /* histogram fixed-point unit: the full mass of one track */
  PV_STATIC_WORKSPACE_BYTES = 16 << 20 /* scratch built into the library for pv_find_static (16 MiB per GPU) */
};

/* event_status bit flags */
enum {
  PV_EVT_TOO_MANY_TRACKS = 1,  /* n_tracks(e) > PV_MAX_TRACKS_PER_EVENT: event skipped, n_vtx = 0 */
  PV_EVT_VTX_OVERFLOW = 2,     /* more seed clusters than max_vtx_per_event: the first max_vtx in z are kept */
  PV_EVT_SINGULAR_FIT = 4,     /* a vertex fit had < 2 active tracks or a non-positive pivot: that vertex is dropped */
  PV_EVT_RECORD_OVERFLOW = 8   /* the workspace cannot hold the event's track records: the multi-vertex flavour needed
                                  more (track, vertex) records than 2 per track of the batch, or n_tracks given to
                                  pv_find is smaller than offsets[n_events]: the event is left without vertices */
};

/* Fill *p with the paper's values (citations on the struct above).  p: HOST.  Returns PV_OK / PV_E_NULL. */
int pv_params_default(pv_params* p);

/* Number of histogram bins implied by p (lrint((z_max - z_min) / dz)), or a negative PV_E_* if p is invalid. */
int pv_nbins(const pv_params* p);

/* Bytes of DEVICE workspace pv_find needs for a batch of this size: 256 B of counters, one 16-byte seed
 * record per (event, vertex slot) and one 32-byte fit-ready track record per track (tracks sorted by seed,
 * in the seed's local frame with W = V^-1 at the seed position) handed from the seed kernel to the
 * fit kernel.  The multi-vertex flavour lists a track once per vertex candidate in its chi2 window: it takes two
 * records per track and 8 more bytes per track (the largest weight of the track and its vertex).  The histograms
 * live in shared memory ("one block per event").  With PV_FILL_TEMPLATE the workspace also holds the table of
 * template histograms (tens of KB; rebuilt by a small kernel at every call: the library keeps no device state).
 * bytes: HOST out. */
int pv_workspace_bytes(int n_events, long long n_tracks, const pv_params* p, size_t* bytes);

/* The hot path a1..a6 over a batch.
 *
 * Inputs (DEVICE, read-only, fp32 SoA, length T = offsets[n_events]; "same data members of all
 * tracks contiguous"): track state x, y, z, tx, ty and the diagonal of its covariance
 * var_x, var_y, var_tx, var_ty (Eq. 2, diagonal form).
 *   offsets   DEVICE int32[n_events + 1], offsets[0] = 0, non-decreasing; event e owns tracks
 *             [offsets[e], offsets[e+1]).
 *   n_tracks  T, as known to the host (only used for validation and sizing; the kernel reads offsets).
 *   params    HOST, copied by value at call time.
 * Outputs (DEVICE, caller-allocated):
 *   vtx_pos      float[n_events][max_vtx][3]   x, y, z of each PV, ordered in z
 *   vtx_cov      float[n_events][max_vtx][6]   upper triangle xx, xy, xz, yy, yz, zz of C (Eq. 14)
 *   vtx_chi2     float[n_events][max_vtx]      sum_i w_i chi2_i of the last iteration (Eq. 6)
 *   vtx_ntracks  int32[n_events][max_vtx]      tracks with w_i > 0 in the last iteration
 *   vtx_niter    int32[n_events][max_vtx]      Newton iterations done
 *   n_vtx        int32[n_events]               PVs found; the first n_vtx[e] slots of event e hold them, the
 *                                              other slots of the event are scratch (pre-cleanup seeds)
 *   trk_weight   float[T]                      Tukey weight w_i of the last iteration (Eq. 18); 0 if unassigned
 *   trk_vertex   int32[T]                      index of the track's PV within its event, -1 = none
 *   event_status uint32[n_events]              PV_EVT_* flags
 *   (trk_weight / trk_vertex also serve as per-track scratch during the call.)
 * workspace: DEVICE, >= pv_workspace_bytes(n_events, n_tracks, params) bytes, 16-byte aligned; scratch.
 * stream: cudaStream_t.
 */
int pv_find(const float* x, const float* y, const float* z, const float* tx, const float* ty,
            const float* var_x, const float* var_y, const float* var_tx, const float* var_ty,
            const int32_t* offsets, int n_events, long long n_tracks, const pv_params* params,
            float* vtx_pos, float* vtx_cov, float* vtx_chi2, int32_t* vtx_ntracks, int32_t* vtx_niter,
            int32_t* n_vtx, float* trk_weight, int32_t* trk_vertex, uint32_t* event_status,
            void* workspace, size_t workspace_bytes, void* stream);

/* Optional x-tx and y-ty elements of the track covariance (Eq. 2: V_xx(z) = V_xx + 2 dz V_xtx + dz^2 V_txtx;
 * x and y are uncorrelated in the simplified track fit).  DEVICE arrays of length T; a NULL struct or
 * member means 0 (the diagonal covariance pv_find assumes).  They enter wherever Eq. 2 is evaluated: W of the
 * vertex fit, the chi2 of the multi-vertex flavour, the IP chi2; sigma_poca (Eq. 3) uses V_xx alone. */
typedef struct pv_track_cov {
  const float* cov_xtx;
  const float* cov_yty;
} pv_track_cov;

/* Impact parameter of every track w.r.t. the PVs of its event ("the distance of closest approach of a track to
 * a vertex, called impact parameter (IP) ... the IP chi2, which is the chi2 difference of a PV reconstructed with and
 * without the track under consideration").  For each track the vertex of its event with the smallest IP chi2 is
 * taken (ties: lower index); the vertex is treated as not containing the track:
 *   r = residual of Eq. 9 at the vertex z, IP = distance of the straight line to the vertex position,
 *   IP chi2 = r^T (V + H C H^T)^-1 r, V from Eq. 2 (diagonal) at the vertex z, H of Eq. 12, C the vertex covariance.
 * Inputs: the track arrays and offsets of pv_find (DEVICE), and its outputs vtx_pos / vtx_cov / n_vtx (DEVICE,
 * stride params->max_vtx_per_event).  Outputs (DEVICE, caller-allocated, length T): ip [mm], ip_chi2, ip_vertex
 * (index within the event); -1 in all three when the event has no vertex usable for the track.
 * cov: optional covariance cross terms (HOST struct of DEVICE pointers, may be NULL).
 * One kernel on `stream`; never allocates or synchronises. */
int pv_track_ip(const float* x, const float* y, const float* z, const float* tx, const float* ty,
                const float* var_x, const float* var_y, const float* var_tx, const float* var_ty,
                const int32_t* offsets, int n_events, long long n_tracks, const pv_params* params,
                const float* vtx_pos, const float* vtx_cov, const int32_t* n_vtx,
                float* ip, float* ip_chi2, int32_t* ip_vertex, const pv_track_cov* cov /* nullable */, void* stream);

/* Parity taps: every member is a nullable DEVICE pointer; no global state. */
typedef struct pv_debug {
  int32_t* hist;          /* [n_hist_events][nbins]: histogram of the first n_hist_events events (a2) */
  int32_t n_hist_events;
  float* z_poca;          /* [T] (a1) */
  float* sigma_poca;      /* [T] (a1) */
  int32_t* trk_bin;       /* [T] central bin, -1 = not assignable (a1) */
  int32_t* n_seeds_raw;   /* [E] clusters found by the peak search before truncation / removal (a3) */
  int32_t* n_seeds;       /* [E] seeds after the removal loop (a4) */
  float* seed_z;          /* [E][max_vtx] (a3, Eq. 4-5) */
  int32_t* seed_bins;     /* [E][max_vtx][3] begin, end, peak (a3) */
  int32_t* trk_seed;      /* [T] pre-cleanup assignment (a4) */
  float* seed_pos;        /* [E][max_vtx][3] fitted position per seed, pre-cleanup (a5) */
  float* seed_cov;        /* [E][max_vtx][6] */
  float* seed_chi2;       /* [E][max_vtx] */
  int32_t* seed_ntrk;     /* [E][max_vtx] */
  int32_t* seed_niter;    /* [E][max_vtx], -1 = singular */
  int32_t* seed_fate;     /* [E][max_vtx] final vertex index, or -1 singular, -2 merged, -3 min tracks, -4 beam distance */
} pv_debug;

/* Same as pv_find, additionally writing the taps selected in *dbg (HOST struct of DEVICE pointers). */
int pv_find_debug(const float* x, const float* y, const float* z, const float* tx, const float* ty,
                  const float* var_x, const float* var_y, const float* var_tx, const float* var_ty,
                  const int32_t* offsets, int n_events, long long n_tracks, const pv_params* params,
                  float* vtx_pos, float* vtx_cov, float* vtx_chi2, int32_t* vtx_ntracks, int32_t* vtx_niter,
                  int32_t* n_vtx, float* trk_weight, int32_t* trk_vertex, uint32_t* event_status,
                  void* workspace, size_t workspace_bytes, void* stream, const pv_debug* dbg);

/* pv_find with the covariance cross terms of Eq. 2 (cov, nullable) and, optionally, the parity taps (dbg, nullable):
 * pv_find(...) == pv_find_ext(..., NULL, NULL). */
int pv_find_ext(const float* x, const float* y, const float* z, const float* tx, const float* ty,
                const float* var_x, const float* var_y, const float* var_tx, const float* var_ty,
                const int32_t* offsets, int n_events, long long n_tracks, const pv_params* params,
                float* vtx_pos, float* vtx_cov, float* vtx_chi2, int32_t* vtx_ntracks, int32_t* vtx_niter,
                int32_t* n_vtx, float* trk_weight, int32_t* trk_vertex, uint32_t* event_status,
                void* workspace, size_t workspace_bytes, void* stream, const pv_track_cov* cov, const pv_debug* dbg);

/* pv_find for callers that have no device memory to give as a workspace and may not allocate any.
 *
 * Who that is: a plug-in inside a host framework that took the GPU's memory at start-up and hands out slices of its
 * own arena only to its own algorithms (the trigger framework the paper runs in works like this, and so does any
 * service with a memory budget fixed at launch), so that a cudaMalloc from a third-party library either fails or
 * breaks the budget; an event loop with a latency bound, whose house rules forbid cudaMalloc / cudaFree after
 * initialisation because both may synchronise the whole device and take an unbounded time; and a plain C caller
 * that simply has no device allocator at hand beyond the buffers it was given for inputs and outputs.
 *
 * Same arguments, same kernels and bit-for-bit the same results as pv_find, except that there is no workspace
 * argument: the scratch (counters, seed records, fit-ready track records, pv_workspace_bytes() of them) lives in an
 * array of PV_STATIC_WORKSPACE_BYTES = 16 MiB that is part of the library's device image.  Every GPU on which the
 * library's kernels are loaded holds those 16 MiB until the process exits, whether or not this entry is ever called.
 * Inputs and outputs are still the caller's DEVICE buffers.
 *
 * Limit: pv_workspace_bytes(n_events, n_tracks, params) must be <= PV_STATIC_WORKSPACE_BYTES, else nothing is
 * enqueued and PV_E_STATIC_LIMIT is returned.  With the default parameters that is about 3 400 events of the paper's
 * mu = 5 mix (117 tracks per event; 256 + 512 B per event + 36 B per track) in the explicit flavour and about 1 800
 * in the multi-vertex flavour (76 B per track) -- several of the paper's batches of "several hundred events".
 * Larger batches: split them, or use pv_find with a workspace of your own.
 *
 * The call makes no cudaMalloc / cudaFree / cudaMallocAsync and calls no library routine that allocates device
 * memory; it refuses to run while pv_kernel_timing(1) is on (PV_E_PARAM), because the timing events would have to be
 * created.  The first call on each device looks up the device address of the array (once per device, with that device
 * current; the caller must have made the device of its buffers current, as for every entry of this header) and, like
 * any first launch, lets the CUDA runtime load the kernels: make that first call during initialisation, before any
 * stream capture and outside the latency-critical loop.
 *
 * Sharing: all calls on one device use the same array, from every thread and stream of the process.  Calls ordered
 * on one stream (or ordered by events) are safe; two calls that can overlap on the GPU race on the scratch and give
 * wrong results without any error.  The array keeps whatever the previous call left in it; no result depends on
 * that: each call clears the counters that must start at zero on `stream` before its first kernel, and takes its
 * results only from records it has written itself. */
int pv_find_static(const float* x, const float* y, const float* z, const float* tx, const float* ty,
                   const float* var_x, const float* var_y, const float* var_tx, const float* var_ty,
                   const int32_t* offsets, int n_events, long long n_tracks, const pv_params* params,
                   float* vtx_pos, float* vtx_cov, float* vtx_chi2, int32_t* vtx_ntracks, int32_t* vtx_niter,
                   int32_t* n_vtx, float* trk_weight, int32_t* trk_vertex, uint32_t* event_status, void* stream);

/* ---- host-buffer entries (the paper's host pipeline: "several streams ... each processing a batch",
 * host->device copies overlapped with compute).  A pv_host_ctx owns device buffers, workspaces, streams and events
 * sized for at most max_events / max_tracks (no host staging: the caller's buffers are copied from and to directly, so
 * they should be pinned, see pv_host_register; pageable memory works but the copies then serialise).
 * pv_find_host() takes HOST pointers everywhere (same meaning and layout as pv_find), splits the batch into n_chunks
 * (1..256) contiguous event ranges whose track counts ramp up and down as 1, 2, 4, 8, 8, ..., 8, 4, 2, 1 (the first
 * kernels start after a short copy, the last results leave after a short one), and for each enqueues H2D copies ->
 * pv_find -> D2H copies on one of the context's streams.  It returns after all results are in the caller's host arrays (it synchronises its
 * own streams only, also on every error path).  `offsets` is validated on the host (offsets[0] = 0, non-decreasing,
 * offsets[n_events] <= max_tracks; else PV_E_SIZE).  Both flavours and both splitting variants are supported (the
 * context is sized for the flavour given at creation); the covariance cross terms of pv_find_ext are not part of
 * these entries. */
typedef struct pv_host_ctx pv_host_ctx;
int pv_host_ctx_create(pv_host_ctx** ctx, int max_events, long long max_tracks, const pv_params* params,
                       int n_streams);
int pv_host_ctx_destroy(pv_host_ctx* ctx);
int pv_find_host(pv_host_ctx* ctx,
                 const float* x, const float* y, const float* z, const float* tx, const float* ty,
                 const float* var_x, const float* var_y, const float* var_tx, const float* var_ty,
                 const int32_t* offsets, int n_events, const pv_params* params,
                 float* vtx_pos, float* vtx_cov, float* vtx_chi2, int32_t* vtx_ntracks, int32_t* vtx_niter,
                 int32_t* n_vtx, float* trk_weight, int32_t* trk_vertex, uint32_t* event_status,
                 int n_chunks);

/* One PV as pv_find_host_compact returns it: the fields of pv_find's vertex arrays side by side (48 bytes). */
typedef struct pv_vertex {
  float pos[3];                 /* x, y, z */
  float cov[6];                 /* xx, xy, xz, yy, yz, zz (Eq. 14) */
  float chi2;
  int32_t ntracks, niter;
} pv_vertex;

/* pv_find_host with a compact read-back: pv_find's fixed-stride vertex arrays are 6/7 scratch at mu = 5 (5 PVs in 32
 * slots), so the PVs of each chunk are packed on the device (exclusive scan of n_vtx + gather, two small kernels per
 * chunk) and only sum(n_vtx) records cross PCIe; the per-track vertex index comes back as int8 (an event holds at
 * most PV_MAX_VTX = 32 PVs).  HOST outputs:
 *   vertices   pv_vertex[vtx_capacity]   the PVs of event e are vertices[vtx_begin[e] .. vtx_begin[e+1]), ordered in z;
 *                                        PV_E_SIZE if the batch holds more than vtx_capacity PVs
 *   vtx_begin  int32[n_events + 1]       exclusive prefix sum of n_vtx
 *   n_vtx, trk_weight, event_status      as pv_find
 *   trk_vertex int8[T]                   index of the track's PV within its event, -1 = none
 * Same values as pv_find / pv_find_host, bit for bit. */
int pv_find_host_compact(pv_host_ctx* ctx,
                         const float* x, const float* y, const float* z, const float* tx, const float* ty,
                         const float* var_x, const float* var_y, const float* var_tx, const float* var_ty,
                         const int32_t* offsets, int n_events, const pv_params* params,
                         pv_vertex* vertices, long long vtx_capacity, int32_t* vtx_begin, int32_t* n_vtx,
                         float* trk_weight, int8_t* trk_vertex, uint32_t* event_status, int n_chunks);
/* Pin / unpin caller host memory so pv_find_host copies run asynchronously (optional). */
int pv_host_register(void* ptr, size_t bytes);
int pv_host_unregister(void* ptr);

/* Launch statistics of the most recent pv_find / pv_find_debug call of this process (for bench.py):
 * kernels launched (4: seed, fit, the small kernel that refits the few ill-conditioned seeds in double, cleanup;
 * 5 with PV_FILL_TEMPLATE: the template table first), and grid size, block size, dynamic shared memory per block of
 * the seed kernel.  All HOST out, nullable. */
int pv_last_launch_info(int* n_kernels, int* grid, int* block, int* smem_bytes);

/* Optional: CUDA events recorded around each kernel of the next pv_find calls on their own stream, so a
 * caller can time the kernels live.  pv_kernel_timing(1) enables, (0) disables; pv_kernel_time_ms()
 * synchronises the last call's events and returns the duration of its three kernels in ms (< 0 if none);
 * pv_kernel_times_ms() writes up to n per-kernel durations (seed a1-a4, fit a5 incl. the refit kernel, cleanup a6) to ms (HOST)
 * and returns the number of kernels (3), or a negative PV_E_*.  With PV_FILL_TEMPLATE the small kernel that builds
 * the table of templates runs inside the first interval: "seed" then means table + seed kernel.
 * Bench / diagnostic use only: the events and the flag are process-global (see "Thread safety" above). */
int pv_kernel_timing(int enable);
float pv_kernel_time_ms(void);
int pv_kernel_times_ms(float* ms, int n);

const char* pv_error_string(int code);
/* Text of the last CUDA error seen by this library in this process ("" if none).  HOST. */
const char* pv_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* PV_FINDER_H */

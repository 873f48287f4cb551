/* pv_oracle.h -- interface of the CPU ORACLE for the primary-vertex finder hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  This is a plain, slow, scalar restatement of what
 * /root/reference/PAPER.md (arXiv:2412.14966) defines, with the readings listed in DESIGN.md
 * section "Readings".  It shares no code, header, table or constant generator with the CUDA
 * product under paper_2412_14966_b200/ ; only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may call it.
 *
 * All pointers are HOST pointers.  Citations "P:Lnn" are line numbers of PAPER.md.
 */
#ifndef PV_ORACLE_H
#define PV_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Parameters; index 0 = pp region (z >= z_split), 1 = p-gas region (z < z_split). */
typedef struct pvo_params {
  float z_min, z_max, dz;              /* -550, 300, 0.25 mm */
  float z_split;                       /* -300 mm                       Table 2 */
  float beam_x, beam_y, beam_tx, beam_ty; /* beamline at z = 0 */
  float max_sigma_poca[2];             /* 1.5, 10 mm                    P:L129, Table 2 */
  float min_bin_content;               /* proto-cluster threshold [tracks/bin]; paper silent: 0.25 */
  float min_dip;                       /* extremum significance [tracks/bin]; paper silent: 0.75 */
  float min_cluster_integral[2];       /* 2.5, 1.75 tracks              Table 2 */
  int32_t min_tracks_seed[2];          /* 3, 2 */
  int32_t min_tracks_pv[2];            /* 4, 3                          Table 2 */
  float chi2_max;                      /* 12; INFINITY = unit weights */
  int32_t max_iter;                    /* 10 */
  float conv_dchi2, conv_dz;           /* 0.01, 0.001 mm */
  float merge_ratio;                   /* 25 */
  float max_beam_dist;                 /* 0.3 mm */
  int32_t max_vtx_per_event;           /* output stride */
  int32_t flavour;                     /* 0: explicit association + Tukey weights (x86, Eq. 18);
                                          1: implicit association + multi-vertex weights (GPU, Eq. 19) */
  float chi2_window;                   /* flavour 1: tracks with chi2 < this at the seed position take part in a
                                          vertex fit (value 25: reading R-13) */
  int32_t split_mode;                  /* proto-cluster splitting: 0 = minima in z order (GPU variant),
                                          1 = smallest minimum between the two largest maxima, recursively (x86) */
  int32_t fill_mode;                   /* histogram fill: 0 = polynomial CDF per track (GPU variant, R-6),
                                          1 = "a finite set of template histograms, selected based on the value of
                                          sigma_poca" (x86 variant, reading R-17) */
} pvo_params;

/* NEXT-2: the x-tx and y-ty elements of the track covariance (Eq. 2: V_xx(z) = V_xx + 2 dz V_xtx + dz^2 V_txtx).
 * Optional everywhere: a NULL struct or member is a diagonal covariance. */
typedef struct pvo_cross { const float *xtx, *yty; } pvo_cross;

enum { PVO_S = 1 << 20 };              /* fixed-point unit: one track's full mass */
enum { PVO_MAX_TRACKS = 2047, PVO_TRACE_STRIDE = 11, PVO_TRACE_ITERS = 16 };
enum { PVO_EVT_TOO_MANY_TRACKS = 1, PVO_EVT_VTX_OVERFLOW = 2, PVO_EVT_SINGULAR_FIT = 4 };
/* track flag bits written by pvo_project */
enum { PVO_TRK_ASSIGNABLE = 1, PVO_TRK_HISTOGRAMMED = 2 };

void pvo_params_default(pvo_params *p);
int pvo_nbins(const pvo_params *p);

/* O1/O2: POCA projection Eq. 1, sigma_poca Eq. 3, acceptance. fp32 contract. */
void pvo_project(int n, const float *x, const float *y, const float *z, const float *tx, const float *ty,
                 const float *var_x, const pvo_params *p,
                 float *z_poca, float *sigma_poca, int32_t *bin, int32_t *flags);

/* O3: fixed-point CDF value at bin edge k for a track (z_poca, sigma_poca).  fp32 contract. */
int32_t pvo_edge_q(int k, float z_poca, float sigma_poca, const pvo_params *p);
/* O3: histogram fill.  H has nbins int32 entries and is ACCUMULATED into.
 * full_range != 0 evaluates every edge of the histogram for every track (the definition);
 * full_range == 0 evaluates a conservative window only (identical result, see tests). */
void pvo_fill(int n, const float *z_poca, const float *sigma_poca, const int32_t *flags,
              const pvo_params *p, int32_t *H, int full_range);
/* O3, x86 variant (reading R-17): the track's bin contents are taken from a TEMPLATE histogram instead of being
 * integrated for its own z_poca and sigma_poca.  Templates exist for sigma classes k = 0, 1, ... with centres
 * sigma_k = 0.08 dz 2^(k/4) (a track takes the class nearest in log sigma, clamped to the classes the sigma cuts allow)
 * and for PVO_TMPL_J = 8 positions of z_poca inside its central bin (the centre of the eighth it falls in).  A template
 * is the fixed-point CDF contract of pvo_edge_q evaluated in bin units for (sigma_k, position): bin i relative to the
 * central bin gets Q(i + 1) - Q(i), i in [-W_k, W_k], W_k = ceil(3 sigma_k / dz); it sums to exactly 2^20.
 * pvo_tmpl_class: class of a sigma_poca; pvo_tmpl_halfwidth: W_k; pvo_tmpl_bin: content of relative bin i of template
 * (k, j); pvo_fill_template: the fill (H accumulated into, like pvo_fill). */
enum { PVO_TMPL_J = 8 };
int pvo_tmpl_class(float sigma_poca, const pvo_params *p);
int pvo_tmpl_halfwidth(int k);
int32_t pvo_tmpl_bin(int k, int j, int i);
void pvo_fill_template(int n, const float *z_poca, const float *sigma_poca, const int32_t *bin, const int32_t *flags,
                       const pvo_params *p, int32_t *H);

/* O3 definition layer L0: exact Gaussian bin integrals via erf in double, untruncated. */
void pvo_fill_exact(int n, const float *z_poca, const float *sigma_poca, const int32_t *flags,
                    const pvo_params *p, double *H0);

/* O4: peak search.  Writes up to cap clusters (begin, end, peak); returns the total
 * number found (may exceed cap). */
int pvo_peaks(const int32_t *H, const pvo_params *p, int cap, int32_t *begin, int32_t *end, int32_t *peak);
/* O5: seed z, Eq. 4-5. */
float pvo_seed_z(const int32_t *H, int peak, const pvo_params *p);

/* O6: assignment with the removal loop.  Seeds are compacted in place; returns the number
 * of seeds left.  trk_seed[i] = seed index or -1. */
int pvo_assign(int n, const int32_t *bin, const int32_t *flags, int n_seeds,
               int32_t *begin, int32_t *end, int32_t *peak, float *z_seed,
               const pvo_params *p, int32_t *trk_seed);

/* O7: adaptive fit of ONE vertex over the m tracks listed in idx[].
 * out_pos[3], out_cov[6] (xx,xy,xz,yy,yz,zz), w[m]; trace (nullable) gets PVO_TRACE_STRIDE doubles
 * per iteration: pos3, cov6, dchi2, dz.  Returns 0, or -1 when the fit is singular. */
int pvo_fit(int m, const int32_t *idx,
            const float *x, const float *y, const float *z, const float *tx, const float *ty,
            const float *var_x, const float *var_y, const float *var_tx, const float *var_ty,
            const double seed[3], const pvo_params *p, const pvo_cross *cx,
            double *out_pos, double *out_cov, double *out_chi2, int32_t *out_ntrk, int32_t *out_niter,
            double *w, double *trace);

/* Eq. 19: multi-vertex weight of a track with chi2_own to this vertex, chi2_others[] to the others. */
double pvo_mv_weight(double chi2_own, double chi2_max, const double *chi2_others, int n_others);
/* chi2 of track i relative to a vertex at pos[3] (Eq. 7 with W from Eq. 2 at pos); < 0 = unusable (R-7). */
double pvo_track_chi2(int i, const float *x, const float *y, const float *z, const float *tx, const float *ty,
                      const float *var_x, const float *var_y, const float *var_tx, const float *var_ty,
                      const pvo_cross *cx, const double pos[3]);
/* O7, multi-vertex flavour: pvo_fit with the weights of Eq. 19; other[j] = exp(-chi2_max / 2) + sum over the
 * other candidates of exp(-chi2_jk / 2) at their seed positions.  out_ntrk = tracks with w >= 1/2. */
int pvo_fit_mv(int m, const int32_t *idx,
               const float *x, const float *y, const float *z, const float *tx, const float *ty,
               const float *var_x, const float *var_y, const float *var_tx, const float *var_ty,
               const double seed[3], const pvo_params *p, const double *other, const pvo_cross *cx,
               double *out_pos, double *out_cov, double *out_chi2, int32_t *out_ntrk, int32_t *out_niter,
               double *w, double *trace);

/* NEXT-4: impact parameter and IP chi2 of track i to a vertex (pos[3], C[6] upper triangle) that does not
 * contain it; returns -1 when the covariance is unusable. */
int pvo_ip_one(int i, const float *x, const float *y, const float *z, const float *tx, const float *ty,
               const float *var_x, const float *var_y, const float *var_tx, const float *var_ty,
               const pvo_cross *cx, const double pos[3], const double C[6], double *ip, double *ip_chi2);
/* per track: the vertex of its event with the smallest IP chi2; -1 if none */
int pvo_track_ip(const float *x, const float *y, const float *z, const float *tx, const float *ty,
                 const float *var_x, const float *var_y, const float *var_tx, const float *var_ty,
                 const pvo_cross *cx, const int32_t *offsets, int n_events, int max_vtx,
                 const double *vtx_pos, const double *vtx_cov, const int32_t *n_vtx,
                 double *ip, double *ip_chi2, int32_t *ip_vertex);

/* Optional taps of the full pipeline (all nullable). */
typedef struct pvo_debug {
  int32_t *hist;        /* [n_hist_events][nbins] */
  int32_t n_hist_events;
  float *z_poca;        /* [T] */
  float *sigma_poca;    /* [T] */
  int32_t *trk_bin;     /* [T] */
  int32_t *trk_flags;   /* [T] */
  int32_t *n_seeds;     /* [E] after removal loop */
  int32_t *n_seeds_raw; /* [E] as found by the peak search (before truncation / removal) */
  float *seed_z;        /* [E][max_vtx] after removal loop */
  int32_t *seed_bins;   /* [E][max_vtx][3] begin,end,peak after removal loop */
  int32_t *trk_seed;    /* [T] pre-cleanup assignment */
  double *seed_pos;     /* [E][max_vtx][3] fitted, pre-cleanup */
  double *seed_cov;     /* [E][max_vtx][6] */
  double *seed_chi2;    /* [E][max_vtx] */
  int32_t *seed_ntrk;   /* [E][max_vtx] */
  int32_t *seed_niter;  /* [E][max_vtx]; -1 = singular */
  int32_t *seed_fate;   /* [E][max_vtx]; final vertex index, or -1 singular, -2 merged, -3 min tracks, -4 beam dist */
  double *trace;        /* [E][max_vtx][PVO_TRACE_ITERS][PVO_TRACE_STRIDE], indexed by seed */
  /* diagnostics for the comparator's near-tie rules (no output depends on them) */
  double *seed_edge_last; /* [E][max_vtx] min over the seed's tracks of |chi2_i / chi2_max - 1| (flavour 0) or |w_i - 1/2|
                             (flavour 1) in the last iteration: how close n_trk is to counting one track more or less */
  double *seed_edge_any;  /* [E][max_vtx] the same, min over all iterations (decides the < 2 active tracks test) */
  double *seed_pivot_min; /* [E][max_vtx] smallest Cholesky pivot / diagonal element over the iterations (<= 0: singular) */
  int32_t *seed_nact_min; /* [E][max_vtx] fewest active tracks in an iteration */
  double *trk_w2;         /* [T] flavour 1: the second largest final weight of the track over the fitted candidates */
  double *trk_w1;         /* [T] flavour 1: the largest one (trk_weight before cleanup releases tracks) */
} pvo_debug;

/* The whole hot path a1..a6 over a batch.  Outputs (host, caller-owned):
 * vtx_pos [E][max_vtx][3], vtx_cov [E][max_vtx][6], vtx_chi2/ntracks/niter [E][max_vtx], n_vtx [E],
 * trk_weight [T], trk_vertex [T], event_status [E].  n_threads > 1 runs events in parallel (OpenMP,
 * timing harness only; results do not depend on it).  Returns 0 or a negative error. */
int pvo_find(const float *x, const float *y, const float *z, const float *tx, const float *ty,
             const float *var_x, const float *var_y, const float *var_tx, const float *var_ty,
             const pvo_cross *cx, const int32_t *offsets, int n_events, const pvo_params *p,
             double *vtx_pos, double *vtx_cov, double *vtx_chi2, int32_t *vtx_ntracks, int32_t *vtx_niter,
             int32_t *n_vtx, double *trk_weight, int32_t *trk_vertex, uint32_t *event_status,
             const pvo_debug *dbg, int n_threads);

#ifdef __cplusplus
}
#endif
#endif

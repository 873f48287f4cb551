/* pv_oracle.c -- CPU ORACLE for the primary-vertex finder hot path of arXiv:2412.14966.
 *
 * TEST INFRASTRUCTURE ONLY (see pv_oracle.h).  Plain scalar C, one event at a time, in the paper's
 * order: project (3.1) -> fill (3.2) -> peak search (3.3) -> associate (3.4) -> fit (3.5) -> cleanup.
 * Floating point is double EXCEPT where a step decides an integer (bin index, fixed-point CDF
 * code, seed position): those follow the fp32 "contract" of DESIGN.md, every operation rounded
 * individually (compile with -ffp-contract=off, no -ffast-math).  Citations "P:Lnn" are PAPER.md lines;
 * "R-n" are the readings listed in DESIGN.md where the paper is silent.
 *
 * Pins (tests/test_oracle_*.py): closed forms, brute force, invariants; none of them calls the CUDA path.
 * Parity status: every function below is pinned; the paper-silent DEFAULT VALUES (min_bin_content,
 * min_dip, the +-3 sigma support, min-bin ownership, loser-track rule) are readings, "parity unpinned"
 * in the sense that no published number fixes them (DESIGN.md lists them).
 */
#include "pv_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

/* ---- O3 frozen constants: odd degree-13 polynomial G(s), s = u/3 -------- */
static const float PVO_G[7] = {
    0x1.3331cep+0f, -0x1.cbf272p+0f, 0x1.32067cp+1f, -0x1.3336f8p+1f,
    0x1.b67296p+0f, -0x1.862240p-1f, 0x1.3e0392p-3f};
#define PVO_U 3.0f

void pvo_params_default(pvo_params *p) {
  p->z_min = -550.0f; p->z_max = 300.0f; p->dz = 0.25f;
  p->z_split = -300.0f;                                          /* Table 2 */
  p->beam_x = p->beam_y = p->beam_tx = p->beam_ty = 0.0f;
  p->max_sigma_poca[0] = 1.5f; p->max_sigma_poca[1] = 10.0f;
  p->min_bin_content = 0.25f; p->min_dip = 0.75f;                /* R-4 */
  p->min_cluster_integral[0] = 2.5f; p->min_cluster_integral[1] = 1.75f; /* Table 2 */
  p->min_tracks_seed[0] = 3; p->min_tracks_seed[1] = 2;
  p->min_tracks_pv[0] = 4; p->min_tracks_pv[1] = 3;              /* Table 2 */
  p->chi2_max = 12.0f;
  p->max_iter = 10; p->conv_dchi2 = 0.01f; p->conv_dz = 0.001f;
  p->merge_ratio = 25.0f;
  p->max_beam_dist = 0.3f;
  p->max_vtx_per_event = 32;
  p->flavour = 0;                                                /* explicit association + Tukey (x86 flavour) */
  p->chi2_window = 25.0f;                                        /* P:L384 "within a certain chi2_i"; value: R-13 */
  p->split_mode = 0;                                             /* z-ordered splitting (GPU variant) */
  p->fill_mode = 0;                                              /* polynomial CDF per track (GPU variant) */
}

int pvo_nbins(const pvo_params *p) {
  return (int)lrint(((double)p->z_max - (double)p->z_min) / (double)p->dz);
}

/* ===================================== O1 / O2 : projection ========================================== */
/* Eq. 1 with the beamline evaluated at the track's z (R-1), Eq. 3 with V_xx = var_x
 * (R-2).  fp32 contract: the exact operation order below is what the CUDA path must reproduce. */
static void project_one(float x, float y, float z, float tx, float ty, float var_x, const pvo_params *p,
                        int nbins, float inv_dz, float *zp_o, float *sp_o, int32_t *bin_o, int32_t *flags_o) {
  float dtx = tx - p->beam_tx;
  float dty = ty - p->beam_ty;
  float den = fmaf(dty, dty, dtx * dtx);
  *zp_o = NAN; *sp_o = NAN; *bin_o = -1; *flags_o = 0;
  if (!(den >= 1e-12f)) return;                      /* R-3: parallel to the beamline (or NaN) */
  float bx = fmaf(p->beam_tx, z, p->beam_x);
  float by = fmaf(p->beam_ty, z, p->beam_y);
  float num = fmaf(dty, by - y, dtx * (bx - x));
  float zp = z + num / den;
  float sp = sqrtf(var_x / den);
  *zp_o = zp; *sp_o = sp;
  float fb = floorf((zp - p->z_min) * inv_dz);
  if (!(fb >= 0.0f && fb < (float)nbins)) return;    /* out of the histogram range, or non-finite */
  *bin_o = (int32_t)fb;
  *flags_o = PVO_TRK_ASSIGNABLE;
  int region = zp < p->z_split ? 1 : 0;              /* R-5: region of a track by its own z_poca */
  float inv = 1.0f / (PVO_U * sp);
  if (sp > 0.0f && sp <= p->max_sigma_poca[region] && isfinite(inv)) *flags_o |= PVO_TRK_HISTOGRAMMED;
}

void pvo_project(int n, const float *x, const float *y, const float *z, const float *tx, const float *ty,
                 const float *var_x, const pvo_params *p,
                 float *z_poca, float *sigma_poca, int32_t *bin, int32_t *flags) {
  int nbins = pvo_nbins(p);
  float inv_dz = 1.0f / p->dz;
  for (int i = 0; i < n; ++i)
    project_one(x[i], y[i], z[i], tx[i], ty[i], var_x[i], p, nbins, inv_dz, &z_poca[i], &sigma_poca[i],
                &bin[i], &flags[i]);
}

/* ===================================== O3 : histogram fill =========================================== */
/* Fixed-point CDF of the truncated, renormalised Gaussian with support +-3 sigma at bin edge k (R-6).
 * F(u) = 0 (u <= -3), 1 (u >= 3), 1/2 + G(u/3) otherwise; Q = rint(F * 2^20). */
int32_t pvo_edge_q(int k, float zp, float sp, const pvo_params *p) {
  float inv = 1.0f / (PVO_U * sp);
  float e = fmaf((float)k, p->dz, p->z_min);
  float s = (e - zp) * inv;
  if (s <= -1.0f) return 0;
  if (s >= 1.0f) return PVO_S;
  float t = s * s;
  float g = PVO_G[6];
  for (int j = 5; j >= 0; --j) g = fmaf(g, t, PVO_G[j]);
  float c = fmaf(s, g, 0.5f);
  if (c < 0.0f) c = 0.0f;
  if (c > 1.0f) c = 1.0f;
  return (int32_t)lrintf(c * 1048576.0f);            /* ties to even */
}

/* Bin i receives Q(i+1) - Q(i) (the integral of the density over the bin), as an integer add. */
void pvo_fill(int n, const float *z_poca, const float *sigma_poca, const int32_t *flags,
              const pvo_params *p, int32_t *H, int full_range) {
  int nbins = pvo_nbins(p);
  for (int i = 0; i < n; ++i) {
    if (!(flags[i] & PVO_TRK_HISTOGRAMMED)) continue;
    int lo = 0, hi = nbins;                          /* edges lo..hi, bins lo..hi-1 */
    if (!full_range) {
      /* "only ... a finite number of bins neighbouring the central bin": conservative window;
       * edges beyond +-3 sigma give exactly 0 or S, so any superset of the support is equivalent. */
      double su = 3.0 * (double)sigma_poca[i];
      double a = floor(((double)z_poca[i] - su - (double)p->z_min) / (double)p->dz) - 2.0;
      double b = floor(((double)z_poca[i] + su - (double)p->z_min) / (double)p->dz) + 3.0;
      if (a > 0.0) lo = a < (double)nbins ? (int)a : nbins;
      if (b < (double)nbins) hi = b > 0.0 ? (int)b : 0;
    }
    if (hi <= lo) continue;
    int32_t q0 = pvo_edge_q(lo, z_poca[i], sigma_poca[i], p);
    for (int b = lo; b < hi; ++b) {
      int32_t q1 = pvo_edge_q(b + 1, z_poca[i], sigma_poca[i], p);
      H[b] += q1 - q0;
      q0 = q1;
    }
  }
}

/* ---- O3, x86 variant: template histograms selected by sigma_poca (reading R-17) ---------------------------
 * fp32 contract like the rest of O3 (every operation rounded once), so that the integer bins are reproducible. */
static const float PVO_TMPL_CENTRE[4] = {1.0f, 0x1.306fe0p+0f, 0x1.6a09e6p+0f, 0x1.ae89fap+0f};   /* 2^(0, 1/4, 1/2, 3/4) */
static const float PVO_TMPL_EDGE[4] = {0x1.172b84p+0f, 0x1.4bfdaep+0f, 0x1.8ace54p+0f, 0x1.d5818ep+0f}; /* 2^(1/8, 3/8, 5/8, 7/8) */

/* centre of sigma class k in bins: 0.08 * 2^(k/4) */
static float tmpl_centre(int k) { return ldexpf(PVO_TMPL_CENTRE[k & 3], k >> 2) * 0.08f; }

/* nearest class in log sigma, before clamping: with v = sigma / (0.08 dz) = m 2^E, m in [1, 2): 4 E + the number of
 * class edges 2^((2 q + 1) / 8) that m has reached */
static int tmpl_class_raw(float sigma, float inv_dz) {
  float v = (sigma * inv_dz) * 12.5f;
  if (!(v >= 1.0f)) return 0;                        /* below the first centre (or NaN) */
  if (!(v < 0x1p+20f)) return 80;                    /* far beyond any sigma cut */
  int E;
  float m = 2.0f * frexpf(v, &E);                    /* v = m 2^(E - 1), m in [1, 2) */
  int k = 4 * (E - 1);
  for (int q = 0; q < 4; ++q) k += (m >= PVO_TMPL_EDGE[q]) ? 1 : 0;
  return k;
}

int pvo_tmpl_class(float sigma_poca, const pvo_params *p) {
  float inv_dz = 1.0f / p->dz;
  float smax = p->max_sigma_poca[0] > p->max_sigma_poca[1] ? p->max_sigma_poca[0] : p->max_sigma_poca[1];
  int kmax = tmpl_class_raw(smax, inv_dz);           /* the finite set: classes 0 .. class of the largest sigma cut */
  int k = tmpl_class_raw(sigma_poca, inv_dz);
  return k < kmax ? k : kmax;
}

int pvo_tmpl_halfwidth(int k) { return (int)ceilf(3.0f * tmpl_centre(k)); }

/* fixed-point CDF (the contract of pvo_edge_q) at bin edge i, in bins relative to the lower edge of the central bin,
 * for a track at zrel inside that bin with 1 / (3 sigma) = inv */
static int32_t tmpl_edge_q(int i, float zrel, float inv) {
  float s = ((float)i - zrel) * inv;
  if (s <= -1.0f) return 0;
  if (s >= 1.0f) return PVO_S;
  float t = s * s;
  float g = PVO_G[6];
  for (int j = 5; j >= 0; --j) g = fmaf(g, t, PVO_G[j]);
  float c = fmaf(s, g, 0.5f);
  if (c < 0.0f) c = 0.0f;
  if (c > 1.0f) c = 1.0f;
  return (int32_t)lrintf(c * 1048576.0f);
}

int32_t pvo_tmpl_bin(int k, int j, int i) {
  float zrel = ((float)j + 0.5f) * (1.0f / (float)PVO_TMPL_J);  /* centre of the j-th eighth of the central bin */
  float inv = 1.0f / (PVO_U * tmpl_centre(k));
  return tmpl_edge_q(i + 1, zrel, inv) - tmpl_edge_q(i, zrel, inv);
}

void pvo_fill_template(int n, const float *z_poca, const float *sigma_poca, const int32_t *bin, const int32_t *flags,
                       const pvo_params *p, int32_t *H) {
  int nbins = pvo_nbins(p);
  float inv_dz = 1.0f / p->dz;
  for (int t = 0; t < n; ++t) {
    if (!(flags[t] & PVO_TRK_HISTOGRAMMED)) continue;
    int k = pvo_tmpl_class(sigma_poca[t], p);         /* "selected based on the value of sigma_poca" */
    float fb = (z_poca[t] - p->z_min) * inv_dz;       /* the expression that gave the central bin (O1) */
    float frac = fb - floorf(fb);
    int j = (int)(frac * (float)PVO_TMPL_J);
    if (j > PVO_TMPL_J - 1) j = PVO_TMPL_J - 1;
    int W = pvo_tmpl_halfwidth(k);
    for (int i = -W; i <= W; ++i) {
      int b = bin[t] + i;
      if (b >= 0 && b < nbins) H[b] += pvo_tmpl_bin(k, j, i);   /* bins beyond the range are dropped, as in pvo_fill */
    }
  }
}

/* Definition layer L0: untruncated Gaussian bin integrals in double with erf. */
void pvo_fill_exact(int n, const float *z_poca, const float *sigma_poca, const int32_t *flags,
                    const pvo_params *p, double *H0) {
  int nbins = pvo_nbins(p);
  for (int i = 0; i < n; ++i) {
    if (!(flags[i] & PVO_TRK_HISTOGRAMMED)) continue;
    double zp = z_poca[i], sp = sigma_poca[i];
    for (int b = 0; b < nbins; ++b) {
      double e0 = (double)p->z_min + (double)b * (double)p->dz;
      double e1 = (double)p->z_min + (double)(b + 1) * (double)p->dz;
      if (e1 < zp - 10.0 * sp || e0 > zp + 10.0 * sp) continue;
      H0[b] += 0.5 * (erf((e1 - zp) / (sp * M_SQRT2)) - erf((e0 - zp) / (sp * M_SQRT2)));
    }
  }
}

/* ===================================== O4 : peak search ============================================== */
static int64_t to_fixed(float tracks) { return (int64_t)llrint((double)tracks * (double)PVO_S); }

static int bin_region(int b, const pvo_params *p) {
  float centre = fmaf((float)b + 0.5f, p->dz, p->z_min);
  return centre < p->z_split ? 1 : 0;
}

static int argmax_bin(const int32_t *H, int b0, int b1) { /* ties -> lowest bin */
  int best = b0;
  for (int b = b0 + 1; b < b1; ++b)
    if (H[b] > H[best]) best = b;
  return best;
}

static int64_t integral(const int32_t *H, int b0, int b1) {
  int64_t s = 0;
  for (int b = b0; b < b1; ++b) s += H[b];
  return s;
}

/* x86 variant of the splitting: "the CPU implementation considers the smallest minimum between the two
 * largest maxima and does the splitting recursively".  Reading R-16: on the bin range [s, e) run the hysteresis
 * sweep of R-4.2; with fewer than two significant maxima the range is a leaf; else take the two highest maxima (ties:
 * lower bin), the lowest significant minimum between them (ties: lower bin), and split there iff BOTH parts carry the
 * minimum cluster integral; recurse into the left part, then the right part (the minimum bin opens the
 * right part, as in R-4.3).  Leaves are seed clusters, emitted in z order. */
typedef struct peak_out { int cap, n; int32_t *begin, *end, *peak; } peak_out;

static void split_recursive(const int32_t *H, int s, int e, const pvo_params *p, int64_t D, const int64_t I_min[2],
                            int *ext_bin, peak_out *out) {
  /* extrema of [s, e): ext_bin[2 j] = bin of MAX j, ext_bin[2 j - 1] = bin of MIN j (between MAX j-1 and MAX j) */
  int n_max = 0;
  int look_max = 1;
  int64_t mx = H[s], mn = 0;
  int mxp = s, mnp = s;
  for (int k = s + 1; k < e; ++k) {
    int64_t h = H[k];
    if (look_max) {
      if (h > mx) { mx = h; mxp = k; }
      else if (h < mx - D) { ext_bin[2 * n_max] = mxp; ++n_max; mn = h; mnp = k; look_max = 0; }
    } else {
      if (h < mn) { mn = h; mnp = k; }
      else if (h > mn + D) { ext_bin[2 * n_max - 1] = mnp; mx = h; mxp = k; look_max = 1; }
    }
  }
  if (look_max) { ext_bin[2 * n_max] = mxp; ++n_max; }
  if (n_max >= 2) {
    int a = 0, b = -1;                                   /* indices of the highest and second highest maximum */
    for (int j = 1; j < n_max; ++j) if (H[ext_bin[2 * j]] > H[ext_bin[2 * a]]) a = j;
    for (int j = 0; j < n_max; ++j) {
      if (j == a) continue;
      if (b < 0 || H[ext_bin[2 * j]] > H[ext_bin[2 * b]]) b = j;
    }
    int lo = a < b ? a : b, hi = a < b ? b : a;
    int c = ext_bin[2 * (lo + 1) - 1];
    for (int j = lo + 2; j <= hi; ++j) if (H[ext_bin[2 * j - 1]] < H[c]) c = ext_bin[2 * j - 1];
    int pl = argmax_bin(H, s, c), pr = argmax_bin(H, c, e);
    if (integral(H, s, c) >= I_min[bin_region(pl, p)] && integral(H, c, e) >= I_min[bin_region(pr, p)]) {
      /* the extrema buffer is reused by the recursion: nothing of this level is needed afterwards */
      split_recursive(H, s, c, p, D, I_min, ext_bin, out);
      split_recursive(H, c, e, p, D, I_min, ext_bin, out);
      return;
    }
  }
  if (out->n < out->cap) { out->begin[out->n] = s; out->end[out->n] = e; out->peak[out->n] = argmax_bin(H, s, e); }
  ++out->n;
}

int pvo_peaks(const int32_t *H, const pvo_params *p, int cap, int32_t *begin, int32_t *end, int32_t *peak) {
  const int nbins = pvo_nbins(p);
  const int64_t T_bin = to_fixed(p->min_bin_content);
  const int64_t D = to_fixed(p->min_dip);
  const int64_t I_min[2] = {to_fixed(p->min_cluster_integral[0]), to_fixed(p->min_cluster_integral[1])};
  int n_out = 0;
  int *minima = (int *)malloc(sizeof(int) * (size_t)(2 * nbins + 2));
  int b = 0;
  while (b < nbins) {
    if (!((int64_t)H[b] > T_bin)) { ++b; continue; }
    /* 1. proto-cluster: maximal run of bins "above a threshold" */
    int b0 = b, b1 = b;
    while (b1 < nbins && (int64_t)H[b1] > T_bin) ++b1;
    if (p->split_mode == 1) {                        /* x86 variant (R-16): recursive splitting */
      int pk = argmax_bin(H, b0, b1);
      if (integral(H, b0, b1) >= I_min[bin_region(pk, p)]) {      /* every seed passes the integral cut */
        peak_out out = {cap, n_out, begin, end, peak};
        split_recursive(H, b0, b1, p, D, I_min, minima, &out);
        n_out = out.n;
      }
      b = b1;
      continue;
    }
    /* 2. "all significant minima and maxima": z-ordered hysteresis sweep (R-4.2).
     *    The emitted extremum list is MAX (MIN MAX)*, only the MINs are needed afterwards. */
    int n_min = 0;
    int look_max = 1;
    int64_t mx = H[b0], mn = 0;
    int mnp = b0;
    for (int k = b0 + 1; k < b1; ++k) {
      int64_t h = H[k];
      if (look_max) {
        if (h > mx) { mx = h; }
        else if (h < mx - D) { mn = h; mnp = k; look_max = 0; }       /* emits MAX */
      } else {
        if (h < mn) { mn = h; mnp = k; }
        else if (h > mn + D) { minima[n_min++] = mnp; mx = h; look_max = 1; } /* emits MIN(mnp) */
      }
    }
    /* 3. split "at minima which have two neighbouring maxima", in z order (GPU variant),
     *    "only ... if the track integral of the resulting seed cluster is above a threshold" */
    int start = b0;
    int first_out = n_out;
    for (int j = 0; j < n_min; ++j) {
      int m = minima[j];
      int pk = argmax_bin(H, start, m);
      if (integral(H, start, m) >= I_min[bin_region(pk, p)]) {
        if (n_out < cap) { begin[n_out] = start; end[n_out] = m; peak[n_out] = pk; }
        ++n_out;
        start = m;                                   /* the minimum bin opens the right-hand cluster */
      }
    }
    {
      int pk = argmax_bin(H, start, b1);
      if (integral(H, start, b1) >= I_min[bin_region(pk, p)]) {
        if (n_out < cap) { begin[n_out] = start; end[n_out] = b1; peak[n_out] = pk; }
        ++n_out;
      } else if (n_out > first_out) {                /* remainder joins the last cluster of this proto-cluster */
        if (n_out - 1 < cap) {
          end[n_out - 1] = b1;
          peak[n_out - 1] = argmax_bin(H, begin[n_out - 1], b1);   /* 4. peak = argmax of the final cluster */
        }
      }                                              /* else: proto-cluster below the integral cut, dropped */
    }
    b = b1;
  }
  free(minima);
  return n_out;
}

/* ===================================== O5 : seed position ============================================ */
/* Eq. 4-5; neighbours are raw histogram bins, 0 beyond the ends (R-10). */
float pvo_seed_z(const int32_t *H, int i, const pvo_params *p) {
  int nbins = pvo_nbins(p);
  int64_t Nm = i > 0 ? H[i - 1] : 0;
  int64_t Np = i < nbins - 1 ? H[i + 1] : 0;
  int64_t N0 = H[i];
  int64_t num = Np - Nm;
  int64_t den = 2 * N0 - Np - Nm;
  float delta = den > 0 ? 0.5f * ((float)num / (float)den) : 0.0f;
  float zi = fmaf((float)i + 0.5f, p->dz, p->z_min);           /* bin midpoint */
  return fmaf(delta, p->dz, zi);
}

/* ===================================== O6 : association ============================================== */
int pvo_assign(int n, const int32_t *bin, const int32_t *flags, int n_seeds,
               int32_t *begin, int32_t *end, int32_t *peak, float *z_seed,
               const pvo_params *p, int32_t *trk_seed) {
  int *cnt = (int *)malloc(sizeof(int) * (size_t)(n_seeds + 1));
  int *part = (int *)malloc(sizeof(int) * (size_t)(n_seeds + 1));
  for (;;) {
    for (int i = 0; i < n; ++i) trk_seed[i] = -1;
    if (n_seeds == 0) break;
    /* partition point = "the bin in between of the upper bound of one cluster and the lower bound of
     * the next cluster"; bins < part[k] belong to seed k, the others to k+1 ... (R-11) */
    for (int k = 0; k + 1 < n_seeds; ++k) part[k] = (end[k] + begin[k + 1]) / 2;
    for (int k = 0; k < n_seeds; ++k) cnt[k] = 0;
    for (int i = 0; i < n; ++i) {
      if (!(flags[i] & PVO_TRK_ASSIGNABLE)) continue;
      int s = 0;
      while (s + 1 < n_seeds && bin[i] >= part[s]) ++s;
      trk_seed[i] = s;
      ++cnt[s];
    }
    /* "In the rare case that this is smaller than a threshold (3 pp / 2 SMOG2) the seed cluster is
     * removed ... and the procedure is repeated": remove the least populated, ties lowest z. */
    int worst = -1;
    for (int k = 0; k < n_seeds; ++k) {
      int region = z_seed[k] < p->z_split ? 1 : 0;
      if (cnt[k] < p->min_tracks_seed[region] && (worst < 0 || cnt[k] < cnt[worst])) worst = k;
    }
    if (worst < 0) break;
    for (int k = worst; k + 1 < n_seeds; ++k) {
      begin[k] = begin[k + 1]; end[k] = end[k + 1]; peak[k] = peak[k + 1]; z_seed[k] = z_seed[k + 1];
    }
    --n_seeds;
  }
  free(cnt); free(part);
  return n_seeds;
}

/* ===================================== O7 : adaptive vertex fit ====================================== */
/* Plain dense Cholesky of a symmetric 3x3, A = L L^T.  Returns -1 if a pivot is <= 0. */
static int chol3(const double A[3][3], double L[3][3], double *min_rel_pivot) {
  memset(L, 0, sizeof(double) * 9);
  for (int j = 0; j < 3; ++j) {
    double d = A[j][j];
    for (int k = 0; k < j; ++k) d -= L[j][k] * L[j][k];
    if (min_rel_pivot) {                              /* diagnostic only: how close the pivot is to its cut (0) */
      double rel = A[j][j] > 0.0 ? d / A[j][j] : 0.0;
      if (rel < *min_rel_pivot) *min_rel_pivot = rel;
    }
    if (!(d > 0.0)) return -1;
    L[j][j] = sqrt(d);
    for (int i = j + 1; i < 3; ++i) {
      double s = A[i][j];
      for (int k = 0; k < j; ++k) s -= L[i][k] * L[j][k];
      L[i][j] = s / L[j][j];
    }
  }
  return 0;
}

static void chol3_solve(const double L[3][3], const double b[3], double x[3]) {
  double y[3];
  for (int i = 0; i < 3; ++i) {
    double s = b[i];
    for (int k = 0; k < i; ++k) s -= L[i][k] * y[k];
    y[i] = s / L[i][i];
  }
  for (int i = 2; i >= 0; --i) {
    double s = y[i];
    for (int k = i + 1; k < 3; ++k) s -= L[k][i] * x[k];
    x[i] = s / L[i][i];
  }
}

/* Eq. 2, one transverse coordinate: V(z) = V_xx + 2 dz V_xtx + dz^2 V_txtx.  The x-y blocks are
 * uncorrelated in the simplified track fit, so V_xy, V_xty, V_txty do not appear.  cx == NULL (or a NULL
 * member) means a diagonal input covariance. */
static double var_at(double v, double vt, const float *cross, int i, double dz) {
  double c = cross ? (double)cross[i] : 0.0;
  return v + 2.0 * dz * c + dz * dz * vt;
}

/* Eq. 19: w_ij = exp(-chi2_ij / 2) / (exp(-chi2_max / 2) + sum_k exp(-chi2_ik / 2)); the sum runs over
 * all vertex candidates k including j itself. */
double pvo_mv_weight(double chi2_own, double chi2_max, const double *chi2_others, int n_others) {
  double den = exp(-0.5 * chi2_max) + exp(-0.5 * chi2_own);
  for (int k = 0; k < n_others; ++k) den += exp(-0.5 * chi2_others[k]);
  return exp(-0.5 * chi2_own) / den;
}
/* The same with the part of the denominator that does not depend on vertex j precomputed:
 * other = exp(-chi2_max / 2) + sum_{k != j} exp(-chi2_ik / 2). */
static double pvo_mv_weight_den(double chi2_own, double other) {
  double E = exp(-0.5 * chi2_own);
  return E / (other + E);
}

/* Diagnostics of one fit for the comparator's near-tie rules (tests only; no output depends on them). */
typedef struct fit_diag {
  double edge_last, edge_any;   /* closest track to the active / associated cut: last iteration, any iteration */
  double pivot_min;             /* smallest Cholesky pivot relative to its diagonal element, over the iterations */
  int nact_min;                 /* fewest active tracks in an iteration */
} fit_diag;

/* One Newton-Raphson iteration (Eq. 6-17) at the vertex position a[]: fills the Tukey weights w[] (Eq. 18),
 * the step (Eq. 13), C (Eq. 14), dchi2 (Eq. 17), chi2 (Eq. 6) and the number of tracks with w > 0.
 * Returns -1 when fewer than 2 tracks are active or the Hessian is not positive definite. */
static int fit_iteration(int m, const int32_t *idx,
                         const float *x, const float *y, const float *z, const float *tx, const float *ty,
                         const double *Wx, const double *Wy, const double a[3], double chi2_max, const double *other,
                         double *w, double step[3], double C[3][3], double *dchi2_o, double *chi2_o, int *nact_o,
                         double *edge_o, double *pivot_o) {
  double A[3][3] = {{0}}, g[3] = {0, 0, 0};
  double chi2 = 0.0;
  int nact = 0;
  double edge = INFINITY;                             /* diagnostic only (comparator near-tie rules): distance of the
                                                         closest track to the cut that decides "active" / "associated":
                                                         |chi2_i / chi2_max - 1| (Eq. 18) or |w_i - 1/2| (Eq. 19, R-13) */
  for (int j = 0; j < m; ++j) {
    int i = idx[j];
    double wi = 0.0;
    if (Wx[j] > 0.0) {
      /* residual Eq. 9 */
      double rx = (double)x[i] + (a[2] - (double)z[i]) * (double)tx[i] - a[0];
      double ry = (double)y[i] + (a[2] - (double)z[i]) * (double)ty[i] - a[1];
      double chi2_i = rx * rx * Wx[j] + ry * ry * Wy[j];            /* Eq. 7 */
      if (other) wi = pvo_mv_weight_den(chi2_i, other[j]);          /* Eq. 19, competitors at their seed positions */
      else if (isinf(chi2_max)) wi = 1.0;
      else if (chi2_i < chi2_max) { double u = 1.0 - chi2_i / chi2_max; wi = u * u; }  /* Eq. 18 */
      {
        double d = other ? fabs(wi - 0.5) : (isinf(chi2_max) ? INFINITY : fabs(chi2_i / chi2_max - 1.0));
        if (d < edge) edge = d;
      }
      /* H_i = [[-1,0,tx],[0,-1,ty]] (Eq. 12); accumulate w H^T W H (Eq. 11 / 2) and w H^T W r (Eq. 10 / 2) */
      double Hm[2][3] = {{-1.0, 0.0, (double)tx[i]}, {0.0, -1.0, (double)ty[i]}};
      double Wd[2] = {Wx[j], Wy[j]}, r[2] = {rx, ry};
      for (int c = 0; c < 2; ++c)
        for (int k = 0; k < 3; ++k) {
          g[k] += wi * Hm[c][k] * Wd[c] * r[c];
          for (int l = 0; l < 3; ++l) A[k][l] += wi * Hm[c][k] * Wd[c] * Hm[c][l];
        }
      chi2 += wi * chi2_i;                                          /* Eq. 6 */
    }
    w[j] = wi;
    if (wi > 0.0) ++nact;
  }
  *chi2_o = chi2; *nact_o = nact;
  if (edge_o) *edge_o = edge;
  if (nact < 2) return -1;
  double L[3][3];
  if (chol3(A, L, pivot_o) != 0) return -1;
  /* Newton-Raphson step Eq. 13: alpha1 = alpha0 - (d2chi2)^-1 dchi2 = alpha0 - A^-1 g */
  double mg[3] = {-g[0], -g[1], -g[2]};
  chol3_solve(L, mg, step);
  /* covariance Eq. 14: C = A^-1, column by column */
  for (int k = 0; k < 3; ++k) {
    double ek[3] = {0, 0, 0}, col[3];
    ek[k] = 1.0;
    chol3_solve(L, ek, col);
    for (int l = 0; l < 3; ++l) C[l][k] = col[l];
  }
  /* Eq. 17: dchi2 = 1/2 (alpha1 - alpha0) . dchi2/dalpha = step . g */
  *dchi2_o = step[0] * g[0] + step[1] * g[1] + step[2] * g[2];
  return 0;
}

static void trace_row(double *trace, int it, const double a[3], double C[3][3], double dchi2, double dz) {
  double *t = trace + (size_t)(it - 1) * PVO_TRACE_STRIDE;
  t[0] = a[0]; t[1] = a[1]; t[2] = a[2];
  t[3] = C[0][0]; t[4] = C[0][1]; t[5] = C[0][2]; t[6] = C[1][1]; t[7] = C[1][2]; t[8] = C[2][2];
  t[9] = dchi2; t[10] = dz;
}

static int fit_core(int m, const int32_t *idx,
                    const float *x, const float *y, const float *z, const float *tx, const float *ty,
                    const float *var_x, const float *var_y, const float *var_tx, const float *var_ty,
                    const double seed[3], const pvo_params *p, const double *other, const pvo_cross *cx,
                    double *out_pos, double *out_cov, double *out_chi2, int32_t *out_ntrk, int32_t *out_niter,
                    double *w, double *trace, fit_diag *diag) {
  double a[3] = {seed[0], seed[1], seed[2]};
  if (diag) { diag->edge_last = INFINITY; diag->edge_any = INFINITY; diag->pivot_min = INFINITY; diag->nact_min = 0x7fffffff; }
  double *Wx = (double *)malloc(sizeof(double) * (size_t)(2 * m + 2));
  double *Wy = Wx + m + 1;
  /* V_i = Eq. 2 at dz = z_seed - z_trk, diagonal input covariance; "evaluated and inverted
   * only once, using the vertex position of the seed". */
  for (int j = 0; j < m; ++j) {
    int i = idx[j];
    double dz = seed[2] - (double)z[i];
    double Vx = var_at((double)var_x[i], (double)var_tx[i], cx ? cx->xtx : NULL, i, dz);
    double Vy = var_at((double)var_y[i], (double)var_ty[i], cx ? cx->yty : NULL, i, dz);
    int ok = (Vx > 0.0) && (Vy > 0.0) && isfinite(Vx) && isfinite(Vy);
    Wx[j] = ok ? 1.0 / Vx : -1.0;                    /* -1 marks an unusable track: w = 0 always (R-7) */
    Wy[j] = ok ? 1.0 / Vy : -1.0;
  }
  const double chi2_max = (double)p->chi2_max;
  int rc = -1, niter = 0, nact = 0;
  double C[3][3] = {{0}}, chi2 = 0.0;
  for (int it = 1; it <= p->max_iter; ++it) {
    double step[3], dchi2;
    double edge = INFINITY, pivot = INFINITY;
    int frc = fit_iteration(m, idx, x, y, z, tx, ty, Wx, Wy, a, chi2_max, other, w, step, C, &dchi2, &chi2, &nact, &edge, &pivot);
    if (diag) {
      diag->edge_last = edge;
      if (edge < diag->edge_any) diag->edge_any = edge;
      if (pivot < diag->pivot_min) diag->pivot_min = pivot;
      if (nact < diag->nact_min) diag->nact_min = nact;
    }
    if (frc != 0) { rc = -1; break; }
    for (int k = 0; k < 3; ++k) a[k] += step[k];
    niter = it; rc = 0;
    if (trace && it <= PVO_TRACE_ITERS) trace_row(trace, it, a, C, dchi2, step[2]);
    /* convergence: x86 flavour |dchi2| < 0.01 and |dz| < 1 um; GPU flavour |dz| < 0.5 um only, which
     * is conv_dchi2 = INFINITY */
    if (fabs(dchi2) < (double)p->conv_dchi2 && fabs(step[2]) < (double)p->conv_dz) break;
  }
  /* Trace only (N1): keep iterating past the stopping point on COPIES, so that a
   * comparator can look up what one more iteration would have given.  Nothing below changes an output. */
  if (trace && rc == 0 && niter < p->max_iter) {
    double at[3] = {a[0], a[1], a[2]}, Ct[3][3], chi2t, dchi2t, stept[3];
    int nactt;
    double *wt = (double *)malloc(sizeof(double) * (size_t)(m + 1));
    for (int it = niter + 1; it <= p->max_iter && it <= PVO_TRACE_ITERS; ++it) {
      if (fit_iteration(m, idx, x, y, z, tx, ty, Wx, Wy, at, chi2_max, other, wt, stept, Ct, &dchi2t, &chi2t, &nactt, NULL, NULL) != 0) break;
      for (int k = 0; k < 3; ++k) at[k] += stept[k];
      trace_row(trace, it, at, Ct, dchi2t, stept[2]);
    }
    free(wt);
  }
  free(Wx);
  if (rc != 0) { *out_niter = -1; *out_ntrk = 0; return -1; }
  out_pos[0] = a[0]; out_pos[1] = a[1]; out_pos[2] = a[2];
  out_cov[0] = C[0][0]; out_cov[1] = C[0][1]; out_cov[2] = C[0][2];
  out_cov[3] = C[1][1]; out_cov[4] = C[1][2]; out_cov[5] = C[2][2];
  *out_chi2 = chi2; *out_ntrk = nact; *out_niter = niter;
  if (other) {                                        /* R-13: "associated" = final weight >= 1/2 */
    int na = 0;
    for (int j = 0; j < m; ++j) if (w[j] >= 0.5) ++na;
    *out_ntrk = na;
  }
  return 0;
}

int pvo_fit(int m, const int32_t *idx,
            const float *x, const float *y, const float *z, const float *tx, const float *ty,
            const float *var_x, const float *var_y, const float *var_tx, const float *var_ty,
            const double seed[3], const pvo_params *p, const pvo_cross *cx,
            double *out_pos, double *out_cov, double *out_chi2, int32_t *out_ntrk, int32_t *out_niter,
            double *w, double *trace) {
  return fit_core(m, idx, x, y, z, tx, ty, var_x, var_y, var_tx, var_ty, seed, p, NULL, cx, out_pos, out_cov, out_chi2,
                  out_ntrk, out_niter, w, trace, NULL);
}

/* Multi-vertex flavour: the same Newton-Raphson fit with the weights of Eq. 19.  other[j] is, for
 * listed track j, exp(-chi2_max / 2) + sum over the OTHER vertex candidates k of exp(-chi2_jk / 2) with chi2_jk
 * taken at their initial (seed) positions ("the weight is always calculated using the initial position of the
 * other vertices").  out_ntrk = tracks with final weight >= 1/2. */
int pvo_fit_mv(int m, const int32_t *idx,
               const float *x, const float *y, const float *z, const float *tx, const float *ty,
               const float *var_x, const float *var_y, const float *var_tx, const float *var_ty,
               const double seed[3], const pvo_params *p, const double *other, const pvo_cross *cx,
               double *out_pos, double *out_cov, double *out_chi2, int32_t *out_ntrk, int32_t *out_niter,
               double *w, double *trace) {
  return fit_core(m, idx, x, y, z, tx, ty, var_x, var_y, var_tx, var_ty, seed, p, other, cx, out_pos, out_cov, out_chi2,
                  out_ntrk, out_niter, w, trace, NULL);
}

/* chi2 of track i relative to a vertex candidate at pos[] "evaluated as in Eq. 7" with W from Eq. 2 at that
 * position; returns a negative number when the extrapolated variance is unusable (R-7). */
double pvo_track_chi2(int i, const float *x, const float *y, const float *z, const float *tx, const float *ty,
                      const float *var_x, const float *var_y, const float *var_tx, const float *var_ty,
                      const pvo_cross *cx, const double pos[3]) {
  double dz = pos[2] - (double)z[i];
  double Vx = var_at((double)var_x[i], (double)var_tx[i], cx ? cx->xtx : NULL, i, dz);
  double Vy = var_at((double)var_y[i], (double)var_ty[i], cx ? cx->yty : NULL, i, dz);
  if (!((Vx > 0.0) && (Vy > 0.0) && isfinite(Vx) && isfinite(Vy))) return -1.0;
  double rx = (double)x[i] + dz * (double)tx[i] - pos[0];
  double ry = (double)y[i] + dz * (double)ty[i] - pos[1];
  return rx * rx / Vx + ry * ry / Vy;
}

/* ===================================== NEXT-4: impact parameter ====================================== */
/* "the distance of closest approach of a track to a vertex, called impact parameter (IP) ... the IP chi2,
 * which is the chi2 difference of a PV reconstructed with and without the track under consideration".
 * For track i and a vertex (pos, C) that does NOT contain the track: r = Eq. 9 residual at the vertex z,
 * IP = distance of the straight line to the point; IP chi2 = r^T (V_i + H C H^T)^-1 r with V_i from Eq. 2 (diagonal)
 * at the vertex z and H of Eq. 12 -- the chi2 increase of the linear least-squares vertex when the track is added.
 * Returns 0, or -1 when the track covariance is unusable there (R-7) or the 2x2 matrix is not positive definite. */
int pvo_ip_one(int i, const float *x, const float *y, const float *z, const float *tx, const float *ty,
               const float *var_x, const float *var_y, const float *var_tx, const float *var_ty,
               const pvo_cross *cx, const double pos[3], const double C[6], double *ip, double *ip_chi2) {
  double dz = pos[2] - (double)z[i];
  double Vx = var_at((double)var_x[i], (double)var_tx[i], cx ? cx->xtx : NULL, i, dz);
  double Vy = var_at((double)var_y[i], (double)var_ty[i], cx ? cx->yty : NULL, i, dz);
  if (!((Vx > 0.0) && (Vy > 0.0) && isfinite(Vx) && isfinite(Vy))) return -1;
  double a = (double)tx[i], b = (double)ty[i];
  double rx = (double)x[i] + dz * a - pos[0];
  double ry = (double)y[i] + dz * b - pos[1];
  /* the point of the line at the vertex z is (rx, ry, 0) away; remove the component along (tx, ty, 1) */
  double along = (rx * a + ry * b) / sqrt(1.0 + a * a + b * b);
  double d2 = rx * rx + ry * ry - along * along;
  *ip = sqrt(d2 > 0.0 ? d2 : 0.0);
  /* H C H^T with H = [[-1, 0, tx], [0, -1, ty]], C = (xx, xy, xz, yy, yz, zz) */
  double Sxx = Vx + C[0] - 2.0 * a * C[2] + a * a * C[5];
  double Syy = Vy + C[3] - 2.0 * b * C[4] + b * b * C[5];
  double Sxy = C[1] - a * C[4] - b * C[2] + a * b * C[5];
  double det = Sxx * Syy - Sxy * Sxy;
  if (!(Sxx > 0.0) || !(det > 0.0)) return -1;
  *ip_chi2 = (Syy * rx * rx - 2.0 * Sxy * rx * ry + Sxx * ry * ry) / det;
  return 0;
}

/* Per track of a batch: the vertex of its event with the smallest IP chi2 (ties: lower index), that chi2 and the IP
 * to that vertex; ip_vertex = -1, ip = ip_chi2 = -1 when the event has no usable vertex for the track. */
int pvo_track_ip(const float *x, const float *y, const float *z, const float *tx, const float *ty,
                 const float *var_x, const float *var_y, const float *var_tx, const float *var_ty,
                 const pvo_cross *cx, const int32_t *offsets, int n_events, int max_vtx,
                 const double *vtx_pos, const double *vtx_cov, const int32_t *n_vtx,
                 double *ip, double *ip_chi2, int32_t *ip_vertex) {
  for (int e = 0; e < n_events; ++e)
    for (int t = offsets[e]; t < offsets[e + 1]; ++t) {
      ip[t] = -1.0; ip_chi2[t] = -1.0; ip_vertex[t] = -1;
      for (int v = 0; v < n_vtx[e] && v < max_vtx; ++v) {
        size_t o = (size_t)e * max_vtx + v;
        double d, c2;
        if (pvo_ip_one(t, x, y, z, tx, ty, var_x, var_y, var_tx, var_ty, cx, vtx_pos + 3 * o, vtx_cov + 6 * o, &d, &c2) != 0) continue;
        if (ip_vertex[t] < 0 || c2 < ip_chi2[t]) { ip[t] = d; ip_chi2[t] = c2; ip_vertex[t] = v; }
      }
    }
  return 0;
}

/* ===================================== whole path, one event ========================================= */
typedef struct scratch {
  int nbins, max_vtx;
  int32_t *H, *bin, *flags, *trk_seed, *cb, *ce, *cp, *idx, *s_ntrk, *s_niter, *fate;
  float *zp, *sp, *zs;
  double *s_pos, *s_cov, *s_chi2, *w, *trace;
  double *Em, *other, *best_w, *second_w;  /* multi-vertex flavour: exp(-chi2_ik / 2) at the seed positions [n][max_vtx] */
} scratch;

static scratch *scratch_new(const pvo_params *p) {
  scratch *s = (scratch *)calloc(1, sizeof(scratch));
  int nb = pvo_nbins(p), mv = p->max_vtx_per_event, nt = PVO_MAX_TRACKS + 1;
  s->nbins = nb; s->max_vtx = mv;
  s->H = (int32_t *)malloc(sizeof(int32_t) * (size_t)nb);
  s->bin = (int32_t *)malloc(sizeof(int32_t) * (size_t)nt * 4);
  s->flags = s->bin + nt; s->trk_seed = s->flags + nt; s->idx = s->trk_seed + nt;
  s->cb = (int32_t *)malloc(sizeof(int32_t) * (size_t)mv * 6);
  s->ce = s->cb + mv; s->cp = s->ce + mv; s->s_ntrk = s->cp + mv; s->s_niter = s->s_ntrk + mv; s->fate = s->s_niter + mv;
  s->zp = (float *)malloc(sizeof(float) * (size_t)nt * 2); s->sp = s->zp + nt;
  s->zs = (float *)malloc(sizeof(float) * (size_t)mv);
  s->s_pos = (double *)malloc(sizeof(double) * (size_t)mv * 10);
  s->s_cov = s->s_pos + 3 * mv; s->s_chi2 = s->s_cov + 6 * mv;
  s->w = (double *)malloc(sizeof(double) * (size_t)nt);
  s->trace = (double *)malloc(sizeof(double) * PVO_TRACE_ITERS * PVO_TRACE_STRIDE);
  s->Em = (double *)malloc(sizeof(double) * ((size_t)nt * (size_t)mv + 3 * (size_t)nt));
  s->other = s->Em + (size_t)nt * (size_t)mv; s->best_w = s->other + nt; s->second_w = s->best_w + nt;
  return s;
}

static void scratch_free(scratch *s) {
  free(s->H); free(s->bin); free(s->cb); free(s->zp); free(s->zs); free(s->s_pos); free(s->w); free(s->trace); free(s->Em); free(s);
}

static void find_event(int e, const float *x, const float *y, const float *z, const float *tx, const float *ty,
                       const float *var_x, const float *var_y, const float *var_tx, const float *var_ty,
                       const pvo_cross *cx_all, const int32_t *offsets, const pvo_params *p, scratch *S,
                       double *vtx_pos, double *vtx_cov, double *vtx_chi2, int32_t *vtx_ntracks, int32_t *vtx_niter,
                       int32_t *n_vtx, double *trk_weight, int32_t *trk_vertex, uint32_t *event_status,
                       const pvo_debug *dbg) {
  const int t0 = offsets[e], n = offsets[e + 1] - offsets[e];
  const int mv = p->max_vtx_per_event, nb = S->nbins;
  pvo_cross cxe = {cx_all && cx_all->xtx ? cx_all->xtx + t0 : NULL, cx_all && cx_all->yty ? cx_all->yty + t0 : NULL};
  const pvo_cross *cx = cx_all ? &cxe : NULL;             /* the event's slice of the cross terms */
  uint32_t status = 0;
  n_vtx[e] = 0;
  for (int i = 0; i < n; ++i) { trk_vertex[t0 + i] = -1; trk_weight[t0 + i] = 0.0; }
  if (dbg) {
    if (dbg->n_seeds) dbg->n_seeds[e] = 0;
    if (dbg->n_seeds_raw) dbg->n_seeds_raw[e] = 0;
    if (dbg->trk_seed) for (int i = 0; i < n; ++i) dbg->trk_seed[t0 + i] = -1;
    if (dbg->seed_niter) for (int k = 0; k < mv; ++k) dbg->seed_niter[(size_t)e * mv + k] = 0;
    if (dbg->seed_fate) for (int k = 0; k < mv; ++k) dbg->seed_fate[(size_t)e * mv + k] = -9;
  }
  if (n > PVO_MAX_TRACKS) { event_status[e] = PVO_EVT_TOO_MANY_TRACKS; return; }

  /* step 1: extrapolation to the point of closest approach */
  pvo_project(n, x + t0, y + t0, z + t0, tx + t0, ty + t0, var_x + t0, p, S->zp, S->sp, S->bin, S->flags);
  /* step 2: histogram filling */
  memset(S->H, 0, sizeof(int32_t) * (size_t)nb);
  if (p->fill_mode == 1) pvo_fill_template(n, S->zp, S->sp, S->bin, S->flags, p, S->H);
  else pvo_fill(n, S->zp, S->sp, S->flags, p, S->H, 0);
  /* step 3: peak search; clusters come out ordered in z */
  int n_raw = pvo_peaks(S->H, p, mv, S->cb, S->ce, S->cp);
  int ns = n_raw;
  if (ns > mv) { ns = mv; status |= PVO_EVT_VTX_OVERFLOW; }      /* first max_vtx in z kept (R-8) */
  for (int k = 0; k < ns; ++k) S->zs[k] = pvo_seed_z(S->H, S->cp[k], p);
  /* step 4: track association */
  const int mvf = p->flavour == 1;                /* multi-vertex (GPU) flavour: implicit association */
  if (!mvf) ns = pvo_assign(n, S->bin, S->flags, ns, S->cb, S->ce, S->cp, S->zs, p, S->trk_seed);
  else for (int i = 0; i < n; ++i) S->trk_seed[i] = -1;

  if (dbg) {
    if (dbg->hist && e < dbg->n_hist_events) memcpy(dbg->hist + (size_t)e * nb, S->H, sizeof(int32_t) * (size_t)nb);
    for (int i = 0; i < n; ++i) {
      if (dbg->z_poca) dbg->z_poca[t0 + i] = S->zp[i];
      if (dbg->sigma_poca) dbg->sigma_poca[t0 + i] = S->sp[i];
      if (dbg->trk_bin) dbg->trk_bin[t0 + i] = S->bin[i];
      if (dbg->trk_flags) dbg->trk_flags[t0 + i] = S->flags[i];
      if (dbg->trk_seed) dbg->trk_seed[t0 + i] = S->trk_seed[i];
    }
    if (dbg->n_seeds) dbg->n_seeds[e] = ns;
    if (dbg->n_seeds_raw) dbg->n_seeds_raw[e] = n_raw;
    for (int k = 0; k < ns; ++k) {
      if (dbg->seed_z) dbg->seed_z[(size_t)e * mv + k] = S->zs[k];
      if (dbg->seed_bins) {
        int32_t *sb = dbg->seed_bins + ((size_t)e * mv + k) * 3;
        sb[0] = S->cb[k]; sb[1] = S->ce[k]; sb[2] = S->cp[k];
      }
    }
  }

  /* step 5: vertex fit, one seed at a time */
  if (mvf) {
    /* R-13/R-14: every assignable track is implicitly associated to every vertex candidate; E_ik =
     * exp(-chi2_ik / 2) with chi2_ik "evaluated as in Eq. 7" at the candidates' initial (seed) positions */
    for (int i = 0; i < n; ++i) {
      S->best_w[i] = 0.0; S->second_w[i] = 0.0;
      for (int k = 0; k < ns; ++k) {
        float zs = S->zs[k];
        double pos[3] = {(double)fmaf(p->beam_tx, zs, p->beam_x), (double)fmaf(p->beam_ty, zs, p->beam_y), (double)zs};
        double c2 = (S->flags[i] & PVO_TRK_ASSIGNABLE)
                        ? pvo_track_chi2(i, x + t0, y + t0, z + t0, tx + t0, ty + t0, var_x + t0, var_y + t0, var_tx + t0, var_ty + t0, cx, pos)
                        : -1.0;
        S->Em[(size_t)i * mv + k] = c2 >= 0.0 ? c2 : -1.0;           /* chi2 kept; negative = not usable */
      }
    }
  }
  for (int k = 0; k < ns; ++k) {
    int m = 0;
    if (!mvf) {
      for (int i = 0; i < n; ++i) if (S->trk_seed[i] == k) S->idx[m++] = i;
    } else {
      /* "only tracks within a certain chi2_i with respect to the vertex candidate are considered" */
      for (int i = 0; i < n; ++i) {
        double c2 = S->Em[(size_t)i * mv + k];
        if (c2 < 0.0 || !(c2 < (double)p->chi2_window)) continue;
        double oth = exp(-0.5 * (double)p->chi2_max);
        for (int l = 0; l < ns; ++l) {
          double cl = S->Em[(size_t)i * mv + l];
          if (l != k && cl >= 0.0) oth += exp(-0.5 * cl);
        }
        S->other[m] = oth;
        S->idx[m++] = i;
      }
    }
    float zs = S->zs[k];
    /* "its xy position is evaluated using the known beamline" */
    double seed[3] = {(double)fmaf(p->beam_tx, zs, p->beam_x), (double)fmaf(p->beam_ty, zs, p->beam_y), (double)zs};
    double chi2 = 0.0;
    memset(S->trace, 0, sizeof(double) * PVO_TRACE_ITERS * PVO_TRACE_STRIDE);
    fit_diag diag;
    int rc = fit_core(m, S->idx, x + t0, y + t0, z + t0, tx + t0, ty + t0, var_x + t0, var_y + t0, var_tx + t0,
                      var_ty + t0, seed, p, mvf ? S->other : NULL, cx, S->s_pos + 3 * k, S->s_cov + 6 * k, &chi2,
                      &S->s_ntrk[k], &S->s_niter[k], S->w, S->trace, &diag);
    S->s_chi2[k] = chi2;
    if (dbg) {
      size_t o = (size_t)e * mv + k;
      if (dbg->seed_edge_last) dbg->seed_edge_last[o] = diag.edge_last;
      if (dbg->seed_edge_any) dbg->seed_edge_any[o] = diag.edge_any;
      if (dbg->seed_pivot_min) dbg->seed_pivot_min[o] = diag.pivot_min;
      if (dbg->seed_nact_min) dbg->seed_nact_min[o] = diag.nact_min;
    }
    if (rc != 0) { status |= PVO_EVT_SINGULAR_FIT; S->s_niter[k] = -1; }
    else if (!mvf) for (int j = 0; j < m; ++j) trk_weight[t0 + S->idx[j]] = S->w[j];
    else for (int j = 0; j < m; ++j) {                 /* R-13: a track follows the candidate with its largest weight */
      int i = S->idx[j];
      if (S->w[j] > S->best_w[i]) { S->second_w[i] = S->best_w[i]; S->best_w[i] = S->w[j]; S->trk_seed[i] = k; }
      else if (S->w[j] > S->second_w[i]) S->second_w[i] = S->w[j];     /* diagnostic only: the runner-up weight */
    }
    if (dbg && dbg->trace)
      memcpy(dbg->trace + ((size_t)e * mv + k) * PVO_TRACE_ITERS * PVO_TRACE_STRIDE, S->trace,
             sizeof(double) * PVO_TRACE_ITERS * PVO_TRACE_STRIDE);
  }
  if (mvf) {
    for (int i = 0; i < n; ++i) trk_weight[t0 + i] = S->trk_seed[i] >= 0 ? S->best_w[i] : 0.0;
    if (dbg && dbg->trk_seed) for (int i = 0; i < n; ++i) dbg->trk_seed[t0 + i] = S->trk_seed[i];
    if (dbg && dbg->trk_w2) for (int i = 0; i < n; ++i) dbg->trk_w2[t0 + i] = S->second_w[i];
    if (dbg && dbg->trk_w1) for (int i = 0; i < n; ++i) dbg->trk_w1[t0 + i] = S->best_w[i];
  }

  /* cleanup O8.  Duplicate removal: greedy sweep in seed (= z) order; duplicate iff
   * (z_v - z_s)^2 / (C_zz,v + C_zz,s) < merge_ratio; the one "with fewer associated tracks" is rejected,
   * ties keep the lower z (R-9). */
  for (int k = 0; k < ns; ++k) S->fate[k] = S->s_niter[k] < 0 ? -1 : 0;
  int s = -1;
  for (int v = 0; v < ns; ++v) {
    if (S->fate[v] != 0) continue;
    if (s < 0) { s = v; continue; }
    double dzv = S->s_pos[3 * v + 2] - S->s_pos[3 * s + 2];
    double ratio = dzv * dzv / (S->s_cov[6 * v + 5] + S->s_cov[6 * s + 5]);
    if (ratio < (double)p->merge_ratio) {
      if (S->s_ntrk[v] > S->s_ntrk[s]) { S->fate[s] = -2; s = v; }
      else S->fate[v] = -2;
    } else s = v;
  }
  /* "Min. tracks in the PV" (Table 2) and the beamline distance cut for pp vertices */
  for (int k = 0; k < ns; ++k) {
    if (S->fate[k] != 0) continue;
    double vz = S->s_pos[3 * k + 2];
    int region = vz < (double)p->z_split ? 1 : 0;
    if (S->s_ntrk[k] < p->min_tracks_pv[region]) { S->fate[k] = -3; continue; }
    if (region == 0) {
      double dx = S->s_pos[3 * k] - ((double)p->beam_x + (double)p->beam_tx * vz);
      double dy = S->s_pos[3 * k + 1] - ((double)p->beam_y + (double)p->beam_ty * vz);
      if (dx * dx + dy * dy > (double)p->max_beam_dist * (double)p->max_beam_dist) S->fate[k] = -4;
    }
  }
  int nv = 0;
  for (int k = 0; k < ns; ++k) {
    if (S->fate[k] != 0) continue;
    size_t o = (size_t)e * mv + nv;
    for (int c = 0; c < 3; ++c) vtx_pos[o * 3 + c] = S->s_pos[3 * k + c];
    for (int c = 0; c < 6; ++c) vtx_cov[o * 6 + c] = S->s_cov[6 * k + c];
    vtx_chi2[o] = S->s_chi2[k]; vtx_ntracks[o] = S->s_ntrk[k]; vtx_niter[o] = S->s_niter[k];
    S->fate[k] = nv + 1000;                          /* temporarily: survivor index + 1000 */
    ++nv;
  }
  n_vtx[e] = nv;
  /* tracks of rejected vertices are released: trk_vertex = -1, weight 0 (R-9) */
  for (int i = 0; i < n; ++i) {
    int k = S->trk_seed[i];
    if (k >= 0 && S->fate[k] >= 1000) trk_vertex[t0 + i] = S->fate[k] - 1000;
    else { trk_vertex[t0 + i] = -1; trk_weight[t0 + i] = 0.0; }
  }
  if (dbg) for (int k = 0; k < ns; ++k) {
    size_t o = (size_t)e * mv + k;
    if (dbg->seed_pos) for (int c = 0; c < 3; ++c) dbg->seed_pos[o * 3 + c] = S->s_pos[3 * k + c];
    if (dbg->seed_cov) for (int c = 0; c < 6; ++c) dbg->seed_cov[o * 6 + c] = S->s_cov[6 * k + c];
    if (dbg->seed_chi2) dbg->seed_chi2[o] = S->s_chi2[k];
    if (dbg->seed_ntrk) dbg->seed_ntrk[o] = S->s_ntrk[k];
    if (dbg->seed_niter) dbg->seed_niter[o] = S->s_niter[k];
    if (dbg->seed_fate) dbg->seed_fate[o] = S->fate[k] >= 1000 ? S->fate[k] - 1000 : S->fate[k];
  }
  event_status[e] = status;
}

int pvo_find(const float *x, const float *y, const float *z, const float *tx, const float *ty,
             const float *var_x, const float *var_y, const float *var_tx, const float *var_ty,
             const pvo_cross *cx, const int32_t *offsets, int n_events, const pvo_params *p,
             double *vtx_pos, double *vtx_cov, double *vtx_chi2, int32_t *vtx_ntracks, int32_t *vtx_niter,
             int32_t *n_vtx, double *trk_weight, int32_t *trk_vertex, uint32_t *event_status,
             const pvo_debug *dbg, int n_threads) {
  if (!p || !offsets || n_events < 0) return -1;
  int nb = pvo_nbins(p);
  if (!(p->dz > 0.0f) || nb <= 0 || p->max_vtx_per_event <= 0 || p->max_iter <= 0) return -2;
  if (fabs((double)nb * (double)p->dz - ((double)p->z_max - (double)p->z_min)) > 1e-6 * (double)p->dz) return -2;
  if (n_threads < 1) n_threads = 1;
#pragma omp parallel num_threads(n_threads)
  {
    scratch *S = scratch_new(p);
#pragma omp for schedule(dynamic, 64)
    for (int e = 0; e < n_events; ++e)
      find_event(e, x, y, z, tx, ty, var_x, var_y, var_tx, var_ty, cx, offsets, p, S, vtx_pos, vtx_cov, vtx_chi2,
                 vtx_ntracks, vtx_niter, n_vtx, trk_weight, trk_vertex, event_status, dbg);
    scratch_free(S);
  }
  return 0;
}

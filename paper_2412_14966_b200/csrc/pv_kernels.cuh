// pv_kernels.cuh -- sm_100a kernels of the PV-finder hot path (arXiv:2412.14966, "P:Lnn" = PAPER.md line nn).
//
// Execution model: ONE WARP PER EVENT.  A persistent grid of one CTA per
// SM holds as many warps as per-event shared-memory histograms fit ("one block per event",
// re-cut for 117-track events: a warp owns an event end to end, so every step is synchronised with
// __syncwarp / shuffles / ballots only and nothing goes through HBM between the steps).  Warps pull
// event indices from a global counter.  Steps a1..a6 of include/pv_finder.h run back to back:
//
//   a1+a2  thread per track: POCA projection (fp32 contract, bit-exact with the CPU oracle) and
//          fixed-point Gaussian bin integrals added to the warp's int32 shared-memory histogram
//   a3     ballot bitmap of bins above threshold -> proto-cluster starts -> one lane per proto-cluster
//          runs the z-ordered hysteresis sweep; warp scan orders the emitted seed clusters in z
//   a4     partition points, per-track seed by comparison, ballot counting, removal loop,
//          match_any counting sort of the tracks by seed
//   a5     8 lanes per vertex (4 vertices per warp pass), tracks register-resident, xor-shuffle
//          reduction of the normal equations, closed-form 3x3 solve of the arrow-shaped Hessian
//   a6     z-ordered duplicate sweep, cuts, compaction, final per-track outputs
//
// This file shares nothing with oracle/ (the frozen CDF coefficients below are the numbers of
// DESIGN.md "CDF contract", restated).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/pv_finder.h"

namespace pvk {

constexpr unsigned FULL = 0xffffffffu;
constexpr int MAX_TRK = PV_MAX_TRACKS_PER_EVENT;
constexpr int MAXV = PV_MAX_VTX;
constexpr int FIT_G = 8;            // lanes per vertex in the fit
constexpr int FIT_VPW = 32 / FIT_G; // vertices per warp pass
constexpr int FIT_KF = 6;           // register-resident tracks per lane (fast path: <= FIT_G*FIT_KF tracks)

// Per-warp shared-memory layout (bytes).  Region 0 holds the histogram during a1-a3 and is re-used
// (the histogram is dead once the seed positions are known) for the seed-sorted track index list and
// the per-vertex fit results during a4-a6.
constexpr int OVL_SIDX_BYTES = 4096;                 // uint16 sidx[2048]
constexpr int OVL_VTX_FIELDS = 13;                   // pos3 cov6 chi2 ntrk niter = 12, +1 spare
constexpr int OVL_MIN_BYTES = OVL_SIDX_BYTES + OVL_VTX_FIELDS * MAXV * 4;
constexpr int R1_BYTES = 1296;                       // peaks: bm[128] sbw[128] cum[130 u16]; assign: cnt cur part off
constexpr int R2_BYTES = 4 * MAXV * 4;               // seeds: begin end peak z

struct KParams {
  float z_min, dz, inv_dz, z_split;
  float beam_x, beam_y, beam_tx, beam_ty;
  float max_sigma[2];
  float win_eps;                 // safety margin of the fill window, in bins
  int nbins, nwords;             // nwords = ceil(nbins / 32)
  int T_bin, D;                  // thresholds in fixed point, clamped to int32
  long long I_min[2];
  int min_tracks_seed[2], min_tracks_pv[2];
  float chi2_max, inv_chi2_max;
  int unit_weights;              // chi2_max == inf
  int max_iter;
  float conv_dchi2, conv_dz, merge_ratio, max_beam_dist2;
  int max_vtx;
  int region0_words;             // int32 words of region 0 (multiple of 4)
  int warp_smem_bytes;
};

struct KArgs {
  const float *x, *y, *z, *tx, *ty, *var_x, *var_y, *var_tx, *var_ty;
  const int32_t* offsets;
  int n_events;
  float *vtx_pos, *vtx_cov, *vtx_chi2;
  int32_t *vtx_ntracks, *vtx_niter, *n_vtx;
  float* trk_weight;
  int32_t* trk_vertex;
  uint32_t* event_status;
  unsigned int* counter;
  pv_debug dbg;
};

// ---- frozen CDF contract: F(u) = 1/2 + s*G(s^2), s = u/3, odd degree-13 polynomial; the seven
// fp32 coefficients are literals inside edge_q() ---------------------------------------------------------------

__device__ __forceinline__ unsigned lanemask_lt() {
  unsigned m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

// Fixed-point CDF at the bin edge with float index kf (contract: every op rounded once).
__device__ __forceinline__ int edge_q(float kf, float zp, float inv, const KParams& P) {
  const float e = __fmaf_rn(kf, P.dz, P.z_min);
  const float s = __fmul_rn(__fsub_rn(e, zp), inv);
  const float t = __fmul_rn(s, s);
  float g = 0x1.3e0392p-3f;
  g = __fmaf_rn(g, t, -0x1.862240p-1f);
  g = __fmaf_rn(g, t, 0x1.b67296p+0f);
  g = __fmaf_rn(g, t, -0x1.3336f8p+1f);
  g = __fmaf_rn(g, t, 0x1.32067cp+1f);
  g = __fmaf_rn(g, t, -0x1.cbf272p+0f);
  g = __fmaf_rn(g, t, 0x1.3331cep+0f);
  float c = __saturatef(__fmaf_rn(s, g, 0.5f));
  int q = __float2int_rn(__fmul_rn(c, 1048576.0f));
  q = (s <= -1.0f) ? 0 : q;
  q = (s >= 1.0f) ? PV_FIXED_ONE : q;
  return q;
}

__device__ __forceinline__ int bin_region(int b, const KParams& P) {
  const float centre = __fmaf_rn(__fadd_rn((float)b, 0.5f), P.dz, P.z_min);
  return centre < P.z_split ? 1 : 0;
}

__device__ __forceinline__ int warp_incl_scan(int v, int lane) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int u = __shfl_up_sync(FULL, v, o);
    if (lane >= o) v += u;
  }
  return v;
}

// ---- a3: z-ordered hysteresis sweep over one proto-cluster starting at bin b0 (R-4) --------
// Returns the number of seed clusters the proto-cluster yields.  With WRITE, cluster j is stored at
// index base + j of (sb, se, sp) when that is < max_vtx.
template <bool WRITE>
__device__ int sweep(const int* __restrict__ H, int b0, const KParams& P, int base, int* sb, int* se, int* sp) {
  int start = b0;
  int h = H[b0];
  bool look_max = true;
  int mx = h, mn = 0, mnp = b0;
  long long sum = h;                         // integral of [start, k]
  int amax = h, amaxp = b0;                  // argmax of [start, k], ties -> lowest bin
  long long snap_sum = 0;                    // the same over [start, mnp)
  int snap_amax = 0, snap_amaxp = b0;
  int smax = h, smaxp = b0;                  // argmax of [mnp, k]
  int count = 0;
  bool have = false;                         // last emitted cluster, held back because the tail may join it
  int lb = 0, le = 0, lp = 0, lpv = 0, lj = 0;
  int k = b0 + 1;
  for (; k < P.nbins; ++k) {
    h = H[k];
    if (!(h > P.T_bin)) break;
    const long long prev_sum = sum;
    const int prev_amax = amax, prev_amaxp = amaxp;
    sum += h;
    if (h > amax) { amax = h; amaxp = k; }
    if (h > smax) { smax = h; smaxp = k; }
    if (look_max) {
      if (h > mx) {
        mx = h;
      } else if (mx - h > P.D) {             // a significant maximum lies behind: start looking for the minimum
        mn = h; mnp = k; look_max = false;
        snap_sum = prev_sum; snap_amax = prev_amax; snap_amaxp = prev_amaxp;
        smax = h; smaxp = k;
      }
    } else {
      if (h < mn) {
        mn = h; mnp = k;
        snap_sum = prev_sum; snap_amax = prev_amax; snap_amaxp = prev_amaxp;
        smax = h; smaxp = k;
      } else if (h - mn > P.D) {             // significant minimum at mnp, with a maximum on either side
        mx = h; look_max = true;
        if (snap_sum >= P.I_min[bin_region(snap_amaxp, P)]) {
          if (WRITE && have && base + lj < P.max_vtx) { sb[base + lj] = lb; se[base + lj] = le; sp[base + lj] = lp; }
          lb = start; le = mnp; lp = snap_amaxp; lpv = snap_amax; lj = count; have = true;
          ++count;
          start = mnp;                       // the minimum bin opens the right-hand cluster
          sum -= snap_sum; amax = smax; amaxp = smaxp;
        }
      }
    }
  }
  // tail [start, k)
  if (sum >= P.I_min[bin_region(amaxp, P)]) {
    if (WRITE && have && base + lj < P.max_vtx) { sb[base + lj] = lb; se[base + lj] = le; sp[base + lj] = lp; }
    lb = start; le = k; lp = amaxp; lj = count; have = true;
    ++count;
  } else if (have) {                         // remainder joins the last cluster of this proto-cluster
    le = k;
    if (amax > lpv) { lp = amaxp; lpv = amax; }
  }
  if (WRITE && have && base + lj < P.max_vtx) { sb[base + lj] = lb; se[base + lj] = le; sp[base + lj] = lp; }
  return count;
}

// ---- a5: one track's contribution to the normal equations (Eq. 6-12, 18) -------------------------------
struct Sums {
  float a, b, c, d, e;     // sum wWx, wWy, wWx tx, wWy ty, w(Wx tx^2 + Wy ty^2)   (Eq. 11 / 2)
  float gx, gy, gz;        // sum wWx rx, wWy ry, w(Wx tx rx + Wy ty ry)           (Eq. 10 / 2, signs in solve)
  float chi2;              // sum w chi2_i                                         (Eq. 6)
  float nact;              // tracks with w > 0
};

__device__ __forceinline__ void sums_zero(Sums& S) {
  S.a = S.b = S.c = S.d = S.e = S.gx = S.gy = S.gz = S.chi2 = S.nact = 0.0f;
}

template <int WIDTH>
__device__ __forceinline__ void sums_reduce(Sums& S) {
#pragma unroll
  for (int o = WIDTH / 2; o > 0; o >>= 1) {
    S.a += __shfl_xor_sync(FULL, S.a, o);
    S.b += __shfl_xor_sync(FULL, S.b, o);
    S.c += __shfl_xor_sync(FULL, S.c, o);
    S.d += __shfl_xor_sync(FULL, S.d, o);
    S.e += __shfl_xor_sync(FULL, S.e, o);
    S.gx += __shfl_xor_sync(FULL, S.gx, o);
    S.gy += __shfl_xor_sync(FULL, S.gy, o);
    S.gz += __shfl_xor_sync(FULL, S.gz, o);
    S.chi2 += __shfl_xor_sync(FULL, S.chi2, o);
    S.nact += __shfl_xor_sync(FULL, S.nact, o);
  }
}

// Returns the Tukey weight of the track at the current vertex (ax, ay, az); Wx < 0 marks an unusable track.
__device__ __forceinline__ float track_accum(float x, float y, float z, float tx, float ty, float Wx, float Wy,
                                             float ax, float ay, float az, const KParams& P, Sums& S) {
  if (!(Wx > 0.0f)) return 0.0f;
  const float dz = az - z;
  const float rx = fmaf(dz, tx, x) - ax;               // residual, Eq. 9
  const float ry = fmaf(dz, ty, y) - ay;
  const float cx = rx * Wx, cy = ry * Wy;
  const float chi = fmaf(rx, cx, ry * cy);             // Eq. 7
  float w;
  if (P.unit_weights) {
    w = 1.0f;
  } else {
    const float u = fmaxf(fmaf(chi, -P.inv_chi2_max, 1.0f), 0.0f);
    w = chi < P.chi2_max ? u * u : 0.0f;               // Tukey bi-square, Eq. 18
  }
  const float wWx = w * Wx, wWy = w * Wy;
  const float p = wWx * tx, q = wWy * ty;
  S.a += wWx; S.b += wWy; S.c += p; S.d += q;
  S.e = fmaf(p, tx, fmaf(q, ty, S.e));
  const float wcx = w * cx, wcy = w * cy;
  S.gx += wcx; S.gy += wcy;
  S.gz = fmaf(wcx, tx, fmaf(wcy, ty, S.gz));
  S.chi2 = fmaf(w, chi, S.chi2);
  S.nact += (w > 0.0f) ? 1.0f : 0.0f;
  return w;
}

// Newton-Raphson step Eq. 13 on the arrow-shaped Hessian A = [[a,0,-c],[0,b,-d],[-c,-d,e]]:
// returns false when the fit is singular (fewer than 2 active tracks or a non-positive pivot).
__device__ __forceinline__ bool newton_step(const Sums& S, float& dx, float& dy, float& dzs, float& dchi2) {
  if (S.nact < 2.0f) return false;
  if (!(S.a > 0.0f) || !(S.b > 0.0f)) return false;
  const float ia = 1.0f / S.a, ib = 1.0f / S.b;
  const float ca = S.c * ia, db = S.d * ib;
  const float sch = S.e - S.c * ca - S.d * db;         // Schur complement = third Cholesky pivot squared
  if (!(sch > 0.0f)) return false;
  dzs = (ca * S.gx + db * S.gy - S.gz) / sch;
  dx = (S.gx + S.c * dzs) * ia;
  dy = (S.gy + S.d * dzs) * ib;
  dchi2 = dzs * S.gz - dx * S.gx - dy * S.gy;          // Eq. 17
  return true;
}

// C = A^-1 (Eq. 14), upper triangle xx xy xz yy yz zz.
__device__ __forceinline__ void covariance(const Sums& S, float* C) {
  const float ia = 1.0f / S.a, ib = 1.0f / S.b;
  const float ca = S.c * ia, db = S.d * ib;
  const float is = 1.0f / (S.e - S.c * ca - S.d * db);
  C[0] = fmaf(ca * ca, is, ia);
  C[1] = ca * db * is;
  C[2] = ca * is;
  C[3] = fmaf(db * db, is, ib);
  C[4] = db * is;
  C[5] = is;
}

// W = V^-1 "evaluated and inverted only once, using the vertex position of the seed", Eq. 2 diagonal.
__device__ __forceinline__ void track_weight_matrix(float zl, float vx, float vy, float vtx, float vty,
                                                    float& Wx, float& Wy) {
  const float dz2 = zl * zl;                               // zl = z_trk - z_seed
  const float Vx = fmaf(dz2, vtx, vx), Vy = fmaf(dz2, vty, vy);
  const bool ok = (Vx > 0.0f) && (Vy > 0.0f) && (Vx < INFINITY) && (Vy < INFINITY);
  Wx = ok ? 1.0f / Vx : -1.0f;
  Wy = ok ? 1.0f / Vy : -1.0f;
}

// ---- one event, one warp ---------------------------------------------------------------------------------
template <bool DBG>
__device__ void process_event(const int e, const KParams& P, const KArgs& A, unsigned char* wsm, const int lane) {
  int* H = reinterpret_cast<int*>(wsm);
  uint16_t* sidx = reinterpret_cast<uint16_t*>(wsm);                       // overlay, valid after a3
  float* V = reinterpret_cast<float*>(wsm + OVL_SIDX_BYTES);              // overlay: V[f * MAXV + k]
  unsigned char* r1 = wsm + (size_t)P.region0_words * 4;
  unsigned* bm = reinterpret_cast<unsigned*>(r1);                          // peaks
  unsigned* sbw = bm + 128;
  uint16_t* cum = reinterpret_cast<uint16_t*>(sbw + 128);
  int* cnt = reinterpret_cast<int*>(r1);                                   // assign (after peaks)
  int* cur = cnt + MAXV;
  int* part = cur + MAXV;
  int* off = part + MAXV;                                                  // MAXV + 1 entries
  int* sb = reinterpret_cast<int*>(r1 + R1_BYTES);
  int* se = sb + MAXV;
  int* sp = se + MAXV;
  float* zs = reinterpret_cast<float*>(sp + MAXV);

  const int t0 = A.offsets[e];
  const int n = A.offsets[e + 1] - t0;
  const size_t ev = (size_t)e * P.max_vtx;
  unsigned status = 0;

  if (n > MAX_TRK) {
    for (int i = lane; i < n; i += 32) { A.trk_vertex[t0 + i] = -1; A.trk_weight[t0 + i] = 0.0f; }
    if (DBG && A.dbg.trk_seed) for (int i = lane; i < n; i += 32) A.dbg.trk_seed[t0 + i] = -1;
    if (lane == 0) {
      A.n_vtx[e] = 0;
      A.event_status[e] = PV_EVT_TOO_MANY_TRACKS;
      if (DBG && A.dbg.n_seeds) A.dbg.n_seeds[e] = 0;
      if (DBG && A.dbg.n_seeds_raw) A.dbg.n_seeds_raw[e] = 0;
    }
    return;
  }

  // ================= a1 + a2: projection (Eq. 1, Eq. 3) and histogram fill ===================
  for (int i = lane; i < n; i += 32) {
    const int t = t0 + i;
    const float x = __ldg(A.x + t), y = __ldg(A.y + t), z = __ldg(A.z + t);
    const float tx = __ldg(A.tx + t), ty = __ldg(A.ty + t), vx = __ldg(A.var_x + t);
    const float dtx = __fsub_rn(tx, P.beam_tx), dty = __fsub_rn(ty, P.beam_ty);
    const float den = __fmaf_rn(dty, dty, __fmul_rn(dtx, dtx));
    float zp = __int_as_float(0x7fc00000), sg = zp;
    int bin = -1;
    bool fill = false;
    float inv = 0.0f;
    if (den >= 1e-12f) {                                  // R-3: not parallel to the beamline
      const float bx = __fmaf_rn(P.beam_tx, z, P.beam_x), by = __fmaf_rn(P.beam_ty, z, P.beam_y);
      const float num = __fmaf_rn(dty, __fsub_rn(by, y), __fmul_rn(dtx, __fsub_rn(bx, x)));
      zp = __fadd_rn(z, __fdiv_rn(num, den));
      sg = __fsqrt_rn(__fdiv_rn(vx, den));
      const float fb = floorf(__fmul_rn(__fsub_rn(zp, P.z_min), P.inv_dz));
      if (fb >= 0.0f && fb < (float)P.nbins) {
        bin = (int)fb;
        const int region = zp < P.z_split ? 1 : 0;
        inv = __fdiv_rn(1.0f, __fmul_rn(3.0f, sg));
        fill = sg > 0.0f && sg <= P.max_sigma[region] && inv < INFINITY;
      }
    }
    A.trk_vertex[t] = bin;                                // scratch: central bin, read back in a4
    if (DBG) {
      if (A.dbg.z_poca) A.dbg.z_poca[t] = zp;
      if (A.dbg.sigma_poca) A.dbg.sigma_poca[t] = sg;
      if (A.dbg.trk_bin) A.dbg.trk_bin[t] = bin;
    }
    if (fill) {
      // window: a superset of the +-3 sigma support; edges outside it give exactly 0 or 2^20
      const float w3 = 3.0f * sg;
      const float fa = floorf((zp - w3 - P.z_min) * P.inv_dz - P.win_eps);
      const float fb2 = floorf((zp + w3 - P.z_min) * P.inv_dz + P.win_eps) + 1.0f;
      const int lo = (int)fmaxf(fa, 0.0f);
      const int hi = (int)fminf(fb2, (float)P.nbins);
      float kf = (float)lo;
      int q0 = edge_q(kf, zp, inv, P);
      for (int b = lo; b < hi; ++b) {
        kf += 1.0f;
        const int q1 = edge_q(kf, zp, inv, P);
        const int d = q1 - q0;
        if (d != 0) atomicAdd(&H[b], d);
        q0 = q1;
      }
    }
  }
  __syncwarp();

  if (DBG && A.dbg.hist && e < A.dbg.n_hist_events)
    for (int b = lane; b < P.nbins; b += 32) A.dbg.hist[(size_t)e * P.nbins + b] = H[b];

  // ================= a3: peak search and seed position (Eq. 4-5) ==============================
  const int nw = P.nwords;
  for (int w = 0; w < nw; ++w) {
    const int b = w * 32 + lane;
    const int v = b < P.nbins ? H[b] : 0;
    const unsigned m = __ballot_sync(FULL, v > P.T_bin);
    if (lane == 0) bm[w] = m;
  }
  __syncwarp();
  int n_proto = 0;
  for (int w0 = 0; w0 < nw; w0 += 32) {
    const int w = w0 + lane;
    unsigned sbits = 0;
    if (w < nw) {
      const unsigned m = bm[w];
      const unsigned prev = w > 0 ? (bm[w - 1] >> 31) : 0u;
      sbits = m & ~((m << 1) | prev);                     // first bin of each run of bins above threshold
      sbw[w] = sbits;
    }
    const int c = __popc(sbits);
    const int inc = warp_incl_scan(c, lane);
    if (w < nw) cum[w] = (uint16_t)(n_proto + inc - c);
    n_proto += __shfl_sync(FULL, inc, 31);
  }
  if (lane == 0) cum[nw] = (uint16_t)n_proto;
  __syncwarp();

  int n_raw = 0;
  for (int p0 = 0; p0 < n_proto; p0 += 32) {
    const int p = p0 + lane;
    int b0 = -1, c = 0;
    if (p < n_proto) {
      int lo = 0, hi = nw;                                // largest w with cum[w] <= p
      while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if ((int)cum[mid] <= p) lo = mid; else hi = mid;
      }
      unsigned sbits = sbw[lo];
      for (int r = p - (int)cum[lo]; r > 0; --r) sbits &= sbits - 1;
      b0 = lo * 32 + __ffs(sbits) - 1;
      c = sweep<false>(H, b0, P, 0, sb, se, sp);
    }
    const int inc = warp_incl_scan(c, lane);
    const int base = n_raw + inc - c;
    if (c > 0 && base < P.max_vtx) sweep<true>(H, b0, P, base, sb, se, sp);
    n_raw += __shfl_sync(FULL, inc, 31);
  }
  int ns = n_raw;
  if (ns > P.max_vtx) { ns = P.max_vtx; status |= PV_EVT_VTX_OVERFLOW; }   // R-8: first max_vtx in z kept
  __syncwarp();
  if (lane < ns) {                                         // Eq. 4-5: neighbours are raw bins, 0 beyond the ends
    const int i = sp[lane];
    const long long Nm = i > 0 ? H[i - 1] : 0;
    const long long Np = i < P.nbins - 1 ? H[i + 1] : 0;
    const long long N0 = H[i];
    const long long num = Np - Nm, den = 2 * N0 - Np - Nm;
    const float delta = den > 0 ? __fmul_rn(0.5f, __fdiv_rn((float)num, (float)den)) : 0.0f;
    const float zi = __fmaf_rn(__fadd_rn((float)i, 0.5f), P.dz, P.z_min);
    zs[lane] = __fmaf_rn(delta, P.dz, zi);
  }
  __syncwarp();                                            // histogram is dead from here on

  // ================= a4: association =========================================================
  int mycnt = 0;
  for (;;) {
    if (ns == 0) break;
    if (lane + 1 < ns) part[lane] = (se[lane] + sb[lane + 1]) / 2;   // bins < part[k] belong to seed <= k
    __syncwarp();
    mycnt = 0;
    for (int i0 = 0; i0 < n; i0 += 32) {
      const int i = i0 + lane;
      int s = -1;
      if (i < n) {
        const int b = A.trk_vertex[t0 + i];
        if (b >= 0) {
          s = 0;
          for (int k = 0; k + 1 < ns; ++k) s += (b >= part[k]) ? 1 : 0;
        }
      }
      for (int k = 0; k < ns; ++k) {
        const int c = __popc(__ballot_sync(FULL, s == k));
        if (lane == k) mycnt += c;
      }
    }
    // "the seed cluster is removed ... and the procedure is repeated": least populated, ties lowest z
    int key = 0x7fffffff;
    if (lane < ns) {
      const int region = zs[lane] < P.z_split ? 1 : 0;
      if (mycnt < P.min_tracks_seed[region]) key = (mycnt << 6) | lane;
    }
    key = __reduce_min_sync(FULL, key);
    if (key == 0x7fffffff) break;
    const int worst = key & 63;
    int nb = 0, ne = 0, np = 0;
    float nz = 0.0f;
    const bool mv = lane >= worst && lane + 1 < ns;
    if (mv) { nb = sb[lane + 1]; ne = se[lane + 1]; np = sp[lane + 1]; nz = zs[lane + 1]; }
    __syncwarp();
    if (mv) { sb[lane] = nb; se[lane] = ne; sp[lane] = np; zs[lane] = nz; }
    --ns;
    __syncwarp();
  }
  // counting sort of the tracks by seed (deterministic: track order is kept inside a seed)
  {
    const int c = lane < ns ? mycnt : 0;
    const int inc = warp_incl_scan(c, lane);
    if (lane < ns) { cnt[lane] = c; off[lane] = inc - c; cur[lane] = inc - c; }
    if (lane == 31) off[ns < MAXV ? ns : MAXV] = inc;
  }
  __syncwarp();
  for (int i0 = 0; i0 < n; i0 += 32) {
    const int i = i0 + lane;
    int s = -1;
    if (i < n) {
      const int b = A.trk_vertex[t0 + i];
      if (b >= 0 && ns > 0) {
        s = 0;
        for (int k = 0; k + 1 < ns; ++k) s += (b >= part[k]) ? 1 : 0;
      }
      A.trk_vertex[t0 + i] = s;                           // scratch: seed index, read back in a6
      if (DBG && A.dbg.trk_seed) A.dbg.trk_seed[t0 + i] = s;
    }
    const unsigned m = __match_any_sync(FULL, s);
    const int rank = __popc(m & lanemask_lt());
    if (s >= 0) sidx[cur[s] + rank] = (uint16_t)i;
    __syncwarp();
    if (s >= 0 && rank == 0) cur[s] += __popc(m);
    __syncwarp();
  }
  if (DBG) {
    if (lane == 0) {
      if (A.dbg.n_seeds) A.dbg.n_seeds[e] = ns;
      if (A.dbg.n_seeds_raw) A.dbg.n_seeds_raw[e] = n_raw;
    }
    if (lane < ns) {
      if (A.dbg.seed_z) A.dbg.seed_z[ev + lane] = zs[lane];
      if (A.dbg.seed_bins) {
        A.dbg.seed_bins[(ev + lane) * 3 + 0] = sb[lane];
        A.dbg.seed_bins[(ev + lane) * 3 + 1] = se[lane];
        A.dbg.seed_bins[(ev + lane) * 3 + 2] = sp[lane];
      }
    }
  }

  // ================= a5: adaptive vertex fit =================================================
  // Fast path: FIT_G lanes per vertex, tracks register-resident.
  for (int v0 = 0; v0 < ns; v0 += FIT_VPW) {
    const int v = v0 + lane / FIT_G, j = lane % FIT_G;
    const bool vact = v < ns;
    int m = vact ? cnt[v] : 0;
    const int o = vact ? off[v] : 0;
    const bool big = m > FIT_G * FIT_KF;
    if (big) m = 0;
    const float zsv = vact ? zs[v] : 0.0f;
    const float sx = __fmaf_rn(P.beam_tx, zsv, P.beam_x);  // "xy position ... using the known beamline"
    const float sy = __fmaf_rn(P.beam_ty, zsv, P.beam_y);
    // The fit runs in the seed's local frame (x - sx, y - sy, z - zseed): every quantity is O(mm), so fp32
    // keeps ~1e-7 mm instead of ulp(550 mm) = 6e-5 mm, and the iterates follow the fp64 oracle.
    float ax = 0.0f, ay = 0.0f, az = 0.0f;
    float fx[FIT_KF], fy[FIT_KF], fz[FIT_KF], ftx[FIT_KF], fty[FIT_KF], fWx[FIT_KF], fWy[FIT_KF], fw[FIT_KF];
#pragma unroll
    for (int s = 0; s < FIT_KF; ++s) {
      const int t = j + FIT_G * s;
      fWx[s] = -1.0f; fWy[s] = -1.0f; fw[s] = 0.0f;
      fx[s] = fy[s] = fz[s] = ftx[s] = fty[s] = 0.0f;
      if (t < m) {
        const int g = t0 + (int)sidx[o + t];
        fx[s] = __ldg(A.x + g) - sx; fy[s] = __ldg(A.y + g) - sy; fz[s] = __ldg(A.z + g) - zsv;
        ftx[s] = __ldg(A.tx + g); fty[s] = __ldg(A.ty + g);
        track_weight_matrix(fz[s], __ldg(A.var_x + g), __ldg(A.var_y + g), __ldg(A.var_tx + g),
                            __ldg(A.var_ty + g), fWx[s], fWy[s]);
      }
    }
    bool run = vact && !big;
    bool sing = false;
    int niter = 0;
    Sums L;                                                // sums of the last iteration done
    sums_zero(L);
    for (int it = 1; it <= P.max_iter; ++it) {
      Sums S;
      sums_zero(S);
      if (run) {
#pragma unroll
        for (int s = 0; s < FIT_KF; ++s)
          fw[s] = track_accum(fx[s], fy[s], fz[s], ftx[s], fty[s], fWx[s], fWy[s], ax, ay, az, P, S);
      }
      sums_reduce<FIT_G>(S);
      if (run) {
        float dx, dy, dzs, dchi2;
        if (!newton_step(S, dx, dy, dzs, dchi2)) {
          sing = true; run = false;
        } else {
          ax += dx; ay += dy; az += dzs;
          L = S; niter = it;
          if (fabsf(dchi2) < P.conv_dchi2 && fabsf(dzs) < P.conv_dz) run = false;
        }
      }
      if (!__any_sync(FULL, run)) break;
    }
    if (vact && !big) {
      if (sing) {
        status |= PV_EVT_SINGULAR_FIT;
        if (j == 0) reinterpret_cast<int*>(V)[11 * MAXV + v] = -1;
      } else {
        if (j == 0) {
          float C[6];
          covariance(L, C);
          V[0 * MAXV + v] = sx + ax; V[1 * MAXV + v] = sy + ay; V[2 * MAXV + v] = zsv + az;
#pragma unroll
          for (int c = 0; c < 6; ++c) V[(3 + c) * MAXV + v] = C[c];
          V[9 * MAXV + v] = L.chi2;
          reinterpret_cast<int*>(V)[10 * MAXV + v] = (int)L.nact;
          reinterpret_cast<int*>(V)[11 * MAXV + v] = niter;
        }
#pragma unroll
        for (int s = 0; s < FIT_KF; ++s) {
          const int t = j + FIT_G * s;
          if (t < m) A.trk_weight[t0 + (int)sidx[o + t]] = fw[s];
        }
      }
    }
  }
  // Slow path: vertices with more tracks than the register-resident path holds; the whole warp strides
  // over the track list and re-reads the tracks (L2-resident) every iteration.
  for (int v = 0; v < ns; ++v) {
    const int m = cnt[v];
    if (m <= FIT_G * FIT_KF) continue;
    const int o = off[v];
    const float zsv = zs[v];
    const float sx = __fmaf_rn(P.beam_tx, zsv, P.beam_x), sy = __fmaf_rn(P.beam_ty, zsv, P.beam_y);
    float ax = 0.0f, ay = 0.0f, az = 0.0f;                 // local frame, as in the fast path
    float px = ax, py = ay, pz = az;                       // vertex position the last weights were taken at
    bool sing = false;
    int niter = 0;
    Sums L;
    sums_zero(L);
    for (int it = 1; it <= P.max_iter; ++it) {
      Sums S;
      sums_zero(S);
      for (int t = lane; t < m; t += 32) {
        const int g = t0 + (int)sidx[o + t];
        const float zl = __ldg(A.z + g) - zsv;
        float Wx, Wy;
        track_weight_matrix(zl, __ldg(A.var_x + g), __ldg(A.var_y + g), __ldg(A.var_tx + g), __ldg(A.var_ty + g), Wx, Wy);
        track_accum(__ldg(A.x + g) - sx, __ldg(A.y + g) - sy, zl, __ldg(A.tx + g), __ldg(A.ty + g), Wx, Wy, ax, ay, az, P, S);
      }
      sums_reduce<32>(S);
      float dx, dy, dzs, dchi2;
      if (!newton_step(S, dx, dy, dzs, dchi2)) { sing = true; break; }
      px = ax; py = ay; pz = az;
      ax += dx; ay += dy; az += dzs;
      L = S; niter = it;
      if (fabsf(dchi2) < P.conv_dchi2 && fabsf(dzs) < P.conv_dz) break;
    }
    if (sing) {
      status |= PV_EVT_SINGULAR_FIT;
      if (lane == 0) reinterpret_cast<int*>(V)[11 * MAXV + v] = -1;
    } else {
      if (lane == 0) {
        float C[6];
        covariance(L, C);
        V[0 * MAXV + v] = sx + ax; V[1 * MAXV + v] = sy + ay; V[2 * MAXV + v] = zsv + az;
        for (int c = 0; c < 6; ++c) V[(3 + c) * MAXV + v] = C[c];
        V[9 * MAXV + v] = L.chi2;
        reinterpret_cast<int*>(V)[10 * MAXV + v] = (int)L.nact;
        reinterpret_cast<int*>(V)[11 * MAXV + v] = niter;
      }
      for (int t = lane; t < m; t += 32) {                 // weights of the last iteration, recomputed
        const int g = t0 + (int)sidx[o + t];
        const float zl = __ldg(A.z + g) - zsv;
        float Wx, Wy;
        track_weight_matrix(zl, __ldg(A.var_x + g), __ldg(A.var_y + g), __ldg(A.var_tx + g), __ldg(A.var_ty + g), Wx, Wy);
        Sums dummy;
        sums_zero(dummy);
        A.trk_weight[g] = track_accum(__ldg(A.x + g) - sx, __ldg(A.y + g) - sy, zl, __ldg(A.tx + g), __ldg(A.ty + g),
                                      Wx, Wy, px, py, pz, P, dummy);
      }
    }
  }
  status = __reduce_or_sync(FULL, status);
  __syncwarp();

  // ================= a6: cleanup (Table 2) =====================================================
  const int* Vi = reinterpret_cast<const int*>(V);
  unsigned alive = 0;                                      // bit k: seed k still a vertex candidate
  {
    const bool ok = lane < ns && Vi[11 * MAXV + lane] >= 0;
    alive = __ballot_sync(FULL, ok);
  }
  unsigned merged = 0;
  {
    // duplicate removal: greedy sweep in z order; duplicate iff dz^2 / (Czz_v + Czz_s) < merge_ratio; the one
    // "with fewer associated tracks" is rejected, ties keep the lower z (R-9).  Every lane runs the same
    // short serial loop on broadcast shared-memory reads.
    int s = -1;
    for (int v = 0; v < ns; ++v) {
      if (!((alive >> v) & 1u)) continue;
      if (s < 0) { s = v; continue; }
      const float dzv = V[2 * MAXV + v] - V[2 * MAXV + s];
      const float ratio = dzv * dzv / (V[8 * MAXV + v] + V[8 * MAXV + s]);
      if (ratio < P.merge_ratio) {
        if (Vi[10 * MAXV + v] > Vi[10 * MAXV + s]) { merged |= 1u << s; s = v; }
        else merged |= 1u << v;
      } else {
        s = v;
      }
    }
  }
  int fate = -9;
  bool keep = false;
  if (lane < ns) {
    if (!((alive >> lane) & 1u)) fate = -1;
    else if ((merged >> lane) & 1u) fate = -2;
    else {
      const float vx = V[0 * MAXV + lane], vy = V[1 * MAXV + lane], vz = V[2 * MAXV + lane];
      const int region = vz < P.z_split ? 1 : 0;
      if (Vi[10 * MAXV + lane] < P.min_tracks_pv[region]) fate = -3;        // Table 2 "Min. tracks in the PV"
      else {
        keep = true;
        if (region == 0) {
          const float dx = vx - fmaf(P.beam_tx, vz, P.beam_x), dy = vy - fmaf(P.beam_ty, vz, P.beam_y);
          if (fmaf(dx, dx, dy * dy) > P.max_beam_dist2) { keep = false; fate = -4; }
        }
      }
    }
  }
  const unsigned kept = __ballot_sync(FULL, keep);
  const int myidx = __popc(kept & lanemask_lt());
  if (keep) {
    fate = myidx;
    const size_t o = ev + myidx;
#pragma unroll
    for (int c = 0; c < 3; ++c) A.vtx_pos[o * 3 + c] = V[c * MAXV + lane];
#pragma unroll
    for (int c = 0; c < 6; ++c) A.vtx_cov[o * 6 + c] = V[(3 + c) * MAXV + lane];
    A.vtx_chi2[o] = V[9 * MAXV + lane];
    A.vtx_ntracks[o] = Vi[10 * MAXV + lane];
    A.vtx_niter[o] = Vi[11 * MAXV + lane];
  }
  if (lane == 0) {
    A.n_vtx[e] = __popc(kept);
    A.event_status[e] = status;
  }
  if (DBG && lane < ns) {
    const size_t o = ev + lane;
    const bool fitted = (alive >> lane) & 1u;
    if (A.dbg.seed_niter) A.dbg.seed_niter[o] = Vi[11 * MAXV + lane];
    if (A.dbg.seed_fate) A.dbg.seed_fate[o] = fate;
    if (fitted) {
      if (A.dbg.seed_pos) for (int c = 0; c < 3; ++c) A.dbg.seed_pos[o * 3 + c] = V[c * MAXV + lane];
      if (A.dbg.seed_cov) for (int c = 0; c < 6; ++c) A.dbg.seed_cov[o * 6 + c] = V[(3 + c) * MAXV + lane];
      if (A.dbg.seed_chi2) A.dbg.seed_chi2[o] = V[9 * MAXV + lane];
      if (A.dbg.seed_ntrk) A.dbg.seed_ntrk[o] = Vi[10 * MAXV + lane];
    }
  }
  // final per-track outputs; tracks of rejected vertices are released (R-9)
  for (int i = lane; i < n; i += 32) {
    const int s = A.trk_vertex[t0 + i];
    int vtx = -1;
    if (s >= 0 && ((kept >> s) & 1u)) vtx = __popc(kept & ((1u << s) - 1u));
    A.trk_vertex[t0 + i] = vtx;
    if (vtx < 0) A.trk_weight[t0 + i] = 0.0f;
  }
  __syncwarp();
  // re-zero region 0 for the next event
  {
    int4* Z = reinterpret_cast<int4*>(wsm);
    const int nq = P.region0_words >> 2;
    for (int i = lane; i < nq; i += 32) Z[i] = make_int4(0, 0, 0, 0);
  }
  __syncwarp();
}

template <bool DBG>
__global__ void __launch_bounds__(512, 1) pv_find_kernel(const __grid_constant__ KParams P,
                                                         const __grid_constant__ KArgs A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  unsigned char* wsm = smem_raw + (size_t)warp * P.warp_smem_bytes;
  {
    int4* Z = reinterpret_cast<int4*>(wsm);
    const int nq = P.region0_words >> 2;
    for (int i = lane; i < nq; i += 32) Z[i] = make_int4(0, 0, 0, 0);
  }
  __syncwarp();
  for (;;) {
    int e = 0;
    if (lane == 0) e = (int)atomicAdd(A.counter, 1u);
    e = __shfl_sync(FULL, e, 0);
    if (e >= A.n_events) break;
    process_event<DBG>(e, P, A, wsm, lane);
  }
}

}  // namespace pvk

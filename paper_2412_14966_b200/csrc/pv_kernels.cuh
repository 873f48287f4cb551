// pv_kernels.cuh -- sm_100a kernels of the PV-finder hot path (arXiv:2412.14966, "P:Lnn" = PAPER.md line nn).
//
// Three kernels per pv_find call:
//
//   seed_kernel     a1..a4  ONE WARP per event, persistent grid, 32 warps (events in flight) per SM, no CTA barrier.
//                           Sparse int32 histograms: the words (32 bins) an event touches are taken from a pool in
//                           shared memory shared by the CTA (bitmap allocator, word map per warp).  POCA projection
//                           (fp32 contract, bit-exact with the CPU oracle), flat list of 6-bin fill units (seven
//                           independent CDF edges per lane, predicated integer adds), one lane per mapped word for the
//                           proto-cluster starts, one lane per proto-cluster for the z-ordered hysteresis sweep, seed
//                           positions, association (explicit with the removal loop, or the multi-vertex chi2 window),
//                           deterministic counting sort -> seed records and fit-ready track records in HBM.
//   fit_kernel      a5      flat over all seeds of the batch (no histogram): a warp counting-sorts a window of seed
//                           records and works through it as a queue, 2 / 4 / ... 32 lanes per seed, tracks staged by
//                           cp.async into conflict-free shared-memory columns; one tick = one Newton iteration of every
//                           seed in flight; a converged seed frees its lanes in the same tick; closed-form solve of the
//                           arrow-shaped 3x3 Hessian; Tukey (Eq. 18) or multi-vertex (Eq. 19) weights.
//   cleanup_kernel  a6      one warp per event: z-ordered duplicate sweep, cuts, compaction, final per-track
//                           vertex index and weight.
//   tmpl_kernel     a2'     table of template histograms for the x86 variant of the fill, rebuilt per call.
//   scan_nvtx_kernel, pack_vertices_kernel   compact read-back of the host pipeline.
//   ip_kernel       NEXT-4  impact parameter / IP chi2 of every track w.r.t. the PVs of its event (pv_track_ip).
//
// The v1 single fused kernel (profiles/r1_v1_fused_kernel.md) was 87 KB of SASS and lost 42 % of its issue
// slots to instruction-cache misses with 14 warps per SM in different phases; each kernel here is smaller.
// Until round 2 the seed kernel gave every event a TEAM of two warps and a dense 13.6 KB histogram (14 events in
// flight per SM, a fifth of the warp time spent at team barriers): profiles/r2_kernels.md has both.
// This file shares nothing with oracle/ (the frozen CDF coefficients below are the numbers of
// DESIGN.md section 3, restated).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/pv_finder.h"

namespace pvk {

constexpr unsigned FULL = 0xffffffffu;
constexpr int MAX_TRK = PV_MAX_TRACKS_PER_EVENT;
constexpr int MAXV = PV_MAX_VTX;
#ifndef PV_MV_KEEP
#define PV_MV_KEEP 4
#endif
constexpr int MV_KEEP = PV_MV_KEEP;   // multi-vertex association: groups of 32 tracks whose candidate masks stay in registers between its two passes
static_assert(MV_KEEP >= 0 && MV_KEEP <= 4, "the association keeps four mask / denominator register pairs (hm0..3, hd0..3)");
#ifndef PV_DET_UNROLL
#define PV_DET_UNROLL 2
#endif
// unroll of the loop that reads a histogram word 16 bytes at a time (a3); measured on configs[1]: 8 (all) 0.632 ms,
// 2 0.620 ms: the kernel is short of issue slots and of instruction cache there, not of parallelism
constexpr int DET_UNROLL = PV_DET_UNROLL;
#ifndef PV_PREFETCH_TRACKS
#define PV_PREFETCH_TRACKS 128    // tracks of a warp's next event pulled into L2 while the current one is associated
#endif
#ifndef PV_BULK_PREFETCH
#define PV_BULK_PREFETCH 0        // 1: that prefetch as nine cp.async.bulk.prefetch.L2 (TMA unit) instead of 9 x 5 prefetch.global.L2
#endif                            // lines; measured on configs[1] (profiles/r3_kernels.md)
#ifndef PV_SEED_WARPS
#define PV_SEED_WARPS 32
#endif
constexpr int SEED_WARPS = PV_SEED_WARPS;      // warps per CTA of seed_kernel = events in flight per SM (one warp per event)
constexpr int CHUNK = 64;           // tracks per fill chunk
constexpr int SLOTS = CHUNK / 32;   // tracks per lane and chunk
#ifndef PV_FIT_UNROLL
#define PV_FIT_UNROLL 2
#endif
#ifndef PV_FIT_UNROLL_MV
#define PV_FIT_UNROLL_MV 4
#endif
#ifndef PV_UNIT
#define PV_UNIT 6
#endif
constexpr int UNIT = PV_UNIT;       // bins per fill unit: a lane evaluates UNIT + 1 independent CDF edges
constexpr int MAX_FILL_UNITS = 512; // units of one track's window: the unit list packs (unit << 7 | staged track) in 16 bits
static_assert(UNIT >= 1 && ((MAX_FILL_UNITS - 1) << 7 | 127) == 0xffff, "unit index: 9 bits above the 7 of the staged track");
// (validate() in pv_api.cu refuses parameters whose widest fill window exceeds MAX_FILL_UNITS * UNIT bins)
constexpr int LIST_CAP = 192;       // fill units of one round (a chunk of median tracks needs ~100)
constexpr int BINS_SM = 128;        // tracks per event whose central bin stays in shared memory (else HBM scratch)
constexpr int SEEDOF_SM = 128;      // ... whose seed index stays in shared memory between the count and the sort of a4
// unroll of the track loop of one fit iteration; with the packed loop, configs[1]: explicit 1 / 2 / 3 / 4 / 8 -> 0.345 / 0.333 /
// 0.339 / 0.338 / 0.345 ms, multi-vertex 2 / 4 -> 0.343 / 0.333 ms
constexpr int FIT_UNROLL = PV_FIT_UNROLL;
constexpr int FIT_UNROLL_MV = PV_FIT_UNROLL_MV;
#ifndef PV_FIT_KF
#define PV_FIT_KF 14
#endif
#ifndef PV_FIT_KF_MV
#define PV_FIT_KF_MV 12
#endif
// track slots per lane in shared memory: G lanes hold a seed of up to G * KF tracks.  Fewer slots send more seeds to
// the next group size but let more warps live on an SM; measured on configs[1], explicit flavour (24 B per slot and
// lane): 16 slots / 18 warps 0.366 ms, 14 / 20 0.344, 12 / 22 0.367, 10 / 26 0.429; multi-vertex (32 B): 16 / 12 0.383, 12 / 16 0.362
constexpr int FIT_KF = PV_FIT_KF;
constexpr int FIT_KF_MV = PV_FIT_KF_MV;
static_assert(FIT_KF >= 2 && FIT_KF <= 15 && FIT_KF_MV >= 2 && FIT_KF_MV <= 15,
              "the fit's sort key is phase * 16 + 16 - slots (slots <= KF), counted in 96 bins");
constexpr int FIT_WIN = 256;        // seed records of one window of the fit (its sorted order is held as 8 bytes per lane)
constexpr int FIT_BLOCK = 64;       // threads per CTA of fit_kernel (warps are autonomous; 12 KB of tracks per warp)
constexpr int FIT_MIN_BLOCKS = 10;  // CTAs per SM: 10 x (21 KB + 1 KB reserved) fill the shared memory
constexpr int FIT_MIN_BLOCKS_MV = 8;  // multi-vertex flavour: 24 KB of staged records per CTA
constexpr int MAX_WORDS = PV_MAX_BINS / 32;   // 128 histogram words of 32 bins
constexpr int PROTO_CAP = 256;      // proto-cluster starts of one sweep round (<= 16 per word)
constexpr int TMPL_J = 8;           // template fill: positions of z_poca inside its central bin
constexpr int TMPL_MAXK = 56;       // template fill: sigma classes (validate() bounds max_sigma_poca / dz)

// Shared memory of seed_kernel: [pool: 1 NULL word + n_pool words of 32 int32 bins][bitmap of the free pool words]
// [SEED_WARPS x WARP_SMEM].  Per warp, in bytes; the 1152 bytes that stage the fill (track windows and the unit list)
// are dead once the histogram is complete: the peak search and the association reuse them.
constexpr int SM_HDR_BYTES = 256;                          // unsigned bm[64]      free words of the pool, one bit each
constexpr int SM_MAP = 0;                                  // uint16 map[128]      histogram word -> pool word (0 = NULL word)
constexpr int SM_TB = SM_MAP + MAX_WORDS * 2;              // uint8 tb[128]        fill: unmapped words of the chunk's windows; peaks: list of the mapped words
constexpr int SM_MISC = SM_TB + MAX_WORDS;                 // unsigned mapped[4]   words that have a pool word (+ spare)
constexpr int SM_BINS = SM_MISC + 64;                      // int16 binsm[128]     central bins of the first 128 tracks
constexpr int SM_STAGE = SM_BINS + BINS_SM * 2;            // fill:  float zp[64], inv[64]; int lonb[64]
constexpr int SM_LIST = SM_STAGE + CHUNK * 12;             // fill:  uint16 list[192]
constexpr int SM_PROTO = SM_STAGE;                         // peaks: uint16 ps[PROTO_CAP]                 (over the stage)
constexpr int SM_CNT = SM_PROTO;                           // a4:    int cnt[32] tracks per seed          (over ps)
constexpr int SM_CUR = SM_CNT + 128;                       // a4:    int cur[32] running record position  (over ps)
constexpr int SM_SEEDOF = SM_CUR + 128;                    // a4:    int8 seedsm[128] seed of the first 128 tracks (over ps)
constexpr int SM_SEED = SM_PROTO + PROTO_CAP * 2;          // peaks..a4: int sb[32], se[32], sp[32]; float zs[32]; int part[32]
constexpr int WARP_SMEM = SM_LIST + LIST_CAP * 2;
static_assert(SM_SEED + 5 * MAXV * 4 <= WARP_SMEM, "the overlays fit the fill stage and unit list");
static_assert(SM_SEEDOF + SEEDOF_SM <= SM_SEED, "cnt, cur and seedsm fit over the proto-cluster list");
static_assert(SM_STAGE % 16 == 0 && SM_SEED % 16 == 0 && WARP_SMEM % 16 == 0, "alignment of the vector accesses");
static_assert(MAX_WORDS <= 128, "mapped[] holds four masks of 32 words");

struct KParams {
  float z_min, dz, inv_dz, z_split;
  float beam_x, beam_y, beam_tx, beam_ty;
  float max_sigma[2];
  float win_eps;                 // safety margin of the fill window, in bins
  int nbins, nwords;             // nwords = ceil(nbins / 32)
  int T_bin, D;                  // thresholds in fixed point, clamped to int32
  int I_min[2];                  // min cluster integral, fixed point clamped to int32 (an event holds < 2^31)
  int min_tracks_seed[2], min_tracks_pv[2];
  float chi2_max, inv_chi2_max;
  int unit_weights;              // chi2_max == inf
  int max_iter;
  float conv_dchi2, conv_dz, merge_ratio, max_beam_dist2;
  int max_vtx;
  int flavour;                   // PV_FLAVOUR_*
  int split_mode;                // PV_SPLIT_*
  float chi2_window;             // multi-vertex flavour: list a track for a seed iff chi2 at the seed position < this
  float mv_e0;                   // exp(-chi2_max / 2), the constant of the denominator of Eq. 19
  int n_pool;                    // words (of 32 bins) in the histogram pool of a CTA of seed_kernel, without the NULL word
  int tmpl_kmax;                 // template fill (R-17): class of the largest sigma cut = last class
  int tmpl_off[TMPL_MAXK];       // first table entry of class k; its TMPL_J templates of 2 W_k + 1 bins follow each other
  short tmpl_w[TMPL_MAXK];       // W_k = ceil(3 sigma_k / dz)
};

// One vertex seed handed from seed_kernel to fit_kernel (16 bytes, read as one int4).
struct SeedRec {
  int e;                         // event
  int k_cnt;                     // seed index within the event | track count << 5
  int begin;                     // first record of the seed's tracks in ftrk[] (absolute)
  float z;                       // z_seed (Eq. 4)
};

struct KArgs {
  const float *x, *y, *z, *tx, *ty, *var_x, *var_y, *var_tx, *var_ty;
  const float *cov_xtx, *cov_yty;  // optional x-tx / y-ty covariance elements (Eq. 2), nullptr = diagonal covariance
  const int32_t* offsets;
  int n_events;
  float *vtx_pos, *vtx_cov, *vtx_chi2;
  int32_t *vtx_ntracks, *vtx_niter, *n_vtx;
  float* trk_weight;
  int32_t* trk_vertex;
  uint32_t* event_status;
  int8_t* trk_vertex8;           // optional (host pipeline): trk_vertex as int8 (an event holds <= 32 PVs), nullptr = not written
  unsigned int* evt_counter;     // workspace: next event of the persistent seed kernel
  unsigned int* seed_counter;    // workspace: seed records written so far
  unsigned int* fit_counter;     // workspace: next window of seed records of the fit kernel
  SeedRec* rec;                  // workspace: [n_events * max_vtx]
  float4* ftrk;                  // workspace: [T or 2 T][2] fit-ready track records sorted by seed
  int32_t* tmpl;                 // workspace, template fill: the table of template histograms (tmpl_kernel)
  float* wrec;                   // workspace, explicit flavour: [T] Tukey weight of every track record (record order)
  unsigned long long* best;      // workspace, multi-vertex flavour: [T] largest weight of the track << 32 | 31 - seed
  unsigned int* trk_counter;     // workspace, multi-vertex flavour: track records allocated so far
  unsigned int* ill_counter;     // workspace: ill-conditioned seeds handed from fit_kernel to ill_kernel (list at the end of rec[])
  unsigned int trk_cap;          // capacity of ftrk in records
  unsigned int n_trk;            // the n_tracks given to pv_find: the per-track parts of the workspace hold this many
  pv_debug dbg;
};

__device__ __forceinline__ unsigned lanemask_lt() {
  unsigned m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

// Fixed-point CDF at the bin edge with float index kf (contract of DESIGN.md section 3: every op rounded
// once).  Returns the BITS of c + 8.0f: in [8, 9] one ulp is 2^-20, so the round-to-nearest-even addition is
// rint(c * 2^20) and the difference of two results is the difference of the two fixed-point values Q.
// The contract's forced Q = 0 for s <= -1 and Q = 2^20 for s >= 1 are reproduced by clamping s to [-1, 1]: the
// frozen polynomial gives G(1) = 0x1.000098p-1 > 1/2 in this Horner order, so fma(+-1, G(1), 0.5) saturates to
// exactly 1 / 0.
__device__ __forceinline__ int cdf_bits(float s);
__device__ __forceinline__ int edge_r(float kf, float zp, float inv, const KParams& P) {
  const float e = __fmaf_rn(kf, P.dz, P.z_min);
  return cdf_bits(__fmul_rn(__fsub_rn(e, zp), inv));
}
// the CDF of the contract at s = (edge - z_poca) / (3 sigma_poca), as the bits of c + 8
__device__ __forceinline__ int cdf_bits(float s) {
  s = fminf(fmaxf(s, -1.0f), 1.0f);
  const float t = __fmul_rn(s, s);
  float g = 0x1.3e0392p-3f;
  g = __fmaf_rn(g, t, -0x1.862240p-1f);
  g = __fmaf_rn(g, t, 0x1.b67296p+0f);
  g = __fmaf_rn(g, t, -0x1.3336f8p+1f);
  g = __fmaf_rn(g, t, 0x1.32067cp+1f);
  g = __fmaf_rn(g, t, -0x1.cbf272p+0f);
  g = __fmaf_rn(g, t, 0x1.3331cep+0f);
  const float c = __saturatef(__fmaf_rn(s, g, 0.5f));
  return __float_as_int(__fadd_rn(c, 8.0f));
}

// Two edges at once with the packed fp32 instructions of sm_100 (FFMA2 / FADD2 / FMUL2: two IEEE fp32 operations, each
// rounded once, in one issue slot): bit for bit the results of edge_r, for half the instructions of the Horner chains.
__device__ __forceinline__ void edge_r2(float kf0, float kf1, float zp, float inv, const KParams& P, int& r0, int& r1) {
  const float2 e = __ffma2_rn(make_float2(kf0, kf1), make_float2(P.dz, P.dz), make_float2(P.z_min, P.z_min));
  float2 s = __fmul2_rn(__fadd2_rn(e, make_float2(-zp, -zp)), make_float2(inv, inv));
  s.x = fminf(fmaxf(s.x, -1.0f), 1.0f);
  s.y = fminf(fmaxf(s.y, -1.0f), 1.0f);
  const float2 t = __fmul2_rn(s, s);
  float2 g = make_float2(0x1.3e0392p-3f, 0x1.3e0392p-3f);
  g = __ffma2_rn(g, t, make_float2(-0x1.862240p-1f, -0x1.862240p-1f));
  g = __ffma2_rn(g, t, make_float2(0x1.b67296p+0f, 0x1.b67296p+0f));
  g = __ffma2_rn(g, t, make_float2(-0x1.3336f8p+1f, -0x1.3336f8p+1f));
  g = __ffma2_rn(g, t, make_float2(0x1.32067cp+1f, 0x1.32067cp+1f));
  g = __ffma2_rn(g, t, make_float2(-0x1.cbf272p+0f, -0x1.cbf272p+0f));
  g = __ffma2_rn(g, t, make_float2(0x1.3331cep+0f, 0x1.3331cep+0f));
  float2 c = __ffma2_rn(s, g, make_float2(0.5f, 0.5f));
  c.x = __saturatef(c.x);
  c.y = __saturatef(c.y);
  const float2 q = __fadd2_rn(c, make_float2(8.0f, 8.0f));
  r0 = __float_as_int(q.x);
  r1 = __float_as_int(q.y);
}

// integer add to a shared-memory bin (byte address in the shared window) unless the addend is zero (ptxas turns the
// predicate into a branch; adding the zeros as well, without any test, was measured slower: 0.630 against 0.620 ms)
__device__ __forceinline__ void red_add_nz(unsigned saddr, int d) {
  asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.s32 q, %1, 0;\n\t@q red.shared.add.s32 [%0], %1;\n\t}" ::"r"(saddr), "r"(d) : "memory");
}

__device__ __forceinline__ int bin_region(int b, const KParams& P) {
  const float centre = __fmaf_rn(__fadd_rn((float)b, 0.5f), P.dz, P.z_min);
  return centre < P.z_split ? 1 : 0;
}

// ---- template fill ("a finite set of template histograms, selected based on the value of sigma_poca"; R-17) ----
// Class k has its centre at sigma_k = 0.08 dz 2^(k/4); a track takes the class nearest in log sigma: with
// v = sigma / (0.08 dz) = m 2^E, m in [1, 2), that is 4 E + the number of class edges 2^((2 q + 1) / 8) m has reached.
__device__ __forceinline__ int tmpl_class_raw(float sigma, float inv_dz) {
  const float v = __fmul_rn(__fmul_rn(sigma, inv_dz), 12.5f);
  if (!(v >= 1.0f)) return 0;
  if (!(v < 0x1p+20f)) return 80;
  const unsigned b = __float_as_uint(v);
  const int E = (int)(b >> 23) - 127;
  const float m = __uint_as_float((b & 0x007fffffu) | 0x3f800000u);
  return 4 * E + (m >= 0x1.172b84p+0f ? 1 : 0) + (m >= 0x1.4bfdaep+0f ? 1 : 0) + (m >= 0x1.8ace54p+0f ? 1 : 0) +
         (m >= 0x1.d5818ep+0f ? 1 : 0);
}
__device__ __forceinline__ float tmpl_centre(int k) {          // sigma_k in bins
  const float c = (k & 3) == 0 ? 1.0f : (k & 3) == 1 ? 0x1.306fe0p+0f : (k & 3) == 2 ? 0x1.6a09e6p+0f : 0x1.ae89fap+0f;
  return __fmul_rn(ldexpf(c, k >> 2), 0.08f);
}

// tmpl_kernel: the table of template histograms, one block per sigma class.  Template (k, j) holds, for the relative
// bins i = -W_k .. W_k, the contract's fixed-point CDF difference Q(i + 1) - Q(i) of a track of width sigma_k whose
// z_poca is the centre of the j-th eighth of the central bin; it sums to exactly 2^20.
__global__ void __launch_bounds__(256) tmpl_kernel(const __grid_constant__ KParams P, int32_t* __restrict__ tab) {
  const int k = blockIdx.x;
  const int W = P.tmpl_w[k], nb = 2 * W + 1;
  const float inv = __fdiv_rn(1.0f, __fmul_rn(3.0f, tmpl_centre(k)));
  for (int idx = threadIdx.x; idx < TMPL_J * nb; idx += blockDim.x) {
    const int j = idx / nb, i = idx - j * nb - W;
    const float zrel = __fmul_rn(__fadd_rn((float)j, 0.5f), 1.0f / (float)TMPL_J);
    const int q0 = cdf_bits(__fmul_rn(__fsub_rn((float)i, zrel), inv));
    const int q1 = cdf_bits(__fmul_rn(__fsub_rn((float)(i + 1), zrel), inv));
    tab[P.tmpl_off[k] + idx] = q1 - q0;
  }
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
// Returns the number of seed clusters the proto-cluster yields.  Clusters 0 and 1 are returned in c0 / c1;
// cluster j is also stored at index wbase + j of (sb, se, sp) when wbase >= 0 and that index is < max_vtx.
// (Single call site, inside a loop, so that the code exists once.)
struct Cl { int b, e, p; };

template <class HT>
__device__ __forceinline__ int sweep(const HT& H, int b0, const KParams& P, int wbase,
                                     int* sb, int* se, int* sp, Cl& c0, Cl& c1) {
  int start = b0;
  int h = H[b0];
  bool look_max = true;
  int mx = h, mn = 0, mnp = b0;
  int sum = h;                               // integral of [start, k]
  int amax = h, amaxp = b0;                  // argmax of [start, k], ties -> lowest bin
  int snap_sum = 0;                          // the same over [start, mnp)
  int snap_amax = 0, snap_amaxp = b0;
  int smax = h, smaxp = b0;                  // argmax of [mnp, k]
  int count = 0;
  bool have = false;                         // last emitted cluster, held back because the tail may join it
  int lb = 0, le = 0, lp = 0, lpv = 0, lj = 0;
  auto flush = [&]() {
    if (lj == 0) { c0.b = lb; c0.e = le; c0.p = lp; }
    if (lj == 1) { c1.b = lb; c1.e = le; c1.p = lp; }
    if (wbase >= 0 && wbase + lj < P.max_vtx) { sb[wbase + lj] = lb; se[wbase + lj] = le; sp[wbase + lj] = lp; }
  };
  int k = b0 + 1;
  // The state machine is written with selects: one step is ~30 straight-line instructions (the branchy form
  // cost ~45 with the register moves at its merge points); only the rare split is a branch.  The next bin is loaded
  // one step ahead: the sweep is a serial chain, and the shared-memory latency would sit on it at every step.
  int hn = H[min(k, P.nbins - 1)];
#pragma unroll 1
  for (; k < P.nbins; ++k) {
    h = hn;
    if (!(h > P.T_bin)) break;
    hn = H[min(k + 1, P.nbins - 1)];
    const bool c_up = h > mx, c_dn = mx - h > P.D, c_lt = h < mn, c_rise = h - mn > P.D;
    const bool to_min = look_max && !c_up && c_dn;          // a significant maximum lies behind: look for the minimum
    const bool new_min = to_min || (!look_max && c_lt);     // this bin is the running minimum
    const bool to_max = !look_max && !c_lt && c_rise;       // significant minimum at mnp, with a maximum on either side
    snap_sum = new_min ? sum : snap_sum;                    // integral and argmax of [start, k): before this bin
    snap_amax = new_min ? amax : snap_amax;
    snap_amaxp = new_min ? amaxp : snap_amaxp;
    sum += h;
    const bool g1 = h > amax;
    amax = g1 ? h : amax; amaxp = g1 ? k : amaxp;
    const bool g2 = new_min || h > smax;
    smax = g2 ? h : smax; smaxp = g2 ? k : smaxp;
    mn = new_min ? h : mn; mnp = new_min ? k : mnp;
    mx = ((look_max && c_up) || to_max) ? h : mx;
    look_max = (look_max && !to_min) || to_max;
    if (to_max && snap_sum >= P.I_min[bin_region(snap_amaxp, P)]) {
      if (have) flush();
      lb = start; le = mnp; lp = snap_amaxp; lpv = snap_amax; lj = count; have = true;
      ++count;
      start = mnp;                                         // the minimum bin opens the right-hand cluster
      sum -= snap_sum; amax = smax; amaxp = smaxp;
    }
  }
  // tail [start, k)
  if (sum >= P.I_min[bin_region(amaxp, P)]) {
    if (have) flush();
    lb = start; le = k; lp = amaxp; lj = count; have = true;
    ++count;
  } else if (have) {                         // remainder joins the last cluster of this proto-cluster
    le = k;
    if (amax > lpv) { lp = amaxp; lpv = amax; }
  }
  if (have) flush();
  return count;
}

// ---- a3, x86 variant of the splitting (reading R-16): "the smallest minimum between the two largest maxima,
// recursively".  Same interface as sweep().  An explicit stack of bin ranges replaces the recursion (left part first,
// so the leaves come out in z order); every range is analysed with the hysteresis sweep of R-4.2: pass 1 finds the
// two highest significant maxima, pass 2 the lowest significant minimum between them, pass 3 the integrals and
// peak bins of the two parts.
struct Part { int sum, amax, amaxp; };

template <class HT>
__device__ __forceinline__ Part part_of(const HT& H, int s, int e) {
  Part r = {0, -1, s};
#pragma unroll 1
  for (int k = s; k < e; ++k) {
    const int h = H[k];
    r.sum += h;
    if (h > r.amax) { r.amax = h; r.amaxp = k; }
  }
  return r;
}

template <class HT>
__device__ int split_x86(const HT& H, int b0, const KParams& P, int wbase,
                         int* sb, int* se, int* sp, Cl& c0, Cl& c1) {
  int b1 = b0 + 1;
#pragma unroll 1
  while (b1 < P.nbins && H[b1] > P.T_bin) ++b1;
  int count = 0;
  {
    const Part root = part_of(H, b0, b1);
    if (root.sum < P.I_min[bin_region(root.amaxp, P)]) return 0;   // every seed passes the integral cut
  }
  constexpr int DEPTH = 32;
  unsigned stack[DEPTH];
  int top = 0;
  stack[top++] = (unsigned)b0 | ((unsigned)b1 << 16);
#pragma unroll 1
  while (top > 0) {
    const unsigned r = stack[--top];
    const int s = (int)(r & 0xffffu), e = (int)(r >> 16);
    // pass 1: significant maxima of [s, e); the highest (ties: lower bin) and the second highest
    int h1 = -1, j1 = -1, h2 = -1, j2 = -1, n_max = 0;
    auto new_max = [&](int h) {
      if (h > h1) { h2 = h1; j2 = j1; h1 = h; j1 = n_max; }
      else if (h > h2) { h2 = h; j2 = n_max; }
      ++n_max;
    };
    {
      bool look_max = true;
      int mx = H[s], mn = 0;
#pragma unroll 1
      for (int k = s + 1; k < e; ++k) {
        const int h = H[k];
        if (look_max) {
          if (h > mx) mx = h;
          else if (mx - h > P.D) { new_max(mx); mn = h; look_max = false; }
        } else {
          if (h < mn) mn = h;
          else if (h - mn > P.D) { mx = h; look_max = true; }
        }
      }
      if (look_max) new_max(mx);
    }
    int c = -1;
    if (n_max >= 2 && top + 2 <= DEPTH) {
      // pass 2: the lowest significant minimum between them (MIN j lies between MAX j-1 and MAX j)
      const int lo = min(j1, j2), hi = max(j1, j2);
      bool look_max = true;
      int mx = H[s], mn = 0, mnp = s, seen = 0, cmin = 0x7fffffff;
#pragma unroll 1
      for (int k = s + 1; k < e; ++k) {
        const int h = H[k];
        if (look_max) {
          if (h > mx) mx = h;
          else if (mx - h > P.D) { ++seen; mn = h; mnp = k; look_max = false; }
        } else {
          if (h < mn) { mn = h; mnp = k; }
          else if (h - mn > P.D) {
            if (seen > lo && seen <= hi && mn < cmin) { cmin = mn; c = mnp; }
            mx = h; look_max = true;
          }
        }
      }
      // pass 3: split iff both parts carry the minimum cluster integral
      const Part L = part_of(H, s, c), R = part_of(H, c, e);
      if (!(L.sum >= P.I_min[bin_region(L.amaxp, P)] && R.sum >= P.I_min[bin_region(R.amaxp, P)])) c = -1;
    }
    if (c >= 0) {
      stack[top++] = (unsigned)c | ((unsigned)e << 16);     // right part, popped after the left one
      stack[top++] = (unsigned)s | ((unsigned)c << 16);
    } else {                                               // leaf: a seed cluster
      const Part leaf = part_of(H, s, e);
      if (count == 0) { c0.b = s; c0.e = e; c0.p = leaf.amaxp; }
      if (count == 1) { c1.b = s; c1.e = e; c1.p = leaf.amaxp; }
      if (wbase >= 0 && wbase + count < P.max_vtx) { sb[wbase + count] = s; se[wbase + count] = e; sp[wbase + count] = leaf.amaxp; }
      ++count;
    }
  }
  return count;
}

// ---- a1: POCA projection of one track (Eq. 1, Eq. 3; fp32 contract of DESIGN.md section 3) ---------------------
struct Proj {
  float zp, sg, inv;             // z_poca, sigma_poca, 1 / (3 sigma_poca)
  float frac;                    // position of z_poca inside its central bin, in bins
  int bin;                       // central bin, -1 = not assignable
  bool fill;                     // enters the histogram
};

__device__ __forceinline__ Proj project(float x, float y, float z, float tx, float ty, float vx, const KParams& P) {
  Proj r;
  r.zp = __int_as_float(0x7fc00000); r.sg = r.zp; r.inv = 0.0f; r.frac = 0.0f; r.bin = -1; r.fill = false;
  const float dtx = __fsub_rn(tx, P.beam_tx), dty = __fsub_rn(ty, P.beam_ty);
  const float den = __fmaf_rn(dty, dty, __fmul_rn(dtx, dtx));
  if (den >= 1e-12f) {                                    // R-3: not parallel to the beamline
    const float bx = __fmaf_rn(P.beam_tx, z, P.beam_x), by = __fmaf_rn(P.beam_ty, z, P.beam_y);
    const float num = __fmaf_rn(dty, __fsub_rn(by, y), __fmul_rn(dtx, __fsub_rn(bx, x)));
    r.zp = __fadd_rn(z, __fdiv_rn(num, den));
    r.sg = __fsqrt_rn(__fdiv_rn(vx, den));
    const float fbin = __fmul_rn(__fsub_rn(r.zp, P.z_min), P.inv_dz);
    const float fb = floorf(fbin);
    if (fb >= 0.0f && fb < (float)P.nbins) {
      r.bin = (int)fb;
      r.frac = __fsub_rn(fbin, fb);
      const int region = r.zp < P.z_split ? 1 : 0;        // R-5
      r.inv = __fdiv_rn(1.0f, __fmul_rn(3.0f, r.sg));
      r.fill = r.sg > 0.0f && r.sg <= P.max_sigma[region] && r.inv < INFINITY;
    }
  }
  return r;
}

// ---- fit-ready track record (written by seed_kernel in seed order, read by fit_kernel) -------------------
// A track in the seed's local frame (x - x_seed, y - y_seed, z - z_seed): every quantity is O(mm), so fp32
// keeps ~1e-7 mm instead of ulp(550 mm) = 6e-5 mm and the iterates follow the fp64 oracle.
// x0 = x - z tx, so the residual Eq. 9 is rx = x0 + az tx - ax.
// W = V^-1 "evaluated and inverted only once, using the vertex position of the seed", Eq. 2 diagonal.
// A slot without a usable track (none, or R-7) is DEAD: with Tukey weights it is {x0 = 1e15, Wx = 1, rest 0},
// so that chi2_i = 1e30 gives w = 0 exactly and every product stays finite and zero -- no select in the loop;
// with unit weights (chi2_max = inf) it is all zeros (W = 0) and the active-track count is taken at load time.
// 32 bytes in HBM: {x0, y0, tx, ty} {Wx, Wy, track index, oth}; oth (multi-vertex flavour only) is the part of the
// denominator of Eq. 19 that does not depend on this vertex: exp(-chi2_max / 2) + sum over the OTHER candidates k of
// exp(-chi2_ik / 2) at their seed positions.
struct Trk { float x0, y0, tx, ty, Wx, Wy, oth; };

__device__ __forceinline__ Trk dead_track(const KParams& P) {
  Trk T;
  T.x0 = P.unit_weights ? 0.0f : 1e15f;
  T.Wx = P.unit_weights ? 0.0f : 1.0f;
  T.y0 = T.tx = T.ty = T.Wy = 0.0f;
  T.oth = 1.0f;
  return T;
}
__device__ __forceinline__ bool track_is_dead(const Trk& T, const KParams& P) {
  return P.unit_weights ? !(T.Wx > 0.0f) : (T.x0 == 1e15f);
}

struct RawTrk { float x, y, z, tx, ty, vx, vy, vtx, vty; };

// Eq. 2 for one coordinate at dz = z - z_trk: V_xx + 2 dz V_xtx + dz^2 V_txtx.  With a cross term the three
// terms cancel when the state is given far from the vertex (at 150 mm they are 25 x the result), so that one expression
// is evaluated in double (once per record, not per iteration); the diagonal case has only positive terms.
// `cross` (warp-uniform: cross terms were passed to the call) keeps the double path out of the diagonal case.
__device__ __forceinline__ float var_at(float v, float vt, float c, float dz, bool cross) {
  if (cross && c != 0.0f) {
    const double d = (double)dz;
    return (float)fma(d, fma(d, (double)vt, 2.0 * (double)c), (double)v);
  }
  return fmaf(dz, dz * vt, v);
}

// cx, cy: the track's V_xtx, V_yty (0 for a diagonal covariance)
__device__ __forceinline__ Trk make_track(const KParams& P, const RawTrk& R, float cx, float cy, float sx, float sy, float zsv,
                                          bool cross) {
  Trk T;
  const float zl = R.z - zsv;
  T.tx = R.tx; T.ty = R.ty;
  if (fabsf(zl) > 4.0f) {
    // a state given far from the vertex: x - zl tx cancels (x ~ 30 mm at 150 mm and a slope of 0.2, against a result
    // of O(0.1 mm)); the fp32 rounding of the large terms (2e-6 mm) is what the Tukey weights of a non-converged fit
    // amplify, so this change of frame is done in double (once per record; never taken for states at their vertex)
    const double zld = (double)R.z - (double)zsv;
    T.x0 = (float)fma(-zld, (double)R.tx, (double)R.x - (double)sx);
    T.y0 = (float)fma(-zld, (double)R.ty, (double)R.y - (double)sy);
  } else {
    T.x0 = fmaf(-zl, R.tx, R.x - sx);
    T.y0 = fmaf(-zl, R.ty, R.y - sy);
  }
  const float Vx = var_at(R.vx, R.vtx, cx, -zl, cross);
  const float Vy = var_at(R.vy, R.vty, cy, -zl, cross);
  const bool ok = (Vx > 0.0f) && (Vy > 0.0f) && (Vx < INFINITY) && (Vy < INFINITY);   // R-7
  T.Wx = __fdividef(1.0f, Vx);
  T.Wy = __fdividef(1.0f, Vy);
  T.oth = 1.0f;
  if (!ok) T = dead_track(P);
  return T;
}

// ---- seed_kernel: a1..a4, ONE WARP per event ---------------------------------------------------------------------
// Persistent grid, one CTA of SEED_WARPS warps per SM, every warp works through whole events on its own (events are
// handed out by an atomic counter): no CTA or team barrier anywhere, __syncwarp only.
// Histograms are SPARSE: an event touches ~13 of its 107 words of 32 bins (configs[1]; ~33 at high pile-up), so a dense
// int32 histogram per event (13.6 KB) would hold the SM to 14 events in flight.  Instead the CTA owns a pool of words;
// a warp maps the histogram words its tracks touch to pool words as it meets them (map[], one uint16 per histogram
// word; pool word 0 is the NULL word, always zero, where every untouched word points) and takes them from a shared
// bitmap.  When the pool runs dry a warp that holds words gives them back and starts its event again (no
// hold-and-wait, hence no deadlock); a warp that holds none simply waits.
struct Hist {
  const int* pool;
  const uint16_t* map;
  __device__ __forceinline__ int operator[](int b) const { return pool[((int)map[b >> 5] << 5) + (b & 31)]; }
};

// k words of the pool into got[0 .. k) (warp-collective): every lane looks at its own two words of the bitmap and
// takes one free bit per round, as many lanes as words are still missing, counted from lane `rot` on (every warp and
// event starts somewhere else, so that the warps of the CTA do not all fight for the same bitmap word).  Returns
// false (nothing kept) when the pool stays dry while this warp holds words (`holding`): the caller gives everything
// back and starts its event again.  A warp that holds nothing waits.
__device__ __forceinline__ bool pool_alloc(unsigned* bm, const int nbw, const int k, const int holding, const int rot,
                                           const int lane, uint16_t* got) {
  const unsigned before = (1u << ((lane - rot) & 31)) - 1u;  // lanes counted before mine, in the rotated order
  int have = 0, spins = 0;
#pragma unroll 1
  while (have < k) {
    const unsigned m0 = reinterpret_cast<volatile unsigned*>(bm)[lane];
    const unsigned m1 = lane + 32 < nbw ? reinterpret_cast<volatile unsigned*>(bm)[lane + 32] : 0u;
    const int idx = m0 ? lane : lane + 32;
    const unsigned m = m0 ? m0 : m1;
    const unsigned cand = __ballot_sync(FULL, m != 0u);
    int mine = -1;
    if (m != 0u && __popc(__funnelshift_r(cand, cand, rot) & before) < k - have) {
      const unsigned bit = 1u << (__ffs(m) - 1);
      if (atomicAnd(&bm[idx], ~bit) & bit) mine = idx * 32 + __ffs(m) - 1;
    }
    const unsigned okm = __ballot_sync(FULL, mine >= 0);
    if (mine >= 0) got[have + __popc(okm & lanemask_lt())] = (uint16_t)(1 + mine);
    have += __popc(okm);
    if (cand == 0u) {                                        // the pool is dry (a lost race is simply tried again)
      if (holding + have > 0 && ++spins > 32) {              // give back what this call took
        __syncwarp();
#pragma unroll 1
        for (int i = lane; i < have; i += 32) { const int w = (int)got[i] - 1; atomicOr(&bm[w >> 5], 1u << (w & 31)); }
        __syncwarp();
        return false;
      }
      __nanosleep(200);
    }
  }
  __syncwarp();
  return true;
}

template <bool DBG, int FLAV, int SPLIT, int FILL>
__device__ void seed_event(const int e, const int nxt, const KParams& P, const KArgs& A, int* pool, unsigned* bm,
                           unsigned char* wsm, const int lane) {
  uint16_t* map = reinterpret_cast<uint16_t*>(wsm + SM_MAP);
  uint8_t* tb = reinterpret_cast<uint8_t*>(wsm + SM_TB);
  unsigned* mapped = reinterpret_cast<unsigned*>(wsm + SM_MISC);   // mapped[c]: words 32 c .. 32 c + 31 that have a pool word
  int16_t* binsm = reinterpret_cast<int16_t*>(wsm + SM_BINS);
  float* st_zp = reinterpret_cast<float*>(wsm + SM_STAGE);
  float* st_inv = st_zp + CHUNK;
  int* st_lonb = reinterpret_cast<int*>(st_inv + CHUNK);
  uint16_t* list = reinterpret_cast<uint16_t*>(wsm + SM_LIST);
  // overlays: stage and list are dead after the fill, the proto-cluster list after the sweeps
  uint16_t* ps = reinterpret_cast<uint16_t*>(wsm + SM_PROTO);
  int* cnt = reinterpret_cast<int*>(wsm + SM_CNT);
  int* cur = reinterpret_cast<int*>(wsm + SM_CUR);
  int8_t* seedsm = reinterpret_cast<int8_t*>(wsm + SM_SEEDOF);
  int* sb = reinterpret_cast<int*>(wsm + SM_SEED);
  int* se = sb + MAXV;
  int* sp = se + MAXV;
  float* zs = reinterpret_cast<float*>(sp + MAXV);
  int* part = reinterpret_cast<int*>(zs + MAXV);
  const Hist H{pool, map};

  const int t0 = __ldg(A.offsets + e);
  const int n = __ldg(A.offsets + e + 1) - t0;
  const size_t ev = (size_t)e * P.max_vtx;
  const bool have_cross = A.cov_xtx != nullptr || A.cov_yty != nullptr;   // Eq. 2 with its x-tx / y-ty elements
  unsigned status = 0;

  // the per-track parts of the workspace (explicit flavour: ftrk[] and wrec[], multi-vertex flavour: best[]) are
  // indexed with the event's own track range and hold the n_tracks given to pv_find: refuse an event beyond them
  const bool no_room = (unsigned)t0 + (unsigned)n > A.n_trk;
  if (n > MAX_TRK || no_room) {
#pragma unroll 1
    for (int i = lane; i < n; i += 32) {
      A.trk_vertex[t0 + i] = -1;
      if (FLAV == PV_FLAVOUR_MULTIVERTEX && !no_room) A.best[t0 + i] = 0ull;   // (cleanup skips best[] of a no_room event)
    }
    if (DBG && A.dbg.trk_seed) for (int i = lane; i < n; i += 32) A.dbg.trk_seed[t0 + i] = -1;
    if (lane == 0) {
      A.n_vtx[e] = 0;
      A.event_status[e] = n > MAX_TRK ? PV_EVT_TOO_MANY_TRACKS : PV_EVT_RECORD_OVERFLOW;
      if (DBG && A.dbg.n_seeds) A.dbg.n_seeds[e] = 0;
      if (DBG && A.dbg.n_seeds_raw) A.dbg.n_seeds_raw[e] = 0;
    }
    return;
  }

  const int nwc = (P.nwords + 31) >> 5;                    // chunks of 32 histogram words
  const int nbw = (P.n_pool + 31) >> 5;                    // words of the pool bitmap
  int nheld = 0;                                           // pool words of this event (warp-uniform)
  // zero my pool words, unmap them and give them back: leaves the warp's histogram state as it is between events.
  // Lane l takes the word 32 c + l, sixteen bytes at a time.
  auto release = [&]() {
#pragma unroll 1
    for (int c = 0; c < nwc; ++c) {
      const unsigned mc = mapped[c];
      if (mc == 0u) continue;
      const bool mine = (mc >> lane) & 1u;
      int id = 0;
      if (mine) {
        id = map[32 * c + lane];
        int4* q = reinterpret_cast<int4*>(pool + (id << 5));
#pragma unroll
        for (int j = 0; j < 8; ++j) q[j] = make_int4(0, 0, 0, 0);
        map[32 * c + lane] = 0;
      }
      __threadfence_block();                               // the zeros are in place before another warp can take the word
      __syncwarp();
      if (mine) atomicOr(&bm[(id - 1) >> 5], 1u << ((id - 1) & 31));
      if (lane == 0) mapped[c] = 0u;
    }
    nheld = 0;
    __syncwarp();
  };

  // ================= a1 + a2: projection (Eq. 1, Eq. 3) and histogram fill ===================
  // Chunks of CHUNK tracks, SLOTS per lane.  The window of a histogrammed track is cut into units of UNIT
  // bins; the units of the chunk form one flat list, and a fill pass gives every lane one unit: UNIT + 1
  // independent CDF edges (instruction-level parallelism instead of one dependent Horner chain) and UNIT
  // predicated integer adds.  The adds are integers, so the order changes nothing.
  const unsigned pool_s = (unsigned)__cvta_generic_to_shared(pool);
  int n_raw = 0;
#pragma unroll 1
  for (;;) {
    bool filled = true;
#pragma unroll 1
    for (int c0 = 0; c0 < n; c0 += CHUNK) {
      float lx[SLOTS], ly[SLOTS], lz[SLOTS], ltx[SLOTS], lty[SLOTS], lvx[SLOTS];
#pragma unroll
      for (int s = 0; s < SLOTS; ++s) {                    // all loads first
        const int t = t0 + min(c0 + s * 32 + lane, n - 1);
        lx[s] = __ldg(A.x + t); ly[s] = __ldg(A.y + t); lz[s] = __ldg(A.z + t);
        ltx[s] = __ldg(A.tx + t); lty[s] = __ldg(A.ty + t); lvx[s] = __ldg(A.var_x + t);
      }
      int nun[SLOTS];                                      // fill units of my tracks
      int myunits = 0;
      bool sawnew = false;
#pragma unroll
      for (int s = 0; s < SLOTS; ++s) {
        const int i = c0 + s * 32 + lane;
        nun[s] = 0;
        if (i < n) {
          const Proj r = project(lx[s], ly[s], lz[s], ltx[s], lty[s], lvx[s], P);
          if (i < BINS_SM) binsm[i] = (int16_t)r.bin; else A.trk_vertex[t0 + i] = r.bin;   // large events: HBM scratch, read back in a4
          if (DBG) {
            if (A.dbg.z_poca) A.dbg.z_poca[t0 + i] = r.zp;
            if (A.dbg.sigma_poca) A.dbg.sigma_poca[t0 + i] = r.sg;
            if (A.dbg.trk_bin) A.dbg.trk_bin[t0 + i] = r.bin;
          }
          int lo = 0, nb = 0;
          if (r.fill && FILL == PV_FILL_TEMPLATE) {
            // template fill (R-17): class of sigma_poca, eighth of the bin z_poca falls in; the units of the
            // window then copy table entries instead of evaluating CDF edges
            const int k = min(tmpl_class_raw(r.sg, P.inv_dz), P.tmpl_kmax);
            const int j = min((int)__fmul_rn(r.frac, (float)TMPL_J), TMPL_J - 1);
            const int W = P.tmpl_w[k];
            lo = max(r.bin - W, 0);
            nb = min(r.bin + W + 1, P.nbins) - lo;
            st_zp[s * 32 + lane] = __int_as_float(P.tmpl_off[k] + j * (2 * W + 1) + (lo - (r.bin - W)));
          } else if (r.fill) {
            // window: a superset of the +-3 sigma support; edges outside it give exactly 0 or 2^20
            const float w3 = 3.0f * r.sg;
            const float fa = floorf((r.zp - w3 - P.z_min) * P.inv_dz - P.win_eps);
            const float fb2 = floorf((r.zp + w3 - P.z_min) * P.inv_dz + P.win_eps) + 1.0f;
            lo = (int)fmaxf(fa, 0.0f);
            nb = (int)fminf(fb2, (float)P.nbins) - lo;
            st_zp[s * 32 + lane] = r.zp; st_inv[s * 32 + lane] = r.inv;
          }
          if (nb > 0) {
            nun[s] = (nb + UNIT - 1) / UNIT;
            st_lonb[s * 32 + lane] = lo | (nb << 12);
#pragma unroll 1
            for (int w = lo >> 5; w <= (lo + nb - 1) >> 5; ++w)   // histogram words of the window without a pool word
              if (map[w] == 0) { tb[w] = 1; sawnew = true; }
          }
        }
        myunits += nun[s];
      }
      __syncwarp();
      // ---- words met for the first time get a pool word (the unit list, not yet built, takes the words from the pool)
      if (__any_sync(FULL, sawnew)) {
        unsigned nm[4];
        int k = 0;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          nm[c] = __ballot_sync(FULL, c < nwc && tb[32 * c + lane] != 0);
          k += __popc(nm[c]);
        }
        if (!pool_alloc(bm, nbw, k, nheld, (e * 7 + c0) & 31, lane, list)) filled = false;   // pool dry: start again
        else {
          int base = 0;
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            if (nm[c] == 0u) continue;
            if ((nm[c] >> lane) & 1u) {
              map[32 * c + lane] = list[base + __popc(nm[c] & lanemask_lt())];
              tb[32 * c + lane] = 0;
            }
            base += __popc(nm[c]);
            if (lane == 0) mapped[c] |= nm[c];
          }
          nheld += k;
        }
        __syncwarp();
      }
      if (!filled) break;
      const int incl = warp_incl_scan(myunits, lane);
      const int total = __shfl_sync(FULL, incl, 31);
      const int first = incl - myunits;                    // list position of my first unit
#pragma unroll 1
      for (int R = 0; R < total; R += LIST_CAP) {          // one round unless the chunk holds very wide tracks
        __syncwarp();
        {
          int g = first - R;
#pragma unroll
          for (int s = 0; s < SLOTS; ++s) {
            const int tk = s * 32 + lane;
#pragma unroll 1
            for (int u = 0; u < nun[s]; ++u, ++g)
              if ((unsigned)g < (unsigned)LIST_CAP) list[g] = (uint16_t)(tk | (u << 7));
          }
        }
        __syncwarp();
        const int nl = min(total - R, LIST_CAP);
#pragma unroll 1
        for (int p0 = 0; p0 < nl; p0 += 32) {
          const int idx = p0 + lane;
          const bool act = idx < nl;
          const int ent = list[act ? idx : nl - 1];
          const int tk = ent & 127, u = ent >> 7;
          const float zp = st_zp[tk], inv = st_inv[tk];
          const int lonb = st_lonb[tk];
          const int b0 = (lonb & 0xfff) + u * UNIT;
          const int rem = act ? (lonb >> 12) - u * UNIT : 0; // bins of this unit: min(rem, UNIT)
          // the unit's bins lie in one or two histogram words: their pool addresses (shared-memory byte addresses)
          const int nfirst = 32 - (b0 & 31);                 // bins before the word boundary
          const unsigned a0 = pool_s + ((unsigned)map[b0 >> 5] << 7) + ((unsigned)(b0 & 31) << 2);
          const unsigned a1 = pool_s + ((unsigned)map[min((b0 >> 5) + 1, MAX_WORDS - 1)] << 7);
          int d[UNIT];
          if constexpr (FILL == PV_FILL_TEMPLATE) {
            const int32_t* tp = A.tmpl + __float_as_int(zp) + u * UNIT;
#pragma unroll
            for (int j = 0; j < UNIT; ++j) d[j] = j < rem ? __ldg(tp + j) : 0;
          } else {
            const float kf = (float)b0;
            int r[UNIT + 1];
#pragma unroll
            for (int j = 0; j + 1 <= UNIT; j += 2) edge_r2(kf + (float)j, kf + (float)(j + 1), zp, inv, P, r[j], r[j + 1]);
            if ((UNIT & 1) == 0) r[UNIT] = edge_r(kf + (float)UNIT, zp, inv, P);
#pragma unroll
            for (int j = 0; j < UNIT; ++j) d[j] = j < rem ? r[j + 1] - r[j] : 0;
          }
#pragma unroll
          for (int j = 0; j < UNIT; ++j) red_add_nz(j < nfirst ? a0 + 4u * j : a1 + 4u * (j - nfirst), d[j]);
        }
      }
      __syncwarp();                                        // the next chunk overwrites the stage
    }
    if (!filled) reinterpret_cast<unsigned*>(tb)[lane] = 0u;
    __syncwarp();
    if (filled) {
      if (DBG && A.dbg.hist && e < A.dbg.n_hist_events)
        for (int b = lane; b < P.nbins; b += 32) A.dbg.hist[(size_t)e * P.nbins + b] = H[b];

      // ================= a3: peak search and seed position (Eq. 4-5) ==============================
      // The mapped words, ascending, are the only ones that can hold bins above the threshold.  One LANE per mapped
      // word reads its 32 bins (sixteen bytes at a time) into a bit mask of the bins above threshold; the first bin
      // of every run (proto-cluster) follows from the mask and the top bit of the word before.  Then one lane per
      // proto-cluster runs the z-ordered hysteresis sweep (select-based state machine: the serial length is the
      // longest proto-cluster).
      {
        uint8_t* twl = tb;                                 // list of the mapped words (the fill's flags are all zero now)
        int ntw = 0;
#pragma unroll 1
        for (int c = 0; c < nwc; ++c) {
          const unsigned mc = mapped[c];
          if ((mc >> lane) & 1u) twl[ntw + __popc(mc & lanemask_lt())] = (uint8_t)(32 * c + lane);
          ntw += __popc(mc);
        }
        __syncwarp();
        int carry_w = -2;                                      // last word of the pass before and its mask
        unsigned carry_m = 0u;
#pragma unroll 1
        for (int r0 = 0; r0 < ntw;) {
          int step = min(32, ntw - r0);
          const int w = lane < step ? (int)twl[r0 + lane] : -5;
          unsigned m = 0u;
          if (lane < step) {
            const int4* q = reinterpret_cast<const int4*>(pool + ((int)map[w] << 5));   // bins beyond nbins are padding and stay 0
#pragma unroll DET_UNROLL
            for (int j = 0; j < 8; ++j) {
              const int4 v = q[j];
              const unsigned nib = (v.x > P.T_bin ? 1u : 0u) | (v.y > P.T_bin ? 2u : 0u) | (v.z > P.T_bin ? 4u : 0u) | (v.w > P.T_bin ? 8u : 0u);
              m |= nib << (4 * j);
            }
          }
          unsigned pm = __shfl_up_sync(FULL, m, 1);
          int pw = __shfl_up_sync(FULL, w, 1);
          if (lane == 0) { pm = carry_m; pw = carry_w; }
          const unsigned carry = (pw == w - 1) ? pm >> 31 : 0u;
          unsigned starts = m & ~((m << 1) | carry);           // first bin of each run of bins above threshold
          int c = __popc(starts);
          int inc = warp_incl_scan(c, lane);
          if (__shfl_sync(FULL, inc, 31) > PROTO_CAP) {        // never with physical histograms: a word starts at most 16 runs
            step = min(step, PROTO_CAP / 16);
            if (lane >= step) { c = 0; starts = 0u; }
            inc = warp_incl_scan(c, lane);
          }
          const int np = __shfl_sync(FULL, inc, 31);
          {
            int o = inc - c;
#pragma unroll 1
            while (starts) {
              ps[o++] = (uint16_t)(32 * w + __ffs(starts) - 1);
              starts &= starts - 1u;
            }
          }
          carry_w = __shfl_sync(FULL, w, step - 1);
          carry_m = __shfl_sync(FULL, m, step - 1);
          r0 += step;
          __syncwarp();
#pragma unroll 1
          for (int p0 = 0; p0 < np; p0 += 32) {                // one lane per proto-cluster
            const int p = p0 + lane;
            const bool act = p < np;
            const int b0 = act ? (int)ps[p] : 0;
            Cl c0 = {0, 0, 0}, c1 = {0, 0, 0};
            int cl = 0, base = 0;
#pragma unroll 1
            for (int rep = 0; rep < 2; ++rep) {                // rep 1 (rare): proto-clusters with three or more seeds
              const bool run = act && (rep == 0 || (cl > 2 && base + 2 < P.max_vtx));
              if (!__any_sync(FULL, run)) break;
              if (run) {
                const int cc = SPLIT ? split_x86(H, b0, P, rep ? base : -1, sb, se, sp, c0, c1)
                                     : sweep(H, b0, P, rep ? base : -1, sb, se, sp, c0, c1);
                if (rep == 0) cl = cc;
              }
              if (rep == 0) {
                const int inc2 = warp_incl_scan(cl, lane);
                base = n_raw + inc2 - cl;
                if (cl > 0 && base < P.max_vtx) { sb[base] = c0.b; se[base] = c0.e; sp[base] = c0.p; }
                if (cl > 1 && base + 1 < P.max_vtx) { sb[base + 1] = c1.b; se[base + 1] = c1.e; sp[base + 1] = c1.p; }
                n_raw += __shfl_sync(FULL, inc2, 31);
              }
            }
          }
          __syncwarp();
        }
        reinterpret_cast<unsigned*>(tb)[lane] = 0u;            // the flags of the next fill start at zero
      }
      if (lane < min(n_raw, P.max_vtx)) {                      // Eq. 4-5: neighbours are raw bins, 0 beyond the ends
        const int i = sp[lane];
        const long long Nm = i > 0 ? H[i - 1] : 0;
        const long long Np = i < P.nbins - 1 ? H[i + 1] : 0;
        const long long N0 = H[i];
        const long long num = Np - Nm, den = 2 * N0 - Np - Nm;
        const float delta = den > 0 ? __fmul_rn(0.5f, __fdiv_rn((float)num, (float)den)) : 0.0f;
        const float zi = __fmaf_rn(__fadd_rn((float)i, 0.5f), P.dz, P.z_min);
        zs[lane] = __fmaf_rn(delta, P.dz, zi);
      }
    }                                                      // if (filled)
    __syncwarp();
    release();                                             // the histogram is dead from here on
    if (filled) break;
    __nanosleep(2000);                                     // the pool ran dry: back off and start the event again
    n_raw = 0;
  }
  {
    // pull the first tracks of my NEXT event (lane 0 holds its index) into L2 while this one is associated
    const int ne = __shfl_sync(FULL, nxt, 0);
    if (ne < A.n_events) {
      const int pt0 = __ldg(A.offsets + ne);
      const int pn = min(__ldg(A.offsets + ne + 1) - pt0, PV_PREFETCH_TRACKS);
#if PV_BULK_PREFETCH
      // the TMA unit's bulk prefetch: lane q < 9 asks for the whole range of array q in one instruction (both ends
      // rounded to 16 bytes inwards / outwards within the event's own range)
      if (lane < 9 && pn > 0) {
        const float* ptr = A.x;
        ptr = lane == 1 ? A.y : ptr; ptr = lane == 2 ? A.z : ptr; ptr = lane == 3 ? A.tx : ptr; ptr = lane == 4 ? A.ty : ptr;
        ptr = lane == 5 ? A.var_x : ptr; ptr = lane == 6 ? A.var_y : ptr; ptr = lane == 7 ? A.var_tx : ptr;
        ptr = lane == 8 ? A.var_ty : ptr;
        const unsigned long long b0 = (unsigned long long)(ptr + pt0) & ~15ull;
        const unsigned long long b1 = (unsigned long long)(ptr + pt0 + pn) & ~15ull;
        if (b1 > b0) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(b0), "r"((unsigned)(b1 - b0)) : "memory");
      }
#else
      if (lane * 32 < pn + 32) {                           // one 128-byte line per lane and array
        const size_t o = (size_t)pt0 + lane * 32;
        const float* arr[9] = {A.x, A.y, A.z, A.tx, A.ty, A.var_x, A.var_y, A.var_tx, A.var_ty};
#pragma unroll
        for (int q = 0; q < 9; ++q) asm volatile("prefetch.global.L2 [%0];" ::"l"(arr[q] + o));
      }
#endif
    }
  }

  int ns = n_raw;
  if (ns > P.max_vtx) { ns = P.max_vtx; status |= PV_EVT_VTX_OVERFLOW; }   // R-8: first max_vtx in z kept
  auto load_raw = [&](const int i) {
    const int g = t0 + min(i, n - 1);
    RawTrk Q;
    Q.x = __ldg(A.x + g); Q.y = __ldg(A.y + g); Q.z = __ldg(A.z + g); Q.tx = __ldg(A.tx + g); Q.ty = __ldg(A.ty + g);
    Q.vx = __ldg(A.var_x + g); Q.vy = __ldg(A.var_y + g); Q.vtx = __ldg(A.var_tx + g); Q.vty = __ldg(A.var_ty + g);
    return Q;
  };
  auto cross_of = [&](const int i, float& cx, float& cy) {   // V_xtx, V_yty of track i (0 = diagonal covariance)
    const int g = t0 + min(i, n - 1);
    cx = A.cov_xtx ? __ldg(A.cov_xtx + g) : 0.0f;
    cy = A.cov_yty ? __ldg(A.cov_yty + g) : 0.0f;
  };
  int myc = 0, myoff = 0;                                  // lane k: records of seed k, its first record within the event
  unsigned rbeg = 0u;                                      // first record of the event in ftrk[]

  // ================= a4', multi-vertex flavour: implicit association (R-13, R-14) =========
  // Every assignable track is a candidate of every seed: E_ik = exp(-chi2_ik / 2) at the seed positions gives the
  // denominator of Eq. 19; the track is listed for (gets a fit-ready record under) every seed with chi2_ik below the
  // window.  No removal loop (that belongs to the explicit association).
  if constexpr (FLAV == PV_FLAVOUR_MULTIVERTEX) {
    auto chi2_at = [&](const RawTrk& R, const float cx, const float cy, const int k) -> float {   // Eq. 7 at seed k, W from Eq. 2; < 0 = unusable (R-7)
      const float zsv = zs[k];
      const float sx = __fmaf_rn(P.beam_tx, zsv, P.beam_x), sy = __fmaf_rn(P.beam_ty, zsv, P.beam_y);
      const float dzv = zsv - R.z;
      const float Vx = var_at(R.vx, R.vtx, cx, dzv, have_cross), Vy = var_at(R.vy, R.vty, cy, dzv, have_cross);
      const bool ok = (Vx > 0.0f) && (Vy > 0.0f) && (Vx < INFINITY) && (Vy < INFINITY);
      const float rx = fmaf(dzv, R.tx, R.x) - sx, ry = fmaf(dzv, R.ty, R.y) - sy;
      const float c = fmaf(rx * rx, __fdividef(1.0f, Vx), ry * ry * __fdividef(1.0f, Vy));
      return ok ? c : -1.0f;
    };
    auto cand = [&](const int i, const RawTrk& R, unsigned& mask, float& den) {
      mask = 0u; den = P.mv_e0;
      const int b = i >= n ? -1 : (i < BINS_SM ? (int)binsm[i] : A.trk_vertex[t0 + i]);
      float cx, cy;
      cross_of(i, cx, cy);
#pragma unroll 1
      for (int k = 0; k < ns; ++k) {
        const float c = chi2_at(R, cx, cy, k);
        if (b >= 0 && c >= 0.0f) {
          den += __expf(-0.5f * c);
          if (c < P.chi2_window) mask |= 1u << k;
        }
      }
    };
    // visits the listed (track, seed) pairs of 32 tracks in a fixed order: f(k, peers) with k = -1 for idle lanes
    auto for_bits = [&](unsigned m, auto&& f) {
#pragma unroll 1
      while (__any_sync(FULL, m != 0u)) {
        const int k = m ? __ffs(m) - 1 : -1;
        m &= m - 1u;
        f(k, __match_any_sync(FULL, k));
        __syncwarp();
      }
    };
    cnt[lane] = 0;
    __syncwarp();
    auto count = [&](int k, unsigned peers) {
      if (k >= 0 && (peers & lanemask_lt()) == 0) cnt[k] += __popc(peers);
    };
    bool ovf = false;
    auto emit = [&](const int i, const RawTrk& R, const unsigned mask, const float den) {
      if (i < n) A.best[t0 + i] = 0ull;
      float cx, cy;
      cross_of(i, cx, cy);
      for_bits(ovf ? 0u : mask, [&](int k, unsigned peers) {
        const int rank = __popc(peers & lanemask_lt());
        if (k >= 0) {
          const float zsv = zs[k];
          const float sx = __fmaf_rn(P.beam_tx, zsv, P.beam_x), sy = __fmaf_rn(P.beam_ty, zsv, P.beam_y);
          const Trk T = make_track(P, R, cx, cy, sx, sy, zsv, have_cross);
          const float oth = fmaxf(den - __expf(-0.5f * chi2_at(R, cx, cy, k)), 0.5f * P.mv_e0);
          float4* o = A.ftrk + 2 * (size_t)(cur[k] + rank);
          o[0] = make_float4(T.x0, T.y0, T.tx, T.ty);
          o[1] = make_float4(T.Wx, T.Wy, __int_as_float(t0 + i), oth);   // (streaming stores were measured: no difference)
        }
        __syncwarp();
        if (k >= 0 && rank == 0) cur[k] += __popc(peers);
      });
    };
    // Two passes over the tracks in the same order: pass 0 counts the (track, seed) pairs per seed, pass 1 writes their
    // records at the counted places.  ONE loop body serves both passes (the candidate and record code exists once: the
    // kernel stays small enough for the instruction cache); the masks and denominators of the first MV_KEEP * 32 tracks
    // are kept in registers from pass 0 to pass 1, the others are computed again.
    unsigned hm0 = 0u, hm1 = 0u, hm2 = 0u, hm3 = 0u;
    float hd0 = 0.0f, hd1 = 0.0f, hd2 = 0.0f, hd3 = 0.0f;
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {
#pragma unroll 1
      for (int it = 0, i0 = 0; i0 < n; ++it, i0 += 32) {
        const int i = i0 + lane;
        const RawTrk Q = load_raw(i);
        unsigned mk = it == 0 ? hm0 : it == 1 ? hm1 : it == 2 ? hm2 : hm3;
        float dn = it == 0 ? hd0 : it == 1 ? hd1 : it == 2 ? hd2 : hd3;
        if (pass == 0 || it >= MV_KEEP) cand(i, Q, mk, dn);
        if (pass == 0) {
          if (it == 0) { hm0 = mk; hd0 = dn; }
          else if (it == 1) { hm1 = mk; hd1 = dn; }
          else if (it == 2) { hm2 = mk; hd2 = dn; }
          else if (it == 3) { hm3 = mk; hd3 = dn; }
          for_bits(mk, count);
        } else {
          emit(i, Q, mk, dn);
        }
      }
      if (pass == 0) {
        __syncwarp();
        myc = lane < ns ? cnt[lane] : 0;
        const int inc = warp_incl_scan(myc, lane);
        const int nrec = __shfl_sync(FULL, inc, 31);         // (track, seed) records of the event
        if (lane == 0) rbeg = atomicAdd(A.trk_counter, (unsigned)nrec);
        rbeg = __shfl_sync(FULL, rbeg, 0);
        ovf = rbeg + (unsigned)nrec > A.trk_cap || rbeg + (unsigned)nrec < rbeg;
        if (ovf) { status |= PV_EVT_RECORD_OVERFLOW; ns = 0; }
        myoff = inc - myc;
        cur[lane] = (int)rbeg + myoff;
        __syncwarp();
      }
    }
  } else {
    // ================= a4: association (R-11) ====================================================
    // Central bins: the first BINS_SM tracks keep them in shared memory, the rest read them back from the
    // trk_vertex scratch.  part[] is padded with INT_MAX to whole groups of four.
    auto seed_of = [&](int i) -> int {                     // seed index of track i, -1 = none
      if (i >= n || ns == 0) return -1;
      const int b = i < BINS_SM ? (int)binsm[i] : A.trk_vertex[t0 + i];
      if (b < 0) return -1;
      int s = 0;
#pragma unroll 1
      for (int k = 0; k + 1 < ns; k += 4) {                // bins < part[k] belong to seed <= k
        const int4 pk = *reinterpret_cast<const int4*>(part + k);
        s += (b >= pk.x ? 1 : 0) + (b >= pk.y ? 1 : 0) + (b >= pk.z ? 1 : 0) + (b >= pk.w ? 1 : 0);
      }
      return s;
    };
#pragma unroll 1
    for (;;) {
      if (ns == 0) break;
      part[lane] = lane + 1 < ns ? (se[lane] + sb[lane + 1]) / 2 : 0x7fffffff;
      cnt[lane] = 0;
      __syncwarp();
#pragma unroll 1
      for (int i0 = 0; i0 < n; i0 += 32) {
        const int s = seed_of(i0 + lane);
        if (i0 + lane < SEEDOF_SM) seedsm[i0 + lane] = (int8_t)s;   // reused by the sort (the last pass of this loop is final)
        if (s >= 0) atomicAdd(&cnt[s], 1);                     // a count: the order does not matter
      }
      __syncwarp();
      // "the seed cluster is removed ... and the procedure is repeated": least populated, ties lowest z
      int key = 0x7fffffff;
      if (lane < ns) {
        const int region = zs[lane] < P.z_split ? 1 : 0;
        const int c = cnt[lane];
        if (c < P.min_tracks_seed[region]) key = (c << 6) | lane;
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
    // counting sort of the tracks by seed (a seed's records are its tracks in track order: deterministic); every
    // assigned track is written as a fit-ready record (local frame of its seed, W at the seed position) at its place
    myc = (ns > 0 && lane < ns) ? cnt[lane] : 0;
    {
      const int inc = warp_incl_scan(myc, lane);
      myoff = inc - myc;
      cur[lane] = myoff;
    }
    rbeg = (unsigned)t0;
    __syncwarp();
#pragma unroll 1
    for (int i0 = 0; i0 < n; i0 += 32) {
      const int i = i0 + lane;
      const RawTrk Q = load_raw(i);                          // issued ahead of the seed look-up
      float cx, cy;
      cross_of(i, cx, cy);
      const int s = ns == 0 ? -1 : (i < SEEDOF_SM ? (i < n ? (int)seedsm[i] : -1) : seed_of(i));
      const unsigned m = __match_any_sync(FULL, s);
      const int rank = __popc(m & lanemask_lt());
      if (i < n) {
        // scratch for cleanup_kernel: seed index | position of the track's record within the event << 5 (the fit
        // leaves the track's weight at that record position)
        A.trk_vertex[t0 + i] = s >= 0 ? (s | ((cur[s] + rank) << 5)) : -1;
        if (DBG && A.dbg.trk_seed) A.dbg.trk_seed[t0 + i] = s;
      }
      if (s >= 0) {
        const float zsv = zs[s];
        const float sx = __fmaf_rn(P.beam_tx, zsv, P.beam_x);  // "xy position ... using the known beamline"
        const float sy = __fmaf_rn(P.beam_ty, zsv, P.beam_y);
        const Trk T = make_track(P, Q, cx, cy, sx, sy, zsv, have_cross);
        float4* o = A.ftrk + 2 * (size_t)(t0 + cur[s] + rank);
        o[0] = make_float4(T.x0, T.y0, T.tx, T.ty);
        o[1] = make_float4(T.Wx, T.Wy, __int_as_float(t0 + i), 0.0f);
      }
      __syncwarp();
      if (s >= 0 && rank == 0) cur[s] += __popc(m);
      __syncwarp();
    }
  }

  // seed records for fit_kernel
  int rbase = 0;
  if (lane == 0 && ns > 0) rbase = (int)atomicAdd(A.seed_counter, (unsigned)ns);
  rbase = __shfl_sync(FULL, rbase, 0);
  if (lane < ns) {
    int4 r;
    r.x = e; r.y = lane | (myc << 5); r.z = (int)rbeg + myoff; r.w = __float_as_int(zs[lane]);
    reinterpret_cast<int4*>(A.rec)[rbase + lane] = r;
    if (myc == 0) A.vtx_niter[ev + lane] = -1;               // nothing listed (or min_tracks_seed < 1): the fit never sees this seed
  }
  if (__any_sync(FULL, lane < ns && myc == 0)) status |= PV_EVT_SINGULAR_FIT;
  if (lane == 0) {
    A.n_vtx[e] = ns;                                       // scratch: seeds of the event, replaced by cleanup_kernel
    A.event_status[e] = status;
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
  __syncwarp();                                            // the next event overwrites the seed arrays
}

template <bool DBG, int FLAV, int SPLIT, int FILL>
__global__ void __launch_bounds__(SEED_WARPS * 32, 1) seed_kernel(const __grid_constant__ KParams P,
                                                                 const __grid_constant__ KArgs A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int* pool = reinterpret_cast<int*>(smem_raw);            // [1 + n_pool] words of 32 bins; word 0 = NULL word
  const int pool_bytes = (1 + P.n_pool) * 128;
  unsigned* bm = reinterpret_cast<unsigned*>(smem_raw + pool_bytes);   // free pool words, one bit each (bit i = pool word 1 + i)
  unsigned char* wsm = smem_raw + pool_bytes + SM_HDR_BYTES + (size_t)warp * WARP_SMEM;
  {
    int4* Z = reinterpret_cast<int4*>(smem_raw);           // the pool and every warp's map / flags start at zero
    const int nq = (pool_bytes + SM_HDR_BYTES + (int)blockDim.x / 32 * WARP_SMEM) >> 4;
#pragma unroll 1
    for (int i = threadIdx.x; i < nq; i += blockDim.x) Z[i] = make_int4(0, 0, 0, 0);
  }
  __syncthreads();
  if (threadIdx.x < SM_HDR_BYTES / 4) {
    const int lo = threadIdx.x * 32;
    bm[threadIdx.x] = P.n_pool >= lo + 32 ? 0xffffffffu : P.n_pool > lo ? (1u << (P.n_pool - lo)) - 1u : 0u;
  }
  __syncthreads();
  int e = 0;
  if (lane == 0) e = (int)atomicAdd(A.evt_counter, 1u);
  e = __shfl_sync(FULL, e, 0);
#pragma unroll 1
  while (e < A.n_events) {
    int nxt = 0x7fffffff;
    if (lane == 0) nxt = (int)atomicAdd(A.evt_counter, 1u);  // issued now, consumed by the prefetch and after this event
    seed_event<DBG, FLAV, SPLIT, FILL>(e, nxt, P, A, pool, bm, wsm, lane);
    e = __shfl_sync(FULL, nxt, 0);
  }
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

// Adds the track to the sums and returns its weight at the current vertex (ax, ay, az): Tukey (Eq. 18) in the
// explicit flavour, the multi-vertex weight of Eq. 19 otherwise.
template <int FLAV>
__device__ __forceinline__ float track_accum(const Trk& T, float ax, float ay, float az, const KParams& P, Sums& S) {
  const float rx = fmaf(az, T.tx, T.x0) - ax;          // residual, Eq. 9
  const float ry = fmaf(az, T.ty, T.y0) - ay;
  const float chi = fmaf(rx * rx, T.Wx, ry * ry * T.Wy);   // Eq. 7
  float w;
  if (FLAV == PV_FLAVOUR_MULTIVERTEX) {
    // Eq. 19 with the competitors frozen at their seed positions; a dead slot has chi = 1e30: E = 0, w = 0
    const float E = __expf(-0.5f * chi);
    w = __fdividef(E, T.oth + E);
  } else {
    // Tukey bi-square, Eq. 18: (1 - chi/chi_max)^2 below chi_max, else 0; inv_chi2_max = 0 gives unit weights
    const float u = fmaxf(fmaf(chi, -P.inv_chi2_max, 1.0f), 0.0f);
    w = u * u;
  }
  const float wWx = w * T.Wx, wWy = w * T.Wy;
  const float p = wWx * T.tx, q = wWy * T.ty;
  S.a += wWx; S.b += wWy; S.c += p; S.d += q;
  S.e = fmaf(p, T.tx, fmaf(q, T.ty, S.e));
  S.gx = fmaf(wWx, rx, S.gx);
  S.gy = fmaf(wWy, ry, S.gy);
  S.gz = fmaf(p, rx, fmaf(q, ry, S.gz));
  S.chi2 = fmaf(w, chi, S.chi2);
  S.nact += __saturatef(w * 1e38f);                    // 1 for w > 0 (a positive weight is >= 3.5e-15 here), else 0
  return w;
}

// The same with the packed fp32 instructions of sm_100: x and y of a track sit side by side in its staged record
// ({x0, y0, tx, ty}, {Wx, Wy}), so residuals, weights and most sums come in pairs -- 18 instead of 27 floating-point
// instructions per track and iteration.  e and gz are kept as two partial sums (x and y part) until the loop ends.
struct Sums2 {
  float2 ab, cd, e2, g, gz2;
  float chi2, nact;
};
__device__ __forceinline__ void sums2_zero(Sums2& S) {
  S.ab = S.cd = S.e2 = S.g = S.gz2 = make_float2(0.0f, 0.0f);
  S.chi2 = S.nact = 0.0f;
}
__device__ __forceinline__ void sums2_close(const Sums2& Q, Sums& S) {
  S.a = Q.ab.x; S.b = Q.ab.y; S.c = Q.cd.x; S.d = Q.cd.y; S.e = Q.e2.x + Q.e2.y;
  S.gx = Q.g.x; S.gy = Q.g.y; S.gz = Q.gz2.x + Q.gz2.y; S.chi2 = Q.chi2; S.nact = Q.nact;
}
template <int FLAV>
__device__ __forceinline__ float track_accum2(const float2 xy0, const float2 txy, const float2 W, const float oth,
                                              const float2 naxy, const float az, const KParams& P, Sums2& S) {
  const float2 r = __fadd2_rn(__ffma2_rn(make_float2(az, az), txy, xy0), naxy);   // residual, Eq. 9 (naxy = -(ax, ay))
  const float2 m = __fmul2_rn(__fmul2_rn(r, r), W);
  const float chi = m.x + m.y;                                                    // Eq. 7
  float w;
  if (FLAV == PV_FLAVOUR_MULTIVERTEX) {
    const float E = __expf(-0.5f * chi);
    w = __fdividef(E, oth + E);
  } else {
    const float u = fmaxf(fmaf(chi, -P.inv_chi2_max, 1.0f), 0.0f);
    w = u * u;
  }
  const float2 wW = __fmul2_rn(make_float2(w, w), W);
  const float2 pq = __fmul2_rn(wW, txy);
  S.ab = __fadd2_rn(S.ab, wW);
  S.cd = __fadd2_rn(S.cd, pq);
  S.e2 = __ffma2_rn(pq, txy, S.e2);
  S.g = __ffma2_rn(wW, r, S.g);
  S.gz2 = __ffma2_rn(pq, r, S.gz2);
  S.chi2 = fmaf(w, chi, S.chi2);
  S.nact += __saturatef(w * 1e38f);
  return w;
}

// Newton-Raphson step Eq. 13 on the arrow-shaped Hessian A = [[a,0,-c],[0,b,-d],[-c,-d,e]]:
// returns false when the fit is singular (fewer than 2 active tracks or a non-positive pivot).
// C = A^-1 (Eq. 14), upper triangle xx xy xz yy yz zz.
// An ILL-CONDITIONED seed (two or three nearly parallel tracks) has e ~ c^2 / a + d^2 / b: the Schur complement and
// the numerator of the z step are then small differences of fp32 sums and lose 1 / r of their digits (r = the pivot
// relative to e; r = 7e-5 seen on configs[4]: C_zz off by 1e-3, iteration counts off).  `ill` (out, optional) reports
// r < ILL_REL (or a non-positive pivot): fit_phase then drops the seed from its queue and puts its record on a list
// that ill_kernel works through after fit_kernel, refitting each in double (fit_ill).  A few seeds in 10^5; every
// other seed keeps the arithmetic (and bits) it always had.
constexpr float ILL_REL = 1.0f / 256.0f;
__device__ __forceinline__ bool newton_step(const Sums& S, float& dx, float& dy, float& dzs, float& dchi2, float* C,
                                            bool* ill = nullptr) {
  if (S.nact < 2.0f) return false;
  if (!(S.a > 0.0f) || !(S.b > 0.0f)) return false;
  const float ia = __fdividef(1.0f, S.a), ib = __fdividef(1.0f, S.b);
  const float ca = S.c * ia, db = S.d * ib;
  const float sch = S.e - S.c * ca - S.d * db;         // Schur complement = third Cholesky pivot squared
  if (ill) *ill = !(sch >= ILL_REL * S.e);
  if (!(sch > 0.0f)) return false;
  const float is = __fdividef(1.0f, sch);
  dzs = (ca * S.gx + db * S.gy - S.gz) * is;
  dx = (S.gx + S.c * dzs) * ia;
  dy = (S.gy + S.d * dzs) * ib;
  dchi2 = dzs * S.gz - dx * S.gx - dy * S.gy;          // Eq. 17
  C[0] = fmaf(ca * ca, is, ia);
  C[1] = ca * db * is;
  C[2] = ca * is;
  C[3] = fmaf(db * db, is, ib);
  C[4] = db * is;
  C[5] = is;
  return true;
}

__device__ __forceinline__ void store_vertex(const KArgs& A, size_t o, float x, float y, float z, const float* C,
                                             float chi2, int ntrk, int niter) {
  A.vtx_pos[o * 3 + 0] = x; A.vtx_pos[o * 3 + 1] = y; A.vtx_pos[o * 3 + 2] = z;
#pragma unroll
  for (int c = 0; c < 6; ++c) A.vtx_cov[o * 6 + c] = C[c];
  A.vtx_chi2[o] = chi2; A.vtx_ntracks[o] = ntrk; A.vtx_niter[o] = niter;
}

// ---- fit_kernel: a5 (R-12) ---------------------------------------------------------------------------
// Warps are autonomous (no CTA barrier).  A warp takes a WINDOW of up to 256 seed records, counting-sorts them by
// (lanes per seed, track slots per lane) and then works through the sorted list as a queue:
//   * G = 2, 4, 8, 16 or 32 lanes per seed (seeds of up to 32, 64, ... 512 tracks), 32 / G seeds in flight; the
//     tracks of a seed sit in the shared-memory columns of its lanes, laid out [slot][lane] so that every iteration
//     reads them back conflict-free (cp.async of 16 + 8 bytes of each fit-ready record);
//   * one TICK of the warp is one Newton-Raphson iteration of every seed in flight.  A seed that has converged
//     spends one more tick writing its track weights (the same arithmetic at the position its last iteration used,
//     hence the same bits), stores its vertex, and its lanes immediately take the next record of the queue: a seed
//     costs its own iterations, not those of the slowest of its neighbours (the round-1 kernel iterated 16 seeds
//     until the last had converged: 9.3 iterations on average for a mean of 5.5);
//   * because the queue is sorted, the seeds in flight need about the same number of slots, and a lane's column
//     only ever holds live tracks below a high-water mark (dead tracks above it), so a tick has no per-slot test.
// Results go to slot (event, seed index) of the vertex arrays; cleanup_kernel compacts them in place.
// Every seed's result depends only on its own tracks and on G: bit-reproducible whatever the scheduling.
__device__ __forceinline__ Trk read_track(const KArgs& A, int rec, int& idx) {
  const float4 a = __ldg(A.ftrk + 2 * (size_t)rec), b = __ldg(A.ftrk + 2 * (size_t)rec + 1);
  Trk T;
  T.x0 = a.x; T.y0 = a.y; T.tx = a.z; T.ty = a.w; T.Wx = b.x; T.Wy = b.y; T.oth = b.w;
  idx = __float_as_int(b.z);
  return T;
}

// second half of a staged record: {Wx, Wy} in the explicit flavour, {Wx, Wy, track index, oth} in the multi-vertex one
template <int FLAV> struct FitB { using type = float2; };
template <> struct FitB<PV_FLAVOUR_MULTIVERTEX> { using type = float4; };

template <int FLAV, class B>
__device__ __forceinline__ Trk slot_track(const float4& qa, const B& qb) {
  Trk T;
  T.x0 = qa.x; T.y0 = qa.y; T.tx = qa.z; T.ty = qa.w; T.Wx = qb.x; T.Wy = qb.y;
  if constexpr (FLAV == PV_FLAVOUR_MULTIVERTEX) T.oth = qb.w; else T.oth = 1.0f;
  return T;
}

// multi-vertex flavour: a track follows the fitted seed with its largest final weight (ties: lower z)
__device__ __forceinline__ void claim_track(const KArgs& A, int idx, float w, int k) {
  atomicMax(A.best + idx, ((unsigned long long)__float_as_uint(w) << 32) | (unsigned)(31 - k));
}

__device__ __forceinline__ void sums_reduce_rt(Sums& S, const int G) {
#pragma unroll 1
  for (int o = G >> 1; o > 0; o >>= 1) {
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

template <int FLAV>
__device__ __forceinline__ void store_dead(float4 (*SA)[32], typename FitB<FLAV>::type (*SB)[32], int s, int lane, const Trk& dead) {
  SA[s][lane] = make_float4(dead.x0, dead.y0, dead.tx, dead.ty);
  if constexpr (FLAV == PV_FLAVOUR_MULTIVERTEX) SB[s][lane] = make_float4(dead.Wx, dead.Wy, 0.0f, dead.oth);
  else SB[s][lane] = make_float2(dead.Wx, dead.Wy);
}

enum { FS_EMPTY = 0, FS_LOAD = 1, FS_ITER = 2, FS_FINAL = 3, FS_DONE = 4 };
#ifndef PV_FIT_WPW
#define PV_FIT_WPW 3        // explicit flavour; measured on configs[1]: 1 -> 0.359 ms, 2 -> 0.338, 3 -> 0.336 (configs[2]: 0.393 -> 0.387)
#endif
#ifndef PV_FIT_WPW_MV
#define PV_FIT_WPW_MV 2     // multi-vertex flavour; measured on configs[1] (round 2, first half): 1 -> 0.540 ms, 2 -> 0.384, 4 -> 0.414
#endif
#ifndef PV_FIT_LOADWAIT
#define PV_FIT_LOADWAIT 0        // ticks a group sits out after starting the copy of its next seed before it waits for the data
                                 // (measured on configs[1]: 0 -> 0.387 ms, 1 -> 0.405 ms; an L2 prefetch one seed ahead did not help)
#endif

// One phase of a window: the records order[pb .. pe) of the window starting at record wb, G = 1 << lg lanes per seed.
// The fit of one ill-conditioned seed (see newton_step) by the whole warp, in double, from its records in global memory
// and from the first iteration on: Eq. 6-18 / 19 as in fit_phase, lane l takes the tracks l, l + 32, ...  Its result
// depends on the seed's own records only.
template <int FLAV>
__device__ void fit_ill(const KParams& P, const KArgs& A, const int4 r, const int lane) {
  const int be = r.x, bk = r.y & 31, bm_ = r.y >> 5, bo = r.z;
  const float bz = __int_as_float(r.w);
  const float bx = __fmaf_rn(P.beam_tx, bz, P.beam_x), by = __fmaf_rn(P.beam_ty, bz, P.beam_y);
  double qx = 0.0, qy = 0.0, qz = 0.0;                 // current position (local frame)
  double px = 0.0, py = 0.0, pz = 0.0;                 // position the last weights were taken at
  double C[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
  double bchi2 = 0.0, bnact = 0.0;
  bool bsing = false;
  int bit = 0;
  auto weight = [&](const Trk& U, const double x, const double y, const double z, double& rx, double& ry, double& chi) {
    rx = (double)U.x0 + z * (double)U.tx - x;          // residual, Eq. 9
    ry = (double)U.y0 + z * (double)U.ty - y;
    chi = rx * rx * (double)U.Wx + ry * ry * (double)U.Wy;   // Eq. 7
    if (FLAV == PV_FLAVOUR_MULTIVERTEX) {
      const double E = exp(-0.5 * chi);                // Eq. 19, competitors frozen at their seed positions
      return E / ((double)U.oth + E);
    }
    if (P.unit_weights) return 1.0;
    const double u = fmax(1.0 - chi * (double)P.inv_chi2_max, 0.0);   // Eq. 18
    return u * u;
  };
#pragma unroll 1
  for (int it = 1; it <= P.max_iter; ++it) {
    double s[10] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};   // a b c d e gx gy gz chi2 nact
    for (int t = lane; t < bm_; t += 32) {
      int idx;
      const Trk U = read_track(A, bo + t, idx);
      if (track_is_dead(U, P)) continue;
      double rx, ry, chi;
      const double w = weight(U, qx, qy, qz, rx, ry, chi);
      const double wWx = w * (double)U.Wx, wWy = w * (double)U.Wy;
      const double p = wWx * (double)U.tx, q = wWy * (double)U.ty;
      s[0] += wWx; s[1] += wWy; s[2] += p; s[3] += q;
      s[4] += p * (double)U.tx + q * (double)U.ty;
      s[5] += wWx * rx; s[6] += wWy * ry; s[7] += p * rx + q * ry;
      s[8] += w * chi;
      s[9] += w > 0.0 ? 1.0 : 0.0;
    }
#pragma unroll
    for (int c = 0; c < 10; ++c)
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) s[c] += __shfl_xor_sync(FULL, s[c], o);
    if (s[9] < 2.0 || !(s[0] > 0.0) || !(s[1] > 0.0)) { bsing = true; break; }
    const double ia = 1.0 / s[0], ib = 1.0 / s[1], ca = s[2] * ia, db = s[3] * ib;
    const double sch = s[4] - s[2] * ca - s[3] * db;
    if (!(sch > 0.0)) { bsing = true; break; }
    const double is = 1.0 / sch;
    const double dzs = (ca * s[5] + db * s[6] - s[7]) * is;   // Eq. 13 on the arrow-shaped Hessian
    const double dx = (s[5] + s[2] * dzs) * ia, dy = (s[6] + s[3] * dzs) * ib;
    const double dchi2 = dzs * s[7] - dx * s[5] - dy * s[6];  // Eq. 17
    C[0] = ca * ca * is + ia; C[1] = ca * db * is; C[2] = ca * is;
    C[3] = db * db * is + ib; C[4] = db * is; C[5] = is;      // Eq. 14
    px = qx; py = qy; pz = qz;
    qx += dx; qy += dy; qz += dzs;
    bchi2 = s[8]; bnact = s[9]; bit = it;
    if (fabs(dchi2) < (double)P.conv_dchi2 && fabs(dzs) < (double)P.conv_dz) break;
  }
  const size_t o = (size_t)be * P.max_vtx + bk;
  float bass = 0.0f;
  if (!bsing) {
    for (int t = lane; t < bm_; t += 32) {             // weights of the last iteration
      int idx;
      const Trk U = read_track(A, bo + t, idx);
      const bool deadt = track_is_dead(U, P);
      double rx, ry, chi;
      const float w = deadt ? 0.0f : (float)weight(U, px, py, pz, rx, ry, chi);
      if constexpr (FLAV == PV_FLAVOUR_MULTIVERTEX) {
        if (!deadt) { claim_track(A, idx, w, bk); bass += (w >= 0.5f) ? 1.0f : 0.0f; }
      } else {
        A.wrec[bo + t] = w;
      }
    }
  }
  if constexpr (FLAV == PV_FLAVOUR_MULTIVERTEX) {
#pragma unroll
    for (int o2 = 16; o2 > 0; o2 >>= 1) bass += __shfl_xor_sync(FULL, bass, o2);
  }
  if (lane == 0) {
    if (bsing) { A.vtx_niter[o] = -1; atomicOr(A.event_status + be, (unsigned)PV_EVT_SINGULAR_FIT); }
    else {
      float Cf[6];
#pragma unroll
      for (int c = 0; c < 6; ++c) Cf[c] = (float)C[c];
      store_vertex(A, o, (float)((double)bx + qx), (float)((double)by + qy), (float)((double)bz + qz), Cf, (float)bchi2,
                   (int)(FLAV ? bass : (float)bnact), bit);
    }
  }
}

// ord0 / ord1: the sorted window (record index within the window, one byte each), 8 entries per lane.
// Explicit flavour: every iteration leaves its Tukey weights at the tracks' record positions in wrec[], so the weights
// of the last iteration are simply what is there when the seed stops (cleanup_kernel moves them to track order);
// a converged seed frees its column in the same tick.  Multi-vertex flavour: one more tick (FS_FINAL) recomputes the
// weights at the position the last iteration used and lets every track claim its best vertex.
template <int FLAV>
__device__ __forceinline__ void fit_phase(const KParams& P, const KArgs& A, float4 (*SA)[32],
                                          typename FitB<FLAV>::type (*SB)[32], const int lg, const int wb, const int pb,
                                          const int pe, const unsigned ord0, const unsigned ord1, int& filled,
                                          const int lane) {
  using BT = typename FitB<FLAV>::type;
  const int G = 1 << lg, j = lane & (G - 1);
  const unsigned below_group = (1u << (lane - j)) - 1u;        // lanes of the groups before mine
  const unsigned leaders = lg == 5 ? 1u : 0xffffffffu / ((1u << G) - 1u);   // lane 0 of every group
  const Trk dead = dead_track(P);
  int qnext = pb;                                              // next queue position to hand out (warp-uniform)
  int st = FS_DONE;                                            // every group starts by taking a record
  int loadwait = 0;
  int4 cur = make_int4(0, 0, 0, 0), nxt = make_int4(0, 0, 0, 0);
  // the record after the current one is fetched one seed ahead, so taking it never waits on memory
  auto fetch = [&](const unsigned wantm, const bool mine) {
    const int q = qnext + __popc(wantm & below_group);
    qnext += __popc(wantm);
    const int qq = min(q, 255);
    const unsigned v0 = __shfl_sync(FULL, ord0, qq >> 3), v1 = __shfl_sync(FULL, ord1, qq >> 3);
    const unsigned idx = (((qq & 4) ? v1 : v0) >> (8 * (qq & 3))) & 0xffu;
    if (mine) {
      nxt = make_int4(0, 0, 0, 0);
      if (q < pe) nxt = __ldg(reinterpret_cast<const int4*>(A.rec) + wb + idx);
    }
  };
  fetch(leaders, true);
  float ax = 0.0f, ay = 0.0f, az = 0.0f;
  float lx = 0.0f, ly = 0.0f, lz = 0.0f;                   // position the weights of the last iteration were taken at
  float C[6] = {0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f};
  float chi2 = 0.0f, nact = 0.0f, nvalid = 0.0f;
  int niter = 0, myslots = 0;
#pragma unroll 1
  for (;;) {
    // ---- groups without a seed take their prefetched record, start the copy of its tracks, prefetch another record
    const bool sw = st == FS_DONE;
    const unsigned swm = __ballot_sync(FULL, sw) & leaders;
    if (swm) {
      if (sw) cur = nxt;
      fetch(swm, sw);
      if (sw) {
        const int m = cur.y >> 5;
        st = FS_EMPTY; myslots = 0;
        if (m > 0) {
          const int mine = m > j ? (m - j + G - 1) >> lg : 0;   // my tracks: j, j + G, ... < m
          const float4* q = A.ftrk + 2 * (size_t)(cur.z + j);
          unsigned da = (unsigned)__cvta_generic_to_shared(&SA[0][lane]);
          unsigned db = (unsigned)__cvta_generic_to_shared(&SB[0][lane]);
          const char* qc = reinterpret_cast<const char*>(q);
          const unsigned qstep = 32u << lg;                    // bytes from my track to my next one
#pragma unroll 2
          for (int s = 0; s < mine; ++s) {
            asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(da), "l"(qc) : "memory");
            if constexpr (FLAV == PV_FLAVOUR_MULTIVERTEX)
              asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(db), "l"(qc + 16) : "memory");
            else
              asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(db), "l"(qc + 16) : "memory");
            qc += qstep; da += 32 * sizeof(float4); db += 32 * sizeof(BT);
          }
#pragma unroll 1
          for (int s = mine; s < filled; ++s) store_dead<FLAV>(SA, SB, s, lane, dead);   // above my tracks: dead
          filled = mine; myslots = mine;
          st = FS_LOAD; loadwait = PV_FIT_LOADWAIT;
          ax = ay = az = 0.0f; niter = 0;
        }
      }
    }
    // ---- has my copy landed?  (a group sits out PV_FIT_LOADWAIT ticks first, so the wait finds the data there)
    if (st == FS_LOAD) {
      if (loadwait > 0) --loadwait;
      else {
        asm volatile("cp.async.wait_all;" ::: "memory");
        st = FS_ITER;
        if (P.unit_weights) {                                // unit weights: the active tracks are the usable ones
          nvalid = 0.0f;
#pragma unroll 1
          for (int s = 0; s < myslots; ++s) nvalid += (SB[s][lane].x > 0.0f) ? 1.0f : 0.0f;
        }
      }
    }
    __syncwarp();
    if (!__any_sync(FULL, st != FS_EMPTY)) break;            // queue empty and nothing in flight
    const bool act = st == FS_ITER || st == FS_FINAL;
    const int nslot_w = __reduce_max_sync(FULL, act ? myslots : 0);
    if (nslot_w == 0) continue;                              // only copies in flight
    const bool fin = st == FS_FINAL;
    const float px = fin ? lx : ax, py = fin ? ly : ay, pz = fin ? lz : az;
    const int e = cur.x, k = cur.y & 31;
    Sums S;
    Sums2 Q;
    sums2_zero(Q);
    const float2 naxy = make_float2(-px, -py);
    float nass = 0.0f;                                       // multi-vertex flavour: tracks with final weight >= 1/2
    float* wp = A.wrec + cur.z + j;                          // explicit flavour: my tracks' places in wrec[]
    char* wq = reinterpret_cast<char*>(wp);                  // walked slot by slot (one pointer add instead of re-deriving
    const unsigned wstep = 4u << lg;                         // the address from the slot index: 8 -> 4 instructions per slot)
    const int wslots = st == FS_ITER ? myslots : 0;
#pragma unroll(FLAV == PV_FLAVOUR_MULTIVERTEX ? FIT_UNROLL_MV : FIT_UNROLL)
    for (int s = 0; s < nslot_w; ++s) {
      const float4 qa = SA[s][lane];
      const BT qb = SB[s][lane];
      float oth = 1.0f;
      if constexpr (FLAV == PV_FLAVOUR_MULTIVERTEX) oth = qb.w;
      const float w = track_accum2<FLAV>(make_float2(qa.x, qa.y), make_float2(qa.z, qa.w), make_float2(qb.x, qb.y), oth, naxy, pz,
                                         P, Q);
      if constexpr (FLAV == PV_FLAVOUR_MULTIVERTEX) {
        const bool deadt = P.unit_weights ? !(qb.x > 0.0f) : (qa.x == 1e15f);
        if (fin && s < myslots && !deadt) {                  // the weights of the last iteration are the outputs
          claim_track(A, __float_as_int(SB[s][lane].z), w, k);
          nass += (w >= 0.5f) ? 1.0f : 0.0f;
        }
      } else {
        if (s < wslots) *reinterpret_cast<float*>(wq) = w;   // a dead track has w = 0 (unit weights: see below)
        wq += wstep;
      }
    }
    sums2_close(Q, S);
    if (P.unit_weights) {
      S.nact = nvalid;
      if (FLAV != PV_FLAVOUR_MULTIVERTEX)                    // unit weights give a dead (R-7) track w = 1: its output is 0
        for (int s = 0; s < wslots; ++s)
          if (!(SB[s][lane].x > 0.0f)) wp[s << lg] = 0.0f;
    }
    sums_reduce_rt(S, G);
    if constexpr (FLAV == PV_FLAVOUR_MULTIVERTEX) {
#pragma unroll 1
      for (int o = G >> 1; o > 0; o >>= 1) nass += __shfl_xor_sync(FULL, nass, o);
    }
    bool store = false;
    if (st == FS_ITER) {
      float dx, dy, dzs, dchi2;
      bool ill = false;
      const bool stepped = newton_step(S, dx, dy, dzs, dchi2, C, &ill);
      if (ill) {                                               // rare: the seed goes to ill_kernel, which refits it in double
        if (j == 0) {
          const unsigned pos = atomicAdd(A.ill_counter, 1u), cap = (unsigned)A.n_events * (unsigned)P.max_vtx;
          if (*A.seed_counter + pos < cap) {                   // the list grows down from the end of rec[], behind the seeds
            reinterpret_cast<int4*>(A.rec)[cap - 1u - pos] = cur;
          } else {                                             // (every slot of the batch holds a seed: no room for a list)
            A.vtx_niter[(size_t)e * P.max_vtx + k] = -1;
            atomicOr(A.event_status + e, (unsigned)PV_EVT_SINGULAR_FIT);
          }
        }
        st = FS_DONE;
      } else if (!stepped) {                                   // singular: the vertex is dropped (R-12)
        if (j == 0) {
          A.vtx_niter[(size_t)e * P.max_vtx + k] = -1;
          atomicOr(A.event_status + e, (unsigned)PV_EVT_SINGULAR_FIT);
        }
        st = FS_DONE;
      } else {
        lx = ax; ly = ay; lz = az;
        ax += dx; ay += dy; az += dzs;
        chi2 = S.chi2; nact = S.nact; ++niter;
        if ((fabsf(dchi2) < P.conv_dchi2 && fabsf(dzs) < P.conv_dz) || niter >= P.max_iter) {
          st = FLAV == PV_FLAVOUR_MULTIVERTEX ? FS_FINAL : FS_DONE;
          store = FLAV != PV_FLAVOUR_MULTIVERTEX;
        }
      }
    } else if (fin) {
      st = FS_DONE;
      store = true;
    }
    if (store && j == 0) {
      const float zsv = __int_as_float(cur.w);
      const float sx = __fmaf_rn(P.beam_tx, zsv, P.beam_x);    // "xy position ... using the known beamline"
      const float sy = __fmaf_rn(P.beam_ty, zsv, P.beam_y);
      store_vertex(A, (size_t)e * P.max_vtx + k, sx + ax, sy + ay, zsv + az, C, chi2, (int)(FLAV ? nass : nact), niter);
    }
  }
}

// Seeds with more tracks than 32 lanes x KF slots hold (> 448 / 384; only constructed events): the whole warp strides
// over the seed's records in global memory (contiguous, L1-resident after the first iteration).
template <int FLAV>
__device__ void fit_huge(const KParams& P, const KArgs& A, const int4 r, const int lane) {
  const int be = r.x, bk = r.y & 31, bm_ = r.y >> 5, bo = r.z;
  const float bz = __int_as_float(r.w);
  const float bx = __fmaf_rn(P.beam_tx, bz, P.beam_x), by = __fmaf_rn(P.beam_ty, bz, P.beam_y);
  float qx = 0.0f, qy = 0.0f, qz = 0.0f;               // current position (local frame)
  float px = 0.0f, py = 0.0f, pz = 0.0f;               // position the last weights were taken at
  float C[6] = {0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f};
  bool bsing = false;
  int bit = 0;
  float bchi2 = 0.0f, bnact = 0.0f;
#pragma unroll 1
  for (int it = 1; it <= P.max_iter; ++it) {
    Sums S;
    sums_zero(S);
    float nv = 0.0f;
    for (int t = lane; t < bm_; t += 32) {
      int idx;
      const Trk U = read_track(A, bo + t, idx);
      nv += track_is_dead(U, P) ? 0.0f : 1.0f;
      track_accum<FLAV>(U, qx, qy, qz, P, S);
    }
    if (P.unit_weights) S.nact = nv;
    sums_reduce_rt(S, 32);
    float dx, dy, dzs, dchi2;
    if (!newton_step(S, dx, dy, dzs, dchi2, C)) { bsing = true; break; }
    px = qx; py = qy; pz = qz;
    qx += dx; qy += dy; qz += dzs;
    bchi2 = S.chi2; bnact = S.nact; bit = it;
    if (fabsf(dchi2) < P.conv_dchi2 && fabsf(dzs) < P.conv_dz) break;
  }
  const size_t o = (size_t)be * P.max_vtx + bk;
  float bass = 0.0f;
  if (!bsing) {
    for (int t = lane; t < bm_; t += 32) {             // weights of the last iteration, recomputed
      int idx;
      const Trk U = read_track(A, bo + t, idx);
      Sums dummy;
      sums_zero(dummy);
      const float w = track_accum<FLAV>(U, px, py, pz, P, dummy);
      if constexpr (FLAV == PV_FLAVOUR_MULTIVERTEX) {
        if (!track_is_dead(U, P)) { claim_track(A, idx, w, bk); bass += (w >= 0.5f) ? 1.0f : 0.0f; }
      } else {
        A.wrec[bo + t] = track_is_dead(U, P) ? 0.0f : w;
      }
    }
  }
  if constexpr (FLAV == PV_FLAVOUR_MULTIVERTEX) {
#pragma unroll
    for (int o2 = 16; o2 > 0; o2 >>= 1) bass += __shfl_xor_sync(FULL, bass, o2);
  }
  if (lane == 0) {
    if (bsing) { A.vtx_niter[o] = -1; atomicOr(A.event_status + be, (unsigned)PV_EVT_SINGULAR_FIT); }
    else store_vertex(A, o, bx + qx, by + qy, bz + qz, C, bchi2, (int)(FLAV ? bass : bnact), bit);
  }
}

template <int FLAV>
__global__ void __launch_bounds__(FIT_BLOCK, FLAV ? FIT_MIN_BLOCKS_MV : FIT_MIN_BLOCKS)
fit_kernel(const __grid_constant__ KParams P, const __grid_constant__ KArgs A) {
  using BT = typename FitB<FLAV>::type;
  constexpr int KF = FLAV == PV_FLAVOUR_MULTIVERTEX ? FIT_KF_MV : FIT_KF;
  __shared__ __align__(16) float4 s_a[FIT_BLOCK / 32][KF][32];       // {x0, y0, tx, ty}
  __shared__ __align__(16) BT s_b[FIT_BLOCK / 32][KF][32];           // {Wx, Wy} or {Wx, Wy, track index, oth}
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  float4(*SA)[32] = s_a[warp];
  BT(*SB)[32] = s_b[warp];
  const int total = (int)*A.seed_counter;
  const int nwarps = (gridDim.x * blockDim.x) >> 5;
  // window size: PV_FIT_WPW windows per warp when the batch allows, claimed one after the other (the windows of a
  // batch take different times; several per warp even that out), at most FIT_WIN records
  constexpr int WPW = FLAV == PV_FLAVOUR_MULTIVERTEX ? PV_FIT_WPW_MV : PV_FIT_WPW;
  int win = (total + WPW * nwarps - 1) / (WPW * nwarps);
  win = min(max((win + 31) & ~31, 32), FIT_WIN);
  const int nwin = (total + win - 1) / win;
  const Trk dead = dead_track(P);
  int filled = KF;                                           // slots of my column that may hold something else than a dead track
#pragma unroll 1
  for (;;) {
    int w = 0;
    if (lane == 0) w = (int)atomicAdd(A.fit_counter, 1u);
    w = __shfl_sync(FULL, w, 0);
    if (w >= nwin) break;
    const int wb = w * win, wn = min(win, total - wb);
    // ---- counting sort of the window's records by key = phase * 16 + 16 - slots per lane (scratch: rows 0, 1 of SA)
    int* hist = reinterpret_cast<int*>(&SA[0][0]);            // 96 counters, then their exclusive scan
    uint8_t* ordb = reinterpret_cast<uint8_t*>(&SA[1][0]);     // the sorted window, one byte per record
    hist[lane] = 0; hist[lane + 32] = 0; hist[lane + 64] = 0;
    __syncwarp();
    int key[FIT_WIN / 32], pos[FIT_WIN / 32];
#pragma unroll
    for (int i = 0; i < FIT_WIN / 32; ++i) {
      const int r = i * 32 + lane;
      key[i] = -1; pos[i] = 0;
      if (r < wn) {
        const int m = __ldg(&A.rec[wb + r].k_cnt) >> 5;
        if (m > 0) {
          const int ph = m <= 2 * KF ? 0 : m <= 4 * KF ? 1 : m <= 8 * KF ? 2 : m <= 16 * KF ? 3 : m <= 32 * KF ? 4 : 5;
          const int slots = ph < 5 ? (m + (2 << ph) - 1) >> (ph + 1) : 1;
          key[i] = ph * 16 + 16 - slots;                         // within a phase: most slots first, so the drain at the
                                                                   // end of the phase (idle lanes) runs on short ticks
          pos[i] = atomicAdd(&hist[key[i]], 1);
        }
      }
    }
    __syncwarp();
    int pendv;                                                // lane ph < 5: end of phase ph in the sorted window; lane 5: all
    {
      const int h0 = hist[3 * lane], h1 = hist[3 * lane + 1], h2 = hist[3 * lane + 2];
      const int tot = h0 + h1 + h2;
      const int inc = warp_incl_scan(tot, lane);
      __syncwarp();
      hist[3 * lane] = inc - tot; hist[3 * lane + 1] = inc - tot + h0; hist[3 * lane + 2] = inc - tot + h0 + h1;
      __syncwarp();
      const int nvalid_w = __shfl_sync(FULL, inc, 31);
      pendv = lane < 5 ? hist[(lane + 1) * 16] : nvalid_w;
    }
#pragma unroll
    for (int i = 0; i < FIT_WIN / 32; ++i)
      if (key[i] >= 0) ordb[hist[key[i]] + pos[i]] = (uint8_t)(i * 32 + lane);
    __syncwarp();
    const unsigned ord0 = reinterpret_cast<const unsigned*>(ordb)[2 * lane], ord1 = reinterpret_cast<const unsigned*>(ordb)[2 * lane + 1];
    __syncwarp();
#pragma unroll 1
    for (int s = 0; s < max(filled, 2); ++s) store_dead<FLAV>(SA, SB, s, lane, dead);
    filled = 0;
    __syncwarp();
    // ---- the queue, phase by phase
    int pb = 0;
#pragma unroll 1
    for (int ph = 0; ph < 5; ++ph) {
      const int pe = __shfl_sync(FULL, pendv, ph);
      if (pe > pb) fit_phase<FLAV>(P, A, SA, SB, ph + 1, wb, pb, pe, ord0, ord1, filled, lane);
      pb = pe;
    }
    const int pall = __shfl_sync(FULL, pendv, 5);
#pragma unroll 1
    for (int q = pb; q < pall; ++q) {
      const unsigned v0 = __shfl_sync(FULL, ord0, q >> 3), v1 = __shfl_sync(FULL, ord1, q >> 3);
      const unsigned idx = (((q & 4) ? v1 : v0) >> (8 * (q & 3))) & 0xffu;
      fit_huge<FLAV>(P, A, __ldg(reinterpret_cast<const int4*>(A.rec) + wb + idx), lane);
    }
  }
}

// ---- ill_kernel: the seeds fit_kernel found ill-conditioned (newton_step), one warp each, in double (fit_ill).  Runs
// between fit_kernel and cleanup_kernel; with an empty list (most small batches) it costs its launch.
template <int FLAV>
__global__ void __launch_bounds__(128) ill_kernel(const __grid_constant__ KParams P, const __grid_constant__ KArgs A) {
  const int lane = threadIdx.x & 31;
  const unsigned warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
  const unsigned cap = (unsigned)A.n_events * (unsigned)P.max_vtx, total = *A.seed_counter;
  unsigned n = *A.ill_counter;
  if (n > cap - total) n = cap - total;
  for (unsigned i = warp; i < n; i += nwarps)
    fit_ill<FLAV>(P, A, __ldg(reinterpret_cast<const int4*>(A.rec) + (cap - 1u - i)), lane);
}

// ---- cleanup_kernel: a6, one warp per event (Table 2, R-9) ------------------------------------
// Lane k holds seed k of the event (position, covariance, ... as fit_kernel left them in slot k of the vertex
// arrays), the duplicate sweep runs on shuffles, survivors are compacted in place in z order, and every
// track gets its final vertex index (weight 0 when it has none).
#ifndef PV_CLEANUP_MIN_BLOCKS
#define PV_CLEANUP_MIN_BLOCKS 8
#endif
template <bool DBG, int FLAV>
__global__ void __launch_bounds__(256, PV_CLEANUP_MIN_BLOCKS) cleanup_kernel(const __grid_constant__ KParams P,
                                                      const __grid_constant__ KArgs A) {
  const int lane = threadIdx.x & 31;
  const int e = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (e >= A.n_events) return;
  const int ns = A.n_vtx[e];                               // seeds of the event (seed_kernel)
  const int t0 = __ldg(A.offsets + e);
  const int n = __ldg(A.offsets + e + 1) - t0;
  const size_t ev = (size_t)e * P.max_vtx;
  // an event beyond the n_tracks given to pv_find (PV_EVT_RECORD_OVERFLOW, no seeds) has no place in wrec[] / best[]
  const int nl = (unsigned)t0 + (unsigned)n > A.n_trk ? 0 : n;
  int sv[4];                                               // seed index of my first four tracks: loads issued now,
#pragma unroll                                             // consumed after the vertex sweep
  for (int q = 0; q < 4; ++q) sv[q] = (lane + 32 * q < n) ? A.trk_vertex[t0 + lane + 32 * q] : -1;
  // explicit flavour: the weight the fit left at the track's record.  The records of an event are the event's own
  // range of wrec[]: its first 128 weights are loaded in order, together with the seed indices (not behind them), and
  // picked from shared memory afterwards: two dependent levels of loads instead of three.
  __shared__ float s_w[8][128];
  float wl[4] = {0.0f, 0.0f, 0.0f, 0.0f};
  if (FLAV != PV_FLAVOUR_MULTIVERTEX) {
#pragma unroll
    for (int q = 0; q < 4; ++q) wl[q] = (lane + 32 * q < nl) ? A.wrec[t0 + lane + 32 * q] : 0.0f;
  }
  unsigned long long bv[4] = {0ull, 0ull, 0ull, 0ull};     // multi-vertex flavour: largest weight << 32 | 31 - seed
  if (FLAV == PV_FLAVOUR_MULTIVERTEX) {
#pragma unroll
    for (int q = 0; q < 4; ++q) bv[q] = (lane + 32 * q < nl) ? A.best[t0 + lane + 32 * q] : 0ull;
  }
  float vp[3] = {0.0f, 0.0f, 0.0f}, vc[6] = {0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f};
  float vchi2 = 0.0f;
  int vntrk = 0, vniter = -1;
  if (lane < ns) {                                         // (a slot the fit never wrote holds niter = -1 and is not used)
    const size_t o = ev + lane;
    vniter = A.vtx_niter[o];
#pragma unroll
    for (int c = 0; c < 3; ++c) vp[c] = A.vtx_pos[o * 3 + c];
#pragma unroll
    for (int c = 0; c < 6; ++c) vc[c] = A.vtx_cov[o * 6 + c];
    vchi2 = A.vtx_chi2[o]; vntrk = A.vtx_ntracks[o];
  }
  float wv[4] = {0.0f, 0.0f, 0.0f, 0.0f};
  if (FLAV != PV_FLAVOUR_MULTIVERTEX) {
    const int warp = (threadIdx.x >> 5) & 7;
#pragma unroll
    for (int q = 0; q < 4; ++q) s_w[warp][lane + 32 * q] = wl[q];
    __syncwarp();
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const int r = sv[q] >> 5;                              // position of the track's record within the event
      wv[q] = sv[q] < 0 ? 0.0f : (r < 128 ? s_w[warp][r] : A.wrec[t0 + r]);
    }
  }
  const unsigned alive = __ballot_sync(FULL, lane < ns && vniter >= 0);
  // duplicate removal: greedy sweep in z order; duplicate iff dz^2 / (Czz_v + Czz_s) < merge_ratio; the one
  // "with fewer associated tracks" is rejected, ties keep the lower z.
  unsigned merged = 0;
  {
    int s = -1;
    float zs_ = 0.0f, cs_ = 0.0f;
    int ns_ = 0;
    unsigned rest = alive;
    while (rest) {
      const int v = __ffs(rest) - 1;
      rest &= rest - 1;
      const float zv = __shfl_sync(FULL, vp[2], v), cv = __shfl_sync(FULL, vc[5], v);
      const int nv = __shfl_sync(FULL, vntrk, v);
      bool take = true;
      if (s >= 0) {
        const float dzv = zv - zs_, csum = cv + cs_;
        // dz^2 / (Czz_v + Czz_s) < merge_ratio without the division (the sum of two variances is positive)
        const bool dup = csum > 0.0f ? dzv * dzv < P.merge_ratio * csum : dzv * dzv / csum < P.merge_ratio;
        if (dup) {
          if (nv > ns_) merged |= 1u << s;
          else { merged |= 1u << v; take = false; }
        }
      }
      if (take) { s = v; zs_ = zv; cs_ = cv; ns_ = nv; }
    }
  }
  int fate = -9;
  bool keep = false;
  if (lane < ns) {
    if (!((alive >> lane) & 1u)) fate = -1;
    else if ((merged >> lane) & 1u) fate = -2;
    else {
      const int region = vp[2] < P.z_split ? 1 : 0;
      if (vntrk < P.min_tracks_pv[region]) fate = -3;                       // Table 2 "Min. tracks in the PV"
      else {
        keep = true;
        if (region == 0) {
          const float dx = vp[0] - fmaf(P.beam_tx, vp[2], P.beam_x), dy = vp[1] - fmaf(P.beam_ty, vp[2], P.beam_y);
          if (fmaf(dx, dx, dy * dy) > P.max_beam_dist2) { keep = false; fate = -4; }
        }
      }
    }
  }
  const unsigned kept = __ballot_sync(FULL, keep);
  const int myidx = __popc(kept & lanemask_lt());
  if (DBG && lane < ns) {
    const size_t o = ev + lane;
    if (A.dbg.seed_niter) A.dbg.seed_niter[o] = vniter;
    if (A.dbg.seed_fate) A.dbg.seed_fate[o] = keep ? myidx : fate;
    if (vniter >= 0) {
      if (A.dbg.seed_pos) for (int c = 0; c < 3; ++c) A.dbg.seed_pos[o * 3 + c] = vp[c];
      if (A.dbg.seed_cov) for (int c = 0; c < 6; ++c) A.dbg.seed_cov[o * 6 + c] = vc[c];
      if (A.dbg.seed_chi2) A.dbg.seed_chi2[o] = vchi2;
      if (A.dbg.seed_ntrk) A.dbg.seed_ntrk[o] = vntrk;
    }
  }
  __syncwarp();                                            // every lane has read its slot: compact in place
  if (keep) {
    const size_t o = ev + myidx;
#pragma unroll
    for (int c = 0; c < 3; ++c) A.vtx_pos[o * 3 + c] = vp[c];
#pragma unroll
    for (int c = 0; c < 6; ++c) A.vtx_cov[o * 6 + c] = vc[c];
    A.vtx_chi2[o] = vchi2; A.vtx_ntracks[o] = vntrk; A.vtx_niter[o] = vniter;
  }
  if (lane == 0) A.n_vtx[e] = __popc(kept);
  // final per-track outputs; tracks of rejected vertices are released (R-9)
  auto finish = [&](int i, int s, unsigned long long b, float w) {
    if (FLAV == PV_FLAVOUR_MULTIVERTEX) {                  // R-13: the track follows the seed with its largest weight
      w = __uint_as_float((unsigned)(b >> 32));
      s = w > 0.0f ? 31 - (int)(b & 31ull) : -1;
      if (DBG && A.dbg.trk_seed) A.dbg.trk_seed[t0 + i] = s;
    } else if (s >= 0) {                                   // explicit flavour: seed | record position << 5 (seed_kernel)
      s &= 31;
    }
    int vtx = -1;
    if (s >= 0 && ((kept >> s) & 1u)) vtx = __popc(kept & ((1u << s) - 1u));
    A.trk_vertex[t0 + i] = vtx;
    if (A.trk_vertex8) A.trk_vertex8[t0 + i] = (int8_t)vtx;
    A.trk_weight[t0 + i] = vtx >= 0 ? w : 0.0f;
  };
#pragma unroll
  for (int q = 0; q < 4; ++q)
    if (lane + 32 * q < n) finish(lane + 32 * q, sv[q], bv[q], wv[q]);
  for (int i = 128 + lane; i < n; i += 32) {
    const int s = A.trk_vertex[t0 + i];
    const float w = (FLAV != PV_FLAVOUR_MULTIVERTEX && s >= 0) ? A.wrec[t0 + (s >> 5)] : 0.0f;
    finish(i, s, (FLAV == PV_FLAVOUR_MULTIVERTEX && i < nl) ? A.best[t0 + i] : 0ull, w);
  }
}

// ---- host pipeline: the PVs of a chunk of events packed into 48-byte records in event order, so that the
// device-to-host copy moves sum(n_vtx) records instead of n_events * max_vtx slots.
// scan_nvtx_kernel: one CTA; begin[e] = sum of n_vtx[0..e), begin[n_events] = total (exclusive scan, tiles of 1024).
__global__ void __launch_bounds__(1024) scan_nvtx_kernel(const int32_t* __restrict__ n_vtx, int n_events,
                                                         int32_t* __restrict__ begin) {
  __shared__ int wsum[32];
  __shared__ int carry_s;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  for (int base = 0; base < n_events; base += 1024) {
    const int e = base + threadIdx.x;
    const int v = e < n_events ? n_vtx[e] : 0;
    const int inc = warp_incl_scan(v, lane);
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    const int carry = carry_s;
    int wv = wsum[lane];
    const int winc = warp_incl_scan(wv, lane);                 // every warp scans the 32 warp totals
    const int woff = __shfl_sync(FULL, winc - wv, warp);
    if (e < n_events) begin[e] = carry + woff + inc - v;
    __syncthreads();
    if (threadIdx.x == 1023) carry_s = carry + woff + inc;
    __syncthreads();
  }
  if (threadIdx.x == 0) begin[n_events] = carry_s;
}

// pack_vertices_kernel: one warp per event, lane k = vertex k of the event -> record begin[e] + k.
__global__ void __launch_bounds__(256) pack_vertices_kernel(const __grid_constant__ KArgs A, int max_vtx,
                                                            const int32_t* __restrict__ begin, pv_vertex* __restrict__ out) {
  const int lane = threadIdx.x & 31;
  const int e = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (e >= A.n_events) return;
  const int b = begin[e], nv = begin[e + 1] - b;
  if (lane < nv) {
    const size_t o = (size_t)e * max_vtx + lane;
    float4 q0, q1, q2;
    q0.x = A.vtx_pos[o * 3 + 0]; q0.y = A.vtx_pos[o * 3 + 1]; q0.z = A.vtx_pos[o * 3 + 2]; q0.w = A.vtx_cov[o * 6 + 0];
    q1.x = A.vtx_cov[o * 6 + 1]; q1.y = A.vtx_cov[o * 6 + 2]; q1.z = A.vtx_cov[o * 6 + 3]; q1.w = A.vtx_cov[o * 6 + 4];
    q2.x = A.vtx_cov[o * 6 + 5]; q2.y = A.vtx_chi2[o];
    q2.z = __int_as_float(A.vtx_ntracks[o]); q2.w = __int_as_float(A.vtx_niter[o]);
    float4* dst = reinterpret_cast<float4*>(out + b + lane);
    dst[0] = q0; dst[1] = q1; dst[2] = q2;
  }
}

// ---- ip_kernel: NEXT-4, impact parameter and IP chi2 of every track w.r.t. the PVs of its event ---------
// One warp per event.  The event's vertices (position, covariance) are staged in shared memory and read back as
// broadcasts; each lane walks its tracks and keeps the vertex with the smallest IP chi2 (ties: lower index).
// For a vertex that does not contain the track: r = Eq. 9 residual at the vertex z, IP = distance of the line to the
// point, IP chi2 = r^T (V + H C H^T)^-1 r with V from Eq. 2 (diagonal) at the vertex z, H of Eq. 12.
// One pass over 36 B/track in, 12 B/track out: HBM-bound.
template <bool CROSS>
__global__ void __launch_bounds__(256) ip_kernel(const __grid_constant__ KParams P, const __grid_constant__ KArgs A,
                                                 const float* __restrict__ vpos, const float* __restrict__ vcov,
                                                 const int32_t* __restrict__ nvtx, float* __restrict__ ip,
                                                 float* __restrict__ ip_chi2, int32_t* __restrict__ ip_vertex) {
  __shared__ float sv[8][MAXV][9];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int e = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  if (e >= A.n_events) return;
  const int t0 = __ldg(A.offsets + e);
  const int n = __ldg(A.offsets + e + 1) - t0;
  const int nv = min(__ldg(nvtx + e), P.max_vtx);
  constexpr bool have_cross = CROSS;                       // compiled twice: the diagonal case carries no double arithmetic
  if (lane < nv) {
    const size_t o = (size_t)e * P.max_vtx + lane;
#pragma unroll
    for (int c = 0; c < 3; ++c) sv[warp][lane][c] = __ldg(vpos + o * 3 + c);
#pragma unroll
    for (int c = 0; c < 6; ++c) sv[warp][lane][3 + c] = __ldg(vcov + o * 6 + c);
  }
  __syncwarp();
  constexpr int U = 2;                                     // tracks per lane in flight: 18 loads before the first use
#pragma unroll 1
  for (int i0 = lane; i0 < n; i0 += 32 * U) {
    float x[U], y[U], z[U], a[U], b[U], vx[U], vy[U], vtx[U], vty[U], cx[U], cy[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int g = t0 + min(i0 + 32 * u, n - 1);
      cx[u] = (CROSS && A.cov_xtx) ? __ldg(A.cov_xtx + g) : 0.0f; cy[u] = (CROSS && A.cov_yty) ? __ldg(A.cov_yty + g) : 0.0f;
      x[u] = __ldg(A.x + g); y[u] = __ldg(A.y + g); z[u] = __ldg(A.z + g); a[u] = __ldg(A.tx + g); b[u] = __ldg(A.ty + g);
      vx[u] = __ldg(A.var_x + g); vy[u] = __ldg(A.var_y + g); vtx[u] = __ldg(A.var_tx + g); vty[u] = __ldg(A.var_ty + g);
    }
    float best_c[U], best_rx[U], best_ry[U];
    int best_v[U];
    bool usable[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      best_c[u] = INFINITY; best_rx[u] = 0.0f; best_ry[u] = 0.0f; best_v[u] = -1;
      usable[u] = true;
    }
    // The two tracks of a lane go through the vertex loop side by side in packed fp32 pairs (FFMA2 / FADD2 / FMUL2 of
    // sm_100): the same operations in the same order as the scalar form, half the floating-point instructions.
    static_assert(U == 2, "the two tracks of a lane are packed in pairs");
    const float2 X = make_float2(x[0], x[1]), Y = make_float2(y[0], y[1]), nZ = make_float2(-z[0], -z[1]);
    const float2 Aa = make_float2(a[0], a[1]), Bb = make_float2(b[0], b[1]), nBb = make_float2(-b[0], -b[1]);
    const float2 VX = make_float2(vx[0], vx[1]), VY = make_float2(vy[0], vy[1]);
    const float2 VTX = make_float2(vtx[0], vtx[1]), VTY = make_float2(vty[0], vty[1]);
    auto dup = [](const float v) { return make_float2(v, v); };
#pragma unroll 1
    for (int v = 0; v < nv; ++v) {
      const float* q = sv[warp][v];
      const float q0 = q[0], q1 = q[1], q2 = q[2], q3 = q[3], q4 = q[4], q5 = q[5], q6 = q[6], q7 = q[7], q8 = q[8];
      const float2 dz = __fadd2_rn(dup(q2), nZ);
      float2 Vx, Vy;
      if (have_cross) {
        Vx = make_float2(var_at(vx[0], vtx[0], cx[0], dz.x, true), var_at(vx[1], vtx[1], cx[1], dz.y, true));
        Vy = make_float2(var_at(vy[0], vty[0], cy[0], dz.x, true), var_at(vy[1], vty[1], cy[1], dz.y, true));
      } else {
        Vx = __ffma2_rn(dz, __fmul2_rn(dz, VTX), VX);
        Vy = __ffma2_rn(dz, __fmul2_rn(dz, VTY), VY);
      }
      const float2 rx = __ffma2_rn(dz, Aa, __fadd2_rn(X, dup(-q0))), ry = __ffma2_rn(dz, Bb, __fadd2_rn(Y, dup(-q1)));
      const float2 Sxx = __ffma2_rn(Aa, __ffma2_rn(Aa, dup(q8), dup(-2.0f * q5)), __fadd2_rn(Vx, dup(q3)));
      const float2 Syy = __ffma2_rn(Bb, __ffma2_rn(Bb, dup(q8), dup(-2.0f * q7)), __fadd2_rn(Vy, dup(q6)));
      const float2 Sxy = __ffma2_rn(Aa, __ffma2_rn(Bb, dup(q8), dup(-q7)), __ffma2_rn(nBb, dup(q5), dup(q4)));
      const float2 sq = __fmul2_rn(Sxy, Sxy);
      const float2 det = __ffma2_rn(Sxx, Syy, make_float2(-sq.x, -sq.y));
      const float2 cr = __fmul2_rn(__fmul2_rn(__fmul2_rn(dup(-2.0f), Sxy), rx), ry);
      const float2 num = __ffma2_rn(__fmul2_rn(Syy, rx), rx, __ffma2_rn(__fmul2_rn(Sxx, ry), ry, cr));
      const float c2[U] = {__fdividef(num.x, det.x), __fdividef(num.y, det.y)};
      const float Vxs[U] = {Vx.x, Vx.y}, Vys[U] = {Vy.x, Vy.y}, Sxxs[U] = {Sxx.x, Sxx.y}, dets[U] = {det.x, det.y};
      const float rxs[U] = {rx.x, rx.y}, rys[U] = {ry.x, ry.y};
#pragma unroll
      for (int u = 0; u < U; ++u) {
        // R-7 and positive definiteness: Vx, Vy positive and finite, Sxx > 0, det > 0 (NaN fails every test)
        const bool ok = usable[u] && Vxs[u] > 0.0f && Vys[u] > 0.0f && Vxs[u] < INFINITY && Vys[u] < INFINITY && Sxxs[u] > 0.0f &&
                        dets[u] > 0.0f;
        if (ok && c2[u] < best_c[u]) { best_c[u] = c2[u]; best_rx[u] = rxs[u]; best_ry[u] = rys[u]; best_v[u] = v; }
      }
    }
    float best_d[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {                          // the IP itself only for the chosen vertex
      const float al = fmaf(best_rx[u], a[u], best_ry[u] * b[u]);
      const float d2 = fmaf(best_rx[u], best_rx[u], best_ry[u] * best_ry[u]) -
                       al * al * __fdividef(1.0f, fmaf(a[u], a[u], fmaf(b[u], b[u], 1.0f)));
      best_d[u] = best_v[u] >= 0 ? sqrtf(fmaxf(d2, 0.0f)) : -1.0f;
      if (best_v[u] < 0) best_c[u] = -1.0f;
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int i = i0 + 32 * u;
      if (i < n) { ip[t0 + i] = best_d[u]; ip_chi2[t0 + i] = best_c[u]; ip_vertex[t0 + i] = best_v[u]; }
    }
  }
}

}  // namespace pvk

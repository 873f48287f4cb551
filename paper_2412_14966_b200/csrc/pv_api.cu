// pv_api.cu -- host side of the C ABI declared in include/pv_finder.h: parameter validation, conversion of
// the paper's thresholds to the fixed-point contract, launch of the three kernels (seed, fit, cleanup), and the
// host-buffer pipeline.  No CPU fallback exists: without a CUDA device every compute entry returns
// PV_E_CUDA.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <mutex>
#include <vector>

#include <nvtx3/nvToolsExt.h>   // header-only; the ranges cost nothing measurable when no profiler is attached

#include "pv_kernels.cuh"

namespace {

// NVTX range around the launches of one stage of pv_find: shows up per stage in a timeline.
struct NvtxRange {
  explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
  ~NvtxRange() { nvtxRangePop(); }
};

thread_local char g_cuda_err[512] = "";
int g_last_kernels = 0, g_last_grid = 0, g_last_block = 0, g_last_smem = 0;
int g_timing = 0;
constexpr int N_KERNELS = 3;
cudaEvent_t g_ev[N_KERNELS + 1] = {nullptr, nullptr, nullptr, nullptr};
bool g_ev_valid = false;

int cuda_fail(cudaError_t err, const char* what) {
  snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", what, cudaGetErrorString(err));
  return PV_E_CUDA;
}
#define CK(call)                                        \
  do {                                                  \
    cudaError_t err__ = (call);                         \
    if (err__ != cudaSuccess) return cuda_fail(err__, #call); \
  } while (0)

struct DeviceInfo {
  int device = -1, sms = 0, max_smem_optin = 0;
  bool attr_set[16] = {false};                         // [debug + 2 flavour + 4 split + 8 fill]
  int attr_smem[16] = {0};
  int fit_blocks_per_sm[2] = {0, 0};                  // [flavour]
};
std::mutex g_mu;
std::vector<DeviceInfo> g_dev;

int get_device_info(DeviceInfo** out) {
  int dev = 0;
  CK(cudaGetDevice(&dev));
  for (auto& d : g_dev)
    if (d.device == dev) { *out = &d; return PV_OK; }
  DeviceInfo d;
  d.device = dev;
  CK(cudaDeviceGetAttribute(&d.sms, cudaDevAttrMultiProcessorCount, dev));
  CK(cudaDeviceGetAttribute(&d.max_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
  g_dev.push_back(d);
  *out = &g_dev.back();
  return PV_OK;
}

long long to_fixed(float tracks) {
  const double v = (double)tracks * (double)PV_FIXED_ONE;
  if (!(v < 9.0e18)) return 0x7fffffffffffffffLL;
  if (!(v > -9.0e18)) return -0x7fffffffffffffffLL;
  return llrint(v);
}
int clamp_i32(long long v) {
  if (v > 0x7fffffffLL) return 0x7fffffff;
  if (v < -0x7fffffffLL) return -0x7fffffff;
  return (int)v;
}

size_t tmpl_layout(const pv_params* p, pvk::KParams* k);

int validate(const pv_params* p, int* nbins_out) {
  if (!p) return PV_E_NULL;
  if (!(p->dz > 0.0f) || !(p->z_max > p->z_min)) return PV_E_PARAM;
  const double nb = ((double)p->z_max - (double)p->z_min) / (double)p->dz;
  if (!(nb >= 1.0) || nb > (double)PV_MAX_BINS + 0.5) return PV_E_PARAM;
  const int nbins = (int)lrint(nb);
  if (nbins < 1 || nbins > PV_MAX_BINS) return PV_E_PARAM;
  if (fabs((double)nbins * (double)p->dz - ((double)p->z_max - (double)p->z_min)) > 1e-6 * (double)p->dz) return PV_E_PARAM;
  if (p->max_vtx_per_event < 1 || p->max_vtx_per_event > PV_MAX_VTX) return PV_E_PARAM;
  if (p->max_iter < 1 || p->max_iter > 16) return PV_E_PARAM;
  if (!(p->chi2_max > 0.0f)) return PV_E_PARAM;
  if (!(p->min_bin_content >= 0.0f)) return PV_E_PARAM;      // only bins a track wrote can start a proto-cluster
  if (p->flavour != PV_FLAVOUR_EXPLICIT && p->flavour != PV_FLAVOUR_MULTIVERTEX) return PV_E_PARAM;
  if (p->split_mode != PV_SPLIT_Z_ORDERED && p->split_mode != PV_SPLIT_RECURSIVE) return PV_E_PARAM;
  if (p->fill_mode != PV_FILL_POLYNOMIAL && p->fill_mode != PV_FILL_TEMPLATE) return PV_E_PARAM;
  if (p->flavour == PV_FLAVOUR_MULTIVERTEX && (!(p->chi2_window > 0.0f) || isinf(p->chi2_max))) return PV_E_PARAM;
  // the fill cuts a track's +-3 sigma window into units of PV_UNIT bins and numbers them with 9 bits
  constexpr int max_window = pvk::MAX_FILL_UNITS * pvk::UNIT;
  for (int r = 0; r < 2; ++r)
    if (!(6.0 * (double)p->max_sigma_poca[r] / (double)p->dz + 4.0 <= (double)max_window)) return PV_E_PARAM;
  // template fill: the window is that of the class centre, up to 2^(1/8) wider than the track's own sigma
  if (p->fill_mode == PV_FILL_TEMPLATE) {
    pvk::KParams k;
    tmpl_layout(p, &k);
    const int widest = 2 * (int)k.tmpl_w[k.tmpl_kmax] + 1;
    if ((widest < nbins ? widest : nbins) > max_window) return PV_E_PARAM;
  }
  if (nbins_out) *nbins_out = nbins;
  return PV_OK;
}

// Template fill (reading R-17): host restatement of the class arithmetic of pv_kernels.cuh (fp32, one rounding
// per operation), used to lay out the table: class of a sigma, centre of a class in bins.
int tmpl_class_raw_host(float sigma, float inv_dz) {
  const float v = (sigma * inv_dz) * 12.5f;
  if (!(v >= 1.0f)) return 0;
  if (!(v < 0x1p+20f)) return 80;
  int E;
  const float m = 2.0f * frexpf(v, &E);
  return 4 * (E - 1) + (m >= 0x1.172b84p+0f ? 1 : 0) + (m >= 0x1.4bfdaep+0f ? 1 : 0) + (m >= 0x1.8ace54p+0f ? 1 : 0) +
         (m >= 0x1.d5818ep+0f ? 1 : 0);
}
float tmpl_centre_host(int k) {
  static const float c[4] = {1.0f, 0x1.306fe0p+0f, 0x1.6a09e6p+0f, 0x1.ae89fap+0f};
  return ldexpf(c[k & 3], k >> 2) * 0.08f;
}

// entries (int32) of the template table for these parameters; fills the layout fields of *k when given
size_t tmpl_layout(const pv_params* p, pvk::KParams* k) {
  const float inv_dz = 1.0f / p->dz;
  const float smax = p->max_sigma_poca[0] > p->max_sigma_poca[1] ? p->max_sigma_poca[0] : p->max_sigma_poca[1];
  int kmax = tmpl_class_raw_host(smax, inv_dz);
  if (kmax > pvk::TMPL_MAXK - 1) kmax = pvk::TMPL_MAXK - 1;       // validate() keeps sigma / dz below 512: class <= 51
  size_t n = 0;
  for (int c = 0; c <= kmax; ++c) {
    const int W = (int)ceilf(3.0f * tmpl_centre_host(c));
    if (k) { k->tmpl_off[c] = (int)n; k->tmpl_w[c] = (short)W; }
    n += (size_t)pvk::TMPL_J * (size_t)(2 * W + 1);
  }
  if (k) k->tmpl_kmax = kmax;
  return n;
}

void make_kparams(const pv_params* p, int nbins, pvk::KParams* k) {
  memset(k, 0, sizeof(*k));
  k->z_min = p->z_min; k->dz = p->dz; k->inv_dz = 1.0f / p->dz; k->z_split = p->z_split;
  k->beam_x = p->beam_x; k->beam_y = p->beam_y; k->beam_tx = p->beam_tx; k->beam_ty = p->beam_ty;
  k->max_sigma[0] = p->max_sigma_poca[0]; k->max_sigma[1] = p->max_sigma_poca[1];
  k->win_eps = 0.0625f + 2e-6f * (float)nbins;
  k->nbins = nbins; k->nwords = (nbins + 31) / 32;
  k->T_bin = clamp_i32(to_fixed(p->min_bin_content));
  k->D = clamp_i32(to_fixed(p->min_dip));
  k->I_min[0] = clamp_i32(to_fixed(p->min_cluster_integral[0]));   // an event holds < 2047 * 2^20 < 2^31
  k->I_min[1] = clamp_i32(to_fixed(p->min_cluster_integral[1]));
  for (int r = 0; r < 2; ++r) { k->min_tracks_seed[r] = p->min_tracks_seed[r]; k->min_tracks_pv[r] = p->min_tracks_pv[r]; }
  k->chi2_max = p->chi2_max;
  k->unit_weights = (isinf(p->chi2_max) && p->flavour == PV_FLAVOUR_EXPLICIT) ? 1 : 0;
  k->flavour = p->flavour;
  k->split_mode = p->split_mode;
  k->chi2_window = p->chi2_window;
  k->mv_e0 = expf(-0.5f * p->chi2_max);
  k->inv_chi2_max = k->unit_weights ? 0.0f : 1.0f / p->chi2_max;
  k->max_iter = p->max_iter;
  k->conv_dchi2 = p->conv_dchi2; k->conv_dz = p->conv_dz; k->merge_ratio = p->merge_ratio;
  k->max_beam_dist2 = p->max_beam_dist * p->max_beam_dist;
  k->max_vtx = p->max_vtx_per_event;
  if (p->fill_mode == PV_FILL_TEMPLATE) tmpl_layout(p, k);
}

// Workspace layout: [0, 256) counters | seed records, 16 B each, n_events * max_vtx | fit-ready track records,
// 32 B each, sorted by seed: one per track (explicit flavour) or up to two per track (multi-vertex flavour, a track
// is listed once per seed in its chi2 window) | explicit flavour: 4 B per track record (its Tukey weight, record order);
// multi-vertex flavour: 8 B per track (largest weight and its seed).
constexpr size_t WS_COUNTERS = 256;
size_t ws_rec_bytes(int n_events, int max_vtx) { return (size_t)n_events * (size_t)max_vtx * sizeof(pvk::SeedRec); }
size_t ws_trk_records(long long n_tracks, int flavour) {
  return (size_t)n_tracks * (flavour == PV_FLAVOUR_MULTIVERTEX ? 2 : 1);
}
size_t ws_core_bytes(int n_events, long long n_tracks, int max_vtx, int flavour) {
  size_t b = WS_COUNTERS + ws_rec_bytes(n_events, max_vtx) + ws_trk_records(n_tracks, flavour) * 32 + 16;
  if (flavour == PV_FLAVOUR_MULTIVERTEX) b += (size_t)n_tracks * 8 + 16;     // best[]
  else b += (size_t)n_tracks * 4 + 16;                                       // wrec[]
  return (b + 15) / 16 * 16;
}
size_t ws_bytes(int n_events, long long n_tracks, const pv_params* p) {
  size_t b = ws_core_bytes(n_events, n_tracks, p->max_vtx_per_event, p->flavour);
  if (p->fill_mode == PV_FILL_TEMPLATE) b += tmpl_layout(p, nullptr) * sizeof(int32_t) + 16;   // template table
  return b;
}


int find_impl(const float* x, const float* y, const float* z, const float* tx, const float* ty,
              const float* var_x, const float* var_y, const float* var_tx, const float* var_ty,
              const int32_t* offsets, int n_events, long long n_tracks, const pv_params* params,
              float* vtx_pos, float* vtx_cov, float* vtx_chi2, int32_t* vtx_ntracks, int32_t* vtx_niter,
              int32_t* n_vtx, float* trk_weight, int32_t* trk_vertex, uint32_t* event_status,
              void* workspace, size_t workspace_bytes, void* stream_, const pv_debug* dbg,
              const pv_track_cov* cov = nullptr, int8_t* trk_vertex8 = nullptr) {
  int nbins = 0;
  int rc = validate(params, &nbins);
  if (rc != PV_OK) return rc;
  if (n_events < 0 || n_tracks < 0 || n_tracks > 0x7fffffffLL) return PV_E_SIZE;
  // multi-vertex flavour: two track records per track, indexed with 32 bits
  if (params->flavour == PV_FLAVOUR_MULTIVERTEX && n_tracks > 0x3fffffffLL) return PV_E_SIZE;
  if (n_events == 0) { g_last_kernels = 0; g_last_grid = 0; return PV_OK; }   // empty batch: nothing to enqueue
  if (!offsets || !n_vtx || !event_status || !vtx_pos || !vtx_cov || !vtx_chi2 || !vtx_ntracks || !vtx_niter || !workspace)
    return PV_E_NULL;
  if (n_tracks > 0 && (!x || !y || !z || !tx || !ty || !var_x || !var_y || !var_tx || !var_ty || !trk_weight || !trk_vertex))
    return PV_E_NULL;
  if (workspace_bytes < ws_bytes(n_events, n_tracks, params)) return PV_E_WORKSPACE;
  if (((uintptr_t)workspace & 15) != 0) return PV_E_PARAM;
  cudaStream_t stream = (cudaStream_t)stream_;

  std::lock_guard<std::mutex> lock(g_mu);
  DeviceInfo* di = nullptr;
  rc = get_device_info(&di);
  if (rc != PV_OK) return rc;

  pvk::KParams kp;
  make_kparams(params, nbins, &kp);
  // seed_kernel: one warp per event, SEED_WARPS of them per CTA; what the warps' own state leaves of the shared memory
  // is the CTA's pool of histogram blocks (a NULL word first)
  int warps = pvk::SEED_WARPS;
#ifdef PV_TUNING                                              // tuning builds only: fewer events in flight per CTA
  if (const char* envw = getenv("PV_WARPS_PER_CTA")) {
    const int w = atoi(envw);
    if (w >= 1 && w < warps) warps = w;
  }
#endif
  const int fixed = 128 + pvk::SM_HDR_BYTES + warps * pvk::WARP_SMEM;
  int n_pool = (di->max_smem_optin - fixed) / 128;            // words of 32 bins
  if (n_pool > pvk::SM_HDR_BYTES * 8) n_pool = pvk::SM_HDR_BYTES * 8;
#ifdef PV_TUNING
  if (const char* envb = getenv("PV_POOL_WORDS")) {
    const int w = atoi(envb);
    if (w >= 1 && w < n_pool) n_pool = w;
  }
#endif
  if (n_pool < pvk::MAX_WORDS) return PV_E_PARAM;             // one event may need every word of the histogram
  kp.n_pool = n_pool;
  const int smem = fixed + n_pool * 128;
  const int mvf = params->flavour == PV_FLAVOUR_MULTIVERTEX ? 1 : 0;
  const int spl = params->split_mode == PV_SPLIT_RECURSIVE ? 1 : 0;
  const int tfl = params->fill_mode == PV_FILL_TEMPLATE ? 1 : 0;
  const int which = (dbg ? 1 : 0) + 2 * mvf + 4 * spl + 8 * tfl;
  static const void* const seed_fn[16] = {
      (const void*)pvk::seed_kernel<false, 0, 0, 0>, (const void*)pvk::seed_kernel<true, 0, 0, 0>,
      (const void*)pvk::seed_kernel<false, 1, 0, 0>, (const void*)pvk::seed_kernel<true, 1, 0, 0>,
      (const void*)pvk::seed_kernel<false, 0, 1, 0>, (const void*)pvk::seed_kernel<true, 0, 1, 0>,
      (const void*)pvk::seed_kernel<false, 1, 1, 0>, (const void*)pvk::seed_kernel<true, 1, 1, 0>,
      (const void*)pvk::seed_kernel<false, 0, 0, 1>, (const void*)pvk::seed_kernel<true, 0, 0, 1>,
      (const void*)pvk::seed_kernel<false, 1, 0, 1>, (const void*)pvk::seed_kernel<true, 1, 0, 1>,
      (const void*)pvk::seed_kernel<false, 0, 1, 1>, (const void*)pvk::seed_kernel<true, 0, 1, 1>,
      (const void*)pvk::seed_kernel<false, 1, 1, 1>, (const void*)pvk::seed_kernel<true, 1, 1, 1>};
  if (!di->attr_set[which] || di->attr_smem[which] < smem) {
    CK(cudaFuncSetAttribute(seed_fn[which], cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    di->attr_set[which] = true;
    di->attr_smem[which] = smem;
  }
  if (di->fit_blocks_per_sm[mvf] == 0) {
    int nb = 0;
    if (mvf) CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, pvk::fit_kernel<1>, pvk::FIT_BLOCK, 0));
    else CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, pvk::fit_kernel<0>, pvk::FIT_BLOCK, 0));
    di->fit_blocks_per_sm[mvf] = nb > 0 ? nb : 1;
  }
  g_last_kernels = 0; g_last_grid = 0; g_last_block = warps * 32; g_last_smem = smem;

  pvk::KArgs ka;
  memset(&ka, 0, sizeof(ka));
  ka.x = x; ka.y = y; ka.z = z; ka.tx = tx; ka.ty = ty;
  ka.var_x = var_x; ka.var_y = var_y; ka.var_tx = var_tx; ka.var_ty = var_ty;
  if (cov) { ka.cov_xtx = cov->cov_xtx; ka.cov_yty = cov->cov_yty; }
  ka.offsets = offsets; ka.n_events = n_events;
  ka.vtx_pos = vtx_pos; ka.vtx_cov = vtx_cov; ka.vtx_chi2 = vtx_chi2;
  ka.vtx_ntracks = vtx_ntracks; ka.vtx_niter = vtx_niter; ka.n_vtx = n_vtx;
  ka.trk_weight = trk_weight; ka.trk_vertex = trk_vertex; ka.event_status = event_status;
  ka.trk_vertex8 = trk_vertex8;
  unsigned char* ws = reinterpret_cast<unsigned char*>(workspace);
  ka.evt_counter = reinterpret_cast<unsigned int*>(ws);
  ka.seed_counter = reinterpret_cast<unsigned int*>(ws + 16);
  ka.rec = reinterpret_cast<pvk::SeedRec*>(ws + WS_COUNTERS);
  ka.trk_counter = reinterpret_cast<unsigned int*>(ws + 32);
  ka.fit_counter = reinterpret_cast<unsigned int*>(ws + 48);
  ka.ill_counter = reinterpret_cast<unsigned int*>(ws + 64);
  ka.ftrk = reinterpret_cast<float4*>(ws + WS_COUNTERS + ws_rec_bytes(n_events, params->max_vtx_per_event));
  ka.trk_cap = (unsigned int)ws_trk_records(n_tracks, params->flavour);
  ka.n_trk = (unsigned int)n_tracks;
  ka.best = reinterpret_cast<unsigned long long*>(reinterpret_cast<unsigned char*>(ka.ftrk) + (size_t)ka.trk_cap * 32 + 16);
  ka.wrec = reinterpret_cast<float*>(ka.best);                // the two flavours use the same place differently
  ka.tmpl = reinterpret_cast<int32_t*>(ws + ws_core_bytes(n_events, n_tracks, params->max_vtx_per_event, params->flavour));
  if (dbg) ka.dbg = *dbg;

  const bool timing = g_timing != 0;
  if (timing && !g_ev[0])
    for (int i = 0; i <= N_KERNELS; ++i) CK(cudaEventCreate(&g_ev[i]));
  CK(cudaMemsetAsync(workspace, 0, 128, stream));
  // a1..a4: persistent, one CTA per SM, one warp per event
  int grid = di->sms;
  const int need = n_events;                                  // a small batch is spread over the SMs, not packed into few CTAs
  if (grid > need) grid = need;
  if (timing) CK(cudaEventRecord(g_ev[0], stream));
  if (tfl) {                                                  // the table of template histograms, ~10^4 entries
    NvtxRange range("pv_find: template table");
    pvk::tmpl_kernel<<<kp.tmpl_kmax + 1, 256, 0, stream>>>(kp, ka.tmpl);
    CK(cudaGetLastError());
  }
  {
    NvtxRange range("pv_find: a1-a4 seed");
    void* kargs[2] = {(void*)&kp, (void*)&ka};
    CK(cudaLaunchKernel(seed_fn[which], dim3(grid), dim3(warps * 32), kargs, (size_t)smem, stream));
  }
  CK(cudaGetLastError());
  if (timing) CK(cudaEventRecord(g_ev[1], stream));
  // a5: autonomous warps work through windows of seed records
  {
    NvtxRange range("pv_find: a5 fit");
    long long fit_grid = (long long)di->sms * di->fit_blocks_per_sm[mvf];
    const long long most = ((long long)n_events * params->max_vtx_per_event + pvk::FIT_BLOCK - 1) / pvk::FIT_BLOCK;
    if (fit_grid > most) fit_grid = most;
    if (fit_grid < 1) fit_grid = 1;
    if (mvf) pvk::fit_kernel<1><<<(int)fit_grid, pvk::FIT_BLOCK, 0, stream>>>(kp, ka);
    else pvk::fit_kernel<0><<<(int)fit_grid, pvk::FIT_BLOCK, 0, stream>>>(kp, ka);
    CK(cudaGetLastError());
    // the few ill-conditioned seeds fit_kernel set aside, refitted in double (timed with the fit)
    if (mvf) pvk::ill_kernel<1><<<32, 128, 0, stream>>>(kp, ka);
    else pvk::ill_kernel<0><<<32, 128, 0, stream>>>(kp, ka);
    CK(cudaGetLastError());
  }
  if (timing) CK(cudaEventRecord(g_ev[2], stream));
  // a6: one warp per event
  {
    NvtxRange range("pv_find: a6 cleanup");
    const int cgrid = (n_events + 7) / 8;
    if (mvf) {
      if (dbg) pvk::cleanup_kernel<true, 1><<<cgrid, 256, 0, stream>>>(kp, ka);
      else pvk::cleanup_kernel<false, 1><<<cgrid, 256, 0, stream>>>(kp, ka);
    } else {
      if (dbg) pvk::cleanup_kernel<true, 0><<<cgrid, 256, 0, stream>>>(kp, ka);
      else pvk::cleanup_kernel<false, 0><<<cgrid, 256, 0, stream>>>(kp, ka);
    }
    CK(cudaGetLastError());
  }
  if (timing) { CK(cudaEventRecord(g_ev[3], stream)); g_ev_valid = true; }
  g_last_kernels = N_KERNELS + 1 + tfl; g_last_grid = grid;
  return PV_OK;
}

}  // namespace

/* ---- pv_find_static: the workspace of callers that cannot allocate device memory (include/pv_finder.h) ----
 * The scratch of the three kernels, as a part of this library's device image: 16 MiB on every GPU that loads it.
 * In host code the name g_static_ws is only a handle for the runtime (a host-side shadow symbol); its value is NOT
 * where the array lives on the GPU, and a kernel given it would fault or scribble over host memory.  The address the
 * kernels need comes from cudaGetSymbolAddress, asked once per device with that device current. */
static __device__ __align__(256) unsigned char g_static_ws[PV_STATIC_WORKSPACE_BYTES];

namespace {

constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mu;
void* g_static_ws_ptr[STATIC_MAX_DEVICES] = {nullptr};   // device address of g_static_ws, per device ordinal

// Device address of g_static_ws on the current device; looked up at the first call on that device.
int static_workspace(void** out) {
  int dev = -1;
  CK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= STATIC_MAX_DEVICES) return PV_E_SIZE;
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_ws_ptr[dev]) {
    void* ptr = nullptr;
    CK(cudaGetSymbolAddress((void**)&ptr, g_static_ws));
    if (!ptr || ((uintptr_t)ptr & 255) != 0) return PV_E_CUDA;
    g_static_ws_ptr[dev] = ptr;
  }
  *out = g_static_ws_ptr[dev];
  return PV_OK;
}

}  // namespace

extern "C" {

int pv_find_static(const float* x, const float* y, const float* z, const float* tx, const float* ty,
                   const float* var_x, const float* var_y, const float* var_tx, const float* var_ty,
                   const int32_t* offsets, int n_events, long long n_tracks, const pv_params* params,
                   float* vtx_pos, float* vtx_cov, float* vtx_chi2, int32_t* vtx_ntracks, int32_t* vtx_niter,
                   int32_t* n_vtx, float* trk_weight, int32_t* trk_vertex, uint32_t* event_status, void* stream) {
  const int rc = validate(params, nullptr);
  if (rc != PV_OK) return rc;
  if (n_events < 0 || n_tracks < 0 || n_tracks > 0x7fffffffLL) return PV_E_SIZE;
  if (g_timing) return PV_E_PARAM;                            // the timing events would have to be created
  if (ws_bytes(n_events, n_tracks, params) > (size_t)PV_STATIC_WORKSPACE_BYTES) return PV_E_STATIC_LIMIT;
  void* ws = nullptr;
  const int src = static_workspace(&ws);
  if (src != PV_OK) return src;
  // from here on the path of pv_find: it clears the 64 bytes of counters at the head of the workspace on `stream`
  // and launches the kernels; none of it allocates
  return find_impl(x, y, z, tx, ty, var_x, var_y, var_tx, var_ty, offsets, n_events, n_tracks, params, vtx_pos, vtx_cov,
                   vtx_chi2, vtx_ntracks, vtx_niter, n_vtx, trk_weight, trk_vertex, event_status, ws,
                   (size_t)PV_STATIC_WORKSPACE_BYTES, stream, nullptr);
}

int pv_params_default(pv_params* p) {
  if (!p) return PV_E_NULL;
  p->z_min = -550.0f; p->z_max = 300.0f; p->dz = 0.25f;
  p->z_split = -300.0f;                                             /* Table 2 */
  p->beam_x = p->beam_y = p->beam_tx = p->beam_ty = 0.0f;
  p->max_sigma_poca[0] = 1.5f; p->max_sigma_poca[1] = 10.0f;
  p->min_bin_content = 0.25f; p->min_dip = 0.75f;                   /* reading R-4 */
  p->min_cluster_integral[0] = 2.5f; p->min_cluster_integral[1] = 1.75f;  /* Table 2 */
  p->min_tracks_seed[0] = 3; p->min_tracks_seed[1] = 2;
  p->min_tracks_pv[0] = 4; p->min_tracks_pv[1] = 3;                 /* Table 2 */
  p->chi2_max = 12.0f;
  p->max_iter = 10; p->conv_dchi2 = 0.01f; p->conv_dz = 0.001f;
  p->merge_ratio = 25.0f;
  p->max_beam_dist = 0.3f;
  p->max_vtx_per_event = 32;
  p->flavour = PV_FLAVOUR_EXPLICIT;
  p->chi2_window = 25.0f;                                           /* P:L384, value: reading R-13 */
  p->split_mode = PV_SPLIT_Z_ORDERED;
  p->fill_mode = PV_FILL_POLYNOMIAL;
  return PV_OK;
}

int pv_nbins(const pv_params* p) {
  int nb = 0;
  const int rc = validate(p, &nb);
  return rc == PV_OK ? nb : rc;
}

int pv_workspace_bytes(int n_events, long long n_tracks, const pv_params* p, size_t* bytes) {
  if (!bytes) return PV_E_NULL;
  const int rc = validate(p, nullptr);
  if (rc != PV_OK) return rc;
  if (n_events < 0 || n_tracks < 0) return PV_E_SIZE;
  if (n_tracks > 0x7fffffffLL) return PV_E_SIZE;
  *bytes = ws_bytes(n_events, n_tracks, p);
  return PV_OK;
}

int pv_find(const float* x, const float* y, const float* z, const float* tx, const float* ty,
            const float* var_x, const float* var_y, const float* var_tx, const float* var_ty,
            const int32_t* offsets, int n_events, long long n_tracks, const pv_params* params,
            float* vtx_pos, float* vtx_cov, float* vtx_chi2, int32_t* vtx_ntracks, int32_t* vtx_niter,
            int32_t* n_vtx, float* trk_weight, int32_t* trk_vertex, uint32_t* event_status,
            void* workspace, size_t workspace_bytes, void* stream) {
  return find_impl(x, y, z, tx, ty, var_x, var_y, var_tx, var_ty, offsets, n_events, n_tracks, params, vtx_pos, vtx_cov,
                   vtx_chi2, vtx_ntracks, vtx_niter, n_vtx, trk_weight, trk_vertex, event_status, workspace,
                   workspace_bytes, stream, nullptr);
}

int pv_find_debug(const float* x, const float* y, const float* z, const float* tx, const float* ty,
                  const float* var_x, const float* var_y, const float* var_tx, const float* var_ty,
                  const int32_t* offsets, int n_events, long long n_tracks, const pv_params* params,
                  float* vtx_pos, float* vtx_cov, float* vtx_chi2, int32_t* vtx_ntracks, int32_t* vtx_niter,
                  int32_t* n_vtx, float* trk_weight, int32_t* trk_vertex, uint32_t* event_status,
                  void* workspace, size_t workspace_bytes, void* stream, const pv_debug* dbg) {
  pv_debug none;
  memset(&none, 0, sizeof(none));
  return find_impl(x, y, z, tx, ty, var_x, var_y, var_tx, var_ty, offsets, n_events, n_tracks, params, vtx_pos, vtx_cov,
                   vtx_chi2, vtx_ntracks, vtx_niter, n_vtx, trk_weight, trk_vertex, event_status, workspace,
                   workspace_bytes, stream, dbg ? dbg : &none);
}

int pv_find_ext(const float* x, const float* y, const float* z, const float* tx, const float* ty,
                const float* var_x, const float* var_y, const float* var_tx, const float* var_ty,
                const int32_t* offsets, int n_events, long long n_tracks, const pv_params* params,
                float* vtx_pos, float* vtx_cov, float* vtx_chi2, int32_t* vtx_ntracks, int32_t* vtx_niter,
                int32_t* n_vtx, float* trk_weight, int32_t* trk_vertex, uint32_t* event_status,
                void* workspace, size_t workspace_bytes, void* stream, const pv_track_cov* cov, const pv_debug* dbg) {
  return find_impl(x, y, z, tx, ty, var_x, var_y, var_tx, var_ty, offsets, n_events, n_tracks, params, vtx_pos, vtx_cov,
                   vtx_chi2, vtx_ntracks, vtx_niter, n_vtx, trk_weight, trk_vertex, event_status, workspace,
                   workspace_bytes, stream, dbg, cov);
}

int pv_track_ip(const float* x, const float* y, const float* z, const float* tx, const float* ty,
                const float* var_x, const float* var_y, const float* var_tx, const float* var_ty,
                const int32_t* offsets, int n_events, long long n_tracks, const pv_params* params,
                const float* vtx_pos, const float* vtx_cov, const int32_t* n_vtx,
                float* ip, float* ip_chi2, int32_t* ip_vertex, const pv_track_cov* cov, void* stream_) {
  int nbins = 0;
  const int rc = validate(params, &nbins);
  if (rc != PV_OK) return rc;
  if (n_events < 0 || n_tracks < 0 || n_tracks > 0x7fffffffLL) return PV_E_SIZE;
  if (n_events == 0) return PV_OK;
  if (!offsets || !vtx_pos || !vtx_cov || !n_vtx) return PV_E_NULL;
  if (n_tracks > 0 && (!x || !y || !z || !tx || !ty || !var_x || !var_y || !var_tx || !var_ty || !ip || !ip_chi2 || !ip_vertex))
    return PV_E_NULL;
  pvk::KParams kp;
  make_kparams(params, nbins, &kp);
  pvk::KArgs ka;
  memset(&ka, 0, sizeof(ka));
  ka.x = x; ka.y = y; ka.z = z; ka.tx = tx; ka.ty = ty;
  ka.var_x = var_x; ka.var_y = var_y; ka.var_tx = var_tx; ka.var_ty = var_ty;
  if (cov) { ka.cov_xtx = cov->cov_xtx; ka.cov_yty = cov->cov_yty; }
  ka.offsets = offsets; ka.n_events = n_events;
  if (ka.cov_xtx || ka.cov_yty)
    pvk::ip_kernel<true><<<(n_events + 7) / 8, 256, 0, (cudaStream_t)stream_>>>(kp, ka, vtx_pos, vtx_cov, n_vtx, ip, ip_chi2, ip_vertex);
  else
    pvk::ip_kernel<false><<<(n_events + 7) / 8, 256, 0, (cudaStream_t)stream_>>>(kp, ka, vtx_pos, vtx_cov, n_vtx, ip, ip_chi2, ip_vertex);
  CK(cudaGetLastError());
  return PV_OK;
}

/* ------------------------------------------- host-buffer pipeline ------------------------------------------- */
constexpr int HOST_MAX_CHUNKS = 256;

struct pv_host_ctx {
  int max_events = 0;
  long long max_tracks = 0;
  int max_vtx = 0;
  int n_streams = 0;
  std::vector<cudaStream_t> streams;
  cudaStream_t h2d_stream = nullptr;          // every input copy, in chunk order: the host-to-device engine never waits
  cudaStream_t d2h_stream = nullptr;          // every fixed-size result copy
  cudaStream_t vtx_stream = nullptr;          // read-back of the packed vertices (sizes known once a chunk is done)
  cudaEvent_t up[HOST_MAX_CHUNKS] = {nullptr};     // inputs of the chunk are on the device
  cudaEvent_t done[HOST_MAX_CHUNKS] = {nullptr};   // kernels of the chunk have finished
  cudaEvent_t back[HOST_MAX_CHUNKS] = {nullptr};   // the chunk's vertex count is on the host
  int32_t* h_total = nullptr;                 // pinned: vertices found per chunk
  float* d_in[9] = {nullptr};
  int32_t* d_off = nullptr;
  float *d_pos = nullptr, *d_cov = nullptr, *d_chi2 = nullptr, *d_w = nullptr;
  int32_t *d_ntrk = nullptr, *d_niter = nullptr, *d_nvtx = nullptr, *d_tv = nullptr;
  int8_t* d_tv8 = nullptr;
  int32_t* d_vbegin = nullptr;                // per chunk: exclusive scan of n_vtx, ne + 1 entries at e0 + chunk index
  pv_vertex* d_packed = nullptr;              // per chunk: its vertices in event order, starting at record e0 * max_vtx
  uint32_t* d_status = nullptr;
  unsigned char* d_ws = nullptr;   // n_streams workspaces of ws_stride bytes each
  size_t ws_stride = 0;
};

int pv_host_ctx_destroy(pv_host_ctx* c) {
  if (!c) return PV_E_NULL;
  for (auto s : c->streams) cudaStreamDestroy(s);
  if (c->vtx_stream) cudaStreamDestroy(c->vtx_stream);
  if (c->h2d_stream) cudaStreamDestroy(c->h2d_stream);
  if (c->d2h_stream) cudaStreamDestroy(c->d2h_stream);
  for (int i = 0; i < HOST_MAX_CHUNKS; ++i) {
    if (c->up[i]) cudaEventDestroy(c->up[i]);
    if (c->done[i]) cudaEventDestroy(c->done[i]);
    if (c->back[i]) cudaEventDestroy(c->back[i]);
  }
  if (c->h_total) cudaFreeHost(c->h_total);
  for (int i = 0; i < 9; ++i) cudaFree(c->d_in[i]);
  cudaFree(c->d_off); cudaFree(c->d_pos); cudaFree(c->d_cov); cudaFree(c->d_chi2); cudaFree(c->d_w);
  cudaFree(c->d_ntrk); cudaFree(c->d_niter); cudaFree(c->d_nvtx); cudaFree(c->d_tv); cudaFree(c->d_status);
  cudaFree(c->d_tv8); cudaFree(c->d_vbegin); cudaFree(c->d_packed);
  cudaFree(c->d_ws);
  delete c;
  return PV_OK;
}

int pv_host_ctx_create(pv_host_ctx** out, int max_events, long long max_tracks, const pv_params* params, int n_streams) {
  if (!out) return PV_E_NULL;
  *out = nullptr;
  const int rc = validate(params, nullptr);
  if (rc != PV_OK) return rc;
  if (max_events < 1 || max_tracks < 0 || max_tracks > 0x7fffffffLL || n_streams < 1 || n_streams > 16) return PV_E_SIZE;
  pv_host_ctx* c = new pv_host_ctx();
  c->max_events = max_events; c->max_tracks = max_tracks; c->max_vtx = params->max_vtx_per_event; c->n_streams = n_streams;
  const size_t T = (size_t)(max_tracks > 0 ? max_tracks : 1), E = (size_t)max_events, mv = (size_t)c->max_vtx;
  cudaError_t err = cudaSuccess;
  auto A = [&](void** p, size_t bytes) { if (err == cudaSuccess) err = cudaMalloc(p, bytes); };
  for (int i = 0; i < 9; ++i) A((void**)&c->d_in[i], T * 4);
  A((void**)&c->d_off, (E + 1) * 4);
  A((void**)&c->d_pos, E * mv * 12); A((void**)&c->d_cov, E * mv * 24); A((void**)&c->d_chi2, E * mv * 4);
  A((void**)&c->d_ntrk, E * mv * 4); A((void**)&c->d_niter, E * mv * 4); A((void**)&c->d_nvtx, E * 4);
  A((void**)&c->d_w, T * 4); A((void**)&c->d_tv, T * 4); A((void**)&c->d_status, E * 4);
  A((void**)&c->d_tv8, T); A((void**)&c->d_vbegin, (E + HOST_MAX_CHUNKS + 1) * 4); A((void**)&c->d_packed, E * mv * sizeof(pv_vertex));
  c->ws_stride = (ws_bytes(max_events, max_tracks, params) + 255) / 256 * 256;
  A((void**)&c->d_ws, (size_t)n_streams * c->ws_stride);
  if (err == cudaSuccess) err = cudaMallocHost((void**)&c->h_total, HOST_MAX_CHUNKS * sizeof(int32_t));
  for (int i = 0; i < n_streams && err == cudaSuccess; ++i) {
    cudaStream_t s = nullptr;
    err = cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking);
    if (err == cudaSuccess) c->streams.push_back(s);
  }
  if (err == cudaSuccess) err = cudaStreamCreateWithFlags(&c->vtx_stream, cudaStreamNonBlocking);
  if (err == cudaSuccess) err = cudaStreamCreateWithFlags(&c->h2d_stream, cudaStreamNonBlocking);
  if (err == cudaSuccess) err = cudaStreamCreateWithFlags(&c->d2h_stream, cudaStreamNonBlocking);
  for (int i = 0; i < HOST_MAX_CHUNKS && err == cudaSuccess; ++i) {
    err = cudaEventCreateWithFlags(&c->up[i], cudaEventDisableTiming);
    if (err == cudaSuccess) err = cudaEventCreateWithFlags(&c->done[i], cudaEventDisableTiming);
    if (err == cudaSuccess) err = cudaEventCreateWithFlags(&c->back[i], cudaEventDisableTiming);
  }
  if (err != cudaSuccess) {
    pv_host_ctx_destroy(c);
    return cuda_fail(err, "pv_host_ctx_create");
  }
  *out = c;
  return PV_OK;
}

namespace {

// Both host entries: H2D -> kernels -> D2H per chunk of events, chunks round-robin over the context's streams.
// compact == false: the fixed-stride [E][max_vtx] vertex arrays come back whole (pv_find_host).
// compact == true:  the vertices of a chunk are packed on the device (scan of n_vtx + gather) and only sum(n_vtx)
//                   48-byte records come back, plus int8 vertex indices per track (pv_find_host_compact).
// No early return once work is enqueued: every error path reaches the synchronisation of all streams, so no copy into
// the caller's buffers is in flight when the call returns.
int host_impl(pv_host_ctx* c, const float* const h_in[9], const int32_t* offsets, int n_events, const pv_params* params,
              bool compact, float* vtx_pos, float* vtx_cov, float* vtx_chi2, int32_t* vtx_ntracks, int32_t* vtx_niter,
              pv_vertex* vertices, long long vtx_capacity, int32_t* vtx_begin, int32_t* n_vtx, float* trk_weight,
              int32_t* trk_vertex, int8_t* trk_vertex8, uint32_t* event_status, int n_chunks) {
  if (!c || !offsets || !params || !n_vtx || !event_status) return PV_E_NULL;
  if (compact ? (!vertices || !vtx_begin || vtx_capacity < 0) : (!vtx_pos || !vtx_cov || !vtx_chi2 || !vtx_ntracks || !vtx_niter))
    return PV_E_NULL;
  if (n_events < 0 || n_events > c->max_events) return PV_E_SIZE;
  if (params->max_vtx_per_event != c->max_vtx) return PV_E_PARAM;
  if (compact) vtx_begin[0] = 0;
  if (n_events == 0) return PV_OK;
  // the offsets are the caller's: one pass checks what every later index relies on
  if (offsets[0] != 0) return PV_E_SIZE;
  for (int e = 0; e < n_events; ++e)
    if (offsets[e + 1] < offsets[e]) return PV_E_SIZE;
  const long long T = offsets[n_events];
  if (T > c->max_tracks) return PV_E_SIZE;
  if (T > 0 && (!trk_weight || (compact ? !trk_vertex8 : !trk_vertex))) return PV_E_NULL;
  for (int i = 0; i < 9; ++i)
    if (T > 0 && !h_in[i]) return PV_E_NULL;
  if (n_chunks < 1) n_chunks = 1;
  if (n_chunks > n_events) n_chunks = n_events;
  if (n_chunks > HOST_MAX_CHUNKS) n_chunks = HOST_MAX_CHUNKS;
  const size_t mv = (size_t)c->max_vtx;
  // chunk boundaries by track count (events are contiguous in the SoA arrays).  The chunks ramp up and down in size
  // (1, 2, 4, 8, 8, ..., 8, 4, 2, 1): the first kernels start after a short copy, the last results leave after a short
  // one, and the bulk moves in few large copies (every cudaMemcpyAsync costs ~5 us of PCIe time on top of its bytes).
  std::vector<int> eb(n_chunks + 1, 0);
  eb[n_chunks] = n_events;
  {
    std::vector<long long> wsum(n_chunks + 1, 0);
    for (int k = 0; k < n_chunks; ++k) {
      const int d = k < n_chunks - 1 - k ? k : n_chunks - 1 - k;   // distance to the nearer end
      wsum[k + 1] = wsum[k] + (1LL << (d < 3 ? d : 3));
    }
    for (int k = 1, e = 0; k < n_chunks; ++k) {
      const long long target = (long long)((double)T * (double)wsum[k] / (double)wsum[n_chunks]);
      while (e < n_events && offsets[e] < target) ++e;
      eb[k] = e < eb[k - 1] ? eb[k - 1] : e;
    }
  }
  int rc = PV_OK;
  auto ck = [&](cudaError_t err, const char* what) {
    if (err != cudaSuccess && rc == PV_OK) rc = cuda_fail(err, what);
    return rc == PV_OK;
  };
  int enqueued = 0;
  for (int k = 0; k < n_chunks && rc == PV_OK; ++k) {
    const int e0 = eb[k], e1 = eb[k + 1];
    c->h_total[k] = 0;
    if (e1 <= e0) continue;
    cudaStream_t s = c->streams[k % c->n_streams];
    const size_t t0 = (size_t)offsets[e0], nt = (size_t)offsets[e1] - t0, ne = (size_t)(e1 - e0);
    // inputs: one stream for all chunks (offsets stay absolute: the kernel indexes the un-shifted SoA base pointers)
    if (!ck(cudaMemcpyAsync(c->d_off + e0, offsets + e0, (ne + 1) * 4, cudaMemcpyHostToDevice, c->h2d_stream), "H2D offsets")) break;
    for (int i = 0; i < 9 && nt > 0 && rc == PV_OK; ++i)
      ck(cudaMemcpyAsync(c->d_in[i] + t0, h_in[i] + t0, nt * 4, cudaMemcpyHostToDevice, c->h2d_stream), "H2D tracks");
    if (rc != PV_OK) break;
    if (!ck(cudaEventRecord(c->up[k], c->h2d_stream), "cudaEventRecord")) break;
    // kernels: round-robin over the compute streams (each with its own workspace)
    if (!ck(cudaStreamWaitEvent(s, c->up[k], 0), "cudaStreamWaitEvent")) break;
    const int frc = find_impl(c->d_in[0], c->d_in[1], c->d_in[2], c->d_in[3], c->d_in[4], c->d_in[5], c->d_in[6], c->d_in[7],
                              c->d_in[8], c->d_off + e0, (int)ne, (long long)c->max_tracks, params, c->d_pos + e0 * mv * 3,
                              c->d_cov + e0 * mv * 6, c->d_chi2 + e0 * mv, c->d_ntrk + e0 * mv, c->d_niter + e0 * mv,
                              c->d_nvtx + e0, c->d_w, c->d_tv, c->d_status + e0,
                              c->d_ws + (size_t)(k % c->n_streams) * c->ws_stride, c->ws_stride, s, nullptr, nullptr,
                              compact ? c->d_tv8 : nullptr);
    if (frc != PV_OK) { rc = frc; break; }
    enqueued = k + 1;
    int32_t* vb = c->d_vbegin + e0 + k;
    if (compact) {
      pvk::KArgs ka;
      memset(&ka, 0, sizeof(ka));
      ka.n_events = (int)ne;
      ka.vtx_pos = c->d_pos + e0 * mv * 3; ka.vtx_cov = c->d_cov + e0 * mv * 6; ka.vtx_chi2 = c->d_chi2 + e0 * mv;
      ka.vtx_ntracks = c->d_ntrk + e0 * mv; ka.vtx_niter = c->d_niter + e0 * mv;
      pvk::scan_nvtx_kernel<<<1, 1024, 0, s>>>(c->d_nvtx + e0, (int)ne, vb);
      pvk::pack_vertices_kernel<<<(unsigned)((ne + 7) / 8), 256, 0, s>>>(ka, (int)mv, vb, c->d_packed + e0 * mv);
      if (!ck(cudaGetLastError(), "pack_vertices_kernel")) break;
    }
    if (!ck(cudaEventRecord(c->done[k], s), "cudaEventRecord")) break;
    // results: one stream for all chunks
    cudaStream_t r = c->d2h_stream;
    if (!ck(cudaStreamWaitEvent(r, c->done[k], 0), "cudaStreamWaitEvent")) break;
    if (compact) {
      ck(cudaMemcpyAsync(c->h_total + k, vb + ne, 4, cudaMemcpyDeviceToHost, r), "D2H chunk total");
      ck(cudaEventRecord(c->back[k], r), "cudaEventRecord");
    } else {
      ck(cudaMemcpyAsync(vtx_pos + e0 * mv * 3, c->d_pos + e0 * mv * 3, ne * mv * 12, cudaMemcpyDeviceToHost, r), "D2H");
      ck(cudaMemcpyAsync(vtx_cov + e0 * mv * 6, c->d_cov + e0 * mv * 6, ne * mv * 24, cudaMemcpyDeviceToHost, r), "D2H");
      ck(cudaMemcpyAsync(vtx_chi2 + e0 * mv, c->d_chi2 + e0 * mv, ne * mv * 4, cudaMemcpyDeviceToHost, r), "D2H");
      ck(cudaMemcpyAsync(vtx_ntracks + e0 * mv, c->d_ntrk + e0 * mv, ne * mv * 4, cudaMemcpyDeviceToHost, r), "D2H");
      ck(cudaMemcpyAsync(vtx_niter + e0 * mv, c->d_niter + e0 * mv, ne * mv * 4, cudaMemcpyDeviceToHost, r), "D2H");
    }
    ck(cudaMemcpyAsync(n_vtx + e0, c->d_nvtx + e0, ne * 4, cudaMemcpyDeviceToHost, r), "D2H");
    ck(cudaMemcpyAsync(event_status + e0, c->d_status + e0, ne * 4, cudaMemcpyDeviceToHost, r), "D2H");
    if (nt > 0) {
      ck(cudaMemcpyAsync(trk_weight + t0, c->d_w + t0, nt * 4, cudaMemcpyDeviceToHost, r), "D2H");
      if (compact) ck(cudaMemcpyAsync(trk_vertex8 + t0, c->d_tv8 + t0, nt, cudaMemcpyDeviceToHost, r), "D2H");
      else ck(cudaMemcpyAsync(trk_vertex + t0, c->d_tv + t0, nt * 4, cudaMemcpyDeviceToHost, r), "D2H");
    }
  }
  // second pass (compact): as each chunk finishes, its vertex count is on the host and its packed records are copied
  // to their final place behind those of the chunks before it
  long long base = 0;
  for (int k = 0; compact && k < enqueued && rc == PV_OK; ++k) {
    const int e0 = eb[k], e1 = eb[k + 1];
    if (e1 <= e0) continue;
    if (!ck(cudaEventSynchronize(c->back[k]), "cudaEventSynchronize")) break;
    const long long nv = c->h_total[k];
    if (base + nv > vtx_capacity) { rc = PV_E_SIZE; break; }
    if (nv > 0)
      ck(cudaMemcpyAsync(vertices + base, c->d_packed + (size_t)e0 * mv, (size_t)nv * sizeof(pv_vertex), cudaMemcpyDeviceToHost,
                         c->vtx_stream), "D2H vertices");
    base += nv;
  }
  ck(cudaStreamSynchronize(c->h2d_stream), "cudaStreamSynchronize");
  ck(cudaStreamSynchronize(c->d2h_stream), "cudaStreamSynchronize");
  for (auto s : c->streams) ck(cudaStreamSynchronize(s), "cudaStreamSynchronize");
  ck(cudaStreamSynchronize(c->vtx_stream), "cudaStreamSynchronize");
  if (rc == PV_OK && compact)
    for (int e = 0; e < n_events; ++e) vtx_begin[e + 1] = vtx_begin[e] + n_vtx[e];
  return rc;
}

}  // namespace

int pv_find_host(pv_host_ctx* c,
                 const float* x, const float* y, const float* z, const float* tx, const float* ty,
                 const float* var_x, const float* var_y, const float* var_tx, const float* var_ty,
                 const int32_t* offsets, int n_events, const pv_params* params,
                 float* vtx_pos, float* vtx_cov, float* vtx_chi2, int32_t* vtx_ntracks, int32_t* vtx_niter,
                 int32_t* n_vtx, float* trk_weight, int32_t* trk_vertex, uint32_t* event_status, int n_chunks) {
  const float* h_in[9] = {x, y, z, tx, ty, var_x, var_y, var_tx, var_ty};
  return host_impl(c, h_in, offsets, n_events, params, false, vtx_pos, vtx_cov, vtx_chi2, vtx_ntracks, vtx_niter, nullptr, 0,
                   nullptr, n_vtx, trk_weight, trk_vertex, nullptr, event_status, n_chunks);
}

int pv_find_host_compact(pv_host_ctx* c,
                         const float* x, const float* y, const float* z, const float* tx, const float* ty,
                         const float* var_x, const float* var_y, const float* var_tx, const float* var_ty,
                         const int32_t* offsets, int n_events, const pv_params* params,
                         pv_vertex* vertices, long long vtx_capacity, int32_t* vtx_begin, int32_t* n_vtx,
                         float* trk_weight, int8_t* trk_vertex, uint32_t* event_status, int n_chunks) {
  const float* h_in[9] = {x, y, z, tx, ty, var_x, var_y, var_tx, var_ty};
  return host_impl(c, h_in, offsets, n_events, params, true, nullptr, nullptr, nullptr, nullptr, nullptr, vertices, vtx_capacity,
                   vtx_begin, n_vtx, trk_weight, nullptr, trk_vertex, event_status, n_chunks);
}

int pv_host_register(void* ptr, size_t bytes) {
  if (!ptr) return PV_E_NULL;
  if (bytes == 0) return PV_OK;
  CK(cudaHostRegister(ptr, bytes, cudaHostRegisterDefault));
  return PV_OK;
}

int pv_host_unregister(void* ptr) {
  if (!ptr) return PV_E_NULL;
  CK(cudaHostUnregister(ptr));
  return PV_OK;
}

int pv_last_launch_info(int* n_kernels, int* grid, int* block, int* smem_bytes) {
  if (n_kernels) *n_kernels = g_last_kernels;
  if (grid) *grid = g_last_grid;
  if (block) *block = g_last_block;
  if (smem_bytes) *smem_bytes = g_last_smem;
  return PV_OK;
}

int pv_kernel_timing(int enable) {
  g_timing = enable ? 1 : 0;
  if (!enable) g_ev_valid = false;
  return PV_OK;
}

float pv_kernel_time_ms(void) {
  if (!g_ev_valid || !g_ev[0]) return -1.0f;
  if (cudaEventSynchronize(g_ev[N_KERNELS]) != cudaSuccess) return -1.0f;
  float ms = -1.0f;
  if (cudaEventElapsedTime(&ms, g_ev[0], g_ev[N_KERNELS]) != cudaSuccess) return -1.0f;
  return ms;
}

int pv_kernel_times_ms(float* ms, int n) {
  if (!ms) return PV_E_NULL;
  if (!g_ev_valid || !g_ev[0]) return PV_E_SIZE;
  CK(cudaEventSynchronize(g_ev[N_KERNELS]));
  for (int i = 0; i < n && i < N_KERNELS; ++i) CK(cudaEventElapsedTime(&ms[i], g_ev[i], g_ev[i + 1]));
  return N_KERNELS;
}

const char* pv_error_string(int code) {
  switch (code) {
    case PV_OK: return "ok";
    case PV_E_NULL: return "a required pointer is NULL";
    case PV_E_PARAM: return "invalid parameter";
    case PV_E_WORKSPACE: return "workspace too small";
    case PV_E_CUDA: return "CUDA error (see pv_last_cuda_error)";
    case PV_E_SIZE: return "invalid size or capacity exceeded";
    case PV_E_STATIC_LIMIT: return "batch needs more scratch than the built-in workspace of pv_find_static (PV_STATIC_WORKSPACE_BYTES): split it or use pv_find";
    default: return "unknown error code";
  }
}

const char* pv_last_cuda_error(void) { return g_cuda_err; }

}  // extern "C"

// libipole_b200.so -- host side of the C ABI declared in include/ipole.h: context, argument checks, buffer
// management, batching of rays through the geodesic path buffer, kernel launches.  All arithmetic of the hot path
// is in the kernels (kernels.cuh); the host only sizes, schedules and copies.
#include "../../include/ipole.h"
#include <cuda_runtime.h>
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <mutex>
#include <new>
#include <vector>
#include "kernels.cuh"
#include "stepop.cuh"
#include "gridsweep.cuh"
#include "geo_f32.cuh"
#include "adaptive.cuh"

using namespace ipole;

namespace {

constexpr int N_QUEUES = 8192;
constexpr int PROBE_TARGET = 4096;   // rays of the probe pass
constexpr int PROBE_EPS_FACTOR = 4;  // the probe integrates with 4 eps and predicts 4x its step count

enum LaunchKind { LK_PROBE = 0, LK_GEO = 1, LK_RT = 2, LK_OTHER = 3, LK_LONG = 4,   // LK_LONG: on the side stream
                  LK_OPS = 5, LK_APPLY = 6 };                                          // split transfer: k_stepop, k_apply

struct TimedSpan { cudaEvent_t a, b; int kind; };

}  // namespace

struct ipole_ctx {
  ipole_camera cam_in;
  CamDev cam;          // host copy of the device camera (after k_camera_setup)
  CamDev* d_cam = nullptr;
  Units units;
  cudaStream_t stream = nullptr;
  int last_cuda = 0;
  int device = 0, n_sm = 0;

  int model = MODEL_NONE;
  void* d_model = nullptr;       // AdafParams / SlabParams / GridParams
  unsigned int* d_occ = nullptr; // stencil occupancy bitmap of the grid
  double* d_grid = nullptr;      // cell-major records
  size_t grid_cells = 0;

  uint64_t opt_path_bytes = 0;
  int opt_sort = 1;
  int opt_path_free = 0;         // PAPER.md:43 bidirectional variant
  int opt_occ = 1;               // grid model: plasma-contact range per ray (IPOLE_NO_OCC=1 in the environment turns it off)
  int last_pf = 0;               // the last image was made path-free
  int opt_unpol = 0;             // unpolarized transfer of I alone
  AdafParams adaf_host;          // host copy of the loaded analytic model (k_apply takes it by value)
  // many cameras per call (ipole_make_images_cameras): device arrays of n_mc cameras, null outside such a call
  CamDev* d_mc_cams = nullptr; Units* d_mc_units = nullptr; double* d_mc_nu3 = nullptr; double* d_mc_scale = nullptr;
  int mc_cap = 0; int n_mc = 0; int64_t mc_rays_per_cam = 0;
  int occ_geo_mc = 0, occ_op_mc = 0, occ_geo_occ_mc = 0, occ_group_mc = 0;
  int opt_geo_fp32 = 0;          // FP32 study (geo_f32.cuh): geodesics in single precision, transfer in FP64
  int occ_geo_f32 = 0;
  int opt_group = 1;             // grid model: transfer with warp-level scheduling (k_transfer_group)
  int occ_group = 0;
  int opt_tight = 1;             // sorted rays: path slots sized batch by batch from the predicted step counts
  int32_t* d_retry = nullptr;    // rays that outgrew their batch's slots (retried with the global S_cap)
  int opt_split = 1;             // stored path, analytic flow: transfer as k_stepop + k_apply (stepop.cuh)
  double* d_ops = nullptr; size_t ops_bytes = 0;   // operator records of one batch
  int32_t* d_irr = nullptr;      // slots of the rays k_stepop leaves to k_transfer
  int32_t *d_rank_pos = nullptr, *d_rank_slot = nullptr;   // k_rank_window: operator-record places of a batch's slots, by position in the order
  int opt_rank = 1;
  int occ_op = 0, occ_ap = 0, occ_ap_edf = 0, occ_ap_unpol = 0, occ_gridop = 0, occ_gridapply = 0, occ_ap_wide = 0;
  EdfDev edf = {0, 128, 3.5, 0.0, nullptr, nullptr};   // electron distribution of the coefficient step (ipole_set_edf); kind 0: thermal fits
  double4* d_edf_nodes = nullptr; double* d_edf_lnnorm = nullptr;
  int occ_unpol[4][2] = {{0, 0}, {0, 0}, {0, 0}, {0, 0}};
  double* d_endp = nullptr; int64_t endp_cap = 0;   // end points of the backward passes, [rays][8]
  long long* d_sum = nullptr;    // forward-step total of the path-free variant
  void* d_sweep_models = nullptr; Units* d_sweep_units = nullptr;   // model sweep: SWEEP_MAX_MODELS entries each (main stream)
  void* d_sweep_models_side = nullptr; Units* d_sweep_units_side = nullptr;   // the same for the long-ray passes on the side stream
  GridParams grid_host; double grid_M_unit = 0.0;   // host copy of the loaded grid model (units are re-derived when the camera's mass changes)
  double* d_sweep_out = nullptr; size_t sweep_out_doubles = 0;            // staging for host outputs of a sweep
  int occ_sweep[4] = {0, 0, 0, 0};
  unsigned char* d_ada = nullptr; size_t ada_bytes = 0;   // adaptive ray tracing: staging planes, list, state, flags
  cudaEvent_t ev_ada0 = nullptr, ev_ada1 = nullptr;

  double* d_path = nullptr; size_t path_bytes = 0;
  double* d_path_long = nullptr; size_t path_long_bytes = 0;   // slots of max_steps for the long-ray passes
  int32_t* d_nsteps_long = nullptr;                             // step counts written by the long-ray passes
  cudaStream_t side = nullptr;                                  // long-ray passes overlap the bulk batches here
  cudaStream_t qstream = nullptr;                               // 4-byte read-backs that must not wait for `side`
  cudaEvent_t ev_geo = nullptr, ev_side = nullptr;
  // bulk batches alternate between `stream` and `lane2`, each with its own half of the path and operator buffers: the
  // persistent kernels of one batch drain while those of the next fill the GPU
  cudaStream_t lane2 = nullptr;
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
  int opt_overlap = 1;
  // retry level on the side stream: its own slots, so that it starts as soon as the last geodesic kernel of the bulk has
  // listed the rays, beside the last transfer kernels, instead of after them (one ray of S_cap steps is ~30 ms of latency)
  cudaEvent_t ev_lastgeo[2] = {nullptr, nullptr};
  double* d_retry_buf = nullptr; size_t retry_buf_bytes = 0;
  double* d_ops_long = nullptr; size_t ops_long_bytes = 0;   // operator records of a long-ray pass through the split kernels (eDF, cameras)
  int opt_side_retry = 1;
  int64_t ray_cap = 0;           // capacity of the per-ray buffers below
  int32_t *d_nsteps = nullptr, *d_nturn = nullptr, *d_order = nullptr, *d_key = nullptr, *d_long = nullptr;
  int2* d_srange = nullptr;      // grid model: per ray, the steps that may cross plasma (k_geodesic<true>)
  double* d_out = nullptr;       // staging for host outputs: 6 planes of ray_cap
  int64_t* d_pixels = nullptr; int64_t pixels_cap = 0;
  int32_t* d_probe = nullptr; int64_t probe_cap = 0;
  unsigned long long* d_queues = nullptr;
  unsigned int* d_hist = nullptr;
  int* d_small = nullptr;        // [0] long_count, [1] probe max, [2] adaptive list length, [4] / [6] irregular rays of a batch (lane 0 / 1), [5] retries
  ReducePartial* d_part = nullptr;
  ReduceOut* d_red = nullptr;

  // Plan of the last full-image call (ipole_set_plan_reuse): what the host had to READ BACK from the device to schedule
  // it -- S_cap and the bin populations of the sort (the ray order itself stays in d_order), the rays that outgrew their
  // slots and the rays longer than S_cap.  All of it depends on the camera and the scheduling options alone, not on the
  // plasma, so a call with the same key replays it without a single host-device synchronisation.
  struct PlanCache {
    bool valid = false;
    ipole_camera cam; int64_t n = 0; size_t budget = 0; unsigned flags = 0;
    int cap = 0, bin_width = 1; std::vector<unsigned int> bin_prefix;
    int n_long = 0, n_retry = 0;
    int32_t* d_long = nullptr; int32_t* d_retry = nullptr; int long_cap = 0, retry_cap = 0;   // the two lists as that call left them
  } plan_cache;
  int opt_plan_reuse = 1;
  int opt_lowlat = 1;            // under-filled launches: kernels built for single-ray latency (IPOLE_NO_LOWLAT=1 turns it off)

  double* totals_scratch = nullptr;   // device address of g_totals_scratch on this context's device (ipole_image_totals_static)
  int totals_scratch_err = 0;         // cudaError_t of the look-up, if it failed

  std::vector<TimedSpan> spans; size_t spans_used = 0;
  bool have_image = false;
  int64_t last_n = 0;
  ipole_stats stats;
  int occ_geo = 0, occ_geo_occ = 0, occ_rt[4] = {0, 0, 0, 0}, occ_pf[4][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
};

namespace {

// IPOLE_DEBUG=1 in the environment: the failing call's line and CUDA's text for the error go to stderr
static void report_cuda_failure(int e, int line) {
  static const bool on = [] { const char* v = std::getenv("IPOLE_DEBUG"); return v && v[0] == '1'; }();
  if (on) std::fprintf(stderr, "ipole: CUDA error %d (%s) at ipole_b200.cu:%d\n", e, cudaGetErrorString((cudaError_t)e), line);
}

#define CK(call)                                                        \
  do {                                                                  \
    cudaError_t e_ = (call);                                            \
    if (e_ != cudaSuccess) { c->last_cuda = (int)e_; report_cuda_failure((int)e_, __LINE__); return IPOLE_ECUDA; } \
  } while (0)

bool is_device_ptr(const void* p) {
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

int check_camera(const ipole_camera* k) {
  if (!(k->spin >= 0.0 && k->spin < 1.0)) return IPOLE_EINVAL;
  if (!(k->inclination_deg > 0.0 && k->inclination_deg < 180.0)) return IPOLE_EINVAL;
  if (!(k->r_cam > 0.0) || !(k->fov > 0.0) || k->nx <= 0 || k->ny <= 0 || !(k->freq_hz > 0.0)) return IPOLE_EINVAL;
  if (k->eps < 0.0 || k->r_esc < 0.0 || k->stop_factor < 0.0 || k->max_steps < 0 || k->hslope < 0.0) return IPOLE_EINVAL;
  if (k->mbh_msun < 0.0 || k->dsource_pc < 0.0) return IPOLE_EINVAL;
  if ((int64_t)k->nx * k->ny > 2147483647LL) return IPOLE_EINVAL;
  return IPOLE_OK;
}

// host part of a camera: what k_camera_setup starts from, and the units that follow from mass, distance and frequency
void fill_camera(const ipole_camera* k, CamDev& C, CameraSetupArgs& a, Units& u) {
  std::memset(&C, 0, sizeof C);
  C.G.a = k->spin;
  C.G.hslope = k->hslope > 0.0 ? k->hslope : 1.0;
  C.G.mass = k->flat_metric ? 0.0 : 1.0;
  C.G.h_is_one = (C.G.hslope == 1.0);
  C.r_cam = k->r_cam;
  C.nx = k->nx; C.ny = k->ny;
  C.pix = k->fov / k->nx;
  C.eps = k->eps > 0.0 ? k->eps : 0.01;
  C.max_steps = k->max_steps > 0 ? k->max_steps : 50000;
  a.inclination_deg = k->inclination_deg;
  a.r_esc = k->r_esc > 0.0 ? k->r_esc : k->r_cam;
  const double stop = k->stop_factor > 0.0 ? k->stop_factor : 1.05;
  a.r_in = k->flat_metric ? 1e-3 : stop * (1.0 + std::sqrt(1.0 - k->spin * k->spin));
  const double M = (k->mbh_msun > 0.0 ? k->mbh_msun : 4.1e6) * IP_MSUN;
  u.nu_obs = k->freq_hz;
  u.L_unit = IP_GNEWT * M / (IP_CL * IP_CL);
  u.D_cm = (k->dsource_pc > 0.0 ? k->dsource_pc : 8000.0) * IP_PC;
  u.dl_unit = u.L_unit / u.nu_obs;
}

int apply_camera(ipole_ctx* c, const ipole_camera* k) {
  CamDev C;
  CameraSetupArgs a;
  Units un;
  fill_camera(k, C, a, un);
  CK(cudaMemcpyAsync(c->d_cam, &C, sizeof C, cudaMemcpyHostToDevice, c->stream));
  k_camera_setup<<<1, 32, 0, c->stream>>>(c->d_cam, a);
  CK(cudaGetLastError());
  CK(cudaMemcpyAsync(&c->cam, c->d_cam, sizeof C, cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  c->cam_in = *k;
  c->units = un;
  c->have_image = false;
  return IPOLE_OK;
}

int ensure_rays(ipole_ctx* c, int64_t n) {
  if (n <= c->ray_cap) return IPOLE_OK;
  c->plan_cache.valid = false;
  cudaFree(c->d_nsteps); cudaFree(c->d_nturn); cudaFree(c->d_order); cudaFree(c->d_key); cudaFree(c->d_long); cudaFree(c->d_out);
  cudaFree(c->d_nsteps_long); cudaFree(c->d_srange); c->d_srange = nullptr; cudaFree(c->d_irr); cudaFree(c->d_retry); c->d_retry = nullptr; cudaFree(c->d_rank_pos); cudaFree(c->d_rank_slot); c->d_rank_pos = c->d_rank_slot = nullptr;
  c->d_nsteps = c->d_nturn = c->d_order = c->d_key = c->d_long = c->d_nsteps_long = c->d_irr = nullptr; c->d_out = nullptr; c->ray_cap = 0;
  CK(cudaMalloc(&c->d_nsteps, n * sizeof(int32_t)));
  CK(cudaMalloc(&c->d_nturn, n * sizeof(int32_t)));
  CK(cudaMalloc(&c->d_order, n * sizeof(int32_t)));
  CK(cudaMalloc(&c->d_key, n * sizeof(int32_t)));
  CK(cudaMalloc(&c->d_long, n * sizeof(int32_t)));
  CK(cudaMalloc(&c->d_nsteps_long, n * sizeof(int32_t)));
  CK(cudaMalloc(&c->d_srange, n * sizeof(int2)));
  CK(cudaMalloc(&c->d_rank_pos, 2 * n * sizeof(int32_t)));    // second half: the retry level on the side stream
  CK(cudaMalloc(&c->d_rank_slot, 2 * n * sizeof(int32_t)));
  CK(cudaMalloc(&c->d_irr, 3 * n * sizeof(int32_t)));   // one list per lane, one for the retry level on the side stream
  CK(cudaMalloc(&c->d_retry, n * sizeof(int32_t)));
  CK(cudaMalloc(&c->d_out, 6 * n * sizeof(double)));
  c->ray_cap = n;
  return IPOLE_OK;
}

int ensure_path(ipole_ctx* c, size_t bytes) {
  if (bytes <= c->path_bytes) return IPOLE_OK;
  cudaFree(c->d_path); c->d_path = nullptr; c->path_bytes = 0;
  cudaError_t e = cudaMalloc(&c->d_path, bytes);
  if (e != cudaSuccess) { c->last_cuda = (int)e; cudaGetLastError(); return IPOLE_ENOMEM; }
  c->path_bytes = bytes;
  return IPOLE_OK;
}

int ensure_ops(ipole_ctx* c, size_t bytes) {
  if (bytes <= c->ops_bytes) return IPOLE_OK;
  cudaFree(c->d_ops); c->d_ops = nullptr; c->ops_bytes = 0;
  cudaError_t e = cudaMalloc(&c->d_ops, bytes);
  if (e != cudaSuccess) { c->last_cuda = (int)e; cudaGetLastError(); return IPOLE_ENOMEM; }
  c->ops_bytes = bytes;
  return IPOLE_OK;
}

int ensure_retry_buf(ipole_ctx* c, size_t bytes) {
  if (bytes <= c->retry_buf_bytes) return IPOLE_OK;
  cudaFree(c->d_retry_buf); c->d_retry_buf = nullptr; c->retry_buf_bytes = 0;
  cudaError_t e = cudaMalloc(&c->d_retry_buf, bytes);
  if (e != cudaSuccess) { c->last_cuda = (int)e; cudaGetLastError(); return IPOLE_ENOMEM; }
  c->retry_buf_bytes = bytes;
  return IPOLE_OK;
}

int ensure_ops_long(ipole_ctx* c, size_t bytes) {
  if (bytes <= c->ops_long_bytes) return IPOLE_OK;
  cudaFree(c->d_ops_long); c->d_ops_long = nullptr; c->ops_long_bytes = 0;
  cudaError_t e = cudaMalloc(&c->d_ops_long, bytes);
  if (e != cudaSuccess) { c->last_cuda = (int)e; cudaGetLastError(); return IPOLE_ENOMEM; }
  c->ops_long_bytes = bytes;
  return IPOLE_OK;
}

int ensure_path_long(ipole_ctx* c, size_t bytes) {
  if (bytes <= c->path_long_bytes) return IPOLE_OK;
  cudaFree(c->d_path_long); c->d_path_long = nullptr; c->path_long_bytes = 0;
  cudaError_t e = cudaMalloc(&c->d_path_long, bytes);
  if (e != cudaSuccess) { c->last_cuda = (int)e; cudaGetLastError(); return IPOLE_ENOMEM; }
  c->path_long_bytes = bytes;
  return IPOLE_OK;
}

size_t path_budget(ipole_ctx* c) {
  if (c->opt_path_bytes) return (size_t)c->opt_path_bytes;
  if (const char* e = std::getenv("IPOLE_PATH_GIB")) { const double gib = std::atof(e); if (gib > 0.0) return (size_t)(gib * 1073741824.0); }
  size_t fr = 0, tot = 0;
  cudaMemGetInfo(&fr, &tot);
  fr += c->path_bytes + c->path_long_bytes + c->ops_bytes + c->retry_buf_bytes + c->ops_long_bytes;  // what we already hold counts as available
  size_t b = (size_t)(0.5 * (double)fr);
  const size_t cap = (size_t)96 << 30;
  return std::min(b, cap);
}

int span_begin(ipole_ctx* c, int kind, cudaStream_t st) {
  if (c->spans_used == c->spans.size()) {
    TimedSpan s; s.kind = kind;
    if (cudaEventCreate(&s.a) != cudaSuccess || cudaEventCreate(&s.b) != cudaSuccess) return -1;
    c->spans.push_back(s);
  }
  TimedSpan* s = &c->spans[c->spans_used++];
  s->kind = kind;
  cudaEventRecord(s->a, st);
  return (int)(c->spans_used - 1);
}
void span_end(ipole_ctx* c, int s, cudaStream_t st) {
  if (s >= 0) cudaEventRecord(c->spans[s].b, st);
}

// `reserve` blocks are left out of a full grid so that the few blocks of a long-ray pass on the side stream find a
// free slot at once instead of waiting for a (persistent) bulk block to exit
int grid_for(ipole_ctx* c, int occ, int threads, int64_t rays, int reserve = 0) {
  const int64_t full = std::max<int64_t>(1, (int64_t)c->n_sm * std::max(occ, 1) - reserve);
  const int64_t need = (rays + threads - 1) / threads;
  return (int)std::max<int64_t>(1, std::min(full, need));
}

int launch_geodesic(ipole_ctx* c, GeoArgs& a, int kind, int64_t rays, cudaStream_t st, int reserve = 0) {
  CK(cudaGetLastError());     // (an error left behind by an unchecked call is reported here, not as this launch's)
  const int s = span_begin(c, kind, st);
  if (c->opt_geo_fp32 && kind != LK_PROBE && !c->n_mc && !a.grid && !a.endp) {
    k_geodesic_f32<<<grid_for(c, c->occ_geo_f32, IPOLE_GEO_THREADS, rays, reserve), IPOLE_GEO_THREADS, 0, st>>>(a);
  } else if (c->n_mc) {
    a.cams = c->d_mc_cams; a.rays_per_cam = c->mc_rays_per_cam;
    if (a.grid) k_geodesic<true, true><<<grid_for(c, c->occ_geo_occ_mc, IPOLE_GEO_THREADS, rays, reserve), IPOLE_GEO_THREADS, 0, st>>>(a);
    else k_geodesic<false, true><<<grid_for(c, c->occ_geo_mc, IPOLE_GEO_THREADS, rays, reserve), IPOLE_GEO_THREADS, 0, st>>>(a);
  } else {
    // a launch that leaves the GPU part empty whatever the kernel: the build that is fastest for a lone ray (kernels.cuh, LOWLAT)
    const bool lowlat = c->opt_lowlat && rays <= (int64_t)c->n_sm * IPOLE_GEO_THREADS * 2;
    if (a.grid) {
      if (lowlat) k_geodesic<true, false, true><<<grid_for(c, 2, IPOLE_GEO_THREADS, rays, reserve), IPOLE_GEO_THREADS, 0, st>>>(a);
      else k_geodesic<true><<<grid_for(c, c->occ_geo_occ, IPOLE_GEO_THREADS, rays, reserve), IPOLE_GEO_THREADS, 0, st>>>(a);
    } else {
      if (lowlat) k_geodesic<false, false, true><<<grid_for(c, 2, IPOLE_GEO_THREADS, rays, reserve), IPOLE_GEO_THREADS, 0, st>>>(a);
      else k_geodesic<false><<<grid_for(c, c->occ_geo, IPOLE_GEO_THREADS, rays, reserve), IPOLE_GEO_THREADS, 0, st>>>(a);
    }
  }
  span_end(c, s, st);
  c->stats.n_launches++;
  CK(cudaGetLastError());
  return IPOLE_OK;
}

// model sweep (ipole_make_images_adaf): n_models parameter sets walked over the same stored paths
struct Sweep {
  int n_models;                 // all of them
  const void* lane_tab;         // host: AdafParams[n_models] or GridScales[n_models]
  size_t lane_bytes;
  const Units* units;           // host
  size_t out_stride;            // doubles between the planes of consecutive models
};

template <int PF>
void launch_transfer_model(int model, int g, cudaStream_t st, const RtArgs& a) {
  if (model == MODEL_ADAF) k_transfer<MODEL_ADAF, PF><<<g, IPOLE_RT_THREADS, 0, st>>>(a);
  else if (model == MODEL_SLAB) k_transfer<MODEL_SLAB, PF><<<g, IPOLE_RT_THREADS, 0, st>>>(a);
  else k_transfer<MODEL_GRID, PF><<<g, IPOLE_RT_THREADS, 0, st>>>(a);
}

int launch_transfer_sweep_split(ipole_ctx* c, const RtArgs& a, int64_t rays, cudaStream_t st, const Sweep* sw);
int launch_transfer_gridsweep_split(ipole_ctx* c, const RtArgs& a, int64_t rays, cudaStream_t st, const Sweep* sw);

// pf: 0 stored path, 1 path-free with eps <= 0.04, 2 path-free with any eps
int launch_transfer(ipole_ctx* c, RtArgs& a, int kind, int64_t rays, cudaStream_t st, int reserve = 0, int pf = 0,
                    const Sweep* sw = nullptr) {
  if (c->opt_unpol && !sw) {
    const int s = span_begin(c, kind, st);
    const int g = grid_for(c, c->occ_unpol[c->model][0], IPOLE_RT_THREADS, rays, reserve);
    if (c->model == MODEL_ADAF) k_transfer_unpol<MODEL_ADAF, false><<<g, IPOLE_RT_THREADS, 0, st>>>(a);
    else if (c->model == MODEL_SLAB) k_transfer_unpol<MODEL_SLAB, false><<<g, IPOLE_RT_THREADS, 0, st>>>(a);
    else k_transfer_unpol<MODEL_GRID, false><<<g, IPOLE_RT_THREADS, 0, st>>>(a);
    span_end(c, s, st);
    c->stats.n_launches++;
    CK(cudaGetLastError());
    return IPOLE_OK;
  }
  if (sw) {
    // chunks of SWEEP_MAX_MODELS parameter sets; the parameter tables are re-sent per chunk on the launching stream
    // (stream order keeps a table alive until the kernel that reads it has finished).  The main stream and the side
    // stream (long-ray passes) each have their own tables: they run concurrently.
    // analytic flow, bulk batches: the operator records are the same for every parameter set -- k_stepop once, k_apply
    // per set (1: a ray with a step outside the split's reach is in the batch; the single kernel below takes it all)
    // (unpolarized: the same records serve I alone; worth k_stepop's full geometry from a few parameter sets on)
    if (c->model == MODEL_ADAF && c->opt_split && (!c->opt_unpol || sw->n_models >= 4) && st != c->side && a.path == c->d_path && c->d_ops) {
      const int r = launch_transfer_sweep_split(c, a, rays, st, sw);
      if (r != 1) return r;
    }
    // grid model, bulk batches: gather, flow, tetrad and leg transport once per call, coefficients and Stokes update per set
    if (c->model == MODEL_GRID && c->opt_split && !c->opt_unpol && st != c->side && a.path == c->d_path && c->d_ops && a.srange)
      return launch_transfer_gridsweep_split(c, a, rays, st, sw);
    void* tab_models = (st == c->side) ? c->d_sweep_models_side : c->d_sweep_models;
    Units* tab_units = (st == c->side) ? c->d_sweep_units_side : c->d_sweep_units;
    RtArgs t = a;
    double* planes[6] = {a.I, a.Q, a.U, a.V, a.tau, a.tauF};
    for (int m0 = 0; m0 < sw->n_models; m0 += SWEEP_MAX_MODELS) {
      const int mc = std::min(SWEEP_MAX_MODELS, sw->n_models - m0);
      const int s = span_begin(c, kind, st);
      CK(cudaMemcpyAsync(tab_models, (const char*)sw->lane_tab + (size_t)m0 * sw->lane_bytes, mc * sw->lane_bytes,
                         cudaMemcpyHostToDevice, st));
      CK(cudaMemcpyAsync(tab_units, sw->units + m0, mc * sizeof(Units), cudaMemcpyHostToDevice, st));
      t.lane_tab = tab_models; t.units_arr = tab_units; t.n_models = mc; t.out_stride = sw->out_stride;
      t.I = planes[0] + (size_t)m0 * sw->out_stride; t.Q = planes[1] + (size_t)m0 * sw->out_stride;
      t.U = planes[2] + (size_t)m0 * sw->out_stride; t.V = planes[3] + (size_t)m0 * sw->out_stride;
      t.tau = planes[4] ? planes[4] + (size_t)m0 * sw->out_stride : nullptr;
      t.tauF = planes[5] ? planes[5] + (size_t)m0 * sw->out_stride : nullptr;
      CK(cudaMemsetAsync(t.queue, 0, sizeof(unsigned long long), st));
      const int g = grid_for(c, c->opt_unpol ? c->occ_unpol[c->model][1] : c->occ_sweep[c->model], IPOLE_RT_THREADS, rays * mc, reserve);
      if (c->opt_unpol) {
        if (c->model == MODEL_ADAF) k_transfer_unpol<MODEL_ADAF, true><<<g, IPOLE_RT_THREADS, 0, st>>>(t);
        else k_transfer_unpol<MODEL_GRID, true><<<g, IPOLE_RT_THREADS, 0, st>>>(t);
      } else if (c->model == MODEL_ADAF) k_transfer<MODEL_ADAF, 0, true><<<g, IPOLE_RT_THREADS, 0, st>>>(t);
      else k_transfer<MODEL_GRID, 0, true><<<g, IPOLE_RT_THREADS, 0, st>>>(t);
      span_end(c, s, st);
      c->stats.n_launches++;
      CK(cudaGetLastError());
    }
    return IPOLE_OK;
  }
  const int s = span_begin(c, kind, st);
  if (pf == 0 && c->model == MODEL_GRID && (c->opt_group || c->n_mc) && !a.slots) {
    // warp-level scheduling: one warp per 32 consecutive rays (kernels.cuh, k_transfer_group)
    const int gg = grid_for(c, c->occ_group, IPOLE_RT_THREADS / 32, (rays + 31) / 32, reserve);
    if (c->opt_rank && a.srange && rays > 32) {
      // the 32 rays of a group walk in lockstep from the group's first plasma contact: windows of 1024 slots are ranked by
      // each ray's contact range, known since k_geodesic<true> (the side stream has its own half of the two arrays)
      const size_t off = (st == c->side) ? (size_t)c->ray_cap : 0;
      RankArgs r = {a.base, a.count, a.count_dev, a.order, a.nsteps, c->d_rank_pos + off, c->d_rank_slot + off, a.srange};
      k_rank_window<<<(unsigned)((rays + RANK_WINDOW - 1) / RANK_WINDOW), RANK_WINDOW, 0, st>>>(r);
      c->stats.n_launches++;
      a.rank_slot = c->d_rank_slot + off;
    }
    if (c->n_mc) {   // many cameras per call: the lanes take frequency, units and camera legs from their ray's camera
      a.cams = c->d_mc_cams; a.units_arr = c->d_mc_units; a.rays_per_cam = c->mc_rays_per_cam;
      k_transfer_group<MODEL_GRID, true><<<grid_for(c, c->occ_group_mc, IPOLE_RT_THREADS / 32, (rays + 31) / 32, reserve), IPOLE_RT_THREADS, 0, st>>>(a);
    } else k_transfer_group<MODEL_GRID><<<gg, IPOLE_RT_THREADS, 0, st>>>(a);
    span_end(c, s, st);
    c->stats.n_launches++;
    CK(cudaGetLastError());
    return IPOLE_OK;
  }
  const int g = grid_for(c, pf ? c->occ_pf[c->model][pf] : c->occ_rt[c->model], IPOLE_RT_THREADS, rays, reserve);
  if (pf == 0) launch_transfer_model<0>(c->model, g, st, a);
  else if (pf == 1) launch_transfer_model<1>(c->model, g, st, a);
  else launch_transfer_model<2>(c->model, g, st, a);
  span_end(c, s, st);
  c->stats.n_launches++;
  CK(cudaGetLastError());
  return IPOLE_OK;
}

// split transfer of one batch (stepop.cuh): k_stepop over the steps, k_apply over the rays, then k_transfer for the
// rays k_stepop could not express (listed on the device; usually none)
int launch_transfer_split(ipole_ctx* c, const RtArgs& a, int64_t rays, cudaStream_t st, int reserve, double* ops, int lane) {
  // lane 0 / 1: the bulk lanes; 2: the retry level on the side stream (its times count as ms_long)
  static const int irr_slot[3] = {4, 6, 3};
  int* irr_count = c->d_small + irr_slot[lane];
  int32_t* irr = c->d_irr + (size_t)lane * c->ray_cap;
  const bool on_side = lane == 2;
  CK(cudaMemsetAsync(irr_count, 0, sizeof(int), st));
  OpArgs o;
  std::memset(&o, 0, sizeof o);
  o.cam = a.cam; o.units = a.units; o.model = a.model; o.cap = a.cap; o.base = a.base; o.count = a.count; o.order = a.order;
  o.count_dev = a.count_dev; o.path = a.path; o.nsteps = a.nsteps; o.queue = a.queue; o.ops = ops; o.irr_slots = irr; o.irr_count = irr_count; o.test_irregular = (c->opt_split == 2);
  const bool rank = c->opt_rank && rays > 32;
  int32_t* rank_pos = c->d_rank_pos + (on_side ? c->ray_cap : 0);     // (the side-stream retry indexes from 0 like a bulk batch)
  int32_t* rank_slot = c->d_rank_slot + (on_side ? c->ray_cap : 0);
  if (rank) {
    RankArgs r = {a.base, a.count, a.count_dev, a.order, a.nsteps, rank_pos, rank_slot, nullptr};
    const int s = span_begin(c, on_side ? LK_LONG : LK_OPS, st);
    k_rank_window<<<(unsigned)((rays + RANK_WINDOW - 1) / RANK_WINDOW), RANK_WINDOW, 0, st>>>(r);
    span_end(c, s, st);
    c->stats.n_launches++;
    CK(cudaGetLastError());
    o.pos = rank_pos;
  }
  {
    const int s = span_begin(c, on_side ? LK_LONG : LK_OPS, st);
    // one warp per ray at a time
    if (c->n_mc) {
      o.cams = c->d_mc_cams; o.units_arr = c->d_mc_units; o.rays_per_cam = c->mc_rays_per_cam;
      k_stepop<MODEL_ADAF, true><<<grid_for(c, c->occ_op_mc, IPOLE_OP_THREADS / 32, rays, reserve), IPOLE_OP_THREADS, 0, st>>>(o);
    } else {
      const int g = grid_for(c, c->occ_op, IPOLE_OP_THREADS / 32, rays, reserve);
      k_stepop<MODEL_ADAF><<<g, IPOLE_OP_THREADS, 0, st>>>(o);
    }
    span_end(c, s, st);
    c->stats.n_launches++;
    CK(cudaGetLastError());
  }
  ApArgs p;
  std::memset(&p, 0, sizeof p);
  p.nu3 = a.units.nu_obs * a.units.nu_obs * a.units.nu_obs;
  p.model = c->adaf_host;
  p.cap = a.cap; p.base = a.base; p.count = a.count; p.count_dev = a.count_dev; p.order = a.order; p.ops = ops; p.nsteps = a.nsteps;
  p.queue = a.queue + 1;
  if (rank) p.slot = rank_slot;
  p.I = a.I; p.Q = a.Q; p.U = a.U; p.V = a.V; p.tau = a.tau; p.tauF = a.tauF;
  {
    const int s = span_begin(c, on_side ? LK_LONG : LK_APPLY, st);
    const int g = grid_for(c, c->occ_ap, IPOLE_AP_THREADS / 32, (rays + 31) / 32, reserve);   // one warp per 32 rays
    p.edf = c->edf;
    if (c->n_mc) { p.nu3_arr = c->d_mc_nu3; p.rays_per_cam = c->mc_rays_per_cam; }
    if (c->edf.kind != 0) k_apply<true><<<grid_for(c, c->occ_ap_edf, IPOLE_AP_THREADS / 32, (rays + 31) / 32, reserve), IPOLE_AP_THREADS, (size_t)c->edf.n_nodes * sizeof(double4), st>>>(p);
    else if (c->opt_lowlat && rays <= 1024)      // a handful of rays (long-ray and retry passes): a warp per ray (stepop.cuh)
      k_apply_wide<32><<<grid_for(c, c->occ_ap_wide, IPOLE_AP_THREADS / 32, rays, reserve), IPOLE_AP_THREADS, 0, st>>>(p);
    else if (c->opt_lowlat && rays <= (int64_t)c->n_sm * IPOLE_AP_THREADS * 2)   // the launch cannot fill the GPU: 8 lanes per ray
      k_apply_wide<8><<<grid_for(c, c->occ_ap_wide, IPOLE_AP_THREADS / 32, (rays + 3) / 4, reserve), IPOLE_AP_THREADS, 0, st>>>(p);
    else k_apply<false><<<g, IPOLE_AP_THREADS, 0, st>>>(p);
    span_end(c, s, st);
    c->stats.n_launches++;
    CK(cudaGetLastError());
  }
  RtArgs t = a;
  t.queue = a.queue + 2; t.count_dev = irr_count; t.slots = irr;
  {
    const int s = span_begin(c, on_side ? LK_LONG : LK_RT, st);
    k_transfer<MODEL_ADAF, 0><<<std::max(1, c->n_sm / 8), IPOLE_RT_THREADS, 0, st>>>(t);
    span_end(c, s, st);
    c->stats.n_launches++;
    CK(cudaGetLastError());
  }
  return IPOLE_OK;
}

// Model sweep of the analytic flow through the split kernels (ipole_make_images_adaf): everything k_stepop computes --
// metric, generator, flow, field direction, tetrad, leg projections -- is the same for every parameter set, so it runs ONCE
// per batch; k_apply then walks the records once per set (work item = ray group x set, the sets of a group back to back so
// that its records come from L2), in chunks of SWEEP_MAX_MODELS sets whose tables are re-sent on the stream.
// Returns 1 (nothing written that matters) when k_stepop met an irregular ray: the caller runs the single sweep kernel.
int launch_transfer_sweep_split(ipole_ctx* c, const RtArgs& a, int64_t rays, cudaStream_t st, const Sweep* sw) {
  int* irr_count = c->d_small + 4;
  CK(cudaMemsetAsync(irr_count, 0, sizeof(int), st));
  void* tab_models = c->d_sweep_models;
  Units* tab_units = c->d_sweep_units;
  auto send_tables = [&](int m0, int mc) -> int {
    CK(cudaMemcpyAsync(tab_models, (const char*)sw->lane_tab + (size_t)m0 * sw->lane_bytes, mc * sw->lane_bytes, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(tab_units, sw->units + m0, mc * sizeof(Units), cudaMemcpyHostToDevice, st));
    return IPOLE_OK;
  };
  int rc;
  const int mc0 = std::min(SWEEP_MAX_MODELS, sw->n_models);
  if ((rc = send_tables(0, mc0)) != IPOLE_OK) return rc;
  OpArgs o;
  std::memset(&o, 0, sizeof o);
  o.cam = a.cam; o.units = a.units; o.model = tab_models;   // (any set: the flow's geometry needs the ISCO radius only)
  o.cap = a.cap; o.base = a.base; o.count = a.count; o.order = a.order;
  o.path = a.path; o.nsteps = a.nsteps; o.queue = a.queue; o.ops = c->d_ops; o.irr_slots = c->d_irr; o.irr_count = irr_count;
  o.test_irregular = (c->opt_split == 2);
  const bool rank = c->opt_rank && rays > 32;
  if (rank) {
    RankArgs r = {a.base, a.count, nullptr, a.order, a.nsteps, c->d_rank_pos, c->d_rank_slot, nullptr};
    const int s = span_begin(c, LK_OPS, st);
    k_rank_window<<<(unsigned)((rays + RANK_WINDOW - 1) / RANK_WINDOW), RANK_WINDOW, 0, st>>>(r);
    span_end(c, s, st);
    c->stats.n_launches++;
    o.pos = c->d_rank_pos;
  }
  {
    const int s = span_begin(c, LK_OPS, st);
    k_stepop<MODEL_ADAF><<<grid_for(c, c->occ_op, IPOLE_OP_THREADS / 32, rays), IPOLE_OP_THREADS, 0, st>>>(o);
    span_end(c, s, st);
    c->stats.n_launches++;
    CK(cudaGetLastError());
  }
  int n_irr = 0;
  CK(cudaMemcpyAsync(&n_irr, irr_count, sizeof(int), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  if (n_irr > 0) return 1;
  ApArgs p;
  std::memset(&p, 0, sizeof p);
  p.cap = a.cap; p.base = a.base; p.count = a.count; p.order = a.order; p.ops = c->d_ops; p.nsteps = a.nsteps;
  p.queue = a.queue + 1;
  if (rank) p.slot = c->d_rank_slot;
  p.lane_tab = (const AdafParams*)tab_models; p.units_arr = tab_units; p.units_ref = a.units; p.out_stride = sw->out_stride;
  double* planes[6] = {a.I, a.Q, a.U, a.V, a.tau, a.tauF};
  for (int m0 = 0; m0 < sw->n_models; m0 += SWEEP_MAX_MODELS) {
    const int mc = std::min(SWEEP_MAX_MODELS, sw->n_models - m0);
    if (m0 > 0 && (rc = send_tables(m0, mc)) != IPOLE_OK) return rc;
    p.n_models = mc;
    p.I = planes[0] + (size_t)m0 * sw->out_stride; p.Q = planes[1] + (size_t)m0 * sw->out_stride;
    p.U = planes[2] + (size_t)m0 * sw->out_stride; p.V = planes[3] + (size_t)m0 * sw->out_stride;
    p.tau = planes[4] ? planes[4] + (size_t)m0 * sw->out_stride : nullptr;
    p.tauF = planes[5] ? planes[5] + (size_t)m0 * sw->out_stride : nullptr;
    CK(cudaMemsetAsync(p.queue, 0, sizeof(unsigned long long), st));
    const int s = span_begin(c, LK_APPLY, st);
    const int ga = grid_for(c, c->opt_unpol ? c->occ_ap_unpol : c->occ_ap, IPOLE_AP_THREADS / 32, ((rays + 31) / 32) * mc);
    if (c->opt_unpol) k_apply_unpol_sweep<<<ga, IPOLE_AP_THREADS, 0, st>>>(p);
    else k_apply<false, true><<<ga, IPOLE_AP_THREADS, 0, st>>>(p);
    span_end(c, s, st);
    c->stats.n_launches++;
    CK(cudaGetLastError());
  }
  return IPOLE_OK;
}

// Model sweep of the grid model with the geometry done once (gridsweep.cuh): k_gridop walks every ray of the batch once and
// leaves a compact record per plasma step, k_gridapply_sweep walks the compact records once per parameter set.
int launch_transfer_gridsweep_split(ipole_ctx* c, const RtArgs& a, int64_t rays, cudaStream_t st, const Sweep* sw) {
  int32_t* npl = c->d_irr;                   // (the irregular-ray lists of the analytic split are not in use here)
  const bool rank = c->opt_rank && rays > 32;
  if (rank) {
    RankArgs r = {a.base, a.count, nullptr, a.order, a.nsteps, c->d_rank_pos, c->d_rank_slot, a.srange};
    const int s = span_begin(c, LK_OPS, st);
    k_rank_window<<<(unsigned)((rays + RANK_WINDOW - 1) / RANK_WINDOW), RANK_WINDOW, 0, st>>>(r);
    span_end(c, s, st);
    c->stats.n_launches++;
  }
  {
    GopArgs o;
    std::memset(&o, 0, sizeof o);
    o.cam = a.cam; o.units = a.units; o.model = a.model; o.cap = a.cap; o.base = a.base; o.count = a.count; o.order = a.order;
    o.path = a.path; o.nsteps = a.nsteps; o.srange = a.srange; o.rank_slot = rank ? c->d_rank_slot : nullptr;
    o.queue = a.queue; o.ops = c->d_ops; o.npl = npl;
    const int s = span_begin(c, LK_OPS, st);
    k_gridop<<<grid_for(c, c->occ_gridop, IPOLE_RT_THREADS / 32, (rays + 31) / 32), IPOLE_RT_THREADS, 0, st>>>(o);
    span_end(c, s, st);
    c->stats.n_launches++;
    CK(cudaGetLastError());
  }
  GapArgs p;
  std::memset(&p, 0, sizeof p);
  p.cap = a.cap; p.base = a.base; p.count = a.count; p.order = a.order; p.rank_slot = rank ? c->d_rank_slot : nullptr;
  p.ops = c->d_ops; p.npl = npl; p.queue = a.queue + 1;
  p.lane_tab = (const GridScales*)c->d_sweep_models; p.units_arr = c->d_sweep_units; p.units_ref = a.units; p.out_stride = sw->out_stride;
  double* planes[6] = {a.I, a.Q, a.U, a.V, a.tau, a.tauF};
  for (int m0 = 0; m0 < sw->n_models; m0 += SWEEP_MAX_MODELS) {
    const int mc = std::min(SWEEP_MAX_MODELS, sw->n_models - m0);
    CK(cudaMemcpyAsync(c->d_sweep_models, (const char*)sw->lane_tab + (size_t)m0 * sw->lane_bytes, mc * sw->lane_bytes, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(c->d_sweep_units, sw->units + m0, mc * sizeof(Units), cudaMemcpyHostToDevice, st));
    p.n_models = mc;
    p.I = planes[0] + (size_t)m0 * sw->out_stride; p.Q = planes[1] + (size_t)m0 * sw->out_stride;
    p.U = planes[2] + (size_t)m0 * sw->out_stride; p.V = planes[3] + (size_t)m0 * sw->out_stride;
    p.tau = planes[4] ? planes[4] + (size_t)m0 * sw->out_stride : nullptr;
    p.tauF = planes[5] ? planes[5] + (size_t)m0 * sw->out_stride : nullptr;
    CK(cudaMemsetAsync(p.queue, 0, sizeof(unsigned long long), st));
    const int s = span_begin(c, LK_APPLY, st);
    k_gridapply_sweep<<<grid_for(c, c->occ_gridapply, IPOLE_AP_THREADS / 32, ((rays + 31) / 32) * mc), IPOLE_AP_THREADS, 0, st>>>(p);
    span_end(c, s, st);
    c->stats.n_launches++;
    CK(cudaGetLastError());
  }
  return IPOLE_OK;
}

GeoArgs geo_args(ipole_ctx* c) {
  GeoArgs g;
  std::memset(&g, 0, sizeof g);
  g.cam = c->cam;
  g.eps = c->cam.eps;
  g.max_steps = c->cam.max_steps;
  g.list_stride = 1;
  return g;
}

// a-9 and the bookkeeping that closes an image
int finish_image(ipole_ctx* c, int64_t n, double* I, double* Q, double* U, double* V, int total) {
  {
    const int s = span_begin(c, LK_OTHER, c->stream);
    const int nb = (int)std::min<int64_t>(REDUCE_BLOCKS, (n + 255) / 256);
    k_reduce_partial<<<nb, 256, 0, c->stream>>>(n, I, Q, U, V, c->d_nsteps, c->d_nturn, c->d_part);
    const double pix_rad = c->cam.pix * c->units.L_unit / c->units.D_cm;
    k_reduce_final<<<1, 32, 0, c->stream>>>(c->d_part, nb, pix_rad * pix_rad * 1e23, c->d_red);
    c->stats.n_launches += 2;
    span_end(c, s, c->stream);
    CK(cudaGetLastError());
  }
  span_end(c, total, c->stream);
  c->have_image = true;
  c->last_n = n;
  return IPOLE_OK;
}


// the whole pipeline for n rays; outputs are DEVICE pointers indexed by ray
int run_rays(ipole_ctx* c, int64_t n, const int64_t* d_pixels, double* I, double* Q, double* U, double* V, double* tau,
             double* tauF, const Sweep* sw = nullptr) {
  int rc;
  if ((rc = ensure_rays(c, n)) != IPOLE_OK) return rc;
  c->spans_used = 0;
  std::memset(&c->stats, 0, sizeof c->stats);
  c->have_image = false;
  c->last_pf = 0;
  CK(cudaMemsetAsync(c->d_queues, 0, N_QUEUES * sizeof(unsigned long long), c->stream));
  CK(cudaMemsetAsync(c->d_small, 0, 2 * sizeof(int), c->stream));
  int qi = 0;
  const int total = span_begin(c, LK_OTHER, c->stream);

  size_t budget = path_budget(c);
  const size_t rec_bytes = REC_DOUBLES * sizeof(double);
  const int max_steps = c->cam.max_steps;
  int cap = max_steps;
  const int32_t* order = nullptr;
  std::vector<unsigned int> bin_prefix;   // sorted rays: number of rays in the bins before each bin (longer rays)
  int bin_width = 1;
  // ---- plan of the previous call (ctx.plan_cache): a full image with the same camera and scheduling options is
  // scheduled from it, with no probe pass and no read-back, so the call returns while the GPU is still working ----
  ipole_ctx::PlanCache& pc = c->plan_cache;
  const unsigned plan_flags = (unsigned)c->opt_sort | (unsigned)c->opt_tight << 2 | (unsigned)(c->opt_split != 0) << 3 | (unsigned)c->opt_overlap << 4 |
                              (unsigned)c->opt_unpol << 5 | (unsigned)c->opt_geo_fp32 << 6 | (unsigned)c->opt_side_retry << 7 |
                              (unsigned)c->opt_occ << 8 | (unsigned)c->opt_rank << 9 | (unsigned)c->model << 12;
  const bool cacheable = c->opt_plan_reuse && !d_pixels && !sw && c->n_mc == 0 && !c->opt_path_free && c->edf.kind == 0 && c->opt_sort != 0;
  const bool replay = cacheable && pc.valid && pc.n == n && pc.flags == plan_flags && std::memcmp(&pc.cam, &c->cam_in, sizeof(ipole_camera)) == 0 &&
                      (budget > pc.budget ? budget - pc.budget : pc.budget - budget) <= pc.budget / 64;
  if (!replay) pc.valid = false;          // (this call may overwrite d_order)
  if (replay) budget = pc.budget;         // the same plan needs the memory that is already there
  c->stats.plan_reused = replay ? 1 : 0;
  const bool fits_all = (double)n * (double)(max_steps + 1) * (double)rec_bytes <= (double)budget;
  const bool probe = !replay && (n >= 32768 || c->opt_sort == 2) && (c->opt_sort || !fits_all);
  if (replay) { cap = pc.cap; bin_width = pc.bin_width; bin_prefix = pc.bin_prefix; order = c->d_order; }

  if (probe) {
    // ---- probe pass: coarse lattice (or strided list), 4 eps, no path storage ----
    GeoArgs g = geo_args(c);
    g.eps = c->cam.eps * PROBE_EPS_FACTOR;
    SortArgs sa;
    std::memset(&sa, 0, sizeof sa);
    int64_t np;
    if (!d_pixels) {
      // one probe lattice per camera (c->n_mc cameras in a call of ipole_make_images_cameras, else one)
      const int stride = std::max(1, (int)std::ceil(std::sqrt((double)n / PROBE_TARGET)));
      const int lnx = std::max(1, c->cam.nx / stride), lny = std::max(1, c->cam.ny / stride);
      np = (int64_t)lnx * lny * std::max(1, c->n_mc);
      g.lattice_stride = stride; g.lattice_nx = lnx; g.lattice_ny = lny;
      sa.lattice_stride = stride; sa.lattice_nx = lnx; sa.lattice_ny = lny; sa.nx = c->cam.nx;
      sa.rays_per_cam = c->n_mc ? c->mc_rays_per_cam : 0;
    } else {
      const int64_t ls = std::max<int64_t>(1, n / PROBE_TARGET);
      np = (n + ls - 1) / ls;
      g.pixels = d_pixels; g.list_stride = ls;
      sa.list_stride = (int)ls;
    }
    if (np > c->probe_cap) {
      cudaFree(c->d_probe); c->d_probe = nullptr; c->probe_cap = 0;
      CK(cudaMalloc(&c->d_probe, np * sizeof(int32_t)));
      c->probe_cap = np;
    }
    g.count = np; g.nsteps = c->d_probe; g.queue = c->d_queues + (qi++);
    if ((rc = launch_geodesic(c, g, LK_PROBE, np, c->stream)) != IPOLE_OK) return rc;
    const int sp = span_begin(c, LK_PROBE, c->stream);
    k_max_i32<<<1, 1024, 0, c->stream>>>(c->d_probe, (int)np, c->d_small + 1);
    c->stats.n_launches++;
    int pmax = 0;
    CK(cudaMemcpyAsync(&pmax, c->d_small + 1, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    cap = (int)std::min<int64_t>(max_steps, (int64_t)(pmax * PROBE_EPS_FACTOR * 1.15) + 64);
    if (c->opt_sort) {
      sa.n = n; sa.probe = c->d_probe; sa.scale = PROBE_EPS_FACTOR;
      sa.bin_width = std::max(1, (cap + SORT_BINS - 1) / SORT_BINS);
      sa.key = c->d_key; sa.hist = c->d_hist; sa.order = c->d_order;
      CK(cudaMemsetAsync(c->d_hist, 0, SORT_BINS * sizeof(unsigned int), c->stream));
      const int gb = (int)std::min<int64_t>((n + 255) / 256, 148 * 8);
      k_predict_hist<<<gb, 256, 0, c->stream>>>(sa);
      k_scan_bins<<<1, 1024, 0, c->stream>>>(c->d_hist);
      // rays before each bin in the sorted order: sizes the path slots batch by batch (below)
      bin_prefix.resize(SORT_BINS);
      CK(cudaMemcpyAsync(bin_prefix.data(), c->d_hist, SORT_BINS * sizeof(unsigned int), cudaMemcpyDeviceToHost, c->stream));
      k_scatter<<<gb, 256, 0, c->stream>>>(sa);
      c->stats.n_launches += 3;
      CK(cudaGetLastError());
      CK(cudaStreamSynchronize(c->stream));
      bin_width = sa.bin_width;
      order = c->d_order;
    }
    span_end(c, sp, c->stream);
  }
  if (!probe && !replay) {
    // everything in flight at once: give each ray what the budget allows
    // (per step: the path record and, where the split transfer will run, the operator record -- so that the slots the
    // plan below can afford hold every ray in ONE batch: a pixel list of an adaptive level is a few thousand rays whose
    // time is the latency of the longest, and two batches are twice that)
    const bool will_split = c->edf.kind != 0 || c->n_mc > 0 || (c->opt_split && (!c->opt_unpol || (sw && sw->n_models >= 4)) && c->model == MODEL_ADAF);
    const bool will_grid = sw && c->opt_split && !c->opt_unpol && c->model == MODEL_GRID && c->opt_occ;
    const size_t per_step = rec_bytes + (will_grid ? GOP_DOUBLES * sizeof(double) : (will_split && !c->opt_path_free) ? OP_DOUBLES * sizeof(double) : 0);
    const int64_t per = (int64_t)(budget / per_step / (size_t)(((n + 31) / 32) * 32)) - 1;
    cap = (int)std::max<int64_t>(64, std::min<int64_t>(max_steps, per));
  }
  if ((c->edf.kind != 0 || c->n_mc) && c->opt_path_free) return IPOLE_EINVAL;
  if (c->opt_path_free && !sw && !c->opt_unpol) {
    // ---- path-free bidirectional variant: one geodesic launch that keeps the end points, one
    // transfer launch that re-integrates forward.  Rays are ordered longest first, so the few very long rays start
    // at once and run beside the bulk. ----
    if (n > c->endp_cap) {
      cudaFree(c->d_endp); c->d_endp = nullptr; c->endp_cap = 0;
      cudaError_t e = cudaMalloc(&c->d_endp, (size_t)n * rec_bytes);
      if (e != cudaSuccess) { c->last_cuda = (int)e; cudaGetLastError(); return IPOLE_ENOMEM; }
      c->endp_cap = n;
    }
    GeoArgs g = geo_args(c);
    g.cap = 0; g.base = 0; g.count = n; g.order = order; g.pixels = d_pixels;
    g.path = nullptr; g.nsteps = c->d_nsteps; g.nturn = c->d_nturn; g.queue = c->d_queues + (qi++);
    g.endp = c->d_endp;
    if ((rc = launch_geodesic(c, g, LK_GEO, n, c->stream)) != IPOLE_OK) return rc;
    RtArgs t;
    std::memset(&t, 0, sizeof t);
    t.cam = c->cam; t.units = c->units; t.model = c->d_model; t.base = 0; t.count = n; t.order = order;
    t.nsteps = c->d_nsteps; t.queue = c->d_queues + (qi++);
    t.I = I; t.Q = Q; t.U = U; t.V = V; t.tau = tau; t.tauF = tauF;
    t.endp = c->d_endp; t.nfwd = c->d_nsteps_long; t.eps = c->cam.eps; t.max_steps = max_steps;
    if ((rc = launch_transfer(c, t, LK_RT, n, c->stream, 0, c->cam.eps <= 0.04 ? 1 : 2)) != IPOLE_OK) return rc;
    c->stats.n_batches = 1;
    c->stats.path_cap = 0;
    c->last_pf = 1;
    CK(cudaMemsetAsync(c->d_sum, 0, sizeof(long long), c->stream));
    k_sum_i32<<<(int)std::min<int64_t>((n + 255) / 256, 592), 256, 0, c->stream>>>(c->d_nsteps_long, n, c->d_sum);
    c->stats.n_launches++;
    CK(cudaGetLastError());
    return finish_image(c, n, I, Q, U, V, total);
  }
  c->stats.path_cap = cap;

  // ---- long-ray passes: rays that overflowed their slot get one of max_steps.  They run on the side stream, as
  // soon as the geodesic kernel of a batch has listed them, concurrently with the remaining bulk batches (one such
  // ray is up to 50 000 sequential steps: its latency is hidden behind the bulk work instead of trailing it). ----
  // grid model: k_geodesic marks the steps that may cross plasma, k_transfer walks only from the first of them
  const bool use_occ = (c->model == MODEL_GRID) && c->opt_occ;
  const size_t lslot = (size_t)(max_steps + 1) * rec_bytes;
  // eDF coefficients and many ADAF cameras live in the split kernels only: their long rays take k_stepop + k_apply here
  // (operator records in d_ops_long) instead of the single kernel
  // (and the long rays of a small call -- an adaptive level, a pixel list, a small image -- of the analytic flow: nothing
  // hides the single kernel's one-lane walk of 50 000 steps there, k_apply_wide is 6x quicker on it)
  const bool long_split = c->edf.kind != 0 || (c->n_mc > 0 && c->model == MODEL_ADAF) ||
                          (c->opt_lowlat && c->opt_split == 1 && !sw && !c->opt_unpol && c->model == MODEL_ADAF && n <= (int64_t)c->n_sm * IPOLE_AP_THREADS * 4 &&
                           budget / 4 >= 128 * lslot);      // (room for 64 long rays with both records per pass)
  int long_done = 0;          // entries of d_long already handed to the side stream
  int64_t LBcap = 0;          // rays that fit the long path buffer
  const int32_t* long_src = replay ? pc.d_long : c->d_long;       // replay: the list the recorded call ended with
  const int32_t* retry_src = replay ? pc.d_retry : c->d_retry;
  auto long_pass = [&](int upto) -> int {
    if (upto <= long_done) return IPOLE_OK;
    if (LBcap == 0) {
      const size_t lbudget = std::max(lslot, std::min<size_t>(budget / 4, (size_t)16 << 30));
      const size_t lboth = long_split ? 2 * lslot : lslot;      // (an operator record is as large as a path record)
      LBcap = std::max<int64_t>(1, std::min<int64_t>(std::max(upto - long_done, 256), (int64_t)(lbudget / lboth)));
      if (!long_split && c->path_long_bytes >= lslot) LBcap = std::max<int64_t>(LBcap, (int64_t)(c->path_long_bytes / lslot));
      if (long_split && LBcap >= 64) LBcap &= ~(int64_t)31;     // whole groups of 32 slots (operator records)
      int rcl = ensure_path_long(c, (size_t)LBcap * lslot);
      if (rcl != IPOLE_OK) return rcl;
      if (long_split && (rcl = ensure_ops_long(c, (size_t)((LBcap + 31) / 32 * 32) * (size_t)(max_steps + 1) * OP_DOUBLES * sizeof(double))) != IPOLE_OK) return rcl;
    }
    for (int64_t base = long_done; base < upto; base += LBcap) {
      const int64_t cnt = std::min<int64_t>(LBcap, upto - base);
      if (qi + 4 > N_QUEUES) return IPOLE_EINVAL;
      GeoArgs g = geo_args(c);
      g.cap = max_steps; g.base = base; g.count = cnt; g.order = long_src; g.pixels = d_pixels;
      g.path = c->d_path_long; g.nsteps = c->d_nsteps_long; g.nturn = c->d_nturn; g.queue = c->d_queues + (qi++);
      if (use_occ) { g.grid = (const GridParams*)c->d_model; g.srange = c->d_srange; }
      int rcl = launch_geodesic(c, g, LK_LONG, cnt, c->side);
      if (rcl != IPOLE_OK) return rcl;
      RtArgs t;
      std::memset(&t, 0, sizeof t);
      t.cam = c->cam; t.units = c->units; t.model = c->d_model; t.cap = max_steps; t.base = base; t.count = cnt;
      t.order = long_src; t.path = c->d_path_long; t.nsteps = c->d_nsteps_long; t.queue = c->d_queues + qi;
      qi += long_split ? 3 : 1;
      if (use_occ) t.srange = c->d_srange;
      t.I = I; t.Q = Q; t.U = U; t.V = V; t.tau = tau; t.tauF = tauF;
      if (long_split) rcl = launch_transfer_split(c, t, cnt, c->side, 0, c->d_ops_long, 2);
      else rcl = launch_transfer(c, t, LK_LONG, cnt, c->side, 0, 0, sw);
      if (rcl != IPOLE_OK) return rcl;
    }
    long_done = upto;
    return IPOLE_OK;
  };
  // number of rays listed so far, read once the geodesic kernel of the current batch has finished
  auto listed = [&](cudaEvent_t geo_done, int& out) -> int {
    CK(cudaEventSynchronize(geo_done));
    CK(cudaMemcpyAsync(&out, c->d_small, sizeof(int), cudaMemcpyDeviceToHost, c->qstream));
    CK(cudaStreamSynchronize(c->qstream));
    return IPOLE_OK;
  };

  // ---- bulk pass in batches ----
  // (Running k_geodesic of batch k+1 on a second stream beside k_transfer of batch k was tried and dropped: the
  // transfer blocks leave no room for useful geodesic occupancy, profiles/r1_notes.md.)
  // split transfer (stepop.cuh): the batch also holds one 96-B operator record per step.
  //
  // Slots per batch: the rays are in order of predicted step count, longest first, so a batch needs slots only as
  // long as the prediction of its FIRST ray (times the same 1.15 margin as the global S_cap).  The longest rays fill
  // the first batch or two; every later batch holds two to three times as many rays in the same memory, and the
  // persistent kernels have that many fewer tails.  A ray that outgrows its batch's slot is listed and retried at
  // the end with the global S_cap (second level); one that outgrows S_cap goes to the long-ray pass as before.
  // numerically integrated eDF coefficients (ipole_set_edf) live in k_apply only: that mode always runs split, and its
  // long rays go through the same kernels on the side stream (long_pass above) instead of the single kernel
  // (many cameras per call, c->n_mc, analytic flow: the same -- only the split kernels know about per-ray cameras)
  // (the grid model's k_transfer_group knows per-ray cameras itself and keeps the ordinary flow)
  if (c->n_mc > 0 && c->model != MODEL_ADAF && (c->model != MODEL_GRID || sw || c->opt_unpol)) return IPOLE_EINVAL;
  const bool edf = c->edf.kind != 0 || (c->n_mc > 0 && c->model == MODEL_ADAF);
  if (edf && (sw || c->opt_unpol || c->model != MODEL_ADAF)) return IPOLE_EINVAL;
  const bool split = edf || (c->opt_split && !sw && !c->opt_unpol && c->model == MODEL_ADAF);
  // the sweep of the analytic flow keeps operator records too (launch_transfer_sweep_split); its batches run through
  // launch_transfer as before
  const bool grid_sweep_split = sw && c->opt_split && !c->opt_unpol && c->model == MODEL_GRID && use_occ;   // gridsweep.cuh
  const bool sweep_split = grid_sweep_split || (sw && c->opt_split && (!c->opt_unpol || sw->n_models >= 4) && c->model == MODEL_ADAF);
  const size_t op_doubles = grid_sweep_split ? GOP_DOUBLES : OP_DOUBLES;
  const size_t step_bytes = rec_bytes + ((split || sweep_split) ? op_doubles * sizeof(double) : 0);
  const bool tight = order != nullptr && !bin_prefix.empty() && c->opt_tight;
  struct Batch { int64_t base, cnt; int cap; };
  std::vector<Batch> plan;
  size_t lane_budget = budget;            // path (+ operator) memory of one lane
  auto make_plan = [&](int64_t total_rays, bool use_bins) {
    plan.clear();
    for (int64_t base = 0; base < total_rays;) {
      int cb = cap;
      if (use_bins) {
        const int bin = (int)(std::upper_bound(bin_prefix.begin(), bin_prefix.end(), (unsigned int)base) - bin_prefix.begin()) - 1;
        const int64_t pred_hi = (int64_t)(SORT_BINS - std::max(bin, 0)) * bin_width;
        cb = (int)std::min<int64_t>(cap, (int64_t)(pred_hi * 1.15) + 64);
      }
      int64_t B = (int64_t)(lane_budget / ((size_t)(cb + 1) * step_bytes));
      if (B >= 64) B &= ~(int64_t)31;           // whole groups of 32 slots (operator records, stepop.cuh)
      B = std::max<int64_t>(1, std::min(B, total_rays - base));
      plan.push_back({base, B, cb});
      if (std::getenv("IPOLE_DEBUG_SPANS")) std::fprintf(stderr, "batch base %lld cnt %lld cap %d\n", (long long)base, (long long)B, cb);
      base += B;
    }
  };
  // Two lanes: consecutive batches alternate between two streams, each with its own half of the path (and operator)
  // memory.  Every kernel of a batch is persistent and ends in a tail during which the GPU drains (the last rays of a
  // geodesic launch are milliseconds long); the other lane's kernels fill those tails.  One lane when a single batch
  // holds everything, and for the sweeps (their parameter tables are per stream).
  int n_lanes = 1;
  make_plan(n, tight);
  // (from three batches on: with two, halving them adds more kernel tails and retried rays than the overlap hides --
  // 64 grid cameras of 128^2: 205 ms on one lane, 220 ms on two)
  if (c->opt_overlap && c->lane2 && !sw && plan.size() >= 3) {
    n_lanes = 2;
    lane_budget = budget / 2;
    make_plan(n, tight);
  }
  c->stats.n_lanes = n_lanes;
  size_t lane_path = 0, lane_ops = 0;     // bytes per lane
  auto prepare = [&](bool with_retry_level) -> int {
    size_t np = 0, no = 0;
    for (const Batch& b : plan) {
      np = std::max(np, (size_t)b.cnt * (size_t)(b.cap + 1) * rec_bytes);
      no = std::max(no, (size_t)((b.cnt + 31) / 32 * 32) * (size_t)(b.cap + 1) * op_doubles * sizeof(double));
    }
    if (with_retry_level) {   // the retry level runs with the global S_cap
      const int64_t Br = std::max<int64_t>(1, (int64_t)(lane_budget / ((size_t)(cap + 1) * step_bytes)));
      const int64_t rr = std::min<int64_t>(Br, std::max<int64_t>(n / 8, 1));   // more than n/8 retries never happen; the buffer grows if they do
      np = std::max(np, (size_t)rr * (size_t)(cap + 1) * rec_bytes);
      no = std::max(no, (size_t)((rr + 31) / 32 * 32) * (size_t)(cap + 1) * op_doubles * sizeof(double));
    }
    lane_path = std::max(lane_path, (np + 255) & ~(size_t)255);
    lane_ops = std::max(lane_ops, (no + 255) & ~(size_t)255);
    int rcp;
    if ((rcp = ensure_path(c, lane_path * n_lanes)) != IPOLE_OK) return rcp;
    if ((split || sweep_split) && (rcp = ensure_ops(c, lane_ops * n_lanes)) != IPOLE_OK) return rcp;
    return IPOLE_OK;
  };
  if ((rc = prepare(tight)) != IPOLE_OK) return rc;
  int n_long = 0;
  int* retry_count = c->d_small + 5;
  // with few batches the long-ray passes cannot wait for kernel boundaries: keep 8 block slots free for them
  const int reserve = (cap < max_steps && plan.size() <= 16) ? 8 : 0;
  auto run_batch = [&](const Batch& b, const int32_t* ord, int lane) -> int {
    if (qi + 4 > N_QUEUES) return IPOLE_EINVAL;
    cudaStream_t st = lane ? c->lane2 : c->stream;
    double* path = c->d_path + (size_t)lane * (lane_path / sizeof(double));
    double* ops = split ? c->d_ops + (size_t)lane * (lane_ops / sizeof(double)) : nullptr;
    const bool top = b.cap >= cap;             // overflow means "longer than S_cap": the long-ray pass
    GeoArgs g = geo_args(c);
    g.cap = b.cap; g.base = b.base; g.count = b.cnt; g.order = ord; g.pixels = d_pixels;
    g.path = path; g.nsteps = c->d_nsteps; g.nturn = c->d_nturn; g.queue = c->d_queues + (qi++);
    if (top) { g.long_list = c->d_long; g.long_count = c->d_small; }
    else { g.long_list = c->d_retry; g.long_count = retry_count; }
    if (use_occ) { g.grid = (const GridParams*)c->d_model; g.srange = c->d_srange; }
    int rcb;
    if ((rcb = launch_geodesic(c, g, LK_GEO, b.cnt, st, reserve)) != IPOLE_OK) return rcb;
    CK(cudaEventRecord(c->ev_lastgeo[lane], st));
    if (top && cap < max_steps && !replay) {
      CK(cudaEventRecord(c->ev_geo, st));
      CK(cudaStreamWaitEvent(c->side, c->ev_geo, 0));
    }
    RtArgs t;
    std::memset(&t, 0, sizeof t);
    t.cam = c->cam; t.units = c->units; t.model = c->d_model; t.cap = b.cap; t.base = b.base; t.count = b.cnt; t.order = ord;
    t.path = path; t.nsteps = c->d_nsteps; t.queue = c->d_queues + qi;
    qi += (split || sweep_split) ? 3 : 1;
    if (use_occ) t.srange = c->d_srange;
    t.I = I; t.Q = Q; t.U = U; t.V = V; t.tau = tau; t.tauF = tauF;
    if (split) rcb = launch_transfer_split(c, t, b.cnt, st, reserve, ops, lane);
    else rcb = launch_transfer(c, t, LK_RT, b.cnt, st, reserve, 0, sw);
    if (rcb != IPOLE_OK) return rcb;
    c->stats.n_batches++;
    if (top && cap < max_steps && !replay) {   // the transfer kernel just queued keeps the GPU busy while the host waits here
      if ((rcb = listed(c->ev_geo, n_long)) != IPOLE_OK) return rcb;
      if ((rcb = long_pass(n_long)) != IPOLE_OK) return rcb;
    }
    return IPOLE_OK;
  };
  // the batches of `plan`, alternating between the lanes; the main stream continues when both are done
  auto run_plan = [&](const int32_t* ord) -> int {
    const bool two = n_lanes == 2 && plan.size() >= 2;
    if (two) {
      CK(cudaEventRecord(c->ev_fork, c->stream));
      CK(cudaStreamWaitEvent(c->lane2, c->ev_fork, 0));
    }
    int k = 0, rcp;
    for (const Batch& b : plan)
      if ((rcp = run_batch(b, ord, two ? (k++ & 1) : 0)) != IPOLE_OK) return rcp;
    if (two) {
      CK(cudaEventRecord(c->ev_join, c->lane2));
      CK(cudaStreamWaitEvent(c->stream, c->ev_join, 0));
    }
    return IPOLE_OK;
  };
  CK(cudaMemsetAsync(retry_count, 0, sizeof(int), c->stream));
  // ---- second level on the side stream: slots of its own for up to R_max retried rays, sized before their number is
  // known (the kernels read the count on the device), so that the pass starts when the LAST geodesic kernel of the bulk
  // has finished and runs beside the last transfer kernels.  What does not fit (never seen) takes the lanes afterwards.
  int64_t R_max = 0;
  if (tight && !sw && c->opt_side_retry && plan.size() >= 2) {
    const size_t slot = (size_t)(cap + 1) * step_bytes;
    R_max = std::max<int64_t>(256, n / 64);     // (what limits it is the memory below: 8 GiB of slots)
    R_max = std::min<int64_t>(R_max, (int64_t)(std::min<size_t>(budget / 8, (size_t)8 << 30) / slot)) & ~(int64_t)31;
    if (R_max >= 32 && ensure_retry_buf(c, (size_t)R_max * slot) != IPOLE_OK) R_max = 0;
    if (R_max < 32) R_max = 0;
  }
  const int n_lanes_bulk = (n_lanes == 2 && plan.size() >= 2) ? 2 : 1;
  // the retry level on the side stream for the first `count` (or *count_dev) entries of `list`
  auto side_retry = [&](const int32_t* list, int64_t count, const int* count_dev) -> int {
    if (qi + 4 > N_QUEUES) return IPOLE_EINVAL;
    double* rpath = c->d_retry_buf;
    double* rops = split ? c->d_retry_buf + (size_t)R_max * (size_t)(cap + 1) * REC_DOUBLES : nullptr;
    GeoArgs g = geo_args(c);
    g.cap = cap; g.base = 0; g.count = count; g.count_dev = count_dev; g.order = list; g.pixels = d_pixels;
    g.path = rpath; g.nsteps = c->d_nsteps_long; g.nturn = c->d_nturn; g.queue = c->d_queues + (qi++);
    g.long_list = c->d_long; g.long_count = c->d_small;
    if (use_occ) { g.grid = (const GridParams*)c->d_model; g.srange = c->d_srange; }
    int rcs;
    if ((rcs = launch_geodesic(c, g, LK_LONG, count, c->side)) != IPOLE_OK) return rcs;
    CK(cudaEventRecord(c->ev_geo, c->side));
    RtArgs t;
    std::memset(&t, 0, sizeof t);
    t.cam = c->cam; t.units = c->units; t.model = c->d_model; t.cap = cap; t.base = 0; t.count = count; t.count_dev = count_dev;
    t.order = list; t.path = rpath; t.nsteps = c->d_nsteps_long; t.queue = c->d_queues + qi;
    qi += split ? 3 : 1;
    if (use_occ) t.srange = c->d_srange;
    t.I = I; t.Q = Q; t.U = U; t.V = V; t.tau = tau; t.tauF = tauF;
    if (split) rcs = launch_transfer_split(c, t, count, c->side, 0, rops, 2);
    else rcs = launch_transfer(c, t, LK_LONG, count, c->side, 0, 0, nullptr);
    return rcs;
  };
  bool side_used = false;
  int n_retry_side = 0;
  if (replay) {
    // Everything the side stream does is known: the retried rays, then the long rays, from the recorded lists, started
    // now, beside the first bulk batches (the retry level first: a retried ray that is also long is marked by it and
    // traced by the long pass, in that order, as in the recorded call).
    CK(cudaEventRecord(c->ev_fork, c->stream));
    CK(cudaStreamWaitEvent(c->side, c->ev_fork, 0));
    n_retry_side = (int)std::min<int64_t>(pc.n_retry, R_max);
    if (n_retry_side > 0 && (rc = side_retry(retry_src, n_retry_side, nullptr)) != IPOLE_OK) return rc;
    n_long = pc.n_long;
    if (n_long > 0 && (rc = long_pass(n_long)) != IPOLE_OK) return rc;
    side_used = n_retry_side > 0;
  }
  if ((rc = run_plan(order)) != IPOLE_OK) return rc;
  if (R_max > 0 && !replay) {
    for (int l = 0; l < n_lanes_bulk; ++l) CK(cudaStreamWaitEvent(c->side, c->ev_lastgeo[l], 0));
    int* rcount = c->d_small + 7;
    k_clamp_count<<<1, 1, 0, c->side>>>(retry_count, (int)R_max, rcount);
    c->stats.n_launches++;
    if ((rc = side_retry(retry_src, R_max, rcount)) != IPOLE_OK) return rc;
    side_used = true;
  }
  int n_retry = 0;
  if (tight) {
    if (replay) n_retry = pc.n_retry;
    else {
      CK(cudaMemcpyAsync(&n_retry, retry_count, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
      CK(cudaStreamSynchronize(c->stream));
      n_retry_side = (int)std::min<int64_t>(n_retry, R_max);
      if (n_retry_side > 0 && cap < max_steps) {
        // retried rays that outgrow S_cap as well: listed by the geodesic kernel above, long-ray pass
        if ((rc = listed(c->ev_geo, n_long)) != IPOLE_OK) return rc;
        if ((rc = long_pass(n_long)) != IPOLE_OK) return rc;
      }
    }
    c->stats.n_retry = n_retry;
    if (n_retry > n_retry_side) {
      // the rest of the second level on the lanes, with the global S_cap
      make_plan(n_retry - n_retry_side, false);
      if ((rc = prepare(false)) != IPOLE_OK) return rc;
      if ((rc = run_plan(retry_src + n_retry_side)) != IPOLE_OK) return rc;
    }
  }
  c->stats.n_long = n_long;
  if (n_long > 0 || side_used) {
    // join the side stream, then publish the step counts of the long and the retried rays (the bulk transfer kernels
    // read nsteps[q] = -1 for them, so the side-stream passes keep theirs apart until every bulk kernel is done)
    CK(cudaEventRecord(c->ev_side, c->side));
    CK(cudaStreamWaitEvent(c->stream, c->ev_side, 0));
    if (n_long > 0) {
      k_merge_long<<<(n_long + 255) / 256, 256, 0, c->stream>>>(n_long, long_src, c->d_nsteps_long, c->d_nsteps);
      c->stats.n_launches++;
    }
    if (n_retry_side > 0) {
      k_merge_long<<<(n_retry_side + 255) / 256, 256, 0, c->stream>>>(n_retry_side, retry_src, c->d_nsteps_long, c->d_nsteps);
      c->stats.n_launches++;
    }
    CK(cudaGetLastError());
  }
  if (cacheable && !replay && order != nullptr && !bin_prefix.empty()) {
    // keep what this call had to read back, and the two lists as they stand now (every kernel that appends has been
    // joined into the stream)
    pc.cam = c->cam_in; pc.n = n; pc.budget = budget; pc.flags = plan_flags;
    pc.cap = cap; pc.bin_width = bin_width; pc.bin_prefix = bin_prefix;
    pc.n_long = c->stats.n_long > 0 ? (int)c->stats.n_long : 0; pc.n_retry = n_retry;
    bool ok = true;
    if (pc.n_long > pc.long_cap) {
      cudaFree(pc.d_long); pc.d_long = nullptr; pc.long_cap = 0;
      if (cudaMalloc(&pc.d_long, (size_t)pc.n_long * sizeof(int32_t)) == cudaSuccess) pc.long_cap = pc.n_long; else { cudaGetLastError(); ok = false; }
    }
    if (pc.n_retry > pc.retry_cap) {
      cudaFree(pc.d_retry); pc.d_retry = nullptr; pc.retry_cap = 0;
      if (cudaMalloc(&pc.d_retry, (size_t)pc.n_retry * sizeof(int32_t)) == cudaSuccess) pc.retry_cap = pc.n_retry; else { cudaGetLastError(); ok = false; }
    }
    if (ok && pc.n_long > 0) CK(cudaMemcpyAsync(pc.d_long, c->d_long, (size_t)pc.n_long * sizeof(int32_t), cudaMemcpyDeviceToDevice, c->stream));
    if (ok && pc.n_retry > 0) CK(cudaMemcpyAsync(pc.d_retry, c->d_retry, (size_t)pc.n_retry * sizeof(int32_t), cudaMemcpyDeviceToDevice, c->stream));
    pc.valid = ok;
  }

  return finish_image(c, n, I, Q, U, V, total);
}

}  // namespace

namespace { void totals_static_setup(ipole_ctx* c); }   // defined with ipole_image_totals_static, below

extern "C" {

int ipole_init(const ipole_camera* cam, ipole_ctx** out) {
  if (!cam || !out) return IPOLE_EINVAL;
  int rc = check_camera(cam);
  if (rc != IPOLE_OK) return rc;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return IPOLE_ECUDA; }
  ipole_ctx* c = new (std::nothrow) ipole_ctx();
  if (!c) return IPOLE_ENOMEM;
  std::memset(&c->stats, 0, sizeof c->stats);
  { const char* e = std::getenv("IPOLE_NO_OCC"); if (e && e[0] == '1') c->opt_occ = 0; }
  auto fail = [&](int code) { ipole_free(c); return code; };
  if (cudaGetDevice(&c->device) != cudaSuccess) return fail(IPOLE_ECUDA);
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, c->device) != cudaSuccess) return fail(IPOLE_ECUDA);
  c->n_sm = prop.multiProcessorCount;
  if (cudaMalloc(&c->d_cam, sizeof(CamDev)) != cudaSuccess) return fail(IPOLE_ENOMEM);
  size_t msz = std::max(sizeof(GridParams), std::max(sizeof(AdafParams), sizeof(SlabParams)));
  if (cudaMalloc(&c->d_model, msz) != cudaSuccess) return fail(IPOLE_ENOMEM);
  if (cudaMalloc(&c->d_queues, N_QUEUES * sizeof(unsigned long long)) != cudaSuccess) return fail(IPOLE_ENOMEM);
  if (cudaMalloc(&c->d_hist, SORT_BINS * sizeof(unsigned int)) != cudaSuccess) return fail(IPOLE_ENOMEM);
  if (cudaMalloc(&c->d_small, 8 * sizeof(int)) != cudaSuccess) return fail(IPOLE_ENOMEM);
  if (cudaMalloc(&c->d_part, REDUCE_BLOCKS * sizeof(ReducePartial)) != cudaSuccess) return fail(IPOLE_ENOMEM);
  if (cudaMalloc(&c->d_red, sizeof(ReduceOut)) != cudaSuccess) return fail(IPOLE_ENOMEM);
  {
    int lo = 0, hi = 0;
    cudaDeviceGetStreamPriorityRange(&lo, &hi);   // hi = greatest priority: the few long-ray blocks go first
    if (cudaStreamCreateWithPriority(&c->side, cudaStreamNonBlocking, hi) != cudaSuccess) return fail(IPOLE_ECUDA);
    if (cudaStreamCreateWithFlags(&c->qstream, cudaStreamNonBlocking) != cudaSuccess) return fail(IPOLE_ECUDA);
    if (cudaEventCreateWithFlags(&c->ev_geo, cudaEventDisableTiming) != cudaSuccess) return fail(IPOLE_ECUDA);
    if (cudaEventCreateWithFlags(&c->ev_side, cudaEventDisableTiming) != cudaSuccess) return fail(IPOLE_ECUDA);
    if (cudaStreamCreateWithFlags(&c->lane2, cudaStreamNonBlocking) != cudaSuccess) return fail(IPOLE_ECUDA);
    if (cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) != cudaSuccess) return fail(IPOLE_ECUDA);
    if (cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming) != cudaSuccess) return fail(IPOLE_ECUDA);
    for (int l = 0; l < 2; ++l)
      if (cudaEventCreateWithFlags(&c->ev_lastgeo[l], cudaEventDisableTiming) != cudaSuccess) return fail(IPOLE_ECUDA);
  }
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_geo, k_geodesic<false>, IPOLE_GEO_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_geo_occ, k_geodesic<true>, IPOLE_GEO_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_rt[MODEL_ADAF], k_transfer<MODEL_ADAF, 0>, IPOLE_RT_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_rt[MODEL_SLAB], k_transfer<MODEL_SLAB, 0>, IPOLE_RT_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_rt[MODEL_GRID], k_transfer<MODEL_GRID, 0>, IPOLE_RT_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_pf[MODEL_ADAF][1], k_transfer<MODEL_ADAF, 1>, IPOLE_RT_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_pf[MODEL_SLAB][1], k_transfer<MODEL_SLAB, 1>, IPOLE_RT_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_pf[MODEL_GRID][1], k_transfer<MODEL_GRID, 1>, IPOLE_RT_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_pf[MODEL_ADAF][2], k_transfer<MODEL_ADAF, 2>, IPOLE_RT_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_pf[MODEL_SLAB][2], k_transfer<MODEL_SLAB, 2>, IPOLE_RT_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_pf[MODEL_GRID][2], k_transfer<MODEL_GRID, 2>, IPOLE_RT_THREADS, 0);
  if (cudaGetLastError() != cudaSuccess) return fail(IPOLE_ECUDA);
  if (cudaMalloc(&c->d_sum, sizeof(long long)) != cudaSuccess) return fail(IPOLE_ENOMEM);
  if (cudaMalloc(&c->d_sweep_models, SWEEP_MAX_MODELS * std::max(sizeof(AdafParams), sizeof(GridScales))) != cudaSuccess) return fail(IPOLE_ENOMEM);
  if (cudaMalloc(&c->d_sweep_units, SWEEP_MAX_MODELS * sizeof(Units)) != cudaSuccess) return fail(IPOLE_ENOMEM);
  if (cudaMalloc(&c->d_sweep_models_side, SWEEP_MAX_MODELS * std::max(sizeof(AdafParams), sizeof(GridScales))) != cudaSuccess) return fail(IPOLE_ENOMEM);
  if (cudaMalloc(&c->d_sweep_units_side, SWEEP_MAX_MODELS * sizeof(Units)) != cudaSuccess) return fail(IPOLE_ENOMEM);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_sweep[MODEL_ADAF], k_transfer<MODEL_ADAF, 0, true>, IPOLE_RT_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_unpol[MODEL_ADAF][0], k_transfer_unpol<MODEL_ADAF, false>, IPOLE_RT_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_unpol[MODEL_SLAB][0], k_transfer_unpol<MODEL_SLAB, false>, IPOLE_RT_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_unpol[MODEL_GRID][0], k_transfer_unpol<MODEL_GRID, false>, IPOLE_RT_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_unpol[MODEL_ADAF][1], k_transfer_unpol<MODEL_ADAF, true>, IPOLE_RT_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_unpol[MODEL_GRID][1], k_transfer_unpol<MODEL_GRID, true>, IPOLE_RT_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_sweep[MODEL_GRID], k_transfer<MODEL_GRID, 0, true>, IPOLE_RT_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_op, k_stepop<MODEL_ADAF>, IPOLE_OP_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_op_mc, k_stepop<MODEL_ADAF, true>, IPOLE_OP_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_geo_mc, k_geodesic<false, true>, IPOLE_GEO_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_geo_occ_mc, k_geodesic<true, true>, IPOLE_GEO_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_group_mc, k_transfer_group<MODEL_GRID, true>, IPOLE_RT_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_geo_f32, k_geodesic_f32, IPOLE_GEO_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_ap, k_apply<false>, IPOLE_AP_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_ap_unpol, k_apply_unpol_sweep, IPOLE_AP_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_ap_wide, k_apply_wide<8>, IPOLE_AP_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_gridop, k_gridop, IPOLE_RT_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_gridapply, k_gridapply_sweep, IPOLE_AP_THREADS, 0);
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_ap_edf, k_apply<true>, IPOLE_AP_THREADS, EDF_MAX_NODES * sizeof(double4));
  { const char* e = std::getenv("IPOLE_NO_SPLIT"); if (e && e[0] == '1') c->opt_split = 0; }
  { const char* e = std::getenv("IPOLE_NO_TIGHT"); if (e && e[0] == '1') c->opt_tight = 0; }
  { const char* e = std::getenv("IPOLE_NO_GROUP"); if (e && e[0] == '1') c->opt_group = 0; }
  { const char* e = std::getenv("IPOLE_NO_OVERLAP"); if (e && e[0] == '1') c->opt_overlap = 0; }
  { const char* e = std::getenv("IPOLE_NO_PLAN_REUSE"); if (e && e[0] == '1') c->opt_plan_reuse = 0; }
  { const char* e = std::getenv("IPOLE_NO_LOWLAT"); if (e && e[0] == '1') c->opt_lowlat = 0; }
  { const char* e = std::getenv("IPOLE_NO_RANK"); if (e && e[0] == '1') c->opt_rank = 0; }
  { const char* e = std::getenv("IPOLE_NO_SIDE_RETRY"); if (e && e[0] == '1') c->opt_side_retry = 0; }
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->occ_group, k_transfer_group<MODEL_GRID>, IPOLE_RT_THREADS, 0);
  rc = apply_camera(c, cam);
  if (rc != IPOLE_OK) return fail(rc);
  totals_static_setup(c);   // address of the static scratch of ipole_image_totals_static on this device (a failure is kept for that call)
  *out = c;
  return IPOLE_OK;
}

int ipole_set_camera(ipole_ctx* c, const ipole_camera* cam) {
  if (!c || !cam) return IPOLE_EINVAL;
  int rc = check_camera(cam);
  if (rc != IPOLE_OK) return rc;
  const double h_new = cam->hslope > 0.0 ? cam->hslope : 1.0;
  if (c->model == MODEL_GRID && h_new != c->cam.G.hslope) return IPOLE_EINVAL;
  if (c->model == MODEL_ADAF && cam->flat_metric) return IPOLE_EINVAL;
  const double a_old = c->cam.G.a, L_old = c->units.L_unit;
  rc = apply_camera(c, cam);
  if (rc != IPOLE_OK) return rc;
  if (c->model == MODEL_GRID && c->units.L_unit != L_old) {
    // the density and field units of the grid model contain the length unit GM/c^2: keep them consistent with the
    // path element dl_unit when the camera's mass changes
    const double L = c->units.L_unit, rho_unit = c->grid_M_unit / (L * L * L);
    c->grid_host.ne_unit = rho_unit / (IP_MP + IP_ME);
    c->grid_host.B_unit = IP_CL * std::sqrt(4.0 * M_PI * rho_unit);
    CK(cudaMemcpyAsync(c->d_model, &c->grid_host, sizeof(GridParams), cudaMemcpyHostToDevice, c->stream));
    CK(cudaStreamSynchronize(c->stream));
  }
  if (c->model == MODEL_ADAF && a_old != cam->spin) {  // r_isco depends on the spin
    c->adaf_host.r_isco = isco_radius(cam->spin);
    CK(cudaMemcpyAsync(c->d_model, &c->adaf_host, sizeof(AdafParams), cudaMemcpyHostToDevice, c->stream));
    CK(cudaStreamSynchronize(c->stream));
  }
  return IPOLE_OK;
}

int ipole_set_stream(ipole_ctx* c, void* s) {
  if (!c) return IPOLE_EINVAL;
  if ((cudaStream_t)s != c->stream) c->plan_cache.valid = false;   // the recorded lists were written in the old stream's order
  c->stream = (cudaStream_t)s;
  return IPOLE_OK;
}

int ipole_set_options(ipole_ctx* c, uint64_t path_bytes, int32_t sort_rays) {
  if (!c) return IPOLE_EINVAL;
  c->opt_path_bytes = path_bytes;
  c->opt_sort = (sort_rays == 2) ? 2 : (sort_rays ? 1 : 0);
  return IPOLE_OK;
}

int ipole_set_unpolarized(ipole_ctx* c, int32_t on) {
  if (!c) return IPOLE_EINVAL;
  c->opt_unpol = on ? 1 : 0;
  return IPOLE_OK;
}

int ipole_set_edf(ipole_ctx* c, const ipole_edf* e) {
  if (!c || !e) return IPOLE_EINVAL;
  if (e->kind < 0 || e->kind > 2) return IPOLE_EINVAL;
  const int nn = e->n_nodes > 0 ? e->n_nodes : 128;
  const double kappa = e->kappa != 0.0 ? e->kappa : 3.5;
  if (e->kind != 0 && (nn > EDF_MAX_NODES || (e->kind == 2 && !(kappa > 1.0)))) return IPOLE_EINVAL;
  c->edf.kind = e->kind; c->edf.n_nodes = nn; c->edf.kappa = kappa; c->edf.dlx = (EDF_LNX_HI - EDF_LNX_LO) / nn;
  if (e->kind == 0) return IPOLE_OK;
  // per-node constants and the normalisation table of this distribution (once per call, not on the hot path)
  if (!c->d_edf_nodes) CK(cudaMalloc(&c->d_edf_nodes, EDF_MAX_NODES * sizeof(double4)));
  if (!c->d_edf_lnnorm) CK(cudaMalloc(&c->d_edf_lnnorm, EDF_TAB_N * sizeof(double)));
  c->edf.nodes = c->d_edf_nodes; c->edf.lnnorm = c->d_edf_lnnorm;
  k_edf_setup_nodes<<<(nn + 127) / 128, 128, 0, c->stream>>>(c->edf, c->d_edf_nodes);
  k_edf_setup_norm<<<(EDF_TAB_N + 127) / 128, 128, 0, c->stream>>>(c->edf, c->d_edf_lnnorm);
  CK(cudaGetLastError());
  return IPOLE_OK;
}

int ipole_set_geodesic_fp32(ipole_ctx* c, int32_t on) {
  if (!c) return IPOLE_EINVAL;
  c->opt_geo_fp32 = on ? 1 : 0;
  return IPOLE_OK;
}

int ipole_set_transfer_split(ipole_ctx* c, int32_t on) {
  if (!c) return IPOLE_EINVAL;
  c->opt_split = (on == 2) ? 2 : (on ? 1 : 0);
  return IPOLE_OK;
}

int ipole_set_plan_reuse(ipole_ctx* c, int32_t on) {
  if (!c) return IPOLE_EINVAL;
  c->opt_plan_reuse = on ? 1 : 0;
  c->plan_cache.valid = false;
  return IPOLE_OK;
}

int ipole_set_batch_overlap(ipole_ctx* c, int32_t on) {
  if (!c) return IPOLE_EINVAL;
  c->opt_overlap = on ? 1 : 0;
  return IPOLE_OK;
}

int ipole_set_path_free(ipole_ctx* c, int32_t on) {
  if (!c) return IPOLE_EINVAL;
  c->opt_path_free = on ? 1 : 0;
  return IPOLE_OK;
}

int ipole_load_model_adaf(ipole_ctx* c, const ipole_adaf_params* p) {
  if (!c || !p) return IPOLE_EINVAL;
  if (c->cam.G.mass == 0.0) return IPOLE_EINVAL;  // the flow is defined on Kerr only
  AdafParams m;
  m.n0 = p->n0; m.p_n = p->p_n; m.Th0 = p->Th0; m.p_T = p->p_T; m.B0 = p->B0; m.p_B = p->p_B;
  m.r_isco = isco_radius(c->cam.G.a);
  c->adaf_host = m;
  CK(cudaMemcpyAsync(c->d_model, &c->adaf_host, sizeof m, cudaMemcpyHostToDevice, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  c->model = MODEL_ADAF;
  return IPOLE_OK;
}

int ipole_load_model_slab(ipole_ctx* c, const ipole_slab_params* p) {
  if (!c || !p || !(p->H > 0.0)) return IPOLE_EINVAL;
  SlabParams m;
  m.H = p->H; m.profile = p->profile;
  const double psi = p->psi_deg * M_PI / 180.0;
  m.cpsi = std::cos(psi); m.spsi = std::sin(psi);
  for (int i = 0; i < 4; ++i) { m.j[i] = p->j[i]; m.al[i] = p->alpha[i]; }
  for (int i = 0; i < 3; ++i) m.rh[i] = p->rho[i];
  CK(cudaMemcpyAsync(c->d_model, &m, sizeof m, cudaMemcpyHostToDevice, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  c->model = MODEL_SLAB;
  return IPOLE_OK;
}

int ipole_load_model_grid(ipole_ctx* c, const ipole_grid_desc* d, const double* const fields[8]) {
  if (!c || !d || !fields) return IPOLE_EINVAL;
  if (d->N1 < 1 || d->N2 < 1 || d->N3 < 1) return IPOLE_EINVAL;
  if (d->hslope != c->cam.G.hslope) return IPOLE_EINVAL;
  for (int q = 0; q < 8; ++q) if (!fields[q]) return IPOLE_EINVAL;
  for (int i = 0; i < 3; ++i) if (!(d->dx[i] > 0.0)) return IPOLE_EINVAL;
  const size_t cells = (size_t)d->N1 * d->N2 * d->N3;
  if (cells != c->grid_cells) {
    cudaFree(c->d_grid); c->d_grid = nullptr; c->grid_cells = 0;
    cudaFree(c->d_occ); c->d_occ = nullptr;
    cudaError_t e = cudaMalloc(&c->d_grid, 8 * cells * sizeof(double));
    if (e != cudaSuccess) { c->last_cuda = (int)e; cudaGetLastError(); return IPOLE_ENOMEM; }
    c->grid_cells = cells;
  }
  GridParams m;
  std::memset(&m, 0, sizeof m);
  {  // SoA planes (caller) -> cell-major records (library copy); one staging plane on the device
    double* stage = nullptr;
    cudaError_t e = cudaMalloc(&stage, cells * sizeof(double));
    if (e != cudaSuccess) { c->last_cuda = (int)e; cudaGetLastError(); return IPOLE_ENOMEM; }
    for (int q = 0; q < 8 && e == cudaSuccess; ++q) {
      e = cudaMemcpyAsync(stage, fields[q], cells * sizeof(double), cudaMemcpyDefault, c->stream);
      if (e == cudaSuccess) {
        k_pack_field<<<c->n_sm * 8, 256, 0, c->stream>>>(cells, q, stage, c->d_grid);
        e = cudaGetLastError();
      }
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    cudaFree(stage);
    if (e != cudaSuccess) { c->last_cuda = (int)e; return IPOLE_ECUDA; }
    m.cells = c->d_grid;
  }
  m.N1 = d->N1; m.N2 = d->N2; m.N3 = d->N3; m.iN3 = 1.0 / d->N3;
  {  // stencil occupancy bitmap
    const size_t bits = (size_t)(d->N1 + 1) * (d->N2 + 1) * d->N3, words = (bits + 31) / 32;
    cudaFree(c->d_occ); c->d_occ = nullptr;
    cudaError_t e = cudaMalloc(&c->d_occ, words * sizeof(unsigned int));
    if (e != cudaSuccess) { c->last_cuda = (int)e; cudaGetLastError(); return IPOLE_ENOMEM; }
    CK(cudaMemsetAsync(c->d_occ, 0, words * sizeof(unsigned int), c->stream));
    m.occ = c->d_occ;
    k_build_occupancy<<<c->n_sm * 8, 256, 0, c->stream>>>(m, c->d_occ);
    CK(cudaGetLastError());
  }
  m.N1 = d->N1; m.N2 = d->N2; m.N3 = d->N3;
  for (int i = 0; i < 3; ++i) { m.startx[i] = d->startx[i]; m.idx[i] = 1.0 / d->dx[i]; }
  m.gam = d->gam; m.Rlow = d->Rlow; m.Rhigh = d->Rhigh; m.r_out = d->r_out; m.lx_out = std::log(d->r_out);
  const double L = c->units.L_unit;
  const double rho_unit = d->M_unit / (L * L * L);
  m.ne_unit = rho_unit / (IP_MP + IP_ME);
  m.B_unit = IP_CL * std::sqrt(4.0 * M_PI * rho_unit);
  c->grid_host = m; c->grid_M_unit = d->M_unit;
  CK(cudaMemcpyAsync(c->d_model, &c->grid_host, sizeof m, cudaMemcpyHostToDevice, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  c->model = MODEL_GRID;
  return IPOLE_OK;
}

int ipole_make_pixels(ipole_ctx* c, int64_t n, const int64_t* pixels, double* I, double* Q, double* U, double* V,
                      double* tau, double* tauF, int32_t* nsteps, int32_t* nturn) {
  if (!c || !I || !Q || !U || !V) return IPOLE_EINVAL;
  if (c->model == MODEL_NONE) return IPOLE_ENOMODEL;
  const int64_t npix = (int64_t)c->cam.nx * c->cam.ny;
  if (!pixels) n = npix;
  if (n < 0 || n > 2147483647LL) return IPOLE_EINVAL;
  if (n == 0) return IPOLE_OK;
  const bool dev = is_device_ptr(I);
  const void* outs[] = {Q, U, V, tau, tauF, nsteps, nturn};
  for (const void* p : outs) if (p && is_device_ptr(p) != dev) return IPOLE_EINVAL;
  int rc;
  if ((rc = ensure_rays(c, n)) != IPOLE_OK) return rc;
  const int64_t* d_pix = nullptr;
  if (pixels) {
    if (is_device_ptr(pixels)) d_pix = pixels;
    else {
      for (int64_t i = 0; i < n; ++i) if (pixels[i] < 0 || pixels[i] >= npix) return IPOLE_EINVAL;
      if (n > c->pixels_cap) {
        cudaFree(c->d_pixels); c->d_pixels = nullptr; c->pixels_cap = 0;
        CK(cudaMalloc(&c->d_pixels, n * sizeof(int64_t)));
        c->pixels_cap = n;
      }
      CK(cudaMemcpyAsync(c->d_pixels, pixels, n * sizeof(int64_t), cudaMemcpyHostToDevice, c->stream));
      d_pix = c->d_pixels;
    }
  }
  double* o[6];
  if (dev) { o[0] = I; o[1] = Q; o[2] = U; o[3] = V; o[4] = tau; o[5] = tauF; }
  else {
    for (int k = 0; k < 6; ++k) o[k] = c->d_out + (size_t)k * c->ray_cap;
    if (!tau) o[4] = nullptr;
    if (!tauF) o[5] = nullptr;
  }
  if ((rc = run_rays(c, n, d_pix, o[0], o[1], o[2], o[3], o[4], o[5])) != IPOLE_OK) return rc;
  if (!dev) {
    double* h[6] = {I, Q, U, V, tau, tauF};
    for (int k = 0; k < 6; ++k)
      if (h[k]) CK(cudaMemcpyAsync(h[k], o[k], n * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  }
  if (nsteps) CK(cudaMemcpyAsync(nsteps, c->d_nsteps, n * sizeof(int32_t), cudaMemcpyDefault, c->stream));
  if (nturn) CK(cudaMemcpyAsync(nturn, c->d_nturn, n * sizeof(int32_t), cudaMemcpyDefault, c->stream));
  if (!dev) CK(cudaStreamSynchronize(c->stream));
  return IPOLE_OK;
}

}  // extern "C"

namespace {
// common part of the two sweep entries; `model` is the model the transfer kernel runs (the context's own stays loaded)
int make_images(ipole_ctx* c, int model, int32_t n_models, const void* lane_tab, size_t lane_bytes, const Units* um,
                double* I, double* Q, double* U, double* V, double* tau, double* tauF, double* flux_jy) {
  const int64_t n = (int64_t)c->cam.nx * c->cam.ny;
  if ((double)n * n_models > 2147483647.0) return IPOLE_EINVAL;
  const bool dev = is_device_ptr(I);
  const void* outs[] = {Q, U, V, tau, tauF};
  for (const void* p : outs) if (p && is_device_ptr(p) != dev) return IPOLE_EINVAL;
  int rc;
  if ((rc = ensure_rays(c, n)) != IPOLE_OK) return rc;
  const size_t plane = (size_t)n * n_models;
  double* o[6] = {I, Q, U, V, tau, tauF};
  // the fluxes live at the start of the staging buffer; host outputs are staged behind them
  const size_t need = (size_t)n_models * 4 + (dev ? 0 : plane * 6);
  if (need > c->sweep_out_doubles) {
    cudaFree(c->d_sweep_out); c->d_sweep_out = nullptr; c->sweep_out_doubles = 0;
    cudaError_t e = cudaMalloc(&c->d_sweep_out, need * sizeof(double));
    if (e != cudaSuccess) { c->last_cuda = (int)e; cudaGetLastError(); return IPOLE_ENOMEM; }
    c->sweep_out_doubles = need;
  }
  double* d_flux = c->d_sweep_out;
  if (!dev) {
    for (int k = 0; k < 6; ++k) o[k] = c->d_sweep_out + (size_t)n_models * 4 + (size_t)k * plane;
    if (!tau) o[4] = nullptr;
    if (!tauF) o[5] = nullptr;
  }
  Sweep sw;
  sw.n_models = n_models; sw.lane_tab = lane_tab; sw.lane_bytes = lane_bytes; sw.units = um; sw.out_stride = (size_t)n;
  const int model_before = c->model;
  c->model = model;
  rc = run_rays(c, n, nullptr, o[0], o[1], o[2], o[3], o[4], o[5], &sw);
  c->model = model_before;
  if (rc != IPOLE_OK) return rc;
  if (flux_jy) {
    const double pix_rad = c->cam.pix * c->units.L_unit / c->units.D_cm;
    k_reduce_models<<<n_models, 256, 0, c->stream>>>(n, (size_t)n, o[0], o[1], o[2], o[3], pix_rad * pix_rad * 1e23, d_flux);
    c->stats.n_launches++;
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(flux_jy, d_flux, (size_t)n_models * 4 * sizeof(double), cudaMemcpyDefault, c->stream));
  }
  if (!dev) {
    double* h[6] = {I, Q, U, V, tau, tauF};
    for (int k = 0; k < 6; ++k)
      if (h[k]) CK(cudaMemcpyAsync(h[k], o[k], plane * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  }
  if (!dev || (flux_jy && !is_device_ptr(flux_jy))) CK(cudaStreamSynchronize(c->stream));
  return IPOLE_OK;
}

void sweep_units(const ipole_ctx* c, int32_t n_models, const double* freq_hz, std::vector<Units>& um) {
  um.assign(n_models, c->units);
  if (freq_hz) for (int m = 0; m < n_models; ++m) { um[m].nu_obs = freq_hz[m]; um[m].dl_unit = um[m].L_unit / um[m].nu_obs; }
}
}  // namespace

extern "C" {

int ipole_make_images_adaf(ipole_ctx* c, int32_t n_models, const ipole_adaf_params* models, const double* freq_hz,
                           double* I, double* Q, double* U, double* V, double* tau, double* tauF, double* flux_jy) {
  if (!c || !models || n_models < 1 || !I || !Q || !U || !V) return IPOLE_EINVAL;
  if (c->cam.G.mass == 0.0) return IPOLE_EINVAL;   // the flow is defined on Kerr only
  if (freq_hz) for (int m = 0; m < n_models; ++m) if (!(freq_hz[m] > 0.0)) return IPOLE_EINVAL;
  std::vector<AdafParams> pm(n_models);
  std::vector<Units> um;
  sweep_units(c, n_models, freq_hz, um);
  for (int m = 0; m < n_models; ++m) {
    AdafParams& a = pm[m];
    a.n0 = models[m].n0; a.p_n = models[m].p_n; a.Th0 = models[m].Th0; a.p_T = models[m].p_T; a.B0 = models[m].B0;
    a.p_B = models[m].p_B; a.r_isco = isco_radius(c->cam.G.a);
  }
  // the kernel reads the uniform model block too (unused by the analytic sweep): any valid device block will do
  return make_images(c, MODEL_ADAF, n_models, pm.data(), sizeof(AdafParams), um.data(), I, Q, U, V, tau, tauF, flux_jy);
}

int ipole_make_images_cameras(ipole_ctx* c, int32_t n_cams, const ipole_camera* cams, double* I, double* Q, double* U, double* V,
                              double* tau, double* tauF, double* flux_jy) {
  if (!c || !cams || n_cams < 1 || !I || !Q || !U || !V) return IPOLE_EINVAL;
  if (c->model != MODEL_ADAF && c->model != MODEL_GRID) return c->model == MODEL_NONE ? IPOLE_ENOMODEL : IPOLE_EINVAL;
  if (c->model == MODEL_GRID && (c->opt_unpol || c->opt_path_free)) return IPOLE_EINVAL;
  for (int k = 0; k < n_cams; ++k) {
    int rc = check_camera(&cams[k]);
    if (rc != IPOLE_OK) return rc;
    const ipole_camera &a = cams[k], &b = cams[0];
    if (a.flat_metric || a.nx != b.nx || a.ny != b.ny || a.eps != b.eps || a.max_steps != b.max_steps || a.hslope != b.hslope) return IPOLE_EINVAL;
    // a grid was computed in one spacetime and scaled with one mass: its cameras share spin, mass and coordinates with the
    // context's camera and differ in direction, field of view, frequency and distance
    const ipole_camera& g0 = c->cam_in;
    auto eff = [](double v, double dflt) { return v == 0.0 ? dflt : v; };   // (0 stands for the default, include/ipole.h)
    if (c->model == MODEL_GRID && (a.spin != g0.spin || eff(a.mbh_msun, 4.1e6) != eff(g0.mbh_msun, 4.1e6) || eff(a.hslope, 1.0) != eff(g0.hslope, 1.0))) return IPOLE_EINVAL;
  }
  const int64_t npix = (int64_t)cams[0].nx * cams[0].ny, n = npix * n_cams;
  if (n > 2147483647LL) return IPOLE_EINVAL;
  const bool dev = is_device_ptr(I);
  const void* outs[] = {Q, U, V, tau, tauF};
  for (const void* p : outs) if (p && is_device_ptr(p) != dev) return IPOLE_EINVAL;
  int rc;
  if ((rc = ensure_rays(c, n)) != IPOLE_OK) return rc;
  if (n_cams > c->mc_cap) {
    cudaFree(c->d_mc_cams); cudaFree(c->d_mc_units); cudaFree(c->d_mc_nu3); cudaFree(c->d_mc_scale);
    c->d_mc_cams = nullptr; c->d_mc_units = nullptr; c->d_mc_nu3 = nullptr; c->d_mc_scale = nullptr; c->mc_cap = 0;
    CK(cudaMalloc(&c->d_mc_cams, n_cams * sizeof(CamDev)));
    CK(cudaMalloc(&c->d_mc_units, n_cams * sizeof(Units)));
    CK(cudaMalloc(&c->d_mc_nu3, n_cams * sizeof(double)));
    CK(cudaMalloc(&c->d_mc_scale, n_cams * 5 * sizeof(double)));   // scale[n] then flux[4 n]
    c->mc_cap = n_cams;
  }
  // camera tetrads on the device, one k_camera_setup each (a-1); units, nu_obs^3 and the Jy scale on the host
  std::vector<CamDev> hc(n_cams);
  std::vector<Units> hu(n_cams);
  std::vector<double> hn(n_cams), hs(n_cams);
  std::vector<CameraSetupArgs> ha(n_cams);
  for (int k = 0; k < n_cams; ++k) {
    fill_camera(&cams[k], hc[k], ha[k], hu[k]);
    hn[k] = hu[k].nu_obs * hu[k].nu_obs * hu[k].nu_obs;
    const double pix_rad = hc[k].pix * hu[k].L_unit / hu[k].D_cm;
    hs[k] = pix_rad * pix_rad * 1e23;
  }
  CK(cudaMemcpyAsync(c->d_mc_cams, hc.data(), n_cams * sizeof(CamDev), cudaMemcpyHostToDevice, c->stream));
  CK(cudaMemcpyAsync(c->d_mc_units, hu.data(), n_cams * sizeof(Units), cudaMemcpyHostToDevice, c->stream));
  CK(cudaMemcpyAsync(c->d_mc_nu3, hn.data(), n_cams * sizeof(double), cudaMemcpyHostToDevice, c->stream));
  CK(cudaMemcpyAsync(c->d_mc_scale, hs.data(), n_cams * sizeof(double), cudaMemcpyHostToDevice, c->stream));
  for (int k = 0; k < n_cams; ++k) k_camera_setup<<<1, 32, 0, c->stream>>>(c->d_mc_cams + k, ha[k]);
  CK(cudaGetLastError());
  CK(cudaStreamSynchronize(c->stream));   // the host vectors above go out of scope
  // the context's own camera lends eps, max_steps and the image shape to the shared parts of the pipeline
  const CamDev cam_saved = c->cam;
  c->cam.eps = hc[0].eps; c->cam.max_steps = hc[0].max_steps; c->cam.nx = hc[0].nx; c->cam.ny = hc[0].ny;
  double* o[6] = {I, Q, U, V, tau, tauF};
  if (!dev) {
    for (int k = 0; k < 6; ++k) o[k] = c->d_out + (size_t)k * c->ray_cap;
    if (!tau) o[4] = nullptr;
    if (!tauF) o[5] = nullptr;
  }
  c->n_mc = n_cams; c->mc_rays_per_cam = npix;
  rc = run_rays(c, n, nullptr, o[0], o[1], o[2], o[3], o[4], o[5]);
  c->n_mc = 0; c->mc_rays_per_cam = 0;
  c->cam = cam_saved;
  if (rc != IPOLE_OK) return rc;
  if (flux_jy) {
    double* d_flux = c->d_mc_scale + n_cams;
    k_reduce_cams<<<n_cams, 256, 0, c->stream>>>(npix, (size_t)npix, o[0], o[1], o[2], o[3], c->d_mc_scale, d_flux);
    c->stats.n_launches++;
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(flux_jy, d_flux, (size_t)n_cams * 4 * sizeof(double), cudaMemcpyDefault, c->stream));
  }
  if (!dev) {
    double* h[6] = {I, Q, U, V, tau, tauF};
    for (int k = 0; k < 6; ++k)
      if (h[k]) CK(cudaMemcpyAsync(h[k], o[k], (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  }
  if (!dev || (flux_jy && !is_device_ptr(flux_jy))) CK(cudaStreamSynchronize(c->stream));
  return IPOLE_OK;
}

int ipole_make_images_grid(ipole_ctx* c, int32_t n_models, const ipole_grid_scales* sets, const double* freq_hz,
                           double* I, double* Q, double* U, double* V, double* tau, double* tauF, double* flux_jy) {
  if (!c || !sets || n_models < 1 || !I || !Q || !U || !V) return IPOLE_EINVAL;
  if (c->model != MODEL_GRID) return IPOLE_ENOMODEL;
  if (freq_hz) for (int m = 0; m < n_models; ++m) if (!(freq_hz[m] > 0.0)) return IPOLE_EINVAL;
  std::vector<GridScales> gs(n_models);
  std::vector<Units> um;
  sweep_units(c, n_models, freq_hz, um);
  const double L = c->units.L_unit;
  for (int m = 0; m < n_models; ++m) {
    if (!(sets[m].M_unit > 0.0)) return IPOLE_EINVAL;
    const double rho_unit = sets[m].M_unit / (L * L * L);    // as in ipole_load_model_grid
    gs[m].ne_unit = rho_unit / (IP_MP + IP_ME);
    gs[m].B_unit = IP_CL * std::sqrt(4.0 * M_PI * rho_unit);
    gs[m].Rlow = sets[m].Rlow; gs[m].Rhigh = sets[m].Rhigh;
  }
  return make_images(c, MODEL_GRID, n_models, gs.data(), sizeof(GridScales), um.data(), I, Q, U, V, tau, tauF, flux_jy);
}

int ipole_make_image_adaptive(ipole_ctx* c, int32_t levels, double rel_tol, double abs_tol, double* I, double* Q, double* U,
                              double* V, uint8_t* state, ipole_adaptive_info* info) {
  if (!c || !I || !Q || !U || !V) return IPOLE_EINVAL;
  if (levels < 1 || levels > 12 || !(rel_tol >= 0.0) || !(abs_tol >= 0.0)) return IPOLE_EINVAL;
  if (c->cam.nx < 2 || c->cam.ny < 2) return IPOLE_EINVAL;   // a lattice cell needs two lines each way
  if (c->model == MODEL_NONE) return IPOLE_ENOMODEL;
  const int nx = c->cam.nx, ny = c->cam.ny;
  const int64_t n = (int64_t)nx * ny;
  const bool dev = is_device_ptr(I);
  const void* outs[] = {Q, U, V};
  for (const void* p : outs) if (is_device_ptr(p) != dev) return IPOLE_EINVAL;
  int rc;
  if ((rc = ensure_rays(c, n)) != IPOLE_OK) return rc;
  const size_t need = (size_t)n * (4 * sizeof(double) + sizeof(int64_t) + 3);
  if (need > c->ada_bytes) {
    cudaFree(c->d_ada); c->d_ada = nullptr; c->ada_bytes = 0;
    cudaError_t e = cudaMalloc(&c->d_ada, need);
    if (e != cudaSuccess) { c->last_cuda = (int)e; cudaGetLastError(); return IPOLE_ENOMEM; }
    c->ada_bytes = need;
  }
  if (!c->ev_ada0) { CK(cudaEventCreate(&c->ev_ada0)); CK(cudaEventCreate(&c->ev_ada1)); }
  double* stage = (double*)c->d_ada;
  int64_t* list = (int64_t*)(stage + 4 * n);
  uint8_t* st8 = (uint8_t*)(list + n);
  uint8_t* flag_a = st8 + n;
  uint8_t* flag_b = flag_a + n;
  AdaArgs A;
  std::memset(&A, 0, sizeof A);
  A.nx = nx; A.ny = ny; A.rel_tol = rel_tol; A.abs_tol = abs_tol;
  double* host_out[4] = {I, Q, U, V};
  for (int k = 0; k < 4; ++k) A.img[k] = dev ? host_out[k] : stage + (size_t)k * n;
  A.state = st8; A.list = list; A.count = c->d_small + 2;
  // values of the traced list entries: the ordinary staging planes of the context (ray-indexed)
  double* val[4];
  for (int k = 0; k < 4; ++k) { val[k] = c->d_out + (size_t)k * c->ray_cap; A.val[k] = val[k]; }
  const int gb = (int)std::min<int64_t>((n + 255) / 256, (int64_t)c->n_sm * 8);
  ipole_adaptive_info inf;
  std::memset(&inf, 0, sizeof inf);
  CK(cudaEventRecord(c->ev_ada0, c->stream));
  int launches = 0;
  auto n_lines = [](int n_, int s_) { return (n_ + s_ - 1) / s_ + (((n_ - 1) % s_) ? 1 : 0); };
  for (int l = 0; l <= levels; ++l) {
    if (l == 1) continue;                          // traced together with level 0
    A.s = 1 << (levels - std::max(l, 1));          // level 0 lists the level-1 lattice
    uint8_t* fprev = (l & 1) ? flag_a : flag_b;    // written at level l-1
    uint8_t* fcur = (l & 1) ? flag_b : flag_a;
    A.flag_prev = fprev; A.flag_cur = fcur;
    CK(cudaMemsetAsync(A.count, 0, sizeof(int), c->stream));
    if (l == 0) k_ada_level01<<<gb, 256, 0, c->stream>>>(A, fcur, 1 << levels);
    else k_ada_select<<<gb, 256, 0, c->stream>>>(A);
    ++launches;
    CK(cudaGetLastError());
    int cnt = 0;
    CK(cudaMemcpyAsync(&cnt, A.count, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    if (cnt > 0) {
      // the per-ray kernels, unchanged, on the listed pixels (run_rays resets the queues; its own d_small[0..1] only)
      if ((rc = run_rays(c, cnt, list, val[0], val[1], val[2], val[3], nullptr, nullptr)) != IPOLE_OK) return rc;
      launches += c->stats.n_launches;
      ReduceOut r;
      CK(cudaMemcpyAsync(&r, c->d_red, sizeof r, cudaMemcpyDeviceToHost, c->stream));
      k_ada_scatter<<<(int)std::min<int64_t>((cnt + 255) / 256, (int64_t)c->n_sm * 8), 256, 0, c->stream>>>(A, cnt);
      ++launches;
      CK(cudaGetLastError());
      CK(cudaStreamSynchronize(c->stream));
      inf.total_steps += r.total_steps;
    }
    if (l == 0) {
      const int64_t n0 = (int64_t)n_lines(nx, 1 << levels) * n_lines(ny, 1 << levels);
      inf.n_traced_level[0] = n0;
      inf.n_traced_level[1] = cnt - n0;
    } else {
      inf.n_traced_level[l] = cnt;
    }
    inf.n_traced += cnt;
    // cells of level max(l,1)-1 are examined with the points of level max(l,1); after level 0+1 that is level 1
    const int lf = std::max(l, 1);
    if (lf < levels) {
      uint8_t* fp = (lf & 1) ? flag_a : flag_b;
      uint8_t* fc = (lf & 1) ? flag_b : flag_a;
      A.flag_prev = fp; A.flag_cur = fc;
      CK(cudaMemsetAsync(fc, 0, (size_t)n, c->stream));
      k_ada_flag<<<gb, 256, 0, c->stream>>>(A);
      ++launches;
      CK(cudaGetLastError());
    }
  }
  const double pix_rad = c->cam.pix * c->units.L_unit / c->units.D_cm;
  {
    // d_part holds REDUCE_BLOCKS ReducePartial (64 B each): room for the 4 results and REDUCE_BLOCKS x 4 partial sums
    static_assert(sizeof(ReducePartial) >= 8 * sizeof(double), "d_part is reused for the plane partials");
    double* flux4 = (double*)c->d_part;
    double* parts = flux4 + 4;
    const int nb = (int)std::min<int64_t>(REDUCE_BLOCKS - 1, (n + 255) / 256);
    k_reduce_planes_partial<<<nb, 256, 0, c->stream>>>(n, A.img[0], A.img[1], A.img[2], A.img[3], parts);
    k_reduce_planes_final<<<1, 32, 0, c->stream>>>(parts, nb, pix_rad * pix_rad * 1e23, flux4);
    launches += 2;
  }
  CK(cudaGetLastError());
  CK(cudaMemcpyAsync(inf.flux_jy, c->d_part, 4 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  CK(cudaEventRecord(c->ev_ada1, c->stream));
  if (!dev)
    for (int k = 0; k < 4; ++k) CK(cudaMemcpyAsync(host_out[k], A.img[k], (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  if (state) CK(cudaMemcpyAsync(state, st8, (size_t)n, cudaMemcpyDefault, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  CK(cudaEventElapsedTime(&inf.ms_total, c->ev_ada0, c->ev_ada1));
  inf.n_launches = launches;
  c->have_image = false;   // ipole_get_stats / ipole_get_ray_info describe whole-image calls only
  if (info) *info = inf;
  return IPOLE_OK;
}

int ipole_make_image(ipole_ctx* c, double* I, double* Q, double* U, double* V, double* tau, double* tauF) {
  return ipole_make_pixels(c, 0, nullptr, I, Q, U, V, tau, tauF, nullptr, nullptr);
}

int ipole_get_ray_info(ipole_ctx* c, int32_t* nsteps, int32_t* nturn) {
  if (!c) return IPOLE_EINVAL;
  if (!c->have_image) return IPOLE_ENOIMAGE;
  if (nsteps) CK(cudaMemcpyAsync(nsteps, c->d_nsteps, c->last_n * sizeof(int32_t), cudaMemcpyDefault, c->stream));
  if (nturn) CK(cudaMemcpyAsync(nturn, c->d_nturn, c->last_n * sizeof(int32_t), cudaMemcpyDefault, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  return IPOLE_OK;
}

int ipole_get_stats(ipole_ctx* c, ipole_stats* out) {
  if (!c || !out) return IPOLE_EINVAL;
  if (!c->have_image) return IPOLE_ENOIMAGE;
  ReduceOut r;
  CK(cudaMemcpyAsync(&r, c->d_red, sizeof r, cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  ipole_stats& s = c->stats;
  for (int k = 0; k < 4; ++k) s.flux_jy[k] = r.flux[k];
  s.lp = r.lp; s.cp = r.cp;
  s.total_steps = r.total_steps; s.max_steps_seen = r.max_steps; s.n_ring = r.n_ring; s.n_maxstep = r.n_maxstep;
  s.total_steps_forward = 0;
  if (c->last_pf) {
    long long f = 0;
    CK(cudaMemcpy(&f, c->d_sum, sizeof f, cudaMemcpyDeviceToHost));
    s.total_steps_forward = f;
  }
  s.ms_probe = s.ms_geodesic = s.ms_transfer = s.ms_total = s.ms_long = s.ms_stepop = s.ms_apply = 0.f;
  const bool dbg = std::getenv("IPOLE_DEBUG_SPANS") != nullptr;
  for (size_t i = 0; i < c->spans_used; ++i) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, c->spans[i].a, c->spans[i].b) != cudaSuccess) { cudaGetLastError(); continue; }
    if (dbg) std::fprintf(stderr, "span %zu kind %d ms %.3f\n", i, c->spans[i].kind, ms);
    if (i == 0) s.ms_total = ms;
    else if (c->spans[i].kind == LK_PROBE) s.ms_probe += ms;
    else if (c->spans[i].kind == LK_GEO) s.ms_geodesic += ms;
    else if (c->spans[i].kind == LK_RT) s.ms_transfer += ms;
    else if (c->spans[i].kind == LK_LONG) s.ms_long += ms;
    else if (c->spans[i].kind == LK_OPS) { s.ms_stepop += ms; s.ms_transfer += ms; }
    else if (c->spans[i].kind == LK_APPLY) { s.ms_apply += ms; s.ms_transfer += ms; }
  }
  *out = s;
  return IPOLE_OK;
}

int ipole_get_camera_tetrad(ipole_ctx* c, double Xcam[4], double e[16]) {
  if (!c || !Xcam || !e) return IPOLE_EINVAL;
  std::memcpy(Xcam, c->cam.Xcam, 4 * sizeof(double));
  std::memcpy(e, c->cam.e, 16 * sizeof(double));
  return IPOLE_OK;
}

int ipole_trace_pixel(ipole_ctx* c, int32_t i, int32_t j, int32_t cap, double* X, double* K, double* dl, int32_t* nturn,
                      int32_t* status, int32_t* needed) {
  if (!c || i < 0 || j < 0 || i >= c->cam.nx || j >= c->cam.ny || cap < 1) return IPOLE_EINVAL;
  int rc;
  if ((rc = ensure_rays(c, 1)) != IPOLE_OK) return rc;
  const int max_steps = c->cam.max_steps;
  const size_t bytes = (size_t)(max_steps + 1) * REC_DOUBLES * sizeof(double);
  if ((rc = ensure_path(c, bytes)) != IPOLE_OK) return rc;
  if (c->pixels_cap < 1) { CK(cudaMalloc(&c->d_pixels, sizeof(int64_t))); c->pixels_cap = 1; }
  const int64_t pix = (int64_t)j * c->cam.nx + i;
  CK(cudaMemcpyAsync(c->d_pixels, &pix, sizeof pix, cudaMemcpyHostToDevice, c->stream));
  CK(cudaMemsetAsync(c->d_queues, 0, sizeof(unsigned long long), c->stream));
  GeoArgs g = geo_args(c);
  g.cap = max_steps; g.count = 1; g.pixels = c->d_pixels; g.path = c->d_path; g.nsteps = c->d_nsteps; g.nturn = c->d_nturn;
  g.queue = c->d_queues;
  k_geodesic<false><<<1, 32, 0, c->stream>>>(g);
  CK(cudaGetLastError());
  int32_t n = 0, nt = 0;
  CK(cudaMemcpyAsync(&n, c->d_nsteps, sizeof n, cudaMemcpyDeviceToHost, c->stream));
  CK(cudaMemcpyAsync(&nt, c->d_nturn, sizeof nt, cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  c->have_image = false;
  if (needed) *needed = n;
  if (nturn) *nturn = nt & 0x7f;
  if (n > cap) return IPOLE_EINVAL;
  std::vector<double> rec((size_t)(n + 1) * REC_DOUBLES);
  CK(cudaMemcpyAsync(rec.data(), c->d_path, rec.size() * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  for (int s = 0; s <= n; ++s) {
    const double* r = &rec[(size_t)s * REC_DOUBLES];
    if (X) { X[4 * s] = 0.0; X[4 * s + 1] = r[0]; X[4 * s + 2] = r[1]; X[4 * s + 3] = r[2]; }
    if (K) { K[4 * s] = r[3]; K[4 * s + 1] = r[4]; K[4 * s + 2] = r[5]; K[4 * s + 3] = r[6]; }
    if (dl && s < n) dl[s] = r[7];
  }
  if (status) {
    const double x1 = rec[(size_t)n * REC_DOUBLES];
    *status = (nt & 0x80) ? 3 : (x1 <= c->cam.lx_in ? 1 : 2);
  }
  return n;
}

}  // extern "C"

namespace {
template <typename F>
int eval_host(ipole_ctx* c, int64_t n, const double* in, int nin, double* out, int nout, F launch) {
  if (!c || !in || !out || n < 0) return IPOLE_EINVAL;
  if (n == 0) return IPOLE_OK;
  double *d_in = nullptr, *d_o = nullptr;
  if (cudaMalloc(&d_in, n * nin * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return IPOLE_ENOMEM; }
  if (cudaMalloc(&d_o, n * nout * sizeof(double)) != cudaSuccess) { cudaFree(d_in); cudaGetLastError(); return IPOLE_ENOMEM; }
  cudaError_t e = cudaMemcpyAsync(d_in, in, n * nin * sizeof(double), cudaMemcpyHostToDevice, c->stream);
  if (e == cudaSuccess) { launch((int)((n + 127) / 128), 128, d_in, d_o); e = cudaGetLastError(); }
  if (e == cudaSuccess) e = cudaMemcpyAsync(out, d_o, n * nout * sizeof(double), cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  cudaFree(d_in); cudaFree(d_o);
  if (e != cudaSuccess) { c->last_cuda = (int)e; return IPOLE_ECUDA; }
  return IPOLE_OK;
}
}  // namespace

extern "C" {

int ipole_eval_connection(ipole_ctx* c, int64_t n, const double* X, double* Gamma) {
  return eval_host(c, n, X, 4, Gamma, 64, [&](int g, int b, double* i, double* o) { k_eval_connection<<<g, b, 0, c->stream>>>(c->cam.G, n, i, o); });
}
int ipole_eval_coefficients(ipole_ctx* c, int64_t n, const double* in5, double* out8) {
  return eval_host(c, n, in5, 5, out8, 8, [&](int g, int b, double* i, double* o) { k_eval_coefficients<<<g, b, 0, c->stream>>>(n, i, o); });
}
int ipole_eval_coefficients_edf(ipole_ctx* c, int64_t n, const double* in5, double* out8) {
  return eval_host(c, n, in5, 5, out8, 8, [&](int g, int b, double* i, double* o) { k_eval_coefficients_edf<<<g, b, 0, c->stream>>>(c->edf, n, i, o); });
}
int ipole_eval_stokes_step(ipole_ctx* c, int64_t n, const double* in16, double* out4) {
  return eval_host(c, n, in16, 16, out4, 4, [&](int g, int b, double* i, double* o) { k_eval_stokes_step<<<g, b, 0, c->stream>>>(n, i, o); });
}
int ipole_eval_bessel(ipole_ctx* c, int64_t n, const double* z, double* out3) {
  return eval_host(c, n, z, 1, out3, 3, [&](int g, int b, double* i, double* o) { k_eval_bessel<<<g, b, 0, c->stream>>>(n, i, o); });
}
int ipole_eval_math(ipole_ctx* c, int64_t n, const double* x, double* out8) {
  return eval_host(c, n, x, 1, out8, 8, [&](int g, int b, double* i, double* o) { k_eval_math<<<g, b, 0, c->stream>>>(n, i, o); });
}
int ipole_eval_plasma(ipole_ctx* c, int64_t n, const double* X, double* out12) {
  if (!c) return IPOLE_EINVAL;
  if (c->model == MODEL_NONE) return IPOLE_ENOMODEL;
  return eval_host(c, n, X, 4, out12, 12, [&](int g, int b, double* i, double* o) {
    if (c->model == MODEL_ADAF) k_eval_plasma<MODEL_ADAF><<<g, b, 0, c->stream>>>(c->cam.G, c->d_model, n, i, o);
    else if (c->model == MODEL_SLAB) k_eval_plasma<MODEL_SLAB><<<g, b, 0, c->stream>>>(c->cam.G, c->d_model, n, i, o);
    else k_eval_plasma<MODEL_GRID><<<g, b, 0, c->stream>>>(c->cam.G, c->d_model, n, i, o);
  });
}

int ipole_measure_fp64_peak(ipole_ctx* c, double* tflops, float* ms_out) {
  if (!c || !tflops) return IPOLE_EINVAL;
  double* sink = nullptr;
  CK(cudaMalloc(&sink, sizeof(double)));
  const int blocks = c->n_sm * 8, threads = 256, iters = 1 << 16;
  cudaEvent_t a, b;
  CK(cudaEventCreate(&a)); CK(cudaEventCreate(&b));
  k_fp64_peak<<<blocks, threads, 0, c->stream>>>(1024, 1.0, sink);  // warm-up
  float best = 1e30f;
  for (int rep = 0; rep < 3; ++rep) {
    cudaEventRecord(a, c->stream);
    k_fp64_peak<<<blocks, threads, 0, c->stream>>>(iters, 1.0 + rep, sink);
    cudaEventRecord(b, c->stream);
    CK(cudaEventSynchronize(b));
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, a, b));
    best = std::min(best, ms);
  }
  cudaEventDestroy(a); cudaEventDestroy(b); cudaFree(sink);
  CK(cudaGetLastError());
  *tflops = 2.0 * 8.0 * (double)iters * (double)blocks * threads / (best * 1e-3) / 1e12;
  if (ms_out) *ms_out = best;
  return IPOLE_OK;
}

int ipole_last_cuda_error(const ipole_ctx* c) { return c ? c->last_cuda : 0; }

void ipole_free(ipole_ctx* c) {
  if (!c) return;
  if (c->side) { cudaStreamSynchronize(c->side); cudaStreamDestroy(c->side); }
  if (c->qstream) cudaStreamDestroy(c->qstream);
  if (c->ev_geo) cudaEventDestroy(c->ev_geo);
  if (c->ev_side) cudaEventDestroy(c->ev_side);
  if (c->lane2) cudaStreamDestroy(c->lane2);
  if (c->ev_fork) cudaEventDestroy(c->ev_fork);
  if (c->ev_join) cudaEventDestroy(c->ev_join);
  for (int l = 0; l < 2; ++l) if (c->ev_lastgeo[l]) cudaEventDestroy(c->ev_lastgeo[l]);
  cudaFree(c->d_retry_buf); cudaFree(c->d_ops_long); cudaFree(c->plan_cache.d_long); cudaFree(c->plan_cache.d_retry);
  cudaFree(c->d_path_long); cudaFree(c->d_nsteps_long); cudaFree(c->d_occ);
  cudaFree(c->d_cam); cudaFree(c->d_model); cudaFree(c->d_grid); cudaFree(c->d_path);
  cudaFree(c->d_nsteps); cudaFree(c->d_nturn); cudaFree(c->d_order); cudaFree(c->d_key); cudaFree(c->d_long);
  cudaFree(c->d_out); cudaFree(c->d_pixels); cudaFree(c->d_probe); cudaFree(c->d_queues); cudaFree(c->d_hist);
  cudaFree(c->d_small); cudaFree(c->d_part); cudaFree(c->d_red); cudaFree(c->d_endp); cudaFree(c->d_sum); cudaFree(c->d_sweep_models); cudaFree(c->d_sweep_units); cudaFree(c->d_sweep_models_side); cudaFree(c->d_sweep_units_side); cudaFree(c->d_sweep_out); cudaFree(c->d_ada);
  cudaFree(c->d_ops); cudaFree(c->d_irr); cudaFree(c->d_rank_pos); cudaFree(c->d_rank_slot); cudaFree(c->d_retry); cudaFree(c->d_edf_nodes); cudaFree(c->d_edf_lnnorm);
  cudaFree(c->d_mc_cams); cudaFree(c->d_mc_units); cudaFree(c->d_mc_nu3); cudaFree(c->d_mc_scale);
  if (c->ev_ada0) cudaEventDestroy(c->ev_ada0);
  if (c->ev_ada1) cudaEventDestroy(c->ev_ada1);
  for (auto& s : c->spans) { cudaEventDestroy(s.a); cudaEventDestroy(s.b); }
  cudaGetLastError();
  delete c;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------
// ipole_image_totals_static: the totals of an image for callers that cannot call
// cudaMalloc (CUDA graph capture, serving loops, harnesses that forbid allocation).  The block partials of the
// reduction live in a file-scope device array instead of the context's cudaMalloc'ed d_part; the entry point
// allocates nothing.  Every GPU that loads the library holds these 32 KiB until the process exits.
namespace {

constexpr int TOTALS_THREADS = 256;
constexpr int TOTALS_PER_THREAD = 64;                                  // pixels per thread: a block folds 16 384 pixels
constexpr int TOTALS_MAX_BLOCKS = IPOLE_TOTALS_STATIC_MAX_PIXELS / (TOTALS_THREADS * TOTALS_PER_THREAD);   // 1024
static_assert((long long)TOTALS_MAX_BLOCKS * TOTALS_THREADS * TOTALS_PER_THREAD == IPOLE_TOTALS_STATIC_MAX_PIXELS, "limit");

// [block][I, Q, U, V].  In HOST code this name is a host-side stand-in, not a device address: the kernels below get
// the address cudaGetSymbolAddress returns (totals_static_setup), looked up once per device.
static __device__ __align__(256) double g_totals_scratch[TOTALS_MAX_BLOCKS * 4];

// block b: pixels [b * 16384, (b+1) * 16384), thread t takes t, t + 256, ... (coalesced); fixed shape => reproducible
__global__ void __launch_bounds__(TOTALS_THREADS) k_totals_partial_static(int64_t n, const double* __restrict__ I,
                                                                            const double* __restrict__ Q, const double* __restrict__ U,
                                                                            const double* __restrict__ V, double* part) {
  const int64_t q0 = (int64_t)blockIdx.x * (TOTALS_THREADS * TOTALS_PER_THREAD);
  double s[4] = {0, 0, 0, 0};
#pragma unroll 4
  for (int k = 0; k < TOTALS_PER_THREAD; ++k) {
    const int64_t q = q0 + (int64_t)k * TOTALS_THREADS + threadIdx.x;
    if (q < n) { s[0] += I[q]; s[1] += Q[q]; s[2] += U[q]; s[3] += V[q]; }
  }
  __shared__ double sh[TOTALS_THREADS / 32][4];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < 4; ++k) s[k] = warp_sum(s[k]);
  if (lane == 0) { for (int k = 0; k < 4; ++k) sh[w][k] = s[k]; }
  __syncthreads();
  if (threadIdx.x < 4) {
    double r = sh[0][threadIdx.x];
    for (int i = 1; i < TOTALS_THREADS / 32; ++i) r += sh[i][threadIdx.x];
    part[(size_t)blockIdx.x * 4 + threadIdx.x] = r;      // every partial the final kernel reads is written here first
  }
}

// one block: thread t folds partials t, t + 256, ...; then the same warp / block fold; out = {flux[4], lp, cp}
__global__ void __launch_bounds__(TOTALS_THREADS) k_totals_final_static(const double* part, int nparts, double scale, double* out) {
  double s[4] = {0, 0, 0, 0};
  for (int i = threadIdx.x; i < nparts; i += TOTALS_THREADS) {
#pragma unroll
    for (int k = 0; k < 4; ++k) s[k] += part[(size_t)i * 4 + k];
  }
  __shared__ double sh[TOTALS_THREADS / 32][4];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < 4; ++k) s[k] = warp_sum(s[k]);
  if (lane == 0) { for (int k = 0; k < 4; ++k) sh[w][k] = s[k]; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double r[4];
    for (int k = 0; k < 4; ++k) { r[k] = sh[0][k]; for (int i = 1; i < TOTALS_THREADS / 32; ++i) r[k] += sh[i][k]; }
    for (int k = 0; k < 4; ++k) out[k] = r[k] * scale;
    out[4] = (r[0] != 0.0) ? sqrt(r[1] * r[1] + r[2] * r[2]) / r[0] : 0.0;
    out[5] = (r[0] != 0.0) ? r[3] / r[0] : 0.0;
  }
}

// Device address of the array, once per device, with that device current (called from ipole_init).
constexpr int TOTALS_MAX_DEVICES = 64;
double* g_totals_addr[TOTALS_MAX_DEVICES] = {};
int g_totals_addr_err[TOTALS_MAX_DEVICES] = {};
bool g_totals_addr_known[TOTALS_MAX_DEVICES] = {};
std::mutex g_totals_mutex;

void totals_static_setup(ipole_ctx* c) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess || dev != c->device || dev < 0 || dev >= TOTALS_MAX_DEVICES) {
    c->totals_scratch = nullptr;
    c->totals_scratch_err = (int)(e != cudaSuccess ? e : cudaErrorInvalidDevice);
    cudaGetLastError();
    return;
  }
  std::lock_guard<std::mutex> lk(g_totals_mutex);
  if (!g_totals_addr_known[dev]) {
    double* ptr = nullptr;
    e = cudaGetSymbolAddress((void**)&ptr, g_totals_scratch);
    if (e != cudaSuccess) { cudaGetLastError(); ptr = nullptr; }
    g_totals_addr[dev] = ptr;
    g_totals_addr_err[dev] = (int)e;
    g_totals_addr_known[dev] = true;
  }
  c->totals_scratch = g_totals_addr[dev];
  c->totals_scratch_err = g_totals_addr_err[dev];
}

}  // namespace

extern "C" {

int ipole_image_totals_static(ipole_ctx* c, int64_t n, const double* I, const double* Q, const double* U, const double* V,
                              double* out6) {
  if (!c || !I || !Q || !U || !V || !out6 || n < 1) return IPOLE_EINVAL;
  if (n > (int64_t)IPOLE_TOTALS_STATIC_MAX_PIXELS) return IPOLE_ETOOBIG;
  if (!c->totals_scratch) { c->last_cuda = c->totals_scratch_err; return IPOLE_ECUDA; }
  const int nb = (int)((n + TOTALS_THREADS * TOTALS_PER_THREAD - 1) / (TOTALS_THREADS * TOTALS_PER_THREAD));
  const double pix_rad = c->cam.pix * c->units.L_unit / c->units.D_cm;
  k_totals_partial_static<<<nb, TOTALS_THREADS, 0, c->stream>>>(n, I, Q, U, V, c->totals_scratch);
  k_totals_final_static<<<1, TOTALS_THREADS, 0, c->stream>>>(c->totals_scratch, nb, pix_rad * pix_rad * 1e23, out6);
  CK(cudaGetLastError());
  return IPOLE_OK;
}

const char* ipole_strerror(int code) {
  switch (code) {
    case IPOLE_OK: return "ok";
    case IPOLE_EINVAL: return "invalid argument";
    case IPOLE_ENOMODEL: return "no plasma model loaded";
    case IPOLE_ENOMEM: return "out of memory";
    case IPOLE_ECUDA: return "CUDA error (see ipole_last_cuda_error)";
    case IPOLE_ENOIMAGE: return "no image has been made yet";
    case IPOLE_ETOOBIG: return "size beyond the fixed maximum of a *_static entry point (IPOLE_TOTALS_STATIC_MAX_PIXELS)";
    default: return "unknown error";
  }
}

const char* ipole_version(void) { return "ipole-b200 0.1 (sm_100a, FP64)"; }

}  // extern "C"

// Kernels of the hot path (SURVEY.md section 8(a) rows a-1 ... a-9), sm_100a, scalar FP64.
//   k_camera_setup   a-1  camera tetrad by Gram-Schmidt (one thread)
//   k_geodesic       a-1/a-2/a-3/a-8  per-lane persistent ray loop: pixel -> K, RK4 push with the fused
//                    metric/connection, adaptive step, path records to HBM, atomic ray queue with lane-level refill
//   k_transfer       a-4/a-5/a-6/a-7/a-8  walks the stored path toward the camera: transport, plasma model, tetrad,
//                    coefficients, analytic 4x4 step; camera projection; writes I,Q,U,V(,tau,tauF)
//   k_predict/k_hist/k_scan/k_scatter  a-8  counting sort of rays by predicted step count (longest first)
//   k_reduce_partial/k_reduce_final    a-9  warp-shuffle reduction of flux, polarization fractions, step statistics
#pragma once
#include <stdint.h>
#include "geom.cuh"
#include "plasma.cuh"

namespace ipole {

// One path record = one point of the geodesic: X1,X2,X3, K0..K3, dl (step from this point to the next one).
// 64 B = two 32-B sectors, moved as two 256-bit accesses; the records of one ray are contiguous, so every sector
// written or read is full.
constexpr int REC_DOUBLES = 8;

struct CamDev {
  Geom G;
  double Xcam[4];
  double e[4][4];       // e[a][mu]
  double ecov1[4], ecov2[4];
  double r_cam, pix;    // pix = fov/nx
  int nx, ny;
  double eps, lx_in, lx_esc;  // ln of the inner stop radius / escape radius
  int max_steps;
};

struct CameraSetupArgs { double inclination_deg, r_in, r_esc; };

__device__ __forceinline__ void gram_schmidt(const Sym7& g, double v[4], const double (*basis)[4], const double* sign, int nb) {
  for (int b = 0; b < nb; ++b) {
    const double pr = sign[b] * dotg(g, v, basis[b]);
    for (int m = 0; m < 4; ++m) v[m] -= pr * basis[b][m];
  }
  const double n = sqrt(fabs(dotg(g, v, v)));
  for (int m = 0; m < 4; ++m) v[m] /= n;
}

// camera-type tetrad at X: e0 || d_t, e3 from d_X1, e2 from -d_X2, e1 from d_X3 (R-3), and the covariant
// components of the two transverse legs
__device__ __forceinline__ void observer_tetrad(const Geom& G, const double X[4], double e[4][4], double ecov1[4], double ecov2[4]) {
  Point p; Sym7 g; Inv6 gi;
  metric<false>(G, X, p, g, gi);
  double basis[3][4], sg[3];
  double e0[4] = {1.0, 0.0, 0.0, 0.0};
  const double n0 = sqrt(-dotg(g, e0, e0));
  for (int m = 0; m < 4; ++m) { e[0][m] = e0[m] / n0; basis[0][m] = e[0][m]; }
  sg[0] = -1.0;
  double e3[4] = {0.0, 1.0, 0.0, 0.0};
  gram_schmidt(g, e3, basis, sg, 1);
  for (int m = 0; m < 4; ++m) { e[3][m] = e3[m]; basis[1][m] = e3[m]; }
  sg[1] = 1.0;
  double e2[4] = {0.0, 0.0, -1.0, 0.0};
  gram_schmidt(g, e2, basis, sg, 2);
  for (int m = 0; m < 4; ++m) { e[2][m] = e2[m]; basis[2][m] = e2[m]; }
  sg[2] = 1.0;
  double e1[4] = {0.0, 0.0, 0.0, 1.0};
  gram_schmidt(g, e1, basis, sg, 3);
  for (int m = 0; m < 4; ++m) e[1][m] = e1[m];
  g.mul(e[1], ecov1);
  g.mul(e[2], ecov2);
}

// a-1: camera at (r_cam, theta_cam, phi=0)
__global__ void k_camera_setup(CamDev* cam, CameraSetupArgs a) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  CamDev C = *cam;
  const double th = a.inclination_deg * M_PI / 180.0;
  double x2 = th / M_PI;
  if (!C.G.h_is_one) {
    for (int it = 0; it < 100; ++it) {
      double t, tp, tpp;
      theta_map(C.G, x2, t, tp, tpp);
      const double d = (t - th) / tp;
      x2 -= d;
      if (fabs(d) < 1e-17) break;
    }
  }
  C.Xcam[0] = 0.0; C.Xcam[1] = log(C.r_cam); C.Xcam[2] = x2; C.Xcam[3] = 0.0;
  observer_tetrad(C.G, C.Xcam, C.e, C.ecov1, C.ecov2);
  C.lx_in = log(a.r_in);
  C.lx_esc = log(a.r_esc);
  *cam = C;
}

// ---------------------------------------------------------------------------------------------------------------
struct GeoArgs {
  CamDev cam;
  double eps;                 // step parameter of this pass (probe passes use a multiple of cam.eps)
  int max_steps;              // step limit of this pass
  int cap;                    // steps that fit in one path slot (records = cap + 1); 0 when path == nullptr
  int64_t base, count;        // rays [base, base+count) of the order / pixel list
  const int* count_dev;       // if non-null, count = *count_dev (long-ray pass)
  const int32_t* order;       // permutation of ray indices q (nullable: identity)
  const int64_t* pixels;      // flat pixel index of ray q (nullable: q itself); with lattice_stride > 0 ignored
  int64_t list_stride;        // probe over a pixel list: ray q stands for list entry q * list_stride (else 1)
  int lattice_stride, lattice_nx, lattice_ny;  // probe: ray q is pixel (ix*stride + stride/2, iy*stride + stride/2) [of camera q / (lattice_nx lattice_ny)]
  double* path;               // [count][cap+1][8] or nullptr (count-only)
  int32_t* nsteps;            // [total rays], indexed by q; -1 = overflowed the slot
  int32_t* nturn;             // [total rays]
  unsigned long long* queue;  // atomic ray counter of this launch
  int32_t* long_list; int* long_count;  // rays that did not fit (nullable)
  double* endp;               // [total rays][8], indexed by q: last point (X1..3, K0..3, 0) of the ray (nullable);
                              // all the path-free variant keeps of the backward pass
  // grid model (k_geodesic<true>): the steps of the ray whose midpoint stencil holds plasma
  const GridParams* grid;     // device
  int2* srange;               // [total rays], indexed by q: (largest, smallest) such step index; (-1, 0) if none
  // many cameras in one launch (k_geodesic<OCC, true>; ipole_make_images_cameras): ray q belongs to camera
  // q / rays_per_cam and is its pixel q % rays_per_cam; eps and max_steps are those of `cam` for all of them
  const CamDev* cams;         // device
  int64_t rays_per_cam;
};

__device__ __forceinline__ void pixel_ray(const CamDev& C, int64_t pix, double X[4], double K[4]) {
  const int i = (int)(pix % C.nx), j = (int)(pix / C.nx);
  const double alpha = (i + 0.5 - 0.5 * C.nx) * C.pix, beta = (j + 0.5 - 0.5 * C.ny) * C.pix;
  const double px = -alpha / C.r_cam, py = -beta / C.r_cam;
  const double nrm = sqrt(1.0 + px * px + py * py);
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    X[m] = C.Xcam[m];
    K[m] = C.e[0][m] + (px * C.e[1][m] + py * C.e[2][m] + C.e[3][m]) / nrm;
  }
}

// 1/dl = (|K1|+d)/eps + (|K2|+d)/(eps min(X2,1-X2)) + (|K3|+d)/eps ; ieps = 1/eps
__device__ __forceinline__ double stepsize(const double X[4], const double K[4], double ieps) {
  const double d = 1e-40;
  const double i13 = (fabs(K[1]) + d) + (fabs(K[3]) + d);
  const double i2 = (fabs(K[2]) + d) * ip_rcp(fabs(fmin(X[2], 1.0 - X[2])));
  return ip_rcp((i13 + i2) * ieps);
}

// classical RK4 on (X^1..3, K^0..3); X^0 is not integrated (static snapshot, R-9).
// SMALL (eps <= 0.04): r, sin/cos theta at the three displaced stage points come from the values at the start of
// the step by short Taylor polynomials in the displacement (point_shift) -- one exp and one or two sincos per step
// instead of four of each; otherwise every stage is evaluated from scratch.
template <bool SMALL>
__device__ __forceinline__ void rk4_push(const Geom& G, double X[4], double K[4], double h) {
  double k1[4], k2[4], k3[4], k4[4], Xt[4], Kt[4];
  Xt[0] = 0.0;
  Point p0, pt;
  point_full(G, X, p0);
  pt = p0;
  geodesic_accel_at(G, pt, K, k1);
#pragma unroll
  for (int m = 0; m < 4; ++m) { Kt[m] = K[m] + 0.5 * h * k1[m]; }
  if (SMALL) point_shift(G, p0, 0.5 * h * K[1], 0.5 * h * K[2], pt);
  else {
#pragma unroll
    for (int m = 1; m < 4; ++m) Xt[m] = X[m] + 0.5 * h * K[m];
    point_full(G, Xt, pt);
  }
  geodesic_accel_at(G, pt, Kt, k2);
  double xs[4];  // x1 + 2 x2 (+ 2 x3 + x4): the X-slopes are the stage K's
#pragma unroll
  for (int m = 1; m < 4; ++m) xs[m] = K[m] + 2.0 * Kt[m];
  if (SMALL) point_shift(G, p0, 0.5 * h * Kt[1], 0.5 * h * Kt[2], pt);
  else {
#pragma unroll
    for (int m = 1; m < 4; ++m) Xt[m] = X[m] + 0.5 * h * Kt[m];
    point_full(G, Xt, pt);
  }
#pragma unroll
  for (int m = 0; m < 4; ++m) { Kt[m] = K[m] + 0.5 * h * k2[m]; }
  geodesic_accel_at(G, pt, Kt, k3);
#pragma unroll
  for (int m = 1; m < 4; ++m) xs[m] += 2.0 * Kt[m];
  if (SMALL) point_shift(G, p0, h * Kt[1], h * Kt[2], pt);
  else {
#pragma unroll
    for (int m = 1; m < 4; ++m) Xt[m] = X[m] + h * Kt[m];
    point_full(G, Xt, pt);
  }
#pragma unroll
  for (int m = 0; m < 4; ++m) { Kt[m] = K[m] + h * k3[m]; }
  geodesic_accel_at(G, pt, Kt, k4);
  const double h6 = h * (1.0 / 6.0);
#pragma unroll
  for (int m = 1; m < 4; ++m) X[m] += h6 * (xs[m] + Kt[m]);
#pragma unroll
  for (int m = 0; m < 4; ++m) K[m] += h6 * (k1[m] + 2.0 * k2[m] + 2.0 * k3[m] + k4[m]);
}

__device__ __forceinline__ void store_record(double* rec, const double X[4], const double K[4], double dl) {
  st_global_v4(rec, X[1], X[2], X[3], K[0]);
  st_global_v4(rec + 4, K[1], K[2], K[3], dl);
}
__device__ __forceinline__ void load_record(const double* rec, double X[4], double K[4], double& dl) {
  X[0] = 0.0;
  ld_global_v4(rec, X[1], X[2], X[3], K[0]);
  ld_global_v4(rec + 4, K[1], K[2], K[3], dl);
}

#ifndef IPOLE_GEO_THREADS
#define IPOLE_GEO_THREADS 128
#endif
#ifndef IPOLE_GEO_MINB
#define IPOLE_GEO_MINB 4
#endif

// a-2, a-3, a-8.  Every lane owns one ray at a time and pulls the next one from the atomic queue as soon as its ray
// ends, so the RK4 body runs with all lanes active whatever the step counts of neighbouring pixels are.
//
// OCC (grid model): every step's midpoint -- the point k_transfer evaluates the plasma at -- is tested against the
// grid's stencil-occupancy bitmap, and the first and last step that may cross plasma are kept per ray.  k_transfer
// then starts a ray at its first contact with plasma instead of its far end (everything before is dark vacuum and
// changes nothing), skips the bitmap test after the last contact, and a ray that meets no plasma is not walked at all.
//
// MC (many cameras per launch: a fit that varies inclination or spin): the geometry and the stop radii are
// per-lane values taken from the ray's own camera at refill; the single-camera instantiation keeps them in the
// constant bank.
//
// LOWLAT: the same code compiled for 2 blocks per SM (180 registers instead of 128).  ptxas then keeps more independent
// operations in flight per thread, which is worth nothing when the SM is full (the 4-block build wins a 4096^2 image by
// 3-10 %) but shortens the dependent chain of a LONE ray: launches that cannot fill the GPU anyway -- long-ray and retry
// passes, probe passes, the levels of an adaptive image, small images -- take it (profiles/r2_notes.md).  Same arithmetic.
template <bool OCC, bool MC = false, bool LOWLAT = false>
__global__ void __launch_bounds__(IPOLE_GEO_THREADS, LOWLAT ? 2 : (MC ? 3 : IPOLE_GEO_MINB)) k_geodesic(const __grid_constant__ GeoArgs A) {
  const CamDev& C = A.cam;
  Geom Gl = C.G;                      // MC: the lane's own
  double lx_in_l = C.lx_in, lx_esc_l = C.lx_esc;
  __shared__ __align__(8) unsigned char grid_smem[OCC ? sizeof(GridParams) : 8];
  if (OCC) {
    for (int i = threadIdx.x; i < (int)sizeof(GridParams); i += blockDim.x) grid_smem[i] = ((const unsigned char*)A.grid)[i];
    __syncthreads();
  }
  const GridParams& GP = *(const GridParams*)grid_smem;
  int s_hi = -1, s_lo = 0;
  const int64_t count = A.count_dev ? (int64_t)*A.count_dev : A.count;
  const size_t slot_doubles = (size_t)(A.cap + 1) * REC_DOUBLES;
  double X[4], K[4];
  double* rec = nullptr;
  int64_t li;
  int32_t q = 0;
  int n = 0, nt = 0;
  bool have = false;

  auto fetch = [&]() {
    li = (int64_t)atomicAdd(A.queue, 1ULL);
    have = li < count;
    if (!have) return;
    q = A.order ? A.order[A.base + li] : (int32_t)(A.base + li);
    int64_t pix;
    if (A.lattice_stride > 0) {
      const int per = A.lattice_nx * A.lattice_ny, cam = MC ? q / per : 0, ql = MC ? q % per : q;
      const int ix = ql % A.lattice_nx, iy = ql / A.lattice_nx;
      pix = (int64_t)(iy * A.lattice_stride + A.lattice_stride / 2) * C.nx + (ix * A.lattice_stride + A.lattice_stride / 2);
      if (MC) pix += (int64_t)cam * A.rays_per_cam;
    } else {
      pix = A.pixels ? A.pixels[(int64_t)q * A.list_stride] : (int64_t)q * A.list_stride;
    }
    if (MC) {
      const CamDev& Cc = A.cams[pix / A.rays_per_cam];
      pixel_ray(Cc, pix % A.rays_per_cam, X, K);
      Gl = Cc.G; lx_in_l = Cc.lx_in; lx_esc_l = Cc.lx_esc;
    } else pixel_ray(C, pix, X, K);
    rec = A.path ? A.path + (size_t)li * slot_doubles : nullptr;
    n = 0; nt = 0;
    s_hi = -1; s_lo = 0;
  };

  const double ieps = 1.0 / A.eps;
  const bool small_steps = A.eps <= 0.04;   // displacements of the RK4 stages within point_shift's range
  fetch();
  while (have) {
    const double dl = stepsize(X, K, ieps);
    if (rec) store_record(rec + (size_t)n * REC_DOUBLES, X, K, dl);
    const double x1_before = X[1];
    const bool k2neg = K[2] < 0.0;
    double Xa[4];
    if (OCC) { Xa[0] = X[0]; Xa[1] = X[1]; Xa[2] = X[2]; Xa[3] = X[3]; }
    if (small_steps) rk4_push<true>(MC ? Gl : C.G, X, K, -dl);
    else rk4_push<false>(MC ? Gl : C.G, X, K, -dl);
    if (OCC) {
      // the midpoint exactly as k_transfer forms it: 0.5 * (X_lo + X_hi) with lo = point n, hi = point n + 1
      double Xm[4];
#pragma unroll
      for (int m = 0; m < 4; ++m) Xm[m] = 0.5 * (Xa[m] + X[m]);
      if (grid_occupied(GP, Xm)) { if (s_hi < 0) s_lo = n; s_hi = n; }
    }
    ++n;
    if ((K[2] < 0.0) != k2neg) ++nt;
    int status = 0;
    if (X[1] <= (MC ? lx_in_l : C.lx_in)) status = 1;
    else if (X[1] > (MC ? lx_esc_l : C.lx_esc) && X[1] > x1_before) status = 2;
    else if (n >= A.max_steps) status = 3;
    const bool overflow = (status == 0) && rec && (n >= A.cap);
    if (status != 0 || overflow) {
      if (overflow) {
        A.nsteps[q] = -1;
        if (A.long_list) { const int w = atomicAdd(A.long_count, 1); A.long_list[w] = q; }
      } else {
        if (rec) store_record(rec + (size_t)n * REC_DOUBLES, X, K, 0.0);
        if (A.endp) store_record(A.endp + (size_t)q * REC_DOUBLES, X, K, 0.0);
        if (OCC && A.srange) A.srange[q] = make_int2(s_hi, s_lo);
        A.nsteps[q] = n;
        if (A.nturn) A.nturn[q] = (nt > 127 ? 127 : nt) | (status == 3 ? 0x80 : 0);
      }
      fetch();
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
struct RtArgs {
  CamDev cam;
  Units units;
  const void* model;          // device pointer to AdafParams / SlabParams / GridParams
  int cap;
  int64_t base, count;
  const int* count_dev;
  const int32_t* order;
  const double* path;
  const int32_t* nsteps;
  unsigned long long* queue;
  double *I, *Q, *U, *V, *tau, *tauF;   // indexed by q
  const int2* srange;         // grid model, stored path: steps that may cross plasma (from k_geodesic<true>; nullable)
  const int32_t* rank_slot;   // k_transfer_group: [base + a] = the slot of the batch that takes place a of its groups (k_rank_window; nullable)
  // path-free variant (PF != 0): no path; the ray restarts from the end point of its backward pass
  const double* endp;         // [total rays][8], indexed by q
  int32_t* nfwd;              // [total rays] steps of the forward pass (nullable)
  double eps; int max_steps;
  // model sweep (SWEEP): work item w = ray * n_models + m; `lane_tab` points at n_models AdafParams (analytic model)
  // or GridScales (grid model; `model` is the shared GridParams), `units_arr` at n_models Units; outputs of model m
  // start at plane + m * out_stride
  int n_models; const void* lane_tab; const Units* units_arr; size_t out_stride;
  // work item -> slot of the batch (nullable: identity): the rays k_stepop left to this kernel (stepop.cuh)
  const int32_t* slots;
  // many cameras per launch (k_transfer_group<MODEL, true>): ray q belongs to camera q / rays_per_cam; the cameras share
  // spin, mass and hslope with `cam` (its geometry serves all) and differ in direction, field of view, frequency, distance
  const CamDev* cams; int64_t rays_per_cam;   // units of camera k: units_arr[k]
};

constexpr int SWEEP_MAX_MODELS = 64;   // parameter sets per transfer launch (shared memory: <= 88 B each)

#ifndef IPOLE_RT_THREADS
#define IPOLE_RT_THREADS 128
#endif
#ifndef IPOLE_RT_MINB
#define IPOLE_RT_MINB 3   // grid model; 2 (254 registers) was better until rays started at their first plasma contact
#endif
#ifndef IPOLE_RT_MINB_ANALYTIC
#define IPOLE_RT_MINB_ANALYTIC 3
#endif
#ifndef IPOLE_PF_MINB_ANALYTIC
#define IPOLE_PF_MINB_ANALYTIC 2   // path-free variant: resident blocks per SM, analytic models / grid model
#endif
#ifndef IPOLE_PF_MINB_GRID
#define IPOLE_PF_MINB_GRID 3         // (measured: profiles/r1_pathfree.md)
#endif
#ifndef IPOLE_RT_SYNC
#define IPOLE_RT_SYNC 0
#endif
#ifndef IPOLE_RT_PREFETCH
#define IPOLE_RT_PREFETCH 1   // prefetch.global.L1 of the next path record: 2-3 % (profiles/r1_notes.md)
#endif

// a-4 ... a-7, a-8.  Lane-level refill as in k_geodesic.  Per step: midpoint (Xm, Km), generator A = Gamma.Km,
// f <- P f, plasma operator, f <- P f  (Strang splitting, R-6).
// Resident blocks per SM: 3 (168 registers, a few spilled doubles) for the analytic models, which ncu shows limited
// by dependent-issue latency, and for the grid model too since k_geodesic<true> marks the plasma-contact range (a
// walked step is now mostly transport and plasma arithmetic, not a dark gather test): 117 -> 102 ms at 1024^2.
//
// PF = 0: the stored path is walked from its far end to the camera.
// PF = 1, 2: path-free bidirectional variant (R-10; 1: eps <= 0.04, RK4 stage points by Taylor
// shifts, 2: any eps).  The ray restarts at the end point of its backward pass and is re-integrated forward, one RK4
// push of +dl per step (dl = the step rule at the point the step starts from), each push followed by the same
// transfer step over its two end points; it stops at r >= r_cam moving outward (or r <= r_in moving inward, or after
// max_steps steps), and the tensor is read in the observer tetrad built at that end point.
//
// SWEEP: many small images for model fitting: the same stored paths are walked once
// per parameter set (analytic model: AdafParams per set; grid model: the four scale numbers GridScales per set over
// the shared grid).  Work item w -> (ray w / n_models, model w % n_models): the lanes of a warp share a ray, so one
// 64-B record load serves up to 32 models and all of them finish the ray on the same step.
template <int MODEL, int PF, bool SWEEP = false>
__global__ void __launch_bounds__(IPOLE_RT_THREADS, (MODEL == MODEL_GRID) ? (PF ? IPOLE_PF_MINB_GRID : IPOLE_RT_MINB)
                                                                           : (PF ? IPOLE_PF_MINB_ANALYTIC : IPOLE_RT_MINB_ANALYTIC))
k_transfer(const __grid_constant__ RtArgs A) {
  static_assert(!SWEEP || (MODEL != MODEL_SLAB && PF == 0), "the sweep is built for the ADAF and grid models on stored paths");
  const CamDev& C = A.cam;
  const int64_t count = (A.count_dev ? (int64_t)*A.count_dev : A.count) * (SWEEP ? A.n_models : 1);
  const size_t slot_doubles = (size_t)(A.cap + 1) * REC_DOUBLES;
  constexpr int MODEL_BYTES = MODEL == MODEL_ADAF ? sizeof(AdafParams) : (MODEL == MODEL_SLAB ? sizeof(SlabParams) : sizeof(GridParams));
  constexpr int LANE_BYTES = MODEL == MODEL_ADAF ? sizeof(AdafParams) : sizeof(GridScales);
  __shared__ __align__(8) unsigned char model_smem[MODEL_BYTES];
  __shared__ __align__(8) unsigned char lane_smem[SWEEP ? LANE_BYTES * SWEEP_MAX_MODELS : 8];
  __shared__ Units units_smem[SWEEP ? SWEEP_MAX_MODELS : 1];
  {
    for (int i = threadIdx.x; i < MODEL_BYTES; i += blockDim.x) model_smem[i] = ((const unsigned char*)A.model)[i];
    if (SWEEP) {
      for (int i = threadIdx.x; i < LANE_BYTES * A.n_models; i += blockDim.x) lane_smem[i] = ((const unsigned char*)A.lane_tab)[i];
      for (int i = threadIdx.x; i < A.n_models; i += blockDim.x) units_smem[i] = A.units_arr[i];
    }
    __syncthreads();
  }
  const void* model = model_smem;
  const void* lane = nullptr;   // SWEEP: the lane's own parameter set
  int mi = 0;                   // SWEEP: its index

  PolState st;
  double Xhi[4], Khi[4];
  const double* rec = nullptr;
  int32_t q = 0;
  int s = -1, s_lo = 0;
  bool have = false, lit = false;

  auto fetch = [&]() {
    for (;;) {
      int64_t li = (int64_t)atomicAdd(A.queue, 1ULL);
      have = li < count;
      if (!have) return;
      if (SWEEP) {
        mi = (int)(li % A.n_models);
        li /= A.n_models;
        lane = lane_smem + (size_t)mi * LANE_BYTES;
      }
      if (A.slots) li = A.slots[li];
      q = A.order ? A.order[A.base + li] : (int32_t)(A.base + li);
      double dl;
      if (PF) {
        load_record(A.endp + (size_t)q * REC_DOUBLES, Xhi, Khi, dl);
        s = 0;   // forward steps taken
      } else {
        int n = A.nsteps[q];
        if (n < 0) continue;  // overflowed its slot: done by the long-ray pass
        if (MODEL == MODEL_GRID && A.srange) {
          const int2 r = A.srange[q];
          s_lo = r.y;
          if (r.x < 0) {      // the ray meets no plasma: dark
            const size_t o = SWEEP ? (size_t)mi * A.out_stride + q : (size_t)q;
            A.I[o] = 0.0; A.Q[o] = 0.0; A.U[o] = 0.0; A.V[o] = 0.0;
            if (A.tau) A.tau[o] = 0.0;
            if (A.tauF) A.tauF[o] = 0.0;
            continue;
          }
          n = r.x + 1;        // start at the first contact with plasma: the steps before it are dark vacuum
        }
        rec = A.path + (size_t)li * slot_doubles;
        load_record(rec + (size_t)n * REC_DOUBLES, Xhi, Khi, dl);
        s = n - 1;
      }
#pragma unroll
      for (int m = 0; m < 4; ++m) { st.f1[m] = 0.0; st.f2[m] = 0.0; st.S[m] = 0.0; }
      st.tau = 0.0; st.tauF = 0.0;
      lit = false;
      return;
    }
  };

  const double ieps = PF ? 1.0 / A.eps : 0.0;
  fetch();
#if IPOLE_RT_SYNC
  // one barrier per step keeps the warps of a block within one iteration of each other, so that they share the
  // instruction-cache lines of the (large) loop body
  while (__syncthreads_or(have)) {
    if (!have) continue;
#else
  while (have) {
#endif
    double Xlo[4], Klo[4], dl;
    if (PF) {
      dl = stepsize(Xhi, Khi, ieps);
#pragma unroll
      for (int m = 0; m < 4; ++m) { Xlo[m] = Xhi[m]; Klo[m] = Khi[m]; }
      rk4_push<PF == 1>(C.G, Xlo, Klo, dl);
    } else {
      load_record(rec + (size_t)s * REC_DOUBLES, Xlo, Klo, dl);
#if IPOLE_RT_PREFETCH
      if (s > 0) asm volatile("prefetch.global.L1 [%0];" ::"l"(rec + (size_t)(s - 1) * REC_DOUBLES));
#endif
    }
    double Xm[4], Km[4];
#pragma unroll
    for (int m = 0; m < 4; ++m) { Xm[m] = 0.5 * (Xlo[m] + Xhi[m]); Km[m] = 0.5 * (Klo[m] + Khi[m]); }
    // `maybe`: this step may cross plasma.  For the grid model the gather comes first (it needs no metric), so a step
    // that is dark so far and crosses no plasma costs eight record loads and nothing else.
    bool maybe = true;
    double prim[8];
    if (MODEL == MODEL_GRID) maybe = (PF != 0 || s >= s_lo) && grid_gather(*(const GridParams*)model, Xm, prim);
    if (lit || maybe) {
      Point p; Sym7 g; Inv6 gi; double Am[4][4];
      transport_generator(C.G, Xm, Km, p, g, gi, Am);
      const double h = 0.5 * dl;
      if (lit) { transport_apply(Am, h, st.f1); transport_apply(Am, h, st.f2); }
      // the tetrad first, then the second half of the transport (applied to the NEW legs), and only then the
      // coefficients and the 4x4 step, which touch the Stokes numbers alone: same result, but the generator and
      // the tetrad are dead while the register-hungry part runs
      PlasmaFrame F;
      const bool applied = maybe && plasma_frame<MODEL>(C.G, model, SWEEP ? lane : nullptr, SWEEP ? units_smem[mi] : A.units, Xm, Km, p, g, gi, prim, st, F);
      lit |= applied;
      if (lit) { transport_apply(Am, h, st.f1); transport_apply(Am, h, st.f2); }
      if (applied) plasma_apply<MODEL>(SWEEP ? units_smem[mi] : A.units, F, dl, st);
    }
    bool done;
    if (PF) {
      ++s;
      done = (Xlo[1] >= C.Xcam[1] && Xlo[1] > Xhi[1]) || (Xlo[1] <= C.lx_in && Xlo[1] < Xhi[1]) || s >= A.max_steps;
    } else {
      --s;
      done = s < 0;
    }
#pragma unroll
    for (int m = 0; m < 4; ++m) { Xhi[m] = Xlo[m]; Khi[m] = Klo[m]; }
    if (done) {
      // a-7: project on the camera's transverse legs, convert the invariant I/nu^3 to specific intensity
      if (PF) {
        double e[4][4], c1[4], c2[4];
        observer_tetrad(C.G, Xhi, e, c1, c2);
        stokes_congruence(dot4(c1, st.f1), dot4(c1, st.f2), dot4(c2, st.f1), dot4(c2, st.f2), st.S);
        if (A.nfwd) A.nfwd[q] = s;
      } else
      stokes_congruence(dot4(C.ecov1, st.f1), dot4(C.ecov1, st.f2), dot4(C.ecov2, st.f1), dot4(C.ecov2, st.f2), st.S);
      const double nu_o = SWEEP ? units_smem[mi].nu_obs : A.units.nu_obs;
      const double nu3 = nu_o * nu_o * nu_o;
      const size_t o = SWEEP ? (size_t)mi * A.out_stride + q : (size_t)q;
      A.I[o] = st.S[0] * nu3; A.Q[o] = st.S[1] * nu3; A.U[o] = st.S[2] * nu3; A.V[o] = st.S[3] * nu3;
      if (A.tau) A.tau[o] = st.tau;
      if (A.tauF) A.tauF[o] = st.tauF;
      fetch();
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// The same transfer on the stored path with WARP-level scheduling: one warp walks 32 consecutive rays of the batch in
// lockstep, lane <-> ray, aligned on the step index s (distance from the camera in steps), from the largest first-contact
// index of the group down to the camera; a lane joins when s reaches its own ray's start.
//
// Why (grid model): a walked step costs ~40 instructions where the stencil is empty and the ray still dark, ~400 in lit
// vacuum (transport only) and ~1200 where it crosses plasma.  With lane-level refill (k_transfer) the lanes of a warp
// drift to unrelated phases of unrelated rays and the warp pays for every kind of step present: 17 of 32 lanes active,
// and the loss grows with the batch length (profiles/r2_notes.md: the same image is 30 % slower in 28 batches than in
// 97).  Rays are ordered by predicted step count, so the 32 rays of a group lie on one ring of the image around the
// spin axis: at equal s they are at nearly equal radius and in the same kind of step.  The arithmetic per ray is that
// of k_transfer, operation for operation (bit-identical images).
// MC (many cameras per launch, grid model: ipole_make_images_cameras): frequency, length unit and the camera's transverse
// legs are the ray's own camera's; the single-camera instantiation is unchanged.
template <int MODEL, bool MC = false>
__global__ void __launch_bounds__(IPOLE_RT_THREADS, IPOLE_RT_MINB) k_transfer_group(const __grid_constant__ RtArgs A) {
  const CamDev& C = A.cam;
  const size_t slot_doubles = (size_t)(A.cap + 1) * REC_DOUBLES;
  constexpr int MODEL_BYTES = MODEL == MODEL_ADAF ? sizeof(AdafParams) : (MODEL == MODEL_SLAB ? sizeof(SlabParams) : sizeof(GridParams));
  __shared__ __align__(8) unsigned char model_smem[MODEL_BYTES];
  for (int i = threadIdx.x; i < MODEL_BYTES; i += blockDim.x) model_smem[i] = ((const unsigned char*)A.model)[i];
  __syncthreads();
  const void* model = model_smem;
  const int lane = threadIdx.x & 31;
  const int64_t count = A.count_dev ? (int64_t)*A.count_dev : A.count;
  const int64_t n_groups = (count + 31) >> 5;

  for (;;) {
    __syncwarp();
    long long grp = 0;
    if (lane == 0) grp = (long long)atomicAdd(A.queue, 1ULL);
    grp = __shfl_sync(0xffffffffu, grp, 0);
    if (grp >= n_groups) break;
    const int64_t li = (grp << 5) + lane;
    PolState st;
    double Xhi[4] = {0, 0, 0, 0}, Khi[4] = {0, 0, 0, 0};
    const double* rec = nullptr;
    int32_t q = 0;
    int s0 = -1, s_lo = 0;       // this lane walks steps s0 ... 0; -1: nothing to walk
    bool lit = false;
    Units Ul = A.units;          // MC: the units of the lane's camera
    int cam_i = 0;
    if (li < count) {
      const int64_t ls = A.rank_slot ? (int64_t)A.rank_slot[A.base + li] : li;    // this lane's slot in the batch
      q = A.order ? A.order[A.base + ls] : (int32_t)(A.base + ls);
      if (MC) { cam_i = (int)(q / A.rays_per_cam); Ul = A.units_arr[cam_i]; }
      int n = A.nsteps[q];
      if (n >= 0) {              // (n < 0: overflowed its slot, done by the long-ray pass)
        if (MODEL == MODEL_GRID && A.srange) {
          const int2 r = A.srange[q];
          s_lo = r.y;
          if (r.x < 0) {         // the ray meets no plasma: dark
            A.I[q] = 0.0; A.Q[q] = 0.0; A.U[q] = 0.0; A.V[q] = 0.0;
            if (A.tau) A.tau[q] = 0.0;
            if (A.tauF) A.tauF[q] = 0.0;
            n = 0;
          } else n = r.x + 1;    // start at the first contact with plasma
        }
        if (n > 0) {
          rec = A.path + (size_t)ls * slot_doubles;
          double dl;
          load_record(rec + (size_t)n * REC_DOUBLES, Xhi, Khi, dl);
          s0 = n - 1;
        }
      }
    }
#pragma unroll
    for (int m = 0; m < 4; ++m) { st.f1[m] = 0.0; st.f2[m] = 0.0; st.S[m] = 0.0; }
    st.tau = 0.0; st.tauF = 0.0;
    int smax = s0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) smax = max(smax, __shfl_xor_sync(0xffffffffu, smax, o));

    for (int s = smax; s >= 0; --s) {
      if (s > s0) continue;
      double Xlo[4], Klo[4], dl;
      load_record(rec + (size_t)s * REC_DOUBLES, Xlo, Klo, dl);
#if IPOLE_RT_PREFETCH
      if (s > 0) asm volatile("prefetch.global.L1 [%0];" ::"l"(rec + (size_t)(s - 1) * REC_DOUBLES));
#endif
      double Xm[4], Km[4];
#pragma unroll
      for (int m = 0; m < 4; ++m) { Xm[m] = 0.5 * (Xlo[m] + Xhi[m]); Km[m] = 0.5 * (Klo[m] + Khi[m]); }
      bool maybe = true;
      double prim[8];
      if (MODEL == MODEL_GRID) maybe = (s >= s_lo) && grid_gather(*(const GridParams*)model, Xm, prim);
      if (lit || maybe) {
        Point p; Sym7 g; Inv6 gi; double Am[4][4];
        transport_generator(C.G, Xm, Km, p, g, gi, Am);
        const double h = 0.5 * dl;
        if (lit) { transport_apply(Am, h, st.f1); transport_apply(Am, h, st.f2); }
        PlasmaFrame F;
        const bool applied = maybe && plasma_frame<MODEL>(C.G, model, nullptr, MC ? Ul : A.units, Xm, Km, p, g, gi, prim, st, F);
        lit |= applied;
        if (lit) { transport_apply(Am, h, st.f1); transport_apply(Am, h, st.f2); }
        if (applied) plasma_apply<MODEL>(MC ? Ul : A.units, F, dl, st);
      }
#pragma unroll
      for (int m = 0; m < 4; ++m) { Xhi[m] = Xlo[m]; Khi[m] = Klo[m]; }
    }
    if (s0 >= 0) {
      const double* ec1 = MC ? A.cams[cam_i].ecov1 : C.ecov1;
      const double* ec2 = MC ? A.cams[cam_i].ecov2 : C.ecov2;
      stokes_congruence(dot4(ec1, st.f1), dot4(ec1, st.f2), dot4(ec2, st.f1), dot4(ec2, st.f2), st.S);
      const double nu_o = MC ? Ul.nu_obs : A.units.nu_obs;
      const double nu3 = nu_o * nu_o * nu_o;
      A.I[q] = st.S[0] * nu3; A.Q[q] = st.S[1] * nu3; A.U[q] = st.S[2] * nu3; A.V[q] = st.S[3] * nu3;
      if (A.tau) A.tau[q] = st.tau;
      if (A.tauF) A.tauF[q] = st.tauF;
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Unpolarized transfer ("nonpolarized images" of the model-fitting loop; R-12): I alone on the
// stored path.  Per step: midpoint, metric (no derivatives, no transport), plasma state, nu = -k.u nu_obs, pitch
// angle, thermal synchrotron j_I and alpha_I, exact scalar step  I <- I e^{-x} + j ds (1 - e^{-x})/x,  x = alpha ds.
// Work items and refill as in k_transfer (SWEEP: (ray, parameter set) pairs, the lanes of a warp share a ray).
#ifndef IPOLE_UNPOL_MINB_ANALYTIC
#define IPOLE_UNPOL_MINB_ANALYTIC 5   // measured: 3..6 blocks, profiles/r1_unpolarized.md
#endif
#ifndef IPOLE_UNPOL_MINB_GRID
#define IPOLE_UNPOL_MINB_GRID 4
#endif
template <int MODEL, bool SWEEP>
__global__ void __launch_bounds__(IPOLE_RT_THREADS, (MODEL == MODEL_GRID) ? IPOLE_UNPOL_MINB_GRID : IPOLE_UNPOL_MINB_ANALYTIC) k_transfer_unpol(const __grid_constant__ RtArgs A) {
  static_assert(!SWEEP || MODEL != MODEL_SLAB, "the sweep is built for the ADAF and grid models");
  const CamDev& C = A.cam;
  const int64_t count = (A.count_dev ? (int64_t)*A.count_dev : A.count) * (SWEEP ? A.n_models : 1);
  const size_t slot_doubles = (size_t)(A.cap + 1) * REC_DOUBLES;
  constexpr int MODEL_BYTES = MODEL == MODEL_ADAF ? sizeof(AdafParams) : (MODEL == MODEL_SLAB ? sizeof(SlabParams) : sizeof(GridParams));
  constexpr int LANE_BYTES = MODEL == MODEL_ADAF ? sizeof(AdafParams) : sizeof(GridScales);
  __shared__ __align__(8) unsigned char model_smem[MODEL_BYTES];
  __shared__ __align__(8) unsigned char lane_smem[SWEEP ? LANE_BYTES * SWEEP_MAX_MODELS : 8];
  __shared__ Units units_smem[SWEEP ? SWEEP_MAX_MODELS : 1];
  {
    for (int i = threadIdx.x; i < MODEL_BYTES; i += blockDim.x) model_smem[i] = ((const unsigned char*)A.model)[i];
    if (SWEEP) {
      for (int i = threadIdx.x; i < LANE_BYTES * A.n_models; i += blockDim.x) lane_smem[i] = ((const unsigned char*)A.lane_tab)[i];
      for (int i = threadIdx.x; i < A.n_models; i += blockDim.x) units_smem[i] = A.units_arr[i];
    }
    __syncthreads();
  }
  const void* model = model_smem;
  const void* lane = nullptr;
  int mi = 0;
  double I = 0.0, tau = 0.0;
  double Xhi[4], Khi[4];
  const double* rec = nullptr;
  int32_t q = 0;
  int s = -1, s_lo = 0;
  bool have = false;

  auto finish = [&]() {
    const double nu_o = SWEEP ? units_smem[mi].nu_obs : A.units.nu_obs;
    const size_t o = SWEEP ? (size_t)mi * A.out_stride + q : (size_t)q;
    A.I[o] = I * (nu_o * nu_o * nu_o); A.Q[o] = 0.0; A.U[o] = 0.0; A.V[o] = 0.0;
    if (A.tau) A.tau[o] = tau;
    if (A.tauF) A.tauF[o] = 0.0;
  };
  auto fetch = [&]() {
    for (;;) {
      int64_t li = (int64_t)atomicAdd(A.queue, 1ULL);
      have = li < count;
      if (!have) return;
      if (SWEEP) { mi = (int)(li % A.n_models); li /= A.n_models; lane = lane_smem + (size_t)mi * LANE_BYTES; }
      q = A.order ? A.order[A.base + li] : (int32_t)(A.base + li);
      int n = A.nsteps[q];
      if (n < 0) continue;   // overflowed its slot: done by the long-ray pass
      I = 0.0; tau = 0.0; s_lo = 0;
      if (MODEL == MODEL_GRID && A.srange) {
        const int2 r = A.srange[q];
        if (r.x < 0) { finish(); continue; }   // the ray meets no plasma
        n = r.x + 1; s_lo = r.y;
      }
      rec = A.path + (size_t)li * slot_doubles;
      double dl;
      load_record(rec + (size_t)n * REC_DOUBLES, Xhi, Khi, dl);
      s = n - 1;
      return;
    }
  };

  fetch();
  while (have) {
    double Xlo[4], Klo[4], dl;
    load_record(rec + (size_t)s * REC_DOUBLES, Xlo, Klo, dl);
    double Xm[4], Km[4];
#pragma unroll
    for (int m = 0; m < 4; ++m) { Xm[m] = 0.5 * (Xlo[m] + Xhi[m]); Km[m] = 0.5 * (Klo[m] + Khi[m]); }
    bool maybe = true;
    double prim[8];
    if (MODEL == MODEL_GRID) maybe = grid_gather(*(const GridParams*)model, Xm, prim);
    if (maybe) {
      Point p; Sym7 g; Inv6 gi;
      metric<true>(C.G, Xm, p, g, gi);
      Plasma P;
      bool present;
      if (MODEL == MODEL_ADAF) present = plasma_adaf(C.G, *(const AdafParams*)(SWEEP ? lane : model), Xm, p, g, gi, P);
      else if (MODEL == MODEL_SLAB) present = plasma_slab(C.G, *(const SlabParams*)model, Xm, p, g, P);
      else {
        const GridParams& M = *(const GridParams*)model;
        if (SWEEP) present = grid_state(C.G, M, *(const GridScales*)lane, prim, p, g, gi, P);
        else { const GridScales S = {M.ne_unit, M.B_unit, M.Rlow, M.Rhigh}; present = grid_state(C.G, M, S, prim, p, g, gi, P); }
      }
      if (present) {
        const Units& U = SWEEP ? units_smem[mi] : A.units;
        double kcov[4];
        g.mul(Km, kcov);
        const double om = -dot4(kcov, P.u);
        if (om > 0.0) {
          const double nu = om * U.nu_obs;
          double ji, ai;
          if (MODEL == MODEL_SLAB) {
            const double inu = ip_rcp(nu);
            ji = P.j[0] * inu * inu; ai = P.al[0] * nu;
          } else {
            double bcov[4];
            g.mul(P.b, bcov);
            const double cosT = fmin(1.0, fmax(-1.0, dot4(bcov, Km) * ip_rcp(om) * ip_rcp(P.B)));
            const Coeff c = synchrotron_invariant(P.ne, P.Th, P.B, cosT, nu);
            ji = c.jI; ai = c.aI;
          }
          const double ds = dl * U.dl_unit;
          const double x = ai * ds;
          const double em = ip_expm1(-x);
          const double E = (x > 0.0) ? -em * ip_rcp(x) : 1.0;
          I = I + I * em + ji * ds * E;
          tau += x;
        }
      }
    }
#pragma unroll
    for (int m = 0; m < 4; ++m) { Xhi[m] = Xlo[m]; Khi[m] = Klo[m]; }
    --s;
    if (s < s_lo) {   // below the last step that may cross plasma nothing changes any more (s_lo = 0 without the range)
      finish();
      fetch();
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// a-8: order rays by predicted step count, longest first (counting sort on 4096 bins)
constexpr int SORT_BINS = 4096;

struct SortArgs {
  int64_t n;                  // rays
  const int32_t* probe;       // step counts of the probe lattice / probe list
  int scale;                  // predicted = probe * scale
  int64_t rays_per_cam;       // many cameras per call: pixel p belongs to camera p / rays_per_cam, one lattice per camera (0: one camera)
  int lattice_stride, lattice_nx, lattice_ny, nx;  // full-image mode: pixel -> nearest lattice point
  const int64_t* pixels;      // list mode with lattice: pixel of ray q (nullable)
  int list_stride;            // list mode without lattice_stride: probe index = q / list_stride
  int bin_width;
  int32_t* key;               // [n] bin of each ray (descending steps = ascending bin)
  unsigned int* hist;         // [SORT_BINS]
  int32_t* order;             // [n] out
};

__global__ void k_predict_hist(SortArgs A) {
  for (int64_t q = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; q < A.n; q += (int64_t)gridDim.x * blockDim.x) {
    int pr;
    if (A.lattice_stride > 0) {
      // the longest of the four probe rays around the pixel (lattice point (ix, iy) is pixel (ix + 1/2) * stride):
      // next to the photon ring the step count jumps by a factor of two to three within one lattice cell, and the
      // per-batch path slots (run_rays) are sized from this prediction
      int64_t pix = A.pixels ? A.pixels[q] : q;
      const int64_t cam = A.rays_per_cam ? pix / A.rays_per_cam : 0;
      pix -= cam * A.rays_per_cam;
      const int32_t* probe = A.probe + cam * (A.lattice_nx * A.lattice_ny);
      const int px = (int)(pix % A.nx) - A.lattice_stride / 2, py = (int)(pix / A.nx) - A.lattice_stride / 2;
      const int ix0 = min(max(px, 0) / A.lattice_stride, A.lattice_nx - 1), iy0 = min(max(py, 0) / A.lattice_stride, A.lattice_ny - 1);
      const int ix1 = min(ix0 + 1, A.lattice_nx - 1), iy1 = min(iy0 + 1, A.lattice_ny - 1);
      pr = max(max(probe[iy0 * A.lattice_nx + ix0], probe[iy0 * A.lattice_nx + ix1]),
               max(probe[iy1 * A.lattice_nx + ix0], probe[iy1 * A.lattice_nx + ix1]));
    } else {
      pr = A.probe[(int)(q / A.list_stride)];
    }
    const int pred = pr * A.scale;
    int bin = SORT_BINS - 1 - min(pred / A.bin_width, SORT_BINS - 1);
    A.key[q] = bin;
    atomicAdd(&A.hist[bin], 1u);
  }
}

__global__ void k_scan_bins(unsigned int* hist) {  // exclusive scan of SORT_BINS counters, one block of 1024
  __shared__ unsigned int part[1024];
  const int t = threadIdx.x;
  unsigned int v[SORT_BINS / 1024], sum = 0;
  for (int i = 0; i < SORT_BINS / 1024; ++i) { v[i] = hist[t * (SORT_BINS / 1024) + i]; sum += v[i]; }
  part[t] = sum;
  __syncthreads();
  for (int off = 1; off < 1024; off <<= 1) {
    const unsigned int x = (t >= off) ? part[t - off] : 0u;
    __syncthreads();
    part[t] += x;
    __syncthreads();
  }
  unsigned int run = part[t] - sum;
  for (int i = 0; i < SORT_BINS / 1024; ++i) { hist[t * (SORT_BINS / 1024) + i] = run; run += v[i]; }
}

__global__ void k_scatter(SortArgs A) {
  for (int64_t q = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; q < A.n; q += (int64_t)gridDim.x * blockDim.x) {
    const unsigned int pos = atomicAdd(&A.hist[A.key[q]], 1u);
    A.order[pos] = (int32_t)q;
  }
}

// ---------------------------------------------------------------------------------------------------------------
// a-9: totals.  Fixed shape: REDUCE_BLOCKS blocks x 256 threads, grid-stride partial sums, warp shuffles, then one
// block folds the partials in index order -> bitwise reproducible for a given image.
constexpr int REDUCE_BLOCKS = 296;

struct ReduceOut {
  double flux[4];          // sum of I,Q,U,V over pixels (times scale in the final kernel)
  double lp, cp;
  long long total_steps;
  int max_steps;
  long long n_ring, n_maxstep;
};

struct ReducePartial { double s[4]; long long steps; int maxs; long long ring, maxed; };

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ long long warp_sum_ll(long long v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ int warp_max(int v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = max(v, __shfl_down_sync(0xffffffffu, v, o));
  return v;
}

__global__ void __launch_bounds__(256) k_reduce_partial(int64_t n, const double* I, const double* Q, const double* U,
                                                        const double* V, const int32_t* nsteps, const int32_t* nturn,
                                                        ReducePartial* part) {
  double s[4] = {0, 0, 0, 0};
  long long steps = 0, ring = 0, maxed = 0;
  int maxs = 0;
  for (int64_t q = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; q < n; q += (int64_t)gridDim.x * blockDim.x) {
    s[0] += I[q]; s[1] += Q[q]; s[2] += U[q]; s[3] += V[q];
    const int ns = nsteps[q], nt = nturn[q];
    steps += ns; maxs = max(maxs, ns);
    ring += ((nt & 0x7f) >= 2); maxed += ((nt & 0x80) != 0);
  }
  __shared__ ReducePartial sh[8];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < 4; ++k) s[k] = warp_sum(s[k]);
  steps = warp_sum_ll(steps); ring = warp_sum_ll(ring); maxed = warp_sum_ll(maxed); maxs = warp_max(maxs);
  if (lane == 0) { for (int k = 0; k < 4; ++k) sh[w].s[k] = s[k]; sh[w].steps = steps; sh[w].maxs = maxs; sh[w].ring = ring; sh[w].maxed = maxed; }
  __syncthreads();
  if (threadIdx.x == 0) {
    ReducePartial r = sh[0];
    for (int i = 1; i < 8; ++i) {
      for (int k = 0; k < 4; ++k) r.s[k] += sh[i].s[k];
      r.steps += sh[i].steps; r.maxs = max(r.maxs, sh[i].maxs); r.ring += sh[i].ring; r.maxed += sh[i].maxed;
    }
    part[blockIdx.x] = r;
  }
}

__global__ void k_reduce_final(const ReducePartial* part, int nparts, double scale, ReduceOut* out) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  ReducePartial r = part[0];
  for (int i = 1; i < nparts; ++i) {
    for (int k = 0; k < 4; ++k) r.s[k] += part[i].s[k];
    r.steps += part[i].steps; r.maxs = max(r.maxs, part[i].maxs); r.ring += part[i].ring; r.maxed += part[i].maxed;
  }
  ReduceOut o;
  for (int k = 0; k < 4; ++k) o.flux[k] = r.s[k] * scale;
  o.lp = (r.s[0] != 0.0) ? sqrt(r.s[1] * r.s[1] + r.s[2] * r.s[2]) / r.s[0] : 0.0;
  o.cp = (r.s[0] != 0.0) ? r.s[3] / r.s[0] : 0.0;
  o.total_steps = r.steps; o.max_steps = r.maxs; o.n_ring = r.ring; o.n_maxstep = r.maxed;
  *out = o;
}

// Flux of ONE large image in two stages (ipole_make_image_adaptive: 16.7 M pixels are too many for the single block per
// image of k_reduce_models below): REDUCE_BLOCKS partial sums, then one block folds them in index order => reproducible.
__global__ void __launch_bounds__(256) k_reduce_planes_partial(int64_t n, const double* I, const double* Q, const double* U,
                                                               const double* V, double* part /* [gridDim.x][4] */) {
  double s[4] = {0, 0, 0, 0};
  for (int64_t q = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; q < n; q += (int64_t)gridDim.x * blockDim.x) {
    s[0] += I[q]; s[1] += Q[q]; s[2] += U[q]; s[3] += V[q];
  }
  __shared__ double sh[8][4];
#pragma unroll
  for (int k = 0; k < 4; ++k) s[k] = warp_sum(s[k]);
  if ((threadIdx.x & 31) == 0) for (int k = 0; k < 4; ++k) sh[threadIdx.x >> 5][k] = s[k];
  __syncthreads();
  if (threadIdx.x < 4) {
    double t = sh[0][threadIdx.x];
    for (int w = 1; w < 8; ++w) t += sh[w][threadIdx.x];
    part[4 * blockIdx.x + threadIdx.x] = t;
  }
}
__global__ void k_reduce_planes_final(const double* part, int nparts, double scale, double* flux /* [4] */) {
  if (threadIdx.x < 4 && blockIdx.x == 0) {
    double t = 0.0;
    for (int i = 0; i < nparts; ++i) t += part[4 * i + threadIdx.x];
    flux[threadIdx.x] = t * scale;
  }
}

// model sweep: flux of every image of the batch, one block per model (fixed shape => reproducible)
__global__ void __launch_bounds__(256) k_reduce_models(int64_t n, size_t stride, const double* I, const double* Q,
                                                       const double* U, const double* V, double scale, double* flux) {
  const size_t o = (size_t)blockIdx.x * stride;
  double s[4] = {0, 0, 0, 0};
  for (int64_t q = threadIdx.x; q < n; q += blockDim.x) { s[0] += I[o + q]; s[1] += Q[o + q]; s[2] += U[o + q]; s[3] += V[o + q]; }
  __shared__ double sh[8][4];
#pragma unroll
  for (int k = 0; k < 4; ++k) s[k] = warp_sum(s[k]);
  if ((threadIdx.x & 31) == 0) for (int k = 0; k < 4; ++k) sh[threadIdx.x >> 5][k] = s[k];
  __syncthreads();
  if (threadIdx.x < 4) {
    double t = sh[0][threadIdx.x];
    for (int w = 1; w < 8; ++w) t += sh[w][threadIdx.x];
    flux[4 * blockIdx.x + threadIdx.x] = t * scale;
  }
}

// the same with one scale per image (many cameras per call: the pixel solid angle is the camera's)
__global__ void __launch_bounds__(256) k_reduce_cams(int64_t n, size_t stride, const double* I, const double* Q, const double* U,
                                                     const double* V, const double* scale, double* flux) {
  const size_t o = (size_t)blockIdx.x * stride;
  double s[4] = {0, 0, 0, 0};
  for (int64_t q = threadIdx.x; q < n; q += blockDim.x) { s[0] += I[o + q]; s[1] += Q[o + q]; s[2] += U[o + q]; s[3] += V[o + q]; }
  __shared__ double sh[8][4];
#pragma unroll
  for (int k = 0; k < 4; ++k) s[k] = warp_sum(s[k]);
  if ((threadIdx.x & 31) == 0) for (int k = 0; k < 4; ++k) sh[threadIdx.x >> 5][k] = s[k];
  __syncthreads();
  if (threadIdx.x < 4) {
    double t = sh[0][threadIdx.x];
    for (int w = 1; w < 8; ++w) t += sh[w][threadIdx.x];
    flux[4 * blockIdx.x + threadIdx.x] = t * scale[blockIdx.x];
  }
}

// out = min(*in, limit): the ray count of a pass sized before the count is known (retry level on the side stream)
__global__ void k_clamp_count(const int* in, int limit, int* out) { *out = min(*in, limit); }

// step counts of the long-ray passes -> nsteps (after every bulk kernel has finished)
__global__ void k_merge_long(int n_long, const int32_t* long_list, const int32_t* nsteps_long, int32_t* nsteps) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n_long) { const int32_t q = long_list[i]; const int32_t v = nsteps_long[q]; if (v >= 0) nsteps[q] = v; }
}

// sum of the forward-step counts of the path-free variant (integer: order-independent)
__global__ void k_sum_i32(const int32_t* v, int64_t n, long long* out) {
  long long s = 0;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) s += v[i];
  s = warp_sum_ll(s);
  if ((threadIdx.x & 31) == 0 && s != 0) atomicAdd((unsigned long long*)out, (unsigned long long)s);
}

__global__ void k_max_i32(const int32_t* v, int n, int* out) {  // probe maximum (one block)
  int m = 0;
  for (int i = threadIdx.x; i < n; i += blockDim.x) m = max(m, v[i]);
  m = warp_max(m);
  __shared__ int sh[32];
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x == 0) { for (int i = 1; i < (int)(blockDim.x >> 5); ++i) m = max(m, sh[i]); *out = m; }
}

// ---------------------------------------------------------------------------------------------------------------
// stage evaluators for the per-stage parity tests
__global__ void k_eval_connection(Geom G, int64_t n, const double* X, double* Gam) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  // Gamma^l_{mn} recovered from the contracted generator: A(K = e_m)^l_n = Gamma^l_{mn}
  for (int m = 0; m < 4; ++m) {
    double K[4] = {0, 0, 0, 0};
    K[m] = 1.0;
    Point p; Sym7 g; Inv6 gi; double A[4][4];
    transport_generator(G, X + 4 * i, K, p, g, gi, A);
    for (int l = 0; l < 4; ++l) for (int nn = 0; nn < 4; ++nn) Gam[64 * i + 16 * l + 4 * m + nn] = A[l][nn];
  }
}
__global__ void k_eval_coefficients(int64_t n, const double* in, double* out) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  const Coeff c = synchrotron_coefficients(in[5 * i], in[5 * i + 1], in[5 * i + 2], in[5 * i + 3], in[5 * i + 4]);
  double* o = out + 8 * i;
  o[0] = c.jI; o[1] = c.jQ; o[2] = c.jV; o[3] = c.aI; o[4] = c.aQ; o[5] = c.aV; o[6] = c.rQ; o[7] = c.rV;
}
__global__ void k_eval_stokes_step(int64_t n, const double* in, double* out) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double* a = in + 16 * i;
  double S[4] = {a[8], a[9], a[10], a[11]};
  if (a[2] == 0.0 && a[5] == 0.0 && a[14] == 0.0)   // aU = rU = jU = 0: the specialised form the transfer kernel uses
    stokes_step_qv<true>(a[0], a[1], a[3], a[4], a[6], a[7], a[12], a[13], a[15], S);
  else
    stokes_step(a, a + 4, a[7], a + 12, S);
  for (int k = 0; k < 4; ++k) out[4 * i + k] = S[k];
}
__global__ void k_eval_bessel(int64_t n, const double* z, double* out) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  double k0, k1;
  bessel_k01_scaled(z[i], k0, k1);
  out[3 * i] = k0; out[3 * i + 1] = k1; out[3 * i + 2] = k0 + 2.0 / z[i] * k1;
}
// re-tile one SoA plane into the cell-major records of GridParams::cells (load time, not on the hot path)
__global__ void k_pack_field(size_t cells, int field, const double* __restrict__ plane, double* __restrict__ out) {
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < cells; i += (size_t)gridDim.x * blockDim.x)
    out[i * 8 + field] = plane[i];
}
// stencil occupancy bitmap of the grid model: bit (ib, jb, k) covers the trilinear stencil whose base cell is
// (ib-1, jb-1, k) before clamping, i.e. exactly the eight cells grid_gather reads there
__global__ void k_build_occupancy(GridParams M, unsigned int* occ) {
  const size_t total = (size_t)(M.N1 + 1) * (M.N2 + 1) * M.N3;
  for (size_t t = blockIdx.x * (size_t)blockDim.x + threadIdx.x; t < total; t += (size_t)gridDim.x * blockDim.x) {
    const int k0 = (int)(t % M.N3);
    const int jb = (int)((t / M.N3) % (M.N2 + 1)), ib = (int)(t / ((size_t)M.N3 * (M.N2 + 1)));
    const int i0 = clampi(ib - 1, 0, M.N1 - 1), i1 = clampi(ib, 0, M.N1 - 1);
    const int j0 = clampi(jb - 1, 0, M.N2 - 1), j1 = clampi(jb, 0, M.N2 - 1);
    const int k1 = (k0 + 1 == M.N3) ? 0 : k0 + 1;
    const int ii[2] = {i0, i1}, jj[2] = {j0, j1}, kk[2] = {k0, k1};
    bool rho = false, u = false;
    for (int a = 0; a < 2; ++a) for (int b = 0; b < 2; ++b) for (int c = 0; c < 2; ++c) {
      const double* rec = M.cells + (((size_t)ii[a] * M.N2 + jj[b]) * M.N3 + kk[c]) * 8;
      rho |= rec[0] > 0.0; u |= rec[1] > 0.0;
    }
    if (rho && u) atomicOr(occ + (t >> 5), 1u << (t & 31));
  }
}
__global__ void k_eval_math(int64_t n, const double* x, double* out) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double v = x[i];
  double* o = out + 8 * i;
  o[0] = ip_exp(v); o[1] = ip_expm1(v); o[2] = ip_log(fabs(v));
  ip_sincos_any(v, &o[3], &o[4]);
  o[5] = ip_rcp(v); o[6] = ip_rsqrt(fabs(v)); o[7] = ip_sqrt(fabs(v));
}
template <int MODEL>
__global__ void k_eval_plasma(Geom G, const void* model, int64_t n, const double* X, double* out) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= n) return;
  Point p; Sym7 g; Inv6 gi;
  metric<true>(G, X + 4 * i, p, g, gi);
  Plasma P;
  P.ne = P.Th = P.B = 0.0;
  for (int m = 0; m < 4; ++m) { P.u[m] = 0.0; P.b[m] = 0.0; }
  bool present;
  if (MODEL == MODEL_ADAF) present = plasma_adaf(G, *(const AdafParams*)model, X + 4 * i, p, g, gi, P);
  else if (MODEL == MODEL_SLAB) present = plasma_slab(G, *(const SlabParams*)model, X + 4 * i, p, g, P);
  else present = plasma_grid(G, *(const GridParams*)model, X + 4 * i, p, g, gi, P);
  double* o = out + 12 * i;
  o[0] = present ? 1.0 : 0.0; o[1] = present ? P.ne : 0.0; o[2] = present ? P.Th : 0.0; o[3] = present ? P.B : 0.0;
  for (int m = 0; m < 4; ++m) { o[4 + m] = present ? P.u[m] : 0.0; o[8 + m] = present ? P.b[m] : 0.0; }
}

// FP64 FMA throughput: 8 independent chains per thread
__global__ void __launch_bounds__(256) k_fp64_peak(int iters, double seed, double* sink) {
  double a0 = seed, a1 = seed + 1, a2 = seed + 2, a3 = seed + 3, a4 = seed + 4, a5 = seed + 5, a6 = seed + 6, a7 = seed + 7;
  const double b = 0.999999 + 1e-9 * threadIdx.x, c = 1e-7;
  for (int i = 0; i < iters; ++i) {
    a0 = fma(a0, b, c); a1 = fma(a1, b, c); a2 = fma(a2, b, c); a3 = fma(a3, b, c);
    a4 = fma(a4, b, c); a5 = fma(a5, b, c); a6 = fma(a6, b, c); a7 = fma(a7, b, c);
  }
  const double r = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
  if (r == 123.456) sink[0] = r;
}

}  // namespace ipole

// Model sweep of the GRID model with the geometry done once (ipole_make_images_grid; what a GRMHD fit varies at
// fixed snapshot and viewing angle is the mass unit, R_low, R_high and the frequency).
//
// Along a stored path the eight-cell gather, the fluid four-velocity, the field direction, the plasma tetrad and the
// transport of the polarization basis do not depend on those numbers: the scales multiply rho and |b|, R(beta) enters
// Theta_e, the frequency multiplies omega.  So one sequential walk per ray (k_gridop, the walk of k_transfer_group without
// coefficients and Stokes numbers) composes the leg transport across the vacuum steps and leaves ONE COMPACT RECORD PER
// PLASMA STEP -- the 2x2 projection of the carried legs on the step's tetrad and the code-unit scalars -- and a second
// kernel (k_gridapply_sweep) walks the compact records once per parameter set.  Only 1 step in 8 crosses plasma, so the
// per-set work is the coefficients and the 4x4 step of those steps alone.
//
// Record k of slot li (walk order: k = 0 is the first plasma contact, far from the camera), three 32-byte parts:
//   part 0  {M11, M12, M21, M22}
//   part 1  {rho, |b| (code units), beta = p_gas / p_mag, (m_p/m_e)(gam - 1) u / rho}
//   part 2  {cos(angle to the field), omega nu_ref, d lambda, 0}
// laid out like the operator records of stepop.cuh with GOP_PARTS parts: the 32 rays of a group side by side.
// Record npl[li] holds the projection on the camera's legs.  npl[li] = -1: the ray is not this pass's (long-ray pass).
#pragma once
#include "stepop.cuh"

namespace ipole {

constexpr int GOP_PARTS = 3;
constexpr int GOP_DOUBLES = 4 * GOP_PARTS;

__device__ __forceinline__ size_t gop_addr(int64_t li, int cap, int k, int j) {
  return ((((size_t)(li >> 5) * (size_t)(cap + 1) + (size_t)k) * GOP_PARTS + j) * 32 + (size_t)(li & 31)) * 4;
}

struct GopArgs {
  CamDev cam; Units units;      // units: the reference the records are written with (the camera's own frequency)
  const void* model;            // GridParams
  int cap;
  int64_t base, count;
  const int32_t* order; const double* path; const int32_t* nsteps; const int2* srange; const int32_t* rank_slot;
  unsigned long long* queue;
  double* ops; int32_t* npl;    // compact records and their number per slot
};

// The walk of k_transfer_group (same scheduling: a warp takes 32 ranked slots in lockstep from the group's first contact).
__global__ void __launch_bounds__(IPOLE_RT_THREADS, IPOLE_RT_MINB) k_gridop(const __grid_constant__ GopArgs A) {
  const CamDev& C = A.cam;
  const size_t slot_doubles = (size_t)(A.cap + 1) * REC_DOUBLES;
  __shared__ __align__(8) unsigned char model_smem[sizeof(GridParams)];
  for (int i = threadIdx.x; i < (int)sizeof(GridParams); i += blockDim.x) model_smem[i] = ((const unsigned char*)A.model)[i];
  __syncthreads();
  const GridParams& GP = *(const GridParams*)model_smem;
  const int lane = threadIdx.x & 31;
  const int64_t n_groups = (A.count + 31) >> 5;
  for (;;) {
    __syncwarp();
    long long grp = 0;
    if (lane == 0) grp = (long long)atomicAdd(A.queue, 1ULL);
    grp = __shfl_sync(0xffffffffu, grp, 0);
    if (grp >= n_groups) break;
    const int64_t li = (grp << 5) + lane;      // place of the group member: where its compact records go
    double f1[4] = {0, 0, 0, 0}, f2[4] = {0, 0, 0, 0};
    double Xhi[4] = {0, 0, 0, 0}, Khi[4] = {0, 0, 0, 0};
    const double* rec = nullptr;
    int s0 = -1, s_lo = 0, k = 0;
    bool lit = false, mine = false;
    if (li < A.count) {
      const int64_t ls = A.rank_slot ? (int64_t)A.rank_slot[A.base + li] : li;
      const int32_t q = A.order ? A.order[A.base + ls] : (int32_t)(A.base + ls);
      int n = A.nsteps[q];
      mine = n >= 0;
      if (mine) {
        const int2 r = A.srange[q];
        s_lo = r.y;
        n = (r.x < 0) ? 0 : r.x + 1;
        if (n > 0) {
          rec = A.path + (size_t)ls * slot_doubles;
          double dl;
          load_record(rec + (size_t)n * REC_DOUBLES, Xhi, Khi, dl);
          s0 = n - 1;
        }
      }
    }
    int smax = s0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) smax = max(smax, __shfl_xor_sync(0xffffffffu, smax, o));
    for (int s = smax; s >= 0; --s) {
      if (s > s0) continue;
      double Xlo[4], Klo[4], dl;
      load_record(rec + (size_t)s * REC_DOUBLES, Xlo, Klo, dl);
      double Xm[4], Km[4];
#pragma unroll
      for (int m = 0; m < 4; ++m) { Xm[m] = 0.5 * (Xlo[m] + Xhi[m]); Km[m] = 0.5 * (Klo[m] + Khi[m]); }
      double prim[8];
      const bool maybe = (s >= s_lo) && grid_gather(GP, Xm, prim);
      if (lit || maybe) {
        Point p; Sym7 g; Inv6 gi; double Am[4][4];
        transport_generator(C.G, Xm, Km, p, g, gi, Am);
        const double h = 0.5 * dl;
        if (lit) { transport_apply(Am, h, f1); transport_apply(Am, h, f2); }
        double e1[4], e2[4], e1c[4], e2c[4];
        PlasmaFrame F;
        const GridScales S1 = {1.0, 1.0, 0.0, 0.0};   // scale-free state: n_e = rho, B = |b|, Theta_e without the R(beta) factor
        const bool applied = maybe && plasma_tetrad<MODEL_GRID, true>(C.G, model_smem, &S1, A.units, Xm, Km, p, g, gi, prim, e1, e2, e1c, e2c, F);
        if (applied) {
          double* o = A.ops + gop_addr(li, A.cap, k, 0);
          st_global_v4(o, dot4(e1c, f1), dot4(e1c, f2), dot4(e2c, f1), dot4(e2c, f2));
          const double beta = 2.0 * (GP.gam - 1.0) * prim[1] * ip_rcp(F.B * F.B);
          st_global_v4(o + 128, F.ne, F.B, beta, F.Th);
          st_global_v4(o + 256, F.cosT, F.nu, dl, 0.0);
          ++k;
#pragma unroll
          for (int m = 0; m < 4; ++m) { f1[m] = e1[m]; f2[m] = e2[m]; }
          lit = true;
        }
        if (lit) { transport_apply(Am, h, f1); transport_apply(Am, h, f2); }
      }
#pragma unroll
      for (int m = 0; m < 4; ++m) { Xhi[m] = Xlo[m]; Khi[m] = Klo[m]; }
    }
    if (li < A.count) {
      if (mine) {
        double* o = A.ops + gop_addr(li, A.cap, k, 0);
        st_global_v4(o, dot4(C.ecov1, f1), dot4(C.ecov1, f2), dot4(C.ecov2, f1), dot4(C.ecov2, f2));
      }
      A.npl[li] = mine ? k : -1;
    }
  }
}

struct GapArgs {
  int cap;
  int64_t base, count;
  const int32_t* order; const int32_t* rank_slot;
  const double* ops; const int32_t* npl;
  unsigned long long* queue;
  int n_models; const GridScales* lane_tab; const Units* units_arr; Units units_ref; size_t out_stride;
  double *I, *Q, *U, *V, *tau, *tauF;
};

// One warp walks the compact records of 32 slots in lockstep for ONE parameter set; the sets of a group follow each
// other in the queue, so its records are re-read from L2.  Per record what k_transfer<grid> does after its geometry:
// scales, R(beta), the eight coefficients, the closed-form 4x4 step.
__global__ void __launch_bounds__(IPOLE_AP_THREADS, 3) k_gridapply_sweep(const __grid_constant__ GapArgs A) {
  const int lane = threadIdx.x & 31;
  const int64_t n_groups = (A.count + 31) >> 5;
  const int64_t n_items = n_groups * A.n_models;
  for (;;) {
    __syncwarp();
    long long g = 0;
    if (lane == 0) g = (long long)atomicAdd(A.queue, 1ULL);
    g = __shfl_sync(0xffffffffu, g, 0);
    if (g >= n_items) break;
    const long long grp = g / A.n_models;
    const int mi = (int)(g - grp * A.n_models);
    const GridScales Sm = A.lane_tab[mi];
    const Units Um = A.units_arr[mi];
    const double nu_r = Um.nu_obs / A.units_ref.nu_obs;
    const size_t oo = (size_t)mi * A.out_stride;
    const int64_t li = (grp << 5) + lane;
    int32_t q = 0;
    int n = -1;                                  // compact records of this lane's ray; -1: not this pass's ray
    if (li < A.count) {
      const int64_t ls = A.rank_slot ? (int64_t)A.rank_slot[A.base + li] : li;
      q = A.order ? A.order[A.base + ls] : (int32_t)(A.base + ls);
      n = A.npl[li];
    }
    int kmax = n;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) kmax = max(kmax, __shfl_xor_sync(0xffffffffu, kmax, o));
    double S[4] = {0, 0, 0, 0}, tau = 0.0, tauF = 0.0;
    const double* base = A.ops + gop_addr(li, A.cap, 0, 0);
    for (int k = 0; k < kmax; ++k) {
      if (k >= n) continue;
      const double* p = base + (size_t)k * (GOP_PARTS * 128);
      double m11, m12, m21, m22, rho, Bc, beta, thf, cosT, nu, dl, z;
      ld_global_v4(p, m11, m12, m21, m22);
      ld_global_v4(p + 128, rho, Bc, beta, thf);
      ld_global_v4(p + 256, cosT, nu, dl, z);
      stokes_congruence(m11, m12, m21, m22, S);
      const double b2 = beta * beta;
      const double R = (Sm.Rhigh * b2 + Sm.Rlow) * ip_rcp(1.0 + b2);
      const Coeff c = synchrotron_invariant(rho * Sm.ne_unit, thf * ip_rcp(1.0 + R), Bc * Sm.B_unit, cosT, nu * nu_r);
      const double ds = dl * Um.dl_unit;
      stokes_step_qv<false>(c.aI, c.aQ, c.aV, c.rQ, c.rV, ds, c.jI, c.jQ, c.jV, S);
      tau += c.aI * ds;
      tauF += fabs(c.rV) * ds;
    }
    if (n >= 0) {
      double m11, m12, m21, m22;
      ld_global_v4(base + (size_t)n * (GOP_PARTS * 128), m11, m12, m21, m22);
      stokes_congruence(m11, m12, m21, m22, S);
      const double nu3 = Um.nu_obs * Um.nu_obs * Um.nu_obs;
      A.I[oo + q] = S[0] * nu3; A.Q[oo + q] = S[1] * nu3; A.U[oo + q] = S[2] * nu3; A.V[oo + q] = S[3] * nu3;
      if (A.tau) A.tau[oo + q] = tau;
      if (A.tauF) A.tauF[oo + q] = tauF;
    }
  }
}

}  // namespace ipole

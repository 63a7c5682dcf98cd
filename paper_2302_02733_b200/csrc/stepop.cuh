// Transfer split in two kernels (SURVEY.md section 8(a) rows a-4 ... a-7; "at every single step ...
// evaluate emission, self-absorption and Faraday coefficients at a given point").
//
// Along a stored path everything a transfer step needs -- the midpoint metric and transport generator, the plasma
// state, the plasma-frame tetrad, the eight coefficients -- depends on the two end points of that step alone, not on
// the polarization state carried by the ray.  Even the 2x2 projection M of the carried legs on a step's new tetrad is
// state-free as long as the previous (farther) step also crossed plasma: the carried legs are then that step's own
// tetrad legs, transported by its P and by this step's P ("factorised coherency tensor").  What
// is sequential is only   S <- C(M) S,   S <- O S + P J   on four Stokes numbers.  So:
//
//   k_stepop  one thread per STEP (a warp takes 31 consecutive steps of one ray plus one halo step, lanes <-> steps):
//             metric, generator, flow, tetrad, leg transport; writes one 64-B operator record per step:
//             M (4), and what the coefficients need: ln r, cos(pitch angle), local frequency, ds.  No loop-carried state.
//   k_apply   one warp per 32 RAYS, lane <-> ray, in lockstep from the far end to the camera: plasma scalars, the eight
//             coefficients, congruence + the analytic 4x4 step, then the camera projection.  Its record stream (64 B per
//             step, coalesced) runs at HBM speed; the coefficient arithmetic lives here because this kernel has the
//             registers to spare for 5 warps per scheduler, which the geometry kernel has not.
//
// A ray with a step that is NOT applied (no plasma there, or a degenerate tetrad) breaks the state-free chain of the
// legs; k_stepop lists such rays (`irregular`) and the single-kernel k_transfer renders them from the same path
// buffer.  With the analytic ADAF flow every step crosses plasma, so the list is empty in practice.
#pragma once
#include "kernels.cuh"
#include "edf.cuh"

namespace ipole {

constexpr int OP_PARTS = 2;        // operator record: two 32-B parts, {M11, M12, M21, M22} and {ln r, cos theta_B, nu, ds}
constexpr int OP_DOUBLES = 4 * OP_PARTS;

// Layout of the operator records of a batch: rays are taken in groups of 32 consecutive slots (one k_apply warp walks
// a group in lockstep, lane <-> ray), and the record of (slot li, step s) is cut in OP_PARTS 32-byte parts j:
//   ops[ (((li/32) * (cap+1) + s) * OP_PARTS + j) * 32 + li%32 ][4 doubles]
// so that for one step the 32 lanes of k_apply read OP_PARTS x 1 KB of contiguous memory (8 full lines per 256-bit load
// instead of 32 partial ones), while k_stepop -- lanes <-> consecutive steps of one ray -- writes full 32-B sectors.
__device__ __forceinline__ size_t op_addr(int64_t li, int cap, int s, int j) {
  return ((((size_t)(li >> 5) * (size_t)(cap + 1) + (size_t)s) * OP_PARTS + j) * 32 + (size_t)(li & 31)) * 4;
}

struct OpArgs {
  CamDev cam;
  Units units;
  const void* model;          // device pointer to AdafParams
  int cap;                    // steps per slot (records = cap + 1) of both the path and the operator buffer
  int64_t base, count;        // rays [base, base+count) of the order
  const int* count_dev;       // if non-null, count = *count_dev (retry level on the side stream)
  const int32_t* order;
  const double* path;         // [count][cap+1][8]
  const int32_t* nsteps;      // indexed by q; -1 = overflowed its slot (long-ray pass)
  unsigned long long* queue;
  double* ops;                // operator records of the batch, layout op_addr(); record n of a ray: camera projection (4), irregular flag (1)
  int32_t* irr_slots; int* irr_count;   // slots (positions in the batch) of the rays left to k_transfer
  int test_irregular;         // tests: declare every 7th slot irregular, so that the hand-over to k_transfer is exercised
  // many cameras per launch (k_stepop<MODEL, true>): ray q belongs to camera q / rays_per_cam
  const CamDev* cams; const Units* units_arr; int64_t rays_per_cam;
  const int32_t* pos;         // [base + li]: where k_apply finds slot li (k_rank_window); null: at li
};

// k_apply walks 32 rays in lockstep, so the rays of a group should be equally long.  The batch is in order of PREDICTED
// length (probe pass); once k_geodesic has run the true step counts are known, and every window of RANK_WINDOW consecutive
// slots is re-ranked by them: pos[base + li] = the place of slot li's operator records, slot[base + a] = the slot at place a.
// The grid model's lockstep kernel (k_transfer_group) uses the same ranking on each ray's plasma-contact range.
constexpr int RANK_WINDOW = 1024;
struct RankArgs {
  int64_t base, count; const int* count_dev; const int32_t* order; const int32_t* nsteps; int32_t* pos; int32_t* slot;
  const int2* srange;         // grid model (k_transfer_group): rank by the plasma-contact range instead (first contact, then last)
};
__global__ void __launch_bounds__(RANK_WINDOW) k_rank_window(RankArgs A) {
  __shared__ unsigned long long key[RANK_WINDOW];
  const int64_t count = A.count_dev ? (int64_t)*A.count_dev : A.count;
  const int64_t w0 = (int64_t)blockIdx.x * RANK_WINDOW;
  if (w0 >= count) return;
  const int t = threadIdx.x;
  unsigned long long k = ~0ULL;                  // padding sorts last
  if (w0 + t < count) {
    const int32_t q = A.order ? A.order[A.base + w0 + t] : (int32_t)(A.base + w0 + t);
    int n = A.nsteps[q], lo = 0;
    if (n < 0) n = 0;
    else if (A.srange) { const int2 r = A.srange[q]; n = r.x + 1; lo = r.y; }   // steps the walk takes; where the plasma ends
    n = min(n, 0x1fffff); lo = min(max(lo, 0), 0x1fffff);
    // longest first, then by the second key, then by slot: a fixed order
    k = ((unsigned long long)(0x1fffff - n) << 31) | ((unsigned long long)lo << 10) | (unsigned)t;
  }
  key[t] = k;
  __syncthreads();
  for (int size = 2; size <= RANK_WINDOW; size <<= 1)
    for (int stride = size >> 1; stride > 0; stride >>= 1) {
      const int partner = t ^ stride;
      if (partner > t) {
        const bool up = (t & size) == 0;
        const unsigned long long a = key[t], b = key[partner];
        if ((a > b) == up) { key[t] = b; key[partner] = a; }
      }
      __syncthreads();
    }
  if (w0 + t < count) {
    const int src = (int)(key[t] & 1023ULL);
    A.slot[A.base + w0 + t] = (int32_t)(w0 + src);
    A.pos[A.base + w0 + src] = (int32_t)(w0 + t);
  }
}

#ifndef IPOLE_OP_THREADS
#define IPOLE_OP_THREADS 128
#endif
#ifndef IPOLE_OP_MINB
#define IPOLE_OP_MINB 3
#endif

__device__ __forceinline__ void shfl_down4(const double v[4], double o[4]) {
#pragma unroll
  for (int m = 0; m < 4; ++m) o[m] = __shfl_down_sync(0xffffffffu, v[m], 1);
}

template <int MODEL, bool MC = false>
__global__ void __launch_bounds__(IPOLE_OP_THREADS, IPOLE_OP_MINB) k_stepop(const __grid_constant__ OpArgs A) {
  static_assert(MODEL == MODEL_ADAF, "the step-parallel pass is built for the analytic flow");
  const CamDev& C0 = A.cam;
  __shared__ __align__(8) unsigned char model_smem[sizeof(AdafParams)];
  for (int i = threadIdx.x; i < (int)sizeof(AdafParams); i += blockDim.x) model_smem[i] = ((const unsigned char*)A.model)[i];
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const int64_t count = A.count_dev ? (int64_t)*A.count_dev : A.count;
  const size_t slot_rec = (size_t)(A.cap + 1) * REC_DOUBLES;
  // MC: the ray's own camera (geometry, transverse legs) and units, and the flow's ISCO for that spin, in registers
  AdafParams model_l = *(const AdafParams*)model_smem;
  Geom Gl = C0.G;
  double ec1[4], ec2[4], nu_obs_l = A.units.nu_obs, dl_unit_l = A.units.dl_unit;
#pragma unroll
  for (int m = 0; m < 4; ++m) { ec1[m] = C0.ecov1[m]; ec2[m] = C0.ecov2[m]; }

  for (;;) {
    // lane 0 leaves the previous iteration later than the others (it writes the ray's last record): without this
    // the warp stays split in 1 + 31 threads and issues every instruction of the body twice
    __syncwarp();
    long long li = 0;
    if (lane == 0) li = (long long)atomicAdd(A.queue, 1ULL);
    li = __shfl_sync(0xffffffffu, li, 0);
    if (li >= count) break;
    const int32_t q = A.order ? A.order[A.base + li] : (int32_t)(A.base + li);
    const int n = A.nsteps[q];
    if (n < 0) continue;                     // overflowed its slot: done by the long-ray pass
    if (MC) {
      const int ci = (int)(q / A.rays_per_cam);
      const CamDev& Cc = A.cams[ci];
      Gl = Cc.G;
#pragma unroll
      for (int m = 0; m < 4; ++m) { ec1[m] = Cc.ecov1[m]; ec2[m] = Cc.ecov2[m]; }
      nu_obs_l = A.units_arr[ci].nu_obs; dl_unit_l = A.units_arr[ci].dl_unit;
      model_l.r_isco = isco_radius(Gl.a);
    }
    const Geom& G = MC ? Gl : C0.G;
    Units Ul = A.units;
    if (MC) { Ul.nu_obs = nu_obs_l; Ul.dl_unit = dl_unit_l; }
    const void* model = MC ? (const void*)&model_l : (const void*)model_smem;
    const double* rec = A.path + (size_t)li * slot_rec;
    const int64_t la = A.pos ? (int64_t)A.pos[A.base + li] : li;   // place of this ray's operator records
    bool regular = true;
    double mc[4] = {0.0, 0.0, 0.0, 0.0};     // lane 0, first chunk: projection of step 0's legs on the camera tetrad

    for (int s0 = 0; s0 < n; s0 += 31) {
      const int s = s0 + lane;               // step s: from point s+1 to point s (point 0 = camera)
      const bool act = s < n;
      // the next chunk's records (lane l: points s0+31+l and, for the halo lane, one more) into L1 while this one computes
      if (s + 31 <= n) asm volatile("prefetch.global.L1 [%0];" ::"l"(rec + (size_t)(s + 31) * REC_DOUBLES));
      if (lane == 31 && s + 32 <= n) asm volatile("prefetch.global.L1 [%0];" ::"l"(rec + (size_t)(s + 32) * REC_DOUBLES));
      // fo: this step's new legs after its second half transport, P e_(a): what the next step towards the camera receives
      double fo1[4] = {0, 0, 0, 0}, fo2[4] = {0, 0, 0, 0};
      double e1c[4], e2c[4], Am[4][4];
      double h = 0.0, dl = 0.0, x1m = 0.0;
      PlasmaFrame F;
      bool applied = false;
      if (act) {
        double Xm[4], Km[4];
        {
          double Xlo[4], Klo[4], Xhi[4], Khi[4], dlh;
          load_record(rec + (size_t)s * REC_DOUBLES, Xlo, Klo, dl);
          load_record(rec + (size_t)(s + 1) * REC_DOUBLES, Xhi, Khi, dlh);
#pragma unroll
          for (int m = 0; m < 4; ++m) { Xm[m] = 0.5 * (Xlo[m] + Xhi[m]); Km[m] = 0.5 * (Klo[m] + Khi[m]); }
        }
        x1m = Xm[1];
        Point p; Sym7 g; Inv6 gi;
        transport_generator(G, Xm, Km, p, g, gi, Am);
        h = 0.5 * dl;
        double e1[4], e2[4];
        applied = plasma_tetrad<MODEL, false>(G, model, nullptr, Ul, Xm, Km, p, g, gi, nullptr, e1, e2, e1c, e2c, F);
        if (applied) {
#pragma unroll
          for (int m = 0; m < 4; ++m) { fo1[m] = e1[m]; fo2[m] = e2[m]; }
          transport_apply(Am, h, fo1);
          transport_apply(Am, h, fo2);
        }
      }
      regular &= (applied || !act);
      // legs arriving at step s = legs leaving step s+1 (the neighbouring lane)
      double fi1[4], fi2[4];
      shfl_down4(fo1, fi1);
      shfl_down4(fo2, fi2);
      if (act && lane < 31) {
        double m11 = 0.0, m12 = 0.0, m21 = 0.0, m22 = 0.0;
        if (s < n - 1 && applied) {          // the far end starts dark: nothing arrives there
          transport_apply(Am, h, fi1);
          transport_apply(Am, h, fi2);
          m11 = dot4(e1c, fi1); m12 = dot4(e1c, fi2); m21 = dot4(e2c, fi1); m22 = dot4(e2c, fi2);
        }
        double* o = A.ops + op_addr(la, A.cap, s, 0);   // part 1 at o + 128
        st_global_v4(o, m11, m12, m21, m22);
        st_global_v4(o + 128, x1m, applied ? F.cosT : 0.0, applied ? F.nu : 0.0, dl * Ul.dl_unit);
        if (s == 0) {
          mc[0] = dot4(MC ? ec1 : C0.ecov1, fo1); mc[1] = dot4(MC ? ec1 : C0.ecov1, fo2);
          mc[2] = dot4(MC ? ec2 : C0.ecov2, fo1); mc[3] = dot4(MC ? ec2 : C0.ecov2, fo2);
        }
      }
    }
    regular = __all_sync(0xffffffffu, regular) && !(A.test_irregular && (li % 7) == 3);
    if (lane == 0) {
      double* o = A.ops + op_addr(la, A.cap, n, 0);
      st_global_v4(o, mc[0], mc[1], mc[2], mc[3]);
      st_global_v4(o + 128, regular ? 0.0 : 1.0, 0.0, 0.0, 0.0);
      if (!regular) { const int w = atomicAdd(A.irr_count, 1); A.irr_slots[w] = (int32_t)li; }
    }
  }
}

struct ApArgs {
  const int32_t* slot;        // [base + a]: the slot whose operator records sit at place a (k_rank_window); null: a
  const double* nu3_arr; int64_t rays_per_cam;   // many cameras per launch: nu_obs^3 of camera q / rays_per_cam (nullable)
  AdafParams model;           // the three power laws (by value: 56 B)
  EdfDev edf;                 // k_apply<true>: j, alpha by quadrature over the electron distribution (edf.cuh)
  double nu3;                 // nu_obs^3: invariant I/nu^3 -> specific intensity at the camera
  int cap;
  int64_t base, count;
  const int* count_dev;       // if non-null, count = *count_dev
  const int32_t* order;
  const double* ops;
  const int32_t* nsteps;
  unsigned long long* queue;
  double *I, *Q, *U, *V, *tau, *tauF;   // indexed by q
  // model sweep (k_apply<false, true>; ipole_make_images_adaf): work item = (group of 32 rays, parameter set m).  The operator
  // records do not depend on the parameter set (flow and field DIRECTION are the model's geometry); its three power laws
  // come from lane_tab[m], its frequency from units_arr[m] relative to units_ref (the units k_stepop wrote the records with);
  // outputs of set m start at plane + m * out_stride
  int n_models; const AdafParams* lane_tab; const Units* units_arr; Units units_ref; size_t out_stride;
};

#ifndef IPOLE_AP_THREADS
#define IPOLE_AP_THREADS 128
#endif
#ifndef IPOLE_AP_MINB
#define IPOLE_AP_MINB 4
#endif

// a step that is not thin (never on the analytic workloads): the closed form, kept out of the slim loop.  Stokes in
// and out by value, so that the caller's S stays in registers.
struct Stokes4 { double I, Q, U, V; };
__device__ __noinline__ Stokes4 stokes_step_qv_closed(double aI, double aQ, double aV, double rQ, double rV, double jI, double jQ,
                                                      double jV, Stokes4 in) {
  double S[4] = {in.I, in.Q, in.U, in.V};
  stokes_step_qv<false>(aI, aQ, aV, rQ, rV, 1.0, jI, jQ, jV, S);
  Stokes4 o = {S[0], S[1], S[2], S[3]};
  return o;
}

// One warp walks a group of 32 consecutive slots of the batch in lockstep, lane <-> ray, from the longest ray's far end
// to the camera; a lane joins when the walk reaches its own far end.  Rays are ordered by predicted step count, so
// the 32 rays of a group have similar lengths.  The record of the next step is loaded (three coalesced 256-bit loads)
// while the current one is applied.
// EDF: the coefficients of a step by numerical integration over the electron distribution function (edf.cuh)
// (2 blocks per SM: the node loop, unrolled 8 times with no branch in its body, wants ~220 registers to keep eight
// reciprocal -> rsqrt -> exp chains in flight; measured faster than 3 blocks at 164, profiles/r2_notes.md)
#ifndef IPOLE_AP_EDF_MINB
#define IPOLE_AP_EDF_MINB 2
#endif
template <bool EDF, bool SWEEP = false>
__global__ void __launch_bounds__(IPOLE_AP_THREADS, EDF ? IPOLE_AP_EDF_MINB : IPOLE_AP_MINB) k_apply(const __grid_constant__ ApArgs A) {
  static_assert(!(EDF && SWEEP), "the sweep is built for the thermal coefficients");
  extern __shared__ double4 edf_nodes_smem[];          // EDF: the per-node constants {x^-1/2, F, G, H} (edf.cuh)
  if (EDF) {
    for (int k = threadIdx.x; k < A.edf.n_nodes; k += blockDim.x) edf_nodes_smem[k] = A.edf.nodes[k];
    __syncthreads();
  }
  const double4* edf_nodes = edf_nodes_smem;
  const int lane = threadIdx.x & 31;
  const int64_t count = A.count_dev ? (int64_t)*A.count_dev : A.count;
  const int64_t n_groups = (count + 31) >> 5;
  const int64_t n_items = SWEEP ? n_groups * A.n_models : n_groups;
  for (;;) {
    __syncwarp();
    long long g = 0;
    if (lane == 0) g = (long long)atomicAdd(A.queue, 1ULL);
    g = __shfl_sync(0xffffffffu, g, 0);
    if (g >= n_items) break;
    // SWEEP: consecutive work items are the parameter sets of one ray group, so its records are re-read from L2
    int mi = 0;
    AdafParams Mm = A.model;
    double nu_r = 1.0, ds_r = 1.0, nu3_m = A.nu3;
    size_t oo = 0;
    if (SWEEP) {
      const long long grp = g / A.n_models;
      mi = (int)(g - grp * A.n_models);
      g = grp;
      Mm = A.lane_tab[mi];
      const Units Um = A.units_arr[mi];
      nu_r = Um.nu_obs / A.units_ref.nu_obs;       // exactly 1 where the set keeps the camera's frequency
      ds_r = Um.dl_unit / A.units_ref.dl_unit;
      nu3_m = Um.nu_obs * Um.nu_obs * Um.nu_obs;
      oo = (size_t)mi * A.out_stride;
    }
    const int64_t li = (g << 5) + lane;          // place in the batch's operator buffer
    int32_t q = 0;
    int n = 0;                                   // steps of this lane's ray; 0: nothing to do
    double mc[4] = {0, 0, 0, 0};
    if (li < count) {
      const int64_t ls = A.slot ? (int64_t)A.slot[A.base + li] : li;
      q = A.order ? A.order[A.base + ls] : (int32_t)(A.base + ls);
      n = A.nsteps[q];
      if (n < 0) n = 0;                          // overflowed its slot: long-ray pass
      else {
        double flag, z0, z1, z2;
        ld_global_v4(A.ops + op_addr(li, A.cap, n, 0), mc[0], mc[1], mc[2], mc[3]);
        ld_global_v4(A.ops + op_addr(li, A.cap, n, 1), flag, z0, z1, z2);
        if (flag != 0.0) n = 0;                  // irregular: rendered by k_transfer
      }
    }
    int smax = n;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) smax = max(smax, __shfl_xor_sync(0xffffffffu, smax, o));
    double S[4] = {0, 0, 0, 0}, tau = 0.0, tauF = 0.0;
    double R[OP_DOUBLES] = {0, 0, 0, 0, 0, 0, 0, 0};
    const double* base = A.ops + op_addr(li, A.cap, 0, 0);   // step s, part j at base + (s*OP_PARTS + j) * 128
    auto load = [&](int s) {
      const double* p = base + (size_t)s * (OP_PARTS * 128);
      ld_global_v4(p, R[0], R[1], R[2], R[3]);
      ld_global_v4(p + 128, R[4], R[5], R[6], R[7]);
    };
    if (smax > 0 && smax - 1 < n) load(smax - 1);   // (a group whose rays all went to another pass has smax = 0)
    for (int s = smax - 1; s >= 0; --s) {
      const bool on = s < n;
      const double m11 = R[0], m12 = R[1], m21 = R[2], m22 = R[3];
      const double x1 = R[4], cosT = R[5], nu = SWEEP ? R[6] * nu_r : R[6], ds = SWEEP ? R[7] * ds_r : R[7];
      if (s > 0 && s - 1 < n) load(s - 1);
      if (on) {
        stokes_congruence(m11, m12, m21, m22, S);
        double ne, Th, B;
        adaf_scalars(SWEEP ? Mm : A.model, x1, ne, Th, B);
        const Coeff c = EDF ? synchrotron_edf_invariant(A.edf, edf_nodes, ne, Th, B, cosT, nu) : synchrotron_invariant(ne, Th, B, cosT, nu);
        // (products rounded on their own, not contracted into the sums of the step: k_apply_wide hands the same eight
        // numbers from lane to lane and must get the same bits)
        const double xI = __dmul_rn(c.aI, ds), xQ = __dmul_rn(c.aQ, ds), xV = __dmul_rn(c.aV, ds), yQ = __dmul_rn(c.rQ, ds), yV = __dmul_rn(c.rV, ds);
        const double eI = __dmul_rn(c.jI, ds), eQ = __dmul_rn(c.jQ, ds), eV = __dmul_rn(c.jV, ds);
        if (IP_UNLIKELY(!stokes_step_qv_series(xI, xQ, xV, yQ, yV, 1.0, eI, eQ, eV, S))) {
          const Stokes4 in = {S[0], S[1], S[2], S[3]};
          const Stokes4 o = stokes_step_qv_closed(xI, xQ, xV, yQ, yV, eI, eQ, eV, in);
          S[0] = o.I; S[1] = o.Q; S[2] = o.U; S[3] = o.V;
        }
        tau = __dadd_rn(tau, xI);                // (no contraction with the product above: k_apply_wide adds the same numbers)
        tauF = __dadd_rn(tauF, fabs(yV));
      }
    }
    if (n > 0) {
      stokes_congruence(mc[0], mc[1], mc[2], mc[3], S);
      const double nu3 = SWEEP ? nu3_m : (A.nu3_arr ? A.nu3_arr[q / A.rays_per_cam] : A.nu3);
      A.I[oo + q] = S[0] * nu3; A.Q[oo + q] = S[1] * nu3; A.U[oo + q] = S[2] * nu3; A.V[oo + q] = S[3] * nu3;
      if (A.tau) A.tau[oo + q] = tau;
      if (A.tauF) A.tauF[oo + q] = tauF;
    }
  }
}

// k_apply for launches that cannot fill the GPU (adaptive levels, retry and long-ray passes, pixel lists, small images):
// LANES LANES PER RAY instead of one.  The lockstep kernel above gives every ray one lane, and a lone photon-ring ray of
// 4 500 steps is then 4 500 x ~560 dependent instructions = 9 ms however empty the GPU is.  Here the LANES lanes of a ray
// take LANES consecutive steps and evaluate their scalars and coefficients side by side (they do not depend on the Stokes
// numbers); only the congruence and the 4x4 step run in sequence, every lane of the ray doing the same update on values
// broadcast from the lane that owns the step.  Per ray the arithmetic and its order are k_apply's (same functions, same
// operands, every rounding spelt out): the same bits.  Dependent instructions per step: (480 + 80 LANES) / LANES -- 95 at
// 32 lanes, 140 at 8; warp instructions per ray step: 15 + 80 LANES / 32 -- 95 at 32 lanes, 35 at 8 (k_apply: 17.5).  So
// 32 lanes for a handful of rays, 8 for a few thousand.
template <int LANES>
__global__ void __launch_bounds__(IPOLE_AP_THREADS, IPOLE_AP_MINB) k_apply_wide(const __grid_constant__ ApArgs A) {
  constexpr int RPW = 32 / LANES;                // rays per warp
  const int lane = threadIdx.x & 31;
  const int sub = lane / LANES, sl = lane % LANES;
  const int64_t count = A.count_dev ? (int64_t)*A.count_dev : A.count;
  const int64_t n_items = (count + RPW - 1) / RPW;
  for (;;) {
    __syncwarp();
    long long g = 0;
    if (lane == 0) g = (long long)atomicAdd(A.queue, 1ULL);
    g = __shfl_sync(0xffffffffu, g, 0);
    if (g >= n_items) break;
    const int64_t li = g * RPW + sub;            // place in the batch's operator buffer
    int32_t q = 0;
    int n = 0;                                   // steps of this ray; 0: nothing to do
    double mc[4] = {0, 0, 0, 0};
    if (li < count) {
      const int64_t ls = A.slot ? (int64_t)A.slot[A.base + li] : li;
      q = A.order ? A.order[A.base + ls] : (int32_t)(A.base + ls);
      n = A.nsteps[q];
      if (n < 0) n = 0;                          // overflowed its slot: long-ray pass
      else {
        double flag, z0, z1, z2;
        ld_global_v4(A.ops + op_addr(li, A.cap, n, 0), mc[0], mc[1], mc[2], mc[3]);
        ld_global_v4(A.ops + op_addr(li, A.cap, n, 1), flag, z0, z1, z2);
        if (flag != 0.0) n = 0;                  // irregular: rendered by k_transfer
      }
    }
    int nmax = n;
    if (RPW > 1) {
#pragma unroll
      for (int o = 16; o >= LANES; o >>= 1) nmax = max(nmax, __shfl_xor_sync(0xffffffffu, nmax, o));
    }
    double S[4] = {0, 0, 0, 0}, tau = 0.0, tauF = 0.0;
    const double* base = A.ops + op_addr(li < count ? li : 0, A.cap, 0, 0);
    for (int done = 0; done < nmax; done += LANES) {
      const int s_top = n - 1 - done;            // the ray's chunk is walked from its lane 0 on; < 0: the ray is through
      const int s = s_top - sl;
      double v[12] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
      if (s >= 0) {
        const double* p = base + (size_t)s * (OP_PARTS * 128);
        double x1, cosT, nu, ds;
        ld_global_v4(p, v[0], v[1], v[2], v[3]);
        ld_global_v4(p + 128, x1, cosT, nu, ds);
        double ne, Th, B;
        adaf_scalars(A.model, x1, ne, Th, B);
        const Coeff c = synchrotron_invariant(ne, Th, B, cosT, nu);
        v[4] = __dmul_rn(c.aI, ds); v[5] = __dmul_rn(c.aQ, ds); v[6] = __dmul_rn(c.aV, ds); v[7] = __dmul_rn(c.rQ, ds); v[8] = __dmul_rn(c.rV, ds);
        v[9] = __dmul_rn(c.jI, ds); v[10] = __dmul_rn(c.jQ, ds); v[11] = __dmul_rn(c.jV, ds);
      }
      const int m = min(LANES, s_top + 1);
      int mmax = m;
      if (RPW > 1) {
#pragma unroll
        for (int o = 16; o >= LANES; o >>= 1) mmax = max(mmax, __shfl_xor_sync(0xffffffffu, mmax, o));
      }
      for (int j = 0; j < mmax; ++j) {
        double w[12];
#pragma unroll
        for (int i = 0; i < 12; ++i) w[i] = __shfl_sync(0xffffffffu, v[i], j, LANES);
        if (j < m) {
          stokes_congruence(w[0], w[1], w[2], w[3], S);
          if (IP_UNLIKELY(!stokes_step_qv_series(w[4], w[5], w[6], w[7], w[8], 1.0, w[9], w[10], w[11], S))) {
            const Stokes4 in = {S[0], S[1], S[2], S[3]};
            const Stokes4 o = stokes_step_qv_closed(w[4], w[5], w[6], w[7], w[8], w[9], w[10], w[11], in);
            S[0] = o.I; S[1] = o.Q; S[2] = o.U; S[3] = o.V;
          }
          tau = __dadd_rn(tau, w[4]);
          tauF = __dadd_rn(tauF, fabs(w[8]));
        }
      }
    }
    if (n > 0 && sl == 0) {
      stokes_congruence(mc[0], mc[1], mc[2], mc[3], S);
      const double nu3 = A.nu3_arr ? A.nu3_arr[q / A.rays_per_cam] : A.nu3;
      A.I[q] = S[0] * nu3; A.Q[q] = S[1] * nu3; A.U[q] = S[2] * nu3; A.V[q] = S[3] * nu3;
      if (A.tau) A.tau[q] = tau;
      if (A.tauF) A.tauF[q] = tauF;
    }
  }
}

// Unpolarized sweep ("nonpolarized images" of the fitting loop; R-12) on the same operator records:
// I alone needs their second half only -- ln r, the angle to the field, the frequency, the step length -- and per
// parameter set the three power laws, j_I, alpha_I and the exact scalar step of k_transfer_unpol:
//   I <- I e^{-x} + j ds (1 - e^{-x})/x,  x = alpha ds.
// Work items and lockstep walk as in k_apply<false, true>.
#ifndef IPOLE_APU_MINB
#define IPOLE_APU_MINB 4
#endif
__global__ void __launch_bounds__(IPOLE_AP_THREADS, IPOLE_APU_MINB) k_apply_unpol_sweep(const __grid_constant__ ApArgs A) {
  const int lane = threadIdx.x & 31;
  const int64_t count = A.count;
  const int64_t n_groups = (count + 31) >> 5;
  const int64_t n_items = n_groups * A.n_models;
  for (;;) {
    __syncwarp();
    long long g = 0;
    if (lane == 0) g = (long long)atomicAdd(A.queue, 1ULL);
    g = __shfl_sync(0xffffffffu, g, 0);
    if (g >= n_items) break;
    const long long grp = g / A.n_models;
    const int mi = (int)(g - grp * A.n_models);
    const AdafParams Mm = A.lane_tab[mi];
    const Units Um = A.units_arr[mi];
    const double nu_r = Um.nu_obs / A.units_ref.nu_obs, ds_r = Um.dl_unit / A.units_ref.dl_unit;
    const size_t oo = (size_t)mi * A.out_stride;
    const int64_t li = (grp << 5) + lane;
    int32_t q = 0;
    int n = 0;
    if (li < count) {
      const int64_t ls = A.slot ? (int64_t)A.slot[A.base + li] : li;
      q = A.order ? A.order[A.base + ls] : (int32_t)(A.base + ls);
      n = A.nsteps[q];
      if (n < 0) n = 0;                          // overflowed its slot: long-ray pass
    }
    int smax = n;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) smax = max(smax, __shfl_xor_sync(0xffffffffu, smax, o));
    double I = 0.0, tau = 0.0;
    double R[4] = {0, 0, 0, 0};
    const double* base = A.ops + op_addr(li, A.cap, 0, 1);   // part 1 of step s at base + s * OP_PARTS * 128
    auto load = [&](int s) { ld_global_v4(base + (size_t)s * (OP_PARTS * 128), R[0], R[1], R[2], R[3]); };
    if (smax > 0 && smax - 1 < n) load(smax - 1);
    for (int s = smax - 1; s >= 0; --s) {
      const bool on = s < n;
      const double x1 = R[0], cosT = R[1], nu = R[2] * nu_r, ds = R[3] * ds_r;
      if (s > 0 && s - 1 < n) load(s - 1);
      if (on) {
        double ne, Th, B;
        adaf_scalars(Mm, x1, ne, Th, B);
        const Coeff c = synchrotron_invariant(ne, Th, B, cosT, nu);
        const double x = c.aI * ds;
        const double em = ip_expm1(-x);
        const double E = (x > 0.0) ? -em * ip_rcp(x) : 1.0;
        I = I + I * em + c.jI * ds * E;
        tau += x;
      }
    }
    if (n > 0) {
      const double nu3 = Um.nu_obs * Um.nu_obs * Um.nu_obs;
      A.I[oo + q] = I * nu3; A.Q[oo + q] = 0.0; A.U[oo + q] = 0.0; A.V[oo + q] = 0.0;
      if (A.tau) A.tau[oo + q] = tau;
      if (A.tauF) A.tauF[oo + q] = 0.0;
    }
  }
}

}  // namespace ipole

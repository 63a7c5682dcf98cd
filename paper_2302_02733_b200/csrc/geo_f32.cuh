// FP32 study kernel ("further code acceleration may be also obtained by switching to
// single precision calculations"; the paper's consumer GPU has 1/64 of its FP32 rate in FP64).
//
// k_geodesic_f32 is k_geodesic with the geodesic state, the metric functions and the RK4 push in single precision: the
// same step rule, stop rules, turning-point count, queue and path-record layout (records are widened to FP64 when stored,
// so the FP64 transfer kernels run on them unchanged -- a mixed-precision image).  It exists to MEASURE what the paper's
// suggestion is worth on this GPU (ipole_set_geodesic_fp32; bench.py --fp32-geodesic; profiles/r2_fp32_study.md): it is
// not a product path and nothing else calls it.  The acceleration uses the Kerr-Schild form of geom.cuh
// (geodesic_accel_ks) typed again in float; every stage point is evaluated in full (expf, sincosf).
#pragma once
#include "kernels.cuh"

namespace ipole {

struct PointF { float r, tp, tpp, s, c; };

__device__ __forceinline__ void point_full_f(const Geom& G, const float X[4], PointF& p) {
  p.r = expf(X[1]);
  float th;
  if (G.h_is_one) { th = 3.14159265358979f * X[2]; p.tp = 3.14159265358979f; p.tpp = 0.f; }
  else {
    float s2, c2;
    sincosf(6.28318530717959f * X[2], &s2, &c2);
    const float q = 1.f - (float)G.hslope;
    th = 3.14159265358979f * X[2] + 0.5f * q * s2;
    p.tp = 3.14159265358979f * (1.f + q * c2);
    p.tpp = -19.7392088021787f * q * s2;
  }
  sincosf(th, &p.s, &p.c);
}

__device__ __forceinline__ void geodesic_accel_f(const Geom& G, const PointF& p, const float K[4], float dK[4]) {
  const float a = (float)G.a, a2 = a * a, m = (float)G.mass;
  const float r = p.r, s2 = p.s * p.s, S2 = 2.f * p.s * p.c, r2 = r * r;
  const float Sig = r2 + a2 * p.c * p.c;
  const float iS = 1.f / Sig, ir = 1.f / r, is2 = 1.f / s2, itp = 1.f / p.tp;
  const float f = 2.f * m * r * iS;
  const float fr = 2.f * m * (a2 * p.c * p.c - r2) * (iS * iS);
  const float ft = f * a2 * S2 * iS;
  const float ut = K[0], ur = r * K[1], uh = p.tp * K[2], up = K[3];
  const float P = ut + ur - a * s2 * up;
  const float hp = uh * up;
  const float W = (fr * ur + ft * uh) * P - f * a * S2 * hp;
  const float ra = r2 + a2;
  const float Rt = -W;
  const float Rr = r * (uh * uh + s2 * up * up) + 0.5f * fr * P * P + a * S2 * hp - W;
  const float Rh = 0.5f * S2 * (ra * up * up - a2 * uh * uh - 2.f * a * up * (ur + f * P)) + 0.5f * ft * P * P
                   - (2.f * r * ur - a2 * S2 * uh) * uh;
  const float Rp = a * S2 * uh * (ur + f * P) + a * s2 * W - (2.f * r * ur * s2 + ra * S2 * uh) * up;
  const float Del = ra - 2.f * m * r;
  dK[0] = f * Rr - (1.f + f) * Rt;
  dK[1] = (f * Rt + iS * (Del * Rr + a * Rp)) * ir - K[1] * K[1];
  dK[2] = (iS * Rh - p.tpp * K[2] * K[2]) * itp;
  dK[3] = iS * (a * Rr + is2 * Rp);
}

__device__ __forceinline__ void rk4_push_f(const Geom& G, float X[4], float K[4], float h) {
  float k1[4], k2[4], k3[4], k4[4], Xt[4], Kt[4];
  PointF p;
  Xt[0] = 0.f;
  point_full_f(G, X, p);
  geodesic_accel_f(G, p, K, k1);
#pragma unroll
  for (int m = 0; m < 4; ++m) Kt[m] = K[m] + 0.5f * h * k1[m];
#pragma unroll
  for (int m = 1; m < 4; ++m) Xt[m] = X[m] + 0.5f * h * K[m];
  float xs[4];
#pragma unroll
  for (int m = 1; m < 4; ++m) xs[m] = K[m] + 2.f * Kt[m];
  point_full_f(G, Xt, p);
  geodesic_accel_f(G, p, Kt, k2);
#pragma unroll
  for (int m = 1; m < 4; ++m) Xt[m] = X[m] + 0.5f * h * Kt[m];
#pragma unroll
  for (int m = 0; m < 4; ++m) Kt[m] = K[m] + 0.5f * h * k2[m];
  point_full_f(G, Xt, p);
  geodesic_accel_f(G, p, Kt, k3);
#pragma unroll
  for (int m = 1; m < 4; ++m) xs[m] += 2.f * Kt[m];
#pragma unroll
  for (int m = 1; m < 4; ++m) Xt[m] = X[m] + h * Kt[m];
#pragma unroll
  for (int m = 0; m < 4; ++m) Kt[m] = K[m] + h * k3[m];
  point_full_f(G, Xt, p);
  geodesic_accel_f(G, p, Kt, k4);
  const float h6 = h * (1.f / 6.f);
#pragma unroll
  for (int m = 1; m < 4; ++m) X[m] += h6 * (xs[m] + Kt[m]);
#pragma unroll
  for (int m = 0; m < 4; ++m) K[m] += h6 * (k1[m] + 2.f * k2[m] + 2.f * k3[m] + k4[m]);
}

__global__ void __launch_bounds__(IPOLE_GEO_THREADS, 6) k_geodesic_f32(const __grid_constant__ GeoArgs A) {
  const CamDev& C = A.cam;
  const int64_t count = A.count_dev ? (int64_t)*A.count_dev : A.count;
  const size_t slot_doubles = (size_t)(A.cap + 1) * REC_DOUBLES;
  float X[4] = {0.f, 0.f, 0.f, 0.f}, K[4] = {0.f, 0.f, 0.f, 0.f};
  double* rec = nullptr;
  int64_t li;
  int32_t q = 0;
  int n = 0, nt = 0;
  bool have = false;
  auto store = [&](double* r, float dl) {
    st_global_v4(r, (double)X[1], (double)X[2], (double)X[3], (double)K[0]);
    st_global_v4(r + 4, (double)K[1], (double)K[2], (double)K[3], (double)dl);
  };
  auto fetch = [&]() {
    li = (int64_t)atomicAdd(A.queue, 1ULL);
    have = li < count;
    if (!have) return;
    q = A.order ? A.order[A.base + li] : (int32_t)(A.base + li);
    int64_t pix;
    if (A.lattice_stride > 0) {
      const int ix = q % A.lattice_nx, iy = q / A.lattice_nx;
      pix = (int64_t)(iy * A.lattice_stride + A.lattice_stride / 2) * C.nx + (ix * A.lattice_stride + A.lattice_stride / 2);
    } else {
      pix = A.pixels ? A.pixels[(int64_t)q * A.list_stride] : (int64_t)q * A.list_stride;
    }
    double Xd[4], Kd[4];
    pixel_ray(C, pix, Xd, Kd);       // the camera ray itself is formed in FP64 (once per ray) and rounded
#pragma unroll
    for (int m = 0; m < 4; ++m) { X[m] = (float)Xd[m]; K[m] = (float)Kd[m]; }
    rec = A.path ? A.path + (size_t)li * slot_doubles : nullptr;
    n = 0; nt = 0;
  };
  const float ieps = (float)(1.0 / A.eps), lx_in = (float)C.lx_in, lx_esc = (float)C.lx_esc;
  fetch();
  while (have) {
    const float i13 = (fabsf(K[1]) + 1e-37f) + (fabsf(K[3]) + 1e-37f);
    const float i2 = (fabsf(K[2]) + 1e-37f) / fabsf(fminf(X[2], 1.f - X[2]));
    const float dl = 1.f / ((i13 + i2) * ieps);
    if (rec) store(rec + (size_t)n * REC_DOUBLES, dl);
    const float x1_before = X[1];
    const bool k2neg = K[2] < 0.f;
    rk4_push_f(C.G, X, K, -dl);
    ++n;
    if ((K[2] < 0.f) != k2neg) ++nt;
    int status = 0;
    if (X[1] <= lx_in) status = 1;
    else if (X[1] > lx_esc && X[1] > x1_before) status = 2;
    else if (n >= A.max_steps) status = 3;
    const bool overflow = (status == 0) && rec && (n >= A.cap);
    if (status != 0 || overflow) {
      if (overflow) {
        A.nsteps[q] = -1;
        if (A.long_list) { const int w = atomicAdd(A.long_count, 1); A.long_list[w] = q; }
      } else {
        if (rec) store(rec + (size_t)n * REC_DOUBLES, 0.f);
        A.nsteps[q] = n;
        if (A.nturn) A.nturn[q] = (nt > 127 ? 127 : nt) | (status == 3 ? 0x80 : 0);
      }
      fetch();
    }
  }
}

}  // namespace ipole

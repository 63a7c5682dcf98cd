// Kerr metric in modified Kerr-Schild (MKS) coordinates: closed-form g_{mu nu}, g^{mu nu}, the two non-zero
// coordinate derivatives d_1 g, d_2 g, and the connection *already contracted* with the wave vector.
//
// DESIGN.md R-2 (north_star stage (1): "null geodesic in the Kerr metric (modified Kerr-Schild coordinates)";
// PAPER.md:35).  X = (t, X1, X2, X3), r = exp(X1), theta = pi X2 + (1-h)/2 sin(2 pi X2), phi = X3.
// Kerr-Schild: Sigma = r^2 + a^2 cos^2, f = 2 m r / Sigma (m = 0 under flat_metric), Delta = r^2 - 2 m r + a^2.
// MKS components g_{mu nu} = J_mu J_nu g^KS_{mu nu}, J = (1, r, theta', 1).  Only 7 covariant and 6 contravariant
// components are non-zero, and only d/dX1, d/dX2 of them, so the 40 Christoffel symbols are never formed:
//   Gamma_{k mn} K^m K^n = K^1 (D1 K)_k + K^2 (D2 K)_k - 1/2 [k=1] K.D1.K - 1/2 [k=2] K.D2.K        (geodesic)
//   Gamma_{l mn} K^m     = 1/2 ( K^1 D1_{ln} + K^2 D2_{ln} + [n=1](D1 K)_l + [n=2](D2 K)_l
//                                - [l=1](D1 K)_n - [l=2](D2 K)_n )                                  (transport)
#pragma once
#include <cuda_runtime.h>
#include <math.h>
#include "fpmath.cuh"

namespace ipole {

struct Geom {
  double a;        // spin
  double hslope;   // h
  double mass;     // 1, or 0 under flat_metric
  int    h_is_one; // theta = pi X2 exactly
};

// sparse symmetric 4x4 with the Kerr-Schild pattern: 00 01 03 11 13 22 33
struct Sym7 {
  double c00, c01, c03, c11, c13, c22, c33;
  __device__ __forceinline__ void mul(const double v[4], double o[4]) const {
    o[0] = c00 * v[0] + c01 * v[1] + c03 * v[3];
    o[1] = c01 * v[0] + c11 * v[1] + c13 * v[3];
    o[2] = c22 * v[2];
    o[3] = c03 * v[0] + c13 * v[1] + c33 * v[3];
  }
};
// inverse metric pattern: 00 01 11 13 22 33 (g^{t phi} = 0 in Kerr-Schild)
struct Inv6 {
  double c00, c01, c11, c13, c22, c33;
  __device__ __forceinline__ void mul(const double v[4], double o[4]) const {
    o[0] = c00 * v[0] + c01 * v[1];
    o[1] = c01 * v[0] + c11 * v[1] + c13 * v[3];
    o[2] = c22 * v[2];
    o[3] = c13 * v[1] + c33 * v[3];
  }
};

struct Point {      // scalar functions of position shared by everything evaluated at X
  double r, th, tp, tpp, s, c, Sig, f, sqrtmg, iSig;
  double s2x, c2x;  // sin, cos of 2 pi X2 (only when hslope != 1)
};

// r, theta(X2) and its derivatives, sin/cos theta: one exp and one (two when hslope != 1) sincos
__device__ __forceinline__ void point_full(const Geom& G, const double X[4], Point& p) {
  p.r = ip_exp(X[1]);
  if (G.h_is_one) {
    p.th = M_PI * X[2]; p.tp = M_PI; p.tpp = 0.0;
    p.s2x = 0.0; p.c2x = 1.0;
  } else {
    ip_sincos(2.0 * M_PI * X[2], &p.s2x, &p.c2x);
    const double q = 1.0 - G.hslope;
    p.th = M_PI * X[2] + 0.5 * q * p.s2x;
    p.tp = M_PI * (1.0 + q * p.c2x);
    p.tpp = -2.0 * M_PI * M_PI * q * p.s2x;
  }
  ip_sincos(p.th, &p.s, &p.c);
}

// sin d and cos d - 1 for |d| <= 0.2 (Taylor to d^13 / d^12: truncation < 1e-19 relative)
__device__ __forceinline__ void sincosm1_small(double d, double& sd, double& cm1) {
  const double w = d * d;
  double ps = 1.6059043836821613e-10;              // 1/13!
  ps = fma(ps, w, -2.5052108385441720e-08);        // -1/11!
  ps = fma(ps, w, 2.7557319223985893e-06);         // 1/9!
  ps = fma(ps, w, -1.9841269841269841e-04);        // -1/7!
  ps = fma(ps, w, 8.3333333333333332e-03);         // 1/5!
  ps = fma(ps, w, -1.6666666666666666e-01);        // -1/3!
  sd = fma(d * w, ps, d);
  double pc = 2.0876756987868100e-09;              // 1/12!
  pc = fma(pc, w, -2.7557319223985888e-07);        // -1/10!
  pc = fma(pc, w, 2.4801587301587302e-05);         // 1/8!
  pc = fma(pc, w, -1.3888888888888889e-03);        // -1/6!
  pc = fma(pc, w, 4.1666666666666664e-02);         // 1/4!
  pc = fma(pc, w, -0.5);
  cm1 = w * pc;
}

// The same scalars at X0 + (0, d1, d2, .) from those at X0, for the small displacements of the RK4 stages
// (|d1| <= 0.06, |2 pi d2| <= 0.2: guaranteed by the step rule for eps <= 0.04, R-4):
//   r = r0 + r0 expm1(d1),   sin(t0 + dt) = s0 + (s0 (cos dt - 1) + c0 sin dt),   cos likewise,
// with short Taylor polynomials in place of one exp and one or two full sincos.  The increments are added to the
// base values, so the relative accuracy of sin(theta) near the axis is that of the base value.
__device__ __forceinline__ void point_shift(const Geom& G, const Point& b, double d1, double d2, Point& p) {
  double e = 2.7557319223985893e-06;               // expm1(d) = d + d^2/2 + ... + d^9/9!
  e = fma(e, d1, 2.4801587301587302e-05);
  e = fma(e, d1, 1.9841269841269841e-04);
  e = fma(e, d1, 1.3888888888888889e-03);
  e = fma(e, d1, 8.3333333333333332e-03);
  e = fma(e, d1, 4.1666666666666664e-02);
  e = fma(e, d1, 1.6666666666666666e-01);
  e = fma(e, d1, 0.5);
  e = fma(d1 * d1, e, d1);
  p.r = fma(b.r, e, b.r);
  double dth;
  if (G.h_is_one) {
    dth = M_PI * d2;
    p.tp = M_PI; p.tpp = 0.0; p.s2x = 0.0; p.c2x = 1.0;
  } else {
    double sa, cam1;
    sincosm1_small(2.0 * M_PI * d2, sa, cam1);
    const double ds2 = fma(b.s2x, cam1, b.c2x * sa), dc2 = fma(b.c2x, cam1, -b.s2x * sa);
    p.s2x = b.s2x + ds2; p.c2x = b.c2x + dc2;
    const double q = 1.0 - G.hslope;
    dth = fma(0.5 * q, ds2, M_PI * d2);
    p.tp = M_PI * (1.0 + q * p.c2x);
    p.tpp = -2.0 * M_PI * M_PI * q * p.s2x;
  }
  p.th = b.th + dth;
  double sd, cm1;
  sincosm1_small(dth, sd, cm1);
  p.s = b.s + fma(b.s, cm1, b.c * sd);
  p.c = b.c + fma(b.c, cm1, -b.s * sd);
}

// g_{mu nu} and g^{mu nu} from the scalars of a filled Point (no derivatives)
template <bool WANT_INV>
__device__ __forceinline__ void metric_assemble(const Geom& G, Point& p, Sym7& g, Inv6& gi) {
  const double a = G.a;
  const double r = p.r, s2 = p.s * p.s;
  p.Sig = r * r + a * a * p.c * p.c;
  const double tp2 = p.tp * p.tp;
  double iS = 0.0, ir = 0.0, iSst = 0.0;
  if (WANT_INV) {
    // one reciprocal of the product instead of four: 1/Sigma, 1/r, 1/sin^2, 1/theta'^2
    const double Sr = p.Sig * r, st = s2 * tp2;
    const double t = ip_rcp(Sr * st);
    iS = t * r * st; ir = t * p.Sig * st; iSst = t * r;   // iSst = 1/(Sigma sin^2 theta'^2)
    p.f = 2.0 * G.mass * r * iS;
    p.iSig = iS;
  } else {
    p.f = 2.0 * G.mass * r / p.Sig;
  }
  const double f = p.f, opf = 1.0 + f;
  g.c00 = -1.0 + f;
  g.c01 = f * r;
  g.c03 = -a * f * s2;
  g.c11 = opf * r * r;
  g.c13 = -a * s2 * opf * r;
  g.c22 = p.Sig * tp2;
  g.c33 = s2 * (p.Sig + a * a * s2 * opf);
  p.sqrtmg = r * p.tp * p.Sig * fabs(p.s);
  if (WANT_INV) {
    const double Del = r * r - 2.0 * G.mass * r + a * a;
    gi.c00 = -opf;
    gi.c01 = f * ir;
    gi.c11 = Del * iS * ir * ir;
    gi.c13 = a * iS * ir;
    gi.c22 = iSst * s2;
    gi.c33 = iSst * tp2;
  }
}

// g_{mu nu} and g^{mu nu} at X (no derivatives)
template <bool WANT_INV>
__device__ __forceinline__ void metric(const Geom& G, const double X[4], Point& p, Sym7& g, Inv6& gi) {
  point_full(G, X, p);
  metric_assemble<WANT_INV>(G, p, g, gi);
}

__device__ __forceinline__ void theta_map(const Geom& G, double x2, double& th, double& tp, double& tpp) {
  if (G.h_is_one) {
    th = M_PI * x2; tp = M_PI; tpp = 0.0;
  } else {
    double s2, c2;
    ip_sincos(2.0 * M_PI * x2, &s2, &c2);
    const double q = 1.0 - G.hslope;
    th = M_PI * x2 + 0.5 * q * s2;
    tp = M_PI * (1.0 + q * c2);
    tpp = -2.0 * M_PI * M_PI * q * s2;
  }
}

// metric, inverse and the derivative matrices D1 = d g / d X1, D2 = d g / d X2
__device__ __forceinline__ void metric_derivs_at(const Geom& G, Point& p, Sym7& g, Inv6& gi, Sym7& D1, Sym7& D2);
__device__ __forceinline__ void metric_derivs(const Geom& G, const double X[4], Point& p, Sym7& g, Inv6& gi,
                                              Sym7& D1, Sym7& D2) {
  point_full(G, X, p);
  metric_derivs_at(G, p, g, gi, D1, D2);
}
// the same from a Point whose scalars (r, theta', theta'', sin, cos) are already filled
__device__ __forceinline__ void metric_derivs_at(const Geom& G, Point& p, Sym7& g, Inv6& gi, Sym7& D1, Sym7& D2) {
  metric_assemble<true>(G, p, g, gi);
  const double a = G.a, r = p.r, s2 = p.s * p.s, f = p.f, opf = 1.0 + f;
  const double a2 = a * a;
  const double iS2 = p.iSig * p.iSig;
  const double fr1 = r * 2.0 * G.mass * (a2 * p.c * p.c - r * r) * iS2;  // r df/dr
  const double cs2 = 2.0 * p.s * p.c * p.tp;                             // theta' d(sin^2)/dtheta
  const double ft2 = 2.0 * G.mass * r * a2 * cs2 * iS2;                  // theta' df/dtheta
  const double St2 = -a2 * cs2;                                          // theta' dSigma/dtheta
  D1.c00 = fr1;
  D1.c01 = r * (f + fr1);
  D1.c03 = -a * s2 * fr1;
  D1.c11 = r * r * (2.0 * opf + fr1);
  D1.c13 = -a * s2 * r * (opf + fr1);
  D1.c22 = 2.0 * r * r * p.tp * p.tp;
  D1.c33 = s2 * (2.0 * r * r + a2 * s2 * fr1);
  const double e = cs2 * opf + s2 * ft2;  // theta' d/dtheta [ s^2 (1+f) ]
  D2.c00 = ft2;
  D2.c01 = r * ft2;
  D2.c03 = -a * (ft2 * s2 + f * cs2);
  D2.c11 = r * r * ft2;
  D2.c13 = -a * r * e;
  D2.c22 = 2.0 * p.tpp * p.tp * p.Sig + p.tp * p.tp * St2;
  D2.c33 = cs2 * (p.Sig + a2 * s2 * opf) + s2 * (St2 + a2 * e);
}

#ifndef IPOLE_GEO_KS
#define IPOLE_GEO_KS 1
#endif

// dK^l / dlambda = - Gamma^l_{mn} K^m K^n, written out for the Kerr-Schild form of the metric instead of through the
// derivative matrices: in (t, r, theta, phi),  g = eta~ + f l l,  l_mu = (1, 1, 0, -a sin^2),  f = 2 m r / Sigma,
//   eta~ = -dt^2 + dr^2 + Sigma dth^2 + (r^2+a^2) sin^2 dph^2 - 2 a sin^2 dr dph .
// With u = dx/dlambda and P = l.u the Euler-Lagrange equations  d/dlambda (g_{kn} u^n) = 1/2 d_k g_{mn} u^m u^n  give
//   g_{kn} du^n/dlambda = R_k = 1/2 d_k g(u,u) - (d eta~_{kn}/dlambda) u^n - W l_k - f P dl_k/dlambda ,
//   W = f (dl/dlambda . u) + (df/dlambda) P ,   dl_phi/dlambda = -a sin(2 theta) dtheta/dlambda  (the only one),
// and the closed-form inverse raises R.  The MKS components follow from r = e^{X1}, theta = theta(X2):
//   dK1 = r''/r - K1^2,   dK2 = (theta'' - theta_XX K2^2) / theta_X .
// The same equations as the contracted Christoffel symbols of geodesic_accel_gamma (identical up to rounding; the
// traced paths are compared with the oracle's to 1e-11 in tests/test_gpu_stages.py), at ~100 instead of ~160 FP64
// instructions per evaluation: k_geodesic is bound by the FP64 pipe, and this is four evaluations per step.
__device__ __forceinline__ void geodesic_accel_ks(const Geom& G, Point& p, const double K[4], double dK[4]) {
  const double a = G.a, a2 = a * a, m = G.mass;
  const double r = p.r, s2 = p.s * p.s, S2 = 2.0 * p.s * p.c, r2 = r * r;
  const double Sig = r2 + a2 * p.c * p.c;
  // one reciprocal for 1/Sigma, 1/r, 1/sin^2, 1/theta_X
  const double Sr = Sig * r, st = s2 * p.tp;
  const double t = ip_rcp(Sr * st);
  const double iS = t * r * st, ir = t * Sig * st, is2 = t * Sr * p.tp, itp = t * Sr * s2;
  const double f = 2.0 * m * r * iS;
  const double fr = 2.0 * m * (a2 * p.c * p.c - r2) * (iS * iS);   // df/dr
  const double ft = f * a2 * S2 * iS;                               // df/dtheta
  const double ut = K[0], ur = r * K[1], uh = p.tp * K[2], up = K[3];
  const double P = ut + ur - a * s2 * up;
  const double hp = uh * up;                       // theta' phi'
  const double W = (fr * ur + ft * uh) * P - f * a * S2 * hp;
  const double ra = r2 + a2;
  const double Rt = -W;
  const double Rr = r * (uh * uh + s2 * up * up) + 0.5 * fr * P * P + a * S2 * hp - W;
  const double Rh = 0.5 * S2 * (ra * up * up - a2 * uh * uh - 2.0 * a * up * (ur + f * P)) + 0.5 * ft * P * P
                    - (2.0 * r * ur - a2 * S2 * uh) * uh;
  const double Rp = a * S2 * uh * (ur + f * P) + a * s2 * W - (2.0 * r * ur * s2 + ra * S2 * uh) * up;
  const double Del = ra - 2.0 * m * r;
  const double tdd = f * Rr - (1.0 + f) * Rt;
  const double rdd = f * Rt + iS * (Del * Rr + a * Rp);
  const double hdd = iS * Rh;
  const double pdd = iS * (a * Rr + is2 * Rp);
  dK[0] = tdd;
  dK[1] = rdd * ir - K[1] * K[1];
  dK[2] = (hdd - p.tpp * K[2] * K[2]) * itp;
  dK[3] = pdd;
}

__device__ __forceinline__ void geodesic_accel_gamma(const Geom& G, Point& p, const double K[4], double dK[4]);
__device__ __forceinline__ void geodesic_accel_at(const Geom& G, Point& p, const double K[4], double dK[4]) {
#if IPOLE_GEO_KS
  geodesic_accel_ks(G, p, K, dK);
#else
  geodesic_accel_gamma(G, p, K, dK);
#endif
}

// the same through the derivative matrices D1, D2 (header of this file)
__device__ __forceinline__ void geodesic_accel_gamma(const Geom& G, Point& p, const double K[4], double dK[4]) {
  Sym7 g, D1, D2; Inv6 gi;
  metric_derivs_at(G, p, g, gi, D1, D2);
  double v1[4], v2[4], F[4];
  D1.mul(K, v1);
  D2.mul(K, v2);
  const double s1 = K[0] * v1[0] + K[1] * v1[1] + K[2] * v1[2] + K[3] * v1[3];
  const double s2 = K[0] * v2[0] + K[1] * v2[1] + K[2] * v2[2] + K[3] * v2[3];
  F[0] = K[1] * v1[0] + K[2] * v2[0];
  F[1] = K[1] * v1[1] + K[2] * v2[1] - 0.5 * s1;
  F[2] = K[1] * v1[2] + K[2] * v2[2] - 0.5 * s2;
  F[3] = K[1] * v1[3] + K[2] * v2[3];
  gi.mul(F, dK);
  dK[0] = -dK[0]; dK[1] = -dK[1]; dK[2] = -dK[2]; dK[3] = -dK[3];
}
__device__ __forceinline__ void geodesic_accel(const Geom& G, const double X[4], const double K[4], double dK[4]) {
  Point p;
  point_full(G, X, p);
  geodesic_accel_at(G, p, K, dK);
}

// A^a_n = Gamma^a_{mn} K^m as a dense 4x4 (row a, column n); also returns the metric at X for the caller
__device__ __forceinline__ void transport_generator_from(const Sym7& D1, const Sym7& D2, const Inv6& gi, const double K[4],
                                                         double A[4][4]);
__device__ __forceinline__ void transport_generator(const Geom& G, const double X[4], const double K[4], Point& p,
                                                    Sym7& g, Inv6& gi, double A[4][4]) {
  Sym7 D1, D2;
  metric_derivs(G, X, p, g, gi, D1, D2);
  transport_generator_from(D1, D2, gi, K, A);
}
// the same from a Point whose scalars are already filled (metric and derivatives are rebuilt from it)
__device__ __forceinline__ void transport_generator_at(const Geom& G, const double K[4], Point& p, double A[4][4]) {
  Sym7 g, D1, D2; Inv6 gi;
  metric_derivs_at(G, p, g, gi, D1, D2);
  transport_generator_from(D1, D2, gi, K, A);
}
__device__ __forceinline__ void transport_generator_from(const Sym7& D1, const Sym7& D2, const Inv6& gi, const double K[4],
                                                         double A[4][4]) {
  double v1[4], v2[4];
  D1.mul(K, v1);
  D2.mul(K, v2);
  const double k1 = K[1], k2 = K[2];
  double L[4][4];  // L_{l n} = Gamma_{l m n} K^m
  L[0][0] = 0.5 * (k1 * D1.c00 + k2 * D2.c00);
  L[0][1] = 0.5 * (k1 * D1.c01 + k2 * D2.c01 + v1[0]);
  L[0][2] = 0.5 * (v2[0]);
  L[0][3] = 0.5 * (k1 * D1.c03 + k2 * D2.c03);
  L[1][0] = 0.5 * (k1 * D1.c01 + k2 * D2.c01 - v1[0]);
  L[1][1] = 0.5 * (k1 * D1.c11 + k2 * D2.c11);                // + v1[1] - v1[1]
  L[1][2] = 0.5 * (v2[1] - v1[2]);
  L[1][3] = 0.5 * (k1 * D1.c13 + k2 * D2.c13 - v1[3]);
  L[2][0] = 0.5 * (-v2[0]);
  L[2][1] = 0.5 * (v1[2] - v2[1]);
  L[2][2] = 0.5 * (k1 * D1.c22 + k2 * D2.c22);                // + v2[2] - v2[2]
  L[2][3] = 0.5 * (-v2[3]);
  L[3][0] = 0.5 * (k1 * D1.c03 + k2 * D2.c03);
  L[3][1] = 0.5 * (k1 * D1.c13 + k2 * D2.c13 + v1[3]);
  L[3][2] = 0.5 * (v2[3]);
  L[3][3] = 0.5 * (k1 * D1.c33 + k2 * D2.c33);
#pragma unroll
  for (int n = 0; n < 4; ++n) {
    A[0][n] = gi.c00 * L[0][n] + gi.c01 * L[1][n];
    A[1][n] = gi.c01 * L[0][n] + gi.c11 * L[1][n] + gi.c13 * L[3][n];
    A[2][n] = gi.c22 * L[2][n];
    A[3][n] = gi.c13 * L[1][n] + gi.c33 * L[3][n];
  }
}

// f <- (1 - h A + h^2 A^2 / 2) f
__device__ __forceinline__ void transport_apply(const double A[4][4], double h, double f[4]) {
  double w[4], w2[4];
#pragma unroll
  for (int a = 0; a < 4; ++a) w[a] = A[a][0] * f[0] + A[a][1] * f[1] + A[a][2] * f[2] + A[a][3] * f[3];
#pragma unroll
  for (int a = 0; a < 4; ++a) w2[a] = A[a][0] * w[0] + A[a][1] * w[1] + A[a][2] * w[2] + A[a][3] * w[3];
  const double hh = 0.5 * h * h;
#pragma unroll
  for (int a = 0; a < 4; ++a) f[a] = f[a] - h * w[a] + hh * w2[a];
}

// c <- (1 - h A + h^2 A^2 / 2)^T c : the pull-back of a covector through the same half step
__device__ __forceinline__ void transport_apply_transposed(const double A[4][4], double h, double c[4]) {
  double w[4], w2[4];
#pragma unroll
  for (int n = 0; n < 4; ++n) w[n] = A[0][n] * c[0] + A[1][n] * c[1] + A[2][n] * c[2] + A[3][n] * c[3];
#pragma unroll
  for (int n = 0; n < 4; ++n) w2[n] = A[0][n] * w[0] + A[1][n] * w[1] + A[2][n] * w[2] + A[3][n] * w[3];
  const double hh = 0.5 * h * h;
#pragma unroll
  for (int n = 0; n < 4; ++n) c[n] = c[n] - h * w[n] + hh * w2[n];
}

__device__ __forceinline__ double dot4(const double u[4], const double v[4]) {
  return u[0] * v[0] + u[1] * v[1] + u[2] * v[2] + u[3] * v[3];
}

__device__ __forceinline__ double horizon_radius(double a) { return 1.0 + sqrt(1.0 - a * a); }

// Bardeen, Press & Teukolsky (1972) prograde ISCO
__device__ __host__ inline double isco_radius(double a) {
  const double z1 = 1.0 + cbrt(1.0 - a * a) * (cbrt(1.0 + a) + cbrt(1.0 - a));
  const double z2 = sqrt(3.0 * a * a + z1 * z1);
  return 3.0 + z2 - sqrt((3.0 - z1) * (3.0 + z1 + 2.0 * z2));
}

}  // namespace ipole

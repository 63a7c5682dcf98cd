// Constant-coefficient solution of the polarized transfer equation over one step,
//   dS/ds = J - Kmat S,  S(s) = O(s) S0 + P(s) J,  O = exp(-Kmat s),  P = int_0^s O,
// applied to vectors (the 4x4 matrices are never formed).  DESIGN.md R-8 (north_star stage (3): "the analytic
// per-step solution of the 4x4 transfer equation"); closed form of Landi Degl'Innocenti & Landi Degl'Innocenti
// (1985):  O = e^{-aI s} { (ch+c)/2 1 - sn M2 - sh M3 + (ch-c)/2 M4 } with, for 3-vectors a = (aQ,aU,aV),
// r = (rQ,rU,rV) and any Stokes vector (S0, s):
//   M2 (S0,s) = ( v2.s , v2 S0 + s x w2 ) / Th,   v2 = L2 a - sg L1 r,  w2 = sg L1 a + L2 r
//   M3 (S0,s) = ( v3.s , v3 S0 + s x w3 ) / Th,   v3 = L1 a + sg L2 r,  w3 = -sg L2 a + L1 r
//   M4 (S0,s) = 2 ( hh S0 + cr.s , -cr S0 + a (a.s) + r (r.s) - hh s ) / Th,  cr = r x a, hh = (|a|^2+|r|^2)/2
// (L1, L2, sg, Th as in the oracle's header; all vectors scaled by m = max |component| first).
#pragma once
#include "geom.cuh"

namespace ipole {


__device__ __forceinline__ void cross3(const double u[3], const double v[3], double o[3]) {
  o[0] = u[1] * v[2] - u[2] * v[1];
  o[1] = u[2] * v[0] - u[0] * v[2];
  o[2] = u[0] * v[1] - u[1] * v[0];
}
__device__ __forceinline__ double dot3(const double u[3], const double v[3]) { return u[0] * v[0] + u[1] * v[1] + u[2] * v[2]; }

// a/b: the fast quotient where b is safely normal, the IEEE division otherwise (coefficients near the subnormal range)
__device__ __forceinline__ double guarded_div(double a, double b) {
  const double ab = fabs(b);
  if (IP_LIKELY(ab > 1e-290 && ab < 1e290)) return ip_div(a, b);
  return a / b;
}

// S <- O(s) S + P(s) J ; al = (aI,aQ,aU,aV), rh = (rQ,rU,rV)
//
// Transcendentals per call: three expm1 and one sincos.  With tp = expm1(-(aI-L1)s), tm = expm1(-(aI+L1)s),
// t0 = expm1(-aI s):  e^{-aI s} cosh(L1 s) = 1 + (tp+tm)/2,  e^{-aI s} sinh(L1 s) = (tp-tm)/2,
// E(aI -+ L1) = -t{p,m}/(aI -+ L1),  1 - cos x = sin^2 x / (1 + cos x) for cos x > 0.
__device__ __forceinline__ void stokes_step(const double al[4], const double rh[3], double s, const double J[4], double S[4]) {
  const double aI = al[0];
  const double m = fmax(fmax(fabs(al[1]), fmax(fabs(al[2]), fabs(al[3]))), fmax(fabs(rh[0]), fmax(fabs(rh[1]), fabs(rh[2]))));
  const double t0 = ip_expm1(-aI * s);
  const double ex = 1.0 + t0;
  if (IP_UNLIKELY(m == 0.0)) {
    const double E = (aI == 0.0) ? s : -guarded_div(t0, aI);
#pragma unroll
    for (int i = 0; i < 4; ++i) S[i] = ex * S[i] + E * J[i];
    return;
  }
  double a[3], r[3];
  if (IP_LIKELY(m > 1e-290)) {
    const double im = ip_rcp(m);
    a[0] = al[1] * im; a[1] = al[2] * im; a[2] = al[3] * im;
    r[0] = rh[0] * im; r[1] = rh[1] * im; r[2] = rh[2] * im;
  } else {  // 1/m would overflow (coefficients in the subnormal range, e.g. far wings of a Gaussian slab)
    a[0] = al[1] / m; a[1] = al[2] / m; a[2] = al[3] / m;
    r[0] = rh[0] / m; r[1] = rh[1] / m; r[2] = rh[2] / m;
  }
  const double a2 = dot3(a, a), r2 = dot3(r, r), ar = dot3(a, r);
  const double sg = (ar >= 0.0) ? 1.0 : -1.0;
  const double d = 0.5 * (a2 - r2);
  const double q = ip_sqrt(d * d + ar * ar);          // >= max scaled component^2 / 2 > 0
  // the larger of l1, l2 from the root (>= 1/sqrt 2 after scaling), the other from l1 l2 = |a.r|
  const double big2 = q + fabs(d);
  const double ibig = ip_rsqrt(big2);
  const double big = big2 * ibig, small = fabs(ar) * ibig;
  const double l1 = (d >= 0.0) ? big : small, l2 = (d >= 0.0) ? small : big;
  const double iTh = 0.5 * ip_rcp(q);                     // Theta = l1^2 + l2^2 = 2 q
  const double L1 = m * l1, L2 = m * l2;
  const double hh = 0.5 * (a2 + r2);
  const double sl1 = sg * l1, sl2 = sg * l2;
  double v2[3], w2[3], v3[3], w3[3], cr[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    v2[i] = l2 * a[i] - sl1 * r[i];
    w2[i] = sl1 * a[i] + l2 * r[i];
    v3[i] = l1 * a[i] + sl2 * r[i];
    w3[i] = l1 * r[i] - sl2 * a[i];
  }
  cross3(r, a, cr);

  double sn, c;
  ip_sincos_any(L2 * s, &sn, &c);
  const double bp = aI - L1, bm = aI + L1;
  const double tp = ip_expm1(-bp * s), tm = ip_expm1(-bm * s);
  const double exch = 1.0 + 0.5 * (tp + tm), exsh = 0.5 * (tp - tm);
  const double Ep = (bp == 0.0) ? s : -guarded_div(tp, bp), Em = (bm == 0.0) ? s : -guarded_div(tm, bm);
  const double Ic1 = 0.5 * (Ep + Em), Is1 = 0.5 * (Ep - Em);
  double Ic2, Is2;
  const double den = aI * aI + L2 * L2;
  if (IP_UNLIKELY(den == 0.0)) { Ic2 = s; Is2 = 0.0; }
  else {
    const double omc = (c > 0.0) ? sn * sn * ip_rcp(1.0 + c) : 1.0 - c;   // 1 - cos(L2 s)
    const double re = omc - t0 * c;                                  // Re(1 - e^{-aI s} e^{i L2 s})
    const double im2 = -ex * sn;
    const double nc = re * aI - im2 * L2, ns = re * L2 + im2 * aI;
    if (IP_LIKELY(den > 1e-280)) { const double iden = ip_rcp(den); Ic2 = nc * iden; Is2 = ns * iden; }
    else { Ic2 = nc / den; Is2 = ns / den; }   // 1/den would overflow (coefficients near the subnormal range)
  }
  // weights of (1, M2, M3, M4) for O and for P
  const double exc = ex * c;
  const double o1 = 0.5 * (exch + exc), o2 = -ex * sn, o3 = -exsh, o4 = 0.5 * (exch - exc);
  const double p1 = 0.5 * (Ic1 + Ic2), p2 = -Is2, p3 = -Is1, p4 = 0.5 * (Ic1 - Ic2);

  double out[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
  for (int pass = 0; pass < 2; ++pass) {
    const double* V = pass ? J : S;
    const double c1 = pass ? p1 : o1, c2 = (pass ? p2 : o2) * iTh, c3 = (pass ? p3 : o3) * iTh,
                 c4 = (pass ? p4 : o4) * 2.0 * iTh;
    const double V0 = V[0];
    const double sv[3] = {V[1], V[2], V[3]};
    double x2[3], x3[3];
    cross3(sv, w2, x2);
    cross3(sv, w3, x3);
    const double as = dot3(a, sv), rs = dot3(r, sv);
    out[0] += c1 * V0 + c2 * dot3(v2, sv) + c3 * dot3(v3, sv) + c4 * (hh * V0 + dot3(cr, sv));
#pragma unroll
    for (int i = 0; i < 3; ++i)
      out[1 + i] += c1 * sv[i] + c2 * (v2[i] * V0 + x2[i]) + c3 * (v3[i] * V0 + x3[i])
                    + c4 * (-cr[i] * V0 + a[i] * as + r[i] * rs - hh * sv[i]);
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) S[i] = out[i];
}

// The same step for aU = rU = jU = 0, which is what the synchrotron coefficients are in the tetrad whose e_(2) lies
// along the projected field (R-6/R-7): a = (aQ, 0, aV), r = (rQ, 0, rV), r x a = (0, rV aQ - rQ aV, 0).
// The operator applied to (V0, x, y, z) = (I, Q, U, V) collapses to ten numbers per weight set (c1..c4):
//   out0 = P0 V0 + Ax x + G y + Az z          P0,1 = c1 +- c4 hh,  A = c2 v2 + c3 v3,  B = c2 w2 + c3 w3,
//   outx = Ax V0 + (P1 + Dxx) x + B2 y + Dxz z          G = c4 (r x a)_U,  D = c4 (a a^T + r r^T)
//   outy = -G V0 - B2 x + P1 y + B0 z
//   outz = Az V0 + Dxz x - B0 y + (P1 + Dzz) z
// Thin step: || Kmat s ||_inf <= nb < 2^-7.  S(s) solves S' = J - Kmat S with constant coefficients, so
//   S(s) = S0 + sum_{n>=1} w_n,   w_1 = s (J - Kmat S0),   w_{n+1} = -(s/(n+1)) Kmat w_n,
// one chain of sparse 4x4 products for O S0 and P J together, no transcendentals and no divisions.  At most seven
// terms: the first dropped one is below nb^7/8! < 5e-20 of w_1.  This is the same matrix exponential the closed form
// evaluates (R-8).  Every step of the analytic ADAF workloads is thin (per-step optical and Faraday
// depths <= 1e-3).  Returns false (S untouched) when the step is not thin: the caller uses the closed form.
__device__ __forceinline__ bool stokes_step_qv_series(double aI, double aQ, double aV, double rQ, double rV, double s,
                                                      double jI, double jQ, double jV, double S[4]) {
  const double nb = fabs(s) * (fabs(aI) + fabs(aQ) + fabs(aV) + fabs(rQ) + fabs(rV));
  if (IP_UNLIKELY(!(nb < 0.0078125))) return false;
  // (every rounding spelt out, as in stokes_congruence: the same bits in every kernel that calls this)
  double w0 = __dmul_rn(s, __dadd_rn(jI, -fma(aV, S[3], fma(aQ, S[1], __dmul_rn(aI, S[0])))));
  double w1 = __dmul_rn(s, __dadd_rn(jQ, -fma(rV, S[2], fma(aI, S[1], __dmul_rn(aQ, S[0])))));
  double w2 = __dmul_rn(s, fma(-rQ, S[3], fma(-aI, S[2], __dmul_rn(rV, S[1]))));
  double w3 = __dmul_rn(s, __dadd_rn(jV, -fma(aI, S[3], fma(-rQ, S[2], __dmul_rn(aV, S[0])))));
  double o0 = w0, o1 = w1, o2 = w2, o3 = w3;
  // The chain is cut where the first dropped term is below 2e-17 of w_1: three terms for nb < 2^-17, five for
  // nb < 2^-10, seven otherwise.  Most steps of the ADAF workloads are in the lowest tier, and a warp whose lanes
  // all are skips the rest of the chain.
  auto term = [&](int n) {
    const double c = __dmul_rn(-s, 1.0 / (double)n);
    const double t0 = fma(aV, w3, fma(aQ, w1, __dmul_rn(aI, w0)));
    const double t1 = fma(rV, w2, fma(aI, w1, __dmul_rn(aQ, w0)));
    const double t2 = fma(rQ, w3, fma(-rV, w1, __dmul_rn(aI, w2)));
    const double t3 = fma(aI, w3, fma(-rQ, w2, __dmul_rn(aV, w0)));
    w0 = __dmul_rn(c, t0); w1 = __dmul_rn(c, t1); w2 = __dmul_rn(c, t2); w3 = __dmul_rn(c, t3);
    o0 = __dadd_rn(o0, w0); o1 = __dadd_rn(o1, w1); o2 = __dadd_rn(o2, w2); o3 = __dadd_rn(o3, w3);
  };
  term(2); term(3);
  if (nb >= 7.62939453125e-06) {          // 2^-17: (2^-17)^3 / 4! = 1.8e-17
    term(4); term(5);
    if (nb >= 9.765625e-4) { term(6); term(7); }   // 2^-10: (2^-10)^5 / 6! = 1.2e-18
  }
  S[0] = __dadd_rn(S[0], o0); S[1] = __dadd_rn(S[1], o1); S[2] = __dadd_rn(S[2], o2); S[3] = __dadd_rn(S[3], o3);
  return true;
}

// THIN_SERIES: try the series first.  The grid model keeps the closed form alone: its plasma steps are 1 in 8 and
// reach depths of order one, and the extra code cost more than it saved there (profiles/r1_notes.md).
template <bool THIN_SERIES>
__device__ __forceinline__ void stokes_step_qv(double aI, double aQ, double aV, double rQ, double rV, double s,
                                               double jI, double jQ, double jV, double S[4]) {
  if (THIN_SERIES) {
    if (stokes_step_qv_series(aI, aQ, aV, rQ, rV, s, jI, jQ, jV, S)) return;
  }
  const double m = fmax(fmax(fabs(aQ), fabs(aV)), fmax(fabs(rQ), fabs(rV)));
  const double t0 = ip_expm1(-aI * s);
  const double ex = 1.0 + t0;
  if (IP_UNLIKELY(m == 0.0)) {
    const double E = (aI == 0.0) ? s : -guarded_div(t0, aI);
    S[0] = ex * S[0] + E * jI; S[1] = ex * S[1] + E * jQ; S[2] = ex * S[2]; S[3] = ex * S[3] + E * jV;
    return;
  }
  double a0, a2, r0, r2;
  if (IP_LIKELY(m > 1e-290)) {
    const double im = ip_rcp(m);
    a0 = aQ * im; a2 = aV * im; r0 = rQ * im; r2 = rV * im;
  } else {
    a0 = aQ / m; a2 = aV / m; r0 = rQ / m; r2 = rV / m;
  }
  const double qa = a0 * a0 + r0 * r0, qz = a2 * a2 + r2 * r2, qxz = a0 * a2 + r0 * r2;
  const double asq = a0 * a0 + a2 * a2, rsq = r0 * r0 + r2 * r2, ar = a0 * r0 + a2 * r2;
  const double sg = (ar >= 0.0) ? 1.0 : -1.0;
  const double d = 0.5 * (asq - rsq);
  const double q = ip_sqrt(d * d + ar * ar);
  const double big2 = q + fabs(d);
  const double ibig = ip_rsqrt(big2);
  const double big = big2 * ibig, small = fabs(ar) * ibig;
  const double l1 = (d >= 0.0) ? big : small, l2 = (d >= 0.0) ? small : big;
  const double iTh = 0.5 * ip_rcp(q);
  const double L1 = m * l1, L2 = m * l2;
  const double hh = 0.5 * (asq + rsq);
  const double sl1 = sg * l1, sl2 = sg * l2;
  const double v2x = l2 * a0 - sl1 * r0, v2z = l2 * a2 - sl1 * r2;
  const double w2x = sl1 * a0 + l2 * r0, w2z = sl1 * a2 + l2 * r2;
  const double v3x = l1 * a0 + sl2 * r0, v3z = l1 * a2 + sl2 * r2;
  const double w3x = l1 * r0 - sl2 * a0, w3z = l1 * r2 - sl2 * a2;
  const double cru = r2 * a0 - r0 * a2;

  double sn, c;
  ip_sincos_any(L2 * s, &sn, &c);
  const double bp = aI - L1, bm = aI + L1;
  const double tp = ip_expm1(-bp * s), tm = ip_expm1(-bm * s);
  const double exch = 1.0 + 0.5 * (tp + tm), exsh = 0.5 * (tp - tm);
  const double Ep = (bp == 0.0) ? s : -guarded_div(tp, bp), Em = (bm == 0.0) ? s : -guarded_div(tm, bm);
  const double Ic1 = 0.5 * (Ep + Em), Is1 = 0.5 * (Ep - Em);
  double Ic2, Is2;
  const double den = aI * aI + L2 * L2;
  if (IP_UNLIKELY(den == 0.0)) { Ic2 = s; Is2 = 0.0; }
  else {
    const double omc = (c > 0.0) ? sn * sn * ip_rcp(1.0 + c) : 1.0 - c;
    const double re = omc - t0 * c;
    const double im2 = -ex * sn;
    const double nc = re * aI - im2 * L2, ns = re * L2 + im2 * aI;
    if (IP_LIKELY(den > 1e-280)) { const double iden = ip_rcp(den); Ic2 = nc * iden; Is2 = ns * iden; }
    else { Ic2 = nc / den; Is2 = ns / den; }
  }
  const double exc = ex * c;
  const double i2Th = 2.0 * iTh;
  // O acting on S
  double o0, ox, oy, oz;
  {
    const double c1 = 0.5 * (exch + exc), c2 = -ex * sn * iTh, c3 = -exsh * iTh, c4 = 0.5 * (exch - exc) * i2Th;
    const double P0 = fma(c4, hh, c1), P1 = fma(-c4, hh, c1);
    const double Ax = c2 * v2x + c3 * v3x, Az = c2 * v2z + c3 * v3z;
    const double B0 = c2 * w2x + c3 * w3x, B2 = c2 * w2z + c3 * w3z;
    const double G = c4 * cru, Dxx = c4 * qa, Dzz = c4 * qz, Dxz = c4 * qxz;
    const double V0 = S[0], x = S[1], y = S[2], z = S[3];
    o0 = P0 * V0 + Ax * x + G * y + Az * z;
    ox = Ax * V0 + (P1 + Dxx) * x + B2 * y + Dxz * z;
    oy = -G * V0 - B2 * x + P1 * y + B0 * z;
    oz = Az * V0 + Dxz * x - B0 * y + (P1 + Dzz) * z;
  }
  // P acting on J = (jI, jQ, 0, jV)
  {
    const double c1 = 0.5 * (Ic1 + Ic2), c2 = -Is2 * iTh, c3 = -Is1 * iTh, c4 = 0.5 * (Ic1 - Ic2) * i2Th;
    const double P0 = fma(c4, hh, c1), P1 = fma(-c4, hh, c1);
    const double Ax = c2 * v2x + c3 * v3x, Az = c2 * v2z + c3 * v3z;
    const double B0 = c2 * w2x + c3 * w3x, B2 = c2 * w2z + c3 * w3z;
    const double G = c4 * cru, Dxx = c4 * qa, Dzz = c4 * qz, Dxz = c4 * qxz;
    o0 += P0 * jI + Ax * jQ + Az * jV;
    ox += Ax * jI + (P1 + Dxx) * jQ + Dxz * jV;
    oy += -G * jI - B2 * jQ + B0 * jV;
    oz += Az * jI + Dxz * jQ + (P1 + Dzz) * jV;
  }
  S[0] = o0; S[1] = ox; S[2] = oy; S[3] = oz;
}

}  // namespace ipole

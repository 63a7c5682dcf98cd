// ORACLE (test infrastructure).  Constant-coefficient solution of the polarized transfer equation
//   dS/ds = J - Kmat S,   S = (I,Q,U,V)^T
//   Kmat = [[aI, aQ, aU, aV], [aQ, aI, rV, -rU], [aU, -rV, aI, rQ], [aV, rU, -rQ, aI]]
// over a path s:  S(s) = O(s) S(0) + P(s) J,  O(s) = exp(-Kmat s),  P(s) = int_0^s O(s') ds'.
//
// BASELINE.json north_star stage (3): "the analytic per-step solution of the 4x4 transfer equation".
// The paper does not print it; reading DESIGN.md R-8 -- the closed form of the
// evolution operator of Landi Degl'Innocenti & Landi Degl'Innocenti (1985):
//   O(s) = e^{-aI s} { 1/2 [cosh(L1 s) + cos(L2 s)] 1 - sin(L2 s) M2 - sinh(L1 s) M3
//                      + 1/2 [cosh(L1 s) - cos(L2 s)] M4 }
//   d = (|a|^2 - |r|^2)/2, q = sqrt(d^2 + (a.r)^2), L1 = sqrt(q + d), L2 = sqrt(q - d),
//   sigma = sign(a.r) (+1 at 0), Theta = L1^2 + L2^2 = 2q,  a = (aQ,aU,aV), r = (rQ,rU,rV)
// and P(s) from the same four scalar integrals.  Pinned against a 50-digit matrix exponential in
// tests/test_oracle_transfer.py (pin T2).
#pragma once
#include <cmath>

namespace iref {

// E(b) = int_0^s exp(-b x) dx
inline double exp_integral(double b, double s) { return (b == 0.0) ? s : -std::expm1(-b * s) / b; }

inline void stokes_operator(const double al[4], const double rh[3], double s, double O[4][4], double P[4][4]) {
  const double aI = al[0];
  const double m = std::fmax(std::fmax(std::fabs(al[1]), std::fmax(std::fabs(al[2]), std::fabs(al[3]))),
                             std::fmax(std::fabs(rh[0]), std::fmax(std::fabs(rh[1]), std::fabs(rh[2]))));
  for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) { O[i][j] = 0.0; P[i][j] = 0.0; }
  if (m == 0.0) {
    const double ex = std::exp(-aI * s), E = exp_integral(aI, s);
    for (int i = 0; i < 4; ++i) { O[i][i] = ex; P[i][i] = E; }
    return;
  }
  // scaled vectors (robust for coefficient magnitudes down to 1e-90 and below)
  const double a[3] = {al[1] / m, al[2] / m, al[3] / m};
  const double r[3] = {rh[0] / m, rh[1] / m, rh[2] / m};
  const double a2 = a[0] * a[0] + a[1] * a[1] + a[2] * a[2];
  const double r2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
  const double ar = a[0] * r[0] + a[1] * r[1] + a[2] * r[2];
  const double sg = (ar >= 0.0) ? 1.0 : -1.0;
  const double d = 0.5 * (a2 - r2);
  const double q = std::sqrt(d * d + ar * ar);
  double l1, l2;  // scaled Lambda_1, Lambda_2; the larger from the root, the other from l1 l2 = |a.r|
  if (d >= 0.0) { l1 = std::sqrt(q + d); l2 = (l1 > 0.0) ? std::fabs(ar) / l1 : 0.0; }
  else          { l2 = std::sqrt(q - d); l1 = (l2 > 0.0) ? std::fabs(ar) / l2 : 0.0; }
  const double Th = l1 * l1 + l2 * l2;
  const double L1 = m * l1, L2 = m * l2;

  double M2[4][4] = {{0}}, M3[4][4] = {{0}}, M4[4][4] = {{0}};
  for (int i = 0; i < 3; ++i) {
    const double v2 = (l2 * a[i] - sg * l1 * r[i]) / Th;
    const double v3 = (l1 * a[i] + sg * l2 * r[i]) / Th;
    M2[0][i + 1] = v2; M2[i + 1][0] = v2;
    M3[0][i + 1] = v3; M3[i + 1][0] = v3;
  }
  // antisymmetric blocks, index 1=Q,2=U,3=V
  const double w2_QU = (sg * l1 * a[2] + l2 * r[2]) / Th, w2_QV = (-sg * l1 * a[1] - l2 * r[1]) / Th,
               w2_UV = (sg * l1 * a[0] + l2 * r[0]) / Th;
  M2[1][2] = w2_QU; M2[2][1] = -w2_QU; M2[1][3] = w2_QV; M2[3][1] = -w2_QV; M2[2][3] = w2_UV; M2[3][2] = -w2_UV;
  const double w3_QU = (-sg * l2 * a[2] + l1 * r[2]) / Th, w3_QV = (sg * l2 * a[1] - l1 * r[1]) / Th,
               w3_UV = (-sg * l2 * a[0] + l1 * r[0]) / Th;
  M3[1][2] = w3_QU; M3[2][1] = -w3_QU; M3[1][3] = w3_QV; M3[3][1] = -w3_QV; M3[2][3] = w3_UV; M3[3][2] = -w3_UV;
  const double hh = 0.5 * (a2 + r2);
  const double cr[3] = {a[2] * r[1] - a[1] * r[2], a[0] * r[2] - a[2] * r[0], a[1] * r[0] - a[0] * r[1]};
  M4[0][0] = 2.0 * hh / Th;
  for (int i = 0; i < 3; ++i) {
    M4[0][i + 1] = 2.0 * cr[i] / Th;
    M4[i + 1][0] = -2.0 * cr[i] / Th;
    for (int j = 0; j < 3; ++j) M4[i + 1][j + 1] = 2.0 * (a[i] * a[j] + r[i] * r[j] - ((i == j) ? hh : 0.0)) / Th;
  }

  const double ex = std::exp(-aI * s);
  const double ch = std::cosh(L1 * s), sh = std::sinh(L1 * s), c = std::cos(L2 * s), sn = std::sin(L2 * s);
  // integrals of e^{-aI x} {cosh, sinh}(L1 x) and e^{-aI x} {cos, sin}(L2 x) over [0,s]
  const double Ep = exp_integral(aI - L1, s), Em = exp_integral(aI + L1, s);
  const double Ic1 = 0.5 * (Ep + Em), Is1 = 0.5 * (Ep - Em);
  double Ic2, Is2;
  const double den = aI * aI + L2 * L2;
  if (den == 0.0) { Ic2 = s; Is2 = 0.0; }
  else {
    // (1 - e^{-aI s} e^{i L2 s}) / (aI - i L2), numerator without cancellation
    const double em1 = std::expm1(-aI * s), hs = std::sin(0.5 * L2 * s);
    const double re = -(em1 * c - 2.0 * hs * hs);
    const double im = -ex * sn;
    Ic2 = (re * aI - im * L2) / den;
    Is2 = (re * L2 + im * aI) / den;
  }
  for (int i = 0; i < 4; ++i)
    for (int j = 0; j < 4; ++j) {
      const double id = (i == j) ? 1.0 : 0.0;
      O[i][j] = ex * (0.5 * (ch + c) * id - sn * M2[i][j] - sh * M3[i][j] + 0.5 * (ch - c) * M4[i][j]);
      P[i][j] = 0.5 * (Ic1 + Ic2) * id - Is2 * M2[i][j] - Is1 * M3[i][j] + 0.5 * (Ic1 - Ic2) * M4[i][j];
    }
}

}  // namespace iref

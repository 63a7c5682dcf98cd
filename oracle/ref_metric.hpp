// ORACLE (test infrastructure).  Kerr metric in modified Kerr-Schild (MKS) coordinates and its
// connection, written the slow generic way: analytic g_{mu nu} and its analytic first derivatives,
// NUMERIC 4x4 inverse, textbook Christoffel formula.
//
// Follows: BASELINE.json north_star stage (1) "null geodesic in the Kerr metric (modified
// Kerr-Schild coordinates)"; PAPER.md:35 (the paper prints no metric); reading DESIGN.md R-2 /
// SURVEY.md 8(c) c-2:
//   X = (t, X1, X2, X3),  r = exp(X1),  theta = pi X2 + (1-h)/2 sin(2 pi X2),  phi = X3
//   Kerr-Schild, Sigma = r^2 + a^2 cos^2(theta), f = 2 r / Sigma (f = 0 under flat_metric):
//   g_tt = -1+f, g_tr = f, g_tphi = -a f s^2, g_rr = 1+f, g_rphi = -a s^2 (1+f),
//   g_thth = Sigma, g_phph = s^2 [Sigma + a^2 s^2 (1+f)],   s = sin(theta)
//   MKS: g_{mu nu} = J_mu J_nu g^KS_{mu nu},  J = (1, r, dtheta/dX2, 1).
#pragma once
#include <cmath>
#include <cstring>

namespace iref {

struct Geom {
  double a;       // spin
  double hslope;  // h
  int flat;       // 1: f == 0 (Minkowski in the same coordinates)
};

inline double theta_of_x2(double h, double x2) { return M_PI * x2 + 0.5 * (1.0 - h) * std::sin(2.0 * M_PI * x2); }
inline double dtheta_dx2(double h, double x2) { return M_PI * (1.0 + (1.0 - h) * std::cos(2.0 * M_PI * x2)); }
inline double d2theta_dx2(double h, double x2) { return -2.0 * M_PI * M_PI * (1.0 - h) * std::sin(2.0 * M_PI * x2); }

inline double x2_of_theta(double h, double th) {
  double x2 = th / M_PI;
  for (int it = 0; it < 100; ++it) {
    double d = (theta_of_x2(h, x2) - th) / dtheta_dx2(h, x2);
    x2 -= d;
    if (std::fabs(d) < 1e-17) break;
  }
  return x2;
}

inline void sym_set(double m[4][4], int i, int j, double v) { m[i][j] = v; m[j][i] = v; }

// Kerr-Schild covariant metric in (t,r,theta,phi) and its r- and theta-derivatives.
inline void ks_metric(const Geom& G, double r, double th, double g[4][4], double gr[4][4], double gt[4][4]) {
  std::memset(g, 0, 16 * sizeof(double));
  std::memset(gr, 0, 16 * sizeof(double));
  std::memset(gt, 0, 16 * sizeof(double));
  const double a = G.a;
  const double s = std::sin(th), c = std::cos(th);
  const double s2 = s * s;
  const double ds2 = 2.0 * s * c;  // d(s^2)/dtheta
  const double Sig = r * r + a * a * c * c;
  const double Sig_r = 2.0 * r;
  const double Sig_t = -2.0 * a * a * s * c;
  double f = 2.0 * r / Sig;
  double f_r = 2.0 / Sig - 2.0 * r * Sig_r / (Sig * Sig);
  double f_t = -2.0 * r * Sig_t / (Sig * Sig);
  if (G.flat) { f = 0.0; f_r = 0.0; f_t = 0.0; }

  sym_set(g, 0, 0, -1.0 + f);
  sym_set(g, 0, 1, f);
  sym_set(g, 0, 3, -a * f * s2);
  sym_set(g, 1, 1, 1.0 + f);
  sym_set(g, 1, 3, -a * s2 * (1.0 + f));
  sym_set(g, 2, 2, Sig);
  const double W = Sig + a * a * s2 * (1.0 + f);
  sym_set(g, 3, 3, s2 * W);

  sym_set(gr, 0, 0, f_r);
  sym_set(gr, 0, 1, f_r);
  sym_set(gr, 0, 3, -a * f_r * s2);
  sym_set(gr, 1, 1, f_r);
  sym_set(gr, 1, 3, -a * s2 * f_r);
  sym_set(gr, 2, 2, Sig_r);
  const double W_r = Sig_r + a * a * s2 * f_r;
  sym_set(gr, 3, 3, s2 * W_r);

  sym_set(gt, 0, 0, f_t);
  sym_set(gt, 0, 1, f_t);
  sym_set(gt, 0, 3, -a * (f_t * s2 + f * ds2));
  sym_set(gt, 1, 1, f_t);
  sym_set(gt, 1, 3, -a * (ds2 * (1.0 + f) + s2 * f_t));
  sym_set(gt, 2, 2, Sig_t);
  const double W_t = Sig_t + a * a * (ds2 * (1.0 + f) + s2 * f_t);
  sym_set(gt, 3, 3, ds2 * W + s2 * W_t);
}

// g_{mu nu}(X) in MKS and dg[k][m][n] = d g_{mn} / d X^k  (k = 0,3 vanish: stationary, axisymmetric)
inline void gcov_and_derivs(const Geom& G, const double X[4], double g[4][4], double dg[4][4][4]) {
  const double r = std::exp(X[1]);
  const double th = theta_of_x2(G.hslope, X[2]);
  const double tp = dtheta_dx2(G.hslope, X[2]);
  const double tpp = d2theta_dx2(G.hslope, X[2]);
  double k[4][4], kr[4][4], kt[4][4];
  ks_metric(G, r, th, k, kr, kt);
  const double J[4] = {1.0, r, tp, 1.0};
  const double dJ1[4] = {0.0, r, 0.0, 0.0};    // dJ/dX1   (dr/dX1 = r)
  const double dJ2[4] = {0.0, 0.0, tpp, 0.0};  // dJ/dX2
  std::memset(dg, 0, 64 * sizeof(double));
  for (int m = 0; m < 4; ++m)
    for (int n = 0; n < 4; ++n) {
      g[m][n] = J[m] * J[n] * k[m][n];
      // chain rule: d/dX1 = r d/dr, d/dX2 = theta' d/dtheta
      dg[1][m][n] = (dJ1[m] * J[n] + J[m] * dJ1[n]) * k[m][n] + J[m] * J[n] * r * kr[m][n];
      dg[2][m][n] = (dJ2[m] * J[n] + J[m] * dJ2[n]) * k[m][n] + J[m] * J[n] * tp * kt[m][n];
    }
}

inline void gcov(const Geom& G, const double X[4], double g[4][4]) {
  double dg[4][4][4];
  gcov_and_derivs(G, X, g, dg);
}

// Gauss-Jordan inverse with partial pivoting; returns determinant of A.
inline double invert4(const double A[4][4], double Ai[4][4]) {
  double M[4][8];
  for (int i = 0; i < 4; ++i)
    for (int j = 0; j < 4; ++j) { M[i][j] = A[i][j]; M[i][4 + j] = (i == j) ? 1.0 : 0.0; }
  double det = 1.0;
  for (int c = 0; c < 4; ++c) {
    int p = c;
    for (int i = c + 1; i < 4; ++i) if (std::fabs(M[i][c]) > std::fabs(M[p][c])) p = i;
    if (p != c) { for (int j = 0; j < 8; ++j) { double t = M[c][j]; M[c][j] = M[p][j]; M[p][j] = t; } det = -det; }
    const double piv = M[c][c];
    det *= piv;
    for (int j = 0; j < 8; ++j) M[c][j] /= piv;
    for (int i = 0; i < 4; ++i) if (i != c) {
      const double fct = M[i][c];
      if (fct != 0.0) for (int j = 0; j < 8; ++j) M[i][j] -= fct * M[c][j];
    }
  }
  for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) Ai[i][j] = M[i][4 + j];
  return det;
}

inline void gcon(const Geom& G, const double X[4], double gi[4][4]) {
  double g[4][4];
  gcov(G, X, g);
  invert4(g, gi);
}

inline double sqrt_minus_g(const double g[4][4]) {
  double gi[4][4];
  return std::sqrt(std::fabs(invert4(g, gi)));
}

// Gamma^l_{mn} = 1/2 g^{lk} (d_m g_{kn} + d_n g_{km} - d_k g_{mn})
inline void connection(const Geom& G, const double X[4], double Gam[4][4][4]) {
  double g[4][4], dg[4][4][4], gi[4][4];
  gcov_and_derivs(G, X, g, dg);
  invert4(g, gi);
  double low[4][4][4];
  for (int k = 0; k < 4; ++k)
    for (int m = 0; m < 4; ++m)
      for (int n = 0; n < 4; ++n) low[k][m][n] = 0.5 * (dg[m][k][n] + dg[n][k][m] - dg[k][m][n]);
  for (int l = 0; l < 4; ++l)
    for (int m = 0; m < 4; ++m)
      for (int n = 0; n < 4; ++n) {
        double s = 0.0;
        for (int k = 0; k < 4; ++k) s += gi[l][k] * low[k][m][n];
        Gam[l][m][n] = s;
      }
}

inline double dot(const double g[4][4], const double u[4], const double v[4]) {
  double s = 0.0;
  for (int m = 0; m < 4; ++m) for (int n = 0; n < 4; ++n) s += g[m][n] * u[m] * v[n];
  return s;
}
inline void lower(const double g[4][4], const double u[4], double ul[4]) {
  for (int m = 0; m < 4; ++m) { double s = 0.0; for (int n = 0; n < 4; ++n) s += g[m][n] * u[n]; ul[m] = s; }
}

inline double horizon_radius(double a) { return 1.0 + std::sqrt(1.0 - a * a); }

// Bardeen, Press & Teukolsky (1972) prograde ISCO radius.
inline double isco_radius(double a) {
  const double z1 = 1.0 + std::cbrt(1.0 - a * a) * (std::cbrt(1.0 + a) + std::cbrt(1.0 - a));
  const double z2 = std::sqrt(3.0 * a * a + z1 * z1);
  return 3.0 + z2 - std::sqrt((3.0 - z1) * (3.0 + z1 + 2.0 * z2));
}

}  // namespace iref

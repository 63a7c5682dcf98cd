// ORACLE (test infrastructure).  Polarized transfer of the complex coherency tensor N^{mu nu} along a
// stored geodesic, toward the observer.
//
// "Once the geodesic integration is over and saved the covariant fully polarized
// radiative-transfer equations are integrated along the geodesic toward the observer ... at every
// single step ... evaluate emission, self-absorption and Faraday coefficients".
// "In ipole the polarization state of light is described in a coordinate frame using
// a coherency matrix N^{alpha beta}, which is a complex quantity".
// The discretisation is not in the paper; reading DESIGN.md R-6.  For the step
// from point s+1 to point s (forward d lambda_s > 0):
//   Xm = (X_s + X_{s+1})/2, Km = (K_s + K_{s+1})/2, A^a_n = Gamma^a_{mn}(Xm) Km^m, h = dl_s/2,
//   P = 1 - h A + h^2 A^2 / 2 (real);  N <- P N P^T;  plasma operator at (Xm, Km) over the whole
//   d l = dl_s L / nu_obs;  N <- P N P^T.
// Plasma operator: omega = -Km.u, nu = omega nu_obs; tetrad e0 = u, e3 = (Km/omega - u) normalised,
//   e2 = b - (b.e3) e3 normalised, e1^mu = [mu a b c] u_a e2_b e3_c / sqrt(-g) ([0123] = +1);
//   N^(a)(b) = e^(a)_mu e^(b)_nu N^{mu nu};  I = N11 + N22, Q = N11 - N22, U = N12 + N21,
//   V = i (N12 - N21);  S <- O S + P J with invariant coefficients j/nu^2, alpha nu, rho nu;
//   N11 = (I+Q)/2, N22 = (I-Q)/2, N12 = (U - iV)/2, N21 = (U + iV)/2, every other tetrad component 0;
//   N^{mu nu} = e_(a)^mu e_(b)^nu N^(a)(b).
#pragma once
#include <complex>
#include "ref_metric.hpp"
#include "ref_geodesic.hpp"
#include "ref_plasma.hpp"
#include "ref_coeff.hpp"
#include "ref_edf.hpp"
#include "ref_stokes_op.hpp"

namespace iref {

typedef std::complex<double> cplx;

struct Model {
  int kind = MODEL_NONE;
  EdfParams edf;       // kind 0: thermal fits; otherwise j, alpha integrated over the eDF (ref_edf.hpp)
  AdafParams adaf;
  SlabParams slab;
  GridParams grid;
};

struct Units {
  double nu_obs;  // Hz
  double L_unit;  // G M / c^2 in cm
  double D_cm;    // distance to the source
};

inline void plasma_at(const Geom& G, const Model& M, const Units& U, const double X[4], Plasma& p) {
  p = Plasma();
  if (M.kind == MODEL_ADAF) plasma_adaf(G, M.adaf, X, p);
  else if (M.kind == MODEL_SLAB) plasma_slab(G, M.slab, X, p);
  else if (M.kind == MODEL_GRID) plasma_grid(G, M.grid, U.L_unit, X, p);
}

// P = 1 - h A + h^2 A^2 / 2 with A^a_n = Gamma^a_{mn}(X) K^m
inline void transport_matrix(const Geom& G, const double X[4], const double K[4], double h, double P[4][4]) {
  double Gam[4][4][4], A[4][4], A2[4][4];
  connection(G, X, Gam);
  for (int a = 0; a < 4; ++a)
    for (int n = 0; n < 4; ++n) {
      double s = 0.0;
      for (int m = 0; m < 4; ++m) s += Gam[a][m][n] * K[m];
      A[a][n] = s;
    }
  for (int a = 0; a < 4; ++a)
    for (int n = 0; n < 4; ++n) {
      double s = 0.0;
      for (int m = 0; m < 4; ++m) s += A[a][m] * A[m][n];
      A2[a][n] = s;
    }
  for (int a = 0; a < 4; ++a)
    for (int n = 0; n < 4; ++n) P[a][n] = ((a == n) ? 1.0 : 0.0) - h * A[a][n] + 0.5 * h * h * A2[a][n];
}

// N <- P N P^T
inline void congruence(const double P[4][4], cplx N[4][4]) {
  cplx T[4][4];
  for (int a = 0; a < 4; ++a)
    for (int n = 0; n < 4; ++n) {
      cplx s = 0.0;
      for (int m = 0; m < 4; ++m) s += P[a][m] * N[m][n];
      T[a][n] = s;
    }
  for (int a = 0; a < 4; ++a)
    for (int b = 0; b < 4; ++b) {
      cplx s = 0.0;
      for (int n = 0; n < 4; ++n) s += T[a][n] * P[b][n];
      N[a][b] = s;
    }
}

inline int levi_civita(int a, int b, int c, int d) {
  const int p[4] = {a, b, c, d};
  int s = 1;
  for (int i = 0; i < 4; ++i)
    for (int j = i + 1; j < 4; ++j) {
      if (p[i] == p[j]) return 0;
      if (p[i] > p[j]) s = -s;
    }
  return s;
}

// plasma tetrad; econ[a][mu] contravariant, ecov[a][mu] = e^(a)_mu (dual basis).  false if it cannot be built.
inline bool plasma_tetrad(const double g[4][4], const double K[4], const double u[4], const double b[4],
                          double econ[4][4], double ecov[4][4], double* omega_out) {
  double kcov[4], ucov[4];
  lower(g, K, kcov);
  lower(g, u, ucov);
  double om = 0.0;
  for (int m = 0; m < 4; ++m) om -= kcov[m] * u[m];
  *omega_out = om;
  if (!(om > 0.0)) return false;
  double e3[4], e2[4];
  for (int m = 0; m < 4; ++m) e3[m] = K[m] / om - u[m];
  const double n3 = dot(g, e3, e3);
  if (!(n3 > 0.0)) return false;
  for (int m = 0; m < 4; ++m) e3[m] /= std::sqrt(n3);
  const double be3 = dot(g, b, e3);
  for (int m = 0; m < 4; ++m) e2[m] = b[m] - be3 * e3[m];
  const double n2 = dot(g, e2, e2);
  if (!(n2 > 0.0)) return false;
  for (int m = 0; m < 4; ++m) e2[m] /= std::sqrt(n2);
  double e2c[4], e3c[4];
  lower(g, e2, e2c);
  lower(g, e3, e3c);
  const double sg = sqrt_minus_g(g);
  for (int m = 0; m < 4; ++m) {
    double s = 0.0;
    for (int a = 0; a < 4; ++a) for (int bb = 0; bb < 4; ++bb) for (int c = 0; c < 4; ++c) {
      const int lc = levi_civita(m, a, bb, c);
      if (lc) s += lc * ucov[a] * e2c[bb] * e3c[c];
    }
    econ[1][m] = s / sg;
    econ[0][m] = u[m]; econ[2][m] = e2[m]; econ[3][m] = e3[m];
  }
  for (int a = 0; a < 4; ++a) {
    lower(g, econ[a], ecov[a]);
    if (a == 0) for (int m = 0; m < 4; ++m) ecov[0][m] = -ecov[0][m];
  }
  return true;
}

inline void project_to_stokes(const double ecov[4][4], const cplx N[4][4], double S[4]) {
  cplx T[3][3];
  for (int a = 1; a <= 2; ++a)
    for (int b = 1; b <= 2; ++b) {
      cplx s = 0.0;
      for (int m = 0; m < 4; ++m) for (int n = 0; n < 4; ++n) s += ecov[a][m] * ecov[b][n] * N[m][n];
      T[a][b] = s;
    }
  S[0] = (T[1][1] + T[2][2]).real();
  S[1] = (T[1][1] - T[2][2]).real();
  S[2] = (T[1][2] + T[2][1]).real();
  S[3] = (cplx(0.0, 1.0) * (T[1][2] - T[2][1])).real();
}

inline void stokes_to_tensor(const double econ[4][4], const double S[4], cplx N[4][4]) {
  cplx T[4][4];
  for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) T[a][b] = 0.0;
  T[1][1] = 0.5 * (S[0] + S[1]);
  T[2][2] = 0.5 * (S[0] - S[1]);
  T[1][2] = 0.5 * cplx(S[2], -S[3]);
  T[2][1] = 0.5 * cplx(S[2], S[3]);
  for (int m = 0; m < 4; ++m)
    for (int n = 0; n < 4; ++n) {
      cplx s = 0.0;
      for (int a = 1; a <= 2; ++a) for (int b = 1; b <= 2; ++b) s += econ[a][m] * econ[b][n] * T[a][b];
      N[m][n] = s;
    }
}

// One application of the plasma operator at (X, K) over affine length dl (>0).  Returns true if applied.
inline bool plasma_operator(const Geom& G, const Model& M, const Units& U, const double X[4], const double K[4],
                            double dl, cplx N[4][4], double* tau, double* tauF) {
  Plasma p;
  plasma_at(G, M, U, X, p);
  if (!p.present) return false;
  double g[4][4], econ[4][4], ecov[4][4], om;
  gcov(G, X, g);
  if (!plasma_tetrad(g, K, p.u, p.b, econ, ecov, &om)) return false;
  const double nu = om * U.nu_obs;
  double jc[4], ac[4], rc[3];  // cgs coefficients in the plasma frame at nu
  if (p.direct) {
    for (int i = 0; i < 4; ++i) { jc[i] = p.j[i]; ac[i] = p.al[i]; }
    for (int i = 0; i < 3; ++i) rc[i] = p.rh[i];
  } else {
    double bcov[4];
    lower(g, p.b, bcov);
    double bk = 0.0;
    for (int m = 0; m < 4; ++m) bk += bcov[m] * K[m];
    double cosT = bk / (om * p.B);
    if (cosT > 1.0) cosT = 1.0;
    if (cosT < -1.0) cosT = -1.0;
    const CoeffCGS c = synchrotron_coefficients_edf(M.edf, p.ne, p.Th, p.B, cosT, nu);
    jc[0] = c.jI; jc[1] = c.jQ; jc[2] = 0.0; jc[3] = c.jV;
    ac[0] = c.aI; ac[1] = c.aQ; ac[2] = 0.0; ac[3] = c.aV;
    rc[0] = c.rQ; rc[1] = 0.0; rc[2] = c.rV;
  }
  // invariant forms: j/nu^2, alpha nu, rho nu; path element dl L / nu_obs
  double ji[4], ai[4], ri[3];
  for (int i = 0; i < 4; ++i) { ji[i] = jc[i] / (nu * nu); ai[i] = ac[i] * nu; }
  for (int i = 0; i < 3; ++i) ri[i] = rc[i] * nu;
  const double ds = dl * U.L_unit / U.nu_obs;
  double O[4][4], Pm[4][4], S[4], S1[4];
  stokes_operator(ai, ri, ds, O, Pm);
  project_to_stokes(ecov, N, S);
  for (int i = 0; i < 4; ++i) {
    double s = 0.0;
    for (int k = 0; k < 4; ++k) s += O[i][k] * S[k] + Pm[i][k] * ji[k];
    S1[i] = s;
  }
  stokes_to_tensor(econ, S1, N);
  if (tau) *tau += ai[0] * ds;
  if (tauF) *tauF += std::fabs(ri[2]) * ds;
  return true;
}

// Walk the stored path from its far end (point n) to the camera (point 0).
inline void transfer_along_path(const Geom& G, const Model& M, const Units& U, const Path& path, cplx N[4][4],
                                double* tau, double* tauF) {
  const int n = (int)path.dl.size();
  for (int s = n - 1; s >= 0; --s) {
    double Xm[4], Km[4], P[4][4];
    for (int m = 0; m < 4; ++m) {
      Xm[m] = 0.5 * (path.X[s][m] + path.X[s + 1][m]);
      Km[m] = 0.5 * (path.K[s][m] + path.K[s + 1][m]);
    }
    transport_matrix(G, Xm, Km, 0.5 * path.dl[s], P);
    congruence(P, N);
    plasma_operator(G, M, U, Xm, Km, path.dl[s], N, tau, tauF);
    congruence(P, N);
  }
}

// Stokes (invariant I/nu^3 units) seen by the camera tetrad e[a][mu] at Xcam
inline void camera_stokes(const Geom& G, const Camera& C, const cplx N[4][4], double S[4]) {
  double g[4][4], ecov[4][4];
  gcov(G, C.Xcam, g);
  for (int a = 0; a < 4; ++a) {
    lower(g, C.e[a], ecov[a]);
    if (a == 0) for (int m = 0; m < 4; ++m) ecov[0][m] = -ecov[0][m];
  }
  project_to_stokes(ecov, N, S);
}

}  // namespace iref
